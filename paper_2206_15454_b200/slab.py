"""z-slab decomposition of one lattice over several GPUs.

Plumbing only: every population that moves is packed, unpacked and updated by the CUDA library
(lbm_step_slab_begin / lbm_step_slab_end); this module decides WHO talks to WHOM and hands the
packed device buffers to torch.distributed (NCCL point-to-point over NVLink) - one exchange of
2 x 5 x nx x ny fp32 per time step ("only information from directly adjacent points is
required") - and sums the [ny][10] raw statistics over the ranks at read-out.

A step is split so that the exchange hides behind the interior update: the library updates the
two boundary planes first, packs the faces and records an event; the exchange runs on a second
CUDA stream that waits for that event while the library's stream updates the interior planes;
the unpack waits for the exchange (lbm.h: lbm_step_slab_begin / _end).

Rank r of W owns the global planes [r nz/W, (r+1) nz/W) plus one ghost plane on either side; z is
periodic, so the ranks form a ring.  Any storage scheme: two-lattice (default), or the single-array
AA / x-balanced AA patterns at half the memory (the in-place odd step pushes into the ghost planes;
the library moves those planes to the neighbour's boundary plane instead - the calls are the
same).  north_star runs on one GPU: this is the path the lattice would take beyond one GPU's
180 GB, verified by emulating the ranks one after another on one GPU (bit-identical to the
undivided lattice) and by gloo ring tests on the CPU.
"""
from __future__ import annotations

import numpy as np

from .binding import Lbm, stats_from_raw


def ring_neighbours(rank: int, world: int):
    """(lower, upper) ranks of a periodic ring."""
    return (rank - 1) % world, (rank + 1) % world


def ring_exchange(hi_send, lo_send, from_lower, from_upper, rank: int, world: int, group=None):
    """Send `hi_send` to the upper and `lo_send` to the lower neighbour; receive the lower
    neighbour's hi into `from_lower` and the upper neighbour's lo into `from_upper`.

    The posting order (hi before lo on the sending side, lower before upper on the receiving
    side) makes the pairing right for world == 2 as well, where both neighbours are the same
    peer and the transport matches messages in order.  world == 1: plain copies."""
    if world == 1:
        from_lower.copy_(hi_send)
        from_upper.copy_(lo_send)
        return
    import torch.distributed as dist

    lower, upper = ring_neighbours(rank, world)
    ops = [dist.P2POp(dist.isend, hi_send, upper, group), dist.P2POp(dist.isend, lo_send, lower, group),
           dist.P2POp(dist.irecv, from_lower, lower, group), dist.P2POp(dist.irecv, from_upper, upper, group)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()


class SlabLbm:
    """One rank's slab.  `cfg` describes the GLOBAL lattice; `exchange` = None uses
    torch.distributed's default group (world == 1: the slab is its own neighbour)."""

    def __init__(self, cfg: dict, rank: int = 0, world: int = 1, device="cuda:0", group=None,
                 emulated: bool = False, storage: str = "two_lattice", vec: int = 0):
        if cfg["nz"] % world:
            raise ValueError(f"nz={cfg['nz']} is not a multiple of the number of slabs {world}")
        self.rank, self.world, self.group = int(rank), int(world), group
        self.emulated = bool(emulated)      # the caller drives the exchange (exchange_emulated)
        self._inited = False                # a state exists (init / set_macros): halo calls are allowed
        self.nz_global = cfg["nz"]
        self.nz_local = cfg["nz"] // world
        self.z_first = self.rank * self.nz_local
        local = dict(cfg)
        local["nz"] = self.nz_local + 2
        if cfg.get("solid") is not None:                        # local planes incl. the two ghosts
            z = np.arange(self.z_first - 1, self.z_first + self.nz_local + 1) % self.nz_global
            local["solid"] = np.asarray(cfg["solid"])[z]
        if storage not in ("two_lattice", "aa", "aax"):
            raise ValueError(f"unknown storage scheme {storage!r}")
        aa = {"two_lattice": False, "aa": True, "aax": "aax"}[storage]
        self.sim = Lbm.from_config(local, aa=aa, vec=vec, halo=True, device=device)
        self.sim.set_z_slab(self.z_first, self.nz_global)
        self.cfg = cfg
        self._send = [self.sim.halo_buffer(), self.sim.halo_buffer()]    # [lo, hi]
        self._recv = [self.sim.halo_buffer(), self.sim.halo_buffer()]    # [from lower, from upper]
        import torch

        with torch.cuda.device(self.sim.device):
            self._comm = torch.cuda.Stream(self.sim.device)              # the exchange runs here
            self._packed = torch.cuda.Event()
            self._ready = torch.cuda.Event()
            # torch creates the CUDA event at the first record(): make the handles real now, they
            # are handed to the library as raw cudaEvent_t
            self._packed.record()
            self._ready.record()

    # -- halo exchange -----------------------------------------------------------------------
    def pack(self):
        self.sim.halo_pack(0, self._send[0])
        self.sim.halo_pack(1, self._send[1])

    def unpack(self):
        self.sim.halo_unpack(0, self._recv[0])     # low ghost plane <- lower neighbour's high face
        self.sim.halo_unpack(1, self._recv[1])     # high ghost plane <- upper neighbour's low face

    def exchange(self):
        if self.emulated:
            return
        self.pack()
        ring_exchange(self._send[1], self._send[0], self._recv[0], self._recv[1], self.rank, self.world,
                      self.group)
        self.unpack()

    # -- the Lbm calls, slab-aware -----------------------------------------------------------
    def init(self, seed: int):
        self.sim.init(seed)
        self._inited = True
        self.exchange()

    def set_macros(self, rho_local, u_local):
        """Fields of the local planes INCLUDING the two ghost planes (nz_local + 2)."""
        self.sim.set_macros(rho_local, u_local)
        self._inited = True
        self.exchange()

    def _local_mask(self, solid_global):
        """The slab's planes of a global [nz][ny][nx] mask, the two ghost planes included."""
        if solid_global is None:
            return None
        z = np.arange(self.z_first - 1, self.z_first + self.nz_local + 1) % self.nz_global
        return np.ascontiguousarray(np.asarray(solid_global)[z])

    def set_solid(self, solid_global):
        """Change the solid mask (GLOBAL [nz][ny][nx], None = no solid cell) on every rank at the same
        time step; on a running slab the flow is kept and the halo exchange is repeated
        (lbm.h: lbm_set_solid on a z slab)."""
        self.sim.set_solid(self._local_mask(solid_global))
        if self._inited:
            self.exchange()

    def stats_accumulate(self, every: int = 1):
        self.sim.stats_accumulate(every)

    def stats_reset(self):
        self.sim.stats_reset()

    def step(self, n: int = 1, overlap: bool = True):
        """n time steps.  overlap=True: boundary planes -> pack -> [exchange on the comm stream ||
        interior planes] -> unpack; overlap=False: the sequential form (same bits)."""
        if self.emulated:
            raise RuntimeError("emulated slabs are advanced together: step_emulated(slabs, n)")
        import torch

        for _ in range(int(n)):
            if not overlap:
                self.sim.step(1)
                self.exchange()
                continue
            self.sim.step_slab_begin(self._send[0], self._send[1], self._packed)
            with torch.cuda.stream(self._comm):
                self._comm.wait_event(self._packed)
                ring_exchange(self._send[1], self._send[0], self._recv[0], self._recv[1], self.rank,
                              self.world, self.group)
                self._ready.record(self._comm)
            self.sim.step_slab_end(self._recv[0], self._recv[1], self._ready)

    def get_macros(self):
        """(rho, u) of the interior planes: shapes (nz_local, ny, nx), (3, nz_local, ny, nx)."""
        rho, u = self.sim.get_macros()
        return rho[1:-1], u[:, 1:-1]

    def stats_raw(self):
        raw, centre, count = self.sim.stats_read_raw()
        assert not centre.any(), "a slab never uses an accumulation centre"
        return raw, count

    def stats_read(self):
        """Plane statistics of the GLOBAL lattice (same table on every rank)."""
        raw, count = self.stats_raw()
        if self.world > 1 and not self.emulated:
            import torch
            import torch.distributed as dist

            backend = dist.get_backend(self.group)
            dev = self.sim.device if backend == "nccl" else "cpu"
            t = torch.from_numpy(np.concatenate([raw.ravel(), [count]])).to(dev)
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            t = t.cpu().numpy()
            raw, count = t[:-1].reshape(raw.shape), float(t[-1])
        return stats_from_raw(raw, count)

    def close(self):
        self.sim.close()


def step_emulated(slabs, n: int = 1, overlap: bool = False):
    """Advance a list of slabs that live in ONE process (all ranks of a ring, e.g. on one GPU, one
    after another - no kernel waits on another): same calls, the exchange done by local copies.
    overlap=True drives the begin / exchange-on-a-second-stream / end form of SlabLbm.step."""
    import torch

    W = len(slabs)
    for _ in range(int(n)):
        if not overlap:
            for s in slabs:
                s.sim.step(1)
            exchange_emulated(slabs)
            continue
        for s in slabs:
            s.sim.step_slab_begin(s._send[0], s._send[1], s._packed)
        for r, s in enumerate(slabs):
            lower, upper = ring_neighbours(r, W)
            with torch.cuda.stream(s._comm):
                s._comm.wait_event(slabs[lower]._packed)
                s._comm.wait_event(slabs[upper]._packed)
                s._recv[0].copy_(slabs[lower]._send[1], non_blocking=True)
                s._recv[1].copy_(slabs[upper]._send[0], non_blocking=True)
                s._ready.record(s._comm)
        for s in slabs:
            s.sim.step_slab_end(s._recv[0], s._recv[1], s._ready)
        # the next begin overwrites the send buffers: it must not overtake this step's copies
        for s in slabs:
            lower, upper = ring_neighbours(slabs.index(s), W)
            torch.cuda.current_stream(s.sim.device).wait_event(slabs[lower]._ready)
            torch.cuda.current_stream(s.sim.device).wait_event(slabs[upper]._ready)


def init_emulated(slabs, seed: int):
    for s in slabs:
        s.init(seed)
    exchange_emulated(slabs)


def set_solid_emulated(slabs, solid_global):
    """SlabLbm.set_solid for a ring of emulated slabs: every slab changes its mask, then one exchange."""
    for s in slabs:
        s.sim.set_solid(s._local_mask(solid_global))
    if slabs[0]._inited:
        exchange_emulated(slabs)


def exchange_emulated(slabs):
    W = len(slabs)
    for s in slabs:
        s.pack()
    for r, s in enumerate(slabs):
        lower, upper = ring_neighbours(r, W)
        s._recv[0].copy_(slabs[lower]._send[1])
        s._recv[1].copy_(slabs[upper]._send[0])
    for s in slabs:
        s.unpack()


def stats_emulated(slabs):
    raws, counts = zip(*(s.stats_raw() for s in slabs))
    return stats_from_raw(np.sum(raws, axis=0), float(np.sum(counts)))
