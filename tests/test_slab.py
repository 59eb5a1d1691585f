"""z-slab decomposition.

GPU: all ranks of a ring emulated one after another on one GPU must reproduce the undivided
lattice bit for bit (same kernels, same arithmetic per cell).  CPU: the ring exchange and the
statistics reduction over torch.distributed with gloo, world sizes 2 and 3."""
import os
import socket
import sys

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


# ---------------------------------------------------------------------------------------------
# CPU: ring exchange over gloo
# ---------------------------------------------------------------------------------------------
def _ring_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_2206_15454_b200.slab import ring_exchange, ring_neighbours

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    hi = torch.full((5, 3, 4), rank * 10.0 + 1.0)
    lo = torch.full((5, 3, 4), rank * 10.0 + 2.0)
    from_lower, from_upper = torch.zeros(5, 3, 4), torch.zeros(5, 3, 4)
    for _ in range(3):                                   # repeated exchanges stay paired
        ring_exchange(hi, lo, from_lower, from_upper, rank, world)
    lower, upper = ring_neighbours(rank, world)
    ok = bool((from_lower == lower * 10.0 + 1.0).all() and (from_upper == upper * 10.0 + 2.0).all())
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t)
    q.put((rank, ok, float(t)))
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_ring_exchange_gloo(world):
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_ring_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=180) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in got)
    assert all(s == world * (world + 1) / 2 for _, _, s in got)


def test_ring_exchange_single_rank_is_self_periodic():
    import torch
    from paper_2206_15454_b200.slab import ring_exchange, ring_neighbours

    hi, lo = torch.ones(2, 2), 2 * torch.ones(2, 2)
    a, b = torch.zeros(2, 2), torch.zeros(2, 2)
    ring_exchange(hi, lo, a, b, 0, 1)
    assert (a == 1).all() and (b == 2).all()
    assert ring_neighbours(0, 4) == (3, 1) and ring_neighbours(3, 4) == (2, 0)


# ---------------------------------------------------------------------------------------------
# GPU: emulated ring == undivided lattice
# ---------------------------------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("storage", ["two_lattice", "aa", "aax"])
@pytest.mark.parametrize("world", [1, 2, 3, 4])
@pytest.mark.parametrize("case", ["forest", "lid+solid", "slip+solid", "periodic"])
def test_emulated_slabs_equal_global_lattice(world, case, storage):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    from paper_2206_15454_b200 import slab

    cfg = wl.small(nx=32, ny=10, nz=12)
    if case == "periodic":
        cfg = wl.small(nx=32, ny=10, nz=12, bottom=wl.PERIODIC, top=wl.PERIODIC)
    if "solid" in case:
        if case == "lid+solid":
            cfg = wl.small(nx=32, ny=10, nz=12, top=wl.FORCED_EQ)
            cfg["U_top"] = (0.06, 0.0, 0.01)
        m = np.zeros((12, 10, 32), bool)
        m[0:2, 0:3, 4:9] = True                          # a box that straddles the z wrap ...
        m[11, 0:3, 4:9] = True
        m[5:7, 2:5, 30:] = True                          # ... and one across a slab face and the x wrap
        m[5:7, 2:5, :2] = True
        m[2:4, 7:10, 12:15] = True                       # ... and one under the top face, across a slab face
        cfg["solid"] = m
    aa = {"two_lattice": False, "aa": True, "aax": "aax"}[storage]
    vec = 4 if world % 2 == 0 else 0        # 4 cells per thread and the small-lattice default (1)
    ref = lb.Lbm.from_config(cfg, aa=aa, vec=vec)
    ref.init(cfg["seed"])
    ref.stats_accumulate(1)
    ref.stats_reset()
    slabs = [slab.SlabLbm(cfg, r, world, emulated=True, storage=storage, vec=vec) for r in range(world)]
    slab.init_emulated(slabs, cfg["seed"])
    for s in slabs:
        s.stats_accumulate(1)
        s.stats_reset()
    for n in (1, 2, 6):
        ref.step(n)
        slab.step_emulated(slabs, n)
        rr, ur = ref.get_macros()
        rs = torch.cat([s.get_macros()[0] for s in slabs], dim=0)
        us = torch.cat([s.get_macros()[1] for s in slabs], dim=1)
        if "solid" not in case:
            assert torch.equal(rs, rr) and torch.equal(us, ur), (world, n)
        else:
            # geometry handles run the plain or the geometry body per thread block (two
            # instantiations of the same arithmetic: ptxas contracts their FMAs differently when the
            # statistics are fused in), so a different block decomposition may round a cell
            # differently: equal to a few ulp, not bit for bit
            assert float((rs - rr).abs().max()) <= 2e-7 and float((us - ur).abs().max()) <= 5e-8, (world, n)
    sr, nr = ref.stats_read()
    ss = slab.stats_emulated(slabs)
    assert nr == 9
    # the undivided run centres its fp32 row sums, the slabs do not: equal to fp32 summation noise
    assert np.abs(ss[:, 0:3] - sr[:, 0:3]).max() <= 1e-6 * cfg["u_bulk"]
    assert np.abs(ss[:, 3:9] - sr[:, 3:9]).max() <= 1e-6 * cfg["u_bulk"] ** 2
    assert np.abs(ss[:, 9] - sr[:, 9]).max() <= 1e-7
    for s in slabs:
        s.close()


@pytest.mark.gpu
def test_single_slab_through_torch_distributed_path():
    """world == 1 through SlabLbm.step itself (self-periodic exchange) == undivided lattice."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    from paper_2206_15454_b200 import slab

    cfg = wl.small(nx=64, ny=8, nz=6)
    ref = lb.Lbm.from_config(cfg, aa=False)
    ref.init(3)
    s = slab.SlabLbm(cfg, 0, 1)
    s.init(3)
    s.stats_accumulate(2)
    ref.stats_accumulate(2)              # the same kernel instantiations on both sides (bit identity)
    ref.step(5)
    s.step(5)
    assert torch.equal(s.get_macros()[1], ref.get_macros()[1])
    st = s.stats_read()
    assert np.isfinite(st).all() and abs(st[:, 9].mean() - 1.0) < 1e-6


@pytest.mark.gpu
def test_halo_flag_rules():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    with pytest.raises(lb.LbmError):
        lb.Lbm(32, 4, 2, 0.01, 0.1, flags=lb.bc_flags("bounce_back", "free_slip", halo=True))
    g = lb.Lbm(32, 4, 6, 0.01, 0.1, flags=lb.bc_flags("bounce_back", "free_slip"))
    with pytest.raises(lb.LbmError):
        g.set_z_slab(0, 4)


@pytest.mark.gpu
@pytest.mark.parametrize("storage", ["two_lattice", "aa"])
@pytest.mark.parametrize("world", [1, 2, 3])
def test_overlapped_slabs_equal_the_lattice_and_the_oracle(orc, world, storage):
    """The begin / exchange-on-a-second-stream / end form (lbm_step_slab_begin/_end): re-assembled
    slab fields against the ORACLE over 20 steps at the north_star tolerance, and to a few ulp
    against the undivided CUDA lattice (a geometry handle: see the note in the test above; without
    geometry the slabs are bit-identical, test_single_slab_overlapped_through_the_comm_stream)."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    from paper_2206_15454_b200 import slab

    cfg = wl.small(nx=64, ny=10, nz=12)
    m = np.zeros((12, 10, 64), bool)
    m[3:5, 0:3, 10:14] = True                            # a trip box across the face between slabs
    cfg["solid"] = m
    o = orc.Oracle.from_config(cfg)
    o.init_from_config(cfg)
    ref = lb.Lbm.from_config(cfg, aa=(storage == "aa"))
    ref.init(cfg["seed"])
    slabs = [slab.SlabLbm(cfg, r, world, emulated=True, storage=storage) for r in range(world)]
    slab.init_emulated(slabs, cfg["seed"])
    for s in slabs:
        s.stats_accumulate(1)
    o.stats_accumulate(1)
    tol = 1e-5 * cfg["u_bulk"]
    for n in (1, 2, 7, 10):
        o.step(n)
        ref.step(n)
        slab.step_emulated(slabs, n, overlap=True)
        torch.cuda.synchronize()
        rs = torch.cat([s.get_macros()[0] for s in slabs], dim=0)
        us = torch.cat([s.get_macros()[1] for s in slabs], dim=1)
        rr, ur = ref.get_macros()
        assert float((rs - rr).abs().max()) <= 2e-7 and float((us - ur).abs().max()) <= 5e-8, (world, n)
        ro, uo = o.get_macros()
        assert np.abs(rs.cpu().numpy() - ro).max() <= tol and np.abs(us.cpu().numpy() - uo).max() <= tol
    so, no = o.stats_read()
    ss = slab.stats_emulated(slabs)
    assert no == 20
    assert np.abs(ss[:, 0:3] - so[:, 0:3]).max() <= tol
    assert np.abs(ss[:, 3:9] - so[:, 3:9]).max() <= tol * cfg["u_bulk"]
    assert np.abs(ss[:, 9] - so[:, 9]).max() <= 1e-6
    # begin twice / end without begin are refused
    with pytest.raises(lb.LbmError):
        slabs[0].sim.step_slab_end(slabs[0]._recv[0], slabs[0]._recv[1])
    slabs[0].sim.step_slab_begin(slabs[0]._send[0], slabs[0]._send[1])
    with pytest.raises(lb.LbmError):
        slabs[0].sim.step_slab_begin(slabs[0]._send[0], slabs[0]._send[1])
    for s in slabs:
        s.close()


@pytest.mark.gpu
@pytest.mark.parametrize("storage", ["two_lattice", "aa", "aax"])
def test_single_slab_overlapped_through_the_comm_stream(storage):
    """world == 1 through SlabLbm.step(overlap=True): the exchange (self-periodic copies) runs on
    the second stream between begin and end."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    from paper_2206_15454_b200 import slab

    cfg = wl.small(nx=64, ny=8, nz=6)
    ref = lb.Lbm.from_config(cfg, aa={"two_lattice": False, "aa": True, "aax": "aax"}[storage])
    ref.init(3)
    a = slab.SlabLbm(cfg, 0, 1, storage=storage)
    b = slab.SlabLbm(cfg, 0, 1, storage=storage)
    a.init(3)
    b.init(3)
    ref.step(9)
    a.step(9, overlap=True)
    b.step(9, overlap=False)
    torch.cuda.synchronize()
    assert torch.equal(a.get_macros()[1], ref.get_macros()[1])
    assert torch.equal(b.get_macros()[1], ref.get_macros()[1])


@pytest.mark.gpu
@pytest.mark.parametrize("storage", ["two_lattice", "aa", "aax"])
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("t_change", [4, 5])
def test_solid_removed_at_run_time_on_slabs(world, storage, t_change):
    """PAPER.md:L226 on a cut lattice: boxes across slab faces are removed (and others put in) on
    running slabs at an even and at an odd time step; the ring must go on like the undivided lattice.
    In the single-array storages at even t the populations between a changed cell and a neighbour
    across a face are converted in the ghost planes and travel with the repeated exchange."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    from paper_2206_15454_b200 import slab

    cfg = wl.small(nx=32, ny=10, nz=12)
    m = np.zeros((12, 10, 32), bool)
    m[0:2, 0:3, 4:9] = True                          # straddles the z wrap ...
    m[11, 0:3, 4:9] = True
    m[3:9, 2:5, 30:] = True                          # ... crosses the slab faces of 2 and 3 slabs and the x wrap
    m[3:9, 2:5, :2] = True
    cfg["solid"] = m
    moved = np.zeros_like(m)
    moved[5:10, 4:8, 10:14] = True                   # new solids across other faces, the old ones gone
    moved[0, 0:2, 20:24] = True
    aa = {"two_lattice": False, "aa": True, "aax": "aax"}[storage]
    ref = lb.Lbm.from_config(cfg, aa=aa, vec=4)
    ref.init(cfg["seed"])
    slabs = [slab.SlabLbm(cfg, r, world, emulated=True, storage=storage, vec=4) for r in range(world)]
    slab.init_emulated(slabs, cfg["seed"])
    ref.step(t_change)
    slab.step_emulated(slabs, t_change)
    part = m.copy()
    part[3:9, 2:5, 30:] = False
    for mask, n in ((part, 3), (None, 2), (moved, 3), (None, 6)):
        ref.set_solid(mask)
        slab.set_solid_emulated(slabs, mask)
        for k in range(n):
            ref.step(1)
            slab.step_emulated(slabs, 1, overlap=bool(k & 1))
            rr, ur = ref.get_macros()
            rs = torch.cat([s.get_macros()[0] for s in slabs], dim=0)
            us = torch.cat([s.get_macros()[1] for s in slabs], dim=1)
            assert float((rs - rr).abs().max()) <= 2e-7 and float((us - ur).abs().max()) <= 5e-8, (mask is None, k)
    for s in slabs:
        s.close()
    ref.close()
