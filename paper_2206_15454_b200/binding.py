"""Thin ctypes binding of the C ABI in include/lbm.h (argument marshalling only).

PyTorch is used for exactly two things: the device workspace (`torch.empty(..., device="cuda")`)
and the CUDA stream the kernels are launched on.  Every step of the method runs in the CUDA
library; there is no CPU fallback: if the shared object or a GPU is missing the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

# bc_flags (mirrors include/lbm.h)
BOTTOM_WALL, BOTTOM_PERIODIC = 0, 1
TOP_WALL, TOP_FREE_SLIP, TOP_PERIODIC, TOP_FORCED_EQ = 0 << 2, 1 << 2, 2 << 2, 3 << 2
DRAG_VECTOR = 1 << 4
SOLID_MASK = 1 << 5
STORAGE_AA = 1 << 6
Z_HALO = 1 << 7
VEC_SHIFT = 8
STORAGE_AAX = 1 << 11
NSTAT = 10

INIT_POWER_LAW, INIT_PARABOLA, INIT_REST = 0, 1, 2

LBM_OK, LBM_EINVAL, LBM_ENOMEM, LBM_ESTATE, LBM_ECUDA, LBM_EDIVERGED = 0, -1, -2, -3, -4, -5

_BOTTOM = {"bounce_back": BOTTOM_WALL, "periodic": BOTTOM_PERIODIC}
_TOP = {"bounce_back": TOP_WALL, "free_slip": TOP_FREE_SLIP, "periodic": TOP_PERIODIC,
        "forced_equilibrium": TOP_FORCED_EQ}

# every symbol include/lbm.h declares
SYMBOLS = [
    "lbm_workspace_bytes", "lbm_create", "lbm_bind", "lbm_set_init", "lbm_init", "lbm_set_macros",
    "lbm_set_macros_host", "lbm_step", "lbm_get_macros", "lbm_get_macros_host",
    "lbm_stats_accumulate", "lbm_stats_read", "lbm_stats_reset", "lbm_get_state", "lbm_time",
    "lbm_launch_count", "lbm_set_launch_shape", "lbm_variant", "lbm_destroy", "lbm_last_error",
    "lbm_lad_profile", "lbm_mix64", "lbm_set_kernel_timing", "lbm_kernel_timing_read",
    "lbm_set_top_velocity", "lbm_set_solid", "lbm_wall_friction_velocity",
    "lbm_forest_friction_velocity", "lbm_stats_normalise", "lbm_wall_units", "lbm_set_graphs", "lbm_set_z_slab",
    "lbm_halo_bytes", "lbm_halo_pack", "lbm_halo_unpack", "lbm_stats_read_raw", "lbm_stats_from_raw",
    "lbm_set_state", "lbm_diverged", "lbm_set_reference_profile", "lbm_get_reference_profile", "lbm_set_tma", "lbm_set_sweep",
    "lbm_set_sgs_rows", "lbm_sgs_van_driest", "lbm_sgs_mean_shear", "lbm_plane_stats_static",
    "lbm_set_forest_codes", "lbm_forest_code", "lbm_lad_eq14", "lbm_step_slab_begin", "lbm_step_slab_end",
]


class LbmError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"lbm error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load (building if needed) liblbm_b200.so.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.LIB if (os.path.exists(_build.LIB) and not _build.needs_build()) else _build.build()
        L = C.CDLL(path)
        vp, dp, fp = C.c_void_p, C.POINTER(C.c_double), C.c_void_p
        L.lbm_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_uint32, C.POINTER(C.c_size_t)]
        L.lbm_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, dp,
                                 C.c_double, dp, C.c_uint32]
        L.lbm_bind.argtypes = [vp, vp, C.c_size_t, vp]
        L.lbm_set_init.argtypes = [vp, C.c_int, C.c_double, C.c_double]
        L.lbm_set_top_velocity.argtypes = [vp, dp]
        L.lbm_set_solid.argtypes = [vp, C.c_void_p]
        L.lbm_set_forest_codes.argtypes = [vp, C.c_void_p, C.c_double]
        L.lbm_forest_code.argtypes = [C.c_int, C.c_int, C.c_double]
        L.lbm_forest_code.restype = C.c_uint32
        L.lbm_set_graphs.argtypes = [vp, C.c_int]
        L.lbm_set_z_slab.argtypes = [vp, C.c_int, C.c_int]
        L.lbm_halo_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
        L.lbm_halo_pack.argtypes = [vp, C.c_int, fp]
        L.lbm_halo_unpack.argtypes = [vp, C.c_int, fp]
        L.lbm_step_slab_begin.argtypes = [vp, fp, fp, vp]
        L.lbm_step_slab_end.argtypes = [vp, fp, fp, vp]
        L.lbm_stats_read_raw.argtypes = [vp, dp, dp, dp]
        L.lbm_stats_from_raw.argtypes = [dp, dp, C.c_int, C.c_double, dp]
        L.lbm_wall_friction_velocity.argtypes = [C.c_double, C.c_double, C.c_double, dp]
        L.lbm_forest_friction_velocity.argtypes = [dp, C.c_int, C.c_int, dp]
        L.lbm_stats_normalise.argtypes = [dp, C.c_int, C.c_double, dp]
        L.lbm_wall_units.argtypes = [C.c_int, C.c_double, C.c_double, dp]
        L.lbm_init.argtypes = [vp, C.c_uint64]
        L.lbm_set_macros.argtypes = [vp, fp, fp]
        L.lbm_set_macros_host.argtypes = [vp, fp, fp]
        L.lbm_step.argtypes = [vp, C.c_int]
        L.lbm_get_macros.argtypes = [vp, fp, fp]
        L.lbm_get_macros_host.argtypes = [vp, fp, fp]
        L.lbm_stats_accumulate.argtypes = [vp, C.c_int]
        L.lbm_stats_read.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        L.lbm_stats_reset.argtypes = [vp]
        L.lbm_get_state.argtypes = [vp, fp]
        L.lbm_set_state.argtypes = [vp, fp, C.c_longlong]
        L.lbm_diverged.argtypes = [vp, C.POINTER(C.c_int)]
        L.lbm_set_reference_profile.argtypes = [vp, dp]
        L.lbm_get_reference_profile.argtypes = [vp, dp]
        L.lbm_set_tma.argtypes = [vp, C.c_int, C.c_int]
        L.lbm_set_sweep.argtypes = [vp, C.c_int]
        L.lbm_set_sgs_rows.argtypes = [vp, vp, vp]
        L.lbm_sgs_van_driest.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, vp]
        L.lbm_sgs_mean_shear.argtypes = [vp, C.c_int, C.c_int, vp]
        L.lbm_plane_stats_static.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, vp, vp]
        L.lbm_time.argtypes = [vp]
        L.lbm_time.restype = C.c_longlong
        L.lbm_launch_count.argtypes = [vp]
        L.lbm_launch_count.restype = C.c_longlong
        L.lbm_set_launch_shape.argtypes = [vp, C.c_int, C.c_int]
        L.lbm_variant.argtypes = [vp]
        L.lbm_variant.restype = C.c_char_p
        L.lbm_destroy.argtypes = [vp]
        L.lbm_destroy.restype = None
        L.lbm_last_error.restype = C.c_char_p
        L.lbm_lad_profile.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, dp]
        L.lbm_lad_eq14.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, dp]
        L.lbm_set_kernel_timing.argtypes = [vp, C.c_int]
        L.lbm_kernel_timing_read.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        L.lbm_mix64.argtypes = [C.c_uint64, C.c_uint64]
        L.lbm_mix64.restype = C.c_uint64
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise LbmError(rc, lib().lbm_last_error().decode())


def bc_flags(bottom: str, top: str, drag_vector: bool = False, aa=False, vec: int = 0,
             solid: bool = False, halo: bool = False) -> int:
    """aa: False = two-lattice, True / "aa" = AA pattern, "aax" = x-balanced AA pattern."""
    storage = STORAGE_AAX if aa == "aax" else (STORAGE_AA if aa else 0)
    return (_BOTTOM[bottom] | _TOP[top] | (DRAG_VECTOR if drag_vector else 0) | storage
            | (SOLID_MASK if solid else 0) | (Z_HALO if halo else 0) | (int(vec) << VEC_SHIFT))


def workspace_bytes(nx: int, ny: int, nz: int, flags: int) -> int:
    out = C.c_size_t(0)
    _check(lib().lbm_workspace_bytes(nx, ny, nz, flags, C.byref(out)))
    return int(out.value)


def lad_profile(h: int, ny: int, LAI: float, eta_m: float = 0.7) -> np.ndarray:
    out = np.zeros(ny)
    _check(lib().lbm_lad_profile(int(h), int(ny), float(LAI), float(eta_m),
                                 out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


def lad_eq14(h: int, ny: int, a_fm: float, eta_m: float = 0.7) -> np.ndarray:
    out = np.zeros(ny)
    _check(lib().lbm_lad_eq14(int(h), int(ny), float(a_fm), float(eta_m),
                              out.ctypes.data_as(C.POINTER(C.c_double))))
    return out


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def wall_friction_velocity(F: float, H: float, rho: float = 1.0) -> float:
    out = C.c_double(0.0)
    _check(lib().lbm_wall_friction_velocity(float(F), float(H), float(rho), C.byref(out)))
    return float(out.value)


def forest_friction_velocity(stats: np.ndarray, h: int) -> float:
    st = np.ascontiguousarray(stats, dtype=np.float64)
    out = C.c_double(0.0)
    _check(lib().lbm_forest_friction_velocity(_dp(st), st.shape[0], int(h), C.byref(out)))
    return float(out.value)


def stats_normalise(stats: np.ndarray, u_ref: float) -> np.ndarray:
    st = np.ascontiguousarray(stats, dtype=np.float64)
    out = np.empty_like(st)
    _check(lib().lbm_stats_normalise(_dp(st), st.shape[0], float(u_ref), _dp(out)))
    return out


def wall_units(ny: int, u_tau: float, nu: float) -> np.ndarray:
    out = np.empty(int(ny))
    _check(lib().lbm_wall_units(int(ny), float(u_tau), float(nu), _dp(out)))
    return out


def stats_from_raw(raw: np.ndarray, count: float, centre=None) -> np.ndarray:
    """The lbm_stats_read table from (summed) raw sums; see include/lbm.h."""
    raw = np.ascontiguousarray(raw, dtype=np.float64)
    out = np.empty_like(raw)
    cp = None if centre is None else _dp(np.ascontiguousarray(centre, dtype=np.float64))
    _check(lib().lbm_stats_from_raw(_dp(raw), cp, raw.shape[0], float(count), _dp(out)))
    return out


STATIC_SCRATCH_BYTES = 16 * 1024 * 1024   # LBM_STATIC_SCRATCH_BYTES of include/lbm.h


def plane_stats_static(rho, u, out=None, stream=None, shape=None):
    """lbm_plane_stats_static: plane statistics of one (rho, u) sample without any allocation inside
    the library (its scratch is a static device array).  rho (nz, ny, nx), u (3, nz, ny, nx): CUDA
    float32 tensors; out: a CUDA float64 tensor (ny, NSTAT), made here when None (the caller's
    allocation, not the library's).  `shape` = (nz, ny, nx) overrides the tensors' shape (tests of
    the size check).  Asynchronous on `stream` (default: torch's current stream)."""
    import torch

    nz, ny, nx = shape if shape is not None else rho.shape
    if out is None:
        out = torch.empty((ny, NSTAT), dtype=torch.float64, device=rho.device)
    if stream is None:
        stream = torch.cuda.current_stream(rho.device)
    for t, dt in ((rho, torch.float32), (u, torch.float32), (out, torch.float64)):
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
            raise ValueError("plane_stats_static needs contiguous CUDA tensors: rho, u float32, out float64")
    _check(lib().lbm_plane_stats_static(C.c_void_p(rho.data_ptr()), C.c_void_p(u.data_ptr()), int(nx), int(ny), int(nz),
                                        C.c_void_p(out.data_ptr()), C.c_void_p(stream.cuda_stream)))
    return out


def sgs_van_driest(ny: int, Cs: float, u_tau: float, nu: float, A_plus: float = 26.0, both_walls: bool = False) -> np.ndarray:
    """C_smag per row with van Driest wall damping (lbm_sgs_van_driest)."""
    out = np.zeros(int(ny))
    _check(lib().lbm_sgs_van_driest(int(ny), float(Cs), float(u_tau), float(nu), float(A_plus),
                                    int(bool(both_walls)), C.c_void_p(out.ctypes.data)))
    return out


def sgs_mean_shear(stats: np.ndarray, top_wall: bool = False) -> np.ndarray:
    """Mean-shear magnitude per row of a statistics table (lbm_sgs_mean_shear)."""
    st = np.ascontiguousarray(stats, dtype=np.float64)
    out = np.zeros(st.shape[0])
    _check(lib().lbm_sgs_mean_shear(C.c_void_p(st.ctypes.data), int(st.shape[0]), int(bool(top_wall)),
                                    C.c_void_p(out.ctypes.data)))
    return out


def mix64(seed: int, ctr: int) -> int:
    return int(lib().lbm_mix64(C.c_uint64(seed), C.c_uint64(ctr)))


def forest_code(h: int, y: int, y_m: float) -> int:
    return int(lib().lbm_forest_code(int(h), int(y), float(y_m)))


def forest_codes_from_spec(spec: dict, shape):
    """(codes (nz, ny, nx) uint32, a_fm) from a workloads `forest_cells` spec: a list of blocks
    {x: (x0, x1), z: (z0, z1), y0, h, y_m} (half-open cell ranges; y_m in cells, 0 = constant LAD)."""
    nz, ny, nx = shape
    codes = np.zeros(shape, dtype=np.uint32)
    for b in spec["blocks"]:
        (x0, x1), (z0, z1) = b["x"], b["z"]
        for j in range(b["h"]):
            if 0 <= b["y0"] + j < ny:
                codes[z0:z1, b["y0"] + j, x0:x1] = forest_code(b["h"], j, b["y_m"])
    return codes, float(spec["a_fm"])


def lad_from_spec(forest, ny: int):
    """lad_profile table from a workloads forest spec (None / uniform / lalic)."""
    if forest is None:
        return None
    if forest["kind"] == "uniform":
        a = np.zeros(ny)
        a[: forest["rows"]] = forest["a"]
        return a
    if forest["kind"] == "lalic":
        return lad_profile(forest["h"], ny, forest["LAI"], forest.get("eta_m", 0.7))
    if forest["kind"] == "eq14":
        return lad_eq14(forest["h"], ny, forest["a_fm"], forest.get("eta_m", 0.7))
    raise ValueError(forest)


class Lbm:
    """One simulation handle.  Arrays: rho (nz, ny, nx), u (3, nz, ny, nx), float32."""

    def __init__(self, nx, ny, nz, nu, Cs, body_force=(0.0, 0.0, 0.0), Cd=0.0, lad=None, flags=0,
                 device="cuda:0", stream=None, guard: int = 0):
        """guard > 0 (debugging aid): the workspace is allocated with `guard` extra bytes on either
        side, filled with a byte pattern; guard_intact() tells whether any kernel wrote outside the
        workspace it was given."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2206_15454_b200 needs a CUDA device; there is no CPU fallback")
        L = lib()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.N = self.nx * self.ny * self.nz
        self.flags = int(flags)
        self.device = torch.device(device)
        bf = np.ascontiguousarray(body_force, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        ladp = None
        if lad is not None:
            lad = np.ascontiguousarray(lad, dtype=np.float64)
            if lad.shape != (self.ny,):
                raise ValueError("lad must have ny entries")
            ladp = lad.ctypes.data_as(dp)
        h = C.c_void_p()
        _check(L.lbm_create(C.byref(h), self.nx, self.ny, self.nz, float(nu), float(Cs),
                            bf.ctypes.data_as(dp), float(Cd), ladp, self.flags))
        self._h = h
        nbytes = workspace_bytes(self.nx, self.ny, self.nz, self.flags)
        self._guard = (int(guard) + 255) // 256 * 256
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256 + 2 * self._guard, dtype=torch.uint8, device=self.device)
            if self._guard:
                self._ws.fill_(0xA5)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self._ws.data_ptr()
        aligned = (base + self._guard + 255) // 256 * 256
        self._ws_span = (aligned - base, nbytes)
        _check(L.lbm_bind(self._h, C.c_void_p(aligned), C.c_size_t(nbytes), C.c_void_p(self._stream.cuda_stream)))

    @classmethod
    def from_config(cls, cfg: dict, aa=None, vec: int = 0, halo: bool = False, **kw) -> "Lbm":
        if aa is None:
            st = cfg.get("storage", "two_lattice")
            aa = "aax" if st == "aax" else (st == "aa")
        flags = bc_flags(cfg["bottom"], cfg["top"], cfg.get("drag_vector", False), aa, vec,
                         solid=cfg.get("solid") is not None or cfg.get("forest_cells") is not None
                         or cfg.get("geometry", False), halo=halo)
        s = cls(cfg["nx"], cfg["ny"], cfg["nz"], cfg["nu"], cfg["Cs"], cfg["body_force"], cfg["Cd"],
                lad_from_spec(cfg["forest"], cfg["ny"]), flags, **kw)
        i = cfg["init"]
        s.set_init(i["kind"], i["U_ref"], i["noise_frac"])
        if cfg.get("U_top") is not None:
            s.set_top_velocity(cfg["U_top"])
        if cfg.get("solid") is not None:
            s.set_solid(cfg["solid"])
        if cfg.get("forest_cells") is not None:
            s.set_forest_codes(*forest_codes_from_spec(cfg["forest_cells"], s.shape))
        return s

    def guard_intact(self) -> bool:
        """True if every byte of the workspace allocation outside the bound range still holds the
        fill pattern (only meaningful for handles created with guard > 0)."""
        import torch

        torch.cuda.synchronize(self.device)
        off, n = self._ws_span
        return bool((self._ws[:off] == 0xA5).all()) and bool((self._ws[off + n:] == 0xA5).all())

    def close(self):
        h = getattr(self, "_h", None)
        if h:
            lib().lbm_destroy(h)
            self._h = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def variant(self) -> str:
        return lib().lbm_variant(self._h).decode()

    @property
    def time(self) -> int:
        return int(lib().lbm_time(self._h))

    @property
    def launch_count(self) -> int:
        return int(lib().lbm_launch_count(self._h))

    def set_launch_shape(self, tx: int, ty: int):
        _check(lib().lbm_set_launch_shape(self._h, int(tx), int(ty)))

    def set_forest_codes(self, codes, a_fm: float = 0.0):
        """codes: (nz, ny, nx) uint32 array of lbm_forest_code values (0 = none); None removes them."""
        if codes is None:
            _check(lib().lbm_set_forest_codes(self._h, None, 0.0))
            return
        c = np.ascontiguousarray(codes, dtype=np.uint32)
        if c.shape != self.shape:
            raise ValueError(f"forest codes must have shape {self.shape}")
        _check(lib().lbm_set_forest_codes(self._h, C.c_void_p(c.ctypes.data), float(a_fm)))

    def set_solid(self, mask):
        """mask: (nz, ny, nx) array, non-zero = solid; None clears.  On a running handle the flow
        is kept (cells that turn fluid start at rest)."""
        if mask is None:
            _check(lib().lbm_set_solid(self._h, None))
            return
        m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.uint8)
        if m.shape != self.shape:
            raise ValueError(f"solid mask must have shape {self.shape}")
        _check(lib().lbm_set_solid(self._h, C.c_void_p(m.ctypes.data)))

    def set_top_velocity(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        if U.shape != (3,):
            raise ValueError("U_top must have 3 components")
        _check(lib().lbm_set_top_velocity(self._h, U.ctypes.data_as(C.POINTER(C.c_double))))

    def set_init(self, kind: int, U_ref: float, noise_frac: float):
        _check(lib().lbm_set_init(self._h, int(kind), float(U_ref), float(noise_frac)))

    def init(self, seed: int):
        _check(lib().lbm_init(self._h, C.c_uint64(seed)))

    def _dev(self, t, shape):
        import torch

        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                and tuple(t.shape) == tuple(shape)):
            raise ValueError(f"expected a contiguous float32 CUDA tensor of shape {shape}")
        return C.c_void_p(t.data_ptr())

    @staticmethod
    def _host(a, shape):
        import torch

        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous() or tuple(a.shape) != tuple(shape):
                raise ValueError(f"expected a contiguous float32 CPU tensor of shape {shape}")
            return C.c_void_p(a.data_ptr())
        if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
                and a.shape == tuple(shape)):
            raise ValueError(f"expected a C-contiguous float32 array of shape {shape}")
        return C.c_void_p(a.ctypes.data)

    def set_macros(self, rho, u):
        """State 0 = f_eq(rho, u) from CUDA tensors."""
        _check(lib().lbm_set_macros(self._h, self._dev(rho, self.shape), self._dev(u, (3,) + self.shape)))

    def set_macros_host(self, rho, u):
        """State 0 = f_eq(rho, u) from host arrays (numpy or CPU tensors; pinned = async copies)."""
        _check(lib().lbm_set_macros_host(self._h, self._host(rho, self.shape), self._host(u, (3,) + self.shape)))

    def step(self, n: int = 1):
        _check(lib().lbm_step(self._h, int(n)))

    def get_macros(self, rho=None, u=None):
        """Sample S_k into CUDA tensors (allocated with torch if not given)."""
        import torch

        if rho is None:
            rho = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        if u is None:
            u = torch.empty((3,) + self.shape, dtype=torch.float32, device=self.device)
        _check(lib().lbm_get_macros(self._h, self._dev(rho, self.shape), self._dev(u, (3,) + self.shape)))
        return rho, u

    def get_macros_host(self, rho=None, u=None):
        if rho is None:
            rho = np.empty(self.shape, dtype=np.float32)
        if u is None:
            u = np.empty((3,) + self.shape, dtype=np.float32)
        _check(lib().lbm_get_macros_host(self._h, self._host(rho, self.shape), self._host(u, (3,) + self.shape)))
        return rho, u

    def get_state(self):
        """(19, nz, ny, nx) CUDA tensor of f_i - w_i, plain post-collision state."""
        import torch

        out = torch.empty((19,) + self.shape, dtype=torch.float32, device=self.device)
        _check(lib().lbm_get_state(self._h, C.c_void_p(out.data_ptr())))
        return out

    def set_tma(self, mode: int, rows: int = 0):
        """Which step kinds stream through the TMA unit (bit 0 AA even, 1 AA odd, 2 pull); rows per tile."""
        _check(lib().lbm_set_tma(self._h, int(mode), int(rows)))

    def set_sgs_rows(self, csmag_row=None, sbar_row=None):
        """Per-row SGS tables (other SGS models): C_smag,j and / or mean shear |<S>|_j; None, None = standard."""
        keep, ptrs = [], []
        for a in (csmag_row, sbar_row):
            if a is None:
                ptrs.append(None)
            else:
                a = np.ascontiguousarray(a, dtype=np.float64)
                if a.shape != (self.ny,):
                    raise ValueError(f"SGS row table must have shape ({self.ny},)")
                keep.append(a)
                ptrs.append(C.c_void_p(a.ctypes.data))
        _check(lib().lbm_set_sgs_rows(self._h, ptrs[0], ptrs[1]))

    def set_sweep(self, mode: int):
        """1 (default): consecutive steps walk the lattice in opposite directions (L2 reuse); 0: forward."""
        _check(lib().lbm_set_sweep(self._h, int(mode)))

    def set_reference_profile(self, jx_ref=None):
        """Per-row momentum reference of the collision arithmetic (rounding only); None = 0."""
        if jx_ref is None:
            _check(lib().lbm_set_reference_profile(self._h, None))
            return
        r = np.ascontiguousarray(jx_ref, dtype=np.float64)
        if r.shape != (self.ny,):
            raise ValueError("jx_ref must have ny entries")
        _check(lib().lbm_set_reference_profile(self._h, _dp(r)))

    def get_reference_profile(self) -> np.ndarray:
        out = np.zeros(self.ny)
        _check(lib().lbm_get_reference_profile(self._h, _dp(out)))
        return out

    def set_state(self, f_minus_w, t: int = 0):
        """Install a (19, nz, ny, nx) CUDA tensor of f_i - w_i as the plain state of step t."""
        _check(lib().lbm_set_state(self._h, self._dev(f_minus_w, (19,) + self.shape), int(t)))

    def save_checkpoint(self, path: str):
        """Write the plain state (lbm_get_state) and the time step to a file (plumbing: one device->host
        copy and torch.save).  A run restarted with load_checkpoint continues bit for bit."""
        import torch

        # the momentum reference of the collision arithmetic is part of the bit-exact state
        torch.save({"shape": self.shape, "t": self.time, "state": self.get_state().cpu(),
                    "jx_ref": torch.from_numpy(self.get_reference_profile())}, path)

    def load_checkpoint(self, path: str):
        """Install a state written by save_checkpoint (lbm_set_state); the lattice shape must match."""
        import torch

        ck = torch.load(path, map_location="cpu")
        if tuple(ck["shape"]) != tuple(self.shape):
            raise ValueError(f"checkpoint is for a {ck['shape']} lattice, this handle is {self.shape}")
        self.set_reference_profile(ck["jx_ref"].numpy())
        self.set_state(ck["state"].to(self.device), int(ck["t"]))

    def diverged(self) -> bool:
        """True once lbm_get_macros* or the statistics reduction has seen a non-finite density."""
        flag = C.c_int(0)
        rc = lib().lbm_diverged(self._h, C.byref(flag))
        if rc not in (LBM_OK, LBM_EDIVERGED):
            _check(rc)
        return bool(flag.value)

    def stats_accumulate(self, every: int = 1):
        _check(lib().lbm_stats_accumulate(self._h, int(every)))

    def stats_reset(self):
        _check(lib().lbm_stats_reset(self._h))

    def stats_read(self):
        out = np.zeros((self.ny, NSTAT))
        n = C.c_longlong(0)
        _check(lib().lbm_stats_read(self._h, out.ctypes.data_as(C.POINTER(C.c_double)), C.byref(n)))
        return out, int(n.value)

    # ---- z-slab halo mode (LBM_Z_HALO) ----
    def set_z_slab(self, z_first: int, nz_global: int):
        _check(lib().lbm_set_z_slab(self._h, int(z_first), int(nz_global)))

    def halo_buffer(self):
        """A CUDA tensor of the size lbm_halo_pack / lbm_halo_unpack move: (5, ny, nx) float32."""
        import torch

        n = C.c_size_t(0)
        _check(lib().lbm_halo_bytes(self._h, C.byref(n)))
        assert n.value == 5 * self.ny * self.nx * 4
        return torch.empty((5, self.ny, self.nx), dtype=torch.float32, device=self.device)

    def halo_pack(self, side: int, buf):
        _check(lib().lbm_halo_pack(self._h, int(side), self._dev(buf, (5, self.ny, self.nx))))

    def halo_unpack(self, side: int, buf):
        _check(lib().lbm_halo_unpack(self._h, int(side), self._dev(buf, (5, self.ny, self.nx))))

    def step_slab_begin(self, send_lo, send_hi, packed_event=None):
        """Boundary planes, pack, record `packed_event` (a torch.cuda.Event), interior planes."""
        ev = C.c_void_p(packed_event.cuda_event) if packed_event is not None else None
        shp = (5, self.ny, self.nx)
        _check(lib().lbm_step_slab_begin(self._h, self._dev(send_lo, shp), self._dev(send_hi, shp), ev))

    def step_slab_end(self, recv_lo, recv_hi, ready_event=None):
        """Wait for `ready_event`, unpack the ghost planes, finish the step."""
        ev = C.c_void_p(ready_event.cuda_event) if ready_event is not None else None
        shp = (5, self.ny, self.nx)
        _check(lib().lbm_step_slab_end(self._h, self._dev(recv_lo, shp), self._dev(recv_hi, shp), ev))

    def stats_read_raw(self):
        """(raw sums [ny][10], centre [ny][3], count) - additive over slabs when the centre is 0."""
        raw = np.zeros((self.ny, NSTAT))
        centre = np.zeros((self.ny, 3))
        cnt = C.c_double(0.0)
        _check(lib().lbm_stats_read_raw(self._h, _dp(raw), _dp(centre), C.byref(cnt)))
        return raw, centre, float(cnt.value)

    def set_graphs(self, mode: int):
        """0 off, 1 on, 2 auto (CUDA graphs of ~32 steps inside lbm_step)."""
        _check(lib().lbm_set_graphs(self._h, int(mode)))

    def set_kernel_timing(self, on: bool):
        _check(lib().lbm_set_kernel_timing(self._h, int(bool(on))))

    def kernel_timing_read(self):
        """(summed step-kernel device time in ms, number of bracketed launches); clears the record."""
        ms = C.c_double(0.0)
        n = C.c_longlong(0)
        _check(lib().lbm_kernel_timing_read(self._h, C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def synchronize(self):
        self._stream.synchronize()
