"""ctypes front-end of the fp64 CPU oracle (oracle/lbm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports
paper_2206_15454_b200 and shares no code with it.

Arrays: rho has shape (nz, ny, nx), u has shape (3, nz, ny, nx), populations (19, nz, ny, nx),
all float64, C-contiguous (cell = x + nx*(y + ny*z)).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_oracle.c")
_LIB = os.path.join(_HERE, "liblbm_oracle.so")

# bc_flags (the oracle's own copy of the layout in DESIGN.md "Boundary")
BOTTOM_WALL, BOTTOM_PERIODIC = 0, 1
TOP_WALL, TOP_FREE_SLIP, TOP_PERIODIC, TOP_FORCED_EQ = 0 << 2, 1 << 2, 2 << 2, 3 << 2
DRAG_VECTOR = 1 << 4
SOLID_MASK = 1 << 5

_BOTTOM = {"bounce_back": BOTTOM_WALL, "periodic": BOTTOM_PERIODIC}
_TOP = {"bounce_back": TOP_WALL, "free_slip": TOP_FREE_SLIP, "periodic": TOP_PERIODIC,
        "forced_equilibrium": TOP_FORCED_EQ}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, dp, C.c_double,
                                 dp, C.c_uint]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_top_velocity.argtypes = [C.c_void_p, dp]
        L.orc_set_solid.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_forest_codes.argtypes = [C.c_void_p, C.c_void_p, C.c_double]
        L.orc_forest_code.restype = C.c_uint32
        L.orc_forest_code.argtypes = [C.c_int, C.c_int, C.c_double]
        L.orc_forest_code_lad.restype = C.c_double
        L.orc_forest_code_lad.argtypes = [C.c_uint32, C.c_double]
        L.orc_set_macros.argtypes = [C.c_void_p, dp, dp]
        L.orc_init_field.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_uint64, dp, dp]
        L.orc_init.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_uint64]
        L.orc_get_populations.argtypes = [C.c_void_p, dp]
        L.orc_set_populations.argtypes = [C.c_void_p, dp]
        L.orc_stream_only.argtypes = [C.c_void_p, dp]
        L.orc_get_macros.argtypes = [C.c_void_p, dp, dp]
        L.orc_stats_accumulate.argtypes = [C.c_void_p, C.c_int]
        L.orc_stats_reset.argtypes = [C.c_void_p]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_stats_read.restype = C.c_longlong
        L.orc_stats_read.argtypes = [C.c_void_p, dp]
        L.orc_stats_raw.argtypes = [C.c_void_p, dp]
        L.orc_time.restype = C.c_longlong
        L.orc_time.argtypes = [C.c_void_p]
        L.orc_tau0.restype = C.c_double
        L.orc_tau0.argtypes = [C.c_void_p]
        L.orc_tables.argtypes = [ip, dp, ip, ip]
        L.orc_feq.argtypes = [C.c_double, dp, dp]
        L.orc_guo.argtypes = [C.c_double, dp, dp, dp]
        L.orc_tau_total.restype = C.c_double
        L.orc_tau_total.argtypes = [C.c_double, C.c_double, C.c_double, dp]
        L.orc_mix64.restype = C.c_uint64
        L.orc_mix64.argtypes = [C.c_uint64, C.c_uint64]
        L.orc_rand01.restype = C.c_double
        L.orc_rand01.argtypes = [C.c_uint64, C.c_uint64]
        L.orc_tau_total_rows.restype = C.c_double
        L.orc_tau_total_rows.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, dp]
        L.orc_sgs_van_driest.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, dp]
        L.orc_sgs_mean_shear.argtypes = [dp, C.c_int, C.c_int, dp]
        L.orc_set_sgs_rows.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_lad_shape.restype = C.c_double
        L.orc_lad_shape.argtypes = [C.c_double, C.c_double]
        L.orc_lad_profile.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, dp]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


# ---- unit functions -------------------------------------------------------------------------

def tables():
    c = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19)
    opp = np.zeros(19, dtype=np.int32)
    mir = np.zeros(19, dtype=np.int32)
    ip = C.POINTER(C.c_int)
    lib().orc_tables(c.ctypes.data_as(ip), _dp(w), opp.ctypes.data_as(ip), mir.ctypes.data_as(ip))
    return c, w, opp, mir


def feq(rho: float, u) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(19)
    lib().orc_feq(float(rho), _dp(u), _dp(out))
    return out


def guo(tau: float, u, F) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float64)
    F = np.ascontiguousarray(F, dtype=np.float64)
    out = np.zeros(19)
    lib().orc_guo(float(tau), _dp(u), _dp(F), _dp(out))
    return out


def tau_total(tau0: float, Csmag: float, rho: float, Pneq6) -> float:
    p = np.ascontiguousarray(Pneq6, dtype=np.float64)
    return lib().orc_tau_total(float(tau0), float(Csmag), float(rho), _dp(p))


def tau_total_rows(tau0: float, C_j: float, Sbar_j: float, rho: float, Pneq6) -> float:
    P = np.ascontiguousarray(Pneq6, dtype=np.float64)
    return float(lib().orc_tau_total_rows(float(tau0), float(C_j), float(Sbar_j), float(rho), _dp(P)))


def sgs_van_driest(ny: int, Cs: float, u_tau: float, nu: float, A_plus: float = 26.0, both_walls: bool = False):
    out = np.zeros(ny)
    lib().orc_sgs_van_driest(int(ny), float(Cs), float(u_tau), float(nu), float(A_plus), int(bool(both_walls)), _dp(out))
    return out


def sgs_mean_shear(stats, top_wall: bool = False):
    st = np.ascontiguousarray(stats, dtype=np.float64)
    out = np.zeros(st.shape[0])
    lib().orc_sgs_mean_shear(_dp(st), int(st.shape[0]), int(bool(top_wall)), _dp(out))
    return out


def mix64(seed: int, ctr: int) -> int:
    return int(lib().orc_mix64(C.c_uint64(seed), C.c_uint64(ctr)))


def rand01(seed: int, ctr: int) -> float:
    return float(lib().orc_rand01(C.c_uint64(seed), C.c_uint64(ctr)))


def lad_shape(eta: float, eta_m: float = 0.7) -> float:
    return float(lib().orc_lad_shape(float(eta), float(eta_m)))


def lad_profile(h: int, ny: int, LAI: float, eta_m: float = 0.7) -> np.ndarray:
    out = np.zeros(ny)
    lib().orc_lad_profile(int(h), int(ny), float(LAI), float(eta_m), _dp(out))
    return out


def forest_code(h: int, y: int, y_m: float) -> int:
    return int(lib().orc_forest_code(int(h), int(y), float(y_m)))


def forest_code_lad(code: int, a_fm: float) -> float:
    return float(lib().orc_forest_code_lad(C.c_uint32(code), float(a_fm)))


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
    if forest["kind"] == "eq14":       # the paper's own normalisation: a_j = a_fm s(eta_j) (Table II)
        h, em = forest["h"], forest.get("eta_m", 0.7)
        a = np.zeros(ny)
        a[:h] = [forest["a_fm"] * (lad_shape((j + 0.5) / h, em) if em > 0 else 1.0) for j in range(h)]
        return a
    raise ValueError(forest)


def bc_flags(bottom: str, top: str, drag_vector: bool = False, solid: bool = False) -> int:
    return (_BOTTOM[bottom] | _TOP[top] | (DRAG_VECTOR if drag_vector else 0)
            | (SOLID_MASK if solid else 0))


# ---- simulation handle ----------------------------------------------------------------------

class Oracle:
    def __init__(self, nx, ny, nz, nu, Cs, body_force=(0.0, 0.0, 0.0), Cd=0.0, lad=None, bc=0):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.N = self.nx * self.ny * self.nz
        bf = np.ascontiguousarray(body_force, dtype=np.float64)
        ladp = None
        if lad is not None:
            lad = np.ascontiguousarray(lad, dtype=np.float64)
            assert lad.shape == (self.ny,)
            ladp = _dp(lad)
        self._h = lib().orc_create(self.nx, self.ny, self.nz, float(nu), float(Cs), _dp(bf),
                                   float(Cd), ladp, int(bc))
        if not self._h:
            raise ValueError("orc_create rejected the arguments")

    @classmethod
    def from_config(cls, cfg: dict) -> "Oracle":
        o = cls(cfg["nx"], cfg["ny"], cfg["nz"], cfg["nu"], cfg["Cs"], cfg["body_force"], cfg["Cd"],
                lad_from_spec(cfg["forest"], cfg["ny"]),
                bc_flags(cfg["bottom"], cfg["top"], cfg.get("drag_vector", False),
                         cfg.get("solid") is not None))
        if cfg.get("U_top") is not None:
            o.set_top_velocity(cfg["U_top"])
        if cfg.get("solid") is not None:
            o.set_solid(cfg["solid"])
        if cfg.get("forest_cells") is not None:
            o.set_forest_codes(*forest_codes_from_spec(cfg["forest_cells"], o.shape))
        return o

    def init_from_config(self, cfg: dict):
        i = cfg["init"]
        self.init(i["kind"], i["U_ref"], i["noise_frac"], cfg["seed"])

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:      # at interpreter shutdown the module globals may be gone
            try:
                _lib.orc_destroy(h)
            except Exception:
                pass
            self._h = None

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    def init(self, kind, U_ref, noise_frac, seed):
        lib().orc_init(self._h, int(kind), float(U_ref), float(noise_frac), C.c_uint64(seed))

    def init_field(self, kind, U_ref, noise_frac, seed):
        rho = np.zeros(self.shape)
        u = np.zeros((3,) + self.shape)
        lib().orc_init_field(self._h, int(kind), float(U_ref), float(noise_frac), C.c_uint64(seed),
                             _dp(rho), _dp(u))
        return rho, u

    def set_macros(self, rho, u):
        rho = np.ascontiguousarray(rho, dtype=np.float64).reshape(self.shape)
        u = np.ascontiguousarray(u, dtype=np.float64).reshape((3,) + self.shape)
        lib().orc_set_macros(self._h, _dp(rho), _dp(u))

    def set_top_velocity(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        lib().orc_set_top_velocity(self._h, _dp(U))

    def set_solid(self, mask):
        """Install / replace / remove (None) the solid cells, keeping the flow."""
        if mask is None:
            lib().orc_set_solid(self._h, None)
        else:
            m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(self.shape)
            lib().orc_set_solid(self._h, m.ctypes.data_as(C.c_void_p))

    def set_forest_codes(self, codes, a_fm: float):
        if codes is None:
            lib().orc_set_forest_codes(self._h, None, 0.0)
        else:
            c = np.ascontiguousarray(codes, dtype=np.uint32).reshape(self.shape)
            lib().orc_set_forest_codes(self._h, c.ctypes.data_as(C.c_void_p), float(a_fm))

    def set_sgs_rows(self, C_row=None, Sbar_row=None):
        """Per-row SGS tables (other SGS models): C_smag,j and / or |<S>|_j; None, None = standard."""
        ptrs = []
        for a in (C_row, Sbar_row):
            if a is None:
                ptrs.append(None)
            else:
                a = np.ascontiguousarray(a, dtype=np.float64)
                assert a.shape == (self.ny,)
                ptrs.append(a.ctypes.data_as(C.c_void_p))
        lib().orc_set_sgs_rows(self._h, ptrs[0], ptrs[1])

    def get_populations(self):
        f = np.zeros((19,) + self.shape)
        lib().orc_get_populations(self._h, _dp(f))
        return f

    def set_populations(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64).reshape((19,) + self.shape)
        lib().orc_set_populations(self._h, _dp(f))

    def stream_only(self):
        f = np.zeros((19,) + self.shape)
        lib().orc_stream_only(self._h, _dp(f))
        return f

    def get_macros(self):
        rho = np.zeros(self.shape)
        u = np.zeros((3,) + self.shape)
        lib().orc_get_macros(self._h, _dp(rho), _dp(u))
        return rho, u

    def step(self, n=1):
        lib().orc_step(self._h, int(n))

    def stats_accumulate(self, every=1):
        lib().orc_stats_accumulate(self._h, int(every))

    def stats_reset(self):
        lib().orc_stats_reset(self._h)

    def stats_read(self):
        out = np.zeros((self.ny, 10))
        n = lib().orc_stats_read(self._h, _dp(out))
        return out, int(n)

    def stats_raw(self):
        out = np.zeros((self.ny, 10))
        lib().orc_stats_raw(self._h, _dp(out))
        return out

    @property
    def time(self):
        return int(lib().orc_time(self._h))

    @property
    def tau0(self):
        return float(lib().orc_tau0(self._h))
