"""CPU-side checks of the CUDA library: it builds for sm_100a, loads, exports every symbol that
include/lbm.h declares, and its host-only entry points behave (no kernel is launched here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def lb():
    import paper_2206_15454_b200 as lb
    lb.lib()
    return lb


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lb):
    names = _declared_symbols()
    assert len(names) >= 20
    L = lb.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/lbm.h but not exported"
    assert sorted(lb.SYMBOLS) == names


def test_sass_is_sm100a_only():
    import subprocess
    from paper_2206_15454_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2206_15454_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "lbm_oracle" not in src, f


def test_create_argument_errors(lb):
    L = lb.lib()
    h = C.c_void_p()
    bf = (C.c_double * 3)(0, 0, 0)
    dp = C.POINTER(C.c_double)

    def create(nx=8, ny=8, nz=8, nu=0.01, Cs=0.1, Cd=0.0, lad=None, flags=0):
        return L.lbm_create(C.byref(h), nx, ny, nz, nu, Cs, C.cast(bf, dp), Cd, lad, flags)

    assert create() == lb.LBM_OK
    L.lbm_destroy(h)
    assert create(nu=0.0) == lb.LBM_EINVAL and b"nu" in L.lbm_last_error()
    assert create(nx=0) == lb.LBM_EINVAL
    assert create(nx=4096, ny=1024, nz=1024) == lb.LBM_EINVAL          # >= 2^31 cells
    assert create(flags=lb.BOTTOM_PERIODIC | lb.TOP_WALL) == lb.LBM_EINVAL  # periodic-y needs both
    assert create(flags=lb.BOTTOM_PERIODIC | lb.TOP_FORCED_EQ) == lb.LBM_EINVAL  # lid needs a wall below
    assert create(flags=lb.TOP_FORCED_EQ) == lb.LBM_OK
    utop = (C.c_double * 3)(0.05, 0.0, 0.0)
    assert L.lbm_set_top_velocity(h, C.cast(utop, dp)) == lb.LBM_OK
    utop[1] = float("nan")
    assert L.lbm_set_top_velocity(h, C.cast(utop, dp)) == lb.LBM_EINVAL
    L.lbm_destroy(h)
    assert create() == lb.LBM_OK
    assert L.lbm_set_top_velocity(h, C.cast(utop, dp)) == lb.LBM_EINVAL   # not a lid handle
    L.lbm_destroy(h)
    assert create(nx=6, flags=4 << 8) == lb.LBM_EINVAL                  # vec=4 does not divide 6
    assert create(flags=1 << 20) == lb.LBM_EINVAL
    bad = (C.c_double * 8)(*([0.1] * 7 + [-1.0]))
    assert create(lad=C.cast(bad, dp)) == lb.LBM_EINVAL
    # calls out of order never touch the GPU
    assert create() == lb.LBM_OK
    assert L.lbm_set_graphs(h, 3) == lb.LBM_EINVAL and L.lbm_set_graphs(h, 1) == lb.LBM_OK
    assert L.lbm_set_solid(h, None) == lb.LBM_EINVAL                     # not a mask handle
    assert L.lbm_step(h, 1) == lb.LBM_ESTATE
    assert L.lbm_init(h, 1) == lb.LBM_ESTATE
    assert L.lbm_bind(h, None, 0, None) == lb.LBM_EINVAL
    assert L.lbm_bind(h, C.c_void_p(256), 16, None) == lb.LBM_ENOMEM
    L.lbm_destroy(h)


def test_workspace_bytes(lb):
    n = 64 * 32 * 32
    two = lb.workspace_bytes(64, 32, 32, 0)
    aa = lb.workspace_bytes(64, 32, 32, lb.STORAGE_AA)
    assert two - aa == 76 * n                     # the second lattice
    assert aa >= 76 * n and aa < 76 * n + 16 * n + (4 << 20)
    # config 5 as an AA single array is a ~46 GB problem (BASELINE.json:configs[4])
    big = lb.workspace_bytes(1536, 384, 1024, lb.STORAGE_AA)
    assert 45.9e9 < big < 47.0e9


def test_mix64_known_answers(lb):
    """The library's own counter-based generator against the published splitmix64 vectors."""
    for line in open(os.path.join(GOLD, "splitmix64_vectors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        seed, n, val = (int(t) for t in line.split())
        assert lb.mix64(seed, n) == val


def test_lad_profile_closed_forms(lb):
    """Eqs. 14-15: peak value 1 at eta_m, zero above h, sum = LAI, and the
    midpoint mean of the shape tends to the quadrature value 0.4601."""
    for h, ny in [(16, 128), (32, 256), (48, 384)]:
        a = lb.lad_profile(h, ny, 2.0, 0.7)
        assert a.shape == (ny,) and np.all(a[h:] == 0) and np.all(a[:h] > 0)
        assert abs(a.sum() - 2.0) < 1e-12
        j = int(np.argmax(a))
        assert abs((j + 0.5) / h - 0.7) <= 0.5 / h + 1e-12
        eta = (np.arange(h) + 0.5) / h
        r = 0.3 / (1 - eta)
        n = np.where(eta < 0.7, 6.0, 0.5)
        shape = r ** n * np.exp(n * (1 - r))
        assert np.allclose(a[:h], 2.0 * shape / shape.sum(), rtol=1e-12)
        assert abs(shape.mean() - 0.4601) < 2e-3
    # peak a_fm for LAI = 2: 0.2726 (h=16), 0.1358 (h=32), 0.0906 (h=48)
    assert abs(lb.lad_profile(16, 128, 2.0).max() - 0.2726) < 2e-3
    assert abs(lb.lad_profile(32, 256, 2.0).max() - 0.1358) < 1e-3
    assert abs(lb.lad_profile(48, 384, 2.0).max() - 0.0906) < 1e-3


def test_no_cpu_fallback(lb):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        lb.Lbm(8, 8, 8, 0.01, 0.1)


def test_normalisation_helpers_closed_forms(lb):
    """NEXT #3 host helpers against the paper's definitions (L179 Eq. 16) and Table I."""
    import os
    g = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_table1.txt")):
        if not line.startswith("#") and line.strip():
            k, v = line.split()
            g[k] = float(v)
    u_tau = lb.wall_friction_velocity(g["F"], g["H"], 1.0)
    assert u_tau * g["H"] / g["nu"] == pytest.approx(177.6, abs=0.1)       # Table I => Re_tau = 177.6
    ny, h = 20, 4
    st = np.zeros((ny, lb.NSTAT))
    st[:, 0] = np.linspace(0.01, 0.08, ny)
    st[:, 3] = 4e-6; st[:, 4] = 1e-6; st[:, 5] = -1e-12                    # tiny negative variance -> 0
    st[:, 6] = -np.arange(ny) * 1e-6
    st[:, 7] = 2e-6
    st[:, 9] = 1.0
    uv = -0.5 * (7 + 8) * 1e-6
    assert lb.forest_friction_velocity(st, h) == pytest.approx((uv ** 2 + (2e-6) ** 2) ** 0.25, rel=1e-14)
    with pytest.raises(lb.LbmError):
        lb.forest_friction_velocity(st, 10)                                # 2h = ny
    n = lb.stats_normalise(st, 0.002)
    assert np.allclose(n[:, 0], st[:, 0] / 0.002) and np.allclose(n[:, 3], 1.0) and np.allclose(n[:, 4], 0.5)
    assert np.all(n[:, 5] == 0.0) and np.allclose(n[:, 6], st[:, 6] / 4e-6) and np.all(n[:, 9] == 1.0)
    with pytest.raises(lb.LbmError):
        lb.stats_normalise(st, 0.0)
    yp = lb.wall_units(4, 0.01, 2e-4)
    assert np.allclose(yp, (np.arange(4) + 0.5) * 50.0)


def test_sgs_row_table_helpers_closed_forms(lb):
    """Host helpers of the row-table SGS models (include/lbm.h lbm_sgs_van_driest,
    lbm_sgs_mean_shear) against their closed forms, written out here independently of oracle/."""
    ny, Cs, ut, nu, Ap = 40, 0.1, 2.5e-3, 2e-4, 26.0
    yp = (np.arange(ny) + 0.5) * ut / nu
    C1 = lb.sgs_van_driest(ny, Cs, ut, nu, Ap)
    assert np.allclose(C1, Cs ** 2 * (1 - np.exp(-yp / Ap)) ** 2, rtol=1e-13, atol=0)
    C2 = lb.sgs_van_driest(ny, Cs, ut, nu, Ap, both_walls=True)
    assert np.allclose(C2, C2[::-1], rtol=1e-15) and np.array_equal(C2[: ny // 2], C1[: ny // 2])
    with pytest.raises(lb.LbmError):
        lb.sgs_van_driest(ny, Cs, ut, 0.0)
    y = np.arange(ny) + 0.5
    st = np.zeros((ny, lb.NSTAT))
    st[:, 0] = 0.2 * (y / ny) * (1 - y / ny)
    st[:, 2] = -0.5 * st[:, 0]
    S = lb.sgs_mean_shear(st, top_wall=True)
    want = np.abs(0.2 / ny * (1 - 2 * y / ny)) * np.sqrt(1.25)
    assert np.allclose(S[1:-1], want[1:-1], rtol=1e-12, atol=1e-18)
    assert np.isclose(S[0], 0.5 * (st[0, 0] + st[1, 0]) * np.sqrt(1.25), rtol=1e-13) and np.isclose(S[-1], S[0], rtol=1e-12)
    S2 = lb.sgs_mean_shear(st, top_wall=False)
    assert np.isclose(S2[-1], 0.5 * abs(st[-1, 0] - st[-2, 0]) * np.sqrt(1.25), rtol=1e-12)


def test_block_shapes_of_the_configs_and_the_paper_meshes(lb):
    """Host logic of lbm_create (no GPU): cells per thread and thread-block shape per lattice width.
    Whole-warp row segments where the width offers them; the paper's meshes (PAPER.md:L171, L244:
    372, 350, 250, 200 cells wide) take one irregular row segment per block; lattices of <= 2^17
    cells run one cell per thread; the x-balanced storage accepts geometry handles."""
    L = lb.lib()
    L.lbm_variant.restype = C.c_char_p
    bf = (C.c_double * 3)(0, 0, 0)
    dp = C.POINTER(C.c_double)
    cases = [
        ((1536, 384, 1024), lb.STORAGE_AAX, "aax/v4/tx128x1"),
        ((1024, 256, 512), lb.STORAGE_AAX | lb.SOLID_MASK, "aax/v4/tx128x1"),
        ((512, 128, 256), 0, "pull2/v4/tx128x1"),
        ((64, 32, 32), 0, "pull2/v1/tx64x2"),
        ((372, 62, 124), 0, "pull2/v4/tx93x1"),
        ((350, 140, 280), lb.STORAGE_AAX, "aax/v2/tx175x1"),
        ((250, 100, 200), lb.STORAGE_AA, "aa/v2/tx125x1"),
        ((200, 80, 160), 0, "pull2/v4/tx50x1"),
    ]
    for (nx, ny, nz), flags, want in cases:
        h = C.c_void_p()
        rc = L.lbm_create(C.byref(h), nx, ny, nz, 1e-4, 0.1, C.cast(bf, dp), 0.0, None, flags | lb.TOP_FREE_SLIP)
        assert rc == 0, (nx, ny, nz, L.lbm_last_error())
        got = L.lbm_variant(h).decode()
        L.lbm_destroy(h)
        assert got == want, ((nx, ny, nz), got, want)
