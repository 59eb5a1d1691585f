"""P11 — statistical parity over long runs that have diverged chaotically (BASELINE.json
north_star: plane-averaged mean profile within 2 %, Reynolds stresses within 5 %).

The CUDA path and the fp64 oracle start from the same seeded field, spin up, then both accumulate
y-plane statistics over the same window.  By then the two trajectories differ locally by far more
than the 100-step tolerance (asserted, so that the test really is about diverged runs); what must
still agree is the statistics.  Differences are normalised by the profile maxima, as north_star's
percentages are read in DESIGN.md §4 ("of the profile maximum"), and additionally point by point
relative to the local value wherever the profile exceeds a fifth of its maximum (near zero
crossings a relative bound means nothing).  Lattices are the ones the oracle finishes in seconds:
these are small-lattice, short-window checks; the full-length config-2 run (20 k + 20 k steps, one
hour of oracle time) is tests/run_p11_cfg2.py, its reports profiles/r01_p11_cfg2.md (round 1,
two-lattice) and profiles/r02_p11_cfg2.md (round 2, the final x-balanced AA kernels).
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    lb.lib()
    return lb


@pytest.fixture(scope="module")
def orc():
    import oracle
    oracle.build()
    return oracle


def _channel_small():
    cfg = wl.get("cfg2")                 # plane channel physics on an oracle-sized lattice
    cfg["nx"], cfg["ny"], cfg["nz"] = 64, 32, 32
    return cfg


@pytest.mark.parametrize("case,aa,spin,window", [
    ("cfg1", True, 2000, 4000), ("cfg1", False, 2000, 4000), ("channel", True, 3000, 3000)])
def test_long_run_statistics(orc, gpu, case, aa, spin, window):
    cfg = wl.get("cfg1") if case == "cfg1" else _channel_small()
    o = orc.Oracle.from_config(cfg)
    o.init_from_config(cfg)
    g = gpu.Lbm.from_config(cfg, aa=aa)
    g.init(cfg["seed"])
    o.step(spin)
    g.step(spin)
    for s in (o, g):
        s.stats_accumulate(1)
        s.stats_reset()
    o.step(window)
    g.step(window)
    _, uo = o.get_macros()
    _, ug = g.get_macros()
    diverged = float(np.abs(ug.cpu().numpy() - uo).max())
    so, no = o.stats_read()
    sg, ng = g.stats_read()
    assert no == ng == window and np.isfinite(sg).all()
    umax = np.abs(so[:, 0]).max()
    d_mean = np.abs(sg[:, 0] - so[:, 0]).max() / umax
    print(f"{case} {g.variant}: local max|du| after {spin + window} steps = {diverged:.2e}; "
          f"mean U differs by {100 * d_mean:.3f} % of max")
    # cfg1 (sheared canopy flow) has left the short-time tolerance far behind by now; the small
    # channel stays closer.  Either way the statistics must agree
    if case == "cfg1":
        assert diverged > 10 * 1e-5 * cfg["u_bulk"]
    assert d_mean <= 0.02

    def pointwise(k):
        """worst |difference| / |oracle value| over the rows whose value exceeds 20 % of the maximum"""
        rows = np.abs(so[:, k]) >= 0.2 * np.abs(so[:, k]).max()
        rel = np.abs(sg[rows, k] - so[rows, k]) / np.abs(so[rows, k])
        j = int(np.flatnonzero(rows)[int(np.argmax(rel))])
        return float(rel.max()), j

    rel, j = pointwise(0)
    print(f"   <U>: worst pointwise relative difference {100 * rel:.3f} % at row {j}")
    assert rel <= 0.02
    for k, name in ((3, "uu"), (4, "vv"), (5, "ww"), (6, "uv")):
        m = np.abs(so[:, k]).max()
        d = np.abs(sg[:, k] - so[:, k]).max() / m
        rel, j = pointwise(k)
        print(f"   <{name}>: max {m:.3e}, differs by {100 * d:.3f} % of max, pointwise {100 * rel:.3f} % at row {j}")
        assert d <= 0.05 and rel <= 0.05
    # the near-zero stresses (vw, uw vanish by symmetry) are compared on the scale of uv
    scale = np.abs(so[:, 6]).max()
    assert np.abs(sg[:, 7:9] - so[:, 7:9]).max() <= 0.05 * scale
    assert np.abs(sg[:, 9] - so[:, 9]).max() <= 1e-5
