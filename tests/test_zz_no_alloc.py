"""lbm_plane_stats_static — the entry point that allocates nothing (include/lbm.h): plane statistics
of one (rho, u) sample with the stage-1 scratch in a static device array, against the existing
path (a handle's fused statistics, lbm_stats_accumulate / lbm_step / lbm_stats_read) on the same
sample, within the tolerances of tests/test_gpu_parity.py (_check_stats), on two calls in a row.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and
after the other tests (it depends on nothing they leave behind: the scratch array keeps the last
call's contents and every call overwrites all it reads)."""
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


def _sample_and_reference(gpu, cfg, aa, presteps):
    """(rho, u) of the sample S_k and the existing path's statistics of exactly that sample."""
    g = gpu.Lbm.from_config(cfg, aa=aa)
    g.init(cfg["seed"])
    g.step(presteps)
    rho, u = g.get_macros()                 # S_k: moments of the streamed state k (R19)
    g.stats_accumulate(1)
    g.stats_reset()
    g.step(1)                               # the fused statistics sample the same S_k
    ref, n = g.stats_read()
    assert n == 1
    g.close()
    return rho, u, ref


def _check(got, ref, u_bulk):
    # the tolerances of tests/test_gpu_parity.py::_check_stats
    assert np.abs(got[:, 0:3] - ref[:, 0:3]).max() <= 1e-5 * u_bulk
    assert np.abs(got[:, 3:9] - ref[:, 3:9]).max() <= 1e-5 * u_bulk ** 2
    assert np.abs(got[:, 9] - ref[:, 9]).max() <= 1e-6


def test_static_scratch_entry_point_matches_the_handle_path_twice_in_a_row(gpu):
    import torch
    # first call: a lattice whose rows span several tiles with a ragged tail; second call, straight
    # after it on the same stream: a SMALLER lattice in another storage scheme, so that stale
    # contents of the shared scratch array from the first call would show
    cases = [(wl.small(nx=100, ny=24, nz=20), True, 6), (wl.small(nx=36, ny=10, nz=7), False, 3)]
    samples = [_sample_and_reference(gpu, cfg, aa, k) for cfg, aa, k in cases]
    outs = [gpu.plane_stats_static(rho, u) for rho, u, _ in samples]          # two calls in a row
    torch.cuda.synchronize()
    for (cfg, _, _), (rho, u, ref), out in zip(cases, samples, outs):
        got = out.cpu().numpy()
        assert got.shape == ref.shape and np.isfinite(got).all()
        _check(got, ref, cfg["u_bulk"])
        # and against the plain definition on the same fields (numpy, fp64); the stage-1 partials are
        # fp32 row sums: relative rounding 6e-8 of |u| <= 0.06, u^2 <= 4e-3, rho ~ 1
        r64, u64 = rho.double().cpu().numpy(), u.double().cpu().numpy()
        mean = u64.mean(axis=(1, 3))                                         # (3, ny)
        assert np.abs(got[:, 0:3] - mean.T).max() <= 1e-8
        assert np.abs(got[:, 3] - ((u64[0] ** 2).mean(axis=(0, 2)) - mean[0] ** 2)).max() <= 2e-9
        assert np.abs(got[:, 6] - ((u64[0] * u64[1]).mean(axis=(0, 2)) - mean[0] * mean[1])).max() <= 2e-9
        assert np.abs(got[:, 9] - r64.mean(axis=(0, 2))).max() <= 2e-7
    # the first case again: same result bit for bit (nothing carried over from the second call)
    again = gpu.plane_stats_static(samples[0][0], samples[0][1])
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])


def test_static_scratch_size_limit_is_an_error(gpu):
    import torch
    rho = torch.zeros((2, 2, 4), dtype=torch.float32, device="cuda")
    u = torch.zeros((3, 2, 2, 4), dtype=torch.float32, device="cuda")
    out = torch.zeros((8, gpu.NSTAT), dtype=torch.float64, device="cuda")
    rows_max = gpu.STATIC_SCRATCH_BYTES // (gpu.NSTAT * 4)
    # one row more than the array holds: rejected before any pointer is touched
    with pytest.raises(gpu.LbmError) as e:
        gpu.plane_stats_static(rho, u, out=out, shape=(rows_max // 1024 + 1, 1024, 4))
    assert e.value.code == gpu.LBM_EINVAL and "static array holds" in str(e.value)
    with pytest.raises(gpu.LbmError):
        gpu.plane_stats_static(rho, u, out=out, shape=(70000, 2, 4))          # nz beyond the grid limit
    with pytest.raises(gpu.LbmError):
        gpu.plane_stats_static(rho, u, out=out, shape=(0, 2, 4))
    # config 5's cross-section (384 x 1024 rows) is within the limit
    assert 384 * 1024 <= rows_max
