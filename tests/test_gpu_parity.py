"""GPU-vs-oracle parity of the CUDA path, through the C ABI (pin P10 of DESIGN.md).

Every test runs the CUDA library (paper_2206_15454_b200) and the fp64 CPU oracle (oracle/) on the
same seeded inputs and compares element by element.  Tolerances:
  * macroscopic rho, u after 1, 10, 100 and 200 steps: max|delta| <= 1e-5 * u_bulk
    (BASELINE.json:north_star fixes the bound "over 100 steps"; SURVEY P10 lists step 200 at the
    same bound, and it holds there too);
  * one-step / few-step population checks: 2e-7 absolute (fp32 rounding of O(0.05) deviations
    from the weights, a few operations deep), far below any indexing or boundary-link mistake,
    which shows up at the 1e-3 level.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

TOL_REL = 1e-5  # north_star: relative to the bulk velocity


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2206_15454_b200 as lb
    lb.lib()
    return lb


def _weights(orc):
    _, w, _, _ = orc.tables()
    return w


def _pair(orc, gpu, cfg, aa, vec, seed=None):
    cfg = dict(cfg)
    if seed is not None:
        cfg["seed"] = seed
    o = orc.Oracle.from_config(cfg)
    o.init_from_config(cfg)
    g = gpu.Lbm.from_config(cfg, aa=aa, vec=vec)
    g.init(cfg["seed"])
    return o, g


def _macro_err(o, g):
    import torch
    ro, uo = o.get_macros()
    rg, ug = g.get_macros()
    torch.cuda.synchronize()
    rg = rg.cpu().numpy().astype(np.float64)
    ug = ug.cpu().numpy().astype(np.float64)
    return float(np.abs(rg - ro).max()), float(np.abs(ug - uo).max())


def _state_err(o, g, w):
    import torch
    fo = o.get_populations() - w[:, None, None, None]
    fg = g.get_state()
    torch.cuda.synchronize()
    return float(np.abs(fg.cpu().numpy().astype(np.float64) - fo).max())


# ---------------------------------------------------------------------------------------------
# small lattices: every storage scheme x vector width x boundary set, ragged widths
# ---------------------------------------------------------------------------------------------
BCS = [(wl.BOUNCE_BACK, wl.FREE_SLIP), (wl.BOUNCE_BACK, wl.BOUNCE_BACK), (wl.PERIODIC, wl.PERIODIC)]


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("nx,vec", [(32, 4), (32, 2), (32, 1), (36, 4), (34, 2), (33, 1), (128, 4),
                                    (256, 4), (4, 4), (2, 2), (1, 1), (200, 4), (1536, 4)])
@pytest.mark.parametrize("bottom,top", BCS, ids=["wall-slip", "wall-wall", "periodic"])
def test_small_state_and_macros(orc, gpu, aa, nx, vec, bottom, top):
    ny, nz = (6, 3) if nx >= 1024 else (12, 6)
    cfg = wl.small(nx=nx, ny=ny, nz=nz, bottom=bottom, top=top, drag_vector=False)
    o, g = _pair(orc, gpu, cfg, aa, vec)
    w = _weights(orc)
    assert f"v{vec}" in g.variant and g.variant.startswith({False: "pull2/", True: "aa/", "aax": "aax/"}[aa])
    assert _state_err(o, g, w) <= 2e-8            # state 0
    er, eu = _macro_err(o, g)
    assert er <= 2e-7 and eu <= 2e-8
    for k in (1, 1, 1, 2, 5):                     # both AA parities, odd and even step counts
        o.step(k)
        g.step(k)
        assert g.time == o.time
        assert _state_err(o, g, w) <= 2e-7
        er, eu = _macro_err(o, g)
        assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
def test_vector_drag_and_general_force(orc, gpu, aa):
    cfg = wl.small(nx=64, ny=10, nz=8, drag_vector=True)
    cfg["body_force"] = (2e-6, -1e-6, 5e-7)
    o, g = _pair(orc, gpu, cfg, aa, 4)
    w = _weights(orc)
    o.step(7)
    g.step(7)
    assert _state_err(o, g, w) <= 2e-7


@pytest.mark.parametrize("shape", [(1, 1, 1), (4, 1, 1), (1, 5, 1), (2, 3, 1), (8, 1, 7), (5, 2, 3), (3, 1, 3),
                                   (1, 1, 6), (12, 2, 1)])
@pytest.mark.parametrize("bottom,top", BCS, ids=["wall-slip", "wall-wall", "periodic"])
def test_degenerate_lattices(orc, gpu, shape, bottom, top):
    """One-cell-thick lattices: the periodic wrap lands on the cell itself, one row touches both
    y faces at once.  Both storage schemes, odd and even step counts."""
    nx, ny, nz = shape
    cfg = wl.small(nx=nx, ny=ny, nz=nz, bottom=bottom, top=top, forest_rows=min(1, ny))
    w = _weights(orc)
    for aa in (False, True, "aax"):
        o, g = _pair(orc, gpu, cfg, aa, 0)
        assert _state_err(o, g, w) <= 5e-8
        for n in (1, 2, 0, 5):
            o.step(n)
            g.step(n)
            assert _state_err(o, g, w) <= 2e-7, (aa, n)
        er, eu = _macro_err(o, g)
        assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]
        assert g.time == 8


def test_single_block_shapes(orc, gpu):
    """Different thread-block shapes (row split across blocks, several rows per block) agree."""
    cfg = wl.small(nx=256, ny=8, nz=4)
    w = _weights(orc)
    o = orc.Oracle.from_config(cfg)
    o.init_from_config(cfg)
    o.stats_accumulate(1)
    o.step(4)
    so, _ = o.stats_read()
    for aa in (False, True, "aax"):
        for tx, ty in [(64, 1), (32, 2), (16, 4), (8, 8), (64, 4), (32, 8)]:
            g = gpu.Lbm.from_config(cfg, aa=aa, vec=4)
            g.set_launch_shape(tx, ty)
            g.init(cfg["seed"])
            g.stats_accumulate(1)
            g.step(4)
            assert _state_err(o, g, w) <= 2e-7, (aa, tx, ty)
            sg, n = g.stats_read()
            assert n == 4
            _check_stats(sg, so, cfg["u_bulk"])


def test_stats_on_ragged_single_row_blocks(orc, gpu):
    """Blocks of one row whose width is not a multiple of a warp - the shape the paper's 350- and
    250-cell meshes run (175 x 1, 125 x 1 threads): the row sums go through shared memory and the
    whole warps of the block finish them.  (A variant that reduced the whole warps in registers and
    sent only the ragged last warp through shared memory was measured on those meshes: -3 % ... +2 %,
    not adopted.)"""
    for nx, vec, shape in [(350, 2, (175, 1)), (250, 2, (125, 1)), (140, 4, (35, 1)), (66, 2, (33, 1)), (372, 4, (93, 1))]:
        cfg = wl.small(nx=nx, ny=6, nz=4)
        o = orc.Oracle.from_config(cfg)
        o.init_from_config(cfg)
        o.stats_accumulate(1)
        o.step(4)
        so, _ = o.stats_read()
        for aa in (False, True, "aax"):
            g = gpu.Lbm.from_config(cfg, aa=aa, vec=vec)
            g.set_launch_shape(*shape)
            g.init(cfg["seed"])
            g.stats_accumulate(1)
            g.step(4)
            assert _state_err(o, g, _weights(orc)) <= 2e-7, (nx, aa)
            sg, n = g.stats_read()
            assert n == 4
            _check_stats(sg, so, cfg["u_bulk"])
            g.close()


# ---------------------------------------------------------------------------------------------
# statistics (S8, S9) against the oracle's O10 on identical samples
# ---------------------------------------------------------------------------------------------
def _check_stats(sg, so, u_bulk):
    # means: relative to u_bulk; second moments: relative to u_bulk^2 (fp32 x-row sums, fp64 beyond)
    assert np.abs(sg[:, 0:3] - so[:, 0:3]).max() <= 1e-5 * u_bulk
    assert np.abs(sg[:, 3:9] - so[:, 3:9]).max() <= 1e-5 * u_bulk ** 2
    assert np.abs(sg[:, 9] - so[:, 9]).max() <= 1e-6


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("nx,vec", [(64, 4), (36, 4), (34, 2), (33, 1), (512, 4)])
def test_stats_parity(orc, gpu, aa, nx, vec):
    cfg = wl.small(nx=nx, ny=10, nz=6)
    o, g = _pair(orc, gpu, cfg, aa, vec)
    o.step(3)
    g.step(3)
    o.stats_accumulate(2)
    g.stats_accumulate(2)
    g.stats_reset()
    o.stats_reset()
    o.step(9)
    g.step(9)
    so, no = o.stats_read()
    sg, ng = g.stats_read()
    assert no == ng == 5
    _check_stats(sg, so, cfg["u_bulk"])
    # switching sampling off keeps the sums
    g.stats_accumulate(0)
    g.step(2)
    sg2, ng2 = g.stats_read()
    assert ng2 == 5 and np.array_equal(sg2, sg)


def test_set_macros_host_and_get_macros_host(orc, gpu):
    import torch
    cfg = wl.small(nx=64, ny=10, nz=12)
    o = orc.Oracle.from_config(cfg)
    rho, u = o.init_field(cfg["init"]["kind"], cfg["init"]["U_ref"], cfg["init"]["noise_frac"], 777)
    rho = rho * (1.0 + 0.01 * np.sin(np.arange(rho.size).reshape(rho.shape)))
    o.set_macros(rho, u)
    w = _weights(orc)
    for aa in (False, True, "aax"):
        g = gpu.Lbm.from_config(cfg, aa=aa)
        g.set_macros_host(rho.astype(np.float32), u.astype(np.float32))
        assert _state_err(o, g, w) <= 5e-8
        g2 = gpu.Lbm.from_config(cfg, aa=aa)
        g2.set_macros(torch.from_numpy(rho.astype(np.float32)).cuda(), torch.from_numpy(u.astype(np.float32)).cuda())
        assert _state_err(o, g2, w) <= 5e-8
        g.step(3)
        rh, uh = g.get_macros_host()
        rd, ud = g.get_macros()
        assert np.array_equal(rh, rd.cpu().numpy()) and np.array_equal(uh, ud.cpu().numpy())


# ---------------------------------------------------------------------------------------------
# config 1 (BASELINE.json:configs[0]) at 1, 10, 100, 200 steps; config 2 at 100 steps
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
def test_cfg1_200_steps(orc, gpu, aa):
    cfg = wl.get("cfg1")
    o, g = _pair(orc, gpu, cfg, aa, 0)
    o.stats_accumulate(1)
    g.stats_accumulate(1)
    tol = TOL_REL * cfg["u_bulk"]
    done = 0
    for target in (1, 10, 100, 200):
        o.step(target - done)
        g.step(target - done)
        done = target
        er, eu = _macro_err(o, g)
        # north_star states the bound over 100 steps; with the momentum reference of the collision
        # arithmetic step 200 meets the same bound (measured 8e-8)
        tol_t = tol
        print(f"cfg1 {g.variant} step {target}: max|drho|={er:.3e} max|du|={eu:.3e} (tol {tol_t:.1e})")
        assert er <= tol_t and eu <= tol_t
    so, no = o.stats_read()
    sg, ng = g.stats_read()
    assert no == ng == 200
    _check_stats(sg, so, cfg["u_bulk"])
    # mass conservation on the GPU side (invariant, any size)
    assert abs(sg[:, 9].mean() - 1.0) < 1e-6


_ORACLE_CACHE = {}


def _oracle_macros_at(orc, cfg, seed, steps):
    """(rho, u) of the oracle's sample S_steps for (config, seed); computed once per session and
    shared by the storage variants (the oracle run is the expensive side)."""
    key = (cfg["name"], seed, steps)
    if key not in _ORACLE_CACHE:
        c = dict(cfg)
        c["seed"] = seed
        o = orc.Oracle.from_config(c)
        o.init_from_config(c)
        o.step(steps)
        _ORACLE_CACHE[key] = o.get_macros()
        del o
    return _ORACLE_CACHE[key]


def _gpu_err_vs(orc, gpu, cfg, seed, steps, aa):
    import torch
    ro, uo = _oracle_macros_at(orc, cfg, seed, steps)
    c = dict(cfg)
    c["seed"] = seed
    g = gpu.Lbm.from_config(c, aa=aa)
    g.init(seed)
    g.step(steps)
    rg, ug = g.get_macros()
    torch.cuda.synchronize()
    er = float((rg.double().cpu() - torch.from_numpy(ro)).abs().max())
    eu = float((ug.double().cpu() - torch.from_numpy(uo)).abs().max())
    variant = g.variant
    g.close()
    return er, eu, variant


# north_star: "Over 100 steps, the macroscopic rho and u must satisfy max|delta| <= 1e-5 relative
# to the bulk velocity".  Several seeds per config: the flow amplifies rounding differences, so
# the margin is a property of the realisation, not only of the arithmetic.
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("seed", [12345, 1, 20220630, 987654321])
def test_cfg1_100_steps_seeds(orc, gpu, aa, seed):
    cfg = wl.get("cfg1")
    tol = TOL_REL * cfg["u_bulk"]
    er, eu, variant = _gpu_err_vs(orc, gpu, cfg, seed, 100, aa)
    print(f"cfg1 {variant} seed {seed} step 100: max|drho|={er:.3e} max|du|={eu:.3e} (tol {tol:.1e})")
    assert er <= tol and eu <= tol


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("seed", [12345, 1, 20220630])
def test_cfg2_100_steps(orc, gpu, aa, seed):
    cfg = wl.get("cfg2")
    tol = TOL_REL * cfg["u_bulk"]
    er, eu, variant = _gpu_err_vs(orc, gpu, cfg, seed, 100, aa)
    print(f"cfg2 {variant} seed {seed} step 100: max|drho|={er:.3e} max|du|={eu:.3e} (tol {tol:.1e})")
    assert er <= tol and eu <= tol


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
def test_cfg3_100_steps(orc, gpu, aa):
    """BASELINE.json:configs[2]: the first config with the Lalic-Mihailovic canopy (PAPER.md:L105-115,
    Eqs. 14-15) at full width, 512x128x256.  The oracle side is ~5 GB and runs once."""
    cfg = wl.get("cfg3")
    tol = TOL_REL * cfg["u_bulk"]
    er, eu, variant = _gpu_err_vs(orc, gpu, cfg, cfg["seed"], 100, aa)
    print(f"cfg3 {variant} step 100: max|drho|={er:.3e} max|du|={eu:.3e} (tol {tol:.1e})")
    assert er <= tol and eu <= tol
    if aa:
        _ORACLE_CACHE.pop((cfg["name"], cfg["seed"], 100), None)   # 0.5 GB of fp64 fields


# ---------------------------------------------------------------------------------------------
# full-size configs in the launch configuration bench.py times: sampled sub-boxes the oracle
# can recompute one step at a time + invariants
# ---------------------------------------------------------------------------------------------
def _subbox_check(orc, gpu, cfg, aa, boxes, presteps):
    """Take GPU state k, cut sub-boxes out of it, let the oracle advance each box one step and
    compare with the GPU's state k+1 on the cells whose neighbours all lie inside the box."""
    import torch
    w = _weights(orc)
    g = gpu.Lbm.from_config(cfg, aa=aa)
    g.init(cfg["seed"])
    g.step(presteps)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    lad = gpu.lad_from_spec(cfg["forest"], ny)
    lad_o = orc.lad_from_spec(cfg["forest"], ny)
    if lad is not None:
        assert np.abs(lad - lad_o).max() <= 1e-14
    S = 8

    def cut(state, x0, y0, z0):
        xi = torch.arange(x0, x0 + S, device=state.device) % nx
        zi = torch.arange(z0, z0 + S, device=state.device) % nz
        sub = state[:, zi][:, :, y0:y0 + S][:, :, :, xi]
        return sub.cpu().numpy().astype(np.float64)

    st = g.get_state()
    before = [cut(st, *b) for b in boxes]
    del st
    g.step(1)
    st = g.get_state()
    after = [cut(st, *b) for b in boxes]
    del st
    torch.cuda.synchronize()
    worst = 0.0
    for (x0, y0, z0), fb, fa in zip(boxes, before, after):
        bottom = wl.BOUNCE_BACK
        top = cfg["top"] if y0 + S == ny else wl.BOUNCE_BACK
        o = orc.Oracle(S, S, S, cfg["nu"], cfg["Cs"], cfg["body_force"], cfg["Cd"],
                       None if lad_o is None else lad_o[y0:y0 + S], orc.bc_flags(bottom, top))
        o.set_populations(fb + w[:, None, None, None])
        o.step(1)
        fo = o.get_populations() - w[:, None, None, None]
        ylo = 0 if y0 == 0 else 1                 # real wall rows are exact, cut faces are not
        yhi = S if y0 + S == ny else S - 1
        d = np.abs(fa - fo)[:, 1:S - 1, ylo:yhi, 1:S - 1]
        worst = max(worst, float(d.max()))
    return worst, g


@pytest.mark.parametrize("name,aa", [("cfg3", False), ("cfg3", True), ("cfg4", True), ("cfg5", True),
                                     ("cfg3", "aax"), ("cfg5", "aax"), ("paper_abl_fine", "aax"),
                                     ("paper_channel", False), ("paper_channel", True),
                                     ("paper_abl_fine", False), ("paper_abl_fine", True)])
def test_full_size_sampled_boxes(orc, gpu, name, aa):
    import torch
    cfg = wl.get(name)
    free, _ = torch.cuda.mem_get_info()
    need = 76 * wl.n_cells(cfg) * (2 if aa else 3) * 1.05          # populations + the get_state copy
    if free < need:
        pytest.skip(f"{name} needs {need / 2**30:.0f} GiB of device memory")
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    h = (cfg["forest"] or {}).get("h", (cfg["forest"] or {}).get("rows", 8))
    boxes = [(0, 0, 0), (nx - 4, 0, nz - 4), (nx // 2 - 3, h - 4, nz // 3), (nx - 8, ny - 8, 0),
             (5, ny - 8, nz - 5), (nx // 3, ny // 2, nz // 2), (124, 0, 1), (nx - 5, ny // 4, nz - 3)]
    for presteps in (2, 3):                       # AA: next step is even / odd
        worst, g = _subbox_check(orc, gpu, cfg, aa, boxes, presteps)
        print(f"{name} {g.variant} presteps={presteps}: worst one-step |delta f| = {worst:.3e}")
        assert worst <= 2e-7
        # invariant at any size: mass is conserved (rho plane means average to 1)
        g.stats_accumulate(1)
        g.stats_reset()
        g.step(2)
        s, n = g.stats_read()
        assert n == 2 and abs(s[:, 9].mean() - 1.0) < 2e-6
        g.close()
        del g
        torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------------------
# forced-equilibrium lid (NEXT #1)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("nx,vec", [(64, 4), (34, 2), (33, 1)])
def test_forced_equilibrium_lid_parity(orc, gpu, aa, nx, vec):
    cfg = wl.small(nx=nx, ny=10, nz=6, top=wl.FORCED_EQ)
    cfg["U_top"] = (0.06, 0.0, 0.01)
    o, g = _pair(orc, gpu, cfg, aa, vec)
    w = _weights(orc)
    assert _state_err(o, g, w) <= 5e-8
    for n in (1, 2, 5, 12):                       # odd and even numbers of steps (AA parities)
        o.step(n)
        g.step(n)
        er, eu = _macro_err(o, g)
        assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]
    # the lid drives the top row: its mean velocity has moved towards U_top
    _, ug = g.get_macros()
    assert float(ug[0, :, -1, :].mean()) > float(ug[0, :, -3, :].mean())


def test_couette_closed_form_on_gpu(gpu):
    """P14's closed form u_j = U (j + 1/2) / (ny + tau - 1/2) reached by the CUDA path itself."""
    ny, nu, U = 12, 0.2, 0.02
    for aa in (False, True, "aax"):
        g = gpu.Lbm(8, ny, 4, nu, 0.0, flags=gpu.bc_flags("bounce_back", "forced_equilibrium", aa=aa))
        g.set_top_velocity([U, 0.0, 0.0])
        g.set_init(gpu.INIT_REST, 0.0, 0.0)
        g.init(1)
        g.step(int(6 * ny * ny / nu) + 1)
        _, u = g.get_macros()
        exact = U * (np.arange(ny) + 0.5) / (ny + 3 * nu)
        assert np.abs(u[0].cpu().numpy() - exact[None, :, None]).max() <= 2e-5 * U


# ---------------------------------------------------------------------------------------------
# per-cell solid mask (NEXT #2)
# ---------------------------------------------------------------------------------------------
def _solid_mask(kind, nx, ny, nz):
    m = np.zeros((nz, ny, nx), bool)
    if kind == "random":
        m = np.random.default_rng(21).uniform(size=m.shape) < 0.12
    elif kind == "boxes":                     # trip boxes on the ground, one across the x wrap
        m[1:4, 0:3, 5:9] = True
        m[2:5, 0:2, nx - 2:] = True
        m[2:5, 0:2, :2] = True
        m[0, 4:6, 30:34] = True               # straddles a 32-cell mask word
    elif kind == "top":
        m[:, -1, ::3] = True                  # solids in the row under the free-slip face
    return m


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("kind", ["random", "boxes", "top"])
@pytest.mark.parametrize("nx,vec", [(64, 4), (96, 4), (64, 2), (32, 1)])
def test_solid_mask_parity(orc, gpu, aa, kind, nx, vec):
    cfg = wl.small(nx=nx, ny=10, nz=6)
    cfg["solid"] = _solid_mask(kind, nx, 10, 6)
    o, g = _pair(orc, gpu, cfg, aa, vec)
    assert g.variant.startswith({False: "pull2/", True: "aa/", "aax": "aax/"}[aa])
    w = _weights(orc)
    assert _state_err(o, g, w) <= 5e-8
    o.stats_accumulate(1)
    g.stats_accumulate(1)
    g.stats_reset()
    o.stats_reset()
    for n in (1, 1, 2, 7):                    # odd and even step counts: both AA parities
        o.step(n)
        g.step(n)
        assert _state_err(o, g, w) <= 2e-7
        er, eu = _macro_err(o, g)
        assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]
    so, no = o.stats_read()
    sg, ng = g.stats_read()
    assert no == ng == 11
    _check_stats(sg, so, cfg["u_bulk"])
    rg, ug = g.get_macros()
    solid = cfg["solid"]
    assert np.all(rg.cpu().numpy()[solid] == 1.0) and np.all(ug.cpu().numpy()[:, solid] == 0.0)


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("nx,vec", [(36, 4), (70, 2), (33, 1), (100, 4)])
def test_solid_mask_on_ragged_rows(orc, gpu, aa, nx, vec):
    """nx not a multiple of 32: the mask rows are padded to whole words (the paper's own meshes are
    372, 350 and 250 cells wide)."""
    cfg = wl.small(nx=nx, ny=8, nz=5)
    m = np.random.default_rng(7).uniform(size=(5, 8, nx)) < 0.1
    m[:, 0:2, nx - 2:] = True                  # a box across the x wrap
    m[:, 0:2, :1] = True
    cfg["solid"] = m
    o, g = _pair(orc, gpu, cfg, aa, vec)
    w = _weights(orc)
    for n in (1, 2, 4):
        o.step(n)
        g.step(n)
        assert _state_err(o, g, w) <= 2e-7


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("t_change", [6, 7])
@pytest.mark.parametrize("nx,vec", [(64, 4), (36, 4), (34, 2)])
def test_solid_removed_at_run_time_keeps_the_flow(orc, gpu, aa, t_change, nx, vec):
    """spin up around trip boxes, remove them, go on.  lbm_set_solid on a running
    handle must agree with the oracle's run-time removal (pin P17) at both AA parities, for a
    partial removal, a complete one and for boxes put back (cells turning solid)."""
    cfg = wl.small(nx=nx, ny=10, nz=6)
    boxes = _solid_mask("boxes", nx, 10, 6)
    cfg["solid"] = boxes
    o, g = _pair(orc, gpu, cfg, aa, vec)
    w = _weights(orc)
    o.step(t_change)
    g.step(t_change)
    part = boxes.copy()
    part[1:4, 0:3, 5:9] = False                 # one box goes
    moved = np.zeros_like(boxes)
    moved[2:5, 3:6, 10:14] = True               # new solids in the middle of the flow, old ones gone
    moved[0, 9, ::2] = True                     # and under the free-slip face
    for mask, nsteps in ((part, 3), (None, 4), (moved, 3), (None, 20)):
        o.set_solid(mask)
        g.set_solid(mask)
        assert g.time == o.time
        assert _state_err(o, g, w) <= 2e-7      # the representation was converted, not re-initialised
        o.step(nsteps)
        g.step(nsteps)
        assert _state_err(o, g, w) <= 3e-7
        er, eu = _macro_err(o, g)
        assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]
    # the flow was kept: the freed cells carry momentum now
    _, ug = g.get_macros()
    assert float(ug[0].cpu().numpy()[boxes].std()) > 1e-4


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("nx,vec", [(64, 4), (36, 4), (34, 2), (33, 1)])
def test_forest_codes_parity(orc, gpu, aa, nx, vec):
    """Per-cell forest codes: a forest edge in x, a clearing in z, two canopy
    heights and both LAD kinds (Eq. 14 and constant), next to a solid box."""
    cfg = wl.small(nx=nx, ny=12, nz=6, forest_rows=0)
    cfg["forest_cells"] = dict(a_fm=0.35, blocks=[
        dict(x=(0, nx // 2), z=(0, 6), y0=0, h=5, y_m=3.5),
        dict(x=(nx // 2 + 3, nx), z=(1, 4), y0=0, h=3, y_m=0.0),
    ])
    cfg["solid"] = np.zeros((6, 12, nx), bool)
    cfg["solid"][2:4, 0:2, nx // 2:nx // 2 + 2] = True
    o, g = _pair(orc, gpu, cfg, aa, vec)
    w = _weights(orc)
    o.stats_accumulate(1)
    g.stats_accumulate(1)
    for n in (1, 2, 6):
        o.step(n)
        g.step(n)
        assert _state_err(o, g, w) <= 2e-7
    er, eu = _macro_err(o, g)
    assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]
    _check_stats(g.stats_read()[0], o.stats_read()[0], cfg["u_bulk"])
    # the codes matter (same run without them differs) and can be taken away again
    o2 = orc.Oracle.from_config({**cfg, "forest_cells": None})
    o2.init_from_config(cfg)
    o2.step(9)
    assert np.abs(o2.get_populations() - o.get_populations()).max() > 1e-6
    g.set_forest_codes(None)
    o.set_forest_codes(None, 0.0)
    o.step(3)
    g.step(3)
    assert _state_err(o, g, w) <= 2e-7


def test_forest_codes_need_a_geometry_handle(gpu):
    g = gpu.Lbm(32, 4, 4, 0.01, 0.1)
    with pytest.raises(gpu.LbmError) as e:
        g.set_forest_codes(np.zeros((4, 4, 32), np.uint32), 0.3)
    assert e.value.code == gpu.LBM_EINVAL
    assert gpu.forest_code(7, 3, 4.9) == 0x2701C03


# ---------------------------------------------------------------------------------------------
# CUDA-graph replay inside lbm_step: same kernels in the same order => bit-identical
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("every", [0, 1, 3, 4])
def test_graph_replay_is_bit_identical(gpu, aa, every):
    import torch
    cfg = wl.get("cfg1")
    out = []
    for mode in (0, 1):
        g = gpu.Lbm.from_config(cfg, aa=aa)
        g.set_graphs(mode)
        g.init(cfg["seed"])
        g.step(1)                               # start from an odd time step
        g.stats_accumulate(every)
        l0 = g.launch_count
        g.step(2)                               # put the sampling phase out of alignment
        g.step(203)
        g.step(77)                              # a second call reuses or rebuilds the graph
        st = g.get_state()
        s, n = g.stats_read()
        torch.cuda.synchronize()
        out.append((st.cpu().numpy(), s, n, g.time, g.launch_count - l0))
        g.close()
    (sa, ta, na, tia, la), (sb, tb, nb, tib, lbb) = out
    assert tia == tib == 283 and na == nb == (0 if every == 0 else -(-282 // every))
    assert la == lbb                             # launches replayed through a graph are counted
    assert np.array_equal(sa, sb) and np.array_equal(ta, tb)


# Sweep direction (lbm_set_sweep): the order in which the blocks visit the rows is free
# (a cell needs the previous state of adjacent cells only) => bit-identical
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("solid", [False, True], ids=["plain", "boxes"])
@pytest.mark.parametrize("nx", [64, 36, 33])
def test_sweep_direction_is_bit_identical(gpu, aa, solid, nx):
    import torch
    cfg = wl.small(nx=nx, ny=12, nz=10)
    if solid:
        m = np.zeros((cfg["nz"], cfg["ny"], cfg["nx"]), dtype=np.uint8)
        m[2:5, 0:3, 5:9] = 1
        m[7:9, 9:12, nx - 3:nx] = 1
        cfg["solid"] = m
    out = []
    for mode in (0, 1):
        g = gpu.Lbm.from_config(cfg, aa=aa, vec=4 if nx % 4 == 0 else 1)   # (the default on lattices this small is 1)
        g.set_sweep(mode)
        g.set_graphs(0)
        g.init(cfg["seed"])
        g.stats_accumulate(2)
        g.step(13)
        st = g.get_state()
        s, n = g.stats_read()
        torch.cuda.synchronize()
        out.append((st.cpu().numpy(), s, n))
        g.close()
    assert out[0][2] == out[1][2] == 7
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    with pytest.raises(gpu.LbmError):
        g2 = gpu.Lbm.from_config(cfg, aa=aa)
        try:
            g2.set_sweep(2)
        finally:
            g2.close()


# ---------------------------------------------------------------------------------------------
# Memory safety and races without compute-sanitizer (closed on this GPU pool):
#  * guard bands: the workspace sits between two regions filled with a byte pattern; no kernel of
#    any call may change a byte of them (an out-of-range store of a boundary / wrap / halo index
#    lands there or faults);
#  * run-to-run bit identity: a data race between lanes or blocks of the in-place AA update (the
#    masked push path mixes vector and element stores to neighbouring lanes' cells) shows as a
#    result that depends on scheduling.
# ---------------------------------------------------------------------------------------------
_GUARD_SHAPES = [(64, 12, 10, 4), (36, 7, 5, 4), (34, 5, 3, 2), (33, 3, 4, 1), (4, 1, 1, 4), (1, 5, 1, 1), (256, 4, 3, 4)]


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("kind", ["plain", "solid", "slab"])
def test_guard_bands_stay_untouched(gpu, aa, kind):
    import torch
    for nx, ny, nz, vec in _GUARD_SHAPES:
        if kind == "slab" and nz < 3:
            continue
        for bottom, top in BCS + [(wl.BOUNCE_BACK, wl.FORCED_EQ)]:
            cfg = wl.small(nx=nx, ny=ny, nz=nz, bottom=bottom, top=top, forest_rows=min(3, ny))
            flags = gpu.bc_flags(bottom, top, aa=aa, vec=vec, solid=(kind == "solid"), halo=(kind == "slab"))
            g = gpu.Lbm(nx, ny, nz, cfg["nu"], cfg["Cs"], cfg["body_force"], cfg["Cd"],
                        gpu.lad_from_spec(cfg["forest"], ny), flags, guard=1 << 16)
            g.set_init(0, 0.05, 0.05)
            if kind == "solid":
                rng = np.random.default_rng(nx * 131 + ny)
                g.set_solid((rng.random((nz, ny, nx)) < 0.15).astype(np.uint8))
            g.init(7)
            g.stats_accumulate(1)
            if kind == "slab":
                bufs = [g.halo_buffer() for _ in range(4)]
                for _ in range(3):
                    g.halo_pack(0, bufs[0]); g.halo_pack(1, bufs[1])
                    g.halo_unpack(0, bufs[1]); g.halo_unpack(1, bufs[0])
                    g.step(1)
                    g.step_slab_begin(bufs[0], bufs[1], None)
                    g.step_slab_end(bufs[1], bufs[0], None)
            else:
                g.set_graphs(0)
                g.step(5)
                g.set_graphs(1)
                g.step(70)
            if kind == "solid":
                g.set_solid(None)
                g.step(3)
            g.get_macros(); g.stats_read(); st = g.get_state()
            g.set_state(st, 3)
            g.step(2)
            rho = torch.empty(g.shape, dtype=torch.float32).pin_memory()
            u = torch.empty((3,) + g.shape, dtype=torch.float32).pin_memory()
            g.get_macros_host(rho, u)
            g.set_macros_host(rho, u)
            g.step(2)
            assert g.guard_intact(), (nx, ny, nz, vec, bottom, top)
            g.close()


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
def test_masked_update_is_run_to_run_bit_identical(gpu, aa):
    """Five runs of a lattice with 15 % random solids (every lane takes the element-store path
    somewhere) and of a plain one: identical to the last bit."""
    import torch
    for solid in (True, False):
        cfg = wl.small(nx=96, ny=16, nz=12)
        if solid:
            rng = np.random.default_rng(5)
            cfg["solid"] = (rng.random((12, 16, 96)) < 0.15).astype(np.uint8)
        ref = None
        for rep in range(5):
            g = gpu.Lbm.from_config(cfg, aa=aa, vec=4)
            g.set_launch_shape(*[(24, 4), (8, 16), (12, 8), (24, 8), (6, 2)][rep]) if not solid else None
            g.init(cfg["seed"])
            g.stats_accumulate(1)
            g.step(41)
            st = g.get_state().cpu().numpy()
            s, _ = g.stats_read()
            g.close()
            if ref is None:
                ref = (st, s)
            else:
                assert np.array_equal(st, ref[0])
                if solid:
                    assert np.array_equal(s, ref[1])      # same block shape: same summation order
                else:
                    assert np.allclose(s, ref[1], rtol=0, atol=1e-9)


def test_step_before_init_is_an_error(gpu):
    g = gpu.Lbm(8, 4, 4, 0.01, 0.1)
    with pytest.raises(gpu.LbmError) as e:
        g.step(1)
    assert e.value.code == gpu.LBM_ESTATE


# ---------------------------------------------------------------------------------------------
# lbm_set_state: checkpoint / restart, and pin P16 through the C ABI
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("t0", [4, 7])
@pytest.mark.parametrize("solid", [False, True])
def test_get_state_set_state_round_trip_is_bit_identical(gpu, aa, t0, solid):
    """get_state -> set_state(t) into a fresh handle -> step continues the run bit for bit."""
    import torch
    cfg = wl.small(nx=64, ny=10, nz=6)
    if solid:
        cfg["solid"] = _solid_mask("boxes", 64, 10, 6)
    a = gpu.Lbm.from_config(cfg, aa=aa)
    a.init(cfg["seed"])
    a.step(t0)
    ck = a.get_state().clone()
    a.step(5)
    want = a.get_state().cpu().numpy()
    b = gpu.Lbm.from_config(cfg, aa=aa)
    b.set_state(ck, t0)
    # the momentum reference is part of a bit-exact checkpoint (it changes rounding only)
    ref = a.get_reference_profile()
    assert np.any(ref != 0) and np.abs(ref - 0.05 * ((np.arange(10) + 0.5) / 10) ** (1 / 7)).max() < 1e-6
    b.set_reference_profile(ref)
    assert np.array_equal(b.get_reference_profile(), ref)
    assert b.time == t0
    assert np.array_equal(b.get_state().cpu().numpy(), ck.cpu().numpy())
    b.step(5)
    torch.cuda.synchronize()
    assert b.time == a.time and np.array_equal(b.get_state().cpu().numpy(), want)
    ra, ua = a.get_macros()
    rb, ub = b.get_macros()
    assert torch.equal(ra, rb) and torch.equal(ua, ub)


@pytest.mark.parametrize("aa", [False, "aax"], ids=["pull2", "aax"])
def test_checkpoint_file_restart_is_bit_identical(gpu, aa, tmp_path):
    """save_checkpoint / load_checkpoint (lbm_get_state, lbm_set_state through a file): the restarted
    run continues exactly like the uninterrupted one, from an odd and from an even time step."""
    import torch
    cfg = wl.small(nx=36, ny=10, nz=6)
    a = gpu.Lbm.from_config(cfg, aa=aa, vec=4)
    a.init(11)
    for t_save in (7, 20):
        a.step(t_save - a.time)
        path = str(tmp_path / f"ck{t_save}.pt")
        a.save_checkpoint(path)
        b = gpu.Lbm.from_config(cfg, aa=aa, vec=4)
        b.load_checkpoint(path)
        assert b.time == t_save
        a.step(9)
        b.step(9)
        torch.cuda.synchronize()
        assert torch.equal(a.get_state(), b.get_state())
        b.close()
    c = gpu.Lbm.from_config(wl.small(nx=32, ny=10, nz=6), aa=aa)
    with pytest.raises(ValueError):
        c.load_checkpoint(path)
    c.close(); a.close()


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("t0", [0, 1])
def test_p16_known_pi_neq_through_the_c_abi(orc, gpu, aa, t0):
    """Pin P16 (tests/test_oracle_pins.py) on the CUDA path: a periodic uniform state with a known
    Pi_neq = A relaxes by (1 - 1/tau_t) in one step (Eq. 11).  t0 selects
    the AA parity (even step / odd step kernel)."""
    import torch
    c, w, _, _ = orc.tables()
    c = c.astype(float)
    rng = np.random.default_rng(61)
    nx, ny, nz = 32, 4, 3
    flags = gpu.bc_flags("periodic", "periodic", aa=aa, vec=4)
    for trial in range(6):
        B = rng.normal(size=(3, 3))
        A = 0.5 * (B + B.T)
        A -= np.trace(A) / 3 * np.eye(3)
        A *= 3e-3 / np.sqrt(np.sum(A * A))
        rho = rng.uniform(0.93, 1.07)
        u = rng.uniform(-0.1, 0.1, 3) + np.array([0.05, 0.0, 0.0])
        nu, Cs = 10 ** rng.uniform(-4, -2.5), 0.17
        tau0 = 3 * nu + 0.5
        cu = c @ u
        feq = w * rho * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * (u @ u))
        fneq = w * 4.5 * np.einsum("iab,ab->i", np.einsum("ia,ib->iab", c, c) - np.eye(3) / 3, A)
        tau_t = 0.5 * (tau0 + np.sqrt(tau0 ** 2 + 18 * np.sqrt(2) * Cs ** 2 * np.sqrt(np.sum(A * A)) / rho))
        want = feq + (1 - 1 / tau_t) * fneq - w
        g = gpu.Lbm(nx, ny, nz, nu, Cs, flags=flags)
        st = torch.from_numpy(np.broadcast_to((feq + fneq - w)[:, None, None, None], (19, nz, ny, nx))
                              .astype(np.float32).copy()).cuda()
        g.set_state(st, t0)
        g.step(1)
        got = g.get_state().double().cpu().numpy()
        err = np.abs(got - want[:, None, None, None]).max()
        teeth = np.abs((1 / tau0 - 1 / tau_t) * fneq).max()
        assert err <= 3e-8 and teeth > 30 * 3e-8, (err, teeth)
        g.close()


# ---------------------------------------------------------------------------------------------
# Row-table SGS models (lbm_set_sgs_rows, pin P19)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("t0", [0, 1])
def test_p19_row_tables_through_the_c_abi(orc, gpu, aa, t0):
    """Pin P19 on the CUDA path: a periodic uniform state with a known Pi_neq relaxes, row by row,
    by (1 - 1/tau_j) with tau_j from the DEFINITION of the closure iterated to its fixed point
    (damped constant, mean shear, clipped rows); then back to the standard model."""
    import torch
    c, w, _, _ = orc.tables()
    c = c.astype(float)
    rng = np.random.default_rng(191)
    nx, ny, nz = 32, 6, 3
    flags = gpu.bc_flags("periodic", "periodic", aa=aa, vec=4)
    B = rng.normal(size=(3, 3))
    A = 0.5 * (B + B.T)
    A -= np.trace(A) / 3 * np.eye(3)
    A *= 3e-3 / np.sqrt(np.sum(A * A))
    rho, u, nu, Cs = 1.04, np.array([0.08, -0.03, 0.02]), 3e-4, 0.17
    tau0 = 3 * nu + 0.5
    Qh = np.sqrt(np.sum(A * A))
    S_now = 3.0 * Qh / (np.sqrt(2.0) * rho * tau0)
    C_row = Cs ** 2 * np.array([0.0, 0.25, 1.0, 1.0, 2.0, 0.6])
    S_row = S_now * np.array([0.0, 0.0, 0.5, 3.0, 0.9, 0.2])
    cu = c @ u
    feq = w * rho * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * (u @ u))
    fneq = w * 4.5 * np.einsum("iab,ab->i", np.einsum("ia,ib->iab", c, c) - np.eye(3) / 3, A)

    def tau_def(Cj, Sj):
        tau = tau0
        for _ in range(200):
            tau = tau0 + 3.0 * Cj * max(3.0 * Qh / (np.sqrt(2.0) * rho * tau) - Sj, 0.0)
        return tau

    g = gpu.Lbm(nx, ny, nz, nu, Cs, flags=flags)
    st = torch.from_numpy(np.broadcast_to((feq + fneq - w)[:, None, None, None], (19, nz, ny, nx))
                          .astype(np.float32).copy()).cuda()
    for tables in ((C_row, S_row), (C_row, None), (None, S_row), (None, None)):
        g.set_sgs_rows(*tables)
        g.set_state(st, t0)
        g.step(1)
        got = g.get_state().double().cpu().numpy()
        taus = []
        for j in range(ny):
            tau_j = tau_def(Cs ** 2 if tables[0] is None else C_row[j], 0.0 if tables[1] is None else S_row[j])
            taus.append(tau_j)
            want = feq + (1 - 1 / tau_j) * fneq - w
            assert np.abs(got[:, :, j, :] - want[:, None, None]).max() <= 3e-8, (tables, j)
        if tables[0] is not None and tables[1] is not None:
            assert taus[3] == tau0 and taus[0] == tau0 and taus[2] > taus[4] > tau0     # clipped / active rows
            assert np.abs((1 / taus[2] - 1 / tau0) * fneq).max() > 20 * 3e-8           # the test has teeth
    with pytest.raises(gpu.LbmError):
        g.set_sgs_rows(-C_row, None)
    g.close()


@pytest.mark.parametrize("aa", [False, True, "aax"], ids=["pull2", "aa", "aax"])
@pytest.mark.parametrize("nx,vec", [(64, 4), (34, 2), (33, 1)])
@pytest.mark.parametrize("model", ["damped", "shear_improved"])
def test_sgs_row_models_parity(orc, gpu, aa, nx, vec, model):
    """Wall-damped and shear-improved Smagorinsky on a forced forest half-channel: 20 steps with
    statistics, populations and plane statistics against the oracle.  The shear-improved table is
    built from each side's own statistics of the first 10 steps (helper against helper too)."""
    import torch
    cfg = wl.small(nx=nx, ny=12, nz=8, Cs=0.17)
    o, g = _pair(orc, gpu, cfg, aa, vec)
    w = _weights(orc)
    o.stats_accumulate(1); g.stats_accumulate(1)
    if model == "damped":
        Co = orc.sgs_van_driest(12, 0.17, 0.004, cfg["nu"], 26.0)
        Cg = gpu.sgs_van_driest(12, 0.17, 0.004, cfg["nu"], 26.0)
        assert np.allclose(Co, Cg, rtol=1e-13, atol=0)
        o.set_sgs_rows(Co, None); g.set_sgs_rows(Cg, None)
        o.step(20); g.step(20)
    else:
        o.step(10); g.step(10)
        so, _ = o.stats_read()
        sg, _ = g.stats_read()
        So, Sg = orc.sgs_mean_shear(so, top_wall=False), gpu.sgs_mean_shear(sg, top_wall=False)
        assert np.abs(So - Sg).max() <= 1e-5 * cfg["u_bulk"] and So.max() > 1e-3
        # scaled down so that the closure is active on some rows and clipped on others
        o.set_sgs_rows(None, 0.02 * So); g.set_sgs_rows(None, 0.02 * So)
        o.step(10); g.step(10)
    assert _state_err(o, g, w) <= 2e-7
    er, eu = _macro_err(o, g)
    assert er <= TOL_REL * cfg["u_bulk"] and eu <= TOL_REL * cfg["u_bulk"]
    so, n1 = o.stats_read()
    sg, n2 = g.stats_read()
    assert n1 == n2 == 20
    assert np.abs(sg[:, :3] - so[:, :3]).max() <= TOL_REL * cfg["u_bulk"]
    # the model really acted: the standard model gives a different state
    o2, g2 = _pair(orc, gpu, cfg, aa, vec)
    g2.step(20)
    torch.cuda.synchronize()
    assert float((g2.get_state() - g.get_state()).abs().max()) > 1e-6
    g.close(); g2.close()


def test_divergence_is_reported(gpu):
    """A deliberately unstable run (nu = 1e-6, Cs = 0, large noise at Ma ~ 0.5) blows up; the
    library must say so: LBM_EDIVERGED from get_macros_host / stats_read, lbm_diverged() true."""
    for aa in (False, True):
        g = gpu.Lbm(32, 16, 16, 1e-6, 0.0, body_force=(1e-3, 0, 0),
                    flags=gpu.bc_flags("bounce_back", "free_slip", aa=aa))
        g.set_init(gpu.INIT_POWER_LAW, 0.3, 1.5)
        g.init(3)
        assert not g.diverged()
        g.stats_accumulate(1)
        for _ in range(40):
            g.step(50)
            g.get_macros()
            if g.diverged():
                break
        assert g.diverged()
        with pytest.raises(gpu.LbmError) as e:
            g.get_macros_host()
        assert e.value.code == gpu.LBM_EDIVERGED
        with pytest.raises(gpu.LbmError) as e:
            g.stats_read()
        assert e.value.code == gpu.LBM_EDIVERGED
        g.init(3)                                  # re-initialising clears the flag
        assert not g.diverged()
        g.close()


def test_chunked_host_transfers(orc, gpu, monkeypatch):
    """Host transfers through a staging area smaller than the lattice (forced with
    LBM_STAGING_BYTES): every row of every chunk is initialised and read back, also when the
    block covers several rows (TY > 1)."""
    monkeypatch.setenv("LBM_STAGING_BYTES", str(16 * 16 * 12 * 3))       # 3 planes of 16 x 12
    cfg = wl.small(nx=16, ny=12, nz=10)
    o = orc.Oracle.from_config(cfg)
    rho, u = o.init_field(cfg["init"]["kind"], cfg["init"]["U_ref"], cfg["init"]["noise_frac"], 5)
    o.set_macros(rho, u)
    w = _weights(orc)
    for aa in (False, True):
        g = gpu.Lbm.from_config(cfg, aa=aa)
        assert "x" in g.variant and int(g.variant.split("x")[-1]) > 1    # several rows per block
        with pytest.raises(gpu.LbmError):
            g.set_launch_shape(4, 8)                                      # 8 does not divide ny = 12
        g.set_macros_host(rho.astype(np.float32), u.astype(np.float32))
        assert _state_err(o, g, w) <= 5e-8
        rh, uh = g.get_macros_host()
        rd, ud = g.get_macros()
        assert np.array_equal(rh, rd.cpu().numpy()) and np.array_equal(uh, ud.cpu().numpy())
        g.close()


# ---------------------------------------------------------------------------------------------
# TMA data path (lbm_tma.cuh) against the per-thread path: same arithmetic => identical bits
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("aa", [False, True], ids=["pull2", "aa"])
@pytest.mark.parametrize("rows", [1, 2, 4])
@pytest.mark.parametrize("nx", [256, 768])
@pytest.mark.parametrize("bottom,top", BCS + [(wl.BOUNCE_BACK, wl.FORCED_EQ)],
                         ids=["wall-slip", "wall-wall", "periodic", "wall-lid"])
def test_tma_path_is_bit_identical_to_the_per_thread_path(orc, gpu, aa, rows, nx, bottom, top):
    import torch
    cfg = wl.small(nx=nx, ny=8, nz=5, bottom=bottom, top=top)
    if top == wl.FORCED_EQ:
        cfg["U_top"] = (0.06, 0.0, 0.01)
    a = gpu.Lbm.from_config(cfg, aa=aa, vec=4)       # (lattices this small default to 1 cell per thread)
    b = gpu.Lbm.from_config(cfg, aa=aa, vec=4)
    a.set_tma(0)
    b.set_tma(7, rows)
    assert "tma" not in a.variant and f"tma7x{rows}" in b.variant
    for g in (a, b):
        g.init(cfg["seed"])
        g.stats_accumulate(1)
    for n in (1, 1, 2, 5):
        a.step(n)
        b.step(n)
        torch.cuda.synchronize()
        assert torch.equal(a.get_state(), b.get_state()), n
    sa, na = a.stats_read()
    sb, nb = b.stats_read()
    assert na == nb == 9
    _check_stats(sb, sa, cfg["u_bulk"])
    # and against the oracle
    o = orc.Oracle.from_config(cfg)
    o.init_from_config(cfg)
    o.step(9)
    assert _state_err(o, b, _weights(orc)) <= 2e-7


def test_tma_is_refused_where_it_cannot_run(gpu):
    v4 = gpu.bc_flags("bounce_back", "bounce_back", vec=4)
    g = gpu.Lbm(64, 4, 4, 0.01, 0.1, flags=v4)
    with pytest.raises(gpu.LbmError) as e:
        g.set_tma(2)
    assert e.value.code == gpu.LBM_EINVAL
    g.set_tma(0)
    g = gpu.Lbm(256, 6, 4, 0.01, 0.1, flags=v4)
    with pytest.raises(gpu.LbmError):
        g.set_tma(7, 4)                      # 4 rows do not divide ny = 6
    g.set_tma(7, 2)
