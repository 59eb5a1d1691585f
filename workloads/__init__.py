"""Seeded synthetic workloads shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no equilibrium, no collision, no LAD
formula, no random-number generator): it only names the problem parameters.  The oracle
(`oracle/`) and the CUDA library (`paper_2206_15454_b200/`) each turn these parameters into
their own `lad_profile` table and their own initial field; neither imports the other.

The five `CONFIGS` stand in for the paper's two flow cases (turbulent channel, PAPER.md:L167-192
§IV Table I; forest ABL, §V.A Table II) with the lattice sizes of
BASELINE.json:configs[0..4]; the body-force values are the derivations of SURVEY.md §8(d)
(the configs give only targets).  `PAPER_SIZED` are the paper's own lattice shapes
(SURVEY.md §8(f) NEXT #3).
"""
from __future__ import annotations

import copy

DEFAULT_SEED = 12345

# Boundary names (each side maps them to its own bc_flags constants).
BOUNCE_BACK = "bounce_back"      # halfway bounce-back no-slip wall
FREE_SLIP = "free_slip"          # specular reflection (BASELINE.json:configs[0,2,3,4])
PERIODIC = "periodic"            # periodic in y (used by the closed-form pins only)
FORCED_EQ = "forced_equilibrium" # paper's ABL top boundary - NEXT #1

# Initial-profile kinds
INIT_POWER_LAW = 0   # U_ref * ((j+1/2)/ny)^(1/7)
INIT_PARABOLA = 1    # U_ref * 4 eta (1-eta), eta = (j+1/2)/ny
INIT_REST = 2        # u = 0 (noise still applies if noise_frac > 0)


def _cfg(name, nx, ny, nz, nu, Cs, Fx, Cd, bottom, top, forest, init_kind, U_ref, noise_frac,
         u_bulk, steps, storage="two_lattice", stats_every=0, note=""):
    return dict(
        name=name, nx=nx, ny=ny, nz=nz, nu=nu, Cs=Cs, body_force=(Fx, 0.0, 0.0), Cd=Cd,
        bottom=bottom, top=top, drag_vector=False, forest=forest,
        init=dict(kind=init_kind, U_ref=U_ref, noise_frac=noise_frac),
        seed=DEFAULT_SEED, u_bulk=u_bulk, steps=steps, storage=storage,
        stats_every=stats_every, note=note,
    )


# forest spec: None | {"kind": "uniform", "a": a, "rows": r} | {"kind": "lalic", "h": h, "LAI": L, "eta_m": 0.7}
CONFIGS = {
    # BASELINE.json:configs[0]
    "cfg1": _cfg("cfg1", 64, 32, 32, 1e-4, 0.1, 3.0e-6, 0.2, BOUNCE_BACK, FREE_SLIP,
                 dict(kind="uniform", a=0.1, rows=4), INIT_POWER_LAW, 0.05, 0.05,
                 u_bulk=0.05, steps=200, note="forest half-channel, oracle-sized"),
    # BASELINE.json:configs[1]; F = u_tau^2/H, H = 64, u_tau = 180 nu / H (Eq. 16)
    "cfg2": _cfg("cfg2", 256, 128, 128, 2e-4, 0.1, 4.9438e-9, 0.0, BOUNCE_BACK, BOUNCE_BACK,
                 None, INIT_PARABOLA, 0.050625, 0.10,
                 u_bulk=0.050625, steps=2000, storage="aax", stats_every=1,
                 note="plane channel, nominal Re_tau=180, single-array AA pattern (x-balanced)"),
    # BASELINE.json:configs[2]
    "cfg3": _cfg("cfg3", 512, 128, 256, 1e-4, 0.1, 3.968e-7, 0.15, BOUNCE_BACK, FREE_SLIP,
                 dict(kind="lalic", h=16, LAI=2.0, eta_m=0.7), INIT_POWER_LAW, 0.08, 0.05,
                 u_bulk=0.08, steps=2000, note="forest ABL, h=16"),
    # BASELINE.json:configs[3]
    "cfg4": _cfg("cfg4", 1024, 256, 512, 1e-4, 0.1, 1.984e-7, 0.15, BOUNCE_BACK, FREE_SLIP,
                 dict(kind="lalic", h=32, LAI=2.0, eta_m=0.7), INIT_POWER_LAW, 0.08, 0.05,
                 u_bulk=0.08, steps=1000, storage="aax", stats_every=1,
                 note="large forest ABL, h=32, single-array AA pattern (x-balanced)"),
    # BASELINE.json:configs[4]
    "cfg5": _cfg("cfg5", 1536, 384, 1024, 1e-4, 0.1, 1.323e-7, 0.15, BOUNCE_BACK, FREE_SLIP,
                 dict(kind="lalic", h=48, LAI=2.0, eta_m=0.7), INIT_POWER_LAW, 0.08, 0.05,
                 u_bulk=0.08, steps=500, storage="aax", stats_every=1,
                 note="HBM-filling forest ABL, h=48, single-array AA pattern (x-balanced)"),
}

# The paper's own lattice shapes and cases.
# Channel: Table I in lattice units, nu_lat = nu dt/dx^2 = 31^2/3250 * 1e-3, F_lat = F dt^2/dx
# (PAPER.md:L185-192); C_smag = 0.01.
# ABL: 1000 x 400 x 800 m, h = 20 m, no-slip ground, periodic x/z, forced-
# equilibrium top moving with the free stream (L216), body force in the whole domain.  Table II:
# case 1 a_f = 0.215 per metre (constant), case 2 Eq. 14 with z_m = 0.7 h and a_fm = 0.38 per metre,
# case 3 no forest.  Table III meshes: 200x80x160, 250x100x200, 350x140x280 (dx = 5, 4, 20/7 m, so
# h = 4, 5, 7 cells); LAD per lattice length = LAD per metre * dx.  The paper's body-force number is
# garbled (L216, R22): F is the SURVEY.md §8(d) balance F (ny - h) = (U_top/12)^2.
def abl_case(name, nx, ny, nz, h, case, note):
    """One of the paper's ABL cases (Table II) on an nx x ny x nz mesh with a canopy of h cells."""
    dx = 1000.0 / nx
    forest = {1: dict(kind="eq14", h=h, a_fm=0.215 * dx, eta_m=0.0),
              2: dict(kind="eq14", h=h, a_fm=0.38 * dx, eta_m=0.7),
              3: None}[case]
    U = 0.08
    c = _cfg(name, nx, ny, nz, 1e-4, 0.1, (U / 12.0) ** 2 / (ny - h), 0.15, BOUNCE_BACK, FORCED_EQ, forest,
             INIT_POWER_LAW, U, 0.05, u_bulk=U, steps=200, note=note)
    c["U_top"] = (U, 0.0, 0.0)
    c["h"] = h
    c["case"] = case
    return c


PAPER_SIZED = {
    "paper_channel": _cfg("paper_channel", 372, 62, 124, 2.9569230769230769e-4, 0.1,
                          9.2566e-8, 0.0, BOUNCE_BACK, BOUNCE_BACK, None, INIT_PARABOLA,
                          0.06, 0.10, u_bulk=0.04, steps=200,
                          note="PAPER.md:L171 (x=372,y=62,z=124), Table I"),
    "paper_abl_fine": _cfg("paper_abl_fine", 350, 140, 280, 1e-4, 0.1, 1.0e-7, 0.15,
                           BOUNCE_BACK, FREE_SLIP, dict(kind="uniform", a=0.215 * 1000.0 / 350.0, rows=7),
                           INIT_POWER_LAW, 0.08, 0.05, u_bulk=0.08, steps=200,
                           note="PAPER.md:L244 Table III fine mesh, Table II case 1 (a_f=0.215/m, h=7 cells), free-slip top"),
    "paper_abl_fine_case1": abl_case("paper_abl_fine_case1", 350, 140, 280, 7, 1,
                                 "Table III fine mesh, Table II case 1 (constant LAD 0.215/m), forced-equilibrium top"),
    "paper_abl_fine_case2": abl_case("paper_abl_fine_case2", 350, 140, 280, 7, 2,
                                 "Table III fine mesh, Table II case 2 (Eq. 14, z_m=0.7h, a_fm=0.38/m)"),
    "paper_abl_fine_case3": abl_case("paper_abl_fine_case3", 350, 140, 280, 7, 3,
                                 "Table III fine mesh, Table II case 3 (no forest)"),
    "paper_abl_medium": abl_case("paper_abl_medium", 250, 100, 200, 5, 2, "Table III medium mesh 250x100x200, case 2"),
    "paper_abl_coarse": abl_case("paper_abl_coarse", 200, 80, 160, 4, 2, "Table III coarse mesh 200x80x160, case 2"),
}


def abl_case_small(case: int, nx=48, ny=28, nz=24, h=7, seed=DEFAULT_SEED) -> dict:
    """An oracle-sized ABL of the paper's structure (Table II case 1, 2 or 3; h = 7 cells as on the
    fine mesh, dx of the fine mesh) for the qualitative checks of PAPER.md:L283-305."""
    c = abl_case(f"abl_small_case{case}", nx, ny, nz, h, case, "oracle-sized Table II case")
    dx = 1000.0 / 350.0
    if c["forest"] is not None:
        c["forest"]["a_fm"] = (0.215 if case == 1 else 0.38) * dx
    c["nu"] = 1e-3
    c["seed"] = seed
    return c


def get(name: str) -> dict:
    """Deep copy of a named config (so callers may edit it)."""
    table = CONFIGS if name in CONFIGS else PAPER_SIZED
    return copy.deepcopy(table[name])


def small(nx=32, ny=12, nz=8, *, bottom=BOUNCE_BACK, top=FREE_SLIP, nu=1e-3, Cs=0.1,
          Fx=2e-6, Cd=0.2, forest_rows=3, forest_a=0.1, init_kind=INIT_POWER_LAW,
          U_ref=0.05, noise_frac=0.05, seed=DEFAULT_SEED, drag_vector=False) -> dict:
    """A tiny forest half-channel for tests; same structure as cfg1."""
    forest = dict(kind="uniform", a=forest_a, rows=forest_rows) if forest_rows > 0 else None
    c = _cfg("small", nx, ny, nz, nu, Cs, Fx, Cd, bottom, top, forest, init_kind, U_ref,
             noise_frac, u_bulk=U_ref, steps=20)
    c["seed"] = seed
    c["drag_vector"] = drag_vector
    return c


def n_cells(cfg: dict) -> int:
    return cfg["nx"] * cfg["ny"] * cfg["nz"]
