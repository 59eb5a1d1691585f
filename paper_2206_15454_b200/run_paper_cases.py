#!/usr/bin/env python
"""Run the paper's ABL cases (Table II) on the GPU and write the normalised
profiles the paper plots: <u>/u_* (Fig. 10) and the stresses / u_*^2 (Fig. 11), with
u_* = [<u'v'>^2 + <v'w'>^2]^(1/4) at y/h = 2 (L210).

    python -m paper_2206_15454_b200.run_paper_cases [--mesh fine|medium|coarse|small]
           [--spinup N] [--window M] [--out report.md] [--boxes] [--sgs standard|damped|shear]

Everything is computed by the CUDA library through its C ABI (lbm_step, lbm_stats_read,
lbm_forest_friction_velocity, lbm_stats_normalise); this script only sequences the calls and
formats the table.  --boxes spins the flow up around 20-cell trip boxes near the inlet and removes
them at run time before the averaging window (L226).  The comparison data of the paper's figures
(field measurements, FVM LES) are not available here; what the text itself states is checked and
reported: the near-ground velocity gradient of case 3 (no forest) exceeds that of cases 1 and 2
(L289), and cases 1 and 2 differ only slightly (L305).  --sgs runs the same cases with one of the
row-table SGS models (L307 "other SGS models"; lbm_set_sgs_rows): `damped` = van Driest wall damping
of the Smagorinsky constant with u_tau = U_top / 12 (the balance the body force is derived from),
`shear` = shear-improved Smagorinsky, the mean-shear table rebuilt from the running statistics every
--refresh steps.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402  (problem parameters only)

MESH = {"fine": "paper_abl_fine", "medium": "paper_abl_medium", "coarse": "paper_abl_coarse"}


def case_config(mesh: str, case: int) -> dict:
    if mesh == "small":
        return wl.abl_case_small(case)
    base = wl.get(MESH[mesh] + ("_case2" if mesh == "fine" else ""))
    cfg = wl.abl_case(f"{MESH[mesh]}_case{case}", base["nx"], base["ny"], base["nz"], base["h"], case,
                  f"Table III {mesh} mesh, Table II case {case}")
    return cfg


def trip_boxes(cfg: dict) -> np.ndarray:
    """A spanwise row of cubic trip boxes near the inlet (L226: "a set of small boxes are set near
    the inlet"; size 20 non-dimensional units, taken as cells, capped at a quarter of the height)."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    b = max(2, min(20, ny // 4))
    m = np.zeros((nz, ny, nx), bool)
    x0 = max(1, nx // 20)
    for z0 in range(b // 2, nz - b, 3 * b):
        m[z0:z0 + b, 0:b, x0:x0 + b] = True
    return m


def advance(lb, sim, n: int, sgs: str, refresh: int, top_wall: bool):
    """n steps; with the shear-improved model the mean-shear table follows the running statistics."""
    if sgs != "shear":
        sim.step(n)
        return
    done = 0
    while done < n:
        k = min(refresh, n - done)
        sim.step(k)
        done += k
        st, ns = sim.stats_read()
        if ns > 0:
            sim.set_sgs_rows(None, lb.sgs_mean_shear(st, top_wall=top_wall))


def run_case(lb, cfg: dict, spinup: int, window: int, boxes: bool, device="cuda:0", sgs="standard", refresh=500):
    """(stats [ny][10], u_star, MLUPS) of one case."""
    import torch

    c = dict(cfg)
    if boxes:
        c["geometry"] = True
    sim = lb.Lbm.from_config(c, aa="aax", device=device)    # single array, x-balanced AA (geometry handles too)
    if boxes:
        sim.set_solid(trip_boxes(cfg))
    sim.init(cfg["seed"])
    top_wall = cfg["top"] == wl.BOUNCE_BACK
    if sgs == "damped":
        u_tau = cfg["init"]["U_ref"] / 12.0
        sim.set_sgs_rows(lb.sgs_van_driest(cfg["ny"], cfg["Cs"], u_tau, cfg["nu"], 26.0, both_walls=top_wall), None)
    if sgs == "shear":
        sim.stats_accumulate(1)                   # the spin-up statistics feed the first tables
    advance(lb, sim, spinup, sgs, refresh, top_wall)
    if boxes:
        sim.set_solid(None)                       # the boxes are removed, the flow is kept (L226)
        advance(lb, sim, max(1, spinup // 4), sgs, refresh, top_wall)
    if sgs == "shear":
        st, ns = sim.stats_read()
        sim.set_sgs_rows(None, lb.sgs_mean_shear(st, top_wall=top_wall))
    sim.stats_accumulate(1)
    sim.stats_reset()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    if sgs == "shear":
        # the table is frozen inside a refresh interval and follows the window's own running mean
        advance(lb, sim, window, sgs, refresh, top_wall)
    else:
        sim.step(window)
    st, n = sim.stats_read()
    dt = time.perf_counter() - t0
    assert n == window
    try:
        u_star = lb.forest_friction_velocity(st, cfg["h"])
    except lb.LbmError:
        u_star = float("nan")
    sim.close()
    return st, u_star, wl.n_cells(cfg) * window / dt / 1e6


def near_ground_gradient(st: np.ndarray, h: int) -> float:
    """Mean d<u>/dy over the canopy layer 0 <= y <= h (lattice units)."""
    return float((st[h, 0] - st[0, 0]) / h)


def text_checks(stats: dict, h: int) -> dict:
    """What the paper's text fixes (L283-305), as numbers."""
    g = {k: near_ground_gradient(s, h) for k, s in stats.items()}
    u = {k: s[:, 0] for k, s in stats.items()}
    top = max(float(np.abs(u[3]).max()), 1e-30)
    d12 = float(np.abs(u[1] - u[2]).max()) / top
    d13 = float(np.abs(u[1] - u[3]).max()) / top
    return {"gradient": g, "case3_gradient_largest": g[3] > g[1] and g[3] > g[2],
            "near_ground_u": {k: float(u[k][:h].mean()) for k in u},
            "case3_near_ground_u_largest": u[3][:h].mean() > u[1][:h].mean() and u[3][:h].mean() > u[2][:h].mean(),
            "max_diff_case1_case2": d12, "max_diff_case1_case3": d13,
            "cases_1_2_differ_slightly": d12 < 0.5 * d13}


def report(mesh, cfgs, stats, ustar, mlups, checks, lb) -> str:
    h = cfgs[1]["h"]
    ny = cfgs[1]["ny"]
    out = [f"# ABL cases of Table II on the {mesh} mesh ({cfgs[1]['nx']}x{ny}x{cfgs[1]['nz']}, h = {h} cells)", ""]
    out.append("| case | u_* (L210, y/h = 2) | d<u>/dy over the canopy | mean <u> below h | MLUPS |")
    out.append("|---|---|---|---|---|")
    for k in (1, 2, 3):
        out.append(f"| {k} | {ustar[k]:.4e} | {checks['gradient'][k]:.4e} | {checks['near_ground_u'][k]:.4e} | {mlups[k]:.0f} |")
    out += ["", f"* case 3 has the largest near-ground gradient (L289): **{checks['case3_gradient_largest']}**",
            f"* case 3 has the largest near-ground velocity (L283-285): **{checks['case3_near_ground_u_largest']}**",
            f"* cases 1 and 2 differ only slightly (L305): max |<u>_1 - <u>_2| / max <u>_3 = "
            f"{checks['max_diff_case1_case2']:.3f} against {checks['max_diff_case1_case3']:.3f} for cases 1 and 3: "
            f"**{checks['cases_1_2_differ_slightly']}**", ""]
    out.append("Normalised profiles (rows up to 3h): y/h, then per case <u>/u_*, u_rms/u_*, v_rms/u_*, <u'v'>/u_*^2")
    out.append("")
    out.append("| y/h | " + " | ".join(f"c{k} <u>/u* | c{k} u_rms/u* | c{k} v_rms/u* | c{k} uv/u*^2" for k in (1, 2, 3)) + " |")
    out.append("|---|" + "---|" * 12)
    norm = {}
    for k in (1, 2, 3):
        ur = ustar[k] if np.isfinite(ustar[k]) and ustar[k] > 0 else 1.0
        norm[k] = lb.stats_normalise(stats[k], ur)
    for j in range(min(ny, 3 * h)):
        row = [f"{(j + 0.5) / h:.3f}"]
        for k in (1, 2, 3):
            n = norm[k][j]
            row += [f"{n[0]:.3f}", f"{n[3]:.3f}", f"{n[4]:.3f}", f"{n[6]:.3f}"]
        out.append("| " + " | ".join(row) + " |")
    return "\n".join(out) + "\n"


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--mesh", choices=["fine", "medium", "coarse", "small"], default="fine")
    ap.add_argument("--spinup", type=int, default=6000)
    ap.add_argument("--window", type=int, default=4000)
    ap.add_argument("--boxes", action="store_true", help="spin up around trip boxes, remove them at run time (L226)")
    ap.add_argument("--sgs", choices=["standard", "damped", "shear"], default="standard",
                    help="SGS closure: the paper's Smagorinsky model, or a row-table model (L307)")
    ap.add_argument("--refresh", type=int, default=500, help="--sgs shear: steps between mean-shear table updates")
    ap.add_argument("--out", default=None, help="write the markdown report here (default: stdout)")
    args = ap.parse_args()

    import paper_2206_15454_b200 as lb

    cfgs = {k: case_config(args.mesh, k) for k in (1, 2, 3)}
    stats, ustar, mlups = {}, {}, {}
    for k in (1, 2, 3):
        stats[k], ustar[k], mlups[k] = run_case(lb, cfgs[k], args.spinup, args.window, args.boxes,
                                                sgs=args.sgs, refresh=args.refresh)
    checks = text_checks(stats, cfgs[1]["h"])
    text = report(args.mesh, cfgs, stats, ustar, mlups, checks, lb)
    text += (f"\nRun: spin-up {args.spinup} steps, window {args.window} steps, trip boxes: {args.boxes}; "
             f"SGS model: {args.sgs}; single-array AA storage, statistics every step.\n")
    if args.out:
        os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
        with open(args.out, "w") as f:
            f.write(text)
    else:
        print(text)
    return 0 if (checks["case3_gradient_largest"] and checks["cases_1_2_differ_slightly"]) else 1


if __name__ == "__main__":
    sys.exit(main())
