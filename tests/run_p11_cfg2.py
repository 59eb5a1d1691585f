#!/usr/bin/env python
"""P11 at full length: config 2 (256x128x128 plane channel), spin-up then a statistics window, on
the CUDA path and on the fp64 oracle from the same seeded field; plus a second CUDA run from
another seed as the sampling-noise floor (SURVEY.md §7 hard part 11).

Not a pytest test (the oracle side takes about an hour on 16 cores):
    python tests/run_p11_cfg2.py [--spin 20000] [--window 20000] [--storage aax|aa|two_lattice]
                                 [--out gpurun_out/p11_cfg2.md]
The report is rewritten every `--every` window steps so that a cut-off run still leaves numbers.
north_star bar: plane-averaged mean within 2 %, Reynolds stresses within 5 % (of the profile maxima).
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import paper_2206_15454_b200 as lb  # noqa: E402
import workloads as wl  # noqa: E402

NAMES = ["<u>", "<v>", "<w>", "<u'u'>", "<v'v'>", "<w'w'>", "<u'v'>", "<v'w'>", "<u'w'>", "<rho>"]


def diffs(a, b):
    """max over y of |a-b| per column, normalised by the column's profile maximum in b."""
    out = []
    for k in range(9):
        m = np.abs(b[:, k]).max()
        out.append((float(np.abs(a[:, k] - b[:, k]).max() / m) if m > 0 else 0.0, float(m)))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--spin", type=int, default=20000)
    ap.add_argument("--window", type=int, default=20000)
    ap.add_argument("--every", type=int, default=2500)
    ap.add_argument("--storage", choices=["aax", "aa", "two_lattice"], default=None,
                    help="storage scheme of the CUDA runs (default: the config's)")
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "p11_cfg2.md"))
    args = ap.parse_args()
    cfg = wl.get("cfg2")
    if args.storage:
        cfg["storage"] = args.storage
    t0 = time.time()

    def gpu_run(seed):
        g = lb.Lbm.from_config(cfg)            # storage scheme from cfg["storage"]
        g.init(seed)
        g.step(args.spin)
        g.stats_accumulate(1)
        g.stats_reset()
        return g

    ga, gb = gpu_run(cfg["seed"]), gpu_run(cfg["seed"] + 1)
    o = oracle.Oracle.from_config(cfg)
    o.init_from_config(cfg)
    o.step(args.spin)
    o.stats_accumulate(1)
    o.stats_reset()
    print(f"spin-up of {args.spin} steps done on all three runs after {time.time() - t0:.0f} s", flush=True)
    done = 0
    while done < args.window:
        n = min(args.every, args.window - done)
        o.step(n)
        ga.step(n)
        gb.step(n)
        done += n
        so, _ = o.stats_read()
        sa, _ = ga.stats_read()
        sb, _ = gb.stats_read()
        d_par, d_floor = diffs(sa, so), diffs(sb, sa)
        lines = [
            "# P11 — config 2 long-run statistical parity (CUDA path vs fp64 oracle)", "",
            f"Command: `python tests/run_p11_cfg2.py --spin {args.spin} --window {args.window} --storage {cfg['storage']}` on one B200 "
            f"+ {os.cpu_count()} host cores; lattice {cfg['nx']}x{cfg['ny']}x{cfg['nz']}, seed {cfg['seed']}; "
            f"variant {ga.variant}.", "",
            f"Window so far: {done} of {args.window} steps after {args.spin} spin-up steps "
            f"({time.time() - t0:.0f} s elapsed).", "",
            "Differences are max over y of |a − b| divided by the column's profile maximum.",
            "Noise floor = two CUDA runs that differ only in the seed of the initial perturbation.", "",
            "| column | profile max (oracle) | GPU vs oracle, same seed | noise floor (GPU seed A vs B) | bar |",
            "|---|---|---|---|---|"]
        for k in range(9):
            bar = "2 %" if k == 0 else ("5 %" if k in (3, 4, 5, 6) else "—")
            lines.append(f"| {NAMES[k]} | {d_par[k][1]:.3e} | {100 * d_par[k][0]:.3f} % | "
                         f"{100 * d_floor[k][0]:.3f} % | {bar} |")
        ok = d_par[0][0] <= 0.02 and all(d_par[k][0] <= 0.05 for k in (3, 4, 5, 6))
        lines += ["", f"Within the north_star bar at this point: **{'yes' if ok else 'no'}**", ""]
        os.makedirs(os.path.dirname(args.out), exist_ok=True)
        with open(args.out, "w") as f:
            f.write("\n".join(lines))
        print(f"window {done}/{args.window}: mean {100 * d_par[0][0]:.3f} %, "
              f"uu {100 * d_par[3][0]:.3f} %, uv {100 * d_par[6][0]:.3f} % "
              f"(floor uu {100 * d_floor[3][0]:.3f} %) [{time.time() - t0:.0f} s]", flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
