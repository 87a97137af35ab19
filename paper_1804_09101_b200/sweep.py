"""Size sweep of gh_rhs (BASELINE.json configs[4]): single shells with N_r = L+1 = n, single cubes
N^3, and the paper's "SingleBH" / "BBH" shell prescriptions, Kerr-Schild a = 0.5 + seeded 1e-4 perturbation.

    python -m paper_1804_09101_b200.sweep [--reps 20] [--markdown] [--fill 2000000]

Per member: points, gh_rhs time (median of `reps` after 5 warm-ups, CUDA events on the library's stream via its
profiling interface), grid-point evaluations/s, derivative-kernel FP64 rate (algorithmic flop of DESIGN.md §6 over
k_cheb + k_ang time; and in the paper's dense convention, Eqs. 29 and 31) and the fused RHS kernel's GB/s.
Sizes are limited by this build's GH_MAX_L = 47 and GH_MAX_CHEB_N = 64.
"""
from __future__ import annotations

import argparse
import json

import numpy as np


def members():
    from . import configs

    out = []
    # the paper's whole-code test problem: 2 shells of (10, 19, 38) points; only its first shell is replicated by --fill
    out.append(("paper test problem, 2 shells (10,19,38)", configs.paper_two_shells()))
    for n in (8, 16, 24, 32, 40, 48):
        out.append((f"shell n={n} (N_r={n}, L={n - 1})", configs.c5_shell(n)))
    for N in (10, 16, 20, 32, 40, 64):
        out.append((f"block {N}^3", configs.c5_block(N)))
    for k in range(0, 11):
        out.append((f"SingleBH k={k}", configs.single_bh(k)))
    for k in range(1, 17):
        out.append((f"BBH k={k}", configs.bbh(k)))
    return out


def run_member(label, cfg, reps, device="cuda:0", fill_points=0):
    import torch

    from . import configs, gh, inputs, opcount

    base = cfg["descs"]
    copies = max(1, -(-fill_points // configs.num_points(base[0]))) if fill_points else 1
    if copies > 1:
        base = base[:1]
    descs = [dict(d) for _ in range(copies) for d in base]   # independent replicas of the member (throughput regime)
    dom = gh.Domain(descs, device=device)
    coords = dom.coords()[:len(base)]
    us, Hs = inputs.initial_data(base, coords, cfg["spin"], cfg["amplitude"], cfg["id"])
    dom.set_gauge_source(dom.pack(list(Hs) * copies))
    dom.set_fields(dom.pack(list(us) * copies), 0.0)
    out = dom.empty(50)
    for _ in range(5):
        dom.rhs(out)
    dom.set_profiling(True)
    tot, der, rhs = [], [], []
    for _ in range(reps):
        dom.profile_reset()
        dom.rhs(out)
        prof = dom.profile_read()
        t_der = prof["k_cheb"][0] + prof["k_ang"][0]
        t_rhs = prof["k_rhs"][0]
        tot.append(t_der + t_rhs); der.append(t_der); rhs.append(t_rhs)
    dom.set_profiling(False)
    torch.cuda.synchronize()
    P = dom.P
    flop = flop_paper = 0
    for d in descs:
        if d["kind"] == "shell":
            n_r, L = d["n"][0], d["n"][1]
            flop += opcount.shell_factored_flop(50, n_r, L)
            flop_paper += opcount.shell_deriv_dense(50, n_r, L + 1, 2 * L + 2)[1]
        else:
            flop += opcount.block_deriv(50, *d["n"])[1]
            flop_paper += opcount.block_deriv(50, *d["n"])[1]
    ms, ms_d, ms_r = float(np.median(tot)), float(np.median(der)), float(np.median(rhs))
    dom.close()
    return {"member": label + (f" x{copies}" if copies > 1 else ""), "points": P, "gh_rhs_ms": ms, "points_per_s": P / (ms * 1e-3),
            "deriv_ms": ms_d, "deriv_TFLOPs": flop / (ms_d * 1e-3) / 1e12,
            "deriv_TFLOPs_paper_convention": flop_paper / (ms_d * 1e-3) / 1e12,
            "k_rhs_ms": ms_r, "k_rhs_GBps": 2128.0 * P / (ms_r * 1e-3) / 1e9}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--markdown", action="store_true")
    ap.add_argument("--fill", type=int, default=0,
                    help="replicate each member until it has at least this many points (throughput regime; 0: single subdomain, latency regime)")
    args = ap.parse_args()
    from . import build

    build.build()
    rows = [run_member(lbl, cfg, args.reps, fill_points=args.fill) for lbl, cfg in members()]
    if args.markdown:
        print("| member | points | gh_rhs ms | points/s | deriv ms | deriv TFLOP/s (executed map) | deriv TFLOP/s (paper's dense count) | k_rhs ms | k_rhs GB/s |")
        print("|---|---|---|---|---|---|---|---|---|")
        for r in rows:
            print(f"| {r['member']} | {r['points']} | {r['gh_rhs_ms']:.4f} | {r['points_per_s']:.3e} | {r['deriv_ms']:.4f} | "
                  f"{r['deriv_TFLOPs']:.2f} | {r['deriv_TFLOPs_paper_convention']:.1f} | {r['k_rhs_ms']:.4f} | {r['k_rhs_GBps']:.0f} |")
    else:
        for r in rows:
            print(json.dumps(r))


if __name__ == "__main__":
    main()
