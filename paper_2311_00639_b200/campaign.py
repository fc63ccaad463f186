"""Disorder-averaged OTOC campaign over sparsities, realizations and temperatures ("the final result is
obtained by averaging over disorder realizations"; BASELINE.json configs[2]: N=48, k in {1,2,4,8} plus dense, 20
realizations per k, beta in {2,5,10}, Krylov dimension 30).

    python -m paper_2311_00639_b200.campaign --N 48 --k 1,2,4,8 --realizations 20 --beta 2,5,10 --krylov-dim 30
           --tmax 10 --nt 11 [--dense-realizations 1 --dense-beta 5 --dense-nt 3] [--dtype c128] [--no-relabel]

Per (k, realization): one Hamiltonian (syk_build_hamiltonian + qubit layout + syk_ham_prepare), one Haar-random state
per realization, one syk_otoc call per beta.  Prints one JSON line per (k, beta) with the mean over
realizations of OTOC(t) = Re F(t)/F(0) (per-sample normalisation, DESIGN.md R-F), its standard error, seconds per curve and
matvec counts, then a markdown summary.  Argument marshalling only: every step runs in the CUDA library.
"""
import argparse
import json
import time

import numpy as np


def run_group(B, torch, inputs, N, k, realizations, betas, t_grid, opts, tdt, code, relabel, seed):
    D = 1 << (N // 2)
    p = 1.0 if not k else inputs.bernoulli_p(N, k)
    iW, jV = N - 1, N - 2
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    psi = torch.empty(D, dtype=tdt, device="cuda")
    wk = None
    ratios = {b: [] for b in betas}
    secs = {b: 0.0 for b in betas}
    matvecs = {b: 0 for b in betas}
    n_terms = []
    t_build = 0.0
    for r in range(realizations):
        t0 = time.perf_counter()
        h = B.syk_build_hamiltonian(N, p, seed, r)
        if relabel:
            B.syk_ham_optimize_layout(h, code)
        B.syk_ham_prepare(h, code)
        t_build += time.perf_counter() - t0
        n_terms.append(h.info()["n_terms"])
        if wk is None:
            wk = torch.empty(B.syk_otoc_workspace_bytes(h, code, opts), dtype=torch.uint8, device="cuda")
        for b in betas:
            B.syk_random_state_h(h, seed, r, psi, scratch)
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            F, st = B.syk_otoc(h, iW, jV, b, t_grid, psi, wk, opts)
            torch.cuda.synchronize()
            secs[b] += time.perf_counter() - t1
            matvecs[b] += st["n_matvec"]
            ratios[b].append((F / F[0]).real)
        h.close()
    out = []
    for b in betas:
        a = np.array(ratios[b])
        out.append({"N": N, "k": k if k else "dense", "beta": b, "realizations": realizations,
                    "mean_terms": float(np.mean(n_terms)), "t": t_grid.tolist(), "otoc_mean": a.mean(axis=0).tolist(),
                    "otoc_stderr": (a.std(axis=0, ddof=1) / np.sqrt(len(a))).tolist() if len(a) > 1 else None,
                    "seconds_per_curve": secs[b] / realizations, "matvecs_per_curve": matvecs[b] / realizations,
                    "seconds_build_per_realization": t_build / realizations})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=48)
    ap.add_argument("--k", default="1,2,4,8")
    ap.add_argument("--realizations", type=int, default=20)
    ap.add_argument("--beta", default="2,5,10")
    ap.add_argument("--krylov-dim", type=int, default=30)
    ap.add_argument("--tmax", type=float, default=10.0)
    ap.add_argument("--nt", type=int, default=11)
    ap.add_argument("--dense-realizations", type=int, default=0)
    ap.add_argument("--dense-beta", default="5")
    ap.add_argument("--dense-nt", type=int, default=3)
    ap.add_argument("--dtype", default="c128", choices=["c128", "c64"])
    ap.add_argument("--tol", type=float, default=0.0)
    ap.add_argument("--no-relabel", action="store_true")
    ap.add_argument("--seed", type=int, default=0)
    args = ap.parse_args()
    import torch
    from . import binding as B, inputs
    if not torch.cuda.is_available():
        raise SystemExit("campaign needs a CUDA device: the library has no CPU path")
    tdt = torch.complex128 if args.dtype == "c128" else torch.complex64
    code = B.SYK_C128 if args.dtype == "c128" else B.SYK_C64
    opts = {"krylov_dim": args.krylov_dim, "tol": args.tol}
    t_grid = np.linspace(0.0, args.tmax, args.nt)
    rows = []
    t_all = time.perf_counter()
    for k in [float(x) for x in args.k.split(",") if x]:
        rows += run_group(B, torch, inputs, args.N, k, args.realizations, [float(b) for b in args.beta.split(",")], t_grid,
                          opts, tdt, code, not args.no_relabel, args.seed)
        for r in rows[-len(args.beta.split(",")):]:
            print(json.dumps(r), flush=True)
    if args.dense_realizations > 0:
        tg = np.linspace(0.0, args.tmax, args.dense_nt)
        dense = run_group(B, torch, inputs, args.N, 0, args.dense_realizations, [float(b) for b in args.dense_beta.split(",")],
                          tg, opts, tdt, code, False, args.seed)
        for r in dense:
            print(json.dumps(r), flush=True)
        rows += dense
    total = time.perf_counter() - t_all
    print(f"\n| k | beta | realizations | mean terms | s / curve | matvecs / curve | OTOC(t_max) mean +- stderr |")
    print("|---|---|---|---|---|---|---|")
    for r in rows:
        se = r["otoc_stderr"][-1] if r["otoc_stderr"] else float("nan")
        print(f"| {r['k']} | {r['beta']} | {r['realizations']} | {r['mean_terms']:.0f} | {r['seconds_per_curve']:.2f} | "
              f"{r['matvecs_per_curve']:.0f} | {r['otoc_mean'][-1]:.4f} +- {se:.4f} (t = {r['t'][-1]:g}, {len(r['t'])} points) |")
    print(f"\ntotal wall time {total:.0f} s; N = {args.N}, Krylov dimension {args.krylov_dim}, dtype {args.dtype}, "
          f"W = gamma_{args.N - 1}, V = gamma_{args.N - 2}")


if __name__ == "__main__":
    main()
