"""One regularised OTOC curve or Green function end to end through the C ABI.

    python -m paper_2311_00639_b200.otoc_run --N 56 --k 4 --beta 5 --tmax 8 --nt 9 [--dtype c128|c64]
           [--krylov-dim 16] [--two-pass] [--tol 1e-10] [--block] [--green] [--seed 0] [--realization 0]
           [--relabel] [--renormalize]

Builds the sparse SYK Hamiltonian (Eq. 1), draws the Haar-random state on the device, runs syk_otoc
(or, with --block, syk_otoc_block on both parity sectors of the same state and adds them) and prints one
JSON line: F(t), OTOC(t) = F(t)/F(0), the seconds per curve and per point (the quantities of the paper's benchmark
tables), matvec counts and the resident device memory.  W = gamma_{N-1}, V = gamma_{N-2} as in the
paper.  Argument marshalling only: every step of the path runs in the CUDA library.
"""
import argparse
import json
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=56)
    ap.add_argument("--k", type=float, default=4.0, help="sparsity k (kN terms on average); 0 = dense")
    ap.add_argument("--beta", type=float, default=5.0)
    ap.add_argument("--tmax", type=float, default=8.0)
    ap.add_argument("--nt", type=int, default=9, help="grid points, t = 0 .. tmax inclusive")
    ap.add_argument("--dtype", default="c128", choices=["c128", "c64"])
    ap.add_argument("--krylov-dim", type=int, default=16)
    ap.add_argument("--two-pass", action="store_true")
    ap.add_argument("--tol", type=float, default=0.0, help="0 = library default (1e-12 / 1e-6)")
    ap.add_argument("--block", action="store_true", help="work in the parity blocks (half-size vectors)")
    ap.add_argument("--green", action="store_true", help="Green function G(t) of gamma_{N-1} instead of the OTOC")
    ap.add_argument("--batch", type=int, default=0, help="disorder realizations 0..batch-1 in lock step (syk_otoc_batched)")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--realization", type=int, default=0)
    ap.add_argument("--relabel", action="store_true", help="qubit layout chosen per Hamiltonian (syk_ham_optimize_layout)")
    ap.add_argument("--renormalize", action="store_true", help="carry the norm separately (large beta in complex64)")
    args = ap.parse_args()

    import torch
    from . import binding as B, inputs

    if not torch.cuda.is_available():
        raise SystemExit("otoc_run needs a CUDA device: the library has no CPU path")
    N, L = args.N, args.N // 2
    tdt = torch.complex128 if args.dtype == "c128" else torch.complex64
    code = B.SYK_C128 if args.dtype == "c128" else B.SYK_C64
    p = 1.0 if args.k == 0 else inputs.bernoulli_p(N, args.k)
    opts = {"krylov_dim": args.krylov_dim, "two_pass": int(args.two_pass), "tol": args.tol,
            "renormalize": int(args.renormalize)}
    t_grid = np.linspace(0.0, args.tmax, args.nt)
    iW, jV = N - 1, N - 2

    if args.batch > 0:
        return run_batch(args, B, torch, N, L, tdt, code, p, opts, t_grid, iW, jV)

    t0 = time.perf_counter()
    h = B.syk_build_hamiltonian(N, p, args.seed, args.realization)
    info = h.info()
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    stats_tot = {"n_matvec": 0, "n_substeps": 0}
    torch.cuda.reset_peak_memory_stats()
    if not args.block:
        if args.relabel:
            B.syk_ham_optimize_layout(h, code)
        B.syk_ham_prepare(h, code)
        psi = torch.empty(1 << L, dtype=tdt, device="cuda")
        B.syk_random_state_h(h, args.seed, args.realization, psi, scratch)
        wk = torch.empty(B.syk_otoc_workspace_bytes(h, code, opts), dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        if args.green:
            F, st = B.syk_green(h, iW, args.beta, t_grid, psi, wk, opts)
        else:
            F, st = B.syk_otoc(h, iW, jV, args.beta, t_grid, psi, wk, opts)
        for key in stats_tot:
            stats_tot[key] += st[key]
    else:
        # the two sector components of the random state are drawn directly as two independent normalised Gaussian
        # vectors with weight 1/2 each (the Haar ensemble up to O(D^-1/2) fluctuations of the sector weights)
        he, ho = B.syk_build_parity_block(h, 0), B.syk_build_parity_block(h, 1)
        if args.relabel:                                       # one layout for both blocks (a gamma maps between them)
            perm = B.syk_ham_optimize_layout(he, code)["perm"]
            B.syk_ham_set_layout(ho, perm)
        half = 1 << (L - 1)
        ps = torch.empty(half, dtype=tdt, device="cuda")       # one sector at a time: N = 66 needs all of the memory
        wk = torch.empty(B.syk_otoc_workspace_bytes(he, code, opts), dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        F = 0
        for s in (0, 1):
            B.syk_random_state_h(he, args.seed, 2 * args.realization + s, ps, scratch)      # norm 1
            if args.green:
                Fs, st = B.syk_green_block(he, ho, s, iW, args.beta, t_grid, ps, wk, opts)
            else:
                Fs, st = B.syk_otoc_block(he, ho, s, iW, jV, args.beta, t_grid, ps, wk, opts)
            F = F + 0.5 * Fs      # F is quadratic in psi: |psi_U|^2 = |psi_D|^2 = 1/2 for the jointly normalised state
            for key in stats_tot:
                stats_tot[key] += st[key]
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    ratio = F / F[0]
    out = {"what": "green" if args.green else "otoc", "N": N, "k": args.k, "beta": args.beta, "dtype": args.dtype,
           "parity_blocks": args.block, "relabelled": args.relabel, "krylov_dim": args.krylov_dim, "two_pass": args.two_pass,
           "n_terms": info["n_terms"], "n_xmasks": info["n_xmasks"], "t": t_grid.tolist(),
           "F_re": F.real.tolist(), "F_im": F.imag.tolist(), "ratio_re": ratio.real.tolist(),
           "seconds_setup": t1 - t0, "seconds_curve": t2 - t1, "seconds_per_point": (t2 - t1) / len(t_grid),
           "n_matvec": stats_tot["n_matvec"], "n_substeps": stats_tot["n_substeps"],
           "peak_device_GB": torch.cuda.max_memory_allocated() / 1e9}
    print(json.dumps(out), flush=True)


def run_batch(args, B, torch, N, L, tdt, code, p, opts, t_grid, iW, jV):
    """BASELINE configs[1] shape: `batch` disorder realizations advanced in lock step (grid.y = realization); prints the
    disorder-averaged curve both ways (mean of ratios, ratio of means: DESIGN.md R-F)."""
    nb, D = args.batch, 1 << L
    t0 = time.perf_counter()
    hams = [B.syk_build_hamiltonian(N, p, args.seed, r) for r in range(nb)]
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    psi = torch.empty((nb, D), dtype=tdt, device="cuda")
    for r in range(nb):
        B.syk_random_state(N, args.seed, r, psi[r], scratch)
    wk = torch.empty(B.syk_otoc_batched_workspace_bytes(hams[0], nb, code, opts), dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    B.syk_launch_count(reset=True)
    t1 = time.perf_counter()
    F, st = B.syk_otoc_batched(hams, iW, jV, args.beta, t_grid, psi, D, wk, opts)
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    ratio = (F / F[:, :1]).real
    out = {"what": "otoc_batched", "N": N, "k": args.k, "beta": args.beta, "dtype": args.dtype, "realizations": nb,
           "krylov_dim": args.krylov_dim, "n_points": len(t_grid), "t_max": float(t_grid[-1]),
           "mean_of_ratios": ratio.mean(axis=0).tolist(),
           "ratio_of_means": (F.mean(axis=0) / F.mean(axis=0)[0]).real.tolist(),
           "std_of_ratios_last": float(ratio[:, -1].std()),
           "seconds_setup": t1 - t0, "seconds_all_curves": t2 - t1, "seconds_per_point_per_realization": (t2 - t1) / len(t_grid) / nb,
           "n_matvec": st["n_matvec"], "rounds": st["n_substeps"], "kernel_launches": B.syk_launch_count(),
           "lanczos_steps_per_s": st["n_matvec"] / (t2 - t1), "peak_device_GB": torch.cuda.max_memory_allocated() / 1e9}
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
