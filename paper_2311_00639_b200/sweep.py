"""Matvec bandwidth sweep of BASELINE.json configs[3] (SURVEY 8(d) "Sweep for config 4"), through the C ABI.

    python -m paper_2311_00639_b200.sweep [--quick] [--relabel] > profiles/<round>_sweep.md

Times plain `syk_apply_H` (CUDA events, 2 warm-up + 5 timed launches, minimum and median) for
  (i)   sparsity k in {1, 2, 4, 8, 16} at N = 56 complex128 -- PAPER.md:327 expects time ~ linear in k;
  (ii)  structured mask sets of equal size at N = 56: all X bits below bit 5 (warp-local), below bit 11
        (tile-local: no second source tile), only above bit 22 (every mask is a separate DRAM stream);
  (iii) N = 40 .. 56 at k = 4 (where the vector leaves L2), and N = 64 complex64 at k in {1, 2, 4};
  (iv)  pure regimes with one term per load (Hamming-code mask sets): all loads L2 hits, all loads DRAM passes, mixtures.
and prints one markdown table.  "model GB/s" = (D_x + 2) V / time; loads / passes are the
tile layout the kernel chose (syk_apply_H_layout).  Argument marshalling only: every number is a kernel time.
"""
import argparse
import sys

import numpy as np


def time_apply(B, torch, h, tdt, N, reps=5, relabel=False):
    D = 1 << (N // 2)
    code = B.SYK_C128 if tdt == torch.complex128 else B.SYK_C64
    if relabel:
        B.syk_ham_optimize_layout(h, code)
    B.syk_ham_prepare(h, code)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    a = torch.empty(D, dtype=tdt, device="cuda")
    b = torch.empty(D, dtype=tdt, device="cuda")
    B.syk_random_state_h(h, 0, 0, a, scratch)
    for _ in range(2):
        B.syk_apply_H(h, a, b)
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        B.syk_apply_H(h, a, b)
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    kind = B.syk_apply_H_kernel_kind(h, code)
    lay = B.syk_apply_H_layout(h, code) if kind == 3 else {"n_loads": None, "n_passes": None}
    info = h.info()
    V = D * (16 if tdt == torch.complex128 else 8)
    ms = min(ts)
    del a, b
    torch.cuda.empty_cache()
    return {"T": info["n_terms"], "Dx": info["n_xmasks"], "kind": kind, "loads": lay["n_loads"],
            "passes": lay["n_passes"], "ms_min": ms, "ms_med": sorted(ts)[len(ts) // 2],
            "model_gbs": (info["n_xmasks"] + 2) * V / (ms * 1e-3) / 1e9, "V": V}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="N <= 48 only (a few seconds)")
    ap.add_argument("--relabel", action="store_true", help="qubit layout chosen per Hamiltonian (syk_ham_optimize_layout)")
    ap.add_argument("--lockstep", action="store_true",
                    help="instead: sweep syk_set_lockstep(epoch, lag) for the two headline workloads and tile kernels")
    args = ap.parse_args()
    import torch
    from . import binding as B, inputs

    if not torch.cuda.is_available():
        raise SystemExit("sweep needs a CUDA device: the library has no CPU path")
    if args.lockstep:
        return lockstep_sweep(B, torch, inputs, args.quick, args.relabel)
    rows = []

    def run(label, N, h, tdt, relabel=None):
        r = time_apply(B, torch, h, tdt, N, relabel=args.relabel if relabel is None else relabel)
        rows.append((label, N, "c128" if tdt == torch.complex128 else "c64", r))
        print(f"# {label} N={N}: {r['ms_min']:.3f} ms", file=sys.stderr, flush=True)

    c128, c64 = torch.complex128, torch.complex64
    Nbig = 48 if args.quick else 56
    for k in (1, 2, 4, 8, 16):
        run(f"(i) k={k}", Nbig, B.syk_build_hamiltonian(Nbig, inputs.bernoulli_p(Nbig, k), 0, 0), c128)
    L = Nbig // 2
    for name, qubits in (("bits<5", range(0, 5)), ("bits<11", range(0, 11)), (f"bits>={L - 6}", range(L - 6, L))):
        q, J = inputs.quartets_on_qubits(list(qubits), 60, seed=9, sigma=0.05)
        run(f"(ii) 60 terms, X {name}", Nbig, B.syk_build_from_terms(Nbig, q, J), c128)
    for N in ((40, 44, 48) if args.quick else (40, 44, 48, 52, 56)):
        run("(iii) k=4", N, B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, 4), 0, 0), c128)
    if not args.quick:
        for k in (1, 2, 4):
            run(f"(iii) k={k}", 64, B.syk_build_hamiltonian(64, inputs.bernoulli_p(64, k), 0, 0), c64)
    # (iv) pure regimes of the tile kernel with ONE term per load: X strings whose masks are the 15 non-zero words of the
    # Hamming(7,4) code on a 7-bit field (any two differ in >= 3 bits, so the kernel's 2 free tile bits cannot merge loads):
    # field inside the L2 window -> every load after the first hits in L2; field on the top bits -> every load is a DRAM pass;
    # products of the two -> runs of 15 (or 4) loads per DRAM pass
    G = (0b1000110, 0b0100101, 0b0010011, 0b0001111)
    code = sorted({(a * G[0]) ^ (b * G[1]) ^ (c * G[2]) ^ (d * G[3]) for a in (0, 1) for b in (0, 1) for c in (0, 1)
                   for d in (0, 1)} - {0})
    lo, hi = 13, L - 7
    for name, terms in (("15 masks in the window", [(w << lo, 0, 0.01) for w in code]),
                        ("15 masks on the top bits", [(w << hi, 0, 0.01) for w in code]),
                        ("15 window x 4 top", [((w1 << lo) | (w2 << hi), 0, 0.01) for w1 in code for w2 in code[:4]]),
                        ("15 window x 15 top", [((w1 << lo) | (w2 << hi), 0, 0.01) for w1 in code for w2 in code])):
        h = B.syk_build_from_pauli_strings(L, terms)
        B.syk_set_apply_H_kernel(h, 3)
        run(f"(iv) {name}", Nbig, h, c128, relabel=False)   # canonical layout: the fields are placed for it

    print("| case | N | dtype | T | D_x | kernel | loads | passes | ms (min) | ms (median) | model GB/s | ms per X-mask |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    for label, N, dt, r in rows:
        print(f"| {label} | {N} | {dt} | {r['T']} | {r['Dx']} | {r['kind']} | {r['loads']} | {r['passes']} | "
              f"{r['ms_min']:.3f} | {r['ms_med']:.3f} | {r['model_gbs']:.0f} | {r['ms_min'] / max(r['Dx'], 1):.4f} |")
    ks = [(r["Dx"], r["ms_min"]) for label, N, dt, r in rows if label.startswith("(i) ")]
    if len(ks) >= 3:
        x = np.array([a for a, _ in ks], dtype=float)
        y = np.array([b for _, b in ks], dtype=float)
        slope, icpt = np.polyfit(x, y, 1)
        resid = float(np.max(np.abs(slope * x + icpt - y) / y))
        print(f"\nAffine fit of (i): time = {icpt:.3f} ms + {slope:.4f} ms x D_x, worst relative residual {resid:.3f}")


def lockstep_sweep(B, torch, inputs, quick, relabel=False):
    """Pacing of the persistent CTAs (syk_set_lockstep): plain syk_apply_H, minimum of 3 launches in ms, for the
    register-tile (kind 2) and scatter-tile (kind 3) kernels; outputs are checked to be bitwise equal across settings."""
    settings = [(0, 0), (1, 1), (2, 1), (2, 2), (4, 1), (4, 2), (8, 1), (8, 2), (16, 1), (32, 1)]
    cases = [(48, 4, torch.complex128)] if quick else [(56, 4, torch.complex128), (64, 2, torch.complex64)]
    print("| workload | kernel | " + " | ".join("free" if e == 0 else f"({e},{lag})" for e, lag in settings) + " |")
    print("|---|---|" + "---|" * len(settings))
    try:
        for N, k, tdt in cases:
            D = 1 << (N // 2)
            h = B.syk_build_hamiltonian(N, inputs.bernoulli_p(N, k), 0, 0)
            if relabel:
                B.syk_ham_optimize_layout(h, B.SYK_C128 if tdt == torch.complex128 else B.SYK_C64)
            scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
            a = torch.empty(D, dtype=tdt, device="cuda")
            b = torch.empty(D, dtype=tdt, device="cuda")
            B.syk_random_state_h(h, 0, 0, a, scratch)
            for kind in (2, 3):
                B.syk_set_apply_H_kernel(h, kind)
                cells, ref = [], None
                for e, lag in settings:
                    B.syk_set_lockstep(e, lag)
                    B.syk_apply_H(h, a, b)
                    torch.cuda.synchronize()
                    ts = []
                    for _ in range(3):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        B.syk_apply_H(h, a, b)
                        e1.record()
                        torch.cuda.synchronize()
                        ts.append(e0.elapsed_time(e1))
                    chk = torch.view_as_real(b[: 1 << 20]).double().sum().item()
                    ref = chk if ref is None else ref
                    cells.append(f"{min(ts):.1f}" + ("" if chk == ref else " (!)"))
                    print(f"# N={N} kind={kind} ({e},{lag}): {min(ts):.2f} ms", file=sys.stderr, flush=True)
                name = "c128" if tdt == torch.complex128 else "c64"
                print(f"| N={N} k={k} {name} | {kind} | " + " | ".join(cells) + " |")
            del a, b
            torch.cuda.empty_cache()
    finally:
        B.syk_set_lockstep(8, 1)


if __name__ == "__main__":
    main()
