"""Timeline of one persistent CTA of the scatter-tile apply_H kernel (syk_apply_H_trace): where a tile's time goes.

    python -m paper_2311_00639_b200.trace [--workload N56_k4_c128|N64_k2_c64] [--cta 0,1,73,147] [--round 2] > profiles/<round>_chunk_trace.md

Per ring chunk (64 KiB = half a source tile) the kernel records when the producer issued its bulk copies, when the first
consumer warp asked for it and when it got it.  The table below groups the chunks by the number of terms their load
serves and reports the time the consumers WORKED on a chunk (from getting it to asking for the next one) and the time they
WAITED for data, in SM clocks.  Measurement only: results of the product are those of syk_apply_H.
"""
import argparse
import sys
from math import comb

import numpy as np


def analyse(tr, window_mask):
    n_loads, rot = tr["n_loads"], tr["rot"]
    nc = len(tr["issue"]) // n_loads
    before, after = tr["before_wait"], tr["after_wait"]
    wait = after - before
    work = np.append(before[1:] - after[:-1], 0)   # the last chunk of the list is followed by the epilogue: not counted
    total = int(after[-1] - before[0])
    run_id = tr["load_xo"] & ~np.uint32(window_mask)
    by_nt = {}
    first_wait, other_wait, n_first, n_other = 0, 0, 0, 0
    for li in range(n_loads):
        l, lp = (li + rot) % n_loads, (li - 1 + rot) % n_loads
        first = li == 0 or run_id[l] != run_id[lp]
        for c in range(nc):
            v = li * nc + c
            if first:
                first_wait += int(wait[v]); n_first += 1
            else:
                other_wait += int(wait[v]); n_other += 1
            if v + 1 < n_loads * nc:
                by_nt.setdefault(int(tr["load_terms"][l]), []).append(int(work[v]))
    if not tr["first_decoded"].any():        # three-stamp trace: no phases
        return {"total": total, "wait": int(wait.sum()), "work": int(work.sum()), "by_nt": by_nt,
                "first_wait": (first_wait, n_first), "other_wait": (other_wait, n_other), "nc": nc, "phases": {}}
    # phases of a chunk as thread 0 of the consumers sees them (means over the chunks of loads with 1, 2, >= 4 terms)
    nt_of = np.repeat(tr["load_terms"][(np.arange(n_loads) + rot) % n_loads], nc)
    phases = {}
    for name, sel in (("1", nt_of == 1), ("2", nt_of == 2), (">= 4", nt_of >= 4)):
        idx = np.where(sel)[0]
        idx = idx[idx + 1 < n_loads * nc]
        if len(idx) == 0:
            continue
        phases[name] = [len(idx)] + [float(np.mean(b[idx] - a[idx])) for a, b in (
            (before, after), (after, tr["first_decoded"]), (tr["first_decoded"], tr["first_issued"]),
            (tr["first_issued"], tr["all_issued"]), (tr["all_issued"], tr["arrived"]))] + [
            float(np.mean(before[idx + 1] - tr["arrived"][idx]))]
    return {"total": total, "wait": int(wait.sum()), "work": int(work.sum()), "by_nt": by_nt,
            "first_wait": (first_wait, n_first), "other_wait": (other_wait, n_other), "nc": nc, "phases": phases}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="N56_k4_c128,N64_k2_c64")
    ap.add_argument("--cta", default="0,1,73,147")
    ap.add_argument("--round", type=int, default=2)
    args = ap.parse_args()
    import torch
    from . import binding as B
    if not torch.cuda.is_available():
        print("needs a CUDA device", file=sys.stderr)
        return 1
    specs = {"N56_k4_c128": (56, 4, torch.complex128), "N64_k2_c64": (64, 2, torch.complex64)}
    print("# Timeline of single persistent CTAs of the scatter-tile kernel (`syk_apply_H_trace`)\n")
    print(f"Command: `python -m paper_2311_00639_b200.trace --workload {args.workload} --cta {args.cta} --round {args.round}`"
          f"  ({torch.cuda.get_device_name(0)}; SM clocks, clock64)\n")
    for name in args.workload.split(","):
        N, k, tdt = specs[name]
        code = B.SYK_C128 if tdt == torch.complex128 else B.SYK_C64
        D = 1 << (N // 2)
        h = B.syk_build_hamiltonian(N, k * N / comb(N, 4), 0, 0)
        B.syk_ham_optimize_layout(h, code)
        B.syk_ham_prepare(h, code)
        lay = B.syk_apply_H_layout(h, code)
        scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
        a = torch.empty(D, dtype=tdt, device="cuda")
        b = torch.empty(D, dtype=tdt, device="cuda")
        B.syk_random_state_h(h, 0, 0, a, scratch)
        for _ in range(2):
            B.syk_apply_H(h, a, b)
        torch.cuda.synchronize()
        info = h.info()
        print(f"## {name}: T = {info['n_terms']} terms, {lay['n_loads']} loads, {lay['n_passes']} passes\n")
        print("| CTA | rotation | clocks for the load list of one tile | consumers worked | waited for data | wait per chunk: first load of a run / other loads |")
        print("|---|---|---|---|---|---|")
        merged = {}
        for cta in [int(x) for x in args.cta.split(",")]:
            tr = B.syk_apply_H_trace(h, a, b, cta=cta, round=args.round)
            r = analyse(tr, lay["window_mask"])
            fw, ow = r["first_wait"], r["other_wait"]
            print(f"| {cta} | {tr['rot']} | {r['total']} | {r['work']} ({100 * r['work'] / r['total']:.1f} %) | {r['wait']} "
                  f"({100 * r['wait'] / r['total']:.1f} %) | {fw[0] / max(fw[1], 1):.0f} / {ow[0] / max(ow[1], 1):.0f} |")
            for nt, v in r["by_nt"].items():
                merged.setdefault(nt, []).extend(v)
        first_cta = int(args.cta.split(",")[0])
        last_phases = analyse(B.syk_apply_H_trace(h, a, b, cta=first_cta, round=args.round, detail=1), lay["window_mask"])["phases"]
        chunk_bytes = 65536
        print("\n| terms of the load | chunks sampled | clocks worked per chunk (mean) | per term | shared-memory bytes read per clock |")
        print("|---|---|---|---|---|")
        for nt in sorted(merged):
            m = float(np.mean(merged[nt]))
            print(f"| {nt} | {len(merged[nt])} | {m:.0f} | {m / nt:.0f} | {nt * chunk_bytes / m:.1f} |")
        xs = np.array([nt for nt in merged for _ in merged[nt]], dtype=np.float64)
        ys = np.array([w for nt in merged for w in merged[nt]], dtype=np.float64)
        A = np.vstack([np.ones_like(xs), xs]).T
        coef, *_ = np.linalg.lstsq(A, ys, rcond=None)
        print(f"\nLeast-squares fit: clocks per chunk = {coef[0]:.0f} + {coef[1]:.0f} x terms "
              f"(an LDS pass over a 64 KiB chunk at 128 B/clk is 512 clocks).\n")
        print(f"Phases of a chunk for thread 0 of the consumers (CTA {first_cta}, seven-stamp build of the kernel: the four extra stamps "
              "lengthen a chunk by ~200 clocks, so read the proportions, not the sums; mean clocks):\n")
        print("| terms of the load | chunks | wait for the chunk | decode of the first term | first term issued (16 LDS.128 + FMAs) | "
              "other terms | last FMAs issued -> arrived on the empty-barrier | -> asks for the next chunk |")
        print("|---|---|---|---|---|---|---|---|")
        for name, ph in last_phases.items():
            print(f"| {name} | {ph[0]} | " + " | ".join(f"{x:.0f}" for x in ph[1:]) + " |")
        print()
        del a, b
        torch.cuda.empty_cache()
    return 0


if __name__ == "__main__":
    sys.exit(main())
