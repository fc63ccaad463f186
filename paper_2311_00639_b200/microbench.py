"""On-chip peaks of this GPU for the roofline of the apply_H kernels (include/syk.h `syk_microbench`).

    python -m paper_2311_00639_b200.microbench [--json]

Prints a markdown table (or one JSON object): L2 -> SM and DRAM -> SM streaming rates of 148 persistent CTAs through the
shared-memory ring of the scatter-tile kernel, the shared-memory read rate of its inner loop, both at once, and the issue
rates that bound the dense-table kernel.  `measure()` is what bench.py calls for its `roofline` denominators.
"""
import json
import sys


def measure(quick=False):
    """Dict of measured peaks.  Rates per SM are per SM CYCLE of the slowest CTA (clock64), chip rates per second of
    device time (CUDA events)."""
    import torch
    from . import binding as B
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    wk = torch.empty(B.syk_microbench_workspace_bytes(), dtype=torch.uint8, device="cuda")
    small = torch.zeros(32 << 20, dtype=torch.uint8, device="cuda")          # L2 resident (126 MB L2)
    n = 2048 if quick else 16384
    out = {"sms": sms}

    def stream(kind, chunks, terms, buf):
        B.syk_microbench(kind, max(chunks // 8, 64), terms, buf, wk)         # warm-up: L2 fill, clocks
        r = B.syk_microbench(kind, chunks, terms, buf, wk)
        d = {"ms": r["ms"], "cycles": r["cycles"]}
        if r["units"]:
            d["load_B_per_clk_per_SM"] = r["units"] / sms / r["cycles"]
            d["load_TB_per_s"] = r["units"] / (r["ms"] * 1e-3) / 1e12
        if r["lds_bytes"]:
            d["lds_B_per_clk_per_SM"] = r["lds_bytes"] / sms / r["cycles"]
            d["lds_TB_per_s"] = r["lds_bytes"] / (r["ms"] * 1e-3) / 1e12
        d["sm_mhz_effective"] = r["cycles"] / (r["ms"] * 1e-3) / 1e6
        return d

    out["l2_to_sm"] = stream(0, n, 0, small)
    out["lds_only"] = stream(1, n // 8, 8, None)
    for t in (1, 2, 3, 4):
        out[f"l2_and_lds_{t}"] = stream(2, n // 2, t, small)
    if not quick:
        free, _ = torch.cuda.mem_get_info()
        big_bytes = 8 << 30 if free > (12 << 30) else 1 << 30
        big = torch.zeros(big_bytes, dtype=torch.uint8, device="cuda")
        out["dram_to_sm"] = stream(0, n, 0, big)
        out["dram_and_lds_2"] = stream(2, n // 2, 2, big)
        del big
    iters = 4000 if quick else 20000
    for name, kind in (("fp64_add", 3), ("dense_term_sequence", 4)):
        B.syk_microbench(kind, iters // 8, 0, None, wk)
        r = B.syk_microbench(kind, iters, 0, None, wk)
        out[name] = {"ms": r["ms"], "cycles": r["cycles"], "adds_per_clk_per_SM": r["units"] / sms / r["cycles"],
                     "adds_per_s": r["units"] / (r["ms"] * 1e-3), "sm_mhz_effective": r["cycles"] / (r["ms"] * 1e-3) / 1e6}
    return out


def main():
    import torch
    assert torch.cuda.is_available(), "needs a CUDA device"
    res = measure(quick="--quick" in sys.argv)
    if "--json" in sys.argv:
        print(json.dumps(res))
        return
    print("| measurement | ms | load B/clk/SM | load TB/s | LDS B/clk/SM | LDS TB/s | adds/clk/SM | effective SM MHz |")
    print("|---|---|---|---|---|---|---|---|")
    for k, v in res.items():
        if not isinstance(v, dict):
            continue
        f = lambda key, fmt: (fmt % v[key]) if key in v else ""
        print(f"| {k} | {v['ms']:.3f} | {f('load_B_per_clk_per_SM', '%.1f')} | {f('load_TB_per_s', '%.2f')} | "
              f"{f('lds_B_per_clk_per_SM', '%.1f')} | {f('lds_TB_per_s', '%.2f')} | {f('adds_per_clk_per_SM', '%.1f')} | "
              f"{v['sm_mhz_effective']:.0f} |")
    print(f"\nSMs: {res['sms']}; {torch.cuda.get_device_name()}")


if __name__ == "__main__":
    main()
