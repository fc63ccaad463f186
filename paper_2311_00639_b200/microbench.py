"""On-chip peaks of this GPU for the roofline of the apply_H kernels (include/syk.h `syk_microbench`).

    python -m paper_2311_00639_b200.microbench [--json] [--quick]
    python -m paper_2311_00639_b200.microbench --sweep       (streaming rate against the size of the source buffer)

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
    for ctas in (74, 37, 8):                                                 # fewer SMs pulling: the per-SM limit
        B.syk_microbench(0, 256, ctas, small, wk)
        r = B.syk_microbench(0, n, ctas, small, wk)
        out[f"l2_to_sm_{ctas}_ctas"] = {"ms": r["ms"], "cycles": r["cycles"], "load_B_per_clk_per_SM": r["units"] / ctas / r["cycles"],
                                        "load_TB_per_s": r["units"] / (r["ms"] * 1e-3) / 1e12,
                                        "sm_mhz_effective": r["cycles"] / (r["ms"] * 1e-3) / 1e6}
    out["lds_only"] = stream(1, n // 8, 8, None)
    for t in (1, 2, 3, 4):
        out[f"l2_and_lds_{t}"] = stream(2, n // 2, t, small)
    if not quick:
        free, _ = torch.cuda.mem_get_info()
        big_bytes = 8 << 30 if free > (12 << 30) else 1 << 30
        big = torch.zeros(big_bytes, dtype=torch.uint8, device="cuda")
        out["dram_to_sm"] = stream(0, n, 0, big)
        out["dram_and_lds_2"] = stream(2, n // 2, 2, big)
        # do the two supplies overlap?  74 CTAs stream from DRAM while 74 stream from an L2-resident region
        for mult in (1, 3):
            B.syk_microbench(5, n // 16, mult, big, wk)
            r = B.syk_microbench(5, n // 2, mult, big, wk)
            out[f"dram_half_and_l2_half_x{mult}"] = {
                "ms": r["ms"], "cycles": r["cycles"], "sm_mhz_effective": r["cycles"] / (r["ms"] * 1e-3) / 1e6,
                "dram_group_TB_per_s": r["units"] / r["cycles_even"] * (r["cycles"] / (r["ms"] * 1e-3)) / 1e12,
                "l2_group_TB_per_s": r["lds_bytes"] / r["cycles_odd"] * (r["cycles"] / (r["ms"] * 1e-3)) / 1e12,
                "dram_group_B_per_clk_per_SM": r["units"] / ((sms + 1) // 2) / r["cycles_even"],
                "l2_group_B_per_clk_per_SM": r["lds_bytes"] / (sms // 2) / r["cycles_odd"]}
        del big
    # global loads against the shared-memory data path (kind 6): LDS alone, LDG alone (L2 hits), both
    it6 = 1000 if quick else 4000
    for name, buf, passes in (("lds_plain", None, 1), ("ldg_l2", small, 0), ("ldg_l2_and_lds_1", small, 1),
                              ("ldg_l2_and_lds_2", small, 2), ("ldg_l2_and_lds_3", small, 3)):
        B.syk_microbench(6, it6 // 8, passes, buf, wk)
        r = B.syk_microbench(6, it6, passes, buf, wk)
        d = {"ms": r["ms"], "cycles": r["cycles"], "sm_mhz_effective": r["cycles"] / (r["ms"] * 1e-3) / 1e6}
        if r["units"]:
            d["load_B_per_clk_per_SM"] = r["units"] / sms / r["cycles"]
            d["load_TB_per_s"] = r["units"] / (r["ms"] * 1e-3) / 1e12
        if r["lds_bytes"]:
            d["lds_B_per_clk_per_SM"] = r["lds_bytes"] / sms / r["cycles"]
            d["lds_TB_per_s"] = r["lds_bytes"] / (r["ms"] * 1e-3) / 1e12
        out[name] = d
    # distributed shared memory (kind 7): the consumers' reads from the own CTA and from the peer CTA of a 2-CTA cluster
    for name, remote in (("dsmem_own_cta", 0), ("dsmem_peer_cta", 1)):
        B.syk_microbench(7, it6 // 8, remote, None, wk)
        r = B.syk_microbench(7, it6, remote, None, wk)
        n_used = sms & ~1
        out[name] = {"ms": r["ms"], "cycles": r["cycles"], "sm_mhz_effective": r["cycles"] / (r["ms"] * 1e-3) / 1e6,
                     "lds_B_per_clk_per_SM": r["lds_bytes"] / n_used / r["cycles"],
                     "lds_TB_per_s": r["lds_bytes"] / (r["ms"] * 1e-3) / 1e12}
    iters = 4000 if quick else 20000
    for name, kind in (("fp64_add", 3), ("dense_term_sequence", 4)):
        B.syk_microbench(kind, iters // 8, 0, None, wk)
        r = B.syk_microbench(kind, iters, 0, None, wk)
        out[name] = {"ms": r["ms"], "cycles": r["cycles"], "adds_per_clk_per_SM": r["units"] / sms / r["cycles"],
                     "adds_per_s": r["units"] / (r["ms"] * 1e-3), "sm_mhz_effective": r["cycles"] / (r["ms"] * 1e-3) / 1e6}
    return out


def sweep():
    """L2 / DRAM -> SM streaming rate (alone and with 1, 2 LDS passes per chunk) against the size of the buffer the 148 CTAs
    walk through: where the working set leaves L2, and that multi-GB buffers (TLB reach) do not cost bandwidth."""
    import torch
    from . import binding as B
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    wk = torch.empty(B.syk_microbench_workspace_bytes(), dtype=torch.uint8, device="cuda")
    free, _ = torch.cuda.mem_get_info()
    print("| buffer | load only B/clk/SM (TB/s) | with 1 LDS pass | with 2 LDS passes |")
    print("|---|---|---|---|")
    for gb in (1 / 32, 1 / 16, 1 / 8, 1 / 4, 1, 8, 32, 64, 128):
        n = int(gb * (1 << 30))
        if n + (4 << 30) > free:
            break
        buf = torch.zeros(n, dtype=torch.uint8, device="cuda")
        B.syk_microbench(0, 2048, 0, buf, wk)
        cells = []
        for kind, terms in ((0, 0), (2, 1), (2, 2)):
            r = B.syk_microbench(kind, 16384, terms, buf, wk)
            cells.append(f"{r['units'] / sms / r['cycles']:.1f} ({r['units'] / (r['ms'] * 1e-3) / 1e12:.2f})")
        print(f"| {gb * 1024:.0f} MiB | " + " | ".join(cells) + " |", flush=True)
        del buf
        torch.cuda.empty_cache()


def main():
    import torch
    assert torch.cuda.is_available(), "needs a CUDA device"
    if "--sweep" in sys.argv:
        return sweep()
    res = measure(quick="--quick" in sys.argv)
    if "--json" in sys.argv:
        print(json.dumps(res))
        return
    print("| measurement | ms | load B/clk/SM | load TB/s | LDS B/clk/SM | LDS TB/s | adds/clk/SM | effective SM MHz |")
    print("|---|---|---|---|---|---|---|---|")
    for k, v in res.items():
        if not isinstance(v, dict):
            continue
        if "dram_group_TB_per_s" in v:
            print(f"| {k} | {v['ms']:.3f} | DRAM half: {v['dram_group_B_per_clk_per_SM']:.1f} | {v['dram_group_TB_per_s']:.2f} | "
                  f"L2 half: {v['l2_group_B_per_clk_per_SM']:.1f} (load) | {v['l2_group_TB_per_s']:.2f} |  | {v['sm_mhz_effective']:.0f} |")
            continue
        f = lambda key, fmt: (fmt % v[key]) if key in v else ""
        print(f"| {k} | {v['ms']:.3f} | {f('load_B_per_clk_per_SM', '%.1f')} | {f('load_TB_per_s', '%.2f')} | "
              f"{f('lds_B_per_clk_per_SM', '%.1f')} | {f('lds_TB_per_s', '%.2f')} | {f('adds_per_clk_per_SM', '%.1f')} | "
              f"{v['sm_mhz_effective']:.0f} |")
    print(f"\nSMs: {res['sms']}; {torch.cuda.get_device_name()}")


if __name__ == "__main__":
    main()
