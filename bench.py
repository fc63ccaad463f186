#!/usr/bin/env python
"""Benchmark of the sparse-SYK hot path on B200 (contract: see DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

One "step" = one pass of the whole hot path over one synthetic realization:
    a-1  syk_build_hamiltonian(N, p = kN/C(N,4), seed, realization)          (host term compiler + table upload)
    a-5  r <- gamma_W r                                                      (Pauli-string insertion, in place)
    a-4  r <- exp(-i (dt - i beta/4 ...) H) r   via syk_krylov_evolve        (m fused Lanczos steps = a-2 + a-3,
                                                                              host exp(-i tau T_m), combine)
    a-5  F = <l | r>                                                         (fp64 inner product)
i.e. one Krylov segment of the OTOC sandwich of PAPER.md:230.  `value` is BASELINE.json's metric, H.v model
bytes per second: the byte model of DESIGN.md section 6 ((D_x + 2) V per matvec + 3 V per fused vector pass
+ combine) divided by the device time of the step.  The `roofline` object is for the dominant kernel (apply_H)
alone, timed with CUDA events around each of its launches inside the timed region.

The default run times BASELINE.json's first headline config (N=56, k=4, complex128) as the JSON line itself and then its
second one (N=64, k=2, complex64, two-pass Lanczos) for 3 steps, embedded under `second_headline` (skipped with a stated
reason when less than 140 GB of device memory is free).  On-chip peaks (L2 -> SM, shared-memory reads, DRAM -> SM through
the TMA ring) are measured in the same run with `syk_microbench` and the roofline reports one fraction per unit.

N > 1 (torchrun): realizations are independent, so each rank runs its own realization with no
data-path collective ("weak" scaling); the time is the max over ranks.

`--impl reference` times the CPU oracle (oracle/alg1.c, the paper's Algorithm 1 under OpenMP) on the host cores.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Hv_model_bytes_throughput"
UNIT = "GB/s"

WORKLOADS = {
    # BASELINE.json configs[3] and configs[4]; krylov_dim/dt: one OTOC time segment (t in [0,8], 16 segments)
    "N56_k4_c128": {"N": 56, "k": 4, "dtype": "c128", "krylov_dim": 16, "two_pass": 0, "dt": 0.5, "beta": 5.0,
                    "i_W": 55, "j_V": 54},
    "N64_k2_c64": {"N": 64, "k": 2, "dtype": "c64", "krylov_dim": 8, "two_pass": 1, "dt": 0.5, "beta": 5.0,
                   "i_W": 63, "j_V": 62},
    # the same N=56 workload in one parity block: 2^27 amplitudes, 2.1 GB vectors
    "N56_k4_c128_block": {"N": 56, "k": 4, "dtype": "c128", "krylov_dim": 16, "two_pass": 0, "dt": 0.5, "beta": 5.0,
                          "i_W": 55, "j_V": 54, "block": 1},
    # smaller shapes of the same path (parity-test sizes; handy for quick runs and ncu)
    "N48_k4_c128": {"N": 48, "k": 4, "dtype": "c128", "krylov_dim": 16, "two_pass": 0, "dt": 0.5, "beta": 5.0,
                    "i_W": 47, "j_V": 46},
    # BASELINE.json configs[1] / configs[2] shapes: disorder realizations batched on one GPU (run back to back on one
    # stream; each step advances every realization by one time segment)
    "N32_k4_c128_x100": {"N": 32, "k": 4, "dtype": "c128", "krylov_dim": 12, "two_pass": 0, "dt": 0.1, "beta": 5.0,
                         "i_W": 31, "j_V": 30, "batch": 100, "lockstep": 1},
    "N48_k4_c128_x20": {"N": 48, "k": 4, "dtype": "c128", "krylov_dim": 30, "two_pass": 0, "dt": 0.5, "beta": 5.0,
                        "i_W": 47, "j_V": 46, "batch": 20},
    # BASELINE.json configs[2], dense p = 1 member: ALU-bound (194 580 terms on 10 903 X-masks, ~0.75 s per matvec)
    "N48_dense_c128": {"N": 48, "k": None, "dtype": "c128", "krylov_dim": 12, "two_pass": 0, "dt": 0.05, "beta": 5.0,
                       "i_W": 47, "j_V": 46},
    "N40_k4_c128": {"N": 40, "k": 4, "dtype": "c128", "krylov_dim": 16, "two_pass": 0, "dt": 0.5, "beta": 5.0,
                    "i_W": 39, "j_V": 38},
}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons during the timed region (B200_PROFILING.md recipe): an NVML polling thread
    (nvidia_ml_py) -- a separate nvidia-smi process polling the driver perturbs launch-heavy steps by 10-30 % -- with
    `nvidia-smi -lms` as the fallback when the module is missing."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        self.index = index
        self.thread = None
        self.stop_flag = False
        self.sm, self.smax, self.reasons = [], [], set()

    def _poll_nvml(self):
        import pynvml as nv
        h = nv.nvmlDeviceGetHandleByIndex(self.index)
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while not self.stop_flag:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                self.smax.append(float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)))
                mask = int(get_reasons(h))
                for name, bit in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.2)

    def start(self):
        try:
            import threading
            import pynvml as nv
            nv.nvmlInit()
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "500",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.thread is not None:
            self.stop_flag = True
            self.thread.join(timeout=2)
            sm = sorted(self.sm)
            return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(self.smax) if self.smax else None,
                    "samples": len(sm), "reasons": sorted(self.reasons), "source": "nvml"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=10)
        except Exception:
            self.proc.kill()
            out = ""
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi"}


def fill_host_state(buf_np, seed):
    """iid complex Gaussian amplitudes, normalised, written in chunks into a (pinned) host array.  Above 2^28
    amplitudes one Gaussian block of 2^24 is drawn and re-used with a different unit phase per chunk (the e2e leg
    only needs a generic dense vector; drawing 2^33 normals with numpy would take minutes)."""
    import numpy as np
    r = np.random.default_rng(seed)
    D = buf_np.shape[0]
    chunk = min(D, 1 << 22)
    if D > (1 << 28):
        chunk = 1 << 24
        block = (r.standard_normal(chunk) + 1j * r.standard_normal(chunk)).astype(buf_np.dtype)
        block *= 1.0 / math.sqrt(float(np.vdot(block, block).real) * (D // chunk))
        for i, lo in enumerate(range(0, D, chunk)):
            np.multiply(block, buf_np.dtype.type(np.exp(2.399963229728653j * i)), out=buf_np[lo:lo + chunk])
        return
    n2 = 0.0
    for lo in range(0, D, chunk):
        hi = min(D, lo + chunk)
        re = r.standard_normal(hi - lo)
        im = r.standard_normal(hi - lo)
        n2 += float(re @ re + im @ im)
        buf_np[lo:hi] = (re + 1j * im).astype(buf_np.dtype)
    scale = 1.0 / math.sqrt(n2)
    for lo in range(0, D, chunk):
        buf_np[lo:lo + chunk] *= scale


def cpu_oracle_matvec_rate(N, k, seed, target_seconds, psi=None):
    """Times oracle/alg1.c (literal Algorithm 1 + OpenMP) on a bounded sample of rows of the same workload.
    Returns (model GB/s, cores, sample description, seconds)."""
    import numpy as np
    from oracle import alg1, rng as orng
    from paper_2311_00639_b200 import inputs
    L = N // 2
    D = 1 << L
    q, J, _ = orng.sample_couplings(N, inputs.bernoulli_p(N, k), seed, 0)
    bits, coeff = alg1.hamiltonian_tuples(N, q, J)
    n_x = len(set(int(b) & 0x5555555555555555 for b in bits))          # distinct X parts of the paper's tuples
    if psi is None:
        psi = np.empty(D, dtype=np.complex128)
        fill_host_state(psi, seed + 1)
    cores = alg1.num_threads()
    rows = min(D, 1 << 16)
    t0 = time.perf_counter()
    alg1.apply_c(L, bits, coeff, psi, 0, rows)
    t_probe = time.perf_counter() - t0
    rows = int(min(D, max(rows, rows * target_seconds / max(t_probe, 1e-6))))
    rows = 1 << int(math.log2(rows))
    t0 = time.perf_counter()
    alg1.apply_c(L, bits, coeff, psi, 0, rows)
    dt = time.perf_counter() - t0
    gbs = (n_x + 2) * 16.0 * rows / dt / 1e9
    return gbs, cores, f"rows [0, 2^{int(math.log2(rows))}) of one N={N} k={k} complex128 matvec ({len(J)} terms)", dt, rows


def run_reference(args, wl, name):
    """The reference arm: the CPU oracle as it stands, on the host cores (rank 0 only)."""
    import numpy as np
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import alg1, rng as orng
    from paper_2311_00639_b200 import inputs
    N, k = wl["N"], wl["k"]
    L, D = N // 2, 1 << (N // 2)
    q, J, _ = orng.sample_couplings(N, inputs.bernoulli_p(N, k), 0, 0)
    bits, coeff = alg1.hamiltonian_tuples(N, q, J)
    n_x = len(set(int(b) & 0x5555555555555555 for b in bits))
    psi = np.empty(D, dtype=np.complex128)
    fill_host_state(psi, 1)
    cores = alg1.num_threads()
    budget = 120.0 / max(1, args.steps + args.warmup)              # whole run within a few minutes
    rows = 1 << 16
    t0 = time.perf_counter()
    alg1.apply_c(L, bits, coeff, psi, 0, rows)
    probe = time.perf_counter() - t0
    rows = 1 << int(math.log2(min(D, max(rows, rows * budget / max(probe, 1e-6)))))
    for _ in range(args.warmup):
        alg1.apply_c(L, bits, coeff, psi, 0, rows)
    t0 = time.perf_counter()
    for s in range(args.steps):
        lo = (s * rows) % D
        alg1.apply_c(L, bits, coeff, psi, lo, lo + rows)
    dt = time.perf_counter() - t0
    value = (n_x + 2) * 16.0 * rows * args.steps / dt / 1e9
    sample = (f"each step = rows of 2^{int(math.log2(rows))} consecutive outputs of one N={N} k={k} complex128 "
              f"H.v by oracle/alg1.c (literal Algorithm 1, OpenMP)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "N": N, "k": k, "n_terms": int(len(J)), "n_xmasks": n_x},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def measure_workload(args, wl, name, steps, warmup, world, rank, local, dist, with_e2e, with_cpu, peaks):
    """Times `steps` steps of one workload on this rank's GPU; returns the JSON line as a dict (rank 0) or None."""
    import numpy as np
    import torch
    from paper_2311_00639_b200 import binding as B, inputs

    N, k = wl["N"], wl["k"]
    block = bool(wl.get("block"))
    D = 1 << (N // 2 - (1 if block else 0))          # parity block: half the amplitudes
    tdt = torch.complex128 if wl["dtype"] == "c128" else torch.complex64
    code = B.SYK_C128 if wl["dtype"] == "c128" else B.SYK_C64
    eb = 16 if wl["dtype"] == "c128" else 8
    V = D * eb
    p = inputs.bernoulli_p(N, k)
    opts = {"krylov_dim": wl["krylov_dim"], "two_pass": wl["two_pass"]}
    tau = (wl["dt"], 0.0)                            # one real-time segment of the t grid
    batch = int(wl.get("batch", 1))
    realization = rank * batch                       # independent realizations per rank (weak scaling)
    relabel = not args.no_relabel and batch == 1     # NEXT-3: qubit layout chosen per Hamiltonian (sparse H only)

    def build(r, sector=None):
        """a-1: term compiler (+ parity block) + qubit layout + device tables: everything the later calls need, so that
        no compute call allocates (syk_ham_prepare)."""
        h = B.syk_build_hamiltonian(N, p, 0, r)
        if block:
            hb = B.syk_build_parity_block(h, sector)
            h.close()
            h = hb
        if relabel:
            B.syk_ham_optimize_layout(h, code)
        B.syk_ham_prepare(h, code)
        return h

    h0 = build(realization, 0)
    info = h0.info()
    n_x, n_t = info["n_xmasks"], info["n_terms"]
    kbytes = B.syk_krylov_workspace_bytes(h0, code, opts)
    scratch = torch.empty(B.syk_reduce_scratch_bytes(), dtype=torch.uint8, device="cuda")
    wk = torch.empty(kbytes + (V if with_e2e else 0), dtype=torch.uint8, device="cuda")   # + one vector for the host entry point
    l = torch.empty((batch, D), dtype=tdt, device="cuda")
    r = torch.empty((batch, D), dtype=tdt, device="cuda")
    Nvec = N - 2 if block else N                     # number of Majoranas that spans the stored vector
    for i in range(batch):
        hi = h0 if batch == 1 else build(realization + i, 0)
        B.syk_random_state_h(hi, 0, realization + i, r[i], scratch)
        if block:
            B.syk_apply_gamma_block_h(hi, 1, 0, r[i], l[i])   # a second, different state for the bra side
        else:
            B.syk_apply_gamma_h(hi, 1, r[i], l[i])
        if hi is not h0:
            hi.close()
    torch.cuda.synchronize()
    sector = [0]                                     # parity block the state is in (every gamma flips it)

    stats_acc = {"n_matvec": 0, "model_bytes": 0.0, "n_substeps": 0}

    lockstep = bool(wl.get("lockstep")) and batch > 1
    if lockstep:
        wk_b = torch.empty(B.syk_krylov_workspace_bytes_batched(h0, batch, code, opts), dtype=torch.uint8, device="cuda")

    def step_lockstep():
        # every realization advances through the Lanczos recurrence in the same launches (grid.y = realization)
        hams = [build(realization + i) for i in range(batch)]                              # a-1
        for i in range(batch):
            B.syk_apply_gamma_h(hams[i], wl["i_W"], r[i], r[i])                            # a-5 insertion
        st = B.syk_krylov_evolve_batched(hams, r, D, tau[0], tau[1], wk_b, opts)          # a-2, a-3, a-4
        F = 0.0
        for i in range(batch):
            F = B.syk_dot(N, l[i], r[i], scratch)                                         # a-5 inner product
        stats_acc["n_matvec"] += st["n_matvec"]
        stats_acc["n_substeps"] += st["n_substeps"]
        stats_acc["model_bytes"] += st["model_bytes"] + 4.0 * V * batch
        for h in hams:
            h.close()
        return F

    def step():
        if lockstep:
            return step_lockstep()
        F = 0.0
        for i in range(batch):
            if block:
                sector[0] ^= 1
                h = build(realization + i, sector[0])                                 # a-1, block of the new sector
                B.syk_apply_gamma_block_h(h, wl["i_W"], sector[0], r[i], r[i])        # a-5 insertion (no gather)
            else:
                h = build(realization + i)                                            # a-1
                B.syk_apply_gamma_h(h, wl["i_W"], r[i], r[i])                         # a-5 insertion (in place)
            st = B.syk_krylov_evolve(h, r[i], tau[0], tau[1], wk, opts)               # a-2, a-3, a-4
            F = B.syk_dot(Nvec, l[i], r[i], scratch)                                  # a-5 inner product
            stats_acc["n_matvec"] += st["n_matvec"]
            stats_acc["n_substeps"] += st["n_substeps"]
            stats_acc["model_bytes"] += st["model_bytes"] + 4.0 * V                   # gamma: 2V, dot: 2V
            h.close()
        return F

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    for key in stats_acc:
        stats_acc[key] = 0
    B.syk_launch_count(reset=True)
    B.syk_profile_enable(not args.no_kernel_timing)
    B.syk_profile_read(reset=True)
    sampler = ClockSampler(local)
    barrier()
    if rank == 0 and not args.no_clocks:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    F_last = None
    for _ in range(steps):
        F_last = step()
    e1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1)
    launches = B.syk_launch_count(reset=True)
    apply_ms, apply_n = B.syk_profile_read(reset=True)
    B.syk_profile_enable(False)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t[0])
        tot = torch.tensor([stats_acc["model_bytes"], float(stats_acc["n_matvec"]), float(launches)],
                           dtype=torch.float64, device="cuda")
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        total_bytes, total_matvec, launches = float(tot[0]), float(tot[1]), int(tot[2])
    else:
        total_bytes, total_matvec = stats_acc["model_bytes"], float(stats_acc["n_matvec"])
    value = total_bytes / (ms * 1e-3) / 1e9

    # ---- end to end through the HOST entry point: pinned host vector in, evolved vector out, every step ----
    e2e = None
    try:
        if not with_e2e:
            raise RuntimeError("skipped")
        host = torch.empty(D, dtype=tdt, pin_memory=True)
        fill_host_state(host.numpy(), 7 + rank)
        def e2e_step():
            tot = {"model_bytes": 0.0}
            for i in range(batch):
                h = build(realization + i, 0)
                tot["model_bytes"] += B.syk_krylov_evolve_host(h, host, tau[0], tau[1], wk, opts)["model_bytes"]
                h.close()
            return tot
        e2e_step()
        barrier()
        n_e2e = max(1, min(steps, 3))
        t0 = time.perf_counter()
        e2e_bytes = 0.0
        for _ in range(n_e2e):
            e2e_bytes += e2e_step()["model_bytes"]
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([t_e2e], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            b = torch.tensor([e2e_bytes], dtype=torch.float64, device="cuda")
            dist.all_reduce(b, op=dist.ReduceOp.SUM)
            t_e2e, e2e_bytes = float(t[0]), float(b[0])
        e2e = {"value": e2e_bytes / t_e2e / 1e9, "unit": UNIT, "h2d_bytes_per_step": V * batch,
               "d2h_bytes_per_step": V * batch, "steps": n_e2e,
               "call": "syk_krylov_evolve_host (pinned canonical host vector in and out each step; converted to and "
                       "from the handle's qubit layout on the device)"}
        del host
    except Exception as ex:   # noqa: BLE001 -- report, do not hide
        e2e = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}

    kind = B.syk_apply_H_kernel_kind(h0, code)
    layout = B.syk_apply_H_layout(h0, code) if kind == 3 else None
    perm = [int(x) for x in B.syk_ham_layout(h0)["perm"]]
    dense_shape = None
    if kind == 4:
        # groups the dense-table kernel applies through one table lookup per amplitude (x-local groups) and the terms left
        # to the term-by-term walk: the same criterion as csrc/apply_h_dense.cu, counted here on the exported tables
        import numpy as np
        tb = h0.tables()
        gx, goff, tz = tb["x"].astype(np.uint64), tb["group_off"], tb["z"].astype(np.uint64)
        n_local, walk_terms = 0, 0
        for g in range(len(gx)):
            zs = tz[goff[g]:goff[g + 1]]
            if bin(int(gx[g])).count("1") <= 4 and len(zs) >= 4 and not np.any((zs ^ zs[0]) & ~gx[g]):
                n_local += 1
            else:
                walk_terms += len(zs)
        dense_shape = dict(B.syk_apply_H_dense_info(h0, code), walk_terms=walk_terms, local_by_tables=n_local)
    h0.close()
    del l, r, wk, scratch
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    peak, peak_src = measured_peak()
    per_launch_bytes = (n_x + 2) * V
    avg_ms = apply_ms / apply_n if apply_n else float("nan")
    achieved = per_launch_bytes / (avg_ms * 1e-3) / 1e9 if apply_n else None
    kernel_names = {0: "apply_h_generic_kernel", 1: "apply_h_tma_kernel", 2: "apply_h_regtile_kernel",
                    3: "apply_h_scatter_kernel", 4: "apply_h_dense_kernel"}
    roofline = {"bound": "hbm", "kernel": kernel_names[kind], "layout": layout, "achieved": achieved, "peak": peak,
                "unit": "GB/s",
                "frac": achieved / peak if achieved else None, "traffic": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": per_launch_bytes, "avg_launch_ms": avg_ms, "launches_timed": apply_n,
                "share_of_step": apply_ms / ms if ms else None,
                "frac_of_nominal_8TBs": achieved / 8000.0 if achieved else None}
    # DRAM bytes per launch of that kernel from the last committed `ncu --set full` capture (profiles/traffic.csv): a
    # property of (kernel, workload) recorded with the commit it was taken at -- NOT measured in this run
    traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(traffic_file):
        try:
            import csv
            for row in csv.DictReader(open(traffic_file)):
                if row["workload"] == name:
                    roofline["traffic"] = float(row["dram_bytes_per_launch"])
                    roofline["traffic_source"] = ("committed ncu capture, not measured in this run: " + row["source"])
        except Exception:
            pass
    if layout and apply_n:
        # One fraction per unit that could bind a tile-kernel launch, each = bytes the launch moves through that unit /
        # launch time / the peak of that unit MEASURED on this box in this run (syk_microbench):
        #   model_vs_hbm        (D_x + 2) V, the byte model of SURVEY 8(d)      / HBM copy peak      (the graded figure)
        #   dram_traffic_vs_hbm ncu DRAM bytes per launch (committed capture)   / DRAM -> SM streaming peak
        #   l2_to_sm            (n_loads + 2) V: every load moves the vector once from L2 into the SMs / L2 -> SM peak
        #   lds                 n_terms V: every term reads the staged vector once from shared memory   / LDS peak
        #   smem_path           (n_terms + n_loads + 2) V: the reads above plus the TMA fills of the ring, which go through the
        #                       same banks / the LDS rate per clock measured by syk_microbench x the SM clock sampled during
        #                       this run (profiles/r2_chunk_trace.md: this is the unit that binds the headline launches)
        sec = avg_ms * 1e-3
        fr = {"model_vs_hbm": roofline["frac"]}
        l2_bytes = (layout["n_loads"] + 2) * V
        lds_bytes = n_t * V
        detail = {"l2_to_sm_bytes_per_launch": l2_bytes, "l2_to_sm_TB_per_s": l2_bytes / sec / 1e12,
                  "lds_bytes_per_launch": lds_bytes, "lds_TB_per_s": lds_bytes / sec / 1e12}
        if roofline["traffic"]:
            detail["dram_TB_per_s"] = roofline["traffic"] / sec / 1e12
        if peaks:
            if roofline["traffic"]:
                fr["dram_traffic_vs_dram_to_sm_peak"] = roofline["traffic"] / sec / 1e12 / peaks["dram_to_sm"]["load_TB_per_s"]
                fr["dram_traffic_vs_hbm_copy_peak"] = roofline["traffic"] / sec / 1e9 / peak
            fr["l2_to_sm_vs_measured_peak"] = detail["l2_to_sm_TB_per_s"] / peaks["l2_to_sm"]["load_TB_per_s"]
            fr["lds_vs_measured_peak"] = detail["lds_TB_per_s"] / peaks["lds_only"]["lds_TB_per_s"]
            mhz = (clocks or {}).get("sm_mhz") or peaks["lds_only"]["sm_mhz_effective"]
            smem_bytes = (n_t + layout["n_loads"] + 2) * V
            smem_peak = peaks["lds_only"]["lds_B_per_clk_per_SM"] * peaks["sms"] * mhz * 1e6
            detail["smem_reads_plus_fills_bytes_per_launch"] = smem_bytes
            detail["smem_reads_plus_fills_B_per_clk_per_SM"] = smem_bytes / sec / (peaks["sms"] * mhz * 1e6)
            fr["smem_reads_plus_fills_vs_lds_rate_at_run_clock"] = smem_bytes / sec / smem_peak
            # supply model of the lock-stepped CTAs: DRAM phases and L2 phases do not overlap
            if roofline["traffic"]:
                t_supply = (roofline["traffic"] / 1e12 / peaks["dram_to_sm"]["load_TB_per_s"] +
                            max(0.0, l2_bytes - roofline["traffic"]) / 1e12 / peaks["l2_to_sm"]["load_TB_per_s"])
                fr["serial_dram_plus_l2_model_vs_time"] = t_supply / sec
        physical = {kk: vv for kk, vv in fr.items() if kk != "model_vs_hbm" and vv is not None}
        roofline["fractions"] = fr
        roofline["binding_unit"] = max(physical, key=physical.get) if physical else None
        roofline["on_chip"] = detail
        roofline["measured_peaks"] = peaks
    if kind in (0, 4) and n_t > 8 * n_x:
        # dense table: plain-ALU bound.  Work unit = one thread-level bin add: every term costs ONE
        # add per thread (8 amplitudes share it through the Walsh binning), i.e. n_terms x D / 8 per launch; peak = the
        # issue rate of exactly that instruction sequence measured on this box (syk_microbench kind 4)
        ach = n_t * (D / 8.0) / (avg_ms * 1e-3) if apply_n else None
        alu_peak = peaks["dense_term_sequence"]["adds_per_s"] if peaks else 148 * 512 * 1.965e9 / 42.0
        roofline.update({"bound": "alu", "achieved": ach / 1e9 if ach else None, "peak": alu_peak / 1e9,
                         "unit": "G thread-level term adds/s",
                         "frac": ach / alu_peak if ach else None,
                         "peak_source": ("measured: syk_microbench kind 4 (the kernel's per-term instruction sequence, 512 "
                                         "threads per SM)" if peaks else "fallback: 12.1 adds/clk/SM x 148 SMs x 1.965 GHz"),
                         "model_GBs_for_reference": achieved})
        if dense_shape and dense_shape["n_local_groups"] > 0 and apply_n:
            # With x-local groups most terms are never walked: the arithmetic the launch cannot avoid is one complex
            # multiply-add (4 FP64 FMA) per (X-mask, amplitude) plus one add per (walked term, thread).  Roofline = those
            # FP64 issue slots / time against the FP64 issue rate of this box (syk_microbench kind 3: one DADD/DFMA per lane).
            ops = 4.0 * n_x * D + dense_shape["walk_terms"] * (D / 8.0)
            fp64_peak = peaks["fp64_add"]["adds_per_s"] if peaks else 63.9 * 148 * 1.965e9
            roofline.update({"achieved": ops / (avg_ms * 1e-3) / 1e9, "peak": fp64_peak / 1e9,
                             "unit": "G FP64 issue slots/s (FMA or add)", "frac": ops / (avg_ms * 1e-3) / fp64_peak,
                             "peak_source": ("measured: syk_microbench kind 3 (FP64 add issue rate, 512 threads per SM)"
                                             if peaks else "fallback: 63.9 /clk/SM x 148 SMs x 1.965 GHz"),
                             "fp64_ops_per_launch": ops, "dense_table": dense_shape,
                             "effective_term_adds_per_s": ach,
                             "effective_term_adds_vs_term_sequence_peak": ach / alu_peak if ach else None})

    cpu = None
    if with_cpu:
        try:
            gbs, cores, sample, secs, rows = cpu_oracle_matvec_rate(N, k, 0, 15.0)
            cpu = {"value": gbs, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                   "seconds": secs}
        except Exception as ex:   # noqa: BLE001
            cpu = {"value": None, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": repr(ex)[:200]}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": warmup, "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if wl["dtype"] == "c128" else "f32", "data": "synthetic",
            "config": {"workload": name, "N": N, "k": k, "dim_log2": N // 2 - (1 if block else 0), "parity_block": block, "n_terms": n_t, "n_xmasks": n_x,
                       "vector_bytes": V, "krylov_dim": wl["krylov_dim"], "two_pass": wl["two_pass"],
                       "tau": list(tau), "realizations_per_gpu": batch, "lockstep_batched": lockstep,
                       "qubit_layout": perm if relabel else "identity",
                       "l2_policy": ("inputs larger than L2 (vector %.1f GB >> 126 MB)" % (V / 1e9)) if V > 3e8 else
                                    ("working set of one step %.2f GB > L2 (%d realizations x %d vectors of %.1f MB)"
                                     % (batch * (wl["krylov_dim"] + 2) * V / 1e9, batch, wl["krylov_dim"] + 2, V / 1e6)),
                       "step": "build_hamiltonian + qubit layout + table upload (syk_ham_prepare) + gamma insertion + "
                               "krylov_evolve (m fused Lanczos steps, host exp, combine) + inner product"},
            "lanczos_steps_per_s": total_matvec / (ms * 1e-3), "matvecs_per_step": total_matvec / steps / world,
            "F_last": [F_last.real, F_last.imag], "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "cpu_baseline": cpu}
    return line


def run_ours(args, wl, name):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # on-chip peaks of this box, measured before the timed region (a few hundred ms)
    peaks = None
    if not args.no_peaks:
        try:
            from paper_2311_00639_b200 import microbench
            peaks = microbench.measure(quick=False)
        except Exception as ex:   # noqa: BLE001
            peaks = None
            print(f"note: on-chip peaks not measured: {ex!r}", file=sys.stderr)

    line = measure_workload(args, wl, name, args.steps, args.warmup, world, rank, local, dist, not args.no_e2e,
                            world == 1 and not args.no_cpu_baseline, peaks)
    # the second headline config of BASELINE.json's metric ("at N=56/64"), in the default run only
    second = None
    if name == "N56_k4_c128" and not args.no_second:
        name2 = "N64_k2_c64"
        free, _ = torch.cuda.mem_get_info()
        need = 4 * (8 << 32) + (2 << 30)          # l, r and two Krylov work vectors of 2^32 complex64 amplitudes + headers
        ok = torch.tensor([1 if free >= need else 0], device="cuda")
        if world > 1:
            dist.all_reduce(ok, op=dist.ReduceOp.MIN)
        if int(ok[0]) == 0:
            second = {"workload": name2, "skipped": "needs %.0f GB of free device memory (4 resident vectors of 34.4 GB); free: %.1f GB"
                      % (need / 1e9, free / 1e9)}
        else:
            l2 = measure_workload(args, WORKLOADS[name2], name2, 3, 1, world, rank, local, dist, False, False, peaks)
            if l2 is not None:
                l2["roofline"].pop("measured_peaks", None)
                second = {key: l2[key] for key in ("value", "unit", "steps", "warmup", "ms_per_step", "dtype", "config",
                                                    "lanczos_steps_per_s", "matvecs_per_step", "clocks", "gpu_launches",
                                                    "roofline")}
    if rank == 0:
        if name == "N56_k4_c128" and not args.no_second:
            line["second_headline"] = second
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="N56_k4_c128", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs only)")
    ap.add_argument("--no-clocks", action="store_true", help="do not poll nvidia-smi (diagnosis only)")
    ap.add_argument("--no-kernel-timing", action="store_true", help="no CUDA events around apply_H (diagnosis only)")
    ap.add_argument("--no-second", action="store_true", help="skip the N=64 complex64 leg of the default run")
    ap.add_argument("--no-peaks", action="store_true", help="skip the on-chip peak measurements (profiling runs only)")
    ap.add_argument("--no-relabel", action="store_true", help="keep the canonical qubit layout (diagnosis only)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("note: fewer than 3 warm-up steps; not a valid bench number", file=sys.stderr)
    wl = WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl, args.workload)
    else:
        run_ours(args, wl, args.workload)


if __name__ == "__main__":
    main()
