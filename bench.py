#!/usr/bin/env python
"""bench.py — E_loc throughput of the hot path on the 76-qubit workload (BASELINE.json `metric`).

A "step" = one pass of the whole hot path (a2-a7: connected configs, Pauli contraction, MADE forward on
every connected configuration, psi-ratio reduction, count-weighted statistics) over ONE
gradient-accumulation mini-batch of 8,192 unique samples of config 5 against ALL unique-flip groups of
the 76-qubit Hamiltonian (the batch is processed "into several mini-batches"; step k of
rank r takes mini-batch (k*N + r) mod 8 of the 65,536 configured samples).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--path auto|simt|tc] [--cfg 5]

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "E_loc throughput (sample*Pauli-term pairs/s) at 76 qubits"
UNIT = "pairs/s"


def algorithmic_flops_per_eval(params):
    """2*nnz(M1, M2, M3) + 2*((n-2)h + 4h) per psi evaluation (masked MACs only; padding,
    masked-zero MACs and extra split-precision passes are overhead, not algorithmic work).  Host-side mask
    count from the degrees — bookkeeping, not method arithmetic."""
    n, h = params.n_qubits, params.hidden
    deg = np.asarray(params.deg_hidden, dtype=np.int64)
    m_in = np.arange(1, n + 1)
    nnz = int((deg[0][:, None] >= m_in[None, :]).sum())
    for k in range(1, deg.shape[0]):
        nnz += int((deg[k][:, None] >= deg[k - 1][None, :]).sum())
    nnz += int((m_in[:, None] > deg[-1][None, :]).sum())
    return 2 * nnz + 2 * ((n - 2) * h + 4 * h)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "tensor_tflops": d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                "tensor_tflops_burst": d["bf16_tflops"], "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "tensor_tflops": 1400.0, "tensor_tflops_burst": 1590.0, "sm_max_mhz": 1965.0,
            "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any(len(r) >= 6 and r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def build_inputs(cfg, need_samples):
    from paper_2208_05637_b200 import workloads as wl
    w = wl.WORKLOADS[cfg]
    h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = wl.jw_pauli_terms(h, g)
    params = wl.make_made_params(w.n_qubits, w.hidden, w.seed_weights)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, need_samples, w.max_count, w.seed_samples, w.unique)
    return w, (x, z, c), params, samples, counts


def time_oracle(w, ham, params, samples, n_samples, one_thread=False):
    """The oracle as it stands (fp64 numpy, memoised mode) on the host cores; returns (pairs/s, seconds, threads).
    one_thread=True pins the BLAS pool the oracle's matmuls run on to a single thread (the oracle is
    timed on all cores and on one)."""
    import contextlib
    from paper_2208_05637_b200 import workloads as wl
    from oracle import eloc as oeloc
    x, z, c = ham
    codes = wl.masks_to_codes(x, z, w.n_qubits)
    limit = contextlib.nullcontext()
    try:
        from threadpoolctl import threadpool_info, threadpool_limits
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
        if one_thread:
            limit, threads = threadpool_limits(limits=1), 1
    except Exception:
        threads = os.cpu_count()
    with limit:
        t0 = time.perf_counter()
        oeloc.local_energy(codes, c, params, samples[:n_samples], memo=True)
        dt = time.perf_counter() - t0
    return n_samples * len(c) / dt, dt, threads


# Constants read from ncu captures (profiles/r3_ncu_counters.md gives the commands).  They describe the kernel SOURCE they
# were captured on: each carries the sha256 (first 16 hex) of the .cu files it depends on, and bench.py reports a constant
# only while those files are unchanged -- a stale capture is omitted, not repeated.
NCU_CAPTURES = {
    # DRAM bytes (read + write) of ONE eloc_tc_kernel launch, keyed by (cfg, samples per launch)
    "eloc_tc_dram_bytes": {"files": ["kernels_tc.cu", "tc_ptx.cuh"], "sha16": "c59e0af701c9581a",
                           "values": {(5, 8192): 1067126912}},      # mean of two launches: 1.046 GB read + 21 MB written
    # thread-level instructions executed per (sample, term) pair by contract_kernel, summed over the 144 launches of one
    # sweep over all groups of cfg 5 (8,192 samples): smsp__thread_inst_executed.sum / (B * K)
    "contract_thread_inst_per_pair": {"files": ["kernels_simt.cu", "nqs_internal.h"], "sha16": "75b0c7f177203c5c",
                                      "values": {5: 23.71}},
}


def _source_sha16(files):
    import hashlib
    h = hashlib.sha256()
    for f in files:
        with open(os.path.join(ROOT, "paper_2208_05637_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_constant(name, key):
    """The captured value, or None when there is no capture for `key` or the kernel source changed since."""
    c = NCU_CAPTURES[name]
    if key not in c["values"] or c["sha16"] != _source_sha16(c["files"]):
        return None
    return c["values"][key]


def time_contraction(nqs, torch, H, xs, stream, clocks_mhz):
    """Standalone Pauli contraction (a3, nqs_pauli_contract) of one mini-batch against ALL groups, in group chunks
    that reuse one output buffer (S is never materialised whole: B x G x 8 bytes would be 38 GB at cfg 5).
    ALU roofline: SMs (device attribute) x 128 INT/FP32 lanes x SM clock.  Two per-pair operation counts are reported:
    the model count of SURVEY.md 8(d) (7 lane-operations: AND, popcount, parity, sign inject, 2 FP32 adds, select), and --
    when a capture of the current kernel source exists -- the thread-level instructions ncu counted per pair (loads,
    address arithmetic, the per-group prologue and store amortised over ~4.8 terms), which is what the lanes actually saw.  The sweep writes B x G x 8 bytes
    of S to HBM, so for groups of ~5 terms the figure is as much a store rate as a popcount rate (hbm_write_gbs)."""
    B, G, K = xs.shape[0], H.G, H.K
    chunk = max(1, min(G, (256 << 20) // (B * 8)))
    out = torch.empty((chunk, B, 2), dtype=torch.float32, device=xs.device)
    L = nqs.lib()

    def sweep():
        for g0 in range(0, G, chunk):
            g1 = min(G, g0 + chunk)
            rc = L.nqs_pauli_contract(H._h, xs.data_ptr(), B, g0, g1, out.data_ptr(), stream.cuda_stream)
            assert rc == 0, rc
    sweep()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    sweep()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    pairs_s = B * K / (ms / 1e3)
    sms = torch.cuda.get_device_properties(xs.device).multi_processor_count
    peak = sms * 128 * clocks_mhz * 1e6
    counted = ncu_constant("contract_thread_inst_per_pair", 5) if (B, K) == (8192, 2802815) else None
    return {"value": pairs_s, "unit": "pairs/s", "ms": ms, "launches": (G + chunk - 1) // chunk, "sms": sms,
            "lane_ops_per_pair_model": 7, "alu_peak_lane_ops_per_s": peak, "alu_frac_model": 7 * pairs_s / peak,
            "thread_inst_per_pair_counted": counted,
            "lane_frac_counted": (counted * pairs_s / peak) if counted else None,
            "hbm_write_gbs": B * G * 8 / (ms / 1e3) / 1e9,
            "note": "standalone nqs_pauli_contract over all groups; S chunks are written to HBM (the fused path keeps them in registers)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="auto", choices=["auto", "simt", "tc"])
    ap.add_argument("--cfg", type=int, default=5)
    ap.add_argument("--oracle-samples", type=int, default=0, help="samples for the cpu_baseline leg (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-contraction", action="store_true", help="skip the standalone contraction figure")
    ap.add_argument("--no-full-config", action="store_true",
                    help="skip the one call over all 65,536 samples as 8 mini-batches (cfg 5: ~20 s)")
    ap.add_argument("--iteration", action="store_true",
                    help="also time one whole VMC iteration through the ABI: sampler -> E_loc -> gradient")
    ap.add_argument("--mb-samples", type=int, default=0,
                    help="profiling aid: samples per step instead of the configured mini-batch (labelled in config)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2208_05637_b200 import workloads as wl
    w = wl.WORKLOADS[args.cfg]
    n_oracle = args.oracle_samples or {1: 256, 2: 64, 3: 16, 4: 4, 5: 2}[args.cfg]
    workload_name = (f"cfg{args.cfg}: {w.n_qubits} qubits, h={w.hidden}, one {args.mb_samples or w.minibatch}-sample "
                     f"mini-batch x all unique-flip groups per step" + (" [REDUCED mini-batch: profiling run]" if args.mb_samples else ""))

    # ---------------- reference arm: the oracle on the host cores (rank 0 only) ----------------
    if args.impl == "reference":
        if rank != 0:
            return
        wq, ham, params, samples, counts = build_inputs(args.cfg, max(n_oracle * (args.steps + args.warmup), n_oracle))
        K = len(ham[2])
        times = []
        for s in range(args.warmup + args.steps):
            sl = samples[s * n_oracle:(s + 1) * n_oracle]
            v, dt, threads = time_oracle(wq, ham, params, sl, n_oracle)
            if s >= args.warmup:
                times.append(dt)
        ms = 1e3 * sum(times) / len(times)
        val = n_oracle * K / (ms / 1e3)
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_name, "n_terms": K,
                           "sample": f"{n_oracle} sample(s) x all {K} terms per step (memoised oracle mode)"},
                "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle",
                                 "sample": f"{n_oracle} of {wq.minibatch} samples of the mini-batch x all {K} terms"},
                "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return

    # ---------------- our arm ----------------
    import torch
    import paper_2208_05637_b200 as nqs
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))

    wq, ham, params, samples, counts = build_inputs(args.cfg, w.batch)
    x, z, c = ham
    H = nqs.ham_compile_packed(wq.n_qubits, x, z, c)
    M = nqs.made_create(params)
    path = {"auto": nqs.PATH_AUTO, "simt": nqs.PATH_SIMT, "tc": nqs.PATH_TC}[args.path]
    mb = args.mb_samples or wq.minibatch
    n_mb = wq.batch // mb
    xs_all = torch.from_numpy(samples.view(np.int64)).to(dev)
    cnt_all = torch.from_numpy(counts).to(dev)
    out = torch.empty((mb, 2), dtype=torch.float32, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)      # > 126 MB L2
    stream = torch.cuda.current_stream()

    from paper_2208_05637_b200.distributed import minibatch_of_step, max_over_ranks, all_reduce_stats

    def step(k):
        b = minibatch_of_step(k, rank, world, n_mb)
        return nqs.local_energy(H, M, xs_all[b * mb:(b + 1) * mb], cnt_all[b * mb:(b + 1) * mb], minibatch=mb,
                                path=path, want_stats=True, stream=stream, out=out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for k in range(args.warmup):
        step(k)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = nqs.kernel_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    chain_ms, chain_launches = 0.0, 0
    job_stats = torch.zeros(5, dtype=torch.float64, device=dev)
    for k in range(args.steps):
        flush.fill_(k & 0xFF)                                                   # L2 flush between timed iterations
        ev[k][0].record(stream)
        _, st_k = step(args.warmup + k)
        ev[k][1].record(stream)
        ms_k, nl = M.last_chain_kernel_ms()
        chain_ms += ms_k
        chain_launches += nl
        st_k = torch.from_numpy(st_k).to(dev)
        job_stats[:4] += st_k[:4]
        job_stats[4] = torch.maximum(job_stats[4], st_k[4])
    # the one exchange of the data-parallel design: the statistics of the mini-batches every rank
    # processed, 4 sums + 1 max, once per accumulation round -- inside the barrier-bracketed region, outside the events
    all_reduce_stats(job_stats)
    barrier()
    launches = nqs.kernel_launch_count() - launches0
    clocks = sampler.stop()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    total_ms = max_over_ranks(total_ms, dev)
    ms_per_step = total_ms / args.steps
    K, G = H.K, H.G
    pairs_per_step = mb * K * world
    value = pairs_per_step / (ms_per_step / 1e3)
    evals_per_s = mb * (G + 1) * world / (ms_per_step / 1e3)

    # ---- e2e: same metric through the host-buffer ABI call (pinned host memory, H2D + D2H inside) ----
    hs = torch.from_numpy(samples.view(np.int64)).pin_memory()
    hc = torch.from_numpy(counts).pin_memory()
    ho = torch.empty((mb, 2), dtype=torch.float32).pin_memory()
    e2e_steps = max(1, min(args.steps, 2))
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        b = minibatch_of_step(k, rank, world, n_mb)
        nqs.local_energy_host(H, M, hs[b * mb:(b + 1) * mb].numpy().view(np.uint64), hc[b * mb:(b + 1) * mb].numpy(),
                              minibatch=mb, path=path, want_stats=True, out=ho.numpy())
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps
    e2e_ms = max_over_ranks(e2e_ms, dev)
    e2e_val = pairs_per_step / (e2e_ms / 1e3)

    # ---- the configuration as BASELINE.json states it: every sample of the batch in ONE call, processed as
    # gradient-accumulation mini-batches (row a7), host buffers in, host buffers out, wall clock ----
    full_config = None
    if not args.no_full_config and not args.mb_samples:
        Bfull = wq.batch
        hof = np.zeros((Bfull, 2), np.float32)
        barrier()
        t0 = time.perf_counter()
        _, st_full = nqs.local_energy_host(H, M, samples, counts, minibatch=mb, path=path, want_stats=True, out=hof)
        full_s = max_over_ranks(time.perf_counter() - t0, dev)
        full_config = {"samples": Bfull, "minibatches": (Bfull + mb - 1) // mb, "seconds": full_s,
                       "value": Bfull * K * world / full_s, "unit": UNIT,
                       "mean_E": [st_full[1] / st_full[0], st_full[2] / st_full[0]],
                       "note": "one nqs_local_energy_host call over the whole configured batch; H2D, all mini-batches, "
                               "statistics and D2H inside the wall-clock region"}

    # ---- one whole iteration through the ABI: sampler -> E_loc -> gradient, each wall-clocked ----
    iteration = None
    if args.iteration:
        M.set_constraint(wq.n_alpha, wq.n_beta)
        n_draws = 1 << 20
        barrier()
        t0 = time.perf_counter()
        s_dev, c_dev = nqs.made_sample(M, n_draws, 2024, max_unique=mb, device=dev)
        torch.cuda.synchronize()
        t_sample = time.perf_counter() - t0
        t0 = time.perf_counter()
        e_it, st_it = nqs.local_energy(H, M, s_dev, c_dev, minibatch=mb, path=path)
        torch.cuda.synchronize()
        t_eloc = time.perf_counter() - t0
        t0 = time.perf_counter()
        g_it, b_it = nqs.energy_grad(M, s_dev, c_dev, e_it, minibatch=mb)
        torch.cuda.synchronize()
        t_grad = time.perf_counter() - t0
        M.set_constraint(-1, -1)
        iteration = {"n_draws": n_draws, "unique_samples": int(s_dev.shape[0]), "constraint": [wq.n_alpha, wq.n_beta],
                     "sample_s": t_sample, "eloc_s": t_eloc, "grad_s": t_grad,
                     "sample_over_eloc": t_sample / t_eloc, "grad_over_eloc": t_grad / t_eloc,
                     "mean_E": [st_it[1] / st_it[0], st_it[2] / st_it[0]], "grad_finite": bool(torch.isfinite(g_it).all().item()),
                     "note": "nqs_made_sample (first call: includes its per-call buffer allocation) -> nqs_local_energy -> "
                             "nqs_energy_grad on the sampler's output, constrained model, wall clock with a synchronise after each"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the MADE-chain / fused E_loc kernel) ----
    peaks = load_peaks()
    used_tc = M.resolved_path(path) == nqs.PATH_TC
    flops_eval = algorithmic_flops_per_eval(params)
    evals_per_launch = mb * (G - 1)                       # rows the chain kernel evaluates (f = 0 group has ratio 1)
    k_ms = chain_ms / max(chain_launches, 1)
    achieved = flops_eval * evals_per_launch / (k_ms / 1e3) / 1e12
    if used_tc:
        roof = {"bound": "tensor", "achieved": achieved, "peak": peaks["tensor_tflops"], "unit": "TFLOP/s",
                "frac": achieved / peaks["tensor_tflops"], "traffic": None,
                "peak_source": f"{peaks['src']} bf16 dense, sustained (fp16 operands run at the bf16 rate)"}
    else:
        clk = (clocks["sm_mhz"] or peaks["sm_max_mhz"]) * 1e6
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        alu_peak = sms * 128 * 2 * clk / 1e12             # FFMA lanes x 2 flop x measured clock
        roof = {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "frac": achieved / alu_peak,
                "traffic": None, "peak_source": f"{sms} SM x 128 FFMA lanes x 2 flop x median SM clock under load"}
    roof.update({"kernel": "eloc_tc_kernel" if used_tc else "eloc_simt_kernel", "kernel_ms_per_launch": k_ms,
                 "algorithmic_flops_per_eval": flops_eval, "evals_per_launch": evals_per_launch,
                 "kernel_share_of_step": chain_ms / total_ms})

    roof["traffic"] = ncu_constant("eloc_tc_dram_bytes", (args.cfg, mb)) if used_tc else None
    roof["traffic_source"] = ("ncu dram__bytes_read.sum + dram__bytes_write.sum of one launch of this kernel source "
                              "(profiles/r3_ncu_counters.md)") if roof["traffic"] else "no ncu capture of the current kernel source"
    if used_tc:
        issued, dense = M.tc_flops()
        roof["issued_flops_per_eval"] = issued                # what the kernel sends to the tensor cores (overhead included)
        roof["issued_over_algorithmic"] = issued / flops_eval
        roof["frac_issued"] = roof["frac"] * issued / flops_eval     # context only: MMA flops the kernel issues / the same peak

    contraction = None
    if not args.no_contraction:
        contraction = time_contraction(nqs, torch, H, xs_all[:mb], stream, clocks["sm_mhz"] or peaks["sm_max_mhz"])

    cpu_baseline = cpu_baseline_1 = None
    if not args.no_cpu_baseline:
        v, dt, threads = time_oracle(wq, ham, params, samples, n_oracle)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": dt,
                        "sample": f"{n_oracle} of {mb} samples of one mini-batch x all {K} terms (memoised oracle mode)"}
        v1, dt1, _ = time_oracle(wq, ham, params, samples[n_oracle:], 1, one_thread=True)
        cpu_baseline_1 = {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt1,
                          "sample": f"1 of {mb} samples x all {K} terms, BLAS pool limited to one thread"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16 operands / f32 accumulate" if used_tc else "f32", "data": "synthetic",
            "config": {"workload": workload_name, "n_qubits": wq.n_qubits, "n_terms": K, "n_groups": G,
                       "minibatch": mb, "hidden": wq.hidden, "path": "tc" if used_tc else "simt",
                       "l2": "flushed between timed steps (256 MiB write)", "parallelism": f"dp{world} over mini-batches"},
            "psi_evals_per_s": evals_per_s, "roofline": roof, "contraction": contraction,
            "cpu_baseline": cpu_baseline, "cpu_baseline_1thread": cpu_baseline_1,
            "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": mb * 16 + mb * 8,
                    "d2h_bytes_per_step": mb * 8 + 5 * 8},
            "full_config": full_config, "iteration": iteration,
            "gpu_launches": int(launches), "clocks": clocks,
            "job_stats": {"sum_n": job_stats[0].item(), "mean_E": [(job_stats[1] / job_stats[0]).item(), (job_stats[2] / job_stats[0]).item()],
                          "note": "count-weighted mean of E_loc over every mini-batch of every rank in the timed steps "
                                  "(all_reduce_stats: 4 sums + 1 max over ranks)"}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
