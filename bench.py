#!/usr/bin/env python3
"""bench.py -- J/K build benchmark (BASELINE.json metric: J/K build ms, screened ERI quartets/s, fraction of
FP64 peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]

A step = one adft_jk_build (max|D|, screening plan, all class ERI kernels with in-kernel digestion, finalise) of the
synthetic workload with D, the basis and the shell-pair table already resident in HBM.  `value` = kept unique shell
quartets per second over the whole job; `e2e` = the same through adft_jk_build_host (pinned host D in, host J, K out,
copies inside the timed region).  The path does not shard (north_star: one GPU, no collectives): under torchrun every
rank runs an independent replica ("replicas only") and `value` adds the replicas up.

--impl reference times the oracle (oracle/, plain C on the host cores) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PAIR_CLASSES = [(la, lb) for la in range(5) for lb in range(la + 1)]       # up to g: 15 pair classes, 120 quartet classes
CLASS_NAMES = []
for X, (la, lb) in enumerate(PAIR_CLASSES):
    for Y, (lc, ld) in enumerate(PAIR_CLASSES[:X + 1]):
        CLASS_NAMES.append("(%s%s|%s%s)" % ("spdfg"[la], "spdfg"[lb], "spdfg"[lc], "spdfg"[ld]))

# classes that run through the block-cooperative Rys kernels (csrc/adft_rys.cu); all others are generated straight-line code
RYS_CLASSES = {"(fp|fp)", "(ff|pp)", "(fd|dp)", "(ff|fs)", "(fp|dd)", "(fd|fp)", "(ff|dp)", "(fd|dd)", "(ff|fp)", "(fd|fd)",
               "(ff|dd)", "(ff|fd)", "(ff|ff)"}
WORKLOAD_NAMES = {0: "cfg0_3atom_13bf", 1: "cfg1_10atom_chain_100bf", 2: "cfg2_60atom_cluster_500bf",
                  3: "cfg3_60atom_cluster_f_940bf", 4: "cfg4_300atom_globular_2500bf"}
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # 148 SMs x 64 DFMA/clk x 2 flops x 1.965 GHz = 37.2
# dram__bytes_read.sum + dram__bytes_write.sum per launch of a class kernel, from the `ncu --set full` captures whose
# summaries are committed under profiles/ (a profiler number, quoted, never measured inside a timed run):
# {workload: {class: (bytes, source)}}.  A dominant kernel without a capture reports "traffic": null.
NCU_DRAM_BYTES = {
    "cfg4_300atom_globular_2500bf": {
        "(dp|pp)": (166.8e9, "profiles/r02_ncu_full_cfg4.md"),
        "(ps|ss)": (4.0e9, "profiles/r02_ncu_full_cfg4.md"),
    },
}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def reduce_max_over_ranks(values, world, device="cpu"):
    """Timing of a multi-rank run = the slowest rank: element-wise MAX of `values` over all ranks (all-reduce on the
    initialised process group: NCCL with a CUDA `device` in the benchmark, gloo on the CPU in tests/)."""
    if world == 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def job_value(kept_per_replica, world, ms_per_step):
    """Whole-job throughput of `world` independent replicas ("replicas only"): every rank builds
    J and K of the same workload, so the job processes world * kept quartets in the time of the slowest rank."""
    return world * kept_per_replica / (ms_per_step * 1e-3)


def oracle_sample(w, seconds_target, seed=7):
    """Time the oracle, as it stands, on a bounded sample of the workload: J and K shell blocks evaluated from the
    definition with the same screen (oracle.jk_block) for random shell pairs until ~seconds_target of wall time."""
    import oracle
    bs = oracle.basis_from_workload(w)
    t0 = time.perf_counter()
    Q = oracle.schwarz(bs)
    t_q = time.perf_counter() - t0
    dm = oracle.dmax(w.D)
    rng = np.random.default_rng(seed)
    nq = npq = nblk = 0
    blocks = []
    t0 = time.perf_counter()
    while True:
        A, B = (int(x) for x in rng.integers(0, bs.nshells, size=2))
        Jb, Kb, (q, p) = oracle.jk_block(bs, w.D, w.tau, Q, dm, A, B, with_work=True)
        blocks.append((A, B, Jb, Kb))
        nq += q; npq += p; nblk += 1
        el = time.perf_counter() - t0
        if el >= seconds_target or nblk >= 4000:
            break
    return {"quartets": nq, "prim_quartets": npq, "seconds": el, "blocks": nblk, "schwarz_seconds": t_q,
            "threads": oracle.num_threads(), "block_values": blocks, "bf_off": bs.bf_off}


def sample_max_abs_err(smp, J, K):
    """Largest |J_gpu - J_oracle|, |K_gpu - K_oracle| over the oracle's sampled shell blocks (host arrays J, K)."""
    o = smp["bf_off"]
    worst = 0.0
    for (A, B, Jb, Kb) in smp["block_values"]:
        worst = max(worst, float(np.abs(J[o[A]:o[A + 1], o[B]:o[B + 1]] - Jb).max()),
                    float(np.abs(K[o[A]:o[A + 1], o[B]:o[B + 1]] - Kb).max()))
    return worst


def run_reference(args, rank, world):
    from paper_2406_11185_b200 import workloads
    if rank != 0:
        return
    w = workloads.make(args.config)
    per_step = max(2.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(w, min(per_step, 2.0))
    tot_q = tot_t = 0.0
    last = None
    for s in range(args.steps):
        last = oracle_sample(w, per_step, seed=100 + s)
        tot_q += last["quartets"]; tot_t += last["seconds"]
    val = tot_q / tot_t
    sample = (f"{last['blocks']} random J+K shell blocks per step from the definition with the same screen "
              f"(oracle.jk_block, long-double core), {per_step:.0f} s per step")
    out = {"impl": "reference", "metric": "screened_eri_quartets_per_s", "value": val, "unit": "quartets/s",
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": WORKLOAD_NAMES[args.config], "nbf": w.nbf, "nshells": w.nshells, "tau": w.tau},
           "cpu_baseline": {"value": val, "unit": "quartets/s", "cores": last["threads"], "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "quartets/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index (default 4 = largest)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="wall seconds of oracle work for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-mixed", action="store_true", help="skip the mixed-precision (f64+f32) measurement reported beside the f64 line")
    ap.add_argument("--prim-threshold", type=float, default=None,
                    help="primitive-pair threshold (default: the library's ADFT_DEFAULT_PRIM_THRESHOLD; 0 = no primitive screening)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2406_11185_b200 import api, workloads
    api.lib()                                 # fail loudly if the extension is missing
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = workloads.make(args.config)
    N = w.nbf
    t0 = time.perf_counter()
    bs = api.Basis.from_workload(w)
    sp = api.ShellPairs(bs, prim_threshold=args.prim_threshold)
    torch.cuda.synchronize()
    t_pairs = time.perf_counter() - t0
    npairs, nprimpairs = sp.counts()
    nprim_nominal, _, prim_thr = sp.prim_counts()
    D = torch.from_numpy(w.D).cuda()
    J = torch.empty_like(D); K = torch.empty_like(D)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream()

    for _ in range(args.warmup):
        sp.jk_build(D, J, K, w.tau)
        torch.cuda.synchronize()
    peak = api.fp64_peak_tflops()

    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    step_ms, class_ms, stats = [], np.zeros(len(CLASS_NAMES)), None
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        flush.zero_()                                   # L2 flush between timed iterations (inputs also exceed L2)
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(stream)
        sp.jk_build(D, J, K, w.tau, stream=stream)
        b.record(stream)
        b.synchronize()
        step_ms.append(a.elapsed_time(b))
        stats = sp.stats()
        class_ms += np.array(stats.class_ms[:])
    e1.record(stream)
    barrier()
    region_ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    ms_step = float(np.mean(step_ms))
    ms_step, region_ms = reduce_max_over_ranks([ms_step, region_ms], world, "cuda")
    kept = int(stats.quartets_kept)
    value = job_value(kept, world, ms_step)

    # end to end: host buffers through adft_jk_build_host (H2D of D, D2H of J and K inside the timed region)
    Dh = torch.from_numpy(w.D).pin_memory(); Jh = torch.empty(N, N, dtype=torch.float64).pin_memory()
    Kh = torch.empty(N, N, dtype=torch.float64).pin_memory()
    e2e_steps = max(1, min(args.steps, 2))
    sp.jk_build_host(Dh.numpy(), Jh.numpy(), Kh.numpy(), w.tau)      # untimed: allocates the library's staging buffers
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sp.jk_build_host(Dh.numpy(), Jh.numpy(), Kh.numpy(), w.tau)
        chk = float(Jh[0, 0])                         # host read of the result
    e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps
    e2e_ms = reduce_max_over_ranks([e2e_ms], world, "cuda")[0]
    e2e_value = job_value(kept, world, e2e_ms)
    assert np.isfinite(chk)

    # beside the f64 headline (never instead of it): the paper's mixed-precision dispatch,
    # quartets with tau <= S < 1e5 tau in single precision.  Same workload, same kept set; timed the same way, and its
    # J, K compared with the f64 J, K of the timed builds above.
    mixed = None
    if not args.no_mixed:
        Jm = torch.empty_like(D); Km = torch.empty_like(D)
        sp.jk_build(D, Jm, Km, w.tau, mixed_precision=True); torch.cuda.synchronize()        # warm-up (module load)
        mx_ms = []
        for _ in range(max(1, min(args.steps, 3))):
            flush.zero_()
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record(stream)
            sp.jk_build(D, Jm, Km, w.tau, stream=stream, mixed_precision=True)
            b.record(stream); b.synchronize()
            mx_ms.append(a.elapsed_time(b))
        sm = sp.stats()
        mms = reduce_max_over_ranks([float(np.mean(mx_ms))], world, "cuda")[0]
        Dl = D.to(torch.float64)
        mixed = {"dtype": "f64+f32", "fp32_band": 1e5, "ms_per_step": mms, "value": job_value(int(sm.quartets_kept), world, mms),
                 "unit": "quartets/s", "speedup_vs_f64": ms_step / mms,
                 "quartets_kept": int(sm.quartets_kept), "quartets_fp32": int(sm.quartets_fp32),
                 "fp32_fraction": int(sm.quartets_fp32) / max(1, int(sm.quartets_kept)),
                 "max_abs_dJ_vs_f64": float((Jm - J).abs().max()), "max_abs_dK_vs_f64": float((Km - K).abs().max()),
                 "dE_J_vs_f64": float(0.5 * (Dl * (Jm - J)).sum()), "dE_K_vs_f64": float(-0.25 * (Dl * (Km - K)).sum()),
                 "E_J": float(0.5 * (Dl * J).sum()), "E_K": float(-0.25 * (Dl * K).sum())}
        sp.jk_build(D, J, K, w.tau); torch.cuda.synchronize()       # leave the stats of an f64 build behind
        stats_after = sp.stats()
        assert int(stats_after.quartets_kept) == kept == mixed["quartets_kept"]

    if rank == 0:
        class_ms /= args.steps
        cq = np.array(stats.class_quartets[:])
        dom = int(np.argmax(class_ms))
        cmf = np.array(stats.class_model_flops[:])
        step_tflops = stats.model_flops / (ms_step * 1e-3) / 1e12
        dom_tflops = cmf[dom] / (class_ms[dom] * 1e-3) / 1e12
        # roofline of the dominant kernel launch: algorithmic (model) FP64 flops of that class launch / its duration
        # measured live with CUDA events on the launching stream (adft_jk_stats.class_ms).  Bound: plain FP64 ALUs.
        roofline = {"bound": "alu", "kernel": f"{'jk_rys_kernel' if (CLASS_NAMES[dom] in RYS_CLASSES or 'g' in CLASS_NAMES[dom]) else 'jk_kernel'}<{CLASS_NAMES[dom]}>", "kernel_ms": float(class_ms[dom]),
                    "kernel_share_of_step": float(class_ms[dom] / ms_step), "kernel_model_flops": float(cmf[dom]),
                    "achieved": dom_tflops, "peak": peak, "unit": "TFLOP/s", "frac": dom_tflops / peak,
                    "whole_step_achieved": step_tflops, "whole_step_frac": step_tflops / peak,
                    "peak_source": "measured on this GPU by adft_fp64_peak_tflops (register-resident DFMA chains, "
                                   f"burst); nominal {NOMINAL_FP64_TFLOPS:.1f} TFLOP/s = 148 SMs x 64 DFMA/clk x 2 x 1.965 GHz; "
                                   "MEASURED_PEAKS.json has no FP64 entry",
                    "traffic": None}
        cap = NCU_DRAM_BYTES.get(WORKLOAD_NAMES[args.config], {}).get(CLASS_NAMES[dom])
        if cap:
            roofline["traffic"] = cap[0]
            roofline["traffic_source"] = f"dram read+write bytes of one launch of this kernel, ncu --set full, {cap[1]}"
        out = {"metric": "screened_eri_quartets_per_s", "value": value, "unit": "quartets/s", "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
               "config": {"workload": WORKLOAD_NAMES[args.config], "nbf": N, "nshells": w.nshells, "natoms": w.natoms,
                          "tau": w.tau, "shell_pairs": npairs, "primitive_pairs": nprimpairs,
                          "quartets_unique": int(stats.quartets_unique), "quartets_kept": kept,
                          "primitive_pairs_nominal": nprim_nominal, "prim_threshold": prim_thr,
                          "prim_quartets": int(stats.prim_quartets),
                          "prim_quartets_evaluated": int(stats.prim_quartets_evaluated), "parallelism": "replicas" if world > 1 else "1gpu",
                          "l2": "flushed between iterations (256 MiB write); pair table + D/J/K exceed L2",
                          "shellpairs_build_s": t_pairs},
               "jk_build_ms": ms_step, "jk_build_ms_min": float(np.min(step_ms)), "jk_build_ms_median": float(np.median(step_ms)),
               "region_ms": region_ms,
               "prim_quartets_per_s": world * int(stats.prim_quartets) / (ms_step * 1e-3),
               "prim_quartets_evaluated_per_s": world * int(stats.prim_quartets_evaluated) / (ms_step * 1e-3),
               "model_tflops": step_tflops, "fp64_peak_fraction": step_tflops / peak,
               "phase_ms": {"dmax": stats.ms_dmax, "plan": stats.ms_plan, "eri": stats.ms_eri, "finalize": stats.ms_finalize},
               # the two HBM-bound phases against the measured copy bandwidth (MEASURED_PEAKS.json: 6496 GB/s on this pool):
               # finalise reads and writes J and K once (4 N^2 doubles); Dmax includes the 16-byte D2H and the host sync
               "phase_gbps": {"finalize": 4.0 * N * N * 8 / (stats.ms_finalize * 1e-3) / 1e9 if stats.ms_finalize > 0 else None,
                              "dmax": N * N * 8 / (stats.ms_dmax * 1e-3) / 1e9 if stats.ms_dmax > 0 else None},
               "class_ms": {CLASS_NAMES[i]: round(float(class_ms[i]), 3) for i in range(len(CLASS_NAMES)) if cq[i]},
               "class_model_tflops": {CLASS_NAMES[i]: round(float(cmf[i] / (class_ms[i] * 1e-3) / 1e12), 2)
                                      for i in range(len(CLASS_NAMES)) if cq[i] and class_ms[i] > 0},
               "roofline": roofline,
               "e2e": {"value": e2e_value, "unit": "quartets/s", "ms_per_step": e2e_ms,
                       "h2d_bytes_per_step": int(N) * N * 8, "d2h_bytes_per_step": 2 * int(N) * N * 8},
               "gpu_launches": int(stats.kernel_launches) * args.steps, "clocks": clocks}
        if mixed is not None:
            out["mixed_precision"] = mixed
        if not args.no_cpu_baseline:
            smp = oracle_sample(w, args.cpu_seconds)
            err = sample_max_abs_err(smp, J.cpu().numpy(), K.cpu().numpy())      # the J, K of the timed builds
            out["cpu_baseline"] = {"value": smp["quartets"] / smp["seconds"], "unit": "quartets/s", "cores": smp["threads"],
                                   "kind": "oracle", "max_abs_err": err,
                                   "sample": f"{smp['blocks']} random J+K shell blocks of the same workload evaluated from "
                                             f"the definition with the same screen (oracle.jk_block), {smp['seconds']:.1f} s, "
                                             f"{smp['quartets']} shell quartets / {smp['prim_quartets']} primitive quartets",
                                   "prim_quartets_per_s": smp["prim_quartets"] / smp["seconds"]}
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
