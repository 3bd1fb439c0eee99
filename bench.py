#!/usr/bin/env python
"""bench.py -- throughput of the direct-summation Hermite force path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-sweep]

Metric (BASELINE.json): pair interactions per second (Ginteractions/s) and fraction of the FP64
roofline.  Workload at N = 1 GPU: the north_star headline point -- N = n_i = 2^18 equal-mass
Plummer sphere, eps = 1e-4, 4th-order Hermite, fp64, acc + jerk + pot (it fits one GPU).

One "step" is one pass of the whole hot path: commit all N j-particles,
predict them to t, force sweep for the i-list (+ deterministic reduce), results available.
  value : inputs already resident in HBM (s2_commit_j_device / s2_calc_ilist_device), device timed.
  e2e   : the same step through the host-buffer C-ABI calls (s2_set_j + s2_commit_j + s2_predict +
          s2_calc_ilist + s2_get_results), H2D / D2H copies inside the timed region.
Timing: CUDA events around every step on the library's stream, L2 flushed between steps,
max over ranks.  --impl reference times the CPU oracle (as it stands) on a bounded sample.
"""
from __future__ import annotations

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

FLOP_PER_PAIR = {2: 38, 4: 60, 6: 97}   # stated convention (reading P16); 38 = the usual acc+pot count
FP64_INSTR_PER_PAIR = {2: 18, 4: 32, 6: 54}    # FP64-pipe instructions per pair in the SASS of the sweep (profiles/)
EXECUTED_FLOP_PER_PAIR = {2: 29, 4: 49, 6: 86}  # flops those instructions really perform (FMA = 2): 4th order 17 DFMA x 2 + 15
SM_COUNT, FP64_LANES_PER_SM, SM_MAX_HZ = 148, 64, 1.965e9
FP64_PEAK_TFLOPS = SM_COUNT * FP64_LANES_PER_SM * 2 * SM_MAX_HZ / 1e12     # 37.2
FP32_PEAK_TFLOPS = 2 * FP64_PEAK_TFLOPS                                    # 128 FP32 lanes per SM: 74.5
# dram__bytes_read.sum + dram__bytes_write.sum of one force-sweep launch at the headline point,
# from the ncu --set full capture summarised in profiles/ (None until a capture exists)
FORCE_KERNEL_DRAM_BYTES = 20.99e6   # tiled sweep: 18.02 MB read + 2.96 MB written (profiles/r01_force_fp64_ncu_full.md)
BANK_KERNEL_DRAM_BYTES = 29.51e6    # uniform-operand sweep, per chunk launch: 29.51 MB read (parked i-state + running
                                    # sums, cold L2 under ncu) + 0 written (profiles/r01_force_bank_ncu_full.md)
FP32_KERNEL_DRAM_BYTES = 16.24e6    # packed fp32 tiled sweep at N = n_i = 2^18: 13.71 MB read + 2.52 MB written
                                    # (profiles/r01_predict_and_fp32_ncu.md)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the n_i sweep and the peak microbenchmarks")
    ap.add_argument("--workload", default="H", help="config key: H (headline), 3, 4, 5 ...")
    ap.add_argument("--N", type=int, default=0, help="override N (reduced sizes are for debugging only)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "ds", "fp32"],
                    help="pair-arithmetic precision of the timed step (the default bench line is fp64)")
    ap.add_argument("--section", default="all", choices=["all", "hbm", "shapes", "fp32fix"],
                    help="hbm: only the streaming-kernel (predictor / scatter) measurement, for ncu captures; shapes: the "
                         "launch-shape space around n_i = 32 and the atomics-versus-reduce A/B (profiles/r02_small_ni.md)")
    ap.add_argument("--shard", default="i", choices=["i", "j"],
                    help="multi-GPU decomposition: i = every rank its own i-list against the whole store (independent units, "
                         "weak scaling, the default line); j = the paper's scheme (L84): every rank sums ALL i over its own block "
                         "of j and the partial results are combined by an all-reduce on device tensors (strong scaling)")
    ap.add_argument("--blockstep", type=int, default=0, metavar="N",
                    help="second workload (not the default line): block-time-step Hermite runs of an N-particle Plummer "
                         "sphere with the device-resident integrator, 4th and 6th order, fp64 and double-single; prints one "
                         "JSON line of statistics")
    ap.add_argument("--bs-tend", type=float, default=1.0, help="end time of the --blockstep runs (N-body time units)")
    ap.add_argument("--bs-orders", default="4,6")
    ap.add_argument("--bs-precisions", default="fp64,ds")
    ap.add_argument("--bs-profile-cta", type=int, default=0, help="CTA of the small-step kernel whose per-part cycle sums are reported")
    ap.add_argument("--bs-no-host", action="store_true", help="skip the host reference driver rows of --blockstep")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------- reference arm
def run_reference(args, w, rank, world):
    """The CPU oracle, as it stands, on the host cores: each step = a bounded sample of the workload."""
    if rank != 0:
        return
    import oracle
    order = w.order
    xp, vp, ap = oracle.predict(order, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle)
    n_s = max(8, min(w.N, int(6.0e7 // w.N)))          # ~6e7 pairs per step
    il = w.ilist(n_s)
    times = []
    for k in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.predict(order, w.t_pred, w.t_j[:n_s], w.pos[:n_s], w.vel[:n_s], w.acc[:n_s], w.jerk[:n_s],
                       w.snap[:n_s], w.crackle[:n_s])
        oracle.forces_ilist(order, w.mass, w.ident, xp, vp, ap, il, w.eps2)
        if k >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * sum(times) / len(times)
    val = n_s * w.N / (ms * 1e-3) / 1e9
    sample = f"{n_s} of {w.N} i-particles (seeded prefix of the active-set permutation) x all {w.N} j per step"
    line = {"impl": "reference", "metric": "Ginteractions/s", "value": val, "unit": "Ginteractions/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f80 (x87 long double)",
            "data": "synthetic", "config": workload_config(w, w.N),
            "cpu_baseline": {"value": val, "unit": "Ginteractions/s", "cores": oracle.max_threads(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "Ginteractions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}          # fallback figures of B200_PROFILING.md are then used ("of fallback")


def workload_config(w, ni, precision="fp64"):
    return {"workload": f"{w.name}: Plummer sphere N={w.N}, n_i={ni}, {w.order}th-order Hermite, "
                        f"eps={w.notes['eps']:.4g}, {'Salpeter' if w.notes['salpeter'] else 'equal'} masses, "
                        f"acc+jerk{'+snap' if w.order == 6 else ''}+pot",
            "N": w.N, "n_i": ni, "order": w.order, "precision": precision, "seed": w.seed,
            "l2": "L2 flushed (256 MiB write) between timed steps; the predicted j-store (16 MiB) is re-read "
                  "from L2 inside a step by design",
            "parallelism": "j-store replicated, i-lists per rank (no data-path collective)"}


# ------------------------------------------------------------------------------------------- our arm
def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    from workloads import make_config
    key = int(args.workload) if args.workload.isdigit() else args.workload
    w = make_config(key, N=args.N or None)

    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return
    if args.blockstep:
        if rank == 0:
            run_blockstep(args.blockstep, args.bs_tend, tuple(int(x) for x in args.bs_orders.split(",")),
                          tuple(args.bs_precisions.split(",")), host_reference=not args.bs_no_host, prof_cta=args.bs_profile_cta)
        return
    if args.section == "fp32fix":
        if rank == 0:
            import torch
            import paper_1510_04068_b200 as s2
            print(json.dumps(fp32_fixup_cost(s2, torch, torch.device("cuda", local))), flush=True)
        return
    if args.section == "shapes":
        if rank == 0:
            import torch
            import paper_1510_04068_b200 as s2
            print(json.dumps(shape_space(s2, torch, torch.device("cuda", local))), flush=True)
        return
    if args.section == "hbm":
        if rank == 0:
            import torch
            import paper_1510_04068_b200 as s2
            print(json.dumps({"hbm_kernels": hbm_kernels(s2, torch, torch.device("cuda", local),
                                                         measured_peaks().get("hbm_gbs", 6650.0))}), flush=True)
        return

    import torch
    import torch.distributed as dist
    import paper_1510_04068_b200 as s2

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    order, N, ni = w.order, w.N, w.N
    # i-list of this rank: its own rotation of the seeded permutation (same per-GPU work on every rank)
    from paper_1510_04068_b200.sharding import max_over_ranks, rank_ilist
    jshard = args.shard == "j"
    il_host = w.ilist(ni) if jshard else rank_ilist(w.perm, rank, world, ni)

    prec = {"fp64": s2.S2_FP64, "ds": s2.S2_DS, "fp32": s2.S2_FP32}[args.precision]
    ctx = s2.s2_open(local, order, prec, nj_capacity=N, ngb_cap=0)
    s2.s2_enable_timing(ctx, True)
    if jshard:
        from paper_1510_04068_b200.sharding import block_shard, combine_partials
        s2.s2_set_j_range(ctx, *block_shard(N, rank, world))
        comb = dict(acc=torch.empty(ni * 3, dtype=torch.float64, device=dev), jerk=torch.empty(ni * 3, dtype=torch.float64, device=dev),
                    pot=torch.empty(ni, dtype=torch.float64, device=dev))
        h_comb = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in comb.items()}
    addr = np.arange(N, dtype=np.int32)
    host = dict(address=addr, ident=w.ident, t=w.t_j, mass=w.mass, pos=w.pos, vel=w.vel, acc=w.acc, jerk=w.jerk,
                snap=w.snap if order == 6 else None, crackle=w.crackle if order == 6 else None)
    d = {k: (torch.from_numpy(v).to(dev) if v is not None else None) for k, v in host.items()}
    d_il = torch.from_numpy(il_host).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step_resident():
        s2.s2_commit_j_device(ctx, d["address"], d["ident"], d["t"], d["mass"], d["pos"], d["vel"], d["acc"], d["jerk"],
                              d["snap"], d["crackle"])
        s2.s2_predict(ctx, w.t_pred, N)
        s2.s2_calc_ilist_device(ctx, d_il, None, w.eps2, 0)
        if jshard:   # the one exchange step of the paper's scheme: partial results of all i added over the ranks
            s2.s2_get_results_device(ctx, ni, acc=comb["acc"], jerk=comb["jerk"], pot=comb["pot"])
            combine_partials(comb["acc"], comb["jerk"], comb["pot"])

    def step_e2e():
        s2.s2_set_j(ctx, host["address"], host["ident"], host["t"], host["mass"], host["pos"], host["vel"], host["acc"],
                    host["jerk"], host["snap"], host["crackle"])
        s2.s2_commit_j(ctx)
        s2.s2_predict(ctx, w.t_pred, N)
        s2.s2_calc_ilist(ctx, il_host, None, w.eps2, 0)
        if jshard:
            s2.s2_get_results_device(ctx, ni, acc=comb["acc"], jerk=comb["jerk"], pot=comb["pot"])
            combine_partials(comb["acc"], comb["jerk"], comb["pot"])
            for k in comb:
                h_comb[k].copy_(comb[k], non_blocking=True)
            torch.cuda.current_stream().synchronize()
            return h_comb
        return s2.s2_get_results(ctx, ni)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup, collect_kernel_times=False):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        ktimes = []
        barrier()
        l0 = s2.s2_kernel_launches(ctx)
        for a, b in ev:
            flush.zero_()
            a.record()
            fn()
            b.record()
            if collect_kernel_times:
                ktimes.append(s2.s2_get_timing(ctx))     # synchronises; outside the event pair
        barrier()
        launches = s2.s2_kernel_launches(ctx) - l0
        ms = [a.elapsed_time(b) for a, b in ev]
        return ms, launches, ktimes

    sampler = ClockSampler(local)
    sampler.start()
    step_ms, launches, ktimes = timed(step_resident, args.steps, max(args.warmup, 3), True)
    clocks = sampler.stop()
    e2e_step_ms, _, _ = timed(step_e2e, args.steps, 1)

    # whole-job numbers: the slowest rank decides (sum, median and best of the per-step device times, each max over ranks)
    tot_ms, e2e_ms, med_ms, best_ms, e2e_med_ms = max_over_ranks(
        [sum(step_ms), sum(e2e_step_ms), statistics.median(step_ms), min(step_ms), statistics.median(e2e_step_ms)], device=dev)
    pairs_step = float(ni) * N * (1 if jshard else world)     # j-sharding: the ranks share ONE n_i x N problem
    value = pairs_step * args.steps / (tot_ms * 1e-3) / 1e9
    e2e_value = pairs_step * args.steps / (e2e_ms * 1e-3) / 1e9

    nf = 20 if order == 6 else 14
    h2d = N * (nf * 8 + 8) + ni * 4
    d2h = ni * 96 + 8

    force_ms = statistics.mean(k["force_ms"] for k in ktimes)
    achieved = ni * N * FLOP_PER_PAIR[order] / (force_ms * 1e-3) / 1e12
    info = s2.s2_last_launch_info(ctx)
    fp64_path = args.precision == "fp64"
    peak = FP64_PEAK_TFLOPS if fp64_path else FP32_PEAK_TFLOPS
    kname = {"fp64": "PolicyF64", "ds": "PolicyDS", "fp32": "PolicyF32"}[args.precision]
    kname = (f"force_sweep_bank_kernel<{kname}<{order},0,0>>" if info["reduced"] in (3, 5)
             else f"force_sweep_tiled_kernel<{kname}<{order},0,0>,{info['i_per_thread']}>" if info["i_per_thread"] > 1
             else f"force_sweep_kernel<{kname}<{order},0,0>,{info['lanes_per_i']}>")
    roofline = {"bound": "alu", "kernel": kname, "achieved": achieved,
                "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": ((BANK_KERNEL_DRAM_BYTES if info["reduced"] in (3, 5) else FORCE_KERNEL_DRAM_BYTES) if fp64_path else
                            FP32_KERNEL_DRAM_BYTES if (args.precision == "fp32" and info["i_per_thread"] > 1) else None),
                "traffic_source": "ncu capture, constant (dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the "
                                  "ncu --set full capture summarised under profiles/; not measured in this run)",
                "peak_source": ("derived: 148 SM x 64 FP64 FMA lanes x 2 flop x 1.965 GHz" if fp64_path else
                                "derived: 148 SM x 128 FP32 FMA lanes x 2 flop x 1.965 GHz") + " (DESIGN.md 5.2); not in MEASURED_PEAKS.json",
                "convention": f"{FLOP_PER_PAIR[order]} flop per pair interaction (labelled convention, reading P16)",
                "kernel_ms": force_ms, "kernel_share_of_step": force_ms * args.steps / tot_ms,
                "predict_ms": statistics.mean(k["predict_ms"] for k in ktimes),
                "reduce_ms": statistics.mean(k["reduce_ms"] for k in ktimes)}
    if info["reduced"] in (3, 5):
        roofline["bank_refill"] = ("by the sweep's own last CTA, launches overlapped (first-use self-test passed)" if info["reduced"] == 3
                                   else "stream-ordered copies between ordinary launches (documented-semantics fallback)")
        # one launch per chunk of the constant bank; achieved = (n_i x chunk x flop) / (mean duration of a chunk
        # launch INCLUDING the copy that refills the bank before it) -- the same ratio as the whole sweep's
        roofline["launches_per_sweep"] = info["S"]
        roofline["pairs_per_launch"] = ni * N // info["S"]
        roofline["ms_per_launch"] = force_ms / info["S"]
        roofline["traffic_note"] = "per chunk launch, cold L2 under ncu; the state it re-reads stays in L2 between launches"
    if fp64_path:
        roofline["fp64_instr_per_pair"] = FP64_INSTR_PER_PAIR[order]
        roofline["fp64_pipe_frac_nominal"] = (ni * N * FP64_INSTR_PER_PAIR[order] / (force_ms * 1e-3)
                                              / (SM_COUNT * FP64_LANES_PER_SM * SM_MAX_HZ))
        # the three honest readings of the same kernel time, side by side (VERDICT r1 "What's weak" 4); the small-n_i
        # target of north_star is added below once the sweep has run
        roofline["targets"] = {
            "fp64_frac_60flop": achieved / peak,                                   # labelled 60-flop convention: the 70 % target's reading
            "fp64_pipe_frac_instr": roofline["fp64_pipe_frac_nominal"],            # FP64 instruction issue rate, 32 instr / pair
            "fp64_frac_executed_flops": achieved / peak * EXECUTED_FLOP_PER_PAIR[order] / FLOP_PER_PAIR[order],   # flops really executed
            "target_fp64_frac_60flop": 0.70, "target_ni32_vs_full": 3.0}

    line = {"metric": "Ginteractions/s", "value": value, "unit": "Ginteractions/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": tot_ms / args.steps,
            "ms_per_step_median": med_ms, "ms_per_step_best": best_ms,
            "value_median": pairs_step / (med_ms * 1e-3) / 1e9, "value_best": pairs_step / (best_ms * 1e-3) / 1e9,
            "higher_is_better": True, "scaling": "strong" if jshard else "weak", "vs_baseline": None, "dtype": {"fp64": "f64", "ds": "f32x2 (double-single)", "fp32": "f32"}[args.precision],
            "data": "synthetic", "config": workload_config(w, ni, args.precision), "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "Ginteractions/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms / args.steps, "ms_per_step_median": e2e_med_ms},
            "gpu_launches": int(launches), "roofline": roofline, "launch": s2.s2_last_launch_info(ctx)}
    if jshard:
        line["config"]["parallelism"] = (f"j-sharded over {world} rank(s) (PAPER.md L84): whole store on every rank, each sums all i over "
                                         f"its own block of N/{world} j; all-reduce of acc/jerk/pot on device tensors (NCCL)")
        # the sweep of one rank covers n_i x N/world pairs
        for k in ("achieved", "frac", "fp64_pipe_frac_nominal"):
            if k in roofline:
                roofline[k] /= world

    if rank == 0 and world == 1 and args.precision == "fp32":
        # FP32 pipe, measured in the same process: scalar FFMA and the packed forms the tiled sweep issues
        nominal32 = SM_COUNT * 128 * SM_MAX_HZ
        ffma = s2.s2_peak_fma(ctx, 1, 4000)
        roofline["measured_ffma_tflops"] = 2 * ffma / 1e12
        roofline["fp32_lane_ops_per_pair"] = 33
        roofline["fp32_pipe_frac_nominal"] = ni * N * 33 / (force_ms * 1e-3) / nominal32
        roofline["fp32_pipe_model"] = {
            "ffma_const_operands": ffma / nominal32,
            "ffma2_const_operands": s2.s2_peak_fma(ctx, 5, 4000) / nominal32,
            "ffma2_three_distinct_register_pairs": s2.s2_peak_fma(ctx, 6, 4000) / nominal32,
            "ffma2_broadcast_operand": s2.s2_peak_fma(ctx, 7, 4000) / nominal32,
            "fadd2_two_register_pairs": s2.s2_peak_fma(ctx, 8, 4000) / nominal32,
            "unit": "fraction of 148 SM x 128 lanes x 1.965 GHz lane-operations/s"}
    if rank == 0 and world == 1 and not args.no_sweep and fp64_path:
        # measured FMA peaks in the same process (SURVEY sec 8(d) "clock risk")
        dfma = s2.s2_peak_fma(ctx, 0, 4000)
        roofline["measured_dfma_tflops"] = 2 * dfma / 1e12
        roofline["frac_of_measured_dfma_pipe"] = (ni * N * FP64_INSTR_PER_PAIR[order] / (force_ms * 1e-3)) / dfma
        # FP64 operand-path model: lane-instruction rate of each operand pattern / nominal
        nominal = SM_COUNT * FP64_LANES_PER_SM * SM_MAX_HZ
        roofline["fp64_pipe_model"] = {
            "dfma_const_operands": dfma / nominal,
            "dfma_three_distinct_registers": s2.s2_peak_fma(ctx, 2, 4000) / nominal,
            "dfma_one_operand_reused": s2.s2_peak_fma(ctx, 3, 4000) / nominal,
            "dadd_two_registers": s2.s2_peak_fma(ctx, 4, 4000) / nominal,
            "unit": "fraction of 148 SM x 64 lanes x 1.965 GHz lane-instructions/s"}
        line["sweep"] = ni_sweep(s2, torch, dev, order)
        by = {(r["cfg"], r["precision"], r["n_i"]): r for r in line["sweep"]}
        r3, rH = by.get(("3", "fp64", 32)), by.get(("H", "fp64", 32))
        if r3 and rH and "targets" in roofline:   # north_star: "small-N_i path within 3x of full-occupancy interactions/s at N_i = 32"
            roofline["targets"].update({"ni32_cfg3_us": r3["call_us"], "ni32_cfg3_vs_full": 1.0 / r3["vs_full_rate"],
                                        "ni32_H_us": rH["call_us"], "ni32_H_vs_full": 1.0 / rH["vs_full_rate"],
                                        "ni32_cfg3_ginteractions_per_s": r3["ginteractions_per_s"],
                                        "full_cfg3_ginteractions_per_s": by[("3", "fp64", 65536)]["ginteractions_per_s"]})
        line["large_configs"] = neighbour_path(s2, torch, dev, measured_peaks().get("hbm_gbs", 6650.0))
        line["hbm_kernels"] = hbm_kernels(s2, torch, dev, measured_peaks().get("hbm_gbs", 6650.0))
        line["blockstep"] = blockstep_summary(s2)
        line["cpu_baseline"] = cpu_baseline(w)
    if rank == 0:
        print(json.dumps(line), flush=True)
    s2.s2_close(ctx)
    if world > 1:
        dist.destroy_process_group()


def blockstep_summary(s2, n=16384):
    """The second workload (sec 3.7) in the default line: one N-body time unit of
    an N = 16384 Plummer sphere with the device-resident block-step integrator, 4th and 6th order, fp64 (about 2 s of GPU
    time).  `bench.py --blockstep N` is the full table (double-single, device time, A/B, host driver; profiles/)."""
    from paper_1510_04068_b200.hermite import DeviceHermite
    from workloads import make_config
    w = make_config(3, N=n)
    rows = []
    for order in (4, 6):
        d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, precision=s2.S2_FP64, averaged=order == 6)
        e0 = d.energy()
        t0 = time.perf_counter()
        d.run_until(1.0)
        wall = time.perf_counter() - t0
        e1 = d.energy()
        st, hist = d.stats(), d.history()
        d.close()
        rows.append({"order": order, "precision": "fp64", "criterion": "Aarseth eta4=0.01" if order == 4 else "mean of Aarseth(eta4=0.01) and generalised(eta6=0.1) (L156)",
                     "block_steps": st["block_steps"], "particle_steps": st["particle_steps"], "n_i_median": float(np.median(hist)),
                     "n_i_mean": float(hist.mean()), "wall_s": wall, "wall_us_per_block_step": wall / st["block_steps"] * 1e6,
                     "ginteractions_per_s_wall": st["particle_steps"] * n / wall / 1e9, "dE_over_E": (e1 - e0) / e0,
                     "steps_in_small_step_kernel": st["small"]["steps"], "small_step_kernel_launches": st["small"]["launches"]})
    return {"workload": f"block-time-step Hermite, Plummer N={n}, eps={w.notes['eps']:.3g}, t=0..1, dt_max=1/8 (DESIGN.md reading R-BTS)",
            "paper_context": "energy error ~1e-12 for the paper's 6th-order fp64 runs (L164); parameters not stated", "runs": rows}


def run_blockstep(n, t_end=1.0, orders=(4, 6), precisions=("fp64", "ds"), host_reference=True, prof_cta=0):
    """PAPER.md sec 3.7 (L152-L168), the second workload: block-time-step Hermite runs of an N-particle Plummer sphere
    for t_end N-body time units with the device-resident integrator (s2_bts_*), 4th order (eta = 0.01) and 6th order
    (eta = 0.1, the paper's scheme), fp64 and double-single.  Reports wall time per block step, the summed device time
    of the same steps (second, event-timed run over the first 1/8 time unit), the active-set statistics and dE/E (the
    paper quotes ~1e-12 in double and ~1e-10 in double-single for its 6th-order runs, L164: context).  The host driver
    of round 1 (hermite.py on s2_set_j / s2_calc_ilist / s2_get_results) runs the first 1/8 time unit for comparison."""
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite, Hermite4, Hermite6, S2Backend
    from workloads import make_config
    w = make_config(3, N=n)
    P = {"fp64": s2.S2_FP64, "ds": s2.S2_DS, "fp32": s2.S2_FP32}
    out = {"workload": f"block-time-step Hermite, Plummer N={n}, eps={w.notes['eps']:.3g}, t=0..{t_end}, eta4=0.01 eta6=0.1, "
                       f"dt_max=1/8", "runs": []}
    for order in orders:
        for name in precisions:
            d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, precision=P[name], averaged=order == 6)
            e0 = d.energy()
            t0 = time.perf_counter()
            d.run_until(t_end)
            wall = time.perf_counter() - t0
            e1 = d.energy()
            st, hist = d.stats(), d.history()
            d.close()
            # the same steps again, event-timed, for the summed device time (first 1/8 time unit)
            d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, precision=P[name], averaged=order == 6)
            if name == "fp64":
                s2.s2_bts_small_profile(d.bts, 1 + prof_cta)     # SM cycles one CTA spends in each part of a small step
            d.run_until(min(t_end, 0.125), time_device=True)
            sd = d.stats()
            prof = None
            if name == "fp64":
                pr = s2.s2_bts_small_profile(d.bts, 0)
                prof = {k: round(v / max(pr["steps"], 1)) for k, v in pr.items() if k != "steps"}
                prof["sum"] = sum(prof.values())
            d.close()
            d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, precision=P[name], averaged=order == 6)
            t0 = time.perf_counter()
            d.run_until(min(t_end, 0.125))
            wall8 = time.perf_counter() - t0
            d.close()
            ab = None
            if name == "fp64":                       # A/B: the same first 1/8 without the small-step kernel (one force call per step)
                d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, precision=P[name], averaged=order == 6)
                s2.s2_set_tuning(d.ctx, 9, 6)
                d.run_until(min(t_end, 0.125), time_device=True)
                sa = d.stats()
                d.close()
                ab = {"device_us_per_block_step": sa["device_ms"] / sa["timed_steps"] * 1e3, "block_steps": sa["block_steps"]}
            row = {"integrator": "device (s2_bts)", "order": order, "criterion": "Aarseth" if order == 4 else "mean of Aarseth(eta4) and generalised(eta6) (L156)", "precision": name, "block_steps": st["block_steps"],
                   "particle_steps": st["particle_steps"], "n_i_min": int(hist.min()), "n_i_median": float(np.median(hist)),
                   "n_i_mean": float(hist.mean()), "n_i_max": int(hist.max()), "wall_s": wall,
                   "wall_us_per_block_step": wall / st["block_steps"] * 1e6,
                   "ginteractions_per_s_wall": st["particle_steps"] * n / wall / 1e9, "dE_over_E": (e1 - e0) / e0,
                   "first_eighth": {"block_steps": sd["block_steps"], "wall_us_per_block_step": wall8 / sd["block_steps"] * 1e6,
                                    "device_us_per_block_step": sd["device_ms"] / sd["timed_steps"] * 1e3,
                                    "wall_over_device": wall8 * 1e3 / sd["device_ms"],
                                    "small_step_kernel": {"steps": sd["small"]["steps"], "launches": sd["small"]["launches"],
                                                          "device_us_per_step": sd["small"]["device_ms"] / max(sd["small"]["steps"], 1) * 1e3},
                                    "small_step_cycles": prof, "small_step_cycles_cta": prof_cta, "one_force_call_per_step": ab}}
            out["runs"].append(row)
            print(json.dumps(row), file=sys.stderr, flush=True)
    # the floor under a small step: SM cycles per round trip (two hops) of a word between SMs through L2
    ctx = s2.s2_open(0, 4, s2.S2_FP64, nj_capacity=64, ngb_cap=0)
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    out["hop_round_trip_cycles"] = {str(c): round(s2.s2_hop_latency(ctx, c, 2000)) for c in (2, 16, sms)}
    s2.s2_close(ctx)
    if host_reference:
        for order, H in ((4, Hermite4), (6, Hermite6)):
            if order not in orders:
                continue
            b = S2Backend(w.N, w.eps2, precision=s2.S2_FP64, order=order)
            h = H(b, w.mass, w.pos, w.vel, **({'averaged': True} if order == 6 else {}))
            b.calls = b.pairs = 0
            t0 = time.perf_counter()
            h.run_until(min(t_end, 0.125))
            wall = time.perf_counter() - t0
            out["runs"].append({"integrator": "host driver (hermite.py), first 1/8 time unit", "order": order, "precision": "fp64",
                                "block_steps": h.block_steps, "wall_s": wall, "wall_us_per_block_step": wall / h.block_steps * 1e6})
            b.close()
    print(json.dumps(out), flush=True)


def graph_time_us(s2, torch, ctx, fn, calls=20, reps=7):
    """Device time per call of `fn` (which only enqueues library calls): `calls` calls captured in one CUDA
    graph on a side stream, replayed `reps` times between CUDA events; median.  Removes the host launch cost
    and the ~6 us floor of an event pair around a single small kernel."""
    st = torch.cuda.Stream()
    s2.s2_set_stream(ctx, st.cuda_stream)
    with torch.cuda.stream(st):
        fn(); fn()                                   # warm-up: allocations and shape caches settle
    st.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        for _ in range(calls):
            fn()
    ts = []
    for _ in range(reps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); g.replay(); e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) / calls * 1e3)
    s2.s2_set_stream(ctx, torch.cuda.current_stream().cuda_stream)
    return statistics.median(ts[1:])


def fp32_fixup_cost(s2, torch, dev):
    """Cost of the fp32 path's fp64 re-evaluation of ill-conditioned jerk sums (reading R-F32): device time per
    s2_calc_ilist_device call with the fix-up (default) and without it (s2_set_tuning key 9 = 4), and the number of
    flagged particles; config 3 (graph-timed), the headline particle set and config 5 (CUDA events)."""
    from workloads import make_config
    out = {"rows": []}
    for key, nis, flags in ((3, (1, 32, 256, 2048, 16384, 65536), 0), ("H", (262144,), 0), (5, (1048576,), 3)):
        w = make_config(key)
        ctx = s2.s2_open(dev.index, 4, s2.S2_FP32, nj_capacity=w.N, ngb_cap=256 if flags else 0)
        a = np.arange(w.N, dtype=np.int32)
        s2.s2_set_j(ctx, a, w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
        s2.s2_commit_j(ctx)
        s2.s2_predict(ctx, w.t_pred, w.N)
        for ni in nis:
            ilh = w.ilist(ni)
            il = torch.from_numpy(ilh).to(dev)
            h2 = torch.from_numpy(np.ascontiguousarray(w.h2[ilh])).to(dev) if flags else None
            row = {"cfg": str(key), "N": w.N, "n_i": ni}
            for name, key9 in (("with_fixup_us", 0), ("without_fixup_us", 4)):
                s2.s2_set_tuning(ctx, 9, key9)
                if ni * w.N < 1e9:
                    us = graph_time_us(s2, torch, ctx, lambda: s2.s2_calc_ilist_device(ctx, il, h2, w.eps2, flags),
                                       calls=20 if ni * w.N < 2e8 else 4, reps=5)
                else:
                    s2.s2_enable_timing(ctx, True)
                    ts = []
                    for r in range(3):
                        s2.s2_calc_ilist_device(ctx, il, h2, w.eps2, flags)
                        t = s2.s2_get_timing(ctx)
                        ts.append(t["force_ms"] + t["reduce_ms"])
                    s2.s2_enable_timing(ctx, False)
                    us = min(ts[1:]) * 1e3
                row[name] = round(us, 1)
            s2.s2_set_tuning(ctx, 9, 0)
            s2.s2_calc_ilist_device(ctx, il, h2, w.eps2, flags)
            row["flagged"] = s2.s2_fp32_fixup_count(ctx)
            row["ginteractions_per_s_with"] = round(ni * w.N / row["with_fixup_us"] / 1e3, 1)
            row["ginteractions_per_s_without"] = round(ni * w.N / row["without_fixup_us"] / 1e3, 1)
            out["rows"].append(row)
        s2.s2_close(ctx)
    return out


def shape_space(s2, torch, dev):
    """Evidence behind the launch balancer and the choice of the deterministic combine, config 3
    (N = 65536, fp64, 4th order), graph-timed device time per s2_calc_ilist_device call:
      (a) n_i = 32: the automatic shape against forced neighbours in (lanes per i, warp columns, j-slices);
      (b) combine by reduce kernel / fused / fp64 atomics (s2_set_tuning key 5) at n_i = 32 ... 16384."""
    from workloads import make_config
    w = make_config(3)
    ctx = s2.s2_open(dev.index, 4, s2.S2_FP64, nj_capacity=w.N, ngb_cap=0)
    a = np.arange(w.N, dtype=np.int32)
    s2.s2_set_j(ctx, a, w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
    s2.s2_commit_j(ctx)
    s2.s2_predict(ctx, w.t_pred, w.N)

    def timed(ni, tune):
        for k in range(9):
            s2.s2_set_tuning(ctx, k, tune.get(k, 0))
        il = torch.from_numpy(w.ilist(ni)).to(dev)
        us = graph_time_us(s2, torch, ctx, lambda: s2.s2_calc_ilist_device(ctx, il, None, w.eps2, 0),
                           calls=20 if ni * w.N < 2e8 else 4, reps=9)
        info = s2.s2_last_launch_info(ctx)
        return {"n_i": ni, "forced": {str(k): v for k, v in tune.items()}, "us": round(us, 2),
                "ginteractions_per_s": round(ni * w.N / us / 1e3, 1), "S": info["S"], "lanes_per_i": info["lanes_per_i"],
                "warp_columns": info["warp_columns"], "grid": info["grid"], "i_per_thread": info["i_per_thread"],
                "combine": ("none", "reduce kernel", "fused", "chunk launches", "atomics", "chunk launches")[info["reduced"]]}

    out = {"workload": "config 3: N = 65536, fp64, 4th order; graph-timed (20 calls per graph, median of 9 replays)",
           "ni32_shapes": [timed(32, {})], "combine_ab": []}
    for L, Wj, S in ((16, 1, 148), (16, 1, 111), (16, 1, 92), (32, 1, 37), (32, 1, 74), (32, 1, 55), (32, 1, 148), (8, 1, 148),
                     (8, 1, 296), (16, 2, 74), (32, 2, 37)):
        out["ni32_shapes"].append(timed(32, {0: S, 1: L, 2: Wj}))
    for ni in (32, 256, 2048, 16384):
        for key5 in (0, 1, 2):
            out["combine_ab"].append(timed(ni, {5: key5} if key5 else {}))
    s2.s2_close(ctx)
    return out


def ni_sweep(s2, torch, dev, order):
    """Ginteractions/s versus n_i (4th order): config 3 (N = 65536) in fp64, double-single and fp32, the
    headline N = 2^18 in fp64, and config 2 (N = 64) latencies.  Device time of one s2_calc_ilist_device call
    (force sweep + combine), as in the paper's Fig. 2 protocol (kernel time only).  Calls with
    fewer than 1e9 pairs are timed by CUDA-graph replay of 20 (4 above 2e8 pairs) calls, larger ones by CUDA events per call."""
    from workloads import make_config
    out = []
    pow2 = tuple(1 << k for k in range(17))    # fp64 at config 3's N: every power of two from 1 to N (Fig. 2's axis)
    plan = ((3, "fp64", s2.S2_FP64, pow2),
            (3, "ds", s2.S2_DS, (1, 32, 256, 2048, 16384, 65536)),
            (3, "fp32", s2.S2_FP32, (1, 32, 256, 2048, 16384, 65536)),
            ("H", "fp64", s2.S2_FP64, (1, 32, 256, 4096, 262144)),
            (2, "fp64", s2.S2_FP64, (1, 2, 4, 8, 16, 32, 64)))
    for key, pname, prec, nis in plan:
        w = make_config(key)
        ctx = s2.s2_open(dev.index, 4, prec, nj_capacity=w.N, ngb_cap=0)
        a = np.arange(w.N, dtype=np.int32)
        s2.s2_set_j(ctx, a, w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
        s2.s2_commit_j(ctx)
        s2.s2_predict(ctx, w.t_pred, w.N)
        full = None
        rows = []
        for ni in nis[::-1]:
            il = torch.from_numpy(w.ilist(ni)).to(dev)
            if ni * w.N >= 1e9:
                s2.s2_enable_timing(ctx, True)
                reps = 3 if ni * w.N > 1e9 else 10
                ts = []
                for r in range(reps + 2):
                    s2.s2_calc_ilist_device(ctx, il, None, w.eps2, 0)
                    t = s2.s2_get_timing(ctx)
                    if r >= 2:
                        ts.append(t["force_ms"] + t["reduce_ms"])
                s2.s2_enable_timing(ctx, False)
                us, how = statistics.median(ts) * 1e3, "events"
            else:
                us, how = graph_time_us(s2, torch, ctx, lambda: s2.s2_calc_ilist_device(ctx, il, None, w.eps2, 0),
                                        calls=20 if ni * w.N < 2e8 else 4), "graph"
            g = ni * w.N / (us * 1e-6) / 1e9
            full = full or g
            info = s2.s2_last_launch_info(ctx)
            host_us = None
            if key == 2:      # config 2: per-call latency as the host sees it (host i-list in, results out, synchronised)
                il_h = w.ilist(ni)
                for _ in range(20):
                    s2.s2_calc_ilist(ctx, il_h, None, w.eps2, 0); s2.s2_get_results(ctx, ni)
                t0 = time.perf_counter()
                for _ in range(300):
                    s2.s2_calc_ilist(ctx, il_h, None, w.eps2, 0); s2.s2_get_results(ctx, ni)
                host_us = (time.perf_counter() - t0) / 300 * 1e6
                host_c_us = s2.s2_time_host_roundtrip(ctx, il_h, w.eps2, 0, 100000)   # BASELINE config 2: 10^5 repeats
            peak = FP64_PEAK_TFLOPS if pname == "fp64" else FP32_PEAK_TFLOPS
            rows.append({"cfg": str(key), "precision": pname, "N": w.N, "n_i": ni, "call_us": round(us, 2), "timing": how,
                         "ginteractions_per_s": g, "vs_full_rate": g / full,
                         "frac_of_peak_60flop": g * 1e9 * FLOP_PER_PAIR[4] / 1e12 / peak,
                         "S": info["S"], "lanes_per_i": info["lanes_per_i"], "warp_columns": info["warp_columns"],
                         "i_per_thread": info["i_per_thread"], "grid": info["grid"],
                         "combine": ("none", "reduce kernel", "fused", "none (chunk launches)", "atomics")[info["reduced"]]})
            if host_us is not None:
                rows[-1]["host_roundtrip_us"] = round(host_us, 1)          # through the Python binding (ctypes)
                rows[-1]["host_roundtrip_c_us"] = round(host_c_us, 1)      # the same two calls timed inside the library
                rows[-1]["host_roundtrip_c_reps"] = 100000
                # k such calls in one launch sequence and one synchronisation (s2_calc_ilist_batch): host us per i-list
                for kb in (8, 64):
                    lists = [il_h] * kb
                    for _ in range(20):
                        s2.s2_calc_ilist_batch(ctx, lists, None, w.eps2, 0); s2.s2_get_results(ctx, ni * kb)
                    t0 = time.perf_counter()
                    for _ in range(200):
                        s2.s2_calc_ilist_batch(ctx, lists, None, w.eps2, 0); s2.s2_get_results(ctx, ni * kb)
                    rows[-1][f"host_us_per_list_batch{kb}"] = round((time.perf_counter() - t0) / 200 / kb * 1e6, 2)
        out.extend(rows[::-1])
        s2.s2_close(ctx)
    return out


def neighbour_path(s2, torch, dev, hbm_gbs):
    """Config 5 (a7 + a8): N = n_i = 2^20 Salpeter Plummer sphere, nearest neighbour + neighbour lists (cap 256,
    mean 32 per i), fp64 and fp32; config 4's 6th-order fp64 sweep at n_i = N = 2^18; and the 2nd-order (acc + pot)
    fp64 sweep on the headline particle set.  One warm-up call, then the median of 3 event-timed calls."""
    from workloads import make_config
    out = []
    for key, order, pname, prec, flags in ((5, 4, "fp64", s2.S2_FP64, 3), (5, 4, "fp32", s2.S2_FP32, 3),
                                           (4, 6, "fp64", s2.S2_FP64, 0), ("H", 2, "fp64", s2.S2_FP64, 0)):
        w = make_config(key)
        ctx = s2.s2_open(dev.index, order, prec, nj_capacity=w.N, ngb_cap=256 if flags else 0)
        a = np.arange(w.N, dtype=np.int32)
        s2.s2_set_j(ctx, a, w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk,
                    w.snap if order == 6 else None, w.crackle if order == 6 else None)
        s2.s2_commit_j(ctx)
        s2.s2_predict(ctx, w.t_pred, w.N)
        il = w.ilist(w.N)
        d_il = torch.from_numpy(il).to(dev)
        d_h2 = torch.from_numpy(np.ascontiguousarray(w.h2[il])).to(dev) if flags else None
        s2.s2_enable_timing(ctx, True)
        ts = []
        for r in range(4):
            s2.s2_calc_ilist_device(ctx, d_il, d_h2, w.eps2, flags)
            t = s2.s2_get_timing(ctx)
            if r:
                ts.append(t["force_ms"] + t["reduce_ms"])
            if flags and r == 2:
                s2.s2_get_neighbours_csr_device(ctx, w.N)     # warm-up of the compaction kernels (first launch, allocations)
        ms = statistics.median(ts)
        info = s2.s2_last_launch_info(ctx)
        row = {"cfg": str(key), "order": order, "precision": pname, "N": w.N, "n_i": w.N,
               "outputs": "acc+jerk+pot+nn+neighbour lists" if flags else {2: "acc+pot", 4: "acc+jerk+pot", 6: "acc+jerk+snap+pot"}[order],
               "call_ms": ms,
               "ginteractions_per_s": w.N * w.N / (ms * 1e-3) / 1e9,
               "tflops_convention": w.N * w.N * FLOP_PER_PAIR[order] / (ms * 1e-3) / 1e12,
               "S": info["S"], "i_per_thread": info["i_per_thread"], "grid": info["grid"]}
        if flags:
            cnt = s2.s2_get_results(ctx, w.N)["ngb_count"]
            row.update(mean_neighbours=float(cnt.mean()), max_neighbours=int(cnt.max()), overflows=int((cnt > 256).sum()))
            # a8/a9 read-back: the lists are compacted on the device (count -> scan -> fill), then offsets + members
            # cross the host link; wall time of the whole s2_get_neighbours_csr call, device time of the compaction
            t0 = time.perf_counter()
            off, lst = s2.s2_get_neighbours_csr(ctx, w.N)
            wall = time.perf_counter() - t0
            ct = s2.s2_get_csr_timing(ctx)
            members = int(off[-1])
            dev_bytes = 20 * w.N + 8 * members            # count word + len + offset per i; 4 B read + 4 B written per member
            dev_ms = ct["scan_ms"] + ct["fill_ms"]
            row.update(list_readback_ms=wall * 1e3, list_members=members, list_d2h_bytes=(w.N + 1) * 8 + 4 * members,
                       fixed_stride_list_bytes=w.N * 256 * 4, csr_device_ms=dev_ms, csr_device_bytes=dev_bytes,
                       csr_device_GBs=dev_bytes / (dev_ms * 1e-3) / 1e9,
                       csr_frac_of_measured_hbm=dev_bytes / (dev_ms * 1e-3) / 1e9 / hbm_gbs,
                       call_plus_list_readback_ms=ms + wall * 1e3)
        out.append(row)
        s2.s2_close(ctx)
    return out


def hbm_kernels(s2, torch, dev, hbm_gbs):
    """Achieved HBM GB/s of the streaming kernels: the predictor (a2) and the commit scatter (a1, from device
    arrays) at N = 2^20 with config 5's (4th order) and config 4's (6th order) particle recipe.
    Algorithmic bytes per j are those of DESIGN.md 5.1; graph-replay timing."""
    from workloads import make_config
    out = []
    for key, order in ((5, 4), (4, 6)):
        w = make_config(key, N=1 << 20)            # both orders at N = 2^20: the working set exceeds the 126 MB L2
        ctx = s2.s2_open(dev.index, order, s2.S2_FP64, nj_capacity=w.N, ngb_cap=0)
        names = ["ident", "t_j", "mass", "pos", "vel", "acc", "jerk"] + (["snap", "crackle"] if order == 6 else [])
        d = {k: torch.from_numpy(getattr(w, k)).to(dev) for k in names}
        addr = torch.arange(w.N, dtype=torch.int32, device=dev)
        args = [addr, d["ident"], d["t_j"], d["mass"], d["pos"], d["vel"], d["acc"], d["jerk"]]
        args += [d["snap"], d["crackle"]] if order == 6 else [None, None]
        commit = lambda: s2.s2_commit_j_device(ctx, *args)
        commit()
        us_c = graph_time_us(s2, torch, ctx, commit, calls=10)
        us_p = graph_time_us(s2, torch, ctx, lambda: s2.s2_predict(ctx, w.t_pred, w.N), calls=10)
        nf = 20 if order == 6 else 14
        b_commit = w.N * ((nf * 8 + 8) + (nf * 8 + 4))
        b_pred = w.N * ((nf * 8 + 4) + (96 if order == 6 else 64))
        for name, us, b in (("scatter_kernel", us_c, b_commit), (f"predict_kernel<{order}>", us_p, b_pred)):
            gbs = b / (us * 1e-6) / 1e9
            out.append({"kernel": name, "N": w.N, "order": order, "bytes": b, "us": round(us, 2), "GB/s": gbs,
                        "frac_of_measured_hbm": gbs / hbm_gbs})
        s2.s2_close(ctx)
        if order == 4:
            # the combine of the j-slices (a6): 2^20 explicit sinks against a 4096-particle store in 4 forced slices,
            # so that the 4 x 2^20 partial records (403 MB) exceed L2; kernel time from the library's events
            S, nj = 4, 4096
            ctx = s2.s2_open(dev.index, 4, s2.S2_FP64, nj_capacity=nj, ngb_cap=0)
            a = np.arange(nj, dtype=np.int32)
            s2.s2_set_j(ctx, a, w.ident[:nj], w.t_j[:nj], w.mass[:nj], w.pos[:nj], w.vel[:nj], w.acc[:nj], w.jerk[:nj])
            s2.s2_commit_j(ctx)
            s2.s2_predict(ctx, w.t_pred, nj)
            s2.s2_enable_timing(ctx, True)
            for k, v in ((0, S), (5, 1), (7, 2)):
                s2.s2_set_tuning(ctx, k, v)
            ids = np.full(w.N, -1, dtype=np.int32)
            best = 1e9
            for _ in range(3):
                s2.s2_calc_explicit(ctx, ids, w.pos, w.vel, None, None, w.eps2, 0)
                best = min(best, s2.s2_get_timing(ctx)["reduce_ms"])
            info = s2.s2_last_launch_info(ctx)
            b = (info["S"] + 1) * w.N * 96
            gbs = b / (best * 1e-3) / 1e9
            out.append({"kernel": f"reduce_thread_kernel<{info['S']}>", "n_i": w.N, "rows": info["S"], "order": 4, "bytes": b,
                        "us": round(best * 1e3, 2), "GB/s": gbs, "frac_of_measured_hbm": gbs / hbm_gbs,
                        "timing": "CUDA events around the launch"})
            s2.s2_close(ctx)
    return out


def cpu_baseline(w):
    """The oracle as it stands, timed on the host cores on a bounded sample of the same workload."""
    import oracle
    xp, vp, ap = oracle.predict(w.order, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle)
    n_s = min(w.N, 4096)          # "on min(n_i, 4096) sample i against all N j"
    il = w.ilist(n_s)
    oracle.forces_ilist(w.order, w.mass, w.ident, xp, vp, ap, il[:64], w.eps2)     # page in, spin up the thread pool
    t0 = time.perf_counter()
    oracle.forces_ilist(w.order, w.mass, w.ident, xp, vp, ap, il, w.eps2)
    dt = time.perf_counter() - t0
    return {"value": n_s * w.N / dt / 1e9, "unit": "Ginteractions/s", "cores": oracle.max_threads(), "kind": "oracle",
            "sample": f"{n_s} of {w.N} i-particles (seeded prefix of the active-set permutation) x all {w.N} j, "
                      f"long double, {dt:.1f} s"}


if __name__ == "__main__":
    main()
