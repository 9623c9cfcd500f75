"""bench.py -- BASELINE.json metric on BASELINE.json configs[4]: the N=48 complete-graph Gaussian instance, S=100.

A "step" is ONE full pass of the hot path over one instance: all 2^48 spin configurations enumerated, filtered,
selected, the survivors re-evaluated in fp64 and the S lowest written.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config k] [--range-log2 r]
                    [--weak] [--n-spins 50|52]

  value          configurations evaluated per second, whole job, inputs resident in HBM, CUDA-event timed
  e2e            same through the host-buffer API: pinned HOST buffers in and out, copies inside the timed region
  roofline       the dominant kernel: the tensor-core screen (zwalk_kernel, one 128x128x128 bf16 tcgen05 GEMM per 2^21
                 configurations, 2 flop per configuration) against the measured cuBLAS bf16 rate of MEASURED_PEAKS.json
  roofline_packed16 / roofline_int32
                 the same full space, same invocation, through the packed 16-bit ALU screen only (ISING_KERNEL=16) and
                 through the int32 kernel (ISING_KERNEL=32: arithmetic no narrower than the paper's), each against the
                 MEASURED rate of its own instruction mix
  cpu_baseline   the CPU oracle, as it stands, on a bounded prefix of the same instance (rank 0, N=1 only)

N > 1 (torchrun): the path shards by ranges of q: ONE instance, one aligned state range per rank,
one all-gather of the per-rank lists, merge on every rank -- "strong" scaling, value = 2^N / (max over ranks of the
device time). --n-spins 50|52 swaps in a complete Gaussian instance of that size so that 8 ranks have seconds of
work each. --weak keeps the other reading (independent instances per rank, no data-path collective).
--impl reference times the CPU oracle (there is no other reference implementation in this tier).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "spin_configs_evaluated_per_s"
UNIT = "configs/s"
# `roofline` (the default path's dominant kernel, zwalk_kernel) is a TENSOR roofline against MEASURED_PEAKS.json.
# The constants below serve the two ALU kernels' own objects, `roofline_packed16` and `roofline_int32` (DESIGN.md
# "Roofline"): VIADDMNMX issues on the ALU pipe at 148 SMs x 4 sub-partitions x 16 lanes/clk (B300_MICROARCH.md "Pipe
# rates") x 1.965 GHz (MEASURED_PEAKS.json); the packed kernel's VIADDMNMX.U16x2 (ISING_KERNEL=16; it also ramps the
# threshold up for the default path) forms two 16-bit add-mins (two configurations) per lane instruction, the int32
# kernel (ISING_KERNEL=32) one. The packed kernel also forms part of its sums as packed adds on the FMA pipe and takes
# the minimum of two of them with one VIMNMX3.U16x2 (4 configurations per ALU lane instruction, 3 issue slots); with
# the ALU pipe at 16 lanes/clk and one warp instruction issued per clock per sub-partition the best possible mix of the
# two forms is 48 configurations/clk/sub-partition = 192 per SM. The `peak` of both ALU objects is the
# MEASURED rate of the kernel's own instruction mix (microbenchmarks run in this invocation); the derived bounds are
# reported beside it.
ALU_LANES_PER_CLK_PER_SM = 64
MIX_BOUND_CONFIGS_PER_CLK_PER_SM = 192
FMA_LANES_PER_CLK_PER_SM = 128


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number (1-based); 5 = N=48")
    ap.add_argument("--range-log2", type=int, default=0,
                    help="development only: enumerate just the first 2^r states per step (0 = the whole space)")
    ap.add_argument("--sharded", action="store_true",
                    help="go through paper_1904_03621_b200/sharded.py even with one rank (default for N > 1): ONE "
                         "instance, one aligned state range per rank, one all-gather, merge on every rank")
    ap.add_argument("--weak", action="store_true",
                    help="N > 1: every rank enumerates its own instance of the ensemble (weak scaling, no collective)")
    ap.add_argument("--n-spins", type=int, default=0,
                    help="replace the config's instance by a complete Gaussian instance of this many spins (S as in the "
                         "config); for multi-GPU runs, e.g. 50 or 52")
    ap.add_argument("--no-int32", action="store_true",
                    help="skip the ALU-kernel passes (one more full enumeration each: packed 16-bit 8 s, int32 18 s at N=48)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def instance_for_rank(k: int, rank: int, n_spins: int = 0):
    from paper_1904_03621_b200 import instances as I
    c = I.baseline_config(k)
    if n_spins:
        J, h = I.complete_gaussian(n_spins, I.SEED_BASE + 100 * n_spins + 1000 * rank)
        return I.Instance(f"complete_gauss_N{n_spins}_rank{rank}", n_spins, c.S, J, h, False)
    if rank == 0:
        return c
    # other ranks: an independent instance of the same ensemble (same generator, rank-specific seed)
    if k in (1, 3, 5):
        J, h = I.complete_gaussian(c.N, I.SEED_BASE + k + 1000 * rank, h_scale=0.5 if k == 3 else 1.0)
        return I.Instance(f"{c.name}_rank{rank}", c.N, c.S, J, h, False)
    return c


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "200",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self, t0: float, t1: float):
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.rows:
            if t < t0 or t > t1:
                continue
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample_rate(inst, seconds_target: float, S: int):
    """Time the oracle, as it stands, on a contiguous prefix of q sized for about `seconds_target` seconds."""
    from oracle import oracle
    cores = oracle.max_threads()
    k = min(inst.N, 20)
    t0 = time.perf_counter()
    oracle.lowest(inst.J, inst.h, S, 0, 1 << k)
    dt = max(time.perf_counter() - t0, 1e-6)
    rate = (1 << k) / dt
    want = rate * seconds_target
    kk = k
    while kk < inst.N and (1 << (kk + 1)) <= want:
        kk += 1
    if kk > k:
        t0 = time.perf_counter()
        oracle.lowest(inst.J, inst.h, S, 0, 1 << kk)
        dt = time.perf_counter() - t0
        rate = (1 << kk) / dt
    return rate, cores, kk, dt


def run_reference(args, rank: int, world: int):
    """--impl reference: the CPU oracle on the box's host cores; each step is a bounded sample of the workload."""
    if rank != 0:
        return
    from oracle import oracle
    inst = instance_for_rank(args.config, 0, args.n_spins)
    cores = oracle.max_threads()
    # size one step for roughly 3 s of oracle time
    rate, _, kk, _ = oracle_sample_rate(inst, 3.0, inst.S)
    n = 1 << kk
    for _ in range(args.warmup):
        oracle.lowest(inst.J, inst.h, inst.S, 0, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.lowest(inst.J, inst.h, inst.S, 0, n)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = (f"oracle.lowest on the first 2^{kk} of 2^{inst.N} states of {inst.name} per step; "
              f"full-space time extrapolated = {float(1 << inst.N) / value:.3e} s")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config - 1}]: {inst.name}, N={inst.N}, S={inst.S}",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1904_03621_b200 import binding as B, build

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    B.load()

    # N > 1: range-sharded on ONE instance unless --weak; N = 1: the plain call (or, with --sharded,
    # the same call through sharded.py, which must give the same number)
    sharded_mode = (world > 1 and not args.weak) or args.sharded
    inst = instance_for_rank(args.config, 0 if sharded_mode else rank, args.n_spins)
    N, S = inst.N, inst.S
    q_end = 1 << N
    if args.range_log2:
        q_end = 1 << max(min(args.range_log2, N), min(N, 20))
    configs_per_step = q_end
    J = torch.from_numpy(inst.J).cuda()
    h = torch.from_numpy(inst.h).cuda()
    out = (torch.empty(S, dtype=torch.int64, device="cuda"), torch.empty(S, dtype=torch.float64, device="cuda"))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")          # > 126 MB L2
    stream = torch.cuda.current_stream()
    if sharded_mode and args.range_log2:
        raise SystemExit("--range-log2 is a single-range development knob; it cannot be combined with the sharded mode")

    def step():
        if sharded_mode:
            from paper_1904_03621_b200 import sharded
            res = sharded.ising_lowest_sharded(J, h, S)    # every rank ends with the global list
            out[0].copy_(res[0]); out[1].copy_(res[1])
        else:
            B.ising_lowest_range(J, h, S, 0, q_end, stream=stream, out=out)
        return B.last_stats()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # roofline denominators measured live on this device (also quoted: the nominal ones DESIGN.md derives)
    fma_peak = B.fma_peak(50.0)
    addmin_peak = B.addmin_peak(50.0)
    addmin16x2_peak = B.addmin16x2_peak(50.0)
    addmin_mix_peak = B.addmin_mix_peak(50.0)

    for _ in range(args.warmup):
        flush.zero_()
        step()

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    barrier()
    t_wall0 = time.perf_counter()
    dev_ms = 0.0
    enum_ms = 0.0
    enum_launches = 0
    launches = 0
    enum_configs = 0
    hit_blocks = false_hit_blocks = 0
    z_ms = 0.0
    z_configs = z_blocks = z_flagged = z_launches = 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(args.steps):
        flush.zero_()                       # L2 flush between timed iterations (outside the event bracket)
        ev0.record(stream)
        st = step()
        ev1.record(stream)
        ev1.synchronize()
        dev_ms += ev0.elapsed_time(ev1)
        enum_ms += st.enum_ms
        enum_configs += st.configs
        enum_launches += st.enum_launches
        launches += st.kernel_launches
        hit_blocks += st.hit_blocks
        false_hit_blocks += st.false_hit_blocks
        z_ms += st.z_ms; z_configs += st.z_configs; z_blocks += st.z_blocks
        z_flagged += st.z_flagged_blocks; z_launches += st.z_launches
    barrier()
    t_wall1 = time.perf_counter()
    clocks = sampler.summary(t_wall0, t_wall1)
    result_states = B.states_to_numpy(out[0]).tolist()

    # ---- end to end: pinned host buffers in, host buffers out (ising_lowest_host; sharded: the same call through
    # sharded.py with the host arrays, every rank copying its result back to the host) ----
    e2e = None
    if not args.no_e2e:
        Jh = torch.from_numpy(inst.J).pin_memory()
        hh = torch.from_numpy(inst.h).pin_memory()
        qh = torch.empty(S, dtype=torch.int64).pin_memory()
        eh = torch.empty(S, dtype=torch.float64).pin_memory()
        out_h = (qh.numpy().view(np.uint64), eh.numpy())
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            if sharded_mode:
                from paper_1904_03621_b200 import sharded
                rq, re_ = sharded.ising_lowest_sharded(Jh.numpy(), hh.numpy(), S)   # H2D of J, h inside the solver call
                qh.copy_(rq, non_blocking=True); eh.copy_(re_, non_blocking=True)
                torch.cuda.synchronize()
            else:
                B.ising_lowest_host(Jh.numpy(), hh.numpy(), S, 0, q_end, stream=stream, out=out_h)
        barrier()
        e2e_s = time.perf_counter() - t0
        assert qh.numpy().view(np.uint64).tolist() == result_states
        e2e = {"seconds": e2e_s, "h2d": (N * N + N) * 8, "d2h": S * 16}

    # ---- the ALU kernels on the same workload, each timed with its own CUDA events; fewer steps (they are 14x and
    # 32x slower than the default path), rank-local like `roofline`: ISING_KERNEL=16 = packed 16-bit screen only (the
    # round-1 default), ISING_KERNEL=32 = 32-bit exact add-min per configuration (no narrower than the paper's) ----
    alu_runs = {}
    if not args.no_int32 and not sharded_mode:
        for kv, nsteps in ((16, 1 if st.kernel_variant == 128 else 0), (32, max(1, min(args.steps, 2)))):
            if nsteps == 0:
                continue
            os.environ["ISING_KERNEL"] = str(kv)
            try:
                msk = ek = 0.0
                ck = 0
                for _ in range(nsteps):
                    ev0.record(stream)
                    qk, _ = B.ising_lowest_range(J, h, S, 0, q_end, stream=stream)
                    ev1.record(stream); ev1.synchronize()
                    stk = B.last_stats()
                    assert stk.kernel_variant == kv
                    msk += ev0.elapsed_time(ev1); ek += stk.enum_ms; ck += stk.configs
                assert B.states_to_numpy(qk).tolist() == result_states       # same list as the default path
                alu_runs[kv] = {"ms_per_step": msk / nsteps, "enum_ms": ek, "configs": ck, "steps": nsteps,
                                "enum_launches": stk.enum_launches}
            finally:
                os.environ.pop("ISING_KERNEL", None)
    sampler.stop()

    # max over ranks of the device time
    times = torch.tensor([dev_ms, e2e["seconds"] if e2e else 0.0], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
    dev_ms_max, e2e_s_max = float(times[0]), float(times[1])
    total_configs = float(configs_per_step) * args.steps * (1 if sharded_mode else world)
    value = total_configs / (dev_ms_max * 1e-3)

    if rank == 0:
        sm_max_hz = 1.965e9
        peaks = None
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            sm_max_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        except Exception:
            peaks = None
        sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        fma_nominal = sms * FMA_LANES_PER_CLK_PER_SM * sm_max_hz       # FMA / s
        derived_mix = sms * MIX_BOUND_CONFIGS_PER_CLK_PER_SM * sm_max_hz

        def profile_number(fname):
            """First number of a one-line file under profiles/ (an ncu capture of one launch; its source says so)."""
            try:
                return float(open(os.path.join(ROOT, "profiles", fname)).read().split()[0])
            except Exception:
                return None

        def alu_roofline(variant, achieved, launches, ms):
            """Roofline object of an ALU enumeration kernel: one add-min per configuration against the MEASURED rate of
            its own instruction forms (register-only microbenchmarks run above, in this invocation)."""
            packed = variant == 16
            fused_live = addmin16x2_peak * 2 if packed else addmin_peak
            peak = max(fused_live, addmin_mix_peak) if packed else fused_live
            fused_nominal = sms * ALU_LANES_PER_CLK_PER_SM * sm_max_hz * (2 if packed else 1)
            r = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "add-min/s", "frac": achieved / peak,
                 "kernel": "ising::walk_kernel<Inner16>" if packed else "ising::walk_kernel<Inner32>",
                 "launches": launches, "avg_launch_ms": ms / max(launches, 1),
                 "peak_source": ("MEASURED in this run: max of ising_addmin16x2_peak x 2 (fused VIADDMNMX.U16x2 only) and "
                                 "ising_addmin_mix_peak (fused + IMAD/IMAD/VIMNMX3.U16x2 mix), register-only loops on the "
                                 "whole GPU" if packed else
                                 "MEASURED in this run: ising_addmin_peak (VIADDMNMX.S32, register-only loop)"),
                 "fused_only_nominal": fused_nominal, "frac_of_fused_only_nominal": achieved / fused_nominal}
            if packed:
                r.update({"fused_only_measured": fused_live, "mix_measured": addmin_mix_peak,
                          "mix_bound_derived": derived_mix, "frac_of_mix_bound_derived": achieved / derived_mix,
                          "mix_bound_note": "derived LP bound (ALU pipe 16 lanes/clk, 1 issue slot/clk per sub-partition); "
                                            "the measured mix does not reach it (DESIGN.md 5.2)"})
            return r

        enum_rate = float(enum_configs) / (enum_ms * 1e-3)     # all enumeration launches of this rank
        if st.kernel_variant == 128:
            # dominant kernel: the tensor-core screen. Algorithmic work = the GEMM: one 128 x 128 x 128 bf16 product per
            # 2^21 configurations = 2 flop per configuration; time = CUDA events around its launches.
            bf16_burst = float(peaks.get("bf16_tflops", 1590.0)) if peaks else 1590.0
            bf16_sust = float(peaks.get("bf16_tflops_sustained", 1400.0)) if peaks else 1400.0
            z_rate = float(z_configs) / (z_ms * 1e-3)
            achieved_tf = 2.0 * z_rate * 1e-12
            traffic = profile_number("zwalk_dram_bytes_per_launch.txt")
            roofline = {"bound": "tensor", "achieved": achieved_tf, "peak": bf16_sust, "unit": "TFLOP/s",
                        "frac": achieved_tf / bf16_sust, "traffic": traffic,
                        "traffic_source": ("ncu --set full capture of one launch of this kernel (dram__bytes_read.sum + "
                                           "dram__bytes_write.sum), stored in profiles/zwalk_dram_bytes_per_launch.txt; "
                                           "not re-measured in this run; algorithmic HBM bytes per configuration: 0")
                                          if traffic is not None else None,
                        "kernel": "ising::zwalk_kernel", "launches": z_launches,
                        "avg_launch_ms": z_ms / max(z_launches, 1),
                        "flop_per_configuration": 2.0, "configs_per_s_in_kernel": z_rate,
                        "share_of_enumeration_time": z_ms / enum_ms, "share_of_configurations": z_configs / enum_configs,
                        "peak_source": ("MEASURED_PEAKS.json bf16_tflops_sustained (cuBLAS bf16 GEMM back to back; the kernel "
                                        "is timed inside a long step)" if peaks else "fallback of B200_PROFILING.md"),
                        "peak_burst": bf16_burst, "frac_of_burst": achieved_tf / bf16_burst,
                        "peak_nominal": 2250.0, "frac_of_nominal": achieved_tf / 2250.0,
                        "blocks_screened": z_blocks, "blocks_flagged": z_flagged,
                        "note": "the GEMM is the algorithmic work of the screen; around it every thread generates its "
                                "operand row and folds its accumulator row on the CUDA cores (DESIGN.md 5.1c), and the "
                                "first 2^35 states go through the packed ALU kernel (roofline_packed16)"}
            dtype = "bf16 tensor-core screen (fp32 accumulate) + int16x2 screen + int32 exact (fp64 output)"
            evaluated = ("bf16 partition-function term per configuration (tensor-core screen of 2^14-configuration blocks); "
                         "exact int32 energy for every configuration of a flagged block and of the packed ramp-up's hit "
                         "blocks; `value` counts configurations SCREENED, `value_int32` configurations whose int32 energy "
                         "is formed one by one (ISING_KERNEL=32)")
        else:
            roofline = alu_roofline(st.kernel_variant, enum_rate, enum_launches, enum_ms)
            traffic = profile_number("enumerate_dram_bytes_per_launch.txt")
            roofline["traffic"] = traffic
            roofline["traffic_source"] = ("ncu --set full capture of one launch of this kernel, stored in "
                                          "profiles/enumerate_dram_bytes_per_launch.txt; not re-measured in this run"
                                          if traffic is not None else None)
            dtype = "int16x2 screen + int32 exact (fp64 output)" if st.kernel_variant == 16 else "int32 (fp64 output)"
            evaluated = ("16-bit lower bound per configuration (packed screen); exact int32 energy for every configuration of "
                         "a hit block" if st.kernel_variant == 16 else "exact int32 energy per configuration")
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong" if (sharded_mode and world > 1) else "weak", "vs_baseline": None,
            "dtype": dtype,
            "evaluated": evaluated,
            "value_int32": None,        # filled below from the int32 pass of this invocation (the strict-reading figure)
            "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}]: {inst.name}, N={N}, S={S}, "
                                   f"states [0, 2^{q_end.bit_length() - 1}) of 2^{N} per step",
                       "instance_sha256": inst.sha256(),
                       "parallelism": (f"one instance, {world} state range(s) + one all-gather + merge (sharded.py)"
                                       if sharded_mode else
                                       f"independent instances x{world}" if world > 1 else "single GPU"),
                       "l2": "256 MiB buffer written between timed steps (inputs are 18 KB; the path has no HBM traffic)",
                       "grid_exponent_p": st.grid_exponent, "epsilon": st.epsilon, "kept": st.keep,
                       "kernel_variant": st.kernel_variant, "screen_shift": st.screen_shift,
                       "candidates": st.candidates, "passes": st.passes,
                       "screened_blocks_formed_exactly": hit_blocks, "of_which_false_hits": false_hit_blocks},
            "time_to_S_lowest_s": dev_ms_max * 1e-3 / args.steps,
            "fp32_fma_roofline": {"definition": "configs/s x N / peak FP32 FMA/s (BASELINE.json metric)",
                                  "frac_of_measured": value / world * N / fma_peak,
                                  "frac_of_nominal": value / world * N / fma_nominal,
                                  "fma_per_s_measured": fma_peak, "fma_per_s_nominal": fma_nominal},
            "roofline": roofline,
            "enumeration_all_launches": {"configs_per_s": enum_rate, "launches": enum_launches, "ms": enum_ms},
            "microbenchmarks_live": {"ffma_per_s": fma_peak, "viaddmnmx_s32_per_s": addmin_peak,
                                     "viaddmnmx_u16x2_inst_per_s": addmin16x2_peak, "addmin_mix_per_s": addmin_mix_peak},
            "gpu_launches": launches,
            "clocks": clocks,
        }
        for kv, key in ((16, "roofline_packed16"), (32, "roofline_int32")):
            if kv in alu_runs:
                rr = alu_runs[kv]
                ak = float(rr["configs"]) / (rr["enum_ms"] * 1e-3)
                obj = alu_roofline(kv, ak, rr["enum_launches"] * rr["steps"], rr["enum_ms"])
                obj.update({"time_to_S_lowest_s": rr["ms_per_step"] * 1e-3,
                            "configs_per_s": float(configs_per_step) / (rr["ms_per_step"] * 1e-3),
                            "steps": rr["steps"], "same_list_as_default_path": True,
                            "dtype": "int16x2 screen + int32 exact (fp64 output)" if kv == 16 else "int32 (fp64 output)"})
                line[key] = obj
                if kv == 32:
                    line["value_int32"] = obj["configs_per_s"]
        if e2e:
            line["e2e"] = {"value": total_configs / e2e_s_max, "unit": UNIT,
                           "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"]}
        if world == 1 and not args.range_log2 and not args.n_spins:
            # north_star: configs/s and time-to-solution for every BASELINE.json config (the other four are
            # parity-test cases, reported here for reference only: median of 5 whole-space calls, CUDA events)
            per = []
            for k in (1, 2, 3, 4):
                ck = instance_for_rank(k, 0)
                Jk = torch.from_numpy(ck.J).cuda(); hk = torch.from_numpy(ck.h).cuda()
                ts = []
                for _ in range(6):
                    ev0.record(stream)
                    B.ising_lowest(Jk, hk, ck.S, stream=stream)
                    ev1.record(stream); ev1.synchronize()
                    ts.append(ev0.elapsed_time(ev1))
                ms = sorted(ts[1:])[2]
                stk = B.last_stats()
                per.append({"config": k, "name": ck.name, "N": ck.N, "S": ck.S, "time_to_S_lowest_ms": ms,
                            "configs_per_s": float(1 << ck.N) / (ms * 1e-3), "exact": bool(stk.exact),
                            "screen_shift": stk.screen_shift, "candidates": stk.candidates,
                            "kernel_launches": stk.kernel_launches,
                            "fp32_fma_roofline_frac": float(1 << ck.N) / (ms * 1e-3) * ck.N / fma_peak})
            per.append({"config": 5, "name": inst.name, "N": N, "S": S, "time_to_S_lowest_ms": dev_ms_max / args.steps,
                        "configs_per_s": value, "exact": bool(st.exact), "screen_shift": st.screen_shift,
                        "candidates": st.candidates, "kernel_launches": st.kernel_launches,
                        "fp32_fma_roofline_frac": value * N / fma_peak})
            line["per_config"] = per
            # "time proportional to 2^N": complete Gaussian instances N = 24 .. 44, configs/s of the whole call
            sweep = []
            for n in (24, 28, 32, 36, 40, 44):
                from paper_1904_03621_b200 import instances as I
                Jn, hn = I.complete_gaussian(n, I.SEED_BASE + 100 * n)
                Jn = torch.from_numpy(Jn).cuda(); hn = torch.from_numpy(hn).cuda()
                ts = []
                for _ in range(3 if n >= 40 else 5):
                    ev0.record(stream)
                    B.ising_lowest(Jn, hn, 100, stream=stream)
                    ev1.record(stream); ev1.synchronize()
                    ts.append(ev0.elapsed_time(ev1))
                ms = sorted(ts[1:])[len(ts[1:]) // 2]
                sweep.append({"N": n, "S": 100, "ms": ms, "configs_per_s": float(1 << n) / (ms * 1e-3)})
            sweep.append({"N": N, "S": S, "ms": dev_ms_max / args.steps, "configs_per_s": value})
            line["n_sweep_complete_gaussian"] = sweep
            # the paper's own pipeline (Algorithm 1) written plainly for this GPU, on a 2^28-state slice of the same
            # instance: the on-box "prior design" figure; not a target, not the reference arm
            n_alg1 = 1 << min(28, N)
            B.ising_lowest_alg1(J, h, S, 0, n_alg1, stream=stream)
            ev0.record(stream)
            B.ising_lowest_alg1(J, h, S, 0, n_alg1, stream=stream)
            ev1.record(stream); ev1.synchronize()
            line["paper_pipeline_on_box"] = {
                "value": float(n_alg1) / (ev0.elapsed_time(ev1) * 1e-3), "unit": UNIT,
                "what": "ising_lowest_alg1: chunks of 2^20 states, eq. (1) directly in fp64 per state, chunk stored, "
                        "S lowest selected by a full sort (PAPER.md:91-114)",
                "sample": f"first 2^{n_alg1.bit_length() - 1} states of {inst.name}"}
        if world == 1 and not args.no_cpu_baseline:
            rate, cores, kk, dt = oracle_sample_rate(inst, 15.0, S)
            line["cpu_baseline"] = {
                "value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": f"oracle.lowest on the first 2^{kk} of 2^{N} states of {inst.name} ({dt:.1f} s); "
                          f"full-space time extrapolated = {float(1 << N) / rate:.3e} s"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
