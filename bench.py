#!/usr/bin/env python
"""bench.py -- integrand evaluations per second of the whole hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--math exact|fast] [--impl reference]

A "step" is one complete tree search (zmc_run: every level's sampling + control kernels) of the
workload; inputs (bounds, parameters, derived keys) are resident on the device for `value`, and pass
through the C ABI from host arrays, with the result read back, for `e2e`. One JSON line on stdout.
DESIGN.md section 7 states the workloads, the ALU roofline and what each key means.

N > 1 (torchrun, one rank per GPU): BASELINE.json rules multi-GPU out of scope ("one GPU only"), so
the ranks are independent replicas of the same problem with seeds seed+rank -- no data-path
collective; torch.distributed only supplies the barrier, the max over ranks of the device time and
the sum of evaluations ("scaling": "weak").
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "integrand_evals_per_s"
UNIT = "evals/s"
PHILOX_IMAD_WIDE_PER_CALL = 20      # 2 IMAD.WIDE.U32 per round, 10 rounds
IMAD_WIDE_CLK_PER_WARP_INST_PER_SM = 1.0   # measured on B200 (zmc_microbench which=0/10), DESIGN.md section 6


def workloads():
    from paper_1902_07916_b200 import workloads as W
    return {
        # BASELINE.json configs[1] with the refinement budget of DESIGN.md R12 (paper semantics need 2.2e14 evals)
        "cfg2_sin6d_depth3_B16": W.config2(depth=3, budget=16),
        # BASELINE.json configs[1], levels 1-2 with the budget off (paper semantics; 6.4e11 evals, ~3 s per step)
        "cfg2_sin6d_depth2": W.config2(depth=2, budget=0),
        "cfg2_sin6d_depth1": W.config2(depth=1, budget=0),
        # BASELINE.json configs[2], whole
        "cfg3_gauss9d": W.config3(),
        # BASELINE.json configs[3] with budget 4 per instance (unbudgeted: ~1.7e12 evals)
        "cfg4_batched4d_B4": W.config4().with_(max_groups_per_level=4),
        # BASELINE.json configs[3] whole, the paper's semantics (about 1.7e12 evaluations, 8e7 level-2 cells, ~5 s)
        "cfg4_batched4d": W.config4().with_(max_cells_per_level=1024 * 1296 * 96),
        # BASELINE.json configs[4], level 1 only (the 5.2e11 evaluations BASELINE.json quotes)
        "cfg5_sin6d_level1": W.config5(depth=1),
        # BASELINE.json configs[4] to its full depth 4 as SURVEY R12 prescribes: level 1 is the whole 262144-cell group (~4e4 cells
        # flagged), the budget keeps one cell per level, so levels 2-4 are three more 262144-cell groups (2.1e12 evaluations, ~8 s)
        "cfg5_sin6d_depth4_B1": W.config5(depth=4, budget=1),
        "cfg1_sin3d_f64": W.config1(),
        # the paper's 12-D Gaussian (Table 4: 47.6 s on one V100), paper's own sizes
        "cfg12_gauss12d": W.gauss12d(),
        # the paper's own parameter sets (context: 38.7 s and 4.8 s on one V100)
        "paper_t3_sin6d": W.paper_table3_sin6d(),
        "paper_t4_gauss9d": W.paper_table4_gauss9d(),
    }


# what each bench workload leaves out of (or adds to) the BASELINE.json config it is named after, stated in the JSON line
DEVIATIONS = {
    "cfg2_sin6d_depth3_B16": "BASELINE.json configs[1] at its full depth 3 with a refinement budget of 16 cells per level (DESIGN.md R12): "
                             "under the paper's rule m = 1.5 flags ~8 % of the cells by chance and depth 3 needs ~2.2e14 evaluations (~14 min); "
                             "cfg2_sin6d_depth2 is the same config without budget, cut at depth 2",
    "cfg2_sin6d_depth2": "BASELINE.json configs[1] under the paper's rule (no budget), depth 2 of 3",
    "cfg2_sin6d_depth1": "BASELINE.json configs[1], level 1 only",
    "cfg4_batched4d_B4": "BASELINE.json configs[3] with a refinement budget of 4 cells per instance; cfg4_batched4d is the config as given",
    "cfg5_sin6d_depth4_B1": "BASELINE.json configs[4] at its full depth 4 with a refinement budget of 1 cell per level (DESIGN.md R12): level 1 flags "
                            "~4e4 of its 262144 cells, the compaction keeps the first; without budget level 2 alone needs > 2e16 evaluations",
    "cfg5_sin6d_level1": "BASELINE.json configs[4], level 1 only (the 5.24e11 evaluations it quotes); deeper levels need > 2e16 evaluations",
}


# total times the paper prints for its own parameter sets on one Tesla V100: context, not a target
PAPER_SECONDS = {"paper_t3_sin6d": 38.7, "paper_t4_gauss9d": 4.8, "cfg12_gauss12d": 47.6}


def capacity_for(w):
    """max_cells_per_level the bench (and the full-size parity tests) run a workload with: what its budget
    or depth bounds, else 0 = the library's automatic capacity."""
    if w.max_cells_per_level:
        return w.max_cells_per_level
    if w.max_groups_per_level:
        return w.k * w.n_instances * max(1, w.max_groups_per_level)
    if w.depth == 1:
        return w.k * w.n_instances
    return 0


def calls_per_eval(dim):
    return dim / 4.0     # flat word stream (R3): D words of 32 bits per sample, 4 words per Philox call


def alu_peak_evals_per_s(dim, n_sm, sm_mhz):
    """IMAD.WIDE-pipe roof: one warp-wide IMAD.WIDE.U32 per SM per clock (measured), 20 per Philox call."""
    clk_per_warp_eval = PHILOX_IMAD_WIDE_PER_CALL * IMAD_WIDE_CLK_PER_WARP_INST_PER_SM * calls_per_eval(dim)
    return n_sm * sm_mhz * 1e6 * 32.0 / clk_per_warp_eval


def imad_wide_issued_per_eval(dim):
    """IMAD.WIDE.U32 the shipped FP32 kernels issue per evaluation (SASS count, confirmed by ncu: profiles/r2_pipe_split.md).
    Of a call's 20 multiplies the unit-constant ones are hoisted (M1*c2 of round 1, M0*c0 of round 2): 18 per call; with
    P0_CARRY (D = 4, 6, 12) the first round's M0*c0 is a 64-bit addition as well: 17 per call."""
    per_call = 17 if dim in (4, 6, 12) else 18
    return per_call * calls_per_eval(dim)


# FP32 instructions (scalar count) and XU conversions per evaluation of the built-in integrands in exact mode (R8):
# map D FFMA; SIN_SUM: D-1 FADD + 11 (zsin); EXP_QUAD: D (quadratic form) + 1 + 10 (zexp). One F2F.F64.F32 per sample on the XU pipe.
def fp32_ops_per_eval(w):
    if w.integrand == "sin_sum":
        return w.dim + (w.dim - 1) + 11
    if w.integrand == "exp_quad":
        return w.dim + w.dim + 1 + 10
    return 2 * w.dim


# FP64 instructions per evaluation of the built-in integrands in FP64 mode (R8; the op sequences of ZmcMapF64 / ZmcIntegrand<.., F64>):
# map 3 per dimension (DADD for (double)w + 0.5, DMUL, DADD); SIN_SUM: D-1 DADD + 15 (zmc_zsin64); EXP_QUAD: 3D - 1 (quadratic form) + 1 +
# ~20 (libdevice exp); 1 DADD into the per-lane sum. The FP64 pipe takes one warp-instruction per 2 clocks per scheduler (profiles/r1_microbench.md).
FP64_CLK_PER_WARP_INST = 2.0


def fp64_ops_per_eval(w):
    if w.integrand == "sin_sum":
        return 3 * w.dim + (w.dim - 1) + 15 + 1
    if w.integrand == "exp_quad":
        return 3 * w.dim + (3 * w.dim - 1) + 1 + 20 + 1
    if w.integrand == "linear":
        return 3 * w.dim + 2 * w.dim + 1
    return 3 * w.dim + 1


def fp64_peak_evals_per_s(w, n_sm, sm_mhz):
    """FP64-pipe roof (C = max(4 n_imad, 2 n_fp64, slots)): evaluations/s if only the FP64 pipe were the limit."""
    return n_sm * 4 * 32.0 * sm_mhz * 1e6 / (FP64_CLK_PER_WARP_INST * fp64_ops_per_eval(w))


def other_roofs(w, n_sm, sm_mhz):
    """The roofs BASELINE.json's metric names, for the integrand's operation mix, next to the IMAD.WIDE roof that binds:
    FP32: 128 lanes per SM per clock; XU (F2F.F64.F32, MUFU): one warp-instruction per 8.5 clocks per scheduler (measured,
    profiles/r1_microbench.md) = 15.06 lanes per SM per clock."""
    f = sm_mhz * 1e6
    if w.precision == "f64":
        return {"imad_wide_gevals_per_s": alu_peak_evals_per_s(w.dim, n_sm, sm_mhz) / 1e9,
                "fp64_pipe_gevals_per_s": fp64_peak_evals_per_s(w, n_sm, sm_mhz) / 1e9,
                "note": "evaluations/s if only that pipe were the limit (FP64 mode: %d FP64 instructions at %g clocks and %g IMAD.WIDE at 4 clocks per "
                        "warp-evaluation; the roof is the lower of the two)" % (fp64_ops_per_eval(w), FP64_CLK_PER_WARP_INST, PHILOX_IMAD_WIDE_PER_CALL * calls_per_eval(w.dim))}
    return {"fp32_fma_gevals_per_s": n_sm * 128.0 * f / fp32_ops_per_eval(w) / 1e9,
            "xu_gevals_per_s": n_sm * 4 * 32.0 / 8.5 * f / 1.0 / 1e9,
            "note": "evaluations/s if only that pipe were the limit (exact mode: %d FP32 instructions and 1 XU conversion per evaluation)" % fp32_ops_per_eval(w)}


def traffic_from_profiles(workload, math):
    """DRAM bytes (read + write) per launch of the sampling kernel from the committed ncu --set full summary
    (profiles/traffic.csv): the mean over the launches captured for this workload, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None, None
    vals, commits = [], set()
    for line in open(path):
        parts = [x.strip() for x in line.split(",")]
        if line.startswith("#") or len(parts) < 5 or parts[0] != workload or parts[1] != math:
            continue
        vals.append(float(parts[3]) + float(parts[4]))
        if len(parts) > 6:
            commits.add(parts[6])
    if not vals:
        return None, None
    return sum(vals) / len(vals), ",".join(sorted(commits))


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.FIELDS,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            busy = sm[len(sm) // 2:]        # the upper half: samples taken under load
            out = {"sm_mhz": busy[len(busy) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                   "power_w_max": max(power), "samples": len(sm)}
        return out


def aggregate(ms_local, evals_local, world_size):
    """max over ranks of the device time, sum over ranks of the evaluations (torch.distributed if N > 1)."""
    if world_size == 1:
        return ms_local, evals_local
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    e = torch.tensor([float(evals_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(e, op=dist.ReduceOp.SUM)
    return float(t.item()), int(e.item())


def oracle_sample(w, n_units, seed_offset=0):
    """Time the oracle, as it stands, on n_units (cell, trial) units of level 1 of workload w (single thread).
    Returns (evals, seconds)."""
    import numpy as np
    import oracle as O
    cfg = O.config_from_workload(w)
    rng = np.random.default_rng(1234 + seed_offset)
    cells = rng.integers(0, w.k, size=n_units)
    t0 = time.perf_counter()
    for i, c in enumerate(cells):
        path, coords = O.path_coords(w.dim, w.g, [int(c)])
        O.unit_sum(cfg, int(i % w.n_instances), path, 1, coords, int(i % w.trials))
    dt = time.perf_counter() - t0
    return n_units * w.n_samples, dt


def _oracle_worker(job):
    """One process of the all-cores oracle baseline (spawned before CUDA is touched)."""
    name, precision, units, offset = job
    w = workloads()[name]
    if precision != "workload":
        w = w.with_(precision=precision)
    ev, sec = oracle_sample(w, units, offset)
    return ev, sec


def oracle_all_cores(name, precision, units_per_core):
    """The oracle, as it stands, in one process per host core (it is single-threaded): aggregate evaluations/s."""
    import concurrent.futures as cf
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    t0 = time.perf_counter()
    with cf.ProcessPoolExecutor(max_workers=cores, mp_context=mp.get_context("spawn")) as ex:
        res = list(ex.map(_oracle_worker, [(name, precision, units_per_core, 1000 + i) for i in range(cores)]))
    wall = time.perf_counter() - t0
    ev = sum(e for e, _ in res)
    busy = max(s for _, s in res)
    return {"value": ev / busy, "unit": UNIT, "cores": cores, "kind": "oracle, one process per core",
            "sample": "%d (cell,trial) units per core, %.1f s busy, %.1f s wall with process start-up" % (units_per_core, busy, wall)}


def run_reference(args, w, name):
    """--impl reference: the oracle on the host cores, same metric/config; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    units = max(1, int(2.0e7 // w.n_samples))        # ~1 s of single-thread work per step
    for i in range(args.warmup):
        oracle_sample(w, max(1, units // 10), i)
    ev, sec = 0, 0.0
    for i in range(args.steps):
        e, s = oracle_sample(w, units, 100 + i)
        ev += e
        sec += s
    val = ev / sec
    sample = "%d (cell,trial) units of level 1 per step, %d samples each, oracle.unit_sum, single thread" % (units, w.n_samples)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if w.precision == "f32" else "f64", "data": "synthetic",
            "config": {"workload": name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2_sin6d_depth3_B16")
    ap.add_argument("--math", default="exact", choices=["exact", "fast"])
    ap.add_argument("--precision", default="workload", choices=["workload", "f32", "f64"], help="override the workload's evaluation precision")
    ap.add_argument("--spread", default="trials", choices=["trials", "samples"], help="DESIGN.md R13")
    ap.add_argument("--budget-order", default="path", choices=["path", "spread"], help="DESIGN.md R14")
    ap.add_argument("--graph", action="store_true", help="replay each step as one CUDA graph (ZMC_OPT_USE_GRAPH)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cpu-all-cores", action="store_true", help="skip the oracle-on-every-host-core baseline (cpu_baseline_all_cores)")
    ap.add_argument("--no-extra", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    wl = workloads()
    w = wl[args.workload]
    if args.precision != "workload":
        w = w.with_(precision=args.precision)

    if args.impl == "reference":
        run_reference(args, w, args.workload)
        return
    all_cores = None
    if (not args.no_cpu_all_cores and not args.no_cpu_baseline and int(os.environ.get("RANK", "0")) == 0
            and int(os.environ.get("WORLD_SIZE", "1")) == 1):      # before CUDA is initialised in this process
        all_cores = oracle_all_cores(args.workload, args.precision, max(1, int(1.0e8 // w.n_samples)))

    import numpy as np
    import torch
    from paper_1902_07916_b200 import binding as B, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    n_dev = torch.cuda.device_count()
    shared = int(os.environ.get("LOCAL_WORLD_SIZE", world)) > n_dev   # more ranks than GPUs (a smoke run of the N > 1 path on one GPU):
    local_dev = local_rank % n_dev                      # the ranks share devices; NCCL cannot, so the plumbing goes over gloo
    torch.cuda.set_device(local_dev)
    if world > 1:
        import torch.distributed as dist
        if shared or os.environ.get("ZMC_BENCH_BACKEND") == "gloo":
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_dev))
    math = B.MATH_EXACT if args.math == "exact" else B.MATH_FAST
    w_rank = w.with_(seed=w.seed + rank)            # replicas differ only in the seed
    cap = capacity_for(w)
    spread = B.SPREAD_SAMPLES if args.spread == "samples" else B.SPREAD_TRIALS
    order = B.BUDGET_LARGEST_SPREAD if args.budget_order == "spread" else B.BUDGET_PATH_ORDER
    it = B.from_workload(w_rank, math=math, max_cells_per_level=cap, use_graph=args.graph, spread=spread, budget_order=order)
    it.use_torch_workspace()
    props = torch.cuda.get_device_properties(local_dev)
    n_sm = props.multi_processor_count
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        flush.zero_()
        it.run(stream.cuda_stream)
    it.result()
    barrier()
    sampler = ClockSampler(local_dev) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_wall = time.perf_counter()
    e0.record(stream)
    for _ in range(args.steps):
        flush.zero_()
        it.run(stream.cuda_stream)
    e1.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall
    ms_local = e0.elapsed_time(e1)
    value_v, value_s = it.result()
    st = it.stats()
    clocks = sampler.stop() if sampler else None
    evals_step = int(st.total_evals)
    ms_total, evals_total = aggregate(ms_local, evals_step * args.steps, world)
    ms_per_step = ms_total / args.steps
    value = evals_total / (ms_total * 1e-3)

    # dominant kernel: the fused sampling kernel, timed by the CUDA events zmc_run records around it on its stream
    samp_ms = sum(st.level[l].sample_ms for l in range(st.levels) if st.level[l].n_cells)
    ctl_ms = sum(st.level[l].control_ms for l in range(st.levels) if st.level[l].n_cells)
    n_sample_launches = sum(1 for l in range(st.levels) if st.level[l].n_cells)
    if args.graph or samp_ms <= 0:      # a graph replay has no events inside: charge the whole step to the sampling kernel
        samp_ms = st.total_ms
    achieved = evals_step / (samp_ms * 1e-3)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak = alu_peak_evals_per_s(w.dim, n_sm, sm_max)
    if w.precision == "f64":      # C = max(4 n_imad, 2 n_fp64): whichever pipe is the slower one
        peak = min(peak, fp64_peak_evals_per_s(w, n_sm, sm_max))
    traffic, traffic_commit = traffic_from_profiles(args.workload, args.math)
    peak_issued = n_sm * sm_max * 1e6 * 32.0 / (IMAD_WIDE_CLK_PER_WARP_INST_PER_SM * imad_wide_issued_per_eval(w.dim))
    roofline = {"bound": "alu", "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": "Gevals/s", "frac": achieved / peak,
                "frac_algorithmic": achieved / peak,
                # the same time against the multiplies the kernel really issues (FP32 built-ins): the share of the time the FMA-heavy pipe spends on them
                "frac_pipe": (achieved / peak_issued) if w.precision == "f32" else None,
                # FP64 mode, measured (profiles/r3_fp64_pipe_split.md): on B200 the FP64 pipe and the FMA-heavy pipe do not overlap -- their busy cycles ADD UP to the
                # elapsed ones -- so the time that cannot be undercut is 4 n_imad + 2 n_fp64 clocks per warp-evaluation, not the larger of the two
                "frac_shared_pipe": (achieved / (1.0 / (1.0 / alu_peak_evals_per_s(w.dim, n_sm, sm_max) + 1.0 / fp64_peak_evals_per_s(w, n_sm, sm_max)))) if w.precision == "f64" else None,
                "imad_wide_per_eval": {"algorithmic": PHILOX_IMAD_WIDE_PER_CALL * calls_per_eval(w.dim), "issued": imad_wide_issued_per_eval(w.dim)},
                "other_roofs": other_roofs(w, n_sm, sm_max),
                "traffic": traffic,
                "traffic_source": ("profiles/traffic.csv: ncu --set full capture at commit %s" % traffic_commit) if traffic is not None else None,
                "kernel": "zmc_sample_kernel", "launches_per_step": n_sample_launches, "avg_launch_ms": samp_ms / max(1, n_sample_launches),
                "share_of_step": samp_ms / (st.total_ms if st.total_ms > 0 else ms_per_step),
                "peak_basis": "IMAD.WIDE.U32 pipe: %d SMs x %.0f MHz (sm_max_mhz, %s) x 32 lanes / (20 IMAD.WIDE per Philox call x %.2f calls per eval x 1 clk)" %
                              (n_sm, sm_max, "MEASURED_PEAKS.json" if peaks else "guide nominal", calls_per_eval(w.dim)),
                "control_ms_per_step": ctl_ms}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if w.precision == "f32" else "f64", "data": "synthetic",
            "config": {"workload": args.workload, "note": w.note, "dim": w.dim, "divisions_per_axis": w.g, "samples_per_cell": w.n_samples,
                       "trials": w.trials, "depth": w.depth, "sigma_multiplier": w.sigma_multiplier, "seed": w.seed,
                       "n_instances": w.n_instances, "max_groups_per_level": w.max_groups_per_level, "math": args.math, "graph": bool(args.graph), "spread": args.spread, "budget_order": args.budget_order,
                       "evals_per_step": evals_step, "l2": "256 MiB buffer written between steps (flush); the path reads ~16 B per cell",
                       "parallelism": "replicas x%d" % world,
                       "deviation": DEVIATIONS.get(args.workload)},
            "result": {"value": float(value_v[0]), "std": float(value_s[0])},
            "wall_ms_per_step": 1e3 * t_wall / args.steps,
            "gpu_launches": int(st.kernel_launches) * args.steps,      # counted by zmc_run as it enqueues them; all the library's own
            "roofline": roofline}
    if clocks is not None:
        line["clocks"] = clocks

    if rank == 0:
        # ---- e2e: the call a user makes, from host arrays to host result, every step
        e2e_steps = max(1, args.steps)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ev = 0
        for i in range(e2e_steps):
            it2 = B.from_workload(w_rank, math=math, max_cells_per_level=cap, spread=spread, budget_order=order)   # host bounds + params -> zmc_create / zmc_set_integrand
            it2.use_torch_workspace()
            it2.run(stream.cuda_stream)                                         # parameters H2D + every kernel
            it2.result()                                                         # D2H of (value, std) per instance + overflow flag
            ev += evals_step
            it2.close()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        npar = 0 if w.params is None else int(np.asarray(w.params).size)
        line["e2e"] = {"value": ev / dt, "unit": UNIT, "h2d_bytes_per_step": 16 * w.dim + 12 * npar,
                       "d2h_bytes_per_step": 16 * w.n_instances + 4, "ms_per_step": 1e3 * dt / e2e_steps,
                       "what": "zmc_create + zmc_set_integrand + zmc_set_option + zmc_set_workspace + zmc_run + zmc_result + zmc_destroy per step, host arrays in, host doubles out"}

        if world == 1 and not args.no_extra:
            # BASELINE.json metric: "time-to-result at 6-D and 9-D" -- one whole tree search each, device time from zmc_stats
            # (first kernel to last kernel), after one untimed run of the same context
            line["time_to_result"] = {args.workload: {"ms": ms_per_step, "value": float(value_v[0]), "std": float(value_s[0])}}
            extra = ["cfg3_gauss9d",            # configs[2] whole, the paper's rule
                     "cfg2_sin6d_depth2",       # configs[1] under the paper's rule (no budget), levels 1-2 of 3 (~2.4 s)
                     "cfg5_sin6d_depth4_B1",    # configs[4] to depth 4 with one refined cell per level (~8 s)
                     "paper_t3_sin6d",          # the paper's own parameter sets (context: 38.7 s, 4.8 s and 47.6 s on one V100,
                     "paper_t4_gauss9d",        #  other hardware, other stack)
                     "cfg12_gauss12d"]
            for name in extra:
                if name == args.workload:
                    continue
                wx = wl[name]
                itx = B.from_workload(wx, math=math, max_cells_per_level=capacity_for(wx))
                n_warm = 2 if wx.name == "cfg3_gauss9d" else 0       # the long ones are their own warm-up: same kernel as the timed steps above
                for _ in range(n_warm + 1):
                    itx.run(stream.cuda_stream)
                vx, sx = itx.result()
                stx = itx.stats()
                line["time_to_result"][name] = {
                    "ms": stx.total_ms, "value": float(vx[0]), "std": float(sx[0]), "evals": int(stx.total_evals),
                    "evals_per_s": stx.total_evals / (stx.total_ms * 1e-3),
                    "cells_per_level": [int(stx.level[l].n_cells) for l in range(stx.levels)],
                    "flagged_per_level": [int(stx.level[l].n_flagged) for l in range(stx.levels)],
                    "refined_per_level": [int(stx.level[l].n_refined) for l in range(stx.levels)],
                    "deviation": DEVIATIONS.get(name)}
                if name in PAPER_SECONDS:
                    line["time_to_result"][name]["paper_seconds_on_one_V100"] = PAPER_SECONDS[name]
                itx.close()
            # BASELINE.json configs[0] is launch-bound (microseconds of arithmetic): kernel by kernel vs one CUDA graph
            w1 = wl["cfg1_sin3d_f64"]
            # ... vs one cooperative launch for the whole tree (ZMC_OPT_SINGLE_LAUNCH; the default for a problem this small)
            for key, graph, single in (("cfg1_sin3d_f64", False, None), ("cfg1_sin3d_f64_multi_launch", False, 0), ("cfg1_sin3d_f64_graph", True, 0)):
                it1 = B.from_workload(w1, math=math, max_cells_per_level=capacity_for(w1), use_graph=graph, single_launch=single)
                for _ in range(3):
                    it1.run(stream.cuda_stream)
                it1.result()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record(stream)
                for _ in range(20):
                    it1.run(stream.cuda_stream)
                g1.record(stream)
                v1, s1 = it1.result()
                line["time_to_result"][key] = {"ms": g0.elapsed_time(g1) / 20, "value": float(v1[0]), "std": float(s1[0]),
                                               "kernel_launches": int(it1.stats().kernel_launches)}
                it1.close()
            # SURVEY 8(f).4 / DESIGN.md R15: a vector-valued user integrand (NVRTC) -- C components from ONE sample stream, against C = 1
            wv = W.vec_moments6d()
            line["vector_valued"] = {"workload": wv.name, "note": wv.note}
            for C_ in (1, 8):
                itv = B.Integrator(wv.dim, wv.lower, wv.upper, wv.g, wv.n_samples, wv.trials, wv.depth, wv.sigma_multiplier, wv.seed)
                itv.set_option(B.OPT_PRECISION, B.F32)
                itv.set_integrand_source_vec(W.VEC_MOMENTS_SRC, W.VEC_MOMENTS_FN, C_, wv.params, 1)
                itv.set_option(B.OPT_MAX_CELLS_PER_LEVEL, wv.k)
                for _ in range(2):
                    itv.run(stream.cuda_stream)
                vv, sv = itv.result()
                stv = itv.stats()
                line["vector_valued"]["C%d" % C_] = {"ms": stv.total_ms, "points_per_s": stv.total_evals / (stv.total_ms * 1e-3),
                                                     "component_evals_per_s": C_ * stv.total_evals / (stv.total_ms * 1e-3),
                                                     "value0": float(vv[0][0]), "std0": float(sv[0][0])}
                itv.close()

        if world == 1 and not args.no_cpu_baseline:
            units = max(1, int(2.0e8 // w.n_samples))
            ev_c, sec_c = oracle_sample(w, units)
            line["cpu_baseline"] = {"value": ev_c / sec_c, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": "%d (cell,trial) units of level 1 of %s, %d samples each, single thread, %.1f s" %
                                              (units, args.workload, w.n_samples, sec_c)}
        if all_cores is not None:
            line["cpu_baseline_all_cores"] = all_cores
        print(json.dumps(line), flush=True)
    it.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
