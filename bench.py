"""bench.py -- BASELINE.json's metric on a B200: edges/s of one Allegro tensor-product layer, forward + force VJP
(fp32, l_max = 2, n = 64) on BASELINE.json:configs[1] (4,096 atoms, ~370k directed edges), seeded synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C1|C1s|C4|C3m]
    torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...     (one rank per GPU)

A "step" is one pass of the whole hot path (all rows) over one system: radial weights -> Y_lm +
environment embedding -> tensor product -> edge energy / cotangent -> tensor-product VJP (gV, gEenv) ->
embedding VJP -> radial chain rule -> force gather -> energy sum.  Every step runs in the library's CUDA kernels.

One JSON line on stdout (rank 0).  `value` = device-timed (CUDA events) edges/s with inputs resident in HBM;
`e2e` = the same step called with HOST buffers (pinned): H2D of the step's inputs and D2H of forces + energy are
inside the timed region; `roofline` = the dominant kernel's algorithmic bytes / its CUDA-event time over the
timed steps, against MEASURED_PEAKS.json; `cpu_baseline` = the float64 oracle timed on the host cores on a
bounded sample of the same workload.  --impl reference times the oracle alone (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
for _p in (ROOT, os.path.join(ROOT, "tests")):
    if _p not in sys.path:
        sys.path.insert(0, _p)

METRIC = "edges/s for Allegro TP fwd+force-VJP (fp32, l_max=2, n=64)"
UNIT = "edges/s"
FALLBACK_HBM_GBS = 6650.0     # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C1")
    ap.add_argument("--force-only", action="store_true", help="skip dE/dV (valid when V does not depend on positions)")
    ap.add_argument("--mode", default="auto", choices=["auto", "separate", "epilogue", "onthefly", "fused"],
                    help="call sequence (pipeline.SingleLayerStep); auto = fused (one kernel for forward + energy + VJP) for l_max <= 2, onthefly for l_max = 3")
    ap.add_argument("--separate-geometry", action="store_true", help="radial / env-embed as four kernels instead of the two fused ones")
    ap.add_argument("--chunks", type=int, default=1, help="process the centres in this many chunks (C3 defaults to 16)")
    ap.add_argument("--no-graph", action="store_true", help="time the eager call sequence instead of CUDA-graph replays of the step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--replicas", action="store_true", help="N > 1: one independent system per rank (weak scaling) instead of one sharded system")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--dense-tp", action="store_true",
                    help="side bench: allegro_tp_forward + allegro_tp_backward alone with DENSE per-path weights on the workload's graph, l_max and n "
                         "(e.g. --workload C3m: the l_max = 3, n = 128 shape of Table 1's large model); not the headline metric")
    ap.add_argument("--dense-edges", type=int, default=200000, help="--dense-tp: leading centres covering about this many edges")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ oracle arm
def _oracle_range(inp, c0, c1):
    """One oracle step (the chain of tests/_chain.oracle_chain without forces) on centres [c0, c1) with their complete
    neighbourhoods (exact sub-problem: every per-edge / per-centre quantity depends on one centre).  -> (edges, seconds)"""
    import _chain
    from workloads.inputs import sub_inputs
    sub = sub_inputs(inp, c0, c1)
    t0 = time.perf_counter()
    _chain.oracle_chain(sub, want_gw=False, forces=False)
    return sub["E"], time.perf_counter() - t0


def _oracle_sample_step(inp, n_centres):
    return _oracle_range(inp, 0, n_centres)


def _oracle_all_cores(inp, n_centres, cores):
    """the same single-threaded oracle over `cores` disjoint centre ranges at once (the C++ oracle runs outside the GIL)
    -> (edges, wall seconds)"""
    import concurrent.futures as cf
    from workloads.inputs import sub_inputs
    bounds = [n_centres * k // cores for k in range(cores + 1)]
    ranges = [(a, b) for a, b in zip(bounds[:-1], bounds[1:]) if b > a]
    subs = [sub_inputs(inp, a, b) for a, b in ranges]          # slicing is not part of the timed work
    import _chain
    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(max_workers=len(subs)) as ex:
        list(ex.map(lambda sb: _chain.oracle_chain(sb, want_gw=False, forces=False), subs))
    return sum(sb["E"] for sb in subs), time.perf_counter() - t0, len(subs)


def cpu_baseline(inp, seconds):
    """The float64 oracle, as it stands, on a bounded sample of the workload: calibrate on 4 centres, one single-threaded leg
    of about seconds / 2, then the same function on all host cores (sched_getaffinity) over disjoint centre ranges."""
    N = inp["N"]
    e_cal, t_cal = _oracle_sample_step(inp, min(4, N))
    rate = e_cal / max(t_cal, 1e-9)
    deg = inp["E"] / max(N, 1)
    nc = int(max(4, min(N, rate * 0.5 * seconds / deg)))
    e1, t1 = _oracle_sample_step(inp, nc)
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    nca = int(max(cores, min(N, nc * cores)))
    ea, ta, used = _oracle_all_cores(inp, nca, cores)
    return {"value": ea / ta, "unit": UNIT, "cores": used, "kind": "oracle", "value_1core": e1 / t1,
            "sample": "float64 C++ oracle chain (radial, env-embed, TP fwd, energy, TP VJP, env VJP; no force gather): all-cores leg on the "
                      "first %d centres = %d edges of %s split into %d ranges, %.1f s wall; single-thread leg on the first %d centres = %d "
                      "edges, %.1f s" % (nca, ea, inp["name"], used, ta, nc, e1, t1)}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    from workloads.inputs import make_inputs
    name = args.workload
    inp = make_inputs(name, features="lazy")
    steps = max(1, args.steps)
    per_step = max(0.5, min(10.0, 120.0 / (steps + args.warmup)))     # wall seconds of oracle work per step
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    e_cal, t_cal = _oracle_sample_step(inp, 4)
    nc = int(max(cores, min(inp["N"], cores * (e_cal / t_cal) * per_step / (inp["E"] / inp["N"]))))
    for _ in range(args.warmup):
        _oracle_all_cores(inp, nc, cores)
    tot_e, tot_t, used = 0, 0.0, cores
    for _ in range(steps):
        e, t, used = _oracle_all_cores(inp, nc, cores)
        tot_e += e
        tot_t += t
    v = tot_e / tot_t
    sample = "first %d centres (%d edges) of %s per step split into %d ranges, float64 C++ oracle, one thread per range" % (nc, tot_e // steps, name, used)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * tot_t / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": name, "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------ CUDA arm
def _dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank, world, local = _dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import ChunkedStep, HostStep, SingleLayerStep, to_device
    from workloads.inputs import make_inputs

    name = args.workload
    if name in ("C2", "C2s"):
        return run_two_layer(args, rank, world, local, dist, barrier_factory=None)
    # multi-GPU: ONE system (seed 0) sharded by centre atom over the ranks -- every rank runs the kernels on its own CSR
    # rows, the only exchange is the halo of cut-edge g_r rows before the owners gather their forces (sharding.py): strong scaling.
    # --replicas: rank r owns the independent system of seed r instead (no data-path collective, weak scaling); C3 (chunked) always.
    sharded = world > 1 and not args.replicas and name != "C3" and args.chunks <= 1
    inp = make_inputs(name, seed=0 if sharded else rank, features="device")
    plan = ab.Plan(inp["lmax"], inp["n"], ab.F64 if inp["dt"] == np.float64 else ab.F32, ab.W_SCALAR)
    sh = None
    if sharded:
        from paper_2504_16068_b200.pipeline import shard_to_device
        from paper_2504_16068_b200.sharding import ShardedForces
        sh = ShardedForces(inp["row_ptr"], inp["rev"], device="cuda", dtype=plan.tdtype)
        dev = shard_to_device(inp, sh)
        args.no_graph = True          # the halo exchange (NCCL send / recv) stays outside a captured graph
    else:
        dev = to_device(inp)
    if args.mode == "auto":      # at l_max = 3 the fused kernel needs 168 registers for one CTA of 8 warps per SM and is slower than the two kernels
        args.mode = "fused" if inp["lmax"] <= 2 else "onthefly"
    chunked = name == "C3" or args.chunks > 1
    if chunked:      # feature tensors that do not fit HBM four times: V resident, work buffers per centre chunk
        step = ChunkedStep(plan, dev, inp["row_ptr"], inp["rc"], inp["kappa"], inp["scale"], n_chunks=max(args.chunks, 16 if name == "C3" else 1), fused=args.mode == "fused",
                           want_gV=not args.force_only)
    else:
        step = SingleLayerStep(plan, dev, inp["rc"], inp["kappa"], inp["scale"], want_gV=not args.force_only, mode=args.mode,
                               fused_geometry=not args.separate_geometry, sharded=sh)
    E, N = step.E, step.N

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing: the step is captured once into a CUDA graph and replayed K times (--no-graph:
    # the eager call sequence).  Per-call times for the roofline come from a second, marked eager pass of K steps.
    for _ in range(max(args.warmup, 3)):
        step.run()
    barrier()
    runner = step
    lib_graph = False
    if not args.no_graph:
        # the library's own step object runs the fused kernel at l_max <= 2 and the two-kernel sequence at l_max = 3: it is the runner
        # only when that is the mode asked for, so that the timed steps and the per-call roofline pass run the same kernels
        lib_mode = "fused" if inp["lmax"] <= 2 else "onthefly"
        if not chunked and args.mode == lib_mode and not args.separate_geometry:
            # the graph is captured INSIDE the library (allegro_layer_step_create): one C-ABI call per MD step, no framework graph
            runner = ab.LayerStepGraph(plan, dev["row_ptr"], dev["rev"], dev["rvec"], dev["V"], dev["W_r"], inp["rc"], dev["q"], inp["kappa"], inp["scale"],
                                       step.F, step.e_tot, want_gV=not args.force_only)
            lib_graph = True
        else:
            from paper_2504_16068_b200.pipeline import GraphedStep
            runner = GraphedStep(step, warmup=1)
        for _ in range(3):
            runner.run()
        barrier()
    clocks = ClockSampler(local)
    clocks.start()
    n0 = ab.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        runner.run()
    ev1.record()
    barrier()
    launches = (runner.kernels_per_step * args.steps) if not args.no_graph else (ab.launch_count() - n0)
    ms_total = ev0.elapsed_time(ev1)
    marks = []
    for _ in range(args.steps):
        step.run(mark=True)
        marks.append(step.marks)
    barrier()
    clk = clocks.stop()
    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    tot = torch.tensor([float(E), float(N)], dtype=torch.float64, device="cuda")     # rank-local edges / atoms: the sum is the whole job
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    E_all, N_all = float(tot[0].item()), float(tot[1].item())
    value = E_all / (ms_step * 1e-3)

    # per-call device time (CUDA events on the launching stream, same timed region)
    per_call = {}
    for mk in marks:          # one list per step; a chunked step has several entries per name: summed per step
        tot = {}
        for nm, a, b in mk:
            tot[nm] = tot.get(nm, 0.0) + a.elapsed_time(b)
        for nm, v in tot.items():
            per_call.setdefault(nm, []).append(v)
    per_call_ms = {k: sum(v) / len(v) for k, v in per_call.items()}
    abytes = step.algorithmic_bytes()
    peak, peak_src = measured_peaks()
    top = max(per_call_ms, key=per_call_ms.get)
    ach = abytes[top] / (per_call_ms[top] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": top, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": _ncu_traffic(name, top) if (args.mode in ("onthefly", "fused") and not args.force_only) else None,
                "traffic_source": "committed ncu --set full capture, profiles/traffic.txt (not re-measured by this run)",
                "peak_source": peak_src, "algorithmic_bytes_per_launch": abytes[top], "ms_per_launch": per_call_ms[top],
                "timing": "eager pass of the same %d steps with CUDA events around every call, run right after the timed graph replays "
                          "(a replay cannot be split per kernel); the calls' sum can exceed ms_per_step by the launch gaps" % args.steps}
    peaks = ab.measure_peaks()
    peaks["hbm_gbs"] = peak
    # FP32 instruction roofline of the sparse CG contraction: FMA + MUL instructions per channel-edge of the generated
    # code (forward nnz + pairs, VJP nnz + 2 pairs) against the FMA-pipe instruction rate measured in this run (fp32 only;
    # nominal: 148 SMs x 128 lanes x 1.965 GHz = 37.2 T lane-instructions/s)
    nnz, pairs = {1: (32, 32), 2: (274, 258), 3: (1222, 1082)}[inp["lmax"]]
    per_ce = {"tp_forward_energy": nnz + pairs, "tp_forward": nnz + pairs, "tp_backward_energy": nnz + 2 * pairs, "tp_backward": nnz + 2 * pairs,
              "tp_fused_energy": (nnz + pairs) + (nnz + 2 * pairs)}
    instr_edge = ((nnz + pairs) + (nnz + 2 * pairs)) * inp["n"]
    alu = None
    if inp["dt"] == np.float32:
        rate = peaks["fp32_fma_tflops"] * 1e12 / 2.0
        src = "measured in this run (allegro_measure_fp32_fma_peak: %.1f TFLOP/s = 2 flops per FFMA)" % peaks["fp32_fma_tflops"]
        alu = {"bound": "alu", "achieved": instr_edge * E_all / world / (ms_step * 1e-3), "peak": rate, "unit": "FP32 lane-instructions/s per GPU",
               "frac": instr_edge * E_all / world / (ms_step * 1e-3) / rate, "instructions_per_edge": instr_edge, "scope": "whole step", "peak_source": src}
        if top in per_ce:
            k_ach = per_ce[top] * inp["n"] * E / (per_call_ms[top] * 1e-3)
            alu["kernel"] = {"name": top, "achieved": k_ach, "frac": k_ach / rate, "instructions_per_channel_edge": per_ce[top]}
    # Which roof binds the dominant kernel follows from its arithmetic: algorithmic instructions / measured FMA rate against algorithmic
    # bytes / measured HBM bandwidth.  The fused kernel (2.5x fewer bytes than the two kernels it replaces) and the l_max = 3 kernels
    # (3,386 instructions per 384 bytes in the VJP) are instruction-bound: their line reports the ALU roofline as `roofline` and
    # keeps the HBM figures under `hbm_roofline`; the two-kernel sequence at l_max <= 2 is HBM-bound.
    hbm_roofline = None
    alu_binds = (alu is not None and "kernel" in alu and
                 per_ce[top] * inp["n"] * E / rate > abytes[top] / (peak * 1e9))
    if alu_binds:
        hbm_roofline = roofline
        roofline = {"bound": "alu", "kernel": top, "achieved": alu["kernel"]["achieved"] / 1e12, "peak": rate / 1e12, "unit": "T FP32 instructions/s",
                    "frac": alu["kernel"]["frac"], "traffic": hbm_roofline["traffic"], "traffic_source": hbm_roofline["traffic_source"],
                    "peak_source": src, "algorithmic_instructions_per_launch": per_ce[top] * inp["n"] * E, "ms_per_launch": per_call_ms[top],
                    "timing": hbm_roofline["timing"],
                    "note": "algorithmic FMA + MUL instructions of the sparse CG contraction / CUDA-event time; at the measured rates this "
                            "kernel's instruction time exceeds its HBM time, so the ALU roof binds; its HBM fraction is under hbm_roofline"}
    # forward only (configs[1]: "forward only, then forward+force VJP")
    fwd = None
    if not chunked:
        for _ in range(3):
            step.run_forward()
        barrier()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        for _ in range(args.steps):
            step.run_forward()
        f1.record()
        barrier()
        fms = f0.elapsed_time(f1) / args.steps
        fwd = {"ms_per_step": fms, "edges_per_s": E / (fms * 1e-3), "GBps_algorithmic": step.forward_bytes() / (fms * 1e-3) / 1e9,
               "frac_of_hbm_peak": step.forward_bytes() / (fms * 1e-3) / 1e9 / peak, "launch": "eager"}
    step_bytes = sum(abytes[k] for k in per_call_ms)
    calls = {k: {"ms": round(per_call_ms[k], 4), "GB/s": round(abytes[k] / (per_call_ms[k] * 1e-3) / 1e9, 1),
                 "share": round(per_call_ms[k] / sum(per_call_ms.values()), 4)} for k in per_call_ms}

    # ---------------- end to end: host buffers in, forces + energy out, copies inside the timed region
    e2e_md = None
    if chunked:
        e2e = None      # the host copy of V alone (86 GB at C3) does not fit pinned memory on the box: no end-to-end arm
    else:
        host = None if sharded else HostStep(step, inp)     # the one-call host entry point is single-GPU
        k_e2e = max(3, min(args.steps, 10))
        e2e_ms = float("nan")
        if host is not None:
            for _ in range(3):
                host.run()
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(k_e2e):
                host.run()
            e1.record()
            barrier()
            t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
            if world > 1:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_ms = float(t.item()) / k_e2e
        e2e = None if host is None else {"value": E_all / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": host.h2d_bytes, "d2h_bytes_per_step": host.d2h_bytes,
                                         "ms_per_step": e2e_ms, "steps": k_e2e,
               "note": "allegro_layer_step_host: EVERY input of the step, the %.2f GB feature tensor V included, is copied from pinned host memory each "
                       "step (PCIe-bound); e2e_md is the MD-shaped variant" % (E * inp["n"] * plan.dV * (4 if inp["dt"] == np.float32 else 8) / 1e9)}
        # MD-shaped end to end: positions (edge vectors) in, forces + energy out, features and weights resident
        h_rvec = torch.empty(dev["rvec"].shape, dtype=dev["rvec"].dtype, pin_memory=True).copy_(dev["rvec"])
        h_F = torch.empty(step.F.shape, dtype=step.F.dtype, pin_memory=True)
        h_e = torch.empty(step.e_tot.shape, dtype=step.e_tot.dtype, pin_memory=True)

        def md_step():
            dev["rvec"].copy_(h_rvec, non_blocking=True)
            runner.run()
            h_F.copy_(step.F, non_blocking=True)
            h_e.copy_(step.e_tot, non_blocking=True)
            torch.cuda.current_stream().synchronize()

        for _ in range(3):
            md_step()
        barrier()
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        m0.record()
        for _ in range(args.steps):
            md_step()
        m1.record()
        barrier()
        t = torch.tensor([m0.elapsed_time(m1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        md_ms = float(t.item()) / args.steps
        e2e_md = {"value": E_all / (md_ms * 1e-3), "unit": UNIT, "ms_per_step": md_ms, "steps": args.steps,
                  "h2d_bytes_per_step": int(h_rvec.numel() * h_rvec.element_size()),
                  "d2h_bytes_per_step": int(h_F.numel() * h_F.element_size() + h_e.numel() * h_e.element_size()),
                  "note": "edge vectors in from pinned host memory, forces and total energy out, host synchronised every step"}
        if sharded:      # the end-to-end arm of a sharded run is the MD-shaped one (every rank: its edge vectors in, its atoms' forces out)
            e2e, e2e_md = e2e_md, None

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f32" if inp["dt"] == np.float32 else "f64", "data": "synthetic",
            "config": {"workload": "%s: BASELINE.json configs recipe, %d atoms, %d directed edges %s, l_max=%d, n=%d, "
                                   "single TP layer forward + %s" % (name, int(N_all) if sharded else N, int(E_all) if sharded else E,
                                                                     "in ONE system sharded over the GPUs" if sharded else "per GPU", inp["lmax"], inp["n"],
                                                                     "force-only VJP" if args.force_only else "full VJP (gV, gEenv) + forces"),
                       "atoms": int(N_all) if sharded else N, "edges": int(E_all) if sharded else E, "l_max": inp["lmax"], "n_channels": inp["n"],
                       "parallelism": ("centres of one system sharded over %d GPUs, halo exchange of %d bytes of cut-edge g_r per step from rank 0"
                                       % (world, sh.halo_bytes)) if sharded else "independent systems per GPU", "mode": args.mode,
                       "l2": "not flushed: every feature tensor (%.2f GB) exceeds the 126 MB L2" % (E * inp["n"] * plan.dV * (4 if inp["dt"] == np.float32 else 8) / 1e9),
                       "fused_geometry": not args.separate_geometry},
            "atom_steps_per_s": N_all / (ms_step * 1e-3),
            "step_GBps_algorithmic": step_bytes / (ms_step * 1e-3) / 1e9, "step_frac_of_hbm_peak": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
            "roofline": roofline, "hbm_roofline": hbm_roofline, "alu_roofline": alu, "calls": calls, "clocks": clk, "e2e": e2e, "e2e_md": e2e_md, "forward_only": fwd, "peaks": peaks,
            "gpu_launches": int(launches),
        }
        line["config"]["launch"] = ("eager call sequence" if args.no_graph else
                                    ("one allegro_layer_step_launch per step: CUDA graph captured inside the library (%d kernels per step)" if lib_graph
                                     else "CUDA graph replay of the step (%d kernels per step)") % runner.kernels_per_step)
        if world == 1 and not args.no_cpu_baseline:
            import oracle
            oracle.build()
            line["cpu_baseline"] = cpu_baseline(inp, args.cpu_seconds)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_two_layer(args, rank, world, local, dist, barrier_factory=None):
    """--workload C2: BASELINE.json:configs[2], two stacked layers with the dense per-path mix, forward + force backward as one MD
    step.  The dominant calls (dense tensor product forward / VJP) are tensor-core bound work: "bound": "tensor"."""
    import numpy as np
    import torch

    import paper_2504_16068_b200 as ab
    from paper_2504_16068_b200.pipeline import TwoLayerStep
    from workloads.inputs import make_model_inputs
    name = args.workload
    sharded = world > 1 and not args.replicas      # one system, centres sharded over the ranks (strong scaling); see run_ours
    inp = make_model_inputs(name, seed=0 if sharded else rank)
    p = inp["params"]
    td = torch.float32 if inp["dt"] == np.float32 else torch.float64
    sh = None
    if sharded:
        from paper_2504_16068_b200.pipeline import shard_to_device
        from paper_2504_16068_b200.sharding import ShardedForces
        sh = ShardedForces(inp["row_ptr"], inp["rev"], device="cuda", dtype=td)
        dev = shard_to_device(inp, sh, keys_edge=("rvec",), keys_full=())
    else:
        dev = {k: torch.from_numpy(np.ascontiguousarray(inp[k])).cuda() for k in ("row_ptr", "rev", "rvec")}
    prm = {k: torch.from_numpy(np.ascontiguousarray(p[k])).to(td).cuda() for k in ("W_x0", "W_v0", "W_w", "W_p", "A_lat", "q")}
    prm.update(rc=p["rc"], scale=p["scale"])
    dt = ab.F32 if inp["dt"] == np.float32 else ab.F64
    # last layer: its output feeds only the readout of the l = 0 outputs (configs[2]), so the plan is restricted to the 0e block
    plan_last = ab.Plan(p["lmax"], p["n"], dt, ab.W_DENSE)
    plan_last.set_out_blocks(0x1)
    # first layer: V0 = v (x) Y(rhat) has the natural-parity blocks only (reading A19), the paths from the other blocks never run
    plan_first = ab.Plan(p["lmax"], p["n"], dt, ab.W_DENSE)
    plan_first.set_in_blocks(0x19)
    step = TwoLayerStep(ab.Plan(p["lmax"], p["n"], dt, ab.W_DENSE), ab.Plan(p["lmax"], p["n"], dt, ab.W_SCALAR), dev, prm, plan_last=plan_last,
                        plan_first=plan_first, sharded=sh)
    E, N = step.E, step.N
    tot = torch.tensor([float(E), float(N)], dtype=torch.float64, device="cuda")     # rank-local edges / atoms: the sum is the whole job
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    E_all, N_all = float(tot[0].item()), float(tot[1].item())

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step.run()
    barrier()
    clocks = ClockSampler(local)
    clocks.start()
    n0 = ab.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    marks = []
    ev0.record()
    for _ in range(args.steps):
        step.run(mark=True)
        marks.append(step.marks)
    ev1.record()
    barrier()
    launches = ab.launch_count() - n0
    clk = clocks.stop()
    t = torch.tensor([ev0.elapsed_time(ev1)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    per_call = {}
    for mk in marks:
        tot = {}
        for nm, a, b in mk:
            tot[nm] = tot.get(nm, 0.0) + a.elapsed_time(b)
        for nm, v in tot.items():
            per_call.setdefault(nm, []).append(v)
    per_call_ms = {k: sum(v) / len(v) for k, v in per_call.items()}
    flops = step.algorithmic_flops()
    top = max(per_call_ms, key=per_call_ms.get)
    # The dense per-path mix runs on the tensor cores (tcgen05.mma kind::tf32, fp32 operands split hi / lo, four products per
    # multiply-add).  Tensor roofline: the TF32 tcgen05 rate measured in this run (M 128, N 256, one CTA per SM); `achieved`
    # counts ALGORITHMIC fp32 flops (one multiply-add per weight element and column), not the four TF32 MMAs each of them costs.
    peaks = ab.measure_peaks()
    hbm_peak, hbm_src = measured_peaks()
    peaks["hbm_gbs"] = hbm_peak
    peak, peak_src = peaks["tf32_mma_tflops"], "measured in this run: tcgen05.mma kind::tf32, M 128 x N 256 x K 8, one CTA per SM (allegro_measure_tf32_mma_peak)"
    abytes = step.algorithmic_bytes()
    tp_ms = per_call_ms.get("tp_forward_dense", 0.0) + per_call_ms.get("tp_backward_dense", 0.0)
    tp_bytes = abytes["tp_forward_dense"] + abytes["tp_backward_dense"]
    ach = flops.get(top, 0) / (per_call_ms[top] * 1e-3) / 1e12
    # end to end: rvec (the positions) in from pinned host memory, forces and energy out, every step
    h_rvec = torch.empty(dev["rvec"].shape, dtype=dev["rvec"].dtype, pin_memory=True).copy_(dev["rvec"])
    h_F = torch.empty(step.F.shape, dtype=step.F.dtype, pin_memory=True)
    h_e = torch.empty(step.e_tot.shape, dtype=step.e_tot.dtype, pin_memory=True)

    def host_step():
        dev["rvec"].copy_(h_rvec, non_blocking=True)
        step.run()
        h_F.copy_(step.F, non_blocking=True)
        h_e.copy_(step.e_tot, non_blocking=True)
        torch.cuda.current_stream().synchronize()

    host_step()
    barrier()
    k_e2e = max(2, min(args.steps, 5))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(k_e2e):
        host_step()
    e1.record()
    barrier()
    e2e_ms = e0.elapsed_time(e1) / k_e2e
    if rank == 0:
        line = {
            "metric": METRIC, "value": E_all / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f32" if inp["dt"] == np.float32 else "f64",
            "data": "synthetic",
            "config": {"workload": "%s: BASELINE.json configs[2] recipe, %d atoms, %d directed edges per GPU, l_max=%d, n=%d, %d layers with dense "
                                   "per-path mix, forward + force backward as one MD step" % (name, N, E, p["lmax"], p["n"], p["n_layers"]),
                       "atoms": int(N_all) if sharded else N, "edges": int(E_all) if sharded else E,
                       "parallelism": ("centres of one system sharded over %d GPUs, halo exchange of cut-edge g_r" % world) if sharded else "independent systems per GPU",
                       "block_subsets": "first layer: paths from the natural-parity blocks of V0 only (15 of 30); last layer: paths into 0e only (3 of 30)",
                       "l2": "not flushed: feature tensors (%.2f GB each) exceed the 126 MB L2" % (E * p["n"] * step.pd.dV * 4 / 1e9)},
            "atom_steps_per_s": N_all / (ms_step * 1e-3),
            "roofline": {"bound": "tensor", "kernel": top, "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                         "traffic": _ncu_traffic(name, top), "traffic_source": "committed ncu --set full capture, profiles/traffic.txt: dram bytes of "
                                                                               "both layers' launches of this call per step (not re-measured by this run)",
                         "peak_source": peak_src, "note": "algorithmic fp32 flops of all layers' calls of this name; every multiply-add costs four TF32 MMAs "
                                                          "(hi / lo split of both operands) on tcgen05",
                         "timing": "CUDA events around every call inside the timed steps"},
            # reading A15 holds the tensor-product part of C2 to the HBM roofline as well: bytes the dense TP calls must move / their time
            "tp_hbm_roofline": {"bound": "hbm", "calls": ["tp_forward_dense", "tp_backward_dense"], "algorithmic_bytes_per_step": tp_bytes,
                                "ms_per_step": tp_ms, "achieved": tp_bytes / (tp_ms * 1e-3) / 1e9 if tp_ms > 0 else None, "peak": hbm_peak, "unit": "GB/s",
                                "frac": tp_bytes / (tp_ms * 1e-3) / 1e9 / hbm_peak if tp_ms > 0 else None, "peak_source": hbm_src},
            "peaks": peaks,
            "calls": {k: {"ms": round(v, 4), "share": round(v / sum(per_call_ms.values()), 4)} for k, v in per_call_ms.items()},
            "clocks": clk,
            "e2e": {"value": E_all / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h_rvec.numel() * h_rvec.element_size()),
                    "d2h_bytes_per_step": int(h_F.numel() * h_F.element_size() + h_e.numel() * h_e.element_size()), "ms_per_step": e2e_ms, "steps": k_e2e},
            "gpu_launches": int(launches),
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_dense_tp(args):
    """Side bench (a4): the dense per-path channel mix alone -- tp_forward + tp_backward (gV, gEenv) with W_p[n, n]
    per path -- on the leading centres of the workload's graph.  One JSON line; flops = 2 n^2 sum_p (2 l3 + 1) per edge and pass."""
    import numpy as np
    import torch

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    import paper_2504_16068_b200 as ab
    from workloads import configs
    g = configs.geometry_for(args.workload)
    spec = g["spec"]
    lmax, n = spec["lmax"], spec["n"]
    dt = ab.F64 if spec["dtype"] == "f64" else ab.F32
    rp = g["row_ptr"]
    c = int(np.searchsorted(rp, min(args.dense_edges, int(rp[-1]))))
    c = max(1, min(c, rp.shape[0] - 1))
    E = int(rp[c])
    plan = ab.Plan(lmax, n, dt, ab.W_DENSE)
    td = plan.tdtype
    gen = torch.Generator(device="cuda").manual_seed(0)
    rnd = lambda *sh: torch.randn(*sh, generator=gen, device="cuda", dtype=td)
    rpd = torch.from_numpy(np.ascontiguousarray(rp[:c + 1])).cuda()
    V, G, Ee, W = rnd(E, n, plan.dV), rnd(E, n, plan.dV), rnd(c, n, plan.dE) * 0.5, rnd(plan.P, n, n) / n ** 0.5
    items = torch.from_numpy(ab.segments_build(rp[:c + 1], 32)).cuda()
    out, gV, gE = torch.empty_like(V), torch.empty_like(V), torch.empty_like(Ee)

    def step():
        ab.tp_forward(plan, rpd, V, Ee, W, out=out, items=items)
        ab.tp_backward(plan, rpd, G, V, Ee, W, gV=gV, gEenv=gE, items=items)
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    clocks = ClockSampler(0)
    clocks.start()
    n0 = ab.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    tf = tb = 0.0
    for _ in range(args.steps):
        ev[0].record()
        ab.tp_forward(plan, rpd, V, Ee, W, out=out, items=items)
        ev[1].record()
        ab.tp_backward(plan, rpd, G, V, Ee, W, gV=gV, gEenv=gE, items=items)
        ev[2].record()
        torch.cuda.synchronize()
        tf += ev[0].elapsed_time(ev[1])
        tb += ev[1].elapsed_time(ev[2])
    launches = ab.launch_count() - n0
    clk = clocks.stop()
    tf, tb = tf / args.steps, tb / args.steps
    pt = plan.paths()
    dT = int(sum(2 * int(l3) + 1 for l3 in pt["l3"]))
    flops = 2.0 * n * n * dT * E
    peaks = ab.measure_peaks()
    tc = lmax == 2 and n == 64 and dt == ab.F32
    peak = peaks["tf32_mma_tflops"] if tc else peaks["fp32_fma_tflops"]
    top, ttop = ("tp_backward_dense", tb) if tb >= tf else ("tp_forward_dense", tf)
    ach = flops / (ttop * 1e-3) / 1e12
    line = {"metric": "edges/s for the dense per-path mix alone (tp_forward + tp_backward, W_p[n, n] per path)", "value": E / ((tf + tb) * 1e-3),
            "unit": "edges/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": tf + tb, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64" if dt == ab.F64 else "f32", "data": "synthetic",
            "config": {"workload": "%s graph (first %d centres, %d edges), l_max=%d, n=%d, %d paths, dense weights; side bench, not the headline "
                                   "metric" % (args.workload, c, E, lmax, n, plan.P),
                       "l2": "inputs of %.1f GB exceed the 126 MB L2" % (3 * V.numel() * V.element_size() / 1e9)},
            "calls": {"tp_forward_dense": {"ms": tf, "TFLOP/s": flops / (tf * 1e-3) / 1e12}, "tp_backward_dense": {"ms": tb, "TFLOP/s": flops / (tb * 1e-3) / 1e12}},
            "roofline": {"bound": "tensor" if tc else "alu", "kernel": top, "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
                         "peak_source": "measured in this run (%s)" % ("allegro_measure_tf32_mma_peak" if tc else "allegro_measure_fp32_fma_peak"),
                         "note": "algorithmic fp32 flops of the n x n mixes (the CG products before them are not counted)"},
            "peaks": peaks, "clocks": clk, "e2e": None, "gpu_launches": launches}      # e2e: the host-buffer arm belongs to the headline step
    print(json.dumps(line))


def _ncu_traffic(workload, kernel):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/traffic.txt), or None"""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f).get(workload, {}).get(kernel)
    return None


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    elif a.dense_tp:
        run_dense_tp(a)
    else:
        run_ours(a)
