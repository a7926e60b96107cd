#!/usr/bin/env python
"""bench.py -- one JSON line for the driver (contract: the task prompt's section 4).

A "step" is one pass of the whole hot path (rows a0..a5) over config 3's
headline call (BASELINE.json configs[2], the one north_star's target is quoted on): Plummer sphere
N = 2^20 in the synthetic block-time-step state, all 2^20 particles active:
    nb_update_j(active)  ->  nb_predict(t)  ->  nb_force(i_list, eps2)  [gather, pairs, reduce]
`value` = interactions/s (N_i x N per call, self pair counted, 60 flop each; R11) with
all inputs resident in HBM; `e2e` = the same step through the host-buffer entry points of the
C-ABI (pinned host arrays in, host arrays out, copies inside the timed region).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg3|cfg2|cfg4|cfg5|small] [--no-cpu-baseline] [--no-e2e]

N > 1 (torchrun, one rank per GPU): the active list is sharded over the ranks (i-particles are
independent), every rank holds all j; the per-rank results are assembled with one
all_gather (paper_1409_5474_b200/sharding.py).  Total work is fixed: "scaling": "strong".

--impl reference: there is no reference code (the paper ships none); this arm times the fp64
oracle, as it stands, on the host cores, each step a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_INTERACTION = 60.0
# "alu" roofline denominator: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x
# clocks.max.sm 1.965 GHz (B200_PROFILING.md unit counts and clocks) = 74.45 Tflop/s.
FP32_LANES_PER_SM = 128
FFMA2_LANES_PER_CLK_SM = 115.6           # measured packed-FMA rate (profiles/r1_pipe_probes.md)
PREDICT_BYTES_PER_PARTICLE = 152.0     # 104 B read + 48 B written


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=["cfg3", "cfg1", "cfg2", "cfg4", "cfg5", "small"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="also time nb_force alone on every active-subset size of the workload "
                         "(config 3: 1, 1024, 16384, 262144, 2^20) and add it as \"sweep\"")
    ap.add_argument("--blockstep", type=int, default=0, metavar="N",
                    help="instead of the default line: time --steps device block steps (nb_step: "
                         "scheduler + predictor + force + corrector) of a Plummer sphere of N "
                         "particles with individual power-of-two steps")
    ap.add_argument("--fp64", action="store_true",
                    help="run the step with the full-double pair loop (nb_set_precision 1); the roofline "
                         "is then the FP64 pipe (64 lanes per SM per clock)")
    ap.add_argument("--order6", action="store_true",
                    help="run the step with the 6th-order pair loop (nb_set_order 6 + nb_force6: acc, jerk, snap, "
                         "pot; 64 FP32 lane-operations per interaction instead of 33)")
    ap.add_argument("--predict", action="store_true",
                    help="instead of the default line: the Hermite predictor alone against the HBM roofline "
                         "(config 5's N = 2^22 + 11, and N = 2^20 alternating between two contexts)")
    ap.add_argument("--shard", default="i", choices=["i", "j", "jx"],
                    help="multi-GPU decomposition: i = active list sharded, j replicated (default); j = the paper's "
                         "scheme (PAPER.md:55): j sharded, every rank evaluates all active particles by value "
                         "against its slice, one all_reduce of [7][N_i]")
    ap.add_argument("--kick", action="store_true",
                    help="instead of the default line: time nb_force_ext on config 4's two galaxies "
                         "(stars of B by value against galaxy A as j-set), with jerk and acc + pot only")
    ap.add_argument("--steps-bound", type=float, default=-1.0,
                    help="with --blockstep: largest N_i x N the persistent kernel of nb_steps takes itself")
    ap.add_argument("--detail", action="store_true", help="with --blockstep: add the per-step sizes and device times")
    ap.add_argument("--scaling", type=int, default=0, metavar="LOG2MAX",
                    help="the direct-code curve of the paper's Fig. 2: one all-active force evaluation for "
                         "N = 2^10 ... 2^LOG2MAX (23: ~2 minutes)")
    ap.add_argument("--fewi", action="store_true",
                    help="instead of the default line: the force call for a handful of active particles "
                         "(N_i = 1..64 of config 3, N = 2^20), nb_force and nb_force_fused, against the HBM roofline")
    ap.add_argument("--midsize", action="store_true",
                    help="instead of the default line: nb_force for N_i = 256 ... 16400 active particles (full i-tiles, "
                         "and i-tiles plus a few) at N = 2^16, 2^17, 2^20, against the FP32 roofline")
    ap.add_argument("--cpu-seconds", type=float, default=12.0,
                    help="target duration of the cpu_baseline sample")
    return ap.parse_args()


def make_case(name):
    """Returns (case, i_list, t, workload string).  Seeded synthetic input (nbgen, DESIGN.md
    section 5): stands in for the paper's own particle sets, which are not available."""
    import nbgen
    if name == "cfg3":
        c = nbgen.config3()
        return c, c.i_lists[-1], c.t_now, "cfg3_plummer_N1048576_blockstep_all_active"
    if name == "cfg1":
        c = nbgen.config1()
        c.a, c.j = nbgen.mean_field(c.x, c.v)
        return c, c.i_lists[1], 2.0 ** -6, "cfg1_plummer_N1024_all_active"
    if name == "cfg2":
        c = nbgen.config2()
        c.a, c.j = nbgen.mean_field(c.x, c.v)
        return c, c.i_lists[0], c.dt, "cfg2_plummer_N65536_hermite_step"
    if name == "cfg4":
        c = nbgen.config4()
        return c, c.i_lists[0], 0.0, "cfg4_merger_N1048578_all_active"
    if name == "cfg5":
        c = nbgen.config5()
        return c, c.i_lists[0], 0.0, "cfg5_group_N4194315_Ni1048576"
    c = nbgen.config3(n=1 << 14, sizes=(1 << 14,))
    return c, c.i_lists[-1], c.t_now, "small_plummer_N16384_all_active"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = "/tmp/nb_bench_clocks_%d_%d.csv" % (os.getpid(), index)

    def start(self):
        try:
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=self.fh, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        self.proc.terminate()          # the exact PID started above
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.fh.close()
        sm, mx, pw, reasons = [], [], [], set()
        with open(self.path) as f:
            for line in f:
                p = [q.strip() for q in line.split(",")]
                if len(p) < 7:
                    continue
                try:
                    sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
                except ValueError:
                    continue
                for name, val in zip(self.NAMES, p[3:7]):
                    if val == "Active":
                        reasons.add(name)
        try:
            os.remove(self.path)
        except OSError:
            pass
        if not sm:
            return None
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(case, il, t, seconds):
    """Time the oracle, as it stands, on a bounded sample of the workload: the predictor on all N
    (once) and the force on the first `ni_s` entries of the active list against all N j.  ni_s is
    calibrated so that the force leg takes about `seconds`."""
    import numpy as np
    import oracle
    fl = case.flags if case.flags.any() else None
    t0 = time.perf_counter()
    xp, vp = oracle.predict(t, case.x, case.v, case.a, case.j, case.t)
    t_pred = time.perf_counter() - t0
    n = case.n
    ni_c = max(1, min(len(il), (1 << 29) // n))           # calibration: ~5.4e8 pairs
    t0 = time.perf_counter()
    oracle.force(case.m, xp, vp, il[:ni_c], case.eps2, fl)
    rate = ni_c * n / (time.perf_counter() - t0)
    ni_s = int(max(1, min(len(il), rate * seconds / n)))
    t0 = time.perf_counter()
    oracle.force(case.m, xp, vp, il[:ni_s], case.eps2, fl)
    dt = time.perf_counter() - t0
    return {"value": ni_s * n / dt, "unit": "interactions/s", "cores": oracle.threads(),
            "kind": "oracle",
            "sample": "first %d of %d active i against all %d j (%.3g interactions, %.1f s); "
                      "predictor on all j took %.3f s" % (ni_s, len(il), n, ni_s * float(n), dt, t_pred),
            "gflops": ni_s * n / dt * FLOP_PER_INTERACTION / 1e9}


def run_reference(args):
    """--impl reference: the oracle on the host cores (no reference code exists)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np
    import oracle
    case, il, t, workload = make_case(args.workload)
    n = case.n
    fl = case.flags if case.flags.any() else None
    # bounded sample per step: ~1.5 s of force work
    xp, vp = oracle.predict(t, case.x, case.v, case.a, case.j, case.t)
    ni_c = max(1, min(len(il), (1 << 29) // n))
    t0 = time.perf_counter()
    oracle.force(case.m, xp, vp, il[:ni_c], case.eps2, fl)
    rate = ni_c * n / (time.perf_counter() - t0)
    ni_s = int(max(1, min(len(il), rate * 1.5 / n)))
    sub = np.ascontiguousarray(il[:ni_s])

    def step():
        xp, vp = oracle.predict(t, case.x, case.v, case.a, case.j, case.t)
        return oracle.force(case.m, xp, vp, sub, case.eps2, fl)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    val = ni_s * n * args.steps / dt
    sample = "each step: oracle predictor on all %d j + oracle force on the first %d of %d active i" % (
        n, ni_s, len(il))
    line = {
        "impl": "reference", "metric": "interactions/s", "value": val, "unit": "interactions/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "gflops": val * FLOP_PER_INTERACTION / 1e9,
        "config": {"workload": workload, "n_j": n, "n_i": int(len(il)), "eps2": case.eps2,
                   "note": "no reference code exists (paper only); this arm is the fp64 oracle on host cores"},
        "cpu_baseline": {"value": val, "unit": "interactions/s", "cores": oracle.threads(),
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "interactions/s", "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def measured_peaks():
    """MEASURED_PEAKS.json (driver-written) or the profiling recipe's stated fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "source": "measured"}
    except (OSError, ValueError, KeyError):
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


# DRAM bytes per launch cannot be measured inside a timed run (they need ncu's counters), so `traffic`
# is quoted from the committed `ncu --set full` captures of this same command, per launch:
# force_kernel, default workload: a call is two launches (whole waves, then the remainder with j split).
# profiles/r2c_cfg3_first.md: the whole-wave launch (7104 CTAs, 87 % of the call's time) moved 68.28 MB
# read + 81.39 MB written = 149.7 MB -- the 46 MB pack plus the 102 MB of partial sums it writes (two
# j-subsets).  profiles/r2b_cfg3_second.md: the remainder launch (7072 CTAs), captured alone: 56.73 MB
# read + 74.69 MB written = 131.4 MB (the pack once more, and most of its 101 MB of partial sums).  Sum:
FORCE_KERNEL_DRAM_TRAFFIC = {"cfg3": 149.67e6 + 131.42e6}
# predict_kernel (profiles/r2_predict_full.md, profiles/r2_cfg3_full.md), by particle count:
# N = 2^22 + 11: 474.04 MB read (= 113 B x N exactly) + 150.20 MB written of the 184.5 MB the kernel
# stores (the rest was still in the L2 when the kernel ended) = 624.2 MB; N = 2^20: 118.5 + 18.3 MB.
PREDICT_DRAM_TRAFFIC = {4194315: 624.25e6, 1048576: 136.84e6}


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import __graft_entry__ as g
    g.build()
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import binding as nb, sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: there is no CPU fallback (use --impl reference "
                         "for the oracle on host cores)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    case, il, t, workload = make_case(args.workload)
    n, ni = case.n, len(il)
    lo, hi = sharding.shard_bounds(ni, rank, world)
    il_loc = np.ascontiguousarray(il[lo:hi])
    ni_loc = hi - lo

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.shard in ("j", "jx"):
        return run_shard_j(args, case, il, t, workload, rank, world, local, dev)
    ctx = nbm.Context(n, max(ni, 1), device=local)
    if args.fp64:
        ctx.precision(1)
    if args.order6:
        ctx.order(6)
    ctx.load_case(case)
    h = ctx.h
    # device-resident step inputs: the active list and the active particles' corrected state (here:
    # their stored state again -- a real integrator writes the corrector's output into these)
    d_il_full = torch.from_numpy(np.ascontiguousarray(il)).to(dev)
    d_il = torch.from_numpy(il_loc).to(dev)
    upd = [torch.from_numpy(np.ascontiguousarray(q[..., il])).to(dev)
           for q in (case.m, case.x, case.v, case.a, case.j, case.t)]
    acc = torch.empty((3, ni_loc), dtype=torch.float64, device=dev)
    jrk = torch.empty((3, ni_loc), dtype=torch.float64, device=dev)
    pot = torch.empty((ni_loc,), dtype=torch.float64, device=dev)
    snp = torch.empty((3, ni_loc), dtype=torch.float64, device=dev) if args.order6 else None

    def step():
        nb.nb_update_j(h, d_il_full, ni, *upd)                     # a0
        nb.nb_predict(h, t)                                        # a1
        if args.order6:
            nb.nb_force6(h, d_il, ni_loc, case.eps2, acc, jrk, snp, pot)
        else:
            nb.nb_force(h, d_il, ni_loc, case.eps2, acc, jrk, pot) # a2..a5
        if world > 1:
            return sharding.gather_forces(acc, jrk, pot, ni)
        return acc, jrk, pot

    def timed(fn, k):
        """k calls of fn between barrier + synchronize, CUDA events on the launching stream."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(k):
            fn()
        e1.record()
        barrier()
        ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item())

    for _ in range(max(args.warmup, 3)):
        step()
    bad = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    for attempt in range(2):
        ctx.profiling(True)
        l0 = ctx.launch_count()
        sampler = ClockSampler(local)
        sampler.start()
        ms = timed(step, args.steps)
        clocks = sampler.stop()
        launches = ctx.launch_count() - l0
        kt = ctx.kernel_times()
        ctx.profiling(False)
        if clocks is None or not (bad & set(clocks["reasons"])):
            break
    nb.nb_sync(h)
    assert bool(torch.isfinite(pot).all()), "non-finite potential"
    value = float(ni) * n * args.steps / (ms * 1e-3)

    # ---- e2e: the same step through the HOST-buffer entry points of the C-ABI -----------------
    e2e = None
    if not args.no_e2e and not args.order6:
        def pin(a):
            return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h_il_full, h_il = pin(il), pin(il_loc)
        h_upd = [pin(q[..., il]) for q in (case.m, case.x, case.v, case.a, case.j, case.t)]
        h_acc = torch.empty((3, ni_loc), dtype=torch.float64).pin_memory()
        h_jrk = torch.empty((3, ni_loc), dtype=torch.float64).pin_memory()
        h_pot = torch.empty((ni_loc,), dtype=torch.float64).pin_memory()
        h2d = ni * 4 + sum(q.numel() * 8 for q in h_upd) + ni_loc * 4
        d2h = (h_acc.numel() + h_jrk.numel() + h_pot.numel()) * 8

        def step_host():
            nb.nb_update_j_host(h, h_il_full, ni, *h_upd)
            nb.nb_predict(h, t)
            nb.nb_force_host(h, h_il, ni_loc, case.eps2, h_acc, h_jrk, h_pot)   # returns synced

        step_host()
        barrier()
        w0 = time.perf_counter()
        ms_h = timed(step_host, args.steps)
        wall = time.perf_counter() - w0
        assert bool(torch.isfinite(h_pot).all())
        # the timed host path against the device-resident result of the same step: bit for bit (the
        # reduction order is fixed, R9); a sample of 256 active particles spread over the list
        samp = np.unique(np.linspace(0, ni_loc - 1, 256).astype(np.int64))
        d_samp = torch.from_numpy(samp).to(dev)
        same = (np.array_equal(h_acc.numpy()[:, samp], acc[:, d_samp].cpu().numpy()) and
                np.array_equal(h_jrk.numpy()[:, samp], jrk[:, d_samp].cpu().numpy()) and
                np.array_equal(h_pot.numpy()[samp], pot[d_samp].cpu().numpy()))
        assert same, "host-buffer path and device-resident path disagree"
        e2e = {"value": float(ni) * n * args.steps / (ms_h * 1e-3), "unit": "interactions/s",
               "checked": "%d sampled i: outputs of the timed host-buffer path are bit-identical to the "
                          "device-resident step's (which tests/test_gpu_configs.py checks against the oracle)" % len(samp),
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": ms_h / args.steps, "wall_ms_per_step": wall / args.steps * 1e3,
               "api": "nb_update_j_host + nb_predict + nb_force_host (pinned host buffers)"}

    sweep = None
    if args.sweep and world == 1:
        # force call alone (gather + pairs + reduce), device-resident, per active-subset size:
        # the few-i regime is bound by streaming the packed j-set (44 B per j), not by FP32
        sweep = []
        for sub in case.i_lists:
            ns = len(sub)
            d_sub = torch.from_numpy(np.ascontiguousarray(sub)).to(dev)
            o = [torch.empty((3, ns), dtype=torch.float64, device=dev),
                 torch.empty((3, ns), dtype=torch.float64, device=dev),
                 torch.empty((ns,), dtype=torch.float64, device=dev)]
            reps = 3 if ns * n > 1e11 else (20 if ns * n > 1e9 else 200)

            def call():
                nb.nb_force(h, d_sub, ns, case.eps2, *o)
            for _ in range(3):
                call()
            best = min(timed(lambda: [call() for _ in range(reps)], 1) for _ in range(3)) / reps
            info = ctx.last_launch()
            ctx.profiling(True)
            for _ in range(min(reps, 50)):
                call()
            kts = ctx.kernel_times()
            ctx.profiling(False)
            sweep.append({"n_i": ns, "ms_per_call": best, "interactions_per_s": ns * n / (best * 1e-3),
                          "frac_fp32_peak": None, "pack_gbs": 44.0 * n / (best * 1e-3) / 1e9,
                          "hbm_frac": 44.0 * n / (best * 1e-3) / 1e9 / measured_peaks()["hbm_gbs"],
                          "j_splits": int(info["j_splits"]), "ctas": int(info["ctas"]),
                          "pair_ms": kts["pair_ms"] / max(kts["n_pair"], 1),
                          "reduce_ms": kts["reduce_ms"] / max(kts["n_reduce"], 1)})

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(dev)
    sm_max = clocks["sm_max_mhz"] if clocks else peaks["sm_max_mhz"]
    fp32_peak_tflops = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    pair_ms = kt["pair_ms"] / max(kt["n_pair"], 1)
    pred_ms = kt["predict_ms"] / max(kt["n_predict"], 1)
    red_ms = kt["reduce_ms"] / max(kt["n_reduce"], 1)
    ach = FLOP_PER_INTERACTION * ni_loc * n / (pair_ms * 1e-3) / 1e12
    roofline = {"kernel": "force_kernel", "bound": "alu", "achieved": ach, "peak": fp32_peak_tflops,
                "unit": "TFLOP/s", "frac": ach / fp32_peak_tflops,
                "traffic": FORCE_KERNEL_DRAM_TRAFFIC.get(args.workload),
                "peak_source": "derived: %d SMs x 128 FP32 lanes x 2 x %.0f MHz (clocks.max.sm)" % (
                    props.multi_processor_count, sm_max),
                "ms_per_launch": pair_ms, "launches_timed": kt["n_pair"],
                "share_of_step": kt["pair_ms"] / ms}
    # what the FMA pipe sustains with the pair kernel's instruction kinds: measured by the committed
    # micro-benchmark bench/micro/pipe_probe.cu (profiles/r1_pipe_probes.md), not re-measured here
    roofline["fma_probe"] = {
        "ffma2_lanes_per_clk_sm": FFMA2_LANES_PER_CLK_SM, "source": "profiles/r1_pipe_probes.md",
        "frac_of_ffma2_rate": (ach * 1e12 / FLOP_PER_INTERACTION * 33.0) /
                              (props.multi_processor_count * FFMA2_LANES_PER_CLK_SM * sm_max * 1e6),
        "note": "the pair body executes 33 FP32 lane-ops per interaction (DESIGN.md 7.2); "
                "frac_of_ffma2_rate = executed lane-ops/s over the measured packed-FMA rate"}
    if args.order6:
        # 64 FP32 lane-operations per interaction (force6.cu) against 128 lanes per SM per clock
        lane_peak = props.multi_processor_count * FP32_LANES_PER_SM * sm_max * 1e6
        rate6 = ni_loc * n / (pair_ms * 1e-3)
        roofline.update({"kernel": "force6_kernel (+ its reduction)", "lane_ops_per_interaction": 64,
                         "frac_of_fp32_lanes": 64.0 * rate6 / lane_peak,
                         "note": "achieved / frac are in 60-flop interactions as for the 4th-order kernel; the "
                                 "6th-order body executes 64 lane-ops per interaction instead of 33, so its "
                                 "ceiling in interactions is 33/64 of that kernel's",
                         "traffic": None})
        roofline["fma_probe"]["frac_of_ffma2_rate"] = (64.0 * rate6) / (
            props.multi_processor_count * FFMA2_LANES_PER_CLK_SM * sm_max * 1e6)
        roofline["fma_probe"]["note"] = "64 lane-ops per interaction (force6.cu)"
    if args.fp64:
        # FP64 pipe: 64 lanes per SM per clock (measured DFMA/DADD rate, profiles/r1_pipe_probes.md)
        p64 = fp32_peak_tflops / 2.0
        roofline.update({"kernel": "force64_kernel", "peak": p64, "frac": ach / p64,
                         "peak_source": "derived: %d SMs x 64 FP64 lanes x 2 x %.0f MHz" % (
                             props.multi_processor_count, sm_max)})
        roofline["fma_probe"]["note"] = "FP32 probe, not applicable to the fp64 loop (35 fp64 ops per interaction)"
        roofline["fma_probe"]["frac_of_ffma2_rate"] = None
    if clocks:
        obs = props.multi_processor_count * FP32_LANES_PER_SM * 2 * clocks["sm_mhz"] * 1e6 / 1e12
        roofline["frac_at_observed_clock"] = ach / (obs / 2.0 if args.fp64 else obs)
    pred_gbs = PREDICT_BYTES_PER_PARTICLE * n / (pred_ms * 1e-3) / 1e9
    roofline_predict = {"kernel": "predict_kernel", "bound": "hbm", "achieved": pred_gbs,
                        "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": pred_gbs / peaks["hbm_gbs"],
                        "traffic": PREDICT_DRAM_TRAFFIC.get(n), "peak_source": peaks["source"], "ms_per_launch": pred_ms,
                        "bytes_per_particle": PREDICT_BYTES_PER_PARTICLE}
    line = {
        "metric": "interactions/s", "value": value, "unit": "interactions/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64" if args.fp64 else "f32",
        "data": "synthetic", "gflops": value * FLOP_PER_INTERACTION / 1e9,
        "config": {"workload": workload + ("_order6" if args.order6 else ""), "n_j": n, "n_i": ni, "eps2": case.eps2,
                   "step": "nb_update_j(active) + nb_predict + %s (gather, pairs, reduce)" % (
                       "nb_force6: acc, jerk, snap, pot" if args.order6 else "nb_force"),
                   "parallelism": "i-sharded x%d, j replicated" % world,
                   "l2": "no flush: per-step working set (j-store %.0f MB + pack %.0f MB + outputs "
                         "%.0f MB) exceeds the L2" % (112e-6 * n, 44e-6 * n, 56e-6 * ni),
                   "arithmetic": ("IEEE double throughout (rsqrt: MUFU + 2 Newton steps)" if args.fp64 else
                                  "two-float (48-bit) position differences, fp32 pair terms, "
                                  "fp32 per-tile sums flushed to fp64")},
        "clocks": ({"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"],
                    "reasons": clocks["reasons"], "power_w_max": clocks["power_w_max"],
                    "samples": clocks["samples"]} if clocks else None),
        "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "roofline_predict": roofline_predict,
        "kernels_ms": {"predict": pred_ms, "pair": pair_ms, "reduce": red_ms},
    }
    if sweep is not None:
        for q in sweep:
            q["frac_fp32_peak"] = q["interactions_per_s"] * FLOP_PER_INTERACTION / 1e12 / fp32_peak_tflops
        line["sweep"] = sweep
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = oracle_sample(case, il, t, args.cpu_seconds)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    print(json.dumps(line))
    return 0


def run_blockstep(args):
    """Block-time-step regime: every step advances only the particles that are
    due, so N_i << N and the O(N) pieces (scheduler, predictor) and launch latency matter."""
    import numpy as np
    import torch
    import __graft_entry__ as g
    g.build()
    import nbgen
    import paper_1409_5474_b200 as nbm
    n = args.blockstep
    eps2, eta, lo, hi = (4.0 / n) ** 2, 0.02, 2.0 ** -24, 2.0 ** -4
    m, x, v = nbgen.plummer(n, nbgen.SEED0 + 6)
    il = np.arange(n, dtype=np.int32)
    def run(mode):
        """The same `--steps` block steps from the same start: mode "step" = one nb_step call per
        block (five launches + a synchronisation each), "steps" = one nb_steps call (persistent
        kernel; the host sees only the blocks above the bound)."""
        with nbm.Context(n) as ctx:
            if args.steps_bound >= 0:
                ctx.steps_bound(int(args.steps_bound))
            ctx.steps_queue({"steps_host": 0, "steps_rounds": 1, "steps_graph": 2}.get(mode, -1))   # "steps": the default
            ctx.set_j(m, x, v)
            ctx.predict(0.0)
            ga, gj, gp = ctx.force(il, eps2)
            ctx.init_steps(il, ga, gj, eta, lo, hi)
            for _ in range(max(args.warmup, 3)):
                ctx.step(eps2, eta, lo, hi)
            ctx.steps(3, eps2, eta, lo, hi)
            ctx.sync()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = ctx.launch_count()
            w0 = time.perf_counter()
            e0.record()
            if mode == "step":
                sz = []
                for _ in range(args.steps):
                    t, ni = ctx.step(eps2, eta, lo, hi)
                    sz.append(ni)
            else:
                done, tl, sz, us = ctx.steps(args.steps, eps2, eta, lo, hi, times=True)
                assert done == args.steps
                t = float(tl[-1])
                {"steps": times, "steps_host": times_host}.get(mode, []).append(np.array(us))
            e1.record()
            ctx.sync()
            return e0.elapsed_time(e1), time.perf_counter() - w0, ctx.launch_count() - l0, list(sz), t

    # A/B inside one process, interleaved: numbers from different gpurun calls differ by +-20 % for a
    # latency-bound loop and must not be compared with each other
    times, times_host = [], []
    runs = [(md, run(md)) for md in ("step", "steps_host", "steps_rounds", "steps_graph", "steps") * 2]
    ms_graph, _, launches_graph, _, _ = min((r for md, r in runs if md == "steps_graph"), key=lambda r: r[0])
    ms_rounds, _, launches_rounds, _, _ = min((r for md, r in runs if md == "steps_rounds"), key=lambda r: r[0])
    ms_step, _, launches_step, _, _ = min((r for md, r in runs if md == "step"), key=lambda r: r[0])
    ms_host, _, launches_host, _, _ = min((r for md, r in runs if md == "steps_host"), key=lambda r: r[0])
    ms, wall, launches, sizes, t = min((r for md, r in runs if md == "steps"), key=lambda r: r[0])
    sizes = np.array(sizes, dtype=np.float64)
    small = (sizes <= 512) & (sizes * n <= (args.steps_bound if args.steps_bound >= 0 else 1.5e7))
    in_kernel = int(small.sum())
    us = np.minimum(times[0], times[1])                    # per-step device time (%globaltimer), best of 2
    floor_us = sizes * n / 1.2408e12 * 1e6                  # pair work at 100 % of the FP32 peak
    line = {"metric": "interactions/s", "value": float(sizes.sum() * n / (ms * 1e-3)),
            "unit": "interactions/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / args.steps, "wall_ms_per_step": wall / args.steps * 1e3,
            "higher_is_better": True, "dtype": "f64 in the persistent kernel, f32 pair terms in large blocks",
            "data": "synthetic",
            "config": {"workload": "blockstep_plummer_N%d" % n, "eta": eta, "eps2": eps2,
                       "step": "nb_steps: scheduler + predictor-in-pair-loop + reduce + corrector per block in "
                               "one persistent kernel; blocks above 512 particles or 1.5e7 pairs: " +
                               ("launch shape planned on the device, predictor + packed fp32 pair kernel + reduction + "
                                "corrector queued ahead of time (no host round trip)" if n < 262144 else
                                "handed to nb_step's launches (one host synchronisation per such block)")},
            "block": {"mean_n_i": float(sizes.mean()), "median_n_i": float(np.median(sizes)),
                      "min_n_i": int(sizes.min()), "max_n_i": int(sizes.max()),
                      "in_persistent_kernel": in_kernel,
                      "us_per_step_in_kernel_mean": float(us[small].mean()) if in_kernel else None,
                      "us_per_step_in_kernel_median": float(np.median(us[small])) if in_kernel else None,
                      "us_per_step_host_path_mean": float(us[~small].mean()) if in_kernel < len(sizes) else None,
                      "us_total_in_kernel": float(us[small].sum()), "us_total_host_path": float(us[~small].sum()),
                      "us_pair_work_at_fp32_peak_total": float(floor_us.sum()),
                      "us_pair_work_at_fp32_peak_host_path": float(floor_us[~small].sum()),
                      "particle_steps_per_s": float(sizes.sum() / (ms * 1e-3)), "t_end": t},
            "ab": {"us_per_block_step_nb_step": ms_step / args.steps * 1e3,
                   "us_per_block_step_nb_steps_host_handover": ms_host / args.steps * 1e3,
                   "us_per_block_step_nb_steps_stream_rounds": ms_rounds / args.steps * 1e3,
                   "us_per_block_step_nb_steps_graph": ms_graph / args.steps * 1e3,
                   "us_per_block_step_nb_steps": ms / args.steps * 1e3,
                   "launches_per_block_nb_steps_graph": launches_graph / args.steps,
                   "launches_per_block_nb_steps_stream_rounds": launches_rounds / args.steps,
                   "launches_per_block_nb_step": launches_step / args.steps,
                   "launches_per_block_nb_steps_host_handover": launches_host / args.steps,
                   "launches_per_block_nb_steps": launches / args.steps,
                   "us_total_host_path_host_handover": float(np.minimum(times_host[0], times_host[1])[~small].sum()),
                   "note": "same process, same start and schedule, best of 2 each, interleaved; "
                           "nb_steps = the library's default (nb_set_steps_queue -1: graph below 262144 particles, "
                           "host_handover from there on), graph = large blocks planned on the device, rounds in the "
                           "WHILE node of one graph (queue 2), stream_rounds = the same rounds queued on the stream (1), "
                           "host_handover = one host synchronisation per large block (queue 0)"},
            "gpu_launches": int(launches)}
    if args.detail:
        line["steps_detail"] = {"n_i": [int(q) for q in sizes], "us": [float(q) for q in us],
                                "us_host_handover": [float(q) for q in np.minimum(times_host[0], times_host[1])]}
    print(json.dumps(line))
    return 0


def run_fewi(args):
    """a handful of active particles.  The call then streams the predicted j-set once
    (44 B per particle, nb_force) or the whole j-store (112 B, nb_force_fused, predictor inside) and
    is bound by HBM and launch latency, not by FP32: reported against the measured copy bandwidth."""
    import numpy as np
    import torch
    import __graft_entry__ as g
    g.build()
    import nbgen
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import binding as nb
    peaks = measured_peaks()
    case, il_all, t, workload = make_case(args.workload)
    n = case.n
    dev = torch.device("cuda", 0)
    rows = []
    n_small = 1024            # the same call on the case's first 1024 particles: what a call costs before any streaming
    with nbm.Context(n, 1 << 10) as ctx, nbm.Context(n_small, 1 << 10) as small:
        ctx.load_case(case)
        sl = slice(0, n_small)
        small.set_j(case.m[sl], case.x[:, sl], case.v[:, sl], case.a[:, sl], case.j[:, sl], case.t[sl])
        flush = torch.zeros(256 << 20, dtype=torch.uint8, device=dev)      # > L2: reading it evicts the pack / store
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def timed(c, call):
            """(a) back to back, the j data resident in L2 as far as it fits; (b) every call after an L2
            flush, timed alone with events around the call (median of 20)."""
            for _ in range(5):
                call()
            c.sync()
            reps = 200
            e0.record()
            for _ in range(reps):
                call()
            e1.record()
            c.sync()
            warm = e0.elapsed_time(e1) / reps * 1e3
            cold = []
            for _ in range(20):
                flush.sum()                 # a READ pass: the L2 then holds clean lines of this buffer only
                e0.record()
                call()
                e1.record()
                c.sync()
                cold.append(e0.elapsed_time(e1) * 1e3)
            return warm, float(np.median(cold))

        for ni in (1, 2, 4, 8, 16, 64):
            il_big = torch.from_numpy(np.ascontiguousarray(il_all[:ni])).to(dev)
            il_small = torch.arange(ni, dtype=torch.int32, device=dev)
            o = [torch.empty((3, ni), dtype=torch.float64, device=dev),
                 torch.empty((3, ni), dtype=torch.float64, device=dev),
                 torch.empty((ni,), dtype=torch.float64, device=dev)]
            for name in ("nb_force", "nb_force_fused"):
                if name == "nb_force_fused" and ni > nb.NB_FUSED_MAX:
                    continue
                res = {}
                for c, d_il, nn in ((ctx, il_big, n), (small, il_small, n_small)):
                    h = c.h
                    if name == "nb_force":
                        nb.nb_predict(h, t)
                        call = lambda: nb.nb_force(h, d_il, ni, case.eps2, *o)
                        per = 44.0
                    else:
                        call = lambda: nb.nb_force_fused(h, t, d_il, ni, case.eps2, *o)
                        per = 112.0
                    res[nn] = timed(c, call)
                warm, cold_us = res[n]
                warm_s, cold_s = res[n_small]
                nbytes = per * n
                info = ctx.last_launch()
                rows.append({"call": name, "n_i": ni, "us_per_call_back_to_back": warm, "us_per_call_after_l2_flush": cold_us,
                             "bytes_per_call": nbytes, "gbs_after_flush": nbytes / cold_us / 1e3,
                             "hbm_frac": nbytes / cold_us / 1e3 / peaks["hbm_gbs"],
                             "gbs_back_to_back": nbytes / warm / 1e3,
                             "us_same_call_n1024_back_to_back": warm_s, "us_same_call_n1024_after_l2_flush": cold_s,
                             "gbs_incremental_after_flush": per * (n - n_small) / max(cold_us - cold_s, 1e-3) / 1e3,
                             "hbm_frac_incremental": per * (n - n_small) / max(cold_us - cold_s, 1e-3) / 1e3 / peaks["hbm_gbs"],
                             "kernels": int(info["kernels"]), "ctas": int(info["ctas"])})
    best = max(r["hbm_frac"] for r in rows if r["n_i"] == 1)
    line = {"metric": "GB/s of the j data streamed by one few-i force call", "value": best * peaks["hbm_gbs"],
            "unit": "GB/s", "n_gpus": 1, "steps": 200, "warmup": 5, "higher_is_better": True, "dtype": "f32/f64",
            "data": "synthetic", "config": {"workload": workload + "_few_i", "n_j": n,
                                            "l2": "hbm_frac rows: the L2 is flushed (a 256 MB buffer is read) before every timed call",
                                            "incremental": "the same call on the first 1024 particles is timed the same way: "
                                                           "hbm_frac_incremental = bytes of the other N - 1024 particles over "
                                                           "the time difference, i.e. the streaming rate without the call's "
                                                           "fixed latency (launch, gather, ticket, reduction, event overhead)"},
            "roofline": {"bound": "hbm", "peak": peaks["hbm_gbs"], "peak_source": peaks["source"], "unit": "GB/s",
                         "achieved": best * peaks["hbm_gbs"], "frac": best, "traffic": None},
            "rows": rows}
    print(json.dumps(line))
    return 0


def run_midsize(args):
    """PAPER.md:51 between the two regimes it names: some hundreds to thousands of active particles (the
    blocks of a block-time-step code at N ~ 1e5 ... 1e6).  One nb_force call, by index, on a Plummer set:
    N_i at multiples of the 256-slot i-tile and a few particles above them, where the last tile would be
    mostly padding and goes to the few-i kernel as a segment of its own."""
    import numpy as np
    import torch
    import __graft_entry__ as g
    g.build()
    import nbgen
    import paper_1409_5474_b200 as nbm
    dev = torch.device("cuda", 0)
    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(dev)
    peak = props.multi_processor_count * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / FLOP_PER_INTERACTION
    rows = []
    for n in (1 << 16, 1 << 17, 1 << 20):
        m, x, v = nbgen.plummer(n, 7)
        zero = np.zeros((3, n))
        with nbm.Context(n, 16400) as ctx:
            ctx.set_j(m, x, v, zero, zero, np.zeros(n))
            ctx.predict(0.0)
            perm = torch.from_numpy(nbgen.permutation(8, n).astype(np.int32)).to(dev)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for ni in (256, 257, 288, 320, 384, 512, 520, 640, 768, 800, 1024, 1056, 2048, 2080, 3100, 4096, 4128, 8192, 8224,
                       16384, 16400):
                il = perm[:ni].contiguous()
                reps = max(5, min(300, int(1e11 / (ni * n))))
                for _ in range(max(args.warmup, 3)):
                    ctx.force(il, 2.0 ** -20)
                ctx.sync()
                e0.record()
                for _ in range(reps):
                    ctx.force(il, 2.0 ** -20)
                e1.record()
                ctx.sync()
                us = e0.elapsed_time(e1) / reps * 1e3
                info = ctx.last_launch()
                rows.append({"n_j": n, "n_i": ni, "us_per_call": us, "interactions_per_s": ni * n / us * 1e6,
                             "frac_fp32_peak": ni * n / us * 1e6 / peak, "kernels": int(info["kernels"]),
                             "ctas": int(info["ctas"])})
    best = max(rows, key=lambda r: r["frac_fp32_peak"])
    line = {"metric": "interactions/s", "value": best["interactions_per_s"], "unit": "interactions/s", "n_gpus": 1,
            "steps": "5..300 calls per row", "warmup": max(args.warmup, 3), "higher_is_better": True, "dtype": "f32",
            "data": "synthetic", "config": {"workload": "plummer_midsize_calls", "value_is": "the best row",
                                            "l2": "no flush: back-to-back calls, the packed j-set (44 B per particle) stays in the L2"},
            "roofline": {"bound": "alu", "unit": "interactions/s", "peak": peak, "achieved": best["interactions_per_s"],
                         "frac": best["frac_fp32_peak"], "traffic": None,
                         "peak_source": "derived: %d SMs x 128 FP32 lanes x 2 x %.0f MHz / 60 flop" % (
                             props.multi_processor_count, peaks["sm_max_mhz"])},
            "rows": rows}
    print(json.dumps(line))
    return 0


def run_predict(args):
    """The Hermite predictor (a1) against the HBM roofline, where its working set cannot sit in the L2:
    (a) config 5's N = 2^22 + 11 (470 MB of j-store, 185 MB of packed records), (b) config 3's
    N = 2^20 alternating between two contexts (2 x 163 MB > 126 MB of L2).  GB/s at the contract's
    152 B per particle and at the 157 B the kernel moves (112 B + 1 flag byte read,
    44 B written)."""
    import numpy as np
    import torch
    import __graft_entry__ as g
    g.build()
    import nbgen
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import binding as nb
    peaks = measured_peaks()
    reps = max(args.steps, 20)

    def time_calls(ctxs, t):
        e = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        for _ in range(max(args.warmup, 3)):
            for c in ctxs:
                nb.nb_predict(c.h, t)
        torch.cuda.synchronize()
        for r in range(reps):
            c = ctxs[r % len(ctxs)]
            e[r][0].record()
            nb.nb_predict(c.h, t)
            e[r][1].record()
        torch.cuda.synchronize()
        ms = np.array([a.elapsed_time(b) for a, b in e])
        return float(np.median(ms)), float(ms.min())

    rows = []
    c5 = nbgen.config5()
    with nbm.Context(c5.n, 1) as ctx:
        ctx.load_case(c5)
        med, best = time_calls([ctx], 2.0 ** -7)
        rows.append({"case": "cfg5_N%d_one_context" % c5.n, "n": c5.n, "ms_median": med, "ms_min": best})
    del c5
    c3 = nbgen.config3(sizes=(1,))
    with nbm.Context(c3.n, 1) as a, nbm.Context(c3.n, 1) as b:
        a.load_case(c3)
        b.load_case(c3)
        med, best = time_calls([a, b], c3.t_now)
        rows.append({"case": "cfg3_N%d_two_contexts_alternating" % c3.n, "n": c3.n, "ms_median": med, "ms_min": best})
    for r in rows:
        r["gbs_152"] = 152.0 * r["n"] / (r["ms_median"] * 1e-3) / 1e9
        r["gbs_157"] = 157.0 * r["n"] / (r["ms_median"] * 1e-3) / 1e9
        r["frac_152"] = r["gbs_152"] / peaks["hbm_gbs"]
        r["frac_157"] = r["gbs_157"] / peaks["hbm_gbs"]
        # DRAM bytes of this launch from the committed ncu capture (profiles/r2_predict_full.md)
        r["traffic"] = PREDICT_DRAM_TRAFFIC.get(r["n"])
    top = rows[0]
    line = {"metric": "GB/s of the Hermite predictor (152 B per particle)", "value": top["gbs_152"], "unit": "GB/s",
            "n_gpus": 1, "steps": reps, "warmup": max(args.warmup, 3), "ms_per_step": top["ms_median"],
            "higher_is_better": True, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "predictor_" + top["case"],
                       "l2": "working set 655 MB (one context) / 2 x 163 MB (two contexts) exceeds the 126 MB L2"},
            "roofline": {"kernel": "predict_kernel", "bound": "hbm", "achieved": top["gbs_152"], "peak": peaks["hbm_gbs"],
                         "unit": "GB/s", "frac": top["frac_152"], "traffic": top["traffic"],
                         "peak_source": peaks["source"], "achieved_at_157_bytes": top["gbs_157"],
                         "frac_at_157_bytes": top["frac_157"]},
            "rows": rows}
    print(json.dumps(line))
    return 0


def run_shard_j(args, case, il, t, workload, rank, world, local, dev):
    """The paper's own multi-GPU scheme: rank r stores and predicts only its slice of j,
    evaluates ALL active particles, received by value, against it (nb_force_ext_ids), and the partial
    forces are summed by one all_reduce of [7][N_i] fp64.  World size 1 runs the same code path."""
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import binding as nb, sharding
    if world == 1 and not dist.is_initialized():
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1, device_id=dev)
    n, ni = case.n, len(il)
    lo, hi = sharding.shard_bounds(n, rank, world)               # this rank's j-slice
    ctx = nbm.Context(hi - lo, ni, device=local)
    sl = slice(lo, hi)
    ctx.set_j(case.m[sl], case.x[:, sl], case.v[:, sl], case.a[:, sl], case.j[:, sl], case.t[sl])
    fl = np.flatnonzero(case.flags[sl]).astype(np.int32)
    if fl.size:
        ctx.set_flags(fl, np.ones(fl.size, np.uint8))
    h = ctx.h
    pos = sharding.owned(il, lo, hi).to(dev)                     # active particles this rank owns
    mine = torch.from_numpy(il.astype(np.int64)).to(dev)[pos]
    flags_dev = torch.from_numpy(case.flags.astype(np.float64)).to(dev)

    fused = args.shard == "jx"
    if fused:
        # the partial forces are exchanged and summed by the kernels over peer memory (nb_xforce)
        torch.cuda.set_device(dev)
        sharding.xchg_connect(ctx, ni)

    def step():
        nb.nb_predict(h, t)
        px, pv = ctx.predicted()
        loc = mine - lo
        state = torch.cat([px[:, loc], pv[:, loc], flags_dev[None, mine], mine[None].to(torch.float64)], 0)
        if fused:
            return sharding.force_j_sharded_xchg(ctx, state, pos, ni, lo, hi, case.eps2)
        return sharding.force_j_sharded(lambda x, v, s_, f_: ctx.force_ext_ids(x, v, s_, f_, case.eps2),
                                        state, pos, ni, lo, hi)

    def small_block(k, reps=200):
        """One force call of the block-step regime (k active particles, state already on every rank):
        partial forces + NCCL all_reduce against nb_xforce (one launch)."""
        sel = torch.from_numpy(il[:k].astype(np.int64)).to(dev)
        px, pv = ctx.predicted()
        own = (sel >= lo) & (sel < hi)
        # the state of particles this rank does not own comes from the case (any value serves the timing)
        xs = torch.from_numpy(np.ascontiguousarray(case.x[:, il[:k]])).to(dev)
        vs = torch.from_numpy(np.ascontiguousarray(case.v[:, il[:k]])).to(dev)
        if bool(own.any()):
            xs[:, own] = px[:, sel[own] - lo]
            vs[:, own] = pv[:, sel[own] - lo]
        sidx = torch.where(own, sel - lo, torch.full_like(sel, -1)).to(torch.int32)
        ifl = torch.zeros(k, dtype=torch.uint8, device=dev)
        out = {}
        for name in ("nccl", "xchg"):
            def call():
                if name == "xchg":
                    return ctx.xforce(xs, vs, sidx, ifl, case.eps2)
                a, j, p = ctx.force_ext_ids(xs, vs, sidx, ifl, case.eps2)
                part = torch.cat([a, j, p.reshape(1, -1)], 0)
                dist.all_reduce(part)
                return part
            for _ in range(10):
                call()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            f0.record()
            for _ in range(reps):
                call()
            f1.record()
            barrier()
            out["us_per_call_" + name] = f0.elapsed_time(f1) * 1e3 / reps
        return out

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        out = step()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = ctx.launch_count()
    barrier()
    e0.record()
    for _ in range(args.steps):
        out = step()
    e1.record()
    barrier()
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms = float(ms.item())
    launches = ctx.launch_count() - l0
    assert bool(torch.isfinite(out[2]).all())
    if rank == 0:
        value = float(ni) * n * args.steps / (ms * 1e-3)
        line = {"metric": "interactions/s", "value": value, "unit": "interactions/s", "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "gflops": value * FLOP_PER_INTERACTION / 1e9,
                "config": {"workload": workload, "n_j": n, "n_i": ni, "eps2": case.eps2,
                           "step": "nb_predict(slice) + all_gather(active state) + nb_force_ext_ids(slice) + "
                                   "all_reduce([7][N_i])",
                           "parallelism": "j-sharded x%d (PAPER.md:55), active particles by value" % world},
                "gpu_launches": int(launches),
                "bytes_all_reduce_per_step": 56 * ni, "bytes_all_gather_per_step": 72 * ni}
        if fused:
            line["config"]["step"] = ("nb_predict(slice) + all_gather(active state) + nb_xforce(slice: pair kernel, "
                                      "reduction, push to the peers' windows, flags, sum in rank order)")
            line["bytes_all_reduce_per_step"] = 0
            line["bytes_pushed_per_step"] = 56 * ni * world
    sb = None
    if fused:
        sb = {"n_i": 4, **small_block(4)}
        sb16 = {"n_i": 16, **small_block(16)}
    if rank == 0:
        if fused:
            line["small_block"] = [sb, sb16]
        print(json.dumps(line))
    ctx.close()
    dist.destroy_process_group()
    return 0


def run_kick(args):
    """NEXT-2: the kick one system receives from another ("completely different set",
    PAPER.md:118-123), i-particles by value."""
    import numpy as np
    import torch
    import __graft_entry__ as g
    g.build()
    import nbgen
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import binding as nb
    c = nbgen.config4()
    na = (c.n // 2)
    dev = torch.device("cuda", 0)
    with nbm.Context(na, c.n - na) as ctx:
        ctx.set_j(c.m[:na].copy(), np.ascontiguousarray(c.x[:, :na]), np.ascontiguousarray(c.v[:, :na]))
        ctx.predict(0.0)
        xb = torch.from_numpy(np.ascontiguousarray(c.x[:, na:])).to(dev)
        vb = torch.from_numpy(np.ascontiguousarray(c.v[:, na:])).to(dev)
        ni = xb.shape[1]
        acc = torch.empty((3, ni), dtype=torch.float64, device=dev)
        jrk = torch.empty((3, ni), dtype=torch.float64, device=dev)
        pot = torch.empty((ni,), dtype=torch.float64, device=dev)
        props = torch.cuda.get_device_properties(dev)
        peak = props.multi_processor_count * FP32_LANES_PER_SM * 1965e6     # lane-ops/s
        out = {}
        for name, v, j, lane_ops in (("acc_jerk_pot", vb, jrk, 33.0), ("acc_pot", None, None, 19.0)):
            def call():
                nb.nb_force_ext(ctx.h, ni, xb, v, c.eps2, acc, j, pot)
            for _ in range(max(args.warmup, 3)):
                call()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.sync()
            e0.record()
            for _ in range(args.steps):
                call()
            e1.record()
            ctx.sync()
            ms = e0.elapsed_time(e1) / args.steps
            rate = float(ni) * na / (ms * 1e-3)
            out[name] = {"ms_per_call": ms, "interactions_per_s": rate,
                         "fp32_lane_ops_per_interaction": lane_ops,
                         "frac_of_fma_pipe": rate * lane_ops / peak}
    line = {"metric": "interactions/s", "value": out["acc_pot"]["interactions_per_s"],
            "unit": "interactions/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": out["acc_pot"]["ms_per_call"], "higher_is_better": True, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": "cfg4_kick_B_from_A", "n_j": int(na), "n_i": int(ni), "eps2": c.eps2},
            "variants": out}
    print(json.dumps(line))
    return 0


def run_scaling(args):
    """The direct-code curve of the paper's Fig. 2 (wall-clock time as a function of the
    number of particles, 10^3 to 10^7, one GPU) on one B200: one all-active force evaluation -- predictor
    + pair kernel + reduction -- of a Plummer sphere of N = 2^10 ... 2^log2max particles."""
    import numpy as np
    import torch
    import __graft_entry__ as g
    g.build()
    import nbgen
    import paper_1409_5474_b200 as nbm
    from paper_1409_5474_b200 import binding as nb
    dev = torch.device("cuda", 0)
    rows = []
    for lg in range(10, args.scaling + 1):
        n = 1 << lg
        m, x, v = nbgen.plummer(n, nbgen.SEED0 + 40 + lg)
        eps2 = (4.0 / n) ** 2
        with nbm.Context(n) as ctx:
            ctx.set_j(m, x, v)
            il = torch.arange(n, dtype=torch.int32, device=dev)
            acc = torch.empty((3, n), dtype=torch.float64, device=dev)
            jrk = torch.empty((3, n), dtype=torch.float64, device=dev)
            pot = torch.empty((n,), dtype=torch.float64, device=dev)

            def call():
                nb.nb_predict(ctx.h, 0.0)
                nb.nb_force(ctx.h, il, n, eps2, acc, jrk, pot)
            pairs = float(n) * n
            reps = 1 if pairs > 2e13 else (3 if pairs > 1e12 else (20 if pairs > 1e10 else 200))
            for _ in range(1 if pairs > 2e13 else 3):
                call()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.sync()
            e0.record()
            for _ in range(reps):
                call()
            e1.record()
            ctx.sync()
            ms = e0.elapsed_time(e1) / reps
            assert bool(torch.isfinite(pot).all())
            rows.append({"n": n, "ms_per_evaluation": ms, "interactions_per_s": pairs / (ms * 1e-3),
                         "frac_fp32_peak": pairs / (ms * 1e-3) / 1.2408e12, "evaluations_timed": reps})
    top = rows[-1]
    line = {"metric": "interactions/s", "value": top["interactions_per_s"], "unit": "interactions/s", "n_gpus": 1,
            "steps": top["evaluations_timed"], "warmup": 3, "ms_per_step": top["ms_per_evaluation"],
            "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "fig2_direct_code_all_active_N_2^10_to_2^%d" % args.scaling,
                       "step": "nb_predict + nb_force on all N particles (one full force evaluation)"},
            "rows": rows}
    print(json.dumps(line))
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.scaling > 0:
        return run_scaling(args)
    if args.kick:
        return run_kick(args)
    if args.fewi:
        return run_fewi(args)
    if args.midsize:
        return run_midsize(args)
    if args.predict:
        return run_predict(args)
    if args.blockstep > 0:
        return run_blockstep(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
