#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on BASELINE.json's config: 6th-order Hermite force interactions/s at
N = 1 048 576 (config 4: Plummer + embedded BH binary, eps = 1e-5), all particles active.

A "step" is one pass of the whole hot path: restore the all-active state, block selection (a-1),
j-predictor (a-2), force (a-3), corrector + new time step (a-4).  `value` = N_act * N * steps / device time, inputs
resident in HBM; `e2e` = the same step through nbody_step_host with pinned HOST buffers (H2D + D2H inside the timed
region); `roofline` = the force kernel against the FP32 ALU peak DESIGN.md derives (2 * 128 lanes * 148 SMs *
1.965 GHz); `cpu_baseline` = the CPU oracle (oracle/, test infrastructure) timed on the host cores on a bounded
sample of the same workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--n N_PARTICLES] [--order P]
For N > 1 launch with torch.distributed.run; ranks i-shard the active list (strong scaling) and all-gather the
corrected rows once per step (paper_1312_1789_b200/parallel.py).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CONV_FLOPS = {4: 60, 6: 97, 8: 144}  # flops per interaction, community convention (R13)
SASS_FLOPS = {4: 41, 6: 78, 8: 127}  # executed: 2 x FFMA + FMUL + FADD + 3 DADD per pair in the loop's SASS (R13)
PACKED_OPS = {4: 24, 6: 46, 8: 76}   # FFMA2 + FMUL2 + FADD2 per (thread, j) = per two pairs
OTHER_OPS = {4: 19.5, 6: 20.5, 8: 21.5}  # DADD, F2F, MUFU, LDS, loop overhead per (thread, j)
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
FP32_PEAK_TFLOPS = 2 * FP32_LANES * SM_COUNT * SM_MAX_GHZ / 1e3  # 74.45, "alu" roofline denominator
METRIC = "6th-order Hermite force interactions/s at N=1M (all active), whole block step"
UNIT = "interactions/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=1048576)
    ap.add_argument("--order", type=int, default=6, choices=[4, 6, 8])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--cpu-sample", type=int, default=12288, help="i-particles of the cpu_baseline leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self._stop, self._th = index, [], False, None

    def _run(self):
        while not self._stop:
            try:
                o = subprocess.run(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-i",
                                    str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if o:
                    self.rows.append([f.strip() for f in o.split(",")])
            except Exception:
                pass
            time.sleep(0.2)

    def start(self):
        self._th = threading.Thread(target=self._run, daemon=True)
        self._th.start()

    def stop(self):
        self._stop = True
        if self._th:
            self._th.join(timeout=10)
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def workload(args):
    """Seeded synthetic stand-in for the paper's initial conditions: config-4 cluster."""
    from paper_1312_1789_b200 import workloads as W
    c = W.cluster(args.config, args.n)
    return W, c


def oracle_step(O, c, D, t, dt, idx, order, eps2, t_now):
    """The oracle's version of one step restricted to the sampled i-particles: predict all N, force on the sample,
    correct the sample.  Returns seconds."""
    t0 = time.perf_counter()
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    acc, jerk, snap, crk, pot = O.force(c["m"], xp, vp, ap, jp, idx, order, eps2)
    ot, odt, ox, ov = t.copy(), dt.copy(), c["x"].copy(), c["v"].copy()
    oD = [d.copy() for d in D] + [np.zeros_like(D[0]) for _ in range(8 - len(D))]
    O.correct(idx, order, t_now, 0.1, 2.0**-30, 2.0**-4, ot, odt, ox, ov, oD, np.zeros(c["n"]), acc, jerk, snap, crk,
              pot, crit_order=4 if order >= 6 else 0)
    return time.perf_counter() - t0, (acc, jerk, snap, crk, pot)


def run_reference(args):
    """--impl reference: the CPU oracle as it stands on the box's host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    W, c = workload(args)
    n, order = c["n"], args.order
    D = W.smooth_field_derivs(c, 6)
    t = np.zeros(n)
    dt = np.full(n, 2.0**-10)
    idx = W.oracle_sample(c, size=min(args.cpu_sample // 3, n))
    for _ in range(max(0, min(args.warmup, 1))):
        oracle_step(O, c, D, t, dt, idx[:64], order, c["eps2"], 2.0**-10)
    secs = []
    for _ in range(args.steps):
        s, _ = oracle_step(O, c, D, t, dt, idx, order, c["eps2"], 2.0**-10)
        secs.append(s)
    tot = sum(secs)
    value = idx.shape[0] * n * args.steps / tot
    sample = "%d i-particles (forced members + seeded draw) x all %d j per step" % (idx.shape[0], n)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config4 Plummer+BH-binary N=%d order %d all-active (oracle on a bounded i-sample)"
                       % (n, order), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1312_1789_b200 import nbody, parallel
    from paper_1312_1789_b200.scheduler import Integrator

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    W, c = workload(args)
    n, order, eps2 = c["n"], args.order, c["eps2"]
    H = 2.0**-10  # every particle is due at t = 2^-10: one all-active block

    # ---- untimed set-up: physically consistent Taylor coefficients from the GPU bootstrap (R9b) ----
    g = Integrator(c["m"], c["x"], c["v"], order, eps2, device=local)
    g.bootstrap(fixed_dt=H)
    torch.cuda.synchronize()
    keep = [a.clone() for a in (g.t, g.dt, g.x, g.v, g.pot, *g.D[:order])]
    live = [g.t, g.dt, g.x, g.v, g.pot, *g.D[:order]]
    scrub = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=g.dev)  # > 126 MB L2
    ev = lambda: torch.cuda.Event(enable_timing=True)
    force_ms, step_ms = [], []

    def one_step(timed):
        scrub.fill_(rank & 0xFF)  # L2 flush between steps (not part of the path)
        e0, e1, f0, f1 = ev(), ev(), ev(), ev()
        e0.record()
        for dst, src in zip(live, keep):
            dst.copy_(src)
        ctx, p = g.ctx, order
        t_next, n_act = ctx.next_block(n, g.t, g.dt, g.active)
        ctx.predict(n, t_next, p, g.t, g.m, g.x, g.v, g.D)
        lo, hi = parallel.shard_bounds(n_act, rank, world)
        act = g.active[lo:hi]
        snap, crk = (g.snap if p >= 6 else None), (g.crk if p >= 8 else None)
        if world > 1:
            ctx.set_option("geometry_n_act", n_act)  # summation order of the unsharded call (bit-identical shards)
        f0.record()
        ctx.force(act, hi - lo, p, eps2, g.acc, g.jerk, snap, crk, g.fpot)
        f1.record()
        if world > 1:
            ctx.set_option("geometry_n_act", 0)
        ctx.correct(act, hi - lo, p, t_next, g.eta, g.dt_min, g.dt_max, g.t, g.dt, g.x, g.v, g.D, g.pot, g.acc, g.jerk,
                    snap, crk, g.fpot)
        sent = parallel.exchange_corrected(g.active, n_act, rank, world, g.t, g.dt, g.pot, g.x, g.v, g.D, p,
                                           ctx=ctx)
        e1.record()
        if timed:
            step_ms.append((e0, e1))
            force_ms.append((f0, f1))
        assert n_act == n and t_next == H
        return n_act, hi - lo, sent

    for _ in range(max(args.warmup, 3)):
        one_step(False)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = g.ctx.launch_count()
    torch.cuda.synchronize()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        n_act, mine, sent = one_step(True)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    wall = time.perf_counter() - w0
    launches = g.ctx.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    dev_s = sum(a.elapsed_time(b) for a, b in step_ms) * 1e-3
    f_s = sum(a.elapsed_time(b) for a, b in force_ms) * 1e-3
    if world > 1:
        tmax = torch.tensor([dev_s, f_s], dtype=torch.float64, device=g.dev)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dev_s, f_s = float(tmax[0]), float(tmax[1])
    value = n_act * n * args.steps / dev_s
    geom = g.ctx.last_force_geometry()

    # ---- roofline of the dominant kernel (K_force), measured live over the timed steps ----
    f_avg = f_s / args.steps
    pairs_per_s = mine * n / f_avg
    achieved = CONV_FLOPS[order] * pairs_per_s / 1e12
    counters = {}
    cj = os.path.join(ROOT, "profiles", "r02_force_counters.json")  # ncu capture of this launch (profiles/r02_force6_1M.md)
    if os.path.exists(cj):
        try:
            counters = json.load(open(cj))
        except Exception:
            counters = {}
    traffic = counters.get("dram_bytes_per_launch") if order == 6 and n == 1048576 and world == 1 else None
    sass = SASS_FLOPS[order]
    roofline = {"bound": "alu", "kernel": "k_force<%d, %d, 0>" % (order, geom["j_lanes"]),
                "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
                "traffic": traffic, "flops_per_interaction": CONV_FLOPS[order],
                "flops_convention": "%d flops per interaction is the community convention for order %d (DESIGN.md R13; "
                                    "not in PAPER.md); the kernel EXECUTES %d (SASS count: FFMA x2 + FMUL + FADD + DADD)"
                                    % (CONV_FLOPS[order], order, sass),
                "flops_sass": sass, "achieved_executed": sass * pairs_per_s / 1e12,
                "frac_executed": sass * pairs_per_s / 1e12 / FP32_PEAK_TFLOPS,
                "peak_source": "nominal 2*128*148*1.965 GHz (DESIGN.md section 6); HBM/bf16 peaks do not bound this kernel",
                "kernel_ms": 1e3 * f_avg, "kernel_share_of_step": f_s / dev_s,
                "pairs_per_s": pairs_per_s}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * dev_s / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32 pair math, f64 differences and accumulation",
            "data": "synthetic",
            "config": {"workload": "config4 Plummer+BH-binary N=%d eps=1e-5 order %d all-active block step "
                                   "(select+predict+force+correct)" % (n, order),
                       "n": n, "n_act": n_act, "order": order, "parallelism": "i-shard x%d" % world,
                       "l2": "256 MiB scrub buffer written between steps; state arrays (%.0f MB) exceed L2"
                             % (sum(a.numel() * 8 for a in keep) / 1e6),
                       "force_geometry": geom, "exchange_bytes_per_step": sent},
            "tflops_conventional": value * CONV_FLOPS[order] / 1e12,
            "frac_fp32_peak_nominal": value * CONV_FLOPS[order] / 1e12 / FP32_PEAK_TFLOPS,
            "wall_s": wall, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}
    return g, c, line, (rank, world, n, order, eps2, H, W), (live, keep)


def e2e_leg(args, g, c, order, eps2, H):
    """The same step through the C-ABI host-buffer call: pinned host state in, updated state out, copies timed."""
    import torch
    n = c["n"]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a.cpu().numpy())).pin_memory()
    names = ["t", "dt", "x", "v", "pot"] + ["D%d" % k for k in range(order)]
    src = [g.t, g.dt, g.x, g.v, g.pot, *g.D[:order]]
    keep = {nm: a.cpu().numpy().copy() for nm, a in zip(names, src)}
    hp = {nm: pin(a) for nm, a in zip(names, src)}
    hn = {nm: hp[nm].numpy() for nm in names}
    m = pin(g.m).numpy()
    ctx = g.ctx
    times, up, down = [], 0, 0
    for it in range(1 + max(1, min(args.steps, 3))):
        for nm in names:
            np.copyto(hn[nm], keep[nm])
        t0 = time.perf_counter()
        tn, na, up, down = ctx.step_host(n, order, eps2, g.eta, g.dt_min, g.dt_max, hn["t"], hn["dt"], m, hn["x"],
                                         hn["v"], [hn["D%d" % k] for k in range(order)], hn["pot"])
        dt_ = time.perf_counter() - t0
        assert na == n and tn == H
        if it > 0:
            times.append(dt_)
    return {"value": n * n / statistics.mean(times), "unit": UNIT, "h2d_bytes_per_step": int(up),
            "d2h_bytes_per_step": int(down), "ms_per_step": 1e3 * statistics.mean(times),
            "api": "nbody_step_host (pinned host buffers; H2D + select + predict + force + correct + D2H)"}


def cpu_leg_impl(args, g, c, W, order, eps2, H, keep_state):
    """The oracle on the host cores on a bounded sample of the same step (cpu_baseline), plus a parity spot check of
    the GPU forces of the timed launch configuration (all-active call) on that sample."""
    from oracle import oracle as O
    n = c["n"]
    idx = W.oracle_sample(c, size=min(args.cpu_sample, n))
    t, dt, D = keep_state["t"], keep_state["dt"], keep_state["D"]
    secs, ref = oracle_step(O, c, D, t, dt, idx, order, eps2, H)
    value = idx.shape[0] * n / secs
    sample = "%d i-particles (BHs, innermost/outermost/nearest-to-BH + seeded draw) x all %d j, one step" % (idx.shape[0], n)
    out = {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample,
           "seconds": secs}
    # parity of the timed launch configuration (all-active call) on the sampled outputs
    import torch
    g.ctx.predict(n, H, order, g.t, g.m, g.x, g.v, g.D)
    g.ctx.force(g.all_idx, n, order, eps2, g.acc, g.jerk, g.snap if order >= 6 else None,
                g.crk if order >= 8 else None, g.fpot)
    torch.cuda.synchronize()
    ii = torch.from_numpy(idx.astype(np.int64)).to(g.dev)
    got = [g.acc[ii].cpu().numpy(), g.jerk[ii].cpu().numpy(), g.snap[ii].cpu().numpy() if order >= 6 else None,
           g.crk[ii].cpu().numpy() if order >= 8 else None, g.fpot[ii].cpu().numpy()]
    rel = lambda a, b: float(np.max(np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)))
    par = {"acc": rel(got[0], ref[0]), "jerk": rel(got[1], ref[1]),
           "pot": float(np.max(np.abs(got[4] - ref[4]) / np.abs(ref[4])))}
    if order >= 6:
        par["snap"] = rel(got[2], ref[2])
    if order >= 8:
        par["crackle"] = rel(got[3], ref[3])
    return out, par


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    g, c, line, (rank, world, n, order, eps2, H, W), (live, keep) = run_ours(args)
    if rank == 0:
        import torch
        for dst, src in zip(live, keep):  # back to the pristine all-active state for the two extra legs
            dst.copy_(src)
        torch.cuda.synchronize()
        keep_state = {"t": g.t.cpu().numpy().copy(), "dt": g.dt.cpu().numpy().copy(),
                      "D": [d.cpu().numpy().copy() for d in g.D[:order - 2]]}
        # instruction-class micro-probes (1e12 thread-ops/s, SM MHz inside the probe): context for the roofline
        names = {0: "ffma", 5: "ffma2_two_fresh_operands", 6: "ffma2_three_fresh_operands", 1: "dadd",
                 2: "f2f_f64_f32_roundtrip", 3: "mufu_rsq"}
        names.update({7: "ffma2_plus_shf_pair", 8: "ffma2_plus_dadd_pair", 9: "ffma2_plus_lds128_pair"})
        line["probes_tera_ops"] = {nm: [round(v, 3) for v in g.ctx.probe_peak(k, 150)] for k, nm in names.items()}
        pr, rl = line["probes_tera_ops"], line["roofline"]
        rl["peak_measured"] = 2.0 * pr["ffma"][0]  # Tflop/s of the FFMA probe on this chip, this run
        rl["frac_measured_peak"] = rl["achieved"] / rl["peak_measured"]
        rl["frac_executed_measured"] = rl["achieved_executed"] / rl["peak_measured"]
        # issue-port model: a packed op holds the sub-partition's issue port for 2 cycles (probes 7-9:
        # an instruction of another pipe next to an FFMA2 is NOT hidden behind its second cycle), so one (warp, j) costs at
        # least 2 x packed + other issue cycles for 64 pairs
        cyc = 2 * PACKED_OPS[order] + OTHER_OPS[order]
        bound = 64.0 / cyc * 4 * SM_COUNT * SM_MAX_GHZ * 1e9
        rl["issue_port_model"] = {"cycles_per_warp_j": cyc, "bound_pairs_per_s": bound,
                                  "frac": rl["pairs_per_s"] / bound,
                                  "fma_pipe_floor_pairs_per_s": 64.0 / (2 * PACKED_OPS[order]) * 4 * SM_COUNT * SM_MAX_GHZ * 1e9,
                                  "pair_cost_vs_ffma2": {k: round(pr["ffma2_two_fresh_operands"][0] / pr[k][0], 3)
                                                         for k in ("ffma2_plus_shf_pair", "ffma2_plus_dadd_pair",
                                                                   "ffma2_plus_lds128_pair") if pr[k][0] > 0}}
        if not args.no_e2e:
            line["e2e"] = e2e_leg(args, g, c, order, eps2, H)
        if not args.no_cpu_baseline and world == 1:
            cb, par = cpu_leg_impl(args, g, c, W, order, eps2, H, keep_state)
            line["cpu_baseline"] = cb
            line["parity_sample"] = par
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
