"""Measurement reports for the BASELINE.json configs beyond bench.py's headline:

    python -m paper_1312_1789_b200.report sweep --config {2,3,4} [--n N]
        force throughput per N_act (config 2: 1..65536 x16; config 3: 4^0..4^9; config 4: all-active + the
        log-uniform block-size histogram 2^0..2^20), one JSON line per call class
    python -m paper_1312_1789_b200.report integrate --config 5 [--n N] [--t-end 0.0625] [--order P] [--driver host|device]
        end-to-end block-time-step integration (bootstrap, then select/predict/force/correct per block) with the
        relative energy error, block-size histogram, time split (host driver) and sustained Tflop/s; --driver device
        runs the blocks through nbody_run_blocks (CUDA graph per block step, no host round trip per block)
    python -m paper_1312_1789_b200.report latency [--config 2] [--n 65536] [--order 4] [--blocks 400]
        microseconds per block step over the same run of blocks: host-driven path against the device-driven path

Product code only (no oracle): every step runs through the C ABI.  Inputs are the seeded synthetic clusters of
workloads.py.
"""
import argparse
import json
import sys
import time

import numpy as np

CONV_FLOPS = {4: 60, 6: 97, 8: 144}
FP32_PEAK = 2 * 128 * 148 * 1.965e9


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _time_call(fn, min_reps=3, budget_ms=300.0):
    import torch
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    fn()
    e1.record()
    torch.cuda.synchronize()
    one = e0.elapsed_time(e1)
    reps = int(max(min_reps, min(200, budget_ms / max(one, 1e-3))))
    ts = []
    for _ in range(reps):
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    return float(np.median(ts)), float(np.min(ts)), reps


def sweep(args):
    import torch
    from . import nbody, workloads as W
    c = W.cluster(args.config, args.n)
    n, order, eps2 = c["n"], (args.order or c["order"]), c["eps2"]
    D = W.smooth_field_derivs(c, 6)
    t, dt = W.predictor_times(c["x"])
    t_now = 2.0**-10
    ctx = nbody.Context(n)
    dD = [_dev(d) for d in D[: order - 2]]
    st = (_dev(t), _dev(c["m"]), _dev(c["x"]), _dev(c["v"]))
    pred = lambda: ctx.predict(n, t_now, order, st[0], st[1], st[2], st[3], dD)
    med, best, _ = _time_call(pred)
    bytes_pp = {4: 112 + 48, 6: 160 + 64, 8: 208 + 64}[order]
    print(json.dumps({"call": "predict", "config": args.config, "n": n, "order": order, "us": med * 1e3,
                      "algorithmic_GBps": bytes_pp * n / (med * 1e-3) / 1e9}), flush=True)
    out = [torch.zeros(n, 3, dtype=torch.float64, device="cuda") for _ in range(4)]
    pot = torch.zeros(n, dtype=torch.float64, device="cuda")
    # the other O(N) kernels of a block step on an all-active block: selection (a-1) and corrector (a-4)
    act = torch.zeros(n, dtype=torch.int32, device="cuda")
    d_dt = _dev(dt)
    med, best, _ = _time_call(lambda: ctx.next_block(n, st[0], d_dt, act))
    print(json.dumps({"call": "next_block", "config": args.config, "n": n, "us": med * 1e3, "us_best": best * 1e3,
                      "note": "one kernel + D2H of the 424-byte control block + stream synchronise", "algorithmic_GBps": 20 * n / (med * 1e-3) / 1e9}),
          flush=True)
    full = [_dev(d) for d in (D + [np.zeros_like(D[0])] * 8)[:8]]
    sx, sv, sp, s_t, s_dt = st[2].clone(), st[3].clone(), torch.zeros(n, dtype=torch.float64, device="cuda"), st[0].clone(), d_dt.clone()
    corr = lambda: ctx.correct(act, n, order, t_now, 0.1, 2.0**-30, 2.0**-4, s_t, s_dt, sx, sv, full, sp, dD[0], dD[1],
                               dD[2] if order >= 6 else None, dD[3] if order >= 8 else None, pot)
    med, best, _ = _time_call(corr)
    bytes_pc = {4: 332, 6: 428, 8: 524}[order]
    print(json.dumps({"call": "correct", "config": args.config, "n": n, "order": order, "n_act": n, "us": med * 1e3,
                      "us_best": best * 1e3, "algorithmic_GBps": bytes_pc * n / (med * 1e-3) / 1e9}), flush=True)
    rng = W.rng_for(args.config, 41)
    if args.config == 2:
        nacts = [1, 16, 256, 4096, 65536]
    elif args.config == 3:
        nacts = [4**k for k in range(10)]
    elif args.config == 5:
        nacts = [1, 16, 256, 4096, 65536, n]
    else:
        nacts = [n]
    for n_act in nacts:
        n_act = min(n_act, n)
        idx = _dev(W.active_list(n, n_act, rng))
        f = lambda: ctx.force(idx, n_act, order, eps2, out[0], out[1], out[2] if order >= 6 else None,
                              out[3] if order >= 8 else None, pot)
        med, best, reps = _time_call(f)
        ips = n_act * n / (med * 1e-3)
        print(json.dumps({"call": "force", "config": args.config, "n": n, "order": order, "n_act": n_act,
                          "us_median": med * 1e3, "us_best": best * 1e3, "reps": reps, "interactions_per_s": ips,
                          "tflops_conventional": ips * CONV_FLOPS[order] / 1e12,
                          "frac_fp32_peak": ips * CONV_FLOPS[order] / FP32_PEAK,
                          "geometry": ctx.last_force_geometry()}), flush=True)
    if args.config == 4:
        sizes = W.block_histogram(n, 64, rng)
        tot_pairs, tot_ms, per_decade = 0, 0.0, {}
        for n_act in sizes:
            n_act = int(n_act)
            idx = _dev(W.active_list(n, n_act, rng))
            f = lambda: ctx.force(idx, n_act, order, eps2, out[0], out[1], out[2], None, pot)
            med, _, _ = _time_call(f, min_reps=3, budget_ms=30.0)
            tot_pairs += n_act * n
            tot_ms += med
            d = per_decade.setdefault(len(str(n_act)) - 1, [0, 0.0, 0])
            d[0] += n_act * n
            d[1] += med
            d[2] += 1
        print(json.dumps({"call": "force_histogram", "config": 4, "n": n, "order": order, "calls": len(sizes),
                          "sum_pairs": tot_pairs, "sum_ms": tot_ms, "interactions_per_s": tot_pairs / (tot_ms * 1e-3),
                          "per_decade_interactions_per_s": {"1e%d" % k: v[0] / (v[1] * 1e-3) for k, v in
                                                            sorted(per_decade.items())},
                          "per_decade_calls": {"1e%d" % k: v[2] for k, v in sorted(per_decade.items())}}), flush=True)
    ctx.close()


def integrate(args):
    import torch
    from . import workloads as W
    from .scheduler import Integrator
    c = W.cluster(args.config, args.n)
    order = args.order or c["order"]
    n, eps2 = c["n"], c["eps2"]
    g = Integrator(c["m"], c["x"], c["v"], order, eps2, eta=args.eta, dt_min=2.0**-args.dt_min_log2,
                   dt_max=2.0**-args.dt_max_log2, step_reject_ratio=args.reject_ratio,
                   corrector_order_limit=args.limit_order)
    t0 = time.perf_counter()
    g.bootstrap()
    torch.cuda.synchronize()
    t_boot = time.perf_counter() - t0
    e0 = g.energy()
    torch.cuda.synchronize()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    marks, hist = [], {}
    w0 = time.perf_counter()
    pairs, rejected, limited = 0, 0, 0
    if args.driver == "device":
        while True:
            r = g.run(args.t_end, max_blocks=1 << 16)
            pairs += r["pairs"]
            rejected += r["rejected"]
            limited += r["limited"]
            for k, v in enumerate(r["hist_log2"]):
                if v:
                    hist[k] = hist.get(k, 0) + v
            if r["stop_reason"] != 3 or (time.perf_counter() - w0) > args.max_seconds:
                break
    else:
        while True:
            t_next, n_act = g.ctx.next_block(n, g.t, g.dt, g.active)
            if t_next > args.t_end or (time.perf_counter() - w0) > args.max_seconds:
                break
            p = order
            a, b, cc, d = ev(), ev(), ev(), ev()
            a.record()
            g.ctx.predict(n, t_next, p, g.t, g.m, g.x, g.v, g.D)
            b.record()
            g.ctx.force(g.active, n_act, p, eps2, g.acc, g.jerk, g.snap if p >= 6 else None, g.crk if p >= 8 else None,
                        g.fpot)
            cc.record()
            g.ctx.correct(g.active, n_act, p, t_next, g.eta, g.dt_min, g.dt_max, g.t, g.dt, g.x, g.v, g.D, g.pot, g.acc,
                          g.jerk, g.snap if p >= 6 else None, g.crk if p >= 8 else None, g.fpot)
            d.record()
            marks.append((a, b, cc, d))
            g.time = t_next
            g.blocks += 1
            pairs += n_act * n
            k = int(n_act).bit_length() - 1
            hist[k] = hist.get(k, 0) + 1
    torch.cuda.synchronize()
    wall = time.perf_counter() - w0
    if args.driver == "host":
        rejected, limited = g.ctx.step_counters()
    t_pred = sum(a.elapsed_time(b) for a, b, _, _ in marks) * 1e-3
    t_force = sum(b.elapsed_time(cc) for _, b, cc, _ in marks) * 1e-3
    t_corr = sum(cc.elapsed_time(d) for _, _, cc, d in marks) * 1e-3
    done = bool((g.t == args.t_end).all())
    e1 = g.energy() if bool((g.t == g.t[0]).all()) else float("nan")
    dts = g.dt.cpu().numpy()
    print(json.dumps({"call": "integrate", "driver": args.driver, "config": args.config, "n": n, "order": order, "eta": args.eta,
                      "dt_criterion_order": g.dt_criterion_order, "step_reject_ratio": args.reject_ratio,
                      "rejected_steps": rejected, "corrector_order_limit": args.limit_order, "order_limited_steps": limited, "dt_max_log2": -args.dt_max_log2, "t_end": args.t_end, "reached_t_end": done,
                      "time_reached": g.time, "blocks": g.blocks, "pairs": pairs, "wall_s": wall,
                      "bootstrap_s": t_boot,
                      "split_s": ({"predict": t_pred, "force": t_force, "correct": t_corr,
                                   "host_and_selection": wall - t_pred - t_force - t_corr} if marks else None),
                      "sustained_tflops_conventional": pairs * CONV_FLOPS[order] / wall / 1e12,
                      "sustained_frac_fp32_peak": pairs * CONV_FLOPS[order] / wall / FP32_PEAK,
                      "force_only_tflops": (pairs * CONV_FLOPS[order] / max(t_force, 1e-9) / 1e12) if marks else None,
                      "E0": e0, "E1": e1, "rel_energy_error": abs((e1 - e0) / e0),
                      "block_size_histogram_log2": {str(k): v for k, v in sorted(hist.items())},
                      "dt_log2_min_median_max": [float(np.log2(dts.min())), float(np.log2(np.median(dts))),
                                                 float(np.log2(dts.max()))]}), flush=True)


def latency(args):
    """us per SMALL block step (n_act <= --small): the host-driven path (one selection round trip and 4-5 launches per
    block) against the device-driven path (nbody_run_blocks), over the same sequence of blocks.  Larger blocks in
    between are stepped untimed.  Wall-clock around synchronised calls."""
    import torch
    from . import workloads as W
    from .scheduler import Integrator
    c = W.cluster(args.config, args.n)
    order = args.order or c["order"]
    mk = lambda: Integrator(c["m"], c["x"], c["v"], order, c["eps2"], dt_max=2.0**-args.dt_max_log2)
    res = {}
    if args.synthetic:
        # A run of small blocks only: `synthetic` particles nearest the centre restart on steps of 2^-16 while everybody
        # else waits on 2^-4, so every block until t = 2^-4 is a subset of those particles (their steps grow back to the
        # criterion's value on the way).  One call per driver over exactly the same blocks.
        r0 = np.argsort(np.linalg.norm(c["x"], axis=1))[: args.synthetic]
        for driver in ("host", "device", "device_nograph", "device_fused"):
            g = mk()
            g.bootstrap()
            g.dt.fill_(2.0**-4)
            g.dt[torch.from_numpy(r0).cuda()] = 2.0**-16
            if driver == "device_nograph":
                g.ctx.set_option("use_graph", 0)
            if driver == "device_fused":
                g.ctx.set_option("use_fused", 1)
            t_stop = 2.0**-4 - 2.0**-17
            g.run(t_stop, max_blocks=args.skip)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if driver == "host":
                b0 = g.blocks
                g.integrate(t_stop, max_blocks=g.blocks + args.blocks)
                torch.cuda.synchronize()
                nb = g.blocks - b0
            else:
                nb = g.run(t_stop, max_blocks=args.blocks)["blocks"]
                torch.cuda.synchronize()
            dt_ = time.perf_counter() - t0
            res[driver] = dict(us_per_block=1e6 * dt_ / max(1, nb), blocks=nb)
            g.ctx.close()
        print(json.dumps({"call": "latency_small_blocks_only", "config": args.config, "n": c["n"], "order": order,
                          "n_act_max": args.synthetic, **res}), flush=True)
        return
    for driver in ("host", "device", "device_nograph"):
        g = mk()
        g.bootstrap()
        if driver == "device_nograph":
            g.ctx.set_option("use_graph", 0)
        g.run(1e9, max_blocks=args.skip)  # leave the synchronised start-up blocks behind
        torch.cuda.synchronize()
        small, t_small, big, sizes = 0, 0.0, 0, []
        while small < args.blocks:
            if driver == "host":
                t0 = time.perf_counter()
                t_next, n_act = g.ctx.next_block(g.n, g.t, g.dt, g.active)
                p = order
                g.ctx.predict(g.n, t_next, p, g.t, g.m, g.x, g.v, g.D)
                g.ctx.force(g.active, n_act, p, g.eps2, g.acc, g.jerk, g.snap if p >= 6 else None,
                            g.crk if p >= 8 else None, g.fpot)
                g.ctx.correct(g.active, n_act, p, t_next, g.eta, g.dt_min, g.dt_max, g.t, g.dt, g.x, g.v, g.D, g.pot,
                              g.acc, g.jerk, g.snap if p >= 6 else None, g.crk if p >= 8 else None, g.fpot)
                torch.cuda.synchronize()
                dt_ = time.perf_counter() - t0
                if n_act <= args.small:
                    small += 1
                    t_small += dt_
                    sizes.append(n_act)
                else:
                    big += 1
            else:
                t0 = time.perf_counter()
                r = g.run(1e9, max_blocks=args.blocks - small, max_n_act=args.small)
                torch.cuda.synchronize()
                t_small += time.perf_counter() - t0
                small += r["blocks"]
                if r["stop_reason"] == 2:
                    g.block_step()
                    big += 1
        res[driver] = dict(us_per_small_block=1e6 * t_small / max(1, small), small_blocks=small, larger_blocks_between=big)
        if sizes:
            res[driver]["median_n_act"] = float(np.median(sizes))
        g.ctx.close()
    print(json.dumps({"call": "latency", "config": args.config, "n": c["n"], "order": order, "small": args.small,
                      "skipped": args.skip, **res}), flush=True)


def main(argv=None):
    ap = argparse.ArgumentParser(prog="paper_1312_1789_b200.report")
    sub = ap.add_subparsers(dest="cmd", required=True)
    s = sub.add_parser("sweep")
    s.add_argument("--config", type=int, required=True, choices=[2, 3, 4, 5])
    s.add_argument("--n", type=int, default=None)
    s.add_argument("--order", type=int, default=None)
    i = sub.add_parser("integrate")
    i.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    i.add_argument("--n", type=int, default=None)
    i.add_argument("--order", type=int, default=None)
    i.add_argument("--t-end", type=float, default=0.0625)
    i.add_argument("--eta", type=float, default=0.1)
    i.add_argument("--dt-min-log2", type=int, default=30)
    i.add_argument("--dt-max-log2", type=int, default=4, help="dt_max = 2^-k (must divide t_end)")
    i.add_argument("--max-seconds", type=float, default=1500.0)
    i.add_argument("--driver", default="host", choices=["host", "device"])
    i.add_argument("--reject-ratio", type=int, default=0, help="R14 a-posteriori step rejection (0 = off)")
    i.add_argument("--limit-order", type=int, default=0, help="R15 corrector order limiter (0 = off, 1 = on)")
    l = sub.add_parser("latency")
    l.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    l.add_argument("--n", type=int, default=65536)
    l.add_argument("--order", type=int, default=None)
    l.add_argument("--blocks", type=int, default=400)
    l.add_argument("--skip", type=int, default=50)
    l.add_argument("--small", type=int, default=16, help="blocks up to this size are timed")
    l.add_argument("--synthetic", type=int, default=0, help="K > 0: a run in which every block has <= K particles")
    l.add_argument("--dt-max-log2", type=int, default=4)
    args = ap.parse_args(argv)
    {"sweep": sweep, "integrate": integrate, "latency": latency}[args.cmd](args)


if __name__ == "__main__":
    main()
