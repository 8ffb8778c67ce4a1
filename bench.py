#!/usr/bin/env python
"""bench.py — events/s of the hot path on B200 (BASELINE.json:metric), with roofline and CPU-oracle baseline.

One "step" = one pass of the whole hot path over one batch of config-3 events (g g -> t tbar g g, sqrt(s) = 1 TeV):
    philox_uniform -> rambo_generate -> apply_cuts -> me_eval
`--workload config4` times vegas_iterate instead (a1-a12 fused; one step = one Vegas iteration).
All inputs are synthetic and seeded (Philox seed 3 / 4), shaped like the paper's LO gg -> ttbar gg benchmark
(PAPER.md:82); there is no dataset.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--events E] [--impl reference]
For N > 1 launch through torch.distributed.run; ranks take disjoint event-index ranges (weak scaling, no
data-path collective — events are independent).
"""
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

METRIC = "gg->ttbar gg |M|^2 events/sec (fp64, 1 B200)"
UNIT = "events/s"
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12  # SMs x DFMA lanes/SM x 2 flop x max SM clock
# dram__bytes_read.sum + dram__bytes_write.sum of me_eval_kernel<gg_ttxgg> per event, from the ncu --set full capture
# of the kernel at HEAD summarised in profiles/r2_me_eval_summary.md (817.7 MB + 37.1 MB for 4 194 304 events;
# algorithmic: 200 B/event)
NCU_DRAM_BYTES_PER_EVENT = {"gg_ttxgg": 202.7, "gg_ttxggg": 228.7, "qqx_ttxgg": 201.4}
NCU_SUMMARY = "profiles/r2_me_eval_summary.md, profiles/r2_n1_n2_summary.md"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "", 1).isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(self.rows[0][1]) if self.rows and self.rows[0][1].isdigit() else None,
                "reasons": sorted(reasons), "samples": len(self.rows), "power_w_max": max(pw) if pw else None}


def oracle_rate(workload, n_sample, first_event=0, blocks=1):
    """Time the tier-1 oracle, as it stands, on the host cores over n_sample events of the workload's own stream:
    `blocks` equally spaced runs of consecutive events starting at first_event (blocks = 1: the first n_sample)."""
    import numpy as np
    from oracle import ref
    w = workload
    per = max(1, n_sample // blocks)
    gap = max(per, (w.n_events - first_event) // blocks)
    r = np.concatenate([ref.philox_uniform(w.seed, 0, first_event + b * gap, w.n_dim, per) for b in range(blocks)])
    n_sample = len(r)
    me = ref.MatrixElementRef(w.process)
    t0 = time.perf_counter()
    mom, wt = ref.rambo_generate(r, w.sqrt_s, w.masses, w.ps_mode)
    ref.cuts(mom, w.is_gluon, 20.0, 0.4)
    out = me.eval(mom)
    dt = time.perf_counter() - t0
    assert np.all(np.isfinite(out))
    return n_sample / dt, dt, ref.get_threads()


def run_reference(args, workload):
    """--impl reference: the oracle on the box's host cores, bounded sample per step (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    rate0, _, cores = oracle_rate(workload, 256)
    budget = float(os.environ.get("MADME_REF_SECONDS", "60"))   # total CPU-arm wall time to aim for
    n = max(256, min(1 << 16, int(rate0 * budget / max(1, args.steps + args.warmup))))
    for _ in range(args.warmup):
        oracle_rate(workload, n)
    t = 0.0
    for k in range(args.steps):
        _, dt, cores = oracle_rate(workload, n, first_event=k * n)
        t += dt
    value = n * args.steps / t
    sample = "%d events/step of %s (Philox seed %d), tier-1 oracle: rambo + cuts + |M|^2" % (n, workload.name, workload.seed)
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": workload.name + " " + workload.process, "events_per_step": n},
                      "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                      "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--events", type=int, default=0, help="events per step per GPU (default: the workload's n_events)")
    ap.add_argument("--workload", default="config3", choices=["config3", "config4", "config4_hadronic", "config2", "config1", "qqx_ttx", "qqx_ttxg", "qg_ttxq",
                                                           "qqx_ttxgg", "qg_ttxqg", "qxg_ttxqxg", "gg_ttxggg"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-vegas-leg", action="store_true", help="skip the config-4 Vegas integration reported beside config 3")
    args = ap.parse_args()

    from paper_2211_14056_b200.workloads import BY_NAME, PARAMS, VEGAS_ALPHA, VEGAS_BINS
    wl = BY_NAME[args.workload]
    if args.impl == "reference":
        run_reference(args, wl)
        return

    import torch
    from paper_2211_14056_b200 import api
    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2211_14056_b200.sharding import weak_shard
    first, n_ev = weak_shard(rank, world, args.events or wl.n_events)  # disjoint global event-index ranges
    h = api.me_init(wl.process, PARAMS)
    stream = torch.cuda.current_stream()
    nf = len(wl.masses)
    vegas = wl.name.startswith("config4")

    # resident buffers
    if vegas:
        grid = api.VegasGrid(wl.n_dim, VEGAS_BINS, VEGAS_ALPHA, wl.seed, wl.ps_mode)
        launches_per_step = 4  # integrand, reduce_chunks, reduce_final, refine
    else:
        rand = torch.empty((n_ev, wl.n_dim), dtype=torch.float64, device="cuda")
        mom = torch.empty((n_ev, nf + 2, 4), dtype=torch.float64, device="cuda")
        wgt = torch.empty(n_ev, dtype=torch.float64, device="cuda")
        passed = torch.empty(n_ev, dtype=torch.int32, device="cuda")
        me2 = torch.empty(n_ev, dtype=torch.float64, device="cuda")
        launches_per_step = 4  # philox, rambo, cuts, me_eval
    me_ms = []

    def step(k, timed):
        if vegas:
            if world > 1:  # strong-sharded iteration over world * n_ev events with the single 3.2 KB exchange (NCCL)
                return api.vegas_iterate_sharded(h, grid, wl.sqrt_s, n_ev * world)
            return api.vegas_iterate(h, grid, wl.sqrt_s, n_ev)
        api.philox_uniform(wl.seed, k, first, wl.n_dim, n_ev, out=rand)
        api.rambo_generate(rand, wl.sqrt_s, wl.masses, wl.ps_mode, momenta=mom, weights=wgt)
        api.apply_cuts(mom, wl.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"], out=passed)
        if timed:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
        api.me_eval(h, mom, me2)
        if timed:
            e1.record(stream)
            me_ms.append((e0, e1))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for k in range(args.warmup):
        step(k, False)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    last = None
    for k in range(args.steps):
        last = step(args.warmup + k, True)
    t1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = torch.tensor([t0.elapsed_time(t1)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_total = float(ms.item())
    value = n_ev * world * args.steps / (ms_total * 1e-3)

    # dominant kernel: me_eval (or the fused integrand), CUDA events on its own stream
    flops_ev = api.me_flops_per_event(h)
    if vegas:   # the roofline is per GPU: this rank's launch evaluated about 1/world of the surviving events
        kern_ms = ms_total / args.steps
        pass_frac = last["n_pass"] / (n_ev * world)
        flops_launch = flops_ev * last["n_pass"] / world
    else:
        kern_ms = sum(a.elapsed_time(b) for a, b in me_ms) / len(me_ms)
        pass_frac = float(passed.float().mean().item())
        flops_launch = flops_ev * n_ev
    achieved = flops_launch / (kern_ms * 1e-3) / 1e12

    # measured fp64 peak: DFMA chain, same process, right after the timed region
    api.fp64_peak_probe(64)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    n_dfma = api.fp64_peak_probe(4096)
    p1.record(stream)
    torch.cuda.synchronize()
    probe_tflops = 2.0 * n_dfma / (p0.elapsed_time(p1) * 1e-3) / 1e12

    # end to end through the public API with HOST buffers: pinned uniforms in, (me2, weight, pass) out, every step
    e2e = None
    if not vegas:
        n_e2e = n_ev          # the same events per step as the device-resident number
        rand_h = torch.empty((n_e2e, wl.n_dim), dtype=torch.float64).pin_memory()
        rand_h.copy_(rand[:n_e2e])
        me2_h = torch.empty(n_e2e, dtype=torch.float64).pin_memory()
        wgt_h = torch.empty(n_e2e, dtype=torch.float64).pin_memory()
        pass_h = torch.empty(n_e2e, dtype=torch.int32).pin_memory()

        # chunked and double-buffered: the H2D copy of chunk k+1 and the D2H copy of chunk k-1 run on their own streams
        # while chunk k is computed (the public API takes a stream; buffers are per chunk, so nothing is overwritten early)
        n_chunks = 8
        cs = n_e2e // n_chunks
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()

        def e2e_step():
            ready = []
            for c in range(n_chunks):
                sl = slice(c * cs, (c + 1) * cs)
                with torch.cuda.stream(s_in):
                    rand[sl].copy_(rand_h[sl], non_blocking=True)
                    ev = torch.cuda.Event()
                    ev.record(s_in)
                    ready.append(ev)
            for c in range(n_chunks):
                sl = slice(c * cs, (c + 1) * cs)
                stream.wait_event(ready[c])
                api.rambo_generate(rand[sl], wl.sqrt_s, wl.masses, wl.ps_mode, momenta=mom[sl], weights=wgt[sl])
                api.apply_cuts(mom[sl], wl.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"], out=passed[sl])
                api.me_eval(h, mom[sl], me2[sl])
                done = torch.cuda.Event()
                done.record(stream)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(done)
                    me2_h[sl].copy_(me2[sl], non_blocking=True)
                    wgt_h[sl].copy_(wgt[sl], non_blocking=True)
                    pass_h[sl].copy_(passed[sl], non_blocking=True)
            fin = torch.cuda.Event()
            fin.record(s_out)
            stream.wait_event(fin)       # the step ends when its results are on the host
            s_in.wait_stream(stream)     # and the next step's uploads may not overwrite inputs still in use
        e2e_step()
        barrier()
        t0.record(stream)
        for _ in range(args.steps):
            e2e_step()
        t1.record(stream)
        barrier()
        ms2 = torch.tensor([t0.elapsed_time(t1)], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(ms2, op=dist.ReduceOp.MAX)
        e2e = {"value": n_e2e * world * args.steps / (float(ms2.item()) * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": rand_h.numel() * 8, "d2h_bytes_per_step": n_e2e * (8 + 8 + 4), "events_per_step": n_e2e}
    else:
        # vegas_iterate takes no bulk input: seeds in, two scalars out; the call itself already ends with a D2H read
        e2e = {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 24,
               "note": "vegas_iterate generates its inputs on the device from the seed; result scalars are read back every step"}

    # config 4 beside the headline: a short extra leg, outside the timed region above — the full
    # Vegas integration of BASELINE.json:configs[4] (5 iterations of the workload's event count, uniform start)
    vegas_leg = None
    if not vegas and world == 1 and wl.name == "config3" and not args.no_vegas_leg:
        from paper_2211_14056_b200.workloads import VEGAS_ITERATIONS
        w4 = BY_NAME["config4"]
        del rand, mom
        torch.cuda.empty_cache()
        n4 = args.events or w4.n_events
        g4 = api.VegasGrid(w4.n_dim, VEGAS_BINS, VEGAS_ALPHA, w4.seed, w4.ps_mode)
        api.me_reserve(h, n4)
        api.vegas_iterate(h, api.VegasGrid(w4.n_dim, VEGAS_BINS, VEGAS_ALPHA, w4.seed, w4.ps_mode), w4.sqrt_s, min(n4, 1 << 20))  # warm-up
        its, evs = [], []
        for _ in range(VEGAS_ITERATIONS):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            its.append(api.vegas_iterate(h, g4, w4.sqrt_s, n4))
            b.record(stream)
            evs.append((a, b))
        torch.cuda.synchronize()
        it_ms = [a.elapsed_time(b) for a, b in evs]
        wts = [1.0 / r["variance"] for r in its]
        comb = sum(r["integral"] * x for r, x in zip(its, wts)) / sum(wts)
        chi2 = sum((r["integral"] - comb) ** 2 * x for r, x in zip(its, wts)) / (len(its) - 1)
        lastv = its[-1]
        tf = flops_ev * lastv["n_pass"] / (it_ms[-1] * 1e-3) / 1e12
        vegas_leg = {"workload": "config4 gg_ttxgg D=%d, %d iterations x %d events, uniform start, seed %d" % (w4.n_dim, len(its), n4, w4.seed),
                     "events_per_s_per_iteration": [n4 / (t * 1e-3) for t in it_ms], "ms_per_iteration": it_ms,
                     "cut_pass_fraction_last": lastv["n_pass"] / n4, "tflops_last": tf, "frac_of_measured_last": tf / probe_tflops,
                     "integral_pb_last": lastv["integral"], "sigma_pb_last": lastv["variance"] ** 0.5,
                     "integral_pb_combined": comb, "sigma_pb_combined": sum(wts) ** -0.5, "chi2_per_dof": chi2}

    # SURVEY §8(f) N1 / N2 beside the headline: me_eval of the quark-initiated 2 -> 4 channels and of g g -> t tbar g g g
    # (the paper's thesis: the gap grows with the number of diagrams), a short extra leg outside the timed
    # region; device-resident RAMBO momenta of each workload's own stream
    channels = None
    if not vegas and world == 1 and wl.name == "config3" and not args.no_vegas_leg:
        channels = {}
        for name in ("qqx_ttxgg", "qg_ttxqg", "gg_ttxggg"):
            wc = BY_NAME[name]
            nc = min(wc.n_events, args.events or wc.n_events)
            hc = api.me_init(wc.process, PARAMS)
            rc = api.philox_uniform(wc.seed, 0, 0, wc.n_dim, nc)
            mc, _ = api.rambo_generate(rc, wc.sqrt_s, wc.masses, wc.ps_mode)
            oc = torch.empty(nc, dtype=torch.float64, device="cuda")
            for _ in range(2):
                api.me_eval(hc, mc, oc)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(3):
                api.me_eval(hc, mc, oc)
            b.record(stream)
            torch.cuda.synchronize()
            msc = a.elapsed_time(b) / 3
            fl = api.me_flops_per_event(hc)
            channels[name] = {"events": nc, "kernel_ms": msc, "events_per_s": nc / (msc * 1e-3), "flops_per_event": fl,
                              "tflops": fl * nc / (msc * 1e-3) / 1e12, "frac_of_measured": fl * nc / (msc * 1e-3) / 1e12 / probe_tflops,
                              "diagrams": api.me_info(hc, 0), "colour_flows": api.me_info(hc, 3), "regs_per_thread": api.me_info(hc, 8),
                              "events_per_cta": api.me_info(hc, 7)}
            del hc, rc, mc, oc
            torch.cuda.empty_cache()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        rate0, _, cores = oracle_rate(wl, 256)
        n_s = int(max(256, min(1 << 16, rate0 * 15.0)))
        rate, dt, cores = oracle_rate(wl, n_s, blocks=64)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "events_per_s_per_core": rate / max(1, cores),
               "sample": "%d events of %s (Philox seed %d) in 64 equally spaced runs over the stream: rambo + cuts + tier-1 |M|^2, %.1f s"
                         % (n_s // 64 * 64, wl.name, wl.seed, dt)}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": "%s %s sqrt_s=%g" % (wl.name, wl.process, wl.sqrt_s), "events_per_step_per_gpu": n_ev,
                      "step": "vegas_iterate (fused a1-a12)" if vegas else "philox_uniform+rambo_generate+apply_cuts+me_eval",
                      "cut_pass_fraction": pass_frac, "l2": "inputs larger than L2 (%.1f GB momenta per step)" % (n_ev * (nf + 2) * 32 / 1e9),
                      "events_per_cta": api.me_info(h, 7), "ctas_per_sm": api.me_info(h, 9), "regs_per_thread": api.me_info(h, 8),
                      "smem_bytes_per_event": api.me_info(h, 6)},
           "roofline": {"bound": "alu", "kernel": "vegas_integrand_kernel" if vegas else "me_eval_kernel", "achieved": achieved,
                        "peak": NOMINAL_FP64_TFLOPS, "unit": "TFLOP/s", "frac": achieved / NOMINAL_FP64_TFLOPS,
                        "peak_source": "nominal fp64: 148 SMs x 64 DFMA lanes x 2 x 1.965 GHz (no fp64 entry in MEASURED_PEAKS.json)",
                        "peak_measured_dfma_chain": probe_tflops, "frac_of_measured": achieved / probe_tflops,
                        "flops_per_event": flops_ev, "kernel_ms": kern_ms,
                        "traffic": (NCU_DRAM_BYTES_PER_EVENT[wl.process] * n_ev if (wl.process in NCU_DRAM_BYTES_PER_EVENT and not vegas) else None),
                        "traffic_unit": "bytes per launch (ncu --set full capture of this kernel, %s)" % NCU_SUMMARY,
                        "hbm_gbs_algorithmic": (32 * (nf + 2) + 8) * n_ev / (kern_ms * 1e-3) / 1e9},
           "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "clocks": clocks}
    if vegas:
        out["vegas"] = last
    elif vegas_leg is not None:
        out["vegas"] = vegas_leg
    if channels:
        out["channels"] = channels
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
