#!/usr/bin/env python
"""bench.py -- throughput of the data-parallel matrix-element hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--precision d|f|m] [--impl reference]

One "step" = one pass of the whole hot path over one batch of synthetic input resident in HBM: on-device Philox +
RAMBO sampler (a0), selection uniforms, then mg_compute (a1-a10: wavefunctions, diagrams, colour sum, helicity sum,
helicity/colour selection, store).  The helicity filter (a9) runs once before the timed region (one-off).
`value` = events / step time (matrix elements per second, whole job); `e2e` = the same through mg_compute_host with
pinned HOST buffers (H2D of momenta and uniforms, compute, D2H of ME and selected indices inside the timed region).
For N > 1 (torchrun) every rank evaluates its own contiguous range of global event indices (weak scaling, no
data-path collective); the good-helicity mask is agreed once by an all-reduce before the timed region.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the same
workload.  Prints ONE JSON line.
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

from paper_2507_21039_b200.workloads import WORKLOADS, SM_PARAMS, PRECISION_CODE  # noqa: E402

# nominal B200 peaks of the plain ALU pipes: 148 SMs x lanes x 2 flop x 1.965 GHz
NOMINAL_PEAK_TFLOPS = {"f64": 148 * 64 * 2 * 1.965e9 / 1e12, "f32": 148 * 128 * 2 * 1.965e9 / 1e12}
ORACLE_SAMPLE = {1: 16384, 2: 524288, 3: 262144, 4: 65536, 5: 4096}      # events per CPU sample (about 10-30 s of CPU work)


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=10)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(self.rows)}


def run_oracle_sample(cfg, nsample, first=0):
    """Time the oracle (as it stands) on `nsample` events of the workload; returns (MEs/s, seconds, threads)."""
    from oracle import binding as O
    wl = WORKLOADS[cfg]
    p, _ = O.rambo(wl.seed, first, nsample, wl.final_masses, wl.sqrt_s)
    u = O.uniforms(wl.seed, first, nsample, 0, 1)
    t0 = time.perf_counter()
    p, _ = O.rambo(wl.seed, first, nsample, wl.final_masses, wl.sqrt_s)
    me, mh2, wcol = O.matrix_elements(wl.process, p, sm=SM_PARAMS)
    O.select(u[:, 0], mh2)
    O.select(u[:, 1], wcol)
    dt = time.perf_counter() - t0
    return nsample / dt, dt, O.num_threads()


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    wl = WORKLOADS[cfg]
    n = ORACLE_SAMPLE[cfg]
    from oracle import binding as O
    O.lib()
    for _ in range(max(1, min(args.warmup, 1))):
        run_oracle_sample(cfg, max(16, n // 8))
    rates, secs = [], []
    steps = min(args.steps, 3)
    for s in range(steps):
        r, dt, nth = run_oracle_sample(cfg, n, first=s * n)
        rates.append(r)
        secs.append(dt)
    value = sum(rates) / len(rates)
    sample = "%d events per step (global indices from 0) of config %d, %d steps" % (n, cfg, steps)
    line = {"impl": "reference", "metric": "matrix elements/s", "value": value, "unit": "MEs/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": 1, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "cfg%d %s, %d events, FP64" % (cfg, wl.name, wl.nevt), "sample": sample},
            "cpu_baseline": {"value": value, "unit": "MEs/s", "cores": nth, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "MEs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# the whole metric (BASELINE.json: "matrix elements/s (FP64, FP32) per process"): every (config, precision) cell it names
PER_CONFIG_CELLS = [(1, "d"), (2, "d"), (3, "d"), (4, "d"), (5, "d"), (2, "f"), (3, "f"), (4, "f"), (5, "f"), (3, "m"),
                    (2, "a"), (3, "a"), (4, "a"), (5, "a"),          # a: the all-FP32 variant, reported beside f
                    (6, "d"), (7, "d"), (8, "d"), (9, "d")]          # Drell-Yan u u~ -> e+ e- + 0..3 g (not a BASELINE config)


def _stats(xs):
    n = len(xs)
    mean = sum(xs) / n
    var = sum((x - mean) ** 2 for x in xs) / (n - 1) if n > 1 else 0.0
    return mean, var ** 0.5


def measure_cell(B, torch, dev, local, cfg, prec, flush, reps=10, warmup=3, e2e_reps=3):
    """One (config, precision) cell at the config's batch size: mg_compute alone and sampler + mg_compute (the paper's throughput
    definition), each as mean +- std over `reps` repetitions timed one by one with CUDA events,
    the amplitude kernel's own time, the roofline fraction and the host-buffer (e2e) rate."""
    wl = WORKLOADS[cfg]
    nevt, lay = wl.nevt, B.MG_LAYOUT_AOS
    ctx = B.Context(wl.process, SM_PARAMS, PRECISION_CODE[prec], local)
    mom, _ = ctx.sample_rambo(wl.seed, 0, nevt, wl.sqrt_s, layout=lay, want_weight=False)
    rh, rc = ctx.sample_uniforms(wl.seed, 0, nevt)
    me = torch.empty(nevt, dtype=torch.float64, device=dev)
    sh = torch.empty(nevt, dtype=torch.int32, device=dev)
    sc = torch.empty(nevt, dtype=torch.int32, device=dev)
    ngood, _ = ctx.filter_helicities(mom, min(nevt, 16384), layout=lay)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def compute():
        ctx.compute(mom, nevt, layout=lay, rnd_hel=rh, rnd_col=rc, me=me, sel_hel=sh, sel_col=sc)

    def sample_compute():
        ctx.sample_rambo(wl.seed, 0, nevt, wl.sqrt_s, layout=lay, momenta=mom, want_weight=False)
        ctx.sample_uniforms(wl.seed, 0, nevt, rnd_hel=rh, rnd_col=rc)
        compute()

    def timed(fn):
        for _ in range(warmup):
            fn()
        out = []
        for _ in range(reps):
            flush.zero_()
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            out.append(e0.elapsed_time(e1))
        return out

    ctx.kernel_time_ms()
    ctx.enable_kernel_timing(True)
    t_c = timed(compute)
    kms, kn = ctx.kernel_time_ms()
    ctx.enable_kernel_timing(False)
    t_sc = timed(sample_compute)
    hmom, hrh, hrc = mom.cpu().pin_memory(), rh.cpu().pin_memory(), rc.cpu().pin_memory()
    hme = torch.empty(nevt, dtype=torch.float64).pin_memory()
    hsh = torch.empty(nevt, dtype=torch.int32).pin_memory()
    hsc = torch.empty(nevt, dtype=torch.int32).pin_memory()
    t_e = timed(lambda: ctx.compute_host(hmom, nevt, layout=lay, rnd_hel=hrh, rnd_col=hrc, me=hme, sel_hel=hsh, sel_col=hsc))[:max(e2e_reps, 1)]
    info = ctx.info
    dtype = {"d": "f64", "f": "f32", "m": "f64", "a": "f32"}[prec]
    kavg = kms / max(kn, 1)
    mc, sc_ = _stats(t_c)
    ms_, ss_ = _stats(t_sc)
    mean_e, _ = _stats(t_e)
    achieved = info.flops_per_event * nevt / (kavg * 1e-3) / 1e12
    ctx.close()
    return {"config": cfg, "process": wl.name, "precision": prec, "nevt": nevt, "ngood": ngood, "reps": reps,
            "mes_per_s": nevt / (mc * 1e-3), "ms_compute_mean": mc, "ms_compute_std": sc_,
            "mes_per_s_with_sampler": nevt / (ms_ * 1e-3), "ms_sampler_compute_mean": ms_, "ms_sampler_compute_std": ss_,
            "kernel_ms": kavg, "flops_per_event_executed": info.flops_per_event, "tflops": achieved,
            "frac": achieved / NOMINAL_PEAK_TFLOPS[dtype], "peak_dtype": dtype,
            "e2e_mes_per_s": nevt / (mean_e * 1e-3), "e2e_ms": mean_e}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config 1..5 (default 5: g g -> t t~ g g g); 6..9: u u~ -> e+ e- + 0..3 g")
    ap.add_argument("--precision", default="d", choices=["d", "f", "m", "a"], help="d FP64, f FP32, m mixed, a all-FP32")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (all other cells of the metric)")
    ap.add_argument("--nevt", type=int, default=0, help="override the batch size (profiling only; the headline uses the config's size)")
    args = ap.parse_args()
    if args.impl == "reference":
        reference_arm(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2507_21039_b200 import binding as B
    from paper_2507_21039_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d: launch N > 1 as `python -m torch.distributed.run --nnodes=1 "
                         "--nproc-per-node N --master-addr 127.0.0.1 bench.py --gpus N ...` (one rank per GPU)" % (args.gpus, world))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg, prec = args.config, args.precision
    wl = WORKLOADS[cfg]
    nevt = args.nevt or wl.nevt                 # per GPU (weak scaling)
    first = rank * nevt                         # global event index of this rank's shard
    ctx = B.Context(wl.process, SM_PARAMS, PRECISION_CODE[prec], local)
    info = ctx.info
    lay = B.MG_LAYOUT_AOS

    mom = torch.empty(ctx.mom_shape(nevt, lay), dtype=torch.float64, device=dev)
    rh = torch.empty(nevt, dtype=torch.float64, device=dev)
    rc = torch.empty(nevt, dtype=torch.float64, device=dev)
    me = torch.empty(nevt, dtype=torch.float64, device=dev)
    sh = torch.empty(nevt, dtype=torch.int32, device=dev)
    sc = torch.empty(nevt, dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    # one-off helicity filter on a first batch; ranks agree on the mask (the only exchange of the path)
    ctx.sample_rambo(wl.seed, first, nevt, wl.sqrt_s, layout=lay, momenta=mom, want_weight=False)
    ngood, good = ctx.filter_helicities(mom, min(nevt, 16384), layout=lay)
    if world > 1:
        m = torch.tensor(list(good), dtype=torch.uint8, device=dev)
        sharding.merge_good_masks(m)
        good = bytes(m.cpu().tolist())
        ngood = ctx.set_good_helicities(good)              # every rank sums over the union

    def step():
        flush.zero_()                                                     # L2 flush between steps
        ctx.sample_rambo(wl.seed, first, nevt, wl.sqrt_s, layout=lay, momenta=mom, want_weight=False)
        ctx.sample_uniforms(wl.seed, first, nevt, rnd_hel=rh, rnd_col=rc)
        ctx.compute(mom, nevt, layout=lay, rnd_hel=rh, rnd_col=rc, me=me, sel_hel=sh, sel_col=sc)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ctx.kernel_time_ms()                         # clear
    ctx.enable_kernel_timing(True)
    clocks = ClockSampler(local)
    clocks.start()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = ctx.launch_count() - l0
    clk = clocks.stop()
    kms, kn = ctx.kernel_time_ms()
    ctx.enable_kernel_timing(False)
    ms_total = sharding.max_over_ranks(ms_total, device=dev)
    ms_step = ms_total / args.steps
    value = world * nevt / (ms_step * 1e-3)

    # end to end through the host-buffer entry point (pinned memory)
    hmom = mom.cpu().pin_memory()
    hrh, hrc = rh.cpu().pin_memory(), rc.cpu().pin_memory()
    hme = torch.empty(nevt, dtype=torch.float64).pin_memory()
    hsh = torch.empty(nevt, dtype=torch.int32).pin_memory()
    hsc = torch.empty(nevt, dtype=torch.int32).pin_memory()
    e2e_steps = max(3, min(args.steps, 5))
    for _ in range(2):
        ctx.compute_host(hmom, nevt, layout=lay, rnd_hel=hrh, rnd_col=hrc, me=hme, sel_hel=hsh, sel_col=hsc)
    barrier()
    e0.record()
    for _ in range(e2e_steps):
        flush.zero_()
        ctx.compute_host(hmom, nevt, layout=lay, rnd_hel=hrh, rnd_col=hrc, me=hme, sel_hel=hsh, sel_col=hsc)
    e1.record()
    barrier()
    e2e_ms = sharding.max_over_ranks(e0.elapsed_time(e1), device=dev) / e2e_steps
    assert torch.equal(hme, me.cpu()), "host-buffer path disagrees with the device path"
    h2d = hmom.numel() * 8 + 2 * nevt * 8
    d2h = nevt * 8 + 2 * nevt * 4

    if rank == 0:
        dtype = {"d": "f64", "f": "f32", "m": "f64", "a": "f32"}[prec]
        fl_exec, fl_canon = info.flops_per_event, info.flops_per_event_canonical
        kavg_ms = kms / max(kn, 1)
        achieved = fl_exec * nevt / (kavg_ms * 1e-3) / 1e12
        peak = NOMINAL_PEAK_TFLOPS[dtype]
        measured_peak = ctx.measure_fma_peak(B.MG_FP64 if dtype == "f64" else B.MG_FP32, 50.0)
        traffic = None
        tpath = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tpath):
            traffic = json.load(open(tpath)).get("cfg%d_%s" % (cfg, prec))
        line = {
            "metric": "matrix elements/s", "value": value, "unit": "MEs/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic",
            "config": {"workload": "cfg%d %s, %d events per GPU, precision %s, sqrt(s)=%g GeV, Philox seed %d" % (cfg, wl.name, nevt, prec, wl.sqrt_s, wl.seed),
                       "step": "mg_sample_rambo + mg_sample_uniforms + mg_compute on device buffers; helicity filter once before timing",
                       "parallelism": "events sharded by global index, no collective in the step" if world > 1 else "1 GPU",
                       "l2": "256 MiB buffer zeroed between steps (inside the timed region)", "layout": "AOS", "ngood": ngood,
                       "flops_per_event_executed": fl_exec, "flops_per_event_canonical": fl_canon},
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": traffic, "kernel": "mg_vm_kernel" if cfg > 1 else "mg_ee_kernel", "kernel_ms": kavg_ms, "kernel_launches": kn,
                         "kernel_share_of_step": kavg_ms / ms_step,
                         "peak_kind": "nominal FMA peak (148 SMs x %d lanes x 2 x 1.965 GHz); MEASURED_PEAKS.json has no %s ALU figure" % (64 if dtype == "f64" else 128, dtype),
                         "peak_measured_fma_chain": measured_peak, "frac_of_measured": achieved / measured_peak if measured_peak else None,
                         "canonical_equivalent_tflops": fl_canon * nevt / (kavg_ms * 1e-3) / 1e12},
            "e2e": {"value": world * nevt / (e2e_ms * 1e-3), "unit": "MEs/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms, "call": "mg_compute_host (pinned host buffers)"},
            "gpu_launches": launches, "clocks": clk,
        }
        if world == 1 and not args.no_per_config:
            cells = []
            for c, pr in PER_CONFIG_CELLS:
                cells.append(measure_cell(B, torch, dev, local, c, pr, flush))
            line["per_config"] = cells
        if world == 1 and not args.no_cpu_baseline:
            n = ORACLE_SAMPLE[cfg]
            r, dt, nth = run_oracle_sample(cfg, n)
            line["cpu_baseline"] = {"value": r, "unit": "MEs/s", "cores": nth, "kind": "oracle",
                                    "sample": "first %d events of the workload, %.1f s" % (n, dt)}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
