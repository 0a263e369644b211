#!/usr/bin/env python
"""bench.py -- throughput of the de-dispersion hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]
                    [--shard beam|dm] [--no-all-configs] [--no-cpu-baseline] [--no-e2e]

A step is one pass of the hot path over one batch of synthetic filterbank data: for the brute-force
workloads one dedisp_execute (SURVEY.md section 8 rows a2/a3 with the plan's a1 table), for cfg4 the two
subband stages (a4+a5), for cfg5 one streaming push of all beams (a3+a6).  The default workload is
BASELINE.json's 4096-DM L-band configuration (cfg3), the one the north-star target is quoted on; the
default run also measures the other four configurations (shorter: `all_configs`) and the register-only
FP32 add microbenchmark that gives the roofline its measured denominator (`fadd_microbench`).

metric  = DM*sample*channel adds per second (nDM * n_out * nchans * nbeams / t), inputs resident
          in HBM, CUDA events on the launching stream, max over ranks.
e2e     = same metric through the C ABI's host-buffer entry (pinned host in/out, H2D and D2H inside
          the timed region); e2e_events = the same with dedisp_execute_detect_host, which ships the
          events instead of the de-dispersed buffer.
roofline: the path is bound by the FP32 add pipe (gather-and-add, no tensor cores); peak =
          SMs * 128 lanes * max SM clock, peak_measured = the microbenchmark.
          frac is taken on the whole device step of the window path (pair-forming pre-pass included).
N > 1   : --shard beam (default): every rank de-disperses its own beam of the same workload, weak
          scaling.  --shard dm: every rank gets the SAME input and a contiguous slice of the DM list
          (PAPER.md:74), strong scaling.  No data-path collective either way; value = adds of all
          ranks / max over ranks of the device time.
"""
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

from paper_1107_2516_b200 import shard, synth  # noqa: E402  (input generators / rank bookkeeping, no arithmetic)

METRIC = "DM*sample*channel adds/s"
UNIT = "adds/s"
WORKLOADS = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, dev):
        self.dev, self.rows, self.proc = dev, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.dev), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [f.strip() for f in line.split(",")]))

    def window(self, t0, t1):
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.05] or [r for (_, r) in self.rows[-3:]]
        sm, mx, pw, reasons = [], [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w": float(np.median(pw)) if pw else None, "samples": len(sm),
                "reasons": sorted(reasons)}

    def stop(self):
        if self.proc:
            self.proc.terminate()


def oracle_sample(cf, budget_adds=3.0e11):
    """A bounded sample of the workload for the CPU oracle: brute-force configs -- every s-th DM row, a
    prefix of the time axis, one beam; the subband config -- a few whole coarse groups on a prefix of the
    time axis through the two-stage oracle.  Sized to about budget_adds additions of the metric."""
    from oracle import dedisp_oracle as orc
    orc.build()
    if cf.nsub:
        n_out = min(cf.n_out, 16384)
        ncoarse = cf.ndm // cf.nfine
        ng = int(min(ncoarse, max(1, budget_adds / (float(n_out) * cf.nchans * cf.nfine))))
        groups = sorted(set(np.linspace(0, ncoarse - 1, ng).astype(int).tolist()))
        tab = orc.subband_tables(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list, cf.nsub, cf.nfine)
        x = synth.make_input(cf, n_out + tab.max_delay)
        desc = "%d of %d coarse groups x %d of %d samples x %d channels, two-stage subband oracle; adds counted as the metric does (nDM*n_out*nchans)" % (
            len(groups), ncoarse, n_out, cf.n_out, cf.nchans)

        def run():
            orc.subband(x, tab, n_out, groups=groups, want_sumabs=False)
        return run, float(len(groups)) * cf.nfine * n_out * cf.nchans, desc, orc.num_threads()
    n_out = min(cf.n_out, 65536)
    rows = max(1, int(budget_adds / (float(n_out) * cf.nchans)))
    rows = min(rows, cf.ndm)
    idx = np.unique(np.linspace(0, cf.ndm - 1, rows).astype(np.int64))
    dm = cf.dm_list[idx]
    tab = orc.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm)
    n_in = n_out + int(tab.max())
    x = synth.make_input(cf, n_in)
    desc = "%d of %d DM rows (evenly spaced) x %d of %d samples x %d channels, 1 beam, %s" % (
        len(idx), cf.ndm, n_out, cf.n_out, cf.nchans, "brute force")

    def run():
        if cf.dtype == "u8":
            orc.brute_u8(x, tab, n_out)
        else:
            orc.brute_f32(x, tab, n_out, want_sumabs=False)
    return run, float(len(idx)) * n_out * cf.nchans, desc, orc.num_threads()


def run_reference(args, cf):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    run, adds, desc, cores = oracle_sample(cf, budget_adds=1.5e10)
    for _ in range(min(args.warmup, 1)):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = time.perf_counter() - t0
    v = adds * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64" if cf.dtype == "f32" else "int64",
            "data": "synthetic", "config": {"workload": cf.name, "sample": desc},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


class Ctx:
    """What every measurement needs: torch, the binding, rank bookkeeping, peaks, the clock sampler."""


def fadd_leg(ctx):
    """Register-only add.f32x2 / add.f32 microbenchmark through the ABI."""
    dd, pk = ctx.dd, ctx.pk
    res = {}
    for name, packed in (("add.f32x2", True), ("add.f32", False)):
        dd.fadd_microbench(packed, iters=2000, repeats=1)
        w0 = time.time()
        ms, adds, nsm = dd.fadd_microbench(packed, iters=20000, repeats=8)
        w1 = time.time()
        ck = ctx.sampler.window(w0, w1) if ctx.sampler else {}
        mhz = ck.get("sm_mhz") or pk["sm_max_mhz"]
        res[name] = {"ms": ms, "adds": adds, "adds_per_s": adds / (ms * 1e-3),
                     "adds_per_clk_per_sm": adds / (ms * 1e-3) / (nsm * mhz * 1e6), "sm_mhz": mhz,
                     "clock_source": "nvidia-smi during the run" if ck.get("sm_mhz") else "clocks.max.sm (no sample)"}
    best = max(res.values(), key=lambda r: r["adds_per_s"])
    return {"kernels": res, "peak_measured_adds_per_s": best["adds_per_s"], "nominal_adds_per_clk_per_sm": 128,
            "how": "dedisp_fadd_microbench: 32 warps per SM, 64 independent fp32 accumulators per thread, 20000 x 8 launches"}


def measure(ctx, cf, args, steps, warmup, primary):
    """One workload: device-resident steps, dominant-kernel timing, e2e, (primary only) the side legs."""
    torch, dd, dist = ctx.torch, ctx.dd, ctx.dist
    world, rank, local, pk = ctx.world, ctx.rank, ctx.local, ctx.pk
    dm_shard = args.shard == "dm" and world > 1
    dm_list = cf.dm_list
    lo, hi = 0, cf.ndm
    if dm_shard:
        lo, hi = shard.dm_slice(cf.ndm, world, rank, multiple=cf.nfine if cf.nsub else 1)
        dm_list = dm_list[lo:hi]
    pa = cf.plan_args()
    pa["dm_list"] = dm_list
    plan = dd.Plan(**pa)
    kern = {"auto": dd.KERNEL_AUTO, "naive": dd.KERNEL_NAIVE, "direct": dd.KERNEL_DIRECT,
            "window": dd.KERNEL_WINDOW, "long": dd.KERNEL_LONG}[args.kernel]
    if primary and args.geometry:
        plan.set_window_geometry(*map(int, args.geometry.split(",")))
    plan.set_kernel(kern)
    ndm_local = hi - lo
    n_out = cf.n_out
    streaming = cf.nchunks > 1
    dtc = dd.U8 if cf.dtype == "u8" else dd.F32
    dt_in = torch.uint8 if cf.dtype == "u8" else torch.float32
    dt_out = torch.int32 if cf.dtype == "u8" else torch.float32
    nb = cf.nbeams
    # the input extent is that of the WHOLE DM list (every rank of a DM-sharded run holds the same buffer)
    full_plan = plan if not dm_shard else dd.Plan(**cf.plan_args())
    M = full_plan.max_delay
    full_tab_max = int(full_plan.shifts().max())
    beam0 = 0 if dm_shard else rank

    # ---- synthetic input, seeded
    t_gen = time.time()
    if streaming:
        n_in = n_out                      # one chunk per step; the driver carries the overlap
        host = np.stack([synth.make_input(cf, n_in, beam=shard.beam_of(beam0, nb, b)) for b in range(nb)])
    else:
        n_in = n_out + max(M, full_tab_max if cf.nsub else 0)
        if cf.nchans * n_in > (1 << 31):   # cfg4: 9 GB of input -- generated on the device (seeded torch generator)
            host = None
        else:
            tab = full_plan.shifts()
            pulses = synth.draw_pulses(cf, n_out, beam=beam0)
            host = synth.make_input(cf, n_in, pulses, {p[0]: tab[p[0]] for p in pulses}, beam=beam0)[None]
    stride = (n_in + 15) // 16 * 16
    if host is not None:
        x = torch.zeros((nb, cf.nchans, stride), dtype=dt_in, device="cuda")
        x[:, :, :n_in] = torch.from_numpy(host).cuda()
    else:
        g = torch.Generator(device="cuda").manual_seed(cf.seed + beam0)
        x = torch.empty((nb, cf.nchans, stride), dtype=torch.float32, device="cuda")
        for c0 in range(0, cf.nchans, 256):
            x[:, c0:c0 + 256].normal_(generator=g)
    t_gen = time.time() - t_gen
    out = torch.empty((nb, ndm_local, n_out), dtype=dt_out, device="cuda")
    stream = dd.Stream(plan, dtc, n_out, nb) if streaming else None
    xin = x[:, :, :n_in].contiguous() if streaming else x
    if not streaming:
        plan.reserve(dtc, n_out, nb)      # tables and scratch up front: execute itself never allocates

    def step():
        if streaming:
            stream.push(xin, out)
        else:
            plan.execute(xin, n_out, out=out)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    launches_per_step = plan.last_launches
    sync_all()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all()
    w0 = time.time()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    sync_all()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = ctx.sampler.window(w0, w1) if ctx.sampler else None
    ms = shard.max_over_ranks(ms, dist if world > 1 else None, "cuda")
    ms_step = ms / steps
    adds_local = float(ndm_local) * float(n_out) * float(cf.nchans) * float(nb)
    adds_job = shard.sum_over_ranks(adds_local, dist if world > 1 else None, "cuda")
    value = adds_job / (ms_step * 1e-3)

    # ---- end to end through the host-buffer ABI entries (pinned host buffers)
    e2e, e2e_events = None, None
    if not args.no_e2e:
        n_host = n_in if streaming else n_out + plan.max_delay      # the extent this plan's host entry expects
        if host is not None:
            hin = torch.from_numpy(np.ascontiguousarray(host[:, :, :n_host])).pin_memory()
        else:
            hin = torch.empty((nb, cf.nchans, n_host), dtype=dt_in).pin_memory()
            hin.copy_(x[:, :, :n_host])
        hout = torch.empty((nb, ndm_local, n_out), dtype=dt_out).pin_memory()
        ksteps = max(1, min(steps, 3))

        def e2e_step():
            if streaming:
                stream.push_host(hin, hout)
            else:
                plan.execute_host(hin, n_out, out=hout)

        def timed(fn):
            fn()
            sync_all()
            t0 = time.perf_counter()
            for _ in range(ksteps):
                fn()
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            return shard.max_over_ranks(dt, dist if world > 1 else None, "cuda")
        dt = timed(e2e_step)
        e2e = {"value": adds_job * ksteps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(hin.numel() * hin.element_size()),
               "d2h_bytes_per_step": int(hout.numel() * hout.element_size()), "steps": ksteps,
               "ms_per_step": 1e3 * dt / ksteps, "entry": "dedisp_stream_push_host" if streaming else "dedisp_execute_host"}
        if not streaming and hasattr(plan, "execute_detect_host"):
            cap = 1 << 20
            last = {}

            def ev_step():
                last["r"] = plan.execute_detect_host(hin, n_out, 5.0, capacity=cap)
            dt = timed(ev_step)
            res, evs = last["r"]
            e2e_events = {"value": adds_job * ksteps / dt, "unit": UNIT, "nsigma": 5.0,
                          "h2d_bytes_per_step": int(hin.numel() * hin.element_size()),
                          "d2h_bytes_per_step": int(sum(32 + 16 * min(r["count"], cap) for r in res)),
                          "events": [r["count"] for r in res], "steps": ksteps, "ms_per_step": 1e3 * dt / ksteps,
                          "entry": "dedisp_execute_detect_host (events and statistics come back, not the buffer)"}
        del hin, hout

    if rank != 0:
        return None

    # ---- dominant kernel alone (roofline): CUDA events recorded by the library on the launching stream
    plan.set_timing(True)
    kms, sms = [], []
    for _ in range(max(3, min(steps, 10))):
        step()
        kms.append(plan.last_kernel_ms())
        try:
            sms.append(plan.last_stage_ms())
        except dd.DedispError:
            pass
    plan.set_timing(False)
    kernel_ms = float(np.mean(kms))
    # the kernel the timed executes really ran (AUTO is size-aware at execute time: cfg 1 goes to the
    # one-thread-per-output kernel although the plan's table fits the register-window kernel)
    resolved = plan.last_kernel
    kname = {dd.KERNEL_WINDOW: "dedisp::window_kernel (all band launches of one execute)",
             dd.KERNEL_DIRECT: "dedisp::direct_kernel", dd.KERNEL_NAIVE: "dedisp::naive_kernel",
             dd.KERNEL_LONG: "dedisp::long_kernel"}.get(resolved, "?")

    props = torch.cuda.get_device_properties(local)
    nsm = props.multi_processor_count
    alu_peak = nsm * 128 * pk["sm_max_mhz"] * 1e6          # adds/s
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        traffic = tj.get("%s:%d" % (cf.name.split("_")[0], resolved))
        traffic_src = "profiles/traffic.json (ncu --set full capture of this kernel, static: not measured in this run)"
    subband = None
    window_parts = None
    if cf.nsub:
        # the two-stage path executes far fewer adds than the brute-force-equivalent count `value`
        # is quoted in: stage 1 = sum_{k,s} (n_out + maxshift2_{k,s}) * nchans/nsub, stage 2 = ndm * n_out * nsub.
        # Stage 1 (the dominant kernel) has no reuse between rows: one shared-memory word per add,
        # so its ceiling is the 128 B/clk/SM shared-memory pipe = a quarter of the add pipe.
        s2tab = plan.subband_shifts()[1].astype(np.float64)
        mks = s2tab.reshape(ndm_local // cf.nfine, cf.nfine, cf.nsub).max(axis=1)          # [ncoarse][nsub]
        s1_samples = float((n_out + mks).sum())                                          # per channel of a subband
        s1_adds = float(nb) * s1_samples * (cf.nchans // cf.nsub)
        s2_adds = float(nb) * ndm_local * float(n_out) * cf.nsub
        s1_ms, s2_ms = (float(np.mean([v[k] for v in sms])) for k in (0, 1))
        s2_bytes = float(nb) * (s1_samples * 4 + float(ndm_local) * n_out * 4)
        smem_peak = nsm * 32 * pk["sm_max_mhz"] * 1e6
        kernel_adds, kernel_ms_dom = s1_adds, s1_ms
        kname = "%s (subband stage 1)" % kname
        subband = {"stage1_ms": s1_ms, "stage2_ms": s2_ms, "stage1_adds": s1_adds, "stage2_adds": s2_adds,
                   "actual_adds_per_s": (s1_adds + s2_adds) / (ms_step * 1e-3),
                   "stage1_smem_pipe": {"peak_adds_per_s": smem_peak, "frac": s1_adds / (s1_ms * 1e-3) / smem_peak,
                                        "how": "%d SMs x 32 words/clk x %.0f MHz, one word per add" % (nsm, pk["sm_max_mhz"])},
                   "stage2_hbm": {"algorithmic_bytes": s2_bytes, "achieved_gbs": s2_bytes / (s2_ms * 1e-3) / 1e9,
                                  "peak_gbs": pk["hbm_gbs"], "frac": s2_bytes / (s2_ms * 1e-3) / 1e9 / pk["hbm_gbs"]}}
    else:
        kernel_adds, kernel_ms_dom = adds_local, kernel_ms
        if resolved == dd.KERNEL_WINDOW and sms:
            window_parts = {"pairify_ms": float(np.mean([v[0] for v in sms])), "bands_ms": float(np.mean([v[1] for v in sms]))}
    per_gpu = kernel_adds / (kernel_ms_dom * 1e-3)
    roof = {"bound": "alu", "achieved": per_gpu / 1e12, "peak": alu_peak / 1e12, "unit": "TFLOP/s",
            "frac": per_gpu / alu_peak, "traffic": traffic, "traffic_source": traffic_src,
            "peak_how": "%d SMs x 128 FP32 lanes x %.0f MHz (1 add = 1 flop; DESIGN.md section 6)" % (nsm, pk["sm_max_mhz"]),
            "kernel": kname, "kernel_ms": kernel_ms_dom, "algorithmic_adds": kernel_adds,
            "frac_of_step": kernel_ms_dom / ms_step,
            "frac_on_step": (kernel_adds / (ms_step * 1e-3)) / alu_peak if not cf.nsub else None,
            "frac_at_observed_clock": (per_gpu / (nsm * 128 * clocks["sm_mhz"] * 1e6)
                                       if clocks and clocks.get("sm_mhz") else None),
            "timed": "all launches of one execute (window path: pair-forming pre-pass + band launches)" if not cf.nsub else "stage 1 launch",
            "window_parts": window_parts}
    if ctx.fadd:
        roof["peak_measured"] = ctx.fadd["peak_measured_adds_per_s"] / 1e12
        roof["frac_of_measured"] = per_gpu / ctx.fadd["peak_measured_adds_per_s"]
    in_bytes = float(nb) * cf.nchans * n_in * (1 if cf.dtype == "u8" else 4)
    out_bytes = float(nb) * ndm_local * n_out * 4
    hbm = {"algorithmic_bytes": in_bytes + out_bytes, "achieved_gbs": (in_bytes + out_bytes) / (ms_step * 1e-3) / 1e9,
           "peak_gbs": pk["hbm_gbs"], "frac": (in_bytes + out_bytes) / (ms_step * 1e-3) / 1e9 / pk["hbm_gbs"],
           "peak_src": pk["src"]}

    res = {"workload": "%s: %d ch, %d DM trials, %d samples%s" % (
               cf.name, cf.nchans, cf.ndm, n_out, ", %d beams, streaming chunk" % nb if streaming else ""),
           "value": value, "ms_per_step": ms_step, "steps": steps, "warmup": warmup,
           "real_time_factor": n_out * cf.t_samp_ms * 1e-3 / (ms_step * 1e-3),
           "dtype": "i32" if cf.dtype == "u8" else "f32",
           "nchans": cf.nchans, "ndm": cf.ndm, "ndm_this_rank": ndm_local, "n_out": n_out, "nbeams": nb, "max_delay": M,
           "resolved_kernel": resolved, "window": plan.window_info() if not cf.nsub else None,
           "l2": "inputs larger than L2 (%.2f GB in, %.2f GB out per step)" % (in_bytes / 1e9, out_bytes / 1e9)
                 if in_bytes + out_bytes > 126e6 else "L2 flushed by nothing: %.1f MB in + out fit the 126 MB L2 (cfg1 is a parity case, timed for completeness)" % ((in_bytes + out_bytes) / 1e6),
           "roofline": roof, "subband": subband, "hbm": hbm, "e2e": e2e, "e2e_events": e2e_events,
           "gpu_launches": launches_per_step * steps, "clocks": clocks, "input_gen_s": t_gen}

    if primary:
        # ---- event detection on the step's output: HBM-bound; timed on
        # its own, not part of the step
        plan.detect(out, 5.0, capacity=1 << 16)
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        d0.record()
        for _ in range(5):
            dres, _ev = plan.detect(out, 5.0, capacity=1 << 16)
        d1.record()
        torch.cuda.synchronize()
        det_ms = d0.elapsed_time(d1) / 5
        det_bytes = 2.0 * float(nb) * ndm_local * n_out * 4
        res["detect"] = {"nsigma": 5.0, "ms": det_ms, "events": [r["count"] for r in dres], "algorithmic_bytes": det_bytes,
                         "achieved_gbs": det_bytes / (det_ms * 1e-3) / 1e9, "peak_gbs": pk["hbm_gbs"],
                         "frac": det_bytes / (det_ms * 1e-3) / 1e9 / pk["hbm_gbs"], "bound": "hbm",
                         "note": "two passes over the buffer; includes the host read-back of 32 bytes of statistics per beam and of the stored events"}
        # ---- power + corner turn and binning (NEXT-2)
        if cf.dtype == "f32":
            ns = int(min(n_in, 1 << 19, (1 << 31) // cf.nchans))
            volt = torch.randn((ns, cf.nchans, 2), dtype=torch.float32, device="cuda")
            vz = torch.view_as_complex(volt)
            pw = dd.power_corner_turn(vz)
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            f0.record()
            for _ in range(5):
                dd.power_corner_turn(vz, out=pw)
            f1.record()
            torch.cuda.synchronize()
            fms = f0.elapsed_time(f1) / 5
            fbytes = 12.0 * ns * cf.nchans
            front = {"op": "power_corner_turn", "spectra": ns, "nchans": cf.nchans, "ms": fms, "algorithmic_bytes": fbytes,
                     "achieved_gbs": fbytes / (fms * 1e-3) / 1e9, "peak_gbs": pk["hbm_gbs"],
                     "frac": fbytes / (fms * 1e-3) / 1e9 / pk["hbm_gbs"], "bound": "hbm"}
            del volt, vz, pw
            bx = x[0]
            dd.bin_samples(bx, 2)
            torch.cuda.synchronize()
            f0.record()
            for _ in range(5):
                dd.bin_samples(bx, 2)
            f1.record()
            torch.cuda.synchronize()
            bms = f0.elapsed_time(f1) / 5
            bbytes = 6.0 * cf.nchans * float(bx.shape[-1])
            front["binning"] = {"nb": 2, "ms": bms, "algorithmic_bytes": bbytes, "achieved_gbs": bbytes / (bms * 1e-3) / 1e9,
                                "frac": bbytes / (bms * 1e-3) / 1e9 / pk["hbm_gbs"], "bound": "hbm",
                                "note": "includes the allocation of the output tensor in the binding"}
            res["front_end"] = front

    if stream is not None:
        stream.close()
    plan.close()
    del x, out
    torch.cuda.empty_cache()

    if not args.no_cpu_baseline:
        run, sadds, desc, cores = oracle_sample(cf, budget_adds=3.0e11 if primary else 5.0e10)
        t0 = time.perf_counter()
        run()
        dt = time.perf_counter() - t0
        res["cpu_baseline"] = {"value": sadds / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                               "seconds": dt}
    else:
        res["cpu_baseline"] = None
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "naive", "direct", "window", "long"])
    ap.add_argument("--geometry", default="", help="T,G,NT,D of the register-window kernel (dedisp_plan_set_window_geometry)")
    ap.add_argument("--shard", default="beam", choices=["beam", "dm"], help="N > 1: one beam per rank (weak) or one DM slice per rank (strong)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true")
    args = ap.parse_args()
    cf = synth.configs()[WORKLOADS[args.workload]]
    if args.impl == "reference":
        return run_reference(args, cf)

    import torch
    import torch.distributed as dist
    import paper_1107_2516_b200 as dd
    from paper_1107_2516_b200 import build as ddbuild

    ctx = Ctx()
    ctx.torch, ctx.dd, ctx.dist = torch, dd, dist
    ctx.world = world = int(os.environ.get("WORLD_SIZE", "1"))
    ctx.rank = rank = int(os.environ.get("RANK", "0"))
    ctx.local = local = int(os.environ.get("LOCAL_RANK", "0"))
    ctx.pk = peaks()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        ddbuild.build()
    if world > 1:
        dist.barrier()
    args.warmup = max(args.warmup, 3)
    ctx.sampler = None
    ctx.fadd = None
    if rank == 0:
        ctx.sampler = ClockSampler(local)
        ctx.sampler.start()
        time.sleep(0.15)
        ctx.fadd = fadd_leg(ctx)

    res = measure(ctx, cf, args, args.steps, args.warmup, primary=True)
    others = {}
    if world == 1 and not args.no_all_configs and args.workload == "cfg3" and args.kernel == "auto":
        for name in ("cfg1", "cfg2", "cfg4", "cfg5"):
            r = measure(ctx, synth.configs()[WORKLOADS[name]], args, 5, 3, primary=False)
            others[name] = r

    if rank == 0:
        ctx.sampler.stop()
        line = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
                "scaling": "strong" if (args.shard == "dm" and world > 1) else "weak",
                "vs_baseline": None, "dtype": res["dtype"], "data": "synthetic",
                "config": {"workload": res["workload"], "nchans": res["nchans"], "ndm": res["ndm"], "n_out": res["n_out"],
                           "nbeams": res["nbeams"], "max_delay": res["max_delay"], "kernel": args.kernel,
                           "resolved_kernel": res["resolved_kernel"], "window": res["window"], "l2": res["l2"],
                           "parallelism": ("single GPU" if world == 1 else
                                           "%d GPUs, same input, contiguous DM slices (PAPER.md:74), no collective" % world
                                           if args.shard == "dm" else "%d GPUs, 1 beam per GPU, no collective" % world)},
                "real_time_factor": res["real_time_factor"], "roofline": res["roofline"], "subband": res["subband"],
                "hbm": res["hbm"], "detect": res.get("detect"), "front_end": res.get("front_end"),
                "cpu_baseline": res["cpu_baseline"], "e2e": res["e2e"], "e2e_events": res["e2e_events"],
                "gpu_launches": res["gpu_launches"], "clocks": res["clocks"], "fadd_microbench": ctx.fadd,
                "all_configs": others or None,
                "paper_context": "paper: 50-200x over one Xeon 2.7 GHz core on a Tesla C1060 (PAPER.md:203), ~1.5e10 adds/s",
                "input_gen_s": res["input_gen_s"]}
        # compact per-config digest as the LAST key: a record that keeps only the tail of this line still
        # carries every config's step time, roofline fraction, end-to-end time and the kernel that ran
        def digest(r):
            return {"ms": round(r["ms_per_step"], 3), "frac": round(r["roofline"]["frac"], 4),
                    "kernel": r["resolved_kernel"], "traffic": r["roofline"]["traffic"],
                    "e2e_ms": round(r["e2e"]["ms_per_step"], 2) if r.get("e2e") else None,
                    "e2e_events_ms": round(r["e2e_events"]["ms_per_step"], 2) if r.get("e2e_events") else None,
                    "stage_ms": [round(r["subband"]["stage1_ms"], 3), round(r["subband"]["stage2_ms"], 3)] if r.get("subband") else None}
        line["summary"] = {args.workload: digest(res)}
        line["summary"].update({k: digest(v) for k, v in others.items()})
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
