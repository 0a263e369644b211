#!/usr/bin/env python
"""bench.py -- throughput of the de-dispersion hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

A step is one pass of the hot path over one batch of synthetic filterbank data: for the brute-force
workloads one dedisp_execute (SURVEY.md §8 rows a2/a3 with the plan's a1 table), for cfg4 the two
subband stages (a4+a5), for cfg5 one streaming push of all beams (a3+a6).  The default workload is
BASELINE.json's 4096-DM L-band configuration (cfg3), the one the north-star target is quoted on.

metric  = DM*sample*channel adds per second (nDM * n_out * nchans * nbeams / t), inputs resident
          in HBM, CUDA events on the launching stream, max over ranks.
e2e     = same metric through the C ABI's host-buffer entry (pinned host in/out, H2D and D2H inside
          the timed region).
roofline: the path is bound by the FP32/INT add pipe (gather-and-add, no tensor cores); peak =
          SMs * 128 lanes * max SM clock.
N > 1   : every rank de-disperses its own beam of the same workload (no data-path collective),
          weak scaling; value is the sum over ranks / max time.
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

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
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


def adds_per_step(cf, n_out):
    return float(cf.ndm) * float(n_out) * float(cf.nchans) * float(cf.nbeams)


def oracle_sample(cf, budget_adds=3.0e11):
    """A bounded sample of the workload for the CPU oracle: every s-th DM row, a prefix of the
    time axis, one beam -- sized to about budget_adds additions."""
    from oracle import dedisp_oracle as orc
    orc.build()
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "naive", "direct", "window", "long"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    cf = synth.configs()[WORKLOADS[args.workload]]
    if args.impl == "reference":
        return run_reference(args, cf)

    import torch
    import torch.distributed as dist
    import paper_1107_2516_b200 as dd
    from paper_1107_2516_b200 import build as ddbuild

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
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

    plan = dd.Plan(**cf.plan_args())
    plan.set_kernel({"auto": dd.KERNEL_AUTO, "naive": dd.KERNEL_NAIVE, "direct": dd.KERNEL_DIRECT,
                     "window": dd.KERNEL_WINDOW, "long": dd.KERNEL_LONG}[args.kernel])
    M = plan.max_delay
    n_out = cf.n_out
    streaming = cf.nchunks > 1
    dt_in = torch.uint8 if cf.dtype == "u8" else torch.float32
    dt_out = torch.int32 if cf.dtype == "u8" else torch.float32
    full_tab_max = int(plan.shifts().max())

    # ---- synthetic input, seeded; beam index = rank so that every rank has its own data
    t_gen = time.time()
    if streaming:
        n_in = n_out                      # one chunk per step; the driver carries the overlap
        host = np.stack([synth.make_input(cf, n_in, beam=shard.beam_of(rank, cf.nbeams, b)) for b in range(cf.nbeams)])
    else:
        n_in = n_out + max(M, full_tab_max if cf.nsub else 0)
        if cf.nchans * n_in > (1 << 31):   # cfg4: 9 GB of input -- generate on the device
            host = None
        else:
            tab = plan.shifts()
            pulses = synth.draw_pulses(cf, n_out, beam=rank)
            host = synth.make_input(cf, n_in, pulses, {p[0]: tab[p[0]] for p in pulses}, beam=rank)[None]
    stride = (n_in + 15) // 16 * 16
    nb = cf.nbeams
    if host is not None:
        x = torch.zeros((nb, cf.nchans, stride), dtype=dt_in, device="cuda")
        x[:, :, :n_in] = torch.from_numpy(host).cuda()
    else:
        g = torch.Generator(device="cuda").manual_seed(cf.seed + rank)
        x = torch.empty((nb, cf.nchans, stride), dtype=torch.float32, device="cuda")
        for c0 in range(0, cf.nchans, 256):
            x[:, c0:c0 + 256].normal_(generator=g)
    t_gen = time.time() - t_gen
    out = torch.empty((nb, cf.ndm, n_out), dtype=dt_out, device="cuda")
    stream = dd.Stream(plan, dd.U8 if cf.dtype == "u8" else dd.F32, n_out, nb) if streaming else None
    xin = x[:, :, :n_in].contiguous() if streaming else x

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

    for _ in range(args.warmup):
        step()
    launches_per_step = plan.last_launches
    sync_all()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all()
    w0 = time.time()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    sync_all()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(w0, w1) if rank == 0 else None
    ms = shard.max_over_ranks(ms, dist if world > 1 else None, "cuda")
    ms_step = ms / args.steps
    adds = adds_per_step(cf, n_out)
    value = adds * world / (ms_step * 1e-3)

    # ---- end to end through the host-buffer ABI entry (pinned host buffers)
    e2e = None
    if not args.no_e2e and host is not None:
        hin = torch.from_numpy(np.ascontiguousarray(host[:, :, :n_in])).pin_memory()
        hout = torch.empty((nb, cf.ndm, n_out), dtype=dt_out).pin_memory()
        ksteps = max(1, min(args.steps, 3))

        def e2e_step():
            if streaming:
                stream.push_host(hin, hout)
            else:
                plan.execute_host(hin, n_out, out=hout)
        e2e_step()
        sync_all()
        t0 = time.perf_counter()
        for _ in range(ksteps):
            e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, dist if world > 1 else None, "cuda")
        e2e = {"value": adds * world * ksteps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(hin.numel() * hin.element_size()),
               "d2h_bytes_per_step": int(hout.numel() * hout.element_size()), "steps": ksteps,
               "ms_per_step": 1e3 * dt / ksteps}
        del hin, hout

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- dominant kernel alone (roofline): CUDA events recorded by the library on the launching
    # stream around the band launches of the register-window kernel (or all launches of the other
    # paths), averaged over the same number of steps
    plan.set_timing(True)
    kms, sms = [], []
    for _ in range(max(3, min(args.steps, 10))):
        step()
        kms.append(plan.last_kernel_ms())
        if cf.nsub:
            sms.append(plan.last_stage_ms())
    plan.set_timing(False)
    kernel_ms = float(np.mean(kms))
    resolved = plan.resolved_kernel(dd.U8 if cf.dtype == "u8" else dd.F32)
    kname = {dd.KERNEL_WINDOW: "dedisp::window_kernel (all band launches of one execute)",
             dd.KERNEL_DIRECT: "dedisp::direct_kernel", dd.KERNEL_NAIVE: "dedisp::naive_kernel",
             dd.KERNEL_LONG: "dedisp::long_kernel"}.get(resolved, "?")

    pk = peaks()
    props = torch.cuda.get_device_properties(local)
    nsm = props.multi_processor_count
    alu_peak = nsm * 128 * pk["sm_max_mhz"] * 1e6          # adds/s
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get("%s:%d" % (args.workload, resolved))
    subband = None
    if cf.nsub:
        # the two-stage path executes far fewer adds than the brute-force-equivalent count `value`
        # is quoted in: stage 1 = sum_{k,s} (n_out + maxshift2_{k,s}) * nchans/nsub, stage 2 = ndm * n_out * nsub.
        # Stage 1 (the dominant kernel) has no reuse between rows: one shared-memory word per add,
        # so its ceiling is the 128 B/clk/SM shared-memory pipe = a quarter of the add pipe.
        # stage 1 forms n_out + max_{d in group k} s2(d, s) samples of subband s in group k (what stage 2 reads)
        s2tab = plan.subband_shifts()[1].astype(np.float64)
        mks = s2tab.reshape(cf.ndm // cf.nfine, cf.nfine, cf.nsub).max(axis=1)          # [ncoarse][nsub]
        s1_samples = float((n_out + mks).sum())                                          # per channel of a subband
        s1_adds = float(nb) * s1_samples * (cf.nchans // cf.nsub)
        s2_adds = float(nb) * cf.ndm * float(n_out) * cf.nsub
        s1_ms, s2_ms = (float(np.mean([v[k] for v in sms])) for k in (0, 1))
        s2_bytes = float(nb) * (s1_samples * 4 + float(cf.ndm) * n_out * 4)
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
        kernel_adds, kernel_ms_dom = adds, kernel_ms
    per_gpu = kernel_adds / (kernel_ms_dom * 1e-3)
    roof = {"bound": "alu", "achieved": per_gpu / 1e12, "peak": alu_peak / 1e12, "unit": "TFLOP/s",
            "frac": per_gpu / alu_peak, "traffic": traffic,
            "peak_how": "%d SMs x 128 FP32 lanes x %.0f MHz (1 add = 1 flop; DESIGN.md section 6)" % (nsm, pk["sm_max_mhz"]),
            "kernel": kname, "kernel_ms": kernel_ms_dom, "algorithmic_adds": kernel_adds,
            "frac_of_step": kernel_ms_dom / ms_step,
            "frac_at_observed_clock": (per_gpu / (nsm * 128 * clocks["sm_mhz"] * 1e6)
                                       if clocks and clocks.get("sm_mhz") else None)}
    in_bytes = float(nb) * cf.nchans * n_in * (1 if cf.dtype == "u8" else 4)
    out_bytes = float(nb) * cf.ndm * n_out * 4
    hbm = {"algorithmic_bytes": in_bytes + out_bytes, "achieved_gbs": (in_bytes + out_bytes) / (ms_step * 1e-3) / 1e9,
           "peak_gbs": pk["hbm_gbs"], "frac": (in_bytes + out_bytes) / (ms_step * 1e-3) / 1e9 / pk["hbm_gbs"],
           "peak_src": pk["src"]}

    # ---- event detection on the step's output: HBM-bound, two
    # passes over out (statistics, threshold scan); timed on its own, not part of the step
    plan.detect(out, 5.0, capacity=1 << 16)
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    d0.record()
    for _ in range(5):
        dres, _ev = plan.detect(out, 5.0, capacity=1 << 16)
    d1.record()
    torch.cuda.synchronize()
    det_ms = d0.elapsed_time(d1) / 5
    det_bytes = 2.0 * float(nb) * cf.ndm * n_out * 4
    detect = {"nsigma": 5.0, "ms": det_ms, "events": [r["count"] for r in dres], "algorithmic_bytes": det_bytes,
              "achieved_gbs": det_bytes / (det_ms * 1e-3) / 1e9, "peak_gbs": pk["hbm_gbs"],
              "frac": det_bytes / (det_ms * 1e-3) / 1e9 / pk["hbm_gbs"], "bound": "hbm",
              "note": "includes the host read-back of 32 bytes of statistics per beam and of the stored events"}

    # ---- power + corner turn: the front-end step that produces the
    # channel-major layout, on a voltage buffer of up to 2^19 spectra (the paper's buffer) x nchans
    front = None
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
        # binning, bin factor 2 on the step's own input
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

    cpu = None
    if not args.no_cpu_baseline:
        run, sadds, desc, cores = oracle_sample(cf)
        t0 = time.perf_counter()
        run()
        dt = time.perf_counter() - t0
        cpu = {"value": sadds / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
               "seconds": dt}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "i32" if cf.dtype == "u8" else "f32", "data": "synthetic",
            "config": {"workload": "%s: %d ch, %d DM trials, %d samples%s" % (
                           cf.name, cf.nchans, cf.ndm, n_out,
                           ", %d beams, streaming chunk" % nb if streaming else ""),
                       "nchans": cf.nchans, "ndm": cf.ndm, "n_out": n_out, "nbeams": nb,
                       "max_delay": M, "kernel": args.kernel, "resolved_kernel": plan.resolved_kernel(dd.U8 if cf.dtype == "u8" else dd.F32),
                       "window": plan.window_info() if not cf.nsub else None,
                       "l2": "inputs larger than L2 (%.2f GB in, %.2f GB out per step)" % (in_bytes / 1e9, out_bytes / 1e9),
                       "parallelism": "1 beam per GPU, no collective" if world > 1 else "single GPU"},
            "real_time_factor": n_out * cf.t_samp_ms * 1e-3 / (ms_step * 1e-3),
            "roofline": roof, "subband": subband, "hbm": hbm, "detect": detect, "front_end": front, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches_per_step * args.steps, "clocks": clocks,
            "paper_context": "paper: 50-200x over one Xeon 2.7 GHz core on a Tesla C1060 (PAPER.md:203), ~1.5e10 adds/s",
            "input_gen_s": t_gen}
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
