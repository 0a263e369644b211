"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Bars (BASELINE.json north_star): shift tables and uint8->int32 bit-exact;
fp32 within |gpu - oracle| <= 1e-5 * sum_c |in[c][t+shift]| per output sample."""
import numpy as np
import pytest

import paper_1107_2516_b200 as dd
from paper_1107_2516_b200 import synth, build as ddbuild

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KERNELS = {"naive": dd.KERNEL_NAIVE, "direct": dd.KERNEL_DIRECT, "auto": dd.KERNEL_AUTO,
           "long": dd.KERNEL_LONG, "window": dd.KERNEL_WINDOW}


@pytest.fixture(scope="module", autouse=True)
def built():
    ddbuild.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"


def to_dev(x, pad_to=16):
    """Host [.., n] -> CUDA tensor whose row stride is a multiple of 16 elements."""
    n = x.shape[-1]
    stride = (n + pad_to - 1) // pad_to * pad_to
    t = torch.zeros(x.shape[:-1] + (stride,), dtype=torch.from_numpy(x[..., :1].copy()).dtype, device="cuda")
    t[..., :n] = torch.from_numpy(x).cuda()
    return t[..., :n] if stride == n else t[..., :n]


def check_f32(got, ref, sumabs):
    err = np.abs(got.astype(np.float64) - ref)
    bound = 1e-5 * sumabs
    bad = err > bound
    assert not bad.any(), "fp32 parity: %d outputs beyond 1e-5*sum|in| (worst ratio %.3g)" % (
        bad.sum(), (err / np.maximum(bound, 1e-300)).max())


def small_cfg(dtype="f32", nchans=96, ndm=70, n_out=3000 + 17, step=0.35, seed=21, **kw):
    return synth.Config("small", nchans, 150.0, 0.1, 0.2, n_out, ndm, step, dtype=dtype, seed=seed,
                        npulses=3, pulse_width_ms=(0.5, 3.0), pulse_amp=(0.5, 2.0), **kw)


def make_case(oracle, cf, n_out=None, beams=1):
    n_out = n_out or cf.n_out
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = n_out + int(tab.max())
    xs = []
    for b in range(beams):
        pulses = synth.draw_pulses(cf, n_out, beam=b)
        xs.append(synth.make_input(cf, n_in, pulses, {p[0]: tab[p[0]] for p in pulses}, beam=b))
    return tab, np.stack(xs)


@pytest.mark.parametrize("kernel", ["naive", "direct", "auto", "long"])
@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_brute_small_ragged(oracle, kernel, dtype):
    cf = small_cfg(dtype)
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    assert (plan.shifts() == tab).all()
    plan.set_kernel(KERNELS[kernel])
    got = plan.execute(to_dev(x), cf.n_out).cpu().numpy()
    assert plan.last_launches >= 1
    for b in range(2):
        if dtype == "u8":
            assert (got[b] == oracle.brute_u8(x[b], tab, cf.n_out)).all()
        else:
            ref, sa = oracle.brute_f32(x[b], tab, cf.n_out)
            check_f32(got[b], ref, sa)


@pytest.mark.parametrize("kernel", ["direct", "auto", "window"])
def test_cfg1_full(oracle, kernel):
    cf = synth.configs()[1]
    tab, x = make_case(oracle, cf)
    plan = dd.Plan(**cf.plan_args())
    plan.set_kernel(KERNELS[kernel])
    got = plan.execute(to_dev(x[0]), cf.n_out).cpu().numpy()
    ref, sa = oracle.brute_f32(x[0], tab, cf.n_out)
    check_f32(got, ref, sa)
    # P7 on the GPU result: the injected pulse is recovered at trial 30
    w = cf.fixed_pulses[0][2]
    box = np.cumsum(np.pad(got.astype(np.float64), ((0, 0), (1, 0))), axis=1)
    assert np.unravel_index(np.argmax(box[:, w:] - box[:, :-w]), (cf.ndm, cf.n_out - w + 1))[0] == 30


@pytest.mark.parametrize("k,ndm,n_out", [(2, 256, 4096 + 40), (3, 320, 8192 + 8), (5, 192, 4096)])
def test_scaled_configs(oracle, k, ndm, n_out):
    """cfg 2/3/5 geometry (band, t_samp, DM step) on a DM/time subset the oracle finishes quickly;
    the DM subset is the TOP of the range, where the shifts and their spread are largest."""
    base = synth.configs()[k]
    cf = synth.scaled(base, n_out=n_out)
    full = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    rows = np.r_[0:ndm // 2, cf.ndm - ndm // 2:cf.ndm]
    dm = cf.dm_list[rows]
    tab = full[rows]
    n_in = n_out + int(tab.max())
    pulses = [(ndm - 5, 100, 20, 1.0), (3, n_out // 2, 8, 2.0)]
    x = synth.make_input(cf, n_in, pulses, {p[0]: tab[p[0]] for p in pulses})
    plan = dd.Plan(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm)
    assert (plan.shifts() == tab).all()
    got = plan.execute(to_dev(x), n_out).cpu().numpy()
    if cf.dtype == "u8":
        assert (got == oracle.brute_u8(x, tab, n_out)).all()
    else:
        ref, sa = oracle.brute_f32(x, tab, n_out)
        check_f32(got, ref, sa)
    # the register-window kernel itself on the contiguous top half of the list (the jump in the middle of
    # `rows` is outside its limits, and AUTO sends a problem this small to the direct kernel anyway)
    top = dd.Plan(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm[ndm // 2:])
    assert top.window_info()["ok"] == 1
    top.set_kernel(dd.KERNEL_WINDOW)
    got = top.execute(to_dev(x), n_out).cpu().numpy()
    if cf.dtype == "u8":
        assert (got == oracle.brute_u8(x, tab[ndm // 2:], n_out)).all()
    else:
        ref, sa = oracle.brute_f32(x, tab[ndm // 2:], n_out)
        check_f32(got, ref, sa)


@pytest.mark.parametrize("dtype,beams,n_out,nchans", [("f32", 1, 100, 384), ("u8", 3, 700, 384),
                                                       ("f32", 2, 1331, 384), ("f32", 1, 1500, 1024)])
def test_window_kernel_forced(oracle, dtype, beams, n_out, nchans):
    """The register-window kernel on its own: cfg-2 band, a DM count that is not a multiple of the
    block's rows, output lengths below / around one warp tile, several beams; the 1024-channel case
    needs several channel bands (accumulating launches)."""
    base = synth.configs()[2]
    cf = synth.scaled(base, dtype=dtype, n_out=n_out, ndm=150, nchans=nchans)
    tab, x = make_case(oracle, cf, beams=beams)
    plan = dd.Plan(**cf.plan_args())
    info = plan.window_info()
    assert info["ok"] == 1 and info["nband"] >= 1
    plan.set_kernel(dd.KERNEL_WINDOW)
    assert plan.resolved_kernel(dd.U8 if dtype == "u8" else dd.F32) == dd.KERNEL_WINDOW
    got = plan.execute(to_dev(x), n_out).cpu().numpy()
    assert plan.last_launches == 1 + info["nband"]
    for b in range(beams):
        if dtype == "u8":
            assert (got[b] == oracle.brute_u8(x[b], tab, n_out)).all()
        else:
            ref, sa = oracle.brute_f32(x[b], tab, n_out)
            check_f32(got[b], ref, sa)
    # running it again accumulates nothing from the previous call (band 0 overwrites)
    again = plan.execute(to_dev(x), n_out).cpu().numpy()
    assert (again == got).all()


GEOMS = [(15, 6, 2, 4), (15, 4, 3, 4), (21, 4, 1, 4), (21, 8, 1, 4), (17, 4, 1, 5), (15, 4, 1, 6), (11, 6, 2, 5),
         (9, 6, 2, 6)]


@pytest.mark.parametrize("geom", GEOMS)
def test_window_geometries(oracle, geom):
    """Every instantiated thread / block shape of the register-window kernel (dedisp_plan_set_window_geometry)
    on the cfg-2 band with 1024 channels: rows drift by tens of slots, so the hand-over of partial sums
    between warp segments and several blocks along time are exercised; uint8 bit-exact, two beams, an output length that ends inside a block."""
    T, G, NT, D = geom
    cf = synth.scaled(synth.configs()[2], dtype="u8", n_out=3 * 2 * NT * 32 * T + 777, ndm=2 * D * G + 3, nchans=1024)
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    try:
        plan.set_window_geometry(T, G, NT, D)
    except dd.DedispError as e:
        assert e.status == dd.binding.ESTATE          # staged segments of this band do not fit this shape's ring
        cf = synth.scaled(cf, nchans=256)             # a quarter of the band: a quarter of the drift
        tab, x = make_case(oracle, cf, beams=2)
        plan = dd.Plan(**cf.plan_args())
        plan.set_window_geometry(T, G, NT, D)
    info = plan.window_info()
    assert info["ok"] == 1 and (info["T"], info["G"], info["NT"], info["D"]) == geom
    assert info["kmax"] > 0 and info["Hb"] == (2 * NT * 32 * T - info["kmax"]) // 2 * 2
    # shallow rings, served by min(4, stages) producer warps: 3 stages with these shapes, 2 with the others
    assert info["ring_stages"] == (3 if geom in ((21, 8, 1, 4), (11, 6, 2, 5), (9, 6, 2, 6)) else 2)
    plan.set_kernel(dd.KERNEL_WINDOW)
    got = plan.execute(to_dev(x), cf.n_out).cpu().numpy()
    assert plan.last_launches == 1 + info["nband"]
    for b in range(2):
        assert (got[b] == oracle.brute_u8(x[b], tab, cf.n_out)).all()
    with pytest.raises(dd.DedispError):
        plan.set_window_geometry(15, 4, 1, 6)          # tables are on the device: too late
    p2 = dd.Plan(**cf.plan_args())
    with pytest.raises(dd.DedispError):
        p2.set_window_geometry(13, 5, 2, 4)            # not an instantiated shape


@pytest.mark.parametrize("dtype", ["u8", "f32"])
def test_window_kernel_several_channel_bands(oracle, dtype):
    """A table whose rows drift too fast for one channel band (cfg-2 band, twice its DM step, 6 rows per
    thread): the register-window kernel runs three launches; bands after the first ADD to the output, and
    their hand-over of partial sums goes through red.global.add on both sides.  Every output against the
    oracle; a second execute on the same buffer must not accumulate on the first."""
    cf = synth.scaled(synth.configs()[2], dtype=dtype, dm_step=0.1, ndm=2 * 36 + 5, nchans=1024, n_out=3 * 1100 + 321)
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    plan.set_window_geometry(9, 6, 2, 6)
    info = plan.window_info()
    assert info["ok"] == 1 and info["nband"] >= 2
    plan.set_kernel(dd.KERNEL_WINDOW)
    xd = to_dev(x)
    for rep in range(2):
        got = plan.execute(xd, cf.n_out).cpu().numpy()
        assert plan.last_launches == 1 + info["nband"]
        for b in range(2):
            if dtype == "u8":
                assert (got[b] == oracle.brute_u8(x[b], tab, cf.n_out)).all()
            else:
                ref, sa = oracle.brute_f32(x[b], tab, cf.n_out)
                check_f32(got[b], ref, sa)
    # detection on a multi-band plan takes the unfused route (an output is final only after the last band)
    out, res, ev = plan.execute_detect(xd, cf.n_out, 4.0)
    mu, sg, thr, evo, val = oracle.detect(out[0].cpu().numpy(), 4.0)
    assert res[0]["count"] == len(evo) and abs(res[0]["sigma"] - sg) <= 1e-11 * sg


@pytest.mark.parametrize("seed", [1, 2, 3, 4, 5, 6])
def test_random_plans_all_kernels(oracle, seed):
    """Seeded random bands, sampling times and DM lists (irregular steps, repeated trials, a DM count
    that is no multiple of any tile) on uint8 input: every kernel the plan accepts must be bit-exact."""
    rng = np.random.default_rng(1107_2516 + seed)
    nchans = int(rng.integers(3, 200))
    f_top = float(rng.uniform(120.0, 1600.0))
    df = float(rng.uniform(0.2, 0.9)) * f_top / nchans * 0.3
    t_samp = float(rng.choice([0.05, 0.064, 0.1, 0.5]))
    ndm = int(rng.integers(1, 90))
    kmax = 4.15e6 * ((f_top - (nchans - 1) * df) ** -2 - f_top ** -2) / t_samp   # samples per unit DM
    steps = rng.uniform(0.0, 2.0, ndm) * (rng.uniform(0.3, 6.0) / max(kmax, 1e-9))
    steps[rng.random(ndm) < 0.1] = 0.0                                           # repeated trials
    dm = np.cumsum(steps)
    n_out = int(rng.integers(1, 3000))
    tab = oracle.shift_table(nchans, f_top, df, t_samp, dm)
    x = rng.integers(0, 256, (nchans, n_out + int(tab.max())), dtype=np.uint8)
    ref = oracle.brute_u8(x, tab, n_out)
    plan = dd.Plan(nchans, f_top, df, t_samp, dm)
    assert (plan.shifts() == tab).all()
    tried = 0
    for name in ("auto", "direct", "long", "naive", "window"):
        try:
            plan.set_kernel(KERNELS.get(name, dd.KERNEL_WINDOW))
        except dd.DedispError:
            assert name == "window" and plan.window_info()["ok"] == 0
            continue
        got = plan.execute(to_dev(x), n_out).cpu().numpy()
        assert (got == ref).all(), name
        tried += 1
    assert tried >= 4


@pytest.mark.parametrize("step,dtype", [(2.0, "f32"), (4.0, "f32"), (6.0, "f32"), (4.0, "u8"), (16.0, "u8")])
def test_long_kernel_ring_depths(oracle, step, dtype):
    """The long-tile kernel with few, widely spaced trials: the 16 rows of a tile are thousands of samples
    apart, so a staged channel segment is large and the shared-memory ring holds 7, 4 (fp32 steps 2 and 4;
    uint8 step 16) or too few slots (fp32 step 6: fewer than four -> the library must fall back to the
    direct kernel instead of running a ring its four producer warps can lap)."""
    cf = synth.Config("wide", 64, 150.0, 0.1, 0.1, 4096 + 2048 + 77, 16, step, dtype=dtype, seed=77)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    spread = int((tab.max(axis=0) - tab.min(axis=0)).max())
    x = synth.make_input(cf, cf.n_out + int(tab.max()))
    plan = dd.Plan(**cf.plan_args())
    assert plan.window_info()["ok"] == 0               # rows this far apart cannot share a register window
    for kernel in (dd.KERNEL_LONG, dd.KERNEL_AUTO):
        plan.set_kernel(kernel)
        got = plan.execute(to_dev(x), cf.n_out).cpu().numpy()
        if dtype == "u8":
            assert (got == oracle.brute_u8(x, tab, cf.n_out)).all(), (kernel, spread)
        else:
            ref, sa = oracle.brute_f32(x, tab, cf.n_out)
            check_f32(got, ref, sa)


@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_detect_matches_oracle(oracle, dtype):
    """dedisp_plan_detect on the GPU's own de-dispersed buffer against oracle.detect on the same
    buffer: mean, sigma, threshold to 1e-12 relative, the event SET exact (order is
    free), intensities bit-equal; two beams; a capacity smaller than the count keeps counting."""
    cf = small_cfg(dtype, nchans=64, ndm=37, n_out=2000 + 3, step=0.4)
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    out = plan.execute(to_dev(x), cf.n_out)
    host = out.cpu().numpy()
    for nsig, cap in ((3.0, 1 << 16), (2.0, 50)):
        results, events = plan.detect(out, nsig, capacity=cap)
        for b in range(2):
            mu, sg, thr, ev, val = oracle.detect(host[b], nsig)
            r = results[b]
            assert abs(r["mean"] - mu) <= 1e-12 * max(1.0, abs(mu)) and abs(r["sigma"] - sg) <= 1e-11 * sg
            assert abs(r["threshold"] - thr) <= 1e-11 * abs(thr)
            assert r["count"] == len(ev) > 0
            got = events[b]
            if len(ev) <= cap:
                order = np.lexsort((got["t"], got["dm"]))
                assert (np.stack([got["t"][order], got["dm"][order]], axis=1) == ev).all()
                assert (got["value"][order] == val.astype(np.float32)).all()
            else:
                assert len(got) == cap
                allowed = set(map(tuple, ev.tolist()))
                assert all((int(t), int(d)) in allowed for t, d in zip(got["t"], got["dm"]))
    with pytest.raises(dd.DedispError):
        plan.detect(out[:, :, 1:], 3.0)            # misaligned view


def _check_detect(oracle, host_out, results, events, nsig, cap):
    for b in range(len(results)):
        mu, sg, thr, ev, val = oracle.detect(host_out[b], nsig)
        r = results[b]
        assert abs(r["mean"] - mu) <= 1e-12 * max(1.0, abs(mu)) and abs(r["sigma"] - sg) <= 1e-11 * sg
        assert abs(r["threshold"] - thr) <= 1e-11 * abs(thr)
        assert r["count"] == len(ev) > 0 and len(ev) <= cap
        got = events[b]
        order = np.lexsort((got["t"], got["dm"]))
        assert (np.stack([got["t"][order], got["dm"][order]], axis=1) == ev).all()
        assert (got["value"][order] == val.astype(np.float32)).all()


@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_execute_detect_fused(oracle, dtype):
    """dedisp_execute_detect / dedisp_execute_detect_host (PAPER.md:76 fused behind the hot path): the
    register-window kernel accumulates the statistics in its flush.  The de-dispersed buffer is checked
    against the brute-force oracle, then mean / sigma / threshold (1e-11) and the event SET against
    oracle.detect on that buffer; the host entry (several time pieces, events only) returns the same
    set; a subband plan takes the unfused route with the same definition."""
    cf = synth.scaled(synth.configs()[1], dtype=dtype, ndm=37, n_out=2 * 32768 + 1000 + 3)     # cfg-1 band and DM grid
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    assert plan.resolved_kernel(dd.U8 if dtype == "u8" else dd.F32) == dd.KERNEL_WINDOW and plan.window_info()["nband"] == 1
    nsig, cap = 3.5, 1 << 16
    out, results, events = plan.execute_detect(to_dev(x), cf.n_out, nsig, capacity=cap)
    assert plan.last_launches == 1 + 2 + 2           # pivot, pairify + one band, finish + threshold scan
    host = out.cpu().numpy()
    for b in range(2):
        if dtype == "u8":
            assert (host[b] == oracle.brute_u8(x[b], tab, cf.n_out)).all()
        else:
            ref, sa = oracle.brute_f32(x[b], tab, cf.n_out)
            check_f32(host[b], ref, sa)
    _check_detect(oracle, host, results, events, nsig, cap)
    # the two-pass detection on the same buffer: same statistics (another summation order), same events
    r2, e2 = plan.detect(out, nsig, capacity=cap)
    for b in range(2):
        assert abs(r2[b]["sigma"] - results[b]["sigma"]) <= 1e-11 * r2[b]["sigma"] and r2[b]["count"] == results[b]["count"]
    # events-only host entry: pieces of 32768 outputs, nothing but triplets and statistics come back
    rh, eh = plan.execute_detect_host(x, cf.n_out, nsig, capacity=cap)
    if dtype == "u8":
        _check_detect(oracle, host, rh, eh, nsig, cap)
    else:
        # The host entry de-disperses in time pieces: tiles, and with them the places where partial sums are
        # handed over, fall elsewhere, so its (device-resident) fp32 buffer may differ from `host` in the
        # last bit of some samples (reading R13).  Statistics agree to fp32 rounding; events may differ
        # only within that rounding of the threshold.
        for b in range(2):
            mu, sg, thr, ev, val = oracle.detect(host[b], nsig)
            assert abs(rh[b]["mean"] - mu) <= 1e-7 * sg and abs(rh[b]["sigma"] - sg) <= 1e-7 * sg
            a = set(zip(eh[b]["t"].tolist(), eh[b]["dm"].tolist()))
            c = set(map(tuple, ev.tolist()))
            for (t, d) in a ^ c:
                assert abs(host[b][d, t] - thr) <= 1e-5 * np.abs(x[b]).sum(axis=0).max()
        # the buffer behind those events (it never left the device): every element against the oracle, and
        # the returned events are exactly oracle.detect's on THAT buffer
        hbuf = plan.host_output(2, cf.n_out, dd.F32).cpu().numpy()
        for b in range(2):
            ref, sa = oracle.brute_f32(x[b], tab, cf.n_out)
            check_f32(hbuf[b], ref, sa)
        _check_detect(oracle, hbuf, rh, eh, nsig, cap)
    with pytest.raises(dd.DedispError):
        plan.host_output(3, cf.n_out)                    # not the shape of the last host call
    plan.close()
    # unfused route (subband plan), same definition
    cs = small_cfg(dtype, nchans=128, ndm=96, n_out=2048 + 33, step=0.25, nsub=8, nfine=12)
    full = oracle.shift_table(cs.nchans, cs.f_top_mhz, cs.df_mhz, cs.t_samp_ms, cs.dm_list)
    xs = synth.make_input(cs, cs.n_out + int(full.max()), [(18, 500, 30, 1.5)], {18: full[18]})[None]
    ps = dd.Plan(**cs.plan_args())
    outs, rs, es = ps.execute_detect(to_dev(xs[:, :, :cs.n_out + ps.max_delay].copy()), cs.n_out, 3.0, capacity=cap)
    _check_detect(oracle, outs.cpu().numpy(), rs, es, 3.0, cap)
    rsh, esh = ps.execute_detect_host(np.ascontiguousarray(xs[:, :, :cs.n_out + ps.max_delay]), cs.n_out, 3.0, capacity=cap)
    _check_detect(oracle, outs.cpu().numpy(), rsh, esh, 3.0, cap)      # one piece, same kernels: same buffer


def test_kernel_timing_hook(oracle):
    cf = small_cfg()
    tab, x = make_case(oracle, cf)
    plan = dd.Plan(**cf.plan_args())
    with pytest.raises(dd.DedispError):
        plan.last_kernel_ms()
    plan.set_timing(True)
    plan.execute(to_dev(x[0]), cf.n_out)
    assert plan.last_kernel_ms() > 0.0


@pytest.mark.parametrize("kernel", ["direct", "long"])
@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_subband_small(oracle, dtype, kernel):
    cf = small_cfg(dtype, nchans=128, ndm=96, n_out=2048 + 33, step=0.25, nsub=8, nfine=12)
    tab = oracle.subband_tables(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list,
                                cf.nsub, cf.nfine)
    full = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = cf.n_out + int(full.max())
    pulses = [(18, 500, 30, 1.5)]
    x = synth.make_input(cf, n_in, pulses, {18: full[18]})
    plan = dd.Plan(**cf.plan_args())
    plan.set_kernel(KERNELS[kernel])
    assert plan.max_delay == tab.max_delay
    plan.set_timing(True)
    got = plan.execute(to_dev(x), cf.n_out).cpu().numpy()
    assert plan.last_launches == 2
    s1_ms, s2_ms = plan.last_stage_ms()
    assert s1_ms > 0.0 and s2_ms > 0.0 and abs(s1_ms + s2_ms - plan.last_kernel_ms()) < 0.05
    ref, sa = oracle.subband(x, tab, cf.n_out)
    if dtype == "u8":
        assert (got == ref).all()
        # P8(i): nominal rows equal brute force exactly
        rows = [k * cf.nfine + cf.nfine // 2 for k in range(tab.ncoarse)]
        assert (got[rows] == oracle.brute_u8(x, full, cf.n_out)[rows]).all()
    else:
        check_f32(got, ref, sa)


def test_cfg4_geometry_subband_scaled(oracle):
    """cfg-4 band and DM grid, 512 of the 4096 channels' subbands kept whole: 4 subbands of 128."""
    base = synth.configs()[4]
    cf = synth.scaled(base, nchans=512, nsub=4, n_out=4096 + 12, ndm=256)
    tab = oracle.subband_tables(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list, 4, 32)
    full = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    x = synth.make_input(cf, cf.n_out + int(full.max()))
    plan = dd.Plan(**cf.plan_args())
    ref, sa = oracle.subband(x, tab, cf.n_out)
    for kernel in ("auto", "direct"):       # auto = the long-tile kernel (rows of >= 4096 samples)
        plan.set_kernel(KERNELS[kernel])
        got = plan.execute(to_dev(x), cf.n_out).cpu().numpy()
        check_f32(got, ref, sa)


@pytest.mark.parametrize("chunk_rel", ["larger", "smaller"])
@pytest.mark.parametrize("dtype", ["u8", "f32"])
@pytest.mark.parametrize("kernel", ["auto", "window"])
def test_streaming_equals_one_shot(oracle, dtype, chunk_rel, kernel):
    cf = small_cfg(dtype, nchans=64, ndm=40, n_out=0, step=0.3) if kernel == "auto" else \
        synth.scaled(synth.configs()[1], dtype=dtype, nchans=64, ndm=40, n_out=0)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    M = int(tab.max())
    C = (M + 200) // 4 * 4 if chunk_rel == "larger" else max(16, (M // 3) // 4 * 4)
    npush, beams = 5, 2
    total = npush * C
    xs = np.stack([synth.make_input(cf, total, [(7, M + 10, 12, 2.0)], {7: tab[7]}, beam=b)
                   for b in range(beams)])
    plan = dd.Plan(**cf.plan_args())
    plan.set_kernel(KERNELS[kernel])
    st = dd.Stream(plan, dd.U8 if dtype == "u8" else dd.F32, C, beams)
    outs = []
    for k in range(npush):
        outs.append(st.push(torch.from_numpy(np.ascontiguousarray(xs[:, :, k * C:(k + 1) * C])).cuda())
                    .cpu().numpy())
    got = np.concatenate(outs, axis=2)[:, :, M:]          # drop the warm-up outputs (reading R9)
    n = total - M
    for b in range(beams):
        if dtype == "u8":
            assert (got[b] == oracle.brute_u8(xs[b], tab, n)).all()
        else:
            ref, sa = oracle.brute_f32(xs[b], tab, n)
            check_f32(got[b], ref, sa)
    # warm-up outputs of push 0 see zeros before the stream start
    st.reset()
    first = st.push(torch.from_numpy(np.ascontiguousarray(xs[:, :, :C])).cuda()).cpu().numpy()
    assert (first == outs[0]).all()
    st.close()
    plan.close()


def test_stream_push_host_pieces(oracle):
    """dedisp_stream_push_host: host chunks copied straight behind the carry in time pieces that
    overlap the kernels; three pushes of 2.2 pieces each equal the one-shot result bit for bit."""
    cf = small_cfg("u8", nchans=48, ndm=24, n_out=0, step=0.6)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    M, C, npush = int(tab.max()), 2 * 16384 + 3000, 3
    xs = synth.make_input(cf, npush * C, [(5, M + 50, 9, 2.0)], {5: tab[5]})[None]
    plan = dd.Plan(**cf.plan_args())
    st = dd.Stream(plan, dd.U8, C, 1)
    outs = []
    for k in range(npush):
        hin = torch.from_numpy(np.ascontiguousarray(xs[:, :, k * C:(k + 1) * C])).pin_memory()
        hout = torch.empty((1, cf.ndm, C), dtype=torch.int32).pin_memory()
        st.push_host(hin, hout)
        outs.append(hout.numpy().copy())
    got = np.concatenate(outs, axis=2)[0][:, M:]
    assert (got == oracle.brute_u8(xs[0], tab, npush * C - M)).all()
    st.close()
    plan.close()


def test_edge_cases(oracle):
    # one channel, one DM, one sample; DM 0 only; nsamp_out = 0
    p = dd.Plan(1, 100.0, 1.0, 1.0, [0.0])
    x = torch.arange(16, dtype=torch.float32, device="cuda").reshape(1, 16)
    assert p.execute(x, 1).cpu().tolist() == [[0.0]]
    assert p.execute(x, 16).cpu().tolist() == [list(map(float, range(16)))]
    assert p.execute(x, 0).shape == (1, 0) and p.last_launches == 0
    # input too short for nsamp_out + max_delay, misaligned stride
    cf = small_cfg()
    plan = dd.Plan(**cf.plan_args())
    M = plan.max_delay
    x = torch.zeros((cf.nchans, (1024 + M + 31) // 16 * 16), dtype=torch.float32, device="cuda")
    with pytest.raises(dd.DedispError) as e:
        plan.execute(x, x.shape[1] - M + 1)            # needs one more input sample than there is
    assert e.value.status == dd.binding.ESHAPE
    with pytest.raises(dd.DedispError) as e:
        plan.execute(x[:, 1:], 512)                    # base pointer not 16-byte aligned
    assert e.value.status == dd.binding.ESHAPE
    with pytest.raises(RuntimeError):
        plan.execute(x.cpu(), 16)
    # constant input (the paper's perf-test buffers): every output = nchans * v
    x.fill_(0.375)
    assert (plan.execute(x, 1024).cpu().numpy() == cf.nchans * 0.375).all()


def test_execute_host_roundtrip(oracle):
    cf = small_cfg("u8", n_out=1500)
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    got = plan.execute_host(x, cf.n_out)
    for b in range(2):
        assert (got[b] == oracle.brute_u8(x[b], tab, cf.n_out)).all()


def test_execute_host_pipelined_chunks(oracle):
    """dedisp_execute_host cuts >= 65536 output samples into time chunks whose copies overlap the
    kernels; ragged last chunk, two beams, bit-exact; pinned and pageable host buffers."""
    cf = synth.scaled(small_cfg("u8", nchans=64, ndm=40, step=0.5), n_out=3 * 32768 + 1234)
    tab, x = make_case(oracle, cf, beams=2)
    plan = dd.Plan(**cf.plan_args())
    got = plan.execute_host(x, cf.n_out)
    xp = torch.from_numpy(x).pin_memory()
    outp = torch.empty((2, cf.ndm, cf.n_out), dtype=torch.int32).pin_memory()
    plan.execute_host(xp, cf.n_out, out=outp)
    for b in range(2):
        ref = oracle.brute_u8(x[b], tab, cf.n_out)
        assert (got[b] == ref).all() and (outp[b].numpy() == ref).all()


def pulse_peak_trial(out_rows, d0, t0, w):
    """argmax over the given DM rows of the boxcar sum over [t0, t0 + w) (P7: SURVEY.md section 8c)."""
    box = np.asarray(out_rows)[:, t0:t0 + w].astype(np.float64).sum(axis=1)
    return d0 + int(np.argmax(box)), box


def test_cfg3_full_size_every_output(oracle):
    """BASELINE cfg 3 at full size in bench.py's launch configuration (AUTO = register-window kernel):
    EVERY one of the 4096 x 262144 outputs against the oracle's triple loop, in slabs of 256 trials
    (1.1e12 oracle adds, about a minute and a half on the box's 16 cores), then P7 on each of the 10
    injected pulses: the boxcar sum over the pulse peaks at its own trial (+-1 where the pulse is wider
    than the sweep difference between neighbouring trials, 10.2 samples at the band bottom)."""
    cf = synth.configs()[3]
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = cf.n_out + int(tab.max())
    pulses = synth.draw_pulses(cf, cf.n_out)
    assert len(pulses) == 10
    x = synth.make_input(cf, n_in, pulses, {p[0]: tab[p[0]] for p in pulses})
    plan = dd.Plan(**cf.plan_args())
    assert plan.resolved_kernel(dd.F32) == dd.KERNEL_WINDOW
    out = plan.execute(to_dev(x), cf.n_out)
    got = out.cpu().numpy()
    del out
    torch.cuda.empty_cache()
    for r0 in range(0, cf.ndm, 256):
        ref, sa = oracle.brute_f32(x, tab[r0:r0 + 256], cf.n_out)
        check_f32(got[r0:r0 + 256], ref, sa)
    for (trial, t0, w, amp) in pulses:
        lo, hi = max(0, trial - 24), min(cf.ndm, trial + 25)
        peak, box = pulse_peak_trial(got[lo:hi], lo, t0, w)
        assert abs(peak - trial) <= 1, (trial, peak, w, amp)
        assert box[trial - lo] > 0.8 * cf.nchans * amp * w      # nchans * a * w plus noise (P7)


def test_cfg2_full_size_every_output(oracle):
    """BASELINE cfg 2 at full size (1024 ch x 2048 trials x 65536 samples, two channel bands in the
    window kernel): every output against the oracle."""
    cf = synth.configs()[2]
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    pulses = synth.draw_pulses(cf, cf.n_out)
    x = synth.make_input(cf, cf.n_out + int(tab.max()), pulses, {p[0]: tab[p[0]] for p in pulses})
    plan = dd.Plan(**cf.plan_args())
    got = plan.execute(to_dev(x), cf.n_out).cpu().numpy()
    for r0 in range(0, cf.ndm, 512):                       # the oracle in slabs of 512 trials (memory)
        ref, sa = oracle.brute_f32(x, tab[r0:r0 + 512], cf.n_out)
        check_f32(got[r0:r0 + 512], ref, sa)


def cfg4_pulses(cf):
    """SURVEY.md section 8d, cfg 4: the 8 drawn pulses, the first 4 moved onto the nominal trial of their
    coarse group (k*32 + 16), the other 4 onto a group edge (k*32 or k*32 + 31)."""
    out = []
    for i, (trial, t0, w, amp) in enumerate(synth.draw_pulses(cf, cf.n_out)):
        k = trial // cf.nfine
        out.append((k * cf.nfine + (cf.nfine // 2 if i < 4 else (0 if i % 2 == 0 else cf.nfine - 1)), t0, w, amp))
    return out


def test_cfg4_full_size_seeded(oracle):
    """BASELINE cfg 4 at full size in bench.py's launch configuration (4096 ch x 555 784 seeded samples =
    9.1 GB, 32 subbands, 128 coarse x 32 fine trials, long-tile kernel for both stages), with the 8 pulses
    of the recipe.  (1) every output of coarse groups 0, 1, 64 and 127 against the stage-by-stage subband
    oracle; (2) P8(i) on the same input: the 128 nominal rows against BRUTE FORCE (oracle.brute_f32);
    (3) the pulses: those on nominal trials peak at their trial with the brute-force sum, those on group
    edges keep most of it ("slight sensitivity loss") and never exceed it by more than noise."""
    cf = synth.configs()[4]
    tab = oracle.subband_tables(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list, cf.nsub, cf.nfine)
    full = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    plan = dd.Plan(**cf.plan_args())
    assert plan.max_delay == tab.max_delay
    n_in = cf.n_out + int(full.max())                   # the brute-force extent (>= the two-stage one)
    pulses = cfg4_pulses(cf)
    x = synth.make_input(cf, n_in, pulses, {p[0]: full[p[0]] for p in pulses})
    stride = (n_in + 15) // 16 * 16
    xd = torch.empty((cf.nchans, stride), dtype=torch.float32, device="cuda")
    for c0 in range(0, cf.nchans, 512):
        xd[c0:c0 + 512, :n_in] = torch.from_numpy(x[c0:c0 + 512]).cuda()
    out = plan.execute(xd[:, :n_in], cf.n_out)
    assert plan.last_launches == 2
    got = out.cpu().numpy()
    del out
    # (4) BRUTE FORCE on the GPU on the same input (BASELINE cfg 4: "also compared against brute force on the
    # same input"): brute-force plans on rows of 4096 channels whose input buffer has 2.28e9
    # elements (> 2^31: 64-bit row offsets) and whose max_delay 424 712 exceeds n_out 131 072.  The direct
    # kernel on the 128 nominal trials + the last 16 (rows 32 DM steps apart: too far for shared staging of the
    # long-tile kernel, which AUTO would therefore not pick), the long-tile kernel on the last 32 contiguous ones.
    nominal = np.arange(tab.ncoarse) * cf.nfine + cf.nfine // 2
    subsets = {"direct": np.concatenate([nominal, np.arange(cf.ndm - 16, cf.ndm)]), "long": np.arange(cf.ndm - 32, cf.ndm)}
    assert cf.nchans * stride > 2 ** 31 and int(full.max()) > cf.n_out
    brute = {}
    for kname, rows in subsets.items():
        bargs = cf.plan_args()
        bargs.update(dm_list=np.asarray(cf.dm_list)[rows], nsub=0, nfine=0)
        bp = dd.Plan(**bargs)
        assert (bp.shifts() == full[rows]).all() and bp.max_delay == int(full.max())
        bp.set_kernel(KERNELS[kname])
        brute[kname] = bp.execute(xd[:, :n_in], cf.n_out).cpu().numpy()
        assert bp.last_kernel == KERNELS[kname] and bp.last_launches == 1
        bp.close()
    del xd
    torch.cuda.empty_cache()
    for kname, rows in subsets.items():
        ref, sa = oracle.brute_f32(x, full[rows], cf.n_out)
        check_f32(brute[kname], ref, sa)
        if kname == "direct":
            bref, bsa = ref, sa
    # (1) subband GPU vs subband oracle, every output of four groups
    for k in (0, 1, 64, 127):
        ref, sa = oracle.subband(x, tab, cf.n_out, groups=[k])
        check_f32(got[k * cf.nfine:(k + 1) * cf.nfine], ref, sa)
    # (2) nominal rows equal brute force (reading R8)
    check_f32(got[nominal], bref[:len(nominal)], bsa[:len(nominal)])
    # (3) pulses
    for i, (trial, t0, w, amp) in enumerate(pulses):
        k = trial // cf.nfine
        bf = oracle.brute_f32(x, full[trial:trial + 1], cf.n_out, want_sumabs=False)[0, t0:t0 + w].sum()
        lo = k * cf.nfine
        peak, box = pulse_peak_trial(got[lo:lo + cf.nfine], lo, t0, w)
        assert bf > 0.9 * cf.nchans * amp * w
        if i < 4:
            assert peak == trial and abs(box[trial - lo] - bf) <= 1e-5 * np.abs(x).max() * cf.nchans * w
        else:
            # an edge trial is 0.75-0.8 DM units off its group's nominal DM: up to ~70 samples of smear
            # inside a subband against pulse widths of 40-200 samples
            ref, sa = oracle.subband(x, tab, cf.n_out, groups=[k])
            check_f32(got[lo:lo + cf.nfine], ref, sa)
            assert 0.2 * bf < box[trial - lo] < bf + 6 * np.sqrt(cf.nchans * w)
    plan.close()


def test_cfg5_full_size_all_pushes(oracle):
    """BASELINE cfg 5 at full size: ALL 16 pushes of 4 beams x 2048 ch x 65536 uint8 samples through
    dedisp_stream_push (3072 trials, max_delay 24 875 carried from chunk to chunk).  Per beam 8 drawn
    pulses plus 3 placed so that their sweep crosses a chunk boundary.  Beam 0: every 8th DM row over the
    whole stream, bit-exact against the one-shot oracle (reading R9: the concatenation of the pushes IS the
    one-shot result); beams 1-3: 400 outputs each, recomputed one by one, spread over all pushes."""
    cf = synth.configs()[5]
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    M, C, nb, npush = int(tab.max()), cf.n_out, cf.nbeams, cf.nchunks
    total = npush * C
    n = total - M                                                # stream times with a full sweep
    xs = []
    for b in range(nb):
        pulses = synth.draw_pulses(cf, n, beam=b)
        for k in (3, 7, 12):                                      # sweep of trial 3000 straddles input chunk k
            pulses.append((3000, k * C - int(tab[3000].max()) // 2, 12, 1.5))
        xs.append(synth.make_input(cf, total, pulses, {p[0]: tab[p[0]] for p in pulses}, beam=b))
    rows = np.arange(0, cf.ndm, 8)
    rng = np.random.default_rng(5)
    sd = np.r_[rng.integers(0, cf.ndm, 380), [0, cf.ndm - 1] * 10]
    st_ = np.r_[rng.integers(0, n, 380), [0, n - 1, C - M - 1, C - M] * 5]       # stream times
    plan = dd.Plan(**cf.plan_args())
    stream = dd.Stream(plan, dd.U8, C, nb)
    out = torch.empty((nb, cf.ndm, C), dtype=torch.int32, device="cuda")
    got0 = np.empty((len(rows), total), dtype=np.int32)
    gots = np.zeros((nb, len(sd)), dtype=np.int64)
    rows_d = torch.from_numpy(rows).cuda()
    for k in range(npush):
        chunk = np.ascontiguousarray(np.stack([x[:, k * C:(k + 1) * C] for x in xs]))
        stream.push(torch.from_numpy(chunk).cuda(), out)
        got0[:, k * C:(k + 1) * C] = out[0][rows_d].cpu().numpy()
        sel = np.nonzero((st_ + M) // C == k)[0]                  # output (d, t) leaves in push (t + M) // C
        if len(sel):
            dd_ = torch.from_numpy(sd[sel]).cuda()
            tl = torch.from_numpy((st_[sel] + M) - k * C).cuda()
            for b in range(1, nb):
                gots[b, sel] = out[b][dd_, tl].cpu().numpy()
    ref0 = oracle.brute_u8(xs[0], tab[rows], n)
    assert (got0[:, M:] == ref0).all()
    for b in range(1, nb):
        ref, _ = oracle.brute_samples(xs[b], tab, sd, st_)
        assert (gots[b] == ref).all()
    # the 3 straddling pulses of beam 0 are recovered at trial 3000 (a row of the checked subset)
    r3000 = int(np.nonzero(rows == 3000)[0][0])
    for k in (3, 7, 12):
        t0 = k * C - int(tab[3000].max()) // 2
        box = got0[:, M + t0:M + t0 + 12].astype(np.int64).sum(axis=1)
        assert abs(int(np.argmax(box)) - r3000) <= 1
    stream.close()
    plan.close()


def test_power_corner_turn_matches_oracle(oracle):
    """dedisp_power_corner_turn: bit-exact against the fp32-defined oracle on ragged
    shapes (tiles of 64 x 64), a strided voltage buffer, and chained into a de-dispersion."""
    rng = np.random.default_rng(11)
    for nsamp, nchans, pad in ((1, 1, 0), (130, 67, 0), (1000, 128, 5), (4099, 200, 0)):
        z = (rng.standard_normal((nsamp, nchans + pad)) + 1j * rng.standard_normal((nsamp, nchans + pad))).astype(np.complex64)
        zd = torch.from_numpy(z).cuda()[:, :nchans]
        got = dd.power_corner_turn(zd).cpu().numpy()
        ref, _ = oracle.power_corner_turn(z[:, :nchans])
        assert got.shape == ref.shape and (got == ref).all()
    with pytest.raises(dd.DedispError):
        dd.power_corner_turn(torch.zeros((4, 4), dtype=torch.float32, device="cuda"))
    # voltages -> power in channel order -> de-dispersion, against the oracle chain
    cf = small_cfg("f32", nchans=64, ndm=20, n_out=1500)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = cf.n_out + int(tab.max())
    z = (rng.standard_normal((n_in, cf.nchans)) + 1j * rng.standard_normal((n_in, cf.nchans))).astype(np.complex64)
    p = dd.power_corner_turn(torch.from_numpy(z).cuda())
    plan = dd.Plan(**cf.plan_args())
    got = plan.execute(p, cf.n_out).cpu().numpy()
    ref, sa = oracle.brute_f32(oracle.power_corner_turn(z)[0], tab, cf.n_out)
    check_f32(got, ref, sa)


def test_binning_matches_oracle_and_feeds_a_pass(oracle):
    """dedisp_bin (eq. 6): bit-exact against the fp32-defined oracle for several bin
    factors and ragged lengths; then one survey pass with bin factor 2 (Table 1): binned input
    de-dispersed by a plan created with 2 * t_samp, against the oracle chain."""
    rng = np.random.default_rng(12)
    x = rng.standard_normal((3, 17, 1003)).astype(np.float32)
    xd = to_dev(x)
    for nb in (1, 2, 3, 4, 8):
        got = dd.bin_samples(xd, nb).cpu().numpy()
        ref, _ = oracle.bin_samples(x, nb)
        assert got.shape == ref.shape and (got == ref).all()
    with pytest.raises(dd.DedispError):
        dd.bin_samples(xd.to(torch.float64), 2)
    cf = small_cfg("f32", nchans=48, ndm=30, n_out=900, step=0.5)
    cfb = synth.scaled(cf, t_samp_ms=2 * cf.t_samp_ms)
    tab = oracle.shift_table(cfb.nchans, cfb.f_top_mhz, cfb.df_mhz, cfb.t_samp_ms, cfb.dm_list)
    n_in = 2 * (cfb.n_out + int(tab.max()))
    raw = synth.make_input(cf, n_in)
    plan = dd.Plan(**cfb.plan_args())
    got = plan.execute(dd.bin_samples(to_dev(raw), 2), cfb.n_out).cpu().numpy()
    ref, sa = oracle.brute_f32(oracle.bin_samples(raw, 2)[0], tab, cfb.n_out)
    check_f32(got, ref, sa)


def test_survey_table4_matches_oracle_chain(oracle):
    """dedisp_survey_execute on the paper's Table 4 plan: 1024 channels over 16 MHz at
    300 MHz, 3 passes (bin 1 / 2 / 4; 22 / 24 / 24 fine trials per nominal DM, i.e. row tiles that are no
    multiple of the long-tile kernel's 16 rows), 3102 trials, 8192 input samples.  Per pass binning ->
    stage 1 -> stage 2 run on the device; every output against oracle.survey (bin_samples -> subband)."""
    from test_oracle_pins import table4_passes
    nch, ft, df, ts, nsub, nsamp = 1024, 308.0, 16.0 / 1024, 0.1, 32, 8192
    passes = table4_passes()
    sv = dd.Survey(nch, ft, df, ts, nsub, passes)
    M = sv.max_delay
    cf = synth.Config("table4", nch, ft, df, ts, nsamp, 1, 0.0, seed=404)
    x = synth.make_input(cf, nsamp + M)
    # a pulse at a nominal trial of pass 3 (unbinned dispersion curve), 12.8 ms wide
    dmp = passes[2][0] + (24 + 12) * passes[2][1]
    row = oracle.shift_table(nch, ft, df, ts, np.array([dmp]))[0]
    for c in range(nch):
        x[c, 1000 + row[c]:1000 + row[c] + 128] += 1.0
    outs = sv.execute(to_dev(x), nsamp)
    assert sv.last_launches == 2 * 3 + 2                     # two stages per pass, binning for bin 2 and 4
    ref = oracle.survey(x, nch, ft, df, ts, nsub, passes, nsamp)
    for i, (o, (r, sa, dm)) in enumerate(zip(outs, ref)):
        assert tuple(o.shape) == r.shape == (passes[i][2], nsamp // passes[i][4])
        check_f32(o.cpu().numpy(), r, sa)
    box = outs[2].cpu().numpy()[:, 1000 // 4:(1000 + 128) // 4].sum(axis=1)
    assert int(np.argmax(box)) == 24 + 12
    sv.close()


def test_survey_small_two_beams(oracle):
    nch, ft, df, ts, nsub, nsamp = 64, 150.0, 0.1, 0.2, 8, 4096 + 40
    passes = [(0.0, 0.25, 24, 12, 1), (6.0, 0.5, 12, 6, 2), (12.0, 1.0, 9, 3, 3)]
    sv = dd.Survey(nch, ft, df, ts, nsub, passes)
    M = sv.max_delay
    rng = np.random.default_rng(9)
    x = rng.standard_normal((2, nch, nsamp + M)).astype(np.float32)
    outs = sv.execute(to_dev(x), nsamp)
    for b in range(2):
        ref = oracle.survey(x[b], nch, ft, df, ts, nsub, passes, nsamp)
        for o, (r, sa, dm) in zip(outs, ref):
            check_f32(o[b].cpu().numpy(), r, sa)
    with pytest.raises(dd.DedispError):
        sv.execute(to_dev(x[:, :, :nsamp + M - 1]), nsamp)        # one input sample short


@pytest.mark.parametrize("world", [2, 3])
def test_dm_sharded_execute_equals_the_whole(oracle, world):
    """"The DM range is split among these threads, such that each will process the same input
    buffer for different DM values."  Every rank's plan is built from its shard.dm_slice of the DM list
    (subband plans: whole coarse groups) and executed on the SAME input; the concatenation of the shards'
    rows is the whole result: against the oracle's one-plan result, brute force (uint8, bit-exact) and
    two-stage (fp32).  The ranks run one after the other on the one GPU: the path has no exchange step."""
    from paper_1107_2516_b200 import shard
    # brute force: cfg-1 band, 67 trials (no multiple of the world size), uint8
    cf = synth.scaled(synth.configs()[1], dtype="u8", ndm=67, n_out=4096 + 100)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    x = synth.make_input(cf, cf.n_out + int(tab.max()))          # the extent of the WHOLE list, on every rank
    xd = to_dev(x)
    parts = []
    for rank in range(world):
        lo, hi = shard.dm_slice(cf.ndm, world, rank)
        plan = dd.Plan(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list[lo:hi])
        assert (plan.shifts() == tab[lo:hi]).all() and plan.max_delay <= int(tab.max())
        parts.append(plan.execute(xd, cf.n_out).cpu().numpy())
    assert (np.concatenate(parts, axis=0) == oracle.brute_u8(x, tab, cf.n_out)).all()
    # two-stage: cfg-4 band, 256 channels in 4 subbands, 5 coarse groups of 32 trials
    cs = synth.scaled(synth.configs()[4], nchans=256, nsub=4, ndm=5 * 32, n_out=4096 + 24)
    t = oracle.subband_tables(cs.nchans, cs.f_top_mhz, cs.df_mhz, cs.t_samp_ms, cs.dm_list, cs.nsub, cs.nfine)
    xs = synth.make_input(cs, cs.n_out + t.max_delay)
    xsd = to_dev(xs)
    parts = []
    for rank in range(world):
        lo, hi = shard.dm_slice(cs.ndm, world, rank, multiple=cs.nfine)
        plan = dd.Plan(cs.nchans, cs.f_top_mhz, cs.df_mhz, cs.t_samp_ms, cs.dm_list[lo:hi], cs.nsub, cs.nfine)
        parts.append(plan.execute(xsd, cs.n_out).cpu().numpy())
    ref, sa = oracle.subband(xs, t, cs.n_out)
    check_f32(np.concatenate(parts, axis=0), ref, sa)


def test_execute_is_asynchronous_and_allocation_free(oracle):
    """include/dedisp.h conventions: after dedisp_plan_reserve, dedisp_execute only
    enqueues on the caller's stream.  A one-second spin kernel is queued on a side stream, then two
    executes: both calls return while the stream is still busy (cudaStreamQuery != cudaSuccess), the
    device allocator is untouched between them, and the result is right once the stream drains.  Without
    a covering reservation execute refuses (DEDISP_ESTATE) instead of allocating."""
    cf = synth.scaled(synth.configs()[1], dtype="u8", ndm=48, n_out=8192)
    tab, x = make_case(oracle, cf)
    plan = dd.Plan(**cf.plan_args())
    xd = to_dev(x[0])
    out = torch.empty((cf.ndm, cf.n_out), dtype=torch.int32, device="cuda")
    L = dd.lib()
    st = L.dedisp_execute(plan._h, xd.data_ptr(), out.data_ptr(), dd.U8, cf.n_out, xd.stride(0), cf.n_out, 1, 0)
    assert st == dd.binding.ESTATE                                   # no reservation: no lazy allocation
    plan.reserve(dd.U8, cf.n_out, 1)
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    with torch.cuda.stream(side):
        torch.cuda._sleep(2_000_000_000)                             # about a second of device time
        for _ in range(2):
            st = L.dedisp_execute(plan._h, xd.data_ptr(), out.data_ptr(), dd.U8, cf.n_out, xd.stride(0), cf.n_out, 1,
                                  side.cuda_stream)
            assert st == dd.binding.OK
            assert not side.query()                                  # returned with the stream still busy
    assert torch.cuda.mem_get_info()[0] == free0                     # nothing allocated or freed by execute
    side.synchronize()
    assert (out.cpu().numpy() == oracle.brute_u8(x[0], tab, cf.n_out)).all()
    st = L.dedisp_execute(plan._h, xd.data_ptr(), out.data_ptr(), dd.U8, 2 * cf.n_out, xd.stride(0), 2 * cf.n_out, 1, 0)
    assert st in (dd.binding.ESTATE, dd.binding.ESHAPE)              # beyond the reservation / the input


def test_reserve_covers_shorter_executes_and_binding_bookkeeping(oracle):
    """dedisp_plan_reserve promises executes of UP TO nsamp_out samples (include/dedisp.h).  (i) A reserve
    beyond the register-window kernel's 32-bit time limit (2 channels x 2^30 samples: 17 GB of pair
    scratch) must still size the pair buffer for the shorter executes that resolve to that kernel.
    (ii) The binding must not take reserve(100, 4 beams) + reserve(1000, 1 beam) for a reservation of
    1000 samples x 4 beams."""
    dm = np.arange(16) * 0.4
    plan = dd.Plan(2, 150.0, 0.1, 0.2, dm)
    plan.reserve(dd.F32, (1 << 30) + 4096, 1)
    assert plan.resolved_kernel(dd.F32) == dd.KERNEL_WINDOW
    tab = oracle.shift_table(2, 150.0, 0.1, 0.2, dm)
    n_out = 450000                                   # >= 148 window tiles, so AUTO keeps the window kernel
    x = np.random.default_rng(5).standard_normal((2, n_out + int(tab.max()))).astype(np.float32)
    got = plan.execute(to_dev(x), n_out).cpu().numpy()     # covered by the reserve above: no second reserve
    assert plan.last_launches == 2 and plan.last_kernel == dd.KERNEL_WINDOW     # pairify + one band
    ref, sa = oracle.brute_f32(x, tab, n_out)
    check_f32(got, ref, sa)
    plan.close()
    torch.cuda.empty_cache()

    cf = small_cfg("u8")
    tab, x = make_case(oracle, cf, n_out=1000, beams=4)
    plan = dd.Plan(**cf.plan_args())
    plan.reserve(dd.U8, 100, 4)
    plan.reserve(dd.U8, 1000, 1)
    got = plan.execute(to_dev(x), 1000).cpu().numpy()
    for b in range(4):
        assert (got[b] == oracle.brute_u8(x[b], tab, 1000)).all()


def test_last_kernel_reports_what_ran(oracle):
    """dedisp_plan_last_kernel follows AUTO's size rule (dedisp_plan_resolved_kernel does not): cfg 1 has 15
    register-window tiles for 148 SMs and runs one thread per output; the host entry judges the whole
    buffer once, so its time pieces all run one kernel -- checked through the result being bit-identical
    to the device entry's (same kernel, same fp32 summation order) on a buffer cut into pieces."""
    cf = synth.configs()[1]
    tab, x = make_case(oracle, cf)
    plan = dd.Plan(**cf.plan_args())
    assert plan.resolved_kernel(dd.F32) == dd.KERNEL_WINDOW and plan.last_kernel == -1
    got = plan.execute(to_dev(x[0]), cf.n_out).cpu().numpy()
    assert plan.last_kernel == dd.KERNEL_NAIVE
    ref, sa = oracle.brute_f32(x[0], tab, cf.n_out)
    check_f32(got, ref, sa)
    # 64 trials x 70000 samples: 4 x 25 window tiles < 148 -> "small" as a whole; the host entry cuts it into
    # 2 pieces (+ the split first one) which must not be judged one by one
    cf2 = synth.scaled(cf, n_out=70000)
    tab2, x2 = make_case(oracle, cf2)
    p2 = dd.Plan(**cf2.plan_args())
    dev = p2.execute(to_dev(x2[0]), cf2.n_out).cpu().numpy()
    k = p2.last_kernel
    assert k in (dd.KERNEL_NAIVE, dd.KERNEL_DIRECT)
    host = p2.execute_host(x2[0], cf2.n_out)
    assert p2.last_kernel == k and (np.asarray(host) == dev).all()


@pytest.mark.parametrize("seed", range(12))
def test_window_kernel_random_stress(oracle, seed):
    """Randomised coverage of the register-window kernel's producer / consumer ring (the class of defect a
    sanitizer would look for; compute-sanitizer is closed on this pool, profiles/r2_sanitizer.md): per seed a
    random instantiated shape, band (cfg 2 / 3 / 5), channel count, DM step, DM offset and count, output
    length from one sample to several blocks, 1-3 beams; uint8, so any lost, doubled or misplaced sample
    changes an integer.  A shape whose ring does not fit the table falls back to the plan's own shape.  Run
    twice on the same buffers: the second execute must reproduce the first bit for bit."""
    rng = np.random.default_rng(7000 + seed)
    T, G, NT, D = GEOMS[int(rng.integers(len(GEOMS)))]
    base = synth.configs()[int(rng.choice([2, 3, 5]))]
    nchans = int(rng.choice([33, 64, 200, 384, 1024]))
    ndm = int(rng.integers(1, 3 * D * G + 1))
    n_out = int(rng.integers(1, 5 * 2 * NT * 32 * T))
    beams = int(rng.integers(1, 4))
    step = float(base.dm_step * rng.choice([0.5, 1.0, 2.0]))
    first = int(rng.integers(0, base.ndm))                 # where in the DM range the rows sit
    dm = (first + np.arange(ndm)) * step
    cf = synth.scaled(base, dtype="u8", n_out=n_out, ndm=ndm, nchans=nchans, dm_step=step, seed=100 + seed)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm)
    n_in = n_out + int(tab.max())
    x = np.stack([synth.make_input(cf, n_in, beam=b) for b in range(beams)])
    plan = dd.Plan(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm)
    assert (plan.shifts() == tab).all()
    try:
        plan.set_window_geometry(T, G, NT, D)
    except dd.DedispError as e:
        assert e.status == dd.binding.ESTATE
    info = plan.window_info()
    if not info["ok"]:
        pytest.skip("table outside the register-window kernel's limits for every shape")
    plan.set_kernel(dd.KERNEL_WINDOW)
    xd = to_dev(x)
    got = plan.execute(xd, n_out).cpu().numpy()
    assert plan.last_launches == 1 + info["nband"]
    for b in range(beams):
        assert (got[b] == oracle.brute_u8(x[b], tab, n_out)).all(), (seed, (T, G, NT, D), nchans, ndm, n_out, beams)
    assert (plan.execute(xd, n_out).cpu().numpy() == got).all()
