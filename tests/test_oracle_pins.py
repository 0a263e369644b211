"""Pins for the CPU oracle (no GPU, no product code): the oracle is checked against what the
paper and the mathematics fix, never against itself.

Pin numbers follow DESIGN.md "Oracle pins" (P1..P9).  PAPER.md citations: eq. 1 :21-24,
definition :26, constant-input perf buffers :191, fake-pulsar recipe :187-189, subband :129-135.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_1107_2516_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append(line.split())
    return out


# ---------------------------------------------------------------- P1: eq. 1 delays
def test_p1_eq1_hand_values(oracle):
    for ft, df, ts, c, dm, x, s in _rows("eq1_delays.txt"):
        ft, df, ts, dm, x = map(float, (ft, df, ts, dm, x))
        c, s = int(c), int(s)
        tab = oracle.shift_table(c + 1, ft, df, ts, [dm])
        assert tab[0, c] == s
        assert abs(oracle.delay_samples(c, ft, df, ts, dm) - x) < 1e-5


def test_p1_exact_rational_agreement(oracle):
    """Every entry of a small table equals floor(x+1/2) with x evaluated in exact rational
    arithmetic from eq. 1 (no entry of this table is within 1e-9 of a tie)."""
    ft, df, ts = "150.0", "0.05", "0.1"
    dms = [Fraction(k, 10) for k in range(0, 64, 7)]
    tab = oracle.shift_table(128, float(ft), float(df), float(ts), [float(d) for d in dms])
    for di, dm in enumerate(dms):
        for c in range(0, 128, 5):
            f_c = Fraction(ft) - c * Fraction(df)
            x = Fraction(4150000) * (1 / f_c ** 2 - 1 / Fraction(ft) ** 2) * dm / Fraction(ts)
            assert abs((x % 1) - Fraction(1, 2)) > Fraction(1, 10 ** 9)
            assert tab[di, c] == (x + Fraction(1, 2)).__floor__()


def test_p1_structure(oracle):
    for k in (1, 2, 5):
        cf = synth.configs()[k]
        tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
        assert (tab[:, 0] == 0).all() and (tab[0, :] == 0).all()
        assert (np.diff(tab, axis=1) >= 0).all()      # lower frequency -> later
        assert (np.diff(tab, axis=0) >= 0).all()      # larger DM -> later
    # |shift - x| <= 0.5 on a sample of entries
    cf = synth.configs()[3]
    dm = cf.dm_list
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm)
    rng = np.random.default_rng(1)
    for _ in range(200):
        d, c = int(rng.integers(cf.ndm)), int(rng.integers(cf.nchans))
        x = oracle.delay_samples(c, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm[d])
        assert abs(tab[d, c] - x) <= 0.5
    assert tab.max() == 41917                       # SURVEY.md §8 table / eq1_delays.txt


def test_p1_max_delay_all_configs(oracle):
    want = {1: 1050, 2: 36275, 3: 41917, 5: 24875}
    for k, m in want.items():
        cf = synth.configs()[k]
        dm = cf.dm_list[-1:]
        tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, dm)
        assert tab.max() == m == tab[0, -1]


def test_p1_ties_follow_the_canonical_order(oracle):
    """Exact .5 ties of cfg 5 (reading R4): the table is defined by the stated fp64 op order."""
    cf = synth.configs()[5]
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    for d, c, s in _rows("ties_cfg5.txt"):
        d, c, s = int(d), int(c), int(s)
        f_c = Fraction(cf.f_top_mhz) - c * Fraction(cf.df_mhz)
        x = (Fraction(4150000) * (1 / f_c ** 2 - 1 / Fraction(cf.f_top_mhz) ** 2)
             * Fraction(cf.dm_list[d]) / Fraction(cf.t_samp_ms))
        # 0.064 is not a dyadic rational: the tie is exact for the decimal t_samp 64/1000
        x_dec = x * Fraction(cf.t_samp_ms) / Fraction(64, 1000)
        assert x_dec.denominator == 2, "golden row is not an exact tie"
        assert tab[d, c] == s
        assert s in (x_dec.__floor__(), x_dec.__ceil__())


def test_shift_table_rejects_bad_arguments(oracle):
    with pytest.raises(ValueError):
        oracle.shift_table(4, 200.0, -25.0, 40.0, [0.0])
    with pytest.raises(ValueError):
        oracle.shift_table(4, 200.0, 25.0, 40.0, [-1.0])
    with pytest.raises(ValueError):
        oracle.shift_table(9, 200.0, 25.0, 40.0, [1.0])      # lowest channel at 0 MHz
    with pytest.raises(ValueError):
        oracle.shift_table(4, 200.0, 25.0, 0.0, [1.0])


# ---------------------------------------------------------------- P6: 4-channel toy
def test_p6_toy4(oracle):
    rows = np.array(_rows("toy4.txt"), dtype=np.int64)
    tab = oracle.shift_table(4, 200.0, 25.0, 40.0, [0.0, 1.0, 2.0, 3.0])
    assert (tab == rows).all()
    n_out, n_in = 50, 50 + 12
    x = (100.0 * np.arange(4)[:, None] + np.arange(n_in)[None, :]).astype(np.float32)
    out, sa = oracle.brute_f32(x, tab, n_out)
    t = np.arange(n_out)
    for d, k in enumerate((600, 607, 614, 620)):      # hand-computed in toy4.txt
        assert (out[d] == k + 4 * t).all()
        assert (sa[d] == k + 4 * t).all()
    xu = (10 * np.arange(4)[:, None] + np.arange(n_in)[None, :]).astype(np.uint8)
    outu = oracle.brute_u8(xu, tab, n_out)
    for d, k in enumerate((60, 67, 74, 80)):
        assert (outu[d] == k + 4 * t).all()


# ---------------------------------------------------------------- P2, P3: DM 0, constant input
def _small_case(oracle, dtype="f32", nchans=24, ndm=9, n_out=301, seed=5):
    cf = synth.Config("small", nchans, 150.0, 0.25, 0.5, n_out, ndm, 1.5, dtype=dtype, seed=seed)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = n_out + int(tab.max())
    x = synth.make_input(cf, n_in, threads=1)
    return cf, tab, x


def test_p2_dm0_is_channel_sum(oracle):
    cf, tab, x = _small_case(oracle)
    out, sa = oracle.brute_f32(x, tab, cf.n_out)
    assert np.allclose(out[0], x[:, :cf.n_out].sum(axis=0, dtype=np.float64), rtol=0, atol=1e-12)
    assert np.allclose(sa[0], np.abs(x[:, :cf.n_out]).sum(axis=0, dtype=np.float64), atol=1e-12)
    cf, tab, x = _small_case(oracle, "u8")
    out = oracle.brute_u8(x, tab, cf.n_out)
    assert (out[0] == x[:, :cf.n_out].astype(np.int64).sum(axis=0)).all()


def test_p3_constant_input(oracle):
    cf, tab, x = _small_case(oracle)
    x[:] = np.float32(0.375)
    out, _ = oracle.brute_f32(x, tab, cf.n_out)
    assert (out == cf.nchans * 0.375).all()
    xu = np.full(x.shape, 201, dtype=np.uint8)
    assert (oracle.brute_u8(xu, tab, cf.n_out) == cf.nchans * 201).all()


# ---------------------------------------------------------------- P4: impulse response
def test_p4_impulse_response_covers_every_table_entry(oracle):
    cf, tab, x = _small_case(oracle, nchans=12, ndm=7, n_out=120)
    n_in = x.shape[1]
    for c0 in range(cf.nchans):
        x[:] = 0
        u0 = int(tab[:, c0].max()) + 17
        x[c0, u0] = 1.0
        out, _ = oracle.brute_f32(x, tab, cf.n_out)
        want = np.zeros_like(out)
        hits = 0
        for d in range(cf.ndm):
            if 0 <= u0 - tab[d, c0] < cf.n_out:
                want[d, u0 - tab[d, c0]] = 1.0
                hits += 1
        assert hits >= 1 and (out == want).all()
    assert n_in == cf.n_out + tab.max()


# ---------------------------------------------------------------- P5: linearity, time shift
def test_p5_linearity_and_time_shift(oracle):
    cf, tab, x = _small_case(oracle, "u8")
    y = synth.make_input(synth.scaled(cf, seed=99), x.shape[1], threads=1)
    a = oracle.brute_u8(x // 2, tab, cf.n_out).astype(np.int64)
    b = oracle.brute_u8(y // 2, tab, cf.n_out).astype(np.int64)
    ab = oracle.brute_u8((x // 2 + y // 2).astype(np.uint8), tab, cf.n_out)
    assert (ab == a + b).all()
    tau = 13
    full = oracle.brute_u8(x, tab, cf.n_out - tau)
    shifted = oracle.brute_u8(np.ascontiguousarray(x[:, tau:]), tab, cf.n_out - tau)
    ref = oracle.brute_u8(x, tab, cf.n_out)
    assert (shifted == ref[:, tau:]).all() and (full == ref[:, :cf.n_out - tau]).all()


def test_brute_samples_equals_definition(oracle):
    cf, tab, x = _small_case(oracle)
    out, sa = oracle.brute_f32(x, tab, cf.n_out)
    rng = np.random.default_rng(3)
    d = rng.integers(0, cf.ndm, 40)
    t = rng.integers(0, cf.n_out, 40)
    o, s = oracle.brute_samples(x, tab, d, t)
    assert np.allclose(o, out[d, t], rtol=0, atol=1e-12) and np.allclose(s, sa[d, t], atol=1e-12)
    # and against a literal python triple loop on a handful
    for i in range(5):
        acc = 0.0
        for c in range(cf.nchans):
            acc += float(x[c, t[i] + tab[d[i], c]])
        assert abs(acc - o[i]) < 1e-12


# ---------------------------------------------------------------- P7: pulse recovery
def test_p7_noise_free_pulse_peaks_at_true_trial(oracle):
    cf = synth.scaled(synth.configs()[1], n_out=2048)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = cf.n_out + int(tab.max())
    trial, t0, w, amp = 30, 700, 10, 3.0
    x = np.zeros((cf.nchans, n_in), dtype=np.float32)
    for c in range(cf.nchans):
        x[c, t0 + tab[trial, c]: t0 + tab[trial, c] + w] += amp
    out, _ = oracle.brute_f32(x, tab, cf.n_out)
    win = out[:, t0:t0 + w].sum(axis=1)
    assert win[trial] == cf.nchans * amp * w
    for d in range(cf.ndm):
        if (tab[d] != tab[trial]).any():
            assert win[d] < win[trial]
    assert out[trial].max() == cf.nchans * amp


def test_p7_cfg1_noisy_pulse_recovered(oracle):
    cf = synth.scaled(synth.configs()[1], n_out=4096)
    tab = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    n_in = cf.n_out + int(tab.max())
    pulses = cf.fixed_pulses
    x = synth.make_input(cf, n_in, pulses, {p[0]: tab[p[0]] for p in pulses}, threads=1)
    out, _ = oracle.brute_f32(x, tab, cf.n_out)
    w = pulses[0][2]
    box = np.cumsum(np.pad(out, ((0, 0), (1, 0))), axis=1)
    sm = box[:, w:] - box[:, :-w]
    d_best, t_best = np.unravel_index(np.argmax(sm), sm.shape)
    assert d_best == pulses[0][0] == 30 and abs(t_best - pulses[0][1]) <= 1
    # per-sample S/N at the true trial: amp*sqrt(nchans) = 3*sqrt(128) = 33.9
    snr = out[30, pulses[0][1]:pulses[0][1] + w].mean() / np.sqrt(cf.nchans)
    assert 30.0 < snr < 38.0


def test_p7_paper_fake_pulsar_statistic(oracle):
    """1024 channels, pulse height 8/sqrt(1024) = 0.25 per channel on N(0,1)
    -> S/N 8 after integrating the channels, at the DM-75 trial (Table 2 parameters)."""
    nch, ft, df, ts = 1024, 156.0, 0.005941, 0.165
    dm = np.arange(70, 81, dtype=np.float64)            # trial 5 = DM 75
    cf = synth.Config("fake", nch, ft, df, ts, 2048, dm.size, 1.0, seed=77)
    tab = oracle.shift_table(nch, ft, df, ts, dm)
    n_in = cf.n_out + int(tab.max())
    w = 60                                              # 1 % duty of P = 1000 ms -> 10 ms
    pulses = [(5, 500, w, 0.25), (5, 1500, w, 0.25)]
    x = synth.make_input(cf, n_in, pulses, {5: tab[5]}, threads=1)
    out, _ = oracle.brute_f32(x, tab, cf.n_out)
    off = np.r_[out[5, :400], out[5, 700:1400]]
    on = np.r_[out[5, 500:500 + w], out[5, 1500:1500 + w]]
    snr = (on.mean() - off.mean()) / off.std()
    assert abs(off.std() - 32.0) < 2.5                  # sqrt(1024)
    assert 7.0 < snr < 9.0                              # paper: S/N of 8
    assert on.mean() > out[0, 500:500 + w].mean() + 100  # smeared away at DM 70


# ---------------------------------------------------------------- P8: subband special cases
def _sub_case(oracle, nsub, nfine=4, nchans=32, ndm=16, n_out=257, dtype="f32"):
    cf = synth.Config("sub", nchans, 150.0, 0.25, 0.25, n_out, ndm, 0.5, dtype=dtype, seed=8,
                      nsub=nsub, nfine=nfine)
    full = oracle.shift_table(nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    tab = oracle.subband_tables(nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list, nsub, nfine)
    n_in = n_out + int(full.max())
    x = synth.make_input(cf, n_in, threads=1)
    return cf, full, tab, x


def test_p8_subband_tables(oracle):
    cf, full, tab, x = _sub_case(oracle, 4)
    cps = cf.nchans // 4
    for k in range(tab.ncoarse):
        dn = k * cf.nfine + cf.nfine // 2
        assert tab.nominal[k] == cf.dm_list[dn]
        for c in range(cf.nchans):
            assert tab.s1[k, c] == full[dn, c] - full[dn, (c // cps) * cps]
    for d in range(cf.ndm):
        for s in range(4):
            assert tab.s2[d, s] == full[d, s * cps]
    eff = tab.s1[np.arange(cf.ndm) // cf.nfine] + tab.s2[:, np.arange(cf.nchans) // cps]
    assert tab.max_delay == eff.max()
    for k in range(tab.ncoarse):
        assert tab.maxshift2[k] == tab.s2[k * cf.nfine:(k + 1) * cf.nfine].max()
    assert (tab.s1[:, ::cps] == 0).all()


def test_p8_nominal_rows_equal_brute_force(oracle):
    for dtype in ("u8", "f32"):
        cf, full, tab, x = _sub_case(oracle, 4, dtype=dtype)
        sub, _ = oracle.subband(x, tab, cf.n_out)
        rows = [k * cf.nfine + cf.nfine // 2 for k in range(tab.ncoarse)]
        if dtype == "u8":
            ref = oracle.brute_u8(x, full, cf.n_out)
            assert (sub[rows] == ref[rows]).all()
            assert (sub != ref).any()                    # and it IS an approximation elsewhere
        else:
            ref, _ = oracle.brute_f32(x, full, cf.n_out)
            assert np.allclose(sub[rows], ref[rows], rtol=0, atol=1e-9)


def test_p8_nsub_equals_nchans_is_brute_force(oracle):
    cf, full, tab, x = _sub_case(oracle, 32, dtype="u8")
    assert (tab.s1 == 0).all() and (tab.s2 == full).all()
    sub, _ = oracle.subband(x, tab, cf.n_out)
    assert (sub == oracle.brute_u8(x, full, cf.n_out)).all()


def test_p8_nsub_one_repeats_the_nominal_row(oracle):
    cf, full, tab, x = _sub_case(oracle, 1, dtype="u8")
    assert (tab.s2 == 0).all()
    sub, _ = oracle.subband(x, tab, cf.n_out)
    ref = oracle.brute_u8(x, full, cf.n_out)
    for d in range(cf.ndm):
        k = d // cf.nfine
        assert (sub[d] == ref[k * cf.nfine + cf.nfine // 2]).all()


def test_p8_effective_shift_error_bound(oracle):
    cf, full, tab, x = _sub_case(oracle, 4, nfine=8, ndm=32)
    cps = cf.nchans // 4
    ft = cf.f_top_mhz
    kc = np.array([4.15e6 * ((ft - c * cf.df_mhz) ** -2 - ft ** -2) for c in range(cf.nchans)])
    for d in range(cf.ndm):
        k = d // cf.nfine
        for c in range(cf.nchans):
            eff = tab.s1[k, c] + tab.s2[d, c // cps]
            bound = np.ceil(abs(kc[c] - kc[(c // cps) * cps]) * abs(cf.dm_list[d] - tab.nominal[k])
                            / cf.t_samp_ms) + 2
            assert abs(eff - full[d, c]) <= bound


def test_p8_effective_shift_error_cfg4(oracle):
    """P8(iv) at BASELINE cfg 4's full geometry: the values SURVEY.md section 8c prints for
    err(c,d) = s1 + s2 - shift(c,d) -- range -67...+72 samples, mean |err| 12.8, per-subband maximum
    37 (top subband) ... 72 (bottom) -- and the analytic bound |k_c - k_ctop| * |DM_d - D_k| / t_samp + 2."""
    cf = synth.configs()[4]
    full = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list).astype(np.int64)
    tab = oracle.subband_tables(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list, cf.nsub, cf.nfine)
    cps = cf.nchans // cf.nsub
    sub = np.arange(cf.nchans) // cps
    k = np.arange(cf.ndm) // cf.nfine
    err = tab.s1[k].astype(np.int64) + tab.s2[:, sub].astype(np.int64) - full
    assert (err.min(), err.max()) == (-67, 72)
    assert abs(np.abs(err).mean() - 12.8) < 0.05
    per_sub = np.abs(err).reshape(cf.ndm, cf.nsub, cps).max(axis=(0, 2))
    assert per_sub[0] == 37 and per_sub[-1] == 72 and (np.diff(per_sub) >= 0).all()
    # nominal rows: exactly brute force (reading R8)
    assert (err[np.arange(tab.ncoarse) * cf.nfine + cf.nfine // 2] == 0).all()
    # analytic bound, channel by channel (delay per unit DM from the oracle's own eq. 1)
    kc = np.array([oracle.delay_samples(c, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, 1.0) for c in range(cf.nchans)])
    ddm = np.abs(cf.dm_list - tab.nominal[k])
    bound = np.ceil(np.abs(kc - kc[sub * cps])[None, :] * ddm[:, None]) + 2
    assert (np.abs(err) <= bound).all()


def test_p8_impulse_through_both_stages(oracle):
    """An impulse at (c0,u0) must land at u0 - s1(c0,k) - s2(d,s(c0)) in every row d."""
    cf, full, tab, x = _sub_case(oracle, 4)
    cps = cf.nchans // 4
    x[:] = 0
    c0 = 21
    u0 = int(full[:, c0].max()) + 9
    x[c0, u0] = 1.0
    sub, _ = oracle.subband(x, tab, cf.n_out)
    hits = 0
    for d in range(cf.ndm):
        want = np.zeros(cf.n_out)
        t = u0 - tab.s1[d // cf.nfine, c0] - tab.s2[d, c0 // cps]
        if 0 <= t < cf.n_out:
            want[t] = 1.0
            hits += 1
        assert (sub[d] == want).all()
    assert hits >= 1


# ---------------------------------------------------------------- P9: streaming definition
def test_p9_chunked_equals_one_shot_on_the_oracle(oracle):
    """Reading R9: push k emits stream times [kC - M, (k+1)C - M); emulate the carry with plain
    numpy concatenation and check it reproduces the one-shot result (C > M and C < M)."""
    cf, tab, x = _small_case(oracle, "u8", n_out=400)
    M = int(tab.max())
    total = x.shape[1]
    one = oracle.brute_u8(x, tab, total - M)
    for C in (M + 37, max(8, M // 3)):
        carry = np.zeros((cf.nchans, M), dtype=np.uint8)
        outs = []
        for k in range(total // C):
            work = np.concatenate([carry, x[:, k * C:(k + 1) * C]], axis=1)
            outs.append(oracle.brute_u8(work, tab, C))
            carry = np.ascontiguousarray(work[:, C:])
        got = np.concatenate(outs, axis=1)[:, M:]
        n = min(got.shape[1], one.shape[1])
        assert n > 0 and (got[:, :n] == one[:, :n]).all()


# ---------------------------------------------------------------- event detection
def test_detect_closed_forms(oracle):
    # constant buffer: sigma = 0, nothing is above the mean
    mu, sg, thr, ev, val = oracle.detect(np.full((7, 33), 4.5, dtype=np.float32), 3.0)
    assert mu == 4.5 and sg == 0.0 and len(ev) == 0
    # one spike of height A in N zeros: mu = A/N, sigma = A*sqrt(N-1)/N
    N, A = 20 * 50, 12.0
    x = np.zeros((20, 50), dtype=np.float32)
    x[13, 7] = A
    mu, sg, thr, ev, val = oracle.detect(x, 5.0)
    assert np.isclose(mu, A / N) and np.isclose(sg, A * np.sqrt(N - 1) / N)
    assert ev.tolist() == [[7, 13]] and val.tolist() == [A]          # (time, DM trial)
    assert len(oracle.detect(x, np.sqrt(N - 1) + 1.0)[3]) == 0        # detected iff sqrt(N-1) > nsigma
    # two equal spikes, threshold strictly above
    x[2, 2] = A
    assert oracle.detect(x, 5.0)[3].tolist() == [[2, 2], [7, 13]]     # sorted by (d, t)
    # Gaussian buffer: about N * Q(3) = N * 1.35e-3 values above 3 sigma
    g = np.random.default_rng(5).standard_normal((64, 8192)).astype(np.float32)
    n3 = len(oracle.detect(g, 3.0)[3])
    assert abs(n3 - g.size * 1.3499e-3) < 5 * np.sqrt(g.size * 1.3499e-3)


def test_detect_paper_fig5_statement(oracle):
    """PAPER.md:197 (Fig. 5): with a 5-sigma threshold on the de-dispersed output of a simulated
    pulsar the data points are at the pulsar's DM; Table-2-like input as in the P7 pin."""
    nch, ft, df, ts = 1024, 156.0, 0.005941, 0.165
    dm = np.arange(70, 81, dtype=np.float64)            # trial 5 = DM 75
    cf = synth.Config("fake", nch, ft, df, ts, 2048, dm.size, 1.0, seed=77)
    tab = oracle.shift_table(nch, ft, df, ts, dm)
    w = 60
    pulses = [(5, 500, w, 0.25), (5, 1500, w, 0.25)]
    x = synth.make_input(cf, cf.n_out + int(tab.max()), pulses, {5: tab[5]}, threads=1)
    out, _ = oracle.brute_f32(x, tab, cf.n_out)
    mu, sg, thr, ev, val = oracle.detect(out, 5.0)
    assert len(ev) > 0.5 * 2 * w                        # most on-pulse samples (S/N 8) pass 5 sigma
    on = ((ev[:, 0] >= 500) & (ev[:, 0] < 500 + w)) | ((ev[:, 0] >= 1500) & (ev[:, 0] < 1500 + w))
    assert (ev[on, 1] == 5).mean() > 0.9 and on.mean() > 0.95   # at the true trial, inside the pulses
    assert (val > thr).all()


def test_subband_sample_indices_equal_the_two_stage_oracle(oracle):
    """The per-sample form of the two-stage sum (used to spot-check full-size GPU runs) against the
    stage-by-stage oracle on every output of a small case, uint8 so that equality is exact."""
    cf, full, tab, x = _sub_case(oracle, nsub=4, dtype="u8", n_out=123)
    ref, _ = oracle.subband(x, tab, cf.n_out)
    d, t = np.divmod(np.arange(cf.ndm * cf.n_out), cf.n_out)
    idx = oracle.subband_sample_indices(tab, d, t)
    got, sa = oracle.sum_samples(x[np.arange(cf.nchans)[None, :], idx])
    assert (got.reshape(cf.ndm, cf.n_out) == ref).all() and (sa == got).all()


def test_power_corner_turn_pins(oracle):
    v = np.zeros((3, 2), dtype=np.complex64)                 # [t][c]
    v[0, 0], v[1, 0], v[2, 1], v[0, 1] = 3 + 4j, 0.5 - 0.25j, -2j, 1e-3 + 0j
    p32, p64 = oracle.power_corner_turn(v)
    assert p32.shape == (2, 3) and p32.dtype == np.float32
    assert p32[0].tolist() == [25.0, 0.3125, 0.0] and p32[1, 2] == 4.0      # out[c][t] <- volt[t][c]
    assert p32[1, 0] == np.float32(np.float32(1e-3) * np.float32(1e-3))
    rng = np.random.default_rng(9)
    z = (rng.standard_normal((50, 7)) + 1j * rng.standard_normal((50, 7))).astype(np.complex64)
    p32, p64 = oracle.power_corner_turn(z)
    assert np.abs(p32 - p64).max() <= 2 * np.spacing(p64.astype(np.float32)).max()
    assert np.isclose(p64.sum(), np.vdot(z.astype(np.complex128), z.astype(np.complex128)).real)


def test_bin_samples_pins(oracle):
    x = np.arange(14, dtype=np.float32).reshape(2, 7)
    assert (oracle.bin_samples(x, 1)[0] == x).all()                               # identity
    assert oracle.bin_samples(x, 2)[0].tolist() == [[0.5, 2.5, 4.5], [7.5, 9.5, 11.5]]   # tail dropped
    assert oracle.bin_samples(x, 4)[0].tolist() == [[1.5], [8.5]]
    assert (oracle.bin_samples(np.full((3, 64), 0.1, np.float32), 4)[0] == np.float32(0.1)).all()
    g = np.random.default_rng(2).standard_normal((5, 999)).astype(np.float32)
    for nb in (2, 3, 4, 8):
        b32, b64 = oracle.bin_samples(g, nb)
        assert b32.shape == (5, 999 // nb)
        assert np.abs(b32 - b64).max() <= nb * np.spacing(np.float32(np.abs(g).max()))


def table4_passes():
    """(dm_low, dm_step, ndm, nfine, bin) per pass from tests/golden/table4_plan.txt (Table 4)."""
    out = []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "table4_plan.txt")):
        f = line.split("#")[0].split()
        if f:
            lo, hi, ddm, b, dsub = float(f[1]), float(f[2]), float(f[3]), int(f[4]), float(f[5])
            out.append((lo, ddm, int(round((hi - lo) / ddm)), int(round(dsub / ddm)), b))
    return out


def test_survey_plan_table4_counts():
    """PAPER.md Table 1 / 4 -> 3102 trials, 136 nominal DMs, 22 / 24 / 24 fine trials per nominal DM
    (SURVEY.md A12), passes contiguous in DM."""
    ps = table4_passes()
    assert [p[2] for p in ps] == [1782, 696, 624] and sum(p[2] for p in ps) == 3102
    assert [p[3] for p in ps] == [22, 24, 24] and [p[4] for p in ps] == [1, 2, 4]
    assert [p[2] // p[3] for p in ps] == [81, 29, 26] and sum(p[2] // p[3] for p in ps) == 136
    for a, b in zip(ps, ps[1:]):
        assert abs(a[0] + a[2] * a[1] - b[0]) < 1e-9


def test_survey_single_pass_is_subband_and_binning_chain(oracle):
    """oracle.survey: one pass with bin 1 IS oracle.subband on that DM list; a pass with bin 2 is
    bin_samples followed by subband with 2 * t_samp (stages (i)-(iii))."""
    nch, ft, df, ts, nsub = 64, 150.0, 0.1, 0.2, 8
    rng = np.random.default_rng(44)
    passes = [(0.0, 0.25, 24, 12, 1), (6.0, 0.5, 12, 6, 2)]
    nsamp = 1000
    M = oracle.survey_max_delay(nch, ft, df, ts, nsub, passes)
    x = rng.standard_normal((nch, nsamp + M)).astype(np.float32)
    res = oracle.survey(x, nch, ft, df, ts, nsub, passes, nsamp)
    dm0 = 0.0 + np.arange(24) * 0.25
    t0 = oracle.subband_tables(nch, ft, df, ts, dm0, nsub, 12)
    ref0, sa0 = oracle.subband(x, t0, nsamp)
    assert (res[0][0] == ref0).all() and (res[0][1] == sa0).all() and (res[0][2] == dm0).all()
    xb = oracle.bin_samples(x, 2)[0]
    dm1 = 6.0 + np.arange(12) * 0.5
    t1 = oracle.subband_tables(nch, ft, df, 2 * ts, dm1, nsub, 6)
    ref1, _ = oracle.subband(np.ascontiguousarray(xb), t1, nsamp // 2)
    assert res[1][0].shape == (12, nsamp // 2) and (res[1][0] == ref1).all()
    assert M == max(t0.max_delay, 2 * t1.max_delay)


def test_survey_recovers_a_pulse_in_each_pass(oracle):
    """A noise-free boxcar pulse injected along the (unbinned) dispersion curve of a trial of each pass is
    recovered by oracle.survey at that trial of that pass (P7 through binning and both subband stages);
    pulses are wider than the binning and the subband smear."""
    nch, ft, df, ts, nsub = 128, 308.0, 16.0 / 128, 0.5, 8
    passes = [(0.0, 0.3, 44, 22, 1), (13.2, 0.5, 48, 24, 2), (37.2, 1.0, 48, 24, 4)]
    nsamp = 4096
    M = oracle.survey_max_delay(nch, ft, df, ts, nsub, passes)
    x = np.zeros((nch, nsamp + M), dtype=np.float32)
    truth = []
    for i, (lo, step, ndm, nfine, b) in enumerate(passes):
        d = nfine + nfine // 2                       # a nominal trial (second group) of the pass
        dm = lo + d * step
        row = oracle.shift_table(nch, ft, df, ts, np.array([dm]))[0]     # unbinned delays at that DM
        t0, w = 400 + 1000 * i, 64
        for c in range(nch):
            x[c, t0 + row[c]:t0 + row[c] + w] += 1.0
        truth.append((d, t0, w, b))
    res = oracle.survey(x, nch, ft, df, ts, nsub, passes, nsamp, want_sumabs=False)
    for (out, _, dm), (d, t0, w, b) in zip(res, truth):
        box = out[:, t0 // b:(t0 + w) // b].sum(axis=1)
        assert int(np.argmax(box)) == d
        assert box[d] > 0.9 * nch * w / b            # binning averages: nch * (w / b) samples of height 1
