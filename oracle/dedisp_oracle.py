"""CPU ORACLE for incoherent de-dispersion -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It never imports the product package
``paper_1107_2516_b200`` and shares no code with the CUDA library.

The arithmetic lives in ``dedisp_oracle.c`` (plain C loops, fp64 accumulation, written from
PAPER.md eq. 1 :21-24, the definition :26, :84, :115-135, :157); this file only marshals numpy
arrays into it, and adds ``brute_samples`` -- the definition written out with numpy indexing for
single output samples (used to spot-check full-size GPU runs).

Pins: see the header of ``dedisp_oracle.c`` and ``tests/test_oracle_pins.py``.  ``brute_samples``
is pinned by equality with ``brute_f32`` / ``brute_u8`` on the pinned small cases; ``survey`` (the
multi-pass plan of PAPER.md Tables 1 / 4: binning -> stage 1 -> stage 2 per pass) has no arithmetic of
its own and is pinned by the single-pass identity, Table 4's counts (tests/golden/table4_plan.txt) and
pulse recovery in every pass.  The absolute sensitivity loss of the subband method is "parity unpinned".
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_oracle.c")
_SO = os.path.join(_HERE, "libdedisp_oracle.so")
_lib = None

_i32p = ctypes.POINTER(ctypes.c_int32)
_f64p = ctypes.POINTER(ctypes.c_double)
_f32p = ctypes.POINTER(ctypes.c_float)
_u8p = ctypes.POINTER(ctypes.c_uint8)


def build(force=False):
    """Compile dedisp_oracle.c with gcc (no FMA contraction: reading R4)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.oracle_delay_samples.restype = ctypes.c_double
        _lib.oracle_delay_samples.argtypes = [ctypes.c_int] + [ctypes.c_double] * 4
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t) if a is not None else None


def num_threads():
    return int(_load().oracle_num_threads())


def shift_table(nchans, f_top_mhz, df_mhz, t_samp_ms, dm_list):
    """int32[ndm][nchans] from eq. 1, readings R1-R4."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    out = np.empty((dm.size, nchans), dtype=np.int32)
    rc = _load().oracle_shift_table(ctypes.c_int(nchans), ctypes.c_double(f_top_mhz),
                                    ctypes.c_double(df_mhz), ctypes.c_double(t_samp_ms),
                                    _p(dm, _f64p), ctypes.c_int(dm.size), _p(out, _i32p))
    if rc != 0:
        raise ValueError("oracle_shift_table: invalid arguments")
    return out


def delay_samples(c, f_top_mhz, df_mhz, t_samp_ms, dm):
    return float(_load().oracle_delay_samples(int(c), float(f_top_mhz), float(df_mhz),
                                              float(t_samp_ms), float(dm)))


def brute_f32(x, shift, n_out, want_sumabs=True):
    """out[d][t] = sum_c x[c][t+shift[d][c]] in fp64.  x: float32 [nchans][n_in]."""
    assert x.dtype == np.float32 and x.ndim == 2 and x.strides[1] == 4
    shift = np.ascontiguousarray(shift, dtype=np.int32)
    ndm, nchans = shift.shape
    assert x.shape[0] == nchans
    out = np.empty((ndm, n_out), dtype=np.float64)
    sa = np.empty((ndm, n_out), dtype=np.float64) if want_sumabs else None
    rc = _load().oracle_dedisperse_f32(_p(x, _f32p), ctypes.c_int64(x.strides[0] // 4),
                                       ctypes.c_int(nchans), _p(shift, _i32p), ctypes.c_int(ndm),
                                       ctypes.c_int64(n_out), _p(out, _f64p), _p(sa, _f64p))
    if rc != 0:
        raise ValueError("oracle_dedisperse_f32: shift + n_out exceeds the input length")
    return (out, sa) if want_sumabs else out


def brute_u8(x, shift, n_out):
    """Exact integer sum for uint8 input (reading R11).  x: uint8 [nchans][n_in] -> int32."""
    assert x.dtype == np.uint8 and x.ndim == 2 and x.strides[1] == 1
    shift = np.ascontiguousarray(shift, dtype=np.int32)
    ndm, nchans = shift.shape
    assert x.shape[0] == nchans
    out = np.empty((ndm, n_out), dtype=np.int32)
    rc = _load().oracle_dedisperse_u8(_p(x, _u8p), ctypes.c_int64(x.strides[0]),
                                      ctypes.c_int(nchans), _p(shift, _i32p), ctypes.c_int(ndm),
                                      ctypes.c_int64(n_out), _p(out, _i32p))
    if rc != 0:
        raise ValueError("oracle_dedisperse_u8: bad shifts or int32 overflow")
    return out


def brute_samples(x, shift, d_idx, t_idx):
    """The definition for single outputs: out[i] = sum_c x[c][t_i + shift[d_i][c]] (fp64 / int64),
    and sum_c |x| beside it.  Plain numpy indexing, one output at a time."""
    nchans = x.shape[0]
    cc = np.arange(nchans)
    is_int = x.dtype == np.uint8
    out = np.empty(len(d_idx), dtype=np.int64 if is_int else np.float64)
    sa = np.empty(len(d_idx), dtype=np.float64)
    for i, (d, t) in enumerate(zip(d_idx, t_idx)):
        v = x[cc, int(t) + shift[int(d)].astype(np.int64)]
        if is_int:
            out[i] = v.astype(np.int64).sum()
            sa[i] = float(out[i])
        else:
            v = v.astype(np.float64)
            out[i] = v.sum()
            sa[i] = np.abs(v).sum()
    return out, sa


def subband_sample_indices(tab, d_idx, t_idx):
    """For single outputs of the two-stage method: the input sample each channel
    contributes, idx[i][c] = t_i + s2[d_i][sub(c)] + s1[k(d_i)][c] (stage 2 reads the partial series
    of subband sub(c) at t + s2, which stage 1 formed from channel c at that time + s1).  The caller
    gathers x[c][idx[i][c]] (from wherever the input lives) and sums in fp64: `sum_samples`.
    Pinned by equality with `subband` on the small P8 cases."""
    nchans = tab.s1.shape[1]
    cps = nchans // tab.s2.shape[1]
    sub = np.arange(nchans) // cps
    d = np.asarray(d_idx, dtype=np.int64)
    k = d // tab.nfine
    return (np.asarray(t_idx, dtype=np.int64)[:, None] + tab.s2[d][:, sub].astype(np.int64)
            + tab.s1[k].astype(np.int64))


def sum_samples(vals):
    """fp64 (int64 for integer input) sum over the channel axis and sum of magnitudes."""
    v = np.asarray(vals)
    if np.issubdtype(v.dtype, np.integer):
        s = v.astype(np.int64).sum(axis=1)
        return s, s.astype(np.float64)
    v = v.astype(np.float64)
    return v.sum(axis=1), np.abs(v).sum(axis=1)


class SubbandTables:
    pass


def subband_tables(nchans, f_top_mhz, df_mhz, t_samp_ms, dm_list, nsub, nfine):
    """s1[ncoarse][nchans], s2[ndm][nsub], nominal[ncoarse], maxshift2[ncoarse], max_delay
    (readings R7, R8, R10)."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    ndm = dm.size
    if nsub <= 0 or nfine <= 0 or nchans % nsub or ndm % nfine:
        raise ValueError("bad subband split")
    nco = ndm // nfine
    t = SubbandTables()
    t.s1 = np.empty((nco, nchans), dtype=np.int32)
    t.s2 = np.empty((ndm, nsub), dtype=np.int32)
    t.nominal = np.empty(nco, dtype=np.float64)
    t.maxshift2 = np.empty(nco, dtype=np.int32)
    md = ctypes.c_int64(0)
    rc = _load().oracle_subband_tables(ctypes.c_int(nchans), ctypes.c_double(f_top_mhz),
                                       ctypes.c_double(df_mhz), ctypes.c_double(t_samp_ms),
                                       _p(dm, _f64p), ctypes.c_int(ndm), ctypes.c_int(nsub),
                                       ctypes.c_int(nfine), _p(t.s1, _i32p), _p(t.s2, _i32p),
                                       _p(t.nominal, _f64p), _p(t.maxshift2, _i32p),
                                       ctypes.byref(md))
    if rc != 0:
        raise ValueError("oracle_subband_tables: invalid arguments")
    t.max_delay = int(md.value)
    t.nsub, t.nfine, t.ncoarse = nsub, nfine, nco
    return t


def subband(x, tab, n_out, groups=None, want_sumabs=True):
    """Two-stage subband de-dispersion, stage by stage in fp64.
    Returns out[len(groups)*nfine][n_out] (+ sumabs) for the coarse groups asked for
    (default: all).  x: float32 or uint8 [nchans][n_in]."""
    lib = _load()
    nchans = x.shape[0]
    nsub, nfine = tab.nsub, tab.nfine
    if groups is None:
        groups = range(tab.ncoarse)
    groups = list(groups)
    out = np.empty((len(groups) * nfine, n_out), dtype=np.float64)
    sa = np.empty_like(out) if want_sumabs else None
    is_u8 = x.dtype == np.uint8
    stride = x.strides[0] // x.itemsize
    for gi, k in enumerate(groups):
        n1 = int(n_out + tab.maxshift2[k])
        sub = np.empty((nsub, n1), dtype=np.float64)
        sabs = np.empty((nsub, n1), dtype=np.float64) if want_sumabs else None
        s1k = np.ascontiguousarray(tab.s1[k])
        rc = lib.oracle_subband_stage1(None if is_u8 else _p(x, _f32p), _p(x, _u8p) if is_u8 else None,
                                       ctypes.c_int64(stride), ctypes.c_int(nchans),
                                       ctypes.c_int(nsub), _p(s1k, _i32p), ctypes.c_int64(n1),
                                       _p(sub, _f64p), _p(sabs, _f64p))
        if rc != 0:
            raise ValueError("oracle_subband_stage1: input too short")
        s2g = np.ascontiguousarray(tab.s2[k * nfine:(k + 1) * nfine])
        o = out[gi * nfine:(gi + 1) * nfine]
        a = sa[gi * nfine:(gi + 1) * nfine] if want_sumabs else None
        rc = lib.oracle_subband_stage2(_p(sub, _f64p), _p(sabs, _f64p), ctypes.c_int64(n1),
                                       ctypes.c_int(nsub), _p(s2g, _i32p), ctypes.c_int(nfine),
                                       ctypes.c_int64(n_out), _p(o, _f64p), _p(a, _f64p))
        if rc != 0:
            raise ValueError("oracle_subband_stage2: intermediate too short")
    return (out, sa) if want_sumabs else out


def detect(out, nsigma):
    """Event detection on one de-dispersed buffer out[ndm][n]: mean and standard
    deviation of the ENTIRE buffer, threshold mu + nsigma * sigma, every value above it as a triplet
    (time, DM trial, intensity).  Readings (R14): population standard deviation (divide by
    N), strict '>', fp64 statistics.  Returns (mu, sigma, threshold, events) with events an int64
    array [k][2] of (t, d) sorted by (d, t) and the intensities out[d][t].
    Pins (tests/test_oracle_pins.py): constant buffer -> no events; one spike of height A in N zeros
    -> mu = A/N, sigma = A*sqrt(N-1)/N, detected iff sqrt(N-1) > nsigma; Gaussian buffer -> count
    near N*Q(nsigma); the paper's Fig. 5 statement: the 5-sigma events of a simulated pulsar sit at
    its DM trial."""
    x = np.asarray(out, dtype=np.float64)
    mu = float(x.mean())
    sigma = float(np.sqrt(((x - mu) ** 2).mean()))
    thr = mu + float(nsigma) * sigma
    d, t = np.nonzero(x > thr)
    return mu, sigma, thr, np.stack([t, d], axis=1).astype(np.int64), np.asarray(out)[d, t]


def power_corner_turn(volt):
    """Total power of complex voltages, transposed into channel order (steps (iii) and
    (iv) of the real-time pipeline): out[c][t] = re(volt[t][c])^2 + im(volt[t][c])^2.  The paper's
    arithmetic is fp32, so the result is DEFINED in fp32 with each product and the sum rounded on its
    own (reading R15); numpy float32 operations round exactly that way.  Also returns the fp64 value.
    Pins: exactly representable hand values ((3,4) -> 25, (0.5,-0.25) -> 0.3125), the layout
    (out[c][t] comes from volt[t][c]), agreement of the fp32 definition with fp64 within 2 ulp."""
    v = np.asarray(volt)
    re = v.real.astype(np.float32)
    im = v.imag.astype(np.float32)
    p32 = (re * re + im * im).astype(np.float32).T.copy()
    p64 = (re.astype(np.float64) ** 2 + im.astype(np.float64) ** 2).T.copy()
    return p32, p64


def bin_samples(x, nb):
    """Binning, stage (i) of the paper's subband scheme ("Binning averages N_b
    consecutive samples"): out[c][j] = (x[c][j*nb] + ... + x[c][j*nb + nb-1]) / nb, floor(n/nb)
    outputs per channel (a ragged tail is dropped).  Reading R16: fp32 like the paper's pipeline, the
    sum taken left to right and divided once, every operation rounded on its own -- so the result is
    defined bit for bit; the fp64 value is returned beside it.
    Pins: nb = 1 is the identity; hand values; constant input stays constant; agreement with the
    fp64 mean within nb ulp."""
    x = np.asarray(x, dtype=np.float32)
    n = x.shape[-1] // nb
    v = x[..., :n * nb].reshape(x.shape[:-1] + (n, nb))
    acc = v[..., 0].copy()
    for i in range(1, nb):
        acc = (acc + v[..., i]).astype(np.float32)
    return (acc / np.float32(nb)).astype(np.float32), v.astype(np.float64).mean(axis=-1)


def survey(x, nchans, f_top_mhz, df_mhz, t_samp_ms, nsub, passes, nsamp, want_sumabs=True):
    """Multi-pass subband survey (PAPER.md:58-60 survey plan; :137-155 the three stages; Tables 1 / 4):
    for every pass (dm_low, dm_step, ndm, nfine, bin), in the paper's order,
      (i)   binning: xb = bin_samples(x, bin)            (fp32-defined, reading R16; bin = 1: x itself)
      (ii)  subband stage 1 and (iii) stage 2: subband(xb, tables for t_samp * bin and the pass's DM list
            dm_low + d * dm_step, nsub, nfine), n_i = nsamp // bin outputs per trial (eq. 8: n_samp / b_i).
    Reading R17: a survey over nsamp input samples needs nsamp + M samples per channel,
    M = max_i bin_i * max_delay_i (unbinned samples); `survey_max_delay` returns it.
    Returns [(out_i, sumabs_i, dm_list_i)].  No arithmetic of its own beyond the DM list: every step is a
    pinned oracle function.  Pins (tests/test_oracle_pins.py): one pass with bin 1 is `subband`; Table 4
    gives 3102 trials and 136 nominal DMs; a noise-free pulse is recovered at its trial in its pass."""
    res = []
    for (dm_low, dm_step, ndm, nfine, b) in passes:
        dm = float(dm_low) + np.arange(int(ndm), dtype=np.float64) * float(dm_step)
        tab = subband_tables(nchans, f_top_mhz, df_mhz, t_samp_ms * b, dm, nsub, int(nfine))
        xb = np.ascontiguousarray(x if b == 1 else bin_samples(x, b)[0])
        n_i = int(nsamp) // b
        if n_i + tab.max_delay > xb.shape[1]:
            raise ValueError("survey: input too short for pass with bin %d" % b)
        r = subband(xb, tab, n_i, want_sumabs=want_sumabs)
        res.append((r[0], r[1], dm) if want_sumabs else (r, None, dm))
    return res


def survey_max_delay(nchans, f_top_mhz, df_mhz, t_samp_ms, nsub, passes):
    """Unbinned input samples a survey needs beyond nsamp: max over passes of bin * max_delay(pass)."""
    m = 0
    for (dm_low, dm_step, ndm, nfine, b) in passes:
        dm = float(dm_low) + np.arange(int(ndm), dtype=np.float64) * float(dm_step)
        m = max(m, b * subband_tables(nchans, f_top_mhz, df_mhz, t_samp_ms * b, dm, nsub, int(nfine)).max_delay)
    return int(m)
