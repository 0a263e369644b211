"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/dedisp.h declares,
and its host-side logic (shift tables, subband tables, argument validation, eq. 3 sizing) matches
the oracle bit for bit.  No kernel is launched here."""
import os
import re
import ctypes

import numpy as np
import pytest

import paper_1107_2516_b200 as dd
from paper_1107_2516_b200 import synth, build as ddbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    ddbuild.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "dedisp.h")).read()
    declared = set(re.findall(r"DEDISP_API[^;(]*?\b(dedisp_\w+)\s*\(", hdr))
    assert len(declared) >= 20
    L = ctypes.CDLL(dd.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(dd.EXPORTS)
    assert "sm_100a" in dd.version()


def test_header_compiles_as_c_and_a_c_caller_works(tmp_path):
    """tests/abi_smoke.c: gcc -std=c99 against include/dedisp.h and the .so, run without a device."""
    import subprocess
    exe = str(tmp_path / "abi_smoke")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I" + os.path.join(ROOT, "include"),
                           os.path.join(ROOT, "tests", "abi_smoke.c"), "-o", exe, dd.LIB_PATH,
                           "-Wl,-rpath," + os.path.dirname(dd.LIB_PATH)])
    out = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr
    assert "abi_smoke ok" in out.stdout and "sm_100a" in out.stdout


def _plan(cf, **kw):
    a = cf.plan_args()
    a.update(kw)
    return dd.Plan(**a)


@pytest.mark.parametrize("k", [1, 2, 3, 5])
def test_shift_tables_bit_exact_vs_oracle(oracle, k):
    cf = synth.configs()[k]
    p = _plan(cf)
    ref = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    got = p.shifts()
    assert got.dtype == np.int32 and (got == ref).all()
    assert p.max_delay == ref.max()
    p.close()


def test_shift_table_cfg4_and_subband_tables_bit_exact(oracle):
    cf = synth.configs()[4]
    p = _plan(cf)
    ref = oracle.shift_table(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list)
    assert (p.shifts() == ref).all()
    tab = oracle.subband_tables(cf.nchans, cf.f_top_mhz, cf.df_mhz, cf.t_samp_ms, cf.dm_list,
                                cf.nsub, cf.nfine)
    s1, s2, nom, m2 = p.subband_shifts()
    assert (s1 == tab.s1).all() and (s2 == tab.s2).all()
    assert (nom == tab.nominal).all() and (m2 == tab.maxshift2).all()
    assert p.max_delay == tab.max_delay == 424645
    assert ref.max() == 424712
    assert p.scratch_bytes(131072) == 128 * 32 * ((131072 + int(m2.max()) + 15) // 16 * 16) * 4
    p.close()


def test_ties_golden(oracle):
    cf = synth.configs()[5]
    got = _plan(cf).shifts()
    for line in open(os.path.join(ROOT, "tests", "golden", "ties_cfg5.txt")):
        line = line.split("#")[0].split()
        if line:
            d, c, s = map(int, line)
            assert got[d, c] == s


def test_random_plans_match_oracle(oracle):
    rng = np.random.default_rng(2516)
    for _ in range(20):
        nch = int(rng.integers(1, 300))
        ft = float(rng.uniform(100, 2000))
        df = float(rng.uniform(0.001, 0.9 * ft / nch))
        ts = float(rng.uniform(0.01, 2.0))
        dm = np.sort(rng.uniform(0, 500, int(rng.integers(1, 50))))
        p = dd.Plan(nch, ft, df, ts, dm)
        assert (p.shifts() == oracle.shift_table(nch, ft, df, ts, dm)).all()
        p.close()


def test_plan_create_rejects_bad_arguments():
    good = dict(nchans=8, f_top_mhz=200.0, df_mhz=1.0, t_samp_ms=1.0, dm_list=[0.0, 1.0])
    for bad in (dict(nchans=0), dict(df_mhz=0.0), dict(df_mhz=-1.0), dict(t_samp_ms=0.0),
                dict(f_top_mhz=7.0), dict(dm_list=[-1.0]), dict(dm_list=[float("nan")]),
                dict(dm_list=[float("inf")]), dict(dm_list=[]), dict(nsub=3, nfine=1),
                dict(nsub=2, nfine=3), dict(nsub=2, nfine=0),
                dict(nsub=2, nfine=2, dm_list=[1.0, 0.0]), dict(t_samp_ms=1e-12, dm_list=[1e6])):
        a = dict(good)
        a.update(bad)
        with pytest.raises(dd.DedispError) as e:
            dd.Plan(**a)
        assert e.value.status == 1


def test_null_handles_and_misc():
    L = dd.lib()
    assert L.dedisp_plan_max_delay(None) == -1 and L.dedisp_plan_nchans(None) == -1
    assert L.dedisp_plan_destroy(None) == 0 and L.dedisp_stream_destroy(None) == 0
    assert L.dedisp_strerror(4).decode().startswith("shape")
    p = dd.Plan(8, 200.0, 1.0, 1.0, [0.0, 1.0])
    with pytest.raises(dd.DedispError) as e:
        p.subband_shifts()
    assert e.value.status == 5
    with pytest.raises(dd.DedispError):
        p.set_kernel(17)
    assert p.resolved_kernel() in (dd.KERNEL_DIRECT, dd.KERNEL_WINDOW)
    assert p.last_kernel == -1 and dd.lib().dedisp_plan_last_kernel(None) == -1     # nothing executed yet
    p.set_kernel(dd.KERNEL_NAIVE)
    assert p.resolved_kernel() == dd.KERNEL_NAIVE


def test_max_chunk_follows_eq3():
    """PAPER.md:90-95 (eq. 3): memory must hold input + maxshift overlap + output."""
    cf = synth.configs()[5]
    p = _plan(cf)
    mem = 40 << 30
    n = p.max_chunk(dd.U8, mem, nbeams=4)
    M = p.max_delay
    used = lambda n: 4 * (2 * cf.nchans * (M + 16 + n) * 1 + cf.ndm * n * 4)
    assert n > 0 and n % 16 == 0 and used(n) <= mem < used(n + 32)
    assert p.max_chunk(dd.U8, 1 << 20, nbeams=4) == 0


def test_survey_tables_match_oracle_table4(oracle):
    """dedisp_survey_create on the paper's Table 4 plan (1024 channels, 16 MHz at 300 MHz; 3102 trials in
    3 passes with bin 1 / 2 / 4 and 22 / 24 / 24 fine trials per nominal DM): every pass's subband tables,
    built for t_samp * bin, equal the oracle's; the survey's input overlap is max_i bin_i * max_delay_i."""
    from test_oracle_pins import table4_passes
    nch, ft, df, ts, nsub = 1024, 308.0, 16.0 / 1024, 0.1, 32
    passes = table4_passes()
    sv = dd.Survey(nch, ft, df, ts, nsub, passes)
    assert sv.max_delay == oracle.survey_max_delay(nch, ft, df, ts, nsub, passes)
    for i, (lo, step, ndm, nfine, b) in enumerate(passes):
        dm = lo + np.arange(ndm, dtype=np.float64) * step
        t = oracle.subband_tables(nch, ft, df, ts * b, dm, nsub, nfine)
        s1, s2, nom, m2, md = sv.pass_tables(i)
        assert (s1 == t.s1).all() and (s2 == t.s2).all() and (nom == t.nominal).all() and (m2 == t.maxshift2).all()
        assert md == t.max_delay
    off, st, no, tot = sv.out_layout(8192, 2)
    assert list(no) == [8192, 4096, 2048] and off[0] == 0 and off[1] == 2 * 1782 * 8192
    assert tot == 2 * (1782 * 8192 + 696 * 4096 + 624 * 2048)
    sv.close()
    for bad in ([(0.0, 0.1, 10, 3, 1)], [(0.0, 0.1, 12, 3, 0)], [(-1.0, 0.1, 12, 3, 1)], []):
        with pytest.raises(dd.DedispError):
            dd.Survey(64, 150.0, 0.1, 0.1, 8, bad)
