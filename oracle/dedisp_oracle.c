/*
 * dedisp_oracle.c -- CPU ORACLE for incoherent de-dispersion.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, link or call this file.  It shares no code, header, table or helper with the CUDA
 * library under paper_1107_2516_b200/csrc/, and the product never routes through it.
 *
 * It is written from Magro et al., "Real-time, fast radio transient searches with GPU
 * de-dispersion" (arXiv 1107.2516), cited as PAPER.md:<line>:
 *
 *   - eq. 1: dt = 4.15e6 ms * (f1^-2 - f2^-2) * DM, f in MHz, DM in pc cm^-3.
 *   - "de-dispersion consists of a relative shift in time of all frequency channels according
 *     to equation 1"; brute force is "the simplest and most accurate"
 *      and is the plain definition, so the oracle for it IS the definition:
 *         out[d][t] = sum_c in[c][t + shift(c,d)]              (triple loop, fp64 accumulator)
 *   - n_samp + maxshift samples must be available.
 *   - channel-major, time-contiguous input.
 *   - subband de-dispersion: "The delays corresponding to the
 *     nominal DM for every channel in a subband, minus the delay at the highest frequency in
 *     that subband, are subtracted from each subband channel", then "Normal de-dispersion is
 *     then used to generate the de-dispersed time series for the rest of the DM values within
 *     the same DM sub-range".  This is an approximation, so the oracle follows it step by
 *     step (stage 1, then stage 2), keeping the intermediate in fp64.
 *
 * Readings of the paper where it is silent (R1..R13) are repeated at
 * the function that uses them.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"):
 *   oracle_shift_table      : pinned (hand values from eq. 1, structure, 4-channel toy)
 *   oracle_dedisperse_f32   : pinned (DM=0 channel sum, constant input, impulse response,
 *                             hand-computed toy, pulse recovery, linearity, time shift)
 *   oracle_dedisperse_u8    : pinned (same, exact integers)
 *   oracle_subband_*        : pinned for the special cases (nominal rows == brute force,
 *                             nsub==nchans, nsub==1, effective-shift error bound);
 *                             the absolute sensitivity loss of the subband method is
 *                             "parity unpinned" (the paper prints no value for it).
 *
 * Arithmetic: plain loops; the only parallelism is an OpenMP "parallel for" over independent
 * DM rows (or (group, subband) pairs).  Compile with -O2 -ffp-contract=off -fopenmp.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * shift(c,d) from eq. 1.
 * Readings: R1 constant exactly 4.15e6 ms MHz^2 cm^3/pc, all times in ms;
 *           R2 f_c = f_top - c*df, channel 0 is the highest frequency, df > 0 is the width;
 *           R3 reference = channel 0, shifts >= 0, lower channels read LATER samples;
 *           R4 fp64, round half up: floor(x + 0.5), evaluated in this order, every operation
 *              rounded on its own (no fused multiply-add):
 *                 f_c = f_top - (double)c * df
 *                 a_c = 1/(f_c*f_c) - 1/(f_top*f_top)
 *                 k_c = 4.15e6 * a_c
 *                 x   = (k_c * DM_d) / t_samp
 * shift is [ndm][nchans].  Returns 0, or -1 on invalid arguments / overflow.
 */
int oracle_shift_table(int nchans, double f_top_mhz, double df_mhz, double t_samp_ms,
                       const double *dm, int ndm, int32_t *shift)
{
    if (nchans <= 0 || ndm <= 0 || !(df_mhz > 0.0) || !(t_samp_ms > 0.0) || !(f_top_mhz > 0.0))
        return -1;
    if (!(f_top_mhz - (double)(nchans - 1) * df_mhz > 0.0))
        return -1;
    for (int d = 0; d < ndm; ++d) {
        if (!(dm[d] >= 0.0) || !isfinite(dm[d]))
            return -1;
        for (int c = 0; c < nchans; ++c) {
            volatile double cdf = (double)c * df_mhz;
            volatile double f_c = f_top_mhz - cdf;
            volatile double fc2 = f_c * f_c;
            volatile double ft2 = f_top_mhz * f_top_mhz;
            volatile double inv_c = 1.0 / fc2;
            volatile double inv_t = 1.0 / ft2;
            volatile double a_c = inv_c - inv_t;
            volatile double k_c = 4.15e6 * a_c;
            volatile double num = k_c * dm[d];
            volatile double x = num / t_samp_ms;
            volatile double xr = x + 0.5;
            double r = floor(xr);
            if (!(r >= 0.0) || r > 2147483647.0)
                return -1;
            shift[(size_t)d * nchans + c] = (int32_t)r;
        }
    }
    return 0;
}

/* The real-valued delay in samples (same operation order, no rounding to integer); used by
 * the pins to check |shift - x| <= 0.5. */
double oracle_delay_samples(int c, double f_top_mhz, double df_mhz, double t_samp_ms, double dm)
{
    volatile double cdf = (double)c * df_mhz;
    volatile double f_c = f_top_mhz - cdf;
    volatile double fc2 = f_c * f_c;
    volatile double ft2 = f_top_mhz * f_top_mhz;
    volatile double inv_c = 1.0 / fc2;
    volatile double inv_t = 1.0 / ft2;
    volatile double a_c = inv_c - inv_t;
    volatile double k_c = 4.15e6 * a_c;
    volatile double num = k_c * dm;
    volatile double x = num / t_samp_ms;
    return x;
}

/*
 * Brute force, fp32 input, fp64 accumulation (R6: raw sum, no 1/nchans).
 *   in     [nchans][in_stride], in_stride >= n_out + max shift
 *   shift  [ndm][nchans]
 *   out    [ndm][n_out]            = sum_c in[c][t + shift(c,d)]
 *   sumabs [ndm][n_out] or NULL    = sum_c |in[c][t + shift(c,d)]|  (the fp32 tolerance scale)
 */
int oracle_dedisperse_f32(const float *in, int64_t in_stride, int nchans, const int32_t *shift,
                          int ndm, int64_t n_out, double *out, double *sumabs)
{
    for (int d = 0; d < ndm; ++d)
        for (int c = 0; c < nchans; ++c) {
            int64_t s = shift[(size_t)d * nchans + c];
            if (s < 0 || s + n_out > in_stride)
                return -1;
        }
#pragma omp parallel for schedule(dynamic, 1)
    for (int d = 0; d < ndm; ++d) {
        double *o = out + (size_t)d * n_out;
        double *a = sumabs ? sumabs + (size_t)d * n_out : NULL;
        for (int64_t t = 0; t < n_out; ++t)
            o[t] = 0.0;
        if (a)
            for (int64_t t = 0; t < n_out; ++t)
                a[t] = 0.0;
        for (int c = 0; c < nchans; ++c) {
            const float *x = in + (size_t)c * in_stride + shift[(size_t)d * nchans + c];
            for (int64_t t = 0; t < n_out; ++t)
                o[t] += (double)x[t];
            if (a)
                for (int64_t t = 0; t < n_out; ++t)
                    a[t] += fabs((double)x[t]);
        }
    }
    return 0;
}

/* Brute force, uint8 input (R11: unsigned 0..255, exact sum, no offset removal).  The sum is
 * taken in int64 and must fit int32. */
int oracle_dedisperse_u8(const uint8_t *in, int64_t in_stride, int nchans, const int32_t *shift,
                         int ndm, int64_t n_out, int32_t *out)
{
    for (int d = 0; d < ndm; ++d)
        for (int c = 0; c < nchans; ++c) {
            int64_t s = shift[(size_t)d * nchans + c];
            if (s < 0 || s + n_out > in_stride)
                return -1;
        }
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int d = 0; d < ndm; ++d) {
        int64_t *acc = (int64_t *)calloc((size_t)n_out, sizeof(int64_t));
        for (int c = 0; c < nchans; ++c) {
            const uint8_t *x = in + (size_t)c * in_stride + shift[(size_t)d * nchans + c];
            for (int64_t t = 0; t < n_out; ++t)
                acc[t] += (int64_t)x[t];
        }
        for (int64_t t = 0; t < n_out; ++t) {
            if (acc[t] > 2147483647LL)
                bad = 1;
            out[(size_t)d * n_out + t] = (int32_t)acc[t];
        }
        free(acc);
    }
    return bad ? -2 : 0;
}

/*
 * Subband tables (readings R7, R8, R10).
 *   dm_list is ncoarse = ndm/nfine consecutive groups of nfine fine DMs.
 *   R7: nominal DM of group k is D_k = dm_list[k*nfine + nfine/2]; subband s is channels
 *       [s*cps, (s+1)*cps), cps = nchans/nsub, represented by its first (highest-frequency)
 *       channel ctop(s) = s*cps.
 *   R8: s1(c,k) = shift(c, D_k) - shift(ctop(s(c)), D_k)   (two entries of the same table)
 *       s2(d,s) = shift(ctop(s), DM_d)
 *   R10: maxshift2[k] = max over s and d in group k of s2(d,s); stage 1 for group k produces
 *       n_out + maxshift2[k] samples ("Maxshift samples have to be preserved").
 *   s1 [ncoarse][nchans], s2 [ndm][nsub], nominal [ncoarse], maxshift2 [ncoarse].
 *   *max_delay = max over c,d of s1 + s2.
 */
int oracle_subband_tables(int nchans, double f_top_mhz, double df_mhz, double t_samp_ms,
                          const double *dm, int ndm, int nsub, int nfine, int32_t *s1,
                          int32_t *s2, double *nominal, int32_t *maxshift2, int64_t *max_delay)
{
    if (nsub <= 0 || nfine <= 0 || nchans % nsub != 0 || ndm % nfine != 0)
        return -1;
    int ncoarse = ndm / nfine, cps = nchans / nsub;
    int32_t *full = (int32_t *)malloc((size_t)ndm * nchans * sizeof(int32_t));
    if (!full)
        return -1;
    if (oracle_shift_table(nchans, f_top_mhz, df_mhz, t_samp_ms, dm, ndm, full) != 0) {
        free(full);
        return -1;
    }
    int64_t md = 0;
    for (int k = 0; k < ncoarse; ++k) {
        int dnom = k * nfine + nfine / 2;
        nominal[k] = dm[dnom];
        for (int c = 0; c < nchans; ++c) {
            int ctop = (c / cps) * cps;
            s1[(size_t)k * nchans + c] =
                full[(size_t)dnom * nchans + c] - full[(size_t)dnom * nchans + ctop];
        }
        int32_t m2 = 0;
        for (int j = 0; j < nfine; ++j) {
            int d = k * nfine + j;
            for (int s = 0; s < nsub; ++s) {
                int32_t v = full[(size_t)d * nchans + s * cps];
                s2[(size_t)d * nsub + s] = v;
                if (v > m2)
                    m2 = v;
            }
            for (int c = 0; c < nchans; ++c) {
                int64_t tot = (int64_t)s1[(size_t)k * nchans + c] + s2[(size_t)d * nsub + c / cps];
                if (tot > md)
                    md = tot;
            }
        }
        maxshift2[k] = m2;
    }
    *max_delay = md;
    free(full);
    return 0;
}

/*
 * Subband stage 1 for ONE coarse group k:
 *   sub[s][t] = sum_{c in subband s} in[c][t + s1(c,k)],  t in [0, n1),  n1 = n_out + maxshift2[k]
 *   s1k [nchans] is row k of the s1 table; sub is [nsub][n1] fp64; sabs likewise (|.| sums) or NULL.
 * in is float (in_u8 == NULL) or uint8 (in_f32 == NULL).
 */
int oracle_subband_stage1(const float *in_f32, const uint8_t *in_u8, int64_t in_stride, int nchans,
                          int nsub, const int32_t *s1k, int64_t n1, double *sub, double *sabs)
{
    int cps = nchans / nsub;
    for (int c = 0; c < nchans; ++c)
        if (s1k[c] < 0 || (int64_t)s1k[c] + n1 > in_stride)
            return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nsub; ++s) {
        double *o = sub + (size_t)s * n1;
        double *a = sabs ? sabs + (size_t)s * n1 : NULL;
        for (int64_t t = 0; t < n1; ++t)
            o[t] = 0.0;
        if (a)
            for (int64_t t = 0; t < n1; ++t)
                a[t] = 0.0;
        for (int c = s * cps; c < (s + 1) * cps; ++c) {
            if (in_f32) {
                const float *x = in_f32 + (size_t)c * in_stride + s1k[c];
                for (int64_t t = 0; t < n1; ++t)
                    o[t] += (double)x[t];
                if (a)
                    for (int64_t t = 0; t < n1; ++t)
                        a[t] += fabs((double)x[t]);
            } else {
                const uint8_t *x = in_u8 + (size_t)c * in_stride + s1k[c];
                for (int64_t t = 0; t < n1; ++t)
                    o[t] += (double)x[t];
                if (a)
                    for (int64_t t = 0; t < n1; ++t)
                        a[t] += (double)x[t];
            }
        }
    }
    return 0;
}

/*
 * Subband stage 2 for ONE coarse group ("Normal de-dispersion is then used..."):
 *   out[j][t] = sum_s sub[s][t + s2(j,s)],  j in [0,nfine), t in [0,n_out)
 *   sub [nsub][n1] fp64, s2g [nfine][nsub] (rows of the s2 table for this group).
 */
int oracle_subband_stage2(const double *sub, const double *sabs, int64_t n1, int nsub,
                          const int32_t *s2g, int nfine, int64_t n_out, double *out, double *sumabs)
{
    for (int j = 0; j < nfine; ++j)
        for (int s = 0; s < nsub; ++s)
            if (s2g[(size_t)j * nsub + s] < 0 || (int64_t)s2g[(size_t)j * nsub + s] + n_out > n1)
                return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < nfine; ++j) {
        double *o = out + (size_t)j * n_out;
        double *a = (sumabs && sabs) ? sumabs + (size_t)j * n_out : NULL;
        for (int64_t t = 0; t < n_out; ++t)
            o[t] = 0.0;
        if (a)
            for (int64_t t = 0; t < n_out; ++t)
                a[t] = 0.0;
        for (int s = 0; s < nsub; ++s) {
            const double *x = sub + (size_t)s * n1 + s2g[(size_t)j * nsub + s];
            for (int64_t t = 0; t < n_out; ++t)
                o[t] += x[t];
            if (a) {
                const double *y = sabs + (size_t)s * n1 + s2g[(size_t)j * nsub + s];
                for (int64_t t = 0; t < n_out; ++t)
                    a[t] += y[t];
            }
        }
    }
    return 0;
}
