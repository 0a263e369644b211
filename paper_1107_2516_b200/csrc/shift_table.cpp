// Integer shift-table builder: eq. 1 of Magro et al.,
//   dt = 4.15e6 ms * (f_c^-2 - f_top^-2) * DM,  shift = nearest integer of dt / t_samp.
// Host code, built with -ffp-contract=off: every fp64 operation below must be rounded on its own,
// because some configurations hit exact .5 ties (reading R4).  The paper evaluates the
// DM-independent factor on the CPU and the per-DM product in fp32 on the GPU (eq. 4/5,
// PAPER.md:97-113); here the whole table is fp64 and is built once per plan.
#include "dedisp_internal.h"

#include <cmath>
#include <thread>
#include <vector>

namespace dedisp {

// k_c = 4.15e6 * (1/f_c^2 - 1/f_top^2)   [ms per unit DM]
static inline double chan_factor(int c, double f_top, double df)
{
    const double cdf = static_cast<double>(c) * df;
    const double f_c = f_top - cdf;
    const double fc2 = f_c * f_c;
    const double ft2 = f_top * f_top;
    const double inv_c = 1.0 / fc2;
    const double inv_t = 1.0 / ft2;
    const double a_c = inv_c - inv_t;
    return 4.15e6 * a_c;
}

bool build_shift_table(int nchans, double f_top, double df, double t_samp, const double* dm,
                       int ndm, std::vector<int32_t>& table, int64_t& max_delay)
{
    table.assign(static_cast<size_t>(ndm) * nchans, 0);
    std::vector<double> k(nchans);
    for (int c = 0; c < nchans; ++c)
        k[c] = chan_factor(c, f_top, df);

    unsigned hw = std::thread::hardware_concurrency();
    int nthr = static_cast<int>(hw ? (hw > 16 ? 16 : hw) : 1);
    if (static_cast<int64_t>(ndm) * nchans < (1 << 16))
        nthr = 1;
    std::vector<int64_t> tmax(nthr, 0);
    std::vector<char> bad(nthr, 0);
    auto work = [&](int tid) {
        int64_t m = 0;
        for (int d = tid; d < ndm; d += nthr) {
            int32_t* row = table.data() + static_cast<size_t>(d) * nchans;
            const double dmd = dm[d];
            for (int c = 0; c < nchans; ++c) {
                const double num = k[c] * dmd;
                const double x = num / t_samp;
                const double xr = x + 0.5;
                const double r = std::floor(xr);
                if (!(r >= 0.0) || r > 2147483647.0) {
                    bad[tid] = 1;
                    return;
                }
                row[c] = static_cast<int32_t>(r);
                if (row[c] > m)
                    m = row[c];
            }
        }
        tmax[tid] = m;
    };
    if (nthr == 1) {
        work(0);
    } else {
        std::vector<std::thread> th;
        for (int i = 0; i < nthr; ++i)
            th.emplace_back(work, i);
        for (auto& t : th)
            t.join();
    }
    max_delay = 0;
    for (int i = 0; i < nthr; ++i) {
        if (bad[i])
            return false;
        if (tmax[i] > max_delay)
            max_delay = tmax[i];
    }
    return true;
}

// Subband tables from the full-band one (readings R7, R8, R10).
void build_subband_tables(const std::vector<int32_t>& full, int nchans, int ndm, int nsub, int nfine,
                          const double* dm, std::vector<int32_t>& s1, std::vector<int32_t>& s2,
                          std::vector<double>& nominal, std::vector<int32_t>& maxshift2,
                          int64_t& max_delay)
{
    const int ncoarse = ndm / nfine, cps = nchans / nsub;
    s1.assign(static_cast<size_t>(ncoarse) * nchans, 0);
    s2.assign(static_cast<size_t>(ndm) * nsub, 0);
    nominal.assign(ncoarse, 0.0);
    maxshift2.assign(ncoarse, 0);
    max_delay = 0;
    for (int k = 0; k < ncoarse; ++k) {
        const int dnom = k * nfine + nfine / 2;
        nominal[k] = dm[dnom];
        const int32_t* nomrow = full.data() + static_cast<size_t>(dnom) * nchans;
        int32_t* s1k = s1.data() + static_cast<size_t>(k) * nchans;
        std::vector<int32_t> s1max(nsub, 0);
        for (int c = 0; c < nchans; ++c) {
            s1k[c] = nomrow[c] - nomrow[(c / cps) * cps];
            if (s1k[c] > s1max[c / cps])
                s1max[c / cps] = s1k[c];
        }
        int32_t m2 = 0;
        for (int j = 0; j < nfine; ++j) {
            const int d = k * nfine + j;
            for (int s = 0; s < nsub; ++s) {
                const int32_t v = full[static_cast<size_t>(d) * nchans + static_cast<size_t>(s) * cps];
                s2[static_cast<size_t>(d) * nsub + s] = v;
                if (v > m2)
                    m2 = v;
                const int64_t tot = static_cast<int64_t>(v) + s1max[s];
                if (tot > max_delay)
                    max_delay = tot;
            }
        }
        maxshift2[k] = m2;
    }
}

}  // namespace dedisp
