// Host planner of the register-window kernel (kernels_window.cu).
//
// The kernel keeps, per thread, kWinD DM rows x kWinT output pairs in registers for the whole
// channel loop and feeds all rows from ONE register window of kWinNW consecutive staged samples.
// That only works if, for every channel c, the samples the kWinD rows need start within
// kWinOMax positions of each other.  Neighbouring DM trials drift apart as the channel frequency
// drops (eq. 1: the delay difference between two DMs grows like f^-2), so each row
// j of a row group carries a skew kappa_j(c): slot p of row j stands for output time p - kappa_j.
// kappa_j only ever grows, one sample at a time ("row shift": the row's accumulators move up one
// slot), and is chosen lazily here so that
//     0 <= [s(c,d_j) - kappa_j(c)] - s(c,d_0) <= 3      for every channel c
// (at most two shifts of a row per channel).
// Everything the kernel needs per (DM tile, channel) is precomputed into WindowPlan::meta.
#include <algorithm>
#include <cstring>

#include "dedisp_internal.h"

namespace dedisp {

bool build_window_plan(const int32_t* shift, int ndm, int nchans, WindowPlan& wp)
{
    wp = WindowPlan();
    if (ndm <= 0 || nchans <= 0)
        return false;
    const int ntile = (ndm + kWinDB - 1) / kWinDB;
    wp.ntile_dm = ntile;
    wp.meta.assign(static_cast<size_t>(ntile) * nchans * kWinMetaWords, 0);
    wp.kfinal.assign(static_cast<size_t>(ntile) * kWinDB, 0);
    int kmax = 0, lmax = 0;
    int64_t maxbase = 0;
    for (int ty = 0; ty < ntile; ++ty) {
        const int32_t* rows[kWinDB];
        for (int r = 0; r < kWinDB; ++r) {
            const int d = std::min(ty * kWinDB + r, ndm - 1);  // tail rows repeat the last trial
            rows[r] = shift + static_cast<size_t>(d) * nchans;
        }
        int kappa[kWinDB];
        std::memset(kappa, 0, sizeof(kappa));
        for (int c = 0; c < nchans; ++c) {
            int32_t* m = wp.meta.data() + (static_cast<size_t>(ty) * nchans + c) * kWinMetaWords;
            int raw0[kWinNG];
            unsigned mask[kWinNG], mask2[kWinNG];
            int64_t base = INT64_MAX;
            for (int g = 0; g < kWinNG; ++g) {
                const int s0 = rows[g * kWinD][c];
                mask[g] = mask2[g] = 0;
                for (int j = 1; j < kWinD; ++j) {
                    int& k = kappa[g * kWinD + j];
                    int diff = rows[g * kWinD + j][c] - s0 - k;
                    // the row shifts by one slot (twice if need be) before this channel is added;
                    // shifting at 3 already leaves room for the +-1 dither of the rounded delays
                    if (diff > 2) {
                        ++k;
                        --diff;
                        mask[g] |= 1u << j;
                    }
                    if (diff > 2) {
                        ++k;
                        --diff;
                        mask2[g] |= 1u << j;
                    }
                    if (diff < 0 || diff > 3)
                        return false;
                }
                raw0[g] = s0;
                base = std::min<int64_t>(base, s0);
            }
            base &= ~static_cast<int64_t>(1);  // staged segments start on an even sample
            int wbmax = 0;
            for (int g = 0; g < kWinNG; ++g) {
                const int e0 = static_cast<int>(raw0[g] - base);
                const int wb = e0 & ~1;  // even: 16-byte aligned LDS.128 of two pairs
                if (wb > 0xffffff)
                    return false;
                unsigned om = 0;
                for (int j = 0; j < kWinD; ++j) {
                    const int o = rows[g * kWinD + j][c] - kappa[g * kWinD + j] - static_cast<int>(base) - wb;
                    if (o < 0 || o > kWinOMax)
                        return false;
                    om |= static_cast<unsigned>(o) << (3 * j);
                }
                om |= mask[g] << 24;
                m[10] |= static_cast<int32_t>(mask2[g] << (8 * g));
                m[2 + g] = wb;
                m[6 + g] = static_cast<int32_t>(om);
                wbmax = std::max(wbmax, wb);
            }
            const int len = kWinNS + wbmax + kWinOMax;  // even
            if (base > INT32_MAX)
                return false;
            m[0] = static_cast<int32_t>(base);
            m[1] = len;
            lmax = std::max(lmax, len);
            maxbase = std::max(maxbase, base);
        }
        for (int r = 0; r < kWinDB; ++r) {
            wp.kfinal[static_cast<size_t>(ty) * kWinDB + r] = kappa[r];
            kmax = std::max(kmax, kappa[r]);
        }
    }
    const int H = (kWinNS - kmax) & ~1;
    if (H < kWinNS / 2)  // more than half of the slots would be skew slack: not worth it
        return false;
    wp.H = H;
    wp.kmax = kmax;
    wp.lmax = lmax;
    wp.maxbase = maxbase;
    wp.ok = true;
    return true;
}

int64_t window_pair_stride(const WindowPlan& wp, int64_t n_out)
{
    const int64_t ntile_t = (n_out + 2 * wp.H - 1) / (2 * wp.H);
    int64_t n = ntile_t * 2 * wp.H + wp.maxbase + wp.lmax;
    return (n + 1) & ~static_cast<int64_t>(1);
}

}  // namespace dedisp
