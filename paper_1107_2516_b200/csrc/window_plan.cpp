// Host planner of the register-window kernel (kernels_window.cu).
//
// A thread keeps D (8 or 4) DM rows x T output pairs in registers and feeds all rows from ONE
// register window of T + 1 consecutive staged pairs per channel: row j adds w[i + o_j] to its
// accumulator i, o_j in {0, 1}.  That needs, for every channel c, the samples of the 8 rows to start
// within one position of a common base.  Neighbouring DM trials drift apart as the frequency drops
// (eq. 1: the delay difference of two DMs grows like f^-2) and the rounded delays
// dither by +-1 around that drift, so
//   * row 0 of a row group is the reference: the window starts at its shift s_0(c);
//   * row j carries base_j(c) = theta_j + kappa_j(c), non-decreasing in c, with
//         o_j(c) = [s_j(c) - s_0(c)] - base_j(c)  in {0, 1};
//     slot p of row j stands for output time  tile_start + p - base_j(c);
//   * kappa_j grows one at a time ("row shift": the row's accumulators move up one slot).  The
//     partial sum that leaves the top of a warp's slot range belongs to the same output sample as
//     the fresh slot that enters at the bottom of the NEXT warp segment in time, so inside a block
//     (2*NT segments of W slots, contiguous in time) nothing is lost: the kernel hands those
//     partial sums over through the output buffer.  Only the block as a whole loses kmax samples,
//     so blocks are Hb = 2*NT*W - kmax samples apart.  The channel loop is cut into BANDS only
//     when a row drifts by more than kcap slots or faster than the kernel can follow; a new band
//     restarts with kappa = 0 and a fresh skew theta_j, and its partial sums are added to the
//     output by a later launch (kernels_window.cu).
// Everything the kernel needs per (DM tile, channel) is precomputed into WindowPlan::meta.
#include <algorithm>
#include <cstring>

#include "dedisp_internal.h"

namespace dedisp {

// Preference order of the thread / block shapes at plan creation: 4 rows x 15 pairs per thread, 12 consumer
// warps (three per scheduler, 160 registers each) in one block per SM.  Three warps along time (NT = 3,
// G = 4 row groups) lose kmax samples per 6 warp segments and measured best on cfg 2, 3 and 5; two warps
// along time with 6 row groups stage shorter channel segments and take over when the NT = 3 ring does not
// fit shared memory.
int window_geom_preferences(WindowGeom* g, int max)
{
    static const int pref[][4] = {{15, 4, 3, 4}, {15, 6, 2, 4}, {21, 8, 1, 4}};
    int n = 0;
    for (const auto& p : pref) {
        if (n == max)
            break;
        g[n].T = p[0];
        g[n].G = p[1];
        g[n].NT = p[2];
        g[n].D = p[3];
        ++n;
    }
    return n;
}

WindowGeom window_default_geom()
{
    WindowGeom g;
    window_geom_preferences(&g, 1);
    return g;
}

namespace {

struct Rows {
    const int32_t* shift;
    int ndm, nchans, RB;
    const int32_t* row(int tile, int r) const
    {
        const int d = std::min(tile * RB + r, ndm - 1);  // tail rows repeat the last trial
        return shift + static_cast<size_t>(d) * nchans;
    }
};

}  // namespace

bool build_window_plan(const int32_t* shift, int ndm, int nchans, const WindowGeom& geom, WindowPlan& wp)
{
    wp = WindowPlan();
    wp.geom = geom;
    if (ndm <= 0 || nchans <= 0 || geom.T <= 0 || geom.G <= 0 || geom.G > 8 || geom.NT <= 0 || geom.D < 2 ||
        geom.D > kWinD)
        return false;
    const int RB = geom.rows(), W = geom.W(), G = geom.G, D = geom.D;
    const int ntile = (ndm + RB - 1) / RB;
    const int kcap = std::max(4, W / 4);  // slots a block may lose (of 2 * NT * W)
    const Rows R{shift, ndm, nchans, RB};
    const size_t nrow = static_cast<size_t>(ntile) * RB;

    // ---- pass 1: band boundaries, common to all DM tiles ------------------------------------------
    std::vector<int32_t> base(nrow), theta(nrow), nb(nrow);
    std::vector<const int32_t*> rp(nrow), r0(nrow);
    for (int ty = 0; ty < ntile; ++ty)
        for (int r = 0; r < RB; ++r) {
            rp[static_cast<size_t>(ty) * RB + r] = R.row(ty, r);
            r0[static_cast<size_t>(ty) * RB + r] = R.row(ty, r / D * D);
        }
    auto start_band = [&](int c) -> bool {
        for (size_t k = 0; k < nrow; ++k) {
            const int diff = rp[k][c] - r0[k][c];
            if (diff < 0)
                return false;  // DM list not monotone inside a row group
            base[k] = theta[k] = std::max(0, diff - 1);
        }
        return true;
    };
    // greedy split with at most `cap` row shifts per band; false: the table does not fit the kernel
    auto split = [&](int cap, std::vector<int32_t>& band, int& kmax_out) -> bool {
        band.assign(1, 0);
        if (!start_band(0))
            return false;
        int km = 0;
        for (int c = 1; c < nchans; ++c) {
            bool cut = false;
            for (size_t k = 0; k < nrow && !cut; ++k) {
                const int diff = rp[k][c] - r0[k][c];
                const int b = std::max(base[k], diff - 1);
                nb[k] = b;
                // infeasible offset, more than two shifts at once, or too many shifts in this band
                if (b > diff || b - base[k] > 2 || b - theta[k] > cap)
                    cut = true;
            }
            if (cut) {
                if (c - band.back() < 4)
                    return false;  // trials drift apart faster than the kernel can follow
                band.push_back(c);
                if (!start_band(c))
                    return false;
            } else {
                for (size_t k = 0; k < nrow; ++k) {
                    base[k] = nb[k];
                    km = std::max(km, base[k] - theta[k]);
                }
            }
        }
        band.push_back(nchans);
        kmax_out = km;
        return true;
    };
    int kmax = 0;
    if (!split(kcap, wp.band, kmax))
        return false;
    {
        // balance: the smallest cap that needs no more bands evens out the band lengths and gives
        // back the slots a looser cap would waste (H = W - kmax)
        const size_t nb0 = wp.band.size();
        int lo = 1, hi = kcap;  // invariant: hi works
        std::vector<int32_t> tb;
        while (lo < hi) {
            const int mid = (lo + hi) / 2;
            int km = 0;
            if (split(mid, tb, km) && tb.size() <= nb0) {
                hi = mid;
                wp.band = tb;
                kmax = km;
            } else {
                lo = mid + 1;
            }
        }
    }
    wp.nband = static_cast<int>(wp.band.size()) - 1;
    if (wp.nband > 64)
        return false;
    wp.Hb = (2 * geom.NT * W - kmax) & ~1;  // even: a block's first pair stays 16-byte aligned for the bulk copies
    wp.kmax = kmax;
    wp.ntile_dm = ntile;

    // ---- pass 2: metadata ---------------------------------------------------------------------------
    wp.meta.assign(static_cast<size_t>(ntile) * nchans * kWinMetaWords, 0);
    wp.kfinal.assign(static_cast<size_t>(ntile) * wp.nband * RB, 0);
    wp.theta.assign(static_cast<size_t>(ntile) * wp.nband * RB, 0);
    int lmax = 0, theta_max = 0;
    int64_t maxbase = 0;
    std::vector<int> bs(RB), th(RB);
    for (int ty = 0; ty < ntile; ++ty) {
        const size_t k0 = static_cast<size_t>(ty) * RB;
        for (int b = 0; b < wp.nband; ++b) {
            for (int c = wp.band[b]; c < wp.band[b + 1]; ++c) {
                int32_t* m = wp.meta.data() + (static_cast<size_t>(ty) * nchans + c) * kWinMetaWords;
                int64_t lo = INT64_MAX, hi = 0;
                for (int g = 0; g < G; ++g) {
                    const int64_t om = r0[k0 + g * D][c];
                    lo = std::min(lo, om);
                    hi = std::max(hi, om);
                }
                const int64_t segbase = lo & ~static_cast<int64_t>(1);
                if (segbase > INT32_MAX)
                    return false;
                int len = static_cast<int>(hi - segbase) + (geom.NT - 1) * W + W + 1;
                len = (len + 1) & ~1;
                m[0] = static_cast<int32_t>(segbase);
                m[1] = len;
                lmax = std::max(lmax, len);
                maxbase = std::max(maxbase, segbase);
                for (int g = 0; g < G; ++g) {
                    const int64_t wb = r0[k0 + g * D][c] - segbase;
                    if (wb + (geom.NT - 1) * W >= (1 << kWinWbBits))
                        return false;
                    unsigned word = static_cast<unsigned>(wb) << 21;
                    for (int j = 1; j < D; ++j) {
                        const int r = g * D + j;
                        const int diff = rp[k0 + r][c] - r0[k0 + r][c];
                        if (c == wp.band[b])
                            bs[r] = th[r] = std::max(0, diff - 1);
                        const int nbase = std::max(bs[r], diff - 1);
                        const int ns = nbase - bs[r], o = diff - nbase;
                        if (o < 0 || o > 1 || ns > 2)
                            return false;  // cannot happen after pass 1
                        bs[r] = nbase;
                        if (o)
                            word |= 1u << (j - 1);
                        if (ns >= 1)
                            word |= 1u << (5 + j - 1);
                        if (ns >= 2)
                            word |= 1u << (10 + j - 1);
                    }
                    m[2 + g] = static_cast<int32_t>(word);
                }
            }
            for (int r = 0; r < RB; ++r) {
                const size_t k = (static_cast<size_t>(ty) * wp.nband + b) * RB + r;
                const bool ref = r % D == 0;
                wp.kfinal[k] = ref ? 0 : bs[r] - th[r];
                wp.theta[k] = ref ? 0 : th[r];
                theta_max = std::max(theta_max, wp.theta[k]);
            }
        }
    }
    // ---- ring of staged segments.  Stage boundaries cost every consumer warp an arrive, a barrier wait
    // and a refill of its pipeline (11.5 % of the kernel with 4-channel stages), so stages should be long;
    // the ring must still hold >= 2 of them.  Measured on cfg 3 (slots of 9.3 / 12.5 KB): 8 channels x 3
    // stages beat 12 x 2, 6 x 4 and 4 x 6; 9 x 2 beats 6 x 3.  Rule: the longest stage <= 12 channels that
    // leaves three stages if that is >= 8 channels, else the longest that leaves two.
    {
        const int sb = (lmax * 8 + 127) & ~127;
        const int budget = (G * geom.NT == 4 ? 113 : 227) * 1024 - kWinFixedBytes;
        auto stage_bytes = [&](int ch) { return (G * ch * 4 + 127) / 128 * 128 + ch * sb; };
        auto longest = [&](int nst) {
            int ch = 0;
            for (int c = 1; c <= kWinChMax; ++c)
                if (nst * stage_bytes(c) <= budget)
                    ch = c;
            return ch;
        };
        int ch = longest(3), nstg = 3;
        if (ch < 8) {
            const int c2 = longest(2);
            if (c2 > ch) {
                ch = c2;
                nstg = 2;
            }
        }
        wp.lmax = lmax;
        wp.slot_bytes = sb;
        // the flush's transpose scratch ([warps][W] pairs per row) overlays the ring
        if (ch < 2 || nstg * stage_bytes(ch) < G * geom.NT * W * 8) {
            wp.ch = wp.nst = wp.hdr_words = 0;  // does not fit shared memory: ok stays false
            return false;
        }
        while ((nstg + 1) * stage_bytes(ch) <= budget && nstg < 8)
            ++nstg;
        wp.ch = ch;
        wp.nst = nstg;
        wp.hdr_words = (G * ch * 4 + 127) / 128 * 32;
    }
    const int CH = wp.ch, HW = wp.hdr_words;
    // ---- stage headers.  A consumer warp carries the
    // current channel's word in a (uniform) register and reads the NEXT channel's word while it adds, so
    // the header of a stage holds, regrouped per row group (hdr[g * CH + c]), the words of the
    // channels one further on; the band's first word comes from `first`.  The word of a channel that
    // opens a stage says whether any channel of that stage has a row shift (the kernel then runs the
    // loop variant that tests for shifts).  Channels past the band's end and one extra stage per band
    // stay zero (the kernel stages a zero segment for them).
    wp.stage0.assign(wp.nband + 1, 0);
    for (int b = 0; b < wp.nband; ++b)
        wp.stage0[b + 1] = wp.stage0[b] + (wp.band[b + 1] - wp.band[b] + CH - 1) / CH + 1;
    const int nst = wp.stage0[wp.nband];
    wp.hdr.assign(static_cast<size_t>(ntile) * nst * HW, 0);
    wp.first.assign(static_cast<size_t>(ntile) * wp.nband * G, 0);
    for (int ty = 0; ty < ntile; ++ty)
        for (int b = 0; b < wp.nband; ++b) {
            const int c0 = wp.band[b], c1 = wp.band[b + 1];
            for (int g = 0; g < G; ++g) {
                auto word_of = [&](int c) -> uint32_t& {
                    return reinterpret_cast<uint32_t&>(wp.meta[(static_cast<size_t>(ty) * nchans + c) * kWinMetaWords + 2 + g]);
                };
                for (int cs = c0; cs < c1; cs += CH) {
                    bool any = false;
                    for (int c = cs; c < std::min(cs + CH, c1); ++c)
                        any = any || (word_of(c) & kWinShiftBits) != 0;
                    if (any)
                        word_of(cs) |= kWinStageShift;
                }
                wp.first[(static_cast<size_t>(ty) * wp.nband + b) * G + g] = static_cast<int32_t>(word_of(c0));
                for (int c = c0; c + 1 < c1; ++c) {
                    const int s = wp.stage0[b] + (c - c0) / CH, cc = (c - c0) % CH;
                    wp.hdr[(static_cast<size_t>(ty) * nst + s) * HW + g * CH + cc] = static_cast<int32_t>(word_of(c + 1));
                }
            }
        }
    wp.maxbase = maxbase;
    wp.theta_max = theta_max;
    wp.ok = true;
    return true;
}

int64_t window_ntile_t(const WindowPlan& wp, int64_t n_out)
{
    return (n_out - 1 + wp.theta_max) / wp.Hb + 1;
}

int64_t window_pair_stride(const WindowPlan& wp, int64_t n_out)
{
    const int64_t n = (window_ntile_t(wp, n_out) - 1) * wp.Hb + 2LL * wp.geom.NT * wp.geom.W() + wp.maxbase + wp.lmax + 2;
    return (n + 1) & ~static_cast<int64_t>(1);
}

}  // namespace dedisp
