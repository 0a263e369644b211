// C ABI of libdedisp_b200.so (include/dedisp.h): plans, execute, the streaming chunk driver.
// Host-side only; the arithmetic lives in shift_table.cpp (tables) and kernels_*.cu (sums).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "dedisp_internal.h"

using namespace dedisp;

namespace {

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
    cudaError_t ensure(size_t n)
    {
        if (n <= bytes)
            return cudaSuccess;
        if (p)
            cudaFree(p);
        p = nullptr;
        bytes = 0;
        cudaError_t e = cudaMalloc(&p, n);
        if (e == cudaSuccess)
            bytes = n;
        return e;
    }
    void release()
    {
        if (p)
            cudaFree(p);
        p = nullptr;
        bytes = 0;
    }
};

// max over row tiles [k*tile, (k+1)*tile) and columns of (max - min) of table[row][col]
int tile_spread(const int32_t* tab, int nrows, int ncols, int64_t row_stride, int tile)
{
    int worst = 0;
    std::vector<int32_t> mn(ncols), mx(ncols);
    for (int r0 = 0; r0 < nrows; r0 += tile) {
        const int r1 = r0 + tile < nrows ? r0 + tile : nrows;
        for (int c = 0; c < ncols; ++c)
            mn[c] = mx[c] = tab[static_cast<int64_t>(r0) * row_stride + c];
        for (int r = r0 + 1; r < r1; ++r) {
            const int32_t* row = tab + static_cast<int64_t>(r) * row_stride;
            for (int c = 0; c < ncols; ++c) {
                mn[c] = row[c] < mn[c] ? row[c] : mn[c];
                mx[c] = row[c] > mx[c] ? row[c] : mx[c];
            }
        }
        for (int c = 0; c < ncols; ++c)
            worst = mx[c] - mn[c] > worst ? mx[c] - mn[c] : worst;
    }
    return worst;
}

int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

}  // namespace

struct dedisp_plan {
    int nchans = 0, ndm = 0, nsub = 0, nfine = 0;
    double f_top = 0, df = 0, t_samp = 0;
    std::vector<double> dm;
    std::vector<int32_t> shift;  // [ndm][nchans]
    int64_t max_delay = 0;       // what the caller must supply (brute: table max; subband: s1+s2)
    int spread_full[3] = {0, 0, 0};
    // subband
    std::vector<int32_t> s1, s2, maxshift2;
    std::vector<int32_t> maxshift2_ks;  // [nsub][ncoarse]: what stage 2 reads of subband s in group k
    std::vector<double> nominal;
    int32_t maxshift2_max = 0;
    int spread_s1[3] = {0, 0, 0}, spread_s2[3] = {0, 0, 0};
    // device side (uploaded by the first execute)
    bool uploaded = false;
    int device = -1, nsm = 148;
    int32_t *d_shift = nullptr, *d_s1 = nullptr, *d_s2 = nullptr, *d_maxshift2 = nullptr, *d_maxshift2_ks = nullptr;
    DevBuf scratch;            // subband intermediate
    DevBuf host_in, host_out;  // staging for dedisp_execute_host
    DevBuf det_partial;        // dedisp_plan_detect / dedisp_execute_detect workspace (per-block partial sums)
    DevBuf det_pivot;          // [nbeams] doubles
    DevBuf det_events, det_results;  // device staging of dedisp_execute_detect_host
    // shape of the de-dispersed data the last *_host entry left in host_out: rows of ho_n samples, ho_stride apart
    int64_t ho_rows = 0, ho_n = 0, ho_stride = 0;
    dedisp_kernel kernel = DEDISP_KERNEL_AUTO;
    int last_launches = 0;
    int last_kernel = -1;  // dedisp_kernel the last execute ran (subband plans: stage 1's), -1 before the first
    int nstreams = 0;
    // register-window kernel (brute-force plans): host plan, device tables, pair scratch
    WindowPlan win;
    bool win_fits = false;
    int32_t *d_win_meta = nullptr, *d_win_kfinal = nullptr, *d_win_theta = nullptr, *d_win_hdr = nullptr, *d_win_first = nullptr;
    void* d_win_zeros = nullptr;
    DevBuf pairs;
    // optional timing of the dominant kernel(s) of an execute (dedisp_plan_set_timing)
    bool timing = false;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};  // start, end, between the subband stages
    bool ev_valid = false, ev_mid_valid = false;
    // dedisp_execute_host pipeline: copy streams and per-chunk events (created on first use)
    static constexpr int kHostChunks = 8;   // time pieces of the host entries (+ 1: the first is split)
    static constexpr int kHostEvents = kHostChunks + 2;
    cudaStream_t copy_st[2] = {nullptr, nullptr};  // H2D, D2H
    cudaEvent_t ev_copy[2 * kHostEvents + 2] = {};
};

struct dedisp_stream {
    dedisp_plan* plan = nullptr;
    dedisp_dtype dtype = DEDISP_F32;
    int64_t chunk = 0, wstride = 0;
    int nbeams = 0;
    DevBuf work[2];
    int cur = 0;
    bool zeroed = false;
    DevBuf host_in, host_out;
};

extern "C" int64_t dedisp_plan_scratch_bytes(const dedisp_plan* p, int64_t nsamp_out, int nbeams);

struct dedisp_survey {
    int nchans = 0, nsub = 0;
    double f_top = 0, df = 0, t_samp = 0;
    std::vector<dedisp_pass> passes;
    std::vector<dedisp_plan*> plans;  // one subband plan per pass, created with t_samp * bin
    int64_t max_delay = 0;            // unbinned input samples beyond nsamp: max_i bin_i * max_delay_i
    DevBuf binned;                    // [nbeams][nchans][stride] of the pass being executed (bin > 1)
    int last_launches = 0;
};

namespace {

size_t in_size(dedisp_dtype t) { return t == DEDISP_F32 ? 4 : 1; }

void free_tables(dedisp_plan* p)
{
    int32_t** tabs[] = {&p->d_shift, &p->d_s1, &p->d_s2, &p->d_maxshift2, &p->d_maxshift2_ks,
                        &p->d_win_meta, &p->d_win_kfinal, &p->d_win_theta, &p->d_win_hdr, &p->d_win_first};
    for (int32_t** t : tabs) {
        if (*t)
            cudaFree(*t);
        *t = nullptr;
    }
    if (p->d_win_zeros)
        cudaFree(p->d_win_zeros);
    p->d_win_zeros = nullptr;
    p->uploaded = false;
}

// copies the plan's tables to the current device (blocking; called by dedisp_plan_reserve only)
dedisp_status upload(dedisp_plan* p)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ECUDA;
    }
    if (p->uploaded)
        return dev == p->device ? DEDISP_OK : DEDISP_ESTATE;  // a plan lives on one device
    auto up = [](int32_t** d, const std::vector<int32_t>& h) -> cudaError_t {
        if (h.empty())
            return cudaSuccess;
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(d), h.size() * sizeof(int32_t));
        if (e != cudaSuccess)
            return e;
        return cudaMemcpy(*d, h.data(), h.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    };
    cudaError_t e = cudaSuccess;
    if (p->nsub == 0) {
        e = up(&p->d_shift, p->shift);
        if (e == cudaSuccess && p->win.ok) {
            e = up(&p->d_win_meta, p->win.meta);
            if (e == cudaSuccess)
                e = up(&p->d_win_kfinal, p->win.kfinal);
            if (e == cudaSuccess)
                e = up(&p->d_win_theta, p->win.theta);
            if (e == cudaSuccess)
                e = up(&p->d_win_hdr, p->win.hdr);
            if (e == cudaSuccess)
                e = up(&p->d_win_first, p->win.first);
            if (e == cudaSuccess) {
                const size_t zb = static_cast<size_t>(p->win.lmax + 16) * 8;
                e = cudaMalloc(&p->d_win_zeros, zb);
                if (e == cudaSuccess)
                    e = cudaMemset(p->d_win_zeros, 0, zb);
            }
        }
    } else {
        e = up(&p->d_s1, p->s1);
        if (e == cudaSuccess)
            e = up(&p->d_s2, p->s2);
        if (e == cudaSuccess)
            e = up(&p->d_maxshift2, p->maxshift2);
        if (e == cudaSuccess)
            e = up(&p->d_maxshift2_ks, p->maxshift2_ks);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        free_tables(p);  // nothing stays behind for a retry to leak
        return e == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA;
    }
    p->device = dev;
    cudaDeviceGetAttribute(&p->nsm, cudaDevAttrMultiProcessorCount, dev);
    p->uploaded = true;
    return DEDISP_OK;
}

bool use_window(const dedisp_plan* p, dedisp_dtype dtype, int64_t nsamp_out);
bool fused_stats_ok(const dedisp_plan* p, dedisp_dtype dtype, int64_t nsamp_out)
{
    return use_window(p, dtype, nsamp_out) && p->win.nband == 1;
}

bool use_window(const dedisp_plan* p, dedisp_dtype dtype, int64_t nsamp_out)
{
    if (p->nsub != 0 || !p->win.ok || !p->win_fits)
        return false;
    // the kernel keeps output times in 32 bits
    if (nsamp_out > 0 && window_pair_stride(p->win, nsamp_out) >= (1LL << 30))
        return false;
    // uint8 sums are carried in fp32, exact while nchans * 255 < 2^24
    if (dtype == DEDISP_U8 && static_cast<int64_t>(p->nchans) * 255 >= (1 << 24))
        return false;
    return p->kernel == DEDISP_KERNEL_AUTO || p->kernel == DEDISP_KERNEL_WINDOW;
}

// request to accumulate the outputs' statistics in the register-window kernel's flush
struct StatReq {
    const double* pivot;
    double* partial;
    int64_t stride, off;  // partials per beam, first partial of this execute
};

// the fused statistics need every output to be final when it is stored: single-band window plans
bool fused_stats_ok(const dedisp_plan* p, dedisp_dtype dtype, int64_t nsamp_out);

// brute force through the register-window kernel: pairify into the plan's scratch, then add
dedisp_status run_window(dedisp_plan* plan, const void* in, void* out, Elem in_t, int64_t nsamp_out,
                         int64_t in_stride, int64_t out_stride, int nbeams, void* stream, const StatReq* sr)
{
    WindowArgs a;
    std::memset(&a, 0, sizeof(a));
    a.pair_stride = window_pair_stride(plan->win, nsamp_out);
    if (static_cast<size_t>(nbeams) * plan->nchans * a.pair_stride * 8 > plan->pairs.bytes)
        return DEDISP_ESTATE;  // dedisp_plan_reserve was not called for this shape
    a.in = in;
    a.out = out;
    a.pairs = plan->pairs.p;
    a.meta = plan->d_win_meta;
    a.kfinal = plan->d_win_kfinal;
    a.theta = plan->d_win_theta;
    a.hdr = plan->d_win_hdr;
    a.first = plan->d_win_first;
    a.zeros = plan->d_win_zeros;
    a.stage0 = plan->win.stage0.data();
    a.stage_total = plan->win.stage0[plan->win.nband];
    a.theta_max = plan->win.theta_max;
    a.ev0 = plan->timing ? plan->ev[0] : nullptr;
    a.ev1 = plan->timing ? plan->ev[1] : nullptr;
    a.ev_mid = plan->timing ? plan->ev[2] : nullptr;
    if (sr) {
        a.pivot = sr->pivot;
        a.stat_partial = sr->partial;
        a.stat_stride = sr->stride;
        a.stat_off = sr->off;
    }
    plan->ev_valid = plan->ev_mid_valid = plan->timing;
    a.nband = plan->win.nband;
    a.band = plan->win.band.data();
    a.geom = plan->win.geom;
    a.in_stride = in_stride;
    a.out_stride = out_stride;
    a.in_len = nsamp_out + plan->max_delay;
    a.n_out = nsamp_out;
    a.nchans = plan->nchans;
    a.ndm = plan->ndm;
    a.nbeams = nbeams;
    a.Hb = plan->win.Hb;
    a.kmax = plan->win.kmax;
    a.lmax = plan->win.lmax;
    a.ch = plan->win.ch;
    a.nst = plan->win.nst;
    a.slot_bytes = plan->win.slot_bytes;
    a.hdr_words = plan->win.hdr_words;
    a.ntile_dm = plan->win.ntile_dm;
    a.ntile_t = static_cast<int>(window_ntile_t(plan->win, nsamp_out));
    {
        // DM tiles per block-order group: a wave of `inflight` blocks = g DM tiles x inflight/g time
        // tiles reads about g * cols_per_tile + (inflight / g) * tile_cols columns of the pair buffer;
        // the g that minimises it
        const double inflight = plan->nsm * (plan->win.geom.G * plan->win.geom.NT == 4 ? 2.0 : 1.0);
        const double tile_cols = plan->win.Hb;
        double mean_last = 0.0;  // mean over channels of the largest delay
        const int32_t* last = plan->shift.data() + static_cast<size_t>(plan->ndm - 1) * plan->nchans;
        for (int c = 0; c < plan->nchans; ++c)
            mean_last += last[c];
        mean_last /= plan->nchans;
        const double cols_per_tile = mean_last / plan->win.ntile_dm + 1.0;
        int g = static_cast<int>(std::sqrt(inflight * tile_cols / cols_per_tile) + 0.5);
        g = g < 1 ? 1 : g > plan->win.ntile_dm ? plan->win.ntile_dm : g;
        a.dm_group = g > plan->win.ntile_dm ? plan->win.ntile_dm : g;
    }
    plan->last_kernel = DEDISP_KERNEL_WINDOW;
    return launch_window(a, in_t, stream, &plan->last_launches) == 0 ? DEDISP_OK : DEDISP_ECUDA;
}

int run_problem(dedisp_plan* plan, const Problem& pr, Elem in_t, const int spread[3], void* stream)
{
    switch (plan->kernel) {
    case DEDISP_KERNEL_NAIVE:
        plan->last_kernel = DEDISP_KERNEL_NAIVE;
        return launch_naive(pr, in_t, stream, &plan->last_launches);
    case DEDISP_KERNEL_DIRECT:
        plan->last_kernel = DEDISP_KERNEL_DIRECT;
        return launch_direct(pr, in_t, spread, stream, &plan->last_launches);
    default: {
        // long tiles pay once a row has a few tiles' worth of samples; short problems keep the
        // 256-sample tiles of the direct kernel
        if (plan->kernel == DEDISP_KERNEL_LONG || pr.n_out >= 4096) {
            const int rc = launch_long(pr, in_t, spread[1], stream, &plan->last_launches);
            if (rc != -1) {
                plan->last_kernel = DEDISP_KERNEL_LONG;
                return rc;
            }
        }
        plan->last_kernel = DEDISP_KERNEL_DIRECT;
        return launch_direct(pr, in_t, spread, stream, &plan->last_launches);
    }
    }
}

dedisp_status execute_device(dedisp_plan* plan, const void* in, void* out, dedisp_dtype dtype,
                             int64_t nsamp_out, int64_t in_stride, int64_t out_stride, int nbeams,
                             void* stream, const StatReq* sr = nullptr, int64_t policy_len = 0)
{
    // policy_len > 0: the host entries cut one buffer into time pieces and pass the length of the WHOLE
    // buffer here, so that AUTO's size rule picks one kernel for all pieces (one fp32 summation order per
    // output buffer) instead of judging every piece by its own length
    if (!plan || nbeams <= 0 || nsamp_out < 0 || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    if (nsamp_out == 0) {
        plan->last_launches = 0;
        return DEDISP_OK;
    }
    if (!in || !out)
        return DEDISP_EINVAL;
    const int64_t vec = 16 / static_cast<int64_t>(in_size(dtype));
    if (in_stride < nsamp_out + plan->max_delay || out_stride < nsamp_out || in_stride % vec != 0 ||
        out_stride % 4 != 0 || (reinterpret_cast<uintptr_t>(in) & 15) != 0 ||
        (reinterpret_cast<uintptr_t>(out) & 15) != 0)
        return DEDISP_ESHAPE;
    plan->last_launches = 0;
    plan->ev_mid_valid = false;
    {
        // never allocates, never blocks: tables and scratch come from dedisp_plan_reserve
        int dev = -1;
        if (!plan->uploaded || cudaGetDevice(&dev) != cudaSuccess || dev != plan->device)
            return DEDISP_ESTATE;
    }
    const Elem in_t = dtype == DEDISP_F32 ? Elem::F32 : Elem::U8;

    Problem pr;
    std::memset(&pr, 0, sizeof(pr));
    pr.nb0 = nbeams;
    pr.in_len = nsamp_out + plan->max_delay;  // the extent seen from `in`: nothing beyond it is read
    int rc = 0;
    // AUTO looks at the size: tiles of the register-window kernel are 24 rows x ~1900 samples, and a
    // problem that yields fewer of them than there are SMs (BASELINE cfg 1: 15) is launch- and
    // latency-bound.  There one thread per output (the paper's own scheme) wins up to
    // ~8192 outputs per SM, the direct kernel's 8..32 rows x 256 samples beyond (measured on cfg 1:
    // naive 0.037 ms, direct 0.054 ms, window 0.069 ms, long 0.078 ms).
    bool small = false;
    const int64_t size_len = policy_len > 0 ? policy_len : nsamp_out;
    if (plan->kernel == DEDISP_KERNEL_AUTO && plan->nsub == 0 && !sr && use_window(plan, dtype, nsamp_out))
        small = static_cast<int64_t>(plan->win.ntile_dm) * window_ntile_t(plan->win, size_len) * nbeams < plan->nsm;
    if (!small && use_window(plan, dtype, nsamp_out))
        return run_window(plan, in, out, in_t, nsamp_out, in_stride, out_stride, nbeams, stream, sr);
    if (sr)
        return DEDISP_ESTATE;  // callers check fused_stats_ok first
    struct Timer {  // the direct / subband kernels are timed as a whole
        dedisp_plan* p;
        cudaStream_t st;
        Timer(dedisp_plan* p_, void* s) : p(p_), st(static_cast<cudaStream_t>(s))
        {
            if (p->timing)
                cudaEventRecord(p->ev[0], st);
        }
        ~Timer()
        {
            if (p->timing) {
                cudaEventRecord(p->ev[1], st);
                p->ev_valid = true;
            }
        }
    } timer(plan, stream);
    if (plan->nsub == 0) {
        pr.in = in;
        pr.out = out;
        pr.shift = plan->d_shift;
        pr.in_chan_stride = in_stride;
        pr.in_b0_stride = in_stride * plan->nchans;
        pr.out_dm_stride = out_stride;
        pr.out_b0_stride = out_stride * plan->ndm;
        pr.shift_dm_stride = plan->nchans;
        pr.n_out = pr.n_base = nsamp_out;
        pr.nchans = plan->nchans;
        pr.ndm = plan->ndm;
        pr.nb1 = 1;
        if (small) {
            const bool tiny = static_cast<int64_t>(plan->ndm) * size_len * nbeams < 8192LL * plan->nsm;
            plan->last_kernel = tiny ? DEDISP_KERNEL_NAIVE : DEDISP_KERNEL_DIRECT;
            rc = tiny ? launch_naive(pr, in_t, stream, &plan->last_launches)
                      : launch_direct(pr, in_t, plan->spread_full, stream, &plan->last_launches);
        } else {
            rc = run_problem(plan, pr, in_t, plan->spread_full, stream);
        }
        return rc == 0 ? DEDISP_OK : DEDISP_ECUDA;
    }

    // two-stage subband: stage 1 into scratch, stage 2 from scratch
    const int ncoarse = plan->ndm / plan->nfine, cps = plan->nchans / plan->nsub;
    const int64_t n1 = round_up(nsamp_out + plan->maxshift2_max, 16);
    if (static_cast<size_t>(nbeams) * ncoarse * plan->nsub * n1 * 4 > plan->scratch.bytes)
        return DEDISP_ESTATE;  // dedisp_plan_reserve was not called for this shape
    // stage 1: b1 = subband s, rows = coarse groups k, channels = the cps channels of s
    pr.in = in;
    pr.out = plan->scratch.p;
    pr.shift = plan->d_s1;
    // stage 1 forms, for subband s of group k, only the samples stage 2 reads: n_out + max_d s2(d, s)
    pr.row_extra = plan->d_maxshift2_ks;
    pr.row_extra_b1_stride = ncoarse;
    pr.in_chan_stride = in_stride;
    pr.in_b0_stride = in_stride * plan->nchans;
    pr.in_b1_stride = in_stride * cps;
    pr.out_dm_stride = n1 * plan->nsub;
    pr.out_b0_stride = n1 * plan->nsub * ncoarse;
    pr.out_b1_stride = n1;
    pr.shift_dm_stride = plan->nchans;
    pr.shift_b1_stride = cps;
    pr.n_base = nsamp_out;
    pr.n_out = nsamp_out + plan->maxshift2_max;
    pr.nchans = cps;
    pr.ndm = ncoarse;
    pr.nb1 = plan->nsub;
    rc = run_problem(plan, pr, in_t, plan->spread_s1, stream);
    if (rc != 0)
        return DEDISP_ECUDA;
    plan->ev_mid_valid = false;
    if (plan->timing) {
        cudaEventRecord(plan->ev[2], static_cast<cudaStream_t>(stream));
        plan->ev_mid_valid = true;
    }
    // stage 2: b1 = coarse group k, rows = its nfine trials, channels = the nsub partial series
    Problem p2;
    std::memset(&p2, 0, sizeof(p2));
    p2.in = plan->scratch.p;
    p2.out = out;
    p2.shift = plan->d_s2;
    p2.in_chan_stride = n1;
    p2.in_b0_stride = n1 * plan->nsub * ncoarse;
    p2.in_b1_stride = n1 * plan->nsub;
    p2.in_len = n1;
    p2.out_dm_stride = out_stride;
    p2.out_b0_stride = out_stride * plan->ndm;
    p2.out_b1_stride = out_stride * plan->nfine;
    p2.shift_dm_stride = plan->nsub;
    p2.shift_b1_stride = static_cast<int64_t>(plan->nsub) * plan->nfine;
    p2.n_out = p2.n_base = nsamp_out;
    p2.nchans = plan->nsub;
    p2.ndm = plan->nfine;
    p2.nb0 = nbeams;
    p2.nb1 = ncoarse;
    const int stage1_kernel = plan->last_kernel;
    rc = run_problem(plan, p2, dtype == DEDISP_F32 ? Elem::F32 : Elem::I32, plan->spread_s2, stream);
    plan->last_kernel = stage1_kernel;
    return rc == 0 ? DEDISP_OK : DEDISP_ECUDA;
}

// tables onto the current device, scratch for executes of up to nsamp_out x nbeams (blocking)
dedisp_status reserve(dedisp_plan* plan, dedisp_dtype dtype, int64_t nsamp_out, int nbeams)
{
    if (!plan || nbeams <= 0 || nsamp_out < 0 || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    dedisp_status st = upload(plan);
    if (st != DEDISP_OK)
        return st;
    size_t pairs = 0, scratch = 0;
    int64_t nwin = 0;  // longest execute <= nsamp_out that runs on the register-window kernel
    if (plan->nsub == 0) {
        // The reservation covers every execute of UP TO nsamp_out samples.  A length beyond the window
        // kernel's 32-bit time limit runs on the long-tile kernel, but shorter executes of the same plan
        // still resolve to the window kernel: size the pair buffer for the longest length it accepts
        // (window_pair_stride grows with the length, so that one covers all shorter ones).
        if (nsamp_out > 0 && use_window(plan, dtype, 0)) {
            nwin = nsamp_out;
            if (!use_window(plan, dtype, nwin)) {
                int64_t lo = 0, hi = nsamp_out;  // accepted at lo, refused at hi
                while (hi - lo > 1) {
                    const int64_t mid = lo + (hi - lo) / 2;
                    (use_window(plan, dtype, mid) ? lo : hi) = mid;
                }
                nwin = lo;
            }
        }
        if (nwin > 0)
            pairs = static_cast<size_t>(nbeams) * plan->nchans * window_pair_stride(plan->win, nwin) * 8;
    } else {
        scratch = static_cast<size_t>(dedisp_plan_scratch_bytes(plan, nsamp_out, nbeams));
    }
    size_t npart = static_cast<size_t>(detect_blocks(plan->ndm));
    if (nwin > 0 && fused_stats_ok(plan, dtype, nwin))
        npart = std::max(npart, static_cast<size_t>(plan->win.ntile_dm) * window_ntile_t(plan->win, nwin));
    const size_t det = static_cast<size_t>(nbeams) * npart * 2 * sizeof(double);
    if (plan->pairs.ensure(pairs) != cudaSuccess || plan->scratch.ensure(scratch) != cudaSuccess ||
        plan->det_partial.ensure(det) != cudaSuccess || plan->det_pivot.ensure(nbeams * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ENOMEM;
    }
    return DEDISP_OK;
}

// Error exit of the host entries: waits for the two copy streams and the caller's stream (errors ignored,
// the call is failing already) so that no DMA touches the caller's host buffers after the return.
void drain_host_streams(dedisp_plan* plan, cudaStream_t st)
{
    for (cudaStream_t q : {plan->copy_st[0], plan->copy_st[1]})
        if (q)
            cudaStreamSynchronize(q);
    cudaStreamSynchronize(st);
    cudaGetLastError();
}

// Time piece i of a host-entry execute: uniform pieces of csize samples, the first one split at a quarter so
// that the first kernel (and with it the first device-to-host copy) starts after a quarter of the wait.
// Returns false past the end.
bool host_piece(int64_t nsamp, int64_t csize, int i, int64_t* t0, int64_t* cn)
{
    const int64_t q = round_up(csize / 4, 64);
    const int64_t b0 = i == 0 ? 0 : i == 1 ? q : static_cast<int64_t>(i - 1) * csize;
    const int64_t b1 = i == 0 ? q : static_cast<int64_t>(i) * csize;
    if (b0 >= nsamp)
        return false;
    *t0 = b0;
    *cn = (b1 < nsamp ? b1 : nsamp) - b0;
    return true;
}

bool ensure_copy_streams(dedisp_plan* plan)
{
    if (plan->copy_st[0])
        return true;
    bool ok = cudaStreamCreateWithFlags(&plan->copy_st[0], cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&plan->copy_st[1], cudaStreamNonBlocking) == cudaSuccess;
    for (auto& e : plan->ev_copy)
        ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
    if (!ok)
        cudaGetLastError();
    return ok;
}

}  // namespace

extern "C" {

dedisp_status dedisp_plan_create(dedisp_plan** plan, int nchans, double f_top_mhz, double df_mhz,
                                 double t_samp_ms, const double* dm_list, int ndm, int nsub, int nfine)
{
    if (!plan)
        return DEDISP_EINVAL;
    *plan = nullptr;
    if (nchans <= 0 || ndm <= 0 || !dm_list || !(f_top_mhz > 0.0) || !(df_mhz > 0.0) ||
        !(t_samp_ms > 0.0) || !std::isfinite(f_top_mhz) || !std::isfinite(df_mhz) ||
        !std::isfinite(t_samp_ms) || nsub < 0)
        return DEDISP_EINVAL;
    if (!(f_top_mhz - static_cast<double>(nchans - 1) * df_mhz > 0.0))
        return DEDISP_EINVAL;
    for (int d = 0; d < ndm; ++d)
        if (!(dm_list[d] >= 0.0) || !std::isfinite(dm_list[d]))
            return DEDISP_EINVAL;
    if (nsub > 0) {
        if (nfine <= 0 || nchans % nsub != 0 || ndm % nfine != 0)
            return DEDISP_EINVAL;
        for (int d = 1; d < ndm; ++d)
            if (dm_list[d] < dm_list[d - 1])
                return DEDISP_EINVAL;
    }
    dedisp_plan* p = new (std::nothrow) dedisp_plan;
    if (!p)
        return DEDISP_ENOMEM;
    try {
        p->nchans = nchans;
        p->ndm = ndm;
        p->nsub = nsub;
        p->nfine = nsub > 0 ? nfine : 0;
        p->f_top = f_top_mhz;
        p->df = df_mhz;
        p->t_samp = t_samp_ms;
        p->dm.assign(dm_list, dm_list + ndm);
        if (!build_shift_table(nchans, f_top_mhz, df_mhz, t_samp_ms, dm_list, ndm, p->shift,
                               p->max_delay)) {
            delete p;
            return DEDISP_EINVAL;
        }
        const int tiles[3] = {32, 16, 8};
        if (nsub == 0) {
            for (int k = 0; k < 3; ++k)
                p->spread_full[k] = tile_spread(p->shift.data(), ndm, nchans, nchans, tiles[k]);
            WindowGeom pref[4];
            const int npref = window_geom_preferences(pref, 4);
            for (int k = 0; k < npref && !p->win_fits; ++k) {
                build_window_plan(p->shift.data(), ndm, nchans, pref[k], p->win);
                p->win_fits = p->win.ok && window_fits_smem(p->win);
            }
        } else {
            build_subband_tables(p->shift, nchans, ndm, nsub, nfine, dm_list, p->s1, p->s2, p->nominal,
                                 p->maxshift2, p->max_delay);
            const int ncoarse = ndm / nfine;
            for (int k = 0; k < ncoarse; ++k)
                p->maxshift2_max = p->maxshift2[k] > p->maxshift2_max ? p->maxshift2[k] : p->maxshift2_max;
            p->maxshift2_ks.assign(static_cast<size_t>(nsub) * ncoarse, 0);
            for (int d = 0; d < ndm; ++d)
                for (int s = 0; s < nsub; ++s) {
                    int32_t& m = p->maxshift2_ks[static_cast<size_t>(s) * ncoarse + d / nfine];
                    const int32_t v = p->s2[static_cast<size_t>(d) * nsub + s];
                    m = v > m ? v : m;
                }
            for (int k = 0; k < 3; ++k) {
                p->spread_s1[k] = tile_spread(p->s1.data(), ncoarse, nchans, nchans, tiles[k]);
                int w = 0;
                for (int g = 0; g < ncoarse; ++g) {
                    const int v = tile_spread(p->s2.data() + static_cast<size_t>(g) * nfine * nsub, nfine,
                                              nsub, nsub, tiles[k]);
                    w = v > w ? v : w;
                }
                p->spread_s2[k] = w;
            }
        }
    } catch (const std::bad_alloc&) {
        delete p;
        return DEDISP_ENOMEM;
    }
    *plan = p;
    return DEDISP_OK;
}

dedisp_status dedisp_plan_destroy(dedisp_plan* p)
{
    if (!p)
        return DEDISP_OK;
    if (p->nstreams != 0)
        return DEDISP_ESTATE;
    free_tables(p);
    if (p->ev[0])
        cudaEventDestroy(p->ev[0]);
    if (p->ev[1])
        cudaEventDestroy(p->ev[1]);
    if (p->ev[2])
        cudaEventDestroy(p->ev[2]);
    for (auto& e : p->ev_copy)
        if (e)
            cudaEventDestroy(e);
    for (auto& c : p->copy_st)
        if (c)
            cudaStreamDestroy(c);
    p->pairs.release();
    p->scratch.release();
    p->host_in.release();
    p->host_out.release();
    p->det_partial.release();
    p->det_pivot.release();
    p->det_events.release();
    p->det_results.release();
    delete p;
    return DEDISP_OK;
}

int64_t dedisp_plan_max_delay(const dedisp_plan* p) { return p ? p->max_delay : -1; }
int dedisp_plan_nchans(const dedisp_plan* p) { return p ? p->nchans : -1; }
int dedisp_plan_ndm(const dedisp_plan* p) { return p ? p->ndm : -1; }
int dedisp_plan_nsub(const dedisp_plan* p) { return p ? p->nsub : -1; }
int dedisp_plan_nfine(const dedisp_plan* p) { return p ? p->nfine : -1; }
int dedisp_plan_last_kernel(const dedisp_plan* p) { return p ? p->last_kernel : -1; }

int dedisp_plan_last_launches(const dedisp_plan* p) { return p ? p->last_launches : -1; }

dedisp_status dedisp_plan_copy_host_output(dedisp_plan* p, void* dst, int64_t bytes, void* cuda_stream)
{
    if (!p || !dst)
        return DEDISP_EINVAL;
    if (p->ho_rows == 0 || !p->host_out.p)
        return DEDISP_ESTATE;
    if (bytes != p->ho_rows * p->ho_n * 4)
        return DEDISP_ESHAPE;
    return cudaMemcpy2DAsync(dst, p->ho_n * 4, p->host_out.p, p->ho_stride * 4, p->ho_n * 4, p->ho_rows,
                             cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess
               ? DEDISP_OK
               : DEDISP_ECUDA;
}

dedisp_status dedisp_plan_set_timing(dedisp_plan* p, int on)
{
    if (!p)
        return DEDISP_EINVAL;
    if (on && !p->ev[0]) {
        if (cudaEventCreate(&p->ev[0]) != cudaSuccess || cudaEventCreate(&p->ev[1]) != cudaSuccess ||
            cudaEventCreate(&p->ev[2]) != cudaSuccess) {
            cudaGetLastError();
            return DEDISP_ECUDA;
        }
    }
    p->timing = on != 0;
    p->ev_valid = p->ev_mid_valid = false;
    return DEDISP_OK;
}

dedisp_status dedisp_plan_last_stage_ms(dedisp_plan* p, float* ms)
{
    if (!p || !ms)
        return DEDISP_EINVAL;
    if (!p->ev_valid || !p->ev_mid_valid)
        return DEDISP_ESTATE;
    if (cudaEventSynchronize(p->ev[1]) != cudaSuccess ||
        cudaEventElapsedTime(&ms[0], p->ev[0], p->ev[2]) != cudaSuccess ||
        cudaEventElapsedTime(&ms[1], p->ev[2], p->ev[1]) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ECUDA;
    }
    return DEDISP_OK;
}

dedisp_status dedisp_plan_last_kernel_ms(dedisp_plan* p, float* ms)
{
    if (!p || !ms)
        return DEDISP_EINVAL;
    if (!p->ev_valid)
        return DEDISP_ESTATE;
    if (cudaEventSynchronize(p->ev[1]) != cudaSuccess || cudaEventElapsedTime(ms, p->ev[0], p->ev[1]) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ECUDA;
    }
    return DEDISP_OK;
}

dedisp_status dedisp_plan_get_shifts(const dedisp_plan* p, int32_t* host_out)
{
    if (!p || !host_out)
        return DEDISP_EINVAL;
    std::memcpy(host_out, p->shift.data(), p->shift.size() * sizeof(int32_t));
    return DEDISP_OK;
}

dedisp_status dedisp_plan_get_subband_shifts(const dedisp_plan* p, int32_t* s1, int32_t* s2,
                                             double* nominal_dm, int32_t* maxshift2)
{
    if (!p)
        return DEDISP_EINVAL;
    if (p->nsub == 0)
        return DEDISP_ESTATE;
    if (s1)
        std::memcpy(s1, p->s1.data(), p->s1.size() * sizeof(int32_t));
    if (s2)
        std::memcpy(s2, p->s2.data(), p->s2.size() * sizeof(int32_t));
    if (nominal_dm)
        std::memcpy(nominal_dm, p->nominal.data(), p->nominal.size() * sizeof(double));
    if (maxshift2)
        std::memcpy(maxshift2, p->maxshift2.data(), p->maxshift2.size() * sizeof(int32_t));
    return DEDISP_OK;
}

dedisp_status dedisp_plan_set_kernel(dedisp_plan* p, dedisp_kernel k)
{
    if (!p || k < DEDISP_KERNEL_AUTO || k > DEDISP_KERNEL_LONG)
        return DEDISP_EINVAL;
    if (k == DEDISP_KERNEL_WINDOW && !(p->nsub == 0 && p->win.ok && p->win_fits))
        return DEDISP_ESTATE;  // the shift table does not fit the register-window kernel's limits
    p->kernel = k;
    return DEDISP_OK;
}

dedisp_status dedisp_plan_set_window_geometry(dedisp_plan* p, int T, int G, int NT, int D)
{
    if (!p)
        return DEDISP_EINVAL;
    if (p->nsub != 0 || p->uploaded)
        return DEDISP_ESTATE;  // brute-force plans, before the first dedisp_plan_reserve
    WindowGeom g;
    g.T = T;
    g.G = G;
    g.NT = NT;
    g.D = D;
    if (!window_geom_supported(g))
        return DEDISP_EINVAL;
    WindowPlan wp;
    if (!build_window_plan(p->shift.data(), p->ndm, p->nchans, g, wp) || !window_fits_smem(wp))
        return DEDISP_ESTATE;  // the table does not fit this geometry; the plan keeps its own
    p->win = std::move(wp);
    p->win_fits = true;
    return DEDISP_OK;
}

int dedisp_plan_resolved_kernel(const dedisp_plan* p, dedisp_dtype dtype)
{
    if (!p || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return -1;
    if (use_window(p, dtype, 0))
        return DEDISP_KERNEL_WINDOW;
    // AUTO without the window kernel: long tiles (the direct kernel below 4096 samples per row)
    return p->kernel == DEDISP_KERNEL_AUTO || p->kernel == DEDISP_KERNEL_WINDOW ? DEDISP_KERNEL_LONG : p->kernel;
}

dedisp_status dedisp_plan_window_info(const dedisp_plan* p, int64_t* info)
{
    if (!p || !info)
        return DEDISP_EINVAL;
    info[0] = p->win.ok && p->win_fits;
    info[1] = p->win.Hb;
    info[2] = p->win.kmax;
    info[3] = p->win.lmax;
    info[4] = p->win.ntile_dm;
    info[5] = p->win.geom.W();
    info[6] = p->win.geom.rows();
    info[7] = p->win.nband;
    info[8] = p->win.geom.T;
    info[9] = p->win.geom.G;
    info[10] = p->win.geom.NT;
    info[11] = p->win.geom.D;
    info[12] = p->win.ch;
    info[13] = p->win.nst;
    return DEDISP_OK;
}

int64_t dedisp_plan_scratch_bytes(const dedisp_plan* p, int64_t nsamp_out, int nbeams)
{
    if (!p || nsamp_out < 0 || nbeams <= 0)
        return -1;
    if (p->nsub == 0)
        return 0;
    const int64_t n1 = round_up(nsamp_out + p->maxshift2_max, 16);
    return static_cast<int64_t>(nbeams) * (p->ndm / p->nfine) * p->nsub * n1 * 4;
}

dedisp_status dedisp_plan_reserve(dedisp_plan* plan, dedisp_dtype dtype, int64_t nsamp_out, int nbeams)
{
    return reserve(plan, dtype, nsamp_out, nbeams);
}

dedisp_status dedisp_execute(dedisp_plan* plan, const void* in, void* out, dedisp_dtype dtype,
                             int64_t nsamp_out, int64_t in_stride, int64_t out_stride, int nbeams,
                             void* cuda_stream)
{
    return execute_device(plan, in, out, dtype, nsamp_out, in_stride, out_stride, nbeams, cuda_stream);
}

dedisp_status dedisp_execute_host(dedisp_plan* plan, const void* host_in, void* host_out,
                                  dedisp_dtype dtype, int64_t nsamp_out, int nbeams, void* cuda_stream)
{
    if (!plan || !host_in || !host_out || nbeams <= 0 || nsamp_out < 0 ||
        (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    if (nsamp_out == 0)
        return DEDISP_OK;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t es = in_size(dtype);
    const int64_t n_in = nsamp_out + plan->max_delay;
    const int64_t in_stride = round_up(n_in, 16), out_stride = round_up(nsamp_out, 4);
    const size_t rows_in = static_cast<size_t>(nbeams) * plan->nchans;
    const size_t rows_out = static_cast<size_t>(nbeams) * plan->ndm;
    if (plan->host_in.ensure(rows_in * in_stride * es) != cudaSuccess ||
        plan->host_out.ensure(rows_out * out_stride * 4) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ENOMEM;
    }
    plan->ho_rows = static_cast<int64_t>(rows_out);
    plan->ho_n = nsamp_out;
    plan->ho_stride = out_stride;
    // Brute-force plans are cut into up to kHostChunks time chunks so that the H2D copy of chunk
    // i+1, the kernels of chunk i and the D2H copy of chunk i-1 overlap (outputs of different times
    // are independent; chunk i reads input columns [t_i, t_i + C_i + max_delay)).
    int nchunk = 1;
    if (plan->nsub == 0) {
        nchunk = static_cast<int>(nsamp_out / 32768);
        nchunk = nchunk < 1 ? 1 : nchunk > dedisp_plan::kHostChunks ? dedisp_plan::kHostChunks : nchunk;
    }
    {
        const int64_t piece = nchunk == 1 ? nsamp_out : round_up((nsamp_out + nchunk - 1) / nchunk, 64);
        const dedisp_status rs = reserve(plan, dtype, piece, nbeams);
        if (rs != DEDISP_OK)
            return rs;
    }
    if (nchunk == 1) {
        if (cudaMemcpy2DAsync(plan->host_in.p, in_stride * es, host_in, n_in * es, n_in * es, rows_in,
                              cudaMemcpyHostToDevice, st) != cudaSuccess)
            return DEDISP_ECUDA;
        // from here on a copy that reads the caller's host_in may be queued: no return without waiting for it
        dedisp_status s = execute_device(plan, plan->host_in.p, plan->host_out.p, dtype, nsamp_out,
                                         in_stride, out_stride, nbeams, cuda_stream);
        if (s == DEDISP_OK && cudaMemcpy2DAsync(host_out, nsamp_out * 4, plan->host_out.p, out_stride * 4, nsamp_out * 4,
                                                rows_out, cudaMemcpyDeviceToHost, st) != cudaSuccess)
            s = DEDISP_ECUDA;
        if (cudaStreamSynchronize(st) != cudaSuccess && s == DEDISP_OK)
            s = DEDISP_ECUDA;
        return s;
    }
    if (!ensure_copy_streams(plan))
        return DEDISP_ECUDA;
    cudaStream_t h2d = plan->copy_st[0], d2h = plan->copy_st[1];
    cudaEvent_t* ev_in = plan->ev_copy;                              // [nchunk] input columns landed
    cudaEvent_t* ev_ex = plan->ev_copy + dedisp_plan::kHostEvents;   // [nchunk] kernels of the chunk done
    cudaEvent_t ev_start = plan->ev_copy[2 * dedisp_plan::kHostEvents];
    cudaEvent_t ev_done = plan->ev_copy[2 * dedisp_plan::kHostEvents + 1];
    const int64_t csize = round_up((nsamp_out + nchunk - 1) / nchunk, 64);
    bool ok = cudaEventRecord(ev_start, st) == cudaSuccess &&
              cudaStreamWaitEvent(h2d, ev_start, 0) == cudaSuccess &&
              cudaStreamWaitEvent(d2h, ev_start, 0) == cudaSuccess;
    const char* hin = static_cast<const char*>(host_in);
    char* din = static_cast<char*>(plan->host_in.p);
    char* dout = static_cast<char*>(plan->host_out.p);
    char* hout = static_cast<char*>(host_out);
    int launches = 0;
    int64_t col = 0;  // input columns copied so far
    dedisp_status exec_status = DEDISP_OK;
    for (int i = 0; i <= nchunk && ok; ++i) {
        int64_t t0, cn;
        if (!host_piece(nsamp_out, csize, i, &t0, &cn))
            break;
        const int64_t need = t0 + cn + plan->max_delay;  // input columns chunk i reads
        if (need > col) {
            ok = cudaMemcpy2DAsync(din + col * es, in_stride * es, hin + col * es, n_in * es, (need - col) * es,
                                   rows_in, cudaMemcpyHostToDevice, h2d) == cudaSuccess;
            col = need;
        }
        ok = ok && cudaEventRecord(ev_in[i], h2d) == cudaSuccess && cudaStreamWaitEvent(st, ev_in[i], 0) == cudaSuccess;
        if (!ok)
            break;
        exec_status = execute_device(plan, din + t0 * es, dout + t0 * 4, dtype, cn, in_stride,
                                     out_stride, nbeams, cuda_stream, nullptr, nsamp_out);
        if (exec_status != DEDISP_OK)
            break;
        launches += plan->last_launches;
        ok = cudaEventRecord(ev_ex[i], st) == cudaSuccess && cudaStreamWaitEvent(d2h, ev_ex[i], 0) == cudaSuccess &&
             cudaMemcpy2DAsync(hout + t0 * 4, nsamp_out * 4, dout + t0 * 4, out_stride * 4, cn * 4, rows_out,
                               cudaMemcpyDeviceToHost, d2h) == cudaSuccess;
    }
    plan->last_launches = launches;
    ok = ok && exec_status == DEDISP_OK;
    ok = ok && cudaEventRecord(ev_done, d2h) == cudaSuccess && cudaStreamWaitEvent(st, ev_done, 0) == cudaSuccess;
    if (!ok) {
        // copies from / to the caller's buffers may still be queued on the private streams, which the
        // caller's stream has not joined: wait for all three before the buffers go back to the caller
        drain_host_streams(plan, st);
        return exec_status != DEDISP_OK ? exec_status : DEDISP_ECUDA;
    }
    return cudaStreamSynchronize(st) == cudaSuccess ? DEDISP_OK : DEDISP_ECUDA;
}

// ---- streaming chunk driver -------------------------------------------------------------------

dedisp_status dedisp_stream_create(dedisp_stream** s, dedisp_plan* plan, dedisp_dtype dtype,
                                   int64_t chunk, int nbeams)
{
    if (!s)
        return DEDISP_EINVAL;
    *s = nullptr;
    if (!plan || chunk <= 0 || nbeams <= 0 || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    if (plan->nsub != 0)
        return DEDISP_ESTATE;
    {
        const dedisp_status rs = reserve(plan, dtype, chunk, nbeams);
        if (rs != DEDISP_OK)
            return rs;
    }
    dedisp_stream* q = new (std::nothrow) dedisp_stream;
    if (!q)
        return DEDISP_ENOMEM;
    q->plan = plan;
    q->dtype = dtype;
    q->chunk = chunk;
    q->nbeams = nbeams;
    q->wstride = round_up(plan->max_delay + chunk, 16);
    const size_t bytes = static_cast<size_t>(nbeams) * plan->nchans * q->wstride * in_size(dtype);
    for (int i = 0; i < 2; ++i)
        if (q->work[i].ensure(bytes) != cudaSuccess) {
            cudaError_t e = cudaGetLastError();
            q->work[0].release();
            q->work[1].release();
            delete q;
            return e == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA;
        }
    ++plan->nstreams;
    *s = q;
    return DEDISP_OK;
}

dedisp_status dedisp_stream_reset(dedisp_stream* s, void* cuda_stream)
{
    if (!s)
        return DEDISP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    for (int i = 0; i < 2; ++i)
        if (cudaMemsetAsync(s->work[i].p, 0, s->work[i].bytes, st) != cudaSuccess)
            return DEDISP_ECUDA;
    s->cur = 0;
    s->zeroed = true;
    return DEDISP_OK;
}

dedisp_status dedisp_stream_push(dedisp_stream* s, const void* chunk_in, void* out, void* cuda_stream)
{
    if (!s || !chunk_in || !out)
        return DEDISP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!s->zeroed) {
        dedisp_status r = dedisp_stream_reset(s, cuda_stream);
        if (r != DEDISP_OK)
            return r;
    }
    dedisp_plan* p = s->plan;
    const size_t es = in_size(s->dtype);
    const size_t rows = static_cast<size_t>(s->nbeams) * p->nchans;
    const int64_t M = p->max_delay, C = s->chunk;
    unsigned char* cur = static_cast<unsigned char*>(s->work[s->cur].p);
    unsigned char* nxt = static_cast<unsigned char*>(s->work[s->cur ^ 1].p);
    // 1. the new chunk goes behind the carried max_delay samples of every channel
    if (cudaMemcpy2DAsync(cur + M * es, s->wstride * es, chunk_in, C * es, C * es, rows,
                          cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return DEDISP_ECUDA;
    // 2. de-disperse the work buffer: outputs for stream times [kC - M, (k+1)C - M)
    dedisp_status r = execute_device(p, cur, out, s->dtype, C, s->wstride, C, s->nbeams, cuda_stream);
    if (r != DEDISP_OK)
        return r;
    // 3. the last max_delay samples become the head of the other buffer (no overlapping copy,
    //    valid for max_delay > chunk as well)
    if (M > 0 && cudaMemcpy2DAsync(nxt, s->wstride * es, cur + C * es, s->wstride * es, M * es, rows,
                                   cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return DEDISP_ECUDA;
    s->cur ^= 1;
    return DEDISP_OK;
}

dedisp_status dedisp_stream_push_host(dedisp_stream* s, const void* host_chunk_in, void* host_out,
                                      void* cuda_stream)
{
    if (!s || !host_chunk_in || !host_out)
        return DEDISP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    dedisp_plan* p = s->plan;
    const size_t es = in_size(s->dtype);
    const size_t nout = static_cast<size_t>(s->nbeams) * p->ndm * s->chunk * 4;
    if (s->chunk % 4 != 0)
        return DEDISP_ESHAPE;
    if (s->host_out.ensure(nout) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ENOMEM;
    }
    if (!s->zeroed) {
        dedisp_status r = dedisp_stream_reset(s, cuda_stream);
        if (r != DEDISP_OK)
            return r;
    }
    // The push is cut into time pieces: the H2D copy of piece j+1 (straight into the work buffer,
    // behind the carry), the kernels of piece j and the D2H copy of piece j-1 overlap.  Piece j
    // emits outputs [j*C', (j+1)*C') and reads work columns [j*C', (j+1)*C' + max_delay).
    if (!ensure_copy_streams(p))
        return DEDISP_ECUDA;
    const int64_t M = p->max_delay, C = s->chunk;
    int npiece = static_cast<int>(C / 16384);
    npiece = npiece < 1 ? 1 : npiece > dedisp_plan::kHostChunks ? dedisp_plan::kHostChunks : npiece;
    const int64_t psize = round_up((C + npiece - 1) / npiece, 64);
    const size_t rows_in = static_cast<size_t>(s->nbeams) * p->nchans;
    const size_t rows_out = static_cast<size_t>(s->nbeams) * p->ndm;
    unsigned char* cur = static_cast<unsigned char*>(s->work[s->cur].p);
    unsigned char* nxt = static_cast<unsigned char*>(s->work[s->cur ^ 1].p);
    const unsigned char* hin = static_cast<const unsigned char*>(host_chunk_in);
    char* dout = static_cast<char*>(s->host_out.p);
    char* hout = static_cast<char*>(host_out);
    cudaStream_t h2d = p->copy_st[0], d2h = p->copy_st[1];
    cudaEvent_t* ev_in = p->ev_copy;
    cudaEvent_t* ev_ex = p->ev_copy + dedisp_plan::kHostEvents;
    cudaEvent_t ev_start = p->ev_copy[2 * dedisp_plan::kHostEvents];
    cudaEvent_t ev_done = p->ev_copy[2 * dedisp_plan::kHostEvents + 1];
    bool ok = cudaEventRecord(ev_start, st) == cudaSuccess && cudaStreamWaitEvent(h2d, ev_start, 0) == cudaSuccess &&
              cudaStreamWaitEvent(d2h, ev_start, 0) == cudaSuccess;
    int launches = 0;
    for (int j = 0; j < npiece && ok; ++j) {
        const int64_t t0 = j * psize;
        if (t0 >= C)
            break;
        const int64_t cn = C - t0 < psize ? C - t0 : psize;
        ok = cudaMemcpy2DAsync(cur + (M + t0) * es, s->wstride * es, hin + t0 * es, C * es, cn * es, rows_in,
                               cudaMemcpyHostToDevice, h2d) == cudaSuccess &&
             cudaEventRecord(ev_in[j], h2d) == cudaSuccess && cudaStreamWaitEvent(st, ev_in[j], 0) == cudaSuccess;
        if (!ok)
            break;
        const dedisp_status r = execute_device(p, cur + t0 * es, dout + t0 * 4, s->dtype, cn, s->wstride, C,
                                               s->nbeams, cuda_stream, nullptr, C);
        if (r != DEDISP_OK) {
            drain_host_streams(p, st);  // copies of the caller's chunk / into the caller's out may be queued
            return r;
        }
        launches += p->last_launches;
        ok = cudaEventRecord(ev_ex[j], st) == cudaSuccess && cudaStreamWaitEvent(d2h, ev_ex[j], 0) == cudaSuccess &&
             cudaMemcpy2DAsync(hout + t0 * 4, C * 4, dout + t0 * 4, C * 4, cn * 4, rows_out, cudaMemcpyDeviceToHost,
                               d2h) == cudaSuccess;
    }
    p->last_launches = launches;
    // the last max_delay samples become the head of the other buffer
    if (ok && M > 0)
        ok = cudaMemcpy2DAsync(nxt, s->wstride * es, cur + C * es, s->wstride * es, M * es, rows_in,
                               cudaMemcpyDeviceToDevice, st) == cudaSuccess;
    s->cur ^= 1;
    ok = ok && cudaEventRecord(ev_done, d2h) == cudaSuccess && cudaStreamWaitEvent(st, ev_done, 0) == cudaSuccess;
    if (!ok) {
        drain_host_streams(p, st);
        return DEDISP_ECUDA;
    }
    return cudaStreamSynchronize(st) == cudaSuccess ? DEDISP_OK : DEDISP_ECUDA;
}

dedisp_status dedisp_stream_destroy(dedisp_stream* s)
{
    if (!s)
        return DEDISP_OK;
    for (int i = 0; i < 2; ++i)
        s->work[i].release();
    s->host_in.release();
    s->host_out.release();
    if (s->plan)
        --s->plan->nstreams;
    delete s;
    return DEDISP_OK;
}

int64_t dedisp_plan_max_chunk(const dedisp_plan* p, dedisp_dtype dtype, int64_t mem_bytes, int nbeams)
{
    if (!p || mem_bytes <= 0 || nbeams <= 0 || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return -1;
    // eq. 3 with element sizes and the driver's two work buffers:
    //   mem >= nbeams * (2 * nchans * (M + n) * in_size + ndm * n * out_size)
    const double es = static_cast<double>(in_size(dtype));
    const double per_beam = static_cast<double>(mem_bytes) / nbeams;
    const double fixed = 2.0 * p->nchans * static_cast<double>(p->max_delay + 16) * es;
    const double per_samp = 2.0 * p->nchans * es + 4.0 * p->ndm;
    const double n = (per_beam - fixed) / per_samp;
    if (!(n >= 1.0))
        return 0;
    return static_cast<int64_t>(n) / 16 * 16;
}

dedisp_status dedisp_plan_detect(dedisp_plan* plan, const void* out, dedisp_dtype dtype, int64_t nsamp_out,
                                 int64_t out_stride, int nbeams, double nsigma, dedisp_event* events,
                                 int64_t capacity, dedisp_detect_result* results, void* cuda_stream)
{
    if (!plan || !out || !results || nbeams <= 0 || nsamp_out <= 0 || capacity < 0 || (capacity > 0 && !events) ||
        !(nsigma == nsigma) || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    if (out_stride < nsamp_out || out_stride % 4 != 0 || (reinterpret_cast<uintptr_t>(out) & 15) != 0)
        return DEDISP_ESHAPE;
    if (static_cast<size_t>(nbeams) * detect_blocks(plan->ndm) * 2 * sizeof(double) > plan->det_partial.bytes)
        return DEDISP_ESTATE;  // dedisp_plan_reserve was not called for this many beams
    plan->last_launches = 0;
    const int rc = launch_detect(out, dtype == DEDISP_F32 ? Elem::F32 : Elem::I32, nbeams, plan->ndm, nsamp_out,
                                 out_stride, nsigma, events, capacity, results,
                                 static_cast<double*>(plan->det_partial.p), cuda_stream, &plan->last_launches);
    return rc == 0 ? DEDISP_OK : DEDISP_ECUDA;
}

dedisp_status dedisp_execute_detect(dedisp_plan* plan, const void* in, void* out, dedisp_dtype dtype, int64_t nsamp_out,
                                    int64_t in_stride, int64_t out_stride, int nbeams, double nsigma,
                                    dedisp_event* events, int64_t capacity, dedisp_detect_result* results,
                                    void* cuda_stream)
{
    if (!plan || !results || nsamp_out <= 0 || capacity < 0 || (capacity > 0 && !events) || !(nsigma == nsigma))
        return DEDISP_EINVAL;
    if (!fused_stats_ok(plan, dtype, nsamp_out)) {
        // subband plans, tables outside the window kernel, several channel bands: de-disperse, then the
        // two-pass detection
        dedisp_status st = execute_device(plan, in, out, dtype, nsamp_out, in_stride, out_stride, nbeams, cuda_stream);
        if (st != DEDISP_OK)
            return st;
        const int launches = plan->last_launches;
        st = dedisp_plan_detect(plan, out, dtype, nsamp_out, out_stride, nbeams, nsigma, events, capacity, results,
                                cuda_stream);
        plan->last_launches += launches;
        return st;
    }
    const int64_t npart = static_cast<int64_t>(plan->win.ntile_dm) * window_ntile_t(plan->win, nsamp_out);
    if (!plan->uploaded || static_cast<size_t>(nbeams) * npart * 2 * sizeof(double) > plan->det_partial.bytes ||
        static_cast<size_t>(nbeams) * sizeof(double) > plan->det_pivot.bytes)
        return DEDISP_ESTATE;  // dedisp_plan_reserve was not called for this shape
    if (!in)
        return DEDISP_EINVAL;
    int launches = 0;
    const Elem in_t = dtype == DEDISP_F32 ? Elem::F32 : Elem::U8;
    double* pivot = static_cast<double*>(plan->det_pivot.p);
    if (launch_detect_pivot(in, in_t, nbeams, plan->nchans, in_stride, pivot, cuda_stream, &launches) != 0)
        return DEDISP_ECUDA;
    const StatReq sr{pivot, static_cast<double*>(plan->det_partial.p), npart, 0};
    const dedisp_status st =
        execute_device(plan, in, out, dtype, nsamp_out, in_stride, out_stride, nbeams, cuda_stream, &sr);
    if (st != DEDISP_OK)
        return st;
    launches += plan->last_launches;
    const int rc = launch_detect_fused(out, dtype == DEDISP_F32 ? Elem::F32 : Elem::I32, nbeams, plan->ndm, nsamp_out,
                                       out_stride, nsigma, events, capacity, results, sr.partial, npart, npart, pivot,
                                       cuda_stream, &launches);
    plan->last_launches = launches;
    return rc == 0 ? DEDISP_OK : DEDISP_ECUDA;
}

dedisp_status dedisp_execute_detect_host(dedisp_plan* plan, const void* host_in, dedisp_dtype dtype, int64_t nsamp_out,
                                         int nbeams, double nsigma, dedisp_event* host_events, int64_t capacity,
                                         dedisp_detect_result* host_results, void* cuda_stream)
{
    if (!plan || !host_in || !host_results || nbeams <= 0 || nsamp_out <= 0 || capacity < 0 ||
        (capacity > 0 && !host_events) || !(nsigma == nsigma) || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t es = in_size(dtype);
    const int64_t n_in = nsamp_out + plan->max_delay;
    const int64_t in_stride = round_up(n_in, 16), out_stride = round_up(nsamp_out, 4);
    const size_t rows_in = static_cast<size_t>(nbeams) * plan->nchans;
    const size_t rows_out = static_cast<size_t>(nbeams) * plan->ndm;
    if (plan->host_in.ensure(rows_in * in_stride * es) != cudaSuccess ||
        plan->host_out.ensure(rows_out * out_stride * 4) != cudaSuccess ||
        plan->det_events.ensure(static_cast<size_t>(nbeams) * capacity * sizeof(dedisp_event) + 16) != cudaSuccess ||
        plan->det_results.ensure(static_cast<size_t>(nbeams) * sizeof(dedisp_detect_result)) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ENOMEM;
    }
    plan->ho_rows = static_cast<int64_t>(rows_out);
    plan->ho_n = nsamp_out;
    plan->ho_stride = out_stride;
    // time pieces as in dedisp_execute_host: the H2D copy of piece i+1 overlaps the kernels of piece i; nothing
    // but the events and 32 bytes of statistics per beam comes back
    int nchunk = 1;
    if (plan->nsub == 0) {
        nchunk = static_cast<int>(nsamp_out / 32768);
        nchunk = nchunk < 1 ? 1 : nchunk > dedisp_plan::kHostChunks ? dedisp_plan::kHostChunks : nchunk;
    }
    const int64_t csize = nchunk == 1 ? nsamp_out : round_up((nsamp_out + nchunk - 1) / nchunk, 64);
    dedisp_status rs = reserve(plan, dtype, csize, nbeams);
    if (rs != DEDISP_OK)
        return rs;
    const bool fused = fused_stats_ok(plan, dtype, csize);
    int64_t npart_total = 0;
    if (fused) {
        int64_t t0, cn;
        for (int i = 0; (nchunk == 1 ? i == 0 : host_piece(nsamp_out, csize, i, &t0, &cn)); ++i)
            npart_total += static_cast<int64_t>(plan->win.ntile_dm) * window_ntile_t(plan->win, nchunk == 1 ? nsamp_out : cn);
        if (plan->det_partial.ensure(static_cast<size_t>(nbeams) * npart_total * 2 * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            return DEDISP_ENOMEM;
        }
    }
    if (!ensure_copy_streams(plan))
        return DEDISP_ECUDA;
    cudaStream_t h2d = plan->copy_st[0];
    cudaEvent_t* ev_in = plan->ev_copy;
    cudaEvent_t ev_start = plan->ev_copy[2 * dedisp_plan::kHostEvents];
    bool ok = cudaEventRecord(ev_start, st) == cudaSuccess && cudaStreamWaitEvent(h2d, ev_start, 0) == cudaSuccess;
    const char* hin = static_cast<const char*>(host_in);
    char* din = static_cast<char*>(plan->host_in.p);
    char* dout = static_cast<char*>(plan->host_out.p);
    double* pivot = static_cast<double*>(plan->det_pivot.p);
    const Elem in_t = dtype == DEDISP_F32 ? Elem::F32 : Elem::U8;
    int launches = 0;
    int64_t col = 0, part_off = 0;
    dedisp_status exec_status = DEDISP_OK;
    for (int i = 0; i <= nchunk && ok; ++i) {
        int64_t t0 = 0, cn = nsamp_out;
        if (nchunk == 1 ? i > 0 : !host_piece(nsamp_out, csize, i, &t0, &cn))
            break;
        const int64_t need = t0 + cn + plan->max_delay;
        if (need > col) {
            ok = cudaMemcpy2DAsync(din + col * es, in_stride * es, hin + col * es, n_in * es, (need - col) * es, rows_in,
                                   cudaMemcpyHostToDevice, h2d) == cudaSuccess;
            col = need;
        }
        ok = ok && cudaEventRecord(ev_in[i], h2d) == cudaSuccess && cudaStreamWaitEvent(st, ev_in[i], 0) == cudaSuccess;
        if (!ok)
            break;
        if (i == 0 && fused && launch_detect_pivot(din, in_t, nbeams, plan->nchans, in_stride, pivot, cuda_stream, &launches) != 0) {
            ok = false;
            break;
        }
        const StatReq sr{pivot, static_cast<double*>(plan->det_partial.p), npart_total, part_off};
        exec_status = execute_device(plan, din + t0 * es, dout + t0 * 4, dtype, cn, in_stride, out_stride, nbeams,
                                     cuda_stream, fused ? &sr : nullptr, nsamp_out);
        if (exec_status != DEDISP_OK)
            break;
        launches += plan->last_launches;
        part_off += static_cast<int64_t>(plan->win.ntile_dm) * (fused ? window_ntile_t(plan->win, cn) : 0);
    }
    if (!ok || exec_status != DEDISP_OK) {
        // host-to-device copies that read the caller's host_in may still be queued on the private copy
        // stream: wait for them before the buffer goes back to the caller
        drain_host_streams(plan, st);
        return exec_status != DEDISP_OK ? exec_status : DEDISP_ECUDA;
    }
    dedisp_event* dev = static_cast<dedisp_event*>(plan->det_events.p);
    dedisp_detect_result* dres = static_cast<dedisp_detect_result*>(plan->det_results.p);
    const Elem out_t = dtype == DEDISP_F32 ? Elem::F32 : Elem::I32;
    int rc;
    if (fused)
        rc = launch_detect_fused(dout, out_t, nbeams, plan->ndm, nsamp_out, out_stride, nsigma, dev, capacity, dres,
                                 static_cast<const double*>(plan->det_partial.p), npart_total, npart_total, pivot,
                                 cuda_stream, &launches);
    else
        rc = launch_detect(dout, out_t, nbeams, plan->ndm, nsamp_out, out_stride, nsigma, dev, capacity, dres,
                           static_cast<double*>(plan->det_partial.p), cuda_stream, &launches);
    plan->last_launches = launches;
    if (rc != 0 ||
        cudaMemcpyAsync(host_results, dres, nbeams * sizeof(dedisp_detect_result), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        drain_host_streams(plan, st);
        return DEDISP_ECUDA;
    }
    for (int b = 0; b < nbeams; ++b) {
        const int64_t k = std::min<int64_t>(host_results[b].count, capacity);
        if (k > 0 && cudaMemcpyAsync(host_events + static_cast<int64_t>(b) * capacity, dev + static_cast<int64_t>(b) * capacity,
                                     k * sizeof(dedisp_event), cudaMemcpyDeviceToHost, st) != cudaSuccess) {
            drain_host_streams(plan, st);
            return DEDISP_ECUDA;
        }
    }
    return cudaStreamSynchronize(st) == cudaSuccess ? DEDISP_OK : DEDISP_ECUDA;
}

dedisp_status dedisp_power_corner_turn(const void* volt, void* out, int nchans, int64_t nsamp, int64_t volt_stride,
                                       int64_t out_stride, void* cuda_stream)
{
    if (!volt || !out || nchans <= 0 || nsamp < 0)
        return DEDISP_EINVAL;
    if (volt_stride < nchans || out_stride < nsamp || (reinterpret_cast<uintptr_t>(volt) & 7) != 0 ||
        (reinterpret_cast<uintptr_t>(out) & 3) != 0)
        return DEDISP_ESHAPE;
    return launch_power_corner_turn(volt, out, nchans, nsamp, volt_stride, out_stride, cuda_stream) == 0 ? DEDISP_OK
                                                                                                         : DEDISP_ECUDA;
}

dedisp_status dedisp_bin(const void* in, void* out, int64_t nrows, int64_t nsamp, int64_t in_stride, int64_t out_stride,
                         int nb, void* cuda_stream)
{
    if (!in || !out || nrows <= 0 || nsamp < 0 || nb <= 0)
        return DEDISP_EINVAL;
    if (in_stride < nsamp || out_stride < nsamp / nb)
        return DEDISP_ESHAPE;
    return launch_bin(in, out, nrows, nsamp / nb, in_stride, out_stride, nb, cuda_stream) == 0 ? DEDISP_OK : DEDISP_ECUDA;
}

// ---- multi-pass subband survey (Tables 1 and 4) ---------------------------

dedisp_status dedisp_survey_create(dedisp_survey** survey, int nchans, double f_top_mhz, double df_mhz, double t_samp_ms,
                                   int nsub, const dedisp_pass* passes, int npass)
{
    if (!survey)
        return DEDISP_EINVAL;
    *survey = nullptr;
    if (!passes || npass <= 0 || nsub <= 0)
        return DEDISP_EINVAL;
    dedisp_survey* s = new (std::nothrow) dedisp_survey;
    if (!s)
        return DEDISP_ENOMEM;
    s->nchans = nchans;
    s->nsub = nsub;
    s->f_top = f_top_mhz;
    s->df = df_mhz;
    s->t_samp = t_samp_ms;
    dedisp_status st = DEDISP_OK;
    try {
        for (int i = 0; i < npass && st == DEDISP_OK; ++i) {
            const dedisp_pass& p = passes[i];
            if (p.ndm <= 0 || p.nfine <= 0 || p.bin <= 0 || !(p.dm_step >= 0.0) || !(p.dm_low >= 0.0)) {
                st = DEDISP_EINVAL;
                break;
            }
            std::vector<double> dm(p.ndm);
            for (int d = 0; d < p.ndm; ++d)
                dm[d] = p.dm_low + static_cast<double>(d) * p.dm_step;  // one multiply, one add, each rounded
            dedisp_plan* plan = nullptr;
            st = dedisp_plan_create(&plan, nchans, f_top_mhz, df_mhz, t_samp_ms * p.bin, dm.data(), p.ndm, nsub, p.nfine);
            if (st == DEDISP_OK) {
                s->passes.push_back(p);
                s->plans.push_back(plan);
                s->max_delay = std::max(s->max_delay, plan->max_delay * p.bin);
            }
        }
    } catch (const std::bad_alloc&) {
        st = DEDISP_ENOMEM;
    }
    if (st != DEDISP_OK) {
        dedisp_survey_destroy(s);
        return st;
    }
    *survey = s;
    return DEDISP_OK;
}

dedisp_status dedisp_survey_destroy(dedisp_survey* s)
{
    if (!s)
        return DEDISP_OK;
    for (dedisp_plan* p : s->plans)
        dedisp_plan_destroy(p);
    s->binned.release();
    delete s;
    return DEDISP_OK;
}

int dedisp_survey_npass(const dedisp_survey* s) { return s ? static_cast<int>(s->plans.size()) : -1; }
int64_t dedisp_survey_max_delay(const dedisp_survey* s) { return s ? s->max_delay : -1; }
int dedisp_survey_last_launches(const dedisp_survey* s) { return s ? s->last_launches : -1; }

const dedisp_plan* dedisp_survey_pass_plan(const dedisp_survey* s, int pass)
{
    return s && pass >= 0 && pass < static_cast<int>(s->plans.size()) ? s->plans[pass] : nullptr;
}

dedisp_status dedisp_survey_out_layout(const dedisp_survey* s, int64_t nsamp, int nbeams, int64_t* offset,
                                       int64_t* stride, int64_t* nout, int64_t* total)
{
    if (!s || nsamp < 0 || nbeams <= 0)
        return DEDISP_EINVAL;
    int64_t off = 0;
    for (size_t i = 0; i < s->plans.size(); ++i) {
        const int64_t n = nsamp / s->passes[i].bin, st = round_up(n, 4);
        if (offset)
            offset[i] = off;
        if (stride)
            stride[i] = st;
        if (nout)
            nout[i] = n;
        off += static_cast<int64_t>(nbeams) * s->plans[i]->ndm * st;
    }
    if (total)
        *total = off;
    return DEDISP_OK;
}

dedisp_status dedisp_survey_reserve(dedisp_survey* s, int64_t nsamp, int nbeams)
{
    if (!s || nsamp < 0 || nbeams <= 0)
        return DEDISP_EINVAL;
    size_t need = 0;
    for (size_t i = 0; i < s->plans.size(); ++i) {
        const int b = s->passes[i].bin;
        const dedisp_status st = reserve(s->plans[i], DEDISP_F32, nsamp / b, nbeams);
        if (st != DEDISP_OK)
            return st;
        if (b > 1)
            need = std::max(need, static_cast<size_t>(nbeams) * s->nchans * round_up((nsamp + s->max_delay) / b, 16) * 4);
    }
    if (s->binned.ensure(need) != cudaSuccess) {
        cudaGetLastError();
        return DEDISP_ENOMEM;
    }
    return DEDISP_OK;
}

dedisp_status dedisp_survey_execute(dedisp_survey* s, const void* in, void* out, int64_t nsamp, int64_t in_stride,
                                    int nbeams, void* cuda_stream)
{
    if (!s || !in || !out || nsamp < 0 || nbeams <= 0)
        return DEDISP_EINVAL;
    if (in_stride < nsamp + s->max_delay || in_stride % 4 != 0 || (reinterpret_cast<uintptr_t>(in) & 15) != 0 ||
        (reinterpret_cast<uintptr_t>(out) & 15) != 0)
        return DEDISP_ESHAPE;
    s->last_launches = 0;
    int64_t off = 0;
    float* o = static_cast<float*>(out);
    for (size_t i = 0; i < s->plans.size(); ++i) {
        dedisp_plan* plan = s->plans[i];
        const int b = s->passes[i].bin;
        const int64_t n = nsamp / b, ostride = round_up(n, 4);
        const void* src = in;
        int64_t sstride = in_stride;
        if (b > 1) {
            // stage (i), on the device: every row of nsamp + max_delay samples -> (nsamp + max_delay) / b
            const int64_t lb = (nsamp + s->max_delay) / b;
            sstride = round_up(lb, 16);
            if (static_cast<size_t>(nbeams) * s->nchans * sstride * 4 > s->binned.bytes)
                return DEDISP_ESTATE;  // dedisp_survey_reserve was not called for this shape
            if (launch_bin(in, s->binned.p, static_cast<int64_t>(nbeams) * s->nchans, lb, in_stride, sstride, b,
                           cuda_stream) != 0)
                return DEDISP_ECUDA;
            ++s->last_launches;
            src = s->binned.p;
        }
        // stages (ii) and (iii): the pass's subband plan (tables for t_samp * b)
        if (n > 0) {
            const dedisp_status st = execute_device(plan, src, o + off, DEDISP_F32, n, sstride, ostride, nbeams, cuda_stream);
            if (st != DEDISP_OK)
                return st;
            s->last_launches += plan->last_launches;
        }
        off += static_cast<int64_t>(nbeams) * plan->ndm * ostride;
    }
    return DEDISP_OK;
}

dedisp_status dedisp_fadd_microbench(int packed, int iters, int repeats, float* ms, double* adds, int* nsm_out,
                                     void* cuda_stream)
{
    if (iters <= 0 || repeats <= 0 || !ms || !adds)
        return DEDISP_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, nsm = 0;
    float* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    bool ok = cudaGetDevice(&dev) == cudaSuccess &&
              cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
              cudaMalloc(reinterpret_cast<void**>(&sink), 64) == cudaSuccess && cudaEventCreate(&e0) == cudaSuccess &&
              cudaEventCreate(&e1) == cudaSuccess;
    double per_launch = 0.0;
    if (ok) {
        ok = launch_fadd_microbench(packed, iters, nsm, sink, st, &per_launch) == 0;  // warm-up launch
        ok = ok && cudaEventRecord(e0, st) == cudaSuccess;
        for (int r = 0; r < repeats && ok; ++r)
            ok = launch_fadd_microbench(packed, iters, nsm, sink, st, &per_launch) == 0;
        ok = ok && cudaEventRecord(e1, st) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess &&
             cudaEventElapsedTime(ms, e0, e1) == cudaSuccess;
    }
    *adds = per_launch * repeats;
    if (nsm_out)
        *nsm_out = nsm;
    if (e0)
        cudaEventDestroy(e0);
    if (e1)
        cudaEventDestroy(e1);
    if (sink)
        cudaFree(sink);
    if (!ok) {
        cudaGetLastError();
        return DEDISP_ECUDA;
    }
    return DEDISP_OK;
}

const char* dedisp_strerror(dedisp_status s)
{
    switch (s) {
    case DEDISP_OK: return "ok";
    case DEDISP_EINVAL: return "invalid argument";
    case DEDISP_ENOMEM: return "out of memory";
    case DEDISP_ECUDA: return "CUDA error";
    case DEDISP_ESHAPE: return "shape, stride or alignment does not match the plan";
    case DEDISP_ESTATE: return "call not valid for this plan or stream";
    case DEDISP_ELIMIT: return "size exceeds the fixed scratch array of an allocation-free entry point";
    }
    return "unknown status";
}

const char* dedisp_version(void) { return "dedisp-b200 0.1 (sm_100a)"; }

}  // extern "C"
