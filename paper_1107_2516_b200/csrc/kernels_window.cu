// Register-window brute-force kernel for sm_100a.
//
//   out[d][t] = sum_c in[c][t + shift(c,d)]
//
// Launches per execute: one pairify, then one window_kernel per channel band.
//  1. pairify_kernel: P[c][u] = (in[c][u], in[c][u + NT*H]) as float2 (uint8 input is widened to
//     fp32 here; sums of < 2^24/255 bytes are exact in fp32).  Two samples NT*H apart that share
//     (c, d) have the same shift, so the main kernel adds two outputs per instruction
//     (add.f32x2 -> FADD2) from naturally aligned 64-bit registers, whatever the shift's parity.
//  2. window_kernel (band b): a block = G row groups x NT warps; a consumer
//     warp owns 8 DM rows x 32*T slots (pairs of output samples) and keeps their 8 x T packed
//     accumulators in registers for the whole band.  Per channel it loads ONE window of T + 1
//     staged pairs (LDS.64, conflict-free for odd T) that feeds all 8 rows: row j adds
//     w[i + o_j], o_j in {0, 1} chosen by a warp-uniform two-way branch (window_rows.inc).  Rows
//     follow the growing delay difference between neighbouring DM trials by moving their
//     accumulators up one slot now and then ("row shift", planned on the host: window_plan.cpp).
//     Channel segments are staged into a ring of shared-memory slots by 1-D TMA bulk copies
//     (cp.async.bulk + mbarrier) issued by thread 0 a few channels ahead.  At the end of the band the
//     accumulators go through a per-warp shared-memory transpose to coalesced global accesses:
//     band 0 stores, later bands add to what is there.
#include <cuda_runtime.h>

#include <cstdlib>

#include "dedisp_internal.h"

namespace dedisp {

typedef unsigned long long u64;

// ------------------------------------------------------------------------------------------------
// 1. pairify
// ------------------------------------------------------------------------------------------------
template <typename InT>
__global__ void __launch_bounds__(256) pairify_kernel(const InT* __restrict__ in, float2* __restrict__ pairs,
                                                      int64_t in_stride, int64_t pair_stride,
                                                      int64_t in_len, int hp)
{
    const int64_t u = (static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x) * 2;
    if (u >= pair_stride)
        return;
    const int64_t row = static_cast<int64_t>(blockIdx.z) * gridDim.y + blockIdx.y;
    const InT* src = in + row * in_stride;
    float v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int64_t idx = u + (k & 1) + (k >> 1) * static_cast<int64_t>(hp);
        v[k] = idx < in_len ? static_cast<float>(src[idx]) : 0.0f;
    }
    // pair_stride is even and the scratch is 16-byte aligned
    *reinterpret_cast<float4*>(pairs + row * pair_stride + u) = make_float4(v[0], v[2], v[1], v[3]);
}

// ------------------------------------------------------------------------------------------------
// PTX helpers: mbarrier, 1-D bulk copy (TMA), packed fp32 add
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p)
{
    return static_cast<unsigned>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_lane0(unsigned bar, int lane)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.eq.s32 p, %1, 0;\n"
        "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n"
        "}\n" ::"r"(bar), "r"(lane) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// producer side: the staging thread shares its scheduler with two consumer warps, so it must not
// spin: try_wait with a suspend-time hint parks the thread in hardware between polls
__device__ __forceinline__ void mbar_wait_backoff(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@!p bra WAIT_%=;\n"
        "}\n" ::"r"(bar), "r"(parity), "r"(20000u) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
#include "window_rows.inc"

// ------------------------------------------------------------------------------------------------
// 2. window kernel
// ------------------------------------------------------------------------------------------------

// the rows in mask (bit j-1 = row j) move their accumulators up one slot; lane 0 gets a fresh one
template <int T, int D> __device__ __forceinline__ void shift_rows(u64 (&acc)[D][T], unsigned mask, int lane)
{
#pragma unroll
    for (int j = 1; j < D; ++j) {
        if (mask & (1u << (j - 1))) {
            const u64 carry = __shfl_up_sync(0xffffffffu, acc[j][T - 1], 1);
            shift_row(acc[j], lane ? carry : 0ull);
        }
    }
}

template <int T> __device__ __forceinline__ void load_window(u64 (&w)[T + 1], const unsigned char* p)
{
    const u64* q = reinterpret_cast<const u64*>(p);
#pragma unroll
    for (int k = 0; k <= T; ++k)
        w[k] = q[k];
}

// band 0 stores; later bands add with a fire-and-forget reduction (one per cell and launch, launches
// are stream-ordered, so the fp32 result does not depend on scheduling)
__device__ __forceinline__ void put(float* p, float v, bool first)
{
    if (first)
        *p = v;
    else
        asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}
// int32 output: the fp32 partial sums are exact integers (nchans * 255 < 2^24)
__device__ __forceinline__ void put(int32_t* p, float v, bool first)
{
    const int iv = __float2int_rn(v);
    if (first)
        *p = iv;
    else
        asm volatile("red.global.add.s32 [%0], %1;" ::"l"(p), "r"(iv) : "memory");
}

// smem layout: [nst] full barriers | [nst] empty barriers | nst stages of { 128-byte header, kWinCh
//              channel slots }; the flush's transpose scratch [NCW][W] u64 overlays the stages
template <int T, int G, int NT, int D, typename OutT>
__global__ void __launch_bounds__((G * NT + 4) * 32, (G * NT == 4 ? 2 : 1))
    window_kernel(const WindowArgs a, const int c_begin, const int c_end, const int band, const int stage0,
                  const int nst, const int slot_bytes)
{
    constexpr int W = 32 * T, NCW = G * NT, RB = D * G;
    // registers per consumer thread once the producer warp group has released its share
    // (blocks of 4 consumer warps run two to an SM and share the register file)
    constexpr int kPool = ((NCW == 4 ? 32768 : 65536) - 4 * 32 * 24) / (NCW * 32) / 8 * 8;
    constexpr int kConsRegs = kPool > 240 ? 240 : kPool;
    static_assert(NCW % 4 == 0, "setmaxnreg works on groups of four warps");
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // Block order: groups of a.dm_group DM tiles; inside a group all time tiles, DM tile fastest.
    // The blocks in flight then read neighbouring delays of a few time tiles: the wave's footprint in
    // the pair buffer fits L2 (DM-fastest over ALL tiles reads a max_delay-wide range per time tile).
    const int beam = blockIdx.z;
    int ty, tt;
    {
        const int lin = blockIdx.x, per_group = a.dm_group * a.ntile_t;
        const int grp = lin / per_group, r = lin - grp * per_group;
        const int g0 = grp * a.dm_group;
        const int gsz = a.ntile_dm - g0 < a.dm_group ? a.ntile_dm - g0 : a.dm_group;  // last group may be short
        tt = r / gsz;
        ty = g0 + r - tt * gsz;
    }
    const int64_t T0 = static_cast<int64_t>(tt) * 2 * NT * a.H;

    const unsigned bar_full = smem_u32(smem);
    const unsigned bar_empty = bar_full + 8u * nst;
    // the flush's transpose scratch [NCW][W] u64 reuses the ring once every consumer has left the loop
    const int stages_off = (16 * nst + 127) & ~127;
    const int tr_off = stages_off;
    const int stage_bytes = kWinHdrWords * 4 + kWinCh * slot_bytes;
    unsigned char* stages = smem + stages_off;

    if (tid == 0) {
        for (int s = 0; s < nst; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, NCW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nch = c_end - c_begin;
    const int nstage = (nch + kWinCh - 1) / kWinCh;
    const int stage_total = a.stage_total;

    if (warp >= NCW) {
        // ---- producer warp group: gives its registers to the consumers; one thread stages kWinCh
        // channels per barrier (padding channels and the extra last stage get zeros)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        {
            // the four warps of the group take the stages in turn (stage s belongs to warp s % 4), so
            // the staging work is spread over the four schedulers instead of loading the one that also
            // runs consumer warps 0, 4, 8
            const int pw = warp - NCW;
            const int32_t* meta = a.meta + (static_cast<int64_t>(ty) * a.nchans + c_begin) * kWinMetaWords;
            const int32_t* hdr = a.hdr + (static_cast<int64_t>(ty) * stage_total + stage0) * kWinHdrWords;
            const float2* prow = static_cast<const float2*>(a.pairs) +
                                 (static_cast<int64_t>(beam) * a.nchans + c_begin) * a.pair_stride + T0;
            const int64_t pair_stride = a.pair_stride;
            const int zlen = ((NT - 1) * a.H + W + 2 + 1) & ~1;  // pairs a padding channel must provide
            for (int s = pw; s < nstage; s += 4) {
                const int ring = s % nst, lap = s / nst;
                // lanes 0 .. kWinCh-1: (base, len) of this stage's channels
                const int k = s * kWinCh + lane;
                int pb = 0, pl = -1;
                if (lane < kWinCh && k < nch) {
                    pb = __ldg(meta + static_cast<int64_t>(k) * kWinMetaWords);
                    pl = __ldg(meta + static_cast<int64_t>(k) * kWinMetaWords + 1);
                }
                int base[kWinCh], len[kWinCh];
#pragma unroll
                for (int ch = 0; ch < kWinCh; ++ch) {
                    base[ch] = __shfl_sync(0xffffffffu, pb, ch);
                    len[ch] = __shfl_sync(0xffffffffu, pl, ch);
                }
                if (lane == 0) {
                    if (lap > 0)
                        mbar_wait_backoff(bar_empty + 8u * ring, (lap - 1) & 1);
                    const unsigned dst = smem_u32(stages) + ring * stage_bytes;
                    const unsigned fb = bar_full + 8u * ring;
                    unsigned bytes = kWinHdrWords * 4;
#pragma unroll
                    for (int ch = 0; ch < kWinCh; ++ch)
                        bytes += (len[ch] < 0 ? zlen : len[ch]) * 8;
                    mbar_expect_tx(fb, bytes);
                    bulk_g2s(dst, hdr + static_cast<int64_t>(s) * kWinHdrWords, kWinHdrWords * 4, fb);
#pragma unroll
                    for (int ch = 0; ch < kWinCh; ++ch) {
                        const unsigned d = dst + kWinHdrWords * 4 + ch * slot_bytes;
                        if (len[ch] < 0)
                            bulk_g2s(d, a.zeros, zlen * 8, fb);
                        else
                            bulk_g2s(d, prow + static_cast<int64_t>(s * kWinCh + ch) * pair_stride + base[ch],
                                     len[ch] * 8, fb);
                    }
                }
                __syncwarp();
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kConsRegs));

    // ---- consumers ------------------------------------------------------------------------------------
    // the warp index through a reduction: ptxas then knows it (and every shared-memory word loaded
    // from an address built from it) is warp-uniform, so the row branches become BRA.U
    const int uwarp = __reduce_or_sync(0xffffffffu, warp);
    const int g = uwarp / NT, wt = uwarp % NT;
    int lane_pinned;  // volatile: not rematerialised (S2R) inside the channel loop
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane_pinned));
    u64 acc[D][T];
#pragma unroll
    for (int j = 0; j < D; ++j)
#pragma unroll
        for (int i = 0; i < T; ++i)
            acc[j][i] = 0ull;

    // per stage: wait for the NEXT stage and read its four metadata words with one LDS.128, then
    // add the four channels of this stage; the window of channel k+1 is loaded while channel k is
    // added (wa / wb alternate).
    const unsigned lane_off = kWinHdrWords * 4 + (wt * a.H + lane_pinned * T) * 8;  // bytes from the slot start
    auto shifts = [&](unsigned m) {
        const unsigned sm = (m >> 7) & 0x3fffu;
        shift_rows<T, D>(acc, sm & 127u, lane_pinned);
        if (sm >> 7)
            shift_rows<T, D>(acc, sm >> 7, lane_pinned);
    };
    auto adds = [&](u64(&w)[T + 1], unsigned m) { rows7(acc, w, m); };
    // Stage loop around a channel loop with a single copy of the add block (ptxas permutes the
    // accumulator registers between copies otherwise).  The bookkeeping that runs once per channel
    // is kept to the window address and the rotation of the stage's four metadata words: every
    // uniform-datapath instruction in that chain costs its full latency with two warps per scheduler.
    // The next stage's barrier wait and metadata load sit between two stages, outside the channel
    // loop: three more bookkeeping instructions per channel cost more than the exposed latency.
    u64 w[T + 1];
    const unsigned hdr_off = 16 * g;
    mbar_wait(bar_full, 0);
    uint4 mq = *reinterpret_cast<const uint4*>(stages + hdr_off);
    const unsigned char* sbase = stages;
    int ring = 0;
    unsigned par = 0;
#pragma unroll 1
    for (int s = 0; s < nstage; ++s) {
        int ring_n = ring + 1;
        unsigned par_n = par;
        if (ring_n == nst) {
            ring_n = 0;
            par_n ^= 1u;
        }
        const unsigned char* sbase_n = stages + ring_n * stage_bytes;
        const unsigned char* sp = sbase + lane_off;
        unsigned m = mq.x;
        if (((mq.x | mq.y) | (mq.z | mq.w)) & 0x1fff80u) {
            // a row shift somewhere in this stage (about a third of the stages)
#pragma unroll 1
            for (int ch = 0; ch < kWinCh; ++ch) {
                load_window<T>(w, sp + (m >> 21) * 8);
                if (m & 0x1fff80u)
                    shifts(m);
                adds(w, m);
                sp += slot_bytes;
                m = mq.y;
                mq.y = mq.z;
                mq.z = mq.w;
            }
        } else {
#pragma unroll 1
            for (int ch = 0; ch < kWinCh; ++ch) {
                load_window<T>(w, sp + (m >> 21) * 8);
                adds(w, m);
                sp += slot_bytes;
                m = mq.y;
                mq.y = mq.z;
                mq.z = mq.w;
            }
        }
        __syncwarp();
        mbar_arrive_lane0(bar_empty + 8u * ring, lane_pinned);
        if (s + 1 < nstage) {
            mbar_wait(bar_full + 8u * ring_n, par_n);
            mq = *reinterpret_cast<const uint4*>(sbase_n + hdr_off);
        }
        ring = ring_n;
        par = par_n;
        sbase = sbase_n;
    }

    // ---- flush: slot p of row r is output time T0 + wt*H + (p - kfinal_r) - theta_r ---------------------
    // The rows go through a shared-memory transpose (overlaying the ring) in passes of `rpp` rows with
    // their own regions: all rows of a pass are written, ONE __syncwarp, then read back and stored.
    // (A sync per row waits for the previous row's global stores every time: 3.5 % of the kernel.)
    asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");  // consumers only: the ring is free now
    const int rpp = a.flush_rows;
    const int32_t* kfp = a.kfinal + (static_cast<int64_t>(ty) * a.nband + band) * RB + g * D;
    const int32_t* thp = a.theta + (static_cast<int64_t>(ty) * a.nband + band) * RB + g * D;
    const int kf_lane = __ldg(kfp + lane_pinned % D), th_lane = __ldg(thp + lane_pinned % D);
    u64* tr = reinterpret_cast<u64*>(smem + tr_off) + static_cast<size_t>(warp) * rpp * W;
    const bool first = band == 0;
    OutT* out = static_cast<OutT*>(a.out) + static_cast<int64_t>(beam) * a.ndm * a.out_stride;
    const int H = a.H;
    const int64_t hp = static_cast<int64_t>(NT) * H;
    const int64_t tw = T0 + wt * H;
    // every sample of this warp's two output ranges inside [0, n_out): no bounds tests
    const bool inside = tw - a.theta_max >= 0 && tw + hp + H <= a.n_out;
    int pass0 = 0;  // first row of the current pass
#pragma unroll
    for (int j = 0; j < D; ++j) {
        u64* trj = tr + (j - pass0) * W;
#pragma unroll
        for (int i = 0; i < T; ++i)
            trj[lane_pinned * T + i] = acc[j][i];
        if (j + 1 - pass0 < rpp && j + 1 < D)
            continue;
        __syncwarp();
#pragma unroll 1
        for (int jj = pass0; jj <= j; ++jj) {
            const int d = ty * RB + g * D + jj;
            const int kf = __shfl_sync(0xffffffffu, kf_lane, jj), th = __shfl_sync(0xffffffffu, th_lane, jj);
            if (d >= a.ndm)
                continue;
            const u64* trr = tr + (jj - pass0) * W + kf;
            OutT* o = out + static_cast<int64_t>(d) * a.out_stride + (tw - th);
            u64 v[T];
#pragma unroll
            for (int k = 0; k < T; ++k) {
                const int q = lane_pinned + 32 * k;
                v[k] = q < H ? trr[q] : 0ull;
            }
            if (inside) {
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    const int q = lane_pinned + 32 * k;
                    if (q < H) {
                        put(o + q, __uint_as_float(static_cast<unsigned>(v[k])), first);
                        put(o + q + hp, __uint_as_float(static_cast<unsigned>(v[k] >> 32)), first);
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    const int q = lane_pinned + 32 * k;
                    const int64_t t = tw - th + q;
                    if (q < H && t >= 0 && t < a.n_out)
                        put(o + q, __uint_as_float(static_cast<unsigned>(v[k])), first);
                    if (q < H && t + hp >= 0 && t + hp < a.n_out)
                        put(o + q + hp, __uint_as_float(static_cast<unsigned>(v[k] >> 32)), first);
                }
            }
        }
        pass0 = j + 1;
        if (j + 1 < D)
            __syncwarp();  // the regions are rewritten by the next pass
    }
}

// ------------------------------------------------------------------------------------------------
// launcher
// ------------------------------------------------------------------------------------------------
// number of pipeline stages that fit into shared memory (0: the kernel cannot run)
static int window_ring(const WindowGeom& g, int lmax, int* slot_bytes)
{
    const int sb = (lmax * 8 + 127) & ~127;
    const int fixed = 256 + 256;  // barriers; the transpose scratch aliases the ring (3 stages > [NCW][W] u64)
    const int budget = (g.G * g.NT == 4 ? 113 : 227) * 1024 - fixed;
    const int stage_bytes = kWinHdrWords * 4 + kWinCh * sb;
    int nst = budget / stage_bytes;
    if (nst > 8)
        nst = 8;
    *slot_bytes = sb;
    if (nst * stage_bytes < g.G * g.NT * g.W() * 8)
        return 0;
    return nst >= 3 ? nst : 0;
}

bool window_fits_smem(const WindowPlan& wp)
{
    int sb;
    return wp.ok && window_ring(wp.geom, wp.lmax, &sb) > 0;
}

template <int T, int G, int NT, int D, typename OutT>
static int launch_bands(const WindowArgs& a, cudaStream_t st, int* launches)
{
    int slot_bytes = 0;
    const int nst = window_ring(a.geom, a.lmax, &slot_bytes);
    if (nst == 0)
        return static_cast<int>(cudaErrorInvalidConfiguration);
    const int stages_off = (16 * nst + 127) & ~127;
    const size_t ring = static_cast<size_t>(nst) * (kWinHdrWords * 4 + kWinCh * slot_bytes);
    const size_t smem = static_cast<size_t>(stages_off) + ring;
    WindowArgs a2 = a;  // rows per flush pass: as many [NCW][W] u64 transposes as the ring holds
    a2.flush_rows = static_cast<int>(ring / (static_cast<size_t>(G) * NT * 32 * T * 8));
    a2.flush_rows = a2.flush_rows > D ? D : a2.flush_rows < 1 ? 1 : a2.flush_rows;
    if (const char* e = std::getenv("DEDISP_WINDOW_FLUSH_ROWS"))  // development override (fewer rows per pass)
        a2.flush_rows = std::atoi(e) >= 1 && std::atoi(e) < a2.flush_rows ? std::atoi(e) : a2.flush_rows;
    cudaError_t e = cudaFuncSetAttribute(window_kernel<T, G, NT, D, OutT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess)
        return static_cast<int>(e);
    dim3 grid(static_cast<unsigned>(a.ntile_dm) * a.ntile_t, 1, a.nbeams);
    for (int b = 0; b < a.nband; ++b) {
        window_kernel<T, G, NT, D, OutT><<<grid, (G * NT + 4) * 32, smem, st>>>(a2, a.band[b], a.band[b + 1], b,
                                                                              a.stage0[b], nst, slot_bytes);
        ++*launches;
        e = cudaGetLastError();
        if (e != cudaSuccess)
            return static_cast<int>(e);
    }
    return 0;
}

template <typename OutT> static int launch_geom(const WindowArgs& a, cudaStream_t st, int* launches)
{
    const WindowGeom& g = a.geom;
#define DEDISP_GEOM(t, gg, nt, dd) \
    if (g.T == t && g.G == gg && g.NT == nt && g.D == dd) \
        return launch_bands<t, gg, nt, dd, OutT>(a, st, launches);
    DEDISP_GEOM(15, 6, 2, 4)
    DEDISP_GEOM(15, 4, 3, 4)
    DEDISP_GEOM(21, 4, 1, 4)
    DEDISP_GEOM(21, 8, 1, 4)
    DEDISP_GEOM(17, 4, 1, 5)
    DEDISP_GEOM(15, 4, 1, 6)
    DEDISP_GEOM(11, 8, 1, 8)
#undef DEDISP_GEOM
    return static_cast<int>(cudaErrorInvalidConfiguration);
}

int launch_window(const WindowArgs& a, Elem in_t, void* stream, int* launches)
{
    if (a.n_out <= 0 || a.ndm <= 0)
        return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    dim3 pgrid(static_cast<unsigned>((a.pair_stride / 2 + 255) / 256), a.nchans, a.nbeams);
    float2* pairs = static_cast<float2*>(a.pairs);
    const int hp = a.geom.NT * a.H;
    if (in_t == Elem::F32)
        pairify_kernel<float><<<pgrid, 256, 0, st>>>(static_cast<const float*>(a.in), pairs, a.in_stride,
                                                     a.pair_stride, a.in_len, hp);
    else
        pairify_kernel<uint8_t><<<pgrid, 256, 0, st>>>(static_cast<const uint8_t*>(a.in), pairs, a.in_stride,
                                                       a.pair_stride, a.in_len, hp);
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess)
        return static_cast<int>(e);
    if (a.ev0)
        cudaEventRecord(static_cast<cudaEvent_t>(a.ev0), st);
    const int rc = in_t == Elem::F32 ? launch_geom<float>(a, st, launches) : launch_geom<int32_t>(a, st, launches);
    if (a.ev1)
        cudaEventRecord(static_cast<cudaEvent_t>(a.ev1), st);
    return rc;
}

}  // namespace dedisp
