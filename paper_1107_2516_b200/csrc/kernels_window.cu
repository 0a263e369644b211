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
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ u64 add2(u64 a, u64 b)
{
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

#include "window_rows.inc"

// ------------------------------------------------------------------------------------------------
// 2. window kernel
// ------------------------------------------------------------------------------------------------
constexpr int kSlotHdr = kWinMetaWords * 4;  // bytes of metadata in front of a staged segment

// the rows in mask (bit j-1 = row j) move their accumulators up one slot; lane 0 gets a fresh one
template <int T> __device__ __forceinline__ void shift_rows(u64 (&acc)[kWinD][T], unsigned mask, int lane)
{
#pragma unroll
    for (int j = 1; j < kWinD; ++j) {
        if (mask & (1u << (j - 1))) {
            const u64 carry = __shfl_up_sync(0xffffffffu, acc[j][T - 1], 1);
#pragma unroll
            for (int i = T - 1; i > 0; --i)
                acc[j][i] = acc[j][i - 1];
            acc[j][0] = lane ? carry : 0ull;
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

// smem layout: [nslot] full barriers | [nslot] empty barriers | transpose scratch [NCW][W] u64 | slots
template <int T, int G, int NT, typename OutT>
__global__ void __launch_bounds__(G * NT * 32, 1)
    window_kernel(const WindowArgs a, const int c_begin, const int c_end, const int band, const int nslot_log2,
                  const int slot_bytes)
{
    constexpr int W = 32 * T, NCW = G * NT, RB = kWinD * G;
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ty = blockIdx.x, beam = blockIdx.z;
    const int64_t T0 = static_cast<int64_t>(blockIdx.y) * 2 * NT * a.H;
    const int nslot = 1 << nslot_log2;

    const unsigned bar_full = smem_u32(smem);
    const unsigned bar_empty = bar_full + 8u * nslot;
    const int tr_off = (16 * nslot + 127) & ~127;
    const int slots_off = (tr_off + NCW * W * 8 + 127) & ~127;
    unsigned char* slots = smem + slots_off;

    if (tid == 0) {
        for (int s = 0; s < nslot; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, NCW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nch = c_end - c_begin;
    const int32_t* meta = a.meta + (static_cast<int64_t>(ty) * a.nchans + c_begin) * kWinMetaWords;

    // ---- producer duty (thread 0): stage channel i into slot i % nslot, kLead channels ahead ------------
    const float2* prow = static_cast<const float2*>(a.pairs) +
                         (static_cast<int64_t>(beam) * a.nchans + c_begin) * a.pair_stride + T0;
    const int64_t pair_stride = a.pair_stride;
    // warp 0 keeps (base, len) of 32 channels in registers (lane L: channel 32*pq + L), loaded one
    // batch ahead of use so that the staging thread never waits for a global load
    int pb = 0, pl = 0, pbn = 0, pln = 0;
    auto fetch_meta = [&](int q, int& b_, int& l_) {
        const int k = q * 32 + lane;
        if (k < nch) {
            b_ = __ldg(meta + static_cast<int64_t>(k) * kWinMetaWords);
            l_ = __ldg(meta + static_cast<int64_t>(k) * kWinMetaWords + 1);
        }
    };
    auto produce = [&](int i) {  // called by all lanes of warp 0
        if ((i & 31) == 0 && i > 0) {
            pb = pbn;
            pl = pln;
        }
        if ((i & 31) == 0)
            fetch_meta((i >> 5) + 1, pbn, pln);
        const int base = __shfl_sync(0xffffffffu, pb, i & 31), len = __shfl_sync(0xffffffffu, pl, i & 31);
        if (lane == 0) {
            const int s = i & (nslot - 1), lap = i >> nslot_log2;
            if (lap > 0)
                mbar_wait(bar_empty + 8u * s, (lap - 1) & 1);
            const int32_t* m = meta + static_cast<int64_t>(i) * kWinMetaWords;
            const unsigned dst = smem_u32(slots + static_cast<size_t>(s) * slot_bytes);
            const unsigned fb = bar_full + 8u * s;
            mbar_expect_tx(fb, kSlotHdr + len * 8);
            bulk_g2s(dst, m, kSlotHdr, fb);
            bulk_g2s(dst + kSlotHdr, prow + static_cast<int64_t>(i) * pair_stride + base, len * 8, fb);
        }
        __syncwarp();
    };
    const int lead = nslot - 4;
    const bool producer = warp == 0;
    if (producer) {
        fetch_meta(0, pb, pl);
        for (int i = 0; i < lead && i < nch; ++i)
            produce(i);
    }

    // ---- consumers ------------------------------------------------------------------------------------
    const int g = warp / NT, wt = warp % NT;
    u64 acc[kWinD][T];
#pragma unroll
    for (int j = 0; j < kWinD; ++j)
#pragma unroll
        for (int i = 0; i < T; ++i)
            acc[j][i] = 0ull;

    const int lane_off = kSlotHdr + (wt * a.H + lane * T) * 8;  // bytes from the slot start
    auto slot_ptr = [&](int i) { return slots + static_cast<size_t>(i & (nslot - 1)) * slot_bytes; };
    auto wait_full = [&](int i) { mbar_wait(bar_full + 8u * (i & (nslot - 1)), (i >> nslot_log2) & 1); };
    auto slot_word = [&](int i) { return reinterpret_cast<const unsigned*>(slot_ptr(i))[2 + g]; };

    // software pipeline: channel i is added from w/m while the window of i+1 and the metadata of
    // i+2 are on their way
    u64 wa[T + 1], wb[T + 1];
    unsigned m = 0, mn = 0, mnn = 0;
    wait_full(0);
    m = slot_word(0);
    if (nch > 1) {
        wait_full(1);
        mn = slot_word(1);
    }
    load_window<T>(wa, slot_ptr(0) + lane_off + (m >> 21) * 8);

    auto step = [&](int i, u64(&w)[T + 1], u64(&wn)[T + 1]) {
        if (producer && i + lead < nch)
            produce(i + lead);
        if (i + 1 < nch)
            load_window<T>(wn, slot_ptr(i + 1) + lane_off + (mn >> 21) * 8);
        if (i + 2 < nch) {
            wait_full(i + 2);
            mnn = slot_word(i + 2);
        }
        const unsigned sm = (m >> 7) & 0x3fffu;
        if (sm) {
            shift_rows<T>(acc, sm & 127u, lane);
            if (sm >> 7)
                shift_rows<T>(acc, sm >> 7, lane);
        }
#pragma unroll
        for (int k = 0; k < T; ++k)
            acc[0][k] = add2(acc[0][k], w[k]);
        rows7(acc, w, m);
        __syncwarp();
        if (lane == 0)
            mbar_arrive(bar_empty + 8u * (i & (nslot - 1)));
        m = mn;
        mn = mnn;
    };
#pragma unroll 1
    for (int i = 0; i < nch; i += 2) {
        step(i, wa, wb);
        if (i + 1 < nch)
            step(i + 1, wb, wa);
    }

    // ---- flush: slot p of row r is output time T0 + wt*H + (p - kfinal_r) - theta_r ---------------------
    u64* tr = reinterpret_cast<u64*>(smem + tr_off) + warp * W;
    const bool first = band == 0;
    const int32_t* kfp = a.kfinal + (static_cast<int64_t>(ty) * a.nband + band) * RB + g * kWinD;
    const int32_t* thp = a.theta + (static_cast<int64_t>(ty) * a.nband + band) * RB + g * kWinD;
    OutT* out = static_cast<OutT*>(a.out) + static_cast<int64_t>(beam) * a.ndm * a.out_stride;
    const int64_t hp = static_cast<int64_t>(NT) * a.H;
#pragma unroll
    for (int j = 0; j < kWinD; ++j) {
        const int d = ty * RB + g * kWinD + j;
        __syncwarp();
#pragma unroll
        for (int i = 0; i < T; ++i)
            tr[lane * T + i] = acc[j][i];
        __syncwarp();
        if (d < a.ndm) {
            const int kf = __ldg(kfp + j), th = __ldg(thp + j);
            OutT* o = out + static_cast<int64_t>(d) * a.out_stride;
            for (int q = lane; q < a.H; q += 32) {
                const u64 v = tr[q + kf];
                const int64_t t = T0 + wt * a.H + q - th;
                if (t >= 0 && t < a.n_out)
                    put(o + t, __uint_as_float(static_cast<unsigned>(v)), first);
                if (t + hp >= 0 && t + hp < a.n_out)
                    put(o + t + hp, __uint_as_float(static_cast<unsigned>(v >> 32)), first);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// launcher
// ------------------------------------------------------------------------------------------------
static int window_ring(const WindowGeom& g, int lmax, int* slot_bytes, int* nslot_log2)
{
    const int sb = (kSlotHdr + lmax * 8 + 127) & ~127;
    const int fixed = 256 + g.G * g.NT * g.W() * 8 + 256;
    const int budget = 227 * 1024 - fixed;
    int lg = 4;  // at most 16 slots
    while (lg > 3 && (sb << lg) > budget)
        --lg;
    *slot_bytes = sb;
    *nslot_log2 = lg;
    return (sb << lg) <= budget ? (1 << lg) : 0;
}

bool window_fits_smem(const WindowPlan& wp)
{
    int sb, lg;
    return wp.ok && window_ring(wp.geom, wp.lmax, &sb, &lg) >= 8;
}

template <int T, int G, int NT, typename OutT>
static int launch_bands(const WindowArgs& a, cudaStream_t st, int* launches)
{
    int slot_bytes = 0, lg = 0;
    const int nslot = window_ring(a.geom, a.lmax, &slot_bytes, &lg);
    if (nslot < 8)
        return static_cast<int>(cudaErrorInvalidConfiguration);
    const int tr_off = (16 * nslot + 127) & ~127;
    const int slots_off = (tr_off + G * NT * 32 * T * 8 + 127) & ~127;
    const size_t smem = static_cast<size_t>(slots_off) + static_cast<size_t>(nslot) * slot_bytes;
    cudaError_t e = cudaFuncSetAttribute(window_kernel<T, G, NT, OutT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess)
        return static_cast<int>(e);
    dim3 grid(a.ntile_dm, a.ntile_t, a.nbeams);
    for (int b = 0; b < a.nband; ++b) {
        window_kernel<T, G, NT, OutT><<<grid, G * NT * 32, smem, st>>>(a, a.band[b], a.band[b + 1], b, lg,
                                                                              slot_bytes);
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
    if (g.T == 9 && g.G == 8 && g.NT == 1)
        return launch_bands<9, 8, 1, OutT>(a, st, launches);
    if (g.T == 5 && g.G == 8 && g.NT == 2)
        return launch_bands<5, 8, 2, OutT>(a, st, launches);
    if (g.T == 7 && g.G == 4 && g.NT == 3)
        return launch_bands<7, 4, 3, OutT>(a, st, launches);
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
    return in_t == Elem::F32 ? launch_geom<float>(a, st, launches) : launch_geom<int32_t>(a, st, launches);
}

}  // namespace dedisp
