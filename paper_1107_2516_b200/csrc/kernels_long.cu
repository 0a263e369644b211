// Long-tile gather-and-add kernel for sm_100a: subband stage 1 and stage 2 (
// PAPER.md:129-135, :157-165) and brute-force tables the register-window kernel cannot take.
//
//   out[d][t] = sum_c in[c][t + shift(d,c)]      for one dedisp::Problem
//
// Neighbouring rows of these problems are far apart in delay (stage 1 of cfg 4: 74-141 samples per
// coarse DM step and channel), so no register window can be shared between rows and every add costs
// one shared-memory word: the kernel is bound by the 128 B/clk/SM shared-memory pipe (32 adds/clk/SM,
// a quarter of the FP32 add pipe).  What is left to win is the traffic BEHIND shared memory: a block
// stages, per channel, the union of the sample ranges its rows need, [t0 + min_j s_j, t0 + L + max_j s_j),
// and that union is only well used when the tile is long compared with the spread of the rows'
// delays.  Hence the shape: R = 16 rows (one consumer warp each) x L = 32*TT = 2048 samples, the
// accumulators of a row in the registers of its warp (lane owns samples lane + 32 i: conflict-free for
// any delay), and four producer warps (one per scheduler, channels in turn) that compute the union per channel and stages it with a 1-D TMA
// bulk copy (cp.async.bulk + mbarrier) into a ring of shared-memory slots.  On cfg 4's stage 1 a
// staged word then serves 16*2048/(2048 + 16*~70) ~ 10 adds instead of 1.7 in the 32 x 256 tile of
// direct_kernel (which drew 8.4 TB/s from L2 and was bound by that).
#include <cuda_runtime.h>

#include <climits>

#include "dedisp_internal.h"

namespace dedisp {

namespace {

template <typename T> struct AccOfL { using type = int32_t; };
template <> struct AccOfL<float> { using type = float; };

__device__ __forceinline__ unsigned smem_addr(const void* p)
{
    return static_cast<unsigned>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void bar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void bar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bar_wait(unsigned bar, unsigned parity)
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
__device__ __forceinline__ void tma_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

constexpr int kLongProducers = 4;  // staging warps, one per scheduler: channel c belongs to warp c % 4

// shared memory: full[nslot], empty[nslot] (mbarriers) | offs[nslot][R] | slots[nslot][cap] InT
__host__ __device__ inline int long_hdr_bytes(int nslot, int R) { return (16 * nslot + 4 * R * nslot + 127) & ~127; }

template <typename InT, int R, int TT>
__global__ void __launch_bounds__((R + kLongProducers) * 32, 1) long_kernel(const Problem p, const int cap, const int nslot, const int nrt)
{
    using AccT = typename AccOfL<InT>::type;
    constexpr int L = 32 * TT;
    constexpr int VEC = 16 / static_cast<int>(sizeof(InT));
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rt = blockIdx.x % nrt;
    const int64_t t0 = static_cast<int64_t>(blockIdx.x / nrt) * L;
    const int d0 = rt * R;
    const int b1 = blockIdx.y, b0 = blockIdx.z;

    // rows of this tile that still have outputs at t0
    unsigned act = 0;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        if (d0 + j < p.ndm) {
            const int64_t len = p.row_extra ? p.n_base + p.row_extra[b1 * p.row_extra_b1_stride + d0 + j] : p.n_out;
            if (t0 < len)
                act |= 1u << j;
        }
    }
    if (act == 0)
        return;

    const unsigned bar_full = smem_addr(smem), bar_empty = bar_full + 8u * nslot;
    int* offs = reinterpret_cast<int*>(smem + 16 * nslot);
    const int hdr = long_hdr_bytes(nslot, R);
    const int slot_bytes = (cap * static_cast<int>(sizeof(InT)) + 127) & ~127;
    if (tid == 0) {
        for (int s = 0; s < nslot; ++s) {
            bar_init(bar_full + 8u * s, 1);
            bar_init(bar_empty + 8u * s, __popc(act));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= R) {
        // ---- producers: per channel the union of the active rows' sample ranges, one bulk copy.  The
        // staging work (16 shuffles and a min/max per channel) is spread over four warps, one per
        // scheduler: a single producer warp made its scheduler (which also runs four consumer warps)
        // the slowest and gated the ring.
        const int pw = warp - R;
        const InT* in = static_cast<const InT*>(p.in) + b0 * p.in_b0_stride + b1 * p.in_b1_stride;
        const int32_t* sh = p.shift + b1 * p.shift_b1_stride;
        for (int c0 = 0; c0 < p.nchans; c0 += 32) {
            int sv[R];  // lane l: shift(d0 + j, c0 + l)
#pragma unroll
            for (int j = 0; j < R; ++j)
                sv[j] = ((act >> j) & 1u) && c0 + lane < p.nchans
                            ? __ldg(sh + static_cast<int64_t>(d0 + j) * p.shift_dm_stride + c0 + lane)
                            : 0;
            const int nc = p.nchans - c0 < 32 ? p.nchans - c0 : 32;
            for (int i = pw; i < nc; i += kLongProducers) {
                const int c = c0 + i;
                const int ring = c % nslot, lap = c / nslot;
                int mn = INT_MAX, mx = 0, mine = 0;
#pragma unroll
                for (int j = 0; j < R; ++j) {
                    const int v = __shfl_sync(0xffffffffu, sv[j], i);
                    if ((act >> j) & 1u) {
                        mn = v < mn ? v : mn;
                        mx = v > mx ? v : mx;
                    }
                    if (lane == j)
                        mine = v;
                }
                const long long g = (t0 + mn) & ~static_cast<long long>(VEC - 1);
                long long end = t0 + L + mx;
                if (end > p.in_len)
                    end = p.in_len;
                const int nv = end > g ? static_cast<int>((end - g + VEC - 1) / VEC) : 0;
                if (lap > 0)
                    bar_wait(bar_empty + 8u * ring, (lap - 1) & 1);
                if (lane < R)
                    offs[ring * R + lane] = static_cast<int>(t0 + mine - g);
                __syncwarp();
                if (lane == 0) {
                    const unsigned fb = bar_full + 8u * ring;
                    if (nv > 0) {
                        bar_expect_tx(fb, static_cast<unsigned>(nv) * 16u);
                        tma_g2s(smem_addr(smem + hdr) + ring * slot_bytes,
                                in + static_cast<int64_t>(c) * p.in_chan_stride + g,
                                static_cast<unsigned>(nv) * 16u, fb);
                    } else {
                        bar_arrive(fb);
                    }
                }
            }
        }
        return;
    }

    // ---- consumers: warp j owns row d0 + j, lane owns samples t0 + lane + 32 i
    if (!((act >> warp) & 1u))
        return;
    AccT acc[TT];
#pragma unroll
    for (int i = 0; i < TT; ++i)
        acc[i] = 0;
    int ring = 0;
    unsigned par = 0;
#pragma unroll 1
    for (int c = 0; c < p.nchans; ++c) {
        bar_wait(bar_full + 8u * ring, par);
        const int off = offs[ring * R + warp];
        const InT* q = reinterpret_cast<const InT*>(smem + hdr + ring * slot_bytes) + off + lane;
#pragma unroll
        for (int i = 0; i < TT; ++i)
            acc[i] += static_cast<AccT>(q[32 * i]);
        __syncwarp();
        if (lane == 0)
            bar_arrive(bar_empty + 8u * ring);
        if (++ring == nslot) {
            ring = 0;
            par ^= 1u;
        }
    }

    const int d = d0 + warp;
    const int64_t len = p.row_extra ? p.n_base + p.row_extra[b1 * p.row_extra_b1_stride + d] : p.n_out;
    AccT* o = static_cast<AccT*>(p.out) + b0 * p.out_b0_stride + b1 * p.out_b1_stride +
              static_cast<int64_t>(d) * p.out_dm_stride + t0 + lane;
    if (t0 + L <= len && !p.accumulate) {
#pragma unroll
        for (int i = 0; i < TT; ++i)
            o[32 * i] = acc[i];
    } else {
#pragma unroll
        for (int i = 0; i < TT; ++i)
            if (t0 + lane + 32 * i < len)
                o[32 * i] = p.accumulate ? o[32 * i] + acc[i] : acc[i];
    }
}

template <typename InT, int R, int TT>
int launch_long_t(const Problem& p, int spread, cudaStream_t st)
{
    constexpr int L = 32 * TT;
    constexpr int VEC = 16 / static_cast<int>(sizeof(InT));
    long long cap = static_cast<long long>(L) + spread + 2 * VEC;
    cap = (cap + VEC - 1) / VEC * VEC;
    const long long slot_bytes = (cap * static_cast<long long>(sizeof(InT)) + 127) & ~127LL;
    int nslot = 8;
    while (nslot > 1 && long_hdr_bytes(nslot, R) + nslot * slot_bytes > 220 * 1024)
        --nslot;
    // Four producer warps take the channels in turn and wait on a slot's empty barrier by parity only:
    // a warp is ordered behind channel c - 4 - nslot, the parity test needs channel c - 2 * nslot
    // consumed, which holds from four slots on (with three, a warp can lap the consumers).
    if (nslot < 4 || p.nb1 > 65535 || p.nb0 > 65535)
        return -1;
    const int nrt = (p.ndm + R - 1) / R;
    const long long ntt = (p.n_out + L - 1) / L;
    if (ntt * nrt > INT_MAX)
        return -1;
    const size_t smem = static_cast<size_t>(long_hdr_bytes(nslot, R)) + static_cast<size_t>(nslot) * slot_bytes;
    cudaError_t e = cudaFuncSetAttribute(long_kernel<InT, R, TT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess)
        return static_cast<int>(e);
    dim3 grid(static_cast<unsigned>(ntt * nrt), p.nb1, p.nb0);
    long_kernel<InT, R, TT><<<grid, (R + kLongProducers) * 32, smem, st>>>(p, static_cast<int>(cap), nslot, nrt);
    return static_cast<int>(cudaGetLastError());
}

template <typename InT> int launch_long_e(const Problem& p, int spread, cudaStream_t st)
{
    return launch_long_t<InT, 16, 64>(p, spread, st);
}

}  // namespace

// spread16: max over tiles of 16 rows and channels of (max shift - min shift).  Returns -1 when the
// staged rows do not fit shared memory (the caller falls back to the direct kernel).
int launch_long(const Problem& p, Elem in_t, int spread16, void* stream, int* launches)
{
    if (p.n_out <= 0 || p.ndm <= 0)
        return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc;
    switch (in_t) {
    case Elem::F32: rc = launch_long_e<float>(p, spread16, st); break;
    case Elem::U8: rc = launch_long_e<uint8_t>(p, spread16, st); break;
    default: rc = launch_long_e<int32_t>(p, spread16, st); break;
    }
    if (rc != -1)
        ++*launches;
    return rc;
}

}  // namespace dedisp
