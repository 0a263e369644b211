// Register-window brute-force kernel for sm_100a.
//
//   out[d][t] = sum_c in[c][t + shift(c,d)]
//
// Two launches per execute:
//  1. pairify_kernel: P[c][u] = (in[c][u], in[c][u+H]) as float2 (uint8 input is widened to fp32
//     here; sums of <= 2^24/255 bytes are exact in fp32).  Pairing two samples H apart that share
//     (c, d) and therefore the same shift lets the main kernel add two outputs per instruction
//     (add.f32x2 -> FADD2) from naturally aligned 64-bit registers, whatever the shift's parity.
//  2. window_kernel: one block = 32 DM rows x 2H output samples.  A thread keeps 8 rows x 10 pairs
//     of accumulators in registers for the whole channel loop; per channel it loads ONE window of
//     14 staged pairs (7 LDS.128) that feeds all 8 rows (row j starts 0..4 pairs into the window,
//     a warp-uniform 5-way branch selects the unrolled variant).  Rows keep up with the growing
//     delay difference between neighbouring DM trials by occasionally moving their accumulators up
//     one slot ("row shift", planned on the host: window_plan.cpp).  Channel segments are staged
//     into a ring of shared-memory slots by 1-D TMA bulk copies (cp.async.bulk + mbarrier) issued
//     by one thread, so the compute warps spend no instructions or registers on staging.
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
                                                      int64_t in_len, int H)
{
    const int64_t u = (static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x) * 2;
    if (u >= pair_stride)
        return;
    const int64_t row = static_cast<int64_t>(blockIdx.z) * gridDim.y + blockIdx.y;
    const InT* src = in + row * in_stride;
    float v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int64_t idx = u + (k & 1) + (k >> 1) * static_cast<int64_t>(H);
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
__device__ __forceinline__ void named_bar(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ------------------------------------------------------------------------------------------------
// 2. window kernel
// ------------------------------------------------------------------------------------------------
constexpr int kWinThreads = kWinNG * kWinNT * 32;  // 256
constexpr int kSlotHdr = 64;                       // bytes of metadata in front of a staged segment
constexpr int kLag = 4;                            // the producer refills the slot used kLag channels ago

template <int O> __device__ __forceinline__ void add_row(u64 (&acc)[kWinT], const u64 (&w)[kWinNW])
{
#pragma unroll
    for (int i = 0; i < kWinT; ++i)
        acc[i] = add2(acc[i], w[O + i]);
}

// smem layout: [nslot] full barriers | [nslot] empty barriers | mailbox [NG][D] u64 | slots
template <typename OutT>
__global__ void __launch_bounds__(kWinThreads, 1) window_kernel(const WindowArgs a, const int nslot,
                                                                 const int slot_bytes)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = warp / kWinNT, wt = warp % kWinNT;
    const int ty = blockIdx.x, beam = blockIdx.z;
    const int64_t tb0 = static_cast<int64_t>(blockIdx.y) * 2 * a.H;

    const unsigned bar_full = smem_u32(smem);
    const unsigned bar_empty = bar_full + 8u * nslot;
    u64* mailbox = reinterpret_cast<u64*>(smem + 16 * nslot);
    const int slots_off = (16 * nslot + kWinNG * kWinD * 8 + 127) & ~127;
    unsigned char* slots = smem + slots_off;

    if (tid == 0) {
        for (int s = 0; s < nslot; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, kWinNG * kWinNT);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int32_t* meta = a.meta + static_cast<int64_t>(ty) * a.nchans * kWinMetaWords;
    const float2* prow = static_cast<const float2*>(a.pairs) + static_cast<int64_t>(beam) * a.nchans * a.pair_stride + tb0;

    // producer state (warp 0, lane 0 only)
    const bool producer = tid == 0;
    int cp = 0;  // next channel to stage
    auto produce = [&](int c) {
        const int s = c % nslot;
        const int32_t* m = meta + static_cast<int64_t>(c) * kWinMetaWords;
        const int base = __ldg(m), len = __ldg(m + 1);
        const unsigned dst = smem_u32(slots + static_cast<size_t>(s) * slot_bytes);
        const unsigned fb = bar_full + 8u * s;
        mbar_expect_tx(fb, kWinMetaWords * 4 + len * 8);
        bulk_g2s(dst, m, kWinMetaWords * 4, fb);
        bulk_g2s(dst + kSlotHdr, prow + static_cast<int64_t>(c) * a.pair_stride + base, len * 8, fb);
    };
    if (producer) {
        const int n0 = min(nslot - kLag, a.nchans);
        for (; cp < n0; ++cp)
            produce(cp);
    }

    u64 acc[kWinD][kWinT];
#pragma unroll
    for (int j = 0; j < kWinD; ++j)
#pragma unroll
        for (int i = 0; i < kWinT; ++i)
            acc[j][i] = 0ull;

    const int p0 = (wt * 32 + lane) * kWinT;  // first slot of this thread

    for (int c = 0; c < a.nchans; ++c) {
        const int s = c % nslot;
        const unsigned ph = (c / nslot) & 1;
        if (producer && cp < a.nchans) {
            // slot of channel cp was last used by channel cp - nslot (<= c - kLag)
            if (cp >= nslot)
                mbar_wait(bar_empty + 8u * (cp % nslot), ((cp / nslot) - 1) & 1);
            produce(cp);
            ++cp;
        }
        mbar_wait(bar_full + 8u * s, ph);
        const unsigned char* slot = slots + static_cast<size_t>(s) * slot_bytes;
        const int wb = reinterpret_cast<const int*>(slot)[2 + g];
        const unsigned om = reinterpret_cast<const unsigned*>(slot)[6 + g];

        // row shifts (uniform over the two warps of this row group): the accumulators of the rows
        // in the mask move up one slot; the pair leaving lane 31 of the first warp reaches lane 0
        // of the second through the mailbox
        unsigned mask = om >> 24;
        if (mask) {
            const unsigned mask2 = (reinterpret_cast<const unsigned*>(slot)[10] >> (8 * g)) & 0xffu;
            for (int pass = 0; pass < 2 && mask; ++pass) {
                if (wt == 0 && lane == 31) {
#pragma unroll
                    for (int j = 1; j < kWinD; ++j)
                        if (mask & (1u << j))
                            mailbox[g * kWinD + j] = acc[j][kWinT - 1];
                }
                named_bar(1 + g, kWinNT * 32);
#pragma unroll
                for (int j = 1; j < kWinD; ++j) {
                    if (mask & (1u << j)) {
                        u64 carry = __shfl_up_sync(0xffffffffu, acc[j][kWinT - 1], 1);
                        if (lane == 0)
                            carry = wt ? mailbox[g * kWinD + j] : 0ull;
#pragma unroll
                        for (int i = kWinT - 1; i > 0; --i)
                            acc[j][i] = acc[j][i - 1];
                        acc[j][0] = carry;
                    }
                }
                named_bar(1 + g, kWinNT * 32);
                mask = mask2;
            }
        }

        u64 w[kWinNW];
        const ulonglong2* wp = reinterpret_cast<const ulonglong2*>(slot + kSlotHdr + static_cast<size_t>(p0 + wb) * 8);
#pragma unroll
        for (int k = 0; k < kWinNW / 2; ++k) {
            const ulonglong2 v = wp[k];
            w[2 * k] = v.x;
            w[2 * k + 1] = v.y;
        }
#pragma unroll
        for (int j = 0; j < kWinD; ++j) {
            switch ((om >> (3 * j)) & 7u) {
            case 0: add_row<0>(acc[j], w); break;
            case 1: add_row<1>(acc[j], w); break;
            case 2: add_row<2>(acc[j], w); break;
            case 3: add_row<3>(acc[j], w); break;
            default: add_row<4>(acc[j], w); break;
            }
        }
        __syncwarp();
        if (lane == 0)
            mbar_arrive(bar_empty + 8u * s);
    }

    // epilogue: slot p of row j is output time p - kfinal_j (valid in [0, H)), pair = (t, t + H)
    OutT* out = static_cast<OutT*>(a.out) + static_cast<int64_t>(beam) * a.ndm * a.out_stride;
#pragma unroll
    for (int j = 0; j < kWinD; ++j) {
        const int r = g * kWinD + j;
        const int d = ty * kWinDB + r;
        if (d >= a.ndm)
            continue;
        const int kf = __ldg(a.kfinal + ty * kWinDB + r);
        OutT* o = out + static_cast<int64_t>(d) * a.out_stride;
#pragma unroll
        for (int i = 0; i < kWinT; ++i) {
            const int tl = p0 + i - kf;
            if (tl < 0 || tl >= a.H)
                continue;
            const int64_t t = tb0 + tl;
            const float lo = __uint_as_float(static_cast<unsigned>(acc[j][i]));
            const float hi = __uint_as_float(static_cast<unsigned>(acc[j][i] >> 32));
            if (t < a.n_out)
                o[t] = static_cast<OutT>(lo);
            if (t + a.H < a.n_out)
                o[t + a.H] = static_cast<OutT>(hi);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// launcher
// ------------------------------------------------------------------------------------------------
static int window_ring(int lmax, int* slot_bytes)
{
    const int sb = (kSlotHdr + lmax * 8 + 127) & ~127;
    const int budget = 227 * 1024 - 1024;
    int nslot = budget / sb;
    if (nslot > 32)
        nslot = 32;
    *slot_bytes = sb;
    return nslot;
}

bool window_fits_smem(int lmax)
{
    int sb;
    return window_ring(lmax, &sb) >= 2 * kLag;
}

int launch_window(const WindowArgs& a, Elem in_t, void* stream, int* launches)
{
    if (a.n_out <= 0 || a.ndm <= 0)
        return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int slot_bytes = 0;
    const int nslot = window_ring(a.lmax, &slot_bytes);
    if (nslot < 2 * kLag)
        return static_cast<int>(cudaErrorInvalidConfiguration);
    const int slots_off = (16 * nslot + kWinNG * kWinD * 8 + 127) & ~127;
    const size_t smem = static_cast<size_t>(slots_off) + static_cast<size_t>(nslot) * slot_bytes;

    dim3 pgrid(static_cast<unsigned>((a.pair_stride / 2 + 255) / 256), a.nchans, a.nbeams);
    float2* pairs = static_cast<float2*>(a.pairs);
    if (in_t == Elem::F32)
        pairify_kernel<float><<<pgrid, 256, 0, st>>>(static_cast<const float*>(a.in), pairs, a.in_stride,
                                                     a.pair_stride, a.in_len, a.H);
    else
        pairify_kernel<uint8_t><<<pgrid, 256, 0, st>>>(static_cast<const uint8_t*>(a.in), pairs, a.in_stride,
                                                       a.pair_stride, a.in_len, a.H);
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess)
        return static_cast<int>(e);

    dim3 grid(a.ntile_dm, a.ntile_t, a.nbeams);
    if (in_t == Elem::F32) {
        e = cudaFuncSetAttribute(window_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 static_cast<int>(smem));
        if (e != cudaSuccess)
            return static_cast<int>(e);
        window_kernel<float><<<grid, kWinThreads, smem, st>>>(a, nslot, slot_bytes);
    } else {
        e = cudaFuncSetAttribute(window_kernel<int32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 static_cast<int>(smem));
        if (e != cudaSuccess)
            return static_cast<int>(e);
        window_kernel<int32_t><<<grid, kWinThreads, smem, st>>>(a, nslot, slot_bytes);
    }
    ++*launches;
    return static_cast<int>(cudaGetLastError());
}

}  // namespace dedisp
