// Naive and direct (shared-memory staged) gather-and-add kernels for sm_100a.
//
// Both compute   out[d][t] = sum_c in[c][t + shift(d,c)] for one
// dedisp::Problem; the same code serves brute force, subband stage 1 and stage 2
// through the strides in Problem.  The paper's own kernel (one thread per output sample, one row
// of the grid per DM, a global read per add) is what launch_naive does; it is
// kept for debugging and as the floor the other kernels are measured against.
#include <cuda_runtime.h>

#include "dedisp_internal.h"

namespace dedisp {

template <typename T> struct AccOf { using type = int32_t; };
template <> struct AccOf<float> { using type = float; };

// ------------------------------------------------------------------------------------------------
// naive: one thread per (d, t); consecutive threads take consecutive t (coalesced reads/writes).
// ------------------------------------------------------------------------------------------------
template <typename InT>
__global__ void __launch_bounds__(256) naive_kernel(Problem p)
{
    using AccT = typename AccOf<InT>::type;
    const int64_t t = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    const int b1 = blockIdx.z % p.nb1, b0 = blockIdx.z / p.nb1;
    const int64_t len = p.row_extra ? p.n_base + p.row_extra[b1 * p.row_extra_b1_stride + d] : p.n_out;
    if (t >= len)
        return;
    const InT* in = static_cast<const InT*>(p.in) + b0 * p.in_b0_stride + b1 * p.in_b1_stride;
    const int32_t* sh = p.shift + b1 * p.shift_b1_stride + d * p.shift_dm_stride;
    AccT acc = 0;
    for (int c = 0; c < p.nchans; ++c)
        acc += static_cast<AccT>(in[c * p.in_chan_stride + t + sh[c]]);
    AccT* o = static_cast<AccT*>(p.out) + b0 * p.out_b0_stride + b1 * p.out_b1_stride +
              d * p.out_dm_stride + t;
    *o = p.accumulate ? *o + acc : acc;
}

int launch_naive(const Problem& p, Elem in_t, void* stream, int* launches)
{
    if (p.n_out <= 0 || p.ndm <= 0)
        return 0;
    dim3 grid(static_cast<unsigned>((p.n_out + 255) / 256), p.ndm, p.nb0 * p.nb1);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (in_t) {
    case Elem::F32: naive_kernel<float><<<grid, 256, 0, st>>>(p); break;
    case Elem::U8: naive_kernel<uint8_t><<<grid, 256, 0, st>>>(p); break;
    case Elem::I32: naive_kernel<int32_t><<<grid, 256, 0, st>>>(p); break;
    }
    ++*launches;
    return static_cast<int>(cudaGetLastError());
}

// ------------------------------------------------------------------------------------------------
// direct: a block owns a tile of DBLK = 8*DT DM rows x TBLK = 32*TT output samples.  Channels are
// processed CH at a time: for each, the union of the samples the tile's rows need,
//     [t0 + min_j shift, t0 + TBLK + max_j shift),
// is copied once into shared memory with 16-byte cp.async (double buffered), so that every sample
// fetched from L2/HBM is reused by all DBLK rows.  Warp w owns rows w*DT..w*DT+DT-1; a lane owns
// the samples lane + 32*i, so shared-memory reads are conflict-free for any shift.
// ------------------------------------------------------------------------------------------------
constexpr int kDirectThreads = 256;
constexpr int kTT = 8;              // samples per thread per row
constexpr int kTBLK = 32 * kTT;     // 256 samples per tile

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    unsigned s = static_cast<unsigned>(__cvta_generic_to_shared(smem));
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::); }

template <typename InT, int DT>
__global__ void __launch_bounds__(kDirectThreads) direct_kernel(Problem p, int cap, int ch)
{
    using AccT = typename AccOf<InT>::type;
    constexpr int DBLK = 8 * DT;
    constexpr int VEC = 16 / sizeof(InT);  // elements per 16-byte copy
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // layout: [2][ch][cap] InT | [2][ch][DBLK] int offsets | [2][ch] long long gstart, int nvec
    InT* buf = reinterpret_cast<InT*>(smem_raw);
    int* off_s = reinterpret_cast<int*>(smem_raw + static_cast<size_t>(2) * ch * cap * sizeof(InT));
    int* nvec_s = off_s + 2 * ch * DBLK;
    long long* gstart_s = reinterpret_cast<long long*>(nvec_s + 2 * ch + ((2 * ch) & 1));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t t0 = static_cast<int64_t>(blockIdx.x) * kTBLK;
    const int d0 = blockIdx.y * DBLK;
    const int b1 = blockIdx.z % p.nb1, b0 = blockIdx.z / p.nb1;
    const InT* in = static_cast<const InT*>(p.in) + b0 * p.in_b0_stride + b1 * p.in_b1_stride;
    const int32_t* sh = p.shift + b1 * p.shift_b1_stride;

    // rows of this tile that exist, and the longest of them: a tile beyond every row's length exits
    int64_t tile_len = 0;
    for (int j = 0; j < DBLK && d0 + j < p.ndm; ++j) {
        const int64_t l = p.row_extra ? p.n_base + p.row_extra[b1 * p.row_extra_b1_stride + d0 + j] : p.n_out;
        tile_len = l > tile_len ? l : tile_len;
    }
    if (t0 >= tile_len)
        return;

    AccT acc[DT][kTT];
#pragma unroll
    for (int j = 0; j < DT; ++j)
#pragma unroll
        for (int i = 0; i < kTT; ++i)
            acc[j][i] = 0;

    const int nstage = (p.nchans + ch - 1) / ch;

    // prepare stage s into buffer b: offsets, then the copies
    auto prepare = [&](int s, int b) {
        // one warp per channel: lane j holds shift(d0+j, c); min/max by shuffles
        for (int cc = warp; cc < ch; cc += kDirectThreads / 32) {
            const int c = s * ch + cc;
            int sv = 0;
            const bool row_ok = lane < DBLK && d0 + lane < p.ndm && c < p.nchans;
            if (row_ok)
                sv = sh[static_cast<int64_t>(d0 + lane) * p.shift_dm_stride + c];
            int mn = row_ok ? sv : 0x7fffffff, mx = row_ok ? sv : 0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
                mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            }
            long long g = 0;
            int nv = 0;
            if (c < p.nchans) {
                g = (t0 + mn) & ~static_cast<long long>(VEC - 1);
                long long end = t0 + kTBLK + mx;
                if (end > p.in_len)
                    end = p.in_len;
                nv = end > g ? static_cast<int>((end - g + VEC - 1) / VEC) : 0;
            }
            if (lane < DBLK)
                off_s[(b * ch + cc) * DBLK + lane] = row_ok ? static_cast<int>(t0 + sv - g) : 0;
            if (lane == 0) {
                gstart_s[b * ch + cc] = g;
                nvec_s[b * ch + cc] = nv;
            }
        }
        __syncthreads();
        for (int cc = 0; cc < ch; ++cc) {
            const int c = s * ch + cc;
            if (c >= p.nchans)
                break;
            const int nv = nvec_s[b * ch + cc];
            const InT* src = in + static_cast<int64_t>(c) * p.in_chan_stride + gstart_s[b * ch + cc];
            InT* dst = buf + (static_cast<size_t>(b) * ch + cc) * cap;
            for (int q = tid; q < nv; q += kDirectThreads)
                cp_async16(dst + static_cast<size_t>(q) * VEC, src + static_cast<size_t>(q) * VEC);
        }
        cp_async_commit();
    };

    prepare(0, 0);
    for (int s = 0; s < nstage; ++s) {
        const int b = s & 1;
        cp_async_wait_all();
        __syncthreads();  // stage s landed; everyone is done computing on buffer b^1
        if (s + 1 < nstage)
            prepare(s + 1, b ^ 1);
        const int nc = min(ch, p.nchans - s * ch);
        for (int cc = 0; cc < nc; ++cc) {
            const InT* row = buf + (static_cast<size_t>(b) * ch + cc) * cap + lane;
            const int* offs = off_s + (b * ch + cc) * DBLK + warp * DT;
#pragma unroll
            for (int j = 0; j < DT; ++j) {
                const InT* r = row + offs[j];
#pragma unroll
                for (int i = 0; i < kTT; ++i)
                    acc[j][i] += static_cast<AccT>(r[32 * i]);
            }
        }
    }

    AccT* out = static_cast<AccT*>(p.out) + b0 * p.out_b0_stride + b1 * p.out_b1_stride;
#pragma unroll
    for (int j = 0; j < DT; ++j) {
        const int d = d0 + warp * DT + j;
        if (d >= p.ndm)
            continue;
        const int64_t len = p.row_extra ? p.n_base + p.row_extra[b1 * p.row_extra_b1_stride + d] : p.n_out;
        AccT* o = out + static_cast<int64_t>(d) * p.out_dm_stride;
#pragma unroll
        for (int i = 0; i < kTT; ++i) {
            const int64_t t = t0 + lane + 32 * i;
            if (t < len)
                o[t] = p.accumulate ? o[t] + acc[j][i] : acc[j][i];
        }
    }
}

// shared memory the direct kernel needs for (cap, ch, DT)
template <typename InT> static size_t direct_smem(int cap, int ch, int dt)
{
    return static_cast<size_t>(2) * ch * cap * sizeof(InT) + static_cast<size_t>(2) * ch * 8 * dt * 4 +
           static_cast<size_t>(2 * ch + 1) * 4 + static_cast<size_t>(2) * ch * 8 + 16;
}

template <typename InT, int DT>
static int launch_direct_t(const Problem& p, int cap, int ch, cudaStream_t st)
{
    const size_t smem = direct_smem<InT>(cap, ch, DT);
    cudaError_t e = cudaFuncSetAttribute(direct_kernel<InT, DT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess)
        return static_cast<int>(e);
    dim3 grid(static_cast<unsigned>((p.n_out + kTBLK - 1) / kTBLK), (p.ndm + 8 * DT - 1) / (8 * DT),
              p.nb0 * p.nb1);
    direct_kernel<InT, DT><<<grid, kDirectThreads, smem, st>>>(p, cap, ch);
    return static_cast<int>(cudaGetLastError());
}

template <typename InT>
static int launch_direct_e(const Problem& p, const int spread[3], cudaStream_t st)
{
    // pick the largest DM tile whose staged rows fit: cap = TBLK + spread + alignment slack
    constexpr int VEC = 16 / sizeof(InT);
    const size_t budget = 96 * 1024;  // two blocks per SM
    const int dts[3] = {4, 2, 1};
    for (int k = 0; k < 3; ++k) {
        const int dt = dts[k];
        long long cap = static_cast<long long>(kTBLK) + spread[k] + 2 * VEC;
        cap = (cap + VEC - 1) / VEC * VEC;
        int ch = 16;
        while (ch > 1 && direct_smem<InT>(static_cast<int>(cap), ch, dt) > budget)
            ch >>= 1;
        if (cap > (1 << 24) || direct_smem<InT>(static_cast<int>(cap), ch, dt) > 200 * 1024)
            continue;
        if (ch > p.nchans) {
            ch = 1;
            while (ch * 2 <= p.nchans)
                ch *= 2;
        }
        switch (dt) {
        case 4: return launch_direct_t<InT, 4>(p, static_cast<int>(cap), ch, st);
        case 2: return launch_direct_t<InT, 2>(p, static_cast<int>(cap), ch, st);
        default: return launch_direct_t<InT, 1>(p, static_cast<int>(cap), ch, st);
        }
    }
    return -1;  // does not fit: the caller falls back to the naive kernel
}

// spread[k]: max over DM tiles of 32, 16, 8 rows and channels of (max shift - min shift) in a tile
int launch_direct(const Problem& p, Elem in_t, const int spread[3], void* stream, int* launches)
{
    if (p.n_out <= 0 || p.ndm <= 0)
        return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc;
    switch (in_t) {
    case Elem::F32: rc = launch_direct_e<float>(p, spread, st); break;
    case Elem::U8: rc = launch_direct_e<uint8_t>(p, spread, st); break;
    default: rc = launch_direct_e<int32_t>(p, spread, st); break;
    }
    if (rc == -1)
        return launch_naive(p, in_t, stream, launches);
    ++*launches;
    return rc;
}

}  // namespace dedisp
