// Power + corner turn ("(iii) channelizes and calculates total
// power (iv) transposes data so that it is in channel order"): complex voltages in spectrum order
// volt[t][c] -> total power in the de-disperser's channel-major layout out[c][t] = re^2 + im^2.
// One fused pass (the paper runs two kernels, Table 6: 20 ms + 112 ms on its C1060): HBM-bound,
// 8 bytes read + 4 written per sample; a 64 x 64 tile goes through shared memory so that both the
// reads (along channels) and the writes (along time) are full 128-byte lines.  Each product and the
// sum are rounded to fp32 on their own (no FMA contraction), so the result is defined bit for bit.
#include <cuda_runtime.h>

#include <cstdint>

#include "dedisp_internal.h"

namespace dedisp {

namespace {

constexpr int kTile = 64;

__global__ void __launch_bounds__(256) power_corner_turn_kernel(const float2* __restrict__ volt, float* __restrict__ out,
                                                                int nchans, int64_t nsamp, int64_t volt_stride,
                                                                int64_t out_stride)
{
    __shared__ float tile[kTile][kTile + 1];
    const int tx = threadIdx.x & 63, ty = threadIdx.x >> 6;  // 64 x 4 threads
    const int64_t t0 = static_cast<int64_t>(blockIdx.x) * kTile;
    const int c0 = blockIdx.y * kTile;
    // all 16 loads of a thread in flight before the first square
    float2 v[kTile / 4];
#pragma unroll
    for (int q = 0; q < kTile / 4; ++q) {
        const int64_t t = t0 + ty + 4 * q;
        const int c = c0 + tx;
        v[q] = t < nsamp && c < nchans ? volt[t * volt_stride + c] : make_float2(0.0f, 0.0f);
    }
#pragma unroll
    for (int q = 0; q < kTile / 4; ++q)
        tile[ty + 4 * q][tx] = __fadd_rn(__fmul_rn(v[q].x, v[q].x), __fmul_rn(v[q].y, v[q].y));
    __syncthreads();
#pragma unroll
    for (int k = ty; k < kTile; k += 4) {
        const int c = c0 + k;
        const int64_t t = t0 + tx;
        if (c < nchans && t < nsamp)
            out[static_cast<int64_t>(c) * out_stride + t] = tile[tx][k];
    }
}

// Binning, stage (i) of the subband scheme ("Binning averages N_b consecutive samples"):
// out[c][j] = (in[c][j*nb] + ... + in[c][j*nb + nb-1]) / nb, the sum left to right, every operation
// rounded on its own.  Four outputs per thread, 256 apart; a warp reads 32*nb consecutive floats per output.  HBM-bound.
__global__ void __launch_bounds__(256) bin_kernel(const float* __restrict__ in, float* __restrict__ out, int64_t nout,
                                                  int64_t in_stride, int64_t out_stride, int nb, int vec)
{
    // four outputs per thread, 256 apart (coalesced), so that enough loads are in flight
    const int64_t j0 = static_cast<int64_t>(blockIdx.x) * 1024 + threadIdx.x;
    const float* row = in + static_cast<int64_t>(blockIdx.y) * in_stride;
    float acc[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int64_t j = j0 + 256 * k;
        acc[k] = 0.0f;
        if (j >= nout)
            continue;
        const float* p = row + j * nb;
        if (nb == 2 && vec) {  // the paper's bin factors (Table 1: 1, 2, 4) with one vector load, same order of adds
            const float2 v = *reinterpret_cast<const float2*>(p);
            acc[k] = __fadd_rn(v.x, v.y);
        } else if (nb == 4 && vec) {
            const float4 v = *reinterpret_cast<const float4*>(p);
            acc[k] = __fadd_rn(__fadd_rn(__fadd_rn(v.x, v.y), v.z), v.w);
        } else {
            float a = p[0];
            for (int i = 1; i < nb; ++i)
                a = __fadd_rn(a, p[i]);
            acc[k] = a;
        }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int64_t j = j0 + 256 * k;
        if (j < nout)
            out[static_cast<int64_t>(blockIdx.y) * out_stride + j] = __fdiv_rn(acc[k], static_cast<float>(nb));
    }
}

}  // namespace

int launch_bin(const void* in, void* out, int64_t nrows, int64_t nout, int64_t in_stride, int64_t out_stride, int nb,
               void* stream)
{
    if (nrows <= 0 || nout <= 0)
        return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // vector loads need rows that start on nb * 4 bytes
    const int vec = (nb == 2 || nb == 4) && in_stride % nb == 0 && (reinterpret_cast<uintptr_t>(in) % (4 * nb)) == 0;
    for (int64_t r0 = 0; r0 < nrows; r0 += 65535) {  // grid.y limit
        const int64_t nr = nrows - r0 < 65535 ? nrows - r0 : 65535;
        dim3 grid(static_cast<unsigned>((nout + 1023) / 1024), static_cast<unsigned>(nr));
        bin_kernel<<<grid, 256, 0, st>>>(static_cast<const float*>(in) + r0 * in_stride,
                                         static_cast<float*>(out) + r0 * out_stride, nout, in_stride, out_stride, nb, vec);
    }
    return static_cast<int>(cudaGetLastError());
}

int launch_power_corner_turn(const void* volt, void* out, int nchans, int64_t nsamp, int64_t volt_stride,
                             int64_t out_stride, void* stream)
{
    if (nchans <= 0 || nsamp <= 0)
        return 0;
    dim3 grid(static_cast<unsigned>((nsamp + kTile - 1) / kTile), (nchans + kTile - 1) / kTile);
    power_corner_turn_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const float2*>(volt), static_cast<float*>(out), nchans, nsamp, volt_stride, out_stride);
    return static_cast<int>(cudaGetLastError());
}

}  // namespace dedisp
