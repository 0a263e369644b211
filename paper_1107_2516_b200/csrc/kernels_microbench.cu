// Register-only FP32 add microbenchmark: the measured denominator of the
// brute-force roofline.  The de-dispersion sum is nchans adds per output sample, so
// its ceiling on B200 is what the FP32 pipe sustains when every issue slot is an add and no operand
// comes from memory: nominally 128 adds / clk / SM.  Each thread keeps 32 packed (add.rn.f32x2 -> FADD2,
// the instruction the register-window kernel uses) or 64 scalar accumulators, all independent, and adds
// a loop-invariant operand to each of them `iters` times.
#include <cuda_runtime.h>

#include "dedisp_internal.h"

namespace dedisp {

namespace {

constexpr int kMbThreads = 256;
constexpr int kMbAcc = 32;  // packed accumulators per thread (64 scalar ones)

template <bool PACKED>
__global__ void __launch_bounds__(kMbThreads) fadd_microbench_kernel(float* __restrict__ sink, int iters, float inc)
{
    unsigned long long acc[kMbAcc];
#pragma unroll
    for (int i = 0; i < kMbAcc; ++i)
        acc[i] = (static_cast<unsigned long long>(__float_as_uint(static_cast<float>(threadIdx.x + i))) << 32) |
                 __float_as_uint(static_cast<float>(i));
    const unsigned long long b = (static_cast<unsigned long long>(__float_as_uint(inc)) << 32) | __float_as_uint(inc);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kMbAcc; ++i) {
            if (PACKED) {
                asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[i]) : "l"(b));
            } else {
                unsigned lo = static_cast<unsigned>(acc[i]), hi = static_cast<unsigned>(acc[i] >> 32);
                asm volatile("add.rn.f32 %0, %0, %2;\n\tadd.rn.f32 %1, %1, %2;" : "+r"(lo), "+r"(hi) : "r"(__float_as_uint(inc)));
                acc[i] = (static_cast<unsigned long long>(hi) << 32) | lo;
            }
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < kMbAcc; ++i)
        s += __uint_as_float(static_cast<unsigned>(acc[i])) + __uint_as_float(static_cast<unsigned>(acc[i] >> 32));
    if (s == 12345.678f)  // keeps the adds alive; practically never true
        sink[0] = s;
}

}  // namespace

// adds executed by one launch; grid = blocks_per_sm blocks of 256 threads on every SM
int launch_fadd_microbench(int packed, int iters, int nsm, float* sink, void* stream, double* adds)
{
    const int blocks_per_sm = 4;  // 32 warps per SM, 8 per scheduler
    const int grid = nsm * blocks_per_sm;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (packed)
        fadd_microbench_kernel<true><<<grid, kMbThreads, 0, st>>>(sink, iters, 1.0f);
    else
        fadd_microbench_kernel<false><<<grid, kMbThreads, 0, st>>>(sink, iters, 1.0f);
    *adds = static_cast<double>(grid) * kMbThreads * static_cast<double>(iters) * kMbAcc * 2.0;
    return static_cast<int>(cudaGetLastError());
}

}  // namespace dedisp
