// Event detection on a de-dispersed buffer: mean and standard
// deviation of the ENTIRE buffer, threshold mu + nsigma * sigma, every value above it emitted as a
// (time, DM trial, intensity) triplet.  HBM-bound: two passes over out[ndm][n] (statistics, then the
// threshold scan), 16-byte loads, fp64 sums reduced in a fixed order (per-thread, warp shuffles,
// per-block partials, one finishing block), so mu, sigma and therefore the event set do not depend
// on scheduling; only the ORDER of the triplets does (an atomic cursor, advanced once per warp and test).
#include <cuda_runtime.h>

#include <mutex>

#include "dedisp_internal.h"

namespace dedisp {

namespace {

constexpr int kDetThreads = 256;

template <typename T> __device__ __forceinline__ double to_f64(T v) { return static_cast<double>(v); }

// sums of (x - pivot) and (x - pivot)^2 over one beam; pivot = first element (keeps the variance
// free of cancellation when the mean is large, e.g. 2048 channels of uint8 around 128)
template <typename T>
__global__ void __launch_bounds__(kDetThreads) detect_stats_kernel(const T* __restrict__ out, int ndm, int64_t n,
                                                                    int64_t stride, int64_t beam_stride,
                                                                    double* __restrict__ partial)
{
    const T* base = out + static_cast<int64_t>(blockIdx.y) * beam_stride;
    const double pivot = to_f64(base[0]);
    double s1 = 0.0, s2 = 0.0;
    const int64_t n4 = n / 4;
    for (int d = blockIdx.x; d < ndm; d += gridDim.x) {
        const T* row = base + static_cast<int64_t>(d) * stride;  // 16-byte aligned (stride % 4 == 0)
        for (int64_t q = threadIdx.x; q < n4; q += kDetThreads) {
            const int4 raw = *reinterpret_cast<const int4*>(row + 4 * q);
            const T* v = reinterpret_cast<const T*>(&raw);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double x = to_f64(v[k]) - pivot;
                s1 += x;
                s2 += x * x;
            }
        }
        for (int64_t t = 4 * n4 + threadIdx.x; t < n; t += kDetThreads) {
            const double x = to_f64(row[t]) - pivot;
            s1 += x;
            s2 += x * x;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    __shared__ double w1[kDetThreads / 32], w2[kDetThreads / 32];
    if ((threadIdx.x & 31) == 0) {
        w1[threadIdx.x >> 5] = s1;
        w2[threadIdx.x >> 5] = s2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < kDetThreads / 32; ++k) {
            a += w1[k];
            b += w2[k];
        }
        double* p = partial + (static_cast<int64_t>(blockIdx.y) * gridDim.x + blockIdx.x) * 2;
        p[0] = a;
        p[1] = b;
    }
}

// one block per beam: partials in index order -> mean, sigma (population), threshold; cursor = 0
template <typename T>
__global__ void detect_finish_kernel(const T* __restrict__ out, int64_t beam_stride, const double* __restrict__ partial,
                                     int nblocks, double count, double nsigma, dedisp_detect_result* __restrict__ res)
{
    if (threadIdx.x != 0)
        return;
    const double* p = partial + static_cast<int64_t>(blockIdx.x) * nblocks * 2;
    double a = 0.0, b = 0.0;
    for (int k = 0; k < nblocks; ++k) {
        a += p[2 * k];
        b += p[2 * k + 1];
    }
    const double pivot = to_f64(out[static_cast<int64_t>(blockIdx.x) * beam_stride]);
    const double m = a / count;
    double var = b / count - m * m;
    var = var > 0.0 ? var : 0.0;
    dedisp_detect_result r;
    r.mean = pivot + m;
    r.sigma = sqrt(var);
    r.threshold = r.mean + nsigma * r.sigma;
    r.count = 0;
    res[blockIdx.x] = r;
}

template <typename T>
__global__ void __launch_bounds__(kDetThreads) detect_emit_kernel(const T* __restrict__ out, int ndm, int64_t n,
                                                                   int64_t stride, int64_t beam_stride,
                                                                   dedisp_detect_result* __restrict__ res,
                                                                   dedisp_event* __restrict__ events, int64_t capacity)
{
    const int beam = blockIdx.y;
    const T* base = out + static_cast<int64_t>(beam) * beam_stride;
    const double thr = res[beam].threshold;
    unsigned long long* cursor = reinterpret_cast<unsigned long long*>(&res[beam].count);
    dedisp_event* ev = events + static_cast<int64_t>(beam) * capacity;
    // one atomic per warp and test: the lanes that found an event take consecutive slots
    const unsigned lane = threadIdx.x & 31;
    auto emit = [&](int64_t t, int d, T v) {
        const unsigned act = __activemask();
        const int leader = __ffs(act) - 1;
        unsigned long long k = 0;
        if (lane == static_cast<unsigned>(leader))
            k = atomicAdd(cursor, static_cast<unsigned long long>(__popc(act)));
        k = __shfl_sync(act, k, leader) + __popc(act & ((1u << lane) - 1u));
        if (static_cast<int64_t>(k) < capacity) {
            dedisp_event e;
            e.t = t;
            e.dm = d;
            e.value = static_cast<float>(v);
            ev[k] = e;
        }
    };
    const int64_t n4 = n / 4;
    for (int d = blockIdx.x; d < ndm; d += gridDim.x) {
        const T* row = base + static_cast<int64_t>(d) * stride;
        // four 16-byte loads in flight per thread before any test
        for (int64_t q0 = threadIdx.x; q0 < n4; q0 += 4 * kDetThreads) {
            int4 raw[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int64_t q = q0 + u * kDetThreads;
                raw[u] = q < n4 ? *reinterpret_cast<const int4*>(row + 4 * q) : make_int4(0, 0, 0, 0);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int64_t q = q0 + u * kDetThreads;
                if (q >= n4)
                    break;
                const T* v = reinterpret_cast<const T*>(&raw[u]);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (to_f64(v[k]) > thr)
                        emit(4 * q + k, d, v[k]);
            }
        }
        for (int64_t t = 4 * n4 + threadIdx.x; t < n; t += kDetThreads)
            if (to_f64(row[t]) > thr)
                emit(t, d, row[t]);
    }
}

// ---- fused path (dedisp_execute_detect): the de-dispersion kernel left per-block sums of (x - pivot) and
// (x - pivot)^2; the pivot is the DM-0 output at t = 0 formed from the input, sum_c in[c][0].
template <typename InT>
__global__ void __launch_bounds__(kDetThreads) detect_pivot_kernel(const InT* __restrict__ in, int nchans, int64_t chan_stride,
                                                                    int64_t beam_stride, double* __restrict__ pivot)
{
    __shared__ double part[kDetThreads];
    const InT* base = in + static_cast<int64_t>(blockIdx.x) * beam_stride;
    double s = 0.0;
    for (int c = threadIdx.x; c < nchans; c += kDetThreads)
        s += static_cast<double>(base[static_cast<int64_t>(c) * chan_stride]);
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int k = 0; k < kDetThreads; ++k)
            a += part[k];
        pivot[blockIdx.x] = a;
    }
}

// one block per beam: thread i adds partials i, i + 256, ... in that order, thread 0 adds the 256 sums in
// index order -> mean, sigma (population), threshold; cursor = 0.  A fixed order: the statistics do not
// depend on scheduling.
__global__ void __launch_bounds__(kDetThreads) detect_finish_fused_kernel(const double* __restrict__ partial, int64_t npart,
                                                                          int64_t part_stride, const double* __restrict__ pivot,
                                                                          double count, double nsigma,
                                                                          dedisp_detect_result* __restrict__ res)
{
    __shared__ double p1[kDetThreads], p2[kDetThreads];
    const double* p = partial + static_cast<int64_t>(blockIdx.x) * part_stride * 2;
    double a = 0.0, b = 0.0;
    for (int64_t k = threadIdx.x; k < npart; k += kDetThreads) {
        a += p[2 * k];
        b += p[2 * k + 1];
    }
    p1[threadIdx.x] = a;
    p2[threadIdx.x] = b;
    __syncthreads();
    if (threadIdx.x != 0)
        return;
    a = b = 0.0;
    for (int k = 0; k < kDetThreads; ++k) {
        a += p1[k];
        b += p2[k];
    }
    const double m = a / count;
    double var = b / count - m * m;
    var = var > 0.0 ? var : 0.0;
    dedisp_detect_result r;
    r.mean = pivot[blockIdx.x] + m;
    r.sigma = sqrt(var);
    r.threshold = r.mean + nsigma * r.sigma;
    r.count = 0;
    res[blockIdx.x] = r;
}

template <typename T>
int launch_detect_t(const void* out, int nbeams, int ndm, int64_t n, int64_t stride, double nsigma,
                    dedisp_event* events, int64_t capacity, dedisp_detect_result* res, double* partial, int nblocks,
                    cudaStream_t st, int* launches)
{
    const T* o = static_cast<const T*>(out);
    const int64_t beam_stride = stride * ndm;
    dim3 grid(nblocks, nbeams);
    detect_stats_kernel<T><<<grid, kDetThreads, 0, st>>>(o, ndm, n, stride, beam_stride, partial);
    detect_finish_kernel<T><<<nbeams, 32, 0, st>>>(o, beam_stride, partial, nblocks, static_cast<double>(ndm) * n, nsigma, res);
    detect_emit_kernel<T><<<grid, kDetThreads, 0, st>>>(o, ndm, n, stride, beam_stride, res, events, capacity);
    *launches += 3;
    return static_cast<int>(cudaGetLastError());
}

}  // namespace

int launch_detect_pivot(const void* in, Elem in_t, int nbeams, int nchans, int64_t chan_stride, double* pivot, void* stream,
                        int* launches)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (in_t == Elem::F32)
        detect_pivot_kernel<float><<<nbeams, kDetThreads, 0, st>>>(static_cast<const float*>(in), nchans, chan_stride,
                                                                  chan_stride * nchans, pivot);
    else
        detect_pivot_kernel<uint8_t><<<nbeams, kDetThreads, 0, st>>>(static_cast<const uint8_t*>(in), nchans, chan_stride,
                                                                    chan_stride * nchans, pivot);
    ++*launches;
    return static_cast<int>(cudaGetLastError());
}

// finish + threshold scan on statistics the de-dispersion kernel accumulated (two launches, one pass over out)
int launch_detect_fused(const void* out, Elem t, int nbeams, int ndm, int64_t n, int64_t stride, double nsigma,
                        dedisp_event* events, int64_t capacity, dedisp_detect_result* res, const double* partial,
                        int64_t npart, int64_t part_stride, const double* pivot, void* stream, int* launches)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    detect_finish_fused_kernel<<<nbeams, kDetThreads, 0, st>>>(partial, npart, part_stride, pivot,
                                                              static_cast<double>(ndm) * n, nsigma, res);
    dim3 grid(detect_blocks(ndm), nbeams);
    const int64_t beam_stride = stride * ndm;
    if (t == Elem::F32)
        detect_emit_kernel<float><<<grid, kDetThreads, 0, st>>>(static_cast<const float*>(out), ndm, n, stride, beam_stride,
                                                               res, events, capacity);
    else
        detect_emit_kernel<int32_t><<<grid, kDetThreads, 0, st>>>(static_cast<const int32_t*>(out), ndm, n, stride,
                                                                 beam_stride, res, events, capacity);
    *launches += 2;
    return static_cast<int>(cudaGetLastError());
}

int detect_blocks(int ndm) { return ndm < 1184 ? ndm : 1184; }  // 8 blocks per SM on 148 SMs, whole rows each

int launch_detect(const void* out, Elem t, int nbeams, int ndm, int64_t n, int64_t stride, double nsigma,
                  dedisp_event* events, int64_t capacity, dedisp_detect_result* res, double* partial, void* stream,
                  int* launches)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int nb = detect_blocks(ndm);
    if (t == Elem::F32)
        return launch_detect_t<float>(out, nbeams, ndm, n, stride, nsigma, events, capacity, res, partial, nb, st, launches);
    return launch_detect_t<int32_t>(out, nbeams, ndm, n, stride, nsigma, events, capacity, res, partial, nb, st, launches);
}

}  // namespace dedisp

// ---- dedisp_detect_static: the two-pass detection above with its per-block partial sums in a fixed
// array that is part of the library image, for callers that must not allocate (include/dedisp.h).
namespace dedisp {
namespace {

// The only scratch the detection needs: two doubles per (beam, block) of detect_stats_kernel.  One copy
// of this array exists on every GPU that loads the library, from module load until the process exits.
constexpr int64_t kStaticSlots = DEDISP_DETECT_STATIC_MAX_SLOTS;
static __device__ __align__(256) double detect_static_scratch[kStaticSlots * 2];

// In host code `detect_static_scratch` is only a handle for the runtime's symbol table, not something a
// kernel can dereference.  The device address differs per GPU, so it is looked up once per device, with
// that device current, and remembered here.
constexpr int kStaticMaxDevices = 64;
std::mutex static_mu;
double* static_ptr[kStaticMaxDevices] = {};

cudaError_t static_scratch(double** ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return e;
    if (dev < 0 || dev >= kStaticMaxDevices)
        return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(static_mu);
    if (!static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, detect_static_scratch);
        if (e != cudaSuccess)
            return e;
        if (!p)
            return cudaErrorInvalidSymbol;
        static_ptr[dev] = static_cast<double*>(p);
    }
    *ptr = static_ptr[dev];
    return cudaSuccess;
}

}  // namespace
}  // namespace dedisp

extern "C" int64_t dedisp_detect_static_max_slots(void) { return dedisp::kStaticSlots; }

extern "C" dedisp_status dedisp_detect_static(const void* out, dedisp_dtype dtype, int ndm, int64_t nsamp_out,
                                              int64_t out_stride, int nbeams, double nsigma, dedisp_event* events,
                                              int64_t capacity, dedisp_detect_result* results, void* cuda_stream)
{
    using namespace dedisp;
    if (!out || !results || ndm <= 0 || nbeams <= 0 || nsamp_out <= 0 || capacity < 0 || (capacity > 0 && !events) ||
        !(nsigma == nsigma) || (dtype != DEDISP_F32 && dtype != DEDISP_U8))
        return DEDISP_EINVAL;
    if (out_stride < nsamp_out || out_stride % 4 != 0 || (reinterpret_cast<uintptr_t>(out) & 15) != 0)
        return DEDISP_ESHAPE;
    // the fixed array cannot grow: refuse, before touching the device, what does not fit
    if (static_cast<int64_t>(nbeams) * detect_blocks(ndm) > kStaticSlots)
        return DEDISP_ELIMIT;
    double* partial = nullptr;
    if (static_scratch(&partial) != cudaSuccess)
        return DEDISP_ECUDA;
    // Nothing in the array has to start at zero: detect_stats_kernel stores both sums of every slot that
    // detect_finish_kernel reads, later on the same stream, so whatever an earlier call left is overwritten
    // first.  The event cursor lives in the caller's `results` and is reset by detect_finish_kernel.
    int launches = 0;
    const int rc = launch_detect(out, dtype == DEDISP_F32 ? Elem::F32 : Elem::I32, nbeams, ndm, nsamp_out, out_stride,
                                 nsigma, events, capacity, results, partial, cuda_stream, &launches);
    return rc == 0 ? DEDISP_OK : DEDISP_ECUDA;
}
