// Register-window brute-force kernel for sm_100a.
//
//   out[d][t] = sum_c in[c][t + shift(c,d)]
//
// Launches per execute: one pairify, then one window_kernel per channel band.
//  1. pairify_kernel: P[c][u] = (in[c][u], in[c][u + NT*W]) as float2 (uint8 input is widened to
//     fp32 here; sums of < 2^24/255 bytes are exact in fp32).  Two samples NT*W apart that share
//     (c, d) have the same shift, so the main kernel adds two outputs per instruction
//     (add.f32x2 -> FADD2) from naturally aligned 64-bit registers, whatever the shift's parity.
//  2. window_kernel (band b): a block = G row groups x NT warps along time (+ a producer warp
//     group); a consumer warp owns D DM rows x 32*T slots (pairs of output samples) and keeps their
//     D x T packed accumulators in registers for the whole band.  Per channel it loads ONE window of
//     T + 1 staged pairs (LDS.64, conflict-free for odd T) that feeds all D rows: row j adds
//     w[i + o_j], o_j in {0, 1}, a warp-uniform choice per row and channel.  4-row shapes run the
//     channels of a pipeline stage as threaded code (chan_loop in window_rows.inc: one indirect
//     branch per channel over the 2^(D-1) offset patterns), 6-row shapes as two chains of row blocks
//     (rows7: one uniform branch per change of offset).  Rows follow the growing delay difference
//     between neighbouring DM trials by moving their accumulators up one slot now and then ("row
//     shift", planned on the host: window_plan.cpp); the partial sum that leaves the top of the
//     warp's slot range is handed, through the output buffer, to the warp segment that follows in
//     time (its fresh bottom slot stands for the same output sample), so a block of 2*NT segments
//     loses kmax samples as a whole, not per segment.  Channel segments are staged into a ring of
//     2-3 pipeline stages of 8-12 channels by 1-D TMA bulk copies (cp.async.bulk + mbarrier), every
//     lane of a producer warp issuing one channel's copy.  At the end of the band the accumulators go
//     through a per-warp shared-memory transpose to coalesced global accesses: band 0 stores (and,
//     for dedisp_execute_detect, sums the outputs' statistics), later bands add to what is there.
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
// one lane of the (converged) warp arrives; elect.sync needs no lane id in a register
__device__ __forceinline__ void mbar_arrive_one(unsigned bar)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "elect.sync _|p, 0xffffffff;\n"
        "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n"
        "}\n" ::"r"(bar) : "memory");
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
__device__ __forceinline__ unsigned lds32(unsigned addr)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
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

// Hand-over state of one consumer warp, in shared memory, touched by lane 31 only: for row j the
// output time (int32 at 8*j; the launcher keeps all times below 2^31) and address (8 bytes at 64 + 8*j) of the NEXT partial sum to leave the
// top slot of the warp's lower segment (the upper segment is hp samples later).  Both move down by
// one sample per row shift.  Kept out of registers: the channel loop has none to spare.
constexpr int kFallBytes = 128;

__device__ __forceinline__ void fall_store(float* p, float v, bool first)
{
    if (first)
        *p = v;
    else
        asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}
__device__ __forceinline__ void fall_store(int32_t* p, float v, bool first)
{
    const int iv = __float2int_rn(v);
    if (first)
        *p = iv;
    else
        asm volatile("red.global.add.s32 [%0], %1;" ::"l"(p), "r"(iv) : "memory");
}

// the rows in mask (bit j-1 = row j) move their accumulators up one slot; lane 0 gets a fresh one and
// lane 31 hands the pair that leaves the top slot over to the following segments (band 0 stores it,
// the flush of that segment adds its own part; later bands add on both sides)
template <int T, int D, typename OutT>
__device__ __forceinline__ void shift_rows(u64 (&acc)[D][T], unsigned mask, int lane, unsigned fall_s, unsigned n_out,
                                           int hp, bool hi_owned, bool first, bool edge)
{
#pragma unroll
    for (int j = 1; j < D; ++j) {
        if (mask & (1u << (j - 1))) {
            if (lane == 31) {
                // before the shuffle, so that its registers are free again when the carry arrives
                unsigned long long pa;
                asm volatile("ld.shared.b64 %0, [%1+64];" : "=l"(pa) : "r"(fall_s + 8u * j));
                OutT* p = reinterpret_cast<OutT*>(pa);
                if (!edge) {
                    fall_store(p, __uint_as_float(static_cast<unsigned>(acc[j][T - 1])), first);
                    if (hi_owned)
                        fall_store(p + hp, __uint_as_float(static_cast<unsigned>(acc[j][T - 1] >> 32)), first);
                } else {
                    // first / last time tiles, tail rows of the last DM tile: test the output time
                    int t;
                    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(t) : "r"(fall_s + 8u * j));
                    if (static_cast<unsigned>(t) < n_out)
                        fall_store(p, __uint_as_float(static_cast<unsigned>(acc[j][T - 1])), first);
                    if (hi_owned && static_cast<unsigned>(t + hp) < n_out)
                        fall_store(p + hp, __uint_as_float(static_cast<unsigned>(acc[j][T - 1] >> 32)), first);
                    asm volatile("st.shared.b32 [%0], %1;" ::"r"(fall_s + 8u * j), "r"(t - 1) : "memory");
                }
                asm volatile("st.shared.b64 [%0+64], %1;" ::"r"(fall_s + 8u * j), "l"(pa - sizeof(OutT)) : "memory");
            }
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

template <typename OutT> __device__ __forceinline__ OutT to_out(float v);
template <> __device__ __forceinline__ float to_out<float>(float v) { return v; }
template <> __device__ __forceinline__ int32_t to_out<int32_t>(float v) { return __float2int_rn(v); }

__device__ __forceinline__ void tile_of(const WindowArgs& a, int lin, int& ty, int& tt)
{
    const int per_group = a.dm_group * a.ntile_t;
    const int grp = lin / per_group, r = lin - grp * per_group;
    const int g0 = grp * a.dm_group;
    const int gsz = a.ntile_dm - g0 < a.dm_group ? a.ntile_dm - g0 : a.dm_group;  // last group may be short
    tt = r / gsz;
    ty = g0 + r - tt * gsz;
}

// smem layout: [nst] full barriers | [nst] empty barriers | Fall[NCW] | nst stages of { 128-byte header,
//              kWinCh channel slots }; the flush's transpose scratch [NCW][W] u64 overlays the stages
static_assert(kWinFixedBytes == 128 + 16 * kFallBytes, "barriers + up to 16 consumer warps' hand-over state");

template <int T, int G, int NT, int D, typename OutT>
__global__ void __launch_bounds__((G * NT + 4) * 32, (G * NT == 4 ? 2 : 1))
    window_kernel(const WindowArgs a, const int c_begin, const int c_end, const int band, const int stage0)
{
    const int nst = a.nst, slot_bytes = a.slot_bytes, CH = a.ch, hdr_bytes = a.hdr_words * 4;
    constexpr int W = 32 * T, NCW = G * NT, RB = D * G;
    // registers per consumer thread once the producer warp group has released its share
    // (blocks of 4 consumer warps run two to an SM and share the register file)
    constexpr int kPool = ((NCW == 4 ? 32768 : 65536) - 4 * 32 * 24) / (NCW * 32) / 8 * 8;
    constexpr int kConsRegs = kPool > 240 ? 240 : kPool;
    static_assert(NCW % 4 == 0, "setmaxnreg works on groups of four warps");
    // setmaxnreg.inc waits until the registers are free in the BLOCK's pool, and that pool is what the block
    // was launched with: threads x the per-thread count ptxas derives from __launch_bounds__ (the largest
    // multiple of 8 that lets the stated number of blocks fit 64 K registers -- cuobjdump -res-usage shows
    // 128 for 512 threads, 168 for 384), not the whole register file.  The consumers' kConsRegs and the
    // producers' 24 must fit it, or the consumers wait for ever.  This is what hung the 16-consumer-warp
    // shapes tried in round 2: 640 threads launch with 96 registers = 61 440, and 512 x 120 + 128 x 24 = 64 512.
    // (They could run with 112, which does not hold D x T >= 60 pairs, so no such shape is instantiated.)
    constexpr int kThreads = (NCW + 4) * 32, kBlocksPerSm = NCW == 4 ? 2 : 1;
    constexpr int kLaunchRegs = 65536 / (kThreads * kBlocksPerSm) / 8 * 8 > 255 ? 255 : 65536 / (kThreads * kBlocksPerSm) / 8 * 8;
    static_assert(NCW * 32 * kConsRegs + 4 * 32 * 24 <= kThreads * kLaunchRegs,
                  "setmaxnreg.inc would never be granted: consumer + producer registers exceed the block's launch pool");
    static_assert(NCW <= 12 && D <= kWinD, "hand-over area holds 16 warps, but 16 consumer warps leave 112 registers each (see above)");
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // Block order: groups of a.dm_group DM tiles; inside a group all time tiles, DM tile fastest.
    // The blocks in flight then read neighbouring delays of a few time tiles: the wave's footprint in
    // the pair buffer fits L2 (DM-fastest over ALL tiles reads a max_delay-wide range per time tile).
    const int beam = blockIdx.z;
    int ty, tt;
    tile_of(a, blockIdx.x, ty, tt);
    // the block's 2*NT warp segments of W slots are contiguous in time from T0 on; blocks are Hb apart
    const int64_t T0 = static_cast<int64_t>(tt) * a.Hb;

    const unsigned bar_full = smem_u32(smem);
    const unsigned bar_empty = bar_full + 8u * nst;
    // the flush's transpose scratch [NCW][W] u64 reuses the ring once every consumer has left the loop
    const int stages_off = kWinFixedBytes;
    const int tr_off = stages_off;
    const int stage_bytes = hdr_bytes + CH * slot_bytes;
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
    const int nstage = (nch + CH - 1) / CH;
    const int stage_total = a.stage_total;

    if (warp >= NCW) {
        // ---- producer warp group: gives its registers to the consumers; one thread stages CH
        // channels per barrier (padding channels and the extra last stage get zeros)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        {
            // the warps of the group take the stages in turn (stage s belongs to warp s % P), so the staging
            // work is spread over the schedulers instead of loading the one that also runs consumer warps
            // 0, 4, 8.  P = min(4, nst): a warp waits on a slot's empty barrier by parity only, it is ordered
            // behind stage s - P - nst, and the parity test needs stage s - 2 * nst consumed (P <= nst).
            const int pw = warp - NCW;
            const int P = nst < 4 ? nst : 4;
            const int32_t* meta = a.meta + (static_cast<int64_t>(ty) * a.nchans + c_begin) * kWinMetaWords;
            const int32_t* hdr = a.hdr + (static_cast<int64_t>(ty) * stage_total + stage0) * a.hdr_words;
            const float2* prow = static_cast<const float2*>(a.pairs) +
                                 (static_cast<int64_t>(beam) * a.nchans + c_begin) * a.pair_stride + T0;
            const int64_t pair_stride = a.pair_stride;
            const int zlen = ((NT - 1) * W + W + 2 + 1) & ~1;  // pairs a padding channel must provide
            for (int s = pw; s < nstage && pw < P; s += P) {
                const int ring = s % nst, lap = s / nst;
                // lanes 0 .. CH-1: (base, len) of this stage's channels
                const int k = s * CH + lane;
                int pb = 0, pl = -1;
                if (lane < CH && k < nch) {
                    pb = __ldg(meta + static_cast<int64_t>(k) * kWinMetaWords);
                    pl = __ldg(meta + static_cast<int64_t>(k) * kWinMetaWords + 1);
                }
                unsigned bytes = lane < CH ? (pl < 0 ? zlen : pl) * 8 : 0;
#pragma unroll
                for (int o = 8; o > 0; o >>= 1)   // CH <= 12 < 16 lanes
                    bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
                if (lane == 0) {
                    if (lap > 0)
                        mbar_wait_backoff(bar_empty + 8u * ring, (lap - 1) & 1);
                    mbar_expect_tx(bar_full + 8u * ring, bytes + hdr_bytes);
                    bulk_g2s(smem_u32(stages) + ring * stage_bytes, hdr + static_cast<int64_t>(s) * a.hdr_words, hdr_bytes,
                             bar_full + 8u * ring);
                }
                __syncwarp();   // the expected byte count is posted before any lane's copy can complete
                if (lane < CH) {
                    const unsigned d = smem_u32(stages) + ring * stage_bytes + hdr_bytes + lane * slot_bytes;
                    if (pl < 0)
                        bulk_g2s(d, a.zeros, zlen * 8, bar_full + 8u * ring);
                    else
                        bulk_g2s(d, prow + static_cast<int64_t>(k) * pair_stride + pb, pl * 8, bar_full + 8u * ring);
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

    const bool first = band == 0;
    constexpr int hp = NT * W;   // a pair is (t, t + hp)
    const unsigned fall_s = smem_u32(smem) + 128u + static_cast<unsigned>(uwarp) * kFallBytes;
    // block-uniform: some hand-over of this block may fall outside [0, n_out) or belong to a tail row
    const bool edge = T0 < a.theta_max + a.kmax || T0 + 2 * NT * W > a.n_out || (ty + 1) * RB > a.ndm;
    if (lane_pinned == 31) {
        // first partial sum to leave row j's top slot: slot W-1 of the lower segment at base theta_j
        const int32_t* thp = a.theta + (static_cast<int64_t>(ty) * a.nband + band) * RB + g * D;
        OutT* out = static_cast<OutT*>(a.out) + static_cast<int64_t>(beam) * a.ndm * a.out_stride;
#pragma unroll
        for (int j = 1; j < D; ++j) {
            const int d = ty * RB + g * D + j;
            const int t = static_cast<int>(T0) + wt * W + (W - 1) - __ldg(thp + j);
            OutT* p = out + static_cast<int64_t>(d) * a.out_stride + t;
            // tail rows of the last DM tile: a time that never passes the bounds test
            asm volatile("st.shared.b32 [%0], %1;\n\tst.shared.b64 [%0+64], %2;" ::"r"(fall_s + 8u * j),
                         "r"(d < a.ndm ? t : -0x40000000), "l"(p)
                         : "memory");
        }
    }
    __syncwarp();

    const unsigned lane_off = hdr_bytes + (wt * W + lane_pinned * T) * 8;  // bytes from the stage start
    auto shifts = [&](unsigned m) {
        // two masks (a row may shift twice at one channel); ONE copy of the shift code: it runs at 2 % of
        // the channels and its instruction fetches miss
        unsigned sm = (m >> 5) & 0x3ffu;
#pragma unroll 1
        do {
            shift_rows<T, D, OutT>(acc, sm & 31u, lane_pinned, fall_s, static_cast<unsigned>(a.n_out), hp, wt < NT - 1, first, edge);
            sm >>= 5;
        } while (sm);
    };
    // Stage loop around the channels of a stage.  (Sequential C++ copies of the add block make ptxas
    // permute the accumulator registers between them -- hundreds of moves -- so the chains keep ONE copy
    // in a rolled loop and the threaded loop is a single PTX statement.)  A warp carries the current channel's word m in a
    // uniform register; the NEXT channel's word is read from the stage's header at the top of the
    // iteration, next to the window loads, and moved into m after the adds, so its latency never shows
    // and a stage boundary is nothing but the barrier traffic (arrive, wait for the next stage).  Every
    // uniform-datapath instruction in the per-channel chain costs its full latency with three warps per
    // scheduler, so that chain is kept to the window address.
    const unsigned hdr_off = 4 * CH * g;
    unsigned m = __ldg(a.first + (static_cast<int64_t>(ty) * a.nband + band) * G + g);
    m = __reduce_or_sync(0xffffffffu, m);   // warp-uniform by construction; this lets ptxas know
    mbar_wait(bar_full, 0);
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
        unsigned hw = smem_u32(sbase) + hdr_off;    // this row group's words of the channels one further on
        if constexpr (D == 4 || (D == 5 && T <= 11)) {
            // threaded code (window_rows.inc, chan_loop): one indirect branch per channel over the 8 offset
            // patterns; runs channels until the stage is done or one needs a row shift
            unsigned spa = smem_u32(sbase) + lane_off;  // this thread's window base in the stage's first slot
            unsigned chn = CH;
            while (true) {
                chan_loop(acc, m, hw, spa, chn, static_cast<unsigned>(slot_bytes));
                if (chn == 0)
                    break;
                shifts(m);
                m &= ~kWinShiftBits;
            }
        } else {
            // two chains of row blocks (rows7), one uniform branch per row whose offset differs from the
            // previous row's
            u64 w[T + 1];
            const unsigned char* sp = sbase + lane_off;
            if (m & kWinStageShift) {
                // a row shift somewhere in this stage (about a third of the stages)
#pragma unroll 1
                for (int ch = 0; ch < CH; ++ch) {
                    const unsigned mn = lds32(hw);
                    load_window<T>(w, sp + (m >> 21) * 8);
                    if (m & kWinShiftBits)
                        shifts(m);
                    rows7(acc, w, m);
                    sp += slot_bytes;
                    hw += 4;
                    m = mn;
                }
            } else {
#pragma unroll 1
                for (int ch = 0; ch < CH; ++ch) {
                    const unsigned mn = lds32(hw);
                    load_window<T>(w, sp + (m >> 21) * 8);
                    rows7(acc, w, m);
                    sp += slot_bytes;
                    hw += 4;
                    m = mn;
                }
            }
        }
        __syncwarp();
        mbar_arrive_one(bar_empty + 8u * ring);
        if (s + 1 < nstage)
            mbar_wait(bar_full + 8u * ring_n, par_n);
        ring = ring_n;
        par = par_n;
        sbase = stages + ring_n * stage_bytes;
    }

    // ---- flush ------------------------------------------------------------------------------------------
    // Slot p of row r in segment seg (seg = wt: lower halves, NT + wt: upper halves) is the output sample
    //     rel = seg * W + p - kfinal_r   of the block's row range, which starts at time T0 - theta_r.
    // The block owns rel in [0, Hb).  Slots p < kfinal_r entered at the bottom during the band: the
    // channels before their entry were summed by segment seg - 1 and handed over through `out`
    // (shift_rows), so band 0 adds what is there; later bands add on both sides anyway.
    // The rows go through a shared-memory transpose (overlaying the ring) in passes of `rpp` rows with
    // their own regions: all rows of a pass are written, ONE __syncwarp, then read back and stored.
    // (A sync per row waits for the previous row's global stores every time: 3.5 % of the kernel.)
    // The barrier also orders the hand-over stores of every segment before the loads below.
    asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");  // consumers only: the ring is free now
    const int rpp = a.flush_rows;
    // the tile is decoded again from a fresh read of the block index: nothing of it stays in registers
    // over the channel loop
    int lin2;
    asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(lin2));
    int ty2, tt2;
    tile_of(a, lin2, ty2, tt2);
    const int64_t tw = static_cast<int64_t>(tt2) * a.Hb + wt * W;   // start of this warp's lower segment
    const int32_t* kfp = a.kfinal + (static_cast<int64_t>(ty2) * a.nband + band) * RB + g * D;
    const int32_t* thp = a.theta + (static_cast<int64_t>(ty2) * a.nband + band) * RB + g * D;
    OutT* out = static_cast<OutT*>(a.out) + static_cast<int64_t>(beam) * a.ndm * a.out_stride;
    const int kf_lane = __ldg(kfp + lane_pinned % D), th_lane = __ldg(thp + lane_pinned % D);
    u64* tr = reinterpret_cast<u64*>(smem + tr_off) + static_cast<size_t>(warp) * rpp * W;
    const int Hb = a.Hb;
    // fused statistics (dedisp_execute_detect): fp64 sums of (x - pivot) and (x - pivot)^2
    const bool stats = first && a.stat_partial != nullptr;
    const double pivot = stats ? a.pivot[beam] : 0.0;
    double s1 = 0.0, s2 = 0.0;
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
            const int d = ty2 * RB + g * D + jj;
            const int kf = __shfl_sync(0xffffffffu, kf_lane, jj), th = __shfl_sync(0xffffffffu, th_lane, jj);
            if (d >= a.ndm)
                continue;
            const u64* trr = tr + (jj - pass0) * W;
            // lower segment: rel = wt * W + p - kf, time = tw - th - kf + p
            const int64_t tb = tw - th - kf;
            OutT* o = out + static_cast<int64_t>(d) * a.out_stride + tb;
            // p ranges owned by the block and inside [0, n_out), per segment
            int lo0 = wt == 0 ? kf : 0, lo1 = W;                                     // lower segment (seg = wt < 2NT - 1)
            int hi0 = 0, hi1 = wt == NT - 1 ? Hb - (2 * NT - 1) * W + kf : W;        // upper segment
            if (tb < 0)
                lo0 = lo0 > -tb ? lo0 : static_cast<int>(-tb < W ? -tb : W);
            if (tb + W > a.n_out)
                lo1 = a.n_out - tb > 0 ? static_cast<int>(a.n_out - tb) : 0;
            if (tb + hp < 0)
                hi0 = static_cast<int>(-(tb + hp) < W ? -(tb + hp) : W);
            if (tb + hp + hi1 > a.n_out)
                hi1 = a.n_out - tb - hp > 0 ? static_cast<int>(a.n_out - tb - hp) : 0;
            u64 v[T];
#pragma unroll
            for (int k = 0; k < T; ++k)
                v[k] = trr[lane_pinned + 32 * k];
            if (first) {
                // What the previous segment handed over for the slots that entered during the band (p < kf:
                // the first KF groups of 32 slots at most) is read first, so that the loads' latency hides
                // behind the stores of the other slots; everything else is plain predicated stores.
                constexpr int KF = (W / 4 + 31) / 32 < T ? (W / 4 + 31) / 32 : T;   // kf <= kmax <= W / 4
                OutT sl[KF], sh[KF];
#pragma unroll
                for (int k = 0; k < KF; ++k) {
                    const int p = lane_pinned + 32 * k;
                    sl[k] = p < kf && p >= lo0 && p < lo1 ? __ldcg(o + p) : OutT(0);
                    sh[k] = p < kf && p >= hi0 && p < hi1 ? __ldcg(o + p + hp) : OutT(0);
                }
#pragma unroll
                for (int k = T - 1; k >= 0; --k) {
                    const int p = lane_pinned + 32 * k;
                    OutT xl = to_out<OutT>(__uint_as_float(static_cast<unsigned>(v[k])));
                    OutT xh = to_out<OutT>(__uint_as_float(static_cast<unsigned>(v[k] >> 32)));
                    if (k < KF) {
                        xl += sl[k];
                        xh += sh[k];
                    }
                    if (p >= lo0 && p < lo1)
                        o[p] = xl;
                    if (p >= hi0 && p < hi1)
                        o[p + hp] = xh;
                    if (stats) {
                        // every output is stored by exactly one lane of one block: its statistics are
                        // taken here, on the final value, and cost no pass over the buffer
                        if (p >= lo0 && p < lo1) {
                            const double dl = static_cast<double>(xl) - pivot;
                            s1 += dl;
                            s2 = fma(dl, dl, s2);
                        }
                        if (p >= hi0 && p < hi1) {
                            const double dh = static_cast<double>(xh) - pivot;
                            s1 += dh;
                            s2 = fma(dh, dh, s2);
                        }
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < T; ++k) {
                    const int p = lane_pinned + 32 * k;
                    if (p >= lo0 && p < lo1)
                        put(o + p, __uint_as_float(static_cast<unsigned>(v[k])), false);
                    if (p >= hi0 && p < hi1)
                        put(o + p + hp, __uint_as_float(static_cast<unsigned>(v[k] >> 32)), false);
                }
            }
        }
        pass0 = j + 1;
        if (j + 1 < D)
            __syncwarp();  // the regions are rewritten by the next pass
    }
    if (stats) {
        // fixed order: lanes by shuffles, warps by index, blocks by the finishing kernel
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        }
        double* wsum = reinterpret_cast<double*>(smem + 128) + 2 * warp;   // the hand-over state is dead by now
        __syncwarp();
        if (lane_pinned == 0) {
            wsum[0] = s1;
            wsum[1] = s2;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NCW * 32) : "memory");
        if (tid == 0) {
            double b1 = 0.0, b2 = 0.0;
            const double* ws = reinterpret_cast<const double*>(smem + 128);
            for (int k = 0; k < NCW; ++k) {
                b1 += ws[2 * k];
                b2 += ws[2 * k + 1];
            }
            double* dst = a.stat_partial + (static_cast<int64_t>(beam) * a.stat_stride + a.stat_off + lin2) * 2;
            dst[0] = b1;
            dst[1] = b2;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// launcher
// ------------------------------------------------------------------------------------------------
bool window_fits_smem(const WindowPlan& wp) { return wp.ok && wp.nst >= 2; }

template <int T, int G, int NT, int D, typename OutT>
static int launch_bands(const WindowArgs& a, cudaStream_t st, int* launches)
{
    const int nst = a.nst, slot_bytes = a.slot_bytes;
    if (nst < 2)
        return static_cast<int>(cudaErrorInvalidConfiguration);
    const int stages_off = kWinFixedBytes;
    const size_t ring = static_cast<size_t>(nst) * (a.hdr_words * 4 + a.ch * slot_bytes);
    const size_t smem = static_cast<size_t>(stages_off) + ring;
    WindowArgs a2 = a;  // rows per flush pass: as many [NCW][W] u64 transposes as the ring holds
    a2.flush_rows = static_cast<int>(ring / (static_cast<size_t>(G) * NT * 32 * T * 8));
    a2.flush_rows = a2.flush_rows > D ? D : a2.flush_rows < 1 ? 1 : a2.flush_rows;
    cudaError_t e = cudaFuncSetAttribute(window_kernel<T, G, NT, D, OutT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess)
        return static_cast<int>(e);
    dim3 grid(static_cast<unsigned>(a.ntile_dm) * a.ntile_t, 1, a.nbeams);
    for (int b = 0; b < a.nband; ++b) {
        window_kernel<T, G, NT, D, OutT><<<grid, (G * NT + 4) * 32, smem, st>>>(a2, a.band[b], a.band[b + 1], b, a.stage0[b]);
        ++*launches;
        e = cudaGetLastError();
        if (e != cudaSuccess)
            return static_cast<int>(e);
    }
    return 0;
}

// instantiated geometries: (T, G, NT, D)
#define DEDISP_GEOMS(X) X(15, 6, 2, 4) X(15, 4, 3, 4) X(21, 4, 1, 4) X(21, 8, 1, 4) X(17, 4, 1, 5) X(15, 4, 1, 6) \
    X(11, 6, 2, 5) X(9, 6, 2, 6)

template <typename OutT> static int launch_geom(const WindowArgs& a, cudaStream_t st, int* launches)
{
    const WindowGeom& g = a.geom;
#define DEDISP_GEOM(t, gg, nt, dd) \
    if (g.T == t && g.G == gg && g.NT == nt && g.D == dd) \
        return launch_bands<t, gg, nt, dd, OutT>(a, st, launches);
    DEDISP_GEOMS(DEDISP_GEOM)
#undef DEDISP_GEOM
    return static_cast<int>(cudaErrorInvalidConfiguration);
}

bool window_geom_supported(const WindowGeom& g)
{
#define DEDISP_GEOM(t, gg, nt, dd) \
    if (g.T == t && g.G == gg && g.NT == nt && g.D == dd) \
        return true;
    DEDISP_GEOMS(DEDISP_GEOM)
#undef DEDISP_GEOM
    return false;
}

int launch_window(const WindowArgs& a, Elem in_t, void* stream, int* launches)
{
    if (a.n_out <= 0 || a.ndm <= 0)
        return 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    dim3 pgrid(static_cast<unsigned>((a.pair_stride / 2 + 255) / 256), a.nchans, a.nbeams);
    float2* pairs = static_cast<float2*>(a.pairs);
    const int hp = a.geom.NT * a.geom.W();
    if (a.ev0)
        cudaEventRecord(static_cast<cudaEvent_t>(a.ev0), st);
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
    if (a.ev_mid)
        cudaEventRecord(static_cast<cudaEvent_t>(a.ev_mid), st);
    const int rc = in_t == Elem::F32 ? launch_geom<float>(a, st, launches) : launch_geom<int32_t>(a, st, launches);
    if (a.ev1)
        cudaEventRecord(static_cast<cudaEvent_t>(a.ev1), st);
    return rc;
}

}  // namespace dedisp
