// Internal declarations shared by the translation units of libdedisp_b200.so.  Not part of the ABI.
#ifndef DEDISP_INTERNAL_H
#define DEDISP_INTERNAL_H

#include <cstdint>
#include <vector>

#include "../../include/dedisp.h"

namespace dedisp {

// ---- shift_table.cpp (host, -ffp-contract=off) ------------------------------------------------
bool build_shift_table(int nchans, double f_top, double df, double t_samp, const double* dm,
                       int ndm, std::vector<int32_t>& table, int64_t& max_delay);
void build_subband_tables(const std::vector<int32_t>& full, int nchans, int ndm, int nsub, int nfine,
                          const double* dm, std::vector<int32_t>& s1, std::vector<int32_t>& s2,
                          std::vector<double>& nominal, std::vector<int32_t>& maxshift2,
                          int64_t& max_delay);

// ---- one gather-and-add problem, as every kernel sees it ---------------------------------------
// out[b0][b1][d][t] = sum_{c < nchans} in[b0][b1][c][t + shift[b1][d][c]],  t < row_len(d)
// Brute force: nb1 = 1.  Subband stage 1: b1 = subband, d = coarse group.  Stage 2: b1 = coarse
// group, c = subband, d = fine trial.  b0 = beam.  All strides are in elements.
struct Problem {
    const void* in;
    void* out;
    const int32_t* shift;    // device
    const int32_t* row_extra;  // device [nb1][ndm] or nullptr: row (b1, d) has n_base + row_extra[b1][d] outputs
    int64_t row_extra_b1_stride;
    int64_t in_chan_stride, in_b0_stride, in_b1_stride;
    int64_t in_len;  // samples that may be read from one channel row
    int64_t out_dm_stride, out_b0_stride, out_b1_stride;
    int64_t shift_dm_stride, shift_b1_stride;
    int64_t n_out;   // outputs per row (the longest row when row_extra is given)
    int64_t n_base;  // see row_extra
    int nchans, ndm, nb0, nb1;
    int accumulate;  // 0: out = sum, 1: out += sum
};

enum class Elem { F32, U8, I32 };

// ---- kernels_*.cu -------------------------------------------------------------------------------
// Each returns the cudaError_t of the launch as int and adds the number of kernels launched to
// *launches.
int launch_naive(const Problem& p, Elem in_t, void* stream, int* launches);
// spread[k], k = 0,1,2: max over DM tiles of 32, 16, 8 rows and over channels of
// (max shift - min shift) inside a tile; decides how many rows share one staged copy.
int launch_direct(const Problem& p, Elem in_t, const int spread[3], void* stream, int* launches);

// kernels_long.cu: 16 rows x 2048 samples per block; spread16 as spread[1] above.  -1: does not fit.
int launch_long(const Problem& p, Elem in_t, int spread16, void* stream, int* launches);

// kernels_detect.cu: statistics, threshold, triplets.  partial: device workspace of
// nbeams * detect_blocks(ndm) * 2 doubles.
int detect_blocks(int ndm);
int launch_detect(const void* out, Elem t, int nbeams, int ndm, int64_t n, int64_t stride, double nsigma,
                  dedisp_event* events, int64_t capacity, dedisp_detect_result* res, double* partial, void* stream,
                  int* launches);

// fused variant: pivot[beam] = sum_c in[beam][c][0]; statistics from the partial sums the register-window
// kernel wrote (WindowArgs::stat_partial), then the threshold scan
int launch_detect_pivot(const void* in, Elem in_t, int nbeams, int nchans, int64_t chan_stride, double* pivot, void* stream,
                        int* launches);
int launch_detect_fused(const void* out, Elem t, int nbeams, int ndm, int64_t n, int64_t stride, double nsigma,
                        dedisp_event* events, int64_t capacity, dedisp_detect_result* res, const double* partial,
                        int64_t npart, int64_t part_stride, const double* pivot, void* stream, int* launches);

// kernels_front.cu: out[c][t] = |volt[t][c]|^2, strides in elements
int launch_power_corner_turn(const void* volt, void* out, int nchans, int64_t nsamp, int64_t volt_stride,
                             int64_t out_stride, void* stream);

int launch_bin(const void* in, void* out, int64_t nrows, int64_t nout, int64_t in_stride, int64_t out_stride, int nb,
               void* stream);

// kernels_microbench.cu: register-only FP32 add throughput
int launch_fadd_microbench(int packed, int iters, int nsm, float* sink, void* stream, double* adds);

// ---- register-window kernel (window_plan.cpp, kernels_window.cu) ---------------------------------
// Geometry: a consumer warp owns the D (4 or 8) DM rows of one
// row group; lane L owns the T consecutive "slots" L*T .. L*T+T-1 of each row, a slot being one
// pair of output samples (t, t + NT*W).  A block has G row groups x NT warps along time
// (+ 1 producer warp); the channel loop is cut into bands, one launch per band.
constexpr int kWinD = 6;            // most DM rows per thread (metadata word: 5 bits per mask)
constexpr int kWinMetaWords = 16;   // per (DM tile, channel) metadata, 64 bytes
constexpr int kWinWbBits = 11;
constexpr unsigned kWinShiftBits = 0x7fe0u;   // bits 5..14 of a channel word: the two row-shift masks
constexpr unsigned kWinStageShift = 0x8000u;  // bit 15: some channel of the stage this channel opens has a row shift
constexpr int kWinChMax = 12;       // most channels per pipeline stage (one mbarrier pair per stage)
constexpr int kWinFixedBytes = 128 + 16 * 128;  // shared memory in front of the ring: barriers + 16 consumer warps' hand-over state

struct WindowGeom {
    int T = 0;   // slots per lane and row (odd: conflict-free LDS.64)
    int G = 0;   // row groups per block (<= 8)
    int NT = 0;  // warps along time per row group
    int D = 8;   // DM rows per thread (row group): 8 with T <= 11, 4 with T <= 21
    int W() const { return 32 * T; }
    int rows() const { return D * G; }
};

struct WindowPlan {
    bool ok = false;
    WindowGeom geom;
    int Hb = 0;         // output samples per block and row: 2 * NT * W - kmax (blocks are Hb samples apart)
    int kmax = 0;       // largest number of row shifts of a row inside one band
    int lmax = 0;       // longest staged channel segment, in pairs
    // ring of the staged segments (sized at the end of build_window_plan): ch channels per pipeline stage,
    // nst >= 2 stages of { hdr_words header words, ch slots of slot_bytes }; nst = 0: the segments do not fit
    // shared memory.  The kernel stages with P = min(4, nst) producer warps, so a ring of 2 or 3 cannot be lapped.
    int ch = 0, nst = 0, slot_bytes = 0, hdr_words = 0;
    int ntile_dm = 0;
    int nband = 0;
    int theta_max = 0;  // largest band skew of a row
    int64_t maxbase = 0;        // largest staged-segment start (pairs, relative to the tile start)
    std::vector<int32_t> band;  // [nband + 1] channel boundaries
    // meta[tile][c] = { base, len, m[G], 0.. }: staged segment start / length in pairs (both even)
    // and, per row group, the channel's word: jitter bits (rows 1..5) | shift mask << 5 | 2nd shift
    // mask << 10 | kWinStageShift if a channel of the 4-channel stage this channel opens has a row
    // shift | window offset << 21
    std::vector<int32_t> meta;
    std::vector<int32_t> stage0;  // [nband + 1] first stage of every band in hdr
    // hdr[tile][stage][g * ch + c] = word of the channel AFTER channel c of that stage (0 past the
    // band's end): a consumer reads the next channel's word from the stage it is working on
    std::vector<int32_t> hdr;     // [tile][stage0[nband]][hdr_words]
    std::vector<int32_t> first;   // [tile][band][G] word of the band's first channel
    std::vector<int32_t> kfinal;  // [tile][band][rows] row shifts of every row at the band's end
    std::vector<int32_t> theta;   // [tile][band][rows] band skew of every row
};
// shift: host table [ndm][nchans].  Returns false (wp.ok = false) when the table does not fit the
// kernel's limits (non-monotone DMs, neighbouring trials drifting apart too fast, ...).
bool build_window_plan(const int32_t* shift, int ndm, int nchans, const WindowGeom& g, WindowPlan& wp);

struct WindowArgs {
    const void* in;       // [nbeams][nchans][in_stride]
    void* out;            // [nbeams][ndm][out_stride]
    void* pairs;          // scratch [nbeams][nchans][pair_stride] float2
    const int32_t* meta;  // device copies of WindowPlan::meta / kfinal / theta
    const int32_t* kfinal;
    const int32_t* theta;
    int64_t in_stride, out_stride, pair_stride, in_len, n_out;
    int nchans, ndm, nbeams, Hb, kmax, lmax, ntile_dm, ntile_t, nband, stage_total, theta_max;
    int ch, nst, slot_bytes, hdr_words;  // ring layout (WindowPlan)
    int flush_rows;  // rows per transpose pass of the flush (set by the launcher)
    int dm_group;  // DM tiles per block-order group (kernels_window.cu)
    const int32_t* band;    // HOST pointer, [nband + 1]
    const int32_t* stage0;  // HOST pointer, [nband + 1]
    const int32_t* hdr;     // device copy of WindowPlan::hdr
    const int32_t* first;   // device copy of WindowPlan::first
    const void* zeros;      // device, >= lmax pairs of zeros (segments of the padding channels)
    WindowGeom geom;
    // fused statistics of the outputs (band 0 of single-band plans only): per beam a pivot, per block two
    // fp64 partial sums at stat_partial[(beam * stat_stride + stat_off + block) * 2]; nullptr: off
    const double* pivot;
    double* stat_partial;
    int64_t stat_stride, stat_off;
    void *ev0, *ev1, *ev_mid;  // cudaEvent_t or nullptr: before the pair-forming pre-pass, after the last band launch, between the two
};
bool window_fits_smem(const WindowPlan& wp);
int64_t window_ntile_t(const WindowPlan& wp, int64_t n_out);
int64_t window_pair_stride(const WindowPlan& wp, int64_t n_out);  // float2 elements per channel row
int launch_window(const WindowArgs& a, Elem in_t, void* stream, int* launches);
WindowGeom window_default_geom();
int window_geom_preferences(WindowGeom* g, int max);  // shapes to try at plan creation, best first
bool window_geom_supported(const WindowGeom& g);  // one of the instantiated kernels

}  // namespace dedisp
#endif
