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
    const int32_t* row_extra;  // device [ndm] or nullptr: row d has n_base + row_extra[d] outputs
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

// ---- register-window kernel (window_plan.cpp, kernels_window.cu) ---------------------------------
// Geometry of the register-window kernel: a block owns kWinDB DM rows; warp (g, wt) owns the kWinD
// rows of row group g and lanes own kWinT consecutive "slots" each, a slot being one pair of output
// samples (t, t + H) of one row.  See DESIGN.md "Register-window kernel".
constexpr int kWinD = 8;                          // DM rows per thread
constexpr int kWinT = 10;                         // slots (sample pairs) per thread and row
constexpr int kWinNG = 4;                         // row groups per block
constexpr int kWinNT = 2;                         // warps along time per row group
constexpr int kWinDB = kWinD * kWinNG;            // 32 DM rows per block
constexpr int kWinNS = kWinNT * 32 * kWinT;       // 640 slots per row and block
constexpr int kWinNW = 14;                        // register window, in pairs
constexpr int kWinOMax = kWinNW - kWinT;          // largest row offset into the window (4)
constexpr int kWinMetaWords = 12;                 // per (DM tile, channel) metadata, 48 bytes

struct WindowPlan {
    bool ok = false;
    int H = 0;          // pairs (t, t+H): a block emits 2H samples per row
    int kmax = 0;       // largest accumulated row skew
    int lmax = 0;       // longest staged channel segment, in pairs
    int ntile_dm = 0;
    int64_t maxbase = 0;  // largest staged-segment start (in samples, relative to the tile start)
    // meta[tile][c] = { base, len, wb[4], om[4], mask2, 0 }: staged segment start/length (pairs),
    // per row group the window start (pairs, even) and 8 x 3-bit row offsets | shift mask << 24;
    // mask2: a second shift of the same channel, one byte per row group
    std::vector<int32_t> meta;
    std::vector<int32_t> kfinal;  // [tile][32] final skew of every row
};
// shift: host table [ndm][nchans].  Returns false (wp.ok = false) when the table does not fit the
// kernel's limits (non-monotone DMs, skew growing by more than one sample per channel, ...).
bool build_window_plan(const int32_t* shift, int ndm, int nchans, WindowPlan& wp);

struct WindowArgs {
    const void* in;       // [nbeams][nchans][in_stride]
    void* out;            // [nbeams][ndm][out_stride]
    void* pairs;          // scratch [nbeams][nchans][pair_stride] float2
    const int32_t* meta;  // device copies of WindowPlan::meta / kfinal
    const int32_t* kfinal;
    int64_t in_stride, out_stride, pair_stride, in_len, n_out;
    int nchans, ndm, nbeams, H, lmax, ntile_dm, ntile_t;
};
bool window_fits_smem(int lmax);  // the staging ring needs >= 8 slots of shared memory
int64_t window_pair_stride(const WindowPlan& wp, int64_t n_out);  // float2 elements per channel row
int launch_window(const WindowArgs& a, Elem in_t, void* stream, int* launches);

}  // namespace dedisp
#endif
