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

}  // namespace dedisp
#endif
