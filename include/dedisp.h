/*
 * dedisp.h -- C ABI of the B200 (sm_100a) incoherent de-dispersion library.
 *
 * The operation is the hot path of Magro et al., "Real-time, fast radio transient searches with
 * GPU de-dispersion" (arXiv 1107.2516); citations are PAPER.md:<line>.
 *
 *   brute force   out[d][t] = sum_c in[c][t + shift(c,d)]
 *   shift(c,d)    = round(4.15e6 ms * (f_c^-2 - f_top^-2) * DM_d / t_samp)  (eq. 1)
 *   two-stage     sub[k][s][t] = sum_{c in subband s} in[c][t + s1(c,k)]
 *                 out[d][t]    = sum_s sub[k(d)][s][t + s2(d,s)]
 *   streaming     the last max_delay samples of every channel are carried from one chunk to
 *                 the next ("n_samp + maxshift" samples per buffer)
 *
 * Conventions
 *   - Plain C types only.  Every pointer is marked HOST or DEVICE.  DEVICE pointers are CUDA
 *     device pointers of the current device, owned by the caller; the library never frees or
 *     reallocates them.  Plans, their device tables, the subband scratch and the streaming carry
 *     buffers are owned by the library and released by the matching *_destroy.
 *   - Data layout: input is channel-major and time-contiguous, channel 0 is the
 *     highest frequency f_top, channel c is at f_top - c*df.  Batches ("beams") are outermost.
 *   - dedisp_execute / dedisp_stream_push / dedisp_plan_detect enqueue work on the given
 *     cudaStream_t and return without synchronising, allocating or freeing: device tables and
 *     scratch are set up beforehand by dedisp_plan_reserve (blocking).  Argument errors are
 *     reported synchronously; a CUDA launch error is reported as DEDISP_ECUDA by the call that
 *     saw it.  The *_host entries and *_create / *_reserve / *_destroy may allocate and block.
 *   - A plan's tables are immutable after creation.  Its scratch (pair buffer, subband
 *     intermediate, detection workspace) and its bookkeeping (last_launches, timing events) are
 *     per plan: ONE execute / push / detect per plan may be in flight at a time, for both kinds
 *     of plan, and calls on one plan must not be made from several threads at once.  Use one
 *     plan per CUDA stream for concurrent work.  A plan lives on the device that was current at
 *     its first dedisp_plan_reserve.
 *   - No exceptions cross this boundary, nothing calls exit(), the library reads no environment
 *     variables and keeps no global state -- with one exception, the fixed device array behind
 *     dedisp_detect_static (described there).
 *   - There is no CPU fallback: without a CUDA device every execute/push returns DEDISP_ECUDA.
 *     Plan creation and the table getters are host-only and work without a device.
 */
#ifndef DEDISP_H
#define DEDISP_H

#include <stdint.h>

#if defined(__GNUC__)
#define DEDISP_API __attribute__((visibility("default")))
#else
#define DEDISP_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dedisp_plan dedisp_plan;     /* opaque, library-owned */
typedef struct dedisp_stream dedisp_stream; /* opaque, library-owned */

typedef enum {
    DEDISP_OK = 0,
    DEDISP_EINVAL = 1, /* bad scalar argument / NULL pointer / bad DM list               */
    DEDISP_ENOMEM = 2, /* host or device allocation failed                                */
    DEDISP_ECUDA = 3,  /* CUDA runtime error (no device, launch failure, ...)             */
    DEDISP_ESHAPE = 4, /* strides / lengths inconsistent with the plan                    */
    DEDISP_ESTATE = 5, /* call not valid for this plan / stream, or no covering reservation   */
    DEDISP_ELIMIT = 6  /* larger than the fixed scratch of an allocation-free entry point     */
} dedisp_status;

typedef enum {
    DEDISP_F32 = 0, /* float input, float output (fp32 adds)                               */
    DEDISP_U8 = 1   /* uint8 input (0..255, no offset removed), int32 output, exact       */
} dedisp_dtype;

/* Kernel choice for dedisp_plan_set_kernel.  AUTO picks, for brute-force plans, the register-window
 * kernel when the plan's shift table fits its limits and the problem fills the device (see
 * dedisp_plan_resolved_kernel); otherwise, and for both stages of subband plans, the long-tile kernel
 * (rows of >= 4096 samples) or the direct kernel (shorter rows). */
typedef enum {
    DEDISP_KERNEL_AUTO = 0,
    DEDISP_KERNEL_NAIVE = 1,  /* one thread per output sample, global loads only (AUTO's choice for tiny problems) */
    DEDISP_KERNEL_DIRECT = 2, /* shared-memory staged, register-blocked DMs x time           */
    DEDISP_KERNEL_WINDOW = 3, /* + one register window shared by the DM rows of a thread     */
    DEDISP_KERNEL_LONG = 4    /* 16 rows x 2048 samples per block, TMA-staged channel unions  */
} dedisp_kernel;

/*
 * dedisp_plan_create -- build the integer shift table(s) of eq. 1 on the host.
 *
 *   nchans      number of frequency channels (> 0)
 *   f_top_mhz   frequency of channel 0, the highest, in MHz (> 0)
 *   df_mhz      magnitude of the channel width in MHz (> 0); f_c = f_top - c*df must stay > 0
 *   t_samp_ms   sampling time in ms (> 0)
 *   dm_list     HOST, ndm doubles, pc cm^-3, finite and >= 0; copied
 *   ndm         number of DM trials (> 0)
 *   nsub        0: brute-force plan.  > 0: two-stage subband plan with nsub subbands of
 *               nchans/nsub consecutive channels (nchans % nsub == 0)
 *   nfine       subband plans only: dm_list is ndm/nfine consecutive groups of nfine trials
 *               (ndm % nfine == 0, dm_list non-decreasing); group k is partially de-dispersed at
 *               its nominal DM dm_list[k*nfine + nfine/2].  Ignored when nsub == 0.
 *
 * shift(c,d) = (int32) floor(x + 0.5), x evaluated in IEEE fp64, every operation rounded on its
 * own, in this order:  f_c = f_top - (double)c*df;  a_c = 1/(f_c*f_c) - 1/(f_top*f_top);
 * k_c = 4.15e6*a_c;  x = (k_c*DM_d)/t_samp.
 * Subband tables: s1(c,k) = shift(c,D_k) - shift(ctop(s),D_k), s2(d,s) = shift(ctop(s),DM_d),
 * ctop(s) = s*nchans/nsub.
 *
 * On success *plan is a new plan.  Errors: DEDISP_EINVAL (any rule above violated, a shift that
 * does not fit int32), DEDISP_ENOMEM.  *plan is NULL on error.
 */
DEDISP_API dedisp_status dedisp_plan_create(dedisp_plan **plan, int nchans, double f_top_mhz, double df_mhz,
                                 double t_samp_ms, const double *dm_list, int ndm, int nsub,
                                 int nfine);

/* Releases the plan, its device tables and scratch.  NULL is accepted.  Streams created from the
 * plan must be destroyed first. */
DEDISP_API dedisp_status dedisp_plan_destroy(dedisp_plan *plan);

/* Number of extra input samples per channel the caller must supply beyond nsamp_out
 * ("maxshift"): the maximum of the integer table (brute force) or of s1+s2
 * (subband).  -1 if plan is NULL. */
DEDISP_API int64_t dedisp_plan_max_delay(const dedisp_plan *plan);

/* Scalar properties; -1 if plan is NULL. */
DEDISP_API int dedisp_plan_nchans(const dedisp_plan *plan);
DEDISP_API int dedisp_plan_ndm(const dedisp_plan *plan);
DEDISP_API int dedisp_plan_nsub(const dedisp_plan *plan);
DEDISP_API int dedisp_plan_nfine(const dedisp_plan *plan);

/* Copies the full-band table shift[ndm][nchans] (row d = DM trial d) to HOST memory.
 * Valid for both kinds of plan (for subband plans it is the table s1/s2 derive from). */
DEDISP_API dedisp_status dedisp_plan_get_shifts(const dedisp_plan *plan, int32_t *host_out);

/* Subband plans: s1 [ncoarse][nchans], s2 [ndm][nsub], nominal_dm [ncoarse],
 * maxshift2 [ncoarse] (overlap stage 1 keeps for stage 2; one argument more than
 * SURVEY.md section 8b's sketch of this call); all HOST; any may be NULL.  DEDISP_ESTATE for
 * brute-force plans. */
DEDISP_API dedisp_status dedisp_plan_get_subband_shifts(const dedisp_plan *plan, int32_t *s1, int32_t *s2,
                                             double *nominal_dm, int32_t *maxshift2);

/* Selects the brute-force kernel (default DEDISP_KERNEL_AUTO).  DEDISP_EINVAL for an unknown
 * value, DEDISP_ESTATE if WINDOW is forced on a plan whose table exceeds its limits.  Scratch is
 * sized for the kernel selected at the time of dedisp_plan_reserve: after changing the kernel call
 * dedisp_plan_reserve again (an execute that lacks its scratch returns DEDISP_ESTATE). */
DEDISP_API dedisp_status dedisp_plan_set_kernel(dedisp_plan *plan, dedisp_kernel kernel);

/* Which kernel AUTO resolves to for this plan and dtype (a dedisp_kernel value), -1 on error.  This is
 * the choice for problems that fill the device; an execute whose (trials x samples x beams) yields fewer
 * register-window tiles than the device has SMs runs the naive kernel (below 8192 outputs per SM) or the
 * direct kernel instead. */
DEDISP_API int dedisp_plan_resolved_kernel(const dedisp_plan *plan, dedisp_dtype dtype);

/* The kernel the last execute / push on this plan actually ran (a dedisp_kernel value other than AUTO;
 * subband plans: the kernel of stage 1), -1 before the first execute or if plan is NULL.  Unlike
 * dedisp_plan_resolved_kernel this reflects AUTO's size rule.  The *_host entries apply that rule once,
 * to the length of the whole buffer, so all time pieces of one buffer run the same kernel. */
DEDISP_API int dedisp_plan_last_kernel(const dedisp_plan *plan);

/* Geometry the register-window kernel would use for this plan, 14 int64 to HOST memory:
 * [0] 1 if the plan's table fits the kernel (else the rest is 0), [1] Hb: output samples per
 * block and DM row (blocks are Hb apart in time), [2] kmax: largest number of row shifts in a
 * channel band = samples a block loses, Hb = 2*NT*W - kmax, [3] longest staged channel segment
 * in pairs, [4] DM tiles, [5] W: slots per row and warp segment, [6] DM rows per block,
 * [7] channel bands (= kernel launches), [8] T, [9] G, [10] NT, [11] D (below), [12] channels per
 * pipeline stage and [13] stages of the shared-memory ring the staged segments go through.
 * Brute-force plans only carry one. */
DEDISP_API dedisp_status dedisp_plan_window_info(const dedisp_plan *plan, int64_t *info);

/* Tuning knob: thread / block shape of the register-window kernel.  A thread owns D DM rows x T
 * sample pairs, a block G row groups x NT warps along time.  Only the instantiated shapes are
 * accepted (DEDISP_EINVAL otherwise): (T,G,NT,D) = (15,4,3,4) [default where it fits], (15,6,2,4), (21,4,1,4),
 * (21,8,1,4), (17,4,1,5), (15,4,1,6), (11,6,2,5), (9,6,2,6).  Brute-force plans, before the first
 * dedisp_plan_reserve (DEDISP_ESTATE otherwise, or when the table does not fit the shape: the
 * plan then keeps the shape it had).  Results do not depend on it beyond fp32 summation order. */
DEDISP_API dedisp_status dedisp_plan_set_window_geometry(dedisp_plan *plan, int T, int G, int NT, int D);

/*
 * dedisp_plan_reserve -- copy the plan's tables to the current device (first call) and size its
 * scratch for executes / pushes / detects of up to nsamp_out output samples and nbeams beams of
 * dtype: the pair buffer of the register-window kernel (2 x 4 bytes per input sample), the subband
 * intermediate (dedisp_plan_scratch_bytes), the detection workspace.  Blocking (cudaMalloc,
 * cudaMemcpy); may be called again with a larger shape while nothing is in flight.  Must precede
 * dedisp_execute / dedisp_plan_detect; dedisp_stream_create and the *_host entries call it
 * themselves.  Errors: DEDISP_EINVAL, DEDISP_ENOMEM, DEDISP_ECUDA, DEDISP_ESTATE (the plan lives
 * on another device).
 */
DEDISP_API dedisp_status dedisp_plan_reserve(dedisp_plan *plan, dedisp_dtype dtype, int64_t nsamp_out, int nbeams);

/* Bytes of device scratch a subband execute of nsamp_out samples and nbeams beams needs
 * (the stage-1 intermediate, fp32 or int32); 0 for brute-force plans; -1 on error. */
DEDISP_API int64_t dedisp_plan_scratch_bytes(const dedisp_plan *plan, int64_t nsamp_out, int nbeams);

/*
 * dedisp_execute -- de-disperse one resident buffer.
 *
 *   in          DEVICE, [nbeams][nchans][in_stride] elements of dtype's input type (float or
 *               uint8); in_stride >= nsamp_out + max_delay; for DEDISP_F32 the pointer and
 *               in_stride*4 must be multiples of 16 bytes, for DEDISP_U8 of 16 bytes as well
 *   out         DEVICE, [nbeams][ndm][out_stride] float (F32) or int32 (U8); out_stride >=
 *               nsamp_out; pointer 16-byte aligned and out_stride a multiple of 4
 *   nsamp_out   output samples per DM trial (>= 0; 0 is a no-op)
 *   cuda_stream a cudaStream_t (NULL = the legacy default stream)
 *
 * Brute-force plans: the register-window kernel (a pair-forming pre-pass into plan-owned scratch,
 * then one launch per channel band) or one long-tile / direct launch.  Subband plans: stage 1
 * into the plan's scratch, then stage 2; stage 1 forms of every (group, subband) series only the
 * samples stage 2 reads.  Input elements beyond nsamp_out + max_delay in a row are never read;
 * output elements beyond nsamp_out in a row are never written.  Asynchronous: no allocation, no
 * synchronisation.  Errors: DEDISP_EINVAL, DEDISP_ESHAPE, DEDISP_ECUDA, DEDISP_ESTATE (no
 * dedisp_plan_reserve covering dtype / nsamp_out / nbeams, or another device is current).
 */
DEDISP_API dedisp_status dedisp_execute(dedisp_plan *plan, const void *in, void *out, dedisp_dtype dtype,
                             int64_t nsamp_out, int64_t in_stride, int64_t out_stride, int nbeams,
                             void *cuda_stream);

/*
 * Host-buffer convenience: same operation with HOST in/out ([nbeams][nchans][nsamp_out+max_delay]
 * dense input, [nbeams][ndm][nsamp_out] dense output).  Allocates device buffers (kept by the
 * plan), copies in, executes, copies out and synchronises the stream.  Brute-force plans with
 * nsamp_out >= 65536 are cut into up to 8 time pieces whose H2D copy, kernels and D2H copy overlap
 * on two plan-owned copy streams (pinned host memory is needed for the overlap, not for
 * correctness).  This is the "end-to-end" entry bench.py times; every arithmetic step still runs
 * in the CUDA kernels.
 */
DEDISP_API dedisp_status dedisp_execute_host(dedisp_plan *plan, const void *host_in, void *host_out,
                                  dedisp_dtype dtype, int64_t nsamp_out, int nbeams,
                                  void *cuda_stream);

/*
 * Streaming chunk driver.  The stream owns a DEVICE work buffer
 * [nbeams][nchans][max_delay + chunk] whose first max_delay samples per channel are the tail of
 * the previous chunks (zeros before the first push).  Push k (k = 0, 1, ...) consumes stream
 * samples [k*chunk, (k+1)*chunk) and produces outputs for stream times
 * [k*chunk - max_delay, (k+1)*chunk - max_delay); outputs at negative times are warm-up values.
 * The concatenation of all pushes equals one dedisp_execute over the whole stream, also when
 * max_delay > chunk.  Brute-force plans only (DEDISP_ESTATE otherwise).
 *
 *   chunk_in    DEVICE, [nbeams][nchans][chunk] dense
 *   out         DEVICE, [nbeams][ndm][chunk] dense
 */
DEDISP_API dedisp_status dedisp_stream_create(dedisp_stream **s, dedisp_plan *plan, dedisp_dtype dtype,
                                   int64_t chunk, int nbeams);
DEDISP_API dedisp_status dedisp_stream_push(dedisp_stream *s, const void *chunk_in, void *out,
                                 void *cuda_stream);
/* Same with HOST chunk_in/out (pinned or pageable): the chunk is copied straight behind the carry
 * in up to 8 time pieces whose H2D copy, kernels and D2H copy overlap; synchronises the stream. */
DEDISP_API dedisp_status dedisp_stream_push_host(dedisp_stream *s, const void *host_chunk_in, void *host_out,
                                      void *cuda_stream);
/* Resets the carry to zeros (asynchronously on cuda_stream). */
DEDISP_API dedisp_status dedisp_stream_reset(dedisp_stream *s, void *cuda_stream);
DEDISP_API dedisp_status dedisp_stream_destroy(dedisp_stream *s);

/* Largest chunk (output samples per push) such that work buffer + output fit in mem_bytes of
 * device memory: the paper's eq. 3,
 * n_samp = (memory - maxshift*n_chans*in_size) / (n_dms*out_size + n_chans*in_size), per beam.
 * Returns <= 0 if nothing fits; -1 on bad arguments. */
DEDISP_API int64_t dedisp_plan_max_chunk(const dedisp_plan *plan, dedisp_dtype dtype, int64_t mem_bytes,
                              int nbeams);

/* Number of kernels the last execute/push on this plan launched (bench.py's gpu_launches). */
DEDISP_API int dedisp_plan_last_launches(const dedisp_plan *plan);

/* Timing for roofline reports.  With timing on, every execute / push records CUDA events on the
 * caller's stream around ALL the kernels it launches (register-window path: the pair-forming pre-pass
 * and the band launches) and one between its two parts.  dedisp_plan_last_kernel_ms waits for the last
 * event and returns the elapsed milliseconds of the last execute; DEDISP_ESTATE if timing was off.
 * Off by default (no events, no overhead). */
DEDISP_API dedisp_status dedisp_plan_set_timing(dedisp_plan *plan, int on);
DEDISP_API dedisp_status dedisp_plan_last_kernel_ms(dedisp_plan *plan, float *ms);
/* The two parts of the last execute, timing on; HOST, 2 floats.  Subband plans: ms[0] = stage 1
 * (partial sums inside subbands), ms[1] = stage 2 (across subbands).  Brute-force
 * plans on the register-window kernel: ms[0] = pair-forming pre-pass, ms[1] = band launches.
 * DEDISP_ESTATE when timing was off or the last execute took another path. */
DEDISP_API dedisp_status dedisp_plan_last_stage_ms(dedisp_plan *plan, float *ms);

/*
 * Event detection on a de-dispersed buffer ("calculate the mean and standard deviation
 * for the entire processed buffer, and use these values to apply a threshold at a particular
 * multiple of the standard deviation.  All values above the threshold are output ... as a list of
 * triplets of the form (time, DM, intensity)").  Per beam: mean and POPULATION standard deviation of
 * all ndm*nsamp_out outputs in fp64, threshold = mean + nsigma*sigma, events = outputs strictly
 * above it.
 *
 *   out        DEVICE, [nbeams][ndm][out_stride] float (DEDISP_F32) or int32 (DEDISP_U8), as written
 *              by dedisp_execute; 16-byte aligned, out_stride a multiple of 4
 *   events     DEVICE, [nbeams][capacity]; the first min(count, capacity) entries of a beam are
 *              valid, in no particular order
 *   results    DEVICE, [nbeams]; count is the number of outputs above the threshold (it may exceed
 *              capacity: the surplus is counted, not stored)
 * Asynchronous on cuda_stream; the plan owns a small workspace sized by dedisp_plan_reserve (one
 * detect per plan in flight).  Errors: DEDISP_EINVAL, DEDISP_ESHAPE, DEDISP_ECUDA, DEDISP_ESTATE
 * (no dedisp_plan_reserve for this many beams).
 */
typedef struct { int64_t t; int32_t dm; float value; } dedisp_event;            /* 16 bytes */
typedef struct { double mean, sigma, threshold; int64_t count; } dedisp_detect_result;
DEDISP_API dedisp_status dedisp_plan_detect(dedisp_plan *plan, const void *out, dedisp_dtype dtype,
                                            int64_t nsamp_out, int64_t out_stride, int nbeams, double nsigma,
                                            dedisp_event *events, int64_t capacity,
                                            dedisp_detect_result *results, void *cuda_stream);

/*
 * dedisp_detect_static -- the event detection of dedisp_plan_detect (same kernels, same
 * definition of mean / sigma / threshold / events, same summation order, hence the same numbers) for
 * callers that cannot let the library allocate device memory.
 *
 * Who that is.  dedisp_plan_detect keeps its per-block partial sums in a workspace that
 * dedisp_plan_reserve obtains with cudaMalloc.  Two kinds of user cannot afford that call:
 *   - the processing thread of a real-time backend (the paper's pipeline): cudaMalloc
 *     and cudaFree serialise on a driver lock, and replacing a workspace by a larger one frees the old
 *     one, which waits for the whole device to go idle -- the copy stream that is receiving the next
 *     buffer from the telescope included -- so a reservation that grows in the middle of an observation
 *     costs samples;
 *   - a host application that claimed the whole of the GPU's memory for its own ring buffers or pool
 *     when it started: whatever the library asks the driver for afterwards simply fails.
 * This entry needs no plan and no reserve.  Its only scratch is an array of
 * DEDISP_DETECT_STATIC_MAX_SLOTS x 16 bytes (296 KiB) that is compiled into the library: every GPU on
 * which the process uses the library holds one copy from the moment the module is loaded until the
 * process ends, whether or not this function is ever called.  The caller supplies everything else.
 *
 *   out, dtype, nsamp_out, out_stride, nbeams, nsigma, events, capacity, results
 *              exactly as for dedisp_plan_detect (all DEVICE pointers, caller-owned)
 *   ndm        DM trials (rows) per beam in `out` (> 0); the plan is not needed for anything else
 *
 * Limit: nbeams * min(ndm, 1184) <= DEDISP_DETECT_STATIC_MAX_SLOTS (18944: e.g. 16 beams of any number
 * of trials, or 74 beams of 256 trials).  Anything larger returns DEDISP_ELIMIT before the device is
 * touched; the array is never enlarged.  dedisp_detect_static_max_slots() returns the same constant for
 * callers that do not compile against this header.
 *
 * First call on a device: the library asks the runtime for the device address of the array
 * (cudaGetSymbolAddress, under a mutex, result cached per device).  That look-up may make the runtime
 * load the library's device code, so make the first call on each GPU during start-up, with that GPU
 * current, and before any stream capture is begun.  Later calls only launch three kernels on
 * cuda_stream; no call ever runs cudaMalloc, cudaFree or an allocating library routine, and none
 * synchronises.
 *
 * Sharing: all calls on one GPU, from every thread and stream, use the same array, and it keeps
 * whatever the previous call wrote.  Nothing in it needs to be zero on entry -- a call overwrites every
 * slot before it reads it -- but two calls that run on the GPU at the same time (different streams with
 * no ordering between them) overwrite each other's sums and return wrong statistics.  Order such calls
 * on one stream or with events.
 *
 * Errors: DEDISP_EINVAL, DEDISP_ESHAPE (as dedisp_plan_detect), DEDISP_ELIMIT, DEDISP_ECUDA (no device,
 * more than 64 devices, the address look-up or a launch failed).
 */
#define DEDISP_DETECT_STATIC_MAX_SLOTS 18944
DEDISP_API dedisp_status dedisp_detect_static(const void *out, dedisp_dtype dtype, int ndm, int64_t nsamp_out,
                                              int64_t out_stride, int nbeams, double nsigma, dedisp_event *events,
                                              int64_t capacity, dedisp_detect_result *results, void *cuda_stream);
DEDISP_API int64_t dedisp_detect_static_max_slots(void);

/*
 * De-dispersion and event detection in one call (PAPER.md:76 is the step right after the hot path).
 * Arguments as dedisp_execute followed by those of dedisp_plan_detect; `out` still receives the whole
 * de-dispersed buffer.  For brute-force plans that run on the register-window kernel with a single
 * channel band, the kernel's flush accumulates the statistics (fp64 sums of x - pivot and (x - pivot)^2,
 * pivot = sum_c in[c][0], reduced in a fixed order), so detection costs ONE pass over the buffer (the
 * threshold scan) instead of two; other plans run dedisp_execute followed by dedisp_plan_detect.  Same
 * definition of mean / sigma / threshold / events either way.  Asynchronous; needs dedisp_plan_reserve.
 */
DEDISP_API dedisp_status dedisp_execute_detect(dedisp_plan *plan, const void *in, void *out, dedisp_dtype dtype,
                                               int64_t nsamp_out, int64_t in_stride, int64_t out_stride, int nbeams,
                                               double nsigma, dedisp_event *events, int64_t capacity,
                                               dedisp_detect_result *results, void *cuda_stream);
/*
 * Events-only end-to-end entry: HOST input as for dedisp_execute_host, HOST events [nbeams][capacity]
 * and HOST results [nbeams].  The input goes to the device in time pieces that overlap the kernels, the
 * de-dispersed buffer stays on the device (plan-owned), and only min(count, capacity) triplets and 32
 * bytes of statistics per beam come back -- instead of nbeams*ndm*nsamp_out*4 bytes.  Allocates
 * plan-owned device buffers, synchronises the stream.
 */
DEDISP_API dedisp_status dedisp_execute_detect_host(dedisp_plan *plan, const void *host_in, dedisp_dtype dtype,
                                                    int64_t nsamp_out, int nbeams, double nsigma,
                                                    dedisp_event *host_events, int64_t capacity,
                                                    dedisp_detect_result *host_results, void *cuda_stream);

/*
 * Copies the de-dispersed buffer that the last dedisp_execute_host / dedisp_execute_detect_host call on
 * this plan left on the device (plan-owned; the events-only entry never sends it to the host, so this is
 * the way to look at the data behind its events) to dst: DEVICE, dense [nbeams][ndm][nsamp_out] float
 * (DEDISP_F32) or int32 (DEDISP_U8) of that call; `bytes` must be exactly its size (DEDISP_ESHAPE
 * otherwise).  Asynchronous on cuda_stream.  DEDISP_ESTATE if no host entry has run on the plan.
 */
DEDISP_API dedisp_status dedisp_plan_copy_host_output(dedisp_plan *plan, void *dst, int64_t bytes, void *cuda_stream);

/*
 * Power + corner turn, the two steps before de-dispersion in the paper's real-time pipeline
 * ("(iii) channelizes and calculates total power (iv) transposes data so that it is
 * in channel order"; Table 6).  One fused kernel:
 *     out[c][t] = re(volt[t][c])^2 + im(volt[t][c])^2     (fp32, each operation rounded on its own)
 *   volt   DEVICE, [nsamp][volt_stride] interleaved (re, im) float pairs, spectrum order, one
 *          polarisation; volt_stride >= nchans (in complex elements); 8-byte aligned
 *   out    DEVICE, [nchans][out_stride] float, the channel-major layout dedisp_execute reads;
 *          out_stride >= nsamp
 * Asynchronous on cuda_stream.  Errors: DEDISP_EINVAL, DEDISP_ESHAPE, DEDISP_ECUDA.
 */
DEDISP_API dedisp_status dedisp_power_corner_turn(const void *volt, void *out, int nchans, int64_t nsamp,
                                                  int64_t volt_stride, int64_t out_stride, void *cuda_stream);

/*
 * Binning, stage (i) of the paper's subband scheme ("Binning averages N_b consecutive
 * samples"; eq. 6): out[r][j] = (in[r][j*nb] + ... + in[r][j*nb + nb-1]) / nb for j < nsamp / nb
 * (a ragged tail is dropped), fp32, the sum left to right, every operation rounded on its own.
 * A survey pass with bin factor b (Table 1) is this call followed by a plan created with
 * t_samp * b.
 *   in     DEVICE, [nrows][in_stride] float (nrows = nbeams * nchans); in_stride >= nsamp
 *   out    DEVICE, [nrows][out_stride] float; out_stride >= nsamp / nb; must not overlap in
 * Asynchronous on cuda_stream.  Errors: DEDISP_EINVAL, DEDISP_ESHAPE, DEDISP_ECUDA.
 */
DEDISP_API dedisp_status dedisp_bin(const void *in, void *out, int64_t nrows, int64_t nsamp, int64_t in_stride,
                                    int64_t out_stride, int nb, void *cuda_stream);

/*
 * Multi-pass subband survey ("each pass will bin the data using a different binning
 * factor ... For each pass the DM range is partitioned, each range being dSub_DM apart"; the three
 * stages of PAPER.md:137-143; Tables 1 and 4).  Pass i covers the trials dm_low + d*dm_step,
 * d = 0 .. ndm-1 (one multiply and one add in fp64), in groups of nfine = dSub_DM / dDM trials around a
 * nominal DM, on the input binned by `bin`.  Per pass, on the device and without a round trip to the
 * host: (i) dedisp_bin by `bin` (skipped for bin 1), (ii) subband stage 1 and
 * (iii) stage 2 of a subband plan created with t_samp * bin (dedisp_plan_create with nsub, nfine).
 *
 * A survey over nsamp input samples per channel needs nsamp + dedisp_survey_max_delay samples
 * (= max over passes of bin * max_delay of the pass's plan, in unbinned samples; R17) and
 * yields nsamp / bin outputs per trial of a pass (eq. 8).
 *
 *   in     DEVICE float [nbeams][nchans][in_stride], in_stride >= nsamp + max_delay, a multiple of 4,
 *          16-byte aligned
 *   out    DEVICE float, dedisp_survey_out_layout's `total` elements: pass i is the dense block
 *          [nbeams][ndm_i][stride_i] at element offset_i, nout_i = nsamp / bin_i valid samples per row
 * dedisp_survey_reserve (blocking) sizes the plans' scratch and the binned buffer; dedisp_survey_execute
 * is asynchronous on cuda_stream and returns DEDISP_ESTATE without a covering reserve.  fp32 input only.
 * One execute per survey in flight.  dedisp_survey_pass_plan lends pass i's plan for the table getters
 * (do not destroy it).
 */
typedef struct dedisp_survey dedisp_survey; /* opaque, library-owned */
typedef struct { double dm_low, dm_step; int ndm, nfine, bin; } dedisp_pass;
DEDISP_API dedisp_status dedisp_survey_create(dedisp_survey **survey, int nchans, double f_top_mhz, double df_mhz,
                                              double t_samp_ms, int nsub, const dedisp_pass *passes, int npass);
DEDISP_API dedisp_status dedisp_survey_destroy(dedisp_survey *survey);
DEDISP_API int dedisp_survey_npass(const dedisp_survey *survey);
DEDISP_API int64_t dedisp_survey_max_delay(const dedisp_survey *survey);
DEDISP_API const dedisp_plan *dedisp_survey_pass_plan(const dedisp_survey *survey, int pass);
/* HOST arrays of npass int64 (any may be NULL) and the total element count of `out`. */
DEDISP_API dedisp_status dedisp_survey_out_layout(const dedisp_survey *survey, int64_t nsamp, int nbeams, int64_t *offset,
                                                  int64_t *stride, int64_t *nout, int64_t *total);
DEDISP_API dedisp_status dedisp_survey_reserve(dedisp_survey *survey, int64_t nsamp, int nbeams);
DEDISP_API dedisp_status dedisp_survey_execute(dedisp_survey *survey, const void *in, void *out, int64_t nsamp,
                                               int64_t in_stride, int nbeams, void *cuda_stream);
DEDISP_API int dedisp_survey_last_launches(const dedisp_survey *survey);

/*
 * Register-only FP32 add microbenchmark: the measured denominator of the brute-force roofline.  The
 * method is nchans adds per output sample ("N_c additions"), so its ceiling is the
 * rate at which the SMs add when no operand comes from memory (nominally
 * 128 adds per clock and SM).  Launches, on every SM, 32 warps whose threads each add a loop-invariant
 * operand to 64 independent fp32 accumulators `iters` times -- as 32 packed add.rn.f32x2 (packed != 0:
 * the instruction the register-window kernel uses) or 64 scalar add.rn.f32 -- `repeats` times after one
 * warm-up launch, and times them with CUDA events on cuda_stream.
 *   ms      HOST, elapsed milliseconds of the `repeats` launches
 *   adds    HOST, fp32 additions they executed
 *   nsm     HOST or NULL, number of SMs of the current device
 * Synchronises the stream, allocates 64 bytes for the call.  Errors: DEDISP_EINVAL, DEDISP_ECUDA.
 */
DEDISP_API dedisp_status dedisp_fadd_microbench(int packed, int iters, int repeats, float *ms, double *adds, int *nsm,
                                                void *cuda_stream);

/* Static string for a status code. */
DEDISP_API const char *dedisp_strerror(dedisp_status status);

/* Library version string, e.g. "dedisp-b200 0.1 (sm_100a)". */
DEDISP_API const char *dedisp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DEDISP_H */
