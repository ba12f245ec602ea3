/*
 * dd.h -- C ABI of the B200-native direct incoherent dedispersion library (libdd_b200.so).
 *
 * The operation is the paper's *direct* dedispersion transform (arXiv:1201.5380; citations are
 * /root/reference/PAPER.md line numbers):
 *
 *     D[d][t] = sum_{c=0}^{nchans-1} A[c][ t + delay[d][c] ]                    eq. 3
 *     delay[d][c] = floor( k_DM * DM[d] * (f_c^-2 - f_top^-2) / dt + 0.5 )      eq. 1, 4, 5
 *     f_c = f_top + c*df,  k_DM = 4.148808e3 MHz^2 pc^-1 cm^3 s
 *
 * over 2/4/8-bit packed unsigned filterbank input.  The API is a plan object in the
 * style the paper describes for its own library ("modeled on FFTW"): create a plan
 * from the observing parameters, give it any list of DM trials, execute it on
 * device-resident data.  Batching over independent beams follows PAPER.md:388 (footnote 5).
 *
 * Conventions
 *   - Plain C types only.  Every pointer argument says whether it is HOST or DEVICE memory.
 *   - All functions return a dd_status (0 = DD_OK, negative = error) unless stated; none aborts.
 *     On error the plan is left unchanged -- with one exception: when the planning of a new DM list / kill mask /
 *     sub-band setting succeeds but the upload of its tables to the device fails (DD_ERR_CUDA), the plan holds the
 *     new setting without device tables, and the next dd_execute* uploads them again.
 *   - A plan is not thread-safe; distinct plans are independent.  The library never frees or
 *     retains caller buffers.  The plan owns its DM list, delay table and tile metadata (host and
 *     device copies) until dd_plan_destroy.
 *   - There is NO CPU fallback: dd_execute* return DD_ERR_CUDA when no CUDA device is usable.
 */
#ifndef DD_B200_H
#define DD_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dd_plan_s *dd_plan; /* opaque, library-owned */
typedef int dd_status;

enum {
    DD_OK = 0,
    DD_ERR_NULL = -1,             /* a required pointer is NULL                                          */
    DD_ERR_INVALID_ARG = -2,      /* nchans<=0, dt<=0, f_top<=0, df>=0, lowest frequency<=0, nbits not in
                                     {2,4,8}, ndm<=0, DM<0 or non-finite, nsamps<=0, out_nbits unknown,
                                     nbeams<=0, negative beam stride                                      */
    DD_ERR_NO_DM_LIST = -3,       /* dd_set_dm_list has not succeeded on this plan yet                    */
    DD_ERR_ALIGNMENT = -4,        /* in_ptr not 16-byte aligned, in_stride or in_beam_stride not a
                                     multiple of 16, out_ptr not aligned to its element size              */
    DD_ERR_STRIDE_TOO_SMALL = -5, /* in_stride*8 < (nsamps + max_delay)*nbits, or a beam stride smaller
                                     than one beam                                                        */
    DD_ERR_OUT_RANGE = -6,        /* nchans*(2^nbits-1) does not fit the requested output type exactly
                                     (>65535 for uint16, >=2^24 for float32)                              */
    DD_ERR_DELAY_OVERFLOW = -7,   /* a delay does not fit int32                                           */
    DD_ERR_SMEM = -8,             /* the delay spread of one DM block does not fit shared memory          */
    DD_ERR_CUDA = -9,             /* a CUDA call failed / no device; text via dd_last_cuda_error          */
    DD_ERR_NOMEM = -10,           /* host allocation failed                                               */
    DD_ERR_TOO_LARGE = -11,       /* dd_execute_static: the call needs more scratch than
                                     DD_STATIC_WORKSPACE_BYTES; text via dd_last_cuda_error               */
    DD_ERR_UNSUPPORTED = -12      /* dd_execute_static: the plan is not one this entry point serves       */
};

/* Output element type codes for `out_nbits` (reading R12 of DESIGN.md): raw sums, no scaling. */
enum {
    DD_OUT_F32 = 32,  /* float32 (exact: sums < 2^24)  */
    DD_OUT_U16 = 16,  /* uint16                         */
    DD_OUT_U32 = -32  /* uint32                         */
};

/*
 * dd_plan_create -- the observing parameters of PAPER.md:55-67 / 384.
 *   plan    HOST out: receives the new plan.
 *   nchans  number of frequency channels N_nu (> 0).
 *   dt      sampling interval in seconds (> 0), e.g. 64e-6.
 *   f_top   frequency of channel 0 in MHz ("start of the band", nu_0; > 0).
 *   df      channel width in MHz, < 0 (descending band; reading R6); f_top + (nchans-1)*df must be > 0.
 *   nbits   bits per input sample: 2, 4 or 8 (unsigned).
 * Host only; touches no device.
 */
dd_status dd_plan_create(dd_plan *plan, int nchans, double dt, double f_top, double df, int nbits);

/* Frees the plan and its host and device tables.  NULL is accepted. */
dd_status dd_plan_destroy(dd_plan plan);

/*
 * dd_set_dm_list -- "any list of DMs": finite, >= 0, any order, pc cm^-3.
 *   dm_list  HOST, ndm doubles; copied.
 * Computes, in double precision on the host (eq. 4-5), the int32 delay table
 * [ndm][nchans] and the per-(DM block, channel) span metadata, then uploads them if a CUDA device
 * is present (may synchronise).  Without a device the host tables are still built (so
 * dd_get_delay_table works) and the upload is retried by the first dd_execute.
 * Replaces any previous list.
 */
dd_status dd_set_dm_list(dd_plan plan, const double *dm_list, int ndm);

/*
 * dd_set_killmask -- the channel "kill mask" of PAPER.md:113: which frequency channels are included in the sum
 * and which are skipped (e.g. channels with radio-frequency interference).  With a mask,
 *     D[d][t] = sum over channels c with mask[c] != 0 of A[c][t + delay[d][c]]
 * i.e. the paper's arithmetic form `sum += data * kill_mask[channel]` with a 0/1 mask.
 *   mask  HOST, nchans int32 (copied): nonzero = summed, 0 = skipped.  NULL removes the mask (all channels summed).
 * May be called before or after dd_set_dm_list; with a DM list present the tile metadata is rebuilt over the
 * surviving channels at once (they are skipped entirely: no copy, no add), and on error the plan is unchanged.
 * The delay table and dd_get_max_delay still cover all channels, and so does the input-row length check of
 * dd_execute; the output-range check counts only the summed channels.  With every channel masked the output is zero.
 */
dd_status dd_set_killmask(dd_plan plan, const int32_t *mask);

/*
 * dd_set_output_stride -- "arbitrary strides through the ... output arrays" (footnote 5): the rows of
 * consecutive DM trials of the output lie out_dm_stride BYTES apart instead of densely, out[beam][d] starting at
 * out_ptr + beam * out_beam_stride + d * out_dm_stride (e.g. rows padded to a power of two for a later FFT, or a
 * window of a larger array).  Applies to dd_execute (device rows) and dd_execute_host (host rows).
 *   out_dm_stride  0 = dense rows of nsamps elements (default); otherwise a multiple of the element size
 *                  (DD_ERR_ALIGNMENT at execute) and >= nsamps * element size (DD_ERR_STRIDE_TOO_SMALL at execute);
 *                  with a batch, out_beam_stride must cover (ndm - 1) * out_dm_stride + nsamps elements.
 *                  Rows that are 16-byte aligned take the fastest store path.  Negative: DD_ERR_INVALID_ARG.
 */
dd_status dd_set_output_stride(dd_plan plan, int64_t out_dm_stride);

/*
 * dd_set_input_max -- the caller's promise that no input sample exceeds vmax (e.g. a series made by adding 2^k
 * 2-bit samples: vmax = 3 * 2^k).  The bit-plane kernel then neither shifts nor adds the planes that
 * cannot be set (bit_length(vmax) of the nbits planes are used).  Results are undefined if the promise is broken.
 *   vmax  1 .. 2^nbits - 1, or 0 to withdraw the promise (DD_ERR_INVALID_ARG otherwise).  Takes effect at the
 *         next dd_execute.  With a DM list already set the tile metadata is planned again (the promise decides which
 *         kernel serves the plan), so the call costs as much as dd_set_dm_list and can return its errors.
 */
dd_status dd_set_input_max(dd_plan plan, int vmax);

/*
 * dd_set_subband -- switches the plan to the SUB-BAND method of PAPER.md:317-321, an approximation of the
 * transform that costs about (1/dm_group + 1/sb_nchans) of the direct one (eq. 30), done as the paper's own
 * implementation did it: "two consecutive calls to the direct dedispersion routine and the addition of a
 * temporary data buffer".  With b = c / sb_nchans the sub-band of channel c and g = d / dm_group
 * the group of trial d, whose nominal DM is the DM of trial min(g*dm_group + dm_group/2, ndm-1):
 *     step 1   S[b][g][t] = sum_{c in sub-band b} A[c][t + delta1[g][c]],
 *              delta1[g][c] = floor(k_DM * DMnom_g * (f_c^-2 - f_{b*sb_nchans}^-2) / dt + 0.5)
 *     step 2   D[d][t]    = sum_b S[b][g][t + delta2[d][b]],   delta2[d][b] = delay[d][b*sb_nchans]   (eq. 4-5)
 * (readings S1-S4 of DESIGN.md section 10).  The result equals the direct transform with the delay
 * delta1 + delta2, which differs from eq. 5 by at most 1 + |DMnom - DM| * (DeltaT(c) - DeltaT(first channel of b)).
 *   sb_nchans  channels per sub-band N'nu: divides nchans; sb_nchans * (2^nbits - 1) <= 255 because the
 *              intermediate series are kept in 8 bits (else DD_ERR_OUT_RANGE).
 *   dm_group   trials per nominal DM N'DM: a multiple of 16.  The DM list is taken in the order given.
 *   (0, 0) returns to the direct transform.
 * Takes effect at once when a DM list is present (else at dd_set_dm_list); on error the plan is unchanged.  Honours
 * the kill mask and dd_set_batch.  dd_execute then needs input rows of nsamps + dd_get_subband_extent() samples,
 * allocates its temporary buffers on first use, and launches three kernels (bit-plane transpose of the input,
 * step 1 writing S as bit planes, step 2).  dd_execute_host runs the method on its staged copy as one time slab.
 */
dd_status dd_set_subband(dd_plan plan, int sb_nchans, int dm_group);

/* Input samples per row beyond nsamps that the two steps read: max_b (max delta2[.][b] + max delta1[.][sub-band b])
 * (>= 0), or a negative status (DD_ERR_INVALID_ARG when the sub-band method is not selected).  Host only. */
int64_t dd_get_subband_extent(dd_plan plan);

/* Copies the sub-band tables (HOST; any pointer may be NULL): nominal[ngroups] trial index of every group's nominal
 * DM, delta1[ngroups][nchans], delta2[ndm][nchans/sb_nchans]; ngroups = ceil(ndm / dm_group).  Host only. */
dd_status dd_get_subband_tables(dd_plan plan, int32_t *nominal, int32_t *delta1, int32_t *delta2);

/* Copies the delay table to `table` (HOST, ndm*nchans int32, row-major [d][c]).  Host only. */
dd_status dd_get_delay_table(dd_plan plan, int32_t *table);

/* max over the delay table (>= 0), or DD_ERR_NO_DM_LIST / DD_ERR_NULL (negative).  Host only. */
int64_t dd_get_max_delay(dd_plan plan);

/*
 * dd_set_batch -- independent beams processed by ONE dd_execute call.
 *   nbeams           >= 1 (default 1).
 *   in_beam_stride   bytes between beam b and b+1 of the input  (multiple of 16; >= nchans*in_stride
 *                    is checked at execute time).  Ignored when nbeams == 1.
 *   out_beam_stride  bytes between beam b and b+1 of the output (>= ndm*nsamps*elem, checked at
 *                    execute time; multiple of the element size).
 * All beams share the plan's delay table.
 */
dd_status dd_set_batch(dd_plan plan, int nbeams, int64_t in_beam_stride, int64_t out_beam_stride);

/*
 * dd_execute -- the dedispersion transform (eq. 3) on device-resident data, asynchronously.
 *   nsamps     number of OUTPUT samples per DM trial (> 0) (reading R8).
 *   in_ptr     DEVICE, 16-byte aligned.  in[beam][c] is a row of at least nsamps + dd_get_max_delay()
 *              samples packed along time, LSB first: sample t is bits [(t*nbits)&7, +nbits) of byte
 *              (t*nbits)>>3 (reading R9).  Rows are in_stride bytes apart and must be READABLE out to
 *              in_stride bytes (the kernel's 16-byte bulk copies may touch the padding).
 *   in_stride  bytes between channel rows; multiple of 16; in_stride*8 >= (nsamps+max_delay)*nbits.
 *   out_ptr    DEVICE.  out[beam][d][t], dense rows of nsamps elements, DM-major, time contiguous.
 *   out_nbits  DD_OUT_F32 (32), DD_OUT_U16 (16) or DD_OUT_U32 (-32).
 *   stream     a cudaStream_t (NULL = default stream).
 * Enqueues on `stream` and returns.  The FIRST call for a given problem size allocates the plan's work buffers (see
 * dd_set_workspace_limit; a call that needs larger ones frees and re-allocates, which synchronises the device), and
 * the first call after a dd_set_dm_list made without a device uploads the tables.  Every later call with the same
 * nsamps and batch only enqueues kernels -- it neither allocates, nor queries the device, nor synchronises -- so it
 * can be captured into a CUDA graph on `stream` and replayed (dd_scrunch_execute likewise).  The caller keeps in/out
 * alive until the stream has passed the enqueued work.  Launch errors are returned as DD_ERR_CUDA; variant 4 runs on
 * two internal streams forked from `stream`, which are joined back to it before the call returns, also on error.
 */
dd_status dd_execute(dd_plan plan, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr,
                     int out_nbits, void *stream);

/*
 * dd_execute_static -- dd_execute for callers that may not allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the same transform (eq. 3) by the bit-plane
 * kernel (variant 3), with the kernel's scratch -- the bit-plane copy of the input that dd_execute keeps
 * in a buffer it allocates on first use -- in a fixed device array of DD_STATIC_WORKSPACE_BYTES bytes that is part of
 * the library image (every GPU that loads the library holds it until the process exits).  Arguments, layouts,
 * alignment rules and the status codes of the argument checks are those of dd_execute.  In addition:
 *   - the plan must run the bit-plane kernel: dd_set_kernel_variant(plan, 3) before dd_set_dm_list, no sub-band
 *     method, and its tables on the CURRENT device (dd_set_dm_list made with that device current); anything else
 *     returns DD_ERR_UNSUPPORTED.  This call never uploads tables.
 *   - the scratch the call needs, about  nbeams * (nchans + 1) * ceil16((nsamps + largest delay of a DM block) * nbits / 8)
 *     bytes, must fit the array: DD_ERR_TOO_LARGE otherwise, with both numbers in dd_last_cuda_error(); nothing is
 *     enqueued.  Larger problems: split the time axis over several calls (each call's input rows start where its
 *     outputs start), or use dd_execute.
 *   - it calls no cudaMalloc, cudaFree or allocating library routine, and does not touch the plan's own work buffers.
 *     The first call on each device looks the array's address up (cudaGetSymbolAddress): make that one call outside
 *     a stream capture; later calls only enqueue two kernels and one memset on `stream`.
 *   - ALL calls, from all plans and threads, share the one array per device, and it keeps what the last call wrote:
 *     each call rewrites every byte it reads (the all-zero rows included), so calls that are ordered on the GPU
 *     (same stream, or joined by events) are independent of one another; calls whose kernels OVERLAP on the GPU
 *     (different streams, no ordering) race on the array and their outputs are undefined.
 */
#define DD_STATIC_WORKSPACE_BYTES (64 * 1024 * 1024)
dd_status dd_execute_static(dd_plan plan, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr,
                            int out_nbits, void *stream);

/*
 * dd_execute_host -- the same transform with HOST buffers (end-to-end path).
 *   in_host / out_host  HOST memory with the layouts of dd_execute (pinned memory gives full PCIe speed).
 * Copies the input to device staging owned by the plan, runs the kernel over time slabs and copies each
 * slab's output back, overlapping copies with compute on internal streams; returns after everything
 * has completed (synchronous).  Staging buffers are (re)allocated when the problem size grows.
 */
dd_status dd_execute_host(dd_plan plan, int64_t nsamps, const void *in_host, int64_t in_stride,
                          void *out_host, int out_nbits);

/*
 * dd_time_scrunch -- "time-scrunching": halves the time resolution of packed rows by adding
 * adjacent pairs of samples, out[r][t] = in[r][2t] + in[r][2t+1], 0 <= t < nsamps_out.  The scrunched rows are
 * packed like the input (LSB first, reading R9) at a width that holds the sums, so that they can be dedispersed by
 * a plan created with 2*dt and nbits_out (the paper applies this beyond the "diagonal" DM, then again at 2x, 4x...).
 *   nrows       rows (channels, or beams * channels when the beams are adjacent) (> 0).
 *   nsamps_out  output samples per row (> 0).
 *   in_ptr      DEVICE, 16-byte aligned; rows in_stride bytes apart (multiple of 16), readable for
 *               ceil16(nsamps_out * nbits_out / 8) * 2 * nbits_in / nbits_out bytes (whole 16-byte groups are read).
 *   out_ptr     DEVICE, 16-byte aligned; rows out_stride bytes apart (multiple of 16, >= ceil16(nsamps_out*nbits_out/8));
 *               the row is written up to that 16-byte boundary.
 *   nbits_in / nbits_out   (2, 4), (2, 8) or (4, 8); DD_ERR_OUT_RANGE when 2*(2^nbits_in - 1) > 2^nbits_out - 1.
 * Asynchronous on `stream`; no plan is involved.
 */
dd_status dd_time_scrunch(int nrows, int64_t nsamps_out, const void *in_ptr, int64_t in_stride, int nbits_in, void *out_ptr,
                          int64_t out_stride, int nbits_out, void *stream);

/*
 * dd_scrunch_* -- the direct transform WITH time-scrunching: "reduce the time
 * resolution by a factor of two when the DM exceeds the diagonal by adding adjacent pairs of time samples ...
 * repeated at 2x the diagonal, 4x etc."  The diagonal DM is the one whose dispersion curve has unit gradient at the
 * end of the band, where the delay is greatest:
 *     DM_diag = 1 / (DeltaT(nchans-1) - DeltaT(nchans-2)),   DeltaT(c) = k_DM (f_c^-2 - f_top^-2) / dt   (samples per unit DM)
 * and, following the order of the paper's procedure (0..DM_diag and DM_diag..2 DM_diag at full
 * resolution, scrunch, 2..4 DM_diag, scrunch, ...) and of its benchmark projection, trial d runs at
 *     factor F_d = 1 for DM_d <= 2 DM_diag,   2^k for 2^k DM_diag < DM_d <= 2^(k+1) DM_diag  (k >= 1)
 * (reading T1 of DESIGN.md section 11), capped at max_factor and at the largest factor whose samples still fit 8
 * bits, F (2^nbits - 1) <= 255.  Level l = the run of trials with the l-th smallest factor F:
 *     A_F[c][t] = sum_{i<F} A[c][F t + i]                         (pairs added log2 F times, packed at 2/4/8 bits)
 *     D_l[d][t] = sum_c A_F[c][t + delay_F[d][c]],  0 <= t < nsamps / F,   delay_F = eq. 4-5 with dt * F
 * An approximation of the transform by design (lower time resolution at high DM); each level is bit-exact against
 * the oracle's scrunched transform.
 *
 * dd_scrunch_create: dm_list HOST, non-decreasing (DD_ERR_INVALID_ARG otherwise), ndm > 0; max_factor a power of two
 *   >= 1 (1 = no scrunching: one level, the plain transform).  The set owns one plan per level.
 * dd_scrunch_set_killmask: the channel kill mask of dd_set_killmask applied to every level; NULL removes it.
 * dd_scrunch_levels: number of levels (>= 1), or a negative status.
 * dd_scrunch_level_info: HOST out, 6 int64: [0] factor F, [1] index of the level's first trial in dm_list,
 *   [2] trials in the level, [3] largest delay in samples of dt*F, [4] bits per sample of A_F, [5] DM_diag * 1e6 rounded.
 * dd_scrunch_required_bytes: bytes per input row that dd_scrunch_execute reads for `nsamps` (a multiple of 16;
 *   in_stride must be at least this; it covers nsamps + the largest F * max delay, rounded up to the 16-byte
 *   groups the pair-adding kernels read), or a negative status.
 * dd_scrunch_execute: in_ptr DEVICE packed rows as for dd_execute (one beam); out_ptrs HOST array of
 *   dd_scrunch_levels() DEVICE pointers, level l receiving dense rows out[d][t] of nsamps / F_l elements for its
 *   trials; out_nbits as for dd_execute.  nsamps >= the largest factor.  Asynchronous on `stream`; the scrunched
 *   rows live in device buffers owned by the set, (re)allocated when nsamps grows.
 */
typedef struct dd_scrunch_s *dd_scrunch;
dd_status dd_scrunch_create(dd_scrunch *set, int nchans, double dt, double f_top, double df, int nbits,
                            const double *dm_list, int ndm, int max_factor);
dd_status dd_scrunch_set_killmask(dd_scrunch set, const int32_t *mask);
int dd_scrunch_levels(dd_scrunch set);
dd_status dd_scrunch_level_info(dd_scrunch set, int level, int64_t *info);
int64_t dd_scrunch_required_bytes(dd_scrunch set, int64_t nsamps);
dd_status dd_scrunch_execute(dd_scrunch set, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *const *out_ptrs,
                             int out_nbits, void *stream);
dd_status dd_scrunch_destroy(dd_scrunch set);

/*
 * dd_tree_* -- the tree dedispersion algorithm (section 3.1, eq. 7-15) and the piecewise linear tree
 * method (section 3.1.1, eq. 16-23).  Readings X1-X5 of DESIGN.md section 12.
 *
 * The tree transforms N = 2^k channel rows into N series along LINEAR trails, D'[d'][t] = sum_c A[c][t + delay(d', c)],
 * d' = 0 .. N - 1, in N log2 N row additions.  The delays are those the recursion of eq. 10-13 applies with Theta
 * (eq. 14) and the shuffle Phi (eq. 15) exactly as printed; they equal eq. 8's round(d' c / (N - 1)) for N <= 8 and
 * lie within one sample of it beyond (reading X1) -- dd_tree_get_delays returns them.  The piecewise linear tree runs
 * the tree on every sub-band of sb_nchans = N' channels (stage 1, eq. 18) and then, for every trial of a DM list, adds
 * one row per sub-band (stage 2, eq. 22):
 *     out[d][t] = sum_n S_n[d'_n(d)][t + Dt''_n(d)],   d'_n(d) = round(DM_d [DeltaT(nu_{n+1}) - DeltaT(nu_n)])  (eq. 20, X3),
 *                                                       Dt''_n(d) = round(DM_d DeltaT(nu_n))                     (eq. 23, X4),
 * DeltaT(c) = k_DM ((f_top + c df)^-2 - f_top^-2) / dt (eq. 4), nu_n = n N'.  An APPROXIMATION of the direct transform
 * (the trail inside a sub-band is a straight line); it is exact in the sense of the paper's own definition, which the
 * tests check element by element.
 *
 * dd_tree_create   sb_nchans a power of two, 2 .. 4096: the channels of one tree; nchans a multiple of it, up to 65536: the
 *                  rows are nchans / sb_nchans trees one after the other -- the sub-bands of one band (== 1: the whole band
 *                  is one tree), or the bands of several beams whose rows lie back to back (without a DM list: stage 2
 *                  sums ALL sub-bands of the rows, so it serves one beam); nbits 2, 4 or 8; other values
 *                  DD_ERR_INVALID_ARG.  No device needed.  (The stages add in
 *                  8- or 16-bit lanes while sb_nchans * (2^nbits - 1) <= 65535, in 32-bit lanes beyond.)
 * dd_tree_create_padded  the frequency-padded tree (section 3.1.2; readings X6-X8): the nchans real channels
 *                  of the band (f_top, df as in dd_plan_create) are placed at the rows nu'(c) of eq. 25 of a stretched band
 *                  of N_pad rows (nu'(nchans) rounded up to a power of two; the other rows are blank), in which the
 *                  quadratic dispersion curves are straight lines, and ONE tree runs over the N_pad rows (the paper scatters
 *                  the input into a zero array; here the first pass reads through the row map and nothing is
 *                  copied).  Trial d' of N_pad is DM(d') = d' / ((N_pad - 1) DeltaT(1)) (eq. 26).  N_pad <= 4096, else
 *                  DD_ERR_INVALID_ARG.  dd_tree_execute then takes nchans input rows of
 *                  nsamps + N_pad - 1 samples and writes N_pad rows; dd_tree_set_dm_list is DD_ERR_UNSUPPORTED.
 * dd_tree_get_padding  returns N_pad (negative status on error; DD_ERR_INVALID_ARG for a tree that is not padded) and, if
 *                  pos is not NULL, writes nu'(c) for the nchans real channels (HOST int32).
 * dd_tree_set_dm_list  selects stage 2 for dm_list (HOST, ndm > 0 finite values >= 0) on the band (dt, f_top, df as in
 *                  dd_plan_create).  A trial with some d'_n(d) >= sb_nchans lies beyond the "diagonal" DM (eq. 21,
 *                  PAPER.md:205-211; reading X5): DD_ERR_OUT_RANGE, the tree unchanged (scrunch the input with
 *                  dd_time_scrunch and make a tree with 2 dt for those trials, as the paper prescribes).
 *                  nchans * (2^nbits - 1) must fit the output type at execute, as for dd_execute.
 * dd_tree_get_tables   HOST arrays [ndm][nchans / sb_nchans] of d'_n(d) and Dt''_n(d) (either may be NULL).
 * dd_tree_get_delays   HOST int32 [sb_nchans][sb_nchans]: delay(d', c) of the tree of one sub-band.
 * dd_tree_required_samples  samples every input row must hold for nsamps outputs: nsamps + sb_nchans - 1 without a DM
 *                  list, nsamps + max Dt'' + sb_nchans - 1 with one; negative status on error.
 * dd_tree_execute  in_ptr DEVICE packed rows as for dd_execute (16-byte aligned, in_stride a multiple of 16 with
 *                  in_stride * 8 >= required samples * nbits, readable out to in_stride).  out_ptr DEVICE dense rows of
 *                  nsamps elements of out_nbits (DD_OUT_*): without a DM list out[n N' + d'][t] = S_n[d'][t] (nchans rows:
 *                  the trees of all sub-bands; with sb_nchans == nchans the tree transform D'[d'][t]); with a DM list
 *                  out[d][t] (ndm rows).  Asynchronous on `stream`; the first call for a given nsamps allocates the
 *                  rows between the passes (8-, 16- or 32-bit, at most 8 nchans (nsamps + sb_nchans) bytes; with a DM list they
 *                  include the stage-1 output), later calls only enqueue kernels.  DD_ERR_CUDA without a device.
 * dd_tree_set_tuning   test knob: key 1 = steps fused by the first pass (1 .. 6, 0 = default), key 2 = steps fused by
 *                  later passes (1 .. 6, 0 = as many as keep the overlap of neighbouring tiles within a quarter of a tile),
 *                  key 3 / 4 = items per thread of the first / of later passes (4: two CTAs per SM, 8: one; 0 = default),
 *                  key 5 = 16: the first pass adds in 16-bit lanes even where 8-bit lanes hold its sums (0 = default),
 *                  key 6 = bit 0: the first two steps of a pass over packed rows are made in shared memory like the
 *                  others instead of in registers while the rows are staged; bit 1: every step makes its own trip through
 *                  shared memory instead of two steps per trip (0 = default).
 *                  Takes effect at the next execute.
 * dd_tree_get_info info[0] = passes, info[1] = kernels enqueued by the last execute, info[2] = device bytes held,
 *                  info[3 + 2 p] / info[4 + 2 p] = steps fused by pass p / columns a tile of it stores (p < 6); int64 x 16.
 */
typedef struct dd_tree_s *dd_tree;
dd_status dd_tree_create(dd_tree *tree, int nchans, int sb_nchans, int nbits);
dd_status dd_tree_create_padded(dd_tree *tree, int nchans, double f_top, double df, int nbits);
int dd_tree_get_padding(dd_tree tree, int32_t *pos);
dd_status dd_tree_set_dm_list(dd_tree tree, double dt, double f_top, double df, const double *dm_list, int ndm);
dd_status dd_tree_get_tables(dd_tree tree, int32_t *dprime, int32_t *dt2);
dd_status dd_tree_get_delays(dd_tree tree, int32_t *delays);
int64_t dd_tree_required_samples(dd_tree tree, int64_t nsamps);
dd_status dd_tree_execute(dd_tree tree, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr, int out_nbits,
                          void *stream);
dd_status dd_tree_set_tuning(dd_tree tree, int key, int value);
dd_status dd_tree_get_info(dd_tree tree, int64_t *info);
dd_status dd_tree_destroy(dd_tree tree);

/*
 * dd_set_kernel_variant -- tuning/testing knob: restrict the plan to one kernel variant.
 *   variant  0 = automatic (default); 1 = generic byte-lane kernel (2/4/8-bit); 2 = 2-bit nibble-lane kernel;
 *            3 = bit-plane carry-save kernel (2/4/8-bit; needs nchans*(2^nbits-1) < 2^12 / 2^16 / 2^20);
 *            4 = pair rows (2/4/8-bit; opt-in, and the fallback of variant 6 for 4- and 8-bit plans): the same kernel
 *                over rows x[c0] + shift(x[c1], delta) made once per
 *                delay difference delta of every pair of adjacent summed channels -- exact, n + 1 plane words per
 *                pair instead of 2 n; costs device memory for the rows of one beam (16x / 26x / 12x its packed
 *                input on the 2-bit / 4-bit / 8-bit survey-shaped configs; twice that with several beams; the time
 *                axis is split into groups if that exceeds the limit of dd_set_workspace_limit) and two more kernels
 *                per group, run on internal streams that are forked from and joined to the caller's stream;
 *            5 = group sums made inside the CTA (2/4/8-bit, opt-in): per group of 2 or 4 adjacent summed channels and
 *                block of 16 trials, one row per pattern of delay differences is built in shared memory from the staged
 *                bit planes by builder warps, and every trial adds the row of its own pattern -- exact like variant 4,
 *                but the rows never reach device memory (slower than variants 3 / 6);
 *            6 = group rows (2/4/8-bit; the DEFAULT for plans of >= 128 channels whenever the planner's cost model says
 *                it pays): one pre-summed row per group of four (or two) adjacent summed channels and tuple of delay
 *                differences of the DM list, n + 2 bit planes added per four channels instead of 4 n -- exact; costs device
 *                memory for the rows (dd_set_workspace_limit) like variant 4 and runs on the same internal streams
 *                (DESIGN.md section 5.5).
 * Takes effect at the next dd_set_dm_list (which returns DD_ERR_SMEM if that variant cannot serve the plan).
 */
dd_status dd_set_kernel_variant(dd_plan plan, int variant);

/*
 * dd_set_tuning -- documented launch-geometry knobs for tests and tuning (the library reads no environment
 * variables).  Results never depend on them.
 *   key    DD_TUNE_SUBBAND_GPC: sub-bands summed one after the other by a CTA of sub-band step 1;
 *            0 = chosen by the library.  Takes effect at the next dd_execute.
 *          DD_TUNE_GROUP_SIZE: channels per group of variants 5 and 6 (2 or 4); 0 = chosen by the planner.
 *          DD_TUNE_GROUPS_PER_STAGE: groups per pipeline stage of variant 5 (one of the compiled shapes: 2-bit 16 pairs
 *            or 4 groups of four, 4-bit 8 or 4, 8-bit 4 / 2 or 2 / 1); 0 = chosen by the planner.
 *            Both take effect at the next dd_set_dm_list (DD_ERR_SMEM if no compiled shape matches or fits).
 *          DD_TUNE_PAIR_TILES: time tiles per group of rows of variants 4 and 6 (their launchers build and transform the
 *            rows group of tiles by group); 0 = as many as the workspace limit allows.  Takes effect at the next dd_execute.
 *          DD_TUNE_TILES_PER_CTA: consecutive time tiles a CTA of the short bit-plane kernel walks (plans with few channels
 *            per group: step 2 of the sub-band method, small transforms); 0 = as many as leave 8 waves of CTAs, at most 8.
 *            Takes effect at the next dd_execute.
 *          DD_TUNE_HOST_SLAB: output samples per time slab of dd_execute_host (rounded up to whole time tiles); 0 = 2^15.
 *            Takes effect at the next dd_execute_host.
 *   value  >= 0.
 * DD_ERR_INVALID_ARG for an unknown key or a negative value.
 */
enum { DD_TUNE_SUBBAND_GPC = 1, DD_TUNE_GROUP_SIZE = 2, DD_TUNE_GROUPS_PER_STAGE = 3, DD_TUNE_PAIR_TILES = 4, DD_TUNE_TILES_PER_CTA = 5,
       DD_TUNE_HOST_SLAB = 6 };
dd_status dd_set_tuning(dd_plan plan, int key, int value);

/*
 * dd_set_workspace_limit / dd_get_workspace_bytes -- device memory the plan takes beside its tables.
 * Every bit-plane variant keeps a bit-plane copy of the packed input (same size as the input).  Variants 6 (the default
 * for larger plans) and 4 also keep the rows of one group of time tiles (two groups when the call has several beams or
 * the time axis is split): 25-105 x the packed input of a beam for variant 6 on the survey-shaped configs (9.6 GB for
 * 1024 channels x 1200 trials x 2^19 2-bit samples, 12.5 GB per 8-bit beam of 2^18 samples) if the whole time axis is one
 * group.  The buffers are allocated by the first dd_execute / dd_execute_host that needs them and re-used afterwards;
 * they grow (cudaFree + cudaMalloc, which synchronise the device) only when a later call needs more.  The split of
 * the time axis is worked out once per launch geometry (time tiles x beams) and kept.
 *   bytes  limit for the pair rows of one group; 0 (default) = 3/4 of the device memory free at the first call.
 *          A limit too small for one time tile's rows makes dd_execute return DD_ERR_CUDA (out of memory).
 * dd_get_workspace_bytes returns the bytes the plan holds on the device right now (work buffers, pair rows, the
 * staging buffers of dd_execute_host; tables not counted).
 */
dd_status dd_set_workspace_limit(dd_plan plan, int64_t bytes);
int64_t dd_get_workspace_bytes(dd_plan plan);

/*
 * dd_get_launch_info -- how the plan tiles the problem (for benchmarks and tests).  Host only.
 *   info  HOST out, 8 int64: [0] DMs per CTA (DB), [1] output samples per CTA (TB), [2] channels per
 *         pipeline stage, [3] dynamic shared memory bytes per CTA, [4] threads per CTA, [5] number of DM
 *         blocks, [6] kernels launched by the last dd_execute (0 if none yet), [7] kernel variant id.
 */
dd_status dd_get_launch_info(dd_plan plan, int64_t *info);

/*
 * dd_profile_enable / dd_profile_read -- optional per-kernel device timing of dd_execute (benchmarks).
 * When enabled, each dd_execute records three CUDA events on the caller's stream: before the first kernel,
 * between the bit-plane pre-pass and the transform kernel (variants without a pre-pass record it right after
 * the first event), and after the last kernel.  Up to `max_executes` calls are recorded; further calls run
 * untimed.  The events cost no synchronisation.
 *   max_executes  > 0: enable (re-arms and drops earlier records); 0: disable and free the events.
 * dd_profile_read waits for the last recorded event, then writes, per recorded dd_execute, the pre-pass and
 * transform-kernel durations in milliseconds and re-arms the recorder.
 *   n_executes  HOST out: number of records written (<= max_executes).
 *   prepass_ms  HOST out, max_executes floats (0 for variants without a pre-pass).
 *   main_ms     HOST out, max_executes floats.
 */
dd_status dd_profile_enable(dd_plan plan, int max_executes);
dd_status dd_profile_read(dd_plan plan, int *n_executes, float *prepass_ms, float *main_ms);

/*
 * dd_int_add_peak -- measures this GPU's 32-bit integer-add throughput (the ALU roofline denominator
 * of DESIGN.md section 6) with a register-resident microbenchmark on all SMs.  Additions are counted, not
 * instructions, and the chains are cross-coupled so that the compiler cannot fold two additions into one.
 *   mode          0: 2-input adds (the compiler spreads them over both integer pipes);
 *                 1: 3-input adds (IADD3: two additions per instruction, ALU pipe only);
 *                 2: IADD3 interleaved 1:1 with multiply-add by a run-time 1 (IMAD on the FMA pipe): both
 *                    pipes busy, three additions per instruction pair -- the highest rate of the three.
 *   adds_per_sec  HOST out: additions per second.
 *   stream        cudaStream_t.  Synchronises.
 */
dd_status dd_int_add_peak(int mode, double *adds_per_sec, void *stream);

/* Static description of a status code. */
const char *dd_strerror(dd_status s);

/* Text of the last CUDA error seen by this library in the calling thread ("" if none). */
const char *dd_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DD_B200_H */
