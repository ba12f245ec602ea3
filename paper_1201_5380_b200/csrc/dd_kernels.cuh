// dd_kernels.cuh -- launch interface between the C ABI (dd_api.cu) and the CUDA kernels (dd_kernels.cu).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "dd_plan.h"

namespace dd {

// Everything one launch of the direct-dedispersion kernel needs (passed by value as a kernel parameter).
struct KernelParams {
    const uint8_t *in;        // device: in[beam][c][byte]
    int64_t in_stride;        // bytes between channel rows
    int64_t in_row_bytes;     // bytes readable from the start of a row (<= in_stride; less for a time slab)
    int64_t in_beam_stride;   // bytes between beams
    uint8_t *out;             // device: out[beam][d][t]
    int64_t out_beam_stride;  // bytes between beams
    int64_t out_dm_stride;    // bytes between the rows of consecutive DM trials (dense: nsamps * element size)
    int64_t nsamps;           // output samples per DM trial
    int32_t out_code;         // DD_OUT_F32 / DD_OUT_U16 / DD_OUT_U32
    int32_t vec_ok;           // rows and base pointers allow 4-sample vector stores
    int32_t vec16_ok;         // ... and 16-byte stores at every multiple of 16 bytes inside a row (coalescing epilogue)
    int32_t nchans;           // channels summed (the live list under a kill mask); span/rel are indexed by list position
    int32_t nrows;            // channel rows of the input
    int32_t ndm, nblk, ntiles, nbeams;
    int32_t cc, nchunks;      // channels per stage, number of stages' worth of channels
    int32_t raw_slot, lane_slot;
    int32_t sub_slot;         // bit planes: bytes per sub-row inside a channel slot
    int32_t ngroups;          // channel groups per beam (sub-bands); the batch index is (beam, group)
    int32_t group_cols;       // span/rel columns per group
    int32_t row_mul;          // input rows per channel index (sub-band step 2: one row per nominal DM), else 1
    int32_t in_blk_div;       // > 0: DM block blk reads the input row  row * row_mul + blk / in_blk_div
    int64_t in_blk_stride;    // bytes between those rows (set by the launcher)
    int32_t nstages;          // ring depth of the staged buffers (bit-plane variant)
    int32_t nchans_pad;       // channels iterated over: nchans padded to a multiple of cc (bit-plane variant)
    const uint8_t *zero;      // raw_slot zero bytes: the span of a padded channel
    const int4 *span;         // [nblk][nchans_pad] {start, nbytes, input row, 0}
    const void *rel;          // [nblk][nchans][DB] entries of var.rel_bytes
    // out_code == kOutPlanes (bit-plane kernel only): `out` is the bit-plane work buffer of an 8-bit plan, rows
    // [beam][group * ndm + d][sub-row 0..1][unit][4 planes]
    int64_t pl_conv;          // bytes per sub-row
    int64_t pl_beam;          // bytes between beams
    int32_t pl_units;         // units (32 samples) per sub-row
    int32_t gpc;              // channel groups summed one after the other by a CTA (>= 1; > 1 only with kOutPlanes)
    int32_t tpc;              // time tiles a CTA of the short bit-plane instantiation walks (>= 1; > 1 only with gpc == 1)
    int32_t rows_per_chunk;   // pair rows (variant 4): rows staged per stage; span is [nblk][nchunks][rows_per_chunk]
    int32_t tile0;            // pair rows: this launch covers the time tiles tile0 .. tile0 + ntiles - 1 ...
    int64_t in_unit0;         // ... and `in` holds the pair rows from unit in_unit0 (32 samples per unit) on
    // group sums (variant 5, dd_kernel_gs.cu): span is [nblk][nchunks][channels per stage], rel [nblk][nchunks][cc][DB]
    const int4 *gs_tab;       // [nblk][nchunks][gs_rows] build entries of 64 bytes each (dd_plan.h: GsEntry)
    int32_t gs_rows;          // rows built per stage
    int32_t gs_row_units;     // units (32 samples) per row slot, a multiple of 4
    int32_t gs_raw_sub;       // bytes per sub-row of a channel slot of the raw stage
    int32_t gs_nsr, gs_nsp;   // ring depths: raw stages, row stages
    int32_t gs_nblk32;        // 32-unit blocks per row = ceil(gs_row_units / 32)
    int32_t gs_magic;         // ceil(65536 / gs_nblk32): item / gs_nblk32 == (item * gs_magic) >> 16 for item < 4096
};

// Geometry of the bit-plane work buffer of a plan for one launch (dd_kernel_bp.cu).
struct BpWork {
    int64_t units;    // 16-byte groups per sub-row
    int64_t conv;     // bytes per sub-row
    int64_t rows;     // rows per beam, the all-zero rows of the padded channels included
    int64_t w_beam;   // bytes per beam
};

// Enqueues the kernel variant chosen by the plan.  Returns the cudaError_t of the launch.
cudaError_t launch_direct(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);

cudaError_t launch_variant1(const dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);
cudaError_t launch_variant2(const dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);
// variant 3 launches two kernels (bit-plane transpose into plan->d_work, then the transform); it may grow d_work.
// planes_ready: plan->d_work already holds the bit planes (written by another launch with kOutPlanes after
// bp_prepare_work): the transpose is skipped.
cudaError_t launch_variant3(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, bool planes_ready = false);
// variant 4 launches three kernels: bit-plane transpose, pair rows (one per delay difference of every channel pair),
// transform over the pair rows.  May grow plan->d_work and plan->d_pairwork.
cudaError_t launch_variant4(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);
// variant 5 (group sums made inside the CTA, dd_kernel_gs.cu): bit-plane transpose, then the transform.
cudaError_t launch_variant5(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);
// Sizes (and grows) plan->d_work for the launch described by kp and keeps its all-zero rows; zero_all: the whole
// buffer is cleared whenever it is new or its layout changed (for a producer that does not write every unit).
cudaError_t bp_prepare_work(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, bool zero_all, BpWork *w);

// variant 6 (group rows in device memory, dd_kernel_gr.cu): transpose, then per group of time tiles row builder + transform.
cudaError_t launch_variant6(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);
// The bit-plane transpose of the packed input into plan->d_work (geometry w from bp_prepare_work).
cudaError_t launch_to_bitplanes(dd_plan_s *plan, const KernelParams &kp, const BpWork &w, cudaStream_t stream);

// dd_execute_static (dd_kernel_bp.cu): variant 3 with its bit-plane work buffer in a file-scope device array of
// DD_STATIC_WORKSPACE_BYTES; no allocation.  static_work_need: bytes of that buffer the launch described by kp takes.
size_t static_work_need(const dd_plan_s *plan, const KernelParams &kp);
cudaError_t launch_variant3_static(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream);

// Time-scrunching of packed rows (dd_scrunch.cu).  out_bytes = bytes of every output row to produce (multiple of 16).
cudaError_t launch_scrunch(int nbits_in, int nbits_out, int nrows, const uint8_t *in, int64_t in_stride, uint8_t *out,
                           int64_t out_stride, int64_t out_bytes, cudaStream_t stream);

// Kernels one launch_direct call enqueues for this plan.
int launches_per_execute(const dd_plan_s *plan);

// DD_ERR_CUDA with the text dd_last_cuda_error returns; the text alone (dd_api.cu).
dd_status report_cuda_error(cudaError_t e, const char *what);
void set_error_text(const std::string &text);

// Integer-add throughput microbenchmark (roofline denominator).  Synchronises `stream`.
cudaError_t int_add_peak(int mode, double *adds_per_sec, cudaStream_t stream);

}  // namespace dd
