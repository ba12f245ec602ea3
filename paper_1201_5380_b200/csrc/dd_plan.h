// dd_plan.h -- internal plan object and host-side planning for libdd_b200 (not part of the C ABI).
//
// Host planning follows PAPER.md:62-67 (eq. 4-5: delay table in double precision) and PAPER.md:115
// (the staged span of a thread block must carry "additional time samples ... to allow for
// differences in delay across a block"): for every (DM block, channel) we record where the staged
// span starts and how many bytes it holds, and for every (DM, channel) the offset of that DM's
// window inside the span.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/dd.h"

namespace dd {

// One CUDA kernel variant: compile-time tile shape, selected at dd_set_dm_list time.
struct Variant {
    int id;           // reported by dd_get_launch_info[7]
    int DB;           // DM trials per CTA
    int TB;           // output samples per CTA
    int threads;      // threads per CTA
    int tail;         // extra samples a thread may read past TB + offset (over-fetch of the aligned loads)
    int rel_bytes;    // bytes per offset-table entry: 2 = sample offset (uint16), 4 = 4 * sample offset (uint32),
                      // 8 = {byte offset of the DM's first window word inside the stage, bit shift} (2 x uint32)
    int lane_bits;    // bits per sample of the unpacked lane buffer in shared memory (== nbits: no lane buffer)
    int lane_stages;  // lane buffers (1 = single, 2 = double-buffered)
    int raw_stages;   // stages of the packed / bit-plane buffer and of the offset table
    int cc[4];        // candidate channels-per-stage, largest first (0 = end)
    int nbits_mask;   // input widths served (bit n set = nbits n)
    int max_sum_bits; // widest sum the accumulators hold: nchans*(2^nbits-1) < 2^max_sum_bits
    bool pad_chunks;  // the kernel always processes whole stages: the channel list is padded to a multiple
                      // of cc with all-zero channels (their spans are staged from a zeroed device buffer)
    bool bitplane;    // stages hold bit planes produced by the transpose pre-pass (dd_kernel_bp.cu)
    int unit_bytes;   // bit planes: bytes per 32-sample unit of a sub-row (4 * planes per sub-row); else 0
    int nsub;         // bit planes: sub-rows per channel (nbits / planes per sub-row); else 1
};

struct SpanMeta {   // per (DM block, live channel); mirrored on the device as int4
    int32_t start;  // first staged sample relative to the tile's first output sample; multiple of 128/nbits.
                    // Bit-plane variants: the same as a byte offset inside a bit-plane sub-row (sample offset in `pad`)
    int32_t nbytes; // packed bytes to stage (multiple of 16); negative (variants 1, 2): a padded channel staged from the
                    // zero buffer; bit-plane variants stage padded channels from the zero row `row` = nchans
    int32_t row;    // the channel's row in the input (differs from its position in the list under a kill mask)
    int32_t pad;
};

// Variant 5: one row to build in a stage (mirrored on the device as 4 x int4).  Row = sum over the group's channels i
// of x[c_i][t + delta_i] for one pattern (delta_1 .. delta_{G-1}) of delay differences, over `nunits` units.
struct GsEntry {
    int32_t dst;      // byte offset of the row slot inside the row stage
    int32_t nunits;   // units to build (0: unused entry)
    int32_t src[4];   // per channel: byte offset, inside the raw stage, of the unit of sub-row 0 that holds the row's first
                      // sample shifted by delta_i (channel slot + whole units of the offset)
    int32_t sh[4];    // per channel: the offset's remainder, 0..31 (sh[0] == 0)
    int32_t pad[6];
};
static_assert(sizeof(GsEntry) == 64, "GsEntry is staged as 4 x 16 bytes");

struct HostStage;   // device staging for dd_execute_host (dd_api.cu)

}  // namespace dd

struct dd_plan_s {
    // observing parameters
    int nchans = 0;
    double dt = 0, f_top = 0, df = 0;
    int nbits = 0;
    // DM trials and the delay table (eq. 4-5)
    int ndm = 0;
    std::vector<double> dm;
    std::vector<int32_t> delay;   // [ndm][nchans]
    int64_t max_delay = -1;
    // channel kill mask: the channels that are summed, in ascending order; all of them by default
    std::vector<uint8_t> keep;    // [nchans] 1 = summed, 0 = skipped; empty = no mask
    std::vector<int32_t> live;    // rows of the summed channels (built by build_tiles)
    int nlive = 0;
    // channel groups: with group_size > 0 every run of group_size consecutive channels is summed on its own (the
    // sub-bands of PAPER.md:317); the launch then treats (beam, group) as the batch index.  0 = one group.
    int group_size = 0;
    int ngroups = 1;       // built by build_tiles
    int group_cols = 0;    // columns of span/rel per group: the largest live count of a group, padded to a multiple of cc
    // sub-band method: two direct steps through sub-plans and a temporary buffer
    int sb_nchans = 0, dm_group = 0;      // channels per sub-band N'nu, trials per nominal DM N'DM; 0 = direct
    dd_plan_s *s1 = nullptr;              // step 1: sub-bands x nominal DMs, uint8 sums (owned)
    dd_plan_s *s2 = nullptr;              // step 2: the miniature filterbanks, 8-bit input (owned)
    std::vector<int32_t> sb_nominal;      // [ngroups of trials] index of the nominal trial
    int64_t sb_max_d2 = 0;                // largest step-2 delay: step 1 computes nsamps + sb_max_d2 samples
    int64_t sb_extent = -1;               // input samples per row beyond nsamps that the two steps read
    void *d_tmp = nullptr;                // intermediate series [beam][sub-band][nominal DM][t], uint8
    size_t tmp_bytes = 0;
    // batching
    int nbeams = 1;
    int64_t in_beam_stride = 0, out_beam_stride = 0;
    int64_t out_dm_stride = 0;   // bytes between output rows (dd_set_output_stride); 0 = dense rows of nsamps elements
    // tiling
    dd::Variant var{};
    int force_variant = 0; // 0 = automatic; otherwise only this variant id is considered (dd_set_kernel_variant)
    int nblk = 0;          // DM blocks
    int cc = 0;            // channels per pipeline stage
    int nchans_pad = 0;    // channels the kernel iterates over (nlive, or padded to a multiple of cc)
    int nstages = 2;       // ring depth of the staged buffers (<= var.raw_stages)
    bool long_mode = false; // bit planes: many channels per group -> the LONG kernel instantiation (flush every FL stages)
    bool patch = false;    // bit planes: epilogue through per-warp shared-memory patches (!long_mode || nbits < 8)
    int64_t max_span_end = 0;   // max over spans of start + staged samples: how far past a tile's t0 a copy reaches
    int raw_slot = 0;      // bytes per channel slot of the packed stage buffer (multiple of 16)
    int sub_slot = 0;      // bit planes: bytes per sub-row inside a channel slot (raw_slot / nsub)
    int lane_slot = 0;     // bytes per channel slot of the unpacked lane buffer
    int64_t smem_bytes = 0;
    // pair rows (variant 4): the CTA adds, per pair of adjacent live channels, ONE row S = x[c0] + shift(x[c1], delta)
    // made beforehand for every delay difference delta = delay[d][c1] - delay[d][c0] that occurs in the table
    bool pairs = false;
    int pair_nbits = 0;                   // width of the consumer layout (4 for 2-bit input, 8 for 4-bit input)
    int pair_planes = 0;                  // planes of a pair sum (nbits + 1)
    int rows_per_chunk = 0;               // pair rows staged per stage (the largest count of any stage, padded rows skipped)
    std::vector<int32_t> prow;            // [n_prows][4] {c0 row, c1 row or -1, delta, 0}
    int64_t n_prows = 0;
    void *d_prow = nullptr;
    void *d_pairwork = nullptr;           // pair rows as bit planes [n_prows + 1][sub][bytes]; the last row is all zero
    size_t pairwork_bytes = 0;
    void *pair_streams[2] = {nullptr, nullptr};   // internal streams: groups of time tiles alternate between them
    void *pair_events[3] = {nullptr, nullptr, nullptr};   // fork, join[2]
    int pair_launches = 0;                // kernels of the last launch (depends on the number of tile groups)
    int pair_tiles = 0;                   // dd_set_tuning(DD_TUNE_PAIR_TILES): time tiles per group of pair rows; 0 = by budget
    int64_t pair_geom[3] = {0, 0, 0};     // {time tiles, beams, tiles per group} the budget was last worked out for
    int64_t ws_limit = 0;                 // dd_set_workspace_limit: bytes the pair rows of one group may take; 0 = 3/4 of free memory
    // group sums (variant 5): per group of G adjacent live channels and DM block, the CTA itself builds one row per
    // pattern of delay differences in shared memory; every trial adds the row of its own pattern
    bool gs = false;
    int gs_G = 0;                         // channels per group (2 or 4); cc = groups per stage
    int gs_force_G = 0, gs_force_cc = 0;  // dd_set_tuning: 0 = chosen by the planner
    int gs_rows = 0;                      // rows built per stage (the largest count of any stage)
    int gs_row_units = 0;                 // units per row slot
    int gs_raw_sub = 0;                   // bytes per sub-row of a raw channel slot
    int gs_nsr = 0, gs_nsp = 0;           // ring depths
    bool gs_patch = false;                // epilogue through shared-memory patches
    std::vector<dd::GsEntry> gs_tab;      // [nblk][nchunks][gs_rows]
    void *d_gs_tab = nullptr;
    // group rows (variant 6): like pair rows, for groups of gs_G = 4 (or 2) adjacent live channels, rows unit-interleaved;
    // prow holds {c_0 .. c_3 (or -1), delta_0 .. delta_3} per row (8 ints), span [nblk][nchunks][rows_per_chunk]
    // {byte offset in the row for tile 0, bytes, row, byte offset in the stage}, raw_slot = bytes of a stage's rows
    bool gr = false;
    int gr_stage_slots = 0;               // stage slots per DM block in span / rel (the largest stage count of any block); every
                                          // block's span list starts with a header entry {stages, groups of the first stage, -, -}
    int bp_tpc = 0;                       // dd_set_tuning: time tiles per CTA of the short bit-plane kernel (0 = chosen by the launcher)
    int host_slab = 0;                    // dd_set_tuning: output samples per time slab of dd_execute_host (0 = the default)
    int sb_gpc = 0;                       // dd_set_tuning: sub-bands per CTA of sub-band step 1 (0 = chosen by the library)
    int in_planes = 0;     // > 0: no input sample reaches 2^in_planes (sub-band step 2: sums of N'nu samples); 0 = nbits
    bool final32 = false;  // sums need 32-bit accumulators (nchans*(2^nbits-1) > 65535)
    std::vector<dd::SpanMeta> span;   // [nblk][nchans_pad] over the live channels (nchans_pad = ngroups * group_cols)
    std::vector<uint8_t> rel;         // [nblk][nchans_pad][DB] entries of var.rel_bytes: delay - span start per DM slot
    // device copies
    int device = -1;
    bool uploaded = false;
    void *d_span = nullptr;
    void *d_rel = nullptr;
    void *d_zero = nullptr;           // raw_slot zero bytes (source of the padded channels)
    void *d_work = nullptr;           // bit-plane copy of the input (variants with `bitplane`), grown on demand
    size_t work_bytes = 0;
    int64_t work_layout[4] = {0, 0, 0, 0};   // {bytes per sub-row, rows, beams, cleared as a whole} d_work's zeros were written for
    int64_t last_launches = 0;
    dd::HostStage *stage = nullptr;
    // optional per-kernel timing of dd_execute (dd_profile_enable): 3 events per recorded call
    std::vector<void *> prof_events;   // cudaEvent_t [3 * prof_cap]
    int prof_cap = 0, prof_n = 0;
    void *prof_mid = nullptr;          // event the launcher records between pre-pass and transform (or null)
};

namespace dd {

// Evaluates eq. 4-5 in double for every (d, c); fills plan->delay / max_delay.  DD_ERR_DELAY_OVERFLOW
// if a delay does not fit int32.
dd_status compute_delay_table(dd_plan_s *p);

// The two sub-plans of the sub-band method for p's DM list, kill mask and (sb_nchans, dm_group): fills s1/s2
// (delay tables + tiles), sb_nominal, sb_max_d2, sb_extent.  s1/s2 must be fresh plans.
dd_status build_subband(const dd_plan_s *p, dd_plan_s *s1, dd_plan_s *s2, std::vector<int32_t> *nominal,
                        int64_t *max_d2, int64_t *extent);

// Chooses the kernel variant and builds span/rel metadata.  DD_ERR_SMEM if no tiling fits.
dd_status build_tiles(dd_plan_s *p);
// Variant 4 (pair rows): 2- and 4-bit input, one channel group.  DD_ERR_SMEM if it cannot serve the plan.
dd_status build_tiles_pairs(dd_plan_s *p);
// Variant 5 (group sums in shared memory), G channels per group, cc groups per stage (0 = the default for the width).
dd_status build_tiles_gs(dd_plan_s *p, int G, int cc);
// Shared-memory bytes of the variant-5 kernel for this geometry (must match the carve-up in dd_kernel_gs.cu).
int64_t gs_smem_bytes(int nbits, int G, int cc, int rows, int row_units, int raw_sub, int nsr, int nsp, bool patch);
bool gs_instance_exists(int nbits, int G, int cc);   // is dd_direct_gs<nbits, G, cc> compiled in?  (dd_kernel_gs.cu)
// Variant 6 (group rows in device memory, dd_kernel_gr.cu): G channels per group (0 = 4).  DD_ERR_SMEM if it cannot serve.
dd_status build_tiles_gr(dd_plan_s *p, int G);
int64_t gr_smem_bytes(int nbits, int G, int nstages, int stage_bytes, bool patch);
// groups between flushes of the pending words / most groups a stage may hold (its offset entries have a fixed slot)
#ifndef DD_GR_NF2
#define DD_GR_NF2 16
#define DD_GR_NF8 8
#endif
constexpr int gr_flush_groups(int nbits, int G) { return nbits == 8 ? DD_GR_NF8 : (nbits == 2 ? DD_GR_NF2 : 16); }
constexpr int gr_max_groups_per_stage(int nbits, int G) { return nbits == 8 ? 8 : 16; }
#ifndef DD_GR_Q4
#define DD_GR_Q4 4
#define DD_GR_Q2 2
#endif
// stages begin and end on multiples of this many groups (the kernel tests for a stage boundary once per quantum)
constexpr int gr_group_quantum(int nbits, int G) { return nbits == 8 ? 1 : (nbits == 4 ? DD_GR_Q4 : DD_GR_Q2); }
// words per 32-sample unit of a group row: the planes (nbits + log2 G) padded so that the lanes of a warp read without
// bank conflicts and units stay 8-byte aligned (dd_kernel_gr.cu)
constexpr int gr_unit_words(int nbits, int G) { return nbits == 2 ? 4 : (nbits == 4 ? 6 : 10); }
#ifndef DD_GR_W2
#define DD_GR_W2 5
#endif
constexpr int kGrW2 = DD_GR_W2;   // units per lane of the 2-bit group-row kernel
constexpr int kGsW2 = 3, kGsW48 = 2;   // variant 5: units (32 samples) per lane for 2-bit / 4- and 8-bit input (tile = 1024 W samples)
constexpr int kGsFlushStages = 4;   // stages between flushes of the pending words (dd_kernel_gs.cu: GS_FL)

// Shared-memory bytes the kernel needs for `cc` channels per stage (must match the kernel's carve-up).
int64_t smem_layout_bytes(const dd_plan_s *p, int cc);

constexpr int64_t kMaxDynSmem = 227 * 1024;   // usable shared memory per CTA on sm_100a
constexpr int kBpPatchBytes = 4096;             // bit-plane kernel epilogue: shared memory per warp (32 lanes x 128 B)
constexpr int kOutU8 = 8;                     // internal output code: uint8 sums, not in the C ABI
constexpr int kOutPlanes = 9;                 // internal output code: the low 8 bit planes of the sums, written in the layout the
                                              // 8-bit bit-plane kernel stages (sub-band intermediate: step 2 needs no pre-pass)

}  // namespace dd
