// dd_kernel_bp.cu -- variant 3: the input as BIT PLANES, summed with carry-save adders.
//
//     D[d][t] = sum_c A[c][t + delay[d][c]]                       (eq. 3)
//
// The paper's bit-level parallelism (several samples per machine word, one word operation
// acting on all of them) taken to its end: ONE BIT per lane.  A pre-pass transposes every 32 consecutive
// n-bit samples of a channel into n 32-bit words, plane k holding bit k of the 32 samples in time order
// (sub-word samples handled by shift and mask).  The sum over channels is then a population
// count per lane, kept as NP bit planes P[0..NP) (P[k] holds bit k of 32 sums) and updated with 3:2
// carry-save adders: sum = a ^ b ^ c, carry = maj(a, b, c), two LOP3 instructions that add one more
// 32-sample word into the counter.  Per channel and 32 outputs that is n funnel shifts (the delay is an
// arbitrary bit offset into the plane words) + ~2.1 n LOP3 for 32 channel-adds, i.e. ~3.1 ALU instructions
// per 32 input bits whatever the sample width.
//
// Layout.  A "unit" is 32 consecutive samples.  Planes are stored in SUB-ROWS of NB planes: unit u of a
// sub-row is NB consecutive words {plane 0 .. plane NB-1} (8 bytes for NB = 2, 16 bytes for NB = 4) so that
// one LDS.64 / LDS.128 fetches all of them.  2- and 4-bit input has one sub-row per channel; 8-bit input
// has two (planes 0-3 and planes 4-7), handled as two 4-plane channels of the same delay whose words carry
// weights 1..8 and 16..128.  With W odd, the lanes of a warp (W units = W * 4 NB bytes apart) fall into
// distinct shared-memory banks.
//
// One CTA = 16 DM trials x (32 * 32 * W) output samples, 16 warps; warp w owns DM slot w, lane l owns the W
// units W l .. W l + W - 1 of the time block (W + 1 loads serve W units).
//   stage  : per channel, the bit-plane span [t0 + start, ...) of the DM block (time block + delay range,
//            PAPER.md:115) arrives by TMA bulk copy; ring of `nstages` stages of CC channels, full/empty
//            mbarriers, no CTA-wide barrier in the channel loop;
//   add    : carry-save counter per unit; words of equal weight are paired as they appear (a binary counter
//            of pending words, resolved at compile time), the pending words left after a stage are rippled
//            into the upper planes;
//   store  : bit-matrix transposes turn NP planes x 32 lanes into 32 integers; float32 / uint32 / uint16,
//            128-bit stores, time contiguous.
#include <mutex>
#include <utility>

#include "dd_bp_core.cuh"

namespace dd {
namespace {

constexpr int BP_DB = 16, BP_NWARPS = 16;

// Tile shape per input width.  FL = stages between flushes of the pending words in the LONG instantiation
// (dd_plan.cpp pads the channel list accordingly: kBpFlushStages there must agree).
#ifndef DD_PAIR_FL
#define DD_PAIR_FL 4   // stages between flushes of the pair-row kernels (dd_plan.cpp: the same)
#endif
#ifndef DD_BP_W2
#define DD_BP_W2 5     // units per lane of the 2-bit kernel (dd_plan.cpp: the tile is 1024 * DD_BP_W2 samples)
#endif
#ifndef DD_BP_FL2
#define DD_BP_FL2 2   // measured on B200: cfg2 8.95 / 8.78 / 9.09 ms for 1 / 2 / 4 stages between flushes
#define DD_BP_FL4 4   //                  cfg4 116.7 / 114.5 / 112.6 ms
#define DD_BP_FL8 2   //                  cfg5 246.4 / 223.7 / 224.8 ms
#endif
// Tile shape per input width.  NP planes hold sums < 2^NP (the plan checks nchans * (2^nbits - 1) < 2^NP).
template <int NBITS>
struct Bp;
template <>
struct Bp<2> {
    static constexpr int NB = 2, NSUB = 1, NP = 12, W = DD_BP_W2, CC = 32, FL = DD_BP_FL2;
};
template <>
struct Bp<3> {   // pair rows of 2-bit input (variant 4): 3 planes per unit (12 bytes, three LDS.32), 8 pairs per stage
    static constexpr int NB = 3, NSUB = 1, NP = 12, W = DD_BP_W2, CC = 8, FL = 4;
};
template <>
struct Bp<4> {
    static constexpr int NB = 4, NSUB = 1, NP = 16, W = 3, CC = 16, FL = DD_BP_FL4;
};
template <>
struct Bp<12> {   // pair rows of 8-bit input (variant 4): 9 planes in three 4-plane sub-rows, 4 pairs per stage
    static constexpr int NB = 4, NSUB = 3, NP = 20, W = 3, CC = 4, FL = 2;
};
template <>
struct Bp<8> {
    static constexpr int NB = 4, NSUB = 2, NP = 20, W = 3, CC = 8, FL = DD_BP_FL8;
};


// ------------------------------------------------------------------------------------------ pre-pass
// bits at even positions of y (y & 0x55555555 == y) -> the low 16 bits, order kept
__device__ __forceinline__ uint32_t compress_even(uint32_t y)
{
    y = (y | (y >> 1)) & 0x33333333u;
    y = (y | (y >> 2)) & 0x0F0F0F0Fu;
    y = (y | (y >> 4)) & 0x00FF00FFu;
    y = (y | (y >> 8)) & 0x0000FFFFu;
    return y;
}
// bits at positions 0, 4, .., 28 of y -> the low 8 bits, order kept
__device__ __forceinline__ uint32_t compress_4th(uint32_t y)
{
    y = (y | (y >> 3)) & 0x03030303u;
    y = (y | (y >> 6)) & 0x000F000Fu;
    y = (y | (y >> 12)) & 0x000000FFu;
    return y;
}
// bits at positions 0, 8, 16, 24 of y -> the low 4 bits, order kept
__device__ __forceinline__ uint32_t compress_8th(uint32_t y) { return (y | (y >> 7) | (y >> 14) | (y >> 21)) & 0xFu; }

// 32 two-bit samples (two packed words, LSB first) -> {plane 0, plane 1}; bit k of a plane = sample k
__device__ __forceinline__ uint2 planes_of(uint32_t x0, uint32_t x1)
{
    const uint32_t m = 0x55555555u;
    return make_uint2(compress_even(x0 & m) | (compress_even(x1 & m) << 16),
                      compress_even((x0 >> 1) & m) | (compress_even((x1 >> 1) & m) << 16));
}

// in: packed rows [beam][c][in_stride]; work: bit-plane rows [beam][c][sub][w_sub bytes].  One thread writes
// 16 bytes of every sub-row of a channel: 64 samples (2 units) of 2-bit input, 32 samples (1 unit) of 4- and
// 8-bit input.  Input bytes at or beyond in_row_bytes read as zero: the bit-plane rows are longer than the input
// (whole tiles plus the longest span), so that the transform kernel never has to clamp a copy.
template <int NBITS>
__global__ void __launch_bounds__(256) dd_to_bitplanes(const uint8_t *__restrict__ in, int64_t in_stride, int64_t in_row_bytes,
                                                       int64_t in_beam_stride, uint8_t *__restrict__ work, int64_t w_sub,
                                                       int64_t w_beam_stride, int32_t groups)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= groups)
        return;
    const int64_t c = blockIdx.y, beam = blockIdx.z;
    const uint8_t *row = in + beam * in_beam_stride + c * in_stride;
    uint8_t *wrow = work + beam * w_beam_stride + c * (Bp<NBITS>::NSUB * w_sub);
    if constexpr (NBITS == 2) {
        const uint4 x = (static_cast<int64_t>(i) * 16 + 16 <= in_row_bytes) ? __ldg(reinterpret_cast<const uint4 *>(row) + i)
                                                                          : make_uint4(0, 0, 0, 0);
        const uint2 a = planes_of(x.x, x.y), b = planes_of(x.z, x.w);
        reinterpret_cast<uint4 *>(wrow)[i] = make_uint4(a.x, a.y, b.x, b.y);
    } else if constexpr (NBITS == 4) {
        const uint4 x = (static_cast<int64_t>(i) * 16 + 16 <= in_row_bytes) ? __ldg(reinterpret_cast<const uint4 *>(row) + i)
                                                                          : make_uint4(0, 0, 0, 0);
        const uint32_t w[4] = {x.x, x.y, x.z, x.w};
        uint32_t pl[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            pl[k] = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q)   // word q = samples 8q .. 8q+7
                pl[k] |= compress_4th((w[q] >> k) & 0x11111111u) << (8 * q);
        }
        reinterpret_cast<uint4 *>(wrow)[i] = make_uint4(pl[0], pl[1], pl[2], pl[3]);
    } else {
        const int64_t b0 = static_cast<int64_t>(i) * 32;
        const uint4 z = make_uint4(0, 0, 0, 0);
        const uint4 xa = (b0 + 16 <= in_row_bytes) ? __ldg(reinterpret_cast<const uint4 *>(row + b0)) : z;
        const uint4 xb = (b0 + 32 <= in_row_bytes) ? __ldg(reinterpret_cast<const uint4 *>(row + b0 + 16)) : z;
        const uint32_t w[8] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
        uint32_t pl[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            pl[k] = 0;
#pragma unroll
            for (int q = 0; q < 8; ++q)   // word q = samples 4q .. 4q+3
                pl[k] |= compress_8th((w[q] >> k) & 0x01010101u) << (4 * q);
        }
        reinterpret_cast<uint4 *>(wrow)[i] = make_uint4(pl[0], pl[1], pl[2], pl[3]);
        reinterpret_cast<uint4 *>(wrow + w_sub)[i] = make_uint4(pl[4], pl[5], pl[6], pl[7]);
    }
}



struct BpShared {
    const uint8_t *lane_base;   // stage base + this lane's byte offset (W units per lane)
    const uint2 *rel;           // this warp's offset entries of the stage: [cl * BP_DB]
    int sub_slot;               // bytes between the sub-rows of a channel slot
    const uint8_t *lane_lone;   // LONE layouts: last sub-row of slot 0 + this lane's offset in it (4 bytes per unit)
};

// plane k of sub-row SUB of a channel, for every unit of the lane; CLS = channels added since the last flush
// PIN: planes of a sample that can be non-zero (NBITS, or fewer for the sub-band intermediate: the rest is skipped)
template <int NBITS, int PIN, int CLS, int SUB, int K, int NP, int NT>
__device__ __forceinline__ void plane_step(const PlaneVec<Bp<NBITS>::NB> (&x)[Bp<NBITS>::W + 1], uint32_t shift,
                                           uint32_t (&P)[Bp<NBITS>::W][NP], uint32_t (&T)[Bp<NBITS>::W][NT])
{
    using C = Bp<NBITS>;
    if constexpr (K < C::NB && SUB * C::NB + K < PIN) {
        constexpr int L = SUB * C::NB + K;                                   // weight 2^L
        constexpr uint32_t VMAX = (1u << PIN) - 1u;
        constexpr uint32_t S = VMAX * CLS + ((1u << L) - 1u);                // weight added to the counter so far
#pragma unroll
        for (int j = 0; j < C::W; ++j)
            csa_add<S, L>(P[j], T[j], __funnelshift_r(x[j].w[K], x[j + 1].w[K], shift));
        plane_step<NBITS, PIN, CLS, SUB, K + 1>(x, shift, P, T);
    }
}

// channel CL of the stage: per sub-row one window of W+1 units serves W units; per unit and plane one funnel
// shift + carry-save adds
// LONE (pair rows of 4- and 8-bit input): the last sub-row holds the carry plane alone, one word per unit; the offset
// entry carries the window's unit offset in e.y >> 8 (the funnel shift takes e.y modulo 32)
template <int NBITS, int PIN, bool LONE, int CLS, int SUB, int NP, int NT>
__device__ __forceinline__ void subrow_step(const BpShared &sh, const uint2 e, uint32_t (&P)[Bp<NBITS>::W][NP],
                                            uint32_t (&T)[Bp<NBITS>::W][NT])
{
    using C = Bp<NBITS>;
    if constexpr (LONE && SUB == C::NSUB - 1) {
        constexpr int L = SUB * C::NB;                                        // weight of the lone plane
        static_assert(PIN == L + 1, "the lone plane is the top plane of a pair sum");
        constexpr uint32_t S = ((1u << PIN) - 1u) * CLS + ((1u << L) - 1u);
        const uint32_t *wp = reinterpret_cast<const uint32_t *>(sh.lane_lone + e.x - (e.y >> 8) * 12u);
        uint32_t x[C::W + 1];
#pragma unroll
        for (int j = 0; j <= C::W; ++j)
            x[j] = wp[j];
#pragma unroll
        for (int j = 0; j < C::W; ++j)
            csa_add<S, L>(P[j], T[j], __funnelshift_r(x[j], x[j + 1], e.y));
    } else if constexpr (SUB < C::NSUB && SUB * C::NB < PIN) {
        const uint8_t *wp = sh.lane_base + e.x + SUB * sh.sub_slot;
        PlaneVec<C::NB> x[C::W + 1];
#pragma unroll
        for (int j = 0; j <= C::W; ++j)
            x[j].load(wp + j * (C::NB * 4));
        plane_step<NBITS, PIN, CLS, SUB, 0>(x, e.y, P, T);
        subrow_step<NBITS, PIN, LONE, CLS, SUB + 1>(sh, e, P, T);
    }
}

// PHASE: stages added since the last flush (the pending words are rippled into the planes every FL stages)
template <int NBITS, int PIN, bool LONE, int PHASE, int NP, int NT, int... CLs>
__device__ __forceinline__ void stage_steps(std::integer_sequence<int, CLs...>, const BpShared &sh,
                                            uint32_t (&P)[Bp<NBITS>::W][NP], uint32_t (&T)[Bp<NBITS>::W][NT])
{
    // rel entry: {byte offset in the stage, bit shift}
    (subrow_step<NBITS, PIN, LONE, PHASE * Bp<NBITS>::CC + CLs, 0>(sh, sh.rel[CLs * BP_DB], P, T), ...);
}





// LONG: the plan found many channels per group.  The pending words are then rippled into the planes only every
// Bp<NBITS>::FL stages (the plan pads the channel list to whole groups of FL stages), and for 8-bit input the
// epilogue stores straight from registers (a deeper stage ring is worth more than coalesced stores there).
// Otherwise: a flush after every stage, and the epilogue goes through per-warp shared-memory patches.
// PIN < NBITS (short instantiation, 8-bit input): only the low PIN planes of a sample can be set (the plan knows the
// largest sample of the sub-band intermediate), the others are neither shifted nor added.
// PAIRS (variant 4): the "channels" are pairs of channels; a stage holds, besides the offset entries of its CC pairs,
// the p.rows_per_chunk pair rows those pairs need for the delay differences of this DM block (span list
// [blk][chunk][rows_per_chunk]); every DM slot's offset entry points into the row of its own difference.
template <int NBITS, bool LONG, int PIN = NBITS, bool PAIRS = false>
__global__ void __launch_bounds__(BP_NWARPS * 32, 1) dd_direct_bp(const KernelParams p)
{
    using C = Bp<NBITS>;
    constexpr int DB = BP_DB, W = C::W, TB = 32 * 32 * W, CC = C::CC, NSUB = C::NSUB;
    // the short instantiation serves fewer than 8 * CC * FL channels per group: 8-bit sums then fit 16 planes and the
    // epilogue transposes 16 x 16 bit matrices instead of 32 x 32
    // (pair rows of 4-bit input: at most 31 per pair and 2114 pairs by plan construction -> 16 planes as well)
    constexpr int NP = (NBITS == 8 && (!LONG || PAIRS)) ? 16 : C::NP;
    static_assert(LONG || static_cast<int64_t>(8 * CC * C::FL) * ((1 << NBITS) - 1) <= (int64_t(1) << NP), "short-mode sums must fit NP planes");
    static_assert(PIN >= 1 && PIN <= NBITS, "planes in use");
    constexpr int UB = C::NB * 4;                                    // bytes per unit of a sub-row
    constexpr bool LONE = PAIRS && (NBITS == 8 || NBITS == 12);      // the last sub-row holds one plane, 4 bytes per unit
    constexpr int FL = LONG ? (PAIRS ? DD_PAIR_FL : C::FL) : 1;   // pair rows: flush every DD_PAIR_FL stages (the plan pads alike)
    constexpr bool PATCH = !LONG || (NBITS < 8 && (!PAIRS || NBITS == 3));   // 4-bit pair rows: the ring needs the shared memory more
    constexpr uint32_t STAGE_SUM = ((1u << PIN) - 1u) * CC;        // largest value one stage adds to a counter
    constexpr int NT = bit_length(FL * STAGE_SUM);                   // pending slots
    static_assert(PAIRS || (CC * NSUB) % BP_NWARPS == 0, "every warp stages the same number of sub-rows");

    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // tile decode: DM block fastest so that CTAs resident together share the same input window (L2)
    const int64_t cta = blockIdx.x;
    const int blk = static_cast<int>(cta % p.nblk);
    const int64_t rest = cta / p.nblk;
    // Short instantiation without pair rows: a CTA walks p.tpc consecutive time tiles of its DM block (the ring of stages
    // runs on across them, so the first copies of a tile and the drain of its output hide behind the tile before and
    // after -- CTAs of a few stages, as in step 2 of the sub-band method, otherwise expose both once per tile)
    constexpr bool MULTI = !LONG && !PAIRS;
    const int ntile_slots = MULTI ? (p.ntiles + p.tpc - 1) / p.tpc : p.ntiles;
    const int tile = MULTI ? static_cast<int>(rest % ntile_slots) * p.tpc : static_cast<int>(rest % p.ntiles) + (PAIRS ? p.tile0 : 0);
    const int batch = static_cast<int>(rest / ntile_slots);       // (beam, set of gpc channel groups); gpc = 1: (beam, group)
    int beam, group, nch_set = 0;   // group: the first one of the set; nch_set: stages this CTA works through
    if constexpr (LONG) {           // always one group per CTA
        beam = batch / p.ngroups, group = batch - beam * p.ngroups;
    } else {
        const int nsets = (p.ngroups + p.gpc - 1) / p.gpc;
        beam = batch / nsets, group = (batch - beam * nsets) * p.gpc;
        nch_set = min(p.gpc, p.ngroups - group) * p.nchunks * (MULTI ? min(p.tpc, p.ntiles - tile) : 1);
    }
    const bool walk = MULTI && p.tpc > 1;   // several tiles per CTA: stage k belongs to tile k / nchunks (gpc == 1 then)
    auto nchunks_cta = [&]() -> int {   // LONG: straight from the parameter bank, no register held across the loop
        if constexpr (LONG)
            return p.nchunks;
        else
            return nch_set;
    };
    const int64_t t0 = static_cast<int64_t>(tile) * TB;

    // shared memory carve-up (must match dd::smem_layout_bytes)
    const int NS = p.nstages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);      // [NS]
    uint64_t *empty = full + 8;                                 // [NS]
    const int rel_stage = static_cast<int>(align128(static_cast<int64_t>(CC) * DB * 8));
    const int raw_stage = static_cast<int>(align128(static_cast<int64_t>(PAIRS ? p.rows_per_chunk : CC) * p.raw_slot));
    uint8_t *rel_base = smem + 128 + (PATCH ? BP_NWARPS * kBpPatchBytes : 0);   // after the warps' output patches
    uint8_t *raw_base = rel_base + NS * rel_stage;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&full[s], BP_NWARPS);
            mbar_init(&empty[s], BP_NWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const uint8_t *in_beam = p.in + static_cast<int64_t>(beam) * p.in_beam_stride +
                             (p.in_blk_div > 0 ? static_cast<int64_t>(blk / p.in_blk_div) * p.in_blk_stride : 0);
    const int64_t unit_t0 = (t0 >> 5) - (PAIRS ? p.in_unit0 : 0);   // the tile's first unit inside the staged-from rows
    const uint8_t *in_tile = in_beam + unit_t0 * UB;   // this tile's first unit in every sub-row
    const int64_t col0 = static_cast<int64_t>(blk) * p.nchans_pad + static_cast<int64_t>(group) * p.group_cols;
    const int4 *span_blk = PAIRS ? p.span + static_cast<int64_t>(blk) * p.nchunks * p.rows_per_chunk : p.span + col0;
    const uint2 *rel_blk = static_cast<const uint2 *>(p.rel) + col0 * DB;

    // producers: EVERY warp stages CPW = CC * NSUB / NWARPS sub-rows of each chunk (its lane 0 issues the bulk
    // copies: a bulk copy takes its operands from uniform registers, so one warp issuing all copies of a chunk
    // serialises over its lanes and falls behind the others); warp 0 also stages the chunk's offset entries.
    // The span metadata of the next chunk to stage is fetched one step early.
    constexpr int CPW = PAIRS ? 3 : CC * NSUB / BP_NWARPS;   // PAIRS: rows per warp and stage (the plan keeps rows_per_chunk <= 48)
    auto load_meta = [&](int chunk, int4 (&m)[CPW]) {
#pragma unroll
        for (int k = 0; k < CPW; ++k) {
            if constexpr (PAIRS) {
                const int slot = warp + BP_NWARPS * k;
                m[k] = (lane == 0 && chunk < nchunks_cta() && slot < p.rows_per_chunk)
                           ? __ldg(&span_blk[static_cast<int64_t>(chunk) * p.rows_per_chunk + slot])
                           : make_int4(0, 0, 0, 0);
            } else {
                const int cm = walk ? chunk % p.nchunks : chunk;
                m[k] = (lane == 0 && chunk < nchunks_cta()) ? __ldg(&span_blk[cm * CC + (warp * CPW + k) / NSUB]) : make_int4(0, 0, 0, 0);
            }
        }
    };
    // chunk = round * NS + s: the ring position is carried along instead of divided out (NS is a run-time value)
    int prod_s = 0, prod_round = 0;
    auto produce = [&](int chunk, const int4 (&m)[CPW]) {
        const int s = prod_s;
        if (lane == 0) {
            if (prod_round > 0)
                mbar_wait(&empty[s], (prod_round - 1) & 1);   // every warp has finished chunk - NS
            // span entry: {byte offset inside the sub-row for tile 0, bytes, row, -}; rows are padded by the launcher
            // so that no copy needs clamping, and padded channels point at an all-zero row
            uint32_t tx = (warp == 0) ? static_cast<uint32_t>(CC * DB * 8) : 0u;
#pragma unroll
            for (int k = 0; k < CPW; ++k)
                tx += PAIRS ? (LONE ? static_cast<uint32_t>(m[k].y) * (NSUB - 1) + static_cast<uint32_t>(m[k].y) / 4u
                                    : static_cast<uint32_t>(m[k].y) * NSUB)
                            : static_cast<uint32_t>(m[k].y);
            mbar_arrive_expect_tx(&full[s], tx);
            if constexpr (PAIRS) {
#pragma unroll
                for (int k = 0; k < CPW; ++k) {
                    if (m[k].y > 0) {
                        const int slot = warp + BP_NWARPS * k;
#pragma unroll
                        for (int sub = 0; sub < NSUB; ++sub) {
                            if (LONE && sub == NSUB - 1)   // the lone plane: a quarter of the bytes at a quarter of the offset
                                tma_bulk_g2s(raw_base + s * raw_stage + slot * p.raw_slot + sub * p.sub_slot,
                                             in_beam + static_cast<int64_t>(m[k].z) * p.in_stride + sub * p.in_row_bytes +
                                                 (unit_t0 * UB + m[k].x) / 4,
                                             static_cast<uint32_t>(m[k].y) / 4u, &full[s]);
                            else
                                tma_bulk_g2s(raw_base + s * raw_stage + slot * p.raw_slot + sub * p.sub_slot,
                                             in_tile + static_cast<int64_t>(m[k].z) * p.in_stride + sub * p.in_row_bytes + m[k].x,
                                             static_cast<uint32_t>(m[k].y), &full[s]);
                        }
                    }
                }
            }
            // several tiles per CTA: the stage belongs to tile chunk / nchunks, its spans lie TB samples per tile further
            const int ct = walk ? chunk / p.nchunks : 0, cm = walk ? chunk - ct * p.nchunks : chunk;
            const uint8_t *in_here = in_tile + static_cast<int64_t>(ct) * (TB / 32) * UB;
#pragma unroll
            for (int k = 0; k < (PAIRS ? 0 : CPW); ++k) {
                const int cl = (warp * CPW + k) / NSUB, sub = (warp * CPW + k) % NSUB;
                const uint8_t *src = in_here + static_cast<int64_t>(m[k].z) * p.in_stride + sub * p.in_row_bytes + m[k].x;
                tma_bulk_g2s(raw_base + s * raw_stage + cl * p.raw_slot + sub * p.sub_slot, src, static_cast<uint32_t>(m[k].y),
                             &full[s]);
            }
            if (warp == 0)
                tma_bulk_g2s(rel_base + s * rel_stage, rel_blk + static_cast<int64_t>(cm) * CC * DB,
                             static_cast<uint32_t>(CC * DB * 8), &full[s]);
        }
        __syncwarp();
        if (++prod_s == NS) {
            prod_s = 0;
            ++prod_round;
        }
    };

    const int dist = NS > 2 ? NS - 2 : 1;   // prefetch distance in chunks (measured: 1 and 2 equal, 3 slower)
    int4 meta[CPW], nxt[CPW];
    load_meta(0, meta);
    for (int k = 0; k < dist && k < nchunks_cta(); ++k) {
        load_meta(k + 1, nxt);
        produce(k, meta);
#pragma unroll
        for (int i = 0; i < CPW; ++i)
            meta[i] = nxt[i];
    }

    uint32_t P[W][NP], T[W][NT];
#pragma unroll
    for (int j = 0; j < W; ++j) {
#pragma unroll
        for (int k = 0; k < NP; ++k)
            P[j][k] = 0;
#pragma unroll
        for (int k = 0; k < NT; ++k)
            T[j][k] = 0;
    }

    int s = 0;
    uint32_t full_parity = 0;
    // one stage: keep the ring fed, wait for the stage, add its CC channels (PHASE = stages since the last flush)
    // FLUSH = weight the counter has taken since the last flush if the pending words are to be rippled in now, else 0
    auto stage = [&](int chunk, auto phase, auto flush) {
        constexpr int PHASE = decltype(phase)::value;
        constexpr uint32_t FLUSH = decltype(flush)::value;
        if (chunk + dist < nchunks_cta()) {
            load_meta(chunk + dist + 1, nxt);
            produce(chunk + dist, meta);
#pragma unroll
            for (int i = 0; i < CPW; ++i)
                meta[i] = nxt[i];
        }
        mbar_wait(&full[s], full_parity);

        BpShared sh;
        sh.lane_base = raw_base + s * raw_stage + lane * (W * UB);
        sh.rel = reinterpret_cast<const uint2 *>(rel_base + s * rel_stage) + warp;
        sh.sub_slot = p.sub_slot;
        sh.lane_lone = raw_base + s * raw_stage + (NSUB - 1) * p.sub_slot + lane * (W * 4);
        stage_steps<NBITS, PIN, LONE, PHASE>(std::make_integer_sequence<int, CC>{}, sh, P, T);
        if constexpr (FLUSH != 0u) {
#pragma unroll
            for (int j = 0; j < W; ++j)
                csa_flush<FLUSH, 0, false>(P[j], T[j], 0u);
        }
        __syncwarp();
        if (lane == 0)
            mbar_arrive(&empty[s]);
        if (++s == NS) {
            s = 0;
            full_parity ^= 1u;
        }
    };
    // groups of FL stages with one flush at the end (nchunks is a multiple of FL by plan construction)
    using NoFlush = std::integral_constant<uint32_t, 0u>;
    using FlushAll = std::integral_constant<uint32_t, FL * STAGE_SUM>;
    // Bit-plane output (kOutPlanes, the intermediate series of the sub-band method): the counter's low 8 planes ARE
    // the 8-bit samples of the next step in the layout its stages want, so they are stored as they stand -- no
    // transposes, no pre-pass afterwards -- and the CTA carries on with its next channel group while the ring keeps
    // the copies of that group in flight.
    [[maybe_unused]] auto store_planes = [&](int g) {
        const int dpl = blk * DB + warp;
        if (dpl < p.ndm) {
            uint8_t *row = p.out + static_cast<int64_t>(beam) * p.pl_beam +
                           (static_cast<int64_t>(g) * p.ndm + dpl) * (2 * p.pl_conv);
            const int64_t u0 = (t0 >> 5) + W * lane;
#pragma unroll
            for (int j = 0; j < W; ++j) {
                if (u0 + j < p.pl_units) {
                    uint8_t *dst = row + (u0 + j) * 16;
                    *reinterpret_cast<uint4 *>(dst) = make_uint4(P[j][0], P[j][1], P[j][2], P[j][3]);
                    *reinterpret_cast<uint4 *>(dst + p.pl_conv) = make_uint4(P[j][4], P[j][5], P[j][6], P[j][7]);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < W; ++j) {
#pragma unroll
            for (int k = 0; k < NP; ++k)
                P[j][k] = 0;
        }
    };
    // ---- epilogue of one tile: thread owns samples t0x + 32*(W*lane + j) + [0, 32) of DM slot `warp`
    // Interior tiles (the whole time block inside the row, vector stores allowed) go through a per-warp patch of
    // shared memory so that every store instruction writes whole 128-byte lines.  The patches lie outside the
    // stage ring: a warp that is done stores while the others are still adding.
    auto store_out = [&](int64_t t0x) {
        const int d = blk * DB + warp;
        if (d >= p.ndm)
            return;
        const int esize = (p.out_code == DD_OUT_U16) ? 2 : (p.out_code == kOutU8 ? 1 : 4);
        uint8_t *orow = p.out + static_cast<int64_t>(batch) * p.out_beam_stride + static_cast<int64_t>(d) * p.out_dm_stride;
        const bool interior = PATCH && p.vec16_ok && (t0x + TB <= p.nsamps);   // 16-byte stores: rows must be 16-byte aligned
        uint8_t *patch = smem + 128 + warp * kBpPatchBytes;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            uint32_t q[32];   // the 32 sums of the unit, in time order
            if constexpr (NP <= 16) {
                uint32_t R[16];
#pragma unroll
                for (int k = 0; k < 16; ++k)
                    R[k] = k < NP ? P[j][k] : 0u;
                transpose16x2(R);
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    q[k] = R[k] & 0xFFFFu;
                    q[16 + k] = R[k] >> 16;
                }
            } else {
#pragma unroll
                for (int k = 0; k < 32; ++k)
                    q[k] = k < NP ? P[j][k] : 0u;
                transpose32(q);
            }
            if (interior) {
                uint8_t *gunit = orow + (t0x + 32 * j) * esize;   // unit j of lane 0; lane s is W * 32 samples further
                if (p.out_code == DD_OUT_F32)
                    store_unit_coalesced<4, true>(q, patch, lane, gunit, W * 32 * 4);
                else if (p.out_code == DD_OUT_U32)
                    store_unit_coalesced<4, false>(q, patch, lane, gunit, W * 32 * 4);
                else if (p.out_code == DD_OUT_U16)
                    store_unit_coalesced<2, false>(q, patch, lane, gunit, W * 32 * 2);
                else
                    store_unit_coalesced<1, false>(q, patch, lane, gunit, W * 32);
            } else {
                const int64_t tunit = t0x + 32 * (W * lane + j);
#pragma unroll
                for (int h = 0; h < 8; ++h) {   // samples 4h .. 4h+3 of the unit
                    const uint32_t q4[4] = {q[4 * h], q[4 * h + 1], q[4 * h + 2], q[4 * h + 3]};
                    store4(p, orow, tunit + 4 * h, q4);
                }
            }
        }
    };
    int cig = 0, gi = 0;   // stages done of the current group / tile, groups / tiles done
    for (int chunk = 0; chunk < nchunks_cta(); chunk += FL) {
        if constexpr (FL == 1) {
            stage(chunk, std::integral_constant<int, 0>{}, FlushAll{});
            if (++cig == p.nchunks) {   // a channel group (bit-plane output) or a time tile is complete
                cig = 0;
                if (p.out_code == kOutPlanes) {
                    store_planes(group + gi);
                } else {
                    store_out(t0 + static_cast<int64_t>(gi) * TB);
#pragma unroll
                    for (int j = 0; j < W; ++j) {
#pragma unroll
                        for (int k = 0; k < NP; ++k)
                            P[j][k] = 0;
                    }
                }
                ++gi;
            }
        } else if constexpr (FL == 2) {
            stage(chunk, std::integral_constant<int, 0>{}, NoFlush{});
            stage(chunk + 1, std::integral_constant<int, 1>{}, FlushAll{});
        } else {
            static_assert(FL == 1 || FL == 2 || FL == 4, "unroll more phases here");
            stage(chunk, std::integral_constant<int, 0>{}, NoFlush{});
            stage(chunk + 1, std::integral_constant<int, 1>{}, NoFlush{});
            stage(chunk + 2, std::integral_constant<int, 2>{}, NoFlush{});
            stage(chunk + 3, std::integral_constant<int, 3>{}, FlushAll{});
        }
    }
    if constexpr (FL > 1)   // (with a flush after every stage the tiles were stored inside the loop)
        store_out(t0);
}

template <int NBITS>
cudaError_t prepare_bp(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, bool zero_all, BpWork *w)
{
    using C = Bp<NBITS>;
    const int64_t TB = plan->var.TB;   // (variant 5 has its own tile length)
    // 16-byte groups of every sub-row the tiles can touch (2 units of 2-bit input, 1 unit otherwise).  The bit-plane
    // rows are as long as the longest span needs, zero beyond the input, so that the kernel's copies need no
    // clamping; behind the nrows input rows of a beam lie row_mul all-zero rows, the source of padded channels.
    const int64_t spg = (16 / (C::NB * 4)) * 32;   // samples per group
    w->units = (static_cast<int64_t>(kp.ntiles - 1) * TB + plan->max_span_end + spg - 1) / spg;
    w->conv = w->units * 16;   // bytes per sub-row
    w->rows = static_cast<int64_t>(kp.nrows) + kp.row_mul;
    w->w_beam = w->rows * C::NSUB * w->conv;
    const size_t need = static_cast<size_t>(kp.nbeams) * static_cast<size_t>(w->w_beam);
    cudaError_t e;
    if (plan->work_bytes < need) {
        if (plan->d_work)
            cudaFree(plan->d_work);   // synchronises with any kernel still reading the old buffer
        plan->d_work = nullptr;
        plan->work_bytes = 0;
        plan->work_layout[0] = 0;
        if ((e = cudaMalloc(&plan->d_work, need)) != cudaSuccess)
            return e;
        plan->work_bytes = need;
    }
    if (plan->work_layout[0] != w->conv || plan->work_layout[1] != w->rows || plan->work_layout[2] != kp.nbeams ||
        plan->work_layout[3] != (zero_all ? 1 : 0)) {
        if (zero_all)
            e = cudaMemsetAsync(plan->d_work, 0, need, stream);
        else
            e = cudaMemset2DAsync(static_cast<uint8_t *>(plan->d_work) + static_cast<int64_t>(kp.nrows) * C::NSUB * w->conv,
                                  static_cast<size_t>(w->w_beam), 0, static_cast<size_t>(kp.row_mul) * C::NSUB * w->conv,
                                  kp.nbeams, stream);
        if (e != cudaSuccess)
            return e;
        plan->work_layout[0] = w->conv;
        plan->work_layout[1] = w->rows;
        plan->work_layout[2] = kp.nbeams;
        plan->work_layout[3] = zero_all ? 1 : 0;
    }
    return cudaSuccess;
}

template <int NBITS>
cudaError_t launch_bp(dd_plan_s *plan, const KernelParams &kp_in, cudaStream_t stream, bool planes_ready)
{
    using C = Bp<NBITS>;
    constexpr int TB = 32 * 32 * C::W;
    if (plan->cc != C::CC || plan->var.TB != TB || plan->var.DB != BP_DB)
        return cudaErrorInvalidValue;
    KernelParams kp = kp_in;
    BpWork w;
    cudaError_t e = prepare_bp<NBITS>(plan, kp, stream, planes_ready, &w);
    if (e != cudaSuccess)
        return e;
    if (!planes_ready) {
        dd_to_bitplanes<NBITS><<<dim3(static_cast<unsigned>((w.units + 255) / 256), kp.nrows, kp.nbeams), 256, 0, stream>>>(
            kp.in, kp.in_stride, kp.in_row_bytes, kp.in_beam_stride, static_cast<uint8_t *>(plan->d_work), w.conv, w.w_beam,
            static_cast<int32_t>(w.units));
        if ((e = cudaGetLastError()) != cudaSuccess)
            return e;
    }
    if (plan->prof_mid)
        cudaEventRecord(static_cast<cudaEvent_t>(plan->prof_mid), stream);
    kp.in = static_cast<const uint8_t *>(plan->d_work);
    kp.in_stride = C::NSUB * w.conv * kp.row_mul;   // between channel indices; sub-rows are in_row_bytes apart
    kp.in_blk_stride = C::NSUB * w.conv;            // between the rows of one channel index (sub-band step 2)
    kp.in_row_bytes = w.conv;
    kp.in_beam_stride = w.w_beam;
    if (kp.out_code == kOutPlanes && plan->long_mode)
        return cudaErrorInvalidValue;   // bit-plane output is compiled into the short instantiation only
    if (kp.gpc < 1 || kp.out_code != kOutPlanes)
        kp.gpc = 1;

    const int64_t nsets = (kp.ngroups + kp.gpc - 1) / kp.gpc;
    // short plans (few stages per tile: step 2 of the sub-band method, small transforms): a CTA walks several time tiles,
    // as many as leave >= 8 waves of CTAs, at most 8 (dd_set_tuning(DD_TUNE_TILES_PER_CTA) overrides)
    kp.tpc = 1;
    if (!plan->long_mode && kp.out_code != kOutPlanes && kp.gpc == 1) {
        int sms = 148;
        (void)cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, plan->device >= 0 ? plan->device : 0);
        const int64_t all = static_cast<int64_t>(kp.nblk) * kp.ntiles * kp.nbeams * nsets;
        int64_t t = plan->bp_tpc > 0 ? plan->bp_tpc : all / (8 * static_cast<int64_t>(sms));
        t = t < 1 ? 1 : (t > 8 && plan->bp_tpc <= 0 ? 8 : t);
        kp.tpc = static_cast<int32_t>(t > kp.ntiles ? kp.ntiles : t);
    }
    const int64_t ctas = static_cast<int64_t>(kp.nblk) * ((kp.ntiles + kp.tpc - 1) / kp.tpc) * kp.nbeams * nsets;
    if (ctas <= 0 || ctas > 0x7FFFFFFFLL)
        return cudaErrorInvalidConfiguration;
    if (plan->long_mode && kp.nchunks % C::FL != 0)
        return cudaErrorInvalidValue;
    auto kernel = plan->long_mode ? dd_direct_bp<NBITS, true> : dd_direct_bp<NBITS, false>;
    // samples known to stay below 2^in_planes (sub-band step 2; scrunched series via dd_set_input_max): the
    // instantiation that skips the planes which cannot be set
    const int pin = plan->in_planes > 0 ? plan->in_planes : NBITS;
    if constexpr (NBITS == 8) {
        if (plan->long_mode)
            kernel = pin <= 5 ? dd_direct_bp<8, true, 5> : pin == 6 ? dd_direct_bp<8, true, 6> : pin == 7 ? dd_direct_bp<8, true, 7> : kernel;
        else
            kernel = pin <= 6 ? dd_direct_bp<8, false, 6> : pin == 7 ? dd_direct_bp<8, false, 7> : kernel;
    } else if constexpr (NBITS == 4) {
        if (plan->long_mode && pin <= 3)
            kernel = dd_direct_bp<4, true, 3>;
    }
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes));
    if (e != cudaSuccess)
        return e;
    kernel<<<dim3(static_cast<unsigned>(ctas)), dim3(BP_NWARPS * 32), plan->smem_bytes, stream>>>(kp);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------ pair rows (variant 4)
// S[t] = x[c0][t] + x[c1][t + delta] in bit planes, for every pair row {c0, c1, delta}: NBITS planes + NBITS planes ->
// NBITS + 1 planes by a ripple of full adders (xor3 / maj3), written in the layout of the consumer kernel
// (2-bit input: 3 planes per unit, 12 bytes; 4-bit input: 2 sub-rows of 4 planes, 5 in use).  One thread per (row, unit).  in: bit-plane rows of the input [c][unit][NBITS
// planes], in_units units per row, zero beyond the input; a killed partner (c1 < 0) contributes nothing.
template <int NBITS>
__global__ void __launch_bounds__(256) dd_make_pair_rows(const uint32_t *__restrict__ in, int64_t in_row_words, int64_t in_units,
                                                         const int4 *__restrict__ prow, uint32_t *__restrict__ out,
                                                         int64_t out_sub_words, int64_t out_units, int64_t ublocks, int64_t unit0)
{
    // out holds the units unit0 .. unit0 + out_units - 1 of every row (a group of time tiles); out_sub_words is the
    // pitch of a 4-plane sub-row of the buffer
    constexpr int NBI = Bp<NBITS>::NB, NSUBI = Bp<NBITS>::NSUB;   // input layout: NSUBI sub-rows of NBI planes per unit
    constexpr int NSUBO = NBITS == 2 ? 1 : (NBITS == 4 ? 2 : 3);
    const int64_t blk = blockIdx.x;
    const int64_t r = blk / ublocks, ul = (blk - r * ublocks) * blockDim.x + threadIdx.x;   // unit inside the buffer
    if (ul >= out_units)
        return;
    const int64_t u = unit0 + ul;                                                           // unit of the row
    const int4 pr = __ldg(&prow[r]);
    const int64_t in_sub_words = in_row_words / NSUBI;
    uint32_t a[NBITS], b[NBITS];
    const uint32_t *ra = in + static_cast<int64_t>(pr.x) * in_row_words;
#pragma unroll
    for (int k = 0; k < NBITS; ++k)
        a[k] = u < in_units ? ra[(k / NBI) * in_sub_words + u * NBI + (k % NBI)] : 0u;
    if (pr.y >= 0) {
        const int64_t ub = u + (pr.z >> 5);
        const uint32_t sh = static_cast<uint32_t>(pr.z) & 31u;
        const uint32_t *rb = in + static_cast<int64_t>(pr.y) * in_row_words;
#pragma unroll
        for (int k = 0; k < NBITS; ++k) {
            const uint32_t *q = rb + (k / NBI) * in_sub_words + ub * NBI + (k % NBI);
            const uint32_t lo = ub < in_units ? q[0] : 0u, hi = ub + 1 < in_units ? q[NBI] : 0u;
            b[k] = __funnelshift_r(lo, hi, sh);
        }
    } else {
#pragma unroll
        for (int k = 0; k < NBITS; ++k)
            b[k] = 0u;
    }
    uint32_t sum[NBITS + 1], cy = 0u;
#pragma unroll
    for (int k = 0; k < NBITS; ++k) {
        sum[k] = xor3(a[k], b[k], cy);
        cy = maj3(a[k], b[k], cy);
    }
    sum[NBITS] = cy;
    if constexpr (NBITS == 2) {   // 3 planes per unit, 12 bytes (consecutive threads write consecutive units)
        uint32_t *o3 = out + r * out_sub_words + ul * 3;
        o3[0] = sum[0], o3[1] = sum[1], o3[2] = sum[2];
    } else {                      // sub-rows of 4 planes, then the carry plane alone at 4 bytes per unit
        uint32_t *o = out + r * ((NSUBO - 1) * out_sub_words + out_sub_words / 4) + ul * 4;
#pragma unroll
        for (int q = 0; q < NSUBO - 1; ++q)
            *reinterpret_cast<uint4 *>(o + q * out_sub_words) = make_uint4(sum[4 * q], sum[4 * q + 1], sum[4 * q + 2], sum[4 * q + 3]);
        out[r * ((NSUBO - 1) * out_sub_words + out_sub_words / 4) + (NSUBO - 1) * out_sub_words + ul] = sum[NBITS];   // the lone carry plane
    }
}

// NBITS: input width; the consumer is the bit-plane kernel with the layout Bp<ENB> and NBITS + 1 planes in use
template <int NBITS>
cudaError_t launch_pairs(dd_plan_s *plan, const KernelParams &kp_in, cudaStream_t stream)
{
    constexpr int ENB = NBITS == 2 ? 3 : (NBITS == 4 ? 8 : 12);   // pair-row layout: 3 planes per unit / 4 + 1 planes / 4 + 4 + 1
    using C = Bp<ENB>;
    using CI = Bp<NBITS>;                      // layout of the input bit planes
    constexpr int TB = 32 * 32 * C::W;
    constexpr int UBO = C::NB * 4;             // bytes per unit of a pair-row sub-row
    constexpr bool LONEL = NBITS != 2;         // last sub-row: the carry plane alone, a quarter of the bytes
    if (!plan->pairs || plan->pair_nbits != ENB || plan->cc != C::CC || plan->var.TB != TB || plan->var.DB != BP_DB ||
        kp_in.ngroups != 1 || !plan->d_prow || kp_in.out_code == kOutPlanes)
        return cudaErrorInvalidValue;
    if (plan->long_mode && kp_in.nchunks % DD_PAIR_FL != 0)
        return cudaErrorInvalidValue;
    cudaError_t e;
    int32_t max_delta = 0;
    for (int64_t r = 0; r < plan->n_prows; ++r)
        max_delta = plan->prow[4 * r + 2] > max_delta ? plan->prow[4 * r + 2] : max_delta;
    // The pair rows are made per beam and per GROUP of time tiles into one of two buffers, on two internal streams that
    // alternate between groups, so that the rows of one group are built while the other is transformed and the device
    // memory taken is two groups' worth whatever the number of beams.  A group is the whole time axis unless its rows
    // would exceed the budget below.  (Groups small enough to keep the rows in L2 -- 1 to 32 tiles on cfg2 -- were
    // measured: 15.5 ... 9.07 ms against 8.77 ms for one group; the launches fragment the machine more than the saved
    // DRAM round trip gives back.)
    const int64_t tile_units = TB / 32;
    const int64_t extra_units = ((plan->max_span_end + 31) / 32 - tile_units + 3) / 4 * 4;   // span beyond a tile's own units
    const int64_t rows_o = plan->n_prows + 1;                                                  // + the all-zero row of padded entries
    auto pitch_of = [&](int64_t units) { return LONEL ? (C::NSUB - 1) * units * UBO + units * UBO / 4 : C::NSUB * units * UBO; };
    // Tiles per group: fixed when the plan first meets this launch geometry (time tiles x beams) and kept afterwards, so
    // that later calls neither query the device nor re-allocate.  The budget of a group's rows is the caller's limit
    // (dd_set_workspace_limit), else 3/4 of the device memory free at that moment; two groups are alive with several
    // beams or a split time axis.  dd_set_tuning(DD_TUNE_PAIR_TILES) overrides the choice (tests).
    int64_t G;
    if (plan->pair_tiles > 0) {
        G = plan->pair_tiles;
    } else if (plan->pair_geom[0] == kp_in.ntiles && plan->pair_geom[1] == kp_in.nbeams && plan->pair_geom[2] > 0) {
        G = plan->pair_geom[2];
    } else {
        const int64_t whole = rows_o * pitch_of(static_cast<int64_t>(kp_in.ntiles) * tile_units + extra_units);
        const int64_t want = kp_in.nbeams > 1 ? 2 * whole : whole;
        int64_t budget = plan->ws_limit;
        if (budget <= 0) {
            size_t free_b = 0, total_b = 0;
            if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) {
                (void)cudaGetLastError();
                free_b = size_t(8) << 30;
            }
            budget = static_cast<int64_t>((free_b + plan->pairwork_bytes) / 4 * 3);
        }
        budget = want <= budget ? whole : budget / 2;
        G = (budget - rows_o * pitch_of(extra_units)) / (rows_o * pitch_of(tile_units));
        if (G < 1)
            return cudaErrorMemoryAllocation;   // not even one tile's rows fit the limit
        G = G > kp_in.ntiles ? kp_in.ntiles : G;
        plan->pair_geom[0] = kp_in.ntiles;
        plan->pair_geom[1] = kp_in.nbeams;
        plan->pair_geom[2] = G;
    }
    G = G < 1 ? 1 : (G > kp_in.ntiles ? kp_in.ntiles : G);
    const int64_t units_g = G * tile_units + extra_units, conv_g = units_g * UBO, pitch_g = pitch_of(units_g);
    const int64_t buf_bytes = rows_o * pitch_g;
    // input bit planes of the whole call (one transpose), long enough for the last group's rows plus the largest difference
    const int64_t all_units = static_cast<int64_t>(kp_in.ntiles) * tile_units + extra_units;
    const int64_t spg = (16 / (CI::NB * 4)) * 32;                            // input samples per 16-byte group of a sub-row
    const int64_t groups_i = (all_units * 32 + max_delta + 64 + spg - 1) / spg;
    const int64_t conv_i = groups_i * 16, in_units = conv_i / (CI::NB * 4);  // bytes per sub-row, units per row
    const int64_t beam_i = static_cast<int64_t>(kp_in.nrows) * CI::NSUB * conv_i;
    const int64_t ngroups_all = static_cast<int64_t>(kp_in.nbeams) * ((kp_in.ntiles + G - 1) / G);
    const int nbuf = ngroups_all >= 2 ? 2 : 1;
    const size_t need_i = static_cast<size_t>(kp_in.nbeams) * beam_i, need_o = static_cast<size_t>(nbuf) * static_cast<size_t>(buf_bytes);
    if (plan->work_bytes < need_i) {
        if (plan->d_work)
            cudaFree(plan->d_work);
        plan->d_work = nullptr;
        plan->work_bytes = 0;
        if ((e = cudaMalloc(&plan->d_work, need_i)) != cudaSuccess)
            return e;
        plan->work_bytes = need_i;
    }
    plan->work_layout[0] = 0;   // the direct launcher must re-establish its zero rows if the plan goes back to it
    if (plan->pairwork_bytes < need_o) {
        if (plan->d_pairwork)
            cudaFree(plan->d_pairwork);
        plan->d_pairwork = nullptr;
        plan->pairwork_bytes = 0;
        if ((e = cudaMalloc(&plan->d_pairwork, need_o)) != cudaSuccess)
            return e;
        plan->pairwork_bytes = need_o;
    }
    for (int i = 0; i < 2; ++i) {   // stored in the plan as they are created: dd_plan_destroy frees whatever exists
        if (!plan->pair_streams[i]) {
            cudaStream_t st;
            if ((e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking)) != cudaSuccess)
                return e;
            plan->pair_streams[i] = st;
        }
    }
    for (int i = 0; i < 3; ++i) {
        if (!plan->pair_events[i]) {
            cudaEvent_t ev;
            if ((e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess)
                return e;
            plan->pair_events[i] = ev;
        }
    }
    cudaStream_t ws[2] = {static_cast<cudaStream_t>(plan->pair_streams[0]), static_cast<cudaStream_t>(plan->pair_streams[1])};
    cudaEvent_t fork = static_cast<cudaEvent_t>(plan->pair_events[0]);
    uint8_t *buf[2] = {static_cast<uint8_t *>(plan->d_pairwork), static_cast<uint8_t *>(plan->d_pairwork) + (nbuf - 1) * buf_bytes};

    dd_to_bitplanes<NBITS><<<dim3(static_cast<unsigned>((groups_i + 255) / 256), kp_in.nrows, kp_in.nbeams), 256, 0, stream>>>(
        kp_in.in, kp_in.in_stride, kp_in.in_row_bytes, kp_in.in_beam_stride, static_cast<uint8_t *>(plan->d_work), conv_i, beam_i,
        static_cast<int32_t>(groups_i));
    if ((e = cudaGetLastError()) != cudaSuccess)
        return e;
    if (plan->prof_mid)
        cudaEventRecord(static_cast<cudaEvent_t>(plan->prof_mid), stream);
    auto kernel = plan->long_mode ? dd_direct_bp<ENB, true, NBITS + 1, true> : dd_direct_bp<ENB, false, NBITS + 1, true>;
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes))) != cudaSuccess)
        return e;
    const int64_t ublocks = (units_g + 255) / 256;
    if (plan->n_prows * ublocks > 0x7FFFFFFFLL || static_cast<int64_t>(kp_in.nblk) * G > 0x7FFFFFFFLL)
        return cudaErrorInvalidConfiguration;
    // fork: both work streams wait for the transpose (and for everything the caller enqueued before).  From here on an
    // error does not return before the join below, so that the caller's stream (and a capture in progress) stays whole.
    cudaEventRecord(fork, stream);
    for (int i = 0; i < 2; ++i)
        cudaStreamWaitEvent(ws[i], fork, 0);
    e = cudaSuccess;
    for (int i = 0; i < nbuf && e == cudaSuccess; ++i)
        e = cudaMemsetAsync(buf[i] + plan->n_prows * pitch_g, 0, static_cast<size_t>(pitch_g), ws[i]);   // the zero row
    int launches = 1, it = 0;
    for (int b = 0; b < kp_in.nbeams && e == cudaSuccess; ++b) {
        for (int64_t c0 = 0; c0 < kp_in.ntiles && e == cudaSuccess; c0 += G, ++it) {
            const int sl = nbuf == 2 ? (it & 1) : 0;
            const int64_t gc = (c0 + G <= kp_in.ntiles) ? G : kp_in.ntiles - c0;
            const int64_t unit0 = c0 * tile_units;
            dd_make_pair_rows<NBITS><<<dim3(static_cast<unsigned>(plan->n_prows * ublocks)), 256, 0, ws[sl]>>>(
                reinterpret_cast<const uint32_t *>(static_cast<const uint8_t *>(plan->d_work) + b * beam_i), CI::NSUB * conv_i / 4,
                in_units, static_cast<const int4 *>(plan->d_prow), reinterpret_cast<uint32_t *>(buf[sl]), conv_g / 4, units_g, ublocks,
                unit0);
            if ((e = cudaGetLastError()) != cudaSuccess)
                break;
            KernelParams kp = kp_in;
            kp.in = buf[sl];
            kp.in_stride = pitch_g;
            kp.in_blk_stride = 0;
            kp.in_row_bytes = conv_g;
            kp.in_beam_stride = 0;
            kp.out = kp_in.out + static_cast<int64_t>(b) * kp_in.out_beam_stride;
            kp.nbeams = 1;
            kp.gpc = 1;
            kp.rows_per_chunk = plan->rows_per_chunk;
            kp.tile0 = static_cast<int32_t>(c0);
            kp.ntiles = static_cast<int32_t>(gc);
            kp.in_unit0 = unit0;
            kernel<<<dim3(static_cast<unsigned>(static_cast<int64_t>(kp.nblk) * gc)), dim3(BP_NWARPS * 32), plan->smem_bytes, ws[sl]>>>(kp);
            e = cudaGetLastError();
            launches += 2;
        }
    }
    // join: the caller's stream continues when both work streams are done
    for (int i = 0; i < 2; ++i) {
        cudaEvent_t jn = static_cast<cudaEvent_t>(plan->pair_events[1 + i]);
        cudaEventRecord(jn, ws[i]);
        cudaStreamWaitEvent(stream, jn, 0);
    }
    if (e != cudaSuccess)
        return e;
    plan->pair_launches = launches;
    return cudaSuccess;
}

}  // namespace

// Two launches: the bit-plane transpose of the rows the tiles will read, then the dedispersion kernel.
cudaError_t launch_variant3(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, bool planes_ready)
{
    if (!plan->var.bitplane)
        return cudaErrorInvalidValue;
    switch (plan->nbits) {
    case 2:
        return launch_bp<2>(plan, kp, stream, planes_ready);
    case 4:
        return launch_bp<4>(plan, kp, stream, planes_ready);
    case 8:
        return launch_bp<8>(plan, kp, stream, planes_ready);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_variant4(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    switch (plan->nbits) {
    case 2:
        return launch_pairs<2>(plan, kp, stream);
    case 4:
        return launch_pairs<4>(plan, kp, stream);
    case 8:
        return launch_pairs<8>(plan, kp, stream);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_to_bitplanes(dd_plan_s *plan, const KernelParams &kp, const BpWork &w, cudaStream_t stream)
{
    const dim3 grid(static_cast<unsigned>((w.units + 255) / 256), kp.nrows, kp.nbeams);
    uint8_t *work = static_cast<uint8_t *>(plan->d_work);
    switch (plan->nbits) {
    case 2:
        dd_to_bitplanes<2><<<grid, 256, 0, stream>>>(kp.in, kp.in_stride, kp.in_row_bytes, kp.in_beam_stride, work, w.conv, w.w_beam,
                                                     static_cast<int32_t>(w.units));
        break;
    case 4:
        dd_to_bitplanes<4><<<grid, 256, 0, stream>>>(kp.in, kp.in_stride, kp.in_row_bytes, kp.in_beam_stride, work, w.conv, w.w_beam,
                                                     static_cast<int32_t>(w.units));
        break;
    case 8:
        dd_to_bitplanes<8><<<grid, 256, 0, stream>>>(kp.in, kp.in_stride, kp.in_row_bytes, kp.in_beam_stride, work, w.conv, w.w_beam,
                                                     static_cast<int32_t>(w.units));
        break;
    default:
        return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t bp_prepare_work(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, bool zero_all, BpWork *w)
{
    if (!plan->var.bitplane)
        return cudaErrorInvalidValue;
    switch (plan->nbits) {
    case 2:
        return prepare_bp<2>(plan, kp, stream, zero_all, w);
    case 4:
        return prepare_bp<4>(plan, kp, stream, zero_all, w);
    case 8:
        return prepare_bp<8>(plan, kp, stream, zero_all, w);
    }
    return cudaErrorInvalidValue;
}

}  // namespace dd

// ------------------------------------------------------------------------------------------ dd_execute_static
// Variant 3 for callers that may not allocate (include/dd.h: dd_execute_static): the bit-plane copy of the input
// lives in this array instead of plan->d_work.  One array per device that loads the library, shared by every call;
// it keeps the last call's contents, so each call writes everything it reads (dd_to_bitplanes every unit of every
// input row, the memset the all-zero rows of the padded channels).  In host code the NAME below is only a handle:
// the device address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char dd_static_work[DD_STATIC_WORKSPACE_BYTES];

namespace dd {
namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
uint8_t *g_static_addr[kStaticMaxDevices] = {};   // device address of dd_static_work on device i, once looked up

// the geometry prepare_bp computes, without its allocation
template <int NBITS>
size_t static_need(const dd_plan_s *plan, const KernelParams &kp)
{
    using C = Bp<NBITS>;
    const int64_t TB = plan->var.TB;
    const int64_t spg = (16 / (C::NB * 4)) * 32;
    const int64_t units = (static_cast<int64_t>(kp.ntiles - 1) * TB + plan->max_span_end + spg - 1) / spg;
    const int64_t rows = static_cast<int64_t>(kp.nrows) + kp.row_mul;
    return static_cast<size_t>(kp.nbeams) * static_cast<size_t>(rows * C::NSUB * units * 16);
}

}  // namespace

size_t static_work_need(const dd_plan_s *plan, const KernelParams &kp)
{
    switch (plan->nbits) {
    case 2:
        return static_need<2>(plan, kp);
    case 4:
        return static_need<4>(plan, kp);
    case 8:
        return static_need<8>(plan, kp);
    }
    return ~static_cast<size_t>(0);
}

cudaError_t launch_variant3_static(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    if (plan->var.id != 3 || !plan->var.bitplane)
        return cudaErrorInvalidValue;
    if (static_work_need(plan, kp) > static_cast<size_t>(DD_STATIC_WORKSPACE_BYTES))
        return cudaErrorInvalidValue;   // (dd_execute_static has reported DD_ERR_TOO_LARGE before it gets here)
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return e;
    if (dev < 0 || dev >= kStaticMaxDevices)
        return cudaErrorInvalidDevice;
    uint8_t *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_addr[dev]) {
            void *q = nullptr;
            if ((e = cudaGetSymbolAddress(&q, dd_static_work)) != cudaSuccess)
                return e;
            g_static_addr[dev] = static_cast<uint8_t *>(q);
        }
        scratch = g_static_addr[dev];
    }
    // The launcher of variant 3 as it stands, with the plan's work buffer swapped for the array for the length of the
    // call: the buffer is large enough, so prepare_bp neither frees nor allocates, and a cleared layout record makes
    // it rewrite the all-zero rows (another plan's call may have left its data there).
    void *const own_work = plan->d_work;
    const size_t own_bytes = plan->work_bytes;
    int64_t own_layout[4];
    for (int i = 0; i < 4; ++i)
        own_layout[i] = plan->work_layout[i];
    plan->d_work = scratch;
    plan->work_bytes = static_cast<size_t>(DD_STATIC_WORKSPACE_BYTES);
    plan->work_layout[0] = 0;
    e = launch_variant3(plan, kp, stream, false);
    plan->d_work = own_work;
    plan->work_bytes = own_bytes;
    for (int i = 0; i < 4; ++i)
        plan->work_layout[i] = own_layout[i];
    return e;
}

}  // namespace dd
