// dd_kernel_gr.cu -- variant 6: GROUP ROWS in device memory.
//
//     D[d][t] = sum_c A[c][t + delay[d][c]]                       (eq. 3)
//
// Variant 4 (pair rows, dd_kernel_bp.cu) shares the sum of two adjacent channels between trials.  Here the channels
// are taken in groups of G = 4 (or 2) adjacent live channels c_0 .. c_3: the tuple of delay differences
// (delay[d][c_i] - delay[d][c_0], i = 1..3) takes a limited number of values over the whole DM list (35 k tuples for the
// 256 groups of the survey band, 1200 trials), so a pre-pass makes, once per tuple, the row
//
//     R[t] = sum_i x[c_i][t + delta_i]                            (n + 2 bit planes for n-bit input)
//
// and every trial adds the row of its own tuple at the delay of c_0: n + 2 plane words per FOUR channels instead of
// 4 n (variant 3) or 2 (n + 1) (variant 4).  Exact: the delay table is used as it stands (the sub-band idea of
// PAPER.md:311-321 without its approximation; PAPER.md:119's bit-level parallelism for the additions themselves).
//
// Rows are stored UNIT-INTERLEAVED: unit u (32 samples) of a row is UW consecutive words {plane 0 .. plane PIN-1, pad},
// so that the span of a row a CTA needs is ONE bulk copy, and UW is chosen so that the lanes of a warp (W units apart)
// read conflict-free: 2-bit groups of four 4 words (LDS.128, W = 5), 4-bit 6 words (3 x LDS.64, W = 3), 8-bit 10 words
// (5 x LDS.64, W = 3).
//
// Kernels: dd_make_group_rows_staged<nbits, G> (pre-pass, one block per group and 256 units) and dd_direct_gr<nbits, G> (16 trials
// x 1024 W samples per CTA, 16 warps, warp = trial; ring of stages with full/empty mbarriers, each holding the rows of as
// many consecutive groups as fit its byte budget; lanes 0-2 of every warp issue the copies of the warp's share of a
// stage's rows).
#include <utility>

#include "dd_bp_core.cuh"

namespace dd {
namespace {

constexpr int GR_DB = 16, GR_NWARPS = 16;

template <int NBITS, int G>
struct Gr {
    static_assert(NBITS == 2 || NBITS == 4 || NBITS == 8, "input width");
    static_assert(G == 2 || G == 4, "channels per group");
    static constexpr int NBR = NBITS == 2 ? 2 : 4;      // input bit planes: planes per unit of a sub-row,
    static constexpr int NSUBR = NBITS / NBR;           // sub-rows per channel (dd_to_bitplanes)
    static constexpr int PIN = NBITS + (G == 2 ? 1 : 2);   // planes of a row
    static constexpr int UW = gr_unit_words(NBITS, G);  // words per unit of a row (dd_plan.h)
    static constexpr int UB = UW * 4;
    static constexpr int W = NBITS == 2 ? kGrW2 : 3;    // units per lane
    static constexpr int NP = NBITS == 2 ? 12 : (NBITS == 4 ? 16 : 20);   // sum planes (8-bit: 18 when the sums fit)
    static constexpr int NF = gr_flush_groups(NBITS, G);              // groups between flushes of the pending words
    static constexpr int GMAX = gr_max_groups_per_stage(NBITS, G);    // most groups a stage holds
    static constexpr int GQ = gr_group_quantum(NBITS, G);             // stages begin on multiples of GQ groups
    static_assert(NF % GQ == 0 && GMAX % GQ == 0, "group quantum");
    static_assert(UW >= PIN && (UW == 4 || UW % 2 == 0), "row unit");
};

// the PIN plane words of one unit of a row in shared memory
template <int UW, int PIN>
__device__ __forceinline__ void gr_load_unit(const uint8_t *q, uint32_t (&w)[PIN])
{
    if constexpr (UW == 4) {
        const uint4 v = *reinterpret_cast<const uint4 *>(q);
        const uint32_t t[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < PIN; ++k)
            w[k] = t[k];
    } else {
#pragma unroll
        for (int h = 0; h < (PIN + 1) / 2; ++h) {
            const uint2 v = *reinterpret_cast<const uint2 *>(q + 8 * h);
            w[2 * h] = v.x;
            if (2 * h + 1 < PIN)
                w[2 * h + 1] = v.y;
        }
    }
}

// ------------------------------------------------------------------------------------------ pre-pass
// in: bit planes of the input [c][sub-row][unit][NBR planes] (dd_to_bitplanes), in_units units per row, zero beyond the
// input.  grow: per row {c_0 .. c_3 (or -1), delta_0 = 0 .. delta_3}.  out holds the units unit0 .. unit0 + out_units - 1 of
// every row (a group of time tiles), out_pitch_words words per row.
// One thread block per (group, block of GR_UBLK units): the spans of the group's G channels are staged in shared memory
// ONCE and every row (tuple) of the group is made from them -- the group's ~140 rows differ only in their bit offsets
// into the same data, which a first kernel with one thread per (row, unit) fetched again per row through L1/L2 (measured
// on cfg5: 5.96 ms per beam for 12.5 GB of rows; L2-bound).  Rows leave through a per-warp shared-memory patch as whole
// 16-byte vectors of consecutive addresses.
//   gbase  [ngroups + 1] first row of every group;  span_units: units staged per channel (GR_UBLK + the largest
//   difference of the plan in units + 2)
constexpr int GR_UBLK = 256;
template <int NBITS, int G>
__global__ void __launch_bounds__(GR_UBLK) dd_make_group_rows_staged(const uint32_t *__restrict__ in, int64_t in_row_words, int64_t in_units,
                                                                     const int4 *__restrict__ grow, const int32_t *__restrict__ gbase,
                                                                     uint32_t *__restrict__ out, int64_t out_pitch_words, int64_t out_units,
                                                                     int64_t ublocks, int64_t unit0, int32_t span_units)
{
    using C = Gr<NBITS, G>;
    extern __shared__ __align__(16) uint32_t gsm[];
    const int64_t blk = blockIdx.x;
    const int64_t q = blk / ublocks, ul0 = (blk - q * ublocks) * GR_UBLK;   // group; first unit (inside the buffer) of this block
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r0 = __ldg(&gbase[q]), r1 = __ldg(&gbase[q + 1]);
    if (r0 >= r1)
        return;
    const int4 gc = __ldg(&grow[2 * r0]);
    const int ch[4] = {gc.x, gc.y, gc.z, gc.w};
    const int64_t in_sub_words = in_row_words / C::NSUBR;
    const int64_t ug0 = unit0 + ul0;   // first unit of the rows this block makes
    // stage: channel i, sub-row s, units ug0 .. ug0 + span_units - 1 -> st[(i * NSUBR + s) * span_units + k] (NBR words each)
    uint32_t *st = gsm;
    uint32_t *patch = gsm + static_cast<size_t>(G) * C::NSUBR * span_units * C::NBR + warp * (32 * C::UW);
    for (int i = 0; i < G; ++i) {
        for (int sub = 0; sub < C::NSUBR; ++sub) {
            uint32_t *dstp = st + static_cast<size_t>(i * C::NSUBR + sub) * span_units * C::NBR;
            const uint32_t *src = ch[i] >= 0 ? in + static_cast<int64_t>(ch[i]) * in_row_words + sub * in_sub_words : nullptr;
            for (int k = tid; k < span_units; k += GR_UBLK) {
                const int64_t ug = ug0 + k;
                if constexpr (C::NBR == 4) {
                    const uint4 v = (src && ug < in_units) ? __ldg(reinterpret_cast<const uint4 *>(src + ug * 4)) : make_uint4(0, 0, 0, 0);
                    *reinterpret_cast<uint4 *>(dstp + k * 4) = v;
                } else {
                    const uint2 v = (src && ug < in_units) ? __ldg(reinterpret_cast<const uint2 *>(src + ug * 2)) : make_uint2(0, 0);
                    *reinterpret_cast<uint2 *>(dstp + k * 2) = v;
                }
            }
        }
    }
    __syncthreads();
    const int64_t ul = ul0 + tid;
    const bool live = ul < out_units;
    // the shifted words of channel i for this thread's unit
    auto shifted = [&](int i, int delta, uint32_t (&x)[NBITS]) {
        const uint32_t sh = static_cast<uint32_t>(delta) & 31u;
#pragma unroll
        for (int sub = 0; sub < C::NSUBR; ++sub) {
            const uint32_t *qp = st + (static_cast<size_t>(i * C::NSUBR + sub) * span_units + tid + (delta >> 5)) * C::NBR;
            if constexpr (C::NBR == 4) {
                const uint4 a = *reinterpret_cast<const uint4 *>(qp), b = *reinterpret_cast<const uint4 *>(qp + 4);
                x[4 * sub] = __funnelshift_r(a.x, b.x, sh), x[4 * sub + 1] = __funnelshift_r(a.y, b.y, sh);
                x[4 * sub + 2] = __funnelshift_r(a.z, b.z, sh), x[4 * sub + 3] = __funnelshift_r(a.w, b.w, sh);
            } else {
                const uint2 a = *reinterpret_cast<const uint2 *>(qp), b = *reinterpret_cast<const uint2 *>(qp + 2);
                x[2 * sub] = __funnelshift_r(a.x, b.x, sh), x[2 * sub + 1] = __funnelshift_r(a.y, b.y, sh);
            }
        }
    };
    // The rows of a group are sorted by (delta_1, delta_2, delta_3): consecutive rows mostly share delta_1 and often
    // delta_2, so x0 is read once, x0 + x1 is kept while delta_1 stays, the shifted x2 while delta_2 stays, and only x3
    // is shifted for every row -- a third of the shared-memory loads and half the ripple adders of making every row anew
    // (cfg5: 3.88 -> 2.31 ms per beam; the builder was bound by the shared-memory pipe and now writes at the HBM rate).
    uint32_t x0[NBITS];
#pragma unroll
    for (int sub = 0; sub < C::NSUBR; ++sub) {   // channel 0 has no shift
        const uint32_t *qp = st + (static_cast<size_t>(sub) * span_units + tid) * C::NBR;
#pragma unroll
        for (int kk = 0; kk < C::NBR; ++kk)
            x0[sub * C::NBR + kk] = qp[kk];
    }
    uint32_t s01[NBITS + 1], x2[NBITS];
    int d1_held = -1, d2_held = -1;
    for (int r = r0; r < r1; ++r) {
        const int4 gd = __ldg(&grow[2 * r + 1]);
        uint32_t o[C::UW];
#pragma unroll
        for (int k = 0; k < C::UW; ++k)
            o[k] = 0u;
        if (gd.y != d1_held) {   // x0 + x1: NBITS + 1 planes
            uint32_t x1[NBITS], cy = 0u;
            shifted(1, gd.y, x1);
#pragma unroll
            for (int k = 0; k < NBITS; ++k) {
                s01[k] = x0[k] ^ x1[k] ^ cy;
                cy = (x0[k] & x1[k]) | (cy & (x0[k] ^ x1[k]));
            }
            s01[NBITS] = cy;
            d1_held = gd.y;
        }
        if constexpr (G == 2) {
#pragma unroll
            for (int k = 0; k <= NBITS; ++k)
                o[k] = s01[k];
        } else {
            if (gd.z != d2_held) {
                shifted(2, gd.z, x2);
                d2_held = gd.z;
            }
            uint32_t x3[NBITS], c23 = 0u, cs = 0u;
            shifted(3, gd.w, x3);
#pragma unroll
            for (int k = 0; k < NBITS; ++k) {   // x2 + x3 ripples beside the sum with x0 + x1
                const uint32_t s23 = x2[k] ^ x3[k] ^ c23;
                c23 = (x2[k] & x3[k]) | (c23 & (x2[k] ^ x3[k]));
                o[k] = s01[k] ^ s23 ^ cs;
                cs = (s01[k] & s23) | (cs & (s01[k] ^ s23));
            }
            o[NBITS] = s01[NBITS] ^ c23 ^ cs;
            o[NBITS + 1] = (s01[NBITS] & c23) | (cs & (s01[NBITS] ^ c23));
        }
        // the warp's 32 units are 32 * UW consecutive words of the row: through the patch, then 16-byte stores in order
        uint32_t *dst = out + static_cast<int64_t>(r) * out_pitch_words + (ul0 + warp * 32) * C::UW;
        if constexpr (C::UW == 4) {
            if (live)
                *reinterpret_cast<uint4 *>(dst + lane * 4) = make_uint4(o[0], o[1], o[2], o[3]);
        } else {
#pragma unroll
            for (int h = 0; h < C::UW / 2; ++h)
                *reinterpret_cast<uint2 *>(patch + lane * C::UW + 2 * h) = make_uint2(o[2 * h], o[2 * h + 1]);
            __syncwarp();
            const int64_t left = out_units - (ul0 + warp * 32);                      // units of this warp inside the buffer
            const int nvec = static_cast<int>((left >= 32 ? 32 : (left > 0 ? left : 0)) * C::UW / 4);   // (rows hold whole 16 bytes)
#pragma unroll
            for (int v = lane; v < 32 * C::UW / 4; v += 32)
                if (v < nvec)
                    *reinterpret_cast<uint4 *>(dst + v * 4) = *reinterpret_cast<const uint4 *>(patch + v * 4);
            __syncwarp();
        }
    }
}

// ------------------------------------------------------------------------------------------ the transform
// one group of the stage for this warp's trial: e = {byte offset, inside the stage, of the unit of the trial's row that
// holds its first sample; bit shift}; W + 1 units loaded for W units, per unit and plane a funnel shift + carry-save adds
// the planes K .. PIN - 1 of one unit: x0 / x1 hold the unit's words and those of the unit after it
template <int NBITS, int G, int CLS, int K, int NP, int NT>
__device__ __forceinline__ void gr_add_planes(const uint32_t (&x0)[Gr<NBITS, G>::PIN], const uint32_t (&x1)[Gr<NBITS, G>::PIN], uint32_t shift,
                                              uint32_t (&P)[NP], uint32_t (&T)[NT])
{
    using C = Gr<NBITS, G>;
    if constexpr (K < C::PIN) {
        // weight the counter has taken since the last flush: CLS whole rows and the planes below this one
        constexpr uint32_t S = ((1u << C::PIN) - 1u) * CLS + ((1u << K) - 1u);
        csa_add<S, K>(P, T, __funnelshift_r(x0[K], x1[K], shift));
        gr_add_planes<NBITS, G, CLS, K + 1>(x0, x1, shift, P, T);
    }
}

// plane K of the units [J0, J1) of the lane (their counters advance side by side: instruction-level parallelism)
template <int NBITS, int G, int CLS, int K, int J0, int J1, int NP, int NT>
__device__ __forceinline__ void gr_add_planes_some(const uint32_t (&x)[Gr<NBITS, G>::W + 1][Gr<NBITS, G>::PIN], uint32_t shift,
                                                   uint32_t (&P)[Gr<NBITS, G>::W][NP], uint32_t (&T)[Gr<NBITS, G>::W][NT])
{
    using C = Gr<NBITS, G>;
    if constexpr (K < C::PIN) {
        constexpr uint32_t S = ((1u << C::PIN) - 1u) * CLS + ((1u << K) - 1u);
#pragma unroll
        for (int j = J0; j < J1; ++j)
            csa_add<S, K>(P[j], T[j], __funnelshift_r(x[j][K], x[j + 1][K], shift));
        gr_add_planes_some<NBITS, G, CLS, K + 1, J0, J1>(x, shift, P, T);
    }
}

// The counters of the W units are independent, so the order of the units is free.  Plane by plane over all units gives
// the most parallelism (measured best for 4-bit input and 8-bit groups of four); unit by unit keeps only two units'
// words live, which the 9-plane rows of 8-bit pairs need to stay clear of spills (cfg3: 196 -> 185 ms).  (The five units
// of 2-bit input in two runs of three and two: 7.91 ms against 7.66 ms on cfg2, no fewer spills.)
template <int NBITS, int G, int CLS, int NP, int NT>
__device__ __forceinline__ void gr_add_group(const uint8_t *lane_base, const uint2 e, uint32_t (&P)[Gr<NBITS, G>::W][NP],
                                             uint32_t (&T)[Gr<NBITS, G>::W][NT])
{
    using C = Gr<NBITS, G>;
    uint32_t x[C::W + 1][C::PIN];
    if constexpr (NBITS == 8 && G == 2) {
        gr_load_unit<C::UW, C::PIN>(lane_base + e.x, x[0]);
#pragma unroll
        for (int j = 0; j < C::W; ++j) {
            gr_load_unit<C::UW, C::PIN>(lane_base + e.x + (j + 1) * C::UB, x[j + 1]);
            gr_add_planes<NBITS, G, CLS, 0>(x[j], x[j + 1], e.y, P[j], T[j]);
        }
    } else {
#pragma unroll
        for (int j = 0; j <= C::W; ++j)
            gr_load_unit<C::UW, C::PIN>(lane_base + e.x + j * C::UB, x[j]);
        gr_add_planes_some<NBITS, G, CLS, 0, 0, C::W>(x, e.y, P, T);
    }
}

template <class F, int... Is>
__device__ __forceinline__ void gr_for_each(F &&f, std::integer_sequence<int, Is...>)
{
    (f(std::integral_constant<int, Is>{}), ...);
}

// Stages hold a VARIABLE number of groups: the planner packs consecutive groups into a stage until the stage's byte
// budget (or 48 rows, or GMAX groups) is reached -- the rows a DM block needs per group vary (1 .. 7 on the survey band,
// 4.1 on average), so stages sized for the worst case of a fixed group count ran at 60 % of their capacity, and the fixed
// cost of a stage (producer chain, barrier round trips: ~650-1200 clocks per SM sub-partition) weighed on too little work.
// The pending words are flushed every NF groups, whatever the stage boundaries are.
// PATCH: the epilogue passes through per-warp shared-memory patches (whole 128-byte lines per store instruction)
// NP: sum planes (sums < 2^NP; 8-bit plans of up to 1028 channels run with 18 instead of 20: six registers fewer, cfg5
// 144.2 -> 141.5 ms)
template <int NBITS, int G, bool PATCH, int NP = Gr<NBITS, G>::NP>
__global__ void __launch_bounds__(GR_NWARPS * 32, 1) dd_direct_gr(const KernelParams p)
{
    using C = Gr<NBITS, G>;
    constexpr int DB = GR_DB, W = C::W, TB = 32 * 32 * W, PIN = C::PIN, UB = C::UB;
    constexpr int NF = C::NF, GMAX = C::GMAX;
    constexpr uint32_t FLUSH_SUM = ((1u << PIN) - 1u) * NF;   // weight the counters take between flushes
    constexpr int NT = bit_length(FLUSH_SUM);                 // pending slots
    constexpr uint32_t REL_BYTES = (GMAX * DB + DB) * 8;      // offset entries of up to GMAX groups + a trailer: groups of the NEXT stage
    constexpr int RPW = 3;                                    // rows a warp stages per stage (the plan keeps rows_per_chunk <= 48)

    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // tile decode: DM block fastest so that CTAs resident together share the same row spans (L2)
    const int64_t cta = blockIdx.x;
    const int blk = static_cast<int>(cta % p.nblk);
    const int tile = static_cast<int>(cta / p.nblk) + p.tile0;   // this launch covers the tiles tile0 .. tile0 + ntiles - 1
    const int64_t t0 = static_cast<int64_t>(tile) * TB;
    const int NS = p.nstages;

    // shared memory carve-up (must match dd::gr_smem_bytes)
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);   // [8]
    uint64_t *empty = full + 8;                              // [8]
    constexpr int rel_slot = static_cast<int>((REL_BYTES + 127) / 128 * 128);
    const int row_slot = p.raw_slot;                         // bytes of a stage's rows (a multiple of 128)
    uint8_t *rel_base = smem + 128 + (PATCH ? GR_NWARPS * kBpPatchBytes : 0);
    uint8_t *row_base = rel_base + NS * rel_slot;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&full[s], GR_NWARPS);
            mbar_init(&empty[s], GR_NWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    // rows of this launch: p.in holds, per row, the units in_unit0 .. of the time axis, rows in_stride bytes apart.
    // Tables per DM block: p.nchunks stage slots (the largest stage count of any block)
    const uint8_t *in_tile = p.in + ((t0 >> 5) - p.in_unit0) * UB;
    const int64_t stage0 = static_cast<int64_t>(blk) * p.nchunks;
    const int4 *span_blk = p.span + (stage0 * p.rows_per_chunk + blk) + 1;   // one header entry ahead of every block's list
    const uint8_t *rel_blk = static_cast<const uint8_t *>(p.rel) + stage0 * REL_BYTES;
    const int4 hdr = __ldg(span_blk - 1);   // {stages of this block, groups of its first stage, -, -}
    const int nstg = hdr.x;

    // producers: lanes 0 .. RPW - 1 of every warp issue the copies of the warp's rows of a stage (lane k: slot warp +
    // 16 k; one span entry per lane, so that the entries cost 8 registers instead of 24); warp 0 also brings the trials'
    // offset entries.  The span entry of the next stage to issue is fetched one step early.
    auto load_meta = [&](int stg) -> int4 {
        const int slot = warp + GR_NWARPS * lane;
        return (lane < RPW && stg < nstg && slot < p.rows_per_chunk)
                   ? __ldg(&span_blk[static_cast<int64_t>(stg) * p.rows_per_chunk + slot])
                   : make_int4(0, 0, 0, 0);
    };
    int prod_s = 0, prod_round = 0;
    // blocking: wait for the slot to be released; otherwise give up (return false) if it has not been yet
    auto produce = [&](int stg, const int4 m, auto blocking_) -> bool {
        constexpr bool BLOCKING = decltype(blocking_)::value;
        const int s = prod_s;
        if constexpr (!BLOCKING) {
            uint32_t ready = 1u;
            if (lane == 0 && prod_round > 0)   // every warp has added stage stg - NS?
                ready = mbar_test(&empty[s], (prod_round - 1) & 1) ? 1u : 0u;
            if (!__shfl_sync(0xFFFFFFFFu, ready, 0))
                return false;
        }
        // span entry: {byte offset inside the row for tile 0, bytes, row, byte offset inside the stage}
        uint32_t tx = static_cast<uint32_t>(m.y);
        tx += __shfl_down_sync(0xFFFFFFFFu, tx, 2);
        tx += __shfl_down_sync(0xFFFFFFFFu, tx, 1);   // lane 0: bytes of lanes 0 .. 2 (RPW == 3; the other lanes hold 0)
        if (lane == 0) {
            if constexpr (BLOCKING) {
                if (prod_round > 0)
                    mbar_wait(&empty[s], (prod_round - 1) & 1);   // every warp has added stage stg - NS
            }
            mbar_arrive_expect_tx(&full[s], tx + (warp == 0 ? REL_BYTES : 0u));
            if (warp == 0)
                tma_bulk_g2s(rel_base + s * rel_slot, rel_blk + static_cast<int64_t>(stg) * REL_BYTES, REL_BYTES, &full[s]);
        }
        __syncwarp();
        if (m.y > 0)
            tma_bulk_g2s(row_base + s * row_slot + m.w, in_tile + static_cast<int64_t>(m.z) * p.in_stride + m.x,
                         static_cast<uint32_t>(m.y), &full[s]);
        __syncwarp();
        if (++prod_s == NS) {
            prod_s = 0;
            ++prod_round;
        }
        return true;
    };
    using Blocking = std::true_type;
    using NonBlocking = std::false_type;
    static_assert(RPW == 3, "the byte count of a warp's copies is summed over lanes 0 .. 2");
    const int dist = NS > 2 ? NS - 2 : 1;   // prefetch distance in stages
    int4 meta = load_meta(0);
    for (int k = 0; k < dist && k < nstg; ++k) {
        const int4 nxt = load_meta(k + 1);
        produce(k, meta, Blocking{});
        meta = nxt;
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
    int s = -1, stg = -1, g_in = 0, n_in = 0, n_next = hdr.y;
    uint32_t full_parity = 1u;
    // the next stage: release the one just finished, keep the ring fed, wait for the rows
    // The copies of stage stg + dist are issued as soon as the slot is free, but a warp does not WAIT for that: it tries at
    // every group quantum and goes on adding meanwhile (the slot is free when the slowest warp has left the stage before;
    // waiting there made every warp as slow as the slowest plus the wait -- a fifth of the warp instructions were spins).
    // (Not for 8-bit input: there the warps -- and with them the CTAs of adjacent DM blocks -- drifting apart cost L2 hits:
    // cfg3 read 250 GB instead of 169 GB from DRAM and took 178 ms instead of 168 ms, cfg5 124 ms instead of 122 ms; cfg4 gained
    // 6.5 %, cfg2 1 %.)
    constexpr bool DEFER = NBITS < 8;
    int pend_stg = -1;   // stage whose copies are still to be issued (its span entry is in `meta`), or -1
    auto try_produce = [&](auto blocking) {
        if (produce(pend_stg, meta, blocking)) {
            meta = load_meta(pend_stg + 1);
            pend_stg = -1;
        }
    };
    auto next_stage = [&]() {
        if (stg >= 0) {
            __syncwarp();
            if (lane == 0)
                mbar_arrive(&empty[s]);
        }
        ++stg;
        if (++s == NS || stg == 0) {
            s = 0;
            full_parity ^= 1u;
        }
        if constexpr (DEFER) {
            if (pend_stg >= 0)   // still not issued, and it is the stage needed next: wait for the slot now
                try_produce(Blocking{});
            if (stg + dist < nstg)
                pend_stg = stg + dist;
        } else if (stg + dist < nstg) {
            const int4 nxt = load_meta(stg + dist + 1);
            produce(stg + dist, meta, Blocking{});
            meta = nxt;
        }
        mbar_wait(&full[s], full_parity);
        n_in = n_next;
        g_in = 0;
        n_next = static_cast<int>(reinterpret_cast<const uint2 *>(rel_base + s * rel_slot)[GMAX * DB].x);   // the trailer
    };
    // one group: CLS = groups added since the last flush
    auto group = [&](auto cls) {
        constexpr int CLS = decltype(cls)::value;
        if constexpr (CLS % C::GQ == 0) {
            if (g_in == n_in)
                next_stage();
            if constexpr (DEFER) {
                if (pend_stg >= 0)
                    try_produce(NonBlocking{});
            }
        }
        gr_add_group<NBITS, G, CLS>(row_base + s * row_slot + lane * (W * UB),
                                    reinterpret_cast<const uint2 *>(rel_base + s * rel_slot)[g_in * DB + warp], P, T);
        ++g_in;
    };
    for (int g = 0; g < p.nchans_pad; g += NF) {   // the group count is a multiple of NF by plan construction
        gr_for_each(group, std::make_integer_sequence<int, NF>{});
#pragma unroll
        for (int j = 0; j < W; ++j)
            csa_flush<FLUSH_SUM, 0, false>(P[j], T[j], 0u);
    }
    __syncwarp();
    if (lane == 0 && stg >= 0)
        mbar_arrive(&empty[s]);

    // ---- epilogue: thread owns samples t0 + 32*(W*lane + j) + [0, 32) of DM slot `warp` (as in dd_kernel_bp.cu)
    const int d = blk * DB + warp;
    if (d >= p.ndm)
        return;
    const int esize = (p.out_code == DD_OUT_U16) ? 2 : 4;
    uint8_t *orow = p.out + static_cast<int64_t>(d) * p.out_dm_stride;
    const bool interior = PATCH && p.vec16_ok && (t0 + TB <= p.nsamps);   // 16-byte stores: rows must be 16-byte aligned
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
            uint8_t *gunit = orow + (t0 + 32 * j) * esize;   // unit j of lane 0; lane s is W * 32 samples further
            if (p.out_code == DD_OUT_F32)
                store_unit_coalesced<4, true>(q, patch, lane, gunit, W * 32 * 4);
            else if (p.out_code == DD_OUT_U32)
                store_unit_coalesced<4, false>(q, patch, lane, gunit, W * 32 * 4);
            else
                store_unit_coalesced<2, false>(q, patch, lane, gunit, W * 32 * 2);
        } else {
            const int64_t tunit = t0 + 32 * (W * lane + j);
#pragma unroll
            for (int h = 0; h < 8; ++h) {   // samples 4h .. 4h+3 of the unit
                const uint32_t q4[4] = {q[4 * h], q[4 * h + 1], q[4 * h + 2], q[4 * h + 3]};
                store4(p, orow, tunit + 4 * h, q4);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ launcher
// As for the pair rows of variant 4 (dd_kernel_bp.cu::launch_pairs): the rows are made per beam and per GROUP of time
// tiles into one of two buffers, on two internal streams that alternate between groups (fork / join by events on the
// caller's stream), so that the rows of one group are built while the other is transformed and the device memory taken
// is two groups' worth whatever the number of beams.  A group is the whole time axis unless its rows exceed the
// workspace limit; the split is worked out once per launch geometry.
template <int NBITS, int G>
cudaError_t launch_group_rows(dd_plan_s *plan, const KernelParams &kp_in, cudaStream_t stream)
{
    using C = Gr<NBITS, G>;
    constexpr int TB = 32 * 32 * C::W, NBI = C::NBR, NSUBI = C::NSUBR;
    if (!plan->gr || plan->gs_G != G || plan->var.TB != TB || kp_in.ngroups != 1 || !plan->d_prow ||
        kp_in.out_code == kOutPlanes || kp_in.out_code == kOutU8 || kp_in.nchans_pad % C::NF != 0 ||
        plan->rows_per_chunk > 48)
        return cudaErrorInvalidValue;
    cudaError_t e;
    int32_t max_delta = 0;
    for (int64_t r = 0; r < plan->n_prows; ++r)
        for (int i = 4; i < 8; ++i)
            max_delta = std::max(max_delta, plan->prow[8 * r + i]);
    const int64_t tile_units = TB / 32;
    const int64_t extra_units = ((plan->max_span_end + 31) / 32 - tile_units + 3) / 4 * 4;   // span beyond a tile's own units
    const int64_t rows_o = plan->n_prows + 1;                                                  // + the all-zero row of padded groups
    auto pitch_of = [&](int64_t units) { return units * C::UB; };
    int64_t GT;   // time tiles per group
    if (plan->pair_tiles > 0) {
        GT = plan->pair_tiles;
    } else if (plan->pair_geom[0] == kp_in.ntiles && plan->pair_geom[1] == kp_in.nbeams && plan->pair_geom[2] > 0) {
        GT = plan->pair_geom[2];
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
        GT = (budget - rows_o * pitch_of(extra_units)) / (rows_o * pitch_of(tile_units));
        if (GT < 1)
            return cudaErrorMemoryAllocation;   // not even one tile's rows fit the limit
        plan->pair_geom[0] = kp_in.ntiles;
        plan->pair_geom[1] = kp_in.nbeams;
        plan->pair_geom[2] = GT > kp_in.ntiles ? kp_in.ntiles : GT;
    }
    GT = GT < 1 ? 1 : (GT > kp_in.ntiles ? kp_in.ntiles : GT);
    const int64_t units_g = GT * tile_units + extra_units, pitch_g = pitch_of(units_g);
    const int64_t buf_bytes = rows_o * pitch_g;
    // input bit planes of the whole call (one transpose), long enough for the last group's rows plus the largest difference
    const int64_t all_units = static_cast<int64_t>(kp_in.ntiles) * tile_units + extra_units;
    const int64_t spg = (16 / (NBI * 4)) * 32;                               // input samples per 16-byte group of a sub-row
    const int64_t groups_i = (all_units * 32 + max_delta + 64 + spg - 1) / spg;
    const int64_t conv_i = groups_i * 16, in_units = conv_i / (NBI * 4);     // bytes per sub-row, units per row
    const int64_t beam_i = static_cast<int64_t>(kp_in.nrows) * NSUBI * conv_i;
    const int64_t ngroups_all = static_cast<int64_t>(kp_in.nbeams) * ((kp_in.ntiles + GT - 1) / GT);
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

    // the transpose of the packed input: d_work rows are conv_i bytes per sub-row here (not the layout of variant 3)
    {
        BpWork w;
        w.units = groups_i;
        w.conv = conv_i;
        w.rows = kp_in.nrows;
        w.w_beam = beam_i;
        if ((e = launch_to_bitplanes(plan, kp_in, w, stream)) != cudaSuccess)
            return e;
    }
    if (plan->prof_mid)
        cudaEventRecord(static_cast<cudaEvent_t>(plan->prof_mid), stream);
    auto kernel = plan->patch ? dd_direct_gr<NBITS, G, true> : dd_direct_gr<NBITS, G, false>;
    if constexpr (NBITS == 8) {
        if (static_cast<int64_t>(plan->nlive) * 255 < (int64_t(1) << 18))
            kernel = dd_direct_gr<8, G, false, 18>;   // (8-bit plans never use the output patches)
    }
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes))) != cudaSuccess)
        return e;
    const int64_t ublocks = (units_g + GR_UBLK - 1) / GR_UBLK;
    const int64_t ngr = static_cast<int64_t>(plan->prow.size()) - 8 * plan->n_prows - 1;   // groups: prow ends with their first rows
    const int32_t span_units = GR_UBLK + (max_delta >> 5) + 2;
    const size_t bsmem = (static_cast<size_t>(G) * NSUBI * span_units * NBI + (GR_UBLK / 32) * 32 * C::UW) * 4;
    if (ngr < 1 || ngr * ublocks > 0x7FFFFFFFLL || static_cast<int64_t>(kp_in.nblk) * GT > 0x7FFFFFFFLL || bsmem > 200 * 1024)
        return cudaErrorInvalidConfiguration;
    if ((e = cudaFuncSetAttribute(dd_make_group_rows_staged<NBITS, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(bsmem))) !=
        cudaSuccess)
        return e;
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
        for (int64_t c0 = 0; c0 < kp_in.ntiles && e == cudaSuccess; c0 += GT, ++it) {
            const int sl = nbuf == 2 ? (it & 1) : 0;
            const int64_t gc = (c0 + GT <= kp_in.ntiles) ? GT : kp_in.ntiles - c0;
            const int64_t unit0 = c0 * tile_units;
            dd_make_group_rows_staged<NBITS, G><<<dim3(static_cast<unsigned>(ngr * ublocks)), GR_UBLK, bsmem, ws[sl]>>>(
                reinterpret_cast<const uint32_t *>(static_cast<const uint8_t *>(plan->d_work) + b * beam_i), NSUBI * conv_i / 4, in_units,
                static_cast<const int4 *>(plan->d_prow), reinterpret_cast<const int32_t *>(plan->d_prow) + 8 * plan->n_prows,
                reinterpret_cast<uint32_t *>(buf[sl]), pitch_g / 4, units_g, ublocks, unit0, span_units);
            if ((e = cudaGetLastError()) != cudaSuccess)
                break;
            KernelParams kp = kp_in;
            kp.in = buf[sl];
            kp.in_stride = pitch_g;
            kp.out = kp_in.out + static_cast<int64_t>(b) * kp_in.out_beam_stride;
            kp.nbeams = 1;
            kp.rows_per_chunk = plan->rows_per_chunk;
            kp.nchunks = plan->gr_stage_slots;
            kp.tile0 = static_cast<int32_t>(c0);
            kp.ntiles = static_cast<int32_t>(gc);
            kp.in_unit0 = unit0;
            kernel<<<dim3(static_cast<unsigned>(static_cast<int64_t>(kp.nblk) * gc)), dim3(GR_NWARPS * 32), plan->smem_bytes, ws[sl]>>>(kp);
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

cudaError_t launch_variant6(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    const int G = plan->gs_G;
    switch (plan->nbits) {
    case 2:
        return G == 4 ? launch_group_rows<2, 4>(plan, kp, stream) : cudaErrorInvalidValue;
    case 4:
        return G == 4 ? launch_group_rows<4, 4>(plan, kp, stream) : launch_group_rows<4, 2>(plan, kp, stream);
    case 8:
        return G == 4 ? launch_group_rows<8, 4>(plan, kp, stream) : launch_group_rows<8, 2>(plan, kp, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace dd
