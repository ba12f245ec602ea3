// dd_kernel_gs.cu -- variant 5: GROUP SUMS made inside the CTA.
//
//     D[d][t] = sum_c A[c][t + delay[d][c]]                       (eq. 3)
//
// The bit-plane kernel (dd_kernel_bp.cu) adds, per trial and channel, n plane words per 32 samples.  Here the
// channels are taken in groups of G adjacent live channels c_0 .. c_{G-1}.  Inside a block of 16 consecutive trials
// the delay differences delta_i = delay[d][c_i] - delay[d][c_0] take only a few distinct patterns (two roundings
// make each difference jitter by one: 1.9 patterns per pair, 4.1 per group of four on the survey band), so the CTA
// builds, once per pattern, the row
//
//     R[t] = sum_i x[c_i][t + delta_i]                            (n + log2 G bit planes)
//
// in shared memory from the staged bit planes of the G channels, and every trial adds the row of its own pattern at
// the delay of c_0: n + log2 G plane words per group instead of G n.  Exact -- the delay table is used as it stands --
// and the rows never leave the SM (this is the sub-band idea of PAPER.md:311-321 without its approximation, and the
// paper's "temporal caching" of PAPER.md:115 applied to partial sums).
//
// One CTA = 16 trials x 1024 W samples; 16 adder warps (warp = trial) and 4 builder warps.  Two rings in shared memory:
//   raw ring  : per stage the bit-plane spans of its G * CC channels (TMA bulk copies) and the build table;
//   row ring  : per stage the rows built from them and the offset entries of the trials,
// with full/empty mbarriers per ring slot (no CTA-wide barrier in the loop).  The builder warps copy and build, the
// adder warps only add (measured with every warp doing all three jobs: per stage and warp ~1000 clocks issuing
// copies, ~2400 building, ~2600 adding -- the latency chains of the first two stalled the adds).
#include <utility>

#include "dd_bp_core.cuh"

namespace dd {
namespace {

constexpr int GS_DB = 16, GS_NWARPS = 16;
#ifndef GS_ILP
#define GS_ILP 2         // items a builder warp takes at a time (their dependency chains interleave)
#endif
constexpr int GS_FL = kGsFlushStages;   // stages between flushes of the pending words

template <int NBITS, int G>
struct Gs {
    static_assert(NBITS == 2 || NBITS == 4 || NBITS == 8, "input width");
    static_assert(G == 2 || G == 4, "channels per group");
    static constexpr int NBR = NBITS == 2 ? 2 : 4;      // planes per unit of a raw sub-row
    static constexpr int NSUBR = NBITS / NBR;           // raw sub-rows per channel
    static constexpr int UBR = NBR * 4;                 // bytes per raw unit
    static constexpr int PIN = NBITS + (G == 2 ? 1 : 2);   // planes of a row
    static constexpr int WF = PIN < 4 ? 2 : 4;          // planes per unit of the full sub-rows of a row
    static constexpr int NF = PIN / WF;                 // full sub-rows
    static constexpr int RW = PIN - NF * WF;            // planes of the last, narrower sub-row (0: none)
    static constexpr int W = NBITS == 2 ? kGsW2 : kGsW48;   // units per lane (16 adder + 4 builder warps: 96 registers per thread)
    static constexpr int NP = NBITS == 2 ? 12 : (NBITS == 4 ? 16 : 20);   // sum planes
    // Row layout in shared memory.  With W odd the lanes of a warp (W units apart) fall into distinct banks when the units
    // of a sub-row lie one after the other.  With W = 2 they would collide two by two, so the units of a sub-row are
    // DE-INTERLEAVED: even units in one array, odd units in a second array row_units / 2 units further -- a lane's units
    // base + 2 l + {0, 1, 2} are then {A_p[h + l], A_(1-p)[h + p + l], A_p[h + l + 1]} (p = base & 1, h = base >> 1) and
    // consecutive lanes read consecutive units of one array: no conflicts (measured without: the adds ran at the speed
    // of the shared-memory pipe, every LDS.128 taking two passes).
    static constexpr int DI = (W % 2 == 0) ? 2 : 1;
    static_assert(W % 2 == 1 || W == 2, "even W: only the two-array layout is written out");
};
// position (in units) of unit u inside a sub-row of row_units units
template <int DI>
__device__ __forceinline__ int gs_unit_pos(int u, int row_units)
{
    if constexpr (DI == 2)
        return (u & 1) * (row_units >> 1) + (u >> 1);
    else
        return u;
}

// ------------------------------------------------------------------------------------------ builder
// One unit (32 samples) of one row: sum over the group's channels of the staged planes, channel i read at the bit
// offset the build entry gives, written as PIN planes in the row layout.  Plane by plane: x0 + x1 and x2 + x3 ripple
// side by side and feed a third ripple adder (G = 4), so that few words are live at a time.
template <int NBITS, int G>
__device__ __forceinline__ void gs_build_unit(const uint8_t *raw, uint8_t *row, const int4 e0, const int4 e1, const int4 e2,
                                              int u, int raw_sub, int row_units)
{
    using C = Gs<NBITS, G>;
    const int src[4] = {e0.z, e0.w, e1.x, e1.y};
    const uint32_t sh[4] = {0u, static_cast<uint32_t>(e1.w), static_cast<uint32_t>(e2.x), static_cast<uint32_t>(e2.y)};
    uint32_t o[C::PIN];
    uint32_t c01 = 0u, c23 = 0u, cs = 0u;
#pragma unroll
    for (int sub = 0; sub < C::NSUBR; ++sub) {
        PlaneVec<C::NBR> a0, lo[G], hi[G];
        a0.load(raw + src[0] + sub * raw_sub + u * C::UBR);
#pragma unroll
        for (int i = 1; i < G; ++i) {
            const uint8_t *q = raw + src[i] + sub * raw_sub + u * C::UBR;
            lo[i].load(q);
            hi[i].load(q + C::UBR);
        }
#pragma unroll
        for (int kk = 0; kk < C::NBR; ++kk) {
            const int k = sub * C::NBR + kk;
            const uint32_t x0 = a0.w[kk];
            const uint32_t x1 = __funnelshift_r(lo[1].w[kk], hi[1].w[kk], sh[1]);
            const uint32_t s01 = x0 ^ x1 ^ c01;
            c01 = (x0 & x1) | (c01 & (x0 ^ x1));
            if constexpr (G == 2) {
                o[k] = s01;
            } else {
                const uint32_t x2 = __funnelshift_r(lo[2].w[kk], hi[2].w[kk], sh[2]);
                const uint32_t x3 = __funnelshift_r(lo[3].w[kk], hi[3].w[kk], sh[3]);
                const uint32_t s23 = x2 ^ x3 ^ c23;
                c23 = (x2 & x3) | (c23 & (x2 ^ x3));
                o[k] = s01 ^ s23 ^ cs;
                cs = (s01 & s23) | (cs & (s01 ^ s23));
            }
        }
    }
    if constexpr (G == 2) {
        o[NBITS] = c01;
    } else {
        o[NBITS] = c01 ^ c23 ^ cs;
        o[NBITS + 1] = (c01 & c23) | (cs & (c01 ^ c23));
    }
    // row layout: NF sub-rows of WF planes per unit, then one sub-row of RW planes per unit
    const int up = gs_unit_pos<C::DI>(u, row_units);
#pragma unroll
    for (int s = 0; s < C::NF; ++s) {
        uint8_t *q = row + e0.x + row_units * (4 * C::WF) * s + up * (4 * C::WF);
        if constexpr (C::WF == 4)
            *reinterpret_cast<uint4 *>(q) = make_uint4(o[4 * s], o[4 * s + 1], o[4 * s + 2], o[4 * s + 3]);
        else
            *reinterpret_cast<uint2 *>(q) = make_uint2(o[2 * s], o[2 * s + 1]);
    }
    if constexpr (C::RW > 0) {
        uint8_t *q = row + e0.x + row_units * (4 * C::WF) * C::NF + up * (4 * C::RW);
        if constexpr (C::RW == 1)
            *reinterpret_cast<uint32_t *>(q) = o[C::NF * C::WF];
        else
            *reinterpret_cast<uint2 *>(q) = make_uint2(o[C::NF * C::WF], o[C::NF * C::WF + 1]);
    }
}

// ------------------------------------------------------------------------------------------ consumer
// plane K of a sub-row holding the planes [L0, L0 + NW) of the row; CLS = groups added since the last flush
template <int NBITS, int G, int CLS, int L0, int NW, int K, int NP, int NT>
__device__ __forceinline__ void gs_add_planes(const PlaneVec<NW> (&x)[Gs<NBITS, G>::W + 1], uint32_t shift,
                                              uint32_t (&P)[Gs<NBITS, G>::W][NP], uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    if constexpr (K < NW) {
        // weight the counter has taken since the last flush: CLS whole rows and the planes below this one
        constexpr uint32_t S = ((1u << C::PIN) - 1u) * CLS + ((1u << (L0 + K)) - 1u);
#pragma unroll
        for (int j = 0; j < C::W; ++j)
            csa_add<S, L0 + K>(P[j], T[j], __funnelshift_r(x[j].w[K], x[j + 1].w[K], shift));
        gs_add_planes<NBITS, G, CLS, L0, NW, K + 1>(x, shift, P, T);
    }
}

// W + 1 units loaded for W units, per unit and plane one funnel shift + carry-save adds.  sub: the sub-row of this row;
// v0, v1: positions (in units) of the lane's first and second unit inside it (DI == 1: v1 unused, units are consecutive)
template <int NBITS, int G, int CLS, int L0, int NW, int NP, int NT>
__device__ __forceinline__ void gs_add_subrow(const uint8_t *sub, int v0, int v1, uint32_t shift,
                                              uint32_t (&P)[Gs<NBITS, G>::W][NP], uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    PlaneVec<NW> x[C::W + 1];
    if constexpr (C::DI == 2) {
        x[0].load(sub + v0 * (4 * NW));
        x[1].load(sub + v1 * (4 * NW));
        x[2].load(sub + v0 * (4 * NW) + 4 * NW);
    } else {
#pragma unroll
        for (int j = 0; j <= C::W; ++j)
            x[j].load(sub + v0 * (4 * NW) + j * (4 * NW));
    }
    gs_add_planes<NBITS, G, CLS, L0, NW, 0>(x, shift, P, T);
}

template <int NBITS, int G, int CLS, int S_, int NP, int NT>
__device__ __forceinline__ void gs_add_full(const uint8_t *rowq, int v0, int v1, int row_units, uint32_t shift,
                                            uint32_t (&P)[Gs<NBITS, G>::W][NP], uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    if constexpr (S_ < C::NF) {
        gs_add_subrow<NBITS, G, CLS, S_ * C::WF, C::WF>(rowq + row_units * (4 * C::WF) * S_, v0, v1, shift, P, T);
        gs_add_full<NBITS, G, CLS, S_ + 1>(rowq, v0, v1, row_units, shift, P, T);
    }
}

// one group of the stage for this warp's trial: e = {byte offset of the row slot, bit shift | v0 << 8 | v1 << 20} with
// v0, v1 the positions of the trial's first and second unit in a sub-row (DI == 1: v0 = the unit offset, v1 = 0)
template <int NBITS, int G, int CLS, int NP, int NT>
__device__ __forceinline__ void gs_add_group(const uint8_t *row_stage, const uint2 e, int lane, int row_units,
                                             uint32_t (&P)[Gs<NBITS, G>::W][NP], uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    const uint8_t *rowq = row_stage + e.x;
    // lane l owns the units base + W l + j: with two arrays that is l positions further in both
    const int v0 = static_cast<int>((e.y >> 8) & 0xFFFu) + (C::DI == 2 ? lane : C::W * lane);
    const int v1 = static_cast<int>(e.y >> 20) + lane;
    gs_add_full<NBITS, G, CLS, 0>(rowq, v0, v1, row_units, e.y, P, T);
    if constexpr (C::RW > 0)
        gs_add_subrow<NBITS, G, CLS, C::NF * C::WF, C::RW>(rowq + row_units * (4 * C::WF) * C::NF, v0, v1, e.y, P, T);
}

template <int NBITS, int G, int CC, int PHASE, int NP, int NT, int... GIs>
__device__ __forceinline__ void gs_add_stage(std::integer_sequence<int, GIs...>, const uint8_t *row_stage, const uint2 *rel,
                                             int lane, int row_units, uint32_t (&P)[Gs<NBITS, G>::W][NP],
                                             uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    (gs_add_group<NBITS, G, PHASE * CC + GIs>(row_stage, rel[GIs * GS_DB], lane, row_units, P, T), ...);
}

// ------------------------------------------------------------------------------------------ the kernel
// Warps 0 .. 15 ADD: warp w owns trial w of the DM block, lane l the units W l .. W l + W - 1; per stage they wait for
// the rows, add them, and release the slot -- nothing else.  Warps 16 .. 16 + NBW - 1 BUILD: they issue the bulk
// copies of the spans (and of the build table and the trials' offset entries) DT stages ahead, and build the rows of
// a stage as soon as its spans have landed and a row slot is free.  The latency chains of copying and building
// (mbarrier round trips, dependent shared-memory loads, ripple carries) thus run beside the adders instead of in them.
// PATCH: the epilogue passes through per-warp shared-memory patches (whole 128-byte lines per store instruction).
template <int NBITS, int G, int CC, int NBW, bool PATCH>
__global__ void __launch_bounds__((GS_NWARPS + NBW) * 32, 1) dd_direct_gs(const KernelParams p)
{
    using C = Gs<NBITS, G>;
    constexpr int DB = GS_DB, W = C::W, TB = 32 * 32 * W, NP = C::NP, PIN = C::PIN;
    constexpr int CHS = G * CC;                                     // channels per stage
    constexpr int NCOPY = CHS * C::NSUBR;                           // bulk copies of spans per stage
    constexpr uint32_t STAGE_SUM = ((1u << PIN) - 1u) * CC;         // weight one stage adds to a counter
    constexpr int NT = bit_length(GS_FL * STAGE_SUM);               // pending slots
    constexpr uint32_t REL_BYTES = CC * DB * 8;
    static_assert(NCOPY + 2 <= 32 * NBW, "one lane per bulk copy");

    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // tile decode: DM block fastest so that CTAs resident together share the same input window (L2)
    const int64_t cta = blockIdx.x;
    const int blk = static_cast<int>(cta % p.nblk);
    const int64_t rest = cta / p.nblk;
    const int tile = static_cast<int>(rest % p.ntiles);
    const int beam = static_cast<int>(rest / p.ntiles);
    const int64_t t0 = static_cast<int64_t>(tile) * TB;
    const int nchunks = p.nchunks;

    // shared memory carve-up (must match dd::gs_smem_bytes)
    const int NSR = p.gs_nsr, NSP = p.gs_nsp;
    uint64_t *raw_full = reinterpret_cast<uint64_t *>(smem);   // [4] each
    uint64_t *raw_empty = raw_full + 4;
    uint64_t *row_full = raw_full + 8;
    uint64_t *row_empty = raw_full + 12;
    const int rel_slot = static_cast<int>(align128(REL_BYTES));
    const int tab_slot = static_cast<int>(align128(static_cast<int64_t>(p.gs_rows) * 64));
    const int raw_slot = static_cast<int>(align128(static_cast<int64_t>(NCOPY) * p.gs_raw_sub));
    const int row_bytes = p.gs_row_units * (4 * PIN);
    const int row_slot = static_cast<int>(align128(static_cast<int64_t>(p.gs_rows) * row_bytes));
    uint8_t *rel_base = smem + 128 + (PATCH ? GS_NWARPS * kBpPatchBytes : 0);
    uint8_t *tab_base = rel_base + NSP * rel_slot;
    uint8_t *raw_base = tab_base + NSR * tab_slot;
    uint8_t *row_base = raw_base + NSR * raw_slot;

    if (tid == 0) {
        for (int s = 0; s < 4; ++s) {
            mbar_init(&raw_full[s], NBW);
            mbar_init(&raw_empty[s], NBW);
            mbar_init(&row_full[s], NBW);
            mbar_init(&row_empty[s], GS_NWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();   // the only CTA-wide barrier: builders and adders part ways below

    if (warp >= GS_NWARPS) {
        // ================================================================== builders
        const int bw = warp - GS_NWARPS;
        const uint8_t *in_beam = p.in + static_cast<int64_t>(beam) * p.in_beam_stride;
        const uint8_t *in_tile = in_beam + (t0 >> 5) * C::UBR;   // this tile's first unit in every sub-row
        const int64_t stage0 = static_cast<int64_t>(blk) * nchunks;
        const int4 *span_blk = p.span + stage0 * CHS;
        const int4 *tab_blk = p.gs_tab + stage0 * p.gs_rows * 4;
        const uint8_t *rel_blk = static_cast<const uint8_t *>(p.rel) + stage0 * REL_BYTES;
        // Copies: lane i of builder warp bw issues copy bw + NBW i -- the spans 0 .. NCOPY - 1 (channel slot / NSUBR, sub-row
        // % NSUBR), then the build table.  Bulk copies take uniform operands, so the lanes of a warp issue theirs one
        // after the other (measured: ~300 clocks per copy; one warp issuing all 17 copies of a stage in turn with the
        // others was slower still -- ~7000 clocks per turn), hence the copies of a stage are spread over all builder warps.
        const int ci = bw + NBW * lane;
        auto load_meta = [&](int chunk) -> int4 {
            return (ci < NCOPY && chunk < nchunks) ? __ldg(&span_blk[static_cast<int64_t>(chunk) * CHS + ci / C::NSUBR])
                                                   : make_int4(0, 0, 0, 0);
        };
        int is = 0, iround = 0;   // ring position of the next chunk to copy
        int4 meta = load_meta(0);
        auto issue = [&](int chunk) {
            if (iround > 0)
                mbar_wait(&raw_empty[is], (iround - 1) & 1);   // the builders are done with chunk - NSR
            const uint32_t bytes = ci < NCOPY ? static_cast<uint32_t>(meta.y) : (ci == NCOPY ? static_cast<uint32_t>(p.gs_rows) * 64u : 0u);
            const uint32_t tx = __reduce_add_sync(0xFFFFFFFFu, bytes);
            if (lane == 0)
                mbar_arrive_expect_tx(&raw_full[is], tx);
            __syncwarp();
            if (ci < NCOPY) {
                // span entry: {byte offset inside a sub-row for tile 0, bytes, input row, -}; the work rows are long enough
                // for every copy, and padded channels point at the all-zero row
                if (meta.y > 0)
                    tma_bulk_g2s(raw_base + is * raw_slot + ci * p.gs_raw_sub,
                                 in_tile + static_cast<int64_t>(meta.z) * p.in_stride + (ci % C::NSUBR) * p.in_row_bytes + meta.x,
                                 static_cast<uint32_t>(meta.y), &raw_full[is]);
            } else if (ci == NCOPY) {
                tma_bulk_g2s(tab_base + is * tab_slot, tab_blk + static_cast<int64_t>(chunk) * p.gs_rows * 4, bytes, &raw_full[is]);
            }
            meta = load_meta(chunk + 1);
            if (++is == NSR) {
                is = 0;
                ++iround;
            }
        };
        const int DT = NSR - 1;   // copies run DT stages ahead of the build
        for (int k = 0; k < DT && k < nchunks; ++k)
            issue(k);
        int bs = 0, bs_round = 0, bp = 0, bp_round = 0;
        for (int chunk = 0; chunk < nchunks; ++chunk) {
            if (chunk + DT < nchunks)
                issue(chunk + DT);
            mbar_wait(&raw_full[bs], bs_round & 1);
            if (bp_round > 0)
                mbar_wait(&row_empty[bp], (bp_round - 1) & 1);   // every adder is done with chunk - NSP
            if (bw == 0 && lane == 0) {   // the trials' offset entries travel with the row slot
                mbar_expect_tx(&row_full[bp], REL_BYTES);
                tma_bulk_g2s(rel_base + bp * rel_slot, rel_blk + static_cast<int64_t>(chunk) * REL_BYTES, REL_BYTES, &row_full[bp]);
            }
            const uint8_t *raw = raw_base + bs * raw_slot;
            uint8_t *row = row_base + bp * row_slot;
            const int4 *tab = reinterpret_cast<const int4 *>(tab_base + bs * tab_slot);
            // items (row, block of 32 units) of the rows in use, dealt round-robin to the builder warps and taken GS_ILP at a
            // time without branches (a lane past the end of a row redoes the row's last unit, a missing item redoes the
            // first), so that their dependency chains interleave
            const int nitems = tab[3].w * p.gs_nblk32;   // GsEntry::pad[5] of entry 0: rows in use in this stage
            for (int it0 = bw; it0 < nitems; it0 += GS_ILP * NBW) {
                int4 e0[GS_ILP], e1[GS_ILP], e2[GS_ILP];
                int u[GS_ILP];
#pragma unroll
                for (int q = 0; q < GS_ILP; ++q) {
                    const int it = it0 + q * NBW < nitems ? it0 + q * NBW : it0;
                    const int r = (it * p.gs_magic) >> 16;
                    e0[q] = tab[4 * r];
                    e1[q] = tab[4 * r + 1];
                    e2[q] = G == 4 ? tab[4 * r + 2] : make_int4(0, 0, 0, 0);
                    u[q] = min((it - r * p.gs_nblk32) * 32 + lane, e0[q].y - 1);
                }
#pragma unroll
                for (int q = 0; q < GS_ILP; ++q)
                    gs_build_unit<NBITS, G>(raw, row, e0[q], e1[q], e2[q], u[q], p.gs_raw_sub, p.gs_row_units);
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&row_full[bp]);
                mbar_arrive(&raw_empty[bs]);
            }
            if (++bs == NSR) {
                bs = 0;
                ++bs_round;
            }
            if (++bp == NSP) {
                bp = 0;
                ++bp_round;
            }
        }
        return;
    }

    // ====================================================================== adders
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
    int cs = 0;
    uint32_t cs_parity = 0;
    auto stage = [&](auto phase, auto flush) {
        constexpr int PHASE = decltype(phase)::value;
        constexpr uint32_t FLUSH = decltype(flush)::value;
        mbar_wait(&row_full[cs], cs_parity);
        gs_add_stage<NBITS, G, CC, PHASE>(std::make_integer_sequence<int, CC>{}, row_base + cs * row_slot,
                                          reinterpret_cast<const uint2 *>(rel_base + cs * rel_slot) + warp, lane, p.gs_row_units,
                                          P, T);
        if constexpr (FLUSH != 0u) {
#pragma unroll
            for (int j = 0; j < W; ++j)
                csa_flush<FLUSH, 0, false>(P[j], T[j], 0u);
        }
        __syncwarp();
        if (lane == 0)
            mbar_arrive(&row_empty[cs]);
        if (++cs == NSP) {
            cs = 0;
            cs_parity ^= 1u;
        }
    };
    using NoFlush = std::integral_constant<uint32_t, 0u>;
    using FlushAll = std::integral_constant<uint32_t, GS_FL * STAGE_SUM>;
    static_assert(GS_FL == 4, "unroll the phases here");
    for (int chunk = 0; chunk < nchunks; chunk += GS_FL) {   // nchunks is a multiple of GS_FL by plan construction
        stage(std::integral_constant<int, 0>{}, NoFlush{});
        stage(std::integral_constant<int, 1>{}, NoFlush{});
        stage(std::integral_constant<int, 2>{}, NoFlush{});
        stage(std::integral_constant<int, 3>{}, FlushAll{});
    }

    // ---- epilogue: thread owns samples t0 + 32*(W*lane + j) + [0, 32) of DM slot `warp` (as in dd_kernel_bp.cu)
    const int d = blk * DB + warp;
    if (d >= p.ndm)
        return;
    const int esize = (p.out_code == DD_OUT_U16) ? 2 : 4;
    uint8_t *orow = p.out + static_cast<int64_t>(beam) * p.out_beam_stride + static_cast<int64_t>(d) * p.out_dm_stride;
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

#ifndef GS_NBW_
#define GS_NBW_ 4
#endif
constexpr int GS_NBW = GS_NBW_;   // builder warps

template <int NBITS, int G, int CC, bool PATCH>
cudaError_t launch_gs_inst(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, int64_t ctas)
{
    auto kernel = dd_direct_gs<NBITS, G, CC, GS_NBW, PATCH>;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes));
    if (e != cudaSuccess)
        return e;
    kernel<<<dim3(static_cast<unsigned>(ctas)), dim3((GS_NWARPS + GS_NBW) * 32), plan->smem_bytes, stream>>>(kp);
    return cudaGetLastError();
}

}  // namespace

// The instantiations compiled in: {nbits, G, groups per stage}; dd_plan.cpp::build_tiles_gs picks among them.
#define DD_GS_INSTANCES(X) \
    X(8, 2, 4) X(8, 2, 2) X(8, 4, 2) X(8, 4, 1) \
    X(4, 2, 8) X(4, 4, 4) \
    X(2, 2, 16) X(2, 4, 4)

bool gs_instance_exists(int nbits, int G, int cc)
{
#define X(NB, GG, C_) \
    if (nbits == NB && G == GG && cc == C_) \
        return true;
    DD_GS_INSTANCES(X)
#undef X
    return false;
}

// Two launches: the bit-plane transpose of the rows the tiles will read, then the transform.
cudaError_t launch_variant5(dd_plan_s *plan, const KernelParams &kp_in, cudaStream_t stream)
{
    if (!plan->gs || !plan->var.bitplane || !plan->d_gs_tab || kp_in.ngroups != 1 || kp_in.out_code == kOutPlanes ||
        kp_in.out_code == kOutU8 || kp_in.nchunks % GS_FL != 0)
        return cudaErrorInvalidValue;
    KernelParams kp = kp_in;
    BpWork w;
    cudaError_t e = bp_prepare_work(plan, kp, stream, false, &w);
    if (e != cudaSuccess)
        return e;
    if ((e = launch_to_bitplanes(plan, kp, w, stream)) != cudaSuccess)
        return e;
    if (plan->prof_mid)
        cudaEventRecord(static_cast<cudaEvent_t>(plan->prof_mid), stream);
    const int nsub = plan->nbits == 8 ? 2 : 1;
    kp.in = static_cast<const uint8_t *>(plan->d_work);
    kp.in_stride = nsub * w.conv;   // between channel rows; sub-rows are in_row_bytes apart
    kp.in_row_bytes = w.conv;
    kp.in_beam_stride = w.w_beam;
    kp.gs_tab = static_cast<const int4 *>(plan->d_gs_tab);
    kp.gs_rows = plan->gs_rows;
    kp.gs_row_units = plan->gs_row_units;
    kp.gs_raw_sub = plan->gs_raw_sub;
    kp.gs_nsr = plan->gs_nsr;
    kp.gs_nsp = plan->gs_nsp;
    kp.gs_nblk32 = (plan->gs_row_units + 31) / 32;
    kp.gs_magic = (65536 + kp.gs_nblk32 - 1) / kp.gs_nblk32;
    const int64_t ctas = static_cast<int64_t>(kp.nblk) * kp.ntiles * kp.nbeams;
    if (ctas <= 0 || ctas > 0x7FFFFFFFLL || kp.gs_rows * kp.gs_nblk32 >= 4096)
        return cudaErrorInvalidConfiguration;
#define X(NB, GG, C_) \
    if (plan->nbits == NB && plan->gs_G == GG && plan->cc == C_) \
        return plan->gs_patch ? launch_gs_inst<NB, GG, C_, true>(plan, kp, stream, ctas) \
                              : launch_gs_inst<NB, GG, C_, false>(plan, kp, stream, ctas);
    DD_GS_INSTANCES(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace dd
