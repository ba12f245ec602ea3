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
// One CTA = 16 trials x 1024 W samples, 16 warps, as in dd_kernel_bp.cu.  Two rings in shared memory:
//   raw ring  : per stage the bit-plane spans of its G * CC channels (TMA bulk copies) and the build table;
//   row ring  : per stage the rows built from them and the offset entries of the trials.
// Every warp takes its share of both jobs, in this order per iteration k:
//   issue the copies of stage k + 1 + DT  |  build its share of the rows of stage k + 1  |  add stage k
// with full/empty mbarriers per ring slot (no CTA-wide barrier in the loop).
#include <cstdio>
#include <utility>

#include "dd_bp_core.cuh"

namespace dd {
namespace {

constexpr int GS_DB = 16, GS_NWARPS = 16;
#ifndef GS_X_SWAP
#define GS_X_SWAP 1      // the two halves of the CTA build at different points of an iteration
#endif
#ifndef GS_X_ILP2
#define GS_X_ILP2 1      // build items two at a time
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
    static constexpr int W = NBITS == 2 ? 5 : 3;        // units per lane
    static constexpr int NP = NBITS == 2 ? 12 : (NBITS == 4 ? 16 : 20);   // sum planes
};

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
#pragma unroll
    for (int s = 0; s < C::NF; ++s) {
        uint8_t *q = row + e0.x + row_units * (4 * C::WF) * s + u * (4 * C::WF);
        if constexpr (C::WF == 4)
            *reinterpret_cast<uint4 *>(q) = make_uint4(o[4 * s], o[4 * s + 1], o[4 * s + 2], o[4 * s + 3]);
        else
            *reinterpret_cast<uint2 *>(q) = make_uint2(o[2 * s], o[2 * s + 1]);
    }
    if constexpr (C::RW > 0) {
        uint8_t *q = row + e0.x + row_units * (4 * C::WF) * C::NF + u * (4 * C::RW);
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

// W + 1 units loaded for W units, per unit and plane one funnel shift + carry-save adds
template <int NBITS, int G, int CLS, int L0, int NW, int NP, int NT>
__device__ __forceinline__ void gs_add_subrow(const uint8_t *q, uint32_t shift, uint32_t (&P)[Gs<NBITS, G>::W][NP],
                                              uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    PlaneVec<NW> x[C::W + 1];
#pragma unroll
    for (int j = 0; j <= C::W; ++j)
        x[j].load(q + j * (4 * NW));
    gs_add_planes<NBITS, G, CLS, L0, NW, 0>(x, shift, P, T);
}

template <int NBITS, int G, int CLS, int S_, int NP, int NT>
__device__ __forceinline__ void gs_add_full(const uint8_t *rowq, int ui, int row_units, uint32_t shift,
                                            uint32_t (&P)[Gs<NBITS, G>::W][NP], uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    if constexpr (S_ < C::NF) {
        gs_add_subrow<NBITS, G, CLS, S_ * C::WF, C::WF>(rowq + row_units * (4 * C::WF) * S_ + ui * (4 * C::WF), shift, P, T);
        gs_add_full<NBITS, G, CLS, S_ + 1>(rowq, ui, row_units, shift, P, T);
    }
}

// one group of the stage for this warp's trial: e = {byte offset of the row slot, (unit offset << 8) | bit shift}
template <int NBITS, int G, int CLS, int NP, int NT>
__device__ __forceinline__ void gs_add_group(const uint8_t *row_stage, const uint2 e, int lane, int row_units,
                                             uint32_t (&P)[Gs<NBITS, G>::W][NP], uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    using C = Gs<NBITS, G>;
    const uint8_t *rowq = row_stage + e.x;
    const int ui = static_cast<int>(e.y >> 8) + C::W * lane;
    gs_add_full<NBITS, G, CLS, 0>(rowq, ui, row_units, e.y, P, T);
    if constexpr (C::RW > 0)
        gs_add_subrow<NBITS, G, CLS, C::NF * C::WF, C::RW>(rowq + row_units * (4 * C::WF) * C::NF + ui * (4 * C::RW), e.y, P, T);
}

template <int NBITS, int G, int CC, int PHASE, int NP, int NT, int... GIs>
__device__ __forceinline__ void gs_add_stage(std::integer_sequence<int, GIs...>, const uint8_t *row_stage, const uint2 *rel,
                                             int lane, int row_units, uint32_t (&P)[Gs<NBITS, G>::W][NP],
                                             uint32_t (&T)[Gs<NBITS, G>::W][NT])
{
    (gs_add_group<NBITS, G, PHASE * CC + GIs>(row_stage, rel[GIs * GS_DB], lane, row_units, P, T), ...);
}

// ------------------------------------------------------------------------------------------ the kernel
// PATCH: the epilogue passes through per-warp shared-memory patches (whole 128-byte lines per store instruction)
template <int NBITS, int G, int CC, bool PATCH>
__global__ void __launch_bounds__(GS_NWARPS * 32, 1) dd_direct_gs(const KernelParams p)
{
    using C = Gs<NBITS, G>;
    constexpr int DB = GS_DB, W = C::W, TB = 32 * 32 * W, NP = C::NP, PIN = C::PIN;
    constexpr int CHS = G * CC;                                     // channels per stage
    constexpr int NCOPY = CHS * C::NSUBR;                           // bulk copies of spans per stage
    constexpr int CPW = (NCOPY + GS_NWARPS - 1) / GS_NWARPS;        // ... per warp
    constexpr uint32_t STAGE_SUM = ((1u << PIN) - 1u) * CC;         // weight one stage adds to a counter
    constexpr int NT = bit_length(GS_FL * STAGE_SUM);               // pending slots
    constexpr uint32_t REL_BYTES = CC * DB * 8;

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

    constexpr int NBUILD = GS_NWARPS;   // every warp builds its share of the rows of a stage
    if (tid == 0) {
        for (int s = 0; s < 4; ++s) {
            mbar_init(&raw_full[s], GS_NWARPS);
            mbar_init(&raw_empty[s], NBUILD);
            mbar_init(&row_full[s], NBUILD);
            mbar_init(&row_empty[s], GS_NWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const uint8_t *in_beam = p.in + static_cast<int64_t>(beam) * p.in_beam_stride;
    const uint8_t *in_tile = in_beam + (t0 >> 5) * C::UBR;   // this tile's first unit in every sub-row
    const int64_t stage0 = static_cast<int64_t>(blk) * nchunks;
    const int4 *span_blk = p.span + stage0 * CHS;
    const int4 *tab_blk = p.gs_tab + stage0 * p.gs_rows * 4;
    const uint8_t *rel_blk = static_cast<const uint8_t *>(p.rel) + stage0 * REL_BYTES;

#ifdef GS_X_TIMING
    uint32_t tm_issue = 0, tm_bwait = 0, tm_build = 0, tm_cwait = 0, tm_add = 0;
#define GS_TICK(acc, t_) { const uint32_t now_ = clock(); acc += now_ - t_; t_ = now_; }
#else
#define GS_TICK(acc, t_)
#endif
    // ring position of a chunk: slot = chunk % depth, round = chunk / depth, by multiplication (depth is 2, 3 or 4 at
    // run time; chunk < 8192 by plan construction), so that no counters are carried through the loop
    const int magic_r = (65536 + NSR - 1) / NSR, magic_p = (65536 + NSP - 1) / NSP;
    auto raw_pos = [&](int chunk, int &slot, int &round) {
        round = (chunk * magic_r) >> 16;
        slot = chunk - round * NSR;
    };
    auto row_pos = [&](int chunk, int &slot, int &round) {
        round = (chunk * magic_p) >> 16;
        slot = chunk - round * NSP;
    };

    // ---- copies: every warp's lane 0 issues its share of the spans of a stage (a bulk copy takes uniform operands,
    // so one warp issuing them all would fall behind); warp 0 also brings the build table.  The span entries of the
    // next stage to issue are fetched one call early.
    int4 meta[CPW];
    auto load_meta = [&](int chunk) {
#pragma unroll
        for (int k = 0; k < CPW; ++k) {
            const int i = warp + GS_NWARPS * k;   // copy index: channel slot i / NSUBR, sub-row i % NSUBR
            meta[k] = (lane == 0 && i < NCOPY && chunk < nchunks) ? __ldg(&span_blk[static_cast<int64_t>(chunk) * CHS + i / C::NSUBR])
                                                                  : make_int4(0, 0, 0, 0);
        }
    };
    auto issue = [&](int chunk) {
        int s, round;
        raw_pos(chunk, s, round);
        if (lane == 0) {
            if (round > 0)
                mbar_wait(&raw_empty[s], (round - 1) & 1);   // the builders of chunk - NSR are done with the slot
            uint32_t tx = (warp == 0) ? static_cast<uint32_t>(p.gs_rows) * 64u : 0u;
#pragma unroll
            for (int k = 0; k < CPW; ++k)
                tx += static_cast<uint32_t>(meta[k].y);
            mbar_arrive_expect_tx(&raw_full[s], tx);
#pragma unroll
            for (int k = 0; k < CPW; ++k) {
                const int i = warp + GS_NWARPS * k;
                if (i < NCOPY && meta[k].y > 0) {
                    const int sub = i % C::NSUBR;
                    // span entry: {byte offset inside a sub-row for tile 0, bytes, input row, -}; the work rows are long
                    // enough for every copy, and padded channels point at the all-zero row
                    tma_bulk_g2s(raw_base + s * raw_slot + i * p.gs_raw_sub,
                                 in_tile + static_cast<int64_t>(meta[k].z) * p.in_stride + sub * p.in_row_bytes + meta[k].x,
                                 static_cast<uint32_t>(meta[k].y), &raw_full[s]);
                }
            }
            if (warp == 0)
                tma_bulk_g2s(tab_base + s * tab_slot, tab_blk + static_cast<int64_t>(chunk) * p.gs_rows * 4,
                             static_cast<uint32_t>(p.gs_rows) * 64u, &raw_full[s]);
        }
        load_meta(chunk + 1);
        __syncwarp();
    };

    // ---- build: this warp's share of the rows of a chunk; items (row, block of 32 units) are dealt round-robin to the
    // warps, two at a time for overlap.  The build is a chain of shared-memory round trips with little arithmetic, so
    // the two halves of the CTA do it at different points of an iteration (see `stage` below): while one half builds,
    // the other adds.
    const int nitems = p.gs_rows * p.gs_nblk32;
    auto build = [&](int chunk) {
        int bs, bs_round, bp, bp_round;
        raw_pos(chunk, bs, bs_round);
        row_pos(chunk, bp, bp_round);
#ifdef GS_X_TIMING
        uint32_t tb = clock();
#endif
        mbar_wait(&raw_full[bs], bs_round & 1);
        if (bp_round > 0)
            mbar_wait(&row_empty[bp], (bp_round - 1) & 1);   // every warp has added chunk - NSP
#ifdef GS_X_TIMING
        tm_bwait += clock() - tb;
#endif
        if (warp == 0 && lane == 0) {   // the trials' offset entries travel with the row slot
            mbar_expect_tx(&row_full[bp], REL_BYTES);
            tma_bulk_g2s(rel_base + bp * rel_slot, rel_blk + static_cast<int64_t>(chunk) * REL_BYTES, REL_BYTES, &row_full[bp]);
        }
        const uint8_t *raw = raw_base + bs * raw_slot;
        uint8_t *row = row_base + bp * row_slot;
        const int4 *tab = reinterpret_cast<const int4 *>(tab_base + bs * tab_slot);
        for (int it = warp; it < nitems; it += (GS_X_ILP2 ? 2 : 1) * NBUILD) {
            const int it2 = GS_X_ILP2 ? it + NBUILD : nitems;
            const int r = (it * p.gs_magic) >> 16, b32 = it - r * p.gs_nblk32;
            const int r2 = it2 < nitems ? (it2 * p.gs_magic) >> 16 : r, b32b = it2 - r2 * p.gs_nblk32;
            const int4 e0 = tab[4 * r], e1 = tab[4 * r + 1], f0 = tab[4 * r2], f1 = tab[4 * r2 + 1];
            int4 e2 = make_int4(0, 0, 0, 0), f2 = make_int4(0, 0, 0, 0);
            if constexpr (G == 4) {
                e2 = tab[4 * r + 2];
                f2 = tab[4 * r2 + 2];
            }
            const int u = b32 * 32 + lane, u2 = b32b * 32 + lane;
#ifndef GS_X_NOBUILD
            if (u < e0.y)
                gs_build_unit<NBITS, G>(raw, row, e0, e1, e2, u, p.gs_raw_sub, p.gs_row_units);
            if (it2 < nitems && u2 < f0.y)
                gs_build_unit<NBITS, G>(raw, row, f0, f1, f2, u2, p.gs_raw_sub, p.gs_row_units);
#endif
        }
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(&row_full[bp]);
            mbar_arrive(&raw_empty[bs]);
        }
    };

    const int DT = NSR - 1;   // copies run DT stages ahead of the build
    const bool early = !GS_X_SWAP || warp < GS_NWARPS / 2;   // this half builds stage k + 1 before it adds stage k, the other half after
    load_meta(0);
    for (int k = 0; k <= DT && k < nchunks; ++k)
        issue(k);
    build(0);

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

    // one iteration: keep the copies flowing, build this warp's share of the next stage's rows, add this stage's rows
    auto stage = [&](int chunk, auto phase, auto flush) {
        constexpr int PHASE = decltype(phase)::value;   // == chunk % 4 (GS_FL == 4)
        constexpr uint32_t FLUSH = decltype(flush)::value;
#ifdef GS_X_TIMING
        uint32_t tk = clock();
#endif
        if (chunk + 1 + DT < nchunks)
            issue(chunk + 1 + DT);
        GS_TICK(tm_issue, tk)
        if (early && chunk + 1 < nchunks)
            build(chunk + 1);
        GS_TICK(tm_build, tk)
        int cs, cs_round;
        row_pos(chunk, cs, cs_round);
        mbar_wait(&row_full[cs], cs_round & 1);
        GS_TICK(tm_cwait, tk)
#ifndef GS_X_NOADD
        gs_add_stage<NBITS, G, CC, PHASE>(std::make_integer_sequence<int, CC>{}, row_base + cs * row_slot,
                                          reinterpret_cast<const uint2 *>(rel_base + cs * rel_slot) + warp, lane, p.gs_row_units,
                                          P, T);
#endif
        if constexpr (FLUSH != 0u) {
#pragma unroll
            for (int j = 0; j < W; ++j)
                csa_flush<FLUSH, 0, false>(P[j], T[j], 0u);
        }
        __syncwarp();
        if (lane == 0)
            mbar_arrive(&row_empty[cs]);
        GS_TICK(tm_add, tk)
        if (!early && chunk + 1 < nchunks)
            build(chunk + 1);
        GS_TICK(tm_build, tk)
    };
    using NoFlush = std::integral_constant<uint32_t, 0u>;
    using FlushAll = std::integral_constant<uint32_t, GS_FL * STAGE_SUM>;
    static_assert(GS_FL == 4, "unroll the phases here");
    for (int chunk = 0; chunk < nchunks; chunk += GS_FL) {   // nchunks is a multiple of GS_FL by plan construction
        stage(chunk, std::integral_constant<int, 0>{}, NoFlush{});
        stage(chunk + 1, std::integral_constant<int, 1>{}, NoFlush{});
        stage(chunk + 2, std::integral_constant<int, 2>{}, NoFlush{});
        stage(chunk + 3, std::integral_constant<int, 3>{}, FlushAll{});
    }

#ifdef GS_X_TIMING
    if (lane == 0 && (cta == 5 || cta == 3000) && (warp == 0 || warp == 6 || warp == 15))
        printf("cta %d warp %d stages %d: per stage issue %u build(total) %u of which waits %u, wait row_full %u, add %u\n", (int)cta, warp,
               nchunks, tm_issue / nchunks, tm_build / nchunks, tm_bwait / nchunks, tm_cwait / nchunks, tm_add / nchunks);
#endif
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

template <int NBITS, int G, int CC, bool PATCH>
cudaError_t launch_gs_inst(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream, int64_t ctas)
{
    auto kernel = dd_direct_gs<NBITS, G, CC, PATCH>;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes));
    if (e != cudaSuccess)
        return e;
    kernel<<<dim3(static_cast<unsigned>(ctas)), dim3(GS_NWARPS * 32), plan->smem_bytes, stream>>>(kp);
    return cudaGetLastError();
}

}  // namespace

// The instantiations compiled in: {nbits, G, groups per stage}; dd_plan.cpp::build_tiles_gs picks among them.
#ifdef GS_X_ONLY
#define DD_GS_INSTANCES(X) X(8, 2, 4)
#else
#define DD_GS_INSTANCES(X) \
    X(8, 2, 4) X(8, 2, 2) X(8, 4, 2) X(8, 4, 1) \
    X(4, 2, 8) X(4, 2, 4) X(4, 4, 4) X(4, 4, 2) \
    X(2, 2, 16) X(2, 2, 8) X(2, 4, 8) X(2, 4, 4)
#endif

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
