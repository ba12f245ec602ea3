// dd_tree.cu -- the tree dedispersion algorithm (eq. 7-15) and the piecewise linear tree method
// (eq. 16-23), and the frequency-padded tree (eq. 25); include/dd.h "dd_tree_*";
// readings X1-X8 of DESIGN.md section 12.
//
// The recursion of eq. 10-13, with Theta (eq. 14) and the shuffle Phi (eq. 15) written out for one step i (r = 2^i):
// the rows of level i lie in blocks of r rows (the tree of r adjacent channels, row m' = trial d' = m' of that block);
// two neighbouring blocks L, U combine into one block of 2r rows,
//
//     out[2 m' + b][t] = L[m'][t] + U[m'][t + m' + b],      m' < r, b = 0, 1                      (eq. 11-12)
//
// (Phi(r, 2 nu) = L's row m', Phi(r, 2 nu + 1) = U's row m', Theta(i, 2 nu + b) = m' + b for nu = r k + m').  log2 N such
// steps over N rows of T samples are N T log2 N additions -- 5.4e9 for 1024 channels and 2^19 samples, 0.1 ms of the
// integer pipes -- against N T (nbits / 8 + 4) bytes in and out: the tree is bound by memory, not by arithmetic, so the
// steps are FUSED in shared memory.  The outputs {2^Q x + o', o' < 2^Q} of Q consecutive steps i0 .. i0 + Q - 1 depend on
// exactly 2^Q rows of level i0 (row x of each of 2^Q neighbouring blocks): a radix-2^Q butterfly, as in an FFT.  One
// kernel, dd_tree_pass<Q>, runs one such pass: a CTA stages R = 2^Q rows x C columns (8- or 16-bit lanes, 64 KB, two CTAs
// per SM) of one butterfly and one time tile, runs the Q steps in place (every thread keeps the sums of its items in registers
// across the barrier between reading and writing a level), and stores the first C - overlap columns.  The first pass
// overlaps its neighbours by 2^Q - 1 columns; later passes stage their rows SKEWED by the delay the pass will apply to
// them (see dd_tree_pass; the pass before stores every row early by what 16-byte staging cannot express), which keeps
// their overlap at 2^Q - 1 as well instead of 2^i0 (2^Q - 1).  The first two steps of a pass over packed rows are made in
// registers while staging.  1024 channels take two passes (Q = 6 in 8-bit lanes for 2-bit samples, then Q = 4).
//
// The piecewise linear tree (section 3.1.1) is the same passes over sub-bands of N' channels (the blocks simply stop
// growing at N' rows: stage 1, eq. 18) followed by dd_tree_stage2 (eq. 22): out[d][t] = sum_n S_n[d'_n(d)][t + Dt''_n(d)].
// The frequency-padded tree is one tree over a stretched band whose first pass reads its rows through a row map.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "dd_common.cuh"
#include "dd_kernels.cuh"

namespace dd {
namespace {

constexpr int TR_THREADS = 512;

struct TreePassParams {
    const uint8_t *in;     // PACKED: rows of nbits-wide samples (nbits = 8: the 8-bit rows of a first pass); else 16-bit rows
    int64_t in_stride;     // bytes between input rows
    int64_t in_bytes;      // PACKED: bytes readable from the start of a row (zero beyond)
    uint8_t *out;          // rows of LB-bit lanes, or rows of the caller's type (LAST)
    int64_t out_stride;    // bytes between output rows
    int64_t out_cols;      // columns to produce: LAST stores exactly these, else whole tiles (up to tt - 1 columns more)
    int32_t nbits;         // PACKED: 2, 4, 8
    int32_t out_code;      // LAST: DD_OUT_*
    int32_t vec_ok;        // LAST: rows allow 16-byte stores
    int32_t i0;            // first step of the pass
    int32_t tt;            // columns a tile stores (multiple of 64)
    int32_t fuse2;         // packed rows: steps 0 and 1 are made while the rows are staged (the step loop starts at 2)
    int32_t radix4;        // pairs of steps in one trip through shared memory (0: every step on its own)
    int32_t next_i0;       // not LAST: the pass that reads these rows starts at step next_i0 and takes next_q steps
    int32_t next_q;        //   (0: no pass follows -- stage 2 reads the rows as they are)
    const int32_t *row_map;   // first pass of a frequency-padded tree: input row of every tree row, -1 = blank; else NULL
};

// words k .. k + 3 of the lane stream w[0..7] (two aligned 16-byte loads) from word E, bit `amount` on, and one lane further
template <int E, int LB>
__device__ __forceinline__ void tree_window(const uint32_t (&w)[8], uint32_t amount, uint32_t (&x0)[4], uint32_t (&x1)[4])
{
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        x0[k] = __funnelshift_rc(w[k + E], w[k + E + 1], amount);
        x1[k] = __funnelshift_rc(w[k + E], w[k + E + 1], amount + LB);   // (32: the next word)
    }
}

// the 128 / LB lanes from lane offset e (0 .. 128 / LB - 1, the same for every thread of a warp) on (x0), and those from
// e + 1 on (x1), of LB-bit lanes
template <int LB>
__device__ __forceinline__ void tree_windows(const uint4 a, const uint4 b, int e, uint32_t (&x0)[4], uint32_t (&x1)[4])
{
    constexpr int LPW = 32 / LB;   // lanes per word
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    const uint32_t amount = (e & (LPW - 1)) * LB;
    switch (e / LPW) {
    case 0:
        tree_window<0, LB>(w, amount, x0, x1);
        break;
    case 1:
        tree_window<1, LB>(w, amount, x0, x1);
        break;
    case 2:
        tree_window<2, LB>(w, amount, x0, x1);
        break;
    default:
        tree_window<3, LB>(w, amount, x0, x1);
        break;
    }
}

__device__ __forceinline__ uint32_t sel4(const uint4 v, int i) { return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w)); }

// 16 bytes of lanes (one chunk: 128 / LB samples) from packed samples, LSB first; kk = index of the chunk inside the 16
// packed bytes v
template <int LB>
__device__ __forceinline__ uint4 tree_unpack_chunk(const uint4 v, int nb, int kk)
{
    uint32_t o[4];
    if constexpr (LB == 32) {   // 4 samples of 8 bits (wider lanes are for sums beyond 65535: 8-bit input only): word kk
        const uint32_t word = sel4(v, kk);
#pragma unroll
        for (int h = 0; h < 4; ++h)
            o[h] = (word >> (8 * h)) & 0xFFu;
    } else if constexpr (LB == 16) {   // 8 samples
        if (nb == 8) {          // words 2 kk, 2 kk + 1
            const uint32_t lo = sel4(v, 2 * kk), hi = sel4(v, 2 * kk + 1);
            o[0] = __byte_perm(lo, 0u, 0x4140), o[1] = __byte_perm(lo, 0u, 0x4342);
            o[2] = __byte_perm(hi, 0u, 0x4140), o[3] = __byte_perm(hi, 0u, 0x4342);
        } else if (nb == 4) {   // word kk, 8 nibbles
            const uint32_t word = sel4(v, kk);
#pragma unroll
            for (int h = 0; h < 4; ++h)
                o[h] = ((word >> (8 * h)) & 0xFu) | (((word >> (8 * h + 4)) & 0xFu) << 16);
        } else {                // half kk & 1 of word kk >> 1, 8 pairs of bits
            const uint32_t word = sel4(v, kk >> 1) >> (16 * (kk & 1));
#pragma unroll
            for (int h = 0; h < 4; ++h)
                o[h] = ((word >> (4 * h)) & 0x3u) | (((word >> (4 * h + 2)) & 0x3u) << 16);
        }
    } else {                    // 16 samples into bytes
        if (nb == 4) {          // words 2 kk, 2 kk + 1: 4 nibbles per output word
            const uint32_t lo = sel4(v, 2 * kk), hi = sel4(v, 2 * kk + 1);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const uint32_t hw = ((h < 2 ? lo : hi) >> (16 * (h & 1))) & 0xFFFFu;
                const uint32_t t = (hw | (hw << 8)) & 0x00FF00FFu;
                o[h] = (t | (t << 4)) & 0x0F0F0F0Fu;
            }
        } else {                // word kk: 4 pairs of bits per output word
            const uint32_t word = sel4(v, kk);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const uint32_t b = (word >> (8 * h)) & 0xFFu;
                const uint32_t t = (b | (b << 12)) & 0x000F000Fu;
                o[h] = (t | (t << 6)) & 0x03030303u;
            }
        }
    }
    return make_uint4(o[0], o[1], o[2], o[3]);
}

// words 0 .. 3 of the lane stream l[0..7] taken S lanes further on (S = 1, 2, 3: the delays of the first two steps)
template <int LB, int S>
__device__ __forceinline__ void tree_lanes_from(const uint32_t (&l)[8], uint32_t (&o)[4])
{
    constexpr int WO = (S * LB) / 32, AM = (S * LB) % 32;
#pragma unroll
    for (int k = 0; k < 4; ++k)
        o[k] = AM == 0 ? l[k + WO] : __funnelshift_r(l[k + WO], l[k + WO + 1], AM);
}

// One pass: steps i0 .. i0 + Q - 1 for one butterfly (R = 2^Q rows) and one time tile.
//   group g = k 2^i0 + x: butterfly x of block k (blocks of B = R 2^i0 rows after the pass)
//   staged row b' (level i0) = global row k B + b' 2^i0 + x;   stored row o' = global row k B + x R + o'
// In local terms step q combines the local blocks of 2^q rows pairwise exactly as the whole tree does, with x 2^q added to
// every delay: out[c][2 o + b] = in[2c][o] + in[2c + 1][o] at + (x 2^q + o + b).
// LB = bits per lane in shared memory: 16, or 8 for a first pass whose sums stay below 256 (2-bit samples: up to 64
// channels) -- half the shared-memory traffic per sample, which bounds the pass, and half the bytes written.
template <int Q, int ITEMS, bool PACKED, bool LAST, int LB>
__global__ void __launch_bounds__(TR_THREADS, ITEMS <= 4 ? 2 : 1) dd_tree_pass(const TreePassParams p)
{
    constexpr int R = 1 << Q;
    constexpr int CPC = 128 / LB;                           // columns per 16-byte chunk
    constexpr int CH = ITEMS * TR_THREADS / (R / 2);        // 16-byte chunks per row (>= 32: a warp stays inside one row)
    constexpr int C = CH * CPC;                             // columns staged per row
    static_assert(CH >= 32 && (CH & (CH - 1)) == 0, "a warp's items must share their row");
    static_assert(LB == 16 || LB == 32 || (LB == 8 && PACKED), "8-bit lanes: first pass only");
    extern __shared__ uint4 smv[];                          // [R][CH] + one chunk of padding
    const int tid = threadIdx.x, lane = tid & 31;
    const int tile = blockIdx.x, g = blockIdx.y;
    const int x = g & ((1 << p.i0) - 1), k = g >> p.i0;
    const int64_t row0 = (static_cast<int64_t>(k) << (p.i0 + Q));
    // SKEWED STAGING (passes after the first).  Step q reads U at t + x 2^q + o + b: the part x 2^q is the same for every
    // row of the step, and over the pass it adds up to x r for staged row r (bit q of r says whether the row is on the U
    // side at step q).  So row r is staged from column t0 + x r instead of t0, and what is left of every shift is o + b --
    // a later pass is the first pass again, for every butterfly alike: the overlap of neighbouring tiles falls from
    // x (R - 1) columns (up to 960 of 2048 for the second pass of 1024 channels) to R - 1, and its first two steps can be
    // made in registers too.  Staging copies whole 16-byte granules (AL columns of the rows read), so the PRODUCER of the
    // rows stores each one (x r) mod AL columns early (its store phase below): column t of the row as stored is column
    // t + (x r) mod AL of the row, and staging from the granule A(x r) = x r - (x r) mod AL on lands on column t0 + x r.
    const bool skew = p.i0 > 0;
    constexpr int AL = PACKED ? 16 : CPC;   // columns per 16 bytes of the rows staged: 8-bit rows / rows of the pass's own lanes
    const int tt = p.tt;
    const int64_t t0 = static_cast<int64_t>(tile) * tt;
    auto first_col = [&](int r) -> int64_t { return skew ? t0 + ((x * r) & ~(AL - 1)) : t0; };

    // ---- stage R rows x C columns
    if (PACKED && p.fuse2) {
        // FIRST TWO STEPS IN REGISTERS.  Their delays are 0 .. 3 samples (eq. 8 for four channels: 0000 / 0011 / 0112 /
        // 0123), so a thread that unpacks one 16-byte chunk of lanes of four adjacent rows, and the three lanes after it,
        // can write the four rows of level 2 straight away: two of the pass's steps never go through shared memory.
        const int nb = p.nbits;
        const int wpc = CPC * nb / 32;                      // packed words per chunk: 1 or 2 (the host checks)
        // (the loads of two items first, then their sums row by row: few registers live -- two CTAs per SM leave 64)
        auto load_item = [&](int id, uint32_t (&w)[4][3]) {
            const int j = id / CH, ch = id & (CH - 1);
#pragma unroll
            for (int rr = 0; rr < 4; ++rr) {
                int64_t row = row0 + (static_cast<int64_t>(4 * j + rr) << p.i0) + x;
                if (p.row_map)
                    row = __ldg(&p.row_map[row]);
                const int64_t off = (first_col(4 * j + rr) + static_cast<int64_t>(ch) * CPC) * nb / 8;   // a multiple of 4
                const uint8_t *src = p.in + row * p.in_stride + off;
#pragma unroll
                for (int k = 0; k < 3; ++k)
                    w[rr][k] = (row >= 0 && k <= wpc && off + 4 * (k + 1) <= p.in_bytes) ? __ldg(reinterpret_cast<const uint32_t *>(src) + k) : 0u;
            }
        };
        auto make_item = [&](int id, const uint32_t (&w)[4][3]) {
            const int j = id / CH, ch = id & (CH - 1);
            uint32_t o[4][4];
            auto lanes_of = [&](int rr, uint32_t (&l)[8]) {   // the chunk, then the lanes that follow it (three are used)
                const uint4 a = tree_unpack_chunk<LB>(make_uint4(w[rr][0], w[rr][1], 0u, 0u), nb, 0);
                const uint4 b = tree_unpack_chunk<LB>(make_uint4(wpc == 1 ? w[rr][1] : w[rr][2], 0u, 0u, 0u), nb, 0);
                l[0] = a.x, l[1] = a.y, l[2] = a.z, l[3] = a.w, l[4] = b.x, l[5] = b.y, l[6] = b.z, l[7] = b.w;
            };
            {   // row 0: delay 0 in all four
                uint32_t l[8];
                lanes_of(0, l);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    o[0][k] = o[1][k] = o[2][k] = o[3][k] = l[k];
            }
            {   // row 1: delays 0 0 1 1
                uint32_t l[8], s1[4];
                lanes_of(1, l);
                tree_lanes_from<LB, 1>(l, s1);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    o[0][k] += l[k], o[1][k] += l[k], o[2][k] += s1[k], o[3][k] += s1[k];
            }
            {   // row 2: delays 0 1 1 2
                uint32_t l[8], s1[4], s2[4];
                lanes_of(2, l);
                tree_lanes_from<LB, 1>(l, s1);
                tree_lanes_from<LB, 2>(l, s2);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    o[0][k] += l[k], o[1][k] += s1[k], o[2][k] += s1[k], o[3][k] += s2[k];
            }
            {   // row 3: delays 0 1 2 3
                uint32_t l[8], s1[4], s2[4], s3[4];
                lanes_of(3, l);
                tree_lanes_from<LB, 1>(l, s1);
                tree_lanes_from<LB, 2>(l, s2);
                tree_lanes_from<LB, 3>(l, s3);
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    o[0][k] += l[k], o[1][k] += s1[k], o[2][k] += s2[k], o[3][k] += s3[k];
            }
#pragma unroll
            for (int rr = 0; rr < 4; ++rr)
                smv[(4 * j + rr) * CH + ch] = make_uint4(o[rr][0], o[rr][1], o[rr][2], o[rr][3]);
        };
        constexpr int NIT = (R / 4) * CH;
        for (int id = tid; id < NIT; id += 2 * TR_THREADS) {
            uint32_t wa[4][3], wb[4][3];
            const bool two = id + TR_THREADS < NIT;
            load_item(id, wa);
            if (two)
                load_item(id + TR_THREADS, wb);
            make_item(id, wa);
            if (two)
                make_item(id + TR_THREADS, wb);
        }
    } else if constexpr (PACKED) {
        // 16 packed bytes hold SUB chunks; they are taken in an order rotated by the lane so that the 16-byte stores of a
        // quarter warp fall into distinct banks.  Up to four loads in flight per thread.
        const int nb = p.nbits;
        const int sub = 128 / (CPC * nb);                   // chunks per 16 packed bytes: 8, 4, 2 (16-bit lanes) / 4, 2 (8-bit)
        const int lg_per_row = 31 - __clz(CH / sub);        // 16-byte loads per row, a power of two
        const int rot = (lane * sub) >> 3;
        auto fetch = [&](int id) {
            const int r = id >> lg_per_row, c16 = id & ((1 << lg_per_row) - 1);
            const int64_t off = first_col(r) * nb / 8 + static_cast<int64_t>(c16) * 16;   // (a multiple of 16)
            int64_t row = row0 + (static_cast<int64_t>(r) << p.i0) + x;
            if (p.row_map)
                row = __ldg(&p.row_map[row]);   // (the stretched band of eq. 25: most rows are blank)
            const uint8_t *src = p.in + row * p.in_stride + off;
            return (row >= 0 && off >= 0 && off + 16 <= p.in_bytes) ? __ldg(reinterpret_cast<const uint4 *>(src)) : make_uint4(0, 0, 0, 0);
        };
        auto unpack = [&](int id, const uint4 v) {
            const int r = id >> lg_per_row, c16 = id & ((1 << lg_per_row) - 1);
            uint4 *dst = smv + r * CH + c16 * sub;
            for (int kk0 = 0; kk0 < sub; ++kk0) {
                const int kk = (kk0 + rot) & (sub - 1);
                dst[kk] = tree_unpack_chunk<LB>(v, nb, kk);
            }
        };
        const int total = R << lg_per_row;   // (a power of two)
        if (total >= 4 * TR_THREADS) {       // four loads in flight per thread
            for (int id = tid; id < total; id += 4 * TR_THREADS) {
                uint4 v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    v[j] = fetch(id + j * TR_THREADS);
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    unpack(id + j * TR_THREADS, v[j]);
            }
        } else {
            for (int id = tid; id < total; id += 2 * TR_THREADS) {
                const bool two = id + TR_THREADS < total;
                const uint4 va = fetch(id);
                const uint4 vb = two ? fetch(id + TR_THREADS) : make_uint4(0, 0, 0, 0);
                unpack(id, va);
                if (two)
                    unpack(id + TR_THREADS, vb);
            }
        }
    } else {
        // 16-bit rows: one bulk copy per row, issued by the first lane of the warps in turn
        __shared__ uint64_t full;
        if (tid == 0) {
            mbar_init(&full, 1);
            mbar_fence_init();
            mbar_arrive_expect_tx(&full, static_cast<uint32_t>(R * CH * 16));
        }
        __syncthreads();
        if (lane == 0) {
            for (int r = tid >> 5; r < R; r += TR_THREADS / 32) {
                const uint8_t *src = p.in + (row0 + (static_cast<int64_t>(r) << p.i0) + x) * p.in_stride + first_col(r) * (LB / 8);
                tma_bulk_g2s(smv + r * CH, src, static_cast<uint32_t>(CH * 16), &full);
            }
        }
        mbar_wait(&full, 0);
    }
    if (tid == 0)
        smv[R * CH] = make_uint4(0, 0, 0, 0);

    // ---- Q steps in place
    // the window of U: CPC lanes of staged row `row` from lane ch CPC + shift on (x0), and from one lane further on (x1)
    auto windows_at = [&](int row, int ch, int shift, uint32_t (&x0)[4], uint32_t (&x1)[4]) {
        int uch = ch + shift / CPC;
        uch = uch < CH - 1 ? uch : CH - 1;   // (columns whose window leaves the tile are never stored)
        const uint4 *u = smv + row * CH + uch;
        const uint4 ua = u[0], ub = u[1];
        tree_windows<LB>(ua, ub, shift & (CPC - 1), x0, x1);
    };
    // one step (eq. 11-12): out[c][2 o + b] = L[o] + U[o] at + (o + b); an item is one pair (L row, U row) x one chunk
    auto radix2 = [&](const int q) {
        uint32_t s0[ITEMS][4], s1[ITEMS][4];
        __syncthreads();
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const int id = it * TR_THREADS + tid;
            const int ch = id & (CH - 1), pair = id / CH;
            const int o = pair & ((1 << q) - 1), c = pair >> q;
            const int lrow = ((2 * c) << q) + o;
            const uint4 l = smv[lrow * CH + ch];
            uint32_t x0[4], x1[4];
            windows_at(lrow + (1 << q), ch, o, x0, x1);   // (+ b for the second sum; the x 2^q of a later pass is in the staging)
            const uint32_t lw[4] = {l.x, l.y, l.z, l.w};
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                s0[it][h] = lw[h] + x0[h];   // 32 / LB lanes per word; the sums stay below 2^LB
                s1[it][h] = lw[h] + x1[h];
            }
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const int id = it * TR_THREADS + tid;
            const int ch = id & (CH - 1), pair = id / CH;
            const int o = pair & ((1 << q) - 1), c = pair >> q;
            uint4 *dst = smv + ((c << (q + 1)) + 2 * o) * CH + ch;
            dst[0] = make_uint4(s0[it][0], s0[it][1], s0[it][2], s0[it][3]);
            dst[CH] = make_uint4(s1[it][0], s1[it][1], s1[it][2], s1[it][3]);
        }
    };
    // TWO steps q, q + 1 in one trip through shared memory: four blocks A, B, C, D of 2^q rows merge into one of 2^(q+2),
    //     out[4 o + 2 b1 + b2] = A[o] + B[o] at + (o + b1) + C[o] at + (2 o + b1 + b2) + D[o] at + (3 o + 2 b1 + b2)
    // (step q makes A + B at o + b1 and C + D at o + b1, step q + 1 adds the second to the first at 2 o + b1 + b2): 11
    // 16-byte loads and 4 stores per item of four rows instead of 2 x (6 + 4) -- the passes are bound by shared memory.
    auto radix4 = [&](const int q) {
        constexpr int NI = ITEMS / 2;
        uint32_t res[NI][4][4];
        __syncthreads();
#pragma unroll
        for (int it = 0; it < NI; ++it) {
            const int id = it * TR_THREADS + tid;
            const int ch = id & (CH - 1), quad = id / CH;
            const int o = quad & ((1 << q) - 1), c = quad >> q;
            const int arow = ((4 * c) << q) + o;
            const uint4 a = smv[arow * CH + ch];
            const uint32_t aw[4] = {a.x, a.y, a.z, a.w};
            uint32_t x0[4], x1[4];
            windows_at(arow + (1 << q), ch, o, x0, x1);                 // B at o, o + 1
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                res[it][0][h] = res[it][1][h] = aw[h] + x0[h];
                res[it][2][h] = res[it][3][h] = aw[h] + x1[h];
            }
            windows_at(arow + (2 << q), ch, 2 * o, x0, x1);             // C at 2 o, 2 o + 1
#pragma unroll
            for (int h = 0; h < 4; ++h)
                res[it][0][h] += x0[h], res[it][1][h] += x1[h], res[it][2][h] += x1[h];
            windows_at(arow + (2 << q), ch, 2 * o + 2, x0, x1);         // C at 2 o + 2
#pragma unroll
            for (int h = 0; h < 4; ++h)
                res[it][3][h] += x0[h];
            windows_at(arow + (3 << q), ch, 3 * o, x0, x1);             // D at 3 o, 3 o + 1
#pragma unroll
            for (int h = 0; h < 4; ++h)
                res[it][0][h] += x0[h], res[it][1][h] += x1[h];
            windows_at(arow + (3 << q), ch, 3 * o + 2, x0, x1);         // D at 3 o + 2, 3 o + 3
#pragma unroll
            for (int h = 0; h < 4; ++h)
                res[it][2][h] += x0[h], res[it][3][h] += x1[h];
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < NI; ++it) {
            const int id = it * TR_THREADS + tid;
            const int ch = id & (CH - 1), quad = id / CH;
            const int o = quad & ((1 << q) - 1), c = quad >> q;
            uint4 *dst = smv + ((c << (q + 2)) + 4 * o) * CH + ch;
#pragma unroll
            for (int k = 0; k < 4; ++k)
                dst[k * CH] = make_uint4(res[it][k][0], res[it][k][1], res[it][k][2], res[it][k][3]);
        }
    };
    const int q0 = (PACKED && p.fuse2) ? 2 : 0;   // (steps 0 and 1 were made while staging)
#pragma unroll
    for (int q = 0; q < Q; q += 2) {
        if (q < q0)
            continue;
        if (q + 1 < Q && p.radix4) {
            radix4(q);
        } else {
            radix2(q);
            if (q + 1 < Q)
                radix2(q + 1);
        }
    }
    __syncthreads();

    // ---- store the first tt columns of every row: a warp per row, consecutive lanes consecutive 16 bytes
    for (int r = tid >> 5; r < R; r += TR_THREADS / 32) {
        uint8_t *orow = p.out + (row0 + (static_cast<int64_t>(x) << Q) + r) * p.out_stride;
        const uint4 *srow = smv + r * CH;
        if constexpr (!LAST) {
            // rows that a later pass stages skewed are stored (x' r') mod CPC columns early, x' and r' being the butterfly
            // and the staged row this row is in that pass (see SKEWED STAGING): 0 .. CPC - 1 lanes, the same for the row
            int early = 0;
            if (p.next_q > 0) {
                const int64_t grow = row0 + (static_cast<int64_t>(x) << Q) + r;
                const int xn = static_cast<int>(grow & ((int64_t(1) << p.next_i0) - 1));
                const int rn = static_cast<int>((grow >> p.next_i0) & ((1 << p.next_q) - 1));
                early = (xn * rn) & (CPC - 1);
            }
            for (int ch = lane; ch < tt / CPC; ch += 32) {
                uint4 v = srow[ch];
                if (early) {
                    uint32_t x0[4], x1[4];
                    tree_windows<LB>(v, srow[ch + 1], early, x0, x1);
                    v = make_uint4(x0[0], x0[1], x0[2], x0[3]);
                }
                *reinterpret_cast<uint4 *>(orow + (t0 + ch * CPC) * (LB / 8)) = v;
            }
        } else if (p.out_code == DD_OUT_U16) {
            // 8 columns per thread: 16 bytes of 16-bit lanes as they are, or 8 bytes of 8-bit lanes widened
            for (int c8 = lane; c8 < tt / 8; c8 += 32) {
                const int64_t col = t0 + c8 * 8;
                if (col >= p.out_cols)
                    break;
                uint4 v;
                if constexpr (LB == 32) {     // (sums beyond 65535 have no uint16 output: dd_tree_execute refuses it)
                    const uint4 a = srow[2 * c8], b = srow[2 * c8 + 1];
                    v = make_uint4(a.x | a.y << 16, a.z | a.w << 16, b.x | b.y << 16, b.z | b.w << 16);
                } else if constexpr (LB == 16) {
                    v = srow[c8];
                } else {
                    const uint2 b = reinterpret_cast<const uint2 *>(srow)[c8];
                    v = make_uint4(__byte_perm(b.x, 0u, 0x4140), __byte_perm(b.x, 0u, 0x4342), __byte_perm(b.y, 0u, 0x4140),
                                   __byte_perm(b.y, 0u, 0x4342));
                }
                if (p.vec_ok && col + 8 <= p.out_cols) {
                    *reinterpret_cast<uint4 *>(orow + col * 2) = v;
                } else {
                    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
                    for (int h = 0; h < 8 && col + h < p.out_cols; ++h)
                        reinterpret_cast<uint16_t *>(orow)[col + h] = static_cast<uint16_t>(w[h >> 1] >> (16 * (h & 1)));
                }
            }
        } else {
            // 4 columns per thread: one 16-byte store of 32-bit elements
            const bool f32 = p.out_code == DD_OUT_F32;
            for (int c4 = lane; c4 < tt / 4; c4 += 32) {
                const int64_t col = t0 + c4 * 4;
                if (col >= p.out_cols)
                    break;
                uint32_t e[4];
                if constexpr (LB == 32) {
                    const uint4 v = srow[c4];
                    e[0] = v.x, e[1] = v.y, e[2] = v.z, e[3] = v.w;
                } else if constexpr (LB == 16) {
                    const uint2 v = reinterpret_cast<const uint2 *>(srow)[c4];
                    e[0] = v.x & 0xFFFFu, e[1] = v.x >> 16, e[2] = v.y & 0xFFFFu, e[3] = v.y >> 16;
                } else {
                    const uint32_t v = reinterpret_cast<const uint32_t *>(srow)[c4];
                    e[0] = v & 0xFFu, e[1] = (v >> 8) & 0xFFu, e[2] = (v >> 16) & 0xFFu, e[3] = v >> 24;
                }
                if (f32) {
#pragma unroll
                    for (int h = 0; h < 4; ++h)
                        e[h] = __float_as_uint(static_cast<float>(e[h]));
                }
                if (p.vec_ok && col + 4 <= p.out_cols)
                    *reinterpret_cast<uint4 *>(orow + col * 4) = make_uint4(e[0], e[1], e[2], e[3]);
                else
                    for (int h = 0; h < 4 && col + h < p.out_cols; ++h)
                        reinterpret_cast<uint32_t *>(orow)[col + h] = e[h];
            }
        }
    }
}

// Stage 2 of the piecewise linear tree (eq. 22): out[d][t] = sum_n S[n N' + d'_n(d)][t + Dt''_n(d)] over rows S of LB-bit
// lanes.  One thread per 128 / LB consecutive samples of one trial; tab[d][n] = {row, offset}.  The offsets of a (trial,
// sub-band) are the same for the whole block, so the windows are cut out of two aligned 16-byte loads as in the passes.
constexpr int TR2_THREADS = 256;
template <int LB>
__global__ void __launch_bounds__(TR2_THREADS) dd_tree_stage2(const uint8_t *__restrict__ S, int64_t pitch, const int2 *__restrict__ tab,
                                                              int ns, uint8_t *__restrict__ out, int64_t out_stride, int64_t nsamps,
                                                              int out_code, int vec_ok)
{
    constexpr int CPC = 128 / LB;
    extern __shared__ int2 stab[];
    const int d = blockIdx.y;
    for (int n = threadIdx.x; n < ns; n += TR2_THREADS)
        stab[n] = __ldg(&tab[static_cast<int64_t>(d) * ns + n]);
    __syncthreads();
    const int64_t col = (static_cast<int64_t>(blockIdx.x) * TR2_THREADS + threadIdx.x) * CPC;
    if (col >= nsamps)
        return;
    uint32_t acc[CPC];
#pragma unroll
    for (int h = 0; h < CPC; ++h)
        acc[h] = 0u;
    for (int n = 0; n < ns; ++n) {
        const int2 e = stab[n];
        const int64_t at = col + e.y;
        const uint8_t *src = S + (static_cast<int64_t>(e.x) * pitch + (at & ~int64_t(CPC - 1))) * (LB / 8);
        const uint4 a = __ldg(reinterpret_cast<const uint4 *>(src)), b = __ldg(reinterpret_cast<const uint4 *>(src + 16));
        uint32_t x0[4], x1[4];
        tree_windows<LB>(a, b, static_cast<int>(at & (CPC - 1)), x0, x1);
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            if constexpr (LB == 32) {
                acc[h] += x0[h];
            } else if constexpr (LB == 16) {
                acc[2 * h] += x0[h] & 0xFFFFu;
                acc[2 * h + 1] += x0[h] >> 16;
            } else {
                acc[4 * h] += x0[h] & 0xFFu;
                acc[4 * h + 1] += (x0[h] >> 8) & 0xFFu;
                acc[4 * h + 2] += (x0[h] >> 16) & 0xFFu;
                acc[4 * h + 3] += x0[h] >> 24;
            }
        }
    }
    uint8_t *orow = out + static_cast<int64_t>(d) * out_stride;
    const bool whole = vec_ok && col + CPC <= nsamps;
    if (out_code == DD_OUT_U16) {
        if (whole && CPC >= 8) {
#pragma unroll
            for (int v = 0; v < CPC / 8; ++v)
                reinterpret_cast<uint4 *>(orow + col * 2)[v] =
                    make_uint4(acc[8 * v] | acc[8 * v + 1] << 16, acc[8 * v + 2] | acc[8 * v + 3] << 16,
                               acc[8 * v + 4] | acc[8 * v + 5] << 16, acc[8 * v + 6] | acc[8 * v + 7] << 16);
        } else {
            for (int h = 0; h < CPC && col + h < nsamps; ++h)
                reinterpret_cast<uint16_t *>(orow)[col + h] = static_cast<uint16_t>(acc[h]);
        }
    } else {
        if (out_code == DD_OUT_F32) {
#pragma unroll
            for (int h = 0; h < CPC; ++h)
                acc[h] = __float_as_uint(static_cast<float>(acc[h]));
        }
        if (whole) {
#pragma unroll
            for (int v = 0; v < CPC / 4; ++v)
                reinterpret_cast<uint4 *>(orow + col * 4)[v] = make_uint4(acc[4 * v], acc[4 * v + 1], acc[4 * v + 2], acc[4 * v + 3]);
        } else {
            for (int h = 0; h < CPC && col + h < nsamps; ++h)
                reinterpret_cast<uint32_t *>(orow)[col + h] = acc[h];
        }
    }
}

// ------------------------------------------------------------------------------------------ host side
struct TreePass {
    int i0 = 0, q = 0, items = 4;
    int lane_bits = 16;               // lanes of the pass in shared memory and of the rows it stores (unless it is the last)
    bool packed = true;               // input: packed samples (the first pass), or the 8-bit rows of the pass before; else 16-bit rows
    int in_bits = 0;                  // packed: bits per sample of the input
    int cols = 0, halo = 0, tt = 0;   // columns staged / overlap of neighbouring tiles / columns a tile stores
    int64_t out_cols = 0;             // columns the pass produces for the current nsamps
    int64_t ntiles = 0;
};

// kind: 0 = 16-bit rows in, 16-bit lanes; 1 = packed in, 16-bit lanes; 2 = packed in, 8-bit lanes; 3 = packed in, 32-bit
// lanes; 4 = 32-bit rows in, 32-bit lanes
template <int Q, int ITEMS>
cudaError_t launch_pass_qi(const TreePassParams &p, int kind, bool last, int64_t groups, int64_t ntiles, cudaStream_t stream)
{
    constexpr int R = 1 << Q;
    const size_t smem = (static_cast<size_t>(R) * (ITEMS * TR_THREADS / (R / 2)) + 1) * 16;
    if (ntiles <= 0 || ntiles > 0x7FFFFFFFLL || groups <= 0 || groups > 65535)
        return cudaErrorInvalidConfiguration;
    auto go = [&](auto kernel) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        if (e != cudaSuccess)
            return e;
        kernel<<<dim3(static_cast<unsigned>(ntiles), static_cast<unsigned>(groups)), TR_THREADS, smem, stream>>>(p);
        return cudaGetLastError();
    };
    if (kind == 4)
        return last ? go(dd_tree_pass<Q, ITEMS, false, true, 32>) : go(dd_tree_pass<Q, ITEMS, false, false, 32>);
    if (kind == 3)
        return last ? go(dd_tree_pass<Q, ITEMS, true, true, 32>) : go(dd_tree_pass<Q, ITEMS, true, false, 32>);
    if (kind == 2)
        return last ? go(dd_tree_pass<Q, ITEMS, true, true, 8>) : go(dd_tree_pass<Q, ITEMS, true, false, 8>);
    if (kind == 1)
        return last ? go(dd_tree_pass<Q, ITEMS, true, true, 16>) : go(dd_tree_pass<Q, ITEMS, true, false, 16>);
    return last ? go(dd_tree_pass<Q, ITEMS, false, true, 16>) : go(dd_tree_pass<Q, ITEMS, false, false, 16>);
}

template <int Q>
cudaError_t launch_pass_q(const TreePassParams &p, int items, int kind, bool last, int64_t groups, int64_t ntiles, cudaStream_t stream)
{
    return items == 4 ? launch_pass_qi<Q, 4>(p, kind, last, groups, ntiles, stream)
                      : launch_pass_qi<Q, 8>(p, kind, last, groups, ntiles, stream);
}

cudaError_t launch_pass(const TreePassParams &p, int q, int items, int kind, bool last, int64_t groups, int64_t ntiles, cudaStream_t stream)
{
    switch (q) {
    case 1:
        return launch_pass_q<1>(p, items, kind, last, groups, ntiles, stream);
    case 2:
        return launch_pass_q<2>(p, items, kind, last, groups, ntiles, stream);
    case 3:
        return launch_pass_q<3>(p, items, kind, last, groups, ntiles, stream);
    case 4:
        return launch_pass_q<4>(p, items, kind, last, groups, ntiles, stream);
    case 5:
        return launch_pass_q<5>(p, items, kind, last, groups, ntiles, stream);
    case 6:
        return launch_pass_q<6>(p, items, kind, last, groups, ntiles, stream);
    }
    return cudaErrorInvalidValue;
}

int pass_cols(int q, int items, int lane_bits) { return items * TR_THREADS * (128 / lane_bits) / ((1 << q) / 2); }

}  // namespace
}  // namespace dd

struct dd_tree_s {
    int nchans = 0, sb = 0, nbits = 0, steps = 0;   // nchans: rows of the tree (the stretched band when padded)
    // frequency-padded tree: the real channels lie at rows pad_pos of a band of nchans rows
    int nchans_in = 0;                  // real channels (0: not padded)
    std::vector<int32_t> pad_pos;       // [nchans_in]
    void *d_row_map = nullptr;          // int32 [nchans]: input row or -1
    int tune[6] = {0, 0, 0, 0, 0, 0};   // steps of the first pass / of later passes, items per thread of the first pass / of later
                                     // passes, lanes of the first pass (16: never 8-bit lanes), 1: no steps fused into staging
    // stage 2 (piecewise linear tree)
    int ndm = 0, ns = 0;
    std::vector<int32_t> dprime, dt2;   // [ndm][ns]
    int64_t max_dt2 = 0;
    void *d_tab = nullptr;              // int2 [ndm][ns] {row of S, offset}
    bool tab_uploaded = false;
    // passes and intermediate rows, sized for `sized_for` output samples with the tuning `sized_tune`
    std::vector<dd::TreePass> passes;
    int64_t sized_for = -1;
    int sized_tune[5] = {-1, -1, -1, -1, -1};
    int sized_ndm = -1;
    void *buf[2] = {nullptr, nullptr};
    size_t buf_bytes[2] = {0, 0};
    int64_t pitch[8] = {};              // columns per row of the output of pass p
    int64_t last_launches = 0;
};

namespace dd {
namespace {

const double kTreeDm = 4.148808e3;   // k_DM in MHz^2 pc^-1 cm^3 s
constexpr int64_t kTreeMargin = 128;  // zero columns in front of every row between the passes

int log2_exact(int v)
{
    int k = 0;
    while ((1 << k) < v)
        ++k;
    return (1 << k) == v ? k : -1;
}

// The passes for t_out output columns of the last pass; false if the tuning leaves a pass without room for a tile.
bool plan_passes(dd_tree_s *t, int64_t t_out)
{
    t->passes.clear();
    const int vmax = (1 << t->nbits) - 1;
    for (int i0 = 0; i0 < t->steps;) {
        const int left = t->steps - i0;
        const int items = (i0 == 0 ? t->tune[2] : t->tune[3]) == 8 ? 8 : 4;   // 4: two CTAs per SM (measured faster on every pass)
        int q = std::min(left, 6);
        if (i0 == 0 && t->tune[0] > 0)
            q = std::min(q, t->tune[0]);
        if (i0 > 0 && t->tune[1] > 0)
            q = std::min(q, t->tune[1]);
        // the first pass adds in 8-bit lanes when its sums stay below 256 (2-bit samples: any first pass; 4-bit: up to 4 steps)
        // (and in 32-bit lanes throughout when the sums of a tree go beyond 16 bits: 8-bit samples, more than 256 channels)
        const bool wide = static_cast<int64_t>(t->sb) * vmax > 65535;
        auto lanes = [&](int qq) { return wide ? 32 : ((i0 == 0 && t->tune[4] != 16 && vmax * (1 << qq) <= 255) ? 8 : 16); };
        // the overlap of neighbouring tiles is 2^q - 1 columns in every pass (later passes stage their rows skewed:
        // dd_tree_pass); later passes, and a first pass in 32-bit lanes, take as many steps as keep it (and the columns a
        // row may be stored early) within a quarter of the columns staged
        auto overlap = [&](int qq) { return (1 << qq) - 1; };
        for (; q > 1; --q) {
            const int cols = pass_cols(q, items, lanes(q));
            if (((i0 == 0 && !wide) || (i0 == 0 ? t->tune[0] : t->tune[1]) > 0 || 4 * (overlap(q) + 128 / lanes(q) - 1) <= cols) &&
                overlap(q) + 16 + 64 <= cols)
                break;
        }
        TreePass ps;
        ps.i0 = i0, ps.q = q, ps.items = items;
        ps.lane_bits = lanes(q);
        ps.packed = i0 == 0 || t->passes.back().lane_bits == 8;
        ps.in_bits = i0 == 0 ? t->nbits : 8;
        ps.cols = pass_cols(q, items, ps.lane_bits);
        ps.halo = overlap(q);
        t->passes.push_back(ps);
        i0 += q;
    }
    if (t->passes.size() > 6)
        return false;
    for (size_t p = 0; p < t->passes.size(); ++p) {
        TreePass &ps = t->passes[p];
        // rows that a later pass stages skewed are stored up to one 16-byte granule of lanes early: that many more columns
        // of the tile have to be complete
        const int early = p + 1 < t->passes.size() ? 128 / ps.lane_bits - 1 : 0;
        ps.tt = (ps.cols - ps.halo - early) & ~63;
        if (ps.tt < 64)
            return false;
    }
    // columns every pass has to produce, backwards: a later pass stages row r of butterfly x from column t0 + x r on
    // (x r < the rows of a block after the pass), cols columns of it
    int64_t need = t_out;
    for (int p = static_cast<int>(t->passes.size()) - 1; p >= 0; --p) {
        TreePass &ps = t->passes[p];
        ps.out_cols = need;
        ps.ntiles = (need + ps.tt - 1) / ps.tt;
        // whole tiles are stored; stage 2 reads up to 47 columns past its last sample; kTreeMargin spare columns in front
        t->pitch[p] = (kTreeMargin + ps.ntiles * ps.tt + 64 + 63) & ~int64_t(63);
        need = (ps.ntiles * ps.tt + (ps.i0 > 0 ? (int64_t(1) << (ps.i0 + ps.q)) : 0) + ps.cols + 63) & ~int64_t(63);
    }
    return true;
}

void tree_free_buffers(dd_tree_s *t)
{
    for (int i = 0; i < 2; ++i) {
        if (t->buf[i])
            cudaFree(t->buf[i]);
        t->buf[i] = nullptr;
        t->buf_bytes[i] = 0;
    }
    t->sized_for = -1;
}

}  // namespace
}  // namespace dd

extern "C" {

dd_status dd_tree_create(dd_tree *tree, int nchans, int sb_nchans, int nbits)
{
    if (!tree)
        return DD_ERR_NULL;
    *tree = nullptr;
    // (the rows are nchans / sb_nchans trees one after the other: sub-bands of one band, or the bands of several beams)
    const int ks = dd::log2_exact(sb_nchans);
    if (nchans < 2 || nchans > 65536 || sb_nchans < 2 || sb_nchans > 4096 || sb_nchans > nchans || ks < 0 || nchans % sb_nchans != 0 ||
        (nbits != 2 && nbits != 4 && nbits != 8))
        return DD_ERR_INVALID_ARG;
    dd_tree_s *t = new (std::nothrow) dd_tree_s;
    if (!t)
        return DD_ERR_NOMEM;
    t->nchans = nchans, t->sb = sb_nchans, t->nbits = nbits, t->steps = ks;
    *tree = t;
    return DD_OK;
}

dd_status dd_tree_destroy(dd_tree tree)
{
    if (!tree)
        return DD_OK;
    dd::tree_free_buffers(tree);
    if (tree->d_tab)
        cudaFree(tree->d_tab);
    if (tree->d_row_map)
        cudaFree(tree->d_row_map);
    delete tree;
    return DD_OK;
}

// Eq. 25: the row of real channel nu in the stretched band, nu' = round(1/2 (nu0 / dnu) [1 - (1 + (dnu / nu0) nu)^-2]); the
// band has nu'(N_nu) rows, rounded up to a power of two (readings X6, X7).
dd_status dd_tree_create_padded(dd_tree *tree, int nchans, double f_top, double df, int nbits)
{
    if (!tree)
        return DD_ERR_NULL;
    *tree = nullptr;
    if (nchans < 2 || nchans > 4096 || !(f_top > 0) || !(df < 0) || !std::isfinite(f_top) || !std::isfinite(df) ||
        !(f_top + static_cast<double>(nchans) * df > 0) || (nbits != 2 && nbits != 4 && nbits != 8))
        return DD_ERR_INVALID_ARG;
    std::vector<int32_t> pos;
    int64_t total = 0;
    try {
        pos.resize(nchans);
        for (int c = 0; c <= nchans; ++c) {
            const double y = 1.0 + (df / f_top) * static_cast<double>(c);
            const double x = 0.5 * (f_top / df) * (1.0 - 1.0 / (y * y));
            const double r = std::floor(x + 0.5);
            if (!(r >= 0) || r > 1e9)
                return DD_ERR_INVALID_ARG;
            if (c < nchans)
                pos[c] = static_cast<int32_t>(r);
            else
                total = static_cast<int64_t>(r);
        }
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
    int64_t npad = 2;
    while (npad < total)
        npad *= 2;
    if (npad > 4096)
        return DD_ERR_INVALID_ARG;   // (the stretched band does not fit the largest tree)
    dd_tree t = nullptr;
    const dd_status st = dd_tree_create(&t, static_cast<int>(npad), static_cast<int>(npad), nbits);
    if (st != DD_OK)
        return st;
    t->nchans_in = nchans;
    t->pad_pos.swap(pos);
    *tree = t;
    return DD_OK;
}

int dd_tree_get_padding(dd_tree tree, int32_t *pos)
{
    if (!tree)
        return DD_ERR_NULL;
    if (tree->nchans_in == 0)
        return DD_ERR_INVALID_ARG;
    if (pos)
        std::copy(tree->pad_pos.begin(), tree->pad_pos.end(), pos);
    return tree->nchans;
}

dd_status dd_tree_set_dm_list(dd_tree tree, double dt, double f_top, double df, const double *dm_list, int ndm)
{
    if (!tree || !dm_list)
        return DD_ERR_NULL;
    if (tree->nchans_in > 0)
        return DD_ERR_UNSUPPORTED;   // (the padded tree is one tree over the stretched band: its trials are fixed, eq. 26)
    if (ndm <= 0 || !(dt > 0) || !(f_top > 0) || !(df < 0) || !std::isfinite(dt) || !std::isfinite(f_top) || !std::isfinite(df) ||
        !(f_top + static_cast<double>(tree->nchans) * df > 0))   // (eq. 20 evaluates DeltaT one channel past the band: X3)
        return DD_ERR_INVALID_ARG;
    for (int d = 0; d < ndm; ++d)
        if (!(dm_list[d] >= 0) || !std::isfinite(dm_list[d]))
            return DD_ERR_INVALID_ARG;
    const int ns = tree->nchans / tree->sb;
    std::vector<int32_t> dprime, dt2;
    int64_t max_dt2 = 0;
    try {
        // DeltaT(nu_n) in samples at the sub-band edges nu_n = n N', n = 0 .. ns (eq. 4)
        std::vector<double> big_t(ns + 1);
        for (int n = 0; n <= ns; ++n) {
            const double edge = f_top + static_cast<double>(n * tree->sb) * df;
            big_t[n] = dd::kTreeDm * (1.0 / (edge * edge) - 1.0 / (f_top * f_top)) / dt;
        }
        dprime.resize(static_cast<size_t>(ndm) * ns);
        dt2.resize(static_cast<size_t>(ndm) * ns);
        for (int d = 0; d < ndm; ++d) {
            for (int n = 0; n < ns; ++n) {
                const double a = std::floor(dm_list[d] * (big_t[n + 1] - big_t[n]) + 0.5);   // eq. 20 (X3): rounded once
                const double b = std::floor(dm_list[d] * big_t[n] + 0.5);                    // eq. 23 (X4): the sum telescopes
                if (!(a >= 0) || !(b >= 0) || b > 2147483000.0)
                    return DD_ERR_DELAY_OVERFLOW;
                if (a >= static_cast<double>(tree->sb))
                    return DD_ERR_OUT_RANGE;   // beyond the diagonal DM (eq. 21, X5)
                dprime[static_cast<size_t>(d) * ns + n] = static_cast<int32_t>(a);
                dt2[static_cast<size_t>(d) * ns + n] = static_cast<int32_t>(b);
                max_dt2 = std::max<int64_t>(max_dt2, static_cast<int64_t>(b));
            }
        }
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
    tree->dprime.swap(dprime);
    tree->dt2.swap(dt2);
    tree->ndm = ndm, tree->ns = ns, tree->max_dt2 = max_dt2;
    tree->tab_uploaded = false;
    return DD_OK;
}

dd_status dd_tree_get_tables(dd_tree tree, int32_t *dprime, int32_t *dt2)
{
    if (!tree)
        return DD_ERR_NULL;
    if (tree->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    if (dprime)
        std::copy(tree->dprime.begin(), tree->dprime.end(), dprime);
    if (dt2)
        std::copy(tree->dt2.begin(), tree->dt2.end(), dt2);
    return DD_OK;
}

// The delays the steps apply, by running them on delay lists: a row of level i holds one delay per channel of its block.
dd_status dd_tree_get_delays(dd_tree tree, int32_t *delays)
{
    if (!tree || !delays)
        return DD_ERR_NULL;
    try {
        const int n = tree->sb;
        std::vector<std::vector<int32_t>> cur(n, std::vector<int32_t>(1, 0)), nxt(n);
        for (int r = 1; r < n; r *= 2) {
            for (int k = 0; k < n / (2 * r); ++k) {
                for (int m = 0; m < r; ++m) {
                    const std::vector<int32_t> &lo = cur[2 * r * k + m], &up = cur[2 * r * k + r + m];
                    for (int b = 0; b < 2; ++b) {
                        std::vector<int32_t> &o = nxt[2 * r * k + 2 * m + b];
                        o = lo;
                        for (int32_t v : up)
                            o.push_back(v + m + b);
                    }
                }
            }
            cur.swap(nxt);
        }
        for (int d = 0; d < n; ++d)
            std::copy(cur[d].begin(), cur[d].end(), delays + static_cast<size_t>(d) * n);
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
    return DD_OK;
}

int64_t dd_tree_required_samples(dd_tree tree, int64_t nsamps)
{
    if (!tree)
        return DD_ERR_NULL;
    if (nsamps <= 0 || nsamps > (int64_t(1) << 40))
        return DD_ERR_INVALID_ARG;
    return nsamps + (tree->ndm > 0 ? tree->max_dt2 : 0) + tree->sb - 1;
}

dd_status dd_tree_set_tuning(dd_tree tree, int key, int value)
{
    if (!tree)
        return DD_ERR_NULL;
    if (key < 1 || key > 6 || value < 0 || (key == 6 && value > 3) || (key <= 2 && value > 6) || ((key == 3 || key == 4) && value != 0 && value != 4 && value != 8) ||
        (key == 5 && value != 0 && value != 16))
        return DD_ERR_INVALID_ARG;
    tree->tune[key - 1] = value;
    return DD_OK;
}

dd_status dd_tree_get_info(dd_tree tree, int64_t *info)
{
    if (!tree || !info)
        return DD_ERR_NULL;
    for (int i = 0; i < 16; ++i)
        info[i] = 0;
    info[0] = static_cast<int64_t>(tree->passes.size());
    info[1] = tree->last_launches;
    info[2] = static_cast<int64_t>(tree->buf_bytes[0] + tree->buf_bytes[1]) +
              (tree->d_tab ? static_cast<int64_t>(tree->ndm) * tree->ns * 8 : 0);
    for (size_t p = 0; p < tree->passes.size() && p < 6; ++p) {
        info[3 + 2 * p] = tree->passes[p].q;
        info[4 + 2 * p] = tree->passes[p].tt;
    }
    return DD_OK;
}

dd_status dd_tree_execute(dd_tree tree, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr, int out_nbits,
                          void *stream)
{
    using namespace dd;
    if (!tree || !in_ptr || !out_ptr)
        return DD_ERR_NULL;
    const int es = out_nbits == DD_OUT_U16 ? 2 : ((out_nbits == DD_OUT_U32 || out_nbits == DD_OUT_F32) ? 4 : 0);
    if (nsamps <= 0 || nsamps > (int64_t(1) << 40) || es == 0)
        return DD_ERR_INVALID_ARG;
    if (in_stride <= 0 || in_stride % 16 != 0 || reinterpret_cast<uintptr_t>(in_ptr) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(out_ptr) % es != 0)
        return DD_ERR_ALIGNMENT;
    const bool stage2 = tree->ndm > 0;
    const int64_t t_out = nsamps + (stage2 ? tree->max_dt2 : 0);   // columns of the stage-1 rows
    const int64_t required = t_out + tree->sb - 1;
    if (in_stride > INT64_MAX / 8 || in_stride * 8 < required * tree->nbits)
        return DD_ERR_STRIDE_TOO_SMALL;
    const int64_t top = static_cast<int64_t>(tree->nchans_in > 0 ? tree->nchans_in : (stage2 ? tree->nchans : tree->sb)) * ((1 << tree->nbits) - 1);
    if (out_nbits == DD_OUT_U16 && top > 65535)
        return DD_ERR_OUT_RANGE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;

    // ---- passes and intermediate rows for this size (first call, or the size / tuning / DM list changed)
    if (tree->sized_for != t_out || tree->sized_ndm != tree->ndm || tree->sized_tune[0] != tree->tune[0] ||
        tree->sized_tune[1] != tree->tune[1] || tree->sized_tune[2] != tree->tune[2] || tree->sized_tune[3] != tree->tune[3] || tree->sized_tune[4] != tree->tune[4]) {
        tree->sized_for = -1;
        if (!plan_passes(tree, t_out)) {
            set_error_text("dd_tree_execute: the tuning leaves a pass without room for a tile");
            return DD_ERR_INVALID_ARG;
        }
        const int np = static_cast<int>(tree->passes.size());
        size_t need[2] = {0, 0};
        for (int p = 0; p < np; ++p)
            if (p + 1 < np || stage2)   // (the last pass of the plain tree writes the caller's rows)
                need[p & 1] = std::max(need[p & 1], static_cast<size_t>(tree->nchans) * static_cast<size_t>(tree->pitch[p]) *
                                                static_cast<size_t>(tree->passes[p].lane_bits / 8));
        for (int i = 0; i < 2; ++i) {
            if (tree->buf_bytes[i] < need[i]) {
                if (tree->buf[i])
                    cudaFree(tree->buf[i]);   // synchronises with kernels still using the old rows
                tree->buf[i] = nullptr;
                tree->buf_bytes[i] = 0;
                if ((e = cudaMalloc(&tree->buf[i], need[i])) != cudaSuccess)
                    return report_cuda_error(e, "dd_tree_execute cudaMalloc(rows)");
                tree->buf_bytes[i] = need[i];
                // columns no pass writes (past the last tile) are staged by the next pass but reach no output: defined all the same
                if ((e = cudaMemsetAsync(tree->buf[i], 0, need[i], st)) != cudaSuccess)
                    return report_cuda_error(e, "dd_tree_execute memset(rows)");
            }
        }
        tree->sized_for = t_out;
        tree->sized_ndm = tree->ndm;
        for (int i = 0; i < 5; ++i)
            tree->sized_tune[i] = tree->tune[i];
    }
    if (tree->nchans_in > 0 && !tree->d_row_map) {
        std::vector<int32_t> map(tree->nchans, -1);
        for (int c = 0; c < tree->nchans_in; ++c)
            map[tree->pad_pos[c]] = c;
        if ((e = cudaMalloc(&tree->d_row_map, map.size() * sizeof(int32_t))) != cudaSuccess ||
            (e = cudaMemcpy(tree->d_row_map, map.data(), map.size() * sizeof(int32_t), cudaMemcpyHostToDevice)) != cudaSuccess) {
            if (tree->d_row_map)
                cudaFree(tree->d_row_map);
            tree->d_row_map = nullptr;
            return report_cuda_error(e, "dd_tree_execute upload(row map)");
        }
    }
    if (stage2 && !tree->tab_uploaded) {
        std::vector<int2> tab(static_cast<size_t>(tree->ndm) * tree->ns);
        for (int d = 0; d < tree->ndm; ++d)
            for (int n = 0; n < tree->ns; ++n) {
                const size_t i = static_cast<size_t>(d) * tree->ns + n;
                tab[i] = make_int2(n * tree->sb + tree->dprime[i], tree->dt2[i]);
            }
        if (tree->d_tab)
            cudaFree(tree->d_tab);
        tree->d_tab = nullptr;
        if ((e = cudaMalloc(&tree->d_tab, tab.size() * sizeof(int2))) != cudaSuccess ||
            (e = cudaMemcpy(tree->d_tab, tab.data(), tab.size() * sizeof(int2), cudaMemcpyHostToDevice)) != cudaSuccess)
            return report_cuda_error(e, "dd_tree_execute upload(stage-2 table)");
        tree->tab_uploaded = true;
    }

    // ---- stage 1: the passes
    const int np = static_cast<int>(tree->passes.size());
    const int64_t out_pitch_bytes = nsamps * es;
    const bool rows16 = reinterpret_cast<uintptr_t>(out_ptr) % 16 == 0 && out_pitch_bytes % 16 == 0;
    int64_t launches = 0;
    for (int p = 0; p < np; ++p) {
        const TreePass &ps = tree->passes[p];
        const bool first = p == 0, last = p + 1 == np && !stage2;
        TreePassParams kp{};
        // (rows between the passes: column 0 lies kTreeMargin columns into the row)
        const int in_lb = first ? 0 : tree->passes[p - 1].lane_bits / 8, out_lb = ps.lane_bits / 8;
        kp.in = first ? static_cast<const uint8_t *>(in_ptr) : static_cast<const uint8_t *>(tree->buf[(p - 1) & 1]) + kTreeMargin * in_lb;
        kp.in_stride = first ? in_stride : tree->pitch[p - 1] * in_lb;
        kp.in_bytes = first ? in_stride : (tree->pitch[p - 1] - kTreeMargin) * in_lb;
        kp.out = last ? static_cast<uint8_t *>(out_ptr) : static_cast<uint8_t *>(tree->buf[p & 1]) + kTreeMargin * out_lb;
        kp.out_stride = last ? out_pitch_bytes : tree->pitch[p] * out_lb;
        kp.out_cols = last ? nsamps : ps.out_cols;
        kp.nbits = ps.in_bits;
        kp.out_code = out_nbits;
        kp.vec_ok = rows16 ? 1 : 0;
        kp.i0 = ps.i0;
        kp.tt = ps.tt;
        kp.row_map = first ? static_cast<const int32_t *>(tree->d_row_map) : nullptr;
        // steps 0 and 1 while staging packed rows (the input, or 8-bit rows): the chunk of a thread must be whole packed words
        // (not 2-bit samples in 16-bit lanes)
        kp.fuse2 = (ps.packed && ps.q >= 2 && (tree->tune[5] & 1) == 0 && (128 / ps.lane_bits) * ps.in_bits >= 32) ? 1 : 0;
        kp.radix4 = (tree->tune[5] & 2) ? 0 : 1;
        kp.next_i0 = p + 1 < np ? tree->passes[p + 1].i0 : 0;
        kp.next_q = p + 1 < np ? tree->passes[p + 1].q : 0;
        const int64_t groups = tree->nchans >> ps.q;
        const int kind = ps.lane_bits == 32 ? (ps.packed ? 3 : 4) : (ps.lane_bits == 8 ? 2 : (ps.packed ? 1 : 0));
        if ((e = launch_pass(kp, ps.q, ps.items, kind, last, groups, ps.ntiles, st)) != cudaSuccess)
            return report_cuda_error(e, "dd_tree_execute pass");
        ++launches;
    }
    // ---- stage 2
    if (stage2) {
        const int lb = tree->passes[np - 1].lane_bits;
        const int cpt = 128 / lb;   // columns per thread
        const dim3 grid(static_cast<unsigned>((nsamps + TR2_THREADS * cpt - 1) / (TR2_THREADS * cpt)), static_cast<unsigned>(tree->ndm));
        auto s2 = lb == 8 ? dd_tree_stage2<8> : (lb == 16 ? dd_tree_stage2<16> : dd_tree_stage2<32>);
        s2<<<grid, TR2_THREADS, static_cast<size_t>(tree->ns) * sizeof(int2), st>>>(
            static_cast<const uint8_t *>(tree->buf[(np - 1) & 1]) + kTreeMargin * (lb / 8), tree->pitch[np - 1], static_cast<const int2 *>(tree->d_tab), tree->ns,
            static_cast<uint8_t *>(out_ptr), out_pitch_bytes, nsamps, out_nbits, rows16 ? 1 : 0);
        if ((e = cudaGetLastError()) != cudaSuccess)
            return report_cuda_error(e, "dd_tree_execute stage 2");
        ++launches;
    }
    tree->last_launches = launches;
    return DD_OK;
}

}  // extern "C"
