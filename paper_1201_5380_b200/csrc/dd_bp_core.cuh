// dd_bp_core.cuh -- device helpers shared by the bit-plane kernels (dd_kernel_bp.cu, dd_kernel_gs.cu): the carry-save
// counter (PAPER.md:119's bit-level parallelism at one bit per lane), plane-vector loads, bit-matrix transposes and
// the output stores of the epilogue (time contiguous).
#pragma once
#include <cstdint>

#include "dd_common.cuh"
#include "dd_kernels.cuh"

namespace dd {

__host__ __device__ constexpr int bit_length(uint32_t v) { return v == 0 ? 0 : 1 + bit_length(v >> 1); }

// ------------------------------------------------------------------------------------------ carry-save counter
__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}

// Adds the word x of weight 2^L to the counter.  S is the compile-time occupancy of the pending slots
// (bit k set: T[k] holds a word of weight 2^k waiting for a partner) -- a binary counter of the words seen.
template <uint32_t S, int L, int NP, int NT>
__device__ __forceinline__ void csa_add(uint32_t (&P)[NP], uint32_t (&T)[NT], uint32_t x)
{
    static_assert(L < NT && L < NP, "carry-save counter overflow");
    if constexpr (((S >> L) & 1u) == 0u) {
        T[L] = x;
    } else {
        const uint32_t a = P[L], b = T[L];
        P[L] = xor3(a, b, x);
        csa_add<S - (1u << L), L + 1>(P, T, maj3(a, b, x));
    }
}

// Empties the pending slots into the planes: ripple-carry addition of the pending number (occupancy S) from
// level L upwards.  CARRY: a carry word `cy` of weight 2^L comes in from below.
template <uint32_t S, int L, bool CARRY, int NP, int NT>
__device__ __forceinline__ void csa_flush(uint32_t (&P)[NP], const uint32_t (&T)[NT], uint32_t cy)
{
    if constexpr (L < NP) {
        constexpr bool pend = L < NT && ((S >> L) & 1u) != 0u;
        if constexpr (pend && CARRY) {
            const uint32_t a = P[L];
            P[L] = xor3(a, T[L], cy);
            csa_flush<S, L + 1, true>(P, T, maj3(a, T[L], cy));
        } else if constexpr (pend || CARRY) {
            const uint32_t a = P[L], b = pend ? T[L < NT ? L : 0] : cy;
            P[L] = a ^ b;
            csa_flush<S, L + 1, true>(P, T, a & b);
        } else {
            csa_flush<S, L + 1, false>(P, T, 0u);
        }
    }
}

// ------------------------------------------------------------------------------------------ the kernel
template <int NB>
struct PlaneVec;
template <>
struct PlaneVec<1> {
    uint32_t w[1];
    __device__ __forceinline__ void load(const uint8_t *p) { w[0] = *reinterpret_cast<const uint32_t *>(p); }
};
template <>
struct PlaneVec<2> {
    uint32_t w[2];
    __device__ __forceinline__ void load(const uint8_t *p)
    {
        const uint2 v = *reinterpret_cast<const uint2 *>(p);
        w[0] = v.x, w[1] = v.y;
    }
};
template <>
struct PlaneVec<3> {
    uint32_t w[3];
    __device__ __forceinline__ void load(const uint8_t *p)
    {
        const uint32_t *q = reinterpret_cast<const uint32_t *>(p);
        w[0] = q[0], w[1] = q[1], w[2] = q[2];
    }
};
template <>
struct PlaneVec<4> {
    uint32_t w[4];
    __device__ __forceinline__ void load(const uint8_t *p)
    {
        const uint4 v = *reinterpret_cast<const uint4 *>(p);
        w[0] = v.x, w[1] = v.y, w[2] = v.z, w[3] = v.w;
    }
};

// adds `bytes` to the transaction count the current phase of the barrier waits for (no arrival)
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
// one try: has the phase of the given parity completed?  (mbar_wait spins on this)
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_addr(bar)), "r"(parity)
        : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}

// 32 x 32 bit-matrix transpose: R[i] bit k  <-  R[k] bit i
__device__ __forceinline__ void transpose32(uint32_t (&R)[32])
{
#pragma unroll
    for (int st = 0; st < 5; ++st) {
        const int sh = 16 >> st;
        const uint32_t m = st == 0 ? 0x0000FFFFu : st == 1 ? 0x00FF00FFu : st == 2 ? 0x0F0F0F0Fu : st == 3 ? 0x33333333u : 0x55555555u;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if (k & sh)
                continue;
            const uint32_t t = ((R[k] >> sh) ^ R[k + sh]) & m;
            R[k + sh] ^= t;
            R[k] ^= t << sh;
        }
    }
}
// 16 x 16 bit-matrix transpose of both half-words at once: afterwards R[k] = {sum of sample 16+k, sum of sample k}
__device__ __forceinline__ void transpose16x2(uint32_t (&R)[16])
{
#pragma unroll
    for (int st = 0; st < 4; ++st) {
        const int sh = 8 >> st;
        const uint32_t m = st == 0 ? 0x00FF00FFu : st == 1 ? 0x0F0F0F0Fu : st == 2 ? 0x33333333u : 0x55555555u;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            if (k & sh)
                continue;
            const uint32_t t = ((R[k] >> sh) ^ R[k + sh]) & m;
            R[k + sh] ^= t;
            R[k] ^= t << sh;
        }
    }
}

// four consecutive sums q[0..3] of DM row `orow` at sample t (a multiple of 4)
__device__ __forceinline__ void store4(const KernelParams &p, uint8_t *orow, int64_t t, const uint32_t (&q)[4])
{
    if (t >= p.nsamps)
        return;
    const bool whole = p.vec_ok && (t + 4 <= p.nsamps);
    if (p.out_code == DD_OUT_F32) {
        float *o = reinterpret_cast<float *>(orow) + t;
        if (whole) {
            *reinterpret_cast<float4 *>(o) =
                make_float4(__uint2float_rn(q[0]), __uint2float_rn(q[1]), __uint2float_rn(q[2]), __uint2float_rn(q[3]));
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k < p.nsamps)
                    o[k] = __uint2float_rn(q[k]);
        }
    } else if (p.out_code == DD_OUT_U32) {
        uint32_t *o = reinterpret_cast<uint32_t *>(orow) + t;
        if (whole) {
            *reinterpret_cast<uint4 *>(o) = make_uint4(q[0], q[1], q[2], q[3]);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k < p.nsamps)
                    o[k] = q[k];
        }
    } else if (p.out_code == kOutU8) {   // internal: the intermediate series of the sub-band method
        uint8_t *o = orow + t;
        if (whole) {
            *reinterpret_cast<uint32_t *>(o) = q[0] | (q[1] << 8) | (q[2] << 16) | (q[3] << 24);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k < p.nsamps)
                    o[k] = static_cast<uint8_t>(q[k]);
        }
    } else {
        uint16_t *o = reinterpret_cast<uint16_t *>(orow) + t;
        if (whole) {
            *reinterpret_cast<uint2 *>(o) = make_uint2(q[0] | (q[1] << 16), q[2] | (q[3] << 16));
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k < p.nsamps)
                    o[k] = static_cast<uint16_t>(q[k]);
        }
    }
}

// One unit (32 consecutive sums per lane) of a warp to global memory through the warp's shared-memory patch.
// Each lane packs its 32 sums into CH = 2 ES chunks of 16 bytes and writes them to its row of the patch; then
// the warp reads the patch back so that consecutive lanes hold consecutive chunks of the SAME unit and stores:
// every STG.128 covers whole 128-byte lines (4 units of float32) instead of 32 scattered 16-byte pieces.
// The chunk index is XOR-swizzled so that both the write and the read phase are free of bank conflicts.
//   ES     bytes per output element (4, 2, 1);  F32: convert to float32
//   gunit  address of this unit of lane 0;  lane s's unit is s * lane_pitch bytes further
template <int ES, bool F32>
__device__ __forceinline__ void store_unit_coalesced(const uint32_t (&q)[32], uint8_t *patch, int lane, uint8_t *gunit,
                                                     int lane_pitch)
{
    constexpr int CH = 2 * ES;            // 16-byte chunks per unit
    constexpr int LPL = 8 / CH;           // lanes per 128 bytes of the patch
    const int swz = (lane / LPL) % CH;
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        uint4 v;
        if constexpr (ES == 4) {
            if constexpr (F32)
                v = make_uint4(__float_as_uint(__uint2float_rn(q[4 * c])), __float_as_uint(__uint2float_rn(q[4 * c + 1])),
                               __float_as_uint(__uint2float_rn(q[4 * c + 2])), __float_as_uint(__uint2float_rn(q[4 * c + 3])));
            else
                v = make_uint4(q[4 * c], q[4 * c + 1], q[4 * c + 2], q[4 * c + 3]);
        } else if constexpr (ES == 2) {
            v = make_uint4(q[8 * c] | (q[8 * c + 1] << 16), q[8 * c + 2] | (q[8 * c + 3] << 16),
                           q[8 * c + 4] | (q[8 * c + 5] << 16), q[8 * c + 6] | (q[8 * c + 7] << 16));
        } else {
            uint32_t w[4];
#pragma unroll
            for (int k = 0; k < 4; ++k)
                w[k] = q[16 * c + 4 * k] | (q[16 * c + 4 * k + 1] << 8) | (q[16 * c + 4 * k + 2] << 16) | (q[16 * c + 4 * k + 3] << 24);
            v = make_uint4(w[0], w[1], w[2], w[3]);
        }
        *reinterpret_cast<uint4 *>(patch + lane * (CH * 16) + ((c ^ swz) * 16)) = v;
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        const int idx = i * 32 + lane, src = idx / CH, c = idx % CH;
        const uint4 v = *reinterpret_cast<const uint4 *>(patch + src * (CH * 16) + ((c ^ ((src / LPL) % CH)) * 16));
        *reinterpret_cast<uint4 *>(gunit + static_cast<int64_t>(src) * lane_pitch + c * 16) = v;
    }
    __syncwarp();
}

}  // namespace dd
