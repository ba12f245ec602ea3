// dd_kernel_bp.cu -- variant 3: 2-bit input as BIT PLANES, summed with carry-save adders.
//
//     D[d][t] = sum_c A[c][t + delay[d][c]]                       (eq. 3)
//
// The paper's bit-level parallelism (several samples per machine word, one word operation
// acting on all of them) taken to its end: ONE BIT per lane.  A pre-pass transposes every 32 consecutive
// 2-bit samples of a channel into two 32-bit words, plane 0 (the low bits) and plane 1 (the high bits), in
// time order (sub-word samples handled by shift and mask).  The sum over channels is then a
// population count per lane, kept as NP bit planes P[0..NP) (P[k] holds bit k of 32 sums) and updated with
// 3:2 carry-save adders: sum = a ^ b ^ c, carry = maj(a, b, c), two LOP3 instructions that add one more
// 32-sample word into the counter.  Per channel and 32 outputs that is 2 funnel shifts (the delay is an
// arbitrary bit offset into the plane words) + ~4.3 LOP3 for 32 channel-adds, against 4 shifts + 2 adds +
// 4 flush operations for the nibble lanes of variant 2, and half the shared-memory traffic.
//
// One CTA = 16 DM trials x 5120 output samples, 16 warps; warp w owns DM slot w, lane l owns the five
// 32-sample units 5l .. 5l+4 of the time block (W = 5: six 8-byte loads serve five units).
//   stage  : per channel, the bit-plane span [t0 + start, ...) of the DM block (time block + delay range,
//            PAPER.md:115) arrives by TMA bulk copy; ring of `nstages` stages of 32 channels, full/empty
//            mbarriers, no CTA-wide barrier in the channel loop;
//   add    : carry-save counter per unit; words of equal weight are paired as they appear (a binary counter
//            of pending words, resolved at compile time), the pending words left after 32 channels are
//            rippled into the upper planes;
//   store  : 16x16 bit-matrix transposes turn 12 planes x 32 lanes into 32 integers; float32 / uint32 /
//            uint16, 128-bit stores, time contiguous.
#include <utility>

#include "dd_common.cuh"
#include "dd_kernels.cuh"

namespace dd {
namespace {

constexpr int BP_DB = 16, BP_W = 5, BP_NWARPS = 16, BP_TB = 32 * 32 * BP_W, BP_CC = 32;
constexpr int BP_NP = 12;                 // planes: sums < 2^12 (plan: nchans * 3 < 4096)
constexpr int BP_NT = 8;                  // pending slots (weights 1 .. 128; 32 channels * 3 = 96 < 256)
constexpr uint32_t BP_WSUM = 3;           // weight added per channel: 2^nbits - 1

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

// 32 two-bit samples (two packed words, LSB first) -> {plane 0, plane 1}; bit k of a plane = sample k
__device__ __forceinline__ uint2 planes_of(uint32_t x0, uint32_t x1)
{
    const uint32_t m = 0x55555555u;
    return make_uint2(compress_even(x0 & m) | (compress_even(x1 & m) << 16),
                      compress_even((x0 >> 1) & m) | (compress_even((x1 >> 1) & m) << 16));
}

// in: packed rows [beam][c][in_stride]; work: bit-plane rows [beam][c][w_stride], unit u of a row is the
// uint2 {plane 0, plane 1} of samples 32u .. 32u+31.  One thread converts 16 bytes (64 samples, 2 units).
__global__ void __launch_bounds__(256) dd_to_bitplanes2(const uint8_t *__restrict__ in, int64_t in_stride,
                                                        int64_t in_beam_stride, uint8_t *__restrict__ work,
                                                        int64_t w_stride, int64_t w_beam_stride, int32_t chunks)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= chunks)
        return;
    const int64_t c = blockIdx.y, beam = blockIdx.z;
    const uint4 x = __ldg(reinterpret_cast<const uint4 *>(in + beam * in_beam_stride + c * in_stride) + i);
    const uint2 a = planes_of(x.x, x.y), b = planes_of(x.z, x.w);
    reinterpret_cast<uint4 *>(work + beam * w_beam_stride + c * w_stride)[i] = make_uint4(a.x, a.y, b.x, b.y);
}

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
template <uint32_t S, int L>
__device__ __forceinline__ void csa_add(uint32_t (&P)[BP_NP], uint32_t (&T)[BP_NT], uint32_t x)
{
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
template <uint32_t S, int L, bool CARRY>
__device__ __forceinline__ void csa_flush(uint32_t (&P)[BP_NP], const uint32_t (&T)[BP_NT], uint32_t cy)
{
    if constexpr (L < BP_NP) {
        constexpr bool pend = L < BP_NT && ((S >> L) & 1u) != 0u;
        if constexpr (pend && CARRY) {
            const uint32_t a = P[L];
            P[L] = xor3(a, T[L], cy);
            csa_flush<S, L + 1, true>(P, T, maj3(a, T[L], cy));
        } else if constexpr (pend || CARRY) {
            const uint32_t a = P[L], b = pend ? T[L < BP_NT ? L : 0] : cy;
            P[L] = a ^ b;
            csa_flush<S, L + 1, true>(P, T, a & b);
        } else {
            csa_flush<S, L + 1, false>(P, T, 0u);
        }
    }
}

// ------------------------------------------------------------------------------------------ the kernel
struct BpShared {
    const uint8_t *lane_base;   // stage base + this lane's byte offset (5 units = 40 bytes per lane)
    const uint2 *rel;           // this warp's offset entries of the stage: [cl * BP_DB]
};

// channel K of the stage: one window of W+1 units serves W units; 2 funnel shifts + carry-save adds per unit
template <int K>
__device__ __forceinline__ void channel_step(const BpShared &sh, uint32_t (&P)[BP_W][BP_NP], uint32_t (&T)[BP_W][BP_NT])
{
    const uint2 e = sh.rel[K * BP_DB];                                        // {byte offset in the stage, bit shift}
    const uint2 *wp = reinterpret_cast<const uint2 *>(sh.lane_base + e.x);
    uint2 x[BP_W + 1];
#pragma unroll
    for (int j = 0; j <= BP_W; ++j)
        x[j] = wp[j];
#pragma unroll
    for (int j = 0; j < BP_W; ++j) {
        const uint32_t b0 = __funnelshift_r(x[j].x, x[j + 1].x, e.y);
        const uint32_t b1 = __funnelshift_r(x[j].y, x[j + 1].y, e.y);
        csa_add<BP_WSUM * K, 0>(P[j], T[j], b0);
        csa_add<BP_WSUM * K + 1u, 1>(P[j], T[j], b1);
    }
}

template <int... Ks>
__device__ __forceinline__ void stage_steps(std::integer_sequence<int, Ks...>, const BpShared &sh,
                                            uint32_t (&P)[BP_W][BP_NP], uint32_t (&T)[BP_W][BP_NT])
{
    (channel_step<Ks>(sh, P, T), ...);
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}

__global__ void __launch_bounds__(BP_NWARPS * 32, 1) dd_direct_bp2(const KernelParams p)
{
    constexpr int DB = BP_DB, W = BP_W, TB = BP_TB, CC = BP_CC, NP = BP_NP;

    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // tile decode: DM block fastest so that CTAs resident together share the same input window (L2)
    const int64_t cta = blockIdx.x;
    const int blk = static_cast<int>(cta % p.nblk);
    const int64_t rest = cta / p.nblk;
    const int tile = static_cast<int>(rest % p.ntiles);
    const int beam = static_cast<int>(rest / p.ntiles);
    const int64_t t0 = static_cast<int64_t>(tile) * TB;

    // shared memory carve-up (must match dd::smem_layout_bytes)
    const int NS = p.nstages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);      // [NS]
    uint64_t *empty = full + 8;                                 // [NS]
    const int rel_stage = static_cast<int>(align128(static_cast<int64_t>(CC) * DB * 8));
    const int raw_stage = static_cast<int>(align128(static_cast<int64_t>(CC) * p.raw_slot));
    uint8_t *rel_base = smem + 128;
    uint8_t *raw_base = rel_base + NS * rel_stage;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&full[s], BP_NWARPS);
            mbar_init(&empty[s], BP_NWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const uint8_t *in_beam = p.in + static_cast<int64_t>(beam) * p.in_beam_stride;
    const int2 *span_blk = p.span + static_cast<int64_t>(blk) * p.nchans_pad;
    const uint2 *rel_blk = static_cast<const uint2 *>(p.rel) + static_cast<int64_t>(blk) * p.nchans_pad * DB;

    // producers: EVERY warp stages CPW = CC / NWARPS channels of each chunk (its lane 0 issues the bulk copies:
    // a bulk copy takes its operands from uniform registers, so one warp issuing all 32 copies of a chunk
    // serialises over its lanes and falls behind the others); warp 0 also stages the chunk's offset entries.
    // The span metadata of the next chunk to stage is fetched one step early.
    constexpr int CPW = CC / BP_NWARPS;
    auto load_meta = [&](int chunk, int2 (&m)[CPW]) {
#pragma unroll
        for (int k = 0; k < CPW; ++k)
            m[k] = (lane == 0 && chunk < p.nchunks) ? __ldg(&span_blk[chunk * CC + warp * CPW + k]) : make_int2(0, 0);
    };
    auto produce = [&](int chunk, const int2 (&m)[CPW]) {
        const int s = chunk % NS;
        if (lane == 0) {
            if (chunk >= NS)
                mbar_wait(&empty[s], ((chunk / NS) - 1) & 1);   // every warp has finished chunk - NS
            const uint8_t *src[CPW];
            uint32_t bytes[CPW], tx = (warp == 0) ? static_cast<uint32_t>(CC * DB * 8) : 0u;
#pragma unroll
            for (int k = 0; k < CPW; ++k) {
                const int c = chunk * CC + warp * CPW + k;
                if (m[k].y < 0) {                                // padded channel: zeros
                    src[k] = p.zero;
                    bytes[k] = static_cast<uint32_t>(-m[k].y);
                } else {
                    const int64_t off = ((t0 + m[k].x) * 2) >> 3;
                    const int64_t avail = p.in_row_bytes - off;
                    bytes[k] = static_cast<uint32_t>(m[k].y < avail ? m[k].y : (avail > 0 ? avail : 0));
                    src[k] = in_beam + static_cast<int64_t>(c) * p.in_stride + off;
                }
                tx += bytes[k];
            }
            mbar_arrive_expect_tx(&full[s], tx);
#pragma unroll
            for (int k = 0; k < CPW; ++k)
                if (bytes[k])
                    tma_bulk_g2s(raw_base + s * raw_stage + (warp * CPW + k) * p.raw_slot, src[k], bytes[k], &full[s]);
            if (warp == 0)
                tma_bulk_g2s(rel_base + s * rel_stage, rel_blk + static_cast<int64_t>(chunk) * CC * DB,
                             static_cast<uint32_t>(CC * DB * 8), &full[s]);
        }
        __syncwarp();
    };

    const int dist = NS > 2 ? NS - 2 : 1;   // prefetch distance in chunks (measured: 1 and 2 equal, 3 slower)
    int2 meta[CPW], nxt[CPW];
    load_meta(0, meta);
    for (int k = 0; k < dist && k < p.nchunks; ++k) {
        load_meta(k + 1, nxt);
        produce(k, meta);
#pragma unroll
        for (int i = 0; i < CPW; ++i)
            meta[i] = nxt[i];
    }

    uint32_t P[W][NP], T[W][BP_NT];
#pragma unroll
    for (int j = 0; j < W; ++j) {
#pragma unroll
        for (int k = 0; k < NP; ++k)
            P[j][k] = 0;
#pragma unroll
        for (int k = 0; k < BP_NT; ++k)
            T[j][k] = 0;
    }

    for (int chunk = 0; chunk < p.nchunks; ++chunk) {
        const int s = chunk % NS;
        if (chunk + dist < p.nchunks) {
            load_meta(chunk + dist + 1, nxt);
            produce(chunk + dist, meta);
#pragma unroll
            for (int i = 0; i < CPW; ++i)
                meta[i] = nxt[i];
        }
        mbar_wait(&full[s], (chunk / NS) & 1);

        BpShared sh;
        sh.lane_base = raw_base + s * raw_stage + lane * (W * 8);
        sh.rel = reinterpret_cast<const uint2 *>(rel_base + s * rel_stage) + warp;
        stage_steps(std::make_integer_sequence<int, CC>{}, sh, P, T);
#pragma unroll
        for (int j = 0; j < W; ++j)
            csa_flush<BP_WSUM * CC, 0, false>(P[j], T[j], 0u);

        __syncwarp();
        if (lane == 0)
            mbar_arrive(&empty[s]);
    }

    // ---- epilogue: thread owns samples t0 + 32*(5*lane + j) + [0, 32) of DM slot `warp`
    const int d = blk * DB + warp;
    if (d >= p.ndm)
        return;
    const int esize = (p.out_code == DD_OUT_U16) ? 2 : 4;
    uint8_t *orow = p.out + static_cast<int64_t>(beam) * p.out_beam_stride + static_cast<int64_t>(d) * p.nsamps * esize;
#pragma unroll
    for (int j = 0; j < W; ++j) {
        // 16x16 bit-matrix transpose of both half-words at once: R[k] = {sum of sample 16+k, sum of sample k}
        uint32_t R[16];
#pragma unroll
        for (int k = 0; k < 16; ++k)
            R[k] = k < NP ? P[j][k] : 0u;
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
        const int64_t tunit = t0 + 32 * (W * lane + j);
#pragma unroll
        for (int h = 0; h < 8; ++h) {   // samples 4h .. 4h+3 of the unit
            const int64_t t = tunit + 4 * h;
            if (t >= p.nsamps)
                continue;
            uint32_t q[4];
#pragma unroll
            for (int k = 0; k < 4; ++k)
                q[k] = h < 4 ? (R[4 * h + k] & 0xFFFFu) : (R[4 * (h - 4) + k] >> 16);
            const bool whole = p.vec_ok && (t + 4 <= p.nsamps);
            if (p.out_code == DD_OUT_F32) {
                float *o = reinterpret_cast<float *>(orow) + t;
                if (whole) {
                    *reinterpret_cast<float4 *>(o) = make_float4(__uint2float_rn(q[0]), __uint2float_rn(q[1]),
                                                                 __uint2float_rn(q[2]), __uint2float_rn(q[3]));
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
    }
}

}  // namespace

// Two launches: the bit-plane transpose of the rows the tiles will read, then the dedispersion kernel.
cudaError_t launch_variant3(dd_plan_s *plan, const KernelParams &kp_in, cudaStream_t stream)
{
    if (plan->nbits != 2 || !plan->var.bitplane || plan->cc != BP_CC)
        return cudaErrorInvalidValue;
    KernelParams kp = kp_in;
    // bytes of every row the tiles can touch, rounded to the 16-byte conversion unit
    int64_t conv = ((static_cast<int64_t>(kp.ntiles - 1) * BP_TB + plan->max_span_end) * 2 + 7) / 8;
    conv = (conv + 15) / 16 * 16;
    if (conv > kp.in_row_bytes)
        conv = kp.in_row_bytes / 16 * 16;
    const size_t need = static_cast<size_t>(kp.nbeams) * kp.nchans * static_cast<size_t>(conv);
    cudaError_t e;
    if (plan->work_bytes < need) {
        if (plan->d_work)
            cudaFree(plan->d_work);   // synchronises with any kernel still reading the old buffer
        plan->d_work = nullptr;
        plan->work_bytes = 0;
        if ((e = cudaMalloc(&plan->d_work, need)) != cudaSuccess)
            return e;
        plan->work_bytes = need;
    }
    const int chunks = static_cast<int>(conv / 16);
    dd_to_bitplanes2<<<dim3((chunks + 255) / 256, kp.nchans, kp.nbeams), 256, 0, stream>>>(
        kp.in, kp.in_stride, kp.in_beam_stride, static_cast<uint8_t *>(plan->d_work), conv,
        static_cast<int64_t>(kp.nchans) * conv, chunks);
    if ((e = cudaGetLastError()) != cudaSuccess)
        return e;
    if (plan->prof_mid)
        cudaEventRecord(static_cast<cudaEvent_t>(plan->prof_mid), stream);
    kp.in = static_cast<const uint8_t *>(plan->d_work);
    kp.in_stride = conv;
    kp.in_row_bytes = conv;
    kp.in_beam_stride = static_cast<int64_t>(kp.nchans) * conv;

    e = cudaFuncSetAttribute(dd_direct_bp2, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes));
    if (e != cudaSuccess)
        return e;
    const int64_t ctas = static_cast<int64_t>(kp.nblk) * kp.ntiles * kp.nbeams;
    if (ctas <= 0 || ctas > 0x7FFFFFFFLL)
        return cudaErrorInvalidConfiguration;
    dd_direct_bp2<<<dim3(static_cast<unsigned>(ctas)), dim3(BP_NWARPS * 32), plan->smem_bytes, stream>>>(kp);
    return cudaGetLastError();
}

}  // namespace dd
