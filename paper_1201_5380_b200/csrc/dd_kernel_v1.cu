// dd_kernel_v1.cu -- variant 1 (generic 2/4/8-bit) of the hand-written sm_100a kernel for the direct dedispersion transform
//     D[d][t] = sum_c A[c][t + delay[d][c]]                       (eq. 3)
//
// Structure of one CTA (variant 1):
//   * owns a (DM block DB=32) x (time block TB=640) output tile, loops over channels sequentially
//     (PAPER.md:83 finding (i): parallel over d and t, sequential over nu);
//   * stages, per channel, the packed input span the tile needs -- the time block plus the DM block's
//     delay range ("additional time samples ... to allow for differences in delay across a
//     block") -- into shared memory with TMA bulk copies (cp.async.bulk + mbarrier complete_tx),
//     double-buffered over chunks of `cc` channels;
//   * unpacks 2/4-bit samples once per staged span into byte lanes (PAPER.md:101 shift/mask, here PRMT/LOP3);
//   * every thread keeps DPW DM trials x 4W consecutive samples in packed register accumulators: 4 x 8-bit
//     lanes per 32-bit add for 2/4-bit input, 2 x 16-bit lanes for 8-bit input (the bit-level
//     parallelism of PAPER.md:119), flushed into wider lanes before they can overflow
//     (85 / 17 / 257 additions for 2 / 4 / 8-bit samples);
//   * converts and writes each DM row's samples with 128-bit stores, time contiguous.
#include "dd_common.cuh"
#include "dd_kernels.cuh"

namespace dd {
namespace {

// ------------------------------------------------------------------------------------------ unpacking
// 16 two-bit samples (LSB first) -> 16 byte lanes.
__device__ __forceinline__ uint4 expand2(uint32_t x)
{
    uint32_t r[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t b = (x >> (8 * k)) & 0xFFu;
        r[k] = (b | (b << 6) | (b << 12) | (b << 18)) & 0x03030303u;
    }
    return make_uint4(r[0], r[1], r[2], r[3]);
}
// 8 four-bit samples (LSB first) -> 8 byte lanes.
__device__ __forceinline__ uint2 expand4(uint32_t x)
{
    const uint32_t e = x & 0x0F0F0F0Fu, o = (x >> 4) & 0x0F0F0F0Fu;
    return make_uint2(__byte_perm(e, o, 0x5140), __byte_perm(e, o, 0x7362));
}

// ------------------------------------------------------------------------------------------ the kernel
constexpr int V1_DB = 32, V1_W = 5, V1_NWARPS = 8, V1_DPW = V1_DB / V1_NWARPS, V1_TB = 128 * V1_W;

template <int NBITS, bool FINAL32>
__global__ void __launch_bounds__(V1_NWARPS * 32, 1) dd_direct_v1(const KernelParams p)
{
    constexpr int DB = V1_DB, W = V1_W, DPW = V1_DPW, TB = V1_TB;
    constexpr int L0N = (NBITS == 8) ? 2 * W : W;                       // narrow accumulator registers per DM
    constexpr bool HAS_WIDE = FINAL32 || NBITS < 8;                       // a second, wider accumulator level
    constexpr int WIDE_N = FINAL32 ? 4 * W : (NBITS < 8 ? 2 * W : 1);
    constexpr int FLUSH = (NBITS == 2) ? 85 : (NBITS == 4 ? 17 : 257);   // (2^lane-1)/(2^nbits-1)

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
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    const int64_t rel_stage = align128(static_cast<int64_t>(p.cc) * DB * 2);
    const int64_t raw_stage = align128(static_cast<int64_t>(p.cc) * p.raw_slot);
    uint8_t *rel_base = smem + 128;
    uint8_t *raw_base = rel_base + 2 * rel_stage;
    uint8_t *lanes_base = raw_base + 2 * raw_stage;

    if (tid == 0) {
        mbar_init(&full[0], 32);
        mbar_init(&full[1], 32);
        mbar_fence_init();
    }
    __syncthreads();

    const uint8_t *in_beam = p.in + static_cast<int64_t>(beam) * p.in_beam_stride;
    const int4 *span_blk = p.span + static_cast<int64_t>(blk) * p.nchans;
    const uint16_t *rel_blk = static_cast<const uint16_t *>(p.rel) + static_cast<int64_t>(blk) * p.nchans * DB;

    // producer: warp 0, lane i stages channel (chunk*cc + i); lane 0 also stages the chunk's offsets
    auto produce = [&](int chunk) {
        const int s = chunk & 1;
        const int c = chunk * p.cc + lane;
        uint32_t bytes = 0;
        const uint8_t *src = nullptr;
        if (lane < p.cc && c < p.nchans) {
            const int4 m = __ldg(&span_blk[c]);
            const int64_t off = ((t0 + m.x) * NBITS) >> 3;
            const int64_t avail = p.in_row_bytes - off;
            bytes = static_cast<uint32_t>(m.y < avail ? m.y : avail);
            src = in_beam + static_cast<int64_t>(m.z) * p.in_stride + off;
        }
        const int nch = min(p.cc, p.nchans - chunk * p.cc);
        const uint32_t rel_bytes = static_cast<uint32_t>(nch) * DB * 2;
        mbar_arrive_expect_tx(&full[s], bytes + (lane == 0 ? rel_bytes : 0u));
        if (bytes)
            tma_bulk_g2s(raw_base + s * raw_stage + static_cast<int64_t>(lane) * p.raw_slot, src, bytes, &full[s]);
        if (lane == 0)
            tma_bulk_g2s(rel_base + s * rel_stage, rel_blk + static_cast<int64_t>(chunk) * p.cc * DB, rel_bytes, &full[s]);
    };

    if (warp == 0) {
        produce(0);
        if (p.nchunks > 1)
            produce(1);
    }

    uint32_t acc0[DPW][L0N];
    uint32_t accw[DPW][WIDE_N];
#pragma unroll
    for (int i = 0; i < DPW; ++i) {
#pragma unroll
        for (int j = 0; j < L0N; ++j)
            acc0[i][j] = 0;
#pragma unroll
        for (int j = 0; j < WIDE_N; ++j)
            accw[i][j] = 0;
    }

    auto flush = [&]() {
        if constexpr (HAS_WIDE) {
#pragma unroll
            for (int i = 0; i < DPW; ++i) {
#pragma unroll
                for (int j = 0; j < L0N; ++j) {
                    const uint32_t a = acc0[i][j];
                    if constexpr (NBITS < 8 && !FINAL32) {          // bytes -> 16-bit lanes (even / odd samples)
                        accw[i][2 * j] += __byte_perm(a, 0, 0x4240);
                        accw[i][2 * j + 1] += __byte_perm(a, 0, 0x4341);
                    } else if constexpr (NBITS < 8) {              // bytes -> 32-bit
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            accw[i][4 * j + k] += (a >> (8 * k)) & 0xFFu;
                    } else {                                        // 16-bit lanes -> 32-bit
                        accw[i][2 * j] += a & 0xFFFFu;
                        accw[i][2 * j + 1] += a >> 16;
                    }
                    acc0[i][j] = 0;
                }
            }
        }
    };

    int since_flush = 0;
    for (int chunk = 0; chunk < p.nchunks; ++chunk) {
        const int s = chunk & 1;
        mbar_wait(&full[s], (chunk >> 1) & 1);
        const uint8_t *raw = raw_base + s * raw_stage;
        const uint8_t *lanes = raw;
        int lane_slot = p.raw_slot;
        if constexpr (NBITS < 8) {
            // unpack the whole stage: raw word i -> 16 (2-bit) or 8 (4-bit) byte lanes, same slot structure
            const int nwords = (p.cc * p.raw_slot) >> 2;
            const uint32_t *rw = reinterpret_cast<const uint32_t *>(raw);
            if constexpr (NBITS == 2) {
                uint4 *lw = reinterpret_cast<uint4 *>(lanes_base);
                for (int i = tid; i < nwords; i += blockDim.x)
                    lw[i] = expand2(rw[i]);
            } else {
                uint2 *lw = reinterpret_cast<uint2 *>(lanes_base);
                for (int i = tid; i < nwords; i += blockDim.x)
                    lw[i] = expand4(rw[i]);
            }
            __syncthreads();
            lanes = lanes_base;
            lane_slot = p.lane_slot;
        }
        const uint16_t *rel_s = reinterpret_cast<const uint16_t *>(rel_base + s * rel_stage);
        const int nch = min(p.cc, p.nchans - chunk * p.cc);

        for (int cl = 0; cl < nch; ++cl) {
            const uint32_t *row = reinterpret_cast<const uint32_t *>(lanes + static_cast<int64_t>(cl) * lane_slot) + lane * W;
            const uint2 r4 = *reinterpret_cast<const uint2 *>(rel_s + cl * DB + warp * DPW);   // DPW == 4 offsets
            const uint32_t offs[4] = {r4.x & 0xFFFFu, r4.x >> 16, r4.y & 0xFFFFu, r4.y >> 16};
#pragma unroll
            for (int i = 0; i < DPW; ++i) {
                const uint32_t off = offs[i];
                const uint32_t *wp = row + (off >> 2);
                const uint32_t sh = (off & 3u) * 8u;
                uint32_t w[W + 1];
#pragma unroll
                for (int j = 0; j <= W; ++j)
                    w[j] = wp[j];
#pragma unroll
                for (int j = 0; j < W; ++j) {
                    const uint32_t v = __funnelshift_r(w[j], w[j + 1], sh);   // 4 consecutive samples, one per byte
                    if constexpr (NBITS < 8) {
                        acc0[i][j] += v;
                    } else {
                        acc0[i][2 * j] += __byte_perm(v, 0, 0x4140);
                        acc0[i][2 * j + 1] += __byte_perm(v, 0, 0x4342);
                    }
                }
            }
            if constexpr (HAS_WIDE) {
                if (++since_flush == FLUSH) {
                    flush();
                    since_flush = 0;
                }
            }
        }
        __syncthreads();   // every warp is done with this stage's lanes, offsets and packed bytes
        if (warp == 0 && chunk + 2 < p.nchunks)
            produce(chunk + 2);
    }
    flush();

    // ---- epilogue: convert and store.  Thread owns samples t0 + lane*4W + [0, 4W) of DPW DM rows.
    const int64_t tbase = t0 + lane * (4 * W);
    uint8_t *out_beam = p.out + static_cast<int64_t>(beam) * p.out_beam_stride;
#pragma unroll
    for (int i = 0; i < DPW; ++i) {
        const int d = blk * DB + warp * DPW + i;
        if (d >= p.ndm)
            continue;
        uint8_t *orow = out_beam + static_cast<int64_t>(d) * p.out_dm_stride;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int64_t t = tbase + 4 * j;
            if (t >= p.nsamps)
                continue;
            uint32_t sv[4];
            if constexpr (FINAL32) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    sv[k] = accw[i][4 * j + k];
            } else if constexpr (NBITS < 8) {
                const uint32_t e = accw[i][2 * j], o = accw[i][2 * j + 1];
                sv[0] = e & 0xFFFFu; sv[1] = o & 0xFFFFu; sv[2] = e >> 16; sv[3] = o >> 16;
            } else {
                const uint32_t lo = acc0[i][2 * j], hi = acc0[i][2 * j + 1];
                sv[0] = lo & 0xFFFFu; sv[1] = lo >> 16; sv[2] = hi & 0xFFFFu; sv[3] = hi >> 16;
            }
            const bool whole = p.vec_ok && (t + 4 <= p.nsamps);
            if (p.out_code == DD_OUT_F32) {
                float *o = reinterpret_cast<float *>(orow) + t;
                if (whole) {
                    *reinterpret_cast<float4 *>(o) = make_float4(__uint2float_rn(sv[0]), __uint2float_rn(sv[1]),
                                                                 __uint2float_rn(sv[2]), __uint2float_rn(sv[3]));
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if (t + k < p.nsamps)
                            o[k] = __uint2float_rn(sv[k]);
                }
            } else if (p.out_code == DD_OUT_U32) {
                uint32_t *o = reinterpret_cast<uint32_t *>(orow) + t;
                if (whole) {
                    *reinterpret_cast<uint4 *>(o) = make_uint4(sv[0], sv[1], sv[2], sv[3]);
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if (t + k < p.nsamps)
                            o[k] = sv[k];
                }
            } else {
                uint16_t *o = reinterpret_cast<uint16_t *>(orow) + t;
                if (whole) {
                    *reinterpret_cast<uint2 *>(o) = make_uint2(sv[0] | (sv[1] << 16), sv[2] | (sv[3] << 16));
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if (t + k < p.nsamps)
                            o[k] = static_cast<uint16_t>(sv[k]);
                }
            }
        }
    }
}

template <int NBITS, bool FINAL32>
cudaError_t launch_v1(const dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    auto kern = dd_direct_v1<NBITS, FINAL32>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(plan->smem_bytes));
    if (e != cudaSuccess)
        return e;
    const int64_t ctas = static_cast<int64_t>(kp.nblk) * kp.ntiles * kp.nbeams;
    if (ctas <= 0 || ctas > 0x7FFFFFFFLL)
        return cudaErrorInvalidConfiguration;
    kern<<<dim3(static_cast<unsigned>(ctas)), dim3(plan->var.threads), plan->smem_bytes, stream>>>(kp);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_variant1(const dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    switch (plan->nbits) {
    case 2:
        return plan->final32 ? launch_v1<2, true>(plan, kp, stream) : launch_v1<2, false>(plan, kp, stream);
    case 4:
        return plan->final32 ? launch_v1<4, true>(plan, kp, stream) : launch_v1<4, false>(plan, kp, stream);
    case 8:
        return plan->final32 ? launch_v1<8, true>(plan, kp, stream) : launch_v1<8, false>(plan, kp, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace dd
