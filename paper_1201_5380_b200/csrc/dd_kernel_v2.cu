// dd_kernel_v2.cu -- variant 2: 2-bit input, nibble-lane SWAR.
//
//     D[d][t] = sum_c A[c][t + delay[d][c]]                       (eq. 3)
//
// One CTA = 32 DM trials x 1280 output samples, 16 warps; warp w owns DM slots 2w, 2w+1 over the whole
// time block; lane l owns 40 consecutive samples (W = 5 words of 8 nibble lanes).
//   stage   : per channel, the packed span [t0 + start, ...) of the DM block (time block + delay range,
//             PAPER.md:115) arrives by TMA bulk copy, double-buffered over chunks of `cc` channels;
//   unpack  : once per staged span, 16 two-bit samples -> two words of eight 4-bit lanes, natural order
//             (PAPER.md:101 shift/mask; here LOP3/SHF/PRMT);
//   add     : acc4 += word(t + delay)   8 channel-adds per 32-bit add (PAPER.md:119 bit-level
//             parallelism).  A 4-bit lane holds 5 additions of values <= 3; after every 5 channels the
//             lanes are split into two words of 8-bit lanes (17 such flushes fit: 17*15 = 255), and
//             after 17 flushes (85 channels) into 16-bit lanes (sums <= 65535 by plan construction);
//   align   : a delay is an arbitrary nibble offset: two adjacent words + one funnel shift (SHF.R);
//   store   : 16-bit lanes -> float32 / uint32 / uint16, 128-bit stores, time contiguous.
#include "dd_common.cuh"
#include "dd_kernels.cuh"

namespace dd {
namespace {

constexpr int V2_DB = 32, V2_W = 5, V2_NWARPS = 16, V2_DPT = V2_DB / V2_NWARPS, V2_TB = 32 * 8 * V2_W;
constexpr int V2_GROUP = 5;       // additions a 4-bit lane can take: floor(15 / 3)
constexpr int V2_FLUSH8 = 17;     // 4->8 bit flushes an 8-bit lane can take: floor(255 / 15)

// 16 two-bit samples (LSB first) -> 2 words of eight 4-bit lanes in natural sample order.
__device__ __forceinline__ uint2 expand2to4(uint32_t x)
{
    const uint32_t y = x >> 4;
    const uint32_t p = (x & 0x03030303u) | ((x << 2) & 0x30303030u);   // bytes (s0,s1) (s4,s5) (s8,s9) (s12,s13)
    const uint32_t q = (y & 0x03030303u) | ((y << 2) & 0x30303030u);   // bytes (s2,s3) (s6,s7) (s10,s11) (s14,s15)
    return make_uint2(__byte_perm(p, q, 0x5140), __byte_perm(p, q, 0x7362));
}

__global__ void __launch_bounds__(V2_NWARPS * 32, 1) dd_direct_v2(const KernelParams p)
{
    constexpr int DB = V2_DB, W = V2_W, DPT = V2_DPT, TB = V2_TB;
    static_assert(DPT == 2, "offset entries are fetched as one 64-bit word per channel");

    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    const int64_t cta = blockIdx.x;
    const int blk = static_cast<int>(cta % p.nblk);
    const int64_t rest = cta / p.nblk;
    const int tile = static_cast<int>(rest % p.ntiles);
    const int beam = static_cast<int>(rest / p.ntiles);
    const int64_t t0 = static_cast<int64_t>(tile) * TB;

    // shared memory carve-up (must match dd::smem_layout_bytes)
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);
    const int rel_stage = static_cast<int>(align128(static_cast<int64_t>(p.cc) * DB * 4));
    const int raw_stage = static_cast<int>(align128(static_cast<int64_t>(p.cc) * p.raw_slot));
    const int lane_stage = static_cast<int>(align128(static_cast<int64_t>(p.cc) * p.lane_slot));
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
    const uint32_t *rel_blk = static_cast<const uint32_t *>(p.rel) + static_cast<int64_t>(blk) * p.nchans * DB;

    // producer (warp 0): lane i stages channels chunk*cc + i, + i + 32; lane 0 also stages the offsets
    auto produce = [&](int chunk) {
        const int s = chunk & 1;
        const int nch = min(p.cc, p.nchans - chunk * p.cc);
        uint32_t tx = (lane == 0) ? static_cast<uint32_t>(nch) * DB * 4u : 0u;
        uint32_t bytes[2] = {0, 0};
        const uint8_t *src[2] = {nullptr, nullptr};
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int cl = lane + 32 * k;
            if (cl < nch) {
                const int c = chunk * p.cc + cl;
                const int4 m = __ldg(&span_blk[c]);
                const int64_t off = ((t0 + m.x) * 2) >> 3;
                const int64_t avail = p.in_row_bytes - off;
                bytes[k] = static_cast<uint32_t>(m.y < avail ? m.y : avail);
                src[k] = in_beam + static_cast<int64_t>(m.z) * p.in_stride + off;
                tx += bytes[k];
            }
        }
        mbar_arrive_expect_tx(&full[s], tx);
#pragma unroll
        for (int k = 0; k < 2; ++k)
            if (bytes[k])
                tma_bulk_g2s(raw_base + s * raw_stage + (lane + 32 * k) * p.raw_slot, src[k], bytes[k], &full[s]);
        if (lane == 0)
            tma_bulk_g2s(rel_base + s * rel_stage, rel_blk + static_cast<int64_t>(chunk) * p.cc * DB,
                         static_cast<uint32_t>(nch) * DB * 4u, &full[s]);
    };

    if (warp == 0)
        produce(0);

    uint32_t acc8[DPT][2 * W];    // 8-bit lanes: [2j] even samples of word j, [2j+1] odd samples
    uint32_t acc16[DPT][4 * W];   // 16-bit lanes: [4j+0] samples 0,4  [4j+1] 2,6  [4j+2] 1,5  [4j+3] 3,7 of word j
#pragma unroll
    for (int i = 0; i < DPT; ++i) {
#pragma unroll
        for (int j = 0; j < 2 * W; ++j)
            acc8[i][j] = 0;
#pragma unroll
        for (int j = 0; j < 4 * W; ++j)
            acc16[i][j] = 0;
    }

    auto flush8 = [&]() {
#pragma unroll
        for (int i = 0; i < DPT; ++i) {
#pragma unroll
            for (int j = 0; j < 2 * W; ++j) {
                const uint32_t a = acc8[i][j];
                acc16[i][2 * j] += a & 0x00FF00FFu;
                acc16[i][2 * j + 1] += (a >> 8) & 0x00FF00FFu;
                acc8[i][j] = 0;
            }
        }
    };
    auto flush4 = [&](int i, const uint32_t(&t)[W]) {
#pragma unroll
        for (int j = 0; j < W; ++j) {
            acc8[i][2 * j] += t[j] & 0x0F0F0F0Fu;
            acc8[i][2 * j + 1] += (t[j] >> 4) & 0x0F0F0F0Fu;
        }
    };
    // one channel of one DM: W aligned words of 8 samples each, starting at nibble offset e/4 of `row`
    auto fetch = [&](const uint8_t *row, uint32_t e, uint32_t(&v)[W]) {
        const uint32_t *wp = reinterpret_cast<const uint32_t *>(row + ((e >> 5) << 2));
        uint32_t w[W + 1];
#pragma unroll
        for (int j = 0; j <= W; ++j)
            w[j] = wp[j];
#pragma unroll
        for (int j = 0; j < W; ++j)
            v[j] = __funnelshift_r(w[j], w[j + 1], e);   // shift amount = e & 31 = 4 * (offset & 7) bits
    };

    int n_flush4 = 0;
    const int lane_byte = lane * (W * 4);
    for (int chunk = 0; chunk < p.nchunks; ++chunk) {
        const int s = chunk & 1;
        mbar_wait(&full[s], (chunk >> 1) & 1);
        {   // unpack the stage: raw word i -> nibble words 2i, 2i+1 (same slot structure, twice the bytes)
            const int nwords = (p.cc * p.raw_slot) >> 2;
            const uint32_t *rw = reinterpret_cast<const uint32_t *>(raw_base + s * raw_stage);
            uint2 *lw = reinterpret_cast<uint2 *>(lanes_base + s * lane_stage);
            for (int i = tid; i < nwords; i += V2_NWARPS * 32)
                lw[i] = expand2to4(rw[i]);
        }
        __syncthreads();   // lanes[s] complete; every warp has finished chunk-1 (frees stage s^1)
        if (warp == 0 && chunk + 1 < p.nchunks)
            produce(chunk + 1);

        const uint8_t *lanes = lanes_base + s * lane_stage + lane_byte;
        const uint2 *rel_s = reinterpret_cast<const uint2 *>(rel_base + s * rel_stage) + warp;   // [cl][DB/2] pairs
        const int nch = min(p.cc, p.nchans - chunk * p.cc);
        const int ngroups = nch / V2_GROUP;

        for (int g = 0; g < ngroups; ++g) {
            uint2 e[V2_GROUP];
#pragma unroll
            for (int k = 0; k < V2_GROUP; ++k)
                e[k] = rel_s[(g * V2_GROUP + k) * (DB / 2)];
#pragma unroll
            for (int i = 0; i < DPT; ++i) {
                uint32_t t[W], v[W];
#pragma unroll
                for (int k = 0; k < V2_GROUP; ++k) {
                    fetch(lanes + (g * V2_GROUP + k) * p.lane_slot, i == 0 ? e[k].x : e[k].y, v);
#pragma unroll
                    for (int j = 0; j < W; ++j)
                        t[j] = (k == 0) ? v[j] : t[j] + v[j];
                }
                flush4(i, t);
            }
            if (++n_flush4 == V2_FLUSH8) {
                flush8();
                n_flush4 = 0;
            }
        }
        // leftover channels of the last chunk (nchans not a multiple of 5): one flush per channel
        for (int cl = ngroups * V2_GROUP; cl < nch; ++cl) {
            const uint2 e1 = rel_s[cl * (DB / 2)];
#pragma unroll
            for (int i = 0; i < DPT; ++i) {
                uint32_t v[W];
                fetch(lanes + cl * p.lane_slot, i == 0 ? e1.x : e1.y, v);
                flush4(i, v);
            }
            if (++n_flush4 == V2_FLUSH8) {
                flush8();
                n_flush4 = 0;
            }
        }
    }
    flush8();

    // ---- epilogue: thread owns samples t0 + lane*8W + [0, 8W) of DM slots 2*warp, 2*warp+1
    const int64_t tbase = t0 + lane * (8 * W);
    uint8_t *out_beam = p.out + static_cast<int64_t>(beam) * p.out_beam_stride;
#pragma unroll
    for (int i = 0; i < DPT; ++i) {
        const int d = blk * DB + warp * DPT + i;
        if (d >= p.ndm)
            continue;
        uint8_t *orow = out_beam + static_cast<int64_t>(d) * p.out_dm_stride;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const uint32_t a = acc16[i][4 * j], b = acc16[i][4 * j + 1], c = acc16[i][4 * j + 2], dd_ = acc16[i][4 * j + 3];
            const uint32_t sv[8] = {a & 0xFFFFu, c & 0xFFFFu, b & 0xFFFFu, dd_ & 0xFFFFu, a >> 16, c >> 16, b >> 16, dd_ >> 16};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int64_t t = tbase + 8 * j + 4 * h;
                if (t >= p.nsamps)
                    continue;
                const uint32_t *q = sv + 4 * h;
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
}

}  // namespace

cudaError_t launch_variant2(const dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    if (plan->nbits != 2 || plan->final32)
        return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(dd_direct_v2, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(plan->smem_bytes));
    if (e != cudaSuccess)
        return e;
    const int64_t ctas = static_cast<int64_t>(kp.nblk) * kp.ntiles * kp.nbeams;
    if (ctas <= 0 || ctas > 0x7FFFFFFFLL)
        return cudaErrorInvalidConfiguration;
    dd_direct_v2<<<dim3(static_cast<unsigned>(ctas)), dim3(V2_NWARPS * 32), plan->smem_bytes, stream>>>(kp);
    return cudaGetLastError();
}

}  // namespace dd
