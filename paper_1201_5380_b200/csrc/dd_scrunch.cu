// dd_scrunch.cu -- time-scrunching: "reduce the time resolution by a factor of two ... by adding
// adjacent pairs of time samples", on packed rows:  out[c][t] = in[c][2t] + in[c][2t+1].
//
// The sums of two n-bit samples need n+1 bits; the output is packed at the next width the transform kernels read
// (2 -> 4, 2 -> 8, 4 -> 8 bits), so that the scrunched series can go straight into a plan made with 2 dt.  Samples
// are LSB first (reading R9), hence the even samples of a word are its even fields and one masked add of the word
// and its shifted copy produces all pair sums at once (shift, mask, several samples per add).
// HBM-bound: every input byte is read once, every output byte written once; one thread handles 16 input bytes.
#include "dd_kernels.cuh"

namespace dd {
namespace {

// pair sums of the 2-bit (4-bit) fields of x, each in a field of twice the width, order kept
__device__ __forceinline__ uint32_t pairs2(uint32_t x) { return (x & 0x33333333u) + ((x >> 2) & 0x33333333u); }
__device__ __forceinline__ uint32_t pairs4(uint32_t x) { return (x & 0x0F0F0F0Fu) + ((x >> 4) & 0x0F0F0F0Fu); }
// the four low (high) nibbles of y -> four bytes
__device__ __forceinline__ uint32_t nib_lo(uint32_t y)
{
    return (y & 0xFu) | ((y & 0xF0u) << 4) | ((y & 0xF00u) << 8) | ((y & 0xF000u) << 12);
}

// pair sums of the bytes of x in 16-bit fields
__device__ __forceinline__ uint32_t pairs8(uint32_t x) { return (x & 0x00FF00FFu) + ((x >> 8) & 0x00FF00FFu); }

// Same-width scrunch (4 -> 4, 8 -> 8 bits) for rows whose pair sums are KNOWN to fit the width: the later stages of
// the scrunch cascade (dd_scrunch_set.cu), where a sample of the series at 2^k dt is at most 2^k (2^nbits - 1).
// 16 input bytes -> 8 output bytes.
template <int NB>
__global__ void __launch_bounds__(256) dd_scrunch_same_kernel(const uint8_t *__restrict__ in, int64_t in_stride,
                                                              uint8_t *__restrict__ out, int64_t out_stride, int64_t out_bytes)
{
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i * 8 >= out_bytes)
        return;
    const uint4 x = __ldg(reinterpret_cast<const uint4 *>(in + static_cast<int64_t>(blockIdx.y) * in_stride) + i);
    const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
    uint32_t h[4];   // 16 output bits per input word
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if constexpr (NB == 4) {
            const uint32_t y = pairs4(xs[k]);   // four sums, one per byte
            h[k] = (y & 0xFu) | ((y >> 4) & 0xF0u) | ((y >> 8) & 0xF00u) | ((y >> 12) & 0xF000u);
        } else {
            const uint32_t y = pairs8(xs[k]);   // two sums, one per half word
            h[k] = (y & 0xFFu) | ((y >> 8) & 0xFF00u);
        }
    }
    *reinterpret_cast<uint2 *>(out + static_cast<int64_t>(blockIdx.y) * out_stride + i * 8) =
        make_uint2(h[0] | (h[1] << 16), h[2] | (h[3] << 16));
}

template <int NIN, int NOUT>
__global__ void __launch_bounds__(256) dd_scrunch_kernel(const uint8_t *__restrict__ in, int64_t in_stride,
                                                         uint8_t *__restrict__ out, int64_t out_stride, int64_t out_bytes)
{
    // 16 input bytes -> OB output bytes
    constexpr int OB = 16 * NOUT / (2 * NIN);
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i * OB >= out_bytes)
        return;
    const uint4 x = __ldg(reinterpret_cast<const uint4 *>(in + static_cast<int64_t>(blockIdx.y) * in_stride) + i);
    uint8_t *o = out + static_cast<int64_t>(blockIdx.y) * out_stride + i * OB;
    uint32_t w[8];
    if constexpr (NIN == 2 && NOUT == 4) {
        w[0] = pairs2(x.x), w[1] = pairs2(x.y), w[2] = pairs2(x.z), w[3] = pairs2(x.w);
    } else if constexpr (NIN == 4 && NOUT == 8) {
        w[0] = pairs4(x.x), w[1] = pairs4(x.y), w[2] = pairs4(x.z), w[3] = pairs4(x.w);
    } else {   // 2 -> 8: nibble sums widened to bytes
        const uint32_t y[4] = {pairs2(x.x), pairs2(x.y), pairs2(x.z), pairs2(x.w)};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            w[2 * k] = nib_lo(y[k]);
            w[2 * k + 1] = nib_lo(y[k] >> 16);
        }
    }
    // the last thread of a row may own fewer than OB bytes (out rows are multiples of 16 bytes, OB is 16 or 32)
    const int64_t left = out_bytes - i * OB;
    reinterpret_cast<uint4 *>(o)[0] = make_uint4(w[0], w[1], w[2], w[3]);
    if (OB == 32 && left > 16)
        reinterpret_cast<uint4 *>(o)[1] = make_uint4(w[4], w[5], w[6], w[7]);
}

}  // namespace

// out_bytes: bytes of every output row to produce (a multiple of 16)
cudaError_t launch_scrunch(int nbits_in, int nbits_out, int nrows, const uint8_t *in, int64_t in_stride, uint8_t *out,
                           int64_t out_stride, int64_t out_bytes, cudaStream_t stream)
{
    const int ob = 16 * nbits_out / (2 * nbits_in);   // output bytes per thread (16 input bytes)
    const int64_t threads = (out_bytes + ob - 1) / ob;
    const dim3 grid(static_cast<unsigned>((threads + 255) / 256), static_cast<unsigned>(nrows));
    if (nbits_in == 2 && nbits_out == 4)
        dd_scrunch_kernel<2, 4><<<grid, 256, 0, stream>>>(in, in_stride, out, out_stride, out_bytes);
    else if (nbits_in == 4 && nbits_out == 8)
        dd_scrunch_kernel<4, 8><<<grid, 256, 0, stream>>>(in, in_stride, out, out_stride, out_bytes);
    else if (nbits_in == 2 && nbits_out == 8)
        dd_scrunch_kernel<2, 8><<<grid, 256, 0, stream>>>(in, in_stride, out, out_stride, out_bytes);
    else if (nbits_in == nbits_out && (nbits_in == 4 || nbits_in == 8)) {   // sums known to fit (scrunch cascade)
        const dim3 g8(static_cast<unsigned>(((out_bytes + 7) / 8 + 255) / 256), static_cast<unsigned>(nrows));
        if (nbits_in == 4)
            dd_scrunch_same_kernel<4><<<g8, 256, 0, stream>>>(in, in_stride, out, out_stride, out_bytes);
        else
            dd_scrunch_same_kernel<8><<<g8, 256, 0, stream>>>(in, in_stride, out, out_stride, out_bytes);
    } else
        return cudaErrorInvalidValue;
    return cudaGetLastError();
}

}  // namespace dd
