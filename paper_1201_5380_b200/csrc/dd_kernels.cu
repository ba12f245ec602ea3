// dd_kernels.cu -- kernel dispatch and the integer-add throughput probe.
#include "dd_kernels.cuh"

namespace dd {
namespace {

// ------------------------------------------------------------------------------------------ ALU peak probe
// Register-resident chains r += q, q += r (cross-coupled, so that no two additions can be folded into one
// multiply-add by the compiler).  Additions are counted, not instructions.
//   mode 0: 2-input adds, ptxas picks the pipe (SASS: IADD3 on the ALU pipe and IMAD.IADD on the FMA pipe)
//   mode 1: 3-input adds (SASS: IADD3, two additions per instruction, ALU pipe only)
//   mode 2: 3-input adds interleaved 1:1 with multiply-adds by a run-time 1 (IADD3 + IMAD: both pipes,
//           three additions per instruction pair) -- the highest integer-add rate the SM sustains
template <int MODE>
__global__ void __launch_bounds__(512) int_add_probe(uint32_t *sink, uint32_t x, uint32_t y, uint32_t one, int iters)
{
    constexpr int NCH = 8;
    uint32_t r[NCH], q[NCH];
#pragma unroll
    for (int i = 0; i < NCH; ++i) {
        r[i] = threadIdx.x * 7u + i;
        q[i] = threadIdx.x * 3u + 5u * i;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
            for (int i = 0; i < NCH; ++i) {
                if (MODE == 0) {
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(r[i]) : "r"(q[i]));
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(q[i]) : "r"(r[i]));
                } else if (MODE == 1) {
                    asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(r[i]) : "r"(q[i]), "r"(x));
                    asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(q[i]) : "r"(r[i]), "r"(y));
                } else {
                    asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(r[i]) : "r"(q[i]), "r"(x));
                    asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(q[i]) : "r"(r[i]), "r"(one));
                }
            }
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < NCH; ++i)
        s ^= r[i] ^ q[i];
    if (s == 0x12345678u)
        sink[0] = s;
}

}  // namespace

cudaError_t launch_direct(dd_plan_s *plan, const KernelParams &kp, cudaStream_t stream)
{
    switch (plan->var.id) {
    case 1:
        return launch_variant1(plan, kp, stream);
    case 2:
        return launch_variant2(plan, kp, stream);
    case 3:
        return launch_variant3(plan, kp, stream);
    case 4:
        return launch_variant4(plan, kp, stream);
    case 5:
        return launch_variant5(plan, kp, stream);
    case 6:
        return launch_variant6(plan, kp, stream);
    }
    return cudaErrorInvalidValue;
}

// bit planes: transpose + transform; pair rows: transpose + (row builder + transform) per group of time tiles
int launches_per_execute(const dd_plan_s *plan)
{
    return (plan->pairs || plan->gr) ? plan->pair_launches : (plan->var.bitplane ? 2 : 1);
}

cudaError_t int_add_peak(int mode, double *adds_per_sec, cudaStream_t stream)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess)
        return e;
    uint32_t *sink = nullptr;
    e = cudaMalloc(&sink, 4);
    if (e != cudaSuccess)
        return e;
    cudaEvent_t ev0, ev1;
    cudaEventCreate(&ev0);
    cudaEventCreate(&ev1);
    const int iters = 2048, blocks = sms * 4, threads = 512;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(ev0, stream);
        if (mode == 0)
            int_add_probe<0><<<blocks, threads, 0, stream>>>(sink, 3u, 5u, 1u, iters);
        else if (mode == 1)
            int_add_probe<1><<<blocks, threads, 0, stream>>>(sink, 3u, 5u, 1u, iters);
        else
            int_add_probe<2><<<blocks, threads, 0, stream>>>(sink, 3u, 5u, 1u, iters);
        cudaEventRecord(ev1, stream);
        e = cudaEventSynchronize(ev1);
        if (e != cudaSuccess)
            break;
        float ms = 0;
        cudaEventElapsedTime(&ms, ev0, ev1);
        if (rep > 0 && ms < best_ms)
            best_ms = ms;
    }
    cudaEventDestroy(ev0);
    cudaEventDestroy(ev1);
    cudaFree(sink);
    if (e != cudaSuccess)
        return e;
    const double adds_per_step = (mode == 0) ? 2.0 : (mode == 1 ? 4.0 : 3.0);   // per chain per repetition
    const double adds = static_cast<double>(blocks) * threads * iters * 8.0 * 8.0 * adds_per_step;
    *adds_per_sec = adds / (static_cast<double>(best_ms) * 1e-3);
    return cudaSuccess;
}

}  // namespace dd
