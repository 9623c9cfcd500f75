// peak.cu -- roofline denominators measured on the device the library runs on (build step 1).
//   which = 0 : FP32 FFMA      (lane-FMAs per second, the BASELINE.json "FP32 FMA roofline")
//   which = 1 : VIADDMNMX.S32  (lane add-min per second: the integer-ALU ceiling of the int32 kernel's inner op)
//   which = 2 : VIADDMNMX.U16x2 (lane instructions per second; each one is TWO 16-bit add-mins: enumerate16.cu)
//   which = 3 : the instruction MIX of DESIGN.md 5.2 -- one fused VIADDMNMX.U16x2 (2 add-mins) per split group
//               IMAD + IMAD + VIMNMX3.U16x2 (4 add-mins): lane ADD-MINS per second. This is the measured counterpart
//               of the derived bound "192 add-mins per clock per SM" (ALU pipe 16 lanes/clk and one issue slot per
//               clock per sub-partition, a = b = 1/4).
// Each thread runs 8 independent dependency chains, 16 deep per loop trip; nothing touches memory inside the loop.
#include "common.cuh"

namespace ising {

template <int WHICH>
__global__ void __launch_bounds__(256) peak_kernel(int iters, float fa, float fb, int ia, int ib, int* sink)
{
    float f[8];
    int v[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) { f[c] = threadIdx.x * 1e-3f + c; v[c] = (int)threadIdx.x - 7 * c; }
    // per-thread addends of the split group (vector registers, as in the kernel: the adds must issue as IMAD)
    const unsigned wa = (unsigned)ia + (threadIdx.x & 1u), wb = (unsigned)ib + (threadIdx.x & 2u);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                if (WHICH == 0) f[c] = fmaf(f[c], fa, fb);
                else if (WHICH == 1) v[c] = __viaddmin_s32(v[c], ia, ib);
                else if (WHICH == 2) v[c] = (int)__viaddmin_u16x2((unsigned)v[c], (unsigned)ia, (unsigned)ib);
                else {
                    // fused group, then split group: two packed sums as 32-bit adds on the FMA pipe (IMAD x*1+y),
                    // one VIMNMX3.U16x2 for the minimum of both and the running minimum
                    unsigned x = __viaddmin_u16x2((unsigned)v[c], (unsigned)ia, (unsigned)ib), a, b;
                    asm("mad.lo.u32 %0, %1, 1, %2;" : "=r"(a) : "r"(x), "r"(wa));
                    asm("mad.lo.u32 %0, %1, 1, %2;" : "=r"(b) : "r"(x), "r"(wb));
                    v[c] = (int)__vimin3_u16x2(x, a, b);
                }
            }
        }
    }
    float fs = 0.f;
    int vs = 0;
#pragma unroll
    for (int c = 0; c < 8; ++c) { fs += f[c]; vs += v[c]; }
    if (fs == 123.456f || vs == 0x7ffffff1) *sink = vs;      // keep the chains alive
}

double run_fma_peak(double ms_target, cudaStream_t st, int which)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1.0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1.0;
    int* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(int)) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    auto launch = [&](int iters) {
        if (which == 0) peak_kernel<0><<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, 1, 1 << 30, sink);
        else if (which == 1) peak_kernel<1><<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, 1, 1 << 30, sink);
        else if (which == 2) peak_kernel<2><<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, 0x00010001, 0x7fff7fff, sink);
        else peak_kernel<3><<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, 0x00010001, 0x00020003, sink);
    };
    auto timed = [&](int iters) -> double {
        cudaEventRecord(e0, st);
        launch(iters);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) return -1.0;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        return ms;
    };
    double result = -1.0;
    launch(64);                                   // warm-up (module load, clocks)
    double ms = timed(2048);
    if (ms > 0.0) {
        if (ms_target < 1.0) ms_target = 1.0;
        long long iters = (long long)(2048.0 * ms_target / ms);
        if (iters < 2048) iters = 2048;
        if (iters > 400000000ll) iters = 400000000ll;
        ms = timed((int)iters);
        // which = 3 counts add-mins: 2 (fused) + 4 (split) per chain step; the others count lane instructions
        if (ms > 0.0) result = (double)iters * 128.0 * (which == 3 ? 6.0 : 1.0) * threads * blocks / (ms * 1e-3);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return -1.0;
    return result;
}

}  // namespace ising
