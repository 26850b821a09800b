// jp_microbench.cu -- FP32 issue-rate microbenchmark for bench.py's roofline denominator ("the builder
// must measure it with an FMA microbenchmark").  NOT part of libjoseph_b200.so or its C ABI: build.py compiles this file
// into libjp_microbench.so, which only bench.py loads.
//
// Every thread runs 8 independent FFMA chains, 16 FFMAs per loop iteration; the caller times the launch with CUDA
// events and divides blocks x 256 x 16 x iters lane-instructions by the time.
#include <cuda_runtime.h>

namespace {
__global__ void __launch_bounds__(256) k_fma_burn(float *out, int iters, float a, float b)
{
    float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456f) out[0] = s; // never true in practice: keeps the chains alive
}
} // namespace

// enqueue blocks x 256 threads x 16 x iters FFMAs on `stream`; scratch: device, one float (not written in practice);
// returns 0 or the cudaError_t of the launch
extern "C" int jp_fma_burn(float *scratch, int blocks, int iters, void *stream)
{
    if (!scratch || blocks < 1 || iters < 1) return -1;
    k_fma_burn<<<blocks, 256, 0, (cudaStream_t)stream>>>(scratch, iters, 0.999f, 0.001f);
    return (int)cudaGetLastError();
}
