// jp_tof_lut.cu -- table of the truncated-Gaussian edge function E(x) = erf(min(x, m) / (sigma sqrt2)),
// x in [0, m], behind the TOF weights of all TOF kernels ("the difference of two error
// functions", :78 "truncated beyond +-3 standard deviations"; the paper itself suggests a 1-D look-up
// table for the TOF kernel).  Built in float64 once per call on the caller's stream.
#include "jp_internal.h"

namespace jp {

__global__ void k_tof_lut(float2 *tab, double m, double isc)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= kLutN) return;
    const double h = m / (double)kLutK;
    const double x0 = fmin((double)k * h, m), x1 = fmin((double)(k + 1) * h, m);
    const double e0 = erf(x0 * isc), e1 = erf(x1 * isc);
    tab[k] = make_float2((float)e0, (float)(e1 - e0));
}

cudaError_t tof_lut_create(const Tof &t, cudaStream_t st, TofLut *out)
{
    float2 *tab = nullptr;
    cudaError_t e = cudaMallocAsync((void **)&tab, sizeof(float2) * kLutN, st);
    if (e != cudaSuccess) return e;
    const double m = (double)t.nsig * (double)t.sigma;
    const double isc = 1.0 / ((double)t.sigma * 1.4142135623730951);
    k_tof_lut<<<(kLutN + 255) / 256, 256, 0, st>>>(tab, m, isc);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        cudaFreeAsync(tab, st);
        return e;
    }
    out->tab = tab;
    out->inv_h = (float)((double)kLutK / m);
    return cudaSuccess;
}

void tof_lut_destroy(TofLut *lut, cudaStream_t st)
{
    if (lut->tab) cudaFreeAsync((void *)lut->tab, st);
    lut->tab = nullptr;
}

} // namespace jp
