// jp_tof_win.cuh -- the table of TOF window weights shared by the TOF sinogram kernels (jp_tof_sino.cu: per-LOR
// sliding window; jp_tof_sino_tile.cu: track tiles of a sinogram plan).
//
// PAPER.md:35, :78 (reading A10): in bin coordinates s = tau / W + (n_tofbins - 1) / 2 (bin k centred at s = k) the
// weight of bin k is G(k - s),
//
//     G(x) = 1/2 [E((x + 1/2) W) - E((x - 1/2) W)],   E(y) = erf(clamp(y, -m, m) / (sigma sqrt2)),
//
// with support |x| < R = m / W + 1/2: at most NBW = ceil(2R) consecutive bins starting at base = ceil(s - R).  With
// phi = base - (s - R) in [0, 1) the arguments of ALL bins of the window are n + phi - R: one row of a table
// T[phi][n] = G(n + phi - R) (kGK rows per unit of phi, (value, slope) pairs, built in float64) gives every weight of
// a plane step with NBW/2 128-bit shared-memory loads and NBW FMAs.
#pragma once
#include "jp_internal.h"

namespace jp {
namespace tofwin {

#ifndef JP_SINO_GK
#define JP_SINO_GK 512
#endif
constexpr int kGK = JP_SINO_GK; // table rows per unit of phi

struct GTab {
    const float2 *tab; // device, (kGK + 2) rows of NBW (value, slope) pairs
    float cbR;         // (n_tofbins - 1) / 2 - R
    float inv_w;       // 1 / W
};

static __global__ void k_tof_gtab(float2 *tab, int nbw, double R, double W, double m, double isc)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (kGK + 2) * nbw) return;
    const int r = e / nbw, n = e - r * nbw;
    auto E = [&](double y) { return erf(fmin(fmax(y, -m), m) * isc); };
    auto G = [&](double x) { return 0.5 * (E((x + 0.5) * W) - E((x - 0.5) * W)); };
    const double x0 = (double)n + (double)r / (double)kGK - R;
    const double g0 = G(x0), g1 = G(x0 + 1.0 / (double)kGK);
    tab[e] = make_float2((float)g0, (float)(g1 - g0));
}

template <int OFF>
__device__ __forceinline__ float4 lds_quad(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "r"(addr), "n"(OFF)
                 : "memory");
    return v;
}

// weights of the NBW window bins from one table row: w[n] = T[n] + f D[n]
template <int NBW, int N>
__device__ __forceinline__ void load_weights(uint32_t row, float f, float (&w)[NBW])
{
    if constexpr (N < NBW) {
        const float4 v = lds_quad<N * 8>(row);
        w[N] = fmaf(f, v.y, v.x);
        w[N + 1] = fmaf(f, v.w, v.z);
        load_weights<NBW, N + 2>(row, f, w);
    }
}

// number of window bins the kernels are compiled for (0: TOF kernel wider than any of them); R = m / W + 1/2
static inline int window_bins(const Tof &t, double *R_out)
{
    const double m = (double)t.nsig * (double)t.sigma;
    const double R = m / (double)t.width + 0.5;
    *R_out = R;
    const int nb = (int)ceil(2.0 * R);
    const int sizes[] = {4, 6, 8, 12};
    for (int s : sizes)
        if (nb <= s) return s;
    return 0;
}

// stream-ordered table for TOF parameters t; *nbw = 0 and cudaErrorNotSupported when the window is too wide
static inline cudaError_t gtab_create(const Tof &t, cudaStream_t st, GTab *out, int *nbw_out)
{
    double R;
    const int nbw = window_bins(t, &R);
    *nbw_out = nbw;
    out->tab = nullptr;
    if (!nbw) return cudaErrorNotSupported;
    float2 *tab = nullptr;
    const int ne = (kGK + 2) * nbw;
    cudaError_t e = cudaMallocAsync((void **)&tab, sizeof(float2) * ne, st);
    if (e != cudaSuccess) return e;
    const double m = (double)t.nsig * (double)t.sigma;
    k_tof_gtab<<<(ne + 255) / 256, 256, 0, st>>>(tab, nbw, R, (double)t.width, m, 1.0 / ((double)t.sigma * 1.4142135623730951));
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        cudaFreeAsync(tab, st);
        return e;
    }
    out->tab = tab;
    out->cbR = (float)(0.5 * (double)(t.nbins - 1) - R);
    out->inv_w = 1.f / t.width;
    return cudaSuccess;
}

static inline void gtab_destroy(GTab *gt, cudaStream_t st)
{
    if (gt->tab) cudaFreeAsync((void *)gt->tab, st);
    gt->tab = nullptr;
}

} // namespace tofwin
} // namespace jp
