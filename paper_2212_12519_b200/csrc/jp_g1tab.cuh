// jp_g1tab.cuh -- table of the TOF weight of ONE bin as a function of the distance from its centre, shared by the
// listmode line tiles (jp_lm_tile.cu) and the listmode brick kernels (jp_brick.cu).
//
// PAPER.md:35 "a Gaussian kernel ... convolved with a rectangular function ..., the difference of two error functions",
// PAPER.md:78 "truncated beyond +-3 standard deviations"; reading A10:
//   G(x) = 1/2 [E((x + 1/2) W) - E((x - 1/2) W)],  E(y) = erf(clamp(y, -m, m) / (sigma sqrt 2)),  m = n_sigmas sigma,
// x = (c - tau) / W in bin widths.  G is even with support |x| < R = m / W + 1/2.
// The table runs in the DISTANCE FROM THE SUPPORT EDGE, x' = R - |x|: the two kinks of the truncated kernel sit at
// x' = 0 and x' = 1, i.e. exactly on table nodes, so the piecewise-linear table never interpolates across one
// (tabulated in |x| the kinks fall inside an interval and the tail weights are off by up to 2.7e-6 absolute).
// Entry k = (intercept, slope) of G on x' in [k, k + 1] / kG1K, built in float64 (k_tof_g1tab, jp_lm_tile.cu).
#pragma once
#include "jp_internal.h"

namespace jp {

constexpr int kG1K = 512; // table intervals per TOF bin width

struct G1Tab {
    const float2 *tab; // device, n entries
    int n;
    float scale; // kG1K / W: mm -> table units
    float xedge; // R kG1K: table position of the support edge
};

// entries needed for this TOF kernel
inline int g1tab_entries(const Tof &t)
{
    const double R = (double)t.nsig * (double)t.sigma / (double)t.width + 0.5;
    return (int)ceil(R * kG1K) + 3;
}

// stream-ordered device scratch: the caller frees out->tab with cudaFreeAsync on the same stream
cudaError_t g1tab_create(const Tof &t, int n, cudaStream_t st, G1Tab *out);

// weight of the event's bin at table position xs = (c - tau) kG1K / W (any sign); gbase: shared-memory address of the
// table copy, biased by -(kMagicI << 3)
__device__ __forceinline__ float g1_weight(uint32_t gbase, float xedge, float xs)
{
    const float xa = fmaxf(xedge - fabsf(xs), 0.f);
    const float tt = __fadd_rd(xa, kMagic);
    const float2 v = lds_pair<0>(gbase + (__float_as_uint(tt) << 3));
    return fmaf(xa, v.y, v.x);
}

} // namespace jp
