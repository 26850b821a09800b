// jp_gauss.cu -- image-based resolution model: 3-D Gaussian smoothing of the image ("a shift-invariant
// image-based resolution model ... 3D isotropic Gaussian kernel of 4.5 mm FWHM"; 68 convolutions per
// OSEM iteration of 34 subsets -- the step that becomes the bottleneck once the projectors are fast).
// Readings R1/R2: taps exp(-(k v_a)^2 / (2 sigma^2)), |k| <= ceil(n_sigmas sigma / v_a), normalised per
// axis, zero outside the image.  The kernel is a product of three 1-D kernels, so it is applied as three passes
// (axis 2, 1, 0); every pass reads and writes the 15 MB image once from L2.  Taps are computed on the host in
// float64 and travel as kernel parameters.
#include <cmath>
#include <cstdint>

#include "jp_internal.h"

namespace jp {

namespace {

constexpr int kMaxRadius = 16;

struct Taps {
    int r;
    float w[2 * kMaxRadius + 1];
};

bool make_taps(double sigma_mm, double nsig, double v, Taps *t)
{
    const int r = (int)std::ceil(nsig * sigma_mm / v);
    if (r < 0 || r > kMaxRadius) return false;
    double g[2 * kMaxRadius + 1], sum = 0.0;
    for (int k = -r; k <= r; ++k) {
        const double x = (double)k * v / sigma_mm;
        g[k + r] = std::exp(-0.5 * x * x);
        sum += g[k + r];
    }
    t->r = r;
    for (int k = 0; k <= 2 * r; ++k) t->w[k] = (float)(g[k] / sum);
    return true;
}

// out[i] = sum_k w[k] in[i - k e_AXIS], zero outside; one thread per voxel (neighbours come from L1 / L2).
// Generic pass: any image shape.
template <int AXIS>
__global__ void __launch_bounds__(256) k_gauss_axis(const float *__restrict__ in, float *__restrict__ out, int n0, int n1,
                                                     int n2, Taps t)
{
    const int64_t i = blockIdx.x * (int64_t)256 + threadIdx.x;
    const int64_t nvox = (int64_t)n0 * n1 * n2;
    if (i >= nvox) return;
    const int i2 = (int)(i % n2);
    const int64_t q = i / n2;
    const int i1 = (int)(q % n1), i0 = (int)(q / n1);
    const int pos = AXIS == 0 ? i0 : AXIS == 1 ? i1 : i2;
    const int len = AXIS == 0 ? n0 : AXIS == 1 ? n1 : n2;
    const int64_t stride = AXIS == 0 ? (int64_t)n1 * n2 : AXIS == 1 ? n2 : 1;
    float acc = 0.f;
    for (int k = -t.r; k <= t.r; ++k) {
        const int j = pos - k;
        if ((unsigned)j < (unsigned)len) acc = fmaf(t.w[k + t.r], __ldg(in + i - k * stride), acc);
    }
    out[i] = acc;
}

// ---- fast path (n2 a multiple of 4, 16-byte aligned images, n2 <= kGZ): two kernels instead of three passes --------
// k_gauss_zy: a CTA takes one image plane i0 and kGY rows of it (+ halo): the axis-2 pass goes from global memory
// into a shared tile, the axis-1 pass out of the tile -- the intermediate image never leaves the SM.
// k_gauss_x4: axis-0 pass, four consecutive voxels of axis 2 per thread (128-bit loads, coalesced).
constexpr int kGY = 32;  // rows per CTA
constexpr int kGZ = 128; // largest n2 of the fast path

__global__ void __launch_bounds__(256) k_gauss_zy(const float *__restrict__ in, float *__restrict__ out, int n0, int n1,
                                                   int n2, Taps tz, Taps ty)
{
    extern __shared__ float tile[]; // [(kGY + 2 ry)][n2]
    const int i0 = blockIdx.y, y0 = blockIdx.x * kGY;
    const int ry = ty.r, rz = tz.r;
    const int rows = kGY + 2 * ry;
    const float *plane = in + (int64_t)i0 * n1 * n2;
    // axis-2 pass of rows y0 - ry .. y0 + kGY + ry - 1 (zero outside the image)
    for (int e = threadIdx.x; e < rows * n2; e += 256) {
        const int r = e / n2, z = e - r * n2;
        const int y = y0 - ry + r;
        float acc = 0.f;
        if ((unsigned)y < (unsigned)n1) {
            const float *row = plane + (int64_t)y * n2;
            for (int k = -rz; k <= rz; ++k) {
                const int j = z - k;
                if ((unsigned)j < (unsigned)n2) acc = fmaf(tz.w[k + rz], __ldg(row + j), acc);
            }
        }
        tile[e] = acc;
    }
    __syncthreads();
    // axis-1 pass out of the tile
    float *oplane = out + (int64_t)i0 * n1 * n2;
    for (int e = threadIdx.x; e < kGY * n2; e += 256) {
        const int r = e / n2, z = e - r * n2;
        const int y = y0 + r;
        if (y >= n1) break;
        float acc = 0.f;
        for (int k = -ry; k <= ry; ++k) acc = fmaf(ty.w[k + ry], tile[(r + ry - k) * n2 + z], acc);
        oplane[(int64_t)y * n2 + z] = acc;
    }
}

__global__ void __launch_bounds__(256) k_gauss_x4(const float4 *__restrict__ in, float4 *__restrict__ out, int n0,
                                                   int plane4 /* n1 n2 / 4 */, Taps t)
{
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= n0 * plane4) return;
    const int i0 = i / plane4;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int k = -t.r; k <= t.r; ++k) {
        const int j = i0 - k;
        if ((unsigned)j < (unsigned)n0) {
            const float4 v = __ldg(in + i - k * plane4);
            const float w = t.w[k + t.r];
            acc.x = fmaf(w, v.x, acc.x);
            acc.y = fmaf(w, v.y, acc.y);
            acc.z = fmaf(w, v.z, acc.z);
            acc.w = fmaf(w, v.w, acc.w);
        }
    }
    out[i] = acc;
}

} // namespace

// tmp: nvox floats of scratch (may not alias in / out); in may alias out.  cudaErrorInvalidValue: radius too large
cudaError_t launch_gauss3d(const float *in, float *out, float *tmp, const Geom &g, float sigma_mm, float nsig,
                           cudaStream_t st)
{
    Taps t[3];
    for (int a = 0; a < 3; ++a)
        if (!make_taps((double)sigma_mm, (double)nsig, (double)g.v[a], &t[a])) return cudaErrorInvalidValue;
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    const bool fast = (g.n[2] % 4 == 0) && g.n[2] <= kGZ && nvox < ((int64_t)1 << 31) &&
                      (((uintptr_t)in | (uintptr_t)out | (uintptr_t)tmp) % 16 == 0);
    if (fast) { // in -> tmp (axes 2 and 1 in one kernel), tmp -> out (axis 0); in may alias out
        const size_t smem = (size_t)(kGY + 2 * t[1].r) * g.n[2] * sizeof(float);
        cudaError_t e = cudaFuncSetAttribute(k_gauss_zy, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        const dim3 grid((unsigned)((g.n[1] + kGY - 1) / kGY), (unsigned)g.n[0]);
        k_gauss_zy<<<grid, 256, smem, st>>>(in, tmp, g.n[0], g.n[1], g.n[2], t[2], t[1]);
        const int plane4 = g.n[1] * g.n[2] / 4;
        k_gauss_x4<<<(unsigned)(((int64_t)g.n[0] * plane4 + 255) / 256), 256, 0, st>>>(
            reinterpret_cast<const float4 *>(tmp), reinterpret_cast<float4 *>(out), g.n[0], plane4, t[0]);
        return cudaGetLastError();
    }
    const unsigned grid = (unsigned)((nvox + 255) / 256);
    // in -> out (axis 2), out -> tmp (axis 1), tmp -> out (axis 0); "in" is dead after the first pass
    if (in == out) {
        k_gauss_axis<2><<<grid, 256, 0, st>>>(in, tmp, g.n[0], g.n[1], g.n[2], t[2]);
        k_gauss_axis<1><<<grid, 256, 0, st>>>(tmp, out, g.n[0], g.n[1], g.n[2], t[1]);
        cudaError_t e = cudaMemcpyAsync(tmp, out, sizeof(float) * (size_t)nvox, cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return e;
        k_gauss_axis<0><<<grid, 256, 0, st>>>(tmp, out, g.n[0], g.n[1], g.n[2], t[0]);
    } else {
        k_gauss_axis<2><<<grid, 256, 0, st>>>(in, out, g.n[0], g.n[1], g.n[2], t[2]);
        k_gauss_axis<1><<<grid, 256, 0, st>>>(out, tmp, g.n[0], g.n[1], g.n[2], t[1]);
        k_gauss_axis<0><<<grid, 256, 0, st>>>(tmp, out, g.n[0], g.n[1], g.n[2], t[0]);
    }
    return cudaGetLastError();
}

// a += b; b = 0
__global__ void k_add_clear(float *__restrict__ a, float *__restrict__ b, int64_t n)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    a[i] += b[i];
    b[i] = 0.f;
}

cudaError_t launch_add_clear(float *a, float *b, int64_t n, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_add_clear<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, b, n);
    return cudaGetLastError();
}

} // namespace jp
