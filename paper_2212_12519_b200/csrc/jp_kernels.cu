// jp_kernels.cu -- generic (unplanned) Joseph kernels: one thread walks one LOR plane by plane.
//
// These are the reference-grade CUDA kernels of the library: they accept any LOR list in any order
// and need no scratch memory.  The planned / sorted kernels (jp_planned.cu) are measured against
// them.  PAPER.md:33 (Joseph), :35/:78 (TOF kernel), :43 (sinogram vs listmode TOF), :44/:46
// (exact adjoint via atomic adds).
#include "jp_internal.h"

namespace jp {

constexpr int kBlock = 128;
constexpr int kLmBlock = 256;

__device__ __forceinline__ int64_t lor_index(const Range &rg, int64_t c) { return rg.first + c * rg.stride; }
__device__ __forceinline__ int64_t io_index(const Range &rg, int64_t c)
{
    if (rg.compact) return c + rg.io_off;
    const int64_t j = lor_index(rg, c);
    return rg.perm ? (int64_t)rg.perm[j] : j;
}

// ---- principal axis only (diagnostic; bit-exact against the oracle) --------------------------------
__global__ void k_classify(Lors l, int64_t n, uint8_t *__restrict__ axis)
{
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= n) return;
    const double d0 = (double)l.xe[j] - (double)l.xs[j];
    const double d1 = (double)l.ye[j] - (double)l.ys[j];
    const double d2 = (double)l.ze[j] - (double)l.zs[j];
    axis[j] = (uint8_t)principal_axis(d0, d1, d2);
}

__global__ void k_plane_steps(Lors l, int64_t n, Geom g, unsigned long long *__restrict__ total)
{
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    unsigned long long nk = 0;
    if (j < n) {
        Ray r;
        ray_setup<false>(l, j, g, 0.f, 0.f, 0.f, r);
        nk = (unsigned long long)r.nk;
    }
    for (int o = 16; o > 0; o >>= 1) nk += __shfl_xor_sync(0xffffffffu, nk, o);
    if ((threadIdx.x & 31) == 0 && nk) atomicAdd(total, nk);
}

// plane-steps of the TOF listmode projectors: planes inside the truncated kernel of the event's own bin
__global__ void k_plane_steps_tof_lm(Lors l, const int16_t *__restrict__ tofbin, int64_t n, Geom g, Tof t,
                                     unsigned long long *__restrict__ total)
{
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    unsigned long long nk = 0;
    if (j < n) {
        const float centre = (float)tofbin[j] * t.width;
        const float reach = 0.5f * t.width + t.nsig * t.sigma;
        Ray r;
        ray_setup<true>(l, j, g, t.coff, centre - reach, centre + reach, r);
        nk = (unsigned long long)r.nk;
    }
    for (int o = 16; o > 0; o >>= 1) nk += __shfl_xor_sync(0xffffffffu, nk, o);
    if ((threadIdx.x & 31) == 0 && nk) atomicAdd(total, nk);
}

// ---- non-TOF ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock) k_fwd(Lors l, Range rg, const float *__restrict__ img, Geom g,
                                                float *__restrict__ p)
{
    const int64_t c = blockIdx.x * (int64_t)kBlock + threadIdx.x;
    if (c >= rg.count) return;
    Ray r;
    ray_setup<false>(l, lor_index(rg, c), g, 0.f, 0.f, 0.f, r);
    float acc = 0.f;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        acc += plane_value(img, r, k, cl);
    }
    p[io_index(rg, c)] = r.cf * acc;
}

__global__ void __launch_bounds__(kBlock) k_back(Lors l, Range rg, const float *__restrict__ y, Geom g,
                                                 float *__restrict__ img)
{
    const int64_t c = blockIdx.x * (int64_t)kBlock + threadIdx.x;
    if (c >= rg.count) return;
    Ray r;
    ray_setup<false>(l, lor_index(rg, c), g, 0.f, 0.f, 0.f, r);
    if (r.nk == 0) return;
    const float x = r.cf * y[io_index(rg, c)];
    if (x == 0.f) return;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        plane_scatter(img, r, k, cl, x);
    }
}

// ---- TOF sinogram ---------------------------------------------------------------------------------------
// All bins of one LOR are accumulated by one thread while it walks the planes.  The
// per-thread bin accumulators live in shared memory, bin-major with a padded row (conflict free),
// and the block's [kBlock][nbins] output tile -- contiguous in global memory -- is written (or, for
// the adjoint, read) fully coalesced.  The image is the zero-padded copy (no bounds tests, PRay).
struct BinWindow {
    int klo, khi;
    float x_lo; // position of the lower edge of bin klo relative to tau
};

__device__ __forceinline__ BinWindow bin_window(const Tof &t, float lim, float inv_w, float cb, float tau)
{
    // bins k with [c_k - W/2, c_k + W/2] meeting [tau - m, tau + m]; k = round(tau'/W + cb)
    BinWindow b;
    b.klo = max(0, (int)floorf((tau - lim) * inv_w + cb + 0.5f));
    b.khi = min(t.nbins - 1, (int)floorf((tau + lim) * inv_w + cb + 0.5f));
    b.x_lo = ((float)b.klo - cb) * t.width - 0.5f * t.width - tau;
    return b;
}

__global__ void __launch_bounds__(kBlock) k_fwd_tof_sino(Lors l, int64_t n, const float *__restrict__ pimg, Geom g,
                                                         Tof t, TofLut lut, float *__restrict__ p)
{
    extern __shared__ __align__(16) float acc[]; // [nbins][kBlock + 1], then the edge-function table
    constexpr int ld = kBlock + 1;
    float2 *lut_sm = reinterpret_cast<float2 *>(acc + ((t.nbins * ld + 3) & ~3));
    const int tid = threadIdx.x;
    const int64_t j0 = blockIdx.x * (int64_t)kBlock;
    const int64_t j = j0 + tid;
    for (int kb = 0; kb < t.nbins; ++kb) acc[kb * ld + tid] = 0.f;
    lut_load(lut, lut_sm);
    __syncthreads();
    const uint32_t lb = lut_base(lut_sm);
    if (j < n) {
        const float lim = t.nsig * t.sigma;
        const float cb = 0.5f * (float)(t.nbins - 1);
        const float inv_w = 1.f / t.width;
        const float reach = cb * t.width + 0.5f * t.width + lim;
        Ray r;
        ray_setup<true>(l, j, g, t.coff, -reach, reach, r);
        const PRay q = pray_from(r, g);
        float fk = 0.f;
        int po = q.off;
        for (int k = 0; k < q.nk; ++k) {
            const PCell cl = pray_cell(q, fk, po);
            const float val = q.cf * pray_value(pimg, q, cl);
            const float tau = fmaf(q.dtau, fk, q.tau0);
            const BinWindow bw = bin_window(t, lim, inv_w, cb, tau);
            float x = bw.x_lo;
            float e_lo = lut_E(lb, lut.inv_h, x);
            for (int kb = bw.klo; kb <= bw.khi; ++kb) {
                x += t.width;
                const float e_hi = lut_E(lb, lut.inv_h, x);
                acc[kb * ld + tid] += val * (0.5f * (e_hi - e_lo));
                e_lo = e_hi;
            }
            fk += 1.f;
            po += q.sp;
        }
    }
    __syncthreads();
    const int nvalid = (int)min((int64_t)kBlock, n - j0);
    float *out = p + j0 * t.nbins;
    for (int x = tid; x < nvalid * t.nbins; x += kBlock) {
        const int lor = x / t.nbins, kb = x - lor * t.nbins;
        out[x] = acc[kb * ld + lor];
    }
}

__global__ void __launch_bounds__(kBlock) k_back_tof_sino(Lors l, int64_t n, const float *__restrict__ y, Geom g,
                                                          Tof t, TofLut lut, float *__restrict__ pimg)
{
    extern __shared__ __align__(16) float ysm[]; // [nbins][kBlock + 1], then the edge-function table
    constexpr int ld = kBlock + 1;
    float2 *lut_sm = reinterpret_cast<float2 *>(ysm + ((t.nbins * ld + 3) & ~3));
    lut_load(lut, lut_sm);
    const int tid = threadIdx.x;
    const int64_t j0 = blockIdx.x * (int64_t)kBlock;
    const int64_t j = j0 + tid;
    const int nvalid = (int)min((int64_t)kBlock, n - j0);
    const float *in = y + j0 * t.nbins;
    for (int x = tid; x < nvalid * t.nbins; x += kBlock) {
        const int lor = x / t.nbins, kb = x - lor * t.nbins;
        ysm[kb * ld + lor] = in[x];
    }
    __syncthreads();
    if (j >= n) return;
    const uint32_t lb = lut_base(lut_sm);
    const float lim = t.nsig * t.sigma;
    const float cb = 0.5f * (float)(t.nbins - 1);
    const float inv_w = 1.f / t.width;
    const float reach = cb * t.width + 0.5f * t.width + lim;
    Ray r;
    ray_setup<true>(l, j, g, t.coff, -reach, reach, r);
    const PRay q = pray_from(r, g);
    float fk = 0.f;
    int po = q.off;
    for (int k = 0; k < q.nk; ++k) {
        const PCell cl = pray_cell(q, fk, po);
        const float tau = fmaf(q.dtau, fk, q.tau0);
        const BinWindow bw = bin_window(t, lim, inv_w, cb, tau);
        float x = bw.x_lo;
        float e_lo = lut_E(lb, lut.inv_h, x);
        float s = 0.f;
        for (int kb = bw.klo; kb <= bw.khi; ++kb) {
            x += t.width;
            const float e_hi = lut_E(lb, lut.inv_h, x);
            s = fmaf(ysm[kb * ld + tid], 0.5f * (e_hi - e_lo), s);
            e_lo = e_hi;
        }
        if (s != 0.f) pray_scatter(pimg, q, cl, q.cf * s);
        fk += 1.f;
        po += q.sp;
    }
}

// ---- TOF listmode ---------------------------------------------------------------------------------------
// Only the planes inside the truncated kernel of the event's own bin are visited.
template <int LM_MODE>
__global__ void __launch_bounds__(kLmBlock) k_fwd_tof_lm(Lors l, const int16_t *__restrict__ tofbin, Range rg,
                                                         const float *__restrict__ pimg, Geom g, Tof t,
                                                         TofLut lut, float *__restrict__ p)
{
    extern __shared__ __align__(16) float2 lut_sm[];
    lut_load(lut, lut_sm);
    __syncthreads();
    const uint32_t lb = lut_base(lut_sm);
    const int64_t c = blockIdx.x * (int64_t)kLmBlock + threadIdx.x;
    if (c >= rg.count) return;
    const int64_t j = lor_index(rg, c);
    const float half_w = 0.5f * t.width;
    const float centre = (float)tofbin[j] * t.width;
    const float reach = half_w + t.nsig * t.sigma;
    Ray r;
    ray_setup<true>(l, j, g, t.coff, centre - reach, centre + reach, r);
    const PRay q = pray_from(r, g);
    float acc = 0.f, fk = 0.f;
    int po = q.off;
    for (int k = 0; k < q.nk; ++k) {
        const PCell cl = pray_cell(q, fk, po);
        const float tau = fmaf(q.dtau, fk, q.tau0);
        acc = fmaf(pray_value(pimg, q, cl), tof_weight(lb, lut.inv_h, half_w, tau, centre), acc);
        fk += 1.f;
        po += q.sp;
    }
    float out = q.cf * acc;
    if (LM_MODE == 1) out = (out > 1e-9f) ? 1.f / out : 0.f;
    p[io_index(rg, c)] = out;
}

__global__ void __launch_bounds__(kLmBlock) k_back_tof_lm(Lors l, const int16_t *__restrict__ tofbin, Range rg,
                                                          const float *__restrict__ y, Geom g, Tof t,
                                                          TofLut lut, float *__restrict__ pimg)
{
    extern __shared__ __align__(16) float2 lut_sm[];
    lut_load(lut, lut_sm);
    __syncthreads();
    const uint32_t lb = lut_base(lut_sm);
    const int64_t c = blockIdx.x * (int64_t)kLmBlock + threadIdx.x;
    if (c >= rg.count) return;
    const int64_t j = lor_index(rg, c);
    const float yj = y[io_index(rg, c)];
    if (yj == 0.f) return;
    const float half_w = 0.5f * t.width;
    const float centre = (float)tofbin[j] * t.width;
    const float reach = half_w + t.nsig * t.sigma;
    Ray r;
    ray_setup<true>(l, j, g, t.coff, centre - reach, centre + reach, r);
    const PRay q = pray_from(r, g);
    const float x = q.cf * yj;
    float fk = 0.f;
    int po = q.off;
    for (int k = 0; k < q.nk; ++k) {
        const PCell cl = pray_cell(q, fk, po);
        const float tau = fmaf(q.dtau, fk, q.tau0);
        const float w = tof_weight(lb, lut.inv_h, half_w, tau, centre);
        if (w != 0.f) pray_scatter(pimg, q, cl, x * w);
        fk += 1.f;
        po += q.sp;
    }
}

// ---- OSEM element-wise update ---------------------------------------------------------------------------
__global__ void k_osem_update(float *__restrict__ x, float *__restrict__ b, const float *__restrict__ sens,
                              float scale, int64_t nvox)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= nvox) return;
    const float s = sens[i];
    x[i] = (s > 0.f) ? x[i] * b[i] * scale / s : 0.f;
    b[i] = 0.f;
}

// ---- launchers --------------------------------------------------------------------------------------------
static inline unsigned grid_for(int64_t n, int block) { return (unsigned)((n + block - 1) / block); }

cudaError_t launch_classify(const Lors &l, int64_t n, uint8_t *axis, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_classify<<<grid_for(n, 256), 256, 0, st>>>(l, n, axis);
    return cudaGetLastError();
}

cudaError_t launch_plane_steps(const Lors &l, int64_t n, const Geom &g, unsigned long long *total, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_plane_steps<<<grid_for(n, 256), 256, 0, st>>>(l, n, g, total);
    return cudaGetLastError();
}

cudaError_t launch_plane_steps_tof_lm(const Lors &l, const int16_t *tofbin, int64_t n, const Geom &g, const Tof &t,
                                      unsigned long long *total, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_plane_steps_tof_lm<<<grid_for(n, 256), 256, 0, st>>>(l, tofbin, n, g, t, total);
    return cudaGetLastError();
}

cudaError_t launch_fwd(const Lors &l, Range rg, const float *img, const Geom &g, float *p, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    k_fwd<<<grid_for(rg.count, kBlock), kBlock, 0, st>>>(l, rg, img, g, p);
    return cudaGetLastError();
}

cudaError_t launch_back(const Lors &l, Range rg, const float *y, const Geom &g, float *img, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    k_back<<<grid_for(rg.count, kBlock), kBlock, 0, st>>>(l, rg, y, g, img);
    return cudaGetLastError();
}

static inline size_t sino_smem(const Tof &t)
{
    return (size_t)((t.nbins * (kBlock + 1) + 3) & ~3) * sizeof(float) + (size_t)kLutN * sizeof(float2);
}

cudaError_t launch_fwd_tof_sino(const Lors &l, Range rg, const float *img, const Geom &g, const Tof &t,
                                const TofLut &lut, float *p, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    if (rg.first != 0 || rg.stride != 1) return cudaErrorInvalidValue;
    const size_t smem = sino_smem(t);
    cudaError_t e = cudaFuncSetAttribute(k_fwd_tof_sino, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_fwd_tof_sino<<<grid_for(rg.count, kBlock), kBlock, smem, st>>>(l, rg.count, img, g, t, lut, p);
    return cudaGetLastError();
}

cudaError_t launch_back_tof_sino(const Lors &l, Range rg, const float *y, const Geom &g, const Tof &t,
                                 const TofLut &lut, float *img, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    if (rg.first != 0 || rg.stride != 1) return cudaErrorInvalidValue;
    const size_t smem = sino_smem(t);
    cudaError_t e = cudaFuncSetAttribute(k_back_tof_sino, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_back_tof_sino<<<grid_for(rg.count, kBlock), kBlock, smem, st>>>(l, rg.count, y, g, t, lut, img);
    return cudaGetLastError();
}

constexpr size_t kLutBytes = (size_t)kLutN * sizeof(float2);

cudaError_t launch_fwd_tof_lm(const Lors &l, const int16_t *tofbin, Range rg, const float *img, const Geom &g,
                              const Tof &t, const TofLut &lut, float *p, int lm_mode, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    if (lm_mode == 1)
        k_fwd_tof_lm<1><<<grid_for(rg.count, kLmBlock), kLmBlock, kLutBytes, st>>>(l, tofbin, rg, img, g, t, lut, p);
    else
        k_fwd_tof_lm<0><<<grid_for(rg.count, kLmBlock), kLmBlock, kLutBytes, st>>>(l, tofbin, rg, img, g, t, lut, p);
    return cudaGetLastError();
}

cudaError_t launch_back_tof_lm(const Lors &l, const int16_t *tofbin, Range rg, const float *y, const Geom &g,
                               const Tof &t, const TofLut &lut, float *img, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    k_back_tof_lm<<<grid_for(rg.count, kLmBlock), kLmBlock, kLutBytes, st>>>(l, tofbin, rg, y, g, t, lut, img);
    return cudaGetLastError();
}

cudaError_t launch_osem_update(float *x, float *b, const float *sens, float scale, int64_t nvox, cudaStream_t st)
{
    if (nvox == 0) return cudaSuccess;
    k_osem_update<<<grid_for(nvox, 256), 256, 0, st>>>(x, b, sens, scale, nvox);
    return cudaGetLastError();
}

} // namespace jp
