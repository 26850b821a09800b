// jp_quad.cu -- TOF listmode projectors on a QUAD image: the kernels behind the planned listmode calls.
//
// Listmode events touch the image at random: measured on B200, a warp-wide gather /
// atomic add of scattered addresses costs one L1 "wavefront" (and one 32-byte sector packet to L2) per
// lane whatever its width -- 289 G gathers/s and 193 G atomic adds/s chip-wide for 4, 8 or 16 bytes alike.
// Joseph's bilinear interpolation reads the 2 x 2 neighbourhood (k1, k1+1) x (k2, k2+1) of the
// crossing point, so the image is re-laid out with that neighbourhood in one aligned 16-byte element:
//
//   Q_p[i0][i1][i2] = ( f[c], f[c + e2], f[c + e1], f[c + e1 + e2] ),   e1 / e2 = unit steps along q1 / q2
//
// (zero outside the image, reading A5; kImgPad voxels of padding as for PRay).  One plane step is then ONE
// 128-bit load instead of four 32-bit loads; the adjoint accumulates the four weights with ONE 128-bit
// atomic add (red.global.add.v4.f32) into B_p[i0][i1][i2] = (to c, to c+e2, to c+e1, to c+e1+e2), and a merge
// pass folds the four taps back into the image.  Q_p depends on the principal axis p through q1, so the plan
// keeps the events of every subset split by axis and the kernels run axis by axis; each array is 4x the
// image (66.6 MB for 200x200x96), L2-resident on its own (126 MB L2), which is why the axes are not mixed.
#include "jp_g1tab.cuh"

namespace jp {

namespace {

constexpr int kQBlock = 256;

__device__ __forceinline__ float padded_at(const float *__restrict__ img, const Geom &g, int i0, int i1, int i2)
{
    // value of the zero-padded image at padded index (i0, i1, i2)
    const int a = i0 - kImgPad, b = i1 - kImgPad, c = i2 - kImgPad;
    if ((unsigned)a >= (unsigned)g.n[0] || (unsigned)b >= (unsigned)g.n[1] || (unsigned)c >= (unsigned)g.n[2]) return 0.f;
    return __ldg(img + ((int64_t)a * g.n[1] + b) * g.n[2] + c);
}

// Q0 (q1 = axis 1) and Q1 (q1 = axis 0) of the padded image, one thread per padded voxel
__global__ void __launch_bounds__(kQBlock) k_quad_build(const float *__restrict__ img, Geom g, int64_t pvox,
                                                        float4 *__restrict__ q0, float4 *__restrict__ q1)
{
    const int64_t i = blockIdx.x * (int64_t)kQBlock + threadIdx.x;
    if (i >= pvox) return;
    const int pn1 = g.n[1] + 2 * kImgPad, pn2 = g.n[2] + 2 * kImgPad;
    const int i2 = (int)(i % pn2);
    const int64_t r = i / pn2;
    const int i1 = (int)(r % pn1), i0 = (int)(r / pn1);
    const float c00 = padded_at(img, g, i0, i1, i2), c01 = padded_at(img, g, i0, i1, i2 + 1);
    if (q0) q0[i] = make_float4(c00, c01, padded_at(img, g, i0, i1 + 1, i2), padded_at(img, g, i0, i1 + 1, i2 + 1));
    if (q1) q1[i] = make_float4(c00, c01, padded_at(img, g, i0 + 1, i1, i2), padded_at(img, g, i0 + 1, i1, i2 + 1));
}

// sum of the four taps of B0 / B1 that belong to image voxel (a, b, c)
__device__ __forceinline__ float quad_taps(const float4 *__restrict__ b0, const float4 *__restrict__ b1, const Geom &g,
                                           int a, int b, int c)
{
    const int pn1 = g.n[1] + 2 * kImgPad, pn2 = g.n[2] + 2 * kImgPad;
    const int64_t s0 = (int64_t)pn1 * pn2, s1 = pn2;
    const int64_t e = ((int64_t)(a + kImgPad) * pn1 + (b + kImgPad)) * pn2 + (c + kImgPad);
    float v = 0.f;
    if (b0) v += b0[e].x + b0[e - 1].y + b0[e - s1].z + b0[e - s1 - 1].w;
    if (b1) v += b1[e].x + b1[e - 1].y + b1[e - s0].z + b1[e - s0 - 1].w;
    return v;
}

__global__ void __launch_bounds__(kQBlock) k_quad_merge(const float4 *__restrict__ b0, const float4 *__restrict__ b1,
                                                        Geom g, int64_t nvox, float *__restrict__ img)
{
    const int64_t i = blockIdx.x * (int64_t)kQBlock + threadIdx.x;
    if (i >= nvox) return;
    const int c = (int)(i % g.n[2]);
    const int64_t r = i / g.n[2];
    img[i] += quad_taps(b0, b1, g, (int)(r / g.n[1]), (int)(r % g.n[1]), c);
}

// OSEM: x = sens > 0 ? x * (b + extra) * scale / sens : 0, with b folded from the quad accumulators
__global__ void __launch_bounds__(kQBlock) k_quad_osem_update(float *__restrict__ x, const float4 *__restrict__ b0,
                                                              const float4 *__restrict__ b1, float *__restrict__ extra,
                                                              const float *__restrict__ sens, float scale, Geom g,
                                                              int64_t nvox)
{
    const int64_t i = blockIdx.x * (int64_t)kQBlock + threadIdx.x;
    if (i >= nvox) return;
    const int c = (int)(i % g.n[2]);
    const int64_t r = i / g.n[2];
    float b = quad_taps(b0, b1, g, (int)(r / g.n[1]), (int)(r % g.n[1]), c);
    if (extra) {
        b += extra[i];
        extra[i] = 0.f;
    }
    const float s = sens[i];
    x[i] = (s > 0.f) ? x[i] * b * scale / s : 0.f;
}

__device__ __forceinline__ float quad_value(const float4 *__restrict__ q, const PCell &c)
{
    const float4 v = __ldg(q + c.off);
    const float lo = fmaf(c.w2, v.y - v.x, v.x);
    const float hi = fmaf(c.w2, v.w - v.z, v.z);
    return fmaf(c.w1, hi - lo, lo);
}

__device__ __forceinline__ void quad_scatter(float4 *__restrict__ b, const PCell &c, float x)
{
    const float xa = x * (1.f - c.w1), xb = x * c.w1;
    const float m2 = 1.f - c.w2;
    atomicAdd(b + c.off, make_float4(xa * m2, xa * c.w2, xb * m2, xb * c.w2));
}

__device__ __forceinline__ int64_t q_io_index(const Range &rg, int64_t c)
{
    if (rg.compact) return c + rg.io_off;
    const int64_t j = rg.first + c * rg.stride;
    return rg.perm ? (int64_t)rg.perm[j] : j;
}

} // namespace

// ---- TOF listmode on the quad image (events of ONE principal axis) --------------------------
template <int LM_MODE>
__global__ void __launch_bounds__(kQBlock) k_fwd_tof_lm_quad(Lors l, const int16_t *__restrict__ tofbin, Range rg,
                                                             const float4 *__restrict__ q, Geom g, Tof t, TofLut lut,
                                                             float *__restrict__ p)
{
    extern __shared__ __align__(16) float2 lut_sm[];
    lut_load(lut, lut_sm);
    __syncthreads();
    const uint32_t lb = lut_base(lut_sm);
    const int64_t c = blockIdx.x * (int64_t)kQBlock + threadIdx.x;
    if (c >= rg.count) return;
    const int64_t j = rg.first + c * rg.stride;
    const float half_w = 0.5f * t.width;
    const float centre = (float)tofbin[j] * t.width;
    const float reach = half_w + t.nsig * t.sigma;
    Ray r;
    ray_setup<true>(l, j, g, t.coff, centre - reach, centre + reach, r);
    const PRay pr = pray_from(r, g);
    float acc = 0.f, fk = 0.f;
    int po = pr.off;
    for (int k = 0; k < pr.nk; ++k) {
        const PCell cl = pray_cell(pr, fk, po);
        const float tau = fmaf(pr.dtau, fk, pr.tau0);
        acc = fmaf(quad_value(q, cl), tof_weight(lb, lut.inv_h, half_w, tau, centre), acc);
        fk += 1.f;
        po += pr.sp;
    }
    float out = pr.cf * acc;
    if (LM_MODE == 1) out = (out > 1e-9f) ? 1.f / out : 0.f;
    p[q_io_index(rg, c)] = out;
}

// Y_MODE 0: y = the values to back project;  1: y = sum_k G bilinear of every event (the forward projection without
// its factor cf, e.g. from the brick kernels) and the OSEM ratio 1 / (cf y) if cf y > 1e-9 else 0 is back projected (A14).
// G1W: the TOF weights come from the one-look-up table of jp_g1tab.cuh, the table the brick forward kernel uses, instead
// of the edge-function table.  An OSEM update divides an event's weights by their own sum: for an event whose expectation
// is made of a few tail weights the two tables' rounding (1e-7 absolute each) does not cancel unless forward and adjoint
// read the SAME table (measured: update rel-L2 1.2e-4 -> 2e-6 on a problem with such events).
template <int Y_MODE, bool G1W>
__global__ void __launch_bounds__(kQBlock) k_back_tof_lm_quad(Lors l, const int16_t *__restrict__ tofbin, Range rg,
                                                              const float *__restrict__ y, Geom g, Tof t, TofLut lut, G1Tab gt,
                                                              float4 *__restrict__ b)
{
    extern __shared__ __align__(16) float2 lut_sm[];
    if (G1W) {
        for (int i = threadIdx.x; i < gt.n; i += kQBlock) lut_sm[i] = __ldg(gt.tab + i);
    } else {
        lut_load(lut, lut_sm);
    }
    __syncthreads();
    const uint32_t lb = lut_base(lut_sm); // (the same bias for both tables: entries are float2)
    const int64_t c = blockIdx.x * (int64_t)kQBlock + threadIdx.x;
    if (c >= rg.count) return;
    const int64_t j = rg.first + c * rg.stride;
    float yj = y[q_io_index(rg, c)];
    if (yj == 0.f) return;
    const float half_w = 0.5f * t.width;
    const float centre = (float)tofbin[j] * t.width;
    const float reach = half_w + t.nsig * t.sigma;
    Ray r;
    ray_setup<true>(l, j, g, t.coff, centre - reach, centre + reach, r);
    const PRay pr = pray_from(r, g);
    if (Y_MODE == 1) {
        const float ybar = pr.cf * yj;
        if (!(ybar > 1e-9f)) return;
        yj = 1.f / ybar;
    }
    const float x = pr.cf * yj;
    const float x0 = (centre - pr.tau0) * gt.scale, dx = -pr.dtau * gt.scale; // G1W: table position of plane k = x0 + dx k
    float fk = 0.f;
    int po = pr.off;
    for (int k = 0; k < pr.nk; ++k) {
        const PCell cl = pray_cell(pr, fk, po);
        const float w = G1W ? g1_weight(lb, gt.xedge, fmaf(dx, fk, x0))
                            : tof_weight(lb, lut.inv_h, half_w, fmaf(pr.dtau, fk, pr.tau0), centre);
        if (w != 0.f) quad_scatter(b, cl, x * w);
        fk += 1.f;
        po += pr.sp;
    }
}


// ---- one OSEM subset update per event in ONE pass (reading A14): ybar_e from the quad image, r_e = 1 / ybar_e, and
// the scatter of cf r_e w along the same planes into the quad accumulator.  The event's set-up (float64) is done
// once instead of twice, the ratio never goes through memory, and gathers (L1-bound) and atomics (L2-bound) of
// different warps overlap in one launch.
__global__ void __launch_bounds__(kQBlock) k_osem_tof_lm_quad(Lors l, const int16_t *__restrict__ tofbin, Range rg,
                                                              const float4 *__restrict__ q, Geom g, Tof t, TofLut lut,
                                                              float4 *__restrict__ b)
{
    extern __shared__ __align__(16) float2 lut_sm[];
    lut_load(lut, lut_sm);
    __syncthreads();
    const uint32_t lb = lut_base(lut_sm);
    const int64_t c = blockIdx.x * (int64_t)kQBlock + threadIdx.x;
    if (c >= rg.count) return;
    const int64_t j = rg.first + c * rg.stride;
    const float half_w = 0.5f * t.width;
    const float centre = (float)tofbin[j] * t.width;
    const float reach = half_w + t.nsig * t.sigma;
    Ray r;
    ray_setup<true>(l, j, g, t.coff, centre - reach, centre + reach, r);
    const PRay pr = pray_from(r, g);
    float acc = 0.f, fk = 0.f;
    int po = pr.off;
    for (int k = 0; k < pr.nk; ++k) {
        const PCell cl = pray_cell(pr, fk, po);
        const float tau = fmaf(pr.dtau, fk, pr.tau0);
        acc = fmaf(quad_value(q, cl), tof_weight(lb, lut.inv_h, half_w, tau, centre), acc);
        fk += 1.f;
        po += pr.sp;
    }
    const float ybar = pr.cf * acc;
    if (!(ybar > 1e-9f)) return;
    const float x = pr.cf * (1.f / ybar);
    fk = 0.f;
    po = pr.off;
    for (int k = 0; k < pr.nk; ++k) {
        const PCell cl = pray_cell(pr, fk, po);
        const float tau = fmaf(pr.dtau, fk, pr.tau0);
        const float w = tof_weight(lb, lut.inv_h, half_w, tau, centre);
        if (w != 0.f) quad_scatter(b, cl, x * w);
        fk += 1.f;
        po += pr.sp;
    }
}

// ---- launchers ------------------------------------------------------------------------------------------------
static inline unsigned grid_for(int64_t n) { return (unsigned)((n + kQBlock - 1) / kQBlock); }
constexpr size_t kLutBytesQ = (size_t)kLutN * sizeof(float2);

cudaError_t launch_quad_build(const float *img, const Geom &g, float4 *q0, float4 *q1, cudaStream_t st)
{
    const int64_t pv = padded_voxels(g);
    k_quad_build<<<grid_for(pv), kQBlock, 0, st>>>(img, g, pv, q0, q1);
    return cudaGetLastError();
}

cudaError_t launch_quad_merge(const float4 *b0, const float4 *b1, const Geom &g, float *img, cudaStream_t st)
{
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    k_quad_merge<<<grid_for(nvox), kQBlock, 0, st>>>(b0, b1, g, nvox, img);
    return cudaGetLastError();
}

cudaError_t launch_quad_osem_update(float *x, const float4 *b0, const float4 *b1, float *extra, const float *sens,
                                    float scale, const Geom &g, cudaStream_t st)
{
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    k_quad_osem_update<<<grid_for(nvox), kQBlock, 0, st>>>(x, b0, b1, extra, sens, scale, g, nvox);
    return cudaGetLastError();
}

cudaError_t launch_fwd_tof_lm_quad(const Lors &l, const int16_t *tofbin, Range rg, const float4 *q, const Geom &g,
                                   const Tof &t, const TofLut &lut, float *p, int lm_mode, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    if (lm_mode == 1)
        k_fwd_tof_lm_quad<1><<<grid_for(rg.count), kQBlock, kLutBytesQ, st>>>(l, tofbin, rg, q, g, t, lut, p);
    else
        k_fwd_tof_lm_quad<0><<<grid_for(rg.count), kQBlock, kLutBytesQ, st>>>(l, tofbin, rg, q, g, t, lut, p);
    return cudaGetLastError();
}

// gt != null: TOF weights from that G1 table (the brick forward kernel's), else from the edge-function table `lut`
cudaError_t launch_back_tof_lm_quad(const Lors &l, const int16_t *tofbin, Range rg, const float *y, const Geom &g,
                                    const Tof &t, const TofLut &lut, float4 *b, cudaStream_t st, int y_mode, const G1Tab *gt)
{
    if (rg.count == 0) return cudaSuccess;
    const unsigned grid = grid_for(rg.count);
    if (gt && sizeof(float2) * (size_t)gt->n <= 40 * 1024) {
        const size_t smem = sizeof(float2) * (size_t)gt->n;
        if (y_mode == 1) k_back_tof_lm_quad<1, true><<<grid, kQBlock, smem, st>>>(l, tofbin, rg, y, g, t, lut, *gt, b);
        else k_back_tof_lm_quad<0, true><<<grid, kQBlock, smem, st>>>(l, tofbin, rg, y, g, t, lut, *gt, b);
    } else {
        const G1Tab none{};
        if (y_mode == 1) k_back_tof_lm_quad<1, false><<<grid, kQBlock, kLutBytesQ, st>>>(l, tofbin, rg, y, g, t, lut, none, b);
        else k_back_tof_lm_quad<0, false><<<grid, kQBlock, kLutBytesQ, st>>>(l, tofbin, rg, y, g, t, lut, none, b);
    }
    return cudaGetLastError();
}

cudaError_t launch_osem_tof_lm_quad(const Lors &l, const int16_t *tofbin, Range rg, const float4 *q, const Geom &g,
                                    const Tof &t, const TofLut &lut, float4 *b, cudaStream_t st)
{
    if (rg.count == 0) return cudaSuccess;
    k_osem_tof_lm_quad<<<grid_for(rg.count), kQBlock, kLutBytesQ, st>>>(l, tofbin, rg, q, g, t, lut, b);
    return cudaGetLastError();
}

} // namespace jp
