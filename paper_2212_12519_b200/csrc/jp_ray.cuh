// jp_ray.cuh -- per-LOR set-up shared by all Joseph kernels (device code only).
//
// PAPER.md:33 (section 2.1): "the algorithm first determines the principal direction in the image
// that is most parallel to the ray and then steps through the image volume plane by plane along this
// principal direction.  In every plane, the intersection point between the ray and the plane is
// calculated ..."  The crossing point is an affine function of the plane index, so the whole set-up
// (principal axis, plane range, affine coefficients, incidence-angle factor, TOF coordinate) is done
// ONCE per LOR in float64 -- every discrete decision (axis, tie, first/last plane of the closed
// segment) is then exact -- and the per-plane hot loop evaluates one float32 FMA per coordinate.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace jp {

struct Geom {
    int n[3];
    float o[3];
    float v[3];
};

struct Tof {
    float width;      // W, TOF bin width (mm)
    float sigma;      // sigma (mm)
    float nsig;       // truncation in sigmas
    int nbins;        // sinogram bins
    float coff;       // centre offset (mm)
};

struct Lors {
    const float *xs, *ys, *zs, *xe, *ye, *ze;
};

// Everything the plane loop needs.  Plane index i = i0 + k, k = 0..nk-1.
struct Ray {
    int p;            // principal axis
    int i0, nk;       // first plane, number of planes (0: nothing to do)
    float a1, b1;     // u_q1(k) = a1 + b1 k   (voxel units along q1)
    float a2, b2;     // u_q2(k) = a2 + b2 k
    float cf;         // v_p |d| / |d_p|
    float tau0, dtau; // tau(k) = tau0 + dtau k  (mm from the LOR midpoint, + towards e, minus centre offset)
    int n1, n2;       // image dims along q1, q2
    int sp, s1, s2;   // element strides of p, q1, q2
};

// 1/x and sqrt(x) in double from a float32 seed and Newton steps (relative error ~1e-16): the double
// precision division and square root of the CUDA library are 30-40 instruction routines, and the
// set-up needs neither correct rounding (its results are rounded to float32) nor exactness (every
// discrete decision is re-checked with exact products).
__device__ __forceinline__ double drcp(double x)
{
    double r = (double)(1.f / (float)x);
    r = fma(r, fma(-x, r, 1.0), r);
    r = fma(r, fma(-x, r, 1.0), r);
    return r;
}

__device__ __forceinline__ double dsqrt_pos(double x) // x > 0
{
    double r = (double)rsqrtf((float)x); // ~ 1/sqrt(x)
    r = r * fma(-0.5 * x * r, r, 1.5);
    r = r * fma(-0.5 * x * r, r, 1.5);
    return x * r;
}

__device__ __forceinline__ int principal_axis(double d0, double d1, double d2)
{
    // argmax |d_a| on the exact differences, ties -> lowest index (reading A3)
    double a0 = fabs(d0), a1 = fabs(d1), a2 = fabs(d2);
    int p = 0;
    double m = a0;
    if (a1 > m) { p = 1; m = a1; }
    if (a2 > m) { p = 2; }
    return p;
}

// The plane range is clipped to the planes whose crossing point has -1 < u_q < n_q for both in-plane
// axes (all other planes contribute exactly zero: their four neighbours are outside the image).
// WITH_TOF: also fill tau0/dtau and clip to the planes with tau_lo <= tau <= tau_hi (outside that
// window every TOF weight the caller needs is exactly zero: the kernel is truncated).
// Both clips are conservative (rounded outwards); they are optimisations, not decisions.
template <bool WITH_TOF>
__device__ __forceinline__ void ray_setup_pts(const double (&s)[3], const double (&e)[3], const Geom &g, float coff,
                                              float tau_lo, float tau_hi, Ray &r)
{
    const double d[3] = {e[0] - s[0], e[1] - s[1], e[2] - s[2]}; // exact
    r.nk = 0;
    r.i0 = 0;
    r.p = principal_axis(d[0], d[1], d[2]);
    const int p = r.p;
    const int q1 = (p == 0) ? 1 : 0;
    const int q2 = (p == 2) ? 1 : 2;
    r.n1 = g.n[q1];
    r.n2 = g.n[q2];
    const int st[3] = {g.n[1] * g.n[2], g.n[2], 1};
    r.sp = st[p];
    r.s1 = st[q1];
    r.s2 = st[q2];
    r.a1 = r.b1 = r.a2 = r.b2 = r.cf = r.tau0 = r.dtau = 0.f;
    if (d[0] == 0.0 && d[1] == 0.0 && d[2] == 0.0) return; // reading A1

    const double op = (double)g.o[p], vp = (double)g.v[p];
    // ---- closed segment rule (reading A4): planes with min(s_p,e_p) <= o_p + i v_p <= max(s_p,e_p)
    const double lo = fmin(s[p], e[p]), hi = fmax(s[p], e[p]);
    const double np1 = (double)(g.n[p] - 1);
    int ilo = 0, ihi = g.n[p] - 1;
    if (!(lo <= op && hi >= op + np1 * vp)) { // an end point inside the image slab (rare)
        const double ivp = drcp(vp);
        double flo = ceil((lo - op) * ivp), fhi = floor((hi - op) * ivp);
        flo = fmin(fmax(flo, 0.0), np1 + 1.0);
        fhi = fmin(fmax(fhi, -1.0), np1);
        ilo = (int)flo;
        ihi = (int)fhi;
        // exact fix-up of the rounded quotients
        if (ilo > 0 && op + (double)(ilo - 1) * vp >= lo) --ilo;
        if (ilo <= g.n[p] - 1 && op + (double)ilo * vp < lo) ++ilo;
        if (ihi < g.n[p] - 1 && op + (double)(ihi + 1) * vp <= hi) ++ihi;
        if (ihi >= 0 && op + (double)ihi * vp > hi) --ihi;
    }

    // ---- crossing point in voxel units: u_q(i) = A_q + B_q i
    const double inv_dp = drcp(d[p]);
    double A[2], B[2];
    const int q[2] = {q1, q2};
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const double ratio = d[q[c]] * inv_dp;
        const double ivq = drcp((double)g.v[q[c]]);
        B[c] = ratio * vp * ivq;
        A[c] = (s[q[c]] - (double)g.o[q[c]] + (op - s[p]) * ratio) * ivq;
        // conservative clip to -1 < u < n_q
        const double nq = (double)g.n[q[c]];
        if (fabs(B[c]) < 1e-12) { // u_q moves by less than 1e-9 voxel over the whole image
            if (A[c] <= -1.0 || A[c] >= nq) ihi = ilo - 1;
        } else {
            const double ivb = drcp(B[c]);
            double ia = (-1.0 - A[c]) * ivb, ib = (nq - A[c]) * ivb;
            double imin = fmin(ia, ib), imax = fmax(ia, ib);
            imin = fmin(fmax(floor(imin), -1.0), np1 + 1.0);
            imax = fmin(fmax(ceil(imax), -1.0), np1 + 1.0);
            ilo = max(ilo, (int)imin);
            ihi = min(ihi, (int)imax);
        }
    }
    const double L = dsqrt_pos(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double tau0 = 0.0, dtau = 0.0;
    if (WITH_TOF) {
        // tau(i) = (t_i - 1/2) L - coff, t_i = (o_p + i v_p - s_p)/d_p   (reading A8)
        dtau = vp * inv_dp * L;
        tau0 = ((op - s[p]) * inv_dp - 0.5) * L - (double)coff;
        const double ivt = drcp(dtau);
        double ia = ((double)tau_lo - tau0) * ivt, ib = ((double)tau_hi - tau0) * ivt;
        double imin = fmin(ia, ib), imax = fmax(ia, ib);
        imin = fmin(fmax(floor(imin), -1.0), np1 + 1.0);
        imax = fmin(fmax(ceil(imax), -1.0), np1 + 1.0);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    if (ihi < ilo) return;
    r.i0 = ilo;
    r.nk = ihi - ilo + 1;
    r.a1 = (float)(A[0] + B[0] * (double)ilo);
    r.b1 = (float)B[0];
    r.a2 = (float)(A[1] + B[1] * (double)ilo);
    r.b2 = (float)B[1];
    r.cf = (float)(vp * L * fabs(inv_dp));
    if (WITH_TOF) {
        r.tau0 = (float)(tau0 + dtau * (double)ilo);
        r.dtau = (float)dtau;
    }
}

template <bool WITH_TOF>
__device__ __forceinline__ void ray_setup(const Lors &l, int64_t j, const Geom &g, float coff,
                                          float tau_lo, float tau_hi, Ray &r)
{
    const double s[3] = {(double)l.xs[j], (double)l.ys[j], (double)l.zs[j]};
    const double e[3] = {(double)l.xe[j], (double)l.ye[j], (double)l.ze[j]};
    ray_setup_pts<WITH_TOF>(s, e, g, coff, tau_lo, tau_hi, r);
}

// One crossed plane: integer cell and bilinear weights of the crossing point.
struct Cell {
    int k1, k2;
    float w1, w2; // fractions along q1, q2
};

__device__ __forceinline__ Cell plane_cell(const Ray &r, int k)
{
    const float fk = (float)k;
    const float u1 = fmaf(r.b1, fk, r.a1);
    const float u2 = fmaf(r.b2, fk, r.a2);
    const float f1 = floorf(u1), f2 = floorf(u2);
    Cell c;
    c.k1 = (int)f1;
    c.k2 = (int)f2;
    c.w1 = u1 - f1;
    c.w2 = u2 - f2;
    return c;
}

// bilinear interpolation of the four nearest neighbours, zero outside the image (reading A5)
__device__ __forceinline__ float plane_value(const float *__restrict__ img, const Ray &r, int k, const Cell &c)
{
    const float *ptr = img + (int64_t)(r.i0 + k) * r.sp + (int64_t)c.k1 * r.s1 + (int64_t)c.k2 * r.s2;
    const bool in1a = (unsigned)c.k1 < (unsigned)r.n1, in1b = (unsigned)(c.k1 + 1) < (unsigned)r.n1;
    const bool in2a = (unsigned)c.k2 < (unsigned)r.n2, in2b = (unsigned)(c.k2 + 1) < (unsigned)r.n2;
    const float v00 = (in1a && in2a) ? __ldg(ptr) : 0.f;
    const float v01 = (in1a && in2b) ? __ldg(ptr + r.s2) : 0.f;
    const float v10 = (in1b && in2a) ? __ldg(ptr + r.s1) : 0.f;
    const float v11 = (in1b && in2b) ? __ldg(ptr + r.s1 + r.s2) : 0.f;
    const float lo = fmaf(c.w2, v01 - v00, v00);
    const float hi = fmaf(c.w2, v11 - v10, v10);
    return fmaf(c.w1, hi - lo, lo);
}

// adjoint of plane_value: img[...] += w x  with atomic adds
__device__ __forceinline__ void plane_scatter(float *__restrict__ img, const Ray &r, int k, const Cell &c, float x)
{
    float *ptr = img + (int64_t)(r.i0 + k) * r.sp + (int64_t)c.k1 * r.s1 + (int64_t)c.k2 * r.s2;
    const bool in1a = (unsigned)c.k1 < (unsigned)r.n1, in1b = (unsigned)(c.k1 + 1) < (unsigned)r.n1;
    const bool in2a = (unsigned)c.k2 < (unsigned)r.n2, in2b = (unsigned)(c.k2 + 1) < (unsigned)r.n2;
    const float xa = x * (1.f - c.w1), xb = x * c.w1;
    const float m2 = 1.f - c.w2;
    if (in1a && in2a) atomicAdd(ptr, xa * m2);
    if (in1a && in2b) atomicAdd(ptr + r.s2, xa * c.w2);
    if (in1b && in2a) atomicAdd(ptr + r.s1, xb * m2);
    if (in1b && in2b) atomicAdd(ptr + r.s1 + r.s2, xb * c.w2);
}

// ---- TOF kernel (reading A10) -----------------------------------------------------
// w(tau, c) = 1/2 [E(c + W/2 - tau) - E(c - W/2 - tau)],  E(x) = erf(clamp(x, -m, m) / (sigma sqrt2)),
// m = n_sigmas sigma.  E is odd and constant beyond m, so it is tabulated on [0, m] only: kLutK
// intervals of h = m / kLutK, entry k = (E(k h), E((k+1) h) - E(k h)) computed in float64 (jp_tof_lut.cu),
// entry kLutK = (E(m), 0).  Linear interpolation error <= h^2/8 max|E''| = 0.06 n_sigmas^2 / kLutK^2
// (1.3e-7 for 3 sigma).  A lookup is 9 instructions (one LDS.64) against ~22 for erff.
constexpr int kLutK = 2048;
constexpr int kLutN = kLutK + 2;
constexpr float kMagic = 12582912.f; // 1.5 * 2^23: fadd_rd(x, kMagic) holds floor(x) in the low mantissa bits
constexpr int kMagicI = 0x4B400000;  // bit pattern of kMagic

struct TofLut {
    const float2 *tab; // device, kLutN entries
    float inv_h;       // kLutK / m
};

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int OFF>
__device__ __forceinline__ float2 lds_pair(uint32_t addr)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(addr), "n"(OFF) : "memory");
    return v;
}

// copy the table into shared memory (all threads of the CTA; caller synchronises)
__device__ __forceinline__ void lut_load(const TofLut &L, float2 *sm)
{
    for (int i = threadIdx.x; i < kLutN; i += blockDim.x) sm[i] = __ldg(L.tab + i);
}

// shared-memory address of the table, biased for lut_E
__device__ __forceinline__ uint32_t lut_base(const float2 *sm) { return smem_addr(sm) - ((uint32_t)kMagicI << 3); }

__device__ __forceinline__ float lut_E(uint32_t base, float inv_h, float x)
{
    const float s = fminf(fabsf(x) * inv_h, (float)kLutK);
    const float tt = __fadd_rd(s, kMagic);
    const float f = s - (tt - kMagic);
    const float2 v = lds_pair<0>(base + (__float_as_uint(tt) << 3));
    return copysignf(fmaf(f, v.y, v.x), x);
}

// weight of the bin centred at c seen from tau
__device__ __forceinline__ float tof_weight(uint32_t base, float inv_h, float half_w, float tau, float c)
{
    const float x = c - tau;
    return 0.5f * (lut_E(base, inv_h, x + half_w) - lut_E(base, inv_h, x - half_w));
}

// ---- padded image: the per-LOR kernels without boundary tests ----------------------------------------
// Reading A5 (neighbours outside the image count as zero) is zero padding.  The per-LOR kernels work on
// a copy of the image with kImgPad zero voxels on every side (jp_pad.cu), so the four neighbour loads /
// atomic adds of a plane need no bounds predicates.  PRay is Ray for that copy: the plane range is
// trimmed (evaluating the end planes with the same float32 FMA as the loop) so that
// -kImgPad <= floor(u_q) and floor(u_q) + 1 <= n_q + kImgPad - 1 on every visited plane -- planes
// trimmed away have all four neighbours outside the image and contribute exactly zero.
constexpr int kImgPad = 2;

struct PRay {
    int nk;           // planes to visit (0: nothing to do)
    int off;          // element offset of (first plane, k1 = 0, k2 = 0) in the padded image, biased for the
                      // magic-number floor: off + bits(t1) * s1 + bits(t2) * s2 addresses the cell
    int sp, s1, s2;   // padded element strides of p, q1, q2
    float a1, b1, a2, b2, cf, tau0, dtau;
};

__device__ __forceinline__ PRay pray_from(const Ray &r, const Geom &g)
{
    PRay q;
    const int pn1 = g.n[1] + 2 * kImgPad, pn2 = g.n[2] + 2 * kImgPad;
    const int st[3] = {pn1 * pn2, pn2, 1};
    const int p = r.p, q1 = (p == 0) ? 1 : 0, q2 = (p == 2) ? 1 : 2;
    q.sp = st[p];
    q.s1 = st[q1];
    q.s2 = st[q2];
    q.b1 = r.b1;
    q.b2 = r.b2;
    q.cf = r.cf;
    q.dtau = r.dtau;
    // trim both ends against the padded range
    const float lo = -(float)kImgPad + 0.1f;
    const float hi1 = (float)(r.n1 + kImgPad - 1) - 0.1f, hi2 = (float)(r.n2 + kImgPad - 1) - 0.1f;
    int k0 = 0, k1 = r.nk - 1;
    while (k0 <= k1) {
        const float u1 = fmaf(r.b1, (float)k0, r.a1), u2 = fmaf(r.b2, (float)k0, r.a2);
        if (u1 > lo && u1 < hi1 && u2 > lo && u2 < hi2) break;
        ++k0;
    }
    while (k0 <= k1) {
        const float u1 = fmaf(r.b1, (float)k1, r.a1), u2 = fmaf(r.b2, (float)k1, r.a2);
        if (u1 > lo && u1 < hi1 && u2 > lo && u2 < hi2) break;
        --k1;
    }
    q.nk = k1 - k0 + 1;
    // rebase the affine coefficients to the first kept plane (one extra float32 rounding)
    q.a1 = fmaf(r.b1, (float)k0, r.a1);
    q.a2 = fmaf(r.b2, (float)k0, r.a2);
    q.tau0 = fmaf(r.dtau, (float)k0, r.tau0);
    q.off = (int)((uint32_t)((r.i0 + k0 + kImgPad) * q.sp + kImgPad * (q.s1 + q.s2)) -
                  (uint32_t)kMagicI * (uint32_t)q.s1 - (uint32_t)kMagicI * (uint32_t)q.s2); // wraps by design
    return q;
}

// one plane of a PRay: cell offset and bilinear fractions (FMA pipe only: the floor is a round-down add)
struct PCell {
    int off;
    float w1, w2;
};

__device__ __forceinline__ PCell pray_cell(const PRay &q, float fk, int plane_off)
{
    const float u1 = fmaf(q.b1, fk, q.a1), u2 = fmaf(q.b2, fk, q.a2);
    const float t1 = __fadd_rd(u1, kMagic), t2 = __fadd_rd(u2, kMagic);
    PCell c;
    c.w1 = u1 - (t1 - kMagic);
    c.w2 = u2 - (t2 - kMagic);
    c.off = (int)((uint32_t)plane_off + __float_as_uint(t1) * (uint32_t)q.s1 + __float_as_uint(t2) * (uint32_t)q.s2);
    return c;
}

__device__ __forceinline__ float pray_value(const float *__restrict__ pimg, const PRay &q, const PCell &c)
{
    const float *ptr = pimg + c.off;
    const float v00 = __ldg(ptr), v01 = __ldg(ptr + q.s2), v10 = __ldg(ptr + q.s1), v11 = __ldg(ptr + q.s1 + q.s2);
    const float lo = fmaf(c.w2, v01 - v00, v00);
    const float hi = fmaf(c.w2, v11 - v10, v10);
    return fmaf(c.w1, hi - lo, lo);
}

__device__ __forceinline__ void pray_scatter(float *__restrict__ pimg, const PRay &q, const PCell &c, float x)
{
    float *ptr = pimg + c.off;
    const float xa = x * (1.f - c.w1), xb = x * c.w1;
    const float m2 = 1.f - c.w2;
    atomicAdd(ptr, xa * m2);
    atomicAdd(ptr + q.s2, xa * c.w2);
    atomicAdd(ptr + q.s1, xb * m2);
    atomicAdd(ptr + q.s1 + q.s2, xb * c.w2);
}

} // namespace jp
