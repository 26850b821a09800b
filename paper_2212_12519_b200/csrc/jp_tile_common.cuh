// jp_tile_common.cuh -- pieces shared by the tiled kernels (jp_tile.cu: sinogram track tiles; jp_lm_tile.cu:
// listmode line tiles): the description of a transaxial track, the q1 cell of each of its planes, the axial
// part of a LOR on that track, and the construction of the (value, slope) rows in shared memory.
// PAPER.md:33 (Joseph's bilinear interpolation); see the header of jp_tile.cu for the factorisation.
#pragma once
#include "jp_internal.h"

namespace jp {
namespace tile {

#ifndef JP_RB
#define JP_RB 2
#endif

constexpr int kThreads = 256;
constexpr int kPerThread = 3;
constexpr int kTile = kThreads * kPerThread;
constexpr int kPad = 4;                // padding columns left of z = 0 in a shared-memory row
constexpr int kPadR = 4;               // columns needed right of z = n2 - 1

// shared per-tile track description, written by thread 0
struct Track {
    int p;          // principal axis (0 or 1)
    int I0, I1;     // plane range of the track (closed segment rule and q1 clip); empty if I1 < I0
    float a1, b1;   // u_q1(i) = a1 + b1 (i - I0)
    double inv_dp;  // 1 / d_p
    double ops;     // o_p - s_p
    float R;        // 1 + (d_q1/d_p)^2
    double iv2;     // 1 / v_2 (axial voxel size), the same for every LOR of the tile
};

// q1 cell of one plane of the track (shared by the whole tile): element offsets of the two image rows
// (i, k1, z = 0) and (i, k1 + 1, z = 0), -1 when the row lies outside the image (reading A5), and the
// two q1 weights
struct __align__(16) RowInfo {
    int base_a, base_b;
    float wa, wb;
};

__device__ __forceinline__ bool same_bits(float a, float b) { return __float_as_uint(a) == __float_as_uint(b); }

// the part of ray_setup that only depends on the shared transaxial end points (float64, once per tile)
static __device__ void track_setup(const Geom &g, float xs, float ys, float xe, float ye, Track &t)
{
    const double s[2] = {(double)xs, (double)ys};
    const double d[2] = {(double)xe - (double)xs, (double)ye - (double)ys};
    const int p = (fabs(d[1]) > fabs(d[0])) ? 1 : 0; // ties -> lowest index
    const int q1 = 1 - p;
    t.p = p;
    const double op = (double)g.o[p], vp = (double)g.v[p];
    const double sp = s[p], ep = s[p] + d[p];
    const double lo = fmin(sp, ep), hi = fmax(sp, ep);
    const double np1 = (double)(g.n[p] - 1);
    int ilo = 0, ihi = g.n[p] - 1;
    if (!(lo <= op && hi >= op + np1 * vp)) { // an end point inside the image slab: closed segment rule (A4)
        const double ivp = drcp(vp);
        double flo = ceil((lo - op) * ivp), fhi = floor((hi - op) * ivp);
        flo = fmin(fmax(flo, 0.0), np1 + 1.0);
        fhi = fmin(fmax(fhi, -1.0), np1);
        ilo = (int)flo;
        ihi = (int)fhi;
        if (ilo > 0 && op + (double)(ilo - 1) * vp >= lo) --ilo;
        if (ilo <= g.n[p] - 1 && op + (double)ilo * vp < lo) ++ilo;
        if (ihi < g.n[p] - 1 && op + (double)(ihi + 1) * vp <= hi) ++ihi;
        if (ihi >= 0 && op + (double)ihi * vp > hi) --ihi;
    }
    const double inv_dp = drcp(d[p]);
    const double ratio = d[q1] * inv_dp;
    const double ivq = drcp((double)g.v[q1]);
    const double B = ratio * vp * ivq;
    const double A = (s[q1] - (double)g.o[q1] + (op - sp) * ratio) * ivq;
    const double nq = (double)g.n[q1];
    if (fabs(B) < 1e-12) { // u_q1 moves by less than 1e-9 voxel over the whole image
        if (A <= -1.0 || A >= nq) ihi = ilo - 1;
    } else {
        const double ivb = drcp(B);
        const double ia = (-1.0 - A) * ivb, ib = (nq - A) * ivb;
        double imin = fmin(ia, ib), imax = fmax(ia, ib);
        imin = fmin(fmax(floor(imin), -1.0), np1 + 1.0);
        imax = fmin(fmax(ceil(imax), -1.0), np1 + 1.0);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    t.I0 = ilo;
    t.I1 = ihi;
    t.a1 = (float)(A + B * (double)ilo);
    t.b1 = (float)B;
    t.inv_dp = inv_dp;
    t.ops = op - sp;
    t.R = (float)(1.0 + ratio * ratio);
    t.iv2 = drcp((double)g.v[2]);
}

__device__ __forceinline__ RowInfo row_info(const Geom &g, const Track &t, int i)
{
    const int q1 = 1 - t.p;
    const int st[2] = {g.n[1] * g.n[2], g.n[2]};
    const float u1 = fmaf(t.b1, (float)(i - t.I0), t.a1);
    const float f1 = floorf(u1);
    const int k1 = (int)f1;
    const float w1 = u1 - f1;
    const bool in_a = (unsigned)k1 < (unsigned)g.n[q1];
    const bool in_b = (unsigned)(k1 + 1) < (unsigned)g.n[q1];
    const int base = i * st[t.p] + k1 * st[q1];
    RowInfo r;
    r.base_a = in_a ? base : -1;
    r.base_b = in_b ? base + st[q1] : -1;
    r.wa = in_a ? 1.f - w1 : 0.f;
    r.wb = in_b ? w1 : 0.f;
    return r;
}

// per-LOR axial part: u2(i) = a2 + b2 (i - i0), planes [i0, i1], incidence factor cf
struct ZRay {
    int i0, i1;
    float a2, b2, cf;
};

// kc: the returned a2 is u2 - kc (kc an integer-valued shift, 0 for the (value, slope) kernels)
__device__ __forceinline__ ZRay z_setup(const Geom &g, const Track &t, float zs, float ze, double kc = 0.0)
{
    ZRay z;
    const double dz = (double)ze - (double)zs;
    const double rz = dz * t.inv_dp;
    const double vp = (double)g.v[t.p];
    const double iv2 = t.iv2;
    const double B = rz * vp * iv2;
    const double A = ((double)zs - (double)g.o[2] + t.ops * rz) * iv2 - kc;
    const float rzf = (float)rz;
    z.cf = g.v[t.p] * sqrtf(fmaf(rzf, rzf, t.R));
    // clip to -1 < u2 < n2 (float32 estimate widened by one plane, then trimmed against the padded row)
    int ilo = t.I0, ihi = t.I1;
    const float kcf = (float)kc;
    const float Af = (float)A, Bf = (float)B, lo = -1.f - kcf, hi = (float)g.n[2] - kcf;
    if (Bf == 0.f) {
        if (Af <= lo || Af >= hi) ihi = ilo - 1;
    } else {
        const float inv = 1.f / Bf;
        const float ia = (lo - Af) * inv, ib = (hi - Af) * inv;
        const float imin = fminf(fmaxf(floorf(fminf(ia, ib)) - 1.f, -1.f), (float)g.n[t.p]);
        const float imax = fminf(fmaxf(ceilf(fmaxf(ia, ib)) + 1.f, -1.f), (float)g.n[t.p]);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    z.b2 = Bf;
    z.a2 = (float)(A + B * (double)ilo);
    // trim: floor(u2) must stay inside the padded row: -2 <= floor(u2) <= n2 (planes trimmed away have
    // all four neighbours outside the image and contribute exactly zero)
    const float umin = lo - 0.9f, umax = hi + 0.9f;
    while (ilo <= ihi) {
        if (z.a2 > umin && z.a2 < umax) break;
        ++ilo;
        z.a2 = (float)(A + B * (double)ilo);
    }
    while (ilo <= ihi) {
        const float u = fmaf(z.b2, (float)(ihi - ilo), z.a2);
        if (u > umin && u < umax) break;
        --ihi;
    }
    z.i0 = ilo;
    z.i1 = ihi;
    return z;
}

// ---- (value, slope) rows of planes [c0, c0 + rows) of track t:  C[z] = wa f[i,k1,z] + wb f[i,k1+1,z],
// pair = (C[z], C[z+1] - C[z]), columns z = -1 .. n2-1 at C2[r * P + kPad + z]  (all threads of the CTA)
// ICPT: store (intercept, slope) instead of (value, slope): pair(z) = (C[z] - (z - kc) D[z], D[z]), D[z] = C[z+1] - C[z],
// so that the interpolant at axial coordinate u (cell z = floor(u)) is  pair.x + (u - kc) pair.y  with no
// fractional part needed; kc (an integer, the middle of the axial range) keeps |u - kc| small.
// PT: row pitch as a template parameter (rows addressed with immediates), or 0: the pitch is the run-time value `prt`
template <int PT, bool ICPT = false, int RB = JP_RB, int NT = kThreads>
__device__ __forceinline__ void build_rows(float2 *C2, const RowInfo *rinfo, const float *__restrict__ img, const Track &t,
                                           int c0, int rows, int n2, int vec_ok, float kc = 0.f, int prt = 0)
{
    const int P = PT > 0 ? PT : prt;
    auto mk = [&](float v, float d, float zrel) { return ICPT ? make_float2(fmaf(-zrel, d, v), d) : make_float2(v, d); };
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
        if (vec_ok) {
            // one warp per row, lanes along z in groups of four voxels; kRB rows in flight per warp
            const int G = n2 >> 2;
            constexpr int kRB = RB, kNW = NT / 32;
            for (int g0 = 0; g0 < G; g0 += 32) {
                const int gq = g0 + lane;
                const bool act = gq < G;
                for (int r0 = warp; r0 < rows; r0 += kRB * kNW) {
                    float4 a[kRB], b[kRB];
#pragma unroll
                    for (int u = 0; u < kRB; ++u) {
                        const int r = r0 + u * kNW;
                        a[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                        b[u] = a[u];
                        if (r < rows && act) {
                            const RowInfo ri = rinfo[c0 - t.I0 + r];
                            if (ri.base_a >= 0) a[u] = __ldg(reinterpret_cast<const float4 *>(img + ri.base_a) + gq);
                            if (ri.base_b >= 0) b[u] = __ldg(reinterpret_cast<const float4 *>(img + ri.base_b) + gq);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < kRB; ++u) {
                        const int r = r0 + u * kNW;
                        if (r >= rows) break; // warp-uniform
                        const RowInfo ri = rinfo[c0 - t.I0 + r];
                        const float c0v = fmaf(ri.wb, b[u].x, ri.wa * a[u].x), c1v = fmaf(ri.wb, b[u].y, ri.wa * a[u].y);
                        const float c2v = fmaf(ri.wb, b[u].z, ri.wa * a[u].z), c3v = fmaf(ri.wb, b[u].w, ri.wa * a[u].w);
                        float c4v = __shfl_down_sync(0xffffffffu, c0v, 1);
                        if (gq >= G - 1) {
                            c4v = 0.f; // z = n2 lies outside the image
                        } else if (lane == 31) { // the neighbour group is in the next pass
                            const float fa = (ri.base_a >= 0) ? __ldg(img + ri.base_a + 4 * gq + 4) : 0.f;
                            const float fb = (ri.base_b >= 0) ? __ldg(img + ri.base_b + 4 * gq + 4) : 0.f;
                            c4v = fmaf(ri.wb, fb, ri.wa * fa);
                        }
                        if (act) {
                            float4 *dst = reinterpret_cast<float4 *>(C2 + r * P + kPad + 4 * gq);
                            const float z0 = (float)(4 * gq) - kc;
                            const float2 e0 = mk(c0v, c1v - c0v, z0), e1 = mk(c1v, c2v - c1v, z0 + 1.f);
                            const float2 e2 = mk(c2v, c3v - c2v, z0 + 2.f), e3 = mk(c3v, c4v - c3v, z0 + 3.f);
                            dst[0] = make_float4(e0.x, e0.y, e1.x, e1.y);
                            dst[1] = make_float4(e2.x, e2.y, e3.x, e3.y);
                            if (gq == 0) C2[r * P + kPad - 1] = mk(0.f, c0v, -1.f - kc);
                        }
                    }
                }
            }
        } else {
            const int ld = n2 + 1; // columns z = -1 .. n2-1
            for (int e = tid; e < rows * ld; e += NT) {
                const int r = e / ld, z = e - r * ld - 1;
                const RowInfo ri = rinfo[c0 - t.I0 + r];
                float v0 = 0.f, v1 = 0.f;
                if (z >= 0) {
                    const float fa = (ri.base_a >= 0) ? __ldg(img + ri.base_a + z) : 0.f;
                    const float fb = (ri.base_b >= 0) ? __ldg(img + ri.base_b + z) : 0.f;
                    v0 = fmaf(ri.wb, fb, ri.wa * fa);
                }
                if (z + 1 < n2) {
                    const float fa = (ri.base_a >= 0) ? __ldg(img + ri.base_a + z + 1) : 0.f;
                    const float fb = (ri.base_b >= 0) ? __ldg(img + ri.base_b + z + 1) : 0.f;
                    v1 = fmaf(ri.wb, fb, ri.wa * fa);
                }
                C2[r * P + kPad + z] = mk(v0, v1 - v0, (float)z - kc);
            }
        }
}

} // namespace tile
} // namespace jp
