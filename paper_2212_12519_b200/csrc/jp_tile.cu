// jp_tile.cu -- non-TOF forward / back projection, tiled: the kernels behind jp_fwd / jp_back.
//
// A CTA takes a tile of 768 consecutive LORs (3 per thread).  LOR lists of ring scanners are full of
// runs of LORs that share their transaxial projection (same xs, ys, xe, ye; only z differs): the ring
// pairs of one sinogram bin (configs[1], [2]: 2304 in a row), or the events of one crystal pair after
// sorting.  For such a *track* tile (checked at run time, bit-exactly) and principal axis x or y, the
// in-plane coordinate along q1, its floor and weight are the same for every LOR of the tile, so
// Joseph's bilinear interpolation factorises:
//
//   forward   C[i][z] = (1-w1(i)) f[i,k1(i),z] + w1(i) f[i,k1(i)+1,z]      built once per tile in shared
//             p_j     = cf_j * sum_i lerp_z(C[i][.], u2_j(i))               memory, 2 LDS + ~13 instr/step
//   adjoint   C[i][z] += cf_j y_j * hat(u2_j(i) - z)                        native int32 shared atomics on a
//             img[i,k1,z] += (1-w1) C[i][z];  img[i,k1+1,z] += w1 C[i][z]   fixed-point tile, then coalesced REDs
//
// Planes are processed in chunks of 64 rows, so shared memory is 64 x (n2+4) x 4 B whatever the image.
// Tiles that are not tracks (ragged tail, principal axis z, unsorted lists) take the generic per-LOR
// path in the same launch.  No plan, no scratch memory, results in caller order.
#include "jp_internal.h"

namespace jp {

namespace {

constexpr int kThreads = 256;
constexpr int kPerThread = 3;
constexpr int kTile = kThreads * kPerThread;
constexpr int kChunk = 64;
constexpr float kMagic = 12582912.f;   // 1.5 * 2^23: (x + kMagic) rounds x to the nearest integer
constexpr int kMagicI = 0x4B400000;    // bit pattern of kMagic
constexpr int kPad = 2;                // zero columns on both sides of a shared-memory row

// shared per-tile track description, written by thread 0
struct Track {
    int p;          // principal axis (0 or 1); -1: not a track tile
    int I0, I1;     // plane range of the track (closed segment rule and q1 clip); empty if I1 < I0
    float a1, b1;   // u_q1(i) = a1 + b1 (i - I0)
    double inv_dp;  // 1 / d_p
    double ops;     // o_p - s_p
    float R;        // 1 + (d_q1/d_p)^2
};

__device__ __forceinline__ bool same_bits(float a, float b) { return __float_as_uint(a) == __float_as_uint(b); }

// the part of ray_setup that only depends on the shared transaxial end points (float64, once per tile)
__device__ void track_setup(const Geom &g, float xs, float ys, float xe, float ye, Track &t)
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
    double flo = ceil((lo - op) / vp), fhi = floor((hi - op) / vp);
    flo = fmin(fmax(flo, 0.0), np1 + 1.0);
    fhi = fmin(fmax(fhi, -1.0), np1);
    int ilo = (int)flo, ihi = (int)fhi;
    if (ilo > 0 && op + (double)(ilo - 1) * vp >= lo) --ilo;
    if (ilo <= g.n[p] - 1 && op + (double)ilo * vp < lo) ++ilo;
    if (ihi < g.n[p] - 1 && op + (double)(ihi + 1) * vp <= hi) ++ihi;
    if (ihi >= 0 && op + (double)ihi * vp > hi) --ihi;
    const double inv_dp = 1.0 / d[p];
    const double ratio = d[q1] * inv_dp;
    const double ivq = 1.0 / (double)g.v[q1];
    const double B = ratio * vp * ivq;
    const double A = (s[q1] - (double)g.o[q1] + (op - sp) * ratio) * ivq;
    const double nq = (double)g.n[q1];
    if (B == 0.0) {
        if (A <= -1.0 || A >= nq) ihi = ilo - 1;
    } else {
        const double ia = (-1.0 - A) / B, ib = (nq - A) / B;
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
}

// per-LOR axial part: u2(i) = a2h + 0.5 + b2 (i - i0), planes [i0, i1], incidence factor cf
struct ZRay {
    int i0, i1;
    float a2h, b2, cf;
};

__device__ __forceinline__ ZRay z_setup(const Geom &g, const Track &t, float zs, float ze)
{
    ZRay z;
    const double dz = (double)ze - (double)zs;
    const double rz = dz * t.inv_dp;
    const double vp = (double)g.v[t.p];
    const double iv2 = 1.0 / (double)g.v[2];
    const double B = rz * vp * iv2;
    const double A = ((double)zs - (double)g.o[2] + t.ops * rz) * iv2;
    const float rzf = (float)rz;
    z.cf = g.v[t.p] * sqrtf(fmaf(rzf, rzf, t.R));
    // clip to -1 < u2 < n2 (float32 estimate widened by one plane, then trimmed against the padded row)
    int ilo = t.I0, ihi = t.I1;
    const float Af = (float)A, Bf = (float)B, n2 = (float)g.n[2];
    if (Bf == 0.f) {
        if (Af <= -1.f || Af >= n2) ihi = ilo - 1;
    } else {
        const float inv = 1.f / Bf;
        const float ia = (-1.f - Af) * inv, ib = (n2 - Af) * inv;
        const float imin = fminf(fmaxf(floorf(fminf(ia, ib)) - 1.f, -1.f), (float)g.n[t.p]);
        const float imax = fminf(fmaxf(ceilf(fmaxf(ia, ib)) + 1.f, -1.f), (float)g.n[t.p]);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    z.b2 = Bf;
    z.a2h = (float)(A + B * (double)ilo - 0.5);
    // trim: the rounded index must stay inside the padded row: -2 <= round(u2 - 1/2) <= n2
    const float hmin = -2.4f, hmax = n2 + 0.4f;
    while (ilo <= ihi) {
        const float h = z.a2h;
        if (h > hmin && h < hmax) break;
        ++ilo;
        z.a2h = (float)(A + B * (double)ilo - 0.5);
    }
    while (ilo <= ihi) {
        const float h = fmaf(z.b2, (float)(ihi - ilo), z.a2h);
        if (h > hmin && h < hmax) break;
        --ihi;
    }
    z.i0 = ilo;
    z.i1 = ihi;
    return z;
}

// generic per-LOR forward / back (any axis, any order): same arithmetic as jp_kernels.cu
__device__ __forceinline__ float generic_fwd(const Lors &l, int64_t j, const Geom &g, const float *__restrict__ img)
{
    Ray r;
    ray_setup<false>(l, j, g, 0.f, 0.f, 0.f, r);
    float acc = 0.f;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        acc += plane_value(img, r, k, cl);
    }
    return r.cf * acc;
}

__device__ __forceinline__ void generic_back(const Lors &l, int64_t j, const Geom &g, float y, float *__restrict__ img)
{
    Ray r;
    ray_setup<false>(l, j, g, 0.f, 0.f, 0.f, r);
    const float x = r.cf * y;
    if (r.nk == 0 || x == 0.f) return;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        plane_scatter(img, r, k, cl, x);
    }
}

// is this tile a track?  all 768 LORs valid, identical transaxial end points, principal axis x or y
__device__ __forceinline__ bool tile_is_track(const Lors &l, int64_t j0, int64_t n, const float (&zs)[kPerThread],
                                              const float (&ze)[kPerThread], float xs0, float ys0, float xe0, float ye0)
{
    bool ok = (j0 + kTile <= n);
    if (ok) {
        const double dmax = fmax(fabs((double)xe0 - (double)xs0), fabs((double)ye0 - (double)ys0));
        ok = dmax > 0.0;
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int64_t j = j0 + m * kThreads + threadIdx.x;
            ok = ok && same_bits(l.xs[j], xs0) && same_bits(l.ys[j], ys0) && same_bits(l.xe[j], xe0) &&
                 same_bits(l.ye[j], ye0) && (fabs((double)ze[m] - (double)zs[m]) <= dmax);
        }
    }
    return __syncthreads_and(ok) != 0;
}

// row r of the chunk: q1 cell of plane i (shared by the whole tile)
struct RowCell {
    int base;     // element offset of (i, k1, z=0)
    float w1;
    bool in_a, in_b;
};

__device__ __forceinline__ RowCell row_cell(const Geom &g, const Track &t, int i)
{
    const int q1 = 1 - t.p;
    const int st[2] = {g.n[1] * g.n[2], g.n[2]};
    const float u1 = fmaf(t.b1, (float)(i - t.I0), t.a1);
    const float f1 = floorf(u1);
    const int k1 = (int)f1;
    RowCell c;
    c.w1 = u1 - f1;
    c.in_a = (unsigned)k1 < (unsigned)g.n[q1];
    c.in_b = (unsigned)(k1 + 1) < (unsigned)g.n[q1];
    c.base = i * st[t.p] + k1 * st[q1];
    return c;
}

} // namespace

// ---- forward ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) k_fwd_tile(Lors l, int64_t n, const float *__restrict__ img, Geom g,
                                                       float *__restrict__ p)
{
    extern __shared__ float C[]; // [kChunk][ld]
    __shared__ Track trk;
    const int tid = threadIdx.x;
    const int64_t j0 = blockIdx.x * (int64_t)kTile;
    const int ld = g.n[2] + 2 * kPad;

    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        const int64_t j = j0 + m * kThreads + tid;
        zs[m] = (j < n) ? l.zs[j] : 0.f;
        ze[m] = (j < n) ? l.ze[j] : 0.f;
    }
    const float xs0 = l.xs[j0], ys0 = l.ys[j0], xe0 = l.xe[j0], ye0 = l.ye[j0];
    if (!tile_is_track(l, j0, n, zs, ze, xs0, ys0, xe0, ye0)) {
#pragma unroll 1
        for (int m = 0; m < kPerThread; ++m) {
            const int64_t j = j0 + m * kThreads + tid;
            if (j < n) p[j] = generic_fwd(l, j, g, img);
        }
        return;
    }
    if (tid == 0) track_setup(g, xs0, ys0, xe0, ye0, trk);
    __syncthreads();
    const Track t = trk;
    if (t.I1 < t.I0) { // the whole track misses the image
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) p[j0 + m * kThreads + tid] = 0.f;
        return;
    }
    ZRay zr[kPerThread];
    float acc[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        zr[m] = z_setup(g, t, zs[m], ze[m]);
        acc[m] = 0.f;
    }
    const int warp = tid >> 5, lane = tid & 31;
    const int s1 = (t.p == 0) ? g.n[2] : g.n[1] * g.n[2];

    for (int c0 = t.I0; c0 <= t.I1; c0 += kChunk) {
        const int rows = min(kChunk, t.I1 - c0 + 1);
        // ---- build C: one warp per row, lanes along z (coalesced image reads)
        for (int r = warp; r < rows; r += kThreads / 32) {
            const RowCell rc = row_cell(g, t, c0 + r);
            const float wa = 1.f - rc.w1, wb = rc.w1;
            const float *ra = img + (rc.in_a ? rc.base : 0);
            const float *rb = img + (rc.in_b ? rc.base + s1 : 0);
            for (int zc = lane; zc < ld; zc += 32) {
                const int z = zc - kPad;
                float v = 0.f;
                if ((unsigned)z < (unsigned)g.n[2]) {
                    const float fa = rc.in_a ? __ldg(ra + z) : 0.f; // neighbours outside the image count as zero
                    const float fb = rc.in_b ? __ldg(rb + z) : 0.f;
                    v = fmaf(wb, fb, wa * fa);
                }
                C[r * ld + zc] = v;
            }
        }
        __syncthreads();
        // ---- consume: every LOR walks its planes of this chunk, interpolating along z only
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int ib = max(zr[m].i0, c0), ie = min(zr[m].i1, c0 + rows - 1);
            if (ib > ie) continue;
            float fk = (float)(ib - zr[m].i0);
            int off = (ib - c0) * ld + kPad - kMagicI;
            const float a2h = zr[m].a2h, b2 = zr[m].b2;
            float a = acc[m];
#pragma unroll 4
            for (int i = ib; i <= ie; ++i) {
                const float h = fmaf(b2, fk, a2h);   // u2 - 1/2
                const float tt = h + kMagic;           // integer part in the low mantissa bits
                const float w = (h - (tt - kMagic)) + 0.5f;
                const int idx = __float_as_int(tt) + off;
                const float v0 = C[idx], v1 = C[idx + 1];
                a += fmaf(w, v1 - v0, v0);
                fk += 1.f;
                off += ld;
            }
            acc[m] = a;
        }
        __syncthreads();
    }
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) p[j0 + m * kThreads + tid] = zr[m].cf * acc[m];
}

// ---- back ------------------------------------------------------------------------------------------------
// Fixed-point staging: contributions are rounded to multiples of 1/S and summed with native int32
// shared-memory atomics (ATOMS.ADD; float shared atomics are CAS loops on sm_100).  S is chosen per
// tile from X = max_j |cf_j y_j| so that neither a single contribution (|c S| < 2^22, the range of the
// magic-number rounding) nor a whole bin (at most one contribution per LOR and plane: |sum| <= 768 X S
// < 2^31) can overflow.  Rounding error per contribution <= X 768 / 2^32 = 1.8e-7 X.
__global__ void __launch_bounds__(kThreads) k_back_tile(Lors l, int64_t n, const float *__restrict__ y, Geom g,
                                                        float *__restrict__ img)
{
    extern __shared__ int Ci[]; // [kChunk][ld]
    __shared__ Track trk;
    __shared__ float red[kThreads / 32];
    const int tid = threadIdx.x;
    const int64_t j0 = blockIdx.x * (int64_t)kTile;
    const int ld = g.n[2] + 2 * kPad;

    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        const int64_t j = j0 + m * kThreads + tid;
        zs[m] = (j < n) ? l.zs[j] : 0.f;
        ze[m] = (j < n) ? l.ze[j] : 0.f;
    }
    const float xs0 = l.xs[j0], ys0 = l.ys[j0], xe0 = l.xe[j0], ye0 = l.ye[j0];
    if (!tile_is_track(l, j0, n, zs, ze, xs0, ys0, xe0, ye0)) {
#pragma unroll 1
        for (int m = 0; m < kPerThread; ++m) {
            const int64_t j = j0 + m * kThreads + tid;
            if (j < n) generic_back(l, j, g, y[j], img);
        }
        return;
    }
    if (tid == 0) track_setup(g, xs0, ys0, xe0, ye0, trk);
    __syncthreads();
    const Track t = trk;
    if (t.I1 < t.I0) return;

    ZRay zr[kPerThread];
    float x[kPerThread];
    float xmax = 0.f;
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        zr[m] = z_setup(g, t, zs[m], ze[m]);
        x[m] = zr[m].cf * y[j0 + m * kThreads + tid];
        if (zr[m].i1 >= zr[m].i0) xmax = fmaxf(xmax, fabsf(x[m]));
    }
    // block max of |x|
    for (int o = 16; o > 0; o >>= 1) xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = xmax;
    for (int e = tid; e < kChunk * ld; e += kThreads) Ci[e] = 0;
    __syncthreads();
    xmax = red[0];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) xmax = fmaxf(xmax, red[w]);
    if (!(xmax > 0.f) || !(xmax < 3.0e38f)) return; // nothing to add (or non-finite input: undefined, skip)
    // S: |c S| <= 2^22 - 2 and 768 |c S| < 2^31  ->  |c S| <= 2^31 / 768 - 1
    const float lim = fminf(4194302.f, 2147483648.f / (float)kTile - 1.f);
    const float S = lim / xmax, invS = xmax / lim;
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) x[m] *= S;

    const int warp = tid >> 5, lane = tid & 31;
    const int s1 = (t.p == 0) ? g.n[2] : g.n[1] * g.n[2];

    for (int c0 = t.I0; c0 <= t.I1; c0 += kChunk) {
        const int rows = min(kChunk, t.I1 - c0 + 1);
        // ---- scatter along z into the fixed-point tile
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int ib = max(zr[m].i0, c0), ie = min(zr[m].i1, c0 + rows - 1);
            if (ib > ie || x[m] == 0.f) continue;
            float fk = (float)(ib - zr[m].i0);
            int off = (ib - c0) * ld + kPad - kMagicI;
            const float a2h = zr[m].a2h, b2 = zr[m].b2, xm = x[m];
#pragma unroll 4
            for (int i = ib; i <= ie; ++i) {
                const float h = fmaf(b2, fk, a2h);
                const float tt = h + kMagic;
                const float w = (h - (tt - kMagic)) + 0.5f;
                const int idx = __float_as_int(tt) + off;
                const int q1 = __float_as_int(fmaf(xm, w, kMagic)) - kMagicI;
                const int q0 = __float_as_int(fmaf(xm, 1.f - w, kMagic)) - kMagicI;
                atomicAdd(&Ci[idx], q0);
                atomicAdd(&Ci[idx + 1], q1);
                fk += 1.f;
                off += ld;
            }
        }
        __syncthreads();
        // ---- flush: spread every row over its two q1 neighbours with coalesced REDs, and clear it
        for (int r = warp; r < rows; r += kThreads / 32) {
            const RowCell rc = row_cell(g, t, c0 + r);
            const float wa = (1.f - rc.w1) * invS, wb = rc.w1 * invS;
            float *ra = img + (rc.in_a ? rc.base : 0);
            float *rb = img + (rc.in_b ? rc.base + s1 : 0);
            for (int zc = lane; zc < ld; zc += 32) {
                const int q = Ci[r * ld + zc];
                if (q == 0) continue;
                Ci[r * ld + zc] = 0;
                const int z = zc - kPad;
                if ((unsigned)z < (unsigned)g.n[2]) {
                    const float v = (float)q;
                    if (rc.in_a) atomicAdd(ra + z, wa * v);
                    if (rc.in_b) atomicAdd(rb + z, wb * v);
                }
            }
        }
        __syncthreads();
    }
}

// ---- launchers ----------------------------------------------------------------------------------------------
static inline size_t tile_smem(const Geom &g) { return (size_t)kChunk * (g.n[2] + 2 * kPad) * sizeof(float); }

cudaError_t launch_fwd_tile(const Lors &l, int64_t n, const float *img, const Geom &g, float *p, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const size_t smem = tile_smem(g);
    static thread_local size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(k_fwd_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    k_fwd_tile<<<(unsigned)((n + kTile - 1) / kTile), kThreads, smem, st>>>(l, n, img, g, p);
    return cudaGetLastError();
}

cudaError_t launch_back_tile(const Lors &l, int64_t n, const float *y, const Geom &g, float *img, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const size_t smem = tile_smem(g);
    static thread_local size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(k_back_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    k_back_tile<<<(unsigned)((n + kTile - 1) / kTile), kThreads, smem, st>>>(l, n, y, g, img);
    return cudaGetLastError();
}

size_t tile_smem_bytes(const Geom &g) { return tile_smem(g); }

} // namespace jp
