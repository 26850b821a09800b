// jp_track.cu -- non-TOF forward / back projection of a REGULAR sinogram plan: one CTA per track.
//
// The list-mode tile kernels of jp_tile.cu cut the list into tiles of 768 LORs and rebuild the shared rows
// C[i][z] = (1-w1(i)) f[i,k1(i),z] + w1(i) f[i,k1(i)+1,z]  (Joseph's interpolation factorised along the
// track, see the header of jp_tile.cu) for every tile: a track of 2304 ring pairs builds (forward) or flushes (adjoint)
// its rows three times, and thread 0 of every tile repeats the float64 set-up of the track.  ncu (profiles/r02, commit
// b60463d): the plane loop itself was 38 % of the forward kernel's instructions, the row builds 30 %, the track set-up
// 9 %, lane mapping and bookkeeping the rest.
//
// With a sinogram plan (jp_sino_plan.cu) everything that repeats is known in advance, so here
//   * a CTA of 256 threads takes a WHOLE track (up to 9 LORs per thread: 2304; longer tracks are cut into equal
//     pieces): rows are built / flushed once per track;
//   * the float64 track set-up runs once per call in its own small kernel (k_track_table, one thread per track) and
//     the CTAs read the result: no serial section, no barrier;
//   * the lane order (which LOR a lane takes: decides the shared-memory wavefronts per plane step, see jp_tile.cu)
//     is computed on the host when the plan is made; the kernels read the axial end points already in that order;
//   * the image rows are combined with all 32 lanes busy (linear (row, 4-voxel group) index instead of one warp per
//     row: 24 groups per 96-voxel row left a quarter of the lanes idle).
// The arithmetic of a plane step, the fixed-point staging of the adjoint and the handling of non-finite values are
// those of jp_tile.cu; results differ from the list kernels only by the order of floating-point additions.
#include "jp_f32x2.cuh"
#include "jp_tile_common.cuh"

namespace jp {

using namespace tile;

namespace {

constexpr int kTT = 256; // threads per CTA

// Launch settings from sweeps on B200 (configs[1], forward / back ms): 3 CTAs per SM and 72 KB of forward rows 3.53 / 4.08;
// 4 CTAs (64 registers, ~80 bytes of spills) and 52 KB 3.41 / 4.04; 48 KB 3.32 / 4.04; 40 KB 3.32; 32 KB 3.42; 5 CTAs
// (48 registers) 3.99 / 4.39.  The forward kernel waits on shared / global loads (24 warps per SM at 3 CTAs): the
// fourth CTA hides more of that than the spills and the extra row chunks cost.
#ifndef JP_TRK_MINB9
#define JP_TRK_MINB9 4 // CTAs per SM with 9 LORs per thread (register budget 64)
#endif
#ifndef JP_TRK_SMEM_KB_FWD
#define JP_TRK_SMEM_KB_FWD 48
#endif
#ifndef JP_TRK_SMEM_KB_BACK
#define JP_TRK_SMEM_KB_BACK 44
#endif

enum : int { kTrackTile = 0, kTrackPerLor = 1, kTrackMiss = 2 };

struct TrkSrc {
    const float4 *trk; // [K] (xs, ys, xe, ye)
    const Track *tab;  // [K] track set-up for this call's image geometry
    const int *kind;   // [K] kTrackTile / kTrackPerLor (a LOR may have principal axis z) / kTrackMiss
    const float2 *zp;  // [npieces][slots] (zs, ze) in lane order
    const int *ord;    // [npieces][slots] index of the slot's LOR inside the track, -1: empty slot
    int T, npieces, slots;
};

// kTrackMiss: the transaxial line stays outside the circle around the footprint of the image extended by one voxel
// (-1 < u < n on both axes) -- no LOR of the track, whatever its axial end points and principal axis, touches a voxel
// (in a ring scanner that is every sinogram bin near the edge of the radial range: short chords far from the centre,
// which are also the ones that may be steeper than they are long).  A zero-length transaxial projection (dmax = 0:
// all LORs parallel to z) is left to the per-LOR path.
__global__ void k_track_table(const float4 *__restrict__ trk, int64_t K, Geom g, double dz_max, Track *__restrict__ tab,
                              int *__restrict__ kind)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= K) return;
    const float4 q = trk[k];
    Track t;
    track_setup(g, q.x, q.y, q.z, q.w, t);
    tab[k] = t;
    const double dx = (double)q.z - (double)q.x, dy = (double)q.w - (double)q.y;
    const double dmax = fmax(fabs(dx), fabs(dy));
    int kd = (dmax > 0.0 && dz_max <= dmax) ? kTrackTile : kTrackPerLor;
    if (dmax > 0.0) {
        const double w0 = 0.5 * (double)(g.n[0] + 1) * (double)g.v[0], w1 = 0.5 * (double)(g.n[1] + 1) * (double)g.v[1];
        const double cx = (double)g.o[0] + 0.5 * (double)(g.n[0] - 1) * (double)g.v[0];
        const double cy = (double)g.o[1] + 0.5 * (double)(g.n[1] - 1) * (double)g.v[1];
        const double cr = dx * (cy - (double)q.y) - dy * (cx - (double)q.x); // |cr| / |d| = distance of the line from the centre
        const double rad = sqrt(w0 * w0 + w1 * w1) * (1.0 + 1e-9) + 1e-6;
        if (cr * cr > rad * rad * (dx * dx + dy * dy)) kd = kTrackMiss;
    }
    kind[k] = kd;
}

__device__ __forceinline__ int pack_planes(int i0, int i1) { return (i1 >= i0) ? (i0 | (i1 << 16)) : 1; } // 1: i0 = 1 > i1 = 0

// ---- (intercept, slope) rows of planes [c0, c0 + rows): all lanes busy ------------------------------------------
// entry e = r G + gq (G = n2 / 4 groups of four voxels per row); magicG = ceil(2^32 / G)
template <int P>
__device__ __forceinline__ void build_rows_lin(float2 *C2, const RowInfo *ri_c, const float *__restrict__ img, int rows,
                                               int n2, float kc, unsigned magicG)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int G = n2 >> 2, total = rows * G;
    auto mk = [&](float v, float d, float zrel) { return make_float2(fmaf(-zrel, d, v), d); };
#pragma unroll 2
    for (int e0 = 0; e0 < total; e0 += kTT) { // warp-uniform trip count
        const int e = e0 + tid;
        const bool act = e < total;
        const int r = act ? (int)__umulhi((unsigned)e, magicG) : 0;
        const int gq = act ? e - r * G : G - 1;
        const RowInfo ri = ri_c[r];
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
        if (act) {
            if (ri.base_a >= 0) a = __ldg(reinterpret_cast<const float4 *>(img + ri.base_a) + gq);
            if (ri.base_b >= 0) b = __ldg(reinterpret_cast<const float4 *>(img + ri.base_b) + gq);
        }
        const float c0v = fmaf(ri.wb, b.x, ri.wa * a.x), c1v = fmaf(ri.wb, b.y, ri.wa * a.y);
        const float c2v = fmaf(ri.wb, b.z, ri.wa * a.z), c3v = fmaf(ri.wb, b.w, ri.wa * a.w);
        float c4v = __shfl_down_sync(0xffffffffu, c0v, 1); // lane + 1 holds (r, gq + 1) when gq < G - 1
        if (gq == G - 1) {
            c4v = 0.f; // z = n2 lies outside the image
        } else if (lane == 31) {
            const float fa = (ri.base_a >= 0) ? __ldg(img + ri.base_a + 4 * gq + 4) : 0.f;
            const float fb = (ri.base_b >= 0) ? __ldg(img + ri.base_b + 4 * gq + 4) : 0.f;
            c4v = fmaf(ri.wb, fb, ri.wa * fa);
        }
        if (act) {
            float4 *dst = reinterpret_cast<float4 *>(C2 + r * P + kPad + 4 * gq);
            const float z0 = (float)(4 * gq) - kc;
            const float2 e0v = mk(c0v, c1v - c0v, z0), e1v = mk(c1v, c2v - c1v, z0 + 1.f);
            const float2 e2v = mk(c2v, c3v - c2v, z0 + 2.f), e3v = mk(c3v, c4v - c3v, z0 + 3.f);
            dst[0] = make_float4(e0v.x, e0v.y, e1v.x, e1v.y);
            dst[1] = make_float4(e2v.x, e2v.y, e3v.x, e3v.y);
            if (gq == 0) C2[r * P + kPad - 1] = mk(0.f, c0v, -1.f - kc);
        }
    }
}

template <int OFF>
__device__ __forceinline__ void reds_add(uint32_t addr, int q)
{
    asm volatile("red.shared.add.s32 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "r"(q) : "memory");
}

__device__ __forceinline__ float generic_fwd_pts(const double (&s)[3], const double (&e)[3], const Geom &g,
                                                 const float *__restrict__ img)
{
    Ray r;
    ray_setup_pts<false>(s, e, g, 0.f, 0.f, 0.f, r);
    float acc = 0.f;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        acc += plane_value(img, r, k, cl);
    }
    return r.cf * acc;
}

__device__ __forceinline__ void generic_back_pts(const double (&s)[3], const double (&e)[3], const Geom &g, float y,
                                                 float *__restrict__ img)
{
    Ray r;
    ray_setup_pts<false>(s, e, g, 0.f, 0.f, 0.f, r);
    const float x = r.cf * y;
    if (r.nk == 0 || x == 0.f) return;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        plane_scatter(img, r, k, cl, x);
    }
}

// chunks of equal size: the planes [I0, I1] of the track in ceil(n / rows_cap) chunks
__device__ __forceinline__ int chunk_rows(int nrows, int rows_cap)
{
    const int nch = (nrows + rows_cap - 1) / rows_cap;
    return (nrows + nch - 1) / nch;
}

} // namespace

// ---- forward ------------------------------------------------------------------------------------------
#define JP_FWD_STEP(K, A2K)                                                    \
    {                                                                          \
        const float u = fmaf(b2, fk, A2K);                                     \
        const float tt = __fadd_rd(u, kMagic);                                 \
        const float2 v = lds_pair<(K) * P * 8>(row + (__float_as_uint(tt) << 3)); \
        acc0 += v.x;                                                           \
        acc1 = fmaf(u, v.y, acc1);                                             \
    }
#define JP_FWD_STEP2(K, A2P)                                                   \
    {                                                                          \
        const F2 U = fma2(b2p, f2(fk), A2P);                                   \
        const F2 TT = add2_rm(U, f2(kMagic));                                  \
        const float2 v0 = lds_pair<(K) * P * 8>(row + (__float_as_uint(f2_lo(TT)) << 3));       \
        const float2 v1 = lds_pair<((K) + 1) * P * 8>(row + (__float_as_uint(f2_hi(TT)) << 3)); \
        acc0 += v0.x;                                                          \
        acc1 = fmaf(f2_lo(U), v0.y, acc1);                                     \
        acc0 += v1.x;                                                          \
        acc1 = fmaf(f2_hi(U), v1.y, acc1);                                     \
    }

template <int P, int NPT>
__global__ void __launch_bounds__(kTT, NPT > 6 ? JP_TRK_MINB9 : 4)
    k_fwd_track(TrkSrc ts, const float *__restrict__ img, Geom g, int rows_cap, int vec_ok, unsigned magicG,
                float *__restrict__ p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *C2 = reinterpret_cast<float2 *>(smem_raw);                                      // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(float2)); // [max(n0,n1)]
    const int tid = threadIdx.x;
    int64_t trk = blockIdx.x;
    int piece = 0;
    if (ts.npieces > 1) {
        trk = blockIdx.x / ts.npieces;
        piece = (int)(blockIdx.x - trk * ts.npieces);
    }
    const float4 q = __ldg(ts.trk + trk);
    const float2 *__restrict__ zp = ts.zp + (size_t)piece * ts.slots;
    const int *__restrict__ ord = ts.ord + (size_t)piece * ts.slots;
    float *__restrict__ pt = p + trk * (int64_t)ts.T;
    const int kind = __ldg(ts.kind + trk);
    if (kind == kTrackPerLor) { // a LOR of the track may have principal axis z
#pragma unroll 1
        for (int m = 0; m < NPT; ++m) {
            const int slot = m * kTT + tid, o = ord[slot];
            if (o < 0) continue;
            const float2 zz = zp[slot];
            const double sp[3] = {(double)q.x, (double)q.y, (double)zz.x}, ep[3] = {(double)q.z, (double)q.w, (double)zz.y};
            pt[o] = generic_fwd_pts(sp, ep, g, img);
        }
        return;
    }
    const Track t = ts.tab[trk];
    if (kind == kTrackMiss || t.I1 < t.I0) { // the whole track misses the image
#pragma unroll 1
        for (int m = 0; m < NPT; ++m) {
            const int o = ord[m * kTT + tid];
            if (o >= 0) pt[o] = 0.f;
        }
        return;
    }
    const int n2 = g.n[2];
    const int kci = n2 >> 1; // axial shift of the (intercept, slope) rows
    const float kc = (float)kci;
    const int nrows = t.I1 - t.I0 + 1;
    for (int r = tid; r < nrows; r += kTT) rinfo[r] = row_info(g, t, t.I0 + r);
    {
        const int ncl = kPad - 1, ncr = P - (n2 + kPad);
        for (int e = tid; e < rows_cap * (ncl + ncr); e += kTT) {
            const int r = e / (ncl + ncr), c = e - r * (ncl + ncr);
            C2[r * P + (c < ncl ? c : n2 + kPad + (c - ncl))] = make_float2(0.f, 0.f);
        }
    }
    float a2[NPT], b2v[NPT], acc0v[NPT], acc1v[NPT];
    int i01[NPT];
#pragma unroll
    for (int m = 0; m < NPT; ++m) {
        const int slot = m * kTT + tid;
        const float2 zz = __ldg(zp + slot);
        const ZRay zr = z_setup(g, t, zz.x, zz.y, (double)kci);
        a2[m] = zr.a2;
        b2v[m] = zr.b2;
        i01[m] = (__ldg(ord + slot) >= 0) ? pack_planes(zr.i0, zr.i1) : 1;
        acc0v[m] = 0.f;
        acc1v[m] = 0.f;
    }
    const uint32_t c2_base = smem_addr(C2) + (uint32_t)(kPad + kci) * 8u - ((uint32_t)kMagicI << 3);
    const int rpc = chunk_rows(nrows, rows_cap);
    __syncthreads();

    for (int c0 = t.I0; c0 <= t.I1; c0 += rpc) {
        const int rows = min(rpc, t.I1 - c0 + 1);
        if (vec_ok) build_rows_lin<P>(C2, rinfo + (c0 - t.I0), img, rows, n2, kc, magicG);
        else build_rows<P, true, 1, kTT>(C2, rinfo, img, t, c0, rows, n2, 0, kc);
        __syncthreads();
#pragma unroll
        for (int m = 0; m < NPT; ++m) {
            const int i0 = i01[m] & 0xffff, i1 = i01[m] >> 16;
            const int ib = max(i0, c0), ie = min(i1, c0 + rows - 1);
            if (ib > ie) continue;
            const float b2 = b2v[m], a2_0 = a2[m];
            const float a2_1 = fmaf(b2, 1.f, a2_0), a2_2 = fmaf(b2, 2.f, a2_0), a2_3 = fmaf(b2, 3.f, a2_0);
            float fk = (float)(ib - i0);
            uint32_t row = c2_base + (uint32_t)((ib - c0) * P) * 8u;
            float acc0 = acc0v[m], acc1 = acc1v[m];
            int left = ie - ib + 1;
            const F2 b2p = f2(b2), a2p01 = f2(a2_0, a2_1), a2p23 = f2(a2_2, a2_3);
            const F2 a2p45 = f2(fmaf(b2, 4.f, a2_0), fmaf(b2, 5.f, a2_0)), a2p67 = f2(fmaf(b2, 6.f, a2_0), fmaf(b2, 7.f, a2_0));
#pragma unroll 1
            for (; left >= 8; left -= 8) {
                JP_FWD_STEP2(0, a2p01)
                JP_FWD_STEP2(2, a2p23)
                JP_FWD_STEP2(4, a2p45)
                JP_FWD_STEP2(6, a2p67)
                fk += 8.f;
                row += 8u * P * 8u;
            }
            if (left >= 4) {
                JP_FWD_STEP2(0, a2p01)
                JP_FWD_STEP2(2, a2p23)
                fk += 4.f;
                row += 4u * P * 8u;
            }
#pragma unroll 1
            for (int it = left & 3; it > 0; --it) {
                JP_FWD_STEP(0, a2_0)
                fk += 1.f;
                row += P * 8u;
            }
            acc0v[m] = acc0;
            acc1v[m] = acc1;
        }
        __syncthreads();
    }
    const float vp = g.v[t.p];
#pragma unroll
    for (int m = 0; m < NPT; ++m) {
        const int slot = m * kTT + tid, o = __ldg(ord + slot);
        if (o < 0) continue;
        const float2 zz = __ldg(zp + slot);
        const float rzf = (float)(((double)zz.y - (double)zz.x) * t.inv_dp); // the incidence factor of z_setup
        pt[o] = vp * sqrtf(fmaf(rzf, rzf, t.R)) * (acc0v[m] + acc1v[m]);
    }
}
#undef JP_FWD_STEP
#undef JP_FWD_STEP2

// ---- back ------------------------------------------------------------------------------------------------
// fixed-point staging as in jp_tile.cu; the bound on a bin's sum uses the LORs of the piece (2 x slots x |c S| < 2^31)
#define JP_BACK_STEP(K, A2K)                                                   \
    {                                                                          \
        const float u = fmaf(b2, fk, A2K);                                     \
        const float tt = __fadd_rd(u, kMagic);                                 \
        const float w = u - (tt - kMagic);                                     \
        const uint32_t a = row + (__float_as_uint(tt) << 2);                   \
        const int bits = __float_as_int(fmaf(xm, w, kMagic));                  \
        reds_add<(K) * P * 4>(a, qxm - bits);                                  \
        reds_add<(K) * P * 4 + 4>(a, bits - kMagicI);                          \
    }
#define JP_BACK_STEP2(K, A2P)                                                  \
    {                                                                          \
        const F2 U = fma2(b2p, f2(fk), A2P);                                   \
        const F2 TT = add2_rm(U, f2(kMagic));                                  \
        const F2 Tm = add2(TT, f2(-kMagic));                                   \
        const F2 W = fma2(Tm, f2(-1.f), U);                                    \
        const F2 B = fma2(xmp, W, f2(kMagic));                                 \
        const uint32_t a0 = row + (__float_as_uint(f2_lo(TT)) << 2);           \
        const uint32_t a1 = row + (__float_as_uint(f2_hi(TT)) << 2);           \
        const int b0 = __float_as_int(f2_lo(B)), b1 = __float_as_int(f2_hi(B)); \
        reds_add<(K) * P * 4>(a0, qxm - b0);                                   \
        reds_add<(K) * P * 4 + 4>(a0, b0 - kMagicI);                           \
        reds_add<((K) + 1) * P * 4>(a1, qxm - b1);                             \
        reds_add<((K) + 1) * P * 4 + 4>(a1, b1 - kMagicI);                     \
    }

template <int P, int NPT>
__global__ void __launch_bounds__(kTT, NPT > 6 ? JP_TRK_MINB9 : 4)
    k_back_track(TrkSrc ts, const float *__restrict__ y, Geom g, int rows_cap, int vec_ok, unsigned magicG,
                 float *__restrict__ img)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int *Ci = reinterpret_cast<int *>(smem_raw);                                        // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(int)); // [max(n0,n1)]
    __shared__ float red[kTT / 32];
    __shared__ int sh_bad;
    const int tid = threadIdx.x;
    int64_t trk = blockIdx.x;
    int piece = 0;
    if (ts.npieces > 1) {
        trk = blockIdx.x / ts.npieces;
        piece = (int)(blockIdx.x - trk * ts.npieces);
    }
    const float4 q = __ldg(ts.trk + trk);
    const float2 *__restrict__ zp = ts.zp + (size_t)piece * ts.slots;
    const int *__restrict__ ord = ts.ord + (size_t)piece * ts.slots;
    const float *__restrict__ yt = y + trk * (int64_t)ts.T;
    const int kind = __ldg(ts.kind + trk);
    if (kind == kTrackMiss) return;
    auto per_lor = [&]() {
#pragma unroll 1
        for (int m = 0; m < NPT; ++m) {
            const int slot = m * kTT + tid, o = ord[slot];
            if (o < 0) continue;
            const float2 zz = zp[slot];
            const double sp[3] = {(double)q.x, (double)q.y, (double)zz.x}, ep[3] = {(double)q.z, (double)q.w, (double)zz.y};
            generic_back_pts(sp, ep, g, yt[o], img);
        }
    };
    if (kind == kTrackPerLor) {
        per_lor();
        return;
    }
    const Track t = ts.tab[trk];
    if (t.I1 < t.I0) return;
    if (tid == 0) sh_bad = 0;
    const int n2 = g.n[2];
    const int nrows = t.I1 - t.I0 + 1;

    float a2[NPT], b2v[NPT], x[NPT];
    int i01[NPT];
    float xmax = 0.f;
    bool bad = false;
#pragma unroll
    for (int m = 0; m < NPT; ++m) {
        const int slot = m * kTT + tid, o = __ldg(ord + slot);
        const float2 zz = __ldg(zp + slot);
        const ZRay zr = z_setup(g, t, zz.x, zz.y);
        a2[m] = zr.a2;
        b2v[m] = zr.b2;
        i01[m] = (o >= 0) ? pack_planes(zr.i0, zr.i1) : 1;
        x[m] = (o >= 0) ? zr.cf * yt[o] : 0.f;
        if (i01[m] != 1) {
            const float ax = fabsf(x[m]);
            bad = bad || !(ax < 3.0e38f); // Inf or NaN (fmaxf would drop a NaN)
            xmax = fmaxf(xmax, ax);
        }
    }
    for (int o = 16; o > 0; o >>= 1) xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
    __syncthreads(); // sh_bad cleared
    if (bad) atomicExch(&sh_bad, 1);
    if ((tid & 31) == 0) red[tid >> 5] = xmax;
    for (int r = tid; r < nrows; r += kTT) rinfo[r] = row_info(g, t, t.I0 + r);
    {
        int4 *z4 = reinterpret_cast<int4 *>(Ci);
        for (int e = tid; e < rows_cap * (P / 4); e += kTT) z4[e] = make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    if (sh_bad) { // non-finite input on a LOR that crosses the image: propagate it as the per-LOR adjoint does
        per_lor();
        return;
    }
    xmax = red[0];
#pragma unroll
    for (int w = 1; w < kTT / 32; ++w) xmax = fmaxf(xmax, red[w]);
    if (!(xmax > 0.f)) return; // nothing to add
    // S: |c S| <= 2^22 - 2 and 2 x (LORs of the piece) |c S| < 2^31
    const float lim = fminf(4194302.f, 2147483648.f / (float)(2 * NPT * kTT) - 1.f);
    const float S = lim / xmax, invS = xmax / lim;
#pragma unroll
    for (int m = 0; m < NPT; ++m) x[m] *= S;

    const uint32_t ci_base = smem_addr(Ci) + kPad * 4u - ((uint32_t)kMagicI << 2);
    const int rpc = chunk_rows(nrows, rows_cap);
    const int G = n2 >> 2;

    for (int c0 = t.I0; c0 <= t.I1; c0 += rpc) {
        const int rows = min(rpc, t.I1 - c0 + 1);
#pragma unroll
        for (int m = 0; m < NPT; ++m) {
            const int i0 = i01[m] & 0xffff, i1 = i01[m] >> 16;
            const int ib = max(i0, c0), ie = min(i1, c0 + rows - 1);
            if (ib > ie || x[m] == 0.f) continue;
            const int nst = ie - ib + 1;
            const float b2 = b2v[m], a2_0 = a2[m], xm = x[m];
            const int qxm = __float2int_rn(xm) + kMagicI;
            const float a2_1 = fmaf(b2, 1.f, a2_0), a2_2 = fmaf(b2, 2.f, a2_0), a2_3 = fmaf(b2, 3.f, a2_0);
            const F2 a2p01 = f2(a2_0, a2_1), a2p23 = f2(a2_2, a2_3), b2p = f2(b2), xmp = f2(xm);
            float fk = (float)(ib - i0);
            uint32_t row = ci_base + (uint32_t)((ib - c0) * P) * 4u;
#pragma unroll 1
            for (int it = nst >> 2; it > 0; --it) {
                JP_BACK_STEP2(0, a2p01)
                JP_BACK_STEP2(2, a2p23)
                fk += 4.f;
                row += 4u * P * 4u;
            }
#pragma unroll 1
            for (int it = nst & 3; it > 0; --it) {
                JP_BACK_STEP(0, a2_0)
                fk += 1.f;
                row += P * 4u;
            }
        }
        __syncthreads();
        // ---- flush: spread every row over its two q1 neighbours with REDs, and clear it
        if (vec_ok) {
            const int total = rows * G;
            const RowInfo *ri_c = rinfo + (c0 - t.I0);
            for (int e = tid; e < total; e += kTT) {
                const int r = (int)__umulhi((unsigned)e, magicG), gq = e - r * G;
                int4 *src4 = reinterpret_cast<int4 *>(Ci + r * P + kPad) + gq;
                const int4 qv = *src4;
                if ((qv.x | qv.y | qv.z | qv.w) == 0) continue;
                *src4 = make_int4(0, 0, 0, 0);
                const RowInfo ri = ri_c[r];
                const float sa = ri.wa * invS, sb = ri.wb * invS;
                const float4 v = make_float4((float)qv.x, (float)qv.y, (float)qv.z, (float)qv.w);
                if (ri.base_a >= 0)
                    atomicAdd(reinterpret_cast<float4 *>(img + ri.base_a) + gq,
                              make_float4(sa * v.x, sa * v.y, sa * v.z, sa * v.w));
                if (ri.base_b >= 0)
                    atomicAdd(reinterpret_cast<float4 *>(img + ri.base_b) + gq,
                              make_float4(sb * v.x, sb * v.y, sb * v.z, sb * v.w));
            }
        } else {
            for (int e = tid; e < rows * n2; e += kTT) {
                const int r = e / n2, z = e - r * n2;
                const int qv = Ci[r * P + kPad + z];
                if (qv == 0) continue;
                Ci[r * P + kPad + z] = 0;
                const RowInfo ri = rinfo[c0 - t.I0 + r];
                const float v = (float)qv * invS;
                if (ri.base_a >= 0) atomicAdd(img + ri.base_a + z, ri.wa * v);
                if (ri.base_b >= 0) atomicAdd(img + ri.base_b + z, ri.wb * v);
            }
        }
        __syncthreads();
    }
}
#undef JP_BACK_STEP
#undef JP_BACK_STEP2

// ---- launchers ----------------------------------------------------------------------------------------------
namespace {

constexpr size_t kSmemMax = 100 * 1024;

struct TrkCfg {
    int P, rows_cap, vec_ok;
    size_t smem;
    unsigned magicG;
};

TrkCfg trk_cfg(const Geom &g, const void *img, size_t elem, size_t budget)
{
    TrkCfg c{};
    const int need = g.n[2] + kPad + kPadR;
    const int pitches[] = {40, 72, 104, 136, 200, 264};
    for (int P : pitches)
        if (need <= P) { c.P = P; break; }
    if (!c.P) return c;
    const int np = g.n[0] > g.n[1] ? g.n[0] : g.n[1];
    if (np > 32767) { c.P = 0; return c; } // plane ranges are packed into 16 + 16 bits
    const size_t rinfo = (size_t)np * sizeof(RowInfo);
    const size_t row = (size_t)c.P * elem;
    if (budget < rinfo + 24 * row) budget = rinfo + 24 * row;
    if (budget > kSmemMax) budget = kSmemMax;
    size_t rows = rinfo + row <= budget ? (budget - rinfo) / row : 0;
    if (rows < 8) { c.P = 0; return c; }
    if (rows > (size_t)np) rows = (size_t)np;
    c.rows_cap = (int)rows;
    c.smem = rows * row + rinfo;
    c.vec_ok = (g.n[2] % 4 == 0) && ((uintptr_t)img % 16 == 0);
    const unsigned G = (unsigned)(g.n[2] >> 2);
    c.magicG = G ? (unsigned)((0x100000000ull + G - 1) / G) : 0u;
    return c;
}

template <typename K>
cudaError_t set_smem(K kernel)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
}

// an unknown P / NPT sets e (a cudaError_t in scope) and falls through: the launchers free their scratch after the switch
#define JP_TRK_DISPATCH_P(CFG, ...)                          \
    switch ((CFG).P) {                                       \
    case 40: { constexpr int P = 40; __VA_ARGS__; } break;   \
    case 72: { constexpr int P = 72; __VA_ARGS__; } break;   \
    case 104: { constexpr int P = 104; __VA_ARGS__; } break; \
    case 136: { constexpr int P = 136; __VA_ARGS__; } break; \
    case 200: { constexpr int P = 200; __VA_ARGS__; } break; \
    case 264: { constexpr int P = 264; __VA_ARGS__; } break; \
    default: e = cudaErrorInvalidValue; break;               \
    }
#define JP_TRK_DISPATCH_NPT(NPTV, ...)                       \
    switch (NPTV) {                                          \
    case 3: { constexpr int NPT = 3; __VA_ARGS__; } break;   \
    case 6: { constexpr int NPT = 6; __VA_ARGS__; } break;   \
    case 9: { constexpr int NPT = 9; __VA_ARGS__; } break;   \
    default: e = cudaErrorInvalidValue; break;               \
    }

// per-call scratch: [K] Track followed by [K] int (stream-ordered allocation)
cudaError_t track_table(const SinoPlanView &pv, const Geom &g, cudaStream_t st, Track **tab, const int **kind)
{
    cudaError_t e = cudaMallocAsync((void **)tab, (sizeof(Track) + sizeof(int)) * (size_t)pv.K, st);
    if (e != cudaSuccess) return e;
    int *kd = reinterpret_cast<int *>(*tab + pv.K);
    k_track_table<<<(unsigned)((pv.K + 127) / 128), 128, 0, st>>>(pv.trk, pv.K, g, pv.dz_max, *tab, kd);
    e = cudaGetLastError();
    if (e != cudaSuccess) cudaFreeAsync(*tab, st);
    *kind = kd;
    return e;
}

} // namespace

// whole-track kernels of a regular plan; cudaErrorNotSupported: image too wide along z (the caller falls back)
cudaError_t launch_fwd_track(const SinoPlanView &pv, const float *img, const Geom &g, float *p, cudaStream_t st)
{
    if (pv.n == 0) return cudaSuccess;
    const TrkCfg c = trk_cfg(g, img, sizeof(float2), JP_TRK_SMEM_KB_FWD * 1024);
    if (!c.P || !pv.regular) return cudaErrorNotSupported;
    const int64_t ctas = pv.K * pv.t_npieces;
    if (ctas >= ((int64_t)1 << 31)) return cudaErrorInvalidValue;
    Track *tab = nullptr;
    const int *kind = nullptr;
    cudaError_t e = track_table(pv, g, st, &tab, &kind);
    if (e != cudaSuccess) return e;
    const TrkSrc ts{pv.trk, tab, kind, pv.t_zp[0], pv.t_ord[0], pv.T, pv.t_npieces, pv.t_npt * kTT};
    JP_TRK_DISPATCH_P(c, JP_TRK_DISPATCH_NPT(pv.t_npt, {
        e = set_smem(k_fwd_track<P, NPT>);
        if (e == cudaSuccess)
            k_fwd_track<P, NPT><<<(unsigned)ctas, kTT, c.smem, st>>>(ts, img, g, c.rows_cap, c.vec_ok, c.magicG, p);
    }))
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaFreeAsync(tab, st);
    return e;
}

cudaError_t launch_back_track(const SinoPlanView &pv, const float *y, const Geom &g, float *img, cudaStream_t st)
{
    if (pv.n == 0) return cudaSuccess;
    const TrkCfg c = trk_cfg(g, img, sizeof(int), JP_TRK_SMEM_KB_BACK * 1024);
    if (!c.P || !pv.regular) return cudaErrorNotSupported;
    const int64_t ctas = pv.K * pv.t_npieces;
    if (ctas >= ((int64_t)1 << 31)) return cudaErrorInvalidValue;
    Track *tab = nullptr;
    const int *kind = nullptr;
    cudaError_t e = track_table(pv, g, st, &tab, &kind);
    if (e != cudaSuccess) return e;
    const TrkSrc ts{pv.trk, tab, kind, pv.t_zp[1], pv.t_ord[1], pv.T, pv.t_npieces, pv.t_npt * kTT};
    JP_TRK_DISPATCH_P(c, JP_TRK_DISPATCH_NPT(pv.t_npt, {
        e = set_smem(k_back_track<P, NPT>);
        if (e == cudaSuccess)
            k_back_track<P, NPT><<<(unsigned)ctas, kTT, c.smem, st>>>(ts, y, g, c.rows_cap, c.vec_ok, c.magicG, img);
    }))
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaFreeAsync(tab, st);
    return e;
}

} // namespace jp
