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
//             p_j     = cf_j * sum_i lerp_z(C[i][.], u2_j(i))               memory as (value, slope) pairs:
//                                                                          one 64-bit LDS + 7 FP32 per step
//   adjoint   C[i][z] += cf_j y_j * hat(u2_j(i) - z)                        native int32 shared atomics on a
//             img[i,k1,z] += (1-w1) C[i][z];  img[i,k1+1,z] += w1 C[i][z]   fixed-point tile, then 128-bit REDs
//
// Planes are processed in chunks of `rows_cap` rows (shared memory = rows_cap x P x 8 or 4 bytes; the
// row pitch P is a template parameter so that the unrolled plane loop addresses rows with immediates).
// Tiles that are not tracks (ragged tail, principal axis z, unsorted lists) take the generic per-LOR
// path in the same launch.  No scratch memory, no state between calls, results in caller order.  With a regular
// sinogram plan (jp_fwd_planned / jp_back_planned) tiles are dealt per track and no end-point array is read.
#include "jp_f32x2.cuh"
#include "jp_tile_common.cuh"

#ifndef JP_PLAN_TRACKS
#define JP_PLAN_TRACKS 1 // regular plans: whole-track kernels (jp_track.cu); 0: the tile kernels, dealt per track
#endif
#ifndef JP_BACK_MAP
#define JP_BACK_MAP 0
#endif // adjoint lane mapping: which neighbouring diagonal the second half-warp takes

namespace jp {

using namespace tile;

namespace {

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


// ---- lane mapping (a performance hint only: any bijection of the tile's LORs onto the threads is correct) ------
// Which LOR a lane works on decides how many shared-memory wavefronts a plane step costs.  In a sinogram the LORs
// of a track form a grid (rows: one axial end point fixed, columns: the other one varies; ring pairs of configs[1]:
// 16 rows x 48 columns per tile).  With consecutive LORs on consecutive lanes a half-warp spans up to 22 axial
// cells at the far side of the image: the 64-bit row loads of the forward kernel then take 2.93 wavefronts
// instead of 2 (profiles/r01_v3: 1.08e9 wavefronts), and the two atomics of the adjoint 4.2 (lanes less than a
// cell apart collide on one address, lanes more than 32 cells apart on one bank).
//   forward: a half-warp takes a block of 2 rows x 8 columns (at most 11 cells wide: conflict-free);
//   adjoint: a half-warp takes a 16-long grid diagonal (lanes exactly one row pitch apart: no equal addresses),
//            the second half-warp the neighbouring diagonal.
// The row length L of the grid is read off the data: the first LOR whose zs or ze changes while the other one
// has been constant so far.  No grid (L = 0): identity mapping.
// forward: half-warp h of the tile <- rows (2 rp, 2 rp + 1) x columns [8 cg, 8 cg + 8)
__device__ __forceinline__ int map_fwd(int idx, int L)
{
    if (L < 8 || (L & 7) || (kTile % (2 * L))) return idx;
    const int h = idx >> 4, l16 = idx & 15, C = L >> 3;
    const int rp = h / C, cg = h - rp * C;
    return rp * 2 * L + (l16 >> 3) * L + cg * 8 + (l16 & 7);
}

// adjoint: warp w of the tile <- rows [16 rb, 16 rb + 16), two neighbouring diagonals (columns wrap)
__device__ __forceinline__ int map_back(int idx, int L)
{
    if (L < 2 || (L & 1) || (kTile % (16 * L))) return idx;
    const int w = idx >> 5, l32 = idx & 31, d = l32 & 15, s = l32 >> 4, half = L >> 1;
    const int rb = w / half, c2 = w - rb * half;
    int col = JP_BACK_MAP ? 2 * c2 + 1 - s + d : 2 * c2 + s + d;
    col %= L; // columns wrap (col < L + 16)
    return (rb * 16 + d) * L + col;
}

// ---- where a tile's LORs come from -------------------------------------------------------------------------------
// LIST: 768 consecutive LORs of the caller's arrays; a tile is a track if all 768 share their transaxial end points
//       (checked at run time, bit-exactly).
// PLAN: a regular sinogram plan (jp_sino_plan.cu): K tracks of T LORs with one axial pattern.  Tiles are dealt PER TRACK
//       (track = tile / tpt, pieces of 768 and one shorter piece when T is not a multiple of 768, e.g. 36 rings: 1296 =
//       768 + 528), the transaxial end points come from the track table and the axial ones from the pattern: no
//       end-point arrays are read at all (24 bytes per LOR of HBM traffic saved) and nothing needs checking.
struct PlanSrc {
    const float4 *trk;  // [K] (xs, ys, xe, ye)
    const float2 *zpat; // [T] (zs, ze)
    int T;
    int tpt;            // tiles per track = ceil(T / kTile)
    double dz_max;      // max |ze - zs| of the pattern: tracks with dz_max > max(|dx|, |dy|) take the per-LOR path
};

template <bool PLAN>
struct TileSrc {
    const Lors &l;
    const PlanSrc &ps;
    int64_t j0; // first LOR of the tile in the list
    int k0;     // PLAN: first pattern index of the tile
    __device__ __forceinline__ float zs(int i) const { return PLAN ? __ldg(ps.zpat + k0 + i).x : l.zs[j0 + i]; }
    __device__ __forceinline__ float ze(int i) const { return PLAN ? __ldg(ps.zpat + k0 + i).y : l.ze[j0 + i]; }
};

// row length of the tile's (zs, ze) grid, see "lane mapping" above (full tiles only)
template <bool PLAN>
__device__ __forceinline__ int detect_row_length(const TileSrc<PLAN> &src, int *sh /* 2 ints */)
{
    const int tid = threadIdx.x;
    if (tid < 2) sh[tid] = kThreads;
    __syncthreads();
    {
        const float zs0 = src.zs(0), ze0 = src.ze(0);
        const bool ds = !same_bits(src.zs(tid), zs0), de = !same_bits(src.ze(tid), ze0);
        const unsigned bs = __ballot_sync(0xffffffffu, ds), be = __ballot_sync(0xffffffffu, de);
        if ((tid & 31) == 0) {
            if (bs) atomicMin(&sh[0], (tid & ~31) + __ffs(bs) - 1);
            if (be) atomicMin(&sh[1], (tid & ~31) + __ffs(be) - 1);
        }
    }
    __syncthreads();
    const int Ls = sh[0], Le = sh[1];
    int L = 0;
    if (Ls == 1 && Le < kThreads) L = Le;       // zs runs along a row, ze is the row's constant
    else if (Le == 1 && Ls < kThreads) L = Ls;  // the other way round
    return L;
}

// is this LIST tile a track?  all 768 LORs valid, identical transaxial end points, principal axis x or y
__device__ __forceinline__ bool tile_is_track_full(const Lors &l, int64_t j0, int64_t n, const int (&jm)[kPerThread],
                                              const float (&zs)[kPerThread], const float (&ze)[kPerThread], float xs0,
                                              float ys0, float xe0, float ye0)
{
    bool ok = (j0 + kTile <= n);
    if (ok) {
        const double dmax = fmax(fabs((double)xe0 - (double)xs0), fabs((double)ye0 - (double)ys0));
        // all loads first (no short-circuit: twelve independent loads in flight), then compare bits
        uint32_t diff = 0;
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int64_t j = j0 + jm[m];
            diff |= (__float_as_uint(l.xs[j]) ^ __float_as_uint(xs0)) | (__float_as_uint(l.ys[j]) ^ __float_as_uint(ys0)) |
                    (__float_as_uint(l.xe[j]) ^ __float_as_uint(xe0)) | (__float_as_uint(l.ye[j]) ^ __float_as_uint(ye0));
            ok = ok && (fabs((double)ze[m] - (double)zs[m]) <= dmax);
        }
        ok = ok && (diff == 0) && (dmax > 0.0);
    }
    return __syncthreads_and(ok) != 0;
}

#ifndef JP_PREFETCH_DIST
#define JP_PREFETCH_DIST 592
#endif
#ifndef JP_RB_TILE
#define JP_RB_TILE 1 // image rows in flight per warp while building the shared rows (measured: 1 beats 2 and 4)
#endif
#ifndef JP_MINB_FWD
#define JP_MINB_FWD 4
#endif
#ifndef JP_MINB_BACK
#define JP_MINB_BACK 5
#endif
#ifndef JP_FWD_UNROLL
#define JP_FWD_UNROLL 8
#endif


// pull the end points of the tile that starts at LOR jt into L2 (one 128-byte line per thread): the CTA
// that will work on it finds them there instead of waiting for HBM
__device__ __forceinline__ void prefetch_tile(const Lors &l, int64_t n, int64_t jt)
{
    if (JP_PREFETCH_DIST == 0 || jt + kTile > n) return;
    const int tid = threadIdx.x;
    constexpr int kLines = kTile * 4 / 128; // lines per coordinate array
    if (tid < 6 * kLines) {
        const int a = tid / kLines, ln = tid - a * kLines;
        const float *base = (a == 0) ? l.xs : (a == 1) ? l.ys : (a == 2) ? l.zs : (a == 3) ? l.xe : (a == 4) ? l.ye : l.ze;
        asm volatile("prefetch.global.L2 [%0];" ::"l"(base + jt + ln * 32));
    }
}

template <int OFF>
__device__ __forceinline__ void reds_add(uint32_t addr, int q)
{
    asm volatile("red.shared.add.s32 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "r"(q) : "memory");
}

} // namespace

// ---- forward ------------------------------------------------------------------------------------------
// One plane step of one LOR against the (intercept, slope) rows in shared memory (build_rows<P, true>): the
// shifted axial coordinate u = u2 - kc (FFMA), its floor in the mantissa of u + magic (FADD.RM), one address LEA,
// one LDS.64, and value = intercept + u slope accumulated in two FP32 instructions -- no fractional part.
#define JP_FWD_STEP(K, A2K)                                                    \
    {                                                                          \
        const float u = fmaf(b2, fk, A2K);                                     \
        const float tt = __fadd_rd(u, kMagic);                                 \
        const float2 v = lds_pair<(K) * P * 8>(row + (__float_as_uint(tt) << 3)); \
        acc0 += v.x;                                                           \
        acc1 = fmaf(u, v.y, acc1);                                             \
    }

// two consecutive planes K, K + 1: the coordinates and their floors on packed pairs (FFMA2, FADD2.RM)
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

// generic per-LOR forward / back from explicit end points (PLAN tiles on tracks that may hold principal-axis-z LORs)
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

// first LOR, pattern offset, length and transaxial end points of the CTA's tile; false: nothing to do
template <bool PLAN>
__device__ __forceinline__ bool tile_of_block(const Lors &l, const PlanSrc &ps, int64_t n, int64_t &j0, int &k0, int &tn,
                                              float &xs0, float &ys0, float &xe0, float &ye0)
{
    if (PLAN) {
        const int64_t trk = blockIdx.x / ps.tpt;
        const int piece = (int)(blockIdx.x - trk * ps.tpt);
        k0 = piece * kTile;
        j0 = trk * (int64_t)ps.T + k0;
        tn = min(kTile, ps.T - k0);
        const float4 q = __ldg(ps.trk + trk);
        xs0 = q.x; ys0 = q.y; xe0 = q.z; ye0 = q.w;
    } else {
        j0 = blockIdx.x * (int64_t)kTile;
        k0 = 0;
        tn = (int)min((int64_t)kTile, n - j0);
        xs0 = l.xs[j0]; ys0 = l.ys[j0]; xe0 = l.xe[j0]; ye0 = l.ye[j0];
    }
    return tn > 0;
}

template <int P, bool PLAN>
__global__ void __launch_bounds__(kThreads, JP_MINB_FWD)
    k_fwd_tile(Lors l, PlanSrc ps, int64_t n, const float *__restrict__ img, Geom g, int rows_cap, int vec_ok,
               int lane_map, float *__restrict__ p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *C2 = reinterpret_cast<float2 *>(smem_raw);                                      // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(float2)); // [max(n0,n1)]
    __shared__ Track trk;
    __shared__ int sh_len[2];
    const int tid = threadIdx.x;
    int64_t j0;
    int k0, tn;
    float xs0, ys0, xe0, ye0;
    if (!PLAN) prefetch_tile(l, n, blockIdx.x * (int64_t)kTile + (int64_t)JP_PREFETCH_DIST * kTile);
    if (!tile_of_block<PLAN>(l, ps, n, j0, k0, tn, xs0, ys0, xe0, ye0)) return;
    TileSrc<PLAN> src{l, ps, j0, k0};
    int jm[kPerThread];
    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        jm[m] = m * kThreads + tid;
        zs[m] = (jm[m] < tn) ? src.zs(jm[m]) : 0.f;
        ze[m] = (jm[m] < tn) ? src.ze(jm[m]) : 0.f;
    }
    bool is_track;
    if (PLAN) {
        const double dmax = fmax(fabs((double)xe0 - (double)xs0), fabs((double)ye0 - (double)ys0));
        is_track = dmax > 0.0 && ps.dz_max <= dmax; // no LOR of the track can have principal axis z
    } else {
        is_track = tile_is_track_full(l, j0, n, jm, zs, ze, xs0, ys0, xe0, ye0);
    }
    if (!is_track) {
#pragma unroll 1
        for (int m = 0; m < kPerThread; ++m) {
            const int i = m * kThreads + tid;
            if (i >= tn) continue;
            if (PLAN) {
                const double sp[3] = {(double)xs0, (double)ys0, (double)zs[m]}, ep[3] = {(double)xe0, (double)ye0, (double)ze[m]};
                p[j0 + i] = generic_fwd_pts(sp, ep, g, img);
            } else {
                p[j0 + i] = generic_fwd(l, j0 + i, g, img);
            }
        }
        return;
    }
    if (tid == 0) track_setup(g, xs0, ys0, xe0, ye0, trk);
    __syncthreads();
    const Track t = trk;
    if (t.I1 < t.I0) { // the whole track misses the image
#pragma unroll
        for (int m = 0; m < kPerThread; ++m)
            if (m * kThreads + tid < tn) p[j0 + m * kThreads + tid] = 0.f;
        return;
    }
    // the tile does work: choose the lane mapping and fetch the axial end points again (from L1) in that order
    const int L = (lane_map && tn == kTile) ? detect_row_length<PLAN>(src, sh_len) : 0;
    if (L) {
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            jm[m] = map_fwd(m * kThreads + tid, L);
            zs[m] = src.zs(jm[m]);
            ze[m] = src.ze(jm[m]);
        }
    }
    const int n2 = g.n[2];
    const int kci = n2 >> 1;          // axial shift of the (intercept, slope) rows
    const float kc = (float)kci;
    // q1 cells of all planes of the track; constant zero columns of the shared rows
    for (int r = tid; r <= t.I1 - t.I0; r += kThreads) rinfo[r] = row_info(g, t, t.I0 + r);
    {
        const int ncl = kPad - 1, ncr = P - (n2 + kPad);
        for (int e = tid; e < rows_cap * (ncl + ncr); e += kThreads) {
            const int r = e / (ncl + ncr), c = e - r * (ncl + ncr);
            C2[r * P + (c < ncl ? c : n2 + kPad + (c - ncl))] = make_float2(0.f, 0.f);
        }
    }
    ZRay zr[kPerThread];
    float acc0[kPerThread], acc1[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        zr[m] = z_setup(g, t, zs[m], ze[m], (double)kci);
        if (jm[m] >= tn) zr[m].i1 = zr[m].i0 - 1; // slot beyond a short tile
        acc0[m] = 0.f;
        acc1[m] = 0.f;
    }
    const uint32_t c2_base = smem_addr(C2) + (uint32_t)(kPad + kci) * 8u - ((uint32_t)kMagicI << 3);
    __syncthreads();

    for (int c0 = t.I0; c0 <= t.I1; c0 += rows_cap) {
        const int rows = min(rows_cap, t.I1 - c0 + 1);
        build_rows<P, true, JP_RB_TILE>(C2, rinfo, img, t, c0, rows, n2, vec_ok, kc);
        __syncthreads();
        // ---- consume: every LOR walks its planes of this chunk, interpolating along z only
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int ib = max(zr[m].i0, c0), ie = min(zr[m].i1, c0 + rows - 1);
            if (ib > ie) continue;
            const int nst = ie - ib + 1;
            const float b2 = zr[m].b2, a2_0 = zr[m].a2;
            const float a2_1 = fmaf(b2, 1.f, a2_0), a2_2 = fmaf(b2, 2.f, a2_0), a2_3 = fmaf(b2, 3.f, a2_0);
            float fk = (float)(ib - zr[m].i0);
            uint32_t row = c2_base + (uint32_t)((ib - c0) * P) * 8u;
            float a0 = acc0[m], a1 = acc1[m];
            {
                float acc0 = a0, acc1 = a1;
                int left = nst;
                const F2 b2p = f2(b2), a2p01 = f2(a2_0, a2_1), a2p23 = f2(a2_2, a2_3);
#if JP_FWD_UNROLL == 8
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
#else
#pragma unroll 1
                for (; left >= 4; left -= 4) {
#endif
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
                a0 = acc0;
                a1 = acc1;
            }
            acc0[m] = a0;
            acc1[m] = a1;
        }
        __syncthreads();
    }
#pragma unroll
    for (int m = 0; m < kPerThread; ++m)
        if (jm[m] < tn) p[j0 + jm[m]] = zr[m].cf * (acc0[m] + acc1[m]);
}
#undef JP_FWD_STEP
#undef JP_FWD_STEP2

// ---- back ------------------------------------------------------------------------------------------------
// Fixed-point staging: contributions are rounded to multiples of 1/S and summed with native int32
// shared-memory atomics (ATOMS.ADD; float shared atomics are CAS loops on sm_100).  S is chosen per
// tile from X = max_j |cf_j y_j| so that neither a single contribution (|c S| < 2^22, the range of the
// magic-number rounding) nor a whole bin (at most two contributions per LOR and plane: |sum| <= 2 x 768 X S
// < 2^31) can overflow.  Rounding error per contribution <= X 768 / 2^31 = 3.6e-7 X.
// Per step the two bins get q1 = round(S x w) and q0 = round(S x) - q1 (their sum is exact).
// A tile whose y holds Inf or NaN (on a LOR that crosses the image) cannot be staged: it takes the per-LOR path with
// float atomics, so non-finite values propagate exactly as they do for LORs that are not in a track tile.
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

// two consecutive planes K, K + 1 at once on packed pairs (FFMA2 / FADD2): 5 floating-point instructions for two
// steps instead of 10; the integer halves (cell index in the mantissa of TT, rounded contribution in B) are the halves
// of the register pairs
#define JP_BACK_STEP2(K, A2P)                                                  \
    {                                                                          \
        const F2 U = fma2(b2p, f2(fk), A2P);                                   \
        const F2 TT = add2_rm(U, f2(kMagic));                                  \
        const F2 T = add2(TT, f2(-kMagic));                                    \
        const F2 W = fma2(T, f2(-1.f), U);                                     \
        const F2 B = fma2(xmp, W, f2(kMagic));                                 \
        const uint32_t a0 = row + (__float_as_uint(f2_lo(TT)) << 2);           \
        const uint32_t a1 = row + (__float_as_uint(f2_hi(TT)) << 2);           \
        const int b0 = __float_as_int(f2_lo(B)), b1 = __float_as_int(f2_hi(B)); \
        reds_add<(K) * P * 4>(a0, qxm - b0);                                   \
        reds_add<(K) * P * 4 + 4>(a0, b0 - kMagicI);                           \
        reds_add<((K) + 1) * P * 4>(a1, qxm - b1);                             \
        reds_add<((K) + 1) * P * 4 + 4>(a1, b1 - kMagicI);                     \
    }

template <int P, bool PLAN>
__global__ void __launch_bounds__(kThreads, JP_MINB_BACK)
    k_back_tile(Lors l, PlanSrc ps, int64_t n, const float *__restrict__ y, Geom g, int rows_cap, int vec_ok,
                int lane_map, float *__restrict__ img)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int *Ci = reinterpret_cast<int *>(smem_raw);                                        // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(int)); // [max(n0,n1)]
    __shared__ Track trk;
    __shared__ float red[kThreads / 32];
    __shared__ int sh_len[2];
    __shared__ int sh_bad;
    const int tid = threadIdx.x;
    int64_t j0;
    int k0, tn;
    float xs0, ys0, xe0, ye0;
    if (!PLAN) prefetch_tile(l, n, blockIdx.x * (int64_t)kTile + (int64_t)JP_PREFETCH_DIST * kTile);
    if (!tile_of_block<PLAN>(l, ps, n, j0, k0, tn, xs0, ys0, xe0, ye0)) return;
    TileSrc<PLAN> src{l, ps, j0, k0};
    int jm[kPerThread];
    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        jm[m] = m * kThreads + tid;
        zs[m] = (jm[m] < tn) ? src.zs(jm[m]) : 0.f;
        ze[m] = (jm[m] < tn) ? src.ze(jm[m]) : 0.f;
    }
    if (tid == 0) sh_bad = 0;
    bool is_track;
    if (PLAN) {
        const double dmax = fmax(fabs((double)xe0 - (double)xs0), fabs((double)ye0 - (double)ys0));
        is_track = dmax > 0.0 && ps.dz_max <= dmax;
    } else {
        is_track = tile_is_track_full(l, j0, n, jm, zs, ze, xs0, ys0, xe0, ye0);
    }
    // per-LOR path for the whole tile (float atomics): not a track, or non-finite values (below)
    auto per_lor = [&]() {
#pragma unroll 1
        for (int m = 0; m < kPerThread; ++m) {
            const int i = m * kThreads + tid;
            if (i >= tn) continue;
            if (PLAN) {
                const float zsi = src.zs(i), zei = src.ze(i);
                const double sp[3] = {(double)xs0, (double)ys0, (double)zsi}, ep[3] = {(double)xe0, (double)ye0, (double)zei};
                generic_back_pts(sp, ep, g, y[j0 + i], img);
            } else {
                generic_back(l, j0 + i, g, y[j0 + i], img);
            }
        }
    };
    if (!is_track) {
        per_lor();
        return;
    }
    if (tid == 0) track_setup(g, xs0, ys0, xe0, ye0, trk);
    __syncthreads();
    const Track t = trk;
    if (t.I1 < t.I0) return;
    const int L = (lane_map && tn == kTile) ? detect_row_length<PLAN>(src, sh_len) : 0;
    if (L) {
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            jm[m] = map_back(m * kThreads + tid, L);
            zs[m] = src.zs(jm[m]);
            ze[m] = src.ze(jm[m]);
        }
    }
    const int n2 = g.n[2];

    ZRay zr[kPerThread];
    float x[kPerThread];
    float xmax = 0.f;
    bool bad = false;
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        zr[m] = z_setup(g, t, zs[m], ze[m]);
        x[m] = (jm[m] < tn) ? zr[m].cf * y[j0 + jm[m]] : 0.f;
        if (jm[m] >= tn) zr[m].i1 = zr[m].i0 - 1; // slot beyond a short tile
        if (zr[m].i1 >= zr[m].i0) {
            const float ax = fabsf(x[m]);
            bad = bad || !(ax < 3.0e38f); // Inf or NaN (fmaxf would drop a NaN)
            xmax = fmaxf(xmax, ax);
        }
    }
    if (bad) atomicExch(&sh_bad, 1);
    // block max of |x|
    for (int o = 16; o > 0; o >>= 1) xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = xmax;
    for (int r = tid; r <= t.I1 - t.I0; r += kThreads) rinfo[r] = row_info(g, t, t.I0 + r);
    {
        int4 *z4 = reinterpret_cast<int4 *>(Ci);
        for (int e = tid; e < rows_cap * (P / 4); e += kThreads) z4[e] = make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    if (sh_bad) { // non-finite input on a LOR that crosses the image: propagate it as the per-LOR adjoint does
        per_lor();
        return;
    }
    xmax = red[0];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) xmax = fmaxf(xmax, red[w]);
    if (!(xmax > 0.f)) return; // nothing to add
    // S: |c S| <= 2^22 - 2 and 2 x 768 |c S| < 2^31
    const float lim = fminf(4194302.f, 2147483648.f / (float)(2 * kTile) - 1.f);
    const float S = lim / xmax, invS = xmax / lim;
    int qx[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        x[m] *= S;
        qx[m] = __float2int_rn(x[m]) + kMagicI;
    }

    const int warp = tid >> 5, lane = tid & 31;
    const uint32_t ci_base = smem_addr(Ci) + kPad * 4u - ((uint32_t)kMagicI << 2);

    for (int c0 = t.I0; c0 <= t.I1; c0 += rows_cap) {
        const int rows = min(rows_cap, t.I1 - c0 + 1);
        // ---- scatter along z into the fixed-point tile
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int ib = max(zr[m].i0, c0), ie = min(zr[m].i1, c0 + rows - 1);
            if (ib > ie || x[m] == 0.f) continue;
            const int nst = ie - ib + 1;
            const float b2 = zr[m].b2, a2_0 = zr[m].a2, xm = x[m];
            const int qxm = qx[m];
            const float a2_1 = fmaf(b2, 1.f, a2_0), a2_2 = fmaf(b2, 2.f, a2_0), a2_3 = fmaf(b2, 3.f, a2_0);
            const F2 a2p01 = f2(a2_0, a2_1), a2p23 = f2(a2_2, a2_3), b2p = f2(b2), xmp = f2(xm);
            float fk = (float)(ib - zr[m].i0);
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
            const int G = n2 >> 2;
            for (int r = warp; r < rows; r += kThreads / 32) {
                const RowInfo ri = rinfo[c0 - t.I0 + r];
                const float sa = ri.wa * invS, sb = ri.wb * invS;
                for (int gq = lane; gq < G; gq += 32) {
                    int4 *src4 = reinterpret_cast<int4 *>(Ci + r * P + kPad) + gq;
                    const int4 q = *src4;
                    if ((q.x | q.y | q.z | q.w) == 0) continue;
                    *src4 = make_int4(0, 0, 0, 0);
                    const float4 v = make_float4((float)q.x, (float)q.y, (float)q.z, (float)q.w);
                    if (ri.base_a >= 0)
                        atomicAdd(reinterpret_cast<float4 *>(img + ri.base_a) + gq,
                                  make_float4(sa * v.x, sa * v.y, sa * v.z, sa * v.w));
                    if (ri.base_b >= 0)
                        atomicAdd(reinterpret_cast<float4 *>(img + ri.base_b) + gq,
                                  make_float4(sb * v.x, sb * v.y, sb * v.z, sb * v.w));
                }
            }
        } else {
            for (int e = tid; e < rows * n2; e += kThreads) {
                const int r = e / n2, z = e - r * n2;
                const int q = Ci[r * P + kPad + z];
                if (q == 0) continue;
                Ci[r * P + kPad + z] = 0;
                const RowInfo ri = rinfo[c0 - t.I0 + r];
                const float v = (float)q * invS;
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

// Shared memory per CTA.  Measured on configs[1] (sweep 20..54 KB): the smaller the tile buffer the larger the L1 that
// serves the end-point and image-row loads, down to ~36 KB where the extra row chunks start to cost more.
#ifndef JP_SMEM_KB_FWD
#define JP_SMEM_KB_FWD 36
#endif
#ifndef JP_SMEM_KB_BACK
#define JP_SMEM_KB_BACK 28
#endif
constexpr size_t kSmemMax = 100 * 1024; // wide images: at least 24 rows per chunk, up to this much

struct TileCfg {
    int P;        // row pitch (0: image too wide along z for the tiled kernels)
    int rows_cap; // rows per chunk
    size_t smem;
    int vec_ok;
};

TileCfg tile_cfg(const Geom &g, const void *img, size_t elem, size_t budget)
{
    TileCfg c{};
    const int need = g.n[2] + kPad + kPadR;
    const int pitches[] = {40, 72, 104, 136, 200, 264};
    for (int P : pitches)
        if (need <= P) { c.P = P; break; }
    if (!c.P) return c;
    const int np = g.n[0] > g.n[1] ? g.n[0] : g.n[1];
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
    return c;
}

template <typename K>
cudaError_t set_smem(K kernel)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
}

PlanSrc plan_src(const SinoPlanView *pv)
{
    PlanSrc ps{};
    if (pv && pv->regular) {
        ps.trk = pv->trk;
        ps.zpat = pv->zpat;
        ps.T = pv->T;
        ps.tpt = (pv->T + kTile - 1) / kTile;
        ps.dz_max = pv->dz_max;
    }
    return ps;
}

} // namespace

// With JP_PLAN_TRACKS a regular plan never reaches the tile kernels (launch_*_track takes it), so their PLAN = true
// instantiations are compiled only without it
#if JP_PLAN_TRACKS
#define JP_IF_PLAN_TILES(...)
#else
#define JP_IF_PLAN_TILES(...) __VA_ARGS__
#endif

#define JP_DISPATCH_P(CFG, ...)                    \
    switch ((CFG).P) {                             \
    case 40: { constexpr int P = 40; __VA_ARGS__; } break;   \
    case 72: { constexpr int P = 72; __VA_ARGS__; } break;   \
    case 104: { constexpr int P = 104; __VA_ARGS__; } break; \
    case 136: { constexpr int P = 136; __VA_ARGS__; } break; \
    case 200: { constexpr int P = 200; __VA_ARGS__; } break; \
    case 264: { constexpr int P = 264; __VA_ARGS__; } break; \
    default: return cudaErrorInvalidValue;         \
    }

// pv == null (or an irregular plan): tiles of 768 consecutive LORs of `l`; a regular plan: tiles per track, `l` unused.
// lane_map = 0 switches the lane mapping off (a performance hint only; the results are the same)
cudaError_t launch_fwd_tile(const Lors &l, int64_t n, const float *img, const Geom &g, float *p, cudaStream_t st,
                            const SinoPlanView *pv, int lane_map)
{
    if (n == 0) return cudaSuccess;
    const bool plan = pv && pv->regular;
    if (plan && JP_PLAN_TRACKS) return launch_fwd_track(*pv, img, g, p, st);
    const TileCfg c = tile_cfg(g, img, sizeof(float2), JP_SMEM_KB_FWD * 1024);
    const PlanSrc ps = plan_src(pv);
    if (!c.P) return plan ? cudaErrorNotSupported : launch_fwd(l, Range{0, 1, n, false, nullptr}, img, g, p, st);
    const int64_t tiles = plan ? pv->K * ps.tpt : (n + kTile - 1) / kTile;
    if (tiles >= ((int64_t)1 << 31)) return cudaErrorInvalidValue;
    cudaError_t e = cudaSuccess;
    JP_DISPATCH_P(c, {
        JP_IF_PLAN_TILES(if (plan) {
            e = set_smem(k_fwd_tile<P, true>);
            if (e == cudaSuccess)
                k_fwd_tile<P, true><<<(unsigned)tiles, kThreads, c.smem, st>>>(l, ps, n, img, g, c.rows_cap, c.vec_ok, lane_map, p);
        } else) {
            e = set_smem(k_fwd_tile<P, false>);
            if (e == cudaSuccess)
                k_fwd_tile<P, false><<<(unsigned)tiles, kThreads, c.smem, st>>>(l, ps, n, img, g, c.rows_cap, c.vec_ok, lane_map, p);
        }
    })
    if (e == cudaSuccess) e = cudaGetLastError();
    return e;
}

cudaError_t launch_back_tile(const Lors &l, int64_t n, const float *y, const Geom &g, float *img, cudaStream_t st,
                             const SinoPlanView *pv, int lane_map)
{
    if (n == 0) return cudaSuccess;
    const bool plan = pv && pv->regular;
    if (plan && JP_PLAN_TRACKS) return launch_back_track(*pv, y, g, img, st);
    const TileCfg c = tile_cfg(g, img, sizeof(int), JP_SMEM_KB_BACK * 1024);
    const PlanSrc ps = plan_src(pv);
    if (!c.P) return plan ? cudaErrorNotSupported : launch_back(l, Range{0, 1, n, false, nullptr}, y, g, img, st);
    const int64_t tiles = plan ? pv->K * ps.tpt : (n + kTile - 1) / kTile;
    if (tiles >= ((int64_t)1 << 31)) return cudaErrorInvalidValue;
    cudaError_t e = cudaSuccess;
    JP_DISPATCH_P(c, {
        JP_IF_PLAN_TILES(if (plan) {
            e = set_smem(k_back_tile<P, true>);
            if (e == cudaSuccess)
                k_back_tile<P, true><<<(unsigned)tiles, kThreads, c.smem, st>>>(l, ps, n, y, g, c.rows_cap, c.vec_ok, lane_map, img);
        } else) {
            e = set_smem(k_back_tile<P, false>);
            if (e == cudaSuccess)
                k_back_tile<P, false><<<(unsigned)tiles, kThreads, c.smem, st>>>(l, ps, n, y, g, c.rows_cap, c.vec_ok, lane_map, img);
        }
    })
    if (e == cudaSuccess) e = cudaGetLastError();
    return e;
}

} // namespace jp
