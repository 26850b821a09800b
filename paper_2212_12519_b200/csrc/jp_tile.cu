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
// path in the same launch.  No plan, no scratch memory, results in caller order.
#include <cstdlib>
#include <mutex>

#include "jp_tile_common.cuh"

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
__device__ __forceinline__ int detect_row_length(const Lors &l, int64_t j0, int64_t n, int *sh /* 2 ints */)
{
    const int tid = threadIdx.x;
    if (tid < 2) sh[tid] = kThreads;
    __syncthreads();
    if (j0 + kTile <= n) {
        const float zs0 = l.zs[j0], ze0 = l.ze[j0];
        const bool ds = !same_bits(l.zs[j0 + tid], zs0), de = !same_bits(l.ze[j0 + tid], ze0);
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

// ---- tiles cut per track ---------------------------------------------------------------------------------------
// A tile is 768 CONSECUTIVE LORs, so a track whose length T is not a multiple of 768 (e.g. 36 rings: 1296 ring
// pairs) would leave every other tile straddling two tracks, i.e. on the per-LOR path.  k_track_probe reads T off
// the head of the list (length of the first run of identical transaxial end points) and, when T > 768 is not a
// multiple of 768, the CUT instantiation of the kernels (persistent CTAs) deals tiles per track instead:
// track k = tile / ceil(T / 768) is cut into pieces of 768 and one shorter piece.  The list is ASSUMED to consist
// of tracks of that length; where it does not, tile_is_track fails and the tile takes the per-LOR path as before.
// *cut_len == 0 selects the plain instantiation (both are launched; the one not selected exits at once).
__global__ void k_track_probe(Lors l, int64_t n, int *cut_len)
{
    __shared__ int first;
    const int tid = threadIdx.x;
    if (tid == 0) first = 0x7fffffff;
    __syncthreads();
    const int64_t lim = n < 8192 ? n : 8192; // tracks longer than this are treated as aligned
    const float xs0 = l.xs[0], ys0 = l.ys[0], xe0 = l.xe[0], ye0 = l.ye[0];
    // 8 positions per thread, all loads independent (one round trip instead of a dependent loop)
    uint32_t d[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int64_t j = (int64_t)u * blockDim.x + tid;
        d[u] = 0;
        if (j < lim)
            d[u] = (__float_as_uint(l.xs[j]) ^ __float_as_uint(xs0)) | (__float_as_uint(l.ys[j]) ^ __float_as_uint(ys0)) |
                   (__float_as_uint(l.xe[j]) ^ __float_as_uint(xe0)) | (__float_as_uint(l.ye[j]) ^ __float_as_uint(ye0));
    }
#pragma unroll
    for (int u = 0; u < 8; ++u)
        if (d[u]) {
            atomicMin(&first, u * (int)blockDim.x + tid);
            break;
        }
    __syncthreads();
    if (tid == 0) {
        const int T = first;
        *cut_len = (T != 0x7fffffff && T > kTile && (T % kTile) != 0) ? T : 0;
    }
}

// first LOR and length of tile number `tile` (CUT: per track, see above); false when the list is exhausted
template <bool CUT>
__device__ __forceinline__ bool tile_span(int64_t tile, int64_t n, int T, int64_t &j0, int &tn)
{
    if (CUT) {
        const int tpt = (T + kTile - 1) / kTile;
        const int64_t k = tile / tpt;
        const int t = (int)(tile - k * tpt);
        j0 = k * (int64_t)T + (int64_t)t * kTile;
        tn = min(kTile, T - t * kTile);
    } else {
        j0 = tile * (int64_t)kTile;
        tn = kTile;
    }
    if (j0 >= n) return false;
    if (j0 + tn > n) tn = (int)(n - j0);
    return true;
}

// is this tile a track?  all 768 LORs valid, identical transaxial end points, principal axis x or y
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

// is this tile a track?  all tn LORs have identical transaxial end points and principal axis x or y
template <bool CUT>
__device__ __forceinline__ bool tile_is_track(const Lors &l, int64_t j0, int tn, const int (&jm)[kPerThread],
                                              const float (&zs)[kPerThread], const float (&ze)[kPerThread], float xs0,
                                              float ys0, float xe0, float ye0)
{
    const double dmax = fmax(fabs((double)xe0 - (double)xs0), fabs((double)ye0 - (double)ys0));
    // all loads first (no short-circuit: twelve independent loads in flight), then compare bits
    uint32_t diff = 0;
    bool ok = (dmax > 0.0) && (CUT || tn == kTile); // plain: full tiles only, so that no slot needs a guard afterwards
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        if (jm[m] < tn) {
            const int64_t j = j0 + jm[m];
            diff |= (__float_as_uint(l.xs[j]) ^ __float_as_uint(xs0)) | (__float_as_uint(l.ys[j]) ^ __float_as_uint(ys0)) |
                    (__float_as_uint(l.xe[j]) ^ __float_as_uint(xe0)) | (__float_as_uint(l.ye[j]) ^ __float_as_uint(ye0));
            ok = ok && (fabs((double)ze[m] - (double)zs[m]) <= dmax);
        }
    }
    ok = ok && (diff == 0);
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

template <int P>
__global__ void __launch_bounds__(kThreads, JP_MINB_FWD)
    k_fwd_tile(Lors l, int64_t n, const float *__restrict__ img, Geom g, int rows_cap, int vec_ok,
               int lane_map, const int *__restrict__ cut_len, float *__restrict__ p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *C2 = reinterpret_cast<float2 *>(smem_raw);                                      // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(float2)); // [max(n0,n1)]
    __shared__ Track trk;
    __shared__ int sh_len[2];
    const int tid = threadIdx.x;
    const int64_t j0 = blockIdx.x * (int64_t)kTile;

    prefetch_tile(l, n, j0 + (int64_t)JP_PREFETCH_DIST * kTile);
    int jm[kPerThread];
    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        jm[m] = m * kThreads + tid;
        const int64_t j = j0 + jm[m];
        zs[m] = (j < n) ? l.zs[j] : 0.f;
        ze[m] = (j < n) ? l.ze[j] : 0.f;
    }
    const float xs0 = l.xs[j0], ys0 = l.ys[j0], xe0 = l.xe[j0], ye0 = l.ye[j0];
    if (cut_len && __ldg(cut_len) != 0) return; // tiles are dealt per track: the _cut kernel does this list
    if (!tile_is_track_full(l, j0, n, jm, zs, ze, xs0, ys0, xe0, ye0)) {
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
    // the tile does work: choose the lane mapping and fetch the axial end points again (from L1) in that order
    const int L = lane_map ? detect_row_length(l, j0, n, sh_len) : 0;
    if (L) {
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            jm[m] = map_fwd(m * kThreads + tid, L);
            zs[m] = l.zs[j0 + jm[m]];
            ze[m] = l.ze[j0 + jm[m]];
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
#if JP_FWD_UNROLL == 8
                const float a2_4 = fmaf(b2, 4.f, a2_0), a2_5 = fmaf(b2, 5.f, a2_0), a2_6 = fmaf(b2, 6.f, a2_0),
                            a2_7 = fmaf(b2, 7.f, a2_0);
#pragma unroll 1
                for (; left >= 8; left -= 8) {
                    JP_FWD_STEP(0, a2_0)
                    JP_FWD_STEP(1, a2_1)
                    JP_FWD_STEP(2, a2_2)
                    JP_FWD_STEP(3, a2_3)
                    JP_FWD_STEP(4, a2_4)
                    JP_FWD_STEP(5, a2_5)
                    JP_FWD_STEP(6, a2_6)
                    JP_FWD_STEP(7, a2_7)
                    fk += 8.f;
                    row += 8u * P * 8u;
                }
                if (left >= 4) {
#else
#pragma unroll 1
                for (; left >= 4; left -= 4) {
#endif
                    JP_FWD_STEP(0, a2_0)
                    JP_FWD_STEP(1, a2_1)
                    JP_FWD_STEP(2, a2_2)
                    JP_FWD_STEP(3, a2_3)
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
    for (int m = 0; m < kPerThread; ++m) p[j0 + map_fwd(m * kThreads + tid, L)] = zr[m].cf * (acc0[m] + acc1[m]);
}

// ---- the same kernel with tiles dealt per track (CUT = true; see k_track_probe) -----------------------------
template <int P, bool CUT>
__global__ void __launch_bounds__(kThreads, JP_MINB_FWD)
    k_fwd_tile_cut(Lors l, int64_t n, const float *__restrict__ img, Geom g, int rows_cap, int vec_ok,
               int lane_map, const int *__restrict__ cut_len, float *__restrict__ p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *C2 = reinterpret_cast<float2 *>(smem_raw);                                      // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(float2)); // [max(n0,n1)]
    __shared__ Track trk;
    __shared__ int sh_len[2];
    const int tid = threadIdx.x;
    const int T = cut_len ? __ldg(cut_len) : 0;
    if (CUT && T == 0) return; // the plain instantiation does this list (it checks after its first loads are in flight)
  // plain: one tile per CTA; CUT: persistent CTAs over the tiles dealt per track
  for (int64_t tile = blockIdx.x; CUT || tile == blockIdx.x; tile += gridDim.x) {
    int64_t j0;
    int tn;
    if (!tile_span<CUT>(tile, n, T, j0, tn)) break;
    if (CUT && tile != blockIdx.x) __syncthreads(); // the shared buffers of the previous tile are free

    prefetch_tile(l, n, j0 + (int64_t)JP_PREFETCH_DIST * kTile);
    int jm[kPerThread];
    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        jm[m] = m * kThreads + tid;
        const int64_t j = j0 + jm[m];
        zs[m] = (jm[m] < tn) ? l.zs[j] : 0.f;
        ze[m] = (jm[m] < tn) ? l.ze[j] : 0.f;
    }
    const float xs0 = l.xs[j0], ys0 = l.ys[j0], xe0 = l.xe[j0], ye0 = l.ye[j0];
    if (!CUT && T != 0) return; // the CUT instantiation does this list
    if (!tile_is_track<CUT>(l, j0, tn, jm, zs, ze, xs0, ys0, xe0, ye0)) {
#pragma unroll 1
        for (int m = 0; m < kPerThread; ++m) {
            const int64_t j = j0 + m * kThreads + tid;
            if (m * kThreads + tid < tn) p[j] = generic_fwd(l, j, g, img);
        }
        continue;
    }
    if (tid == 0) track_setup(g, xs0, ys0, xe0, ye0, trk);
    __syncthreads();
    const Track t = trk;
    if (t.I1 < t.I0) { // the whole track misses the image
#pragma unroll
        for (int m = 0; m < kPerThread; ++m)
            if (!CUT || m * kThreads + tid < tn) p[j0 + m * kThreads + tid] = 0.f;
        continue;
    }
    // the tile does work: choose the lane mapping and fetch the axial end points again (from L1) in that order
    const int L = (lane_map && (!CUT || tn == kTile)) ? detect_row_length(l, j0, n, sh_len) : 0;
    if (L) {
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            jm[m] = map_fwd(m * kThreads + tid, L);
            zs[m] = l.zs[j0 + jm[m]];
            ze[m] = l.ze[j0 + jm[m]];
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
        if (CUT && jm[m] >= tn) zr[m].i1 = zr[m].i0 - 1; // slot beyond a short tile
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
#if JP_FWD_UNROLL == 8
                const float a2_4 = fmaf(b2, 4.f, a2_0), a2_5 = fmaf(b2, 5.f, a2_0), a2_6 = fmaf(b2, 6.f, a2_0),
                            a2_7 = fmaf(b2, 7.f, a2_0);
#pragma unroll 1
                for (; left >= 8; left -= 8) {
                    JP_FWD_STEP(0, a2_0)
                    JP_FWD_STEP(1, a2_1)
                    JP_FWD_STEP(2, a2_2)
                    JP_FWD_STEP(3, a2_3)
                    JP_FWD_STEP(4, a2_4)
                    JP_FWD_STEP(5, a2_5)
                    JP_FWD_STEP(6, a2_6)
                    JP_FWD_STEP(7, a2_7)
                    fk += 8.f;
                    row += 8u * P * 8u;
                }
                if (left >= 4) {
#else
#pragma unroll 1
                for (; left >= 4; left -= 4) {
#endif
                    JP_FWD_STEP(0, a2_0)
                    JP_FWD_STEP(1, a2_1)
                    JP_FWD_STEP(2, a2_2)
                    JP_FWD_STEP(3, a2_3)
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
    for (int m = 0; m < kPerThread; ++m) {
        const int jl = CUT ? jm[m] : map_fwd(m * kThreads + tid, L);
        if (!CUT || jl < tn) p[j0 + jl] = zr[m].cf * (acc0[m] + acc1[m]);
    }
  }
}
#undef JP_FWD_STEP

// ---- back ------------------------------------------------------------------------------------------------
// Fixed-point staging: contributions are rounded to multiples of 1/S and summed with native int32
// shared-memory atomics (ATOMS.ADD; float shared atomics are CAS loops on sm_100).  S is chosen per
// tile from X = max_j |cf_j y_j| so that neither a single contribution (|c S| < 2^22, the range of the
// magic-number rounding) nor a whole bin (at most two contributions per LOR and plane: |sum| <= 2 x 768 X S
// < 2^31) can overflow.  Rounding error per contribution <= X 768 / 2^31 = 3.6e-7 X.
// Per step the two bins get q1 = round(S x w) and q0 = round(S x) - q1 (their sum is exact).
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

template <int P>
__global__ void __launch_bounds__(kThreads, JP_MINB_BACK)
    k_back_tile(Lors l, int64_t n, const float *__restrict__ y, Geom g, int rows_cap, int vec_ok,
                int lane_map, const int *__restrict__ cut_len, float *__restrict__ img)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int *Ci = reinterpret_cast<int *>(smem_raw);                                        // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(int)); // [max(n0,n1)]
    __shared__ Track trk;
    __shared__ float red[kThreads / 32];
    __shared__ int sh_len[2];
    const int tid = threadIdx.x;
    const int64_t j0 = blockIdx.x * (int64_t)kTile;

    prefetch_tile(l, n, j0 + (int64_t)JP_PREFETCH_DIST * kTile);
    int jm[kPerThread];
    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        jm[m] = m * kThreads + tid;
        const int64_t j = j0 + jm[m];
        zs[m] = (j < n) ? l.zs[j] : 0.f;
        ze[m] = (j < n) ? l.ze[j] : 0.f;
    }
    const float xs0 = l.xs[j0], ys0 = l.ys[j0], xe0 = l.xe[j0], ye0 = l.ye[j0];
    if (cut_len && __ldg(cut_len) != 0) return; // tiles are dealt per track: the _cut kernel does this list
    if (!tile_is_track_full(l, j0, n, jm, zs, ze, xs0, ys0, xe0, ye0)) {
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
    const int L = lane_map ? detect_row_length(l, j0, n, sh_len) : 0;
    if (L) {
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            jm[m] = map_back(m * kThreads + tid, L);
            zs[m] = l.zs[j0 + jm[m]];
            ze[m] = l.ze[j0 + jm[m]];
        }
    }
    const int n2 = g.n[2];

    ZRay zr[kPerThread];
    float x[kPerThread];
    float xmax = 0.f;
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        zr[m] = z_setup(g, t, zs[m], ze[m]);
        x[m] = zr[m].cf * y[j0 + jm[m]];
        if (zr[m].i1 >= zr[m].i0) xmax = fmaxf(xmax, fabsf(x[m]));
    }
    // block max of |x|
    for (int o = 16; o > 0; o >>= 1) xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = xmax;
    for (int r = tid; r <= t.I1 - t.I0; r += kThreads) rinfo[r] = row_info(g, t, t.I0 + r);
    {
        int4 *z4 = reinterpret_cast<int4 *>(Ci);
        for (int e = tid; e < rows_cap * (P / 4); e += kThreads) z4[e] = make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    xmax = red[0];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) xmax = fmaxf(xmax, red[w]);
    if (!(xmax > 0.f) || !(xmax < 3.0e38f)) return; // nothing to add (or non-finite input: undefined, skip)
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
            float fk = (float)(ib - zr[m].i0);
            uint32_t row = ci_base + (uint32_t)((ib - c0) * P) * 4u;
#pragma unroll 1
            for (int it = nst >> 2; it > 0; --it) {
                JP_BACK_STEP(0, a2_0)
                JP_BACK_STEP(1, a2_1)
                JP_BACK_STEP(2, a2_2)
                JP_BACK_STEP(3, a2_3)
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
                    int4 *src = reinterpret_cast<int4 *>(Ci + r * P + kPad) + gq;
                    const int4 q = *src;
                    if ((q.x | q.y | q.z | q.w) == 0) continue;
                    *src = make_int4(0, 0, 0, 0);
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

// ---- the same kernel with tiles dealt per track (CUT = true) --------------------------------------------------
template <int P, bool CUT>
__global__ void __launch_bounds__(kThreads, JP_MINB_BACK)
    k_back_tile_cut(Lors l, int64_t n, const float *__restrict__ y, Geom g, int rows_cap, int vec_ok,
                int lane_map, const int *__restrict__ cut_len, float *__restrict__ img)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int *Ci = reinterpret_cast<int *>(smem_raw);                                        // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(int)); // [max(n0,n1)]
    __shared__ Track trk;
    __shared__ float red[kThreads / 32];
    __shared__ int sh_len[2];
    const int tid = threadIdx.x;
    const int T = cut_len ? __ldg(cut_len) : 0;
    if (CUT && T == 0) return; // the plain instantiation does this list (it checks after its first loads are in flight)
  for (int64_t tile = blockIdx.x; CUT || tile == blockIdx.x; tile += gridDim.x) {
    int64_t j0;
    int tn;
    if (!tile_span<CUT>(tile, n, T, j0, tn)) break;
    if (CUT && tile != blockIdx.x) __syncthreads(); // the shared buffers of the previous tile are free

    prefetch_tile(l, n, j0 + (int64_t)JP_PREFETCH_DIST * kTile);
    int jm[kPerThread];
    float zs[kPerThread], ze[kPerThread];
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        jm[m] = m * kThreads + tid;
        const int64_t j = j0 + jm[m];
        zs[m] = (jm[m] < tn) ? l.zs[j] : 0.f;
        ze[m] = (jm[m] < tn) ? l.ze[j] : 0.f;
    }
    const float xs0 = l.xs[j0], ys0 = l.ys[j0], xe0 = l.xe[j0], ye0 = l.ye[j0];
    if (!CUT && T != 0) return; // the CUT instantiation does this list
    if (!tile_is_track<CUT>(l, j0, tn, jm, zs, ze, xs0, ys0, xe0, ye0)) {
#pragma unroll 1
        for (int m = 0; m < kPerThread; ++m) {
            const int64_t j = j0 + m * kThreads + tid;
            if (m * kThreads + tid < tn) generic_back(l, j, g, y[j], img);
        }
        continue;
    }
    if (tid == 0) track_setup(g, xs0, ys0, xe0, ye0, trk);
    __syncthreads();
    const Track t = trk;
    if (t.I1 < t.I0) continue;
    const int L = (lane_map && (!CUT || tn == kTile)) ? detect_row_length(l, j0, n, sh_len) : 0;
    if (L) {
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            jm[m] = map_back(m * kThreads + tid, L);
            zs[m] = l.zs[j0 + jm[m]];
            ze[m] = l.ze[j0 + jm[m]];
        }
    }
    const int n2 = g.n[2];

    ZRay zr[kPerThread];
    float x[kPerThread];
    float xmax = 0.f;
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) {
        zr[m] = z_setup(g, t, zs[m], ze[m]);
        x[m] = (!CUT || jm[m] < tn) ? zr[m].cf * y[j0 + jm[m]] : 0.f;
        if (CUT && jm[m] >= tn) zr[m].i1 = zr[m].i0 - 1; // slot beyond a short tile
        if (zr[m].i1 >= zr[m].i0) xmax = fmaxf(xmax, fabsf(x[m]));
    }
    // block max of |x|
    for (int o = 16; o > 0; o >>= 1) xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
    if ((tid & 31) == 0) red[tid >> 5] = xmax;
    for (int r = tid; r <= t.I1 - t.I0; r += kThreads) rinfo[r] = row_info(g, t, t.I0 + r);
    {
        int4 *z4 = reinterpret_cast<int4 *>(Ci);
        for (int e = tid; e < rows_cap * (P / 4); e += kThreads) z4[e] = make_int4(0, 0, 0, 0);
    }
    __syncthreads();
    xmax = red[0];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) xmax = fmaxf(xmax, red[w]);
    if (!(xmax > 0.f) || !(xmax < 3.0e38f)) continue; // nothing to add (or non-finite input: undefined, skip)
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
            float fk = (float)(ib - zr[m].i0);
            uint32_t row = ci_base + (uint32_t)((ib - c0) * P) * 4u;
#pragma unroll 1
            for (int it = nst >> 2; it > 0; --it) {
                JP_BACK_STEP(0, a2_0)
                JP_BACK_STEP(1, a2_1)
                JP_BACK_STEP(2, a2_2)
                JP_BACK_STEP(3, a2_3)
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
                    int4 *src = reinterpret_cast<int4 *>(Ci + r * P + kPad) + gq;
                    const int4 q = *src;
                    if ((q.x | q.y | q.z | q.w) == 0) continue;
                    *src = make_int4(0, 0, 0, 0);
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
}
#undef JP_BACK_STEP

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

// JP_LANE_MAP=0 in the environment switches the lane mapping off (A/B measurements; results are the same)
int lane_map_on()
{
    const char *e = getenv("JP_LANE_MAP");
    return !(e && e[0] == '0');
}

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
cudaError_t set_smem(K kernel, size_t smem)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
}

} // namespace

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

// probe of the track length (lists long enough for it to matter); *out = device int (stream-ordered scratch) or null
// The probe result is cached per LOR list, keyed by (device, address of xs, n): repeated projections of the same
// list (every OSEM iteration, every benchmark step) skip the probe launch, which would otherwise sit in front of the
// tile kernel on the stream.  Only the ADDRESS is remembered, nothing is dereferenced later; a stale hit (another
// list at the same address) can only cost speed, never correctness: both instantiations read the same int, and
// any track length partitions the list.  Events order the int between streams: `ready` after the probe, `used`
// after the last kernels that read it (an entry is recycled only behind that event).
struct ProbeEntry {
    int dev = -1;
    const void *key = nullptr;
    int64_t n = 0;
    int *cut = nullptr;
    cudaEvent_t ready = nullptr, used = nullptr;
    unsigned long long stamp = 0;
};
static std::mutex g_probe_mu;
static ProbeEntry g_probe[16];
static unsigned long long g_probe_clock = 0;

static cudaError_t probe_tracks(const Lors &l, int64_t n, cudaStream_t st, int **out, cudaEvent_t *used)
{
    *out = nullptr;
    *used = nullptr;
    if (n < 8 * kTile) return cudaSuccess;
    const char *env = getenv("JP_TRACK_PROBE"); // JP_TRACK_PROBE=0: assume aligned tracks (A/B measurements)
    if (env && env[0] == '0') return cudaSuccess;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone)
        return cudaSuccess; // inside a graph capture: no allocation, no cross-stream events -- plain tiles (always correct)
    std::lock_guard<std::mutex> lock(g_probe_mu);
    ProbeEntry *hit = nullptr, *lru = &g_probe[0];
    for (ProbeEntry &p : g_probe) {
        if (p.cut && p.dev == dev && p.key == (const void *)l.xs && p.n == n) hit = &p;
        if (p.stamp < lru->stamp) lru = &p;
    }
    if (hit) {
        hit->stamp = ++g_probe_clock;
        if ((e = cudaStreamWaitEvent(st, hit->ready, 0)) != cudaSuccess) return e;
        // chain the users of an entry (a no-op on the same stream), so that `used` always covers all of them
        if ((e = cudaStreamWaitEvent(st, hit->used, 0)) != cudaSuccess) return e;
        *out = hit->cut;
        *used = hit->used;
        return cudaSuccess;
    }
    ProbeEntry &p = *lru;
    if (!p.cut || p.dev != dev) { // first use of the slot (or another device: the old int is left to that device)
        p = ProbeEntry{};
        if ((e = cudaMalloc((void **)&p.cut, sizeof(int))) != cudaSuccess) return e;
        if ((e = cudaEventCreateWithFlags(&p.ready, cudaEventDisableTiming)) != cudaSuccess) return e;
        if ((e = cudaEventCreateWithFlags(&p.used, cudaEventDisableTiming)) != cudaSuccess) return e;
    } else if ((e = cudaStreamWaitEvent(st, p.used, 0)) != cudaSuccess) { // kernels of the evicted list may still read it
        return e;
    }
    p.dev = dev;
    p.key = (const void *)l.xs;
    p.n = n;
    p.stamp = ++g_probe_clock;
    k_track_probe<<<1, 1024, 0, st>>>(l, n, p.cut);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = cudaEventRecord(p.ready, st)) != cudaSuccess) return e;
    *out = p.cut;
    *used = p.used;
    return cudaSuccess;
}

static unsigned persistent_grid(int per_sm)
{
    int dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    return (unsigned)(nsm > 0 ? nsm * per_sm : 148 * per_sm);
}

cudaError_t launch_fwd_tile(const Lors &l, int64_t n, const float *img, const Geom &g, float *p, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const TileCfg c = tile_cfg(g, img, sizeof(float2), JP_SMEM_KB_FWD * 1024);
    if (!c.P) return launch_fwd(l, Range{0, 1, n, false, nullptr}, img, g, p, st);
    const unsigned grid = (unsigned)((n + kTile - 1) / kTile);
    int *cut = nullptr;
    cudaEvent_t used = nullptr;
    cudaError_t e = probe_tracks(l, n, st, &cut, &used);
    if (e != cudaSuccess) return e;
    JP_DISPATCH_P(c, {
        e = set_smem(k_fwd_tile<P>, c.smem);
        if (e == cudaSuccess && cut) e = set_smem(k_fwd_tile_cut<P, true>, c.smem);
        if (e == cudaSuccess) {
            k_fwd_tile<P><<<grid, kThreads, c.smem, st>>>(l, n, img, g, c.rows_cap, c.vec_ok, lane_map_on(), cut, p);
            if (cut)
                k_fwd_tile_cut<P, true><<<persistent_grid(JP_MINB_FWD), kThreads, c.smem, st>>>(l, n, img, g, c.rows_cap, c.vec_ok,
                                                                                         lane_map_on(), cut, p);
        }
    })
    if (e == cudaSuccess) e = cudaGetLastError();
    if (used && e == cudaSuccess) e = cudaEventRecord(used, st);
    return e;
}

cudaError_t launch_back_tile(const Lors &l, int64_t n, const float *y, const Geom &g, float *img, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const TileCfg c = tile_cfg(g, img, sizeof(int), JP_SMEM_KB_BACK * 1024);
    if (!c.P) return launch_back(l, Range{0, 1, n, false, nullptr}, y, g, img, st);
    const unsigned grid = (unsigned)((n + kTile - 1) / kTile);
    int *cut = nullptr;
    cudaEvent_t used = nullptr;
    cudaError_t e = probe_tracks(l, n, st, &cut, &used);
    if (e != cudaSuccess) return e;
    JP_DISPATCH_P(c, {
        e = set_smem(k_back_tile<P>, c.smem);
        if (e == cudaSuccess && cut) e = set_smem(k_back_tile_cut<P, true>, c.smem);
        if (e == cudaSuccess) {
            k_back_tile<P><<<grid, kThreads, c.smem, st>>>(l, n, y, g, c.rows_cap, c.vec_ok, lane_map_on(), cut, img);
            if (cut)
                k_back_tile_cut<P, true><<<persistent_grid(JP_MINB_BACK), kThreads, c.smem, st>>>(l, n, y, g, c.rows_cap, c.vec_ok,
                                                                                           lane_map_on(), cut, img);
        }
    })
    if (e == cudaSuccess) e = cudaGetLastError();
    if (used && e == cudaSuccess) e = cudaEventRecord(used, st);
    return e;
}

} // namespace jp
