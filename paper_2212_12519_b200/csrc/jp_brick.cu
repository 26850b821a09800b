// jp_brick.cu -- TOF listmode projections of SPARSE event sets on image BRICKS held in shared memory: the kernels
// behind the planned listmode OSEM (BASELINE.json configs[4]) and the planned projections of sparsely populated lists.
//
// An OSEM subset of a listmode acquisition (40e6 events in 20 - 34 subsets) puts ~20 events on a
// transaxial line, so nothing is shared along a line (the line tiles of jp_lm_tile.cu need hundreds), and a TOF event
// only touches the ~46 planes around its TOF bin ("only affected by a few voxels"): its 4 gathers / 4 atomic
// adds per plane land on random sectors of the 15 MB image.  Measured on B200 such a walk runs at the L1 gather rate
// (one 128-byte line per clock and SM) and at the L2 atomic rate, whatever the order of the events.
// But every voxel is still touched ~100 times per subset.  The reuse is spatial, not per line, so the image is cut into
// bricks of kBrP x kBr1 x kBr2 cells (principal axis, other transaxial axis, axial) and every event into PIECES, the
// maximal runs of consecutive planes whose interpolation cell lies in one brick (3.5 per event for 32 x 32 x 16).  The
// plan (set-up, "pre-sorting") sorts the pieces of every subset by brick and length and stores, per piece,
// the affine plane loop in BRICK-LOCAL coordinates (32 bytes, float64 set-up as in jp_ray.cuh).  A CTA takes a chunk of
// <= kBrChunk pieces of one brick:
//   forward   brick (+ one column of neighbours) -> shared memory; per piece  acc[event] += sum_k G(k) bilinear(k)
//   adjoint   float atomics on the quad accumulators (jp_quad.cu), reading the same TOF table as the forward kernel.
//             (Rounds 1-2 also shipped an adjoint staged in the bricks in int32 fixed point, one scale per chunk.  One
//             scale cannot carry the dynamic range of OSEM ratios: on a low-count reconstruction the update amplified
//             its rounding to 2e-3 of the image maximum, over the 1e-3 bound, so it was taken out in round 3.)
// Shared-memory gathers of 32 random banks cost ~3.5 wavefronts per load instead of 32 L1 wavefronts per gather.
#include <cuda.h> // CUtensorMap (types only: the encoder is fetched with cudaGetDriverEntryPoint, libcuda is not linked)

#include <cub/device/device_scan.cuh>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

#include "jp_g1tab.cuh"

namespace jp {

namespace {

#ifndef JP_BR_P
#define JP_BR_P 32
#endif
#ifndef JP_BR_1
#define JP_BR_1 32
#endif
#ifndef JP_BR_2
#define JP_BR_2 16
#endif
#ifndef JP_BR_CHUNK
#define JP_BR_CHUNK 4096
#endif
#ifndef JP_BR_THREADS
#define JP_BR_THREADS 768
#endif
#ifndef JP_BR_ROUND_ROBIN
#define JP_BR_ROUND_ROBIN 1
#endif
#ifndef JP_BR_MINB
#define JP_BR_MINB 2
#endif
constexpr int kBrP = JP_BR_P, kBr1 = JP_BR_1, kBr2 = JP_BR_2; // cells of a brick along p, q1, q2 (axial)
// columns held per brick row: the cells, the bilinear neighbour (+1) and one safety column (the float32 plane loop may
// land one cell above the cell the float64 set-up assigned to the brick; below is excluded by construction)
constexpr int kBrC1 = kBr1 + 2, kBrC2 = kBr2 + 2;
// cells are shifted before they are cut into bricks: local column c <-> voxel b kBr - kOff + c.  Along q1 one column of
// padding is what cell -1 needs; along z four, so that every brick starts at a multiple of 4 voxels (16 bytes: the TMA
// box of the forward kernel needs that alignment)
constexpr int kOff1 = 1, kOff2 = 4;
constexpr int kBrChunk = JP_BR_CHUNK;         // pieces per CTA
constexpr int kBrT = JP_BR_THREADS;
constexpr int kBrPer = (kBrChunk + kBrT - 1) / kBrT; // pieces per thread
constexpr int kLenBits = 6;                   // key bits of the piece length (kBrP <= 64)
static_assert(kBrP <= 64 && kBrP < 256, "piece length must fit its key / record field");
static_assert(kBr2 % 4 == 0, "the TMA box needs bricks aligned to 4 axial voxels");

// one piece: planes k = 0 .. nk-1 of the brick-local loop
//   u1(k) = a1 + b1 k, u2(k) = a2 + b2 k   cell (floor u1, floor u2) of brick plane pl0 + k, local column c <-> voxel
//                                          b kBr - kOff + c
//   x(k)  = x0 + dx k                      position in the G1 table (jp_g1tab.cuh)
struct __align__(16) BrickPiece {
    float a1, b1, a2, b2;
    float x0, dx;
    int pl_nk; // pl0 << 8 | nk
    int ev;    // position of the event in the plan's sorted list
};
static_assert(sizeof(BrickPiece) == 32, "piece record is two 16-byte loads");

struct __align__(8) BrickChunk {
    int first, count;   // pieces [first, first + count) of the sorted piece list
    short bp, b1, b2;   // brick coordinates
    short axis;         // principal axis (0 or 1)
    int pad;            // host side: slice number of the chunk inside its brick (launch order)
    int pad2;
};

// brick grid of the image for principal axis a: cells kk = k + kOff in [kOff - 1, n_q + kOff) along q1 / q2, planes [0, n_p)
struct BrickGrid {
    int nb[2][3];
    int NB; // max over the axes of the number of bricks
};

BrickGrid brick_grid(const Geom &g)
{
    BrickGrid bg{};
    for (int a = 0; a < 2; ++a) {
        const int q1 = 1 - a;
        bg.nb[a][0] = (g.n[a] + kBrP - 1) / kBrP;
        bg.nb[a][1] = (g.n[q1] + kOff1 + kBr1 - 1) / kBr1;
        bg.nb[a][2] = (g.n[2] + kOff2 + kBr2 - 1) / kBr2;
        const int nb = bg.nb[a][0] * bg.nb[a][1] * bg.nb[a][2];
        if (nb > bg.NB) bg.NB = nb;
    }
    return bg;
}

// ---- plan-time set-up of one event in float64 (same formulae and the same discrete decisions as ray_setup_pts) ----
struct DRay {
    int p;          // principal axis
    int ilo, ihi;   // planes visited (closed segment rule, TOF window, crossing point strictly inside (-1, n) x (-1, n))
    double A1, B1;  // u_q1(i) = A1 + B1 i, i the plane index
    double A2, B2;
    double tau0, dtau; // tau(i) = tau0 + dtau i
    float cf;
};

__device__ bool dray_setup(const Lors &l, int64_t e, const int16_t *__restrict__ tb, const Geom &g, const Tof &t, DRay &R)
{
    const float centre = (float)tb[e] * t.width;
    const float reach = 0.5f * t.width + t.nsig * t.sigma;
    const double s[3] = {(double)l.xs[e], (double)l.ys[e], (double)l.zs[e]};
    const double en[3] = {(double)l.xe[e], (double)l.ye[e], (double)l.ze[e]};
    Ray r;
    ray_setup_pts<true>(s, en, g, t.coff, centre - reach, centre + reach, r);
    R.p = r.p;
    R.cf = r.cf;
    R.ilo = 0;
    R.ihi = -1;
    if (r.nk == 0 || r.p == 2) return false;
    const int p = r.p, q1 = 1 - p;
    const double d[3] = {en[0] - s[0], en[1] - s[1], en[2] - s[2]};
    const double op = (double)g.o[p], vp = (double)g.v[p];
    const double inv_dp = drcp(d[p]);
    const double r1 = d[q1] * inv_dp, r2 = d[2] * inv_dp;
    const double iv1 = drcp((double)g.v[q1]), iv2 = drcp((double)g.v[2]);
    R.B1 = r1 * vp * iv1;
    R.A1 = (s[q1] - (double)g.o[q1] + (op - s[p]) * r1) * iv1;
    R.B2 = r2 * vp * iv2;
    R.A2 = (s[2] - (double)g.o[2] + (op - s[p]) * r2) * iv2;
    const double L = dsqrt_pos(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    R.dtau = vp * inv_dp * L;
    R.tau0 = ((op - s[p]) * inv_dp - 0.5) * L - (double)t.coff;
    // the clips of ray_setup are rounded outwards: drop end planes whose crossing point is not strictly inside
    // (-1, n_q1) x (-1, n_2) (all four neighbours outside the image: they contribute exactly zero, reading A5)
    const double n1 = (double)g.n[q1], n2 = (double)g.n[2];
    int ilo = r.i0, ihi = r.i0 + r.nk - 1;
    auto inside = [&](int i) {
        const double u1 = fma(R.B1, (double)i, R.A1), u2 = fma(R.B2, (double)i, R.A2);
        return u1 > -1.0 && u1 < n1 && u2 > -1.0 && u2 < n2;
    };
    while (ilo <= ihi && !inside(ilo)) ++ilo;
    while (ihi >= ilo && !inside(ihi)) --ihi;
    R.ilo = ilo;
    R.ihi = ihi;
    return ihi >= ilo;
}

__device__ __forceinline__ int dray_brick(const DRay &R, int i, const int (&nb)[3])
{
    const int bp = i / kBrP;
    const int k1 = (int)floor(fma(R.B1, (double)i, R.A1) + (double)kOff1), k2 = (int)floor(fma(R.B2, (double)i, R.A2) + (double)kOff2);
    return (bp * nb[1] + k1 / kBr1) * nb[2] + k2 / kBr2;
}

// The pieces are ordered by a COUNTING sort on  bin = ((subset * 2 + axis) * NB + brick) << kLenBits | (nk - 1):
// pass 1 (k_brick_pieces<false>) counts the pieces of every bin, an exclusive scan turns the counts into offsets, and
// pass 2 (k_brick_pieces<true>) writes every piece's record straight to its final place (one atomic ticket per piece).
// The order of the pieces inside a bin (same brick, same length) is arbitrary.
__device__ __forceinline__ void brick_piece_record(const DRay &R, const int16_t *__restrict__ tb, const Tof &t, float scale,
                                                   const int (&nb)[3], int e, int brick, int i0, int nk, BrickPiece &pc)
{
    const int b2 = brick % nb[2], b1 = (brick / nb[2]) % nb[1], bp = brick / (nb[2] * nb[1]);
    // local coordinates: column c <-> voxel b kBr - kOff + c, so u' = u + kOff - b kBr lies in [0, kBr) for the brick's cells
    const double a1 = fma(R.B1, (double)i0, R.A1) + (double)kOff1 - (double)(b1 * kBr1);
    const double a2 = fma(R.B2, (double)i0, R.A2) + (double)kOff2 - (double)(b2 * kBr2);
    pc.b1 = (float)R.B1;
    pc.b2 = (float)R.B2;
    pc.a1 = fmaxf((float)a1, 0.f);
    pc.a2 = fmaxf((float)a2, 0.f);
    // the plane loop evaluates fmaf(b, k, a) in float32: keep its last plane (the other extreme of a monotone
    // sequence) at or above 0 as well; the shift is a few ulp of a (<= 4e-6 voxel)
    const float kl = (float)(nk - 1);
    for (int it = 0; it < 64 && fmaf(pc.b1, kl, pc.a1) < 0.f; ++it) pc.a1 = nextafterf(pc.a1, 1e30f);
    for (int it = 0; it < 64 && fmaf(pc.b2, kl, pc.a2) < 0.f; ++it) pc.a2 = nextafterf(pc.a2, 1e30f);
    const double centre = (double)((float)tb[e] * t.width);
    pc.x0 = (float)((centre - fma(R.dtau, (double)i0, R.tau0)) * (double)scale);
    pc.dx = (float)(-R.dtau * (double)scale);
    pc.pl_nk = ((i0 - bp * kBrP) << 8) | nk;
    pc.ev = e;
}

// events [first, first + count) of the sorted list = subset `subset`.  EMIT false: bins[bin] += 1 per piece, cf per event,
// *total += pieces;  EMIT true: bins holds the running offsets (tickets), the records go to pieces[ticket].
template <bool EMIT>
__global__ void __launch_bounds__(256) k_brick_pieces(Lors l, const int16_t *__restrict__ tb, int64_t first, int64_t count,
                                                       int subset, Geom g, Tof t, BrickGrid bg, float scale,
                                                       int *__restrict__ bins, float *__restrict__ cf,
                                                       unsigned long long *__restrict__ total, BrickPiece *__restrict__ pieces)
{
    const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int cnt = 0;
    if (c < count) {
        const int64_t e = first + c;
        DRay R;
        const bool hit = dray_setup(l, e, tb, g, t, R);
        if (!EMIT) cf[e] = R.cf;
        if (hit) {
            const int (&nb)[3] = bg.nb[R.p];
            const unsigned sab0 = (unsigned)(subset * 2 + R.p) * (unsigned)bg.NB;
            int prev = dray_brick(R, R.ilo, nb), i0 = R.ilo;
            for (int i = R.ilo + 1; i <= R.ihi + 1; ++i) {
                const int b = (i <= R.ihi) ? dray_brick(R, i, nb) : -1;
                if (b != prev) {
                    const int nk = i - i0;
                    const unsigned bin = ((sab0 + (unsigned)prev) << kLenBits) | (unsigned)(nk - 1);
                    if (EMIT) {
                        BrickPiece pc;
                        brick_piece_record(R, tb, t, scale, nb, (int)e, prev, i0, nk, pc);
                        pieces[atomicAdd(&bins[bin], 1)] = pc;
                    } else {
                        atomicAdd(&bins[bin], 1);
                        ++cnt;
                    }
                    prev = b;
                    i0 = i;
                }
            }
        }
    }
    if (!EMIT) {
        for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
        if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(total, (unsigned long long)cnt);
    }
}

// ---- hot kernels ---------------------------------------------------------------------------------------------------
template <int OFF>
__device__ __forceinline__ float lds_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(addr), "n"(OFF) : "memory");
    return v;
}

struct BrickOrg {
    int p, q1;
    int sp, s1;            // element strides of the image along p and q1 (axial stride 1)
    int i0, k1_0, k2_0;    // image indices of local (plane 0, column 0, column 0)
    int np, n1, n2;
};

__device__ __forceinline__ BrickOrg brick_org(const BrickChunk &ch, const Geom &g)
{
    BrickOrg o;
    o.p = ch.axis;
    o.q1 = 1 - o.p;
    const int s_x = g.n[1] * g.n[2], s_y = g.n[2];
    o.sp = o.p == 0 ? s_x : s_y;
    o.s1 = o.p == 0 ? s_y : s_x;
    o.i0 = ch.bp * kBrP;
    o.k1_0 = ch.b1 * kBr1 - kOff1;
    o.k2_0 = ch.b2 * kBr2 - kOff2;
    o.np = o.p == 0 ? g.n[0] : g.n[1];
    o.n1 = o.p == 0 ? g.n[1] : g.n[0];
    o.n2 = g.n[2];
    return o;
}

// ---- forward -------------------------------------------------------------------------------------------------------
// The brick is a 3-D box of the image: ONE TMA tile load (cp.async.bulk.tensor.3d) brings it into shared memory, the
// hardware zero-fills whatever lies outside the image (reading A5), and no thread spends instructions or LSU wavefronts
// on it.  Box rows are kFwRow floats (a multiple of 16 bytes).  The box follows the image's axis order, so the plane /
// q1 strides of the shared copy depend on the principal axis: axis 0: [plane][q1][z], axis 1: [q1][plane][z].
constexpr int kFwRow = (kBrC2 + 3) / 4 * 4;
constexpr int kFwVox = kFwRow * kBrC1 * kBrP;

__device__ __forceinline__ void mbar_init(uint32_t mbar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "JP_MBAR_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra JP_MBAR_WAIT_%=;\n"
        "}\n" ::"r"(mbar), "r"(parity)
        : "memory");
}

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, uint32_t mbar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
                 "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(mbar)
                 : "memory");
}

// the pieces of one chunk on the shared brick; SP / S1: element strides of a plane / a q1 row of the shared copy
template <int SP, int S1>
__device__ __forceinline__ void brick_fwd_pieces(const BrickChunk &ch, const BrickPiece *__restrict__ pieces, uint32_t bsm,
                                                 uint32_t gbase, float xedge, int ev0, float *__restrict__ acc)
{
    const uint32_t bbase = bsm - (uint32_t)kMagicI * (uint32_t)((S1 + 1) * 4);
    for (int j = threadIdx.x; j < ch.count; j += kBrT) {
        const float4 *rec = reinterpret_cast<const float4 *>(pieces + ch.first + j);
        const float4 r0 = __ldg(rec), r1 = __ldg(rec + 1);
        const float a1 = r0.x, b1 = r0.y, a2 = r0.z, b2 = r0.w, x0 = r1.x, dx = r1.y;
        const int pl_nk = __float_as_int(r1.z), ev = __float_as_int(r1.w);
        const int nk = pl_nk & 0xff;
        uint32_t row = bbase + (uint32_t)(pl_nk >> 8) * (uint32_t)(SP * 4);
        float fk = 0.f, sum = 0.f;
#pragma unroll 2
        for (int k = 0; k < nk; ++k) {
            const float u1 = fmaf(b1, fk, a1), u2 = fmaf(b2, fk, a2);
            const float t1 = __fadd_rd(u1, kMagic), t2 = __fadd_rd(u2, kMagic);
            const float w1 = u1 - (t1 - kMagic), w2 = u2 - (t2 - kMagic);
            const uint32_t ad = row + __float_as_uint(t1) * (uint32_t)(S1 * 4) + (__float_as_uint(t2) << 2);
            const float v00 = lds_f32<0>(ad), v01 = lds_f32<4>(ad);
            const float v10 = lds_f32<S1 * 4>(ad), v11 = lds_f32<S1 * 4 + 4>(ad);
            const float lo = fmaf(w2, v01 - v00, v00), hi = fmaf(w2, v11 - v10, v10);
            const float wt = g1_weight(gbase, xedge, fmaf(dx, fk, x0));
            sum = fmaf(fmaf(w1, hi - lo, lo), wt, sum);
            fk += 1.f;
            row += SP * 4;
        }
        atomicAdd(acc + (ev - ev0), sum);
    }
}

// forward: acc[ev - ev0] += sum over the piece's planes of  G * bilinear  (the factor cf is applied per event later)
__global__ void __launch_bounds__(kBrT, JP_BR_MINB)
    k_brick_fwd(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, int use_tma,
                const BrickChunk *__restrict__ chunks, const BrickPiece *__restrict__ pieces, const float *__restrict__ img,
                Geom g, G1Tab gt, int ev0, float *__restrict__ acc)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *B = reinterpret_cast<float *>(smem_raw);
    float2 *g1 = reinterpret_cast<float2 *>(smem_raw + sizeof(float) * kFwVox);
    __shared__ __align__(8) unsigned long long mbar_sm;
    const int tid = threadIdx.x;
    const BrickChunk ch = chunks[blockIdx.x];
    const BrickOrg o = brick_org(ch, g);
    const int SP = (o.p == 0) ? kBrC1 * kFwRow : kFwRow;  // element strides of the shared copy
    const int S1 = (o.p == 0) ? kFwRow : kBrP * kFwRow;
    const uint32_t mbar = smem_addr(&mbar_sm);
    if (use_tma) {
        if (tid == 0) mbar_init(mbar, 1);
        __syncthreads();
        if (tid == 0) {
            mbar_expect_tx(mbar, (uint32_t)(sizeof(float) * kFwVox));
            if (o.p == 0) tma_load_3d(smem_addr(B), &tm0, o.k2_0, o.k1_0, o.i0, mbar);
            else tma_load_3d(smem_addr(B), &tm1, o.k2_0, o.i0, o.k1_0, mbar);
        }
    } else { // images the tensor map cannot describe (axial size not a multiple of 4, unaligned base)
        for (int idx = tid; idx < kBrP * kBrC1 * kBrC2; idx += kBrT) {
            const int c2 = idx % kBrC2, r = idx / kBrC2;
            const int c1 = r % kBrC1, pl = r / kBrC1;
            const int i = o.i0 + pl, k1 = o.k1_0 + c1, k2 = o.k2_0 + c2;
            float v = 0.f;
            if (i < o.np && (unsigned)k1 < (unsigned)o.n1 && (unsigned)k2 < (unsigned)o.n2)
                v = __ldg(img + (int64_t)i * o.sp + (int64_t)k1 * o.s1 + k2);
            B[pl * SP + c1 * S1 + c2] = v;
        }
    }
    for (int i = tid; i < gt.n; i += kBrT) g1[i] = __ldg(gt.tab + i);
    __syncthreads();
    if (use_tma) mbar_wait(mbar, 0);
    const uint32_t gbase = smem_addr(g1) - ((uint32_t)kMagicI << 3);
    // the strides are compile-time constants inside the loop (immediates): one instantiation per principal axis
    if (o.p == 0) brick_fwd_pieces<kBrC1 * kFwRow, kFwRow>(ch, pieces, smem_addr(B), gbase, gt.xedge, ev0, acc);
    else brick_fwd_pieces<kFwRow, kBrP * kFwRow>(ch, pieces, smem_addr(B), gbase, gt.xedge, ev0, acc);
}

// p[io] = cf acc  (MODE 0)  or the OSEM ratio 1 / (cf acc)  (MODE 1) for the events [first, first + count) of the sorted
// list that have pieces (principal axis 0 / 1)
__global__ void __launch_bounds__(256) k_brick_finish(const float *__restrict__ cf, const float *__restrict__ acc, int64_t first,
                                                       int64_t count, int ev0, const int *__restrict__ perm, int64_t io_off,
                                                       int mode, float *__restrict__ p)
{
    const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c >= count) return;
    const int64_t e = first + c;
    float out = cf[e] * acc[e - ev0];
    if (mode == 1) out = (out > 1e-9f) ? 1.f / out : 0.f;
    p[perm ? (int64_t)perm[e] : c + io_off] = out;
}

constexpr size_t brick_smem_fwd(int g1n) { return sizeof(float) * (size_t)kFwVox + sizeof(float2) * (size_t)g1n; }

} // namespace

// ---- the brick set of a listmode plan --------------------------------------------------------------------------------
struct BrickSet {
    int64_t n_pieces = 0;
    BrickPiece *pieces = nullptr;
    BrickChunk *chunks = nullptr;
    float *cf = nullptr;                       // [n] incidence factor of every sorted event
    float *acc = nullptr;                      // [n] scratch of the planned forward projection: the events' sums
    std::vector<int> chunk_first, chunk_count; // per subset
    int g1n = 0;
    float gmax = 1.f;
    int64_t n_chunks = 0;
};

bool brick_supported(const Geom &g, const Tof &t, int n_subsets)
{
    const BrickGrid bg = brick_grid(g);
    if (bg.NB > 32767) return false; // brick coordinates are stored as shorts
    // the counting sort keeps one int per (subset, axis, brick, length) bin and scans them with an int count: at most
    // 2^26 bins (256 MB of histogram); larger problems take the line-tile path of the plan
    if (((uint64_t)n_subsets * 2u * (uint64_t)bg.NB << kLenBits) >= ((uint64_t)1 << 26)) return false;
    if (g.n[0] >= (1 << 23) || g.n[1] >= (1 << 23)) return false;
    if (brick_smem_fwd(g1tab_entries(t)) > 110 * 1024) return false; // two CTAs per SM
    return true;
}

void brick_set_destroy(BrickSet *bs)
{
    if (!bs) return;
    cudaFree(bs->pieces);
    cudaFree(bs->chunks);
    cudaFree(bs->cf);
    cudaFree(bs->acc);
    delete bs;
}

int64_t brick_set_pieces(const BrickSet *bs) { return bs->n_pieces; }

// l / tb: the plan's SORTED events (subset-major, then principal axis); sub_first[m], sub_count[m]: events of subset m.
// Synchronises `st` (piece counts and the per-brick bounds are read back).  cudaErrorNotSupported: too many pieces.
cudaError_t brick_set_create(const Lors &l, const int16_t *tb, int64_t n, const Geom &g, const Tof &t, int n_subsets,
                             const int64_t *sub_first, const int64_t *sub_count, cudaStream_t st, BrickSet **out)
{
    *out = nullptr;
    if (!brick_supported(g, t, n_subsets)) return cudaErrorNotSupported;
    BrickSet *bs = new BrickSet;
    const BrickGrid bg = brick_grid(g);
    bs->g1n = g1tab_entries(t);
    {   // G(0): the largest TOF weight
        const double m = (double)t.nsig * (double)t.sigma, h = 0.5 * (double)t.width;
        bs->gmax = (float)(std::erf(std::fmin(h, m) / ((double)t.sigma * 1.4142135623730951)) * 1.0001);
    }
    bs->chunk_first.assign((size_t)n_subsets, 0);
    bs->chunk_count.assign((size_t)n_subsets, 0);
    *out = bs;
    if (n == 0) return cudaSuccess;
    cudaError_t e;
    int *bins = nullptr;
    unsigned long long *total = nullptr;
    void *tmp = nullptr;
    size_t tmp_bytes = 0;
    const size_t n_sab = (size_t)n_subsets * 2 * (size_t)bg.NB;
    const size_t n_bins = n_sab << kLenBits;
    const float scale = (float)((double)kG1K / (double)t.width);
    std::vector<int> h_first(n_sab + 1, 0); // first piece of every (subset, axis, brick)
    std::vector<BrickChunk> h_chunks;
#define JP_BR_TRY(x)                     \
    do {                                 \
        e = (x);                         \
        if (e != cudaSuccess) goto fail; \
    } while (0)
    JP_BR_TRY(cudaMalloc((void **)&bs->cf, sizeof(float) * (size_t)n));
    JP_BR_TRY(cudaMalloc((void **)&bs->acc, sizeof(float) * (size_t)n));
    JP_BR_TRY(cudaMalloc((void **)&bins, sizeof(int) * (n_bins + 1)));
    JP_BR_TRY(cudaMemsetAsync(bins, 0, sizeof(int) * (n_bins + 1), st));
    JP_BR_TRY(cudaMalloc((void **)&total, sizeof(unsigned long long)));
    JP_BR_TRY(cudaMemsetAsync(total, 0, sizeof(unsigned long long), st));
    for (int m = 0; m < n_subsets; ++m) {
        if (sub_count[m] == 0) continue;
        k_brick_pieces<false><<<(unsigned)((sub_count[m] + 255) / 256), 256, 0, st>>>(l, tb, sub_first[m], sub_count[m], m, g, t, bg,
                                                                                     scale, bins, bs->cf, total, nullptr);
        JP_BR_TRY(cudaGetLastError());
    }
    {
        unsigned long long h_total = 0;
        JP_BR_TRY(cudaMemcpyAsync(&h_total, total, sizeof(h_total), cudaMemcpyDeviceToHost, st));
        JP_BR_TRY(cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, bins, bins, (int)(n_bins + 1), st));
        JP_BR_TRY(cudaMalloc(&tmp, tmp_bytes));
        JP_BR_TRY(cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, bins, bins, (int)(n_bins + 1), st));
        // offsets of the bricks' first bins (every 2^kLenBits-th entry) and the total, one strided copy
        JP_BR_TRY(cudaMemcpy2DAsync(h_first.data(), sizeof(int), bins, sizeof(int) << kLenBits, sizeof(int), n_sab + 1,
                                    cudaMemcpyDeviceToHost, st));
        JP_BR_TRY(cudaStreamSynchronize(st));
        if (h_total >= ((unsigned long long)1 << 31)) {
            e = cudaErrorNotSupported;
            goto fail;
        }
        bs->n_pieces = (int64_t)h_total;
    }
    if (bs->n_pieces > 0) {
        JP_BR_TRY(cudaMalloc((void **)&bs->pieces, sizeof(BrickPiece) * (size_t)bs->n_pieces));
        for (int m = 0; m < n_subsets; ++m) {
            if (sub_count[m] == 0) continue;
            k_brick_pieces<true><<<(unsigned)((sub_count[m] + 255) / 256), 256, 0, st>>>(l, tb, sub_first[m], sub_count[m], m, g, t,
                                                                                        bg, scale, bins, nullptr, nullptr, bs->pieces);
            JP_BR_TRY(cudaGetLastError());
        }
        // chunks: every (subset, axis, brick) run of the sorted pieces, cut into slices of <= kBrChunk pieces
        for (int m = 0; m < n_subsets; ++m) {
            bs->chunk_first[(size_t)m] = (int)h_chunks.size();
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < bg.NB; ++b) {
                    const size_t s = ((size_t)m * 2 + a) * (size_t)bg.NB + b;
                    const int64_t cnt = (int64_t)h_first[s + 1] - h_first[s];
                    if (cnt == 0) continue;
                    const int (&nb)[3] = bg.nb[a];
                    for (int64_t at = 0; at < cnt; at += kBrChunk) {
                        BrickChunk c;
                        c.first = (int)(h_first[s] + at);
                        c.count = (int)std::min<int64_t>(kBrChunk, cnt - at);
                        c.b2 = (short)(b % nb[2]);
                        c.b1 = (short)((b / nb[2]) % nb[1]);
                        c.bp = (short)(b / (nb[2] * nb[1]));
                        c.axis = (short)a;
                        c.pad = (int)(at / kBrChunk); // slice number inside its brick (launch order, below)
                        h_chunks.push_back(c);
                    }
                }
            bs->chunk_count[(size_t)m] = (int)h_chunks.size() - bs->chunk_first[(size_t)m];
            // launch order: the k-th slices of all bricks before the (k+1)-th, so that the CTAs in flight at any time
            // work on different bricks instead of ~40 chunks of one central brick side by side: the brick loads do not
            // pile up on one brick's voxels (a small effect: configs[4] iteration 16.43 -> 16.39 ms, A/B in one run)
#if JP_BR_ROUND_ROBIN
            std::stable_sort(h_chunks.begin() + bs->chunk_first[(size_t)m], h_chunks.end(), [&](const BrickChunk &x, const BrickChunk &y) {
                return (x.pad < y.pad);
            });
#endif
        }
        for (BrickChunk &c : h_chunks) c.pad = 0;
        if (!h_chunks.empty()) {
            JP_BR_TRY(cudaMalloc((void **)&bs->chunks, sizeof(BrickChunk) * h_chunks.size()));
            JP_BR_TRY(cudaMemcpyAsync(bs->chunks, h_chunks.data(), sizeof(BrickChunk) * h_chunks.size(), cudaMemcpyHostToDevice, st));
            JP_BR_TRY(cudaStreamSynchronize(st)); // h_chunks goes out of scope
        }
        bs->n_chunks = (int64_t)h_chunks.size();
    }
    e = cudaSuccess;
fail:
    cudaStreamSynchronize(st); // the temporaries are plain cudaMalloc memory (cheaper than stream-ordered at this size)
    cudaFree(tmp);
    cudaFree(total);
    cudaFree(bins);
    if (e != cudaSuccess) {
        brick_set_destroy(bs);
        *out = nullptr;
    }
    return e;
#undef JP_BR_TRY
}

const float *brick_set_cf(const BrickSet *bs) { return bs->cf; }
float *brick_set_acc(const BrickSet *bs) { return bs->acc; }

// function attributes belong to the current device: set on every launch, like the other launchers (a process-wide
// "done" flag would leave the second GPU of a hybrid handle at the 48 KB default)
static cudaError_t brick_attr()
{
    return cudaFuncSetAttribute(k_brick_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024);
}

// acc[e - ev0] += sum_k G bilinear over the pieces of subset m (acc: zeroed by the caller, one float per event of the
// subset, ev0 = position of the subset's first event in the sorted list)
// tensor maps of the image for the brick boxes of principal axis 0 / 1; false: the image cannot be described (the
// kernel then loads the brick with plain loads)
static bool brick_tensor_maps(const float *img, const Geom &g, CUtensorMap *tm0, CUtensorMap *tm1)
{
    typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    static bool looked = false;
    if (!looked) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            encode = reinterpret_cast<EncodeFn>(fn);
        else
            (void)cudaGetLastError();
        looked = true;
    }
    if (!encode || g.n[2] % 4 != 0 || (uintptr_t)img % 16 != 0) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.n[2], (cuuint64_t)g.n[1], (cuuint64_t)g.n[0]};
    const cuuint64_t strides[2] = {(cuuint64_t)g.n[2] * 4u, (cuuint64_t)g.n[1] * (cuuint64_t)g.n[2] * 4u};
    const cuuint32_t es[3] = {1, 1, 1};
    const cuuint32_t box0[3] = {(cuuint32_t)kFwRow, (cuuint32_t)kBrC1, (cuuint32_t)kBrP}; // principal axis 0: q1 = axis 1
    const cuuint32_t box1[3] = {(cuuint32_t)kFwRow, (cuuint32_t)kBrP, (cuuint32_t)kBrC1}; // principal axis 1: q1 = axis 0
    void *base = const_cast<float *>(img);
    if (encode(tm0, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims, strides, box0, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    if (encode(tm1, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims, strides, box1, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    return true;
}

// acc[e - ev0] += sum_k G bilinear over the pieces of subset m (acc: zeroed by the caller, one float per event of the
// subset, ev0 = position of the subset's first event in the sorted list)
cudaError_t launch_brick_fwd(const BrickSet *bs, int m, const float *img, const Geom &g, const Tof &t, int64_t ev0, float *acc,
                             cudaStream_t st, const G1Tab *table)
{
    const int nc = bs->chunk_count[(size_t)m];
    if (nc == 0) return cudaSuccess;
    cudaError_t e = brick_attr();
    if (e != cudaSuccess) return e;
    G1Tab gt{};
    if (table && table->n == bs->g1n) gt = *table; // the caller's table (a driver that loops over subsets makes it once)
    else e = g1tab_create(t, bs->g1n, st, &gt);
    if (e != cudaSuccess) return e;
    CUtensorMap tm0, tm1;
    memset(&tm0, 0, sizeof(tm0));
    memset(&tm1, 0, sizeof(tm1));
    const int use_tma = brick_tensor_maps(img, g, &tm0, &tm1) ? 1 : 0;
    k_brick_fwd<<<(unsigned)nc, kBrT, brick_smem_fwd(bs->g1n), st>>>(tm0, tm1, use_tma, bs->chunks + bs->chunk_first[(size_t)m],
                                                                    bs->pieces, img, g, gt, (int)ev0, acc);
    e = cudaGetLastError();
    if (!(table && table->n == bs->g1n)) cudaFreeAsync((void *)gt.tab, st);
    return e;
}

cudaError_t launch_brick_finish(const BrickSet *bs, const float *acc, int64_t first, int64_t count, int64_t ev0, const int *perm,
                                int64_t io_off, int mode, float *p, cudaStream_t st)
{
    if (count == 0) return cudaSuccess;
    k_brick_finish<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(bs->cf, acc, first, count, (int)ev0, perm, io_off, mode, p);
    return cudaGetLastError();
}

} // namespace jp
