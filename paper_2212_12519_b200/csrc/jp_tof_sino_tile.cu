// jp_tof_sino_tile.cu -- TOF sinogram forward / back projection and the fused OSEM subset pass on the TRACK TILES of a
// regular sinogram plan (jp_sino_plan.cu): the kernels behind jp_fwd_tof_sino_planned / jp_back_tof_sino_planned /
// jp_sino_osem_tof_planned.
//
// PAPER.md:33 (Joseph), :35 / :78 (TOF kernel: Gaussian integrated over the bin, truncated), :43 (sinogram mode: every
// plane step contributes to ALL TOF bins along the ray), :44 / :46 (exact adjoint by atomic adds).  BASELINE.json
// north_star (b): "back projection that uses warp-level aggregation or shared-memory tile staging before global
// atomicAdd".
//
// A CTA takes a SLICE of one track: kTS LORs that share their transaxial end points.  As in jp_tile.cu the q1 half of
// the bilinear interpolation is common to the slice:
//
//   forward   C[i][z] = (1-w1(i)) f[i,k1(i),z] + w1(i) f[i,k1(i)+1,z]    rows in shared memory, (intercept, slope) form;
//             a plane step of a LOR is one 64-bit shared load and one FMA instead of four global gathers;
//   adjoint   C[i][z] += cf (sum_k w_k y[j,k]) hat(u2(i) - z)              fixed-point shared atomics, then every row is
//             spread over its two image rows with 128-bit REDs -- one global atomic per (plane, 4 voxels) of the
//             slice instead of four per LOR and plane.
//
// The slice is not kTS consecutive LORs but kTS consecutive entries of the plan's LANE ORDER (LORs sorted by axial
// tilt |ze - zs|): the lanes of a warp then have the same LOR length, hence the same TOF coordinate on every plane,
// so the row of the TOF weight table (jp_tof_win.cuh) a warp reads per step is a shared-memory broadcast and its
// TOF window slides in lockstep.  The TOF bins of the window live in registers (a bin is written / its y read once,
// when the window passes it); the slice's [n_tofbins][kTS] values are staged through shared memory and moved
// to / from global memory one LOR row (n_tofbins contiguous floats) per warp instruction.
// Planes are walked in the direction of increasing TOF coordinate ("walk order" r = 0 .. I1 - I0), in chunks of
// rows_cap rows.  Tracks on which a LOR could have principal axis z, slices whose y holds a non-finite value, and
// images too wide for the shared rows take a per-LOR path with the same table and window.
#include "jp_tile_common.cuh"
#include "jp_tof_win.cuh"

namespace jp {

using namespace tile;
using namespace tofwin;

namespace {

constexpr int kTS = kSinoSlice;  // threads per CTA = LORs per slice
constexpr int kTSLd = kTS + 1;
constexpr int kNW = kTS / 32;

struct TrackX {
    Track t;
    double Rd;  // 1 + (d_q1 / d_p)^2
    double adp; // |d_p|
    int dir;    // +1: the TOF coordinate increases with the plane index
    int generic;
    float xs, ys, xe, ye;
    int rmin, rmax; // union of the LORs' walk ranges
};

// axial + TOF part of one LOR on track X, in walk order r (plane i(r) = I0 + r or I1 - r)
struct SRay {
    int r_lo, r_hi; // empty if r_hi < r_lo
    float a2, b2;   // u2(r) - kc = a2 + b2 (r - r_lo)
    float a2u;      // u2(r_lo), not shifted (the fixed-point rows of the adjoint)
    float cf;
    float q0, dq;   // kGK x (bin coordinate minus R) at r_lo; increment per plane (>= 0)
    float qr0;      // the same at walk position r = 0 (identical for all LORs of the track with the same |ze - zs|)
};

__device__ __forceinline__ SRay sino_setup(const Geom &g, const TrackX &X, float zs, float ze, const Tof &t, float cbR,
                                           float reach, double kc)
{
    const Track &tr = X.t;
    SRay z;
    const double dz = (double)ze - (double)zs;
    const double rz = dz * tr.inv_dp;
    const double vp = (double)g.v[tr.p];
    const double B = rz * vp * tr.iv2;
    const double A = ((double)zs - (double)g.o[2] + tr.ops * rz) * tr.iv2 - kc;
    const double Ln = dsqrt_pos(X.Rd + rz * rz); // L / |d_p|
    z.cf = (float)(vp * Ln);
    const double L = Ln * X.adp;
    const double dtau = vp * tr.inv_dp * L;                            // per plane (reading A8)
    const double tau0 = (tr.ops * tr.inv_dp - 0.5) * L - (double)t.coff; // at plane 0
    int ilo = tr.I0, ihi = tr.I1;
    { // planes inside the reach of the TOF bins, rounded outwards (outside it every weight is exactly zero)
        const double ivt = drcp(dtau);
        const double ia = (-(double)reach - tau0) * ivt, ib = ((double)reach - tau0) * ivt;
        const double np = (double)g.n[tr.p];
        const double imin = fmin(fmax(floor(fmin(ia, ib)), -1.0), np), imax = fmin(fmax(ceil(fmax(ia, ib)), -1.0), np);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    const float kcf = (float)kc;
    const float Af = (float)A, Bf = (float)B, ulo = -1.f - kcf, uhi = (float)g.n[2] - kcf;
    if (Bf == 0.f) {
        if (Af <= ulo || Af >= uhi) ihi = ilo - 1;
    } else {
        const float inv = 1.f / Bf;
        const float ia = (ulo - Af) * inv, ib = (uhi - Af) * inv;
        const float imin = fminf(fmaxf(floorf(fminf(ia, ib)) - 1.f, -1.f), (float)g.n[tr.p]);
        const float imax = fminf(fmaxf(ceilf(fmaxf(ia, ib)) + 1.f, -1.f), (float)g.n[tr.p]);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    // walk order
    const int dir = X.dir;
    int r_lo = dir > 0 ? ilo - tr.I0 : tr.I1 - ihi;
    int r_hi = dir > 0 ? ihi - tr.I0 : tr.I1 - ilo;
    const int ifirst = dir > 0 ? tr.I0 : tr.I1;
    auto u_at = [&](int r) { return (float)(A + B * (double)(ifirst + dir * r)); };
    z.b2 = (float)(B * (double)dir);
    z.a2 = u_at(r_lo);
    // trim: floor(u2) must stay inside the padded shared row, -2 <= floor(u2) <= n2, evaluated with the loop's own FMA
    // (planes trimmed away have all four neighbours outside the image and contribute exactly zero)
    const float umin = ulo - 0.9f, umax = uhi + 0.9f;
    while (r_lo <= r_hi) {
        if (z.a2 > umin && z.a2 < umax) break;
        ++r_lo;
        z.a2 = u_at(r_lo);
    }
    while (r_lo <= r_hi) {
        const float u = fmaf(z.b2, (float)(r_hi - r_lo), z.a2);
        if (u > umin && u < umax) break;
        --r_hi;
    }
    z.r_lo = r_lo;
    z.r_hi = r_hi;
    z.a2u = (float)(A + kc + B * (double)(ifirst + dir * r_lo));
    const double sc = (double)tofwin::kGK / (double)t.width, off = (double)cbR * (double)tofwin::kGK;
    z.dq = (float)(fabs(dtau) * sc);
    z.qr0 = (float)((tau0 + dtau * (double)ifirst) * sc + off);
    z.q0 = (float)((tau0 + dtau * (double)(ifirst + dir * r_lo)) * sc + off);
    return z;
}

template <int OFF>
__device__ __forceinline__ void reds_add_s(uint32_t addr, int q)
{
    asm volatile("red.shared.add.s32 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "r"(q) : "memory");
}

// TOF bin coordinates are carried scaled by kGK (table rows): q = kGK (s - R).  kMagicG = 1.5 x 2^23 x kGK: adding it
// rounds q to a multiple of kGK, so  cq = (q + kMagicG)_ru - kMagicG = kGK ceil(s - R)  and  cq - q  is the table row.
constexpr float kMagicG = 12582912.f * (float)kGK;
constexpr float kGKf = (float)kGK;
constexpr int kGMax = kSinoGroupsMax; // groups (LORs of equal |ze - zs|) per slice that get shared weight rows

// TOF window of one LOR: NBW bins starting at `base`, values in registers
template <int NBW>
struct Win {
    float a[NBW];
    float baseq; // kGK * base
    int base;
};

// slide the window up to scaled bin coordinate cq (forward: retire bins into the stage; back: fetch the bins entering)
template <int NBW, bool BACK>
__device__ __forceinline__ void win_slide(Win<NBW> &w, float cq, float *__restrict__ stage, int slot, int nbins, float cf)
{
#pragma unroll 1
    while (cq > w.baseq) { // false for NaN
        if (BACK) {
#pragma unroll
            for (int n = 0; n + 1 < NBW; ++n) w.a[n] = w.a[n + 1];
            w.a[NBW - 1] = ((unsigned)(w.base + NBW) < (unsigned)nbins) ? stage[(w.base + NBW) * kTSLd + slot] : 0.f;
        } else {
            if ((unsigned)w.base < (unsigned)nbins) stage[w.base * kTSLd + slot] = cf * w.a[0];
#pragma unroll
            for (int n = 0; n + 1 < NBW; ++n) w.a[n] = w.a[n + 1];
            w.a[NBW - 1] = 0.f;
        }
        w.baseq += kGKf;
        ++w.base;
    }
}

template <int NBW, bool BACK>
__device__ __forceinline__ void win_init(Win<NBW> &w, float q0, const float *__restrict__ stage, int slot, int nbins)
{
    w.baseq = __fadd_ru(q0, kMagicG) - kMagicG; // kGK ceil(s - R)
    w.base = (int)(w.baseq * (1.f / kGKf));
#pragma unroll
    for (int n = 0; n < NBW; ++n)
        w.a[n] = (BACK && (unsigned)(w.base + n) < (unsigned)nbins) ? stage[(w.base + n) * kTSLd + slot] : 0.f;
}

template <int NBW>
__device__ __forceinline__ void win_flush(const Win<NBW> &w, float *__restrict__ stage, int slot, int nbins, float cf)
{
#pragma unroll
    for (int n = 0; n < NBW; ++n)
        if ((unsigned)(w.base + n) < (unsigned)nbins) stage[(w.base + n) * kTSLd + slot] = cf * w.a[n];
}

// weights of the window bins on a plane with scaled bin coordinate q, from the table; returns cq = kGK ceil(s - R)
template <int NBW>
__device__ __forceinline__ float tab_weights(float q, uint32_t tab_addr, float (&wt)[NBW])
{
    const float cq = __fadd_ru(q, kMagicG) - kMagicG;
    const float tk = cq - q;
    const float tt = __fadd_rd(tk, kMagic);
    const float f = tk - (tt - kMagic);
    const uint32_t row = tab_addr + __float_as_uint(tt) * (uint32_t)(NBW * 8);
    load_weights<NBW, 0>(row, f, wt);
    return cq;
}

// ---- shared weight rows: one entry per (group, plane of the chunk) = the NBW weights and cq -------------------------
template <int NBW>
struct WEntry {
    static constexpr int kFloats = ((NBW + 1 + 3) / 4) * 4;
};

template <int NBW, int N>
__device__ __forceinline__ void load_wentry(uint32_t addr, float (&v)[WEntry<NBW>::kFloats])
{
    if constexpr (N < WEntry<NBW>::kFloats) {
        const float4 x = lds_quad<N * 4>(addr);
        v[N] = x.x;
        v[N + 1] = x.y;
        v[N + 2] = x.z;
        v[N + 3] = x.w;
        load_wentry<NBW, N + 4>(addr, v);
    }
}

// per-LOR path (any principal axis, global gathers / atomics on the unpadded image): same table, same window
template <int NBW, bool BACK>
__device__ __forceinline__ void generic_walk(const double (&s)[3], const double (&e)[3], const Geom &g, const Tof &t,
                                             const GTab &gt, uint32_t tab_addr, float *__restrict__ stage, int slot,
                                             float reach, const float *__restrict__ img_r, float *__restrict__ img_w)
{
    Ray r;
    ray_setup_pts<true>(s, e, g, t.coff, -reach, reach, r);
    if (r.nk == 0) return;
    const int nbins = t.nbins;
    const float dq = r.dtau * gt.inv_w * kGKf;
    const float q0 = fmaf(r.tau0, gt.inv_w, gt.cbR) * kGKf;
    int k = 0, dk = 1;
    if (dq < 0.f) {
        k = r.nk - 1;
        dk = -1;
    }
    Win<NBW> w;
    win_init<NBW, BACK>(w, fmaf(dq, (float)k, q0), stage, slot, nbins);
    for (int it = 0; it < r.nk; ++it, k += dk) {
        float wt[NBW];
        const float cq = tab_weights<NBW>(fmaf(dq, (float)k, q0), tab_addr, wt);
        win_slide<NBW, BACK>(w, cq, stage, slot, nbins, r.cf);
        const Cell cl = plane_cell(r, k);
        if (BACK) {
            float sm = 0.f;
#pragma unroll
            for (int n = 0; n < NBW; ++n) sm = fmaf(w.a[n], wt[n], sm);
            if (sm != 0.f) plane_scatter(img_w, r, k, cl, r.cf * sm);
        } else {
            const float val = plane_value(img_r, r, k, cl);
#pragma unroll
            for (int n = 0; n < NBW; ++n) w.a[n] = fmaf(val, wt[n], w.a[n]);
        }
    }
    if (!BACK) win_flush<NBW>(w, stage, slot, nbins, r.cf);
}

struct TileArgs {
    const float4 *trk;
    const float2 *zpat;
    const int *order;
    const unsigned char *slot_grp; // [T] group of every entry of the lane order, numbered from 0 inside its slice
    const int *slice_ng;           // [slices] groups of the slice (0: more than kGMax -> per-lane weights)
    int T;
    double dz_max;
    int64_t k0, nk; // tracks
    const float *img_r;
    float *img_w;
    Geom g;
    Tof t;
    GTab gt;
    int P;        // row pitch (0: image too wide for shared rows -> per-LOR path)
    int rows_cap; // rows per chunk
    int vec_r, vec_w;
    float *p;
    const float *y;
    SinoEpi epi;
};

// MODE 0: forward, 1: back, 2: OSEM subset pass (forward, ratio, back)
template <int NBW, int MODE>
__global__ void __launch_bounds__(kTS, 2) k_tof_sino_tile(TileArgs A)
{
    constexpr int WE = WEntry<NBW>::kFloats;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nbins = A.t.nbins;
    const int np = max(A.g.n[0], A.g.n[1]);
    const int rows_cap = A.rows_cap;
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);                                         // [(kGK + 2)][NBW]
    float *stage = reinterpret_cast<float *>(smem_raw + (size_t)(kGK + 2) * NBW * sizeof(float2)); // [nbins][kTSLd]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(stage + (((size_t)nbins * kTSLd + 3) & ~(size_t)3)); // [np], walk order
    int *kidx = reinterpret_cast<int *>(rinfo + np);                                            // [kTS]
    float *Wt = reinterpret_cast<float *>(kidx + kTS);                                          // [kGMax][rows_cap][WE]
    unsigned char *rows_raw = reinterpret_cast<unsigned char *>(Wt + (size_t)kGMax * rows_cap * WE); // float2 / int [rows_cap][P]
    float2 *C2 = reinterpret_cast<float2 *>(rows_raw);
    int *Ci = reinterpret_cast<int *>(rows_raw);
    __shared__ TrackX X;
    __shared__ float red[kNW];
    __shared__ float2 grpq[kGMax]; // per group: scaled bin coordinate at walk position 0, increment per plane
    __shared__ int flag_nonfinite;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const Geom &g = A.g;
    const Tof &t = A.t;
    const int P = A.P, n2 = g.n[2];
    for (int i = tid; i < (kGK + 2) * NBW; i += kTS) tab[i] = __ldg(A.gt.tab + i);
    for (int i = tid; i < nbins * kTSLd; i += kTS) stage[i] = 0.f;
    uint32_t tab_addr = smem_addr(tab) - (uint32_t)kMagicI * (uint32_t)(NBW * 8);
    const float reach = 0.5f * (float)(nbins - 1) * t.width + 0.5f * t.width + t.nsig * t.sigma;
    const int kci = n2 >> 1;
    uint32_t c2_base = smem_addr(C2) + (uint32_t)(kPad + kci) * 8u - ((uint32_t)kMagicI << 3);
    uint32_t ci_base = smem_addr(Ci) + kPad * 4u - ((uint32_t)kMagicI << 2);
    uint32_t wt_base = smem_addr(Wt);
    // keep the biased shared-memory addresses in registers: left to itself the compiler rematerialises them (an S2R
    // and three integer adds) inside the plane loops
    asm volatile("" : "+r"(tab_addr), "+r"(c2_base), "+r"(ci_base), "+r"(wt_base));
    const int T = A.T;
    const int nsl = (T + kTS - 1) / kTS;
    const int64_t items = A.nk * nsl;

    for (int64_t item = blockIdx.x; item < items; item += gridDim.x) {
        const int64_t trk = A.k0 + item / nsl;
        const int sl = (int)(item % nsl);
        const int64_t j0 = trk * (int64_t)T;
        const int nv = min(kTS, T - sl * kTS);
        __syncthreads(); // the previous item is done with X, the stage and the rows
        if (tid == 0) {
            const float4 q = __ldg(A.trk + trk);
            X.xs = q.x; X.ys = q.y; X.xe = q.z; X.ye = q.w;
            const double dxy[2] = {(double)q.z - (double)q.x, (double)q.w - (double)q.y};
            const double dmax = fmax(fabs(dxy[0]), fabs(dxy[1]));
            X.generic = (P == 0 || !(dmax > 0.0) || A.dz_max > dmax) ? 1 : 0; // some LOR may have principal axis z
            X.rmin = 0x7fffffff;
            X.rmax = -1;
            flag_nonfinite = 0;
            if (!X.generic) {
                track_setup(g, q.x, q.y, q.z, q.w, X.t);
                const double ratio = dxy[1 - X.t.p] * X.t.inv_dp;
                X.Rd = 1.0 + ratio * ratio;
                X.adp = fabs(dxy[X.t.p]);
                X.dir = (dxy[X.t.p] > 0.0) ? 1 : -1;
            }
        }
        __syncthreads();
        const bool generic = X.generic != 0;
        const bool miss = !generic && X.t.I1 < X.t.I0;
        if (miss) { // the whole track misses the image
            if (MODE == 0) { // zeros, in list order (a flat range)
                float *out = A.p + (j0 + (int64_t)sl * kTS) * nbins;
                const int tot = nv * nbins;
                if ((((uintptr_t)out) & 15) == 0) {
                    float4 *o4 = reinterpret_cast<float4 *>(out);
                    for (int x = tid; x < tot / 4; x += kTS) o4[x] = make_float4(0.f, 0.f, 0.f, 0.f);
                    for (int x = (tot & ~3) + tid; x < tot; x += kTS) out[x] = 0.f;
                } else {
                    for (int x = tid; x < tot; x += kTS) out[x] = 0.f;
                }
            }
            continue;
        }
        // ---- this thread's LOR: slot tid of the slice = entry sl * kTS + tid of the lane order
        const int kk = (tid < nv) ? __ldg(A.order + sl * kTS + tid) : -1;
        kidx[tid] = kk;
        const int NG = generic ? 0 : __ldg(A.slice_ng + sl); // 0: weights per lane
        const int gid = (NG > 0 && kk >= 0) ? (int)__ldg(A.slot_grp + sl * kTS + tid) : 0;
        float zs = 0.f, ze = 0.f;
        if (kk >= 0) {
            const float2 zz = __ldg(A.zpat + kk);
            zs = zz.x;
            ze = zz.y;
        }
        SRay zr;
        zr.r_lo = 0;
        zr.r_hi = -1;
        zr.a2 = zr.b2 = zr.a2u = zr.cf = zr.q0 = zr.dq = zr.qr0 = 0.f;
        if (!generic) {
            if (kk >= 0) {
                zr = sino_setup(g, X, zs, ze, t, A.gt.cbR, reach, (double)kci);
                if (NG > 0) grpq[gid] = make_float2(zr.qr0, zr.dq); // the same bits from every LOR of the group
            }
            int lo = zr.r_hi >= zr.r_lo ? zr.r_lo : 0x7fffffff, hi = zr.r_hi >= zr.r_lo ? zr.r_hi : -1;
            for (int o = 16; o > 0; o >>= 1) {
                lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
                hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
            }
            if (lane == 0 && hi >= lo) {
                atomicMin(&X.rmin, lo);
                atomicMax(&X.rmax, hi);
            }
            const Track &tr = X.t;
            const int nr = tr.I1 - tr.I0;
            for (int r = tid; r <= nr; r += kTS) rinfo[r] = row_info(g, tr, X.dir > 0 ? tr.I0 + r : tr.I1 - r);
        }
        __syncthreads(); // kidx, rinfo, grpq, X.rmin / rmax
        const double sp[3] = {(double)X.xs, (double)X.ys, (double)zs}, ep[3] = {(double)X.xe, (double)X.ye, (double)ze};
        const bool live = zr.r_hi >= zr.r_lo;
        // scaled bin coordinate of the first plane: with shared weight rows the SAME float32 expression that builds the
        // rows, so that the window a lane opens and the window the row was made for cannot differ by a rounding
        const float q_init = NG > 0 ? fmaf(grpq[gid].y, (float)zr.r_lo, grpq[gid].x) : zr.q0;

        // the weight rows of chunk [r0, r0 + rows): thread e -> (group, plane)
        auto build_wt = [&](int r0, int rows) {
            if (tid < NG * rows) {
                const int gq = tid / rows, rr = tid - gq * rows;
                const float2 gp = grpq[gq];
                float wt[NBW];
                const float cq = tab_weights<NBW>(fmaf(gp.y, (float)(r0 + rr), gp.x), tab_addr, wt);
                float *dst = Wt + (size_t)(gq * rows_cap + rr) * WE;
#pragma unroll
                for (int n = 0; n < NBW; ++n) dst[n] = wt[n];
                dst[NBW] = cq;
            }
        };

        // ======== forward (MODE 0, 2): walk into the window registers, retire bins into the stage =======================
        if (MODE != 1) {
            if (generic) {
                if (kk >= 0) generic_walk<NBW, false>(sp, ep, g, t, A.gt, tab_addr, stage, tid, reach, A.img_r, nullptr);
            } else if (X.rmax >= X.rmin) {
                // constant zero columns of the shared rows
                {
                    const int ncl = kPad - 1, ncr = P - (n2 + kPad);
                    for (int e = tid; e < rows_cap * (ncl + ncr); e += kTS) {
                        const int r = e / (ncl + ncr), c = e - r * (ncl + ncr);
                        C2[r * P + (c < ncl ? c : n2 + kPad + (c - ncl))] = make_float2(0.f, 0.f);
                    }
                }
                Win<NBW> w;
                win_init<NBW, false>(w, q_init, stage, tid, nbins);
                const int R0 = X.rmin, R1 = X.rmax;
                for (int r0 = R0; r0 <= R1; r0 += rows_cap) {
                    const int rows = min(rows_cap, R1 - r0 + 1);
                    __syncthreads(); // the previous chunk's rows are no longer read
                    build_rows<0, true, 1, kTS>(C2, rinfo, A.img_r, X.t, X.t.I0 + r0, rows, n2, A.vec_r, (float)kci, P);
                    build_wt(r0, rows);
                    __syncthreads();
                    const int rb = max(zr.r_lo, r0), re = min(zr.r_hi, r0 + rows - 1);
                    if (rb <= re) {
                        float fk = (float)(rb - zr.r_lo);
                        uint32_t row = c2_base + (uint32_t)((rb - r0) * P) * 8u;
                        if (NG > 0) {
                            uint32_t wrow = wt_base + (uint32_t)((gid * rows_cap + (rb - r0)) * WE) * 4u;
#pragma unroll 2
                            for (int it = re - rb + 1; it > 0; --it) {
                                const float u = fmaf(zr.b2, fk, zr.a2);
                                const float tt = __fadd_rd(u, kMagic);
                                const float2 v = lds_pair<0>(row + (__float_as_uint(tt) << 3));
                                float wv[WE];
                                load_wentry<NBW, 0>(wrow, wv);
                                win_slide<NBW, false>(w, wv[NBW], stage, tid, nbins, zr.cf);
                                const float val = fmaf(u, v.y, v.x);
#pragma unroll
                                for (int n = 0; n < NBW; ++n) w.a[n] = fmaf(val, wv[n], w.a[n]);
                                fk += 1.f;
                                row += (uint32_t)P * 8u;
                                wrow += WE * 4u;
                            }
                        } else {
#pragma unroll 1
                            for (int it = re - rb + 1; it > 0; --it) {
                                const float u = fmaf(zr.b2, fk, zr.a2);
                                const float tt = __fadd_rd(u, kMagic);
                                const float2 v = lds_pair<0>(row + (__float_as_uint(tt) << 3));
                                float wt[NBW];
                                const float cq = tab_weights<NBW>(fmaf(zr.dq, fk, zr.q0), tab_addr, wt);
                                win_slide<NBW, false>(w, cq, stage, tid, nbins, zr.cf);
                                const float val = fmaf(u, v.y, v.x);
#pragma unroll
                                for (int n = 0; n < NBW; ++n) w.a[n] = fmaf(val, wt[n], w.a[n]);
                                fk += 1.f;
                                row += (uint32_t)P * 8u;
                            }
                        }
                    }
                }
                if (live) win_flush<NBW>(w, stage, tid, nbins, zr.cf);
            }
            __syncthreads(); // the stage holds p[slot][:] of the slice
        }

        // ======== forward: write the LOR rows (and clear the stage) ==========================================================
        if (MODE == 0) {
            float *st_lo = stage + lane * kTSLd, *st_hi = stage + (lane + 32) * kTSLd; // JP_MAX_TOFBINS = 64: two halves
            const bool lo_ok = lane < nbins, hi_ok = lane + 32 < nbins;
#pragma unroll 4
            for (int s0 = warp; s0 < nv; s0 += kNW) {
                float *out = A.p + (j0 + kidx[s0]) * nbins + lane;
                if (lo_ok) {
                    out[0] = st_lo[s0];
                    st_lo[s0] = 0.f;
                }
                if (hi_ok) {
                    out[32] = st_hi[s0];
                    st_hi[s0] = 0.f;
                }
            }
            continue;
        }

        // ======== back (MODE 1): stage the y rows (or the broadcast values of a sensitivity image) ======================
        if (MODE == 1) {
            if (A.epi.mult_bcast || A.epi.ones_bcast) {
                const float v = (kk >= 0) ? (A.epi.mult_bcast ? A.epi.mult_bcast[j0 + kk] : 1.f) : 0.f;
                for (int b = 0; b < nbins; ++b) stage[b * kTSLd + tid] = v;
            } else {
                for (int s0 = warp; s0 < kTS; s0 += 4 * kNW) {
                    float v[4][2];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int sx = s0 + u * kNW;
                        const int64_t j = j0 + (sx < nv ? kidx[sx] : 0);
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int b = lane + 32 * h;
                            v[u][h] = (sx < nv && b < nbins) ? A.y[j * nbins + b] : 0.f;
                        }
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int sx = s0 + u * kNW;
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int b = lane + 32 * h;
                            if (sx < kTS && b < nbins) stage[b * kTSLd + sx] = v[u][h];
                        }
                    }
                }
            }
            __syncthreads();
        }

        // ======== OSEM (MODE 2): the ratio in place (reading S2) =========================================================
        if (MODE == 2) {
            const bool lo_ok = lane < nbins, hi_ok = lane + 32 < nbins;
#pragma unroll 2
            for (int s0 = warp; s0 < nv; s0 += kNW) {
                const int64_t j = j0 + kidx[s0];
                const float mv = A.epi.mult ? A.epi.mult[j] : 1.f;
                const int64_t e = j * nbins + lane;
                float y0 = 0.f, y1 = 0.f, c0 = 0.f, c1 = 0.f;
                if (lo_ok) y0 = A.epi.y_em[e];
                if (hi_ok) y1 = A.epi.y_em[e + 32];
                if (A.epi.contam) {
                    if (lo_ok) c0 = A.epi.contam[e];
                    if (hi_ok) c1 = A.epi.contam[e + 32];
                }
                if (lo_ok) {
                    float *sp2 = stage + lane * kTSLd + s0;
                    const float yb = fmaf(mv, *sp2, c0);
                    *sp2 = (yb > 1e-9f) ? mv * y0 / yb : 0.f;
                }
                if (hi_ok) {
                    float *sp2 = stage + (lane + 32) * kTSLd + s0;
                    const float yb = fmaf(mv, *sp2, c1);
                    *sp2 = (yb > 1e-9f) ? mv * y1 / yb : 0.f;
                }
            }
            __syncthreads();
        }

        // ======== back walk (MODE 1, 2) ==================================================================================
        bool use_generic = generic;
        bool any_value = true;
        if (!generic) {
            // Inf / NaN anywhere in the values of a LOR that crosses the image -> per-LOR float path for the slice
            float xm = 0.f;
            if (live) {
                bool bad = false;
                for (int b = 0; b < nbins; ++b) {
                    const float v = fabsf(stage[b * kTSLd + tid]);
                    bad = bad || !(v < 3.0e38f); // Inf or NaN (fmaxf would drop a NaN)
                    xm = fmaxf(xm, v);
                }
                if (bad) atomicExch(&flag_nonfinite, 1);
            }
            for (int o = 16; o > 0; o >>= 1) xm = fmaxf(xm, __shfl_xor_sync(0xffffffffu, xm, o));
            if (lane == 0) red[warp] = xm;
            // zero the fixed-point rows (MODE 2: the forward rows are dead)
            {
                int4 *z4 = reinterpret_cast<int4 *>(Ci);
                for (int e = tid; e < rows_cap * (P / 4); e += kTS) z4[e] = make_int4(0, 0, 0, 0);
            }
            __syncthreads();
            xm = red[0];
#pragma unroll
            for (int w2 = 1; w2 < kNW; ++w2) xm = fmaxf(xm, red[w2]);
            use_generic = flag_nonfinite != 0; // propagate Inf / NaN exactly as the per-LOR adjoint does
            any_value = xm > 0.f;
        }
        if (use_generic) {
            if (kk >= 0) generic_walk<NBW, true>(sp, ep, g, t, A.gt, tab_addr, stage, tid, reach, nullptr, A.img_w);
        } else if (any_value && X.rmax >= X.rmin) {
            // Fixed-point staging with a scale per CHUNK of planes: S = lim / Xc, Xc = max over the slice's LORs of
            // cf x max |value| over the TOF bins whose window is open on the chunk's planes (the weights of a step sum
            // to <= 1, so |cf sum_k w_k value_k| <= Xc).  Rounding error per contribution <= 2.4e-7 Xc.
            Win<NBW> w;
            win_init<NBW, true>(w, q_init, stage, tid, nbins);
            const int R0 = X.rmin, R1 = X.rmax;
            const float lim = 4194302.f; // |c S| <= 2^22 - 2 and kTS |c S| < 2^31
            for (int r0 = R0; r0 <= R1; r0 += rows_cap) {
                const int rows = min(rows_cap, R1 - r0 + 1);
                const int rb = max(zr.r_lo, r0), re = min(zr.r_hi, r0 + rows - 1);
                build_wt(r0, rows);
                { // bound of this LOR's contributions in the chunk
                    float xm = 0.f;
                    if (rb <= re) {
                        const float qe = fmaf(zr.dq, (float)(re - zr.r_lo), zr.q0);
                        const int k_hi = min(nbins - 1, (int)((__fadd_ru(qe, kMagicG) - kMagicG) * (1.f / kGKf)) + NBW);
                        for (int k = max(w.base, 0); k <= k_hi; ++k) xm = fmaxf(xm, fabsf(stage[k * kTSLd + tid]));
                        xm *= zr.cf;
                    }
                    for (int o = 16; o > 0; o >>= 1) xm = fmaxf(xm, __shfl_xor_sync(0xffffffffu, xm, o));
                    if (lane == 0) red[warp] = xm;
                }
                __syncthreads(); // weight rows, red; the previous chunk's flush is complete
                float xc = red[0];
#pragma unroll
                for (int w2 = 1; w2 < kNW; ++w2) xc = fmaxf(xc, red[w2]);
                if (!(xc > 0.f)) { // nothing to add on these planes (block-uniform)
                    __syncthreads(); // red is rewritten by the next chunk
                    continue;
                }
                const float S = lim / xc, invS = xc / lim;
                if (rb <= re) {
                    const float xs_ = zr.cf * S;
                    float fk = (float)(rb - zr.r_lo);
                    uint32_t row = ci_base + (uint32_t)((rb - r0) * P) * 4u;
                    if (NG > 0) {
                        uint32_t wrow = wt_base + (uint32_t)((gid * rows_cap + (rb - r0)) * WE) * 4u;
#pragma unroll 2
                        for (int it = re - rb + 1; it > 0; --it) {
                            const float u = fmaf(zr.b2, fk, zr.a2u);
                            const float tt = __fadd_rd(u, kMagic);
                            const float wz = u - (tt - kMagic);
                            const uint32_t a = row + (__float_as_uint(tt) << 2);
                            float wv[WE];
                            load_wentry<NBW, 0>(wrow, wv);
                            win_slide<NBW, true>(w, wv[NBW], stage, tid, nbins, zr.cf);
                            float sm = 0.f;
#pragma unroll
                            for (int n = 0; n < NBW; ++n) sm = fmaf(w.a[n], wv[n], sm);
                            const float xw = xs_ * sm;
                            const int qxw = __float_as_int(xw + kMagic);
                            const int bits = __float_as_int(fmaf(xw, wz, kMagic));
                            reds_add_s<0>(a, qxw - bits);
                            reds_add_s<4>(a, bits - kMagicI);
                            fk += 1.f;
                            row += (uint32_t)P * 4u;
                            wrow += WE * 4u;
                        }
                    } else {
#pragma unroll 1
                        for (int it = re - rb + 1; it > 0; --it) {
                            const float u = fmaf(zr.b2, fk, zr.a2u);
                            const float tt = __fadd_rd(u, kMagic);
                            const float wz = u - (tt - kMagic);
                            const uint32_t a = row + (__float_as_uint(tt) << 2);
                            float wt[NBW];
                            const float cq = tab_weights<NBW>(fmaf(zr.dq, fk, zr.q0), tab_addr, wt);
                            win_slide<NBW, true>(w, cq, stage, tid, nbins, zr.cf);
                            float sm = 0.f;
#pragma unroll
                            for (int n = 0; n < NBW; ++n) sm = fmaf(w.a[n], wt[n], sm);
                            const float xw = xs_ * sm;
                            const int qxw = __float_as_int(xw + kMagic);
                            const int bits = __float_as_int(fmaf(xw, wz, kMagic));
                            reds_add_s<0>(a, qxw - bits);
                            reds_add_s<4>(a, bits - kMagicI);
                            fk += 1.f;
                            row += (uint32_t)P * 4u;
                        }
                    }
                }
                __syncthreads();
                // ---- flush: spread every row over its two q1 neighbours with REDs, and clear it
                if (A.vec_w) {
                    const int G = n2 >> 2;
                    for (int r = warp; r < rows; r += kNW) {
                        const RowInfo ri = rinfo[r0 + r];
                        const float sa = ri.wa * invS, sb = ri.wb * invS;
                        for (int gq = lane; gq < G; gq += 32) {
                            int4 *src = reinterpret_cast<int4 *>(Ci + r * P + kPad) + gq;
                            const int4 q = *src;
                            if ((q.x | q.y | q.z | q.w) == 0) continue;
                            *src = make_int4(0, 0, 0, 0);
                            const float4 v = make_float4((float)q.x, (float)q.y, (float)q.z, (float)q.w);
                            if (ri.base_a >= 0)
                                atomicAdd(reinterpret_cast<float4 *>(A.img_w + ri.base_a) + gq,
                                          make_float4(sa * v.x, sa * v.y, sa * v.z, sa * v.w));
                            if (ri.base_b >= 0)
                                atomicAdd(reinterpret_cast<float4 *>(A.img_w + ri.base_b) + gq,
                                          make_float4(sb * v.x, sb * v.y, sb * v.z, sb * v.w));
                        }
                    }
                } else {
                    for (int e = tid; e < rows * n2; e += kTS) {
                        const int r = e / n2, z = e - r * n2;
                        const int q = Ci[r * P + kPad + z];
                        if (q == 0) continue;
                        Ci[r * P + kPad + z] = 0;
                        const RowInfo ri = rinfo[r0 + r];
                        const float v = (float)q * invS;
                        if (ri.base_a >= 0) atomicAdd(A.img_w + ri.base_a + z, ri.wa * v);
                        if (ri.base_b >= 0) atomicAdd(A.img_w + ri.base_b + z, ri.wb * v);
                    }
                }
                // (the barrier at the top of the next chunk, or of the next item, orders the flush against the next scatter)
            }
        }
        if (MODE == 2) { // the forward walk of the next item starts from zeros
            __syncthreads();
            for (int i = tid; i < nbins * kTSLd; i += kTS) stage[i] = 0.f;
        }
    }
}

struct TileCfgS {
    int P, rows_cap, vec_r, vec_w;
    size_t smem;
};

TileCfgS tile_cfg_s(const Geom &g, int nbw, int nbins, int mode, const void *img_r, const void *img_w)
{
    TileCfgS c{};
    const int need = g.n[2] + kPad + kPadR;
    const int pitches[] = {40, 72, 104, 136, 200, 264};
    for (int P : pitches)
        if (need <= P) { c.P = P; break; }
    const int np = g.n[0] > g.n[1] ? g.n[0] : g.n[1];
    const size_t we = (size_t)((nbw + 1 + 3) / 4) * 4;
    const size_t fixed = (size_t)(kGK + 2) * nbw * sizeof(float2) + ((((size_t)nbins * kTSLd + 3) & ~(size_t)3)) * sizeof(float) +
                         (size_t)np * sizeof(RowInfo) + (size_t)kTS * sizeof(int);
    const size_t elem = (mode == 1) ? sizeof(int) : sizeof(float2);
    const size_t wrow = (size_t)kGMax * we * sizeof(float); // weight rows of one plane
    const size_t budget = 110 * 1024;                       // two CTAs per SM
    size_t rows = 0;
    if (c.P) {
        const size_t row = (size_t)c.P * elem + wrow;
        rows = fixed + 8 * row <= budget ? (budget - fixed) / row : 0;
        if (rows > (size_t)(kTS / kGMax)) rows = kTS / kGMax; // one thread per (group, plane) builds the weight rows
        if (rows > (size_t)np) rows = (size_t)np;
        if (rows < 8) { c.P = 0; rows = 0; }
    }
    c.rows_cap = (int)rows;
    c.smem = fixed + rows * ((size_t)c.P * elem + wrow);
    c.vec_r = (g.n[2] % 4 == 0) && ((uintptr_t)img_r % 16 == 0);
    c.vec_w = (g.n[2] % 4 == 0) && ((uintptr_t)img_w % 16 == 0);
    return c;
}

template <int NBW, int MODE>
cudaError_t launch_tile(const TileArgs &A, size_t smem, cudaStream_t st)
{
    auto kern = k_tof_sino_tile<NBW, MODE>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, nsm = 0, per_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kTS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorNotSupported;
    const int nsl = (A.T + kTS - 1) / kTS;
    const int64_t items = A.nk * nsl, cap = (int64_t)nsm * per_sm;
    kern<<<(unsigned)(items < cap ? items : cap), kTS, smem, st>>>(A);
    return cudaGetLastError();
}

} // namespace

int tof_window_bins(const Tof &t, double *R_out) { return window_bins(t, R_out); }

cudaError_t launch_tof_sino_tile(int mode, const SinoPlanView &pv, int64_t k0, int64_t nk, const float *img_r, float *img_w,
                                 const Geom &g, const Tof &t, float *p, const float *y, const SinoEpi *epi_in, cudaStream_t st)
{
    if (nk == 0) return cudaSuccess;
    if (!pv.regular) return cudaErrorNotSupported;
    GTab gt{};
    int nbw = 0;
    cudaError_t e = gtab_create(t, st, &gt, &nbw);
    if (e != cudaSuccess) return e;
    const TileCfgS c = tile_cfg_s(g, nbw, t.nbins, mode, img_r, img_w);
    if (c.smem > 200 * 1024) {
        gtab_destroy(&gt, st);
        return cudaErrorNotSupported;
    }
    TileArgs A{};
    A.trk = pv.trk; A.zpat = pv.zpat; A.order = pv.order; A.slot_grp = pv.slot_grp; A.slice_ng = pv.slice_ng;
    A.T = pv.T; A.dz_max = pv.dz_max;
    if (pv.slice_len != kTS) { // the plan's slices are not ours (never happens: both come from kSinoSlice)
        gtab_destroy(&gt, st);
        return cudaErrorNotSupported;
    }
    A.k0 = k0; A.nk = nk; A.img_r = img_r; A.img_w = img_w; A.g = g; A.t = t; A.gt = gt;
    A.P = c.P; A.rows_cap = c.rows_cap; A.vec_r = c.vec_r; A.vec_w = c.vec_w; A.p = p; A.y = y;
    A.epi = epi_in ? *epi_in : SinoEpi{};
#define JP_TILE_MODE(NB)                                          \
    case NB:                                                      \
        e = mode == 0 ? launch_tile<NB, 0>(A, c.smem, st)         \
          : mode == 1 ? launch_tile<NB, 1>(A, c.smem, st)         \
                      : launch_tile<NB, 2>(A, c.smem, st);        \
        break;
    switch (nbw) {
        JP_TILE_MODE(4)
        JP_TILE_MODE(6)
        JP_TILE_MODE(8)
        JP_TILE_MODE(12)
    default: e = cudaErrorNotSupported;
    }
#undef JP_TILE_MODE
    gtab_destroy(&gt, st);
    return e;
}

} // namespace jp
