// jp_lm_tile.cu -- TOF listmode forward / back projection on LINE TILES: the planned listmode calls over a
// sorted event list whose runs of events share their transaxial line.
//
// A ring scanner snaps events to crystal centres, so after the plan's sort (jp_plan.cu) thousands of events
// of configs[3] share the same transaxial projection (same crystal pair, any ring pair, any TOF bin, either
// orientation).  For such a run the q1 half of Joseph's bilinear interpolation is common to
// all its events, exactly as for the ring pairs of one sinogram bin (jp_tile.cu):
//
//   forward   C[i][z] = (1-w1(i)) f[i,k1(i),z] + w1(i) f[i,k1(i)+1,z]   rows built once per run in shared memory;
//             p_e     = cf_e sum_{i in TOF window of e} G_e(i) lerp_z(C[i][.], u2_e(i))
//   adjoint   C[i][z] += cf_e y_e G_e(i) hat(u2_e(i) - z)  (fixed-point shared atomics), then each row is
//             spread over its two image rows with 128-bit REDs: one global atomic per (plane, 4 voxels) of the
//             run instead of one per event and plane (north_star: shared-memory tile staging)
//
// G_e(i) is the TOF weight of the event's own bin, from a float64-built table of
// G(x) = 1/2 [E((x + 1/2) W) - E((x - 1/2) W)] over x = |c - tau| / W (reading A10).
// A CTA takes 768 consecutive sorted events, finds the runs inside them (bit-exact comparison of the
// canonically ordered transaxial end points) and processes run after run; an event given as (e, s) instead of
// (s, e) is walked in the canonical orientation with its axial end points swapped and its TOF centre negated
// (the kernel is even).  Runs shorter than kMinRun, and events whose principal axis is z, take the per-LOR path.
#include "jp_g1tab.cuh"
#include "jp_tile_common.cuh"

namespace jp {

using namespace tile;

namespace {

#ifndef JP_LMT_BACK_UNROLL
#define JP_LMT_BACK_UNROLL 2
#endif
#ifndef JP_LMT_MINB_FWD
#define JP_LMT_MINB_FWD 4
#endif
#ifndef JP_LMT_MINB_BACK
#define JP_LMT_MINB_BACK 5
#endif
constexpr int kMinRun = 48; // shorter runs are not worth a row build

// The table runs in the DISTANCE FROM THE SUPPORT EDGE, x' = R - |x| (bin widths, R = n_sigmas sigma / W + 1/2): the two
// kinks of the truncated kernel (A4: erf argument clamped at +- n_sigmas sigma) sit at x' = 0 and x' = 1, i.e. exactly
// on table nodes, so the piecewise-linear table never interpolates across one (tabulated in |x| the kinks fall inside
// an interval and the tail weights are off by up to 2.7e-6 absolute, 10 % of a 1e-5 weight)
__global__ void k_tof_g1tab(float2 *tab, int n, double W, double m, double isc)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const double R = m / W + 0.5;
    auto E = [&](double y) { return erf(fmin(fmax(y, -m), m) * isc); };
    auto G = [&](double xp) { const double x = R - xp; return 0.5 * (E((x + 0.5) * W) - E((x - 0.5) * W)); };
    const double g0 = k == 0 ? 0.0 : G((double)k / kG1K), g1 = G((double)(k + 1) / kG1K);
    tab[k] = make_float2((float)(g0 - (double)k * (g1 - g0)), (float)(g1 - g0)); // (intercept, slope): G = .x + x' .y
}


// canonical orientation of the transaxial end points: start = the lexicographically smaller (x, y)
__device__ __forceinline__ bool is_swapped(float xs, float ys, float xe, float ye)
{
    return !((xs < xe) || (xs == xe && ys <= ye));
}


// per-event axial + TOF part on track t (canonical orientation)
struct LmRay {
    int i0, i1;     // planes inside the image along z AND inside the TOF window of the event's bin
    float a2, b2;   // u2(i) = a2 + b2 (i - i0)
    float cf;
    float x0, dx;   // table position of plane i: x0 + dx (i - i0)
};

struct LineExtra {
    double Rd;      // 1 + (d_q1 / d_p)^2
};

template <bool TOF>
__device__ __forceinline__ LmRay lm_setup(const Geom &g, const Track &t, double Rd, float zs, float ze, float centre,
                                          float reach, float scale, double kc = 0.0) // kc: a2 is u2 - kc
{
    LmRay z;
    const double dz = (double)ze - (double)zs;
    const double rz = dz * t.inv_dp;
    const double vp = (double)g.v[t.p];
    const double iv2 = t.iv2;
    const double B = rz * vp * iv2;
    const double A = ((double)zs - (double)g.o[2] + t.ops * rz) * iv2 - kc;
    const double Ln = dsqrt_pos(Rd + rz * rz);   // L / |d_p|
    z.cf = (float)(vp * Ln);
    // tau(i) = ((ops + i vp) inv_dp - 1/2) L,  L = Ln / |inv_dp|
    const double L = Ln * fabs(drcp(t.inv_dp));
    const double dtau = vp * t.inv_dp * L;
    const double tau_at0 = (t.ops * t.inv_dp - 0.5) * L;
    int ilo = t.I0, ihi = t.I1;
    if (TOF) { // TOF window: |tau(i) - centre| <= reach, rounded outwards
        const double ivt = drcp(dtau);
        const double ia = ((double)centre - (double)reach - tau_at0) * ivt, ib = ((double)centre + (double)reach - tau_at0) * ivt;
        const double np = (double)g.n[t.p];
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
        const float imin = fminf(fmaxf(floorf(fminf(ia, ib)) - 1.f, -1.f), (float)g.n[t.p]);
        const float imax = fminf(fmaxf(ceilf(fmaxf(ia, ib)) + 1.f, -1.f), (float)g.n[t.p]);
        ilo = max(ilo, (int)imin);
        ihi = min(ihi, (int)imax);
    }
    z.b2 = Bf;
    z.a2 = (float)(A + B * (double)ilo);
    const float umin = ulo - 0.9f, umax = uhi + 0.9f;
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
    z.x0 = TOF ? (float)(((double)centre - (tau_at0 + dtau * (double)ilo)) * (double)scale) : 0.f;
    z.dx = TOF ? (float)(-dtau * (double)scale) : 0.f;
    return z;
}

// per-LOR path (short runs, principal axis z): same arithmetic as jp_kernels.cu on the unpadded image
template <bool TOF>
__device__ __forceinline__ float generic_fwd_lm(const Lors &l, int64_t j, float centre, float reach, const Geom &g,
                                                const Tof &t, const float *__restrict__ img, uint32_t gbase,
                                                const G1Tab &gt)
{
    Ray r;
    ray_setup<TOF>(l, j, g, t.coff, centre - reach, centre + reach, r);
    float acc = 0.f;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        const float tau = fmaf(r.dtau, (float)k, r.tau0);
        const float w = TOF ? g1_weight(gbase, gt.xedge, (centre - tau) * gt.scale) : 1.f;
        acc = fmaf(plane_value(img, r, k, cl), w, acc);
    }
    return r.cf * acc;
}

template <bool TOF>
__device__ __forceinline__ void generic_back_lm(const Lors &l, int64_t j, float centre, float reach, float y, const Geom &g,
                                                const Tof &t, float *__restrict__ img, uint32_t gbase, const G1Tab &gt)
{
    Ray r;
    ray_setup<TOF>(l, j, g, t.coff, centre - reach, centre + reach, r);
    const float x = r.cf * y;
    if (r.nk == 0 || x == 0.f) return;
    for (int k = 0; k < r.nk; ++k) {
        const Cell cl = plane_cell(r, k);
        const float tau = fmaf(r.dtau, (float)k, r.tau0);
        const float w = TOF ? g1_weight(gbase, gt.xedge, (centre - tau) * gt.scale) : 1.f;
        if (w != 0.f) plane_scatter(img, r, k, cl, x * w);
    }
}

// shared bookkeeping of a CTA
constexpr int kMaxLong = (kTile + kMinRun - 1) / kMinRun; // long runs (>= kMinRun events) of a window: slot = start / kMinRun

struct TileState {
    Track trk;      // adjoint kernel: the current run's track
    LineExtra ex;
    int nruns;
    int imin, imax;
    int bad;        // adjoint kernel: the current run holds a non-finite value on an event that crosses the image
    unsigned short starts[kTile + 1];
    // forward kernel: the tracks of ALL long runs of the window, set up in parallel before the run loop
    Track trks[kMaxLong];
    double Rds[kMaxLong];
    int imins[kMaxLong], imaxs[kMaxLong];
};

// runs of events with identical canonical transaxial end points among the CTA's nev events; canon = smem scratch
// of kTile uint4 (may alias the row buffer).  All threads; ends with a barrier.
__device__ __forceinline__ void find_runs(TileState &S, uint4 *canon, const uint4 (&mine)[kPerThread], int nev)
{
    const int tid = threadIdx.x;
#pragma unroll
    for (int m = 0; m < kPerThread; ++m) canon[m * kThreads + tid] = mine[m];
    __syncthreads();
    if (tid < 32) {
        int n = 0;
        for (int b0 = 0; b0 < nev; b0 += 32) {
            const int pos = b0 + tid;
            bool flag = false;
            if (pos < nev) {
                if (pos == 0) {
                    flag = true;
                } else {
                    const uint4 a = canon[pos], b = canon[pos - 1];
                    flag = (a.x != b.x) | (a.y != b.y) | (a.z != b.z) | (a.w != b.w);
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, flag);
            if (flag) S.starts[n + __popc(bal & ((1u << tid) - 1u))] = (unsigned short)pos;
            n += __popc(bal);
        }
        if (tid == 0) {
            S.starts[n] = (unsigned short)nev;
            S.nruns = n;
        }
    }
    __syncthreads();
}

__device__ __forceinline__ int64_t out_index(const int *__restrict__ perm, int64_t io_off, int64_t first, int64_t e)
{
    return perm ? (int64_t)perm[e] : (e - first) + io_off;
}

} // namespace

// ---- forward ------------------------------------------------------------------------------------------------
#define JP_LM_FWD_STEP(K, A2K, X0K)                                             \
    {                                                                           \
        const float u = fmaf(b2, fk, A2K);                                      \
        const float tt = __fadd_rd(u, kMagic);                                  \
        const float2 v = lds_pair<(K) * P * 8>(row + (__float_as_uint(tt) << 3)); \
        const float wt = TOF ? g1_weight(gbase, xedge, fmaf(dx, fk, X0K)) : 1.f; \
        acc = fmaf(fmaf(u, v.y, v.x), wt, acc);                                 \
    }

template <int P, int LM_MODE, bool TOF>
__global__ void __launch_bounds__(kThreads, JP_LMT_MINB_FWD)
    k_fwd_tof_lm_tile(Lors l, const int16_t *__restrict__ tofbin, int64_t first, int64_t count,
                      const int *__restrict__ perm, int64_t io_off, const float *__restrict__ img, Geom g, Tof t,
                      G1Tab gt, int rows_cap, int vec_ok, float *__restrict__ p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *C2 = reinterpret_cast<float2 *>(smem_raw);                                             // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(float2)); // [max(n0,n1)]
    const int np = max(g.n[0], g.n[1]);
    float2 *g1 = reinterpret_cast<float2 *>(rinfo + np);                                           // [gt.n]
    __shared__ TileState S;
    const int tid = threadIdx.x;
    const int64_t c0 = first + blockIdx.x * (int64_t)kTile;
    const int nev = (int)min((int64_t)kTile, first + count - c0);
    const float reach = 0.5f * t.width + t.nsig * t.sigma;

    if (TOF)
        for (int i = tid; i < gt.n; i += kThreads) g1[i] = __ldg(gt.tab + i);
    const uint32_t gbase = smem_addr(g1) - ((uint32_t)kMagicI << 3);
    const float xedge = gt.xedge;

    // ---- canonical transaxial end points of the CTA's events -> runs
    {
        uint4 canon[kPerThread];
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int pos = m * kThreads + tid;
            canon[m] = make_uint4(0xffffffffu, pos, 0, 0); // invalid slots never match
            if (pos < nev) {
                const int64_t e = c0 + pos;
                float xs = l.xs[e], ys = l.ys[e], xe = l.xe[e], ye = l.ye[e];
                const double dx = (double)xe - (double)xs, dy = (double)ye - (double)ys;
                const double dz = (double)l.ze[e] - (double)l.zs[e];
                if (is_swapped(xs, ys, xe, ye)) {
                    float tmp = xs; xs = xe; xe = tmp;
                    tmp = ys; ys = ye; ye = tmp;
                }
                canon[m] = (principal_axis(dx, dy, dz) != 2)
                               ? make_uint4(__float_as_uint(xs), __float_as_uint(ys), __float_as_uint(xe), __float_as_uint(ye))
                               : make_uint4(0xffffffffu, pos, 1, 0); // principal axis z: a run of one
            }
        }
        find_runs(S, reinterpret_cast<uint4 *>(C2), canon, nev);
    }
    const int nruns = S.nruns;
    // constant zero columns of the shared rows (after the scratch use of C2)
    {
        const int ncl = kPad - 1, ncr = P - (g.n[2] + kPad);
        for (int e = tid; e < rows_cap * (ncl + ncr); e += kThreads) {
            const int r = e / (ncl + ncr), c = e - r * (ncl + ncr);
            C2[r * P + (c < ncl ? c : g.n[2] + kPad + (c - ncl))] = make_float2(0.f, 0.f);
        }
    }
    const int n2 = g.n[2];
    const int kci = n2 >> 1; // axial shift of the (intercept, slope) rows (build_rows<P, true>)
    const uint32_t c2_base = smem_addr(C2) + (uint32_t)(kPad + kci) * 8u - ((uint32_t)kMagicI << 3);

    // tracks of all long runs at once (one thread per run) instead of one serial set-up + barrier per run
    for (int k = tid; k < nruns; k += kThreads) {
        const int ra = S.starts[k], rb = S.starts[k + 1];
        if (rb - ra < kMinRun) continue;
        const int slot = ra / kMinRun;
        const int64_t e = c0 + ra;
        float xs = l.xs[e], ys = l.ys[e], xe = l.xe[e], ye = l.ye[e];
        if (is_swapped(xs, ys, xe, ye)) {
            float tmp = xs; xs = xe; xe = tmp;
            tmp = ys; ys = ye; ye = tmp;
        }
        track_setup(g, xs, ys, xe, ye, S.trks[slot]);
        const double dxy[2] = {(double)xe - (double)xs, (double)ye - (double)ys};
        const double ratio = dxy[1 - S.trks[slot].p] * S.trks[slot].inv_dp;
        S.Rds[slot] = 1.0 + ratio * ratio;
        S.imins[slot] = 0x7fffffff;
        S.imaxs[slot] = -1;
    }
    __syncthreads();

    for (int k = 0; k < nruns; ++k) {
        const int ra = S.starts[k], rb = S.starts[k + 1];
        bool active[kPerThread]; // the run's events are dealt to the threads: event ra + m kThreads + tid
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) active[m] = ra + m * kThreads + tid < rb;
        if (rb - ra < kMinRun) { // per-LOR path (also every event whose principal axis is z: runs of one)
#pragma unroll 1
            for (int m = 0; m < kPerThread; ++m)
                if (active[m]) {
                    const int64_t e = c0 + ra + m * kThreads + tid;
                    const float c = TOF ? (float)tofbin[e] * t.width : 0.f;
                    float out = generic_fwd_lm<TOF>(l, e, c, reach, g, t, img, gbase, gt);
                    if (LM_MODE == 1) out = (out > 1e-9f) ? 1.f / out : 0.f;
                    p[out_index(perm, io_off, first, e)] = out;
                }
            continue;
        }
        // ---- the run's track (set up before the loop)
        const int slot = ra / kMinRun;
        const Track trk = S.trks[slot];
        LmRay zr[kPerThread];
        float acc_[kPerThread];
        if (trk.I1 >= trk.I0) {
            const double Rd = S.Rds[slot];
            int lo = 0x7fffffff, hi = -1;
#pragma unroll
            for (int m = 0; m < kPerThread; ++m) {
                acc_[m] = 0.f;
                zr[m].i0 = 0;
                zr[m].i1 = -1;
                if (active[m]) {
                    const int64_t e = c0 + ra + m * kThreads + tid;
                    float zs = l.zs[e], ze = l.ze[e];
                    float centre = TOF ? fmaf((float)tofbin[e], t.width, t.coff) : 0.f; // bin centre on the canonical tau axis
                    if (is_swapped(l.xs[e], l.ys[e], l.xe[e], l.ye[e])) {   // (e, s): walk it as (s, e), mirrored
                        const float tmp = zs; zs = ze; ze = tmp;
                        centre = -centre;
                    }
                    zr[m] = lm_setup<TOF>(g, trk, Rd, zs, ze, centre, reach, gt.scale, (double)kci);
                    if (zr[m].i1 >= zr[m].i0) {
                        lo = min(lo, zr[m].i0);
                        hi = max(hi, zr[m].i1);
                    }
                }
            }
            if (hi >= lo) {
                atomicMin(&S.imins[slot], lo);
                atomicMax(&S.imaxs[slot], hi);
            }
            for (int r = tid; r <= trk.I1 - trk.I0; r += kThreads) rinfo[r] = row_info(g, trk, trk.I0 + r);
        }
        __syncthreads();
        if (trk.I1 >= trk.I0) {
            const int I0 = S.imins[slot], I1 = S.imaxs[slot];
            for (int cc = I0; cc <= I1; cc += rows_cap) {
                const int rows = min(rows_cap, I1 - cc + 1);
                build_rows<P, true>(C2, rinfo, img, trk, cc, rows, n2, vec_ok, (float)kci);
                __syncthreads();
#pragma unroll
                for (int m = 0; m < kPerThread; ++m) {
                    const int ib = max(zr[m].i0, cc), ie = min(zr[m].i1, cc + rows - 1);
                    if (ib > ie) continue;
                    const int nst = ie - ib + 1;
                    const float b2 = zr[m].b2, a2_0 = zr[m].a2, dx = zr[m].dx, x0_0 = zr[m].x0;
                    const float a2_1 = fmaf(b2, 1.f, a2_0), x0_1 = fmaf(dx, 1.f, x0_0);
                    float fk = (float)(ib - zr[m].i0);
                    uint32_t row = c2_base + (uint32_t)((ib - cc) * P) * 8u;
                    float acc = acc_[m];
#pragma unroll 1
                    for (int it = nst >> 1; it > 0; --it) {
                        JP_LM_FWD_STEP(0, a2_0, x0_0)
                        JP_LM_FWD_STEP(1, a2_1, x0_1)
                        fk += 2.f;
                        row += 2u * P * 8u;
                    }
                    if (nst & 1) JP_LM_FWD_STEP(0, a2_0, x0_0)
                    acc_[m] = acc;
                }
                __syncthreads();
            }
        }
#pragma unroll
        for (int m = 0; m < kPerThread; ++m)
            if (active[m]) {
                float out = (trk.I1 >= trk.I0) ? zr[m].cf * acc_[m] : 0.f;
                if (LM_MODE == 1) out = (out > 1e-9f) ? 1.f / out : 0.f;
                p[out_index(perm, io_off, first, c0 + ra + m * kThreads + tid)] = out;
            }
    }
}
#undef JP_LM_FWD_STEP

// ---- back ------------------------------------------------------------------------------------------------------
// Fixed-point staging as in jp_tile.cu (native int32 shared atomics; scale from max |cf y| over the run: the TOF
// weight is <= 1, a bin receives at most two contributions per event and plane, a run has at most kTile events).
template <int OFF>
__device__ __forceinline__ void reds_add_lm(uint32_t addr, int q)
{
    asm volatile("red.shared.add.s32 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "r"(q) : "memory");
}

#define JP_LM_BACK_STEP(K, A2K, X0K)                                            \
    {                                                                           \
        const float u = fmaf(b2, fk, A2K);                                      \
        const float tt = __fadd_rd(u, kMagic);                                  \
        const float w = u - (tt - kMagic);                                      \
        const uint32_t a = row + (__float_as_uint(tt) << 2);                    \
        const float xw = TOF ? xm * g1_weight(gbase, xedge, fmaf(dx, fk, X0K)) : xm; \
        const int qxw = __float_as_int(xw + kMagic);                            \
        const int bits = __float_as_int(fmaf(xw, w, kMagic));                   \
        reds_add_lm<(K) * P * 4>(a, qxw - bits);                                \
        reds_add_lm<(K) * P * 4 + 4>(a, bits - kMagicI);                        \
    }

template <int P, bool TOF>
__global__ void __launch_bounds__(kThreads, JP_LMT_MINB_BACK)
    k_back_tof_lm_tile(Lors l, const int16_t *__restrict__ tofbin, int64_t first, int64_t count,
                       const int *__restrict__ perm, int64_t io_off, const float *__restrict__ y, Geom g, Tof t,
                       G1Tab gt, int rows_cap, int vec_ok, float *__restrict__ img)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int *Ci = reinterpret_cast<int *>(smem_raw);                                                 // [rows_cap][P]
    RowInfo *rinfo = reinterpret_cast<RowInfo *>(smem_raw + (size_t)rows_cap * P * sizeof(int)); // [max(n0,n1)]
    const int np = max(g.n[0], g.n[1]);
    float2 *g1 = reinterpret_cast<float2 *>(rinfo + np);                                         // [gt.n]
    __shared__ TileState S;
    __shared__ float red[kThreads / 32];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int64_t c0 = first + blockIdx.x * (int64_t)kTile;
    const int nev = (int)min((int64_t)kTile, first + count - c0);
    const float reach = 0.5f * t.width + t.nsig * t.sigma;

    if (TOF)
        for (int i = tid; i < gt.n; i += kThreads) g1[i] = __ldg(gt.tab + i);
    const uint32_t gbase = smem_addr(g1) - ((uint32_t)kMagicI << 3);
    const float xedge = gt.xedge;
    {
        uint4 canon[kPerThread];
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) {
            const int pos = m * kThreads + tid;
            canon[m] = make_uint4(0xffffffffu, pos, 0, 0);
            if (pos < nev) {
                const int64_t e = c0 + pos;
                float xs = l.xs[e], ys = l.ys[e], xe = l.xe[e], ye = l.ye[e];
                const double dx = (double)xe - (double)xs, dy = (double)ye - (double)ys;
                const double dz = (double)l.ze[e] - (double)l.zs[e];
                if (is_swapped(xs, ys, xe, ye)) {
                    float tmp = xs; xs = xe; xe = tmp;
                    tmp = ys; ys = ye; ye = tmp;
                }
                canon[m] = (principal_axis(dx, dy, dz) != 2)
                               ? make_uint4(__float_as_uint(xs), __float_as_uint(ys), __float_as_uint(xe), __float_as_uint(ye))
                               : make_uint4(0xffffffffu, pos, 1, 0);
            }
        }
        find_runs(S, reinterpret_cast<uint4 *>(Ci), canon, nev);
    }
    const int nruns = S.nruns;
    {
        int4 *z4 = reinterpret_cast<int4 *>(Ci);
        for (int e = tid; e < rows_cap * (P / 4); e += kThreads) z4[e] = make_int4(0, 0, 0, 0);
    }
    const uint32_t ci_base = smem_addr(Ci) + kPad * 4u - ((uint32_t)kMagicI << 2);
    const int n2 = g.n[2];
    __syncthreads();

    for (int k = 0; k < nruns; ++k) {
        const int ra = S.starts[k], rb = S.starts[k + 1];
        bool active[kPerThread];
#pragma unroll
        for (int m = 0; m < kPerThread; ++m) active[m] = ra + m * kThreads + tid < rb;
        if (rb - ra < kMinRun) {
#pragma unroll 1
            for (int m = 0; m < kPerThread; ++m)
                if (active[m]) {
                    const int64_t e = c0 + ra + m * kThreads + tid;
                    const float yv = y[out_index(perm, io_off, first, e)];
                    if (yv != 0.f)
                        generic_back_lm<TOF>(l, e, TOF ? (float)tofbin[e] * t.width : 0.f, reach, yv, g, t, img, gbase, gt);
                }
            continue;
        }
        if (tid == 0) {
            const int64_t e = c0 + ra;
            float xs = l.xs[e], ys = l.ys[e], xe = l.xe[e], ye = l.ye[e];
            if (is_swapped(xs, ys, xe, ye)) {
                float tmp = xs; xs = xe; xe = tmp;
                tmp = ys; ys = ye; ye = tmp;
            }
            track_setup(g, xs, ys, xe, ye, S.trk);
            const double dxy[2] = {(double)xe - (double)xs, (double)ye - (double)ys};
            const double ratio = dxy[1 - S.trk.p] * S.trk.inv_dp;
            S.ex.Rd = 1.0 + ratio * ratio;
            S.imin = 0x7fffffff;
            S.imax = -1;
            S.bad = 0;
        }
        __syncthreads();
        const Track trk = S.trk;
        if (trk.I1 < trk.I0) {
            __syncthreads();
            continue;
        }
        LmRay zr[kPerThread];
        float x[kPerThread];
        float xm_ = 0.f;
        bool bad = false;
        {
            const double Rd = S.ex.Rd;
            int lo = 0x7fffffff, hi = -1;
#pragma unroll
            for (int m = 0; m < kPerThread; ++m) {
                x[m] = 0.f;
                zr[m].i0 = 0;
                zr[m].i1 = -1;
                if (active[m]) {
                    const int64_t e = c0 + ra + m * kThreads + tid;
                    float zs = l.zs[e], ze = l.ze[e];
                    float centre = TOF ? fmaf((float)tofbin[e], t.width, t.coff) : 0.f;
                    if (is_swapped(l.xs[e], l.ys[e], l.xe[e], l.ye[e])) {
                        const float tmp = zs; zs = ze; ze = tmp;
                        centre = -centre;
                    }
                    zr[m] = lm_setup<TOF>(g, trk, Rd, zs, ze, centre, reach, gt.scale);
                    x[m] = zr[m].cf * y[out_index(perm, io_off, first, e)];
                    if (zr[m].i1 >= zr[m].i0 && x[m] != 0.f) {
                        lo = min(lo, zr[m].i0);
                        hi = max(hi, zr[m].i1);
                        bad = bad || !(fabsf(x[m]) < 3.0e38f); // Inf or NaN (fmaxf would drop a NaN)
                        xm_ = fmaxf(xm_, fabsf(x[m]));
                    } else {
                        zr[m].i1 = zr[m].i0 - 1;
                    }
                }
            }
            if (hi >= lo) {
                atomicMin(&S.imin, lo);
                atomicMax(&S.imax, hi);
            }
            if (bad) atomicExch(&S.bad, 1);
        }
        for (int o = 16; o > 0; o >>= 1) xm_ = fmaxf(xm_, __shfl_xor_sync(0xffffffffu, xm_, o));
        if (lane == 0) red[warp] = xm_;
        for (int r = tid; r <= trk.I1 - trk.I0; r += kThreads) rinfo[r] = row_info(g, trk, trk.I0 + r);
        __syncthreads();
        xm_ = red[0];
#pragma unroll
        for (int w = 1; w < kThreads / 32; ++w) xm_ = fmaxf(xm_, red[w]);
        const int I0 = S.imin, I1 = S.imax;
        if (S.bad) { // a non-finite value cannot be staged in fixed point: the run takes the per-LOR float path, so that
                     // Inf / NaN propagate exactly as they do for events outside a line tile
#pragma unroll 1
            for (int m = 0; m < kPerThread; ++m)
                if (active[m]) {
                    const int64_t e = c0 + ra + m * kThreads + tid;
                    const float yv = y[out_index(perm, io_off, first, e)];
                    if (yv != 0.f)
                        generic_back_lm<TOF>(l, e, TOF ? (float)tofbin[e] * t.width : 0.f, reach, yv, g, t, img, gbase, gt);
                }
        } else if (xm_ > 0.f && I1 >= I0) {
            const float lim = fminf(4194302.f, 2147483648.f / (float)(2 * kTile) - 1.f);
            const float Sc = lim / xm_, invS = xm_ / lim;
            for (int cc = I0; cc <= I1; cc += rows_cap) {
                const int rows = min(rows_cap, I1 - cc + 1);
#pragma unroll
                for (int m = 0; m < kPerThread; ++m) {
                    const int ib = max(zr[m].i0, cc), ie = min(zr[m].i1, cc + rows - 1);
                    if (ib > ie) continue;
                    const int nst = ie - ib + 1;
                    const float b2 = zr[m].b2, a2_0 = zr[m].a2, dx = zr[m].dx, x0_0 = zr[m].x0, xm = x[m] * Sc;
                    const float a2_1 = fmaf(b2, 1.f, a2_0), x0_1 = fmaf(dx, 1.f, x0_0);
                    float fk = (float)(ib - zr[m].i0);
                    uint32_t row = ci_base + (uint32_t)((ib - cc) * P) * 4u;
                    int left = nst;
#if JP_LMT_BACK_UNROLL == 4
                    const float a2_2 = fmaf(b2, 2.f, a2_0), x0_2 = fmaf(dx, 2.f, x0_0);
                    const float a2_3 = fmaf(b2, 3.f, a2_0), x0_3 = fmaf(dx, 3.f, x0_0);
#pragma unroll 1
                    for (; left >= 4; left -= 4) {
                        JP_LM_BACK_STEP(0, a2_0, x0_0)
                        JP_LM_BACK_STEP(1, a2_1, x0_1)
                        JP_LM_BACK_STEP(2, a2_2, x0_2)
                        JP_LM_BACK_STEP(3, a2_3, x0_3)
                        fk += 4.f;
                        row += 4u * P * 4u;
                    }
                    if (left >= 2) {
#else
#pragma unroll 1
                    for (; left >= 2; left -= 2) {
#endif
                        JP_LM_BACK_STEP(0, a2_0, x0_0)
                        JP_LM_BACK_STEP(1, a2_1, x0_1)
                        fk += 2.f;
                        row += 2u * P * 4u;
                    }
                    if (left & 1) JP_LM_BACK_STEP(0, a2_0, x0_0)
                }
                __syncthreads();
                // ---- flush: spread every row over its two q1 neighbours with REDs, and clear it
                if (vec_ok) {
                    const int G = n2 >> 2;
                    for (int r = warp; r < rows; r += kThreads / 32) {
                        const RowInfo ri = rinfo[cc - trk.I0 + r];
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
                        const RowInfo ri = rinfo[cc - trk.I0 + r];
                        const float v = (float)q * invS;
                        if (ri.base_a >= 0) atomicAdd(img + ri.base_a + z, ri.wa * v);
                        if (ri.base_b >= 0) atomicAdd(img + ri.base_b + z, ri.wb * v);
                    }
                }
                __syncthreads();
            }
        }
        __syncthreads(); // S.trk / red are rewritten by the next run
    }
}
#undef JP_LM_BACK_STEP

// ---- launchers ----------------------------------------------------------------------------------------------
namespace {

#ifndef JP_LMT_SMEM_KB_FWD
#define JP_LMT_SMEM_KB_FWD 52
#endif
#ifndef JP_LMT_SMEM_KB_BACK
#define JP_LMT_SMEM_KB_BACK 28
#endif
constexpr size_t kSmemMax = 64 * 1024;

struct LmTileCfg {
    int P, rows_cap, vec_ok, g1n;
    size_t smem;
};

// elem: bytes per row element (8: forward pairs, 4: back fixed point)
LmTileCfg lm_tile_cfg(const Geom &g, const Tof &t, const void *img, size_t elem, size_t kSmemBudget)
{
    LmTileCfg c{};
    const int need = g.n[2] + kPad + kPadR;
    const int pitches[] = {40, 72, 104, 136, 200, 264};
    for (int P : pitches)
        if (need <= P) { c.P = P; break; }
    if (!c.P) return c;
    c.g1n = g1tab_entries(t);
    const int np = g.n[0] > g.n[1] ? g.n[0] : g.n[1];
    const size_t fixed = (size_t)np * sizeof(RowInfo) + (size_t)c.g1n * sizeof(float2);
    const size_t row = (size_t)c.P * elem;
    if (kSmemBudget > kSmemMax) kSmemBudget = kSmemMax;
    size_t rows = fixed + row <= kSmemBudget ? (kSmemBudget - fixed) / row : 0;
    if (rows * row < (size_t)kTile * sizeof(uint4) || rows < 8) { c.P = 0; return c; } // also the run-detection scratch
    if (rows > (size_t)np) rows = (size_t)np;
    if (rows * row < (size_t)kTile * sizeof(uint4)) rows = ((size_t)kTile * sizeof(uint4) + row - 1) / row;
    c.rows_cap = (int)rows;
    c.smem = rows * row + fixed;
    c.vec_ok = (g.n[2] % 4 == 0) && ((uintptr_t)img % 16 == 0);
    return c;
}

} // namespace

// can the line-tile kernels take this image / TOF kernel at all?  (the planned calls use the quad or per-LOR path if not)
bool lm_tile_supported(const Geom &g, const Tof &t_in, bool tof)
{
    const Tof t = tof ? t_in : Tof{1.f, 1.f, 1.f, 1, 0.f};
    return lm_tile_cfg(g, t, nullptr, sizeof(float2), JP_LMT_SMEM_KB_FWD * 1024).P != 0 &&
           lm_tile_cfg(g, t, nullptr, sizeof(int), JP_LMT_SMEM_KB_BACK * 1024).P != 0;
}

cudaError_t g1tab_create(const Tof &t, int n, cudaStream_t st, G1Tab *out)
{
    float2 *tab = nullptr;
    cudaError_t e = cudaMallocAsync((void **)&tab, sizeof(float2) * n, st);
    if (e != cudaSuccess) return e;
    const double m = (double)t.nsig * (double)t.sigma;
    k_tof_g1tab<<<(n + 255) / 256, 256, 0, st>>>(tab, n, (double)t.width, m, 1.0 / ((double)t.sigma * 1.4142135623730951));
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        cudaFreeAsync(tab, st);
        return e;
    }
    out->tab = tab;
    out->n = n;
    out->scale = (float)((double)kG1K / (double)t.width);
    out->xedge = (float)(((double)t.nsig * (double)t.sigma / (double)t.width + 0.5) * kG1K);
    return cudaSuccess;
}

#define JP_LM_DISPATCH_P(CFG, ...)                           \
    switch ((CFG).P) {                                       \
    case 40: { constexpr int P = 40; __VA_ARGS__; } break;   \
    case 72: { constexpr int P = 72; __VA_ARGS__; } break;   \
    case 104: { constexpr int P = 104; __VA_ARGS__; } break; \
    case 136: { constexpr int P = 136; __VA_ARGS__; } break; \
    case 200: { constexpr int P = 200; __VA_ARGS__; } break; \
    case 264: { constexpr int P = 264; __VA_ARGS__; } break; \
    default: return cudaErrorNotSupported;                   \
    }

// events [first, first + count) of the sorted list l / tofbin; outputs p[perm[e]] (perm != null) or
// p[io_off + e - first].  cudaErrorNotSupported: image too wide for the tiled kernel.
// tofbin == nullptr: NON-TOF listmode (every plane of the LOR, weight 1; t is ignored)
cudaError_t launch_fwd_tof_lm_tile(const Lors &l, const int16_t *tofbin, int64_t first, int64_t count, const int *perm,
                                   int64_t io_off, const float *img, const Geom &g, const Tof &t_in, float *p, int lm_mode,
                                   cudaStream_t st)
{
    if (count == 0) return cudaSuccess;
    const bool tof = tofbin != nullptr;
    const Tof t = tof ? t_in : Tof{1.f, 1.f, 1.f, 1, 0.f};
    const LmTileCfg c = lm_tile_cfg(g, t, img, sizeof(float2), JP_LMT_SMEM_KB_FWD * 1024);
    if (!c.P) return cudaErrorNotSupported;
    G1Tab gt{};
    cudaError_t e = tof ? g1tab_create(t, c.g1n, st, &gt) : cudaSuccess;
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((count + kTile - 1) / kTile);
#define JP_LM_LAUNCH_FWD(MODE, TOFF)                                                                                   \
    {                                                                                                                  \
        e = cudaFuncSetAttribute(k_fwd_tof_lm_tile<P, MODE, TOFF>, cudaFuncAttributeMaxDynamicSharedMemorySize,        \
                                 (int)kSmemMax);                                                                    \
        if (e == cudaSuccess)                                                                                          \
            k_fwd_tof_lm_tile<P, MODE, TOFF><<<grid, kThreads, c.smem, st>>>(l, tofbin, first, count, perm, io_off, img, \
                                                                             g, t, gt, c.rows_cap, c.vec_ok, p);       \
    }
    JP_LM_DISPATCH_P(c, {
        if (!tof) JP_LM_LAUNCH_FWD(0, false)
        else if (lm_mode == 1) JP_LM_LAUNCH_FWD(1, true)
        else JP_LM_LAUNCH_FWD(0, true)
    })
#undef JP_LM_LAUNCH_FWD
    if (e == cudaSuccess) e = cudaGetLastError();
    if (gt.tab) cudaFreeAsync((void *)gt.tab, st);
    return e;
}

cudaError_t launch_back_tof_lm_tile(const Lors &l, const int16_t *tofbin, int64_t first, int64_t count, const int *perm,
                                    int64_t io_off, const float *y, const Geom &g, const Tof &t_in, float *img,
                                    cudaStream_t st)
{
    if (count == 0) return cudaSuccess;
    const bool tof = tofbin != nullptr;
    const Tof t = tof ? t_in : Tof{1.f, 1.f, 1.f, 1, 0.f};
    const LmTileCfg c = lm_tile_cfg(g, t, img, sizeof(int), JP_LMT_SMEM_KB_BACK * 1024);
    if (!c.P) return cudaErrorNotSupported;
    G1Tab gt{};
    cudaError_t e = tof ? g1tab_create(t, c.g1n, st, &gt) : cudaSuccess;
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((count + kTile - 1) / kTile);
#define JP_LM_LAUNCH_BACK(TOFF)                                                                                         \
    {                                                                                                                   \
        e = cudaFuncSetAttribute(k_back_tof_lm_tile<P, TOFF>, cudaFuncAttributeMaxDynamicSharedMemorySize,              \
                                 (int)kSmemMax);                                                                     \
        if (e == cudaSuccess)                                                                                           \
            k_back_tof_lm_tile<P, TOFF><<<grid, kThreads, c.smem, st>>>(l, tofbin, first, count, perm, io_off, y, g, t, \
                                                                        gt, c.rows_cap, c.vec_ok, img);                 \
    }
    JP_LM_DISPATCH_P(c, {
        if (tof) JP_LM_LAUNCH_BACK(true)
        else JP_LM_LAUNCH_BACK(false)
    })
#undef JP_LM_LAUNCH_BACK
    if (e == cudaSuccess) e = cudaGetLastError();
    if (gt.tab) cudaFreeAsync((void *)gt.tab, st);
    return e;
}

} // namespace jp
