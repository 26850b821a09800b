// jp_tof_sino.cu -- TOF sinogram forward / back projection with a sliding register window of TOF bins:
// the kernels behind jp_fwd_tof_sino / jp_back_tof_sino.
//
// in sinogram mode every plane step contributes to ALL TOF bins along the ray; PAPER.md:35,
// :78: the weight of a bin is the Gaussian integrated over the bin (difference of two error functions),
// truncated at n_sigmas.  In bin coordinates s = tau / W + (n_tofbins - 1) / 2 (bin k centred at s = k) the
// weight of bin k is G(k - s),
//
//     G(x) = 1/2 [E((x + 1/2) W) - E((x - 1/2) W)],   E(y) = erf(clamp(y, -m, m) / (sigma sqrt2)),
//
// with support |x| < R = m / W + 1/2: at most ceil(2R) consecutive bins starting at base = ceil(s - R).
// Two facts shape the kernels:
//   * with phi = base - (s - R) in [0, 1), the arguments of ALL bins of the window are n + phi - R: one row
//     of a table T[phi][n] = G(n + phi - R) (512 rows, (value, slope) pairs, built in float64) gives every
//     weight of the step with NBW/2 128-bit shared-memory loads and NBW FMAs -- instead of one edge-function
//     look-up per bin edge;
//   * s is monotone along the ray (the planes are walked in the direction of increasing tau), so base never
//     decreases: the NBW bins of the window are accumulated in REGISTERS and a bin is written (forward) /
//     its y value read (back) exactly once, when the window slides past it.
// Persistent CTAs (one table copy per CTA) loop over blocks of 256 consecutive LORs; the block's
// [256][n_tofbins] tile is staged through shared memory so that global reads / writes are coalesced, and
// blocks whose LORs all miss the image skip the walk (forward: zero fill; back: y is not even read).
// Images are the zero-padded copies of jp_pad.cu (PRay).
#include "jp_tof_win.cuh"

namespace jp {

using namespace tofwin;

namespace {

constexpr int kSBlock = 256;
constexpr int kSLd = kSBlock + 1;
#ifndef JP_SINO_IO
#define JP_SINO_IO 4 // tile elements per thread in flight
#endif
#ifndef JP_SINO_MINB
#define JP_SINO_MINB 4
#endif

// the walk of one LOR; FWD: a[] accumulates value x weight per window bin, flushed into acc (shared, [bin][kSLd]);
// BACK: yv[] holds the y values of the window bins (from ysm), the step's sum is scattered with atomic adds
// S2ONE: the q2 axis is the contiguous image axis (principal axis x or y), neighbours along q2 are 4 bytes apart
template <int NBW, bool BACK, bool S2ONE>
__device__ __forceinline__ void walk(const PRay &q, const GTab &gt, uint32_t tab_addr, float *__restrict__ stage,
                                     int nbins, const float *__restrict__ pimg_r, float *__restrict__ pimg_w)
{
    const int tid = threadIdx.x;
    const float ds = q.dtau * gt.inv_w;
    const float sR0 = fmaf(q.tau0, gt.inv_w, gt.cbR);
    // walk in the direction of increasing s
    float fk = 0.f, dfk = 1.f;
    int po = q.off, dpo = q.sp;
    if (ds < 0.f) {
        fk = (float)(q.nk - 1);
        dfk = -1.f;
        po = q.off + (q.nk - 1) * q.sp;
        dpo = -q.sp;
    }
    float sR = fmaf(ds, fk, sR0);
    float basef = __fadd_ru(sR, kMagic) - kMagic; // ceil(s - R)
    int base = (int)basef;
    float a[NBW];
#pragma unroll
    for (int n = 0; n < NBW; ++n) {
        if (BACK)
            a[n] = ((unsigned)(base + n) < (unsigned)nbins) ? stage[(base + n) * kSLd + tid] : 0.f;
        else
            a[n] = 0.f;
    }
    const int s2 = S2ONE ? 1 : q.s2;
    PCell cl = pray_cell(q, fk, po);
    for (int it = 0; it < q.nk; ++it) {
        sR = fmaf(ds, fk, sR0);
        const float cur = __fadd_ru(sR, kMagic) - kMagic;
#pragma unroll 1
        while (cur > basef) { // slide the window by one bin (false for NaN)
            if (BACK) {
#pragma unroll
                for (int n = 0; n + 1 < NBW; ++n) a[n] = a[n + 1];
                a[NBW - 1] = ((unsigned)(base + NBW) < (unsigned)nbins) ? stage[(base + NBW) * kSLd + tid] : 0.f;
            } else {
                if ((unsigned)base < (unsigned)nbins) stage[base * kSLd + tid] = q.cf * a[0];
#pragma unroll
                for (int n = 0; n + 1 < NBW; ++n) a[n] = a[n + 1];
                a[NBW - 1] = 0.f;
            }
            basef += 1.f;
            ++base;
        }
        const float tk = (cur - sR) * (float)kGK;
        const float tt = __fadd_rd(tk, kMagic);
        const float f = tk - (tt - kMagic);
        const uint32_t row = tab_addr + __float_as_uint(tt) * (uint32_t)(NBW * 8);
        float w[NBW];
        load_weights<NBW, 0>(row, f, w);
        fk += dfk;
        po += dpo;
        if (BACK) {
            float s = 0.f;
#pragma unroll
            for (int n = 0; n < NBW; ++n) s = fmaf(a[n], w[n], s);
            if (s != 0.f) {
                const float x = q.cf * s;
                float *p0 = pimg_w + cl.off, *p1 = p0 + q.s1;
                const float xa = x * (1.f - cl.w1), xb = x * cl.w1, m2 = 1.f - cl.w2;
                atomicAdd(p0, xa * m2);
                atomicAdd(p0 + s2, xa * cl.w2);
                atomicAdd(p1, xb * m2);
                atomicAdd(p1 + s2, xb * cl.w2);
            }
            cl = pray_cell(q, fk, po);
        } else {
            const float *p0 = pimg_r + cl.off, *p1 = p0 + q.s1;
            const float v00 = __ldg(p0), v01 = __ldg(p0 + s2), v10 = __ldg(p1), v11 = __ldg(p1 + s2);
            const float lo = fmaf(cl.w2, v01 - v00, v00), hi = fmaf(cl.w2, v11 - v10, v10);
            const float val = fmaf(cl.w1, hi - lo, lo);
#pragma unroll
            for (int n = 0; n < NBW; ++n) a[n] = fmaf(val, w[n], a[n]);
            cl = pray_cell(q, fk, po);
        }
    }
    if (!BACK) {
#pragma unroll
        for (int n = 0; n < NBW; ++n)
            if ((unsigned)(base + n) < (unsigned)nbins) stage[(base + n) * kSLd + tid] = q.cf * a[n];
    }
}

// The block's [nvalid][nbins] tile in global memory is contiguous: thread t visits elements t, t + 256, ... (fully
// coalesced), four at a time so that four independent loads are in flight; (lor, bin) of an element advance by
// (256 / nbins, 256 % nbins) from one visit to the next, no division in the loop.
struct TileIdx {
    int x, lor, kb;
};
__device__ __forceinline__ TileIdx tile_first(int tid, int nbins)
{
    TileIdx i;
    i.x = tid;
    i.lor = tid / nbins;
    i.kb = tid - i.lor * nbins;
    return i;
}
__device__ __forceinline__ void tile_next(TileIdx &i, int dq, int dr, int nbins)
{
    i.x += kSBlock;
    i.lor += dq;
    i.kb += dr;
    if (i.kb >= nbins) {
        i.kb -= nbins;
        ++i.lor;
    }
}

template <int NBW, bool BACK>
__global__ void __launch_bounds__(kSBlock, JP_SINO_MINB)
    k_tof_sino_win(Lors l, int64_t n, int64_t nblocks, const float *__restrict__ pimg_r, float *__restrict__ pimg_w,
                   Geom g, Tof t, GTab gt, float *__restrict__ p, const float *__restrict__ y, SinoEpi epi)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);                                       // [(kGK + 2)][NBW]
    float *stage = reinterpret_cast<float *>(smem_raw + (size_t)(kGK + 2) * NBW * sizeof(float2)); // [nbins][kSLd]
    const int tid = threadIdx.x;
    const int nbins = t.nbins;
    const int dq = kSBlock / nbins, dr = kSBlock % nbins; // (lor, bin) step of the flattened tile walk
    for (int i = tid; i < (kGK + 2) * NBW; i += kSBlock) tab[i] = __ldg(gt.tab + i);
    if (!BACK)
        for (int i = tid; i < nbins * kSLd; i += kSBlock) stage[i] = 0.f;
    const uint32_t tab_addr = smem_addr(tab) - (uint32_t)kMagicI * (uint32_t)(NBW * 8);
    const float lim = t.nsig * t.sigma;
    const float reach = 0.5f * (float)(nbins - 1) * t.width + 0.5f * t.width + lim;
    __syncthreads();

    for (int64_t blk = blockIdx.x; blk < nblocks; blk += gridDim.x) {
        const int64_t j0 = blk * kSBlock, j = j0 + tid;
        const int nvalid = (int)min((int64_t)kSBlock, n - j0);
        PRay q;
        q.nk = 0;
        if (j < n) {
            Ray r;
            ray_setup<true>(l, j, g, t.coff, -reach, reach, r);
            q = pray_from(r, g);
        }
        const bool any = __syncthreads_or(q.nk > 0) != 0;
        // pull into L2 what the block will read at its end (forward: the emission / contamination tile of the OSEM
        // ratio) or what the next block of this CTA reads at its start (back: its y tile), one 128-byte line per thread
        if (!BACK && any && epi.y_em) {
            const int64_t o = j0 * nbins + (int64_t)tid * 32;
            if (o < (j0 + nvalid) * nbins) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(epi.y_em + o));
                if (epi.contam) asm volatile("prefetch.global.L2 [%0];" ::"l"(epi.contam + o));
            }
        }
        if (BACK && y && blk + gridDim.x < nblocks) {
            const int64_t jn = (blk + gridDim.x) * kSBlock;
            const int64_t o = jn * nbins + (int64_t)tid * 32;
            if (o < min(n, jn + kSBlock) * nbins) asm volatile("prefetch.global.L2 [%0];" ::"l"(y + o));
        }
        if (!any) {
            if (!BACK) { // the whole block misses the image: zeros
                float *out = p + j0 * nbins;
                const int tot = nvalid * nbins;
                if (nvalid == kSBlock && (((uintptr_t)out) & 15) == 0) {
                    float4 *o4 = reinterpret_cast<float4 *>(out);
                    for (int x = tid; x < tot / 4; x += kSBlock) o4[x] = make_float4(0.f, 0.f, 0.f, 0.f);
                    for (int x = (tot & ~3) + tid; x < tot; x += kSBlock) out[x] = 0.f;
                } else {
                    for (int x = tid; x < tot; x += kSBlock) out[x] = 0.f;
                }
            }
            continue;
        }
        if (BACK) { // stage y[j0 .. j0 + nvalid)[nbins]: one warp per LOR, lanes along the bins
            if (epi.mult_bcast || epi.ones_bcast) {
                const float v = (tid < nvalid) ? (epi.mult_bcast ? epi.mult_bcast[j0 + tid] : 1.f) : 0.f;
                for (int kb = 0; kb < nbins; ++kb) stage[kb * kSLd + tid] = v;
            } else {
                const float *in = y + j0 * nbins;
                const int tot = nvalid * nbins;
                TileIdx it = tile_first(tid, nbins);
                while (it.x < tot) {
                    TileIdx e[JP_SINO_IO];
                    float v[JP_SINO_IO];
#pragma unroll
                    for (int u = 0; u < JP_SINO_IO; ++u) {
                        e[u] = it;
                        v[u] = (it.x < tot) ? in[it.x] : 0.f;
                        tile_next(it, dq, dr, nbins);
                    }
#pragma unroll
                    for (int u = 0; u < JP_SINO_IO; ++u)
                        if (e[u].x < tot) stage[e[u].kb * kSLd + e[u].lor] = v[u];
                }
            }
            __syncthreads();
        }
        if (q.nk > 0) {
            if (q.s2 == 1)
                walk<NBW, BACK, true>(q, gt, tab_addr, stage, nbins, pimg_r, pimg_w);
            else
                walk<NBW, BACK, false>(q, gt, tab_addr, stage, nbins, pimg_r, pimg_w);
        }
        __syncthreads();
        if (!BACK) { // write the tile (and clear it for the next block)
            float *out = p + j0 * nbins;
            const int tot = nvalid * nbins;
            TileIdx it = tile_first(tid, nbins);
            if (epi.y_em) { // OSEM ratio instead of the projection (reading S2)
                const float *ye = epi.y_em + j0 * nbins;
                const float *ct = epi.contam ? epi.contam + j0 * nbins : nullptr;
                while (it.x < tot) {
                    TileIdx e[JP_SINO_IO];
                    float yv[JP_SINO_IO], cv[JP_SINO_IO], mv[JP_SINO_IO];
#pragma unroll
                    for (int u = 0; u < JP_SINO_IO; ++u) {
                        e[u] = it;
                        const bool ok = it.x < tot;
                        yv[u] = ok ? ye[it.x] : 0.f;
                        cv[u] = (ok && ct) ? ct[it.x] : 0.f;
                        mv[u] = (ok && epi.mult) ? epi.mult[j0 + it.lor] : 1.f;
                        tile_next(it, dq, dr, nbins);
                    }
#pragma unroll
                    for (int u = 0; u < JP_SINO_IO; ++u)
                        if (e[u].x < tot) {
                            const int sidx = e[u].kb * kSLd + e[u].lor;
                            const float yb = fmaf(mv[u], stage[sidx], cv[u]);
                            out[e[u].x] = (yb > 1e-9f) ? mv[u] * yv[u] / yb : 0.f;
                            stage[sidx] = 0.f;
                        }
                }
            } else {
                while (it.x < tot) {
                    const int sidx = it.kb * kSLd + it.lor;
                    out[it.x] = stage[sidx];
                    stage[sidx] = 0.f;
                    tile_next(it, dq, dr, nbins);
                }
            }
            __syncthreads();
        }
    }
}

// ---- one OSEM subset update per LOR in ONE pass (readings S1-S3): forward walk into the shared tile, ratio in place
// (mult y / (mult p + contam), emission and contamination tiles read as flat coalesced ranges), back walk out of the
// same tile.  The ratio sinogram never goes through global memory and the float64 ray set-up is done once.
template <int NBW>
__global__ void __launch_bounds__(kSBlock, JP_SINO_MINB)
    k_tof_sino_osem(Lors l, int64_t n, int64_t nblocks, const float *__restrict__ pimg_r, float *__restrict__ pimg_w,
                    Geom g, Tof t, GTab gt, SinoEpi epi)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tab = reinterpret_cast<float2 *>(smem_raw);                                       // [(kGK + 2)][NBW]
    float *stage = reinterpret_cast<float *>(smem_raw + (size_t)(kGK + 2) * NBW * sizeof(float2)); // [nbins][kSLd]
    const int tid = threadIdx.x;
    const int nbins = t.nbins;
    const int dq = kSBlock / nbins, dr = kSBlock % nbins;
    for (int i = tid; i < (kGK + 2) * NBW; i += kSBlock) tab[i] = __ldg(gt.tab + i);
    for (int i = tid; i < nbins * kSLd; i += kSBlock) stage[i] = 0.f;
    const uint32_t tab_addr = smem_addr(tab) - (uint32_t)kMagicI * (uint32_t)(NBW * 8);
    const float lim = t.nsig * t.sigma;
    const float reach = 0.5f * (float)(nbins - 1) * t.width + 0.5f * t.width + lim;
    __syncthreads();

    for (int64_t blk = blockIdx.x; blk < nblocks; blk += gridDim.x) {
        const int64_t j0 = blk * kSBlock, j = j0 + tid;
        const int nvalid = (int)min((int64_t)kSBlock, n - j0);
        PRay q;
        q.nk = 0;
        if (j < n) {
            Ray r;
            ray_setup<true>(l, j, g, t.coff, -reach, reach, r);
            q = pray_from(r, g);
        }
        const bool any = __syncthreads_or(q.nk > 0) != 0;
        if (!any) continue; // no LOR of the block meets the image: nothing to add
        const int tot = nvalid * nbins;
        { // the tiles the ratio stage will read, one 128-byte line per thread
            const int64_t o = j0 * nbins + (int64_t)tid * 32;
            if (o < (j0 + nvalid) * nbins) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(epi.y_em + o));
                if (epi.contam) asm volatile("prefetch.global.L2 [%0];" ::"l"(epi.contam + o));
            }
        }
        if (q.nk > 0) {
            if (q.s2 == 1)
                walk<NBW, false, true>(q, gt, tab_addr, stage, nbins, pimg_r, nullptr);
            else
                walk<NBW, false, false>(q, gt, tab_addr, stage, nbins, pimg_r, nullptr);
        }
        __syncthreads();
        { // ratio in place (LORs that miss the image keep p = 0: their ratio is never walked)
            const float *ye = epi.y_em + j0 * nbins;
            const float *ct = epi.contam ? epi.contam + j0 * nbins : nullptr;
            TileIdx it = tile_first(tid, nbins);
            while (it.x < tot) {
                TileIdx e[JP_SINO_IO];
                float yv[JP_SINO_IO], cv[JP_SINO_IO], mv[JP_SINO_IO];
#pragma unroll
                for (int u = 0; u < JP_SINO_IO; ++u) {
                    e[u] = it;
                    const bool ok = it.x < tot;
                    yv[u] = ok ? ye[it.x] : 0.f;
                    cv[u] = (ok && ct) ? ct[it.x] : 0.f;
                    mv[u] = (ok && epi.mult) ? epi.mult[j0 + it.lor] : 1.f;
                    tile_next(it, dq, dr, nbins);
                }
#pragma unroll
                for (int u = 0; u < JP_SINO_IO; ++u)
                    if (e[u].x < tot) {
                        const int sidx = e[u].kb * kSLd + e[u].lor;
                        const float yb = fmaf(mv[u], stage[sidx], cv[u]);
                        stage[sidx] = (yb > 1e-9f) ? mv[u] * yv[u] / yb : 0.f;
                    }
            }
        }
        __syncthreads();
        if (q.nk > 0) {
            if (q.s2 == 1)
                walk<NBW, true, true>(q, gt, tab_addr, stage, nbins, nullptr, pimg_w);
            else
                walk<NBW, true, false>(q, gt, tab_addr, stage, nbins, nullptr, pimg_w);
        }
        __syncthreads();
        for (int i = tid; i < nbins * kSLd; i += kSBlock) stage[i] = 0.f; // the forward walk of the next block starts from zeros
        __syncthreads();
    }
}

size_t win_smem(int nbw, int nbins) { return (size_t)(kGK + 2) * nbw * sizeof(float2) + (size_t)nbins * kSLd * sizeof(float); }

template <int NBW, bool BACK>
cudaError_t launch_win(const Lors &l, int64_t n, const float *pimg_r, float *pimg_w, const Geom &g, const Tof &t,
                       const GTab &gt, float *p, const float *y, const SinoEpi &epi, cudaStream_t st)
{
    const size_t smem = win_smem(NBW, t.nbins);
    auto kern = k_tof_sino_win<NBW, BACK>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, nsm = 0, per_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kSBlock, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    const int64_t nblocks = (n + kSBlock - 1) / kSBlock;
    const int64_t cap = (int64_t)nsm * per_sm;
    const unsigned grid = (unsigned)(nblocks < cap ? nblocks : cap);
    kern<<<grid, kSBlock, smem, st>>>(l, n, nblocks, pimg_r, pimg_w, g, t, gt, p, y, epi);
    return cudaGetLastError();
}

} // namespace

// returns cudaErrorNotSupported when the TOF window is wider than the compiled sizes or the tile does not fit
// in shared memory (the caller then uses the generic kernels of jp_kernels.cu)
cudaError_t launch_tof_sino_win(bool back, const Lors &l, int64_t n, const float *pimg_r, float *pimg_w, const Geom &g,
                                const Tof &t, float *p, const float *y, cudaStream_t st, const SinoEpi *epi_in)
{
    const SinoEpi epi = epi_in ? *epi_in : SinoEpi{};
    if (n == 0) return cudaSuccess;
    double R;
    int nbw = window_bins(t, &R);
    if (!nbw || win_smem(nbw, t.nbins) > 72 * 1024) return cudaErrorNotSupported;
    GTab gt{};
    cudaError_t e = gtab_create(t, st, &gt, &nbw);
    if (e == cudaSuccess) {
#define JP_WIN(NB)                                                                                           \
    case NB:                                                                                                 \
        e = back ? launch_win<NB, true>(l, n, pimg_r, pimg_w, g, t, gt, p, y, epi, st)                             \
                 : launch_win<NB, false>(l, n, pimg_r, pimg_w, g, t, gt, p, y, epi, st);                           \
        break;
        switch (nbw) {
            JP_WIN(4)
            JP_WIN(6)
            JP_WIN(8)
            JP_WIN(12)
        default: e = cudaErrorNotSupported;
        }
#undef JP_WIN
    }
    gtab_destroy(&gt, st);
    return e;
}

// fused OSEM subset pass (forward + ratio + back); cudaErrorNotSupported as for launch_tof_sino_win
namespace {
template <int NBW>
cudaError_t launch_osem_win(const Lors &l, int64_t n, const float *pimg_r, float *pimg_w, const Geom &g, const Tof &t,
                            const GTab &gt, const SinoEpi &epi, cudaStream_t st)
{
    const size_t smem = win_smem(NBW, t.nbins);
    auto kern = k_tof_sino_osem<NBW>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, nsm = 0, per_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kSBlock, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    const int64_t nblocks = (n + kSBlock - 1) / kSBlock;
    const int64_t cap = (int64_t)nsm * per_sm;
    kern<<<(unsigned)(nblocks < cap ? nblocks : cap), kSBlock, smem, st>>>(l, n, nblocks, pimg_r, pimg_w, g, t, gt, epi);
    return cudaGetLastError();
}
} // namespace

cudaError_t launch_tof_sino_osem(const Lors &l, int64_t n, const float *pimg_r, float *pimg_w, const Geom &g, const Tof &t,
                                 const SinoEpi &epi, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    double R;
    int nbw = window_bins(t, &R);
    if (!nbw || win_smem(nbw, t.nbins) > 72 * 1024) return cudaErrorNotSupported;
    GTab gt{};
    cudaError_t e = gtab_create(t, st, &gt, &nbw);
    if (e == cudaSuccess) {
        switch (nbw) {
        case 4: e = launch_osem_win<4>(l, n, pimg_r, pimg_w, g, t, gt, epi, st); break;
        case 6: e = launch_osem_win<6>(l, n, pimg_r, pimg_w, g, t, gt, epi, st); break;
        case 8: e = launch_osem_win<8>(l, n, pimg_r, pimg_w, g, t, gt, epi, st); break;
        case 12: e = launch_osem_win<12>(l, n, pimg_r, pimg_w, g, t, gt, epi, st); break;
        default: e = cudaErrorNotSupported;
        }
    }
    gtab_destroy(&gt, st);
    return e;
}

// ---- unfused stages for the generic TOF sinogram kernels (TOF window wider than the compiled register windows) ----
namespace {
__global__ void k_sino_ratio(float *__restrict__ r, const float *__restrict__ y, const float *__restrict__ mult,
                             const float *__restrict__ contam, int64_t n, int nbins)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n * nbins) return;
    const float mj = mult ? mult[i / nbins] : 1.f;
    const float yb = fmaf(mj, r[i], contam ? contam[i] : 0.f);
    r[i] = (yb > 1e-9f) ? mj * y[i] / yb : 0.f;
}
__global__ void k_sino_bcast(float *__restrict__ r, const float *__restrict__ mult, int64_t n, int nbins)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n * nbins) return;
    r[i] = mult ? mult[i / nbins] : 1.f;
}
} // namespace

cudaError_t launch_sino_ratio(float *r, const float *y, const float *mult, const float *contam, int64_t n, int nbins,
                              cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_sino_ratio<<<(unsigned)((n * nbins + 255) / 256), 256, 0, st>>>(r, y, mult, contam, n, nbins);
    return cudaGetLastError();
}

cudaError_t launch_sino_bcast(float *r, const float *mult, int64_t n, int nbins, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_sino_bcast<<<(unsigned)((n * nbins + 255) / 256), 256, 0, st>>>(r, mult, n, nbins);
    return cudaGetLastError();
}

} // namespace jp
