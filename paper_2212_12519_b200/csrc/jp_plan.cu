// jp_plan.cu -- listmode plan: the events of every OSEM subset, reordered so that neighbouring threads
// walk nearby voxels (BASELINE.json north_star: "LORs sorted or binned by principal axis and direction
// so neighbouring threads walk nearby voxels"; the paper names pre-sorting of listmode events as the way
// to speed up the projections).
//
// Events arrive in acquisition order (random access).  The image is stored with the axial
// axis fastest, so a warp's four gathers per plane touch few 128-byte lines only when its lanes sit on
// the same transaxial line (same plane, same row) -- and its lanes stay converged only when their TOF
// windows cover the same planes.  The sort key, most significant field first:
//
//   subset (e mod n_subsets) | principal axis | transaxial slope d_q1/d_p (11 bits) | transaxial
//   intercept at the image centre plane (11 bits) | hash of the transaxial end points (20 bits) | plane of
//   the TOF bin centre (6 bits) | axial position of the TOF bin centre (6 bits)
//
// It is purely geometric (no scanner model): crystal-snapped events of one crystal pair get the same
// slope/intercept cell, continuous events get neighbours.  The plan owns a sorted SoA copy of the end
// points and TOF bins (coalesced loads) and the permutation (results are returned in caller order).
// The sort itself is CUB's device radix sort (a library primitive used for set-up); key generation,
// gather and all projections are this library's kernels.
#include <cub/device/device_radix_sort.cuh>

#include <vector>

#include "jp_internal.h"

namespace jp {

__global__ void k_lm_keys(Lors l, const int16_t *__restrict__ tofbin, int64_t n, Geom g, Tof t, int n_subsets,
                          unsigned long long *__restrict__ keys, int *__restrict__ idx, int *__restrict__ counts)
{
    // events per (subset, principal axis): block-level counters, then one global atomic per non-empty counter
    extern __shared__ int cnt_sm[]; // [n_subsets][4]
    for (int i = threadIdx.x; i < n_subsets * 4; i += blockDim.x) cnt_sm[i] = 0;
    __syncthreads();
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j < n) {
    const float s[3] = {l.xs[j], l.ys[j], l.zs[j]};
    const float e[3] = {l.xe[j], l.ye[j], l.ze[j]};
    const double d0 = (double)e[0] - (double)s[0], d1 = (double)e[1] - (double)s[1], d2 = (double)e[2] - (double)s[2];
    const int p = principal_axis(d0, d1, d2);
    const float d[3] = {(float)d0, (float)d1, (float)d2};
    unsigned long long key = (unsigned long long)(j % n_subsets) << 56 | (unsigned long long)p << 54;
    const float L = sqrtf(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (L > 0.f) {
        const int q1 = (p == 0) ? 1 : 0, q2 = (p == 2) ? 1 : 2;
        const float inv_dp = 1.f / d[p];
        // transaxial line in slope / intercept form (the same for both orientations of the event)
        const float slope = d[q1] * inv_dp; // in [-1, 1]
        const float cp = g.o[p] + 0.5f * (float)(g.n[p] - 1) * g.v[p];
        const float cq = g.o[q1] + 0.5f * (float)(g.n[q1] - 1) * g.v[q1];
        const float icpt = s[q1] + (cp - s[p]) * slope - cq;              // mm from the image centre
        const float half = 0.75f * (float)g.n[q1] * g.v[q1];              // covers the image with margin
        const int ks = min(2047, max(0, (int)((slope + 1.f) * 1023.5f)));
        const int ki = min(2047, max(0, (int)((icpt / half + 1.f) * 1023.5f)));
        // TOF bin centre: tau_c mm from the midpoint towards e
        const float tau_c = (float)tofbin[j] * t.width + t.coff;
        const float f = 0.5f + tau_c / L;
        const float xc = s[p] + f * d[p], zc = s[q2] + f * d[q2];
        const int kp = min(63, max(0, (int)((xc - g.o[p]) / (g.v[p] * (float)g.n[p]) * 64.f)));
        const int kz = min(63, max(0, (int)((zc - g.o[q2]) / (g.v[q2] * (float)g.n[q2]) * 64.f)));
        // 20-bit hash of the canonically ordered transaxial end points: events of one crystal pair (either
        // orientation) that share a slope / intercept cell with another pair still form ONE contiguous run
        // (the line tiles of jp_lm_tile.cu need that; a hash collision only costs a tile its coherence)
        const bool sw = !((s[0] < e[0]) || (s[0] == e[0] && s[1] <= e[1]));
        const unsigned ax = __float_as_uint(sw ? e[0] : s[0]), ay = __float_as_uint(sw ? e[1] : s[1]);
        const unsigned bx = __float_as_uint(sw ? s[0] : e[0]), by = __float_as_uint(sw ? s[1] : e[1]);
        unsigned h = ax * 0x9E3779B1u;
        h = (h ^ (h >> 15) ^ ay) * 0x85EBCA77u;
        h = (h ^ (h >> 13) ^ bx) * 0xC2B2AE3Du;
        h = (h ^ (h >> 16) ^ by) * 0x27D4EB2Fu;
        h ^= h >> 15;
        key |= (unsigned long long)ks << 43 | (unsigned long long)ki << 32 | (unsigned long long)(h & 0xFFFFFu) << 12 |
               (unsigned long long)kp << 6 | (unsigned long long)kz;
    }
    keys[j] = key;
    idx[j] = (int)j;
    atomicAdd(&cnt_sm[(int)(j % n_subsets) * 4 + p], 1);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_subsets * 4; i += blockDim.x)
        if (cnt_sm[i]) atomicAdd(&counts[i], cnt_sm[i]);
}

// sorted SoA copy of the events.  A gather of seven arrays through the permutation touches seven 32-byte sectors per
// event; packing the event into ONE 32-byte record first (coalesced) makes it one sector per event.
__global__ void k_lm_pack(Lors l, const int16_t *__restrict__ tofbin, int64_t n, float4 *__restrict__ rec)
{
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= n) return;
    rec[2 * j] = make_float4(l.xs[j], l.ys[j], l.zs[j], l.xe[j]);
    rec[2 * j + 1] = make_float4(l.ye[j], l.ze[j], __int_as_float((int)tofbin[j]), 0.f);
}

__global__ void k_lm_gather(const float4 *__restrict__ rec, const int *__restrict__ perm, int64_t n,
                            float *__restrict__ xs, float *__restrict__ ys, float *__restrict__ zs,
                            float *__restrict__ xe, float *__restrict__ ye, float *__restrict__ ze,
                            int16_t *__restrict__ tb)
{
    const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c >= n) return;
    const int64_t j = perm[c];
    const float4 a = __ldg(rec + 2 * j), b = __ldg(rec + 2 * j + 1);
    xs[c] = a.x;
    ys[c] = a.y;
    zs[c] = a.z;
    xe[c] = a.w;
    ye[c] = b.x;
    ze[c] = b.y;
    tb[c] = (int16_t)__float_as_int(b.z);
}

__global__ void k_lm_permute(const int *__restrict__ perm, const float *__restrict__ in, float *__restrict__ out, int64_t n,
                             int to_plan)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int j = perm[k];
    if (to_plan) out[k] = in[j];
    else out[j] = in[k];
}

// number of runs of consecutive sorted events with the same (canonically ordered) transaxial end points
__global__ void k_lm_count_runs(const float *__restrict__ xs, const float *__restrict__ ys, const float *__restrict__ xe,
                                const float *__restrict__ ye, int64_t n, unsigned long long *__restrict__ runs)
{
    const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    bool flag = false;
    if (c < n) {
        flag = (c == 0);
        if (!flag) {
            float a[4] = {xs[c], ys[c], xe[c], ye[c]}, b[4] = {xs[c - 1], ys[c - 1], xe[c - 1], ye[c - 1]};
            if (!((a[0] < a[2]) || (a[0] == a[2] && a[1] <= a[3]))) { float t = a[0]; a[0] = a[2]; a[2] = t; t = a[1]; a[1] = a[3]; a[3] = t; }
            if (!((b[0] < b[2]) || (b[0] == b[2] && b[1] <= b[3]))) { float t = b[0]; b[0] = b[2]; b[2] = t; t = b[1]; b[1] = b[3]; b[3] = t; }
            flag = (a[0] != b[0]) || (a[1] != b[1]) || (a[2] != b[2]) || (a[3] != b[3]);
        }
    }
    const unsigned bal = __ballot_sync(0xffffffffu, flag);
    if ((threadIdx.x & 31) == 0 && bal) atomicAdd(runs, (unsigned long long)__popc(bal));
}

struct LmPlan {
    int64_t n = 0;
    int64_t n_runs = 0;     // runs of events sharing their transaxial line in the sorted list
    int n_subsets = 1;
    int path = 0;           // 0: automatic, 1: line tiles, 2: quad image (jp_lm_plan_set_path)
    Geom g{};
    Tof t{};
    float *coord = nullptr; // 6 arrays of n floats: xs ys zs xe ye ze, sorted
    int16_t *tb = nullptr;  // sorted TOF bins
    int *perm = nullptr;    // sorted position -> caller index
    std::vector<int64_t> seg_first, seg_count; // [n_subsets][4]: run of (subset, principal axis) in the sorted list
    float4 *quad[4] = {nullptr, nullptr, nullptr, nullptr}; // Q0, Q1, B0, B1 (allocated on first use)
    BrickSet *bricks = nullptr; // pieces of the events per image brick (jp_brick.cu), built by lm_plan_bricks
    bool bricks_tried = false;  // a failed build is not repeated
};

static int bits_for(int v)
{
    int b = 0;
    while ((1 << b) < v) ++b;
    return b;
}

cudaError_t lm_plan_create(const Lors &l, const int16_t *tofbin, int64_t n, const Geom &g, const Tof &t,
                           int n_subsets, cudaStream_t st, LmPlan **out)
{
    LmPlan *pl = new LmPlan;
    pl->n = n;
    pl->n_subsets = n_subsets;
    pl->g = g;
    pl->t = t;
    *out = pl;
    pl->seg_first.assign((size_t)n_subsets * 4, 0);
    pl->seg_count.assign((size_t)n_subsets * 4, 0);
    if (n == 0) return cudaSuccess;
    cudaError_t e;
    unsigned long long *keys = nullptr, *keys2 = nullptr;
    int *idx = nullptr, *counts = nullptr;
    float4 *rec = nullptr;
    void *tmp = nullptr;
    size_t tmp_bytes = 0;
#define JP_PLAN_TRY(x)                  \
    do {                                \
        e = (x);                        \
        if (e != cudaSuccess) goto fail; \
    } while (0)
    JP_PLAN_TRY(cudaMalloc((void **)&pl->coord, sizeof(float) * 6 * (size_t)n));
    JP_PLAN_TRY(cudaMalloc((void **)&pl->tb, sizeof(int16_t) * (size_t)n));
    JP_PLAN_TRY(cudaMalloc((void **)&pl->perm, sizeof(int) * (size_t)n));
    JP_PLAN_TRY(cudaMalloc((void **)&keys, sizeof(unsigned long long) * (size_t)n));
    JP_PLAN_TRY(cudaMalloc((void **)&keys2, sizeof(unsigned long long) * (size_t)n));
    JP_PLAN_TRY(cudaMalloc((void **)&idx, sizeof(int) * (size_t)n));
    JP_PLAN_TRY(cudaMalloc((void **)&counts, sizeof(int) * (size_t)n_subsets * 4));
    JP_PLAN_TRY(cudaMemsetAsync(counts, 0, sizeof(int) * (size_t)n_subsets * 4, st));
    {
        const unsigned grid = (unsigned)((n + 255) / 256);
        k_lm_keys<<<grid, 256, sizeof(int) * (size_t)n_subsets * 4, st>>>(l, tofbin, n, g, t, n_subsets, keys, idx, counts);
        JP_PLAN_TRY(cudaGetLastError());
        {   // the sorted list is ordered by (subset, axis, ...): turn the counts into runs (host, synchronises)
            std::vector<int> h((size_t)n_subsets * 4);
            JP_PLAN_TRY(cudaMemcpyAsync(h.data(), counts, sizeof(int) * h.size(), cudaMemcpyDeviceToHost, st));
            JP_PLAN_TRY(cudaStreamSynchronize(st));
            int64_t at = 0;
            for (size_t i = 0; i < h.size(); ++i) {
                pl->seg_first[i] = at;
                pl->seg_count[i] = h[i];
                at += h[i];
            }
        }
        const int end_bit = 56 + bits_for(n_subsets);
        JP_PLAN_TRY(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, idx, pl->perm, (int)n, 0, end_bit, st));
        JP_PLAN_TRY(cudaMalloc(&tmp, tmp_bytes));
        JP_PLAN_TRY(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys2, idx, pl->perm, (int)n, 0, end_bit, st));
        float *c = pl->coord;
        JP_PLAN_TRY(cudaMalloc((void **)&rec, sizeof(float4) * 2 * (size_t)n));
        k_lm_pack<<<grid, 256, 0, st>>>(l, tofbin, n, rec);
        JP_PLAN_TRY(cudaGetLastError());
        k_lm_gather<<<grid, 256, 0, st>>>(rec, pl->perm, n, c, c + n, c + 2 * n, c + 3 * n, c + 4 * n, c + 5 * n, pl->tb);
        JP_PLAN_TRY(cudaGetLastError());
        {   // run statistics of the sorted list: decides between line tiles and the quad kernels
            unsigned long long *runs = reinterpret_cast<unsigned long long *>(keys); // scratch, keys are dead
            unsigned long long h = 0;
            JP_PLAN_TRY(cudaMemsetAsync(runs, 0, sizeof(unsigned long long), st));
            k_lm_count_runs<<<grid, 256, 0, st>>>(c, c + n, c + 3 * n, c + 4 * n, n, runs);
            JP_PLAN_TRY(cudaGetLastError());
            JP_PLAN_TRY(cudaMemcpyAsync(&h, runs, sizeof(h), cudaMemcpyDeviceToHost, st));
            JP_PLAN_TRY(cudaStreamSynchronize(st));
            pl->n_runs = (int64_t)h;
        }
    }
    // (the stream has just been synchronised: the temporaries are idle.  Plain cudaMalloc / cudaFree on purpose: a
    // stream-ordered allocation of this size costs ~6 ms per GB to map and as much to trim at the next synchronisation)
    cudaFree(rec);
    cudaFree(tmp);
    cudaFree(counts);
    cudaFree(idx);
    cudaFree(keys2);
    cudaFree(keys);
    return cudaSuccess;
fail:
    cudaStreamSynchronize(st);
    cudaFree(rec);
    cudaFree(tmp);
    cudaFree(counts);
    cudaFree(idx);
    cudaFree(keys2);
    cudaFree(keys);
    lm_plan_destroy(pl);
    *out = nullptr;
    return e;
#undef JP_PLAN_TRY
}

void lm_plan_destroy(LmPlan *pl)
{
    if (!pl) return;
    cudaFree(pl->coord);
    cudaFree(pl->tb);
    cudaFree(pl->perm);
    for (float4 *q : pl->quad) cudaFree(q);
    brick_set_destroy(pl->bricks);
    delete pl;
}

void lm_plan_segment(const LmPlan *pl, int m, int a, int64_t *first, int64_t *count)
{
    *first = pl->seg_first[(size_t)m * 4 + a];
    *count = pl->seg_count[(size_t)m * 4 + a];
}

cudaError_t lm_plan_quad(LmPlan *pl, int which, float4 **out)
{
    if (!pl->quad[which]) {
        cudaError_t e = cudaMalloc((void **)&pl->quad[which], sizeof(float4) * (size_t)padded_voxels(pl->g));
        if (e != cudaSuccess) return e;
    }
    *out = pl->quad[which];
    return cudaSuccess;
}

// the plan's brick set, built on first use (allocates and synchronises `st`); *out = null when the image / TOF kernel /
// event count is outside what the brick kernels take (the callers then use the quad path)
cudaError_t lm_plan_bricks(LmPlan *pl, cudaStream_t st, const BrickSet **out)
{
    *out = nullptr;
    if (!pl->bricks && !pl->bricks_tried) {
        pl->bricks_tried = true;
        std::vector<int64_t> first((size_t)pl->n_subsets), count((size_t)pl->n_subsets);
        Lors l;
        const int16_t *tb;
        Range rg;
        for (int m = 0; m < pl->n_subsets; ++m) {
            lm_plan_view(pl, m, true, &l, &tb, &rg);
            first[(size_t)m] = rg.first;
            count[(size_t)m] = rg.count;
        }
        const cudaError_t e = brick_set_create(l, tb, pl->n, pl->g, pl->t, pl->n_subsets, first.data(), count.data(), st, &pl->bricks);
        if (e == cudaErrorMemoryAllocation) (void)cudaGetLastError(); // no room for the pieces: the plan works without them
        else if (e != cudaSuccess && e != cudaErrorNotSupported) return e;
    }
    *out = pl->bricks;
    return cudaSuccess;
}

cudaError_t lm_plan_permute(const LmPlan *pl, const float *in, float *out, bool to_plan_order, cudaStream_t st)
{
    if (pl->n == 0) return cudaSuccess;
    k_lm_permute<<<(unsigned)((pl->n + 255) / 256), 256, 0, st>>>(pl->perm, in, out, pl->n, to_plan_order ? 1 : 0);
    return cudaGetLastError();
}

int64_t lm_plan_n(const LmPlan *pl) { return pl->n; }
int64_t lm_plan_runs(const LmPlan *pl) { return pl->n_runs; }
int lm_plan_subsets(const LmPlan *pl) { return pl->n_subsets; }
int lm_plan_path(const LmPlan *pl) { return pl->path; }
void lm_plan_set_path(LmPlan *pl, int path) { pl->path = path; }
const Geom &lm_plan_geom(const LmPlan *pl) { return pl->g; }
const Tof &lm_plan_tof(const LmPlan *pl) { return pl->t; }

// sorted events of subset m (m < 0: all subsets) as a LOR list + range; per-event inputs / outputs are
// addressed through the permutation (caller order) unless `compact`
void lm_plan_view(const LmPlan *pl, int m, bool compact, Lors *l, const int16_t **tb, Range *rg)
{
    const int64_t n = pl->n;
    const float *c = pl->coord;
    l->xs = c;
    l->ys = c + n;
    l->zs = c + 2 * n;
    l->xe = c + 3 * n;
    l->ye = c + 4 * n;
    l->ze = c + 5 * n;
    *tb = pl->tb;
    int64_t first = 0, count = n;
    if (m >= 0) {
        const int ns = pl->n_subsets;
        // subset k holds the events {e : e mod ns == k}: ceil((n - k) / ns) of them, stored in subset order
        for (int k = 0; k < m; ++k) first += (n > k) ? (n - k + ns - 1) / ns : 0;
        count = (n > m) ? (n - m + ns - 1) / ns : 0;
    }
    rg->first = first;
    rg->stride = 1;
    rg->count = count;
    rg->compact = compact;
    rg->perm = compact ? nullptr : pl->perm;
}

} // namespace jp
