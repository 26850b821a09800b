// jp_sino_plan.cu -- sinogram plan: the structure of a LOR list, found once (set-up; BASELINE.json north_star (b):
// "LORs sorted or binned by principal axis and direction so neighbouring threads walk nearby voxels").
//
// The projectors take a plain list of LOR end points and know nothing about the scanner.  The lists a
// ring scanner produces are nevertheless highly regular: the sinogram of configs[1] is 65,792 TRACKS (one per
// (view, radial) bin: identical transaxial end points) of 2304 LORs (the ring pairs), and every track has the SAME
// axial pattern (zs, ze)[2304].  The plan detects exactly that, from the data alone:
//
//   T        length of the first run of LORs with bit-identical (xs, ys, xe, ye);
//   regular  n is a multiple of T, every block of T LORs is such a run, and (zs, ze)[j] == (zs, ze)[j mod T] bit for bit.
//
// A regular plan keeps K = n / T end-point quadruples, the pattern and a LANE ORDER: the pattern indices sorted by
// |ze - zs|.  LORs of one track with equal |ze - zs| have the same length, hence the same TOF coordinate on every
// plane (the TOF weight depends on the distance along the LOR), so a warp that takes 32 consecutive
// entries of that order reads ONE row of the TOF weight table per plane step (a shared-memory broadcast) and slides
// its TOF window in lockstep.  24 bytes per LOR shrink to 16 bytes per track.  Any other list is kept as a plain SoA
// copy and the planned calls run the unplanned kernels on it.
#include <algorithm>
#include <cmath>
#include <vector>

#include "jp_internal.h"

namespace jp {

namespace {

constexpr int kProbeMax = 1 << 16; // longest track the probe looks for

// first index in [1, lim) whose transaxial end points differ from LOR 0 (lim if none)
__global__ void k_sino_probe(Lors l, int lim, int *first)
{
    const uint32_t xs0 = __float_as_uint(l.xs[0]), ys0 = __float_as_uint(l.ys[0]);
    const uint32_t xe0 = __float_as_uint(l.xe[0]), ye0 = __float_as_uint(l.ye[0]);
    int mine = lim;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < lim; j += gridDim.x * blockDim.x) {
        const uint32_t d = (__float_as_uint(l.xs[j]) ^ xs0) | (__float_as_uint(l.ys[j]) ^ ys0) |
                           (__float_as_uint(l.xe[j]) ^ xe0) | (__float_as_uint(l.ye[j]) ^ ye0);
        if (d) {
            mine = j;
            break;
        }
    }
    for (int o = 16; o > 0; o >>= 1) mine = min(mine, __shfl_xor_sync(0xffffffffu, mine, o));
    if ((threadIdx.x & 31) == 0 && mine < lim) atomicMin(first, mine);
}

// ok[0] = 0 unless every block of T LORs is a track with the axial pattern of the first block
__global__ void k_sino_check(Lors l, int64_t n, int T, int *ok)
{
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    bool bad = false;
    if (j < n) {
        const int64_t h = (j / T) * T;
        const int i = (int)(j - h);
        const uint32_t d = (__float_as_uint(l.xs[j]) ^ __float_as_uint(l.xs[h])) | (__float_as_uint(l.ys[j]) ^ __float_as_uint(l.ys[h])) |
                           (__float_as_uint(l.xe[j]) ^ __float_as_uint(l.xe[h])) | (__float_as_uint(l.ye[j]) ^ __float_as_uint(l.ye[h])) |
                           (__float_as_uint(l.zs[j]) ^ __float_as_uint(l.zs[i])) | (__float_as_uint(l.ze[j]) ^ __float_as_uint(l.ze[i]));
        bad = d != 0;
    }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicExch(ok, 0);
}

__global__ void k_sino_extract(Lors l, int64_t K, int T, float4 *trk, float2 *zpat)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < K) {
        const int64_t h = i * T;
        trk[i] = make_float4(l.xs[h], l.ys[h], l.xe[h], l.ye[h]);
    }
    if (i < T) zpat[i] = make_float2(l.zs[i], l.ze[i]);
}

__global__ void k_sino_expand(const float4 *__restrict__ trk, const float2 *__restrict__ zpat, int T, int64_t first,
                              int64_t count, float *__restrict__ c)
{
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= count) return;
    const int64_t j = first + e;
    const float4 t = __ldg(trk + j / T);
    const float2 z = __ldg(zpat + (int)(j % T));
    c[e] = t.x;
    c[count + e] = t.y;
    c[2 * count + e] = z.x;
    c[3 * count + e] = t.z;
    c[4 * count + e] = t.w;
    c[5 * count + e] = z.y;
}

} // namespace

struct SinoPlan {
    SinoPlanView v;
    float4 *trk = nullptr;
    float2 *zpat = nullptr;
    int *order = nullptr;
    unsigned char *slot_grp = nullptr;
    int *slice_ng = nullptr;
    float2 *t_zp = nullptr; // both lane orders of the whole-track kernels, one allocation each
    int *t_ord = nullptr;
    float *coord = nullptr;
};

void sino_plan_destroy(SinoPlan *pl)
{
    if (!pl) return;
    cudaFree(pl->trk);
    cudaFree(pl->zpat);
    cudaFree(pl->order);
    cudaFree(pl->slot_grp);
    cudaFree(pl->slice_ng);
    cudaFree(pl->t_zp);
    cudaFree(pl->t_ord);
    cudaFree(pl->coord);
    delete pl;
}

SinoPlanView sino_plan_view(const SinoPlan *pl) { return pl->v; }

cudaError_t sino_plan_create(const Lors &l, int64_t n, cudaStream_t st, SinoPlan **out)
{
    SinoPlan *pl = new SinoPlan;
    *out = pl;
    pl->v.n = n;
    if (n == 0) return cudaSuccess;
    cudaError_t e = cudaSuccess;
    int *flag = nullptr;
    int T = 0, regular = 0;
#define JP_SP_TRY(x)                     \
    do {                                 \
        e = (x);                         \
        if (e != cudaSuccess) goto fail; \
    } while (0)
    JP_SP_TRY(cudaMallocAsync((void **)&flag, 2 * sizeof(int), st));
    {
        const int lim = (int)std::min<int64_t>(n, kProbeMax);
        int h[2] = {lim, 1};
        JP_SP_TRY(cudaMemcpyAsync(flag, h, sizeof(h), cudaMemcpyHostToDevice, st));
        k_sino_probe<<<64, 256, 0, st>>>(l, lim, flag);
        JP_SP_TRY(cudaGetLastError());
        JP_SP_TRY(cudaMemcpyAsync(h, flag, sizeof(int), cudaMemcpyDeviceToHost, st));
        JP_SP_TRY(cudaStreamSynchronize(st));
        T = h[0];
        // a run that reaches the probe limit without ending is not a track length we can trust (unless it is the list)
        if (T == lim && n > lim) T = 0;
        if (T >= 32 && n % T == 0) {
            k_sino_check<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(l, n, T, flag + 1);
            JP_SP_TRY(cudaGetLastError());
            JP_SP_TRY(cudaMemcpyAsync(h, flag + 1, sizeof(int), cudaMemcpyDeviceToHost, st));
            JP_SP_TRY(cudaStreamSynchronize(st));
            regular = h[0];
        }
    }
    if (regular) {
        const int64_t K = n / T;
        JP_SP_TRY(cudaMalloc((void **)&pl->trk, sizeof(float4) * (size_t)K));
        JP_SP_TRY(cudaMalloc((void **)&pl->zpat, sizeof(float2) * (size_t)T));
        JP_SP_TRY(cudaMalloc((void **)&pl->order, sizeof(int) * (size_t)T));
        const int64_t m = std::max<int64_t>(K, T);
        k_sino_extract<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(l, K, T, pl->trk, pl->zpat);
        JP_SP_TRY(cudaGetLastError());
        std::vector<float2> zp((size_t)T);
        JP_SP_TRY(cudaMemcpyAsync(zp.data(), pl->zpat, sizeof(float2) * (size_t)T, cudaMemcpyDeviceToHost, st));
        JP_SP_TRY(cudaStreamSynchronize(st));
        // ---- lane order (a performance hint only: any permutation of 0..T-1 gives the same results).
        // Groups = pattern entries of equal |dz| (exact in double), inside a group ordered by sign of dz, then zs.
        // Slices of kSinoSlice entries are filled with whole groups, largest first, each into the slice with the most
        // room (a group that fits nowhere is split), so that every slice holds few groups: the tile kernels build
        // ONE row of TOF weights per (group, plane).
        std::vector<int> ord((size_t)T);
        double dzmax = 0.0;
        auto dz_of = [&](int i) { return (double)zp[(size_t)i].y - (double)zp[(size_t)i].x; };
        for (int i = 0; i < T; ++i) {
            ord[(size_t)i] = i;
            dzmax = std::max(dzmax, std::fabs(dz_of(i)));
        }
        std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) {
            const double da = dz_of(a), db = dz_of(b);
            if (std::fabs(da) != std::fabs(db)) return std::fabs(da) < std::fabs(db);
            if ((da < 0) != (db < 0)) return da < 0;
            return zp[(size_t)a].x < zp[(size_t)b].x;
        });
        struct Grp { int first, count; };
        std::vector<Grp> grps;
        for (int i = 0; i < T;) {
            int j = i + 1;
            while (j < T && std::fabs(dz_of(ord[(size_t)j])) == std::fabs(dz_of(ord[(size_t)i]))) ++j;
            grps.push_back(Grp{i, j - i});
            i = j;
        }
        std::stable_sort(grps.begin(), grps.end(), [](const Grp &a, const Grp &b) { return a.count > b.count; });
        const int nsl = (T + kSinoSlice - 1) / kSinoSlice;
        std::vector<int> room((size_t)nsl, kSinoSlice), ngr((size_t)nsl, 0);
        room[(size_t)nsl - 1] = T - (nsl - 1) * kSinoSlice;
        std::vector<std::vector<int>> members((size_t)nsl);      // pattern indices per slice
        std::vector<std::vector<unsigned char>> mgrp((size_t)nsl);
        for (const Grp &gr : grps) {
            int first = gr.first, left = gr.count;
            while (left > 0) {
                int best = 0;
                for (int s2 = 1; s2 < nsl; ++s2)
                    if (room[(size_t)s2] > room[(size_t)best]) best = s2;
                const int take = std::min(left, room[(size_t)best]);
                const int gi = ngr[(size_t)best]++;
                for (int k = 0; k < take; ++k) {
                    members[(size_t)best].push_back(ord[(size_t)(first + k)]);
                    mgrp[(size_t)best].push_back((unsigned char)std::min(gi, 255));
                }
                room[(size_t)best] -= take;
                first += take;
                left -= take;
            }
        }
        std::vector<int> order_h((size_t)T), ng_h((size_t)nsl);
        std::vector<unsigned char> grp_h((size_t)T);
        for (int s2 = 0; s2 < nsl; ++s2) {
            ng_h[(size_t)s2] = ngr[(size_t)s2] <= kSinoGroupsMax ? ngr[(size_t)s2] : 0;
            for (size_t k = 0; k < members[(size_t)s2].size(); ++k) {
                order_h[(size_t)s2 * kSinoSlice + k] = members[(size_t)s2][k];
                grp_h[(size_t)s2 * kSinoSlice + k] = mgrp[(size_t)s2][k];
            }
        }
        JP_SP_TRY(cudaMalloc((void **)&pl->slot_grp, (size_t)T));
        JP_SP_TRY(cudaMalloc((void **)&pl->slice_ng, sizeof(int) * (size_t)nsl));
        JP_SP_TRY(cudaMemcpyAsync(pl->order, order_h.data(), sizeof(int) * (size_t)T, cudaMemcpyHostToDevice, st));
        JP_SP_TRY(cudaMemcpyAsync(pl->slot_grp, grp_h.data(), (size_t)T, cudaMemcpyHostToDevice, st));
        JP_SP_TRY(cudaMemcpyAsync(pl->slice_ng, ng_h.data(), sizeof(int) * (size_t)nsl, cudaMemcpyHostToDevice, st));
        // ---- lane orders of the whole-track kernels (jp_track.cu; again a performance hint only).  A track is cut into
        // equal pieces of at most 2304 LORs (9 per thread).  Inside a piece the LORs of a sinogram form a grid (rows: one
        // axial end point fixed, the other one varies: L columns).  Forward: a half-warp takes a block of 2 rows x 8
        // columns (at most ~11 axial cells wide: its 64-bit row loads stay conflict-free).  Adjoint: a half-warp takes a
        // 16-long grid diagonal (lanes one row pitch apart never hit one address), the next half-warp the next diagonal.
        const int kTrkSlotsMax = 9 * 256;
        const int npieces = (T + kTrkSlotsMax - 1) / kTrkSlotsMax;
        const int piece_len = (T + npieces - 1) / npieces;
        const int npt = piece_len <= 3 * 256 ? 3 : piece_len <= 6 * 256 ? 6 : 9;
        const int slots = npt * 256;
        std::vector<float2> tzp((size_t)2 * npieces * slots, make_float2(0.f, 0.f));
        std::vector<int> tord((size_t)2 * npieces * slots, -1);
        for (int pc = 0; pc < npieces; ++pc) {
            const int first = pc * piece_len, cnt = std::min(piece_len, T - first);
            // row length of the grid: the first entry whose zs (or ze) changes while the other one has been constant
            int Ls = cnt, Le = cnt;
            for (int i = 1; i < cnt && Ls == cnt; ++i)
                if (zp[(size_t)(first + i)].x != zp[(size_t)first].x) Ls = i;
            for (int i = 1; i < cnt && Le == cnt; ++i)
                if (zp[(size_t)(first + i)].y != zp[(size_t)first].y) Le = i;
            int L = 0;
            if (Ls == 1 && Le < cnt) L = Le;
            else if (Le == 1 && Ls < cnt) L = Ls;
            if (L < 2 || cnt % L) L = 0;
            std::vector<int> of, ob;
            of.reserve((size_t)cnt);
            ob.reserve((size_t)cnt);
            if (L) {
                const int R = cnt / L;
                for (int r0 = 0; r0 < R; r0 += 2)
                    for (int cb = 0; cb < L; cb += 8)
                        for (int r = r0; r < std::min(R, r0 + 2); ++r)
                            for (int c = cb; c < std::min(L, cb + 8); ++c) of.push_back(r * L + c);
                for (int r0 = 0; r0 < R; r0 += 16) {
                    const int nr = std::min(16, R - r0);
                    for (int c0 = 0; c0 < L; ++c0)
                        for (int d = 0; d < nr; ++d) ob.push_back((r0 + d) * L + (c0 + d) % L);
                }
            } else {
                for (int i = 0; i < cnt; ++i) {
                    of.push_back(i);
                    ob.push_back(i);
                }
            }
            for (int dir = 0; dir < 2; ++dir) {
                const std::vector<int> &o = dir ? ob : of;
                const size_t base = ((size_t)dir * npieces + pc) * slots;
                for (int i = 0; i < cnt; ++i) {
                    tord[base + i] = first + o[(size_t)i];
                    tzp[base + i] = zp[(size_t)(first + o[(size_t)i])];
                }
            }
        }
        JP_SP_TRY(cudaMalloc((void **)&pl->t_zp, sizeof(float2) * tzp.size()));
        JP_SP_TRY(cudaMalloc((void **)&pl->t_ord, sizeof(int) * tord.size()));
        JP_SP_TRY(cudaMemcpyAsync(pl->t_zp, tzp.data(), sizeof(float2) * tzp.size(), cudaMemcpyHostToDevice, st));
        JP_SP_TRY(cudaMemcpyAsync(pl->t_ord, tord.data(), sizeof(int) * tord.size(), cudaMemcpyHostToDevice, st));
        JP_SP_TRY(cudaStreamSynchronize(st)); // the vectors are host temporaries
        pl->v.t_npieces = npieces;
        pl->v.t_npt = npt;
        for (int dir = 0; dir < 2; ++dir) {
            pl->v.t_zp[dir] = pl->t_zp + (size_t)dir * npieces * slots;
            pl->v.t_ord[dir] = pl->t_ord + (size_t)dir * npieces * slots;
        }
        pl->v.K = K;
        pl->v.T = T;
        pl->v.regular = 1;
        pl->v.dz_max = dzmax;
        pl->v.trk = pl->trk;
        pl->v.zpat = pl->zpat;
        pl->v.order = pl->order;
        pl->v.slot_grp = pl->slot_grp;
        pl->v.slice_ng = pl->slice_ng;
    } else {
        JP_SP_TRY(cudaMalloc((void **)&pl->coord, sizeof(float) * 6 * (size_t)n));
        const float *src[6] = {l.xs, l.ys, l.zs, l.xe, l.ye, l.ze};
        for (int a = 0; a < 6; ++a)
            JP_SP_TRY(cudaMemcpyAsync(pl->coord + (size_t)a * n, src[a], sizeof(float) * (size_t)n, cudaMemcpyDeviceToDevice, st));
        float *c = pl->coord;
        pl->v.lors = Lors{c, c + n, c + 2 * n, c + 3 * n, c + 4 * n, c + 5 * n};
    }
    cudaFreeAsync(flag, st);
    return cudaSuccess;
fail:
    if (flag) cudaFreeAsync(flag, st);
    sino_plan_destroy(pl);
    *out = nullptr;
    return e;
#undef JP_SP_TRY
}

cudaError_t sino_plan_expand(const SinoPlanView &pv, int64_t first, int64_t count, float *coord6, cudaStream_t st, Lors *out)
{
    if (count > 0) {
        k_sino_expand<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(pv.trk, pv.zpat, pv.T, first, count, coord6);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    *out = Lors{coord6, coord6 + count, coord6 + 2 * count, coord6 + 3 * count, coord6 + 4 * count, coord6 + 5 * count};
    return cudaSuccess;
}

} // namespace jp
