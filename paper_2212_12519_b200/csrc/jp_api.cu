// jp_api.cu -- the extern "C" boundary of libjoseph_b200.so (see include/joseph_b200.h).
// Argument validation, error text, and dispatch to the kernel launchers; no arithmetic here.
#include <cstdio>
#include <cstring>

#include "../../include/joseph_b200.h"
#include "jp_internal.h"

namespace jp {
thread_local char g_err_buf[512] = "";
char *err_buf() { return g_err_buf; }
} // namespace jp

namespace {

#define g_err jp::g_err_buf

int fail_cuda(cudaError_t e, const char *where)
{
    snprintf(g_err, 512, "%s: %s (%s)", where, cudaGetErrorString(e), cudaGetErrorName(e));
    return JP_ERR_CUDA;
}

int fail(int code, const char *msg)
{
    snprintf(g_err, 512, "%s", msg);
    return code;
}

int check_geom(const jp_geom *g, jp::Geom &out)
{
    if (!g) return fail(JP_ERR_POINTER, "geom is NULL");
    int64_t nvox = 1;
    for (int a = 0; a < 3; ++a) {
        if (g->n[a] <= 0) return fail(JP_ERR_SIZE, "image dim <= 0");
        if (!(g->voxsize[a] > 0.f)) return fail(JP_ERR_SIZE, "voxsize <= 0");
        out.n[a] = g->n[a];
        out.o[a] = g->origin[a];
        out.v[a] = g->voxsize[a];
        nvox *= g->n[a];
    }
    if (nvox >= (int64_t)1 << 31) return fail(JP_ERR_SIZE, "image has >= 2^31 voxels");
    return JP_OK;
}

int check_tof(const jp_tof *t, bool sino, jp::Tof &out)
{
    if (!t) return fail(JP_ERR_POINTER, "tof is NULL");
    if (!(t->tofbin_width_mm > 0.f)) return fail(JP_ERR_SIZE, "tofbin_width <= 0");
    if (!(t->sigma_tof_mm > 0.f)) return fail(JP_ERR_SIZE, "sigma_tof <= 0");
    if (!(t->n_sigmas > 0.f)) return fail(JP_ERR_SIZE, "n_sigmas <= 0");
    if (sino && (t->n_tofbins < 1 || t->n_tofbins > JP_MAX_TOFBINS)) return fail(JP_ERR_SIZE, "n_tofbins out of range");
    out.width = t->tofbin_width_mm;
    out.sigma = t->sigma_tof_mm;
    out.nsig = t->n_sigmas;
    out.nbins = t->n_tofbins;
    out.coff = t->center_offset_mm;
    return JP_OK;
}

int check_lors(const jp_lors *l, jp::Lors &out)
{
    if (!l) return fail(JP_ERR_POINTER, "lors is NULL");
    if (l->n < 0) return fail(JP_ERR_SIZE, "n < 0");
    if (l->n > 0 && (!l->xs || !l->ys || !l->zs || !l->xe || !l->ye || !l->ze))
        return fail(JP_ERR_POINTER, "LOR coordinate array is NULL");
    out.xs = l->xs; out.ys = l->ys; out.zs = l->zs;
    out.xe = l->xe; out.ye = l->ye; out.ze = l->ze;
    return JP_OK;
}

inline jp::Range whole(int64_t n) { return jp::Range{0, 1, n, false, nullptr}; }

#define JP_TRY(expr)                  \
    do {                              \
        int rc__ = (expr);            \
        if (rc__ != JP_OK) return rc__; \
    } while (0)

#define JP_CUDA(expr, where)                              \
    do {                                                  \
        cudaError_t e__ = (expr);                         \
        if (e__ != cudaSuccess) return fail_cuda(e__, where); \
    } while (0)

} // namespace

extern "C" {

const char *jp_last_error(void) { return g_err; }
int jp_version(void) { return 100; }

int jp_classify(const jp_lors *lors, uint8_t *principal_axis, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    JP_TRY(check_lors(lors, l));
    if (lors->n > 0 && !principal_axis) return fail(JP_ERR_POINTER, "principal_axis is NULL");
    JP_CUDA(jp::launch_classify(l, lors->n, principal_axis, (cudaStream_t)stream), "jp_classify");
    return JP_OK;
}

int jp_plane_steps(const jp_lors *lors, const jp_geom *geom, unsigned long long *total, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    if (!total) return fail(JP_ERR_POINTER, "total is NULL");
    JP_CUDA(jp::launch_plane_steps(l, lors->n, g, total, (cudaStream_t)stream), "jp_plane_steps");
    return JP_OK;
}

int jp_fwd(const jp_lors *lors, const float *img, const jp_geom *geom, float *p, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    if (!img || (lors->n > 0 && !p)) return fail(JP_ERR_POINTER, "img or p is NULL");
    JP_CUDA(jp::launch_fwd_tile(l, lors->n, img, g, p, (cudaStream_t)stream), "jp_fwd");
    return JP_OK;
}

int jp_back(const jp_lors *lors, const float *y, const jp_geom *geom, float *img, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    if (!img || (lors->n > 0 && !y)) return fail(JP_ERR_POINTER, "img or y is NULL");
    JP_CUDA(jp::launch_back_tile(l, lors->n, y, g, img, (cudaStream_t)stream), "jp_back");
    return JP_OK;
}

int jp_fwd_tof_sino(const jp_lors *lors, const float *img, const jp_geom *geom, const jp_tof *tof, float *p,
                    void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    if (!img || (lors->n > 0 && !p)) return fail(JP_ERR_POINTER, "img or p is NULL");
    if (lors->n == 0) return JP_OK;
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, (cudaStream_t)stream, &lut), "jp_fwd_tof_sino (table)");
    const cudaError_t e = jp::launch_fwd_tof_sino(l, whole(lors->n), img, g, t, lut, p, (cudaStream_t)stream);
    jp::tof_lut_destroy(&lut, (cudaStream_t)stream);
    JP_CUDA(e, "jp_fwd_tof_sino");
    return JP_OK;
}

int jp_back_tof_sino(const jp_lors *lors, const float *y, const jp_geom *geom, const jp_tof *tof, float *img,
                     void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    if (!img || (lors->n > 0 && !y)) return fail(JP_ERR_POINTER, "img or y is NULL");
    if (lors->n == 0) return JP_OK;
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, (cudaStream_t)stream, &lut), "jp_back_tof_sino (table)");
    const cudaError_t e = jp::launch_back_tof_sino(l, whole(lors->n), y, g, t, lut, img, (cudaStream_t)stream);
    jp::tof_lut_destroy(&lut, (cudaStream_t)stream);
    JP_CUDA(e, "jp_back_tof_sino");
    return JP_OK;
}

int jp_fwd_tof_lm(const jp_lors *lors, const int16_t *tofbin, const float *img, const jp_geom *geom,
                  const jp_tof *tof, float *p, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, false, t));
    if (!img || (lors->n > 0 && (!p || !tofbin))) return fail(JP_ERR_POINTER, "img, p or tofbin is NULL");
    if (lors->n == 0) return JP_OK;
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, (cudaStream_t)stream, &lut), "jp_fwd_tof_lm (table)");
    const cudaError_t e = jp::launch_fwd_tof_lm(l, tofbin, whole(lors->n), img, g, t, lut, p, 0, (cudaStream_t)stream);
    jp::tof_lut_destroy(&lut, (cudaStream_t)stream);
    JP_CUDA(e, "jp_fwd_tof_lm");
    return JP_OK;
}

int jp_back_tof_lm(const jp_lors *lors, const int16_t *tofbin, const float *y, const jp_geom *geom,
                   const jp_tof *tof, float *img, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, false, t));
    if (!img || (lors->n > 0 && (!y || !tofbin))) return fail(JP_ERR_POINTER, "img, y or tofbin is NULL");
    if (lors->n == 0) return JP_OK;
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, (cudaStream_t)stream, &lut), "jp_back_tof_lm (table)");
    const cudaError_t e = jp::launch_back_tof_lm(l, tofbin, whole(lors->n), y, g, t, lut, img, (cudaStream_t)stream);
    jp::tof_lut_destroy(&lut, (cudaStream_t)stream);
    JP_CUDA(e, "jp_back_tof_lm");
    return JP_OK;
}

// workspace layout: [b: nvox floats][r: ceil(n_events / n_subsets) floats]
size_t jp_lm_osem_workspace_bytes(int64_t n_events, const jp_geom *geom, int n_subsets)
{
    if (!geom || n_events < 0 || n_subsets < 1) return 0;
    const int64_t nvox = (int64_t)geom->n[0] * geom->n[1] * geom->n[2];
    const int64_t per = (n_events + n_subsets - 1) / n_subsets;
    return (size_t)(nvox + per + 64) * sizeof(float);
}

int jp_lm_osem(const jp_lors *events, const int16_t *tofbin, const jp_geom *geom, const jp_tof *tof,
               const float *sens, float *img, int n_subsets, int n_iter, void *workspace, size_t workspace_bytes,
               void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(events, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, false, t));
    if (n_subsets < 1 || n_iter < 0) return fail(JP_ERR_SIZE, "n_subsets < 1 or n_iter < 0");
    if (!sens || !img || !workspace || (events->n > 0 && !tofbin)) return fail(JP_ERR_POINTER, "NULL argument");
    if (workspace_bytes < jp_lm_osem_workspace_bytes(events->n, geom, n_subsets))
        return fail(JP_ERR_SIZE, "workspace too small");
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n = events->n;
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    float *b = (float *)workspace;
    float *r = b + ((nvox + 31) / 32) * 32;
    JP_CUDA(cudaMemsetAsync(b, 0, (size_t)nvox * sizeof(float), st), "jp_lm_osem memset");
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, st, &lut), "jp_lm_osem (table)");
    cudaError_t e = cudaSuccess;
    for (int it = 0; it < n_iter && e == cudaSuccess; ++it) {
        for (int m = 0; m < n_subsets && e == cudaSuccess; ++m) {
            const int64_t count = (n > m) ? (n - m + n_subsets - 1) / n_subsets : 0;
            const jp::Range rg{m, n_subsets, count, true, nullptr};
            e = jp::launch_fwd_tof_lm(l, tofbin, rg, img, g, t, lut, r, 1, st);
            if (e == cudaSuccess) e = jp::launch_back_tof_lm(l, tofbin, rg, r, g, t, lut, b, st);
            if (e == cudaSuccess) e = jp::launch_osem_update(img, b, sens, (float)n_subsets, nvox, st);
        }
    }
    jp::tof_lut_destroy(&lut, st);
    JP_CUDA(e, "jp_lm_osem");
    return JP_OK;
}


// ---- listmode plan ------------------------------------------------------------------------------------------
struct jp_plan {
    jp::LmPlan *lm;
};

int jp_lm_plan_create(const jp_lors *events, const int16_t *tofbin, const jp_geom *geom, const jp_tof *tof,
                      int n_subsets, void *stream, jp_plan **plan)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(events, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, false, t));
    if (!plan) return fail(JP_ERR_POINTER, "plan is NULL");
    *plan = nullptr;
    if (n_subsets < 1 || n_subsets > 255) return fail(JP_ERR_SIZE, "n_subsets must be in 1..255");
    if (events->n >= ((int64_t)1 << 31)) return fail(JP_ERR_SIZE, "a plan holds fewer than 2^31 events");
    if (events->n > 0 && !tofbin) return fail(JP_ERR_POINTER, "tofbin is NULL");
    jp::LmPlan *lm = nullptr;
    JP_CUDA(jp::lm_plan_create(l, tofbin, events->n, g, t, n_subsets, (cudaStream_t)stream, &lm), "jp_lm_plan_create");
    jp_plan *pl = new jp_plan;
    pl->lm = lm;
    *plan = pl;
    return JP_OK;
}

int jp_lm_plan_destroy(jp_plan *plan)
{
    g_err[0] = 0;
    if (!plan) return JP_OK;
    if (!plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    jp::lm_plan_destroy(plan->lm);
    plan->lm = nullptr;
    delete plan;
    return JP_OK;
}

int64_t jp_lm_plan_subset_count(const jp_plan *plan, int subset)
{
    if (!plan || !plan->lm) return -1;
    jp::Lors l;
    const int16_t *tb;
    jp::Range rg;
    if (subset >= jp::lm_plan_subsets(plan->lm)) return -1;
    jp::lm_plan_view(plan->lm, subset, true, &l, &tb, &rg);
    return rg.count;
}

int jp_fwd_tof_lm_planned(const jp_plan *plan, int subset, const float *img, float *p, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    jp::Lors l;
    const int16_t *tb;
    jp::Range rg;
    jp::lm_plan_view(plan->lm, subset, false, &l, &tb, &rg);
    if (rg.count == 0) return JP_OK;
    if (!img || !p) return fail(JP_ERR_POINTER, "img or p is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const jp::Tof &t = jp::lm_plan_tof(plan->lm);
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, st, &lut), "jp_fwd_tof_lm_planned (table)");
    const cudaError_t e = jp::launch_fwd_tof_lm(l, tb, rg, img, jp::lm_plan_geom(plan->lm), t, lut, p, 0, st);
    jp::tof_lut_destroy(&lut, st);
    JP_CUDA(e, "jp_fwd_tof_lm_planned");
    return JP_OK;
}

int jp_back_tof_lm_planned(const jp_plan *plan, int subset, const float *y, float *img, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    jp::Lors l;
    const int16_t *tb;
    jp::Range rg;
    jp::lm_plan_view(plan->lm, subset, false, &l, &tb, &rg);
    if (rg.count == 0) return JP_OK;
    if (!img || !y) return fail(JP_ERR_POINTER, "img or y is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const jp::Tof &t = jp::lm_plan_tof(plan->lm);
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, st, &lut), "jp_back_tof_lm_planned (table)");
    const cudaError_t e = jp::launch_back_tof_lm(l, tb, rg, y, jp::lm_plan_geom(plan->lm), t, lut, img, st);
    jp::tof_lut_destroy(&lut, st);
    JP_CUDA(e, "jp_back_tof_lm_planned");
    return JP_OK;
}

size_t jp_lm_osem_planned_workspace_bytes(const jp_plan *plan)
{
    if (!plan || !plan->lm) return 0;
    const jp::Geom &g = jp::lm_plan_geom(plan->lm);
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    const int64_t n = jp::lm_plan_n(plan->lm);
    const int ns = jp::lm_plan_subsets(plan->lm);
    return (size_t)(nvox + (n + ns - 1) / ns + 64) * sizeof(float);
}

int jp_lm_osem_planned(const jp_plan *plan, const float *sens, float *img, int n_iter, void *workspace,
                       size_t workspace_bytes, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (n_iter < 0) return fail(JP_ERR_SIZE, "n_iter < 0");
    if (!sens || !img || !workspace) return fail(JP_ERR_POINTER, "NULL argument");
    if (workspace_bytes < jp_lm_osem_planned_workspace_bytes(plan)) return fail(JP_ERR_SIZE, "workspace too small");
    cudaStream_t st = (cudaStream_t)stream;
    const jp::Geom &g = jp::lm_plan_geom(plan->lm);
    const jp::Tof &t = jp::lm_plan_tof(plan->lm);
    const int ns = jp::lm_plan_subsets(plan->lm);
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    float *b = (float *)workspace;
    float *r = b + ((nvox + 31) / 32) * 32;
    JP_CUDA(cudaMemsetAsync(b, 0, (size_t)nvox * sizeof(float), st), "jp_lm_osem_planned memset");
    jp::TofLut lut{};
    JP_CUDA(jp::tof_lut_create(t, st, &lut), "jp_lm_osem_planned (table)");
    cudaError_t e = cudaSuccess;
    for (int it = 0; it < n_iter && e == cudaSuccess; ++it) {
        for (int m = 0; m < ns && e == cudaSuccess; ++m) {
            jp::Lors l;
            const int16_t *tb;
            jp::Range rg;
            jp::lm_plan_view(plan->lm, m, true, &l, &tb, &rg); // r is indexed in sorted order: no permutation
            e = jp::launch_fwd_tof_lm(l, tb, rg, img, g, t, lut, r, 1, st);
            if (e == cudaSuccess) e = jp::launch_back_tof_lm(l, tb, rg, r, g, t, lut, b, st);
            if (e == cudaSuccess) e = jp::launch_osem_update(img, b, sens, (float)ns, nvox, st);
        }
    }
    jp::tof_lut_destroy(&lut, st);
    JP_CUDA(e, "jp_lm_osem_planned");
    return JP_OK;
}

} // extern "C"
