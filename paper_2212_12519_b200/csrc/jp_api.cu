// jp_api.cu -- the extern "C" boundary of libjoseph_b200.so (see include/joseph_b200.h).
// Argument validation, error text, and dispatch to the kernel launchers; no arithmetic here.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "../../include/joseph_b200.h"
#include "jp_g1tab.cuh"

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

// stream-ordered scratch of one TOF call: the edge-function table and a zero-padded image
struct TofCtx {
    jp::TofLut lut{};
    jp::G1Tab g1{};       // the brick kernels' TOF table, when the adjoint has to read the same weights (g1_init)
    float *pimg = nullptr;
    cudaStream_t st = nullptr;
    cudaError_t g1_init(const jp::Tof &t) { return jp::g1tab_create(t, jp::g1tab_entries(t), st, &g1); }
    ~TofCtx()
    {
        jp::tof_lut_destroy(&lut, st);
        jp::padded_destroy(pimg, st);
        if (g1.tab) cudaFreeAsync((void *)g1.tab, st);
    }
};

// mode 0: pimg = padded copy of img (forward); 1: pimg = zero accumulator (back)
static int tof_ctx_init(TofCtx &c, const jp::Tof &t, const jp::Geom &g, const float *img, int mode, cudaStream_t st,
                        const char *where)
{
    c.st = st;
    if (jp::padded_voxels(g) >= ((int64_t)1 << 31)) return fail(JP_ERR_SIZE, "padded image has >= 2^31 voxels");
    JP_CUDA(jp::tof_lut_create(t, st, &c.lut), where);
    JP_CUDA(jp::padded_create(img, g, mode == 1, st, &c.pimg), where);
    return JP_OK;
}

static int lm_fwd(const jp::Lors &l, const int16_t *tb, const jp::Range &rg, const float *img, const jp::Geom &g,
                  const jp::Tof &t, float *p, cudaStream_t st, const char *where)
{
    TofCtx c;
    JP_TRY(tof_ctx_init(c, t, g, img, 0, st, where));
    JP_CUDA(jp::launch_fwd_tof_lm(l, tb, rg, c.pimg, g, t, c.lut, p, 0, st), where);
    return JP_OK;
}

static int lm_back(const jp::Lors &l, const int16_t *tb, const jp::Range &rg, const float *y, const jp::Geom &g,
                   const jp::Tof &t, float *img, cudaStream_t st, const char *where)
{
    TofCtx c;
    JP_TRY(tof_ctx_init(c, t, g, nullptr, 1, st, where));
    JP_CUDA(jp::launch_back_tof_lm(l, tb, rg, y, g, t, c.lut, c.pimg, st), where);
    JP_CUDA(jp::padded_add_to(c.pimg, g, img, st), where);
    return JP_OK;
}

// OSEM subset loop on padded copies of x and b (allocated here, stream-ordered); r = per-event ratios
template <typename View>
static int lm_osem_loop(View view, int n_subsets, int n_iter, const jp::Geom &g, const jp::Tof &t, const float *sens,
                        float *img, float *r, cudaStream_t st, const char *where)
{
    TofCtx cx, cb; // cx.pimg = padded x, cb.pimg = padded b
    JP_TRY(tof_ctx_init(cx, t, g, img, 0, st, where));
    cb.st = st;
    JP_CUDA(jp::padded_create(nullptr, g, true, st, &cb.pimg), where);
    for (int it = 0; it < n_iter; ++it) {
        for (int m = 0; m < n_subsets; ++m) {
            jp::Lors l;
            const int16_t *tb;
            jp::Range rg;
            view(m, &l, &tb, &rg);
            JP_CUDA(jp::launch_fwd_tof_lm(l, tb, rg, cx.pimg, g, t, cx.lut, r, 1, st), where);
            JP_CUDA(jp::launch_back_tof_lm(l, tb, rg, r, g, t, cx.lut, cb.pimg, st), where);
            JP_CUDA(jp::launch_osem_update_padded(img, cx.pimg, cb.pimg, sens, (float)n_subsets, g, st), where);
        }
    }
    return JP_OK;
}

// Which kernels a planned listmode call uses.  Line tiles (jp_lm_tile.cu) pay when the sorted events come in long runs
// on one transaxial line (crystal-snapped events, all subsets together: ~2500 per run for configs[3]); sparsely
// populated lines (one OSEM subset of 20: ~120 per run) take the image bricks (jp_brick.cu), and whatever the bricks
// cannot hold takes the quad image (jp_quad.cu).  jp_lm_plan_set_path overrides the rule.
bool lm_tiles_wanted(const jp::LmPlan *lm, bool tof)
{
    if (!jp::lm_tile_supported(jp::lm_plan_geom(lm), jp::lm_plan_tof(lm), tof)) return false;
    const int path = jp::lm_plan_path(lm);
    if (path == 1) return true;
    if (path >= 2) return false;
    const int64_t runs = jp::lm_plan_runs(lm);
    return runs > 0 && jp::lm_plan_n(lm) / runs >= 512;
}

// the plan's brick set if the call should use it (path 0 / 3 and the plan could build one), else null.  The forward
// projection runs on the bricks; the adjoint keeps float atomics on the quad accumulators.
cudaError_t lm_bricks_wanted(jp::LmPlan *lm, cudaStream_t st, const jp::BrickSet **bs)
{
    *bs = nullptr;
    const int path = jp::lm_plan_path(lm);
    if (path == 1 || path == 2) return cudaSuccess;
    return jp::lm_plan_bricks(lm, st, bs);
}

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

int jp_plane_steps_tof_lm(const jp_lors *lors, const int16_t *tofbin, const jp_geom *geom, const jp_tof *tof,
                          unsigned long long *total, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, false, t));
    if (!total || (lors->n > 0 && !tofbin)) return fail(JP_ERR_POINTER, "total or tofbin is NULL");
    JP_CUDA(jp::launch_plane_steps_tof_lm(l, tofbin, lors->n, g, t, total, (cudaStream_t)stream),
            "jp_plane_steps_tof_lm");
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

// bodies of the unplanned TOF sinogram calls (also the fallback of the planned ones)
static int sino_fwd_impl(const jp::Lors &l, int64_t n, const float *img, const jp::Geom &g, const jp::Tof &t, float *p,
                         cudaStream_t st)
{
    if (n == 0) return JP_OK;
    TofCtx c;
    JP_TRY(tof_ctx_init(c, t, g, img, 0, st, "jp_fwd_tof_sino (scratch)"));
    cudaError_t e = jp::launch_tof_sino_win(false, l, n, c.pimg, nullptr, g, t, p, nullptr, st);
    if (e == cudaErrorNotSupported) // TOF window wider than the compiled register windows: generic kernel
        e = jp::launch_fwd_tof_sino(l, whole(n), c.pimg, g, t, c.lut, p, st);
    JP_CUDA(e, "jp_fwd_tof_sino");
    return JP_OK;
}

static int sino_back_impl(const jp::Lors &l, int64_t n, const float *y, const jp::Geom &g, const jp::Tof &t, float *img,
                          cudaStream_t st)
{
    if (n == 0) return JP_OK;
    TofCtx c;
    JP_TRY(tof_ctx_init(c, t, g, nullptr, 1, st, "jp_back_tof_sino (scratch)"));
    cudaError_t e = jp::launch_tof_sino_win(true, l, n, nullptr, c.pimg, g, t, nullptr, y, st);
    if (e == cudaErrorNotSupported)
        e = jp::launch_back_tof_sino(l, whole(n), y, g, t, c.lut, c.pimg, st);
    JP_CUDA(e, "jp_back_tof_sino");
    JP_CUDA(jp::padded_add_to(c.pimg, g, img, st), "jp_back_tof_sino (unpad)");
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
    return sino_fwd_impl(l, lors->n, img, g, t, p, (cudaStream_t)stream);
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
    return sino_back_impl(l, lors->n, y, g, t, img, (cudaStream_t)stream);
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
    return lm_fwd(l, tofbin, whole(lors->n), img, g, t, p, (cudaStream_t)stream, "jp_fwd_tof_lm");
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
    return lm_back(l, tofbin, whole(lors->n), y, g, t, img, (cudaStream_t)stream, "jp_back_tof_lm");
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
    (void)b;
    auto view = [&](int m, jp::Lors *lo, const int16_t **tb, jp::Range *rg) {
        *lo = l;
        *tb = tofbin;
        const int64_t count = (n > m) ? (n - m + n_subsets - 1) / n_subsets : 0;
        *rg = jp::Range{m, n_subsets, count, true, nullptr};
    };
    JP_TRY(lm_osem_loop(view, n_subsets, n_iter, g, t, sens, img, r, st, "jp_lm_osem"));
    return JP_OK;
}


// ---- listmode plan ------------------------------------------------------------------------------------------
struct jp_plan {
    jp::LmPlan *lm = nullptr;     // listmode plan (jp_lm_plan_create)
    jp::SinoPlan *sino = nullptr; // sinogram plan (jp_sino_plan_create)
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
    if (!lm_tiles_wanted(lm, true)) { // sparsely populated lines: the planned calls will want the brick pieces
        const jp::BrickSet *bs;
        const cudaError_t e = jp::lm_plan_bricks(lm, (cudaStream_t)stream, &bs);
        if (e != cudaSuccess) {
            jp_plan_destroy(pl);
            return fail_cuda(e, "jp_lm_plan_create (bricks)");
        }
    }
    *plan = pl;
    return JP_OK;
}

int jp_plan_destroy(jp_plan *plan)
{
    g_err[0] = 0;
    if (!plan) return JP_OK;
    if (!plan->lm && !plan->sino) return fail(JP_ERR_PLAN, "invalid plan");
    if (plan->lm) jp::lm_plan_destroy(plan->lm);
    if (plan->sino) jp::sino_plan_destroy(plan->sino);
    plan->lm = nullptr;
    plan->sino = nullptr;
    delete plan;
    return JP_OK;
}

int jp_lm_plan_destroy(jp_plan *plan) { return jp_plan_destroy(plan); }

int jp_lm_plan_set_path(jp_plan *plan, int path)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "not a listmode plan");
    if (path < 0 || path > 3)
        return fail(JP_ERR_SIZE, "path must be 0 (automatic), 1 (line tiles), 2 (quad image) or 3 (bricks forward, float adjoint)");
    jp::lm_plan_set_path(plan->lm, path);
    if (path == 3) { // builds the pieces now if the plan has none yet (allocates, synchronises the NULL stream)
        const jp::BrickSet *bs;
        JP_CUDA(jp::lm_plan_bricks(plan->lm, nullptr, &bs), "jp_lm_plan_set_path (bricks)");
    }
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

// ---- planned calls: quad image, axis by axis (jp_quad.cu) --------------------------------------------------------
namespace {

struct PlanCtx {
    jp::LmPlan *lm;
    jp::Lors l;
    const int16_t *tb;
    jp::Range all;          // the whole sorted list (perm set)
    int ns;
    jp::Geom g;
    jp::Tof t;
    explicit PlanCtx(const jp_plan *plan) : lm(plan->lm)
    {
        jp::lm_plan_view(lm, -1, false, &l, &tb, &all);
        ns = jp::lm_plan_subsets(lm);
        g = jp::lm_plan_geom(lm);
        t = jp::lm_plan_tof(lm);
    }
    // run of (subset m, axis a); compact: per-event arrays indexed from the start of subset m
    jp::Range seg(int m, int a, bool compact) const
    {
        int64_t first, count, sfirst, dummy;
        jp::lm_plan_segment(lm, m, a, &first, &count);
        jp::lm_plan_segment(lm, m, 0, &sfirst, &dummy);
        jp::Range rg{first, 1, count, compact, compact ? nullptr : all.perm};
        rg.io_off = first - sfirst;
        return rg;
    }
    // the same run with per-event arrays in PLAN order (index = position in the sorted list), or in caller order
    jp::Range seg_io(int m, int a, bool sorted_io) const
    {
        jp::Range rg = seg(m, a, sorted_io);
        if (sorted_io) rg.io_off = rg.first;
        return rg;
    }
    // all events of subset m (a contiguous run of the sorted list), per-event arrays indexed from its start
    jp::Range subset(int m) const
    {
        jp::Lors ll;
        const int16_t *tt;
        jp::Range rg;
        jp::lm_plan_view(lm, m, true, &ll, &tt, &rg);
        return rg;
    }
    bool has_axis2(int subset) const
    {
        for (int m = 0; m < ns; ++m)
            if (subset < 0 || m == subset) {
                int64_t f, c;
                jp::lm_plan_segment(lm, m, 2, &f, &c);
                if (c) return true;
            }
        return false;
    }
};

} // namespace

} // extern "C"

// the planned TOF listmode projectors as internal calls (also used by the hybrid handle, jp_host.cu)
namespace jp {

#define JP_E(x)                           \
    do {                                  \
        const cudaError_t e__ = (x);      \
        if (e__ != cudaSuccess) return e__; \
    } while (0)

cudaError_t lm_plan_fwd_tof(LmPlan *lm, int subset, const float *img, float *p, cudaStream_t st, bool sorted_io)
{
    jp_plan tmp;
    tmp.lm = lm;
    PlanCtx c(&tmp);
    TofCtx tc;
    tc.st = st;
    JP_E(jp::tof_lut_create(c.t, st, &tc.lut));
    const bool tiles = lm_tiles_wanted(c.lm, true);
    const jp::BrickSet *bs = nullptr;
    if (!tiles) JP_E(lm_bricks_wanted(c.lm, st, &bs));
    if (bs) { // image bricks: per-event sums of every subset in the plan's scratch array, then p = cf sum
        float *acc = jp::brick_set_acc(bs); // the plan's scratch (a plan is used from one stream at a time)
        cudaError_t e = cudaMemsetAsync(acc, 0, sizeof(float) * (size_t)jp::lm_plan_n(c.lm), st);
        for (int m = 0; m < c.ns && e == cudaSuccess; ++m)
            if (subset < 0 || m == subset) {
                e = jp::launch_brick_fwd(bs, m, img, c.g, c.t, 0, acc, st);
                for (int a = 0; a < 2 && e == cudaSuccess; ++a) {
                    const jp::Range rg = c.seg_io(m, a, sorted_io);
                    e = jp::launch_brick_finish(bs, acc, rg.first, rg.count, 0, rg.perm, rg.io_off, 0, p, st);
                }
            }
        JP_E(e);
    }
    float4 *q[2] = {nullptr, nullptr};
    if (!tiles && !bs) {
        JP_E(jp::lm_plan_quad(c.lm, 0, &q[0]));
        JP_E(jp::lm_plan_quad(c.lm, 1, &q[1]));
        JP_E(jp::launch_quad_build(img, c.g, q[0], q[1], st));
    }
    for (int a = 0; a < 2 && !bs; ++a)
        for (int m = 0; m < c.ns; ++m)
            if (subset < 0 || m == subset) {
                const jp::Range rg = c.seg_io(m, a, sorted_io);
                if (tiles)
                    JP_E(jp::launch_fwd_tof_lm_tile(c.l, c.tb, rg.first, rg.count, rg.perm, rg.io_off, img, c.g, c.t, p, 0, st));
                else
                    JP_E(jp::launch_fwd_tof_lm_quad(c.l, c.tb, rg, q[a], c.g, c.t, tc.lut, p, 0, st));
            }
    if (c.has_axis2(subset)) { // principal axis z: per-LOR kernels on the padded scalar image
        JP_E(jp::padded_create(img, c.g, false, st, &tc.pimg));
        for (int m = 0; m < c.ns; ++m)
            if (subset < 0 || m == subset)
                JP_E(jp::launch_fwd_tof_lm(c.l, c.tb, c.seg_io(m, 2, sorted_io), tc.pimg, c.g, c.t, tc.lut, p, 0, st));
    }
    return cudaSuccess;
}

cudaError_t lm_plan_back_tof(LmPlan *lm, int subset, const float *y, float *img, cudaStream_t st, bool sorted_io)
{
    jp_plan tmp;
    tmp.lm = lm;
    PlanCtx c(&tmp);
    TofCtx tc;
    tc.st = st;
    JP_E(jp::tof_lut_create(c.t, st, &tc.lut));
    const bool tiles = lm_tiles_wanted(c.lm, true);
    const jp::BrickSet *bs = nullptr;
    if (!tiles) JP_E(lm_bricks_wanted(c.lm, st, &bs));
    if (bs) JP_E(tc.g1_init(c.t)); // float adjoint of the brick forward projection: the same TOF table
    if (tiles) {
        for (int a = 0; a < 2; ++a)
            for (int m = 0; m < c.ns; ++m)
                if (subset < 0 || m == subset) {
                    const jp::Range rg = c.seg_io(m, a, sorted_io);
                    JP_E(jp::launch_back_tof_lm_tile(c.l, c.tb, rg.first, rg.count, rg.perm, rg.io_off, y, c.g, c.t, img, st));
                }
    } else {
        float4 *b[2];
        const size_t qbytes = sizeof(float4) * (size_t)jp::padded_voxels(c.g);
        for (int a = 0; a < 2; ++a) {
            JP_E(jp::lm_plan_quad(c.lm, 2 + a, &b[a]));
            JP_E(cudaMemsetAsync(b[a], 0, qbytes, st));
            for (int m = 0; m < c.ns; ++m)
                if (subset < 0 || m == subset)
                    JP_E(jp::launch_back_tof_lm_quad(c.l, c.tb, c.seg_io(m, a, sorted_io), y, c.g, c.t, tc.lut, b[a], st, 0,
                                                     tc.g1.tab ? &tc.g1 : nullptr));
        }
        JP_E(jp::launch_quad_merge(b[0], b[1], c.g, img, st));
    }
    if (c.has_axis2(subset)) {
        JP_E(jp::padded_create(nullptr, c.g, true, st, &tc.pimg));
        for (int m = 0; m < c.ns; ++m)
            if (subset < 0 || m == subset)
                JP_E(jp::launch_back_tof_lm(c.l, c.tb, c.seg_io(m, 2, sorted_io), y, c.g, c.t, tc.lut, tc.pimg, st));
        JP_E(jp::padded_add_to(tc.pimg, c.g, img, st));
    }
    return cudaSuccess;
}
#undef JP_E

} // namespace jp

extern "C" {

int jp_fwd_tof_lm_planned(const jp_plan *plan, int subset, const float *img, float *p, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!img || !p) return fail(JP_ERR_POINTER, "img or p is NULL");
    JP_CUDA(jp::lm_plan_fwd_tof(plan->lm, subset, img, p, (cudaStream_t)stream, false), "jp_fwd_tof_lm_planned");
    return JP_OK;
}

int jp_fwd_tof_lm_planned_sorted(const jp_plan *plan, int subset, const float *img, float *p_sorted, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!img || !p_sorted) return fail(JP_ERR_POINTER, "img or p is NULL");
    JP_CUDA(jp::lm_plan_fwd_tof(plan->lm, subset, img, p_sorted, (cudaStream_t)stream, true), "jp_fwd_tof_lm_planned_sorted");
    return JP_OK;
}

int jp_back_tof_lm_planned_sorted(const jp_plan *plan, int subset, const float *y_sorted, float *img, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!img || !y_sorted) return fail(JP_ERR_POINTER, "img or y is NULL");
    JP_CUDA(jp::lm_plan_back_tof(plan->lm, subset, y_sorted, img, (cudaStream_t)stream, true), "jp_back_tof_lm_planned_sorted");
    return JP_OK;
}

int jp_lm_plan_permute(const jp_plan *plan, const float *in, float *out, int to_plan_order, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!in || !out || in == out) return fail(JP_ERR_POINTER, "in / out is NULL, or in == out");
    JP_CUDA(jp::lm_plan_permute(plan->lm, in, out, to_plan_order != 0, (cudaStream_t)stream), "jp_lm_plan_permute");
    return JP_OK;
}

int jp_back_tof_lm_planned(const jp_plan *plan, int subset, const float *y, float *img, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!img || !y) return fail(JP_ERR_POINTER, "img or y is NULL");
    JP_CUDA(jp::lm_plan_back_tof(plan->lm, subset, y, img, (cudaStream_t)stream, false), "jp_back_tof_lm_planned");
    return JP_OK;
}

// ---- non-TOF listmode over the plan's sorted events ----------------------
int jp_fwd_lm_planned(const jp_plan *plan, int subset, const float *img, float *p, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!img || !p) return fail(JP_ERR_POINTER, "img or p is NULL");
    const char *where = "jp_fwd_lm_planned";
    cudaStream_t st = (cudaStream_t)stream;
    PlanCtx c(plan);
    const bool tiles = lm_tiles_wanted(c.lm, false);
    for (int a = 0; a < 3; ++a)
        for (int m = 0; m < c.ns; ++m)
            if (subset < 0 || m == subset) {
                const jp::Range rg = c.seg(m, a, false);
                cudaError_t e = cudaErrorNotSupported;
                if (tiles && a < 2)
                    e = jp::launch_fwd_tof_lm_tile(c.l, nullptr, rg.first, rg.count, rg.perm, 0, img, c.g, c.t, p, 0, st);
                if (e == cudaErrorNotSupported) e = jp::launch_fwd(c.l, rg, img, c.g, p, st);
                JP_CUDA(e, where);
            }
    return JP_OK;
}

int jp_back_lm_planned(const jp_plan *plan, int subset, const float *y, float *img, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    if (!img || !y) return fail(JP_ERR_POINTER, "img or y is NULL");
    const char *where = "jp_back_lm_planned";
    cudaStream_t st = (cudaStream_t)stream;
    PlanCtx c(plan);
    const bool tiles = lm_tiles_wanted(c.lm, false);
    for (int a = 0; a < 3; ++a)
        for (int m = 0; m < c.ns; ++m)
            if (subset < 0 || m == subset) {
                const jp::Range rg = c.seg(m, a, false);
                cudaError_t e = cudaErrorNotSupported;
                if (tiles && a < 2)
                    e = jp::launch_back_tof_lm_tile(c.l, nullptr, rg.first, rg.count, rg.perm, 0, y, c.g, c.t, img, st);
                if (e == cudaErrorNotSupported) e = jp::launch_back(c.l, rg, y, c.g, img, st);
                JP_CUDA(e, where);
            }
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

static int lm_osem_planned_impl(const jp_plan *plan, const float *sens, float *img, int n_iter, float res_sigma,
                                float res_nsig, void *workspace, size_t workspace_bytes, void *stream)
{
    g_err[0] = 0;
    const bool res = res_sigma > 0.f;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (n_iter < 0) return fail(JP_ERR_SIZE, "n_iter < 0");
    if (!sens || !img || !workspace) return fail(JP_ERR_POINTER, "NULL argument");
    if (workspace_bytes < jp_lm_osem_planned_workspace_bytes(plan)) return fail(JP_ERR_SIZE, "workspace too small");
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    const char *where = "jp_lm_osem_planned";
    cudaStream_t st = (cudaStream_t)stream;
    PlanCtx c(plan);
    const int64_t nvox = (int64_t)c.g.n[0] * c.g.n[1] * c.g.n[2];
    float *bz = (float *)workspace;              // image-sized accumulator of the principal-axis-z events
    float *r = bz + ((nvox + 31) / 32) * 32;     // per-event ratios of one subset, in sorted order
    TofCtx tc;
    tc.st = st;
    JP_CUDA(jp::tof_lut_create(c.t, st, &tc.lut), where);
    // bs: forward sums on the image bricks (the adjoint: float atomics on the quad accumulators either way)
    const jp::BrickSet *bs = nullptr;
    JP_CUDA(lm_bricks_wanted(c.lm, st, &bs), where);
    if (bs) JP_CUDA(tc.g1_init(c.t), where); // forward and adjoint must read the same TOF table (jp_quad.cu)
    float4 *q[2] = {nullptr, nullptr}, *b[2] = {nullptr, nullptr};
    const size_t qbytes = sizeof(float4) * (size_t)jp::padded_voxels(c.g);
    for (int a = 0; a < 2; ++a) {
        if (!bs) JP_CUDA(jp::lm_plan_quad(c.lm, a, &q[a]), where);
        JP_CUDA(jp::lm_plan_quad(c.lm, 2 + a, &b[a]), where);
    }
    const bool z_events = c.has_axis2(-1);
    if (z_events) JP_CUDA(cudaMemsetAsync(bz, 0, sizeof(float) * (size_t)nvox, st), where);
    // resolution model: xb = G x feeds the forward projection, G folds the back projection (stream-ordered scratch)
    struct Scratch {
        float *p = nullptr;
        cudaStream_t st = nullptr;
        ~Scratch() { if (p) cudaFreeAsync(p, st); }
    } sc;
    float *xb = nullptr, *bb = nullptr, *tmp = nullptr;
    if (res) {
        sc.st = st;
        JP_CUDA(cudaMallocAsync((void **)&sc.p, sizeof(float) * 3 * (size_t)nvox, st), where);
        xb = sc.p;
        bb = sc.p + nvox;
        tmp = sc.p + 2 * nvox;
    }
    // per subset: fwd (ratio fused) and back axis by axis on the quad arrays, then the multiplicative update
    for (int it = 0; it < n_iter; ++it) {
        for (int m = 0; m < c.ns; ++m) {
            const float *xin = img;
            if (res) {
                JP_CUDA(jp::launch_gauss3d(img, xb, tmp, c.g, res_sigma, res_nsig, st), where);
                xin = xb;
            }
            if (bs) { // bricks: forward sums per event; ratio + back projection with float atomics on the quad accumulators
                const jp::Range sub = c.subset(m);
                JP_CUDA(cudaMemsetAsync(r, 0, sizeof(float) * (size_t)sub.count, st), where);
                JP_CUDA(jp::launch_brick_fwd(bs, m, xin, c.g, c.t, sub.first, r, st, tc.g1.tab ? &tc.g1 : nullptr), where);
                for (int a = 0; a < 2; ++a) {
                    JP_CUDA(cudaMemsetAsync(b[a], 0, qbytes, st), where);
                    JP_CUDA(jp::launch_back_tof_lm_quad(c.l, c.tb, c.seg(m, a, true), r, c.g, c.t, tc.lut, b[a], st, 1, &tc.g1), where);
                }
            } else {
                JP_CUDA(jp::launch_quad_build(xin, c.g, q[0], q[1], st), where);
                for (int a = 0; a < 2; ++a) { // forward, ratio and back of the subset's events in one pass per axis
                    JP_CUDA(cudaMemsetAsync(b[a], 0, qbytes, st), where);
                    JP_CUDA(jp::launch_osem_tof_lm_quad(c.l, c.tb, c.seg(m, a, true), q[a], c.g, c.t, tc.lut, b[a], st), where);
                }
            }
            if (z_events) {
                float *px = nullptr, *pb = nullptr;
                JP_CUDA(jp::padded_create(xin, c.g, false, st, &px), where);
                cudaError_t e = jp::padded_create(nullptr, c.g, true, st, &pb);
                if (e == cudaSuccess) e = jp::launch_fwd_tof_lm(c.l, c.tb, c.seg(m, 2, true), px, c.g, c.t, tc.lut, r, 1, st);
                if (e == cudaSuccess) e = jp::launch_back_tof_lm(c.l, c.tb, c.seg(m, 2, true), r, c.g, c.t, tc.lut, pb, st);
                if (e == cudaSuccess) e = jp::padded_add_to(pb, c.g, bz, st);
                jp::padded_destroy(px, st);
                jp::padded_destroy(pb, st);
                JP_CUDA(e, where);
            }
            if (!res) {
                JP_CUDA(jp::launch_quad_osem_update(img, b[0], b[1], z_events ? bz : nullptr, sens, (float)c.ns, c.g, st), where);
            } else {
                JP_CUDA(cudaMemsetAsync(bb, 0, sizeof(float) * (size_t)nvox, st), where);
                JP_CUDA(jp::launch_quad_merge(b[0], b[1], c.g, bb, st), where);
                if (z_events) JP_CUDA(jp::launch_add_clear(bb, bz, nvox, st), where);
                JP_CUDA(jp::launch_gauss3d(bb, bb, tmp, c.g, res_sigma, res_nsig, st), where);
                JP_CUDA(jp::launch_osem_update(img, bb, sens, (float)c.ns, nvox, st), where);
            }
        }
    }
    return JP_OK;
}

int jp_lm_osem_planned(const jp_plan *plan, const float *sens, float *img, int n_iter, void *workspace,
                       size_t workspace_bytes, void *stream)
{
    return lm_osem_planned_impl(plan, sens, img, n_iter, 0.f, 0.f, workspace, workspace_bytes, stream);
}

int jp_lm_osem_planned_res(const jp_plan *plan, const float *sens, float *img, int n_iter, float res_sigma_mm,
                           float res_n_sigmas, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!(res_sigma_mm > 0.f) || !(res_n_sigmas > 0.f)) return fail(JP_ERR_SIZE, "res_sigma_mm <= 0 or res_n_sigmas <= 0");
    return lm_osem_planned_impl(plan, sens, img, n_iter, res_sigma_mm, res_n_sigmas, workspace, workspace_bytes, stream);
}

int jp_gauss3d(const float *in, float *out, const jp_geom *geom, float sigma_mm, float n_sigmas, void *stream)
{
    g_err[0] = 0;
    jp::Geom g;
    JP_TRY(check_geom(geom, g));
    if (!in || !out) return fail(JP_ERR_POINTER, "in or out is NULL");
    if (!(sigma_mm > 0.f) || !(n_sigmas > 0.f)) return fail(JP_ERR_SIZE, "sigma_mm <= 0 or n_sigmas <= 0");
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    float *tmp = nullptr;
    JP_CUDA(cudaMallocAsync((void **)&tmp, sizeof(float) * (size_t)nvox, st), "jp_gauss3d (scratch)");
    const cudaError_t e = jp::launch_gauss3d(in, out, tmp, g, sigma_mm, n_sigmas, st);
    cudaFreeAsync(tmp, st);
    if (e == cudaErrorInvalidValue) return fail(JP_ERR_SIZE, "Gaussian kernel radius > 16 voxels");
    JP_CUDA(e, "jp_gauss3d");
    return JP_OK;
}

// ---- TOF sinogram OSEM -------------------------------------------------------------------
static int check_subsets(const int64_t *off, int n_subsets, int64_t n, int64_t *max_count)
{
    if (!off) return fail(JP_ERR_POINTER, "subset_offsets is NULL");
    if (n_subsets < 1) return fail(JP_ERR_SIZE, "n_subsets < 1");
    int64_t mx = 0;
    if (off[0] < 0 || off[n_subsets] > n) return fail(JP_ERR_SIZE, "subset_offsets outside [0, n]");
    for (int m = 0; m < n_subsets; ++m) {
        if (off[m + 1] < off[m]) return fail(JP_ERR_SIZE, "subset_offsets not non-decreasing");
        if (off[m + 1] - off[m] > mx) mx = off[m + 1] - off[m];
    }
    *max_count = mx;
    return JP_OK;
}

static jp::Lors lors_at(const jp::Lors &l, int64_t a)
{
    return jp::Lors{l.xs + a, l.ys + a, l.zs + a, l.xe + a, l.ye + a, l.ze + a};
}

size_t jp_sino_osem_tof_workspace_bytes(const int64_t *subset_offsets, int n_subsets, int64_t n, const jp_tof *tof)
{
    int64_t mx = 0;
    if (!tof || tof->n_tofbins < 1 || check_subsets(subset_offsets, n_subsets, n, &mx) != JP_OK) return 0;
    return (size_t)(mx * tof->n_tofbins + 64) * sizeof(float);
}

static int sino_sens_impl(const jp::Lors &l, const int64_t *subset_offsets, int n_subsets, const float *mult,
                          const jp::Geom &g, const jp::Tof &t, float *sens, void *workspace, size_t workspace_bytes,
                          cudaStream_t st)
{
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    JP_CUDA(cudaMemsetAsync(sens, 0, sizeof(float) * (size_t)nvox * n_subsets, st), "jp_sino_sens_tof (zero)");
    TofCtx c;
    JP_TRY(tof_ctx_init(c, t, g, nullptr, 1, st, "jp_sino_sens_tof (scratch)"));
    jp::SinoEpi epi;
    epi.mult_bcast = mult;
    epi.ones_bcast = mult ? 0 : 1;
    for (int m = 0; m < n_subsets; ++m) {
        const int64_t a = subset_offsets[m], cnt = subset_offsets[m + 1] - a;
        if (cnt == 0) continue;
        jp::SinoEpi e = epi;
        if (mult) e.mult_bcast = mult + a;
        cudaError_t rc = jp::launch_tof_sino_win(true, lors_at(l, a), cnt, nullptr, c.pimg, g, t, nullptr, nullptr, st, &e);
        if (rc == cudaErrorNotSupported) { // generic kernels: expand mult over the bins in the workspace first
            if (!workspace || workspace_bytes < (size_t)(cnt * t.nbins) * sizeof(float))
                return fail(JP_ERR_SIZE, "jp_sino_sens_tof: workspace needed (TOF window wider than the fused kernels)");
            float *r = (float *)workspace;
            rc = jp::launch_sino_bcast(r, mult ? mult + a : nullptr, cnt, t.nbins, st);
            if (rc == cudaSuccess) rc = jp::launch_back_tof_sino(lors_at(l, a), whole(cnt), r, g, t, c.lut, c.pimg, st);
        }
        JP_CUDA(rc, "jp_sino_sens_tof");
        JP_CUDA(jp::padded_add_to(c.pimg, g, sens + (size_t)m * nvox, st), "jp_sino_sens_tof (unpad)");
        JP_CUDA(cudaMemsetAsync(c.pimg, 0, sizeof(float) * (size_t)jp::padded_voxels(g), st), "jp_sino_sens_tof (clear)");
    }
    return JP_OK;
}

static int sino_osem_impl(const jp::Lors &l, const int64_t *subset_offsets, int n_subsets, const float *y,
                          const float *mult, const float *contam, const float *sens, const jp::Geom &g, const jp::Tof &t,
                          float *img, int n_iter, void *workspace, cudaStream_t st)
{
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    const int nb = t.nbins;
    float *r = (float *)workspace;
    TofCtx cx, cb; // cx.pimg = padded x, cb.pimg = padded b
    JP_TRY(tof_ctx_init(cx, t, g, img, 0, st, "jp_sino_osem_tof (scratch)"));
    cb.st = st;
    JP_CUDA(jp::padded_create(nullptr, g, true, st, &cb.pimg), "jp_sino_osem_tof (scratch)");
    for (int it = 0; it < n_iter; ++it) {
        for (int m = 0; m < n_subsets; ++m) {
            const int64_t a = subset_offsets[m], cnt = subset_offsets[m + 1] - a;
            if (cnt > 0) {
                const jp::Lors ls = lors_at(l, a);
                jp::SinoEpi e;
                e.y_em = y + (size_t)a * nb;
                e.mult = mult ? mult + a : nullptr;
                e.contam = contam ? contam + (size_t)a * nb : nullptr;
                // one fused pass (forward, ratio, back); the unfused generic kernels when the TOF window is too wide
                cudaError_t rc = jp::launch_tof_sino_osem(ls, cnt, cx.pimg, cb.pimg, g, t, e, st);
                if (rc == cudaErrorNotSupported) {
                    rc = jp::launch_fwd_tof_sino(ls, whole(cnt), cx.pimg, g, t, cx.lut, r, st);
                    if (rc == cudaSuccess) rc = jp::launch_sino_ratio(r, e.y_em, e.mult, e.contam, cnt, nb, st);
                    if (rc == cudaSuccess) rc = jp::launch_back_tof_sino(ls, whole(cnt), r, g, t, cx.lut, cb.pimg, st);
                }
                JP_CUDA(rc, "jp_sino_osem_tof (subset pass)");
            }
            JP_CUDA(jp::launch_osem_update_padded(img, cx.pimg, cb.pimg, sens + (size_t)m * nvox, 1.f, g, st),
                    "jp_sino_osem_tof (update)");
        }
    }
    return JP_OK;
}

int jp_sino_sens_tof(const jp_lors *lors, const int64_t *subset_offsets, int n_subsets, const float *mult,
                     const jp_geom *geom, const jp_tof *tof, float *sens, void *workspace, size_t workspace_bytes,
                     void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    int64_t mx = 0;
    JP_TRY(check_subsets(subset_offsets, n_subsets, lors->n, &mx));
    if (!sens) return fail(JP_ERR_POINTER, "sens is NULL");
    return sino_sens_impl(l, subset_offsets, n_subsets, mult, g, t, sens, workspace, workspace_bytes, (cudaStream_t)stream);
}

int jp_sino_osem_tof(const jp_lors *lors, const int64_t *subset_offsets, int n_subsets, const float *y,
                     const float *mult, const float *contam, const float *sens, const jp_geom *geom, const jp_tof *tof,
                     float *img, int n_iter, void *workspace, size_t workspace_bytes, void *stream)
{
    g_err[0] = 0;
    jp::Lors l;
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_lors(lors, l));
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    int64_t mx = 0;
    JP_TRY(check_subsets(subset_offsets, n_subsets, lors->n, &mx));
    if (n_iter < 0) return fail(JP_ERR_SIZE, "n_iter < 0");
    if (!sens || !img || !workspace || (lors->n > 0 && !y)) return fail(JP_ERR_POINTER, "NULL argument");
    if (workspace_bytes < jp_sino_osem_tof_workspace_bytes(subset_offsets, n_subsets, lors->n, tof))
        return fail(JP_ERR_SIZE, "workspace too small");
    return sino_osem_impl(l, subset_offsets, n_subsets, y, mult, contam, sens, g, t, img, n_iter, workspace,
                          (cudaStream_t)stream);
}

// ---- sinogram plan and the planned TOF sinogram calls (jp_sino_plan.cu, jp_tof_sino_tile.cu) ---------------------------
int jp_sino_plan_create(const jp_lors *lors, void *stream, jp_plan **plan)
{
    g_err[0] = 0;
    jp::Lors l;
    JP_TRY(check_lors(lors, l));
    if (!plan) return fail(JP_ERR_POINTER, "plan is NULL");
    *plan = nullptr;
    jp::SinoPlan *sp = nullptr;
    JP_CUDA(jp::sino_plan_create(l, lors->n, (cudaStream_t)stream, &sp), "jp_sino_plan_create");
    jp_plan *pl = new jp_plan;
    pl->sino = sp;
    *plan = pl;
    return JP_OK;
}

int jp_sino_plan_info(const jp_plan *plan, int64_t *n_lors, int64_t *n_tracks, int32_t *track_length)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    if (n_lors) *n_lors = v.n;
    if (n_tracks) *n_tracks = v.regular ? v.K : 0;
    if (track_length) *track_length = v.regular ? v.T : 0;
    return JP_OK;
}

namespace {

// the LOR list of a sinogram plan as arrays: the plan's own copy (irregular) or stream-ordered scratch filled from the
// track table and the axial pattern (regular plans on a path that needs per-LOR arrays)
struct PlanLors {
    jp::Lors l{};
    float *scratch = nullptr;
    cudaStream_t st = nullptr;
    ~PlanLors() { if (scratch) cudaFreeAsync(scratch, st); }
    cudaError_t init(const jp::SinoPlanView &v, cudaStream_t s)
    {
        st = s;
        if (!v.regular) {
            l = v.lors;
            return cudaSuccess;
        }
        cudaError_t e = cudaMallocAsync((void **)&scratch, sizeof(float) * 6 * (size_t)v.n, s);
        if (e != cudaSuccess) return e;
        return jp::sino_plan_expand(v, 0, v.n, scratch, s, &l);
    }
};

// subsets of a regular plan must consist of whole tracks for the tile kernels
bool subsets_on_tracks(const int64_t *off, int n_subsets, int T)
{
    for (int m = 0; m <= n_subsets; ++m)
        if (off[m] % T) return false;
    return true;
}

} // namespace

// non-TOF projections of a sinogram plan's LORs: per-track tiles read the track table and the axial pattern only
int jp_fwd_planned(const jp_plan *plan, const float *img, const jp_geom *geom, float *p, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    jp::Geom g;
    JP_TRY(check_geom(geom, g));
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    if (!img || (v.n > 0 && !p)) return fail(JP_ERR_POINTER, "img or p is NULL");
    if (v.n == 0) return JP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if (v.regular) {
        const cudaError_t e = jp::launch_fwd_tile(jp::Lors{}, v.n, img, g, p, st, &v);
        if (e != cudaErrorNotSupported) {
            JP_CUDA(e, "jp_fwd_planned");
            return JP_OK;
        }
    }
    PlanLors pl;
    JP_CUDA(pl.init(v, st), "jp_fwd_planned (LOR list)");
    JP_CUDA(jp::launch_fwd_tile(pl.l, v.n, img, g, p, st), "jp_fwd_planned");
    return JP_OK;
}

int jp_back_planned(const jp_plan *plan, const float *y, const jp_geom *geom, float *img, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    jp::Geom g;
    JP_TRY(check_geom(geom, g));
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    if (!img || (v.n > 0 && !y)) return fail(JP_ERR_POINTER, "img or y is NULL");
    if (v.n == 0) return JP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if (v.regular) {
        const cudaError_t e = jp::launch_back_tile(jp::Lors{}, v.n, y, g, img, st, &v);
        if (e != cudaErrorNotSupported) {
            JP_CUDA(e, "jp_back_planned");
            return JP_OK;
        }
    }
    PlanLors pl;
    JP_CUDA(pl.init(v, st), "jp_back_planned (LOR list)");
    JP_CUDA(jp::launch_back_tile(pl.l, v.n, y, g, img, st), "jp_back_planned");
    return JP_OK;
}

int jp_fwd_tof_sino_planned(const jp_plan *plan, const float *img, const jp_geom *geom, const jp_tof *tof, float *p,
                            void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    if (!img || (v.n > 0 && !p)) return fail(JP_ERR_POINTER, "img or p is NULL");
    if (v.n == 0) return JP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if (v.regular) {
        const cudaError_t e = jp::launch_tof_sino_tile(0, v, 0, v.K, img, nullptr, g, t, p, nullptr, nullptr, st);
        if (e != cudaErrorNotSupported) {
            JP_CUDA(e, "jp_fwd_tof_sino_planned");
            return JP_OK;
        }
    }
    PlanLors pl;
    JP_CUDA(pl.init(v, st), "jp_fwd_tof_sino_planned (LOR list)");
    return sino_fwd_impl(pl.l, v.n, img, g, t, p, st);
}

int jp_back_tof_sino_planned(const jp_plan *plan, const float *y, const jp_geom *geom, const jp_tof *tof, float *img,
                             void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    if (!img || (v.n > 0 && !y)) return fail(JP_ERR_POINTER, "img or y is NULL");
    if (v.n == 0) return JP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if (v.regular) {
        const cudaError_t e = jp::launch_tof_sino_tile(1, v, 0, v.K, nullptr, img, g, t, nullptr, y, nullptr, st);
        if (e != cudaErrorNotSupported) {
            JP_CUDA(e, "jp_back_tof_sino_planned");
            return JP_OK;
        }
    }
    PlanLors pl;
    JP_CUDA(pl.init(v, st), "jp_back_tof_sino_planned (LOR list)");
    return sino_back_impl(pl.l, v.n, y, g, t, img, st);
}

int jp_sino_sens_tof_planned(const jp_plan *plan, const int64_t *subset_offsets, int n_subsets, const float *mult,
                             const jp_geom *geom, const jp_tof *tof, float *sens, void *workspace, size_t workspace_bytes,
                             void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    int64_t mx = 0;
    JP_TRY(check_subsets(subset_offsets, n_subsets, v.n, &mx));
    if (!sens) return fail(JP_ERR_POINTER, "sens is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    if (v.regular && subsets_on_tracks(subset_offsets, n_subsets, v.T)) {
        JP_CUDA(cudaMemsetAsync(sens, 0, sizeof(float) * (size_t)nvox * n_subsets, st), "jp_sino_sens_tof_planned (zero)");
        jp::SinoEpi epi;
        epi.mult_bcast = mult;
        epi.ones_bcast = mult ? 0 : 1;
        cudaError_t e = cudaSuccess;
        for (int m = 0; m < n_subsets && e == cudaSuccess; ++m) {
            const int64_t k0 = subset_offsets[m] / v.T, nk = subset_offsets[m + 1] / v.T - k0;
            e = jp::launch_tof_sino_tile(1, v, k0, nk, nullptr, sens + (size_t)m * nvox, g, t, nullptr, nullptr, &epi, st);
        }
        if (e != cudaErrorNotSupported) {
            JP_CUDA(e, "jp_sino_sens_tof_planned");
            return JP_OK;
        }
    }
    PlanLors pl;
    JP_CUDA(pl.init(v, st), "jp_sino_sens_tof_planned (LOR list)");
    return sino_sens_impl(pl.l, subset_offsets, n_subsets, mult, g, t, sens, workspace, workspace_bytes, st);
}

int jp_sino_osem_tof_planned(const jp_plan *plan, const int64_t *subset_offsets, int n_subsets, const float *y,
                             const float *mult, const float *contam, const float *sens, const jp_geom *geom,
                             const jp_tof *tof, float *img, int n_iter, void *workspace, size_t workspace_bytes, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->sino) return fail(JP_ERR_PLAN, "not a sinogram plan");
    jp::Geom g;
    jp::Tof t;
    JP_TRY(check_geom(geom, g));
    JP_TRY(check_tof(tof, true, t));
    const jp::SinoPlanView v = jp::sino_plan_view(plan->sino);
    int64_t mx = 0;
    JP_TRY(check_subsets(subset_offsets, n_subsets, v.n, &mx));
    if (n_iter < 0) return fail(JP_ERR_SIZE, "n_iter < 0");
    if (!sens || !img || !workspace || (v.n > 0 && !y)) return fail(JP_ERR_POINTER, "NULL argument");
    if (workspace_bytes < jp_sino_osem_tof_workspace_bytes(subset_offsets, n_subsets, v.n, tof))
        return fail(JP_ERR_SIZE, "workspace too small");
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    double R;
    jp::Tof tt = t;
    if (v.regular && subsets_on_tracks(subset_offsets, n_subsets, v.T) && jp::tof_window_bins(tt, &R) > 0) {
        // per subset: ONE fused kernel on the unpadded images (forward, ratio, back), then the multiplicative update
        struct Scratch {
            float *p = nullptr;
            cudaStream_t st = nullptr;
            ~Scratch() { if (p) cudaFreeAsync(p, st); }
        } b;
        b.st = st;
        JP_CUDA(cudaMallocAsync((void **)&b.p, sizeof(float) * (size_t)nvox, st), "jp_sino_osem_tof_planned (scratch)");
        JP_CUDA(cudaMemsetAsync(b.p, 0, sizeof(float) * (size_t)nvox, st), "jp_sino_osem_tof_planned (scratch)");
        jp::SinoEpi epi;
        epi.y_em = y;
        epi.mult = mult;
        epi.contam = contam;
        // launch_tof_sino_tile decides "not supported" on its first NON-EMPTY subset (an empty one returns at once).
        // Until then only updates of empty subsets have been enqueued (x <- x 0 / sens = 0, which the unplanned
        // path repeats with the same result), so the fall-back may still start over from subset 0.
        bool unsupported = false, launched = false;
        for (int it = 0; it < n_iter && !unsupported; ++it) {
            for (int m = 0; m < n_subsets; ++m) {
                const int64_t k0 = subset_offsets[m] / v.T, nk = subset_offsets[m + 1] / v.T - k0;
                const cudaError_t e = jp::launch_tof_sino_tile(2, v, k0, nk, img, b.p, g, t, nullptr, nullptr, &epi, st);
                if (e == cudaErrorNotSupported && !launched) { // no projection enqueued yet: take the unplanned path
                    unsupported = true;
                    break;
                }
                if (nk > 0) launched = true;
                JP_CUDA(e, "jp_sino_osem_tof_planned (subset pass)");
                JP_CUDA(jp::launch_osem_update(img, b.p, sens + (size_t)m * nvox, 1.f, nvox, st),
                        "jp_sino_osem_tof_planned (update)");
            }
        }
        if (!unsupported) return JP_OK;
    }
    PlanLors pl;
    JP_CUDA(pl.init(v, st), "jp_sino_osem_tof_planned (LOR list)");
    return sino_osem_impl(pl.l, subset_offsets, n_subsets, y, mult, contam, sens, g, t, img, n_iter, workspace, st);
}

// ---- pieces of one OSEM subset update, for callers that exchange b between the two halves (multi-GPU) ----------
int jp_lm_osem_planned_backratio(const jp_plan *plan, int subset, const float *x, float *b, void *workspace,
                                 size_t workspace_bytes, void *stream)
{
    g_err[0] = 0;
    if (!plan || !plan->lm) return fail(JP_ERR_PLAN, "invalid plan");
    if (subset < 0 || subset >= jp::lm_plan_subsets(plan->lm)) return fail(JP_ERR_SIZE, "subset out of range");
    if (!x || !b || !workspace) return fail(JP_ERR_POINTER, "NULL argument");
    if (workspace_bytes < jp_lm_osem_planned_workspace_bytes(plan)) return fail(JP_ERR_SIZE, "workspace too small");
    const char *where = "jp_lm_osem_planned_backratio";
    cudaStream_t st = (cudaStream_t)stream;
    PlanCtx c(plan);
    const int64_t nvox = (int64_t)c.g.n[0] * c.g.n[1] * c.g.n[2];
    JP_CUDA(cudaMemsetAsync(b, 0, sizeof(float) * (size_t)nvox, st), where);
    if (jp::lm_plan_n(plan->lm) == 0) return JP_OK;
    float *r = (float *)workspace + ((nvox + 31) / 32) * 32; // per-event ratios of the subset, in sorted order
    TofCtx tc;
    tc.st = st;
    JP_CUDA(jp::tof_lut_create(c.t, st, &tc.lut), where);
    const int m = subset;
    const jp::BrickSet *bs = nullptr;
    JP_CUDA(lm_bricks_wanted(c.lm, st, &bs), where);
    if (bs) {
        const jp::Range sub = c.subset(m);
        JP_CUDA(cudaMemsetAsync(r, 0, sizeof(float) * (size_t)sub.count, st), where);
        JP_CUDA(jp::launch_brick_fwd(bs, m, x, c.g, c.t, sub.first, r, st), where);
    }
    if (bs) {
        JP_CUDA(tc.g1_init(c.t), where);
        float4 *qb[2];
        const size_t qbytes = sizeof(float4) * (size_t)jp::padded_voxels(c.g);
        for (int a = 0; a < 2; ++a) {
            JP_CUDA(jp::lm_plan_quad(c.lm, 2 + a, &qb[a]), where);
            JP_CUDA(cudaMemsetAsync(qb[a], 0, qbytes, st), where);
            JP_CUDA(jp::launch_back_tof_lm_quad(c.l, c.tb, c.seg(m, a, true), r, c.g, c.t, tc.lut, qb[a], st, 1, &tc.g1), where);
        }
        JP_CUDA(jp::launch_quad_merge(qb[0], qb[1], c.g, b, st), where);
    } else {
        float4 *q[2], *qb[2];
        const size_t qbytes = sizeof(float4) * (size_t)jp::padded_voxels(c.g);
        for (int a = 0; a < 2; ++a) {
            JP_CUDA(jp::lm_plan_quad(c.lm, a, &q[a]), where);
            JP_CUDA(jp::lm_plan_quad(c.lm, 2 + a, &qb[a]), where);
        }
        JP_CUDA(jp::launch_quad_build(x, c.g, q[0], q[1], st), where);
        for (int a = 0; a < 2; ++a) {
            JP_CUDA(cudaMemsetAsync(qb[a], 0, qbytes, st), where);
            JP_CUDA(jp::launch_osem_tof_lm_quad(c.l, c.tb, c.seg(m, a, true), q[a], c.g, c.t, tc.lut, qb[a], st), where);
        }
        JP_CUDA(jp::launch_quad_merge(qb[0], qb[1], c.g, b, st), where);
    }
    if (c.has_axis2(m)) {
        float *px = nullptr, *pb = nullptr;
        JP_CUDA(jp::padded_create(x, c.g, false, st, &px), where);
        cudaError_t e = jp::padded_create(nullptr, c.g, true, st, &pb);
        if (e == cudaSuccess) e = jp::launch_fwd_tof_lm(c.l, c.tb, c.seg(m, 2, true), px, c.g, c.t, tc.lut, r, 1, st);
        if (e == cudaSuccess) e = jp::launch_back_tof_lm(c.l, c.tb, c.seg(m, 2, true), r, c.g, c.t, tc.lut, pb, st);
        if (e == cudaSuccess) e = jp::padded_add_to(pb, c.g, b, st);
        jp::padded_destroy(px, st);
        jp::padded_destroy(pb, st);
        JP_CUDA(e, where);
    }
    return JP_OK;
}

int jp_osem_update(float *x, float *b, const float *sens, float scale, const jp_geom *geom, void *stream)
{
    g_err[0] = 0;
    jp::Geom g;
    JP_TRY(check_geom(geom, g));
    if (!x || !b || !sens) return fail(JP_ERR_POINTER, "NULL argument");
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    JP_CUDA(jp::launch_osem_update(x, b, sens, scale, nvox, (cudaStream_t)stream), "jp_osem_update");
    return JP_OK;
}

} // extern "C"
