// jp_host.cu -- "hybrid" mode: HOST buffers in, HOST buffers out, over ALL visible GPUs ("hybrid
// CPU/GPU mode": "data transfer from the host to all available GPUs, execution of projection kernels on the GPUs, and
// transfer of the results back"; the projections split naturally over LOR chunks).
//
// A jp_hybrid handle owns one WORKER per device it was created over: a host thread per call and worker, two CUDA
// streams, and device buffers that are kept between calls (the LOR shard, per-LOR values, two images; grown on demand,
// freed with the handle).  jp_hybrid_set_lors splits the host LOR list into contiguous shards -- cut at multiples of
// the list's track length when it has one, so that every shard is a regular sinogram (jp_sino_plan.cu) -- uploads
// each shard ONCE and builds the shard's plan (sinogram plan; listmode plan when TOF bins are given).  The projection
// calls then move only what changes: the image (to every GPU), the per-LOR values of each shard, the results back.
// Forward results are disjoint (no exchange).  A back projection leaves one partial image per worker; they are copied
// to pinned host memory and added on the host in worker order (n_workers x 15 MB: nothing next to the PCIe time of
// the values), then accumulated into the caller's image.  A device may be listed more than once (several workers on
// one GPU): that is how the single-GPU tests exercise the fan-out and the summation.
//
// The one-shot jp_*_host calls of round 1 are kept: each makes a handle over all visible devices, sets the list, runs
// and destroys it (they allocate and synchronise by their nature; callers that project a list more than once use the
// handle).
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <thread>
#include <vector>

#include "../../include/joseph_b200.h"
#include "jp_internal.h"

struct jp_plan; // the C-ABI handle type (jp_api.cu); not used here

namespace {

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
        const cudaError_t e = cudaMalloc(&p, bytes);
        if (e == cudaSuccess) cap = bytes;
        return e;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
};

struct Worker {
    int dev = 0;
    cudaStream_t st = nullptr;
    int64_t lo = 0, hi = 0; // shard [lo, hi) of the list
    DevBuf coord, tb, val, img, img2;
    float *host_img = nullptr; // pinned, partial back projection of this worker
    size_t host_img_cap = 0;
    jp::SinoPlan *sp = nullptr;
    jp::LmPlan *lp = nullptr;
    cudaError_t err = cudaSuccess;
    const char *where = "";
};

} // namespace

struct jp_hybrid {
    std::vector<Worker> w;
    int64_t n = 0;
    bool have_lors = false, have_tb = false;
    jp::Geom g_lm{};
    jp::Tof t_lm{};
};

namespace {

int hfail(int code, const char *msg)
{
    snprintf(jp::err_buf(), 512, "%s", msg);
    return code;
}

bool geom_ok(const jp_geom *g, jp::Geom &out, int64_t &nvox)
{
    if (!g) return false;
    nvox = 1;
    for (int a = 0; a < 3; ++a) {
        if (g->n[a] <= 0 || !(g->voxsize[a] > 0.f)) return false;
        out.n[a] = g->n[a];
        out.o[a] = g->origin[a];
        out.v[a] = g->voxsize[a];
        nvox *= g->n[a];
    }
    return nvox < ((int64_t)1 << 31);
}

bool tof_ok(const jp_tof *t, bool sino, jp::Tof &out)
{
    if (!t || !(t->tofbin_width_mm > 0.f) || !(t->sigma_tof_mm > 0.f) || !(t->n_sigmas > 0.f)) return false;
    if (sino && (t->n_tofbins < 1 || t->n_tofbins > JP_MAX_TOFBINS)) return false;
    out.width = t->tofbin_width_mm;
    out.sigma = t->sigma_tof_mm;
    out.nsig = t->n_sigmas;
    out.nbins = t->n_tofbins;
    out.coff = t->center_offset_mm;
    return true;
}

// run f(worker) on every worker of h, each in its own host thread bound to the worker's device; first error wins
template <typename F>
int run_all(jp_hybrid *h, F f, const char *where)
{
    std::vector<std::thread> th;
    th.reserve(h->w.size());
    for (Worker &wk : h->w)
        th.emplace_back([&wk, &f, where]() {
            wk.err = cudaSetDevice(wk.dev);
            wk.where = where;
            if (wk.err == cudaSuccess) wk.err = f(wk);
            if (wk.err == cudaSuccess) wk.err = cudaStreamSynchronize(wk.st);
        });
    for (std::thread &t : th) t.join();
    for (Worker &wk : h->w)
        if (wk.err != cudaSuccess) {
            snprintf(jp::err_buf(), 512, "%s (device %d): %s", where, wk.dev, cudaGetErrorString(wk.err));
            return JP_ERR_CUDA;
        }
    return JP_OK;
}

void drop_plans(Worker &wk)
{
    if (wk.sp) jp::sino_plan_destroy(wk.sp);
    if (wk.lp) jp::lm_plan_destroy(wk.lp);
    wk.sp = nullptr;
    wk.lp = nullptr;
}

// length of the first run of LORs with identical transaxial end points (0: none within the probe limit)
int64_t host_track_length(const jp_lors *l)
{
    const int64_t lim = std::min<int64_t>(l->n, 1 << 16);
    for (int64_t j = 1; j < lim; ++j)
        if (memcmp(l->xs + j, l->xs, 4) || memcmp(l->ys + j, l->ys, 4) || memcmp(l->xe + j, l->xe, 4) || memcmp(l->ye + j, l->ye, 4))
            return j;
    return l->n <= lim ? l->n : 0;
}

jp::Lors shard_lors(const Worker &wk)
{
    const int64_t m = wk.hi - wk.lo;
    float *c = (float *)wk.coord.p;
    return jp::Lors{c, c + m, c + 2 * m, c + 3 * m, c + 4 * m, c + 5 * m};
}

cudaError_t upload_image(Worker &wk, const float *img_host, int64_t nvox)
{
    cudaError_t e = wk.img.ensure(sizeof(float) * (size_t)nvox);
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(wk.img.p, img_host, sizeof(float) * (size_t)nvox, cudaMemcpyHostToDevice, wk.st);
}

cudaError_t zero_partial(Worker &wk, int64_t nvox)
{
    cudaError_t e = wk.img2.ensure(sizeof(float) * (size_t)nvox);
    if (e != cudaSuccess) return e;
    if (wk.host_img_cap < (size_t)nvox) {
        if (wk.host_img) cudaFreeHost(wk.host_img);
        wk.host_img = nullptr;
        wk.host_img_cap = 0;
        if ((e = cudaMallocHost((void **)&wk.host_img, sizeof(float) * (size_t)nvox)) != cudaSuccess) return e;
        wk.host_img_cap = (size_t)nvox;
    }
    return cudaMemsetAsync(wk.img2.p, 0, sizeof(float) * (size_t)nvox, wk.st);
}

cudaError_t download_partial(Worker &wk, int64_t nvox)
{
    return cudaMemcpyAsync(wk.host_img, wk.img2.p, sizeof(float) * (size_t)nvox, cudaMemcpyDeviceToHost, wk.st);
}

// img_host += sum of the workers' partial images, in worker order (deterministic for a given set of workers)
void add_partials(jp_hybrid *h, int64_t nvox, float *img_host)
{
    for (Worker &wk : h->w) {
        if (wk.hi <= wk.lo) continue;
        const float *src = wk.host_img;
        for (int64_t i = 0; i < nvox; ++i) img_host[i] += src[i];
    }
}

int check_ready(const jp_hybrid *h, bool need_tb)
{
    if (!h) return hfail(JP_ERR_PLAN, "hybrid handle is NULL");
    if (!h->have_lors) return hfail(JP_ERR_PLAN, "jp_hybrid_set_lors has not been called");
    if (need_tb && !h->have_tb) return hfail(JP_ERR_PLAN, "the handle's LOR list was set without TOF bins");
    return JP_OK;
}

} // namespace

extern "C" {

int jp_hybrid_create(const int *devices, int n_devices, jp_hybrid **out)
{
    jp::err_buf()[0] = 0;
    if (!out) return JP_ERR_POINTER;
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) return hfail(JP_ERR_CUDA, "jp_hybrid_create: no CUDA device");
    std::vector<int> devs;
    if (devices) {
        if (n_devices < 1) return hfail(JP_ERR_SIZE, "jp_hybrid_create: n_devices < 1");
        for (int i = 0; i < n_devices; ++i) {
            if (devices[i] < 0 || devices[i] >= ndev) return hfail(JP_ERR_SIZE, "jp_hybrid_create: device ordinal out of range");
            devs.push_back(devices[i]);
        }
    } else {
        for (int i = 0; i < ndev; ++i) devs.push_back(i);
    }
    int cur = 0;
    cudaGetDevice(&cur);
    jp_hybrid *h = new jp_hybrid;
    h->w.resize(devs.size());
    for (size_t i = 0; i < devs.size() && e == cudaSuccess; ++i) {
        h->w[i].dev = devs[i];
        e = cudaSetDevice(devs[i]);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->w[i].st, cudaStreamNonBlocking);
    }
    cudaSetDevice(cur);
    if (e != cudaSuccess) {
        snprintf(jp::err_buf(), 512, "jp_hybrid_create: %s", cudaGetErrorString(e));
        jp_hybrid_destroy(h);
        return JP_ERR_CUDA;
    }
    *out = h;
    return JP_OK;
}

int jp_hybrid_destroy(jp_hybrid *h)
{
    if (!h) return JP_OK;
    int cur = 0;
    cudaGetDevice(&cur);
    for (Worker &wk : h->w) {
        cudaSetDevice(wk.dev);
        if (wk.st) cudaStreamSynchronize(wk.st);
        drop_plans(wk);
        wk.coord.release();
        wk.tb.release();
        wk.val.release();
        wk.img.release();
        wk.img2.release();
        if (wk.host_img) cudaFreeHost(wk.host_img);
        if (wk.st) cudaStreamDestroy(wk.st);
    }
    cudaSetDevice(cur);
    delete h;
    return JP_OK;
}

int jp_hybrid_worker_count(const jp_hybrid *h) { return h ? (int)h->w.size() : -1; }

int jp_hybrid_set_lors(jp_hybrid *h, const jp_lors *lors_host, const int16_t *tofbin_host, const jp_geom *geom,
                       const jp_tof *tof)
{
    jp::err_buf()[0] = 0;
    if (!h) return hfail(JP_ERR_PLAN, "hybrid handle is NULL");
    if (!lors_host) return JP_ERR_POINTER;
    const int64_t n = lors_host->n;
    if (n < 0) return JP_ERR_SIZE;
    if (n > 0 && (!lors_host->xs || !lors_host->ys || !lors_host->zs || !lors_host->xe || !lors_host->ye || !lors_host->ze))
        return JP_ERR_POINTER;
    jp::Geom g{};
    jp::Tof t{};
    int64_t nvox = 0;
    if (tofbin_host) { // a listmode plan needs the image geometry and the TOF parameters
        if (!geom_ok(geom, g, nvox) || !tof_ok(tof, false, t)) return hfail(JP_ERR_SIZE, "jp_hybrid_set_lors: geom / tof needed with TOF bins");
        if (n >= ((int64_t)1 << 31)) return JP_ERR_SIZE;
    }
    // shards: contiguous, cut at multiples of the track length (when the list has one) and of 768 LORs
    const int64_t T = n > 0 ? host_track_length(lors_host) : 0;
    int64_t align = 768;
    if (T >= 32 && n % T == 0) {
        int64_t a = T, b = 768;
        while (b) { const int64_t r = a % b; a = b; b = r; }
        align = T / a * 768;
    }
    const int64_t nw = (int64_t)h->w.size();
    int64_t per = (n + nw - 1) / nw;
    per = (per + align - 1) / align * align;
    for (int64_t i = 0; i < nw; ++i) {
        h->w[(size_t)i].lo = std::min(n, i * per);
        h->w[(size_t)i].hi = std::min(n, (i + 1) * per);
    }
    h->n = n;
    h->have_tb = tofbin_host != nullptr;
    h->g_lm = g;
    h->t_lm = t;
    h->have_lors = false;
    const int rc = run_all(h, [&](Worker &wk) -> cudaError_t {
        drop_plans(wk);
        const int64_t m = wk.hi - wk.lo;
        if (m <= 0) return cudaSuccess;
        cudaError_t e = wk.coord.ensure(sizeof(float) * 6 * (size_t)m);
        if (e != cudaSuccess) return e;
        const float *src[6] = {lors_host->xs, lors_host->ys, lors_host->zs, lors_host->xe, lors_host->ye, lors_host->ze};
        for (int a = 0; a < 6; ++a)
            if ((e = cudaMemcpyAsync((float *)wk.coord.p + (size_t)a * m, src[a] + wk.lo, sizeof(float) * (size_t)m,
                                     cudaMemcpyHostToDevice, wk.st)) != cudaSuccess)
                return e;
        const jp::Lors l = shard_lors(wk);
        if (tofbin_host) {
            if ((e = wk.tb.ensure(sizeof(int16_t) * (size_t)m)) != cudaSuccess) return e;
            if ((e = cudaMemcpyAsync(wk.tb.p, tofbin_host + wk.lo, sizeof(int16_t) * (size_t)m, cudaMemcpyHostToDevice, wk.st)) != cudaSuccess)
                return e;
            return jp::lm_plan_create(l, (const int16_t *)wk.tb.p, m, g, t, 1, wk.st, &wk.lp);
        }
        return jp::sino_plan_create(l, m, wk.st, &wk.sp);
    }, "jp_hybrid_set_lors");
    if (rc == JP_OK) h->have_lors = true;
    return rc;
}

int jp_hybrid_fwd(jp_hybrid *h, const float *img_host, const jp_geom *geom, float *p_host)
{
    jp::err_buf()[0] = 0;
    int rc = check_ready(h, false);
    if (rc != JP_OK) return rc;
    jp::Geom g;
    int64_t nvox;
    if (!img_host || !geom) return JP_ERR_POINTER;
    if (!geom_ok(geom, g, nvox)) return JP_ERR_SIZE;
    if (h->n == 0) return JP_OK;
    if (!p_host) return JP_ERR_POINTER;
    return run_all(h, [&](Worker &wk) -> cudaError_t {
        const int64_t m = wk.hi - wk.lo;
        if (m <= 0) return cudaSuccess;
        cudaError_t e = upload_image(wk, img_host, nvox);
        if (e == cudaSuccess) e = wk.val.ensure(sizeof(float) * (size_t)m);
        if (e != cudaSuccess) return e;
        const jp::Lors l = shard_lors(wk);
        e = cudaErrorNotSupported;
        if (wk.sp) {
            const jp::SinoPlanView v = jp::sino_plan_view(wk.sp);
            if (v.regular) e = jp::launch_fwd_tile(l, m, (const float *)wk.img.p, g, (float *)wk.val.p, wk.st, &v);
        }
        if (e == cudaErrorNotSupported) e = jp::launch_fwd_tile(l, m, (const float *)wk.img.p, g, (float *)wk.val.p, wk.st);
        if (e != cudaSuccess) return e;
        return cudaMemcpyAsync(p_host + wk.lo, wk.val.p, sizeof(float) * (size_t)m, cudaMemcpyDeviceToHost, wk.st);
    }, "jp_hybrid_fwd");
}

int jp_hybrid_back(jp_hybrid *h, const float *y_host, const jp_geom *geom, float *img_host)
{
    jp::err_buf()[0] = 0;
    int rc = check_ready(h, false);
    if (rc != JP_OK) return rc;
    jp::Geom g;
    int64_t nvox;
    if (!img_host || !geom) return JP_ERR_POINTER;
    if (!geom_ok(geom, g, nvox)) return JP_ERR_SIZE;
    if (h->n == 0) return JP_OK;
    if (!y_host) return JP_ERR_POINTER;
    rc = run_all(h, [&](Worker &wk) -> cudaError_t {
        const int64_t m = wk.hi - wk.lo;
        if (m <= 0) return cudaSuccess;
        cudaError_t e = zero_partial(wk, nvox);
        if (e == cudaSuccess) e = wk.val.ensure(sizeof(float) * (size_t)m);
        if (e == cudaSuccess) e = cudaMemcpyAsync(wk.val.p, y_host + wk.lo, sizeof(float) * (size_t)m, cudaMemcpyHostToDevice, wk.st);
        if (e != cudaSuccess) return e;
        const jp::Lors l = shard_lors(wk);
        e = cudaErrorNotSupported;
        if (wk.sp) {
            const jp::SinoPlanView v = jp::sino_plan_view(wk.sp);
            if (v.regular) e = jp::launch_back_tile(l, m, (const float *)wk.val.p, g, (float *)wk.img2.p, wk.st, &v);
        }
        if (e == cudaErrorNotSupported) e = jp::launch_back_tile(l, m, (const float *)wk.val.p, g, (float *)wk.img2.p, wk.st);
        if (e != cudaSuccess) return e;
        return download_partial(wk, nvox);
    }, "jp_hybrid_back");
    if (rc == JP_OK) add_partials(h, nvox, img_host);
    return rc;
}

} // extern "C"

// ---- TOF calls on the handle ---------------------------------------------------------------------------------------
namespace {

// the unplanned TOF sinogram kernels on a worker's shard (irregular shards, TOF kernels too wide for the tile kernels)
cudaError_t tof_sino_generic(Worker &wk, bool back, const jp::Lors &l, int64_t m, const jp::Geom &g, const jp::Tof &t)
{
    jp::TofLut lut{};
    float *pimg = nullptr;
    cudaError_t e = jp::tof_lut_create(t, wk.st, &lut);
    if (e == cudaSuccess) e = jp::padded_create(back ? nullptr : (const float *)wk.img.p, g, back, wk.st, &pimg);
    if (e == cudaSuccess) {
        e = jp::launch_tof_sino_win(back, l, m, back ? nullptr : pimg, back ? pimg : nullptr, g, t, back ? nullptr : (float *)wk.val.p,
                                    back ? (const float *)wk.val.p : nullptr, wk.st);
        if (e == cudaErrorNotSupported) {
            const jp::Range rg{0, 1, m, false, nullptr};
            e = back ? jp::launch_back_tof_sino(l, rg, (const float *)wk.val.p, g, t, lut, pimg, wk.st)
                     : jp::launch_fwd_tof_sino(l, rg, pimg, g, t, lut, (float *)wk.val.p, wk.st);
        }
    }
    if (e == cudaSuccess && back) e = jp::padded_add_to(pimg, g, (float *)wk.img2.p, wk.st);
    jp::padded_destroy(pimg, wk.st);
    jp::tof_lut_destroy(&lut, wk.st);
    return e;
}

int hybrid_tof_sino(jp_hybrid *h, bool back, const float *vals_in, float *vals_out, const float *img_in, float *img_out,
                    const jp_geom *geom, const jp_tof *tof, const char *where)
{
    jp::err_buf()[0] = 0;
    int rc = check_ready(h, false);
    if (rc != JP_OK) return rc;
    jp::Geom g;
    jp::Tof t;
    int64_t nvox;
    if (!geom || !tof || (back ? !img_out : !img_in)) return JP_ERR_POINTER;
    if (!geom_ok(geom, g, nvox) || !tof_ok(tof, true, t)) return JP_ERR_SIZE;
    if (jp::padded_voxels(g) >= ((int64_t)1 << 31)) return JP_ERR_SIZE;
    if (h->n == 0) return JP_OK;
    if (back ? !vals_in : !vals_out) return JP_ERR_POINTER;
    const int nb = t.nbins;
    rc = run_all(h, [&](Worker &wk) -> cudaError_t {
        const int64_t m = wk.hi - wk.lo;
        if (m <= 0) return cudaSuccess;
        cudaError_t e = back ? zero_partial(wk, nvox) : upload_image(wk, img_in, nvox);
        if (e == cudaSuccess) e = wk.val.ensure(sizeof(float) * (size_t)m * nb);
        if (e == cudaSuccess && back)
            e = cudaMemcpyAsync(wk.val.p, vals_in + wk.lo * nb, sizeof(float) * (size_t)m * nb, cudaMemcpyHostToDevice, wk.st);
        if (e != cudaSuccess) return e;
        const jp::Lors l = shard_lors(wk);
        e = cudaErrorNotSupported;
        if (wk.sp) {
            const jp::SinoPlanView v = jp::sino_plan_view(wk.sp);
            if (v.regular)
                e = jp::launch_tof_sino_tile(back ? 1 : 0, v, 0, v.K, (const float *)wk.img.p, (float *)wk.img2.p, g, t,
                                             (float *)wk.val.p, (const float *)wk.val.p, nullptr, wk.st);
        }
        if (e == cudaErrorNotSupported) e = tof_sino_generic(wk, back, l, m, g, t);
        if (e != cudaSuccess) return e;
        return back ? download_partial(wk, nvox)
                    : cudaMemcpyAsync(vals_out + wk.lo * nb, wk.val.p, sizeof(float) * (size_t)m * nb, cudaMemcpyDeviceToHost, wk.st);
    }, where);
    if (rc == JP_OK && back) add_partials(h, nvox, img_out);
    return rc;
}

int hybrid_tof_lm(jp_hybrid *h, bool back, const float *vals_in, float *vals_out, const float *img_in, float *img_out,
                  const char *where)
{
    jp::err_buf()[0] = 0;
    int rc = check_ready(h, true);
    if (rc != JP_OK) return rc;
    const jp::Geom g = h->g_lm;
    const jp::Tof t = h->t_lm;
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    if (back ? !img_out : !img_in) return JP_ERR_POINTER;
    if (h->n == 0) return JP_OK;
    if (back ? !vals_in : !vals_out) return JP_ERR_POINTER;
    rc = run_all(h, [&](Worker &wk) -> cudaError_t {
        const int64_t m = wk.hi - wk.lo;
        if (m <= 0) return cudaSuccess;
        cudaError_t e = back ? zero_partial(wk, nvox) : upload_image(wk, img_in, nvox);
        if (e == cudaSuccess) e = wk.val.ensure(sizeof(float) * (size_t)m);
        if (e == cudaSuccess && back)
            e = cudaMemcpyAsync(wk.val.p, vals_in + wk.lo, sizeof(float) * (size_t)m, cudaMemcpyHostToDevice, wk.st);
        if (e != cudaSuccess) return e;
        e = back ? jp::lm_plan_back_tof(wk.lp, -1, (const float *)wk.val.p, (float *)wk.img2.p, wk.st)
                 : jp::lm_plan_fwd_tof(wk.lp, -1, (const float *)wk.img.p, (float *)wk.val.p, wk.st);
        if (e != cudaSuccess) return e;
        return back ? download_partial(wk, nvox)
                    : cudaMemcpyAsync(vals_out + wk.lo, wk.val.p, sizeof(float) * (size_t)m, cudaMemcpyDeviceToHost, wk.st);
    }, where);
    if (rc == JP_OK && back) add_partials(h, nvox, img_out);
    return rc;
}

// one-shot calls: a handle over all visible devices for the duration of the call
struct OneShot {
    jp_hybrid *h = nullptr;
    ~OneShot() { jp_hybrid_destroy(h); }
};

// argument errors are reported before any device is touched
int oneshot_check(const jp_lors *l, const jp_geom *geom, const jp_tof *tof, bool need_tof, bool sino, const void *a, const void *b)
{
    jp::err_buf()[0] = 0;
    if (!l || !geom || (need_tof && !tof) || !a) return JP_ERR_POINTER;
    jp::Geom g;
    jp::Tof t;
    int64_t nvox;
    if (l->n < 0 || !geom_ok(geom, g, nvox) || (need_tof && !tof_ok(tof, sino, t))) return JP_ERR_SIZE;
    if (l->n > 0 && (!b || !l->xs || !l->ys || !l->zs || !l->xe || !l->ye || !l->ze)) return JP_ERR_POINTER;
    return JP_OK;
}

} // namespace

extern "C" {

int jp_hybrid_fwd_tof_sino(jp_hybrid *h, const float *img_host, const jp_geom *geom, const jp_tof *tof, float *p_host)
{
    return hybrid_tof_sino(h, false, nullptr, p_host, img_host, nullptr, geom, tof, "jp_hybrid_fwd_tof_sino");
}

int jp_hybrid_back_tof_sino(jp_hybrid *h, const float *y_host, const jp_geom *geom, const jp_tof *tof, float *img_host)
{
    return hybrid_tof_sino(h, true, y_host, nullptr, nullptr, img_host, geom, tof, "jp_hybrid_back_tof_sino");
}

int jp_hybrid_fwd_tof_lm(jp_hybrid *h, const float *img_host, float *p_host)
{
    return hybrid_tof_lm(h, false, nullptr, p_host, img_host, nullptr, "jp_hybrid_fwd_tof_lm");
}

int jp_hybrid_back_tof_lm(jp_hybrid *h, const float *y_host, float *img_host)
{
    return hybrid_tof_lm(h, true, y_host, nullptr, nullptr, img_host, "jp_hybrid_back_tof_lm");
}

int jp_fwd_host(const jp_lors *lors_host, const float *img_host, const jp_geom *geom, float *p_host)
{
    { const int rc0 = oneshot_check(lors_host, geom, nullptr, false, false, img_host, p_host); if (rc0 != JP_OK) return rc0; }
    OneShot o;
    int rc = jp_hybrid_create(nullptr, 0, &o.h);
    if (rc == JP_OK) rc = jp_hybrid_set_lors(o.h, lors_host, nullptr, nullptr, nullptr);
    if (rc == JP_OK) rc = jp_hybrid_fwd(o.h, img_host, geom, p_host);
    return rc;
}

int jp_back_host(const jp_lors *lors_host, const float *y_host, const jp_geom *geom, float *img_host)
{
    { const int rc0 = oneshot_check(lors_host, geom, nullptr, false, false, img_host, y_host); if (rc0 != JP_OK) return rc0; }
    OneShot o;
    int rc = jp_hybrid_create(nullptr, 0, &o.h);
    if (rc == JP_OK) rc = jp_hybrid_set_lors(o.h, lors_host, nullptr, nullptr, nullptr);
    if (rc == JP_OK) rc = jp_hybrid_back(o.h, y_host, geom, img_host);
    return rc;
}

int jp_fwd_tof_sino_host(const jp_lors *lors_host, const float *img_host, const jp_geom *geom, const jp_tof *tof,
                         float *p_host)
{
    { const int rc0 = oneshot_check(lors_host, geom, tof, true, true, img_host, p_host); if (rc0 != JP_OK) return rc0; }
    OneShot o;
    int rc = jp_hybrid_create(nullptr, 0, &o.h);
    if (rc == JP_OK) rc = jp_hybrid_set_lors(o.h, lors_host, nullptr, nullptr, nullptr);
    if (rc == JP_OK) rc = jp_hybrid_fwd_tof_sino(o.h, img_host, geom, tof, p_host);
    return rc;
}

int jp_back_tof_sino_host(const jp_lors *lors_host, const float *y_host, const jp_geom *geom, const jp_tof *tof,
                          float *img_host)
{
    { const int rc0 = oneshot_check(lors_host, geom, tof, true, true, img_host, y_host); if (rc0 != JP_OK) return rc0; }
    OneShot o;
    int rc = jp_hybrid_create(nullptr, 0, &o.h);
    if (rc == JP_OK) rc = jp_hybrid_set_lors(o.h, lors_host, nullptr, nullptr, nullptr);
    if (rc == JP_OK) rc = jp_hybrid_back_tof_sino(o.h, y_host, geom, tof, img_host);
    return rc;
}

int jp_fwd_tof_lm_host(const jp_lors *lors_host, const int16_t *tofbin_host, const float *img_host, const jp_geom *geom,
                       const jp_tof *tof, float *p_host)
{
    if (lors_host && lors_host->n > 0 && !tofbin_host) return JP_ERR_POINTER;
    { const int rc0 = oneshot_check(lors_host, geom, tof, true, false, img_host, p_host); if (rc0 != JP_OK) return rc0; }
    OneShot o;
    int rc = jp_hybrid_create(nullptr, 0, &o.h);
    if (rc == JP_OK) rc = jp_hybrid_set_lors(o.h, lors_host, tofbin_host, geom, tof);
    if (rc == JP_OK) rc = jp_hybrid_fwd_tof_lm(o.h, img_host, p_host);
    return rc;
}

int jp_back_tof_lm_host(const jp_lors *lors_host, const int16_t *tofbin_host, const float *y_host, const jp_geom *geom,
                        const jp_tof *tof, float *img_host)
{
    if (lors_host && lors_host->n > 0 && !tofbin_host) return JP_ERR_POINTER;
    { const int rc0 = oneshot_check(lors_host, geom, tof, true, false, img_host, y_host); if (rc0 != JP_OK) return rc0; }
    OneShot o;
    int rc = jp_hybrid_create(nullptr, 0, &o.h);
    if (rc == JP_OK) rc = jp_hybrid_set_lors(o.h, lors_host, tofbin_host, geom, tof);
    if (rc == JP_OK) rc = jp_hybrid_back_tof_lm(o.h, y_host, img_host);
    return rc;
}

} // extern "C"
