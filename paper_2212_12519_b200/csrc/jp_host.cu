// jp_host.cu -- "hybrid" entry points: HOST buffers in, HOST buffers out ("hybrid
// CPU/GPU mode": host -> device transfer, projection kernels, transfer of the result back).
//
// The LOR list is streamed through the GPU in chunks on two CUDA streams, so the host->device copy
// of chunk c+1 overlaps the kernel of chunk c and the device->host copy of chunk c-1 (PAPER.md:124
// "chunk-wise").  Copies are truly asynchronous only from page-locked host memory; pageable memory
// works but serialises.  The calls return after the result is in host memory.
#include <algorithm>
#include <cstdio>

#include "../../include/joseph_b200.h"
#include "jp_internal.h"

namespace {

constexpr int kStreams = 2;
// LORs per chunk: 8.4 M x 28 B = 224 MiB of device staging per stream.  A multiple of 768 (the tile of jp_tile.cu) and
// of 2304, so that chunk boundaries do not cut the tracks of a 48-ring sinogram into straddling tiles.
constexpr int64_t kChunk = 2304 * 3641;
constexpr int64_t kChunkTofSino = 2304 * 455; // x n_tofbins values per LOR

struct HostPipe {
    cudaStream_t st[kStreams] = {};
    float *coord[kStreams] = {}; // 6 * chunk floats
    float *val[kStreams] = {};   // chunk floats (p out, or y in)
    float *img = nullptr;
    cudaError_t err = cudaSuccess;

    int16_t *tb[kStreams] = {}; // chunk TOF bins (listmode)

    cudaError_t init(int64_t chunk, int64_t nvox, int vals_per_lor = 1, bool with_tb = false)
    {
        for (int s = 0; s < kStreams; ++s) {
            if ((err = cudaStreamCreateWithFlags(&st[s], cudaStreamNonBlocking)) != cudaSuccess) return err;
            if ((err = cudaMalloc(&coord[s], sizeof(float) * 6 * chunk)) != cudaSuccess) return err;
            if ((err = cudaMalloc(&val[s], sizeof(float) * chunk * vals_per_lor)) != cudaSuccess) return err;
            if (with_tb && (err = cudaMalloc(&tb[s], sizeof(int16_t) * chunk)) != cudaSuccess) return err;
        }
        return err = cudaMalloc(&img, sizeof(float) * nvox);
    }
    ~HostPipe()
    {
        for (int s = 0; s < kStreams; ++s) {
            if (coord[s]) cudaFree(coord[s]);
            if (val[s]) cudaFree(val[s]);
            if (tb[s]) cudaFree(tb[s]);
            if (st[s]) cudaStreamDestroy(st[s]);
        }
        if (img) cudaFree(img);
    }
};

int host_fail(cudaError_t e, const char *where)
{
    snprintf(jp::err_buf(), 512, "%s: %s", where, cudaGetErrorString(e));
    return JP_ERR_CUDA;
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

// stage chunk [c0, c0+m) of the six host coordinate arrays into dev (SoA with row length `chunk`)
cudaError_t stage_coords(const jp_lors *h, int64_t c0, int64_t m, float *dev, int64_t chunk, cudaStream_t st, jp::Lors &l)
{
    const float *src[6] = {h->xs, h->ys, h->zs, h->xe, h->ye, h->ze};
    for (int a = 0; a < 6; ++a) {
        cudaError_t e = cudaMemcpyAsync(dev + a * chunk, src[a] + c0, sizeof(float) * m, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return e;
    }
    l.xs = dev; l.ys = dev + chunk; l.zs = dev + 2 * chunk;
    l.xe = dev + 3 * chunk; l.ye = dev + 4 * chunk; l.ze = dev + 5 * chunk;
    return cudaSuccess;
}

} // namespace

extern "C" {

int jp_fwd_host(const jp_lors *lors_host, const float *img_host, const jp_geom *geom, float *p_host)
{
    jp::err_buf()[0] = 0;
    jp::Geom g;
    int64_t nvox;
    if (!lors_host || !img_host || !geom) return JP_ERR_POINTER;
    if (lors_host->n < 0 || !geom_ok(geom, g, nvox)) return JP_ERR_SIZE;
    const int64_t n = lors_host->n;
    if (n == 0) return JP_OK;
    if (!p_host || !lors_host->xs || !lors_host->ys || !lors_host->zs || !lors_host->xe || !lors_host->ye || !lors_host->ze)
        return JP_ERR_POINTER;
    const int64_t chunk = std::min(kChunk, n);
    HostPipe hp;
    if (hp.init(chunk, nvox) != cudaSuccess) return host_fail(hp.err, "jp_fwd_host alloc");
    cudaError_t e = cudaMemcpy(hp.img, img_host, sizeof(float) * nvox, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return host_fail(e, "jp_fwd_host img copy");
    int s = 0;
    for (int64_t c0 = 0; c0 < n; c0 += chunk, s = (s + 1) % kStreams) {
        const int64_t m = std::min(chunk, n - c0);
        jp::Lors l;
        if ((e = stage_coords(lors_host, c0, m, hp.coord[s], chunk, hp.st[s], l)) != cudaSuccess) break;
        if ((e = jp::launch_fwd_tile(l, m, hp.img, g, hp.val[s], hp.st[s])) != cudaSuccess) break;
        if ((e = cudaMemcpyAsync(p_host + c0, hp.val[s], sizeof(float) * m, cudaMemcpyDeviceToHost, hp.st[s])) != cudaSuccess) break;
    }
    for (int k = 0; k < kStreams; ++k) {
        cudaError_t e2 = cudaStreamSynchronize(hp.st[k]);
        if (e == cudaSuccess) e = e2;
    }
    return e == cudaSuccess ? JP_OK : host_fail(e, "jp_fwd_host");
}

int jp_back_host(const jp_lors *lors_host, const float *y_host, const jp_geom *geom, float *img_host)
{
    jp::err_buf()[0] = 0;
    jp::Geom g;
    int64_t nvox;
    if (!lors_host || !img_host || !geom) return JP_ERR_POINTER;
    if (lors_host->n < 0 || !geom_ok(geom, g, nvox)) return JP_ERR_SIZE;
    const int64_t n = lors_host->n;
    if (n == 0) return JP_OK;
    if (!y_host || !lors_host->xs || !lors_host->ys || !lors_host->zs || !lors_host->xe || !lors_host->ye || !lors_host->ze)
        return JP_ERR_POINTER;
    const int64_t chunk = std::min(kChunk, n);
    HostPipe hp;
    if (hp.init(chunk, nvox) != cudaSuccess) return host_fail(hp.err, "jp_back_host alloc");
    // ACCUMULATE semantics: start from the caller's image
    cudaError_t e = cudaMemcpy(hp.img, img_host, sizeof(float) * nvox, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return host_fail(e, "jp_back_host img copy");
    int s = 0;
    for (int64_t c0 = 0; c0 < n; c0 += chunk, s = (s + 1) % kStreams) {
        const int64_t m = std::min(chunk, n - c0);
        jp::Lors l;
        if ((e = stage_coords(lors_host, c0, m, hp.coord[s], chunk, hp.st[s], l)) != cudaSuccess) break;
        if ((e = cudaMemcpyAsync(hp.val[s], y_host + c0, sizeof(float) * m, cudaMemcpyHostToDevice, hp.st[s])) != cudaSuccess) break;
        if ((e = jp::launch_back_tile(l, m, hp.val[s], g, hp.img, hp.st[s])) != cudaSuccess) break;
    }
    for (int k = 0; k < kStreams; ++k) {
        cudaError_t e2 = cudaStreamSynchronize(hp.st[k]);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaMemcpy(img_host, hp.img, sizeof(float) * nvox, cudaMemcpyDeviceToHost);
    return e == cudaSuccess ? JP_OK : host_fail(e, "jp_back_host");
}

} // extern "C"

// ---- TOF hybrid calls: one pipeline, four modes ---------------------------------------------------------------------
namespace {

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

// sino: values are [n][n_tofbins]; listmode: [n] + tofbin[n].  back: vals = y (in), img accumulates; else vals = p (out)
int tof_host(bool sino, bool back, const jp_lors *h, const int16_t *tofbin_host, const float *vals_in, float *vals_out,
             const float *img_in, float *img_out, const jp_geom *geom, const jp_tof *tof, const char *where)
{
    jp::err_buf()[0] = 0;
    jp::Geom g;
    jp::Tof t;
    int64_t nvox;
    if (!h || !geom || !tof || !img_in) return JP_ERR_POINTER;
    if (h->n < 0 || !geom_ok(geom, g, nvox) || !tof_ok(tof, sino, t)) return JP_ERR_SIZE;
    if (jp::padded_voxels(g) >= ((int64_t)1 << 31)) return JP_ERR_SIZE;
    const int64_t n = h->n;
    if (n == 0) return JP_OK;
    if (!h->xs || !h->ys || !h->zs || !h->xe || !h->ye || !h->ze || (back ? !vals_in : !vals_out) || (!sino && !tofbin_host))
        return JP_ERR_POINTER;
    const int nv = sino ? t.nbins : 1;
    const int64_t chunk = std::min(sino ? kChunkTofSino : kChunk, n);
    HostPipe hp;
    if (hp.init(chunk, nvox, nv, !sino) != cudaSuccess) return host_fail(hp.err, where);
    cudaError_t e = cudaMemcpy(hp.img, img_in, sizeof(float) * nvox, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return host_fail(e, where);
    // scratch shared by all chunks: TOF edge table and the zero-padded image (forward: copy, back: accumulator)
    jp::TofLut lut{};
    float *pimg = nullptr;
    cudaStream_t s0 = hp.st[0];
    e = jp::tof_lut_create(t, s0, &lut);
    if (e == cudaSuccess) e = jp::padded_create(back ? nullptr : hp.img, g, back, s0, &pimg);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s0);
    int s = 0;
    for (int64_t c0 = 0; e == cudaSuccess && c0 < n; c0 += chunk, s = (s + 1) % kStreams) {
        const int64_t m = std::min(chunk, n - c0);
        cudaStream_t st = hp.st[s];
        jp::Lors l;
        if ((e = stage_coords(h, c0, m, hp.coord[s], chunk, st, l)) != cudaSuccess) break;
        if (!sino && (e = cudaMemcpyAsync(hp.tb[s], tofbin_host + c0, sizeof(int16_t) * m, cudaMemcpyHostToDevice, st)) != cudaSuccess) break;
        if (back && (e = cudaMemcpyAsync(hp.val[s], vals_in + c0 * nv, sizeof(float) * m * nv, cudaMemcpyHostToDevice, st)) != cudaSuccess) break;
        const jp::Range rg{0, 1, m, false, nullptr};
        if (sino) {
            e = jp::launch_tof_sino_win(back, l, m, back ? nullptr : pimg, back ? pimg : nullptr, g, t, back ? nullptr : hp.val[s],
                                        back ? hp.val[s] : nullptr, st);
            if (e == cudaErrorNotSupported)
                e = back ? jp::launch_back_tof_sino(l, rg, hp.val[s], g, t, lut, pimg, st)
                         : jp::launch_fwd_tof_sino(l, rg, pimg, g, t, lut, hp.val[s], st);
        } else {
            e = back ? jp::launch_back_tof_lm(l, hp.tb[s], rg, hp.val[s], g, t, lut, pimg, st)
                     : jp::launch_fwd_tof_lm(l, hp.tb[s], rg, pimg, g, t, lut, hp.val[s], 0, st);
        }
        if (e != cudaSuccess) break;
        if (!back) e = cudaMemcpyAsync(vals_out + c0 * nv, hp.val[s], sizeof(float) * m * nv, cudaMemcpyDeviceToHost, st);
    }
    for (int k = 0; k < kStreams; ++k) {
        cudaError_t e2 = cudaStreamSynchronize(hp.st[k]);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess && back) { // hp.img still holds the caller's image: ACCUMULATE
        e = jp::padded_add_to(pimg, g, hp.img, s0);
        if (e == cudaSuccess) e = cudaMemcpyAsync(img_out, hp.img, sizeof(float) * nvox, cudaMemcpyDeviceToHost, s0);
    }
    jp::padded_destroy(pimg, s0);
    jp::tof_lut_destroy(&lut, s0);
    cudaError_t e3 = cudaStreamSynchronize(s0);
    if (e == cudaSuccess) e = e3;
    return e == cudaSuccess ? JP_OK : host_fail(e, where);
}

} // namespace

extern "C" {

int jp_fwd_tof_sino_host(const jp_lors *lors_host, const float *img_host, const jp_geom *geom, const jp_tof *tof,
                         float *p_host)
{
    return tof_host(true, false, lors_host, nullptr, nullptr, p_host, img_host, nullptr, geom, tof, "jp_fwd_tof_sino_host");
}

int jp_back_tof_sino_host(const jp_lors *lors_host, const float *y_host, const jp_geom *geom, const jp_tof *tof,
                          float *img_host)
{
    return tof_host(true, true, lors_host, nullptr, y_host, nullptr, img_host, img_host, geom, tof, "jp_back_tof_sino_host");
}

int jp_fwd_tof_lm_host(const jp_lors *lors_host, const int16_t *tofbin_host, const float *img_host, const jp_geom *geom,
                       const jp_tof *tof, float *p_host)
{
    return tof_host(false, false, lors_host, tofbin_host, nullptr, p_host, img_host, nullptr, geom, tof, "jp_fwd_tof_lm_host");
}

int jp_back_tof_lm_host(const jp_lors *lors_host, const int16_t *tofbin_host, const float *y_host, const jp_geom *geom,
                        const jp_tof *tof, float *img_host)
{
    return tof_host(false, true, lors_host, tofbin_host, y_host, nullptr, img_host, img_host, geom, tof, "jp_back_tof_lm_host");
}

} // extern "C"
