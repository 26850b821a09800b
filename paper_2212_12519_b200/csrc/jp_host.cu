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
constexpr int64_t kChunk = 8 << 20; // LORs per chunk: 8 Mi x 28 B = 224 MiB of device staging per stream

struct HostPipe {
    cudaStream_t st[kStreams] = {};
    float *coord[kStreams] = {}; // 6 * chunk floats
    float *val[kStreams] = {};   // chunk floats (p out, or y in)
    float *img = nullptr;
    cudaError_t err = cudaSuccess;

    cudaError_t init(int64_t chunk, int64_t nvox)
    {
        for (int s = 0; s < kStreams; ++s) {
            if ((err = cudaStreamCreateWithFlags(&st[s], cudaStreamNonBlocking)) != cudaSuccess) return err;
            if ((err = cudaMalloc(&coord[s], sizeof(float) * 6 * chunk)) != cudaSuccess) return err;
            if ((err = cudaMalloc(&val[s], sizeof(float) * chunk)) != cudaSuccess) return err;
        }
        return err = cudaMalloc(&img, sizeof(float) * nvox);
    }
    ~HostPipe()
    {
        for (int s = 0; s < kStreams; ++s) {
            if (coord[s]) cudaFree(coord[s]);
            if (val[s]) cudaFree(val[s]);
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
