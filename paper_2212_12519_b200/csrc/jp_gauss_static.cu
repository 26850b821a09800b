// jp_gauss_static.cu -- jp_gauss3d_static: the resolution-model smoothing of jp_gauss3d for
// callers that must not allocate device memory.
//
// Who that is: code that runs where the CUDA allocator is off limits -- a reconstruction loop whose memory budget
// was fixed at start-up and handed out completely (the pool is full, cudaMalloc would fail or evict), a host
// thread inside a latency-critical acquisition loop (cudaMalloc / cudaFree take a device-wide lock and may
// synchronise), or an application whose stream has no memory pool configured (a device or driver set-up without
// stream-ordered allocation, where the cudaMallocAsync inside jp_gauss3d returns cudaErrorNotSupported).
//
// The three separable passes need one image-sized intermediate.  jp_gauss3d takes it from cudaMallocAsync; here
// it is a fixed array in the library's own device data segment, JP_GAUSS3D_STATIC_MAX_VOXELS floats (16 MiB),
// which every GPU that loads libjoseph_b200.so holds until the process exits.  The kernels are the ones
// jp_gauss3d launches (jp_gauss.cu, unchanged): results are bit-identical.
#include <cstdio>
#include <mutex>

#include "../../include/joseph_b200.h"
#include "jp_internal.h"

namespace {

// The intermediate image.  256-byte aligned: the fused two-kernel path of launch_gauss3d moves float4s.
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and must never
// be passed to a kernel as it stands.
static __device__ __align__(256) float g_gauss_scratch[JP_GAUSS3D_STATIC_MAX_VOXELS];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
float *g_scratch_addr[kMaxDevices] = {}; // device address of g_gauss_scratch on device d; null until the first call there

// Address of the array on the CURRENT device (every device has its own copy of the library's globals, at its own
// address).  Looked up once per device, under a lock; later calls only read the cached pointer.
cudaError_t scratch_on_current_device(float **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        float *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_gauss_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

int sfail(int code, const char *msg)
{
    snprintf(jp::err_buf(), 512, "%s", msg);
    return code;
}

int sfail_cuda(cudaError_t e, const char *where)
{
    snprintf(jp::err_buf(), 512, "%s: %s (%s)", where, cudaGetErrorString(e), cudaGetErrorName(e));
    return JP_ERR_CUDA;
}

} // namespace

extern "C" int jp_gauss3d_static(const float *in, float *out, const jp_geom *geom, float sigma_mm, float n_sigmas,
                                 void *stream)
{
    jp::err_buf()[0] = 0;
    if (!geom) return sfail(JP_ERR_POINTER, "geom is NULL");
    jp::Geom g;
    int64_t nvox = 1;
    for (int a = 0; a < 3; ++a) {
        if (geom->n[a] <= 0) return sfail(JP_ERR_SIZE, "image dim <= 0");
        if (!(geom->voxsize[a] > 0.f)) return sfail(JP_ERR_SIZE, "voxsize <= 0");
        g.n[a] = geom->n[a];
        g.o[a] = geom->origin[a];
        g.v[a] = geom->voxsize[a];
        nvox *= geom->n[a];
    }
    if (nvox > (int64_t)JP_GAUSS3D_STATIC_MAX_VOXELS) {
        snprintf(jp::err_buf(), 512,
                 "jp_gauss3d_static: image of %lld voxels exceeds the built-in scratch of %lld voxels "
                 "(JP_GAUSS3D_STATIC_MAX_VOXELS); use jp_gauss3d, which allocates its scratch",
                 (long long)nvox, (long long)JP_GAUSS3D_STATIC_MAX_VOXELS);
        return JP_ERR_SIZE;
    }
    if (!in || !out) return sfail(JP_ERR_POINTER, "in or out is NULL");
    if (!(sigma_mm > 0.f) || !(n_sigmas > 0.f)) return sfail(JP_ERR_SIZE, "sigma_mm <= 0 or n_sigmas <= 0");
    float *tmp = nullptr;
    cudaError_t e = scratch_on_current_device(&tmp);
    if (e != cudaSuccess) return sfail_cuda(e, "jp_gauss3d_static (address of the built-in scratch)");
    // every pass writes all nvox elements of its destination before the next pass reads them: what an earlier
    // call left in the array is never read, so nothing has to be cleared
    e = jp::launch_gauss3d(in, out, tmp, g, sigma_mm, n_sigmas, (cudaStream_t)stream);
    if (e == cudaErrorInvalidValue) return sfail(JP_ERR_SIZE, "Gaussian kernel radius > 16 voxels");
    if (e != cudaSuccess) return sfail_cuda(e, "jp_gauss3d_static");
    return JP_OK;
}
