// jp_pad.cu -- zero-padded copies of the image for the per-LOR kernels (see PRay in jp_ray.cuh):
// pad (image -> padded copy), unpad-add (image += interior of the padded accumulator), and the OSEM
// update on a padded pair (x, b).
#include "jp_internal.h"

namespace jp {

__device__ __forceinline__ int64_t padded_index(const Geom &g, int64_t i, int &i2)
{
    const int n2 = g.n[2], n1 = g.n[1];
    i2 = (int)(i % n2);
    const int64_t r = i / n2;
    const int i1 = (int)(r % n1), i0 = (int)(r / n1);
    const int pn1 = n1 + 2 * kImgPad, pn2 = n2 + 2 * kImgPad;
    return ((int64_t)(i0 + kImgPad) * pn1 + (i1 + kImgPad)) * pn2 + (i2 + kImgPad);
}

__global__ void k_pad(const float *__restrict__ img, Geom g, int64_t nvox, float *__restrict__ pimg)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= nvox) return;
    int i2;
    pimg[padded_index(g, i, i2)] = img[i];
}

__global__ void k_unpad_add(const float *__restrict__ pimg, Geom g, int64_t nvox, float *__restrict__ img)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= nvox) return;
    int i2;
    img[i] += pimg[padded_index(g, i, i2)];
}

// x = sens > 0 ? x * b * scale / sens : 0 on the image and on its padded copy; b (padded) = 0
__global__ void k_osem_update_padded(float *__restrict__ x, float *__restrict__ px, float *__restrict__ pb,
                                     const float *__restrict__ sens, float scale, Geom g, int64_t nvox)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= nvox) return;
    int i2;
    const int64_t pi = padded_index(g, i, i2);
    const float s = sens[i];
    const float v = (s > 0.f) ? x[i] * pb[pi] * scale / s : 0.f;
    x[i] = v;
    px[pi] = v;
    pb[pi] = 0.f;
}

int64_t padded_voxels(const Geom &g)
{
    return (int64_t)(g.n[0] + 2 * kImgPad) * (g.n[1] + 2 * kImgPad) * (g.n[2] + 2 * kImgPad);
}

static inline unsigned grid_for(int64_t n) { return (unsigned)((n + 255) / 256); }

// padded copy of img in stream-ordered scratch (zero border); zero_only: an all-zero accumulator
cudaError_t padded_create(const float *img, const Geom &g, bool zero_only, cudaStream_t st, float **out)
{
    const int64_t pv = padded_voxels(g), nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    float *p = nullptr;
    cudaError_t e = cudaMallocAsync((void **)&p, sizeof(float) * (size_t)pv, st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(p, 0, sizeof(float) * (size_t)pv, st);
    if (e == cudaSuccess && !zero_only) {
        k_pad<<<grid_for(nvox), 256, 0, st>>>(img, g, nvox, p);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        cudaFreeAsync(p, st);
        return e;
    }
    *out = p;
    return cudaSuccess;
}

cudaError_t padded_add_to(const float *pimg, const Geom &g, float *img, cudaStream_t st)
{
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    k_unpad_add<<<grid_for(nvox), 256, 0, st>>>(pimg, g, nvox, img);
    return cudaGetLastError();
}

void padded_destroy(float *p, cudaStream_t st)
{
    if (p) cudaFreeAsync(p, st);
}

cudaError_t launch_osem_update_padded(float *x, float *px, float *pb, const float *sens, float scale, const Geom &g,
                                      cudaStream_t st)
{
    const int64_t nvox = (int64_t)g.n[0] * g.n[1] * g.n[2];
    k_osem_update_padded<<<grid_for(nvox), 256, 0, st>>>(x, px, pb, sens, scale, g, nvox);
    return cudaGetLastError();
}

} // namespace jp
