__global__ void k(unsigned long long *out, const int *idx, const long long *v)
{
    __shared__ unsigned long long s[256];
    s[threadIdx.x] = 0;
    __syncthreads();
    unsigned a = (unsigned)__cvta_generic_to_shared(&s[idx[threadIdx.x]]);
    asm volatile("red.shared.add.u64 [%0], %1;" ::"r"(a), "l"(v[threadIdx.x]) : "memory");
    __syncthreads();
    out[threadIdx.x] = s[threadIdx.x];
}
