// Test-only third opinion for Philox4x32-10 (SURVEY 8(c) O4 / pin 13): NVIDIA's cuRAND device API.
// Not part of the product and not used by it.  For each i, initialises a
// curandStatePhilox4_32_10_t with (seed, subsequence, offset) and returns the first curand4() block,
// which by cuRAND's definition is Philox4x32-10 of counter (offset/4 lo, offset/4 hi, subsequence lo,
// subsequence hi) under key (seed lo, seed hi).
//   nvcc -gencode arch=compute_100a,code=sm_100a -shared -Xcompiler -fPIC curand_philox_ref.cu -o libcurand_philox_ref.so
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <stdint.h>

__global__ void curand_ref_kernel(int n, const unsigned long long* seed, const unsigned long long* subsequence,
                                  const unsigned long long* offset, uint32_t* out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    curandStatePhilox4_32_10_t st;
    curand_init(seed[i], subsequence[i], offset[i], &st);
    const uint4 r = curand4(&st);
    out[4 * i] = r.x;
    out[4 * i + 1] = r.y;
    out[4 * i + 2] = r.z;
    out[4 * i + 3] = r.w;
}

extern "C" int curand_philox_ref(int n, const void* dev_seed, const void* dev_subsequence, const void* dev_offset,
                                 void* dev_out, void* stream)
{
    curand_ref_kernel<<<(n + 127) / 128, 128, 0, static_cast<cudaStream_t>(stream)>>>(
        n, static_cast<const unsigned long long*>(dev_seed), static_cast<const unsigned long long*>(dev_subsequence),
        static_cast<const unsigned long long*>(dev_offset), static_cast<uint32_t*>(dev_out));
    return (int)cudaGetLastError();
}
