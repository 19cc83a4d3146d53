// gen.cu -- device twin of inputs/__init__.py:uniform_rhs (same 64-bit integer mixer, so the bits
// match the numpy generator exactly).  Holds none of the solver's arithmetic.
#include <cuda_runtime.h>
#include <stdint.h>

__host__ __device__ static inline uint64_t mix64(uint64_t z)
{
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

template <typename T>
__global__ void fill_uniform(T *out, int n, long long batch, long long j0, uint64_t s0, double scale)
{
    const long long total = (long long)n * batch;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long i = idx / batch, j = idx - i * batch;
        const uint64_t z = mix64(mix64(s0 + (uint64_t)(j0 + j)) + (uint64_t)i);
        double v = (double)(z >> 11) * (2.0 * 1.1102230246251565e-16) - 1.0;  // 2 * 2^-53
        if (scale != 1.0) v *= scale;
        out[idx] = (T)v;
    }
}

extern "C" __attribute__((visibility("default"))) int btps_inputs_fill_uniform(
    void *d_out, int elem_bytes, int n, long long batch, long long j0, unsigned long long seed,
    unsigned long long tag, double scale, void *stream)
{
    const uint64_t s0 = mix64((uint64_t)seed + (uint64_t)tag * 0x9E3779B97F4A7C15ULL);
    const long long total = (long long)n * batch;
    const int block = 256;
    long long grid = (total + block - 1) / block;
    if (grid > 148 * 32) grid = 148 * 32;
    if (grid < 1) grid = 1;
    if (elem_bytes == 8)
        fill_uniform<double><<<(unsigned)grid, block, 0, (cudaStream_t)stream>>>((double *)d_out, n, batch, j0, s0, scale);
    else
        fill_uniform<float><<<(unsigned)grid, block, 0, (cudaStream_t)stream>>>((float *)d_out, n, batch, j0, s0, scale);
    return (int)cudaGetLastError();
}
