// Test helper: exposes cuRAND's own Philox4x32-10 (curand_philox4x32_x.h, shipped with the CUDA
// toolkit, independent of both the oracle and the product kernels) as a HOST function, so the CPU
// test-suite can cross-check the oracle's generator without a GPU.
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>

extern "C" void curand_philox_host(const unsigned* ctr, const unsigned* key, unsigned* out, unsigned long long n)
{
    for (unsigned long long i = 0; i < n; ++i) {
        uint4 c = make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
        uint2 k = make_uint2(key[2 * i], key[2 * i + 1]);
        uint4 r = curand_Philox4x32_10(c, k);
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}
