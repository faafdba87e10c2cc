// Test helper: cuRAND's own Philox4x32-10 (library code, /usr/local/cuda/include/curand_philox4x32_x.h)
// compiled for the HOST so that the CPU oracle's restatement can be pinned against a library routine
// without a GPU.  Built by tests/test_oracle_philox.py with nvcc; not part of the product or the oracle.
#define QUALIFIERS static inline __host__ __device__
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>

extern "C" void curand_philox_host(const unsigned* ctr, const unsigned* key, unsigned* out)
{
    uint4 c = make_uint4(ctr[0], ctr[1], ctr[2], ctr[3]);
    uint2 k = make_uint2(key[0], key[1]);
    uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
