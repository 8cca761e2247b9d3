// Test helper: exposes cuRAND's own Philox4x32-10 (host code path of
// curand_philox4x32_x.h) so the oracle's Philox can be pinned to an independent
// library routine.  Contains no code of the oracle or of the CUDA path.
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>
#include <stdint.h>

extern "C" void curand_philox_batch(int64_t n, const uint32_t* ctr /*4n*/, const uint32_t* key /*2n*/,
                                    uint32_t* out /*4n*/)
{
    for (int64_t t = 0; t < n; ++t) {
        uint4 c = make_uint4(ctr[4 * t], ctr[4 * t + 1], ctr[4 * t + 2], ctr[4 * t + 3]);
        uint2 k = make_uint2(key[2 * t], key[2 * t + 1]);
        uint4 r = curand_Philox4x32_10(c, k);
        out[4 * t] = r.x; out[4 * t + 1] = r.y; out[4 * t + 2] = r.z; out[4 * t + 3] = r.w;
    }
}
