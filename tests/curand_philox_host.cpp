// Test helper: calls cuRAND's own Philox4x32-10 (curand_philox4x32_x.h, a library routine that is
// independent of oracle/ and of the CUDA path) on the host, for tests/test_oracle_noise.py.
#include <stdint.h>
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
extern "C" void curand_philox_host(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int64_t n) {
    for (int64_t i = 0; i < n; ++i) {
        uint4 c = {ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]};
        uint2 k = {key[2 * i], key[2 * i + 1]};
        uint4 r = curand_Philox4x32_10(c, k);
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}
