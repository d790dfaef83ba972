// Test helper (not product, not oracle): exposes cuRAND's own Philox4x32-10 block function on the
// HOST, as a black box, so the oracle's Philox can be pinned against a library routine without a GPU.
// cuRAND's header provides a host code path when QUALIFIERS is overridable (curand_philox4x32_x.h).
#define QUALIFIERS static inline __host__ __device__
#include <curand_kernel.h>
#include <curand_philox4x32_x.h>
#include <cstdint>

extern "C" void curand_philox_block(uint64_t n, const uint32_t* ctrs, const uint32_t* key, uint32_t* out) {
    for (uint64_t i = 0; i < n; ++i) {
        uint4 c = make_uint4(ctrs[4 * i], ctrs[4 * i + 1], ctrs[4 * i + 2], ctrs[4 * i + 3]);
        uint2 k = make_uint2(key[0], key[1]);
        uint4 r = curand_Philox4x32_10(c, k);
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}
