// c8ph_philox.cuh — the counter-based generator of libc8ph (device code shared by the kernels).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace c8ph {

// ---- Philox4x32-10 (Salmon et al.; thesis ref. [66]), round keys precomputed ---------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const uint2 (&key)[10])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ key[r].x;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ key[r].y;
        c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

}  // namespace c8ph
