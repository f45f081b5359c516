// Philox4x32-10 device function (Salmon et al., SC'11).  Internal to libcloak.so.
#pragma once
#include <stdint.h>

namespace cloak {

// r_i of O2: words o0:o1 of Philox(ctr = (i, 0, s_lo, s_hi), key = (k0, k1)).
__device__ __forceinline__ uint64_t philox_key64(uint32_t i, uint32_t s_lo, uint32_t s_hi, uint32_t k0, uint32_t k1) {
    uint32_t c0 = i, c1 = 0u, c2 = s_lo, c3 = s_hi;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return ((uint64_t)c0 << 32) | c1;
}

}  // namespace cloak
