// noise.cuh -- Gaussian increments of the Brownian term of Eq. (1a) in the additive approximation the
// paper advocates: dW = sqrt(2 k_B T dt / (6 pi mu a)) z, z ~ N(0,1) independent per sphere, component and
// step (Eq. 1b, 1c).  z is a pure function of (seed, step n, system w, state element 3 alpha + i): Philox4x32-10
// (Salmon, Moraes, Dror, Shaw, SC'11) with counter (n lo, n hi, element, w) and key (seed lo, seed hi); the first two
// output words feed a Box-Muller transform.  No state, no tables: the integrator tail draws what it needs.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ds {

__device__ __forceinline__ void philox_round(uint32_t (&c)[4], uint32_t k0, uint32_t k1) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c[0]), lo0 = 0xD2511F53u * c[0];
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c[2]), lo1 = 0xCD9E8D57u * c[2];
    const uint32_t n0 = hi1 ^ c[1] ^ k0, n2 = hi0 ^ c[3] ^ k1;
    c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
}

__device__ __noinline__ double noise_normal(unsigned long long seed, long long n, int system, long long element) {
    uint32_t c[4] = {(uint32_t)((unsigned long long)n & 0xffffffffu), (uint32_t)((unsigned long long)n >> 32), (uint32_t)element,
                     (uint32_t)system};
    uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c, k0, k1);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    const double U1 = ((double)c[0] + 0.5) * (1.0 / 4294967296.0), U2 = ((double)c[1] + 0.5) * (1.0 / 4294967296.0);
    return sqrt(-2.0 * log(U1)) * cos(6.283185307179586476925286766559 * U2);
}

}  // namespace ds
