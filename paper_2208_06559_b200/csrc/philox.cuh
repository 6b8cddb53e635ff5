// philox.cuh -- device-side Philox4x32-10 + Box-Muller (BASELINE.json north_star noise definition;
// replaces the paper's cuRAND uniform stream).  Written independently of oracle/.
//
// counter = (pair index p, chain id, step low 32, step high 28 | purpose << 28), key = seed (lo, hi)
// purpose 0: Brownian noise, 1: initial conformation.
// 128 output bits -> x1 = w1:w0, x2 = w3:w2 -> u = (2 (x >> 12) + 1) 2^-53 in (0,1).
#pragma once
#include <stdint.h>

struct Philox2 { double u1, u2; };

__device__ __forceinline__ Philox2 philox_uniform_pair(uint64_t seed, uint32_t pair, uint64_t chain,
                                                       uint64_t step, uint32_t purpose)
{
    uint32_t c0 = pair;
    uint32_t c1 = (uint32_t)chain;
    uint32_t c2 = (uint32_t)step;
    uint32_t c3 = ((uint32_t)(step >> 32) & 0x0FFFFFFFu) | (purpose << 28);
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    const uint64_t x1 = ((uint64_t)c1 << 32) | c0;
    const uint64_t x2 = ((uint64_t)c3 << 32) | c2;
    Philox2 r;
    r.u1 = (double)(((x1 >> 12) << 1) | 1ull) * 0x1.0p-53;
    r.u2 = (double)(((x2 >> 12) << 1) | 1ull) * 0x1.0p-53;
    return r;
}

// two Brownian increments dW_{2p}, dW_{2p+1} of (chain, step).
// kind 0: sqrt(2 dt) * (rho cos theta, rho sin theta); kind 1: sqrt(6 dt) * (2u1-1, 2u2-1) (Eq. 2).
__device__ __forceinline__ void brownian_pair(uint64_t seed, uint32_t pair, uint64_t chain, uint64_t step,
                                              int kind, double dt, double& w0, double& w1)
{
    Philox2 u = philox_uniform_pair(seed, pair, chain, step, 0u);
    if (kind == 1) {
        const double s = sqrt(6.0 * dt);
        w0 = s * (2.0 * u.u1 - 1.0);
        w1 = s * (2.0 * u.u2 - 1.0);
    } else {
        const double rho = sqrt(-2.0 * log(u.u1));
        double sn, cs;
        sincos(6.283185307179586 * u.u2, &sn, &cs);
        const double s = sqrt(2.0 * dt);
        w0 = s * (rho * cs);
        w1 = s * (rho * sn);
    }
}
