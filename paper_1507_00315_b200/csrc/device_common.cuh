// Device helpers shared by the generic and the SWAR kernels: 32-bit Montgomery arithmetic
// (R = 2^32, odd p < 2^31) and the block-level reduction + row write (§8(a) row a6).
#pragma once
#include "internal.h"
#include <cuda_runtime.h>
#include <stdint.h>

namespace pairings {

// a*b < p*2^32  ->  a*b*2^{-32} mod p in [0,p)
__device__ __forceinline__ uint32_t montmul(uint32_t a, uint32_t b, uint32_t p, uint32_t pinv_neg) {
    const uint64_t t = (uint64_t)a * b;
    const uint32_t m = (uint32_t)t * pinv_neg;
    const uint32_t u = (uint32_t)((t + (uint64_t)m * p) >> 32);   // < 2p < 2^32
    return u >= p ? u - p : u;
}

// out[idx] = (out[idx] + v) mod p, atomically (several blocks may share one chunk row)
__device__ __forceinline__ void atomic_add_mod(uint32_t* addr, uint32_t v, uint32_t p) {
    uint32_t old = *addr, assumed;
    do {
        assumed = old;
        uint32_t s = assumed + v; if (s >= p) s -= p;
        old = atomicCAS(addr, assumed, s);
    } while (old != assumed);
}

// Block-level sum of per-thread residues (vals[i] < p_i) and the row write.
// red: shared scratch of (blockDim/32) * PAIRINGS_MAX_MODULI uint64.
__device__ __forceinline__ void block_reduce_write(const KernelParams& kp, const uint32_t* vals,
                                                   unsigned long long nz, unsigned long long* red,
                                                   uint64_t chunk_local) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    for (int i = 0; i < kp.n_moduli; i++) {
        unsigned long long v = vals[i];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp * PAIRINGS_MAX_MODULI + i] = v;
    }
    for (int o = 16; o > 0; o >>= 1) nz += __shfl_xor_sync(0xffffffffu, nz, o);
    if (lane == 0 && kp.nonzero && nz) atomicAdd(kp.nonzero, nz);
    __syncthreads();
    if ((int)threadIdx.x < kp.n_moduli) {
        const int i = threadIdx.x;
        unsigned long long s = 0;
        for (int w = 0; w < nwarps; w++) s += red[w * PAIRINGS_MAX_MODULI + i];
        const uint32_t p = kp.primes[i].p;
        const uint32_t r = (uint32_t)(s % p);
        uint32_t* dst = kp.out + chunk_local * (uint64_t)kp.n_moduli + (uint64_t)i;
        if (kp.log2_bpc == 0) *dst = r; else atomic_add_mod(dst, r, p);
    }
}

}  // namespace pairings
