// Internal declarations shared by the translation units of libpairings_b200.so (not installed).
#ifndef PAIRINGS_INTERNAL_H
#define PAIRINGS_INTERNAL_H
#include <stdint.h>
#include "pairings.h"

#ifndef __CUDACC__
#define __host__
#define __device__
#endif

namespace pairings {

// pair distance d_k: k (Skolem) or k+1 (Langford)
__host__ __device__ inline constexpr int dist(int kind, int k) { return kind == PAIRINGS_SKOLEM ? k : k + 1; }

int check_kind_n(int kind, int n);
int check_moduli(const uint32_t* moduli, int n_moduli);
int check_chunks(int n, int chunk_bits, uint64_t begin, uint64_t end);

// Per-modulus Montgomery constants, R = 2^32 (p odd, 2^30 < p < 2^31).
struct MontPrime {
    uint32_t p;
    uint32_t pinv_neg;  // -p^{-1} mod 2^32
    uint32_t r1;        // 2^32 mod p  (Montgomery form of 1)
    uint32_t r2;        // 2^64 mod p  (montmul(w, r2) = w * 2^32 mod p for any 32-bit w)
    uint32_t r3;        // 2^96 mod p
    uint32_t pad[3];
};

// Kernel parameter block, passed by value (__grid_constant__).
struct KernelParams {
    int kind, n;
    int chunk_bits;       // C
    int gray_bits;        // g
    int log2_bpc;         // log2(blocks per chunk)
    int n_moduli;
    uint32_t c80;         // 0x80808080, passed as data so that it stays in a register (SWAR drain: one LOP3 per masked operand)
    uint32_t ztab_shared; // SWAR: 1 = every block copies the zero-step tables (24 KB) into shared memory (long-lived blocks)
    uint64_t chunk_begin;
    uint64_t n_chunks;
    uint32_t* out;        // DEVICE rows
    unsigned long long* nonzero;  // DEVICE or nullptr
    MontPrime primes[PAIRINGS_MAX_MODULI];
};

// Launchers implemented in the .cu files.  Return cudaError_t as int.
typedef int (*swar_launch_fn)(const KernelParams& kp, int block_threads, unsigned grid, void* stream);
swar_launch_fn swar_lookup(int kind, int n);   // nullptr if not compiled for (kind, n)
int swar_min_gray_bits();                      // unrolled inner bits h
const char* swar_list();                       // "S12 S13 ... L28"

}  // namespace pairings
#endif
