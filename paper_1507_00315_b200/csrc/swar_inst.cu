// One SWAR specialisation per compilation: -DPAIRINGS_SWAR_KIND=<0|1> -DPAIRINGS_SWAR_N=<n>.
#include "swar_kernel.cuh"

#ifndef PAIRINGS_SWAR_KIND
#error "compile with -DPAIRINGS_SWAR_KIND=.. -DPAIRINGS_SWAR_N=.."
#endif

#define PAIRINGS_CAT3(a, b, c) a##b##_##c
#define PAIRINGS_NAME(k, n) PAIRINGS_CAT3(swar_launch_, k, n)

namespace pairings {
int PAIRINGS_NAME(PAIRINGS_SWAR_KIND, PAIRINGS_SWAR_N)(const KernelParams& kp, int block_threads, unsigned grid, void* stream) {
    return swar::launch<PAIRINGS_SWAR_KIND, PAIRINGS_SWAR_N>(kp, block_threads, grid, stream);
}
}  // namespace pairings
