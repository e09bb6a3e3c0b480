// Integer-issue calibration kernels for the roofline denominator: independent
// dependency chains of one instruction class, ILP = 8 per thread.  MEASURED_PEAKS.json has no
// integer figure, so bench.py measures IADD3-only, LOP3-only, IMAD-only and a 1:1 IADD3:IMAD mix
// next to the formula peak 148 SM x 128 lanes x f_SM.
//
// A measurement helper of bench.py, NOT part of the product: it is built into its own
// libpairings_probe.so (paper_1507_00315_b200/build.py: build_probe) and libpairings_b200.so does not export it.
//
//   int pairings_issue_probe(int mode, int blocks, int threads, int iters, uint32_t* out_dev, void* stream,
//                            uint64_t* thread_instructions);
//   mode 0: IADD3, 1: LOP3, 2: IMAD, 3: IADD3:IMAD 1:1.  out_dev: DEVICE scratch, one uint32.  Enqueues one kernel and
//   reports how many thread-instructions of that class it executes.  Returns 0, -10 (bad argument), -5 (NULL), -6 (CUDA).
#include <stdint.h>

#include <cuda_runtime.h>

namespace pairings_probe {

constexpr int PROBE_ILP = 8;
constexpr int PROBE_UNROLL = 16;   // instructions per chain per loop iteration

template <int MODE>
__global__ void __launch_bounds__(256) issue_probe_kernel(int iters, uint32_t seed, uint32_t* out) {
    uint32_t a[PROBE_ILP];
    const uint32_t b = seed | 1u, c = seed * 2654435761u + threadIdx.x;
#pragma unroll
    for (int i = 0; i < PROBE_ILP; i++) a[i] = seed + threadIdx.x * 977u + i;
#pragma unroll 1
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; u++) {
#pragma unroll
            for (int i = 0; i < PROBE_ILP; i++) {
                if (MODE == 0) asm volatile("add.u32 %0, %0, %1;\n\tadd.u32 %0, %0, %2;" : "+r"(a[i]) : "r"(b), "r"(c)); // one IADD3
                else if (MODE == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b), "r"(c)); // LOP3
                else if (MODE == 2) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));   // IMAD
                else {
                    if ((i & 1) == 0) asm volatile("add.u32 %0, %0, %1;\n\tadd.u32 %0, %0, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
                    else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b), "r"(c));
                }
            }
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int i = 0; i < PROBE_ILP; i++) r ^= a[i];
    if (r == 0x12345678u) out[0] = r;   // practically never: keeps the chains alive
}

}  // namespace pairings_probe

using namespace pairings_probe;

extern "C" int pairings_issue_probe(int mode, int blocks, int threads, int iters, uint32_t* out_dev, void* stream,
                                    uint64_t* thread_instructions) {
    if (mode < 0 || mode > 3 || blocks < 1 || threads < 32 || threads > 256 || iters < 1) return -10;
    if (!out_dev || !thread_instructions) return -5;
    cudaStream_t s = (cudaStream_t)stream;
    (void)cudaGetLastError();
    switch (mode) {
        case 0: issue_probe_kernel<0><<<blocks, threads, 0, s>>>(iters, 12345u, out_dev); break;
        case 1: issue_probe_kernel<1><<<blocks, threads, 0, s>>>(iters, 12345u, out_dev); break;
        case 2: issue_probe_kernel<2><<<blocks, threads, 0, s>>>(iters, 12345u, out_dev); break;
        default: issue_probe_kernel<3><<<blocks, threads, 0, s>>>(iters, 12345u, out_dev); break;
    }
    if (cudaGetLastError() != cudaSuccess) return -6;
    *thread_instructions = (uint64_t)blocks * (uint64_t)threads * (uint64_t)iters * PROBE_UNROLL * PROBE_ILP;
    return 0;
}
