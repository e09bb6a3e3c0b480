// Approximate counting by parallel tempering (§3, :259-325; Algorithm 2, :291-319) —
// SURVEY.md §8(f) NEXT #4, a second workload beside the exact count.
//
// One thread runs one replica of Algorithm 2: M configurations (one per inverse temperature), per
// iteration (in the paper's order) the ratio sample of every level, one Metropolis move per level,
// then the exchanges of neighbouring levels j = 1..M-1 in sequence.  Replicas are independent, so a
// launch is embarrassingly parallel; what comes back is integer only:
//     hist[j][E]  how often level j was seen with E empty bins  (Ratio(j) = sum_E hist[j][E] w_j(E), host)
//     moves[j], swaps[j]  accepted moves / exchanges (the W1, W2 columns of Table 6)
// Every random decision is "u < threshold" on 32-bit integers, the thresholds floor(p 2^32) are computed
// once on the host, and the generator is counter-based (readings C1-C3 in DESIGN.md), so the counters
// are reproducible bit for bit — that is what the parity tests compare with the oracle.
//
// State of a replica lives in shared memory, byte-interleaved over the block's threads:
//   pos[slot][k]   position a_k of colour k (bins a_k and a_k + d_k)            M x n bytes
//   occ[slot][b]   balls in bin b                                                M x (2n+1) bytes, or nibbles for n <= 15
//                  (a bin holds at most n balls; 4-bit counts shrink the state of S(12) x 12 levels from 468 to 324 bytes
//                  per replica: 10 instead of 7 blocks of 64 threads per SM — measured no faster, 8.5e10 moves/s either
//                  way: the kernel is bound by its dependent instruction chains, not by residency)
//   lev[j] = slot holding level j's configuration, E[j] its energy               2 M bytes
// An exchange swaps lev / E entries, not configurations.  The energy change of a move is counted
// incrementally from the occupancy of the four affected bins: bins that become empty minus bins that
// become occupied.
#include "pairings.h"
#include "internal.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstring>
#include <mutex>
#include <vector>

namespace pairings {

constexpr int PT_THREADS = 64;

struct PtParams {
    int kind, n, M;
    uint64_t replica_begin, replica_end, iterations, burn_in, seed;
    const uint64_t* move_thr;    // DEVICE, M x 2: threshold for dE = 1, 2
    const uint64_t* swap_thr;    // DEVICE, (M-1) x (2n+1): threshold for dE = E_j - E_{j+1} > 0
    unsigned long long *hist, *moves, *swaps;   // DEVICE
};

__device__ __forceinline__ uint64_t pt_mix64(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
__device__ __forceinline__ uint64_t pt_draw(uint64_t seed, uint64_t ctr) {
    return pt_mix64(seed + 0x9E3779B97F4A7C15ULL * (ctr + 1));
}

template <bool NIB>
__global__ void __launch_bounds__(PT_THREADS) pt_kernel(const PtParams p) {
    extern __shared__ unsigned char smem_raw[];
    const int n = p.n, N = 2 * n, M = p.M, kind = p.kind;
    const int tid = threadIdx.x, BD = PT_THREADS;
    // block counters first (32-bit, flushed at the end), then the byte-interleaved replica state
    unsigned int* shist = reinterpret_cast<unsigned int*>(smem_raw);           // M x (N+1)
    unsigned int* smoves = shist + M * (N + 1);                                 // M
    unsigned int* sswaps = smoves + M;                                          // M
    unsigned char* st = reinterpret_cast<unsigned char*>(sswaps + M);
    const int OB = NIB ? (N + 2) / 2 : N + 1;                                   // occupancy bytes per configuration
    const int POS = 0, OCC = M * n, LEV = OCC + M * OB, EN = LEV + M;           // byte offsets of the per-thread state
#define ST(i) st[(i) * BD + tid]
    auto occ_get = [&](int ob, int b) -> int {
        if (NIB) return ((int)ST(ob + (b >> 1)) >> ((b & 1) * 4)) & 15;
        return (int)ST(ob + b);
    };
    auto occ_add = [&](int ob, int b, int delta) {       // a count stays in [0, n]: no carry or borrow leaves its nibble
        if (NIB) ST(ob + (b >> 1)) = (unsigned char)((int)ST(ob + (b >> 1)) + delta * (1 << ((b & 1) * 4)));
        else ST(ob + b) = (unsigned char)((int)ST(ob + b) + delta);
    };
    for (int i = tid; i < M * (N + 1) + 2 * M; i += BD) shist[i] = 0;
    __syncthreads();

    const uint64_t r = p.replica_begin + (uint64_t)blockIdx.x * BD + tid;
    const bool active = r < p.replica_end;
    const uint64_t S = n > 3 ? n : 3, T = p.iterations, seed = p.seed;

    if (active) {
        // ---- "C(i) <- a random configuration"
        for (int j = 0; j < M; j++) {
            for (int b = 0; b < OB; b++) ST(OCC + j * OB + b) = 0;
            for (int k = 1; k <= n; k++) {
                const int d = dist(kind, k);
                const uint64_t u = pt_draw(seed, ((r * (T + 1)) * M + j) * S + (k - 1)) >> 32;
                const int a = 1 + (int)((u * (uint64_t)(N - d)) >> 32);
                ST(POS + j * n + (k - 1)) = (unsigned char)a;
                occ_add(OCC + j * OB, a, 1);
                occ_add(OCC + j * OB, a + d, 1);
            }
            int e = 0;
            for (int b = 1; b <= N; b++) e += (occ_get(OCC + j * OB, b) == 0);
            ST(LEV + j) = (unsigned char)j;
            ST(EN + j) = (unsigned char)e;
        }
        for (uint64_t t = 0; t < T; t++) {
            const uint64_t base = (r * (T + 1) + (t + 1)) * M;
            // ---- step 1: ratio samples
            const bool counted = t >= p.burn_in;
            // (Measured: without these atomics the kernel is 6 % faster; electing one lane per distinct energy with
            // match.any costs more than the same-address atomics it saves: 7.4e10 against 8.5e10 moves/s.)
            if (counted) for (int j = 0; j < M; j++) atomicAdd(&shist[j * (N + 1) + ST(EN + j)], 1u);
            // ---- step 2: one move per level.  A move is evaluated from loads only (the four affected bins and
            // the old position), so the moves of two levels — different configurations — are evaluated together
            // and their dependent load chains overlap; shared memory is written only when a move is accepted.
            // (Four levels at a time measured no faster: 8.3e10 against 8.5-8.7e10 moves/s.)
            struct Move { int slot, k, d, a0, a1, dE, j; };
            auto evaluate = [&](int j) -> Move {
                Move m; m.j = j;
                m.slot = ST(LEV + j);
                const uint64_t w = pt_draw(seed, (base + j) * S + 0);
                m.k = 1 + (int)(((w & 0xFFFFFFFFULL) * (uint64_t)n) >> 32);
                m.d = dist(kind, m.k);
                m.a1 = 1 + (int)(((w >> 32) * (uint64_t)(N - m.d)) >> 32);
                m.a0 = ST(POS + m.slot * n + (m.k - 1));
                const int ob = OCC + m.slot * OB;
                const int c0 = occ_get(ob, m.a0), c1 = occ_get(ob, m.a0 + m.d), c2 = occ_get(ob, m.a1), c3 = occ_get(ob, m.a1 + m.d);
                // bins that become empty when the pair leaves (a0 != a0+d), minus bins that are empty after that
                // and become occupied when it lands (a1 != a1+d); a bin left and re-entered counts in both
                const int e2 = (m.a1 == m.a0) + (m.a1 == m.a0 + m.d), e3 = (m.a1 + m.d == m.a0) + (m.a1 + m.d == m.a0 + m.d);
                m.dE = (c0 == 1) + (c1 == 1) - (c2 - e2 == 0) - (c3 - e3 == 0);
                return m;
            };
            auto commit = [&](const Move& m) {
                bool accept = m.dE <= 0;
                if (!accept) {
                    const uint64_t u = pt_draw(seed, (base + m.j) * S + 1) >> 32;
                    accept = u < p.move_thr[m.j * 2 + (m.dE - 1)];
                }
                if (accept) {
                    const int ob = OCC + m.slot * OB;
                    occ_add(ob, m.a0, -1); occ_add(ob, m.a0 + m.d, -1); occ_add(ob, m.a1, 1); occ_add(ob, m.a1 + m.d, 1);
                    ST(POS + m.slot * n + (m.k - 1)) = (unsigned char)m.a1;
                    ST(EN + m.j) = (unsigned char)((int)ST(EN + m.j) + m.dE);
                    if (counted) atomicAdd(&smoves[m.j], 1u);
                }
            };
            int j2 = 0;
            for (; j2 + 1 < M; j2 += 2) {
                const Move ma = evaluate(j2), mb = evaluate(j2 + 1);
                commit(ma); commit(mb);
            }
            if (j2 < M) commit(evaluate(j2));
            // ---- step 3: exchanges j, j+1 in sequence
            for (int j = 0; j + 1 < M; j++) {
                const int e0 = ST(EN + j), e1 = ST(EN + j + 1), dE = e0 - e1;
                bool accept = dE <= 0;
                if (!accept) {
                    const uint64_t u = pt_draw(seed, (base + j) * S + 2) >> 32;
                    accept = u < p.swap_thr[j * (N + 1) + dE];
                }
                if (accept) {
                    const unsigned char l0 = ST(LEV + j);
                    ST(LEV + j) = ST(LEV + j + 1); ST(LEV + j + 1) = l0;
                    ST(EN + j) = (unsigned char)e1; ST(EN + j + 1) = (unsigned char)e0;
                    if (counted) atomicAdd(&sswaps[j], 1u);
                }
            }
        }
    }
#undef ST
    __syncthreads();
    for (int i = tid; i < M * (N + 1); i += BD) if (shist[i]) atomicAdd(&p.hist[i], (unsigned long long)shist[i]);
    for (int i = tid; i < M; i += BD) {
        if (smoves[i]) atomicAdd(&p.moves[i], (unsigned long long)smoves[i]);
        if (sswaps[i]) atomicAdd(&p.swaps[i], (unsigned long long)sswaps[i]);
    }
}

static uint64_t pt_threshold(double prob) {
    if (prob >= 1.0) return 1ULL << 32;
    return (uint64_t)std::floor(prob * 4294967296.0);
}

static int pt_check(int kind, int n, const double* betas, int n_levels) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    if (!betas) return PAIRINGS_ENULL;
    if (n_levels < 1 || n_levels > PAIRINGS_PT_MAX_LEVELS) return PAIRINGS_EINVAL_OPTS;
    if (betas[0] != 0.0) return PAIRINGS_EINVAL_OPTS;                 // Z(0) is the closed form the estimate starts from
    for (int j = 1; j < n_levels; j++) if (!(betas[j] > betas[j - 1]) || !std::isfinite(betas[j])) return PAIRINGS_EINVAL_OPTS;
    return PAIRINGS_OK;
}

// ---- pairings_pt_run_noalloc: the threshold table in a fixed array of the library's own instead of cudaMallocAsync.
// Every GPU that loads this library holds these 16 KiB until the process exits.  The name is usable as it stands only
// in device code: on the host it is a stand-in symbol, not a device pointer — a kernel handed `pt_static_thr` itself
// would fault (or quietly read host memory on systems where the GPU can reach it).  Host code therefore asks the
// runtime for the real address, once per device with that device current, and passes that to the kernel.
static __device__ __align__(256) unsigned long long pt_static_thr[PAIRINGS_PT_STATIC_WORDS];

// Device address of pt_static_thr on the current device (looked up on the first call per device, then remembered).
static int pt_static_address(uint64_t** out) {
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static uint64_t* known[MAX_DEV] = {};
    int dev = -1;
    (void)cudaGetLastError();
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    std::lock_guard<std::mutex> lock(mu);
    if (dev < MAX_DEV && known[dev]) { *out = known[dev]; return PAIRINGS_OK; }
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, pt_static_thr);
    if (e != cudaSuccess || ptr == nullptr) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    if (dev < MAX_DEV) known[dev] = (uint64_t*)ptr;
    *out = (uint64_t*)ptr;
    return PAIRINGS_OK;
}

}  // namespace pairings

using namespace pairings;

extern "C" {

int pairings_pt_run(int kind, int n, const double* betas, int n_levels,
                    uint64_t replica_begin, uint64_t replica_end, uint64_t iterations, uint64_t burn_in, uint64_t seed,
                    uint64_t* hist_dev, uint64_t* moves_dev, uint64_t* swaps_dev, void* stream) {
    int rc = pt_check(kind, n, betas, n_levels); if (rc) return rc;
    if (replica_begin > replica_end || iterations == 0 || iterations > (1ULL << 25) || burn_in >= iterations) return PAIRINGS_EINVAL_OPTS;
    if (replica_end > (1ULL << 30)) return PAIRINGS_EINVAL_OPTS;
    {   // the draw counter ((r (T+1) + tt) M + j) S + slot, S = max(n, 3), must stay below 2^64: otherwise it wraps and two
        // replicas share a random stream (the oracle wraps the same way, so parity would not show it)
        const unsigned __int128 span = (unsigned __int128)replica_end * (iterations + 1) * (unsigned)n_levels * (unsigned)(n > 3 ? n : 3);
        if (span >> 64) return PAIRINGS_EINVAL_OPTS;
    }
    if (!hist_dev || !moves_dev || !swaps_dev) return PAIRINGS_ENULL;
    if (replica_begin == replica_end) return PAIRINGS_OK;
    const int M = n_levels, N = 2 * n;
    std::vector<uint64_t> thr((size_t)(M * 2 + M * (N + 1)), 0);
    for (int j = 0; j < M; j++)
        for (int dE = 1; dE <= 2; dE++) thr[(size_t)(j * 2 + dE - 1)] = pt_threshold(std::exp(-betas[j] * (double)dE));
    for (int j = 0; j + 1 < M; j++)
        for (int dE = 1; dE <= N; dE++)
            thr[(size_t)(M * 2 + j * (N + 1) + dE)] = pt_threshold(std::exp(-(betas[j + 1] - betas[j]) * (double)dE));

    cudaStream_t s = (cudaStream_t)stream;
    (void)cudaGetLastError();
    uint64_t* dthr = nullptr;
    if (cudaMallocAsync((void**)&dthr, thr.size() * sizeof(uint64_t), s) != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    cudaError_t e = cudaMemcpyAsync(dthr, thr.data(), thr.size() * sizeof(uint64_t), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);               // thr is a local: the copy must have left it
    PtParams p; std::memset(&p, 0, sizeof p);
    p.kind = kind; p.n = n; p.M = M;
    p.replica_begin = replica_begin; p.replica_end = replica_end; p.iterations = iterations; p.burn_in = burn_in; p.seed = seed;
    p.move_thr = dthr; p.swap_thr = dthr + M * 2;
    p.hist = (unsigned long long*)hist_dev; p.moves = (unsigned long long*)moves_dev; p.swaps = (unsigned long long*)swaps_dev;
    const bool nib = n <= 15;                                         // a bin holds at most n balls: 4-bit counts
    const size_t occ_bytes = nib ? (size_t)(N + 2) / 2 : (size_t)(N + 1);
    const size_t smem = (size_t)(M * (N + 1) + 2 * M) * sizeof(unsigned int)
                      + (size_t)PT_THREADS * ((size_t)M * n + (size_t)M * occ_bytes + 2 * (size_t)M);
    auto kernel = nib ? pt_kernel<true> : pt_kernel<false>;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) {
        const uint64_t blocks = (replica_end - replica_begin + PT_THREADS - 1) / PT_THREADS;
        kernel<<<(unsigned)blocks, PT_THREADS, smem, s>>>(p);
        e = cudaGetLastError();
    }
    cudaError_t e2 = cudaFreeAsync(dthr, s);
    if (e != cudaSuccess || e2 != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    return PAIRINGS_OK;
}

// Same replicas, same kernel, same counters as pairings_pt_run, for callers that may not allocate on the device
// (include/pairings.h says who and why).  No cudaMalloc*/cudaFree*, no std::vector: the table is built in a stack
// array and staged into pt_static_thr, which every call on this device shares — see the header for the race rule.
int pairings_pt_run_noalloc(int kind, int n, const double* betas, int n_levels,
                            uint64_t replica_begin, uint64_t replica_end, uint64_t iterations, uint64_t burn_in, uint64_t seed,
                            uint64_t* hist_dev, uint64_t* moves_dev, uint64_t* swaps_dev, void* stream) {
    int rc = pt_check(kind, n, betas, n_levels); if (rc) return rc;
    if (replica_begin > replica_end || iterations == 0 || iterations > (1ULL << 25) || burn_in >= iterations) return PAIRINGS_EINVAL_OPTS;
    if (replica_end > (1ULL << 30)) return PAIRINGS_EINVAL_OPTS;
    {   // the draw counter must not wrap (as in pairings_pt_run)
        const unsigned __int128 span = (unsigned __int128)replica_end * (iterations + 1) * (unsigned)n_levels * (unsigned)(n > 3 ? n : 3);
        if (span >> 64) return PAIRINGS_EINVAL_OPTS;
    }
    const int M = n_levels, N = 2 * n;
    const size_t words = (size_t)M * 2 + (size_t)M * (size_t)(N + 1);          // move thresholds, then exchange thresholds
    if (words > (size_t)PAIRINGS_PT_STATIC_WORDS) return PAIRINGS_ETOOBIG;     // refused before anything is enqueued
    if (!hist_dev || !moves_dev || !swaps_dev) return PAIRINGS_ENULL;
    if (replica_begin == replica_end) return PAIRINGS_OK;

    // All `words` entries are written, also the ones no decision ever reads (dE = 0, the row above the last level):
    // the array still holds the previous call's table and none of it may survive inside this call's extent.
    uint64_t thr[PAIRINGS_PT_STATIC_WORDS];
    for (size_t i = 0; i < words; i++) thr[i] = 0;
    for (int j = 0; j < M; j++)
        for (int dE = 1; dE <= 2; dE++) thr[(size_t)(j * 2 + dE - 1)] = pt_threshold(std::exp(-betas[j] * (double)dE));
    for (int j = 0; j + 1 < M; j++)
        for (int dE = 1; dE <= N; dE++)
            thr[(size_t)(M * 2 + j * (N + 1) + dE)] = pt_threshold(std::exp(-(betas[j + 1] - betas[j]) * (double)dE));

    uint64_t* table = nullptr;                                                 // DEVICE address of pt_static_thr
    rc = pt_static_address(&table); if (rc) return rc;                         // first call on this device: the set-up

    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(table, thr, words * sizeof(uint64_t), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);                        // thr is a local: the copy must have left it
    PtParams p; std::memset(&p, 0, sizeof p);
    p.kind = kind; p.n = n; p.M = M;
    p.replica_begin = replica_begin; p.replica_end = replica_end; p.iterations = iterations; p.burn_in = burn_in; p.seed = seed;
    p.move_thr = table; p.swap_thr = table + M * 2;
    p.hist = (unsigned long long*)hist_dev; p.moves = (unsigned long long*)moves_dev; p.swaps = (unsigned long long*)swaps_dev;
    const bool nib = n <= 15;
    const size_t occ_bytes = nib ? (size_t)(N + 2) / 2 : (size_t)(N + 1);
    const size_t smem = (size_t)(M * (N + 1) + 2 * M) * sizeof(unsigned int)
                      + (size_t)PT_THREADS * ((size_t)M * n + (size_t)M * occ_bytes + 2 * (size_t)M);
    auto kernel = nib ? pt_kernel<true> : pt_kernel<false>;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) {
        const uint64_t blocks = (replica_end - replica_begin + PT_THREADS - 1) / PT_THREADS;
        kernel<<<(unsigned)blocks, PT_THREADS, smem, s>>>(p);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    return PAIRINGS_OK;
}

// Ladder choice ("the inverse temperatures are chosen such that the acceptance rates for the
// configuration exchanges are no smaller than one half", with as few levels as that allows).  Built level by
// level: a short pilot run of the ladder so far gives the energy distribution p(E) of its last level; the next
// beta is the one for which the predicted exchange acceptance
//     A(db) = sum_{E,E'} p(E) q(E') min[1, exp(-db (E - E'))],   q(E') ~ p(E') exp(-db E')   (p reweighted to beta + db)
// equals the target (bisection; A falls from 1 as db grows; at most a doubling of beta per level).  Stops when the
// last level sits at E = 0 with probability >= 0.98 or beta >= 32 (the remaining factor to beta = infinity is ~1).
int pairings_pt_ladder(int kind, int n, double target_exchange, uint64_t pilot_replicas, uint64_t pilot_iterations,
                       uint64_t seed, double* betas_out, int cap_levels, void* stream) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    if (!betas_out) return PAIRINGS_ENULL;
    if (!(target_exchange > 0.05 && target_exchange < 0.95) || cap_levels < 1 || pilot_replicas == 0 ||
        pilot_iterations < 2 || pilot_iterations > (1ULL << 25)) return PAIRINGS_EINVAL_OPTS;
    const int N = 2 * n, cap = cap_levels < PAIRINGS_PT_MAX_LEVELS ? cap_levels : PAIRINGS_PT_MAX_LEVELS;
    cudaStream_t s = (cudaStream_t)stream;
    std::vector<double> betas(1, 0.0);
    const size_t words = (size_t)PAIRINGS_PT_MAX_LEVELS * (size_t)(N + 1) + 2 * PAIRINGS_PT_MAX_LEVELS;
    uint64_t* dev = nullptr;
    (void)cudaGetLastError();
    if (cudaMallocAsync((void**)&dev, words * sizeof(uint64_t), s) != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    std::vector<uint64_t> host(words);
    int result = PAIRINGS_ERANGE;                                      // cap reached before the ladder is cold enough
    for (;;) {
        const int M = (int)betas.size();
        cudaError_t e = cudaMemsetAsync(dev, 0, words * sizeof(uint64_t), s);
        if (e != cudaSuccess) { result = PAIRINGS_ECUDA; break; }
        rc = pairings_pt_run(kind, n, betas.data(), M, 0, pilot_replicas, pilot_iterations, pilot_iterations / 2,
                             seed + (uint64_t)M, dev, dev + (size_t)PAIRINGS_PT_MAX_LEVELS * (N + 1),
                             dev + (size_t)PAIRINGS_PT_MAX_LEVELS * (N + 1) + PAIRINGS_PT_MAX_LEVELS, s);
        if (rc) { result = rc; break; }
        e = cudaMemcpyAsync(host.data(), dev, words * sizeof(uint64_t), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { result = PAIRINGS_ECUDA; break; }
        std::vector<double> pE((size_t)N + 1);
        double tot = 0;
        for (int E = 0; E <= N; E++) { pE[E] = (double)host[(size_t)(M - 1) * (N + 1) + E]; tot += pE[E]; }
        for (int E = 0; E <= N; E++) pE[E] /= tot;
        if (pE[0] >= 0.98 || betas.back() >= 32.0) { result = M; break; }   // cold enough: the factor to beta = infinity is ~1
        if (M == cap) break;
        auto acceptance = [&](double db) {
            std::vector<double> q((size_t)N + 1);
            double z = 0;
            for (int E = 0; E <= N; E++) { q[E] = pE[E] * std::exp(-db * E); z += q[E]; }
            double a = 0;
            for (int E = 0; E <= N; E++)
                for (int F = 0; F <= N; F++)
                    a += pE[E] * (q[F] / z) * (E <= F ? 1.0 : std::exp(-db * (double)(E - F)));
            return a;
        };
        // at most a doubling per level (the cold end of Table 6 goes 8.1, 16, 32): with only E in {0, 1} left the
        // predicted acceptance no longer falls to the target
        double lo = 0.0, hi = betas.back() > 1.0 ? betas.back() : 1.0;
        for (int it = 0; it < 60; it++) {
            const double mid = 0.5 * (lo + hi);
            if (acceptance(mid) > target_exchange) lo = mid; else hi = mid;
        }
        betas.push_back(betas.back() + 0.5 * (lo + hi));
    }
    cudaError_t e2 = cudaFreeAsync(dev, s);
    cudaError_t e3 = cudaStreamSynchronize(s);
    if (result > 0 && (e2 != cudaSuccess || e3 != cudaSuccess)) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    if (result > 0) for (int j = 0; j < result; j++) betas_out[j] = betas[(size_t)j];
    return result;
}

int pairings_pt_estimate(int kind, int n, const double* betas, int n_levels, const uint64_t* hist_host,
                         double* ratios_out, double* log_distinct_out) {
    int rc = pt_check(kind, n, betas, n_levels); if (rc) return rc;
    if (!hist_host || !ratios_out || !log_distinct_out) return PAIRINGS_ENULL;
    const int N = 2 * n;
    double logz = 0.0;                                                  // log Z(0) = sum_k log(2n - d_k)
    for (int k = 1; k <= n; k++) logz += std::log((double)(N - dist(kind, k)));
    for (int j = 0; j < n_levels; j++) {
        long double num = 0, den = 0;
        for (int E = 0; E <= N; E++) {
            const long double h = (long double)hist_host[(size_t)j * (N + 1) + E];
            den += h;
            if (j + 1 < n_levels) num += h * (long double)std::exp(-(betas[j + 1] - betas[j]) * (double)E);
            else if (E == 0) num += h;                                  // beta(M+1) = infinity
        }
        if (den == 0 || num == 0) return PAIRINGS_ERANGE;               // no samples, or a ratio estimated as zero
        ratios_out[j] = (double)(num / den);
        logz += std::log(ratios_out[j]);
    }
    *log_distinct_out = logz;
    return PAIRINGS_OK;
}

int pairings_pt_counts(int n, double log_distinct, double* distinct_out, double* identified_out) {
    if (n < 2 || n > 32) return PAIRINGS_EINVAL_N;
    if (!distinct_out || !identified_out) return PAIRINGS_ENULL;
    if (!std::isfinite(log_distinct)) return PAIRINGS_ERANGE;
    *distinct_out = std::exp(log_distinct);
    *identified_out = 0.5 * *distinct_out;          // n > 1: a pairing is never its own reflection
    return PAIRINGS_OK;
}

}  // extern "C"
