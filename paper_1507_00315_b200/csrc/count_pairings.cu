// count_pairings: argument validation, Montgomery constants, launch geometry, the GENERIC kernel
// (any kind, any 2 <= n <= 32), the host-buffer variant and the whole-job host driver.
//
// The generic kernel is north_star's description taken literally:
//   a2  each thread evaluates its prefix's n pair-sums directly (popcount of X ^ (X >> d_k)),
//   a3  walks its low g bits in binary-reflected Gray-code order, updating every
//       P_k by  -2 x_j (x_{j-d_k} + x_{j+d_k})  with both neighbours boundary-guarded,
//   a4  skips terms with a zero factor,
//   a5  multiplies the rest as exact <= 60-bit group products and one 32-bit Montgomery chain per
//       modulus ("calculations modulo number of co-primes"),
//   a6  reduces per thread -> warp shuffles -> shared memory -> one row per chunk.
// The specialised SWAR kernels (swar_kernel.cuh) are the fast path; this one is the fallback for
// every (kind, n) they are not compiled for and an independent second implementation of the rows.
#include "pairings.h"
#include "internal.h"
#include "device_common.cuh"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

namespace pairings {

// ------------------------------------------------------------------------------------------------
// host: Montgomery constants
// ------------------------------------------------------------------------------------------------
static MontPrime make_prime(uint32_t p) {
    MontPrime mp; std::memset(&mp, 0, sizeof mp);
    mp.p = p;
    uint32_t inv = p;                                  // Newton: inv = p^{-1} mod 2^32 (p odd; 3 correct bits to start)
    for (int i = 0; i < 5; i++) inv *= 2u - p * inv;
    mp.pinv_neg = 0u - inv;
    uint64_t r = 1;
    for (int i = 0; i < 32; i++) r = (r * 2) % p;
    mp.r1 = (uint32_t)r;
    for (int i = 0; i < 32; i++) r = (r * 2) % p;
    mp.r2 = (uint32_t)r;
    for (int i = 0; i < 32; i++) r = (r * 2) % p;
    mp.r3 = (uint32_t)r;
    return mp;
}

// ------------------------------------------------------------------------------------------------
// device helpers (montmul, atomic_add_mod, block_reduce_write: device_common.cuh)
// ------------------------------------------------------------------------------------------------
// Montgomery form (value * 2^32 mod p) of a signed 64-bit integer with |g| < 2^62
__device__ __forceinline__ uint32_t to_mont64(long long g, const MontPrime& mp) {
    const bool neg = g < 0;
    const unsigned long long a = neg ? 0ULL - (unsigned long long)g : (unsigned long long)g;
    uint32_t r = montmul((uint32_t)a, mp.r2, mp.p, mp.pinv_neg) + montmul((uint32_t)(a >> 32), mp.r3, mp.p, mp.pinv_neg);
    if (r >= mp.p) r -= mp.p;
    if (neg && r) r = mp.p - r;
    return r;
}

// ------------------------------------------------------------------------------------------------
// GENERIC kernel
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
generic_kernel(const __grid_constant__ KernelParams kp) {
    __shared__ unsigned long long red[8 * PAIRINGS_MAX_MODULI];
    const int n = kp.n, N = 2 * n, B = N - 1, C = kp.chunk_bits, g = kp.gray_bits;
    const int kind = kp.kind, M = kp.n_moduli;
    const uint64_t chunk_local = (uint64_t)blockIdx.x >> kp.log2_bpc;
    const uint64_t sub = (uint64_t)blockIdx.x & ((1ULL << kp.log2_bpc) - 1);
    const uint64_t chunk = kp.chunk_begin + chunk_local;
    const int tb = B - C;                               // index bits inside one chunk
    const uint64_t prefixes = 1ULL << (tb - g);          // thread prefixes per chunk
    const uint64_t per_block = prefixes >> kp.log2_bpc;  // >= 1 by construction
    const uint64_t chunk_base = (tb >= 64) ? 0 : (chunk << tb);

    unsigned long long acc[PAIRINGS_MAX_MODULI];
#pragma unroll
    for (int i = 0; i < PAIRINGS_MAX_MODULI; i++) acc[i] = 0;
    unsigned long long nz = 0;

    for (uint64_t q = sub * per_block + threadIdx.x; q < (sub + 1) * per_block; q += blockDim.x) {
        uint64_t V = chunk_base | (q << g);             // bit b <-> position N-b, set <-> x = -1
        int P[32];
#pragma unroll
        for (int k = 1; k <= 32; k++) {
            P[k - 1] = 1;
            if (k <= n) {
                const int d = dist(kind, k), cnt = N - d;          // cnt summands, 1 <= cnt <= 63
                const uint64_t mask = (1ULL << cnt) - 1;
                P[k - 1] = cnt - 2 * __popcll((V ^ (V >> d)) & mask);
            }
        }
        int sign = (__popcll(V) & 1) ? -1 : 1;
        const uint64_t steps = 1ULL << g;
        for (uint64_t t = 0; t < steps; t++) {
            // ---- a4: zero-factor test, a5: signed product -> residues
            bool zero = false;
#pragma unroll
            for (int k = 0; k < 32; k++) zero |= (P[k] == 0);
            if (!zero) {
                nz++;
                long long G0 = sign, G1 = 1, G2 = 1, G3 = 1;       // <= 10 factors of |P| <= 63 each: < 2^60
#pragma unroll
                for (int k = 0; k < 32; k++) {
                    if (k < 10) G0 *= P[k]; else if (k < 20) G1 *= P[k]; else if (k < 30) G2 *= P[k]; else G3 *= P[k];
                }
                for (int i = 0; i < M; i++) {
                    const MontPrime& mp = kp.primes[i];
                    uint32_t r = to_mont64(G0, mp);
                    if (n > 10) r = montmul(r, to_mont64(G1, mp), mp.p, mp.pinv_neg);
                    if (n > 20) r = montmul(r, to_mont64(G2, mp), mp.p, mp.pinv_neg);
                    if (n > 30) r = montmul(r, to_mont64(G3, mp), mp.p, mp.pinv_neg);
                    acc[i] += r;                                  // Montgomery form, < p < 2^31
                }
            }
            // ---- a3: Gray step t -> t+1 flips index bit ctz(t+1), i.e. position j = N - b
            if (t + 1 < steps) {
                const int b = __ffsll((long long)(t + 1)) - 1;
                const int xj = 1 - 2 * (int)((V >> b) & 1ULL);
#pragma unroll
                for (int k = 1; k <= 32; k++) {
                    if (k <= n) {
                        const int d = dist(kind, k);
                        int nb = 0;
                        if (b + d <= N - 1) nb += 1 - 2 * (int)((V >> (b + d)) & 1ULL);   // x_{j-d}, exists iff j-d >= 1
                        if (b - d >= 0) nb += 1 - 2 * (int)((V >> (b - d)) & 1ULL);       // x_{j+d}, exists iff j+d <= N
                        P[k - 1] -= 2 * xj * nb;
                    }
                }
                V ^= 1ULL << b;
                sign = -sign;
            }
        }
        // keep the 64-bit accumulators far from overflow across prefixes
#pragma unroll
        for (int i = 0; i < PAIRINGS_MAX_MODULI; i++) if (i < M && acc[i] >= (1ULL << 62)) acc[i] %= kp.primes[i].p;
    }

    uint32_t vals[PAIRINGS_MAX_MODULI];
#pragma unroll
    for (int i = 0; i < PAIRINGS_MAX_MODULI; i++) {
        vals[i] = 0;
        if (i < M) {
            const MontPrime& mp = kp.primes[i];
            vals[i] = montmul((uint32_t)(acc[i] % mp.p), 1u, mp.p, mp.pinv_neg);   // out of Montgomery form
        }
    }
    block_reduce_write(kp, vals, nz, red, chunk_local);
}

// ------------------------------------------------------------------------------------------------
// host: geometry + launch
// ------------------------------------------------------------------------------------------------
static int ilog2_floor(uint64_t v) { int r = 0; while (v >>= 1) r++; return r; }
static bool is_pow2(uint64_t v) { return v && !(v & (v - 1)); }

struct Geometry { int variant, g, threads, log2_bpc; };

static int choose_geometry(int kind, int n, int chunk_bits, uint64_t n_chunks,
                           const pairings_launch_opts* o, Geometry* out) {
    const int tb = 2 * n - 1 - chunk_bits;               // index bits inside one chunk
    int variant = o ? o->variant : PAIRINGS_VARIANT_AUTO;
    if (variant < 0 || variant > PAIRINGS_VARIANT_SWAR) return PAIRINGS_EINVAL_OPTS;
    int g = o ? o->gray_bits : 0, threads = o ? o->block_threads : 0, bpc = o ? o->blocks_per_chunk : 0;
    if (g < 0 || threads < 0 || bpc < 0) return PAIRINGS_EINVAL_OPTS;
    if (threads != 0 && (threads < 32 || threads > 256 || threads % 32)) return PAIRINGS_EINVAL_OPTS;
    if (bpc != 0 && (!is_pow2((uint64_t)bpc) || bpc > (1 << 20))) return PAIRINGS_EINVAL_OPTS;
    const int total_bits = tb + ilog2_floor(std::max<uint64_t>(n_chunks, 1));

    // ---- SWAR: whole warps of prefixes per block, every left neighbour of a walked bit exists
    // (g <= n-2), power-of-two threads, at most 2^32 steps per thread (accumulator width).
    const int h = swar_min_gray_bits();
    const int swar_gmax = std::min(std::min(n - 2, 24), tb - 5);
    bool swar_ok = swar_lookup(kind, n) != nullptr && swar_gmax >= h;
    if (swar_ok && g != 0 && (g < h || g > swar_gmax)) swar_ok = false;
    if (swar_ok && threads != 0 && !is_pow2((uint64_t)threads)) swar_ok = false;
    if (swar_ok) {
        // Gray bits per thread prefix: about 2^19 threads per launch (a few waves of blocks) with at most 2^14 steps each;
        // small jobs take at least 2^7 steps per prefix so that the direct evaluation of the prefix (~300 instructions)
        // and the per-thread residue reduction are amortised (measured: L(12) 28 -> 19 us, S(13) 57 -> 46 us per count)
        int sg = g ? g : std::max(h, std::min(std::max(total_bits - 19, 7), std::min(swar_gmax, 14)));
        const int pb = tb - sg;                           // log2(prefixes per chunk) >= 5
        int st = threads ? threads : std::min(256, 1 << std::min(pb, 8));
        int sb = bpc;
        if (sb == 0) {
            sb = 1;
            const uint64_t want_blocks = 148ULL * 8;
            while (n_chunks * (uint64_t)sb < want_blocks && pb - ilog2_floor((uint64_t)sb) - 1 >= ilog2_floor((uint64_t)st) && sb < (1 << 20)) sb *= 2;
            while (tb - ilog2_floor((uint64_t)sb) - ilog2_floor((uint64_t)st) > 32 && sb < (1 << 20)) sb *= 2;
            // long chunks (2^27 sign vectors at n = 24, C = 20) as several blocks of at most 2^24: a block then runs
            // ~25 ms instead of 200 ms and the last, partly filled wave of a launch costs 1 % instead of 8 %
            while (tb - ilog2_floor((uint64_t)sb) > 24 && pb - ilog2_floor((uint64_t)sb) - 1 >= ilog2_floor((uint64_t)st) && sb < (1 << 20)) sb *= 2;
        }
        const int lb = ilog2_floor((uint64_t)sb);
        if (pb - lb < ilog2_floor((uint64_t)st) || tb - lb - ilog2_floor((uint64_t)st) > 32) swar_ok = false;
        else if (variant != PAIRINGS_VARIANT_GENERIC) {
            out->variant = PAIRINGS_VARIANT_SWAR; out->g = sg; out->threads = st; out->log2_bpc = lb;
            return PAIRINGS_OK;
        }
    }
    if (variant == PAIRINGS_VARIANT_SWAR) return PAIRINGS_EINVAL_OPTS;

    // ---- generic
    const int gmax = std::min(tb, 32);                    // 2^g residues below 2^31 plus the 2^62 carried between prefixes stay below 2^64
    if (g != 0) { if (g > gmax) return PAIRINGS_EINVAL_OPTS; }
    else g = std::max(0, std::min(total_bits - 20, std::min(gmax, 12)));
    if (threads == 0) {
        threads = 256;
        const int pb = tb - g;
        if (pb < 8) threads = std::max(32, 1 << pb);
    }
    const uint64_t prefixes = 1ULL << std::min(tb - g, 62);
    if (bpc != 0) { if ((uint64_t)bpc > prefixes) return PAIRINGS_EINVAL_OPTS; }
    else {
        bpc = 1;
        const uint64_t want_blocks = 148ULL * 16;
        while (n_chunks * (uint64_t)bpc < want_blocks && (uint64_t)bpc * 2 * (uint64_t)threads <= prefixes && bpc < (1 << 20)) bpc *= 2;
    }
    out->variant = PAIRINGS_VARIANT_GENERIC; out->g = g; out->threads = threads; out->log2_bpc = ilog2_floor((uint64_t)bpc);
    return PAIRINGS_OK;
}

static int validate(int kind, int n, int chunk_bits, uint64_t b, uint64_t e, const uint32_t* moduli, int n_moduli, const void* out) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, b, e); if (rc) return rc;
    rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    if (!out && e > b) return PAIRINGS_ENULL;
    return PAIRINGS_OK;
}

// One memory pool per device for count_pairings_host's staging rows (created on first use, never destroyed).
static cudaMemPool_t staging_pool() {
    static std::mutex mu;
    static cudaMemPool_t pools[64] = {};
    static bool tried[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!tried[dev]) {
        tried[dev] = true;
        cudaMemPoolProps props; std::memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t p = nullptr;
        if (cudaMemPoolCreate(&p, &props) == cudaSuccess) {
            unsigned long long keep = 64ULL << 20;
            (void)cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
            pools[dev] = p;
        } else (void)cudaGetLastError();
    }
    return pools[dev];
}

static int launch_range(int kind, int n, int chunk_bits, uint64_t chunk_begin, uint64_t chunk_end,
                        const uint32_t* moduli, int n_moduli, uint32_t* out, cudaStream_t stream,
                        const pairings_launch_opts* opts) {
    const uint64_t n_chunks = chunk_end - chunk_begin;
    if (n_chunks == 0) return PAIRINGS_OK;
    Geometry geo;
    int rc = choose_geometry(kind, n, chunk_bits, n_chunks, opts, &geo); if (rc) return rc;

    KernelParams kp; std::memset(&kp, 0, sizeof kp);
    kp.kind = kind; kp.n = n; kp.chunk_bits = chunk_bits; kp.gray_bits = geo.g; kp.log2_bpc = geo.log2_bpc;
    kp.n_moduli = n_moduli; kp.c80 = 0x80808080u;
    // SWAR: a block that evaluates at least 2^22 sign vectors copies the zero-step tables into shared memory (measured:
    // L(20) +3.4 %, S(24) +4.2 %; the 24 KB copy costs short-lived blocks more than it saves: L(12) 19 -> 25 us)
    kp.ztab_shared = (2 * n - 1 - chunk_bits - geo.log2_bpc >= 22) ? 1u : 0u;
    kp.nonzero = opts ? (unsigned long long*)opts->nonzero_terms : nullptr;
    for (int i = 0; i < n_moduli; i++) kp.primes[i] = make_prime(moduli[i]);

    (void)cudaGetLastError();
    if (geo.log2_bpc > 0) {
        if (cudaMemsetAsync(out, 0, n_chunks * (uint64_t)n_moduli * sizeof(uint32_t), stream) != cudaSuccess) {
            (void)cudaGetLastError(); return PAIRINGS_ECUDA;
        }
    }
    // at most 2^30 blocks per launch
    const uint64_t max_chunks_per_launch = std::max<uint64_t>(1, (1ULL << 30) >> geo.log2_bpc);
    swar_launch_fn swar = geo.variant == PAIRINGS_VARIANT_SWAR ? swar_lookup(kind, n) : nullptr;
    for (uint64_t off = 0; off < n_chunks; off += max_chunks_per_launch) {
        const uint64_t cnt = std::min(max_chunks_per_launch, n_chunks - off);
        kp.chunk_begin = chunk_begin + off; kp.n_chunks = cnt;
        kp.out = out + off * (uint64_t)n_moduli;
        const unsigned grid = (unsigned)(cnt << geo.log2_bpc);
        cudaError_t err;
        if (swar) err = (cudaError_t)swar(kp, geo.threads, grid, (void*)stream);
        else { generic_kernel<<<grid, geo.threads, 0, stream>>>(kp); err = cudaGetLastError(); }
        if (err != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    }
    return PAIRINGS_OK;
}

}  // namespace pairings

using namespace pairings;

extern "C" {

int count_pairings_ex(int kind, int n, int chunk_bits, uint64_t chunk_begin, uint64_t chunk_end,
                      const uint32_t* moduli, int n_moduli, uint32_t* out_residues, void* stream,
                      const pairings_launch_opts* opts) {
    int rc = validate(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, n_moduli, out_residues); if (rc) return rc;
    return launch_range(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, n_moduli, out_residues, (cudaStream_t)stream, opts);
}

int count_pairings(int kind, int n, int chunk_bits, uint64_t chunk_begin, uint64_t chunk_end,
                   const uint32_t* moduli, int n_moduli, uint32_t* out_residues, void* stream) {
    return count_pairings_ex(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, n_moduli, out_residues, stream, nullptr);
}

int pairings_query_geometry(int kind, int n, int chunk_bits, uint64_t n_chunks, const pairings_launch_opts* opts,
                            int* variant_out, int* gray_bits_out, int* block_threads_out, int* blocks_per_chunk_out) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, 0, 0); if (rc) return rc;
    if (n_chunks == 0 || (chunk_bits < 64 && n_chunks > (1ULL << chunk_bits))) return PAIRINGS_EINVAL_CHUNK;
    Geometry geo; rc = choose_geometry(kind, n, chunk_bits, n_chunks, opts, &geo); if (rc) return rc;
    if (variant_out) *variant_out = geo.variant;
    if (gray_bits_out) *gray_bits_out = geo.g;
    if (block_threads_out) *block_threads_out = geo.threads;
    if (blocks_per_chunk_out) *blocks_per_chunk_out = 1 << geo.log2_bpc;
    return PAIRINGS_OK;
}

int pairings_has_swar(int kind, int n) {
    if (check_kind_n(kind, n)) return 0;
    return swar_lookup(kind, n) != nullptr ? 1 : 0;
}

int count_pairings_host(int kind, int n, int chunk_bits, uint64_t chunk_begin, uint64_t chunk_end,
                        const uint32_t* moduli, int n_moduli, uint32_t* out_residues_host, void* stream,
                        const pairings_launch_opts* opts) {
    int rc = validate(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, n_moduli, out_residues_host); if (rc) return rc;
    const uint64_t n_chunks = chunk_end - chunk_begin;
    if (n_chunks == 0) return PAIRINGS_OK;
    {   // options are validated before anything is allocated
        Geometry geo; rc = choose_geometry(kind, n, chunk_bits, n_chunks, opts, &geo); if (rc) return rc;
    }
    cudaStream_t s = (cudaStream_t)stream;
    const size_t bytes = n_chunks * (size_t)n_moduli * sizeof(uint32_t);
    uint32_t* dev = nullptr;
    (void)cudaGetLastError();
    // The staging rows come from a pool of the library's own that keeps up to 64 MiB between calls: with the
    // default pool (release threshold 0) every synchronise hands the memory back to the driver, and the next
    // call's allocation was measured to cost up to 0.5 s.
    cudaMemPool_t pool = staging_pool();
    cudaError_t ea = pool ? cudaMallocFromPoolAsync((void**)&dev, bytes, pool, s) : cudaMallocAsync((void**)&dev, bytes, s);
    if (ea != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    rc = launch_range(kind, n, chunk_bits, chunk_begin, chunk_end, moduli, n_moduli, dev, s, opts);
    cudaError_t e1 = cudaSuccess;
    if (rc == PAIRINGS_OK) e1 = cudaMemcpyAsync(out_residues_host, dev, bytes, cudaMemcpyDeviceToHost, s);
    cudaError_t e2 = cudaFreeAsync(dev, s);
    cudaError_t e3 = cudaStreamSynchronize(s);
    if (rc) return rc;
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) { (void)cudaGetLastError(); return PAIRINGS_ECUDA; }
    return PAIRINGS_OK;
}

// the host driver; apply_symmetry: double the complete x_2 = +1 half (pairings_run_ex) or leave the raw sum (a slice)
static int run_impl(int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli,
                    uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                    void* stream, const pairings_launch_opts* opts, unsigned flags,
                    uint64_t slice_begin, uint64_t slice_end, bool apply_symmetry,
                    uint32_t* total_out, uint64_t* chunks_done_out, uint64_t* chunks_needed_out,
                    uint64_t* duplicate_mismatches_out) {
    int rc = validate(kind, n, chunk_bits, slice_begin, slice_end, moduli, n_moduli, total_out); if (rc) return rc;
    if (!total_out || !chunks_done_out) return PAIRINGS_ENULL;
    if (chunks_per_call == 0) return PAIRINGS_EINVAL_CHUNK;
    if (flags & ~(unsigned)(PAIRINGS_RUN_LEMMA24 | PAIRINGS_RUN_DUPLICATE | PAIRINGS_RUN_AUDIT)) return PAIRINGS_EINVAL_OPTS;
    for (int i = 0; i < n_moduli; i++) total_out[i] = 0;
    *chunks_done_out = 0;
    if (duplicate_mismatches_out) *duplicate_mismatches_out = 0;

    // Lemma 2.4: negating the even positions maps the x_2 = +1 half of every
    // sum onto the x_2 = -1 half, term for term (up to the sign pairings_lemma24 reports).  The most
    // significant chunk bit is x_2, so the x_2 = +1 half is the chunk range [0, 2^{C-1}).
    // pairings_mode_chunks (host_math.cpp) is the one statement of that rule: chunks [0, needed), factor 1, 2 or 0
    // (the two halves cancel: H = 0, nothing to evaluate).
    uint64_t needed = 0;
    const int multiplier = pairings_mode_chunks(kind, n, chunk_bits, flags, &needed);
    if (multiplier < 0) return multiplier;
    // a slice (one job of a chunk farm): only chunks of [slice_begin, slice_end) that this mode evaluates
    const uint64_t sb = std::min(slice_begin, needed), se = std::min(slice_end, needed);
    const bool whole = (sb == 0 && se == needed);
    if (chunks_needed_out) *chunks_needed_out = se - sb;
    if (se == sb) return PAIRINGS_OK;

    // a1: what is already journalled
    std::vector<uint64_t> done;
    if (journal_path) {
        uint32_t jt[PAIRINGS_MAX_MODULI];
        int64_t nd = pairings_journal_load(journal_path, kind, n, chunk_bits, moduli, n_moduli, nullptr, 0, jt);
        if (nd < 0) return (int)nd;
        done.resize((size_t)(2 * nd) + 2);
        nd = pairings_journal_load(journal_path, kind, n, chunk_bits, moduli, n_moduli, done.data(), nd, total_out);
        if (nd < 0) return (int)nd;
        done.resize((size_t)(2 * nd));
        for (int64_t j = 0; j < nd; j++) {
            if (done[(size_t)(2 * j + 1)] > needed) return PAIRINGS_EJOURNAL;   // journal of a run without the symmetry
            if (done[(size_t)(2 * j)] < sb || done[(size_t)(2 * j + 1)] > se) return PAIRINGS_EJOURNAL;   // journal of another slice
            *chunks_done_out += done[(size_t)(2 * j + 1)] - done[(size_t)(2 * j)];
        }
    }
    if (se < (1ULL << chunk_bits)) { done.push_back(se); done.push_back(1ULL << chunk_bits); }   // not to be evaluated
    if (sb > 0) { done.push_back(0); done.push_back(sb); }
    // a1: the remaining ranges
    int64_t need = pairings_partition(chunk_bits, chunks_per_call, done.data(), (int)(done.size() / 2), nullptr, 0);
    if (need < 0) return (int)need;
    std::vector<uint64_t> ranges((size_t)(2 * need) + 2);
    need = pairings_partition(chunk_bits, chunks_per_call, done.data(), (int)(done.size() / 2), ranges.data(), need);
    if (need < 0) return (int)need;

    std::vector<uint32_t> rows;
    int64_t calls = 0;
    for (int64_t r = 0; r < need; r++) {
        if (max_calls > 0 && calls >= max_calls) break;
        const uint64_t b = ranges[(size_t)(2 * r)], e = ranges[(size_t)(2 * r + 1)];
        rows.resize((size_t)(e - b) * (size_t)n_moduli);
        // another launch geometry of the same kernel variant: the nearest admissible Gray-bit count (other thread <->
        // term mapping, other summation order); if none exists (tiny jobs) the same geometry again
        auto rerun_other_geometry = [&](int first_dg, uint64_t rb, uint64_t re, uint32_t* dst,
                                        const pairings_launch_opts* base) -> int {
            Geometry geo; int rc2 = choose_geometry(kind, n, chunk_bits, re - rb, base, &geo); if (rc2) return rc2;
            pairings_launch_opts alt; std::memset(&alt, 0, sizeof alt);
            alt.variant = geo.variant;
            rc2 = PAIRINGS_EINVAL_OPTS;
            for (int dg = first_dg; dg <= first_dg + 4 && rc2 == PAIRINGS_EINVAL_OPTS; dg += 2) {
                alt.gray_bits = geo.g - dg > 0 ? geo.g - dg : geo.g + dg;
                rc2 = count_pairings_host(kind, n, chunk_bits, rb, re, moduli, n_moduli, dst, stream, &alt);
            }
            if (rc2 == PAIRINGS_EINVAL_OPTS) rc2 = count_pairings_host(kind, n, chunk_bits, rb, re, moduli, n_moduli, dst, stream, base);
            return rc2;
        };
        if (flags & PAIRINGS_RUN_DUPLICATE) {
            // "every GPU job was ran twice ... a third time to establish a match" (silent GPU errors).  With
            // one GPU the second and third runs use other launch geometries, so a repeatable fault of one mapping does
            // not hide itself.  The vote itself is pairings_duplicate_vote (host_math.cpp).
            struct Ctx { decltype(rerun_other_geometry)* rerun; uint64_t b, e; int kind, n, C; const uint32_t* moduli; int m;
                         void* stream; const pairings_launch_opts* opts; } ctx{&rerun_other_geometry, b, e, kind, n, chunk_bits, moduli, n_moduli, stream, opts};
            auto eval = [](void* c, int attempt, uint32_t* out) -> int {
                Ctx* x = static_cast<Ctx*>(c);
                if (attempt == 0) return count_pairings_host(x->kind, x->n, x->C, x->b, x->e, x->moduli, x->m, out, x->stream, x->opts);
                return (*x->rerun)(attempt, x->b, x->e, out, x->opts);
            };
            int mismatch = 0;
            rc = pairings_duplicate_vote(eval, &ctx, (uint64_t)rows.size(), rows.data(), &mismatch); if (rc) return rc;
            if (mismatch && duplicate_mismatches_out) ++*duplicate_mismatches_out;
        } else {
            rc = count_pairings_host(kind, n, chunk_bits, b, e, moduli, n_moduli, rows.data(), stream, opts);
            if (rc) return rc;
        }
        if (flags & PAIRINGS_RUN_AUDIT) {
            // the generic kernel as auditor of the first and of one seeded chunk of the range
            uint64_t z = b * 0x9E3779B97F4A7C15ULL + 0xD1B54A32D192ED03ULL; z ^= z >> 29; z *= 0xBF58476D1CE4E5B9ULL; z ^= z >> 32;
            const uint64_t picks[2] = {b, b + z % (e - b)};
            pairings_launch_opts gen; std::memset(&gen, 0, sizeof gen); gen.variant = PAIRINGS_VARIANT_GENERIC;
            for (int a = 0; a < (picks[1] == picks[0] ? 1 : 2); a++) {
                const uint64_t c = picks[a];
                uint32_t second[PAIRINGS_MAX_MODULI], third[PAIRINGS_MAX_MODULI];
                rc = count_pairings_host(kind, n, chunk_bits, c, c + 1, moduli, n_moduli, second, stream, &gen); if (rc) return rc;
                const uint32_t* first = rows.data() + (size_t)(c - b) * (size_t)n_moduli;
                if (pairings_vote_rows(first, second, nullptr, (uint64_t)n_moduli) == 0) continue;
                if (duplicate_mismatches_out) ++*duplicate_mismatches_out;
                // The tie is broken by the INDEPENDENT implementation, never by the audited one: a deterministic bug
                // of the fast kernel (a wrong drain, a wrong zero table, a bad new instance) reproduces itself at
                // any geometry and would out-vote the auditor.  The generic kernel runs once more at another
                // Gray-bit count; the range stands only if that run sides with the fast row (then the auditor's
                // first run was the transient fault).  Generic reproducing its own row = the fast row is wrong.
                rc = rerun_other_geometry(1, c, c + 1, third, &gen); if (rc) return rc;
                if (pairings_vote_rows(first, second, third, (uint64_t)n_moduli) != 0) return PAIRINGS_ECHECK;
            }
        }
        uint32_t row_sum[PAIRINGS_MAX_MODULI] = {0};
        rc = pairings_sum_rows(rows.data(), e - b, moduli, n_moduli, row_sum); if (rc) return rc;
        if (journal_path) {
            rc = pairings_journal_append(journal_path, kind, n, chunk_bits, moduli, n_moduli, b, e, row_sum);
            if (rc) return rc;
        }
        rc = pairings_sum_rows(row_sum, 1, moduli, n_moduli, total_out); if (rc) return rc;
        *chunks_done_out += e - b;
        calls++;
    }
    if (apply_symmetry && whole && *chunks_done_out == needed && multiplier == 2) {       // complete: H = 2 * (x_2 = +1 half)
        rc = pairings_sum_rows(total_out, 1, moduli, n_moduli, total_out); if (rc) return rc;
    }
    return PAIRINGS_OK;
}

int pairings_run_ex(int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli,
                    uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                    void* stream, const pairings_launch_opts* opts, unsigned flags,
                    uint32_t* total_out, uint64_t* chunks_done_out, uint64_t* chunks_needed_out,
                    uint64_t* duplicate_mismatches_out) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, 0, 0); if (rc) return rc;
    return run_impl(kind, n, chunk_bits, moduli, n_moduli, chunks_per_call, journal_path, max_calls, stream, opts,
                    flags, 0, 1ULL << chunk_bits, true, total_out, chunks_done_out, chunks_needed_out, duplicate_mismatches_out);
}

int pairings_run_slice(int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli,
                       uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                       void* stream, const pairings_launch_opts* opts, unsigned flags,
                       uint64_t slice_begin, uint64_t slice_end,
                       uint32_t* total_out, uint64_t* chunks_done_out, uint64_t* chunks_needed_out,
                       uint64_t* duplicate_mismatches_out) {
    return run_impl(kind, n, chunk_bits, moduli, n_moduli, chunks_per_call, journal_path, max_calls, stream, opts,
                    flags, slice_begin, slice_end, false, total_out, chunks_done_out, chunks_needed_out, duplicate_mismatches_out);
}

int pairings_run(int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli,
                 uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                 void* stream, const pairings_launch_opts* opts,
                 uint32_t* total_out, uint64_t* chunks_done_out) {
    return pairings_run_ex(kind, n, chunk_bits, moduli, n_moduli, chunks_per_call, journal_path, max_calls,
                           stream, opts, 0u, total_out, chunks_done_out, nullptr, nullptr);
}

const char* pairings_build_info(void) {
    static const std::string info = [] {
        char buf[512];
        std::snprintf(buf, sizeof buf, "pairings_b200 0.1 sm_100a cuda %d swar[h=%d]: %s", CUDART_VERSION,
                      swar_min_gray_bits(), swar_list());
        return std::string(buf);
    }();
    return info.c_str();
}

}  // extern "C"
