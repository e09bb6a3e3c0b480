// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow CPU implementation of the paper's approximate counter (§3, :259-325,
// Algorithm 2 "Approximate Counting", :291-319), written from the paper text.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline leg may load it; it shares no code with the CUDA
// path under paper_1507_00315_b200/.
//
// The statistical system: n pairs of coloured balls in 2n bins, colour k at bins
// a_k and a_k + d_k (d_k = k Skolem, k+1 Langford), a_k in [1, 2n - d_k]; bins may hold several balls.
// There are prod_k (2n - d_k) = (2n-1)!/(n-1)! configurations (Skolem); the energy E(C) is
// the number of EMPTY bins; E = 0 configurations are exactly the pairings.
//
// One iteration, in the paper's order (Algorithm 2), for M levels beta(1) = 0 < ... < beta(M):
//   1. Ratio(j) += exp(-(beta(j+1) - beta(j)) E(C(j)))  — kept here as the integer histogram
//      hist[j][E(C(j))] += 1; the weights are applied afterwards (pt_ratios), beta(M+1) = infinity
//      (weight [E = 0]; reading C1 in DESIGN.md: "0 = beta_1 < ... < beta_m < beta").
//   2. every level j: N = random neighbour of C(j): a colour k uniformly at random, its pair moved to a
//      position uniformly at random; accepted with probability min[1, exp(-beta(j) dE)]
//      (the algorithm box prints the test reversed, "if p <= random" — reading C2:
//      accept iff random < p).
//   3. j = 1 .. M-1 in this order: C(j), C(j+1) exchanged with probability
//      min[1, exp(-(beta(j+1) - beta(j)) (E(C(j)) - E(C(j+1))))].
//
// Random numbers (reading C3: the paper names no generator): a counter-based generator that both
// sides implement from this description — draw(seed, ctr) = mix(seed + 0x9E3779B97F4A7C15 (ctr + 1)),
// mix = the SplitMix64 output function.  ctr = ((r (T + 1) + tt) M + j) S + slot with r the replica,
// T the iterations, tt = 0 for the initial configuration (slot k-1 places colour k) and tt = t + 1 for
// iteration t (slot 0: colour from the low, position from the high 32 bits; slot 1: acceptance;
// slot 2: exchange of levels j, j+1), S = max(n, 3).  A uniform integer in [0, m) from 32 bits u is
// floor(u m / 2^32); an event of probability p happens iff u < floor(p 2^32) (u = high 32 bits).
//
// Pins (tests/test_pt_oracle_pins.py): the density of states g(E) by exhaustive enumeration for small
// n (g sums to (2n-1)!/(n-1)!, g(0) = the paper's counts); the E-histogram of the beta = 0 level against
// g(E)/Z(0) and every level's ratio against the exact Z(beta(j+1))/Z(beta(j)) within the statistical
// error estimated from independent replicas; the final estimate of S(12) with the ladder of Table 6
// within the paper's "less than one percent" of 227,968.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

inline int dist(int kind, int k) { return kind == 0 ? k : k + 1; }

inline uint64_t mix64(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
inline uint64_t draw(uint64_t seed, uint64_t ctr) { return mix64(seed + 0x9E3779B97F4A7C15ULL * (ctr + 1)); }

// number of empty bins of a configuration a[1..n] — the plain definition, recomputed every time
int energy(int kind, int n, const int* a) {
    int balls[65]; std::memset(balls, 0, sizeof balls);
    for (int k = 1; k <= n; k++) { balls[a[k]]++; balls[a[k] + dist(kind, k)]++; }
    int e = 0;
    for (int b = 1; b <= 2 * n; b++) if (balls[b] == 0) e++;
    return e;
}

inline uint64_t threshold(double p) {                 // event iff (32-bit u) < threshold
    if (p >= 1.0) return 1ULL << 32;
    return (uint64_t)std::floor(p * 4294967296.0);
}

}  // namespace

extern "C" {

uint64_t pt_draw(uint64_t seed, uint64_t ctr) { return draw(seed, ctr); }

// Runs `replicas` independent copies of Algorithm 2 for `iterations` iterations each.
// hist: n_levels x (2n+1) counters (+=), moves_acc / swaps_acc: n_levels counters (+=).
// burn_in: the first burn_in iterations of every replica are run but not counted (0 = Algorithm 2 as printed;
// reading C4: without it a replica of T iterations is biased by O(relaxation time / T)).
int pt_run(int kind, int n, const double* beta, int n_levels, uint64_t replicas, uint64_t iterations,
           uint64_t burn_in, uint64_t seed, uint64_t* hist, uint64_t* moves_acc, uint64_t* swaps_acc) {
    if (kind < 0 || kind > 1 || n < 2 || n > 32 || n_levels < 1 || n_levels > 64) return -1;
    const int M = n_levels, N = 2 * n;
    const uint64_t S = n > 3 ? n : 3, T = iterations;
    std::vector<std::vector<int>> C(M, std::vector<int>(n + 1, 0));
    std::vector<int> E(M);
    for (uint64_t r = 0; r < replicas; r++) {
        for (int j = 0; j < M; j++) {                                     // "C(i) <- a random configuration"
            for (int k = 1; k <= n; k++) {
                const uint64_t u = draw(seed, ((r * (T + 1) + 0) * M + j) * S + (k - 1)) >> 32;
                C[j][k] = 1 + (int)((u * (uint64_t)(N - dist(kind, k))) >> 32);
            }
            E[j] = energy(kind, n, C[j].data());
        }
        for (uint64_t t = 0; t < T; t++) {
            const uint64_t base = (r * (T + 1) + (t + 1)) * M;
            const bool counted = t >= burn_in;
            for (int j = 0; j < M; j++) if (counted) hist[j * (N + 1) + E[j]]++;   // step 1
            for (int j = 0; j < M; j++) {                                 // step 2
                const uint64_t w = draw(seed, (base + j) * S + 0);
                const int k = 1 + (int)(((w & 0xFFFFFFFFULL) * (uint64_t)n) >> 32);
                const int pos = 1 + (int)(((w >> 32) * (uint64_t)(N - dist(kind, k))) >> 32);
                std::vector<int> Nb = C[j];
                Nb[k] = pos;
                const int dE = energy(kind, n, Nb.data()) - E[j];
                const uint64_t u = draw(seed, (base + j) * S + 1) >> 32;
                const double p = dE <= 0 ? 1.0 : std::exp(-beta[j] * (double)dE);
                if (u < threshold(p)) { C[j] = Nb; E[j] += dE; if (counted) moves_acc[j]++; }
            }
            for (int j = 0; j + 1 < M; j++) {                             // step 3
                const int dE = E[j] - E[j + 1];
                const uint64_t u = draw(seed, (base + j) * S + 2) >> 32;
                const double p = dE <= 0 ? 1.0 : std::exp(-(beta[j + 1] - beta[j]) * (double)dE);
                if (u < threshold(p)) { C[j].swap(C[j + 1]); std::swap(E[j], E[j + 1]); if (counted) swaps_acc[j]++; }
            }
        }
    }
    return 0;
}

// Ratio(j)/iterations of Algorithm 2 from the histogram: sum_E hist[j][E] exp(-(beta(j+1)-beta(j)) E) / samples,
// with beta(M+1) = infinity for the last level.  Returns log( Z(0) * prod_j ratio_j ), the natural logarithm
// of the estimated number of E = 0 configurations (reflections distinct); ratios_out: n_levels values.
double pt_ratios(int kind, int n, const double* beta, int n_levels, const uint64_t* hist, double* ratios_out) {
    const int N = 2 * n;
    double logz = 0.0;
    for (int k = 1; k <= n; k++) logz += std::log((double)(N - dist(kind, k)));   // Z(0) = prod_k (2n - d_k)
    for (int j = 0; j < n_levels; j++) {
        double num = 0.0, den = 0.0;
        for (int e = 0; e <= N; e++) {
            const double h = (double)hist[j * (N + 1) + e];
            den += h;
            if (j + 1 < n_levels) num += h * std::exp(-(beta[j + 1] - beta[j]) * (double)e);
            else if (e == 0) num += h;
        }
        ratios_out[j] = den > 0 ? num / den : 0.0;
        logz += std::log(ratios_out[j]);
    }
    return logz;
}

// Exhaustive density of states: g[E] = number of configurations with E empty bins (small n only).
int pt_density_of_states(int kind, int n, uint64_t* g /* 2n+1 */) {
    if (kind < 0 || kind > 1 || n < 2 || n > 8) return -1;
    const int N = 2 * n;
    for (int e = 0; e <= N; e++) g[e] = 0;
    int a[33];
    for (int k = 1; k <= n; k++) a[k] = 1;
    for (;;) {
        g[energy(kind, n, a)]++;
        int k = 1;
        while (k <= n) {                                   // odometer over a_k in [1, 2n - d_k]
            if (a[k] < N - dist(kind, k)) { a[k]++; break; }
            a[k] = 1; k++;
        }
        if (k > n) break;
    }
    return 0;
}

}  // extern "C"
