// ASan / UBSan driver: the host side of the library (csrc/host_math.cpp) and the two CPU oracles are
// compiled with -fsanitize=address,undefined and exercised on what untrusted input reaches them — journal files of every
// kind of damage, argument extremes — plus the CRT round trips and small-n pins.  Built three times by
// tests/test_sanitizers.py: -DDRIVE_HOST (links host_math.cpp), -DDRIVE_ORACLE (godfrey_oracle.cpp), -DDRIVE_PT
// (pt_oracle.cpp); each build shares nothing with the others.  Exit code 0 = every check held and no sanitizer report.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#define CHECK(c) do { if (!(c)) { std::fprintf(stderr, "CHECK failed line %d: %s\n", __LINE__, #c); std::exit(1); } } while (0)

static uint64_t rng_state = 150700315ULL;
static uint64_t rnd() {
    uint64_t z = (rng_state += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL; z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL; return z ^ (z >> 31);
}

#ifdef DRIVE_HOST
#include "pairings.h"

static void write_file(const std::string& path, const std::string& data) {
    FILE* f = std::fopen(path.c_str(), "wb"); CHECK(f);
    std::fwrite(data.data(), 1, data.size(), f); std::fclose(f);
}

static int vote_script[3][4];
static int vote_calls;
static int vote_eval(void*, int attempt, uint32_t* out) {
    vote_calls++;
    for (int i = 0; i < 4; i++) out[i] = (uint32_t)vote_script[attempt][i];
    return 0;
}

int main(int argc, char** argv) {
    CHECK(argc == 2);
    const std::string dir = argv[1];
    uint32_t p[PAIRINGS_MAX_MODULI];
    CHECK(pairings_default_moduli(p, PAIRINGS_MAX_MODULI) == 0 && p[0] == 2147483647u);
    for (int kind = 0; kind < 2; kind++)
        for (int n = 2; n <= 32; n++) {
            const int m = pairings_min_moduli(kind, n), b = pairings_bound_moduli(kind, n);
            CHECK(m >= 1 && b >= m && b < PAIRINGS_MAX_MODULI);
            CHECK(pairings_lemma24(kind, n) == 0 || pairings_lemma24(kind, n) == 1);
        }
    CHECK(pairings_min_moduli(0, 1) < 0 && pairings_min_moduli(2, 8) < 0 && pairings_min_moduli(0, 33) < 0);

    // CRT: L(12) = 108,144: H = D * 2^23, residues by plain 64-bit arithmetic
    {
        const uint64_t H = 216288ULL << 23;
        uint32_t r[4]; for (int i = 0; i < 4; i++) r[i] = (uint32_t)(H % p[i]);
        char d[64], s[64];
        CHECK(pairings_reconstruct(1, 12, p, 4, r, d, s, sizeof d) == 0 && !std::strcmp(d, "216288") && !std::strcmp(s, "108144"));
        CHECK(pairings_reconstruct(1, 12, p, 4, r, d, s, 3) == PAIRINGS_ERANGE);
        r[3] ^= 1; CHECK(pairings_reconstruct(1, 12, p, 4, r, d, s, sizeof d) == PAIRINGS_ECHECK); r[3] ^= 1;
        uint32_t r2[4]; for (int i = 0; i < 4; i++) r2[i] = (uint32_t)((H + 1) % p[i]);
        CHECK(pairings_reconstruct(1, 12, p, 4, r2, d, s, sizeof d) == PAIRINGS_EINEXACT);
        CHECK(pairings_reconstruct(1, 12, p, 1, r, d, s, sizeof d) == PAIRINGS_EINVAL_MODULUS);
        CHECK(pairings_reconstruct(1, 12, p, 2, r, d, s, sizeof d) == PAIRINGS_ERANGE);
        // signed lift: random small signed values through all 16 primes
        for (int t = 0; t < 200; t++) {
            const int64_t v = (int64_t)(rnd() >> 2) - (int64_t)(1ULL << 61);
            uint32_t rr[PAIRINGS_MAX_MODULI];
            for (int i = 0; i < PAIRINGS_MAX_MODULI; i++) { int64_t q = v % (int64_t)p[i]; if (q < 0) q += p[i]; rr[i] = (uint32_t)q; }
            char out[256];
            const int m = 3 + (int)(rnd() % 14);
            CHECK(pairings_crt_signed(p, m, rr, out, sizeof out) == 0);
            CHECK(std::strtoll(out, nullptr, 10) == v);
        }
    }
    // partition / rank ranges / row sums on random inputs
    for (int t = 0; t < 200; t++) {
        const int C = (int)(rnd() % 12);
        uint64_t done[16]; const int nd = (int)(rnd() % 8);
        for (int j = 0; j < nd; j++) { uint64_t a = rnd() % ((1ULL << C) + 1), b = rnd() % ((1ULL << C) + 1); done[2 * j] = a < b ? a : b; done[2 * j + 1] = a < b ? b : a; }
        const uint64_t mx = 1 + rnd() % 37;
        const int64_t need = pairings_partition(C, mx, done, nd, nullptr, 0);
        CHECK(need >= 0);
        std::vector<uint64_t> out((size_t)(2 * need) + 2);
        CHECK(pairings_partition(C, mx, done, nd, out.data(), need) == need);
        for (int64_t j = 0; j < need; j++) CHECK(out[2 * j] < out[2 * j + 1] && out[2 * j + 1] - out[2 * j] <= mx && out[2 * j + 1] <= (1ULL << C));
        uint64_t b, e; const int world = 1 + (int)(rnd() % 9);
        uint64_t prev = 0;
        for (int r = 0; r < world; r++) { CHECK(pairings_rank_range(C, r, world, &b, &e) == 0 && b == prev && e >= b); prev = e; }
        CHECK(prev == (1ULL << C));
    }
    CHECK(pairings_partition(64, 1, nullptr, 0, nullptr, 0) < 0 && pairings_partition(4, 0, nullptr, 0, nullptr, 0) < 0);

    // journal: healthy round trip, then every kind of damage — load must answer (>= 0 or PAIRINGS_EJOURNAL), never crash
    const std::string j = dir + "/j.txt";
    uint32_t row[4] = {1, 2, 3, 4}, tot[4];
    CHECK(pairings_journal_append(j.c_str(), 1, 12, 6, p, 4, 0, 8, row) == 0);
    CHECK(pairings_journal_append(j.c_str(), 1, 12, 6, p, 4, 8, 64, row) == 0);
    uint64_t rg[8];
    CHECK(pairings_journal_load(j.c_str(), 1, 12, 6, p, 4, rg, 4, tot) == 2 && tot[0] == 2 && rg[3] == 64);
    std::string good;
    { FILE* f = std::fopen(j.c_str(), "rb"); char buf[4096]; size_t g = std::fread(buf, 1, sizeof buf, f); std::fclose(f); good.assign(buf, g); }
    const std::string header = good.substr(0, good.find('\n') + 1);
    std::vector<std::string> damaged = {
        "", "\n", header, header.substr(0, header.size() - 1), header + "0 8 1 2 3", header + "0 8 1 2 3 4 5\n", header + "0 8 1 2 3\n",
        header + "99999999999999999999999999 8 1 2 3 4\n", header + "0 8 -1 2 3 4\n", header + std::string(100000, '7') + "\n",
        header + std::string(70000, ' ') + "0 8 1 2 3 4\n", header + "0 8 1 2 3 4\n0 8 1 2 3 4\n", header + "\n\n\n",
        std::string("\0\0\0\0binary\xff\xfe\n", 13), header + std::string("0 8 1 2 \0 4\n", 12), good.substr(0, good.size() / 2),
        header + "0 8 4294967296 2 3 4\n", header + "8 0 1 2 3 4\n", header + "0 65 1 2 3 4\n"};
    for (size_t k = 0; k < damaged.size(); k++) {
        const std::string path = dir + "/d" + std::to_string(k) + ".txt";
        write_file(path, damaged[k]);
        const int64_t rc = pairings_journal_load(path.c_str(), 1, 12, 6, p, 4, rg, 4, tot);
        CHECK(rc >= 0 || rc == PAIRINGS_EJOURNAL);
        const int ra = pairings_journal_append(path.c_str(), 1, 12, 6, p, 4, 16, 24, row);   // append on top of the damage
        CHECK(ra == 0 || ra == PAIRINGS_EJOURNAL);
        const int64_t rc2 = pairings_journal_load(path.c_str(), 1, 12, 6, p, 4, rg, 4, tot);
        CHECK(rc2 >= 0 || rc2 == PAIRINGS_EJOURNAL);
    }
    for (int t = 0; t < 300; t++) {                       // random byte flips of a healthy journal
        std::string d = good;
        for (int f = 0; f < 3; f++) d[rnd() % d.size()] = (char)rnd();
        if (rnd() % 4 == 0) d.resize(rnd() % (d.size() + 1));
        const std::string path = dir + "/fuzz.txt";
        write_file(path, d);
        const int64_t rc = pairings_journal_load(path.c_str(), 1, 12, 6, p, 4, rg, 4, tot);
        CHECK(rc >= 0 || rc == PAIRINGS_EJOURNAL);
    }
    {   // merge + vote
        const std::string a = dir + "/a.txt", b = dir + "/b.txt", m = dir + "/m.txt";
        CHECK(pairings_journal_append(a.c_str(), 1, 12, 6, p, 4, 0, 32, row) == 0);
        CHECK(pairings_journal_append(b.c_str(), 1, 12, 6, p, 4, 32, 64, row) == 0);
        const char* paths[3] = {b.c_str(), a.c_str(), a.c_str()};
        uint64_t cov = 0;
        CHECK(pairings_journal_merge(paths, 2, m.c_str(), 1, 12, 6, p, 4, tot, &cov) == 2 && cov == 64 && tot[3] == 8);
        CHECK(pairings_journal_merge(paths, 3, nullptr, 1, 12, 6, p, 4, tot, &cov) == PAIRINGS_EJOURNAL);
        CHECK(pairings_journal_merge(paths, 0, nullptr, 1, 12, 6, p, 4, tot, &cov) == PAIRINGS_ENULL);
        // the mode of a job: b.txt lies in the x_2 = -1 half, which a Lemma 2.4 job does not evaluate
        uint64_t need = 0;
        CHECK(pairings_mode_chunks(1, 12, 6, PAIRINGS_RUN_LEMMA24, &need) == 2 && need == 32);
        CHECK(pairings_mode_chunks(0, 14, 6, PAIRINGS_RUN_LEMMA24, &need) == 0 && need == 0);
        CHECK(pairings_mode_chunks(1, 12, 6, 0, nullptr) == PAIRINGS_ENULL);
        CHECK(pairings_journal_merge_mode(paths, 2, nullptr, 1, 12, 6, p, 4, PAIRINGS_RUN_LEMMA24, tot, &cov, &need) == PAIRINGS_EJOURNAL);
        CHECK(pairings_journal_merge_mode(paths + 1, 1, nullptr, 1, 12, 6, p, 4, PAIRINGS_RUN_LEMMA24, tot, &cov, &need) == 1 && cov == 32 && need == 32);
        CHECK(pairings_finish_total(1, 12, 6, PAIRINGS_RUN_LEMMA24, cov, p, 4, tot) == 1 && tot[3] == 2 * row[3] % p[3]);
        CHECK(pairings_finish_total(1, 12, 6, PAIRINGS_RUN_LEMMA24, 31, p, 4, tot) == 0);
        CHECK(pairings_finish_total(1, 12, 6, PAIRINGS_RUN_LEMMA24, 33, p, 4, tot) == PAIRINGS_EINVAL_CHUNK);
        CHECK(pairings_finish_total(1, 12, 6, 0, 64, p, 4, nullptr) == PAIRINGS_ENULL);
        uint32_t x[4] = {1, 2, 3, 4}, y[4] = {1, 2, 3, 5}, z[4] = {7, 7, 7, 7};
        CHECK(pairings_vote_rows(x, x, nullptr, 4) == 0 && pairings_vote_rows(x, y, nullptr, 4) == 3);
        CHECK(pairings_vote_rows(x, y, x, 4) == 0 && pairings_vote_rows(x, y, y, 4) == 1 && pairings_vote_rows(x, y, z, 4) == PAIRINGS_ECHECK);
        CHECK(pairings_vote_rows(nullptr, y, z, 4) == PAIRINGS_ENULL && pairings_vote_rows(x, y, nullptr, 0) == 0);
        const int scripts[4][3][4] = {{{1, 2, 3, 4}, {1, 2, 3, 4}, {0, 0, 0, 0}}, {{1, 2, 3, 4}, {1, 2, 3, 5}, {1, 2, 3, 4}},
                                      {{1, 2, 3, 4}, {1, 2, 3, 5}, {1, 2, 3, 5}}, {{1, 2, 3, 4}, {1, 2, 3, 5}, {9, 9, 9, 9}}};
        const int want_rc[4] = {0, 0, 0, PAIRINGS_ECHECK}, want_calls[4] = {2, 3, 3, 3}, want_last[4] = {4, 4, 5, 0};
        for (int s = 0; s < 4; s++) {
            std::memcpy(vote_script, scripts[s], sizeof vote_script);
            vote_calls = 0;
            uint32_t rows[4]; int mm = -1;
            CHECK(pairings_duplicate_vote(vote_eval, nullptr, 4, rows, &mm) == want_rc[s] && vote_calls == want_calls[s]);
            if (want_rc[s] == 0) CHECK(rows[3] == (uint32_t)want_last[s] && mm == (s > 0));
        }
    }
    for (int code = -12; code <= 1; code++) CHECK(pairings_strerror(code) != nullptr);
    std::puts("host ok");
    return 0;
}
#endif

#ifdef DRIVE_ORACLE
extern "C" {
int godfrey_term(int kind, int n, uint64_t xbits, char* out_dec, size_t cap);
int godfrey_F(int kind, int n, uint64_t xbits, char* out_dec, size_t cap);
int godfrey_range(int kind, int n, uint64_t index_begin, uint64_t index_end, char* out_sum_dec, size_t cap, uint64_t* out_nonzero,
                  const uint32_t* moduli, int n_moduli, uint32_t* out_residues);
uint64_t brute_count(int kind, int n);
uint64_t brute_list(int kind, int n, int* out_seq, int max_solutions);
}
int main() {
    char buf[256];
    const uint32_t mod[2] = {2147483647u, 2147483629u};
    // formula == backtracking for every kind, n <= 7; S(4) = 3, S(5) = 5, L(3) = L(4) = 1, L(7) = 26
    for (int kind = 0; kind < 2; kind++)
        for (int n = 2; n <= 7; n++) {
            uint64_t nz = 0; uint32_t res[2];
            CHECK(godfrey_range(kind, n, 0, 1ULL << (2 * n), buf, sizeof buf, &nz, mod, 2, res) == 0);
            const long long total = std::strtoll(buf, nullptr, 10);
            CHECK(total % (1LL << (2 * n)) == 0 && (uint64_t)(total >> (2 * n)) == brute_count(kind, n));
            CHECK(res[0] == (uint32_t)(total % mod[0]));
        }
    CHECK(brute_count(0, 4) == 6 && brute_count(0, 5) == 10 && brute_count(1, 3) == 2 && brute_count(1, 4) == 2 && brute_count(1, 7) == 52);
    int seq[6 * 8];
    CHECK(brute_list(0, 4, seq, 6) == 6 && brute_list(0, 4, seq, 2) == 6);
    // extremes: n = 32 terms (big integers ~2^177), all-(+1) and all-(-1); tiny output buffers; bad arguments
    for (int kind = 0; kind < 2; kind++) {
        CHECK(godfrey_term(kind, 32, 0, buf, sizeof buf) == 0 && std::strlen(buf) > 40);
        CHECK(godfrey_term(kind, 32, ~0ULL, buf, sizeof buf) == 0);
        CHECK(godfrey_F(kind, 32, 0x5555555555555555ULL, buf, sizeof buf) == 0);
        CHECK(godfrey_term(kind, 32, 0, buf, 4) != 0);
        for (int t = 0; t < 50; t++) CHECK(godfrey_term(kind, 2 + (int)(rnd() % 31), rnd(), buf, sizeof buf) == 0);
    }
    CHECK(godfrey_term(2, 8, 0, buf, sizeof buf) != 0 && godfrey_term(0, 33, 0, buf, sizeof buf) != 0 && godfrey_term(0, 0, 0, buf, sizeof buf) != 0);
    CHECK(godfrey_range(0, 8, 5, 4, buf, sizeof buf, nullptr, mod, 0, nullptr) != 0);
    CHECK(godfrey_range(0, 32, (1ULL << 63) - 3, (1ULL << 63) + 3, buf, sizeof buf, nullptr, mod, 0, nullptr) == 0);
    CHECK(brute_count(0, 0) == 0 && brute_count(3, 4) == 0);
    std::puts("oracle ok");
    return 0;
}
#endif

#ifdef DRIVE_PT
extern "C" {
uint64_t pt_draw(uint64_t seed, uint64_t ctr);
int pt_run(int kind, int n, const double* beta, int n_levels, uint64_t replicas, uint64_t iterations, uint64_t burn_in, uint64_t seed,
           uint64_t* hist, uint64_t* moves_acc, uint64_t* swaps_acc);
double pt_ratios(int kind, int n, const double* beta, int n_levels, const uint64_t* hist, double* ratios_out);
int pt_density_of_states(int kind, int n, uint64_t* g);
}
int main() {
    CHECK(pt_draw(0, 0) == 0xE220A8397B1DCDAFULL);      // first output of SplitMix64 seeded with 0 (the published test vector)
    const double beta[5] = {0, 0.8, 1.8, 3.0, 6.0};
    for (int kind = 0; kind < 2; kind++)
        for (int n : {2, 3, 8, 17, 32}) {
            const int N = 2 * n;
            std::vector<uint64_t> hist((size_t)5 * (N + 1), 0), mv(5, 0), sw(5, 0);
            CHECK(pt_run(kind, n, beta, 5, 7, 200, 20, 99, hist.data(), mv.data(), sw.data()) == 0);
            for (int j = 0; j < 5; j++) {
                uint64_t s = 0; for (int e = 0; e <= N; e++) s += hist[(size_t)j * (N + 1) + e];
                CHECK(s == 7ULL * 180ULL && mv[j] <= 7ULL * 180ULL);
            }
            double r[5]; (void)pt_ratios(kind, n, beta, 5, hist.data(), r);
            CHECK(r[0] > 0 && r[0] <= 1.0);
        }
    CHECK(pt_run(0, 1, beta, 5, 1, 1, 0, 0, nullptr, nullptr, nullptr) != 0 && pt_run(2, 8, beta, 5, 1, 1, 0, 0, nullptr, nullptr, nullptr) != 0);
    uint64_t g[17];
    for (int n = 2; n <= 5; n++) {                      // sum_E g(E) = prod_k (2n - k) = (2n-1)!/(n-1)!
        CHECK(pt_density_of_states(0, n, g) == 0);
        uint64_t s = 0, want = 1; for (int e = 0; e <= 2 * n; e++) s += g[e];
        for (int k = 1; k <= n; k++) want *= (uint64_t)(2 * n - k);
        CHECK(s == want);
    }
    CHECK(pt_density_of_states(0, 9, g) != 0);
    std::puts("pt ok");
    return 0;
}
#endif
