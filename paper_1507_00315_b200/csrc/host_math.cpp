// Host side of the path: moduli, prefix partitioner, journal, row sums, Garner CRT.
// (§8(a) rows a1 and a7 of SURVEY.md; PAPER.md:253 for the splitting, PAPER.md:257 for the
// modular arithmetic + Chinese remainder theorem, PAPER.md:168 for the exact division.)
// Plain C++17, no CUDA.  Shares nothing with oracle/.
#include "pairings.h"
#include "internal.h"

#include <algorithm>
#include <cerrno>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include <fcntl.h>
#include <unistd.h>

namespace pairings {

// ------------------------------------------------------------------------------------------------
// argument checks
// ------------------------------------------------------------------------------------------------
int check_kind_n(int kind, int n) {
    if (kind != PAIRINGS_SKOLEM && kind != PAIRINGS_LANGFORD) return PAIRINGS_EINVAL_KIND;
    if (n < 2 || n > 32) return PAIRINGS_EINVAL_N;
    return PAIRINGS_OK;
}

int check_moduli(const uint32_t* moduli, int n_moduli) {
    if (!moduli) return PAIRINGS_ENULL;
    if (n_moduli < 1 || n_moduli > PAIRINGS_MAX_MODULI) return PAIRINGS_EINVAL_MODULUS;
    for (int i = 0; i < n_moduli; i++) {
        uint32_t p = moduli[i];
        if ((p & 1u) == 0 || p <= (1u << 30) || p >= (1u << 31)) return PAIRINGS_EINVAL_MODULUS;
        for (int j = 0; j < i; j++) if (moduli[j] == p) return PAIRINGS_EINVAL_MODULUS;
    }
    return PAIRINGS_OK;
}

int check_chunks(int n, int chunk_bits, uint64_t begin, uint64_t end) {
    const int B = 2 * n - 1;
    if (chunk_bits < 0 || chunk_bits > B) return PAIRINGS_EINVAL_CHUNK;
    const uint64_t total = (chunk_bits >= 64) ? 0 : (1ULL << chunk_bits);  // B <= 63
    if (begin > end || end > total) return PAIRINGS_EINVAL_CHUNK;
    return PAIRINGS_OK;
}

// ------------------------------------------------------------------------------------------------
// 32-bit modular helpers (host)
// ------------------------------------------------------------------------------------------------
static inline uint32_t mulmod(uint32_t a, uint32_t b, uint32_t p) { return (uint32_t)((uint64_t)a * b % p); }

static uint32_t powmod(uint32_t a, uint64_t e, uint32_t p) {
    uint32_t r = 1 % p; a %= p;
    while (e) { if (e & 1) r = mulmod(r, a, p); a = mulmod(a, a, p); e >>= 1; }
    return r;
}

// deterministic Miller-Rabin for 32-bit integers (bases 2, 7, 61)
static bool is_prime32(uint32_t v) {
    if (v < 2) return false;
    for (uint32_t q : {2u, 3u, 5u, 7u, 11u, 13u, 17u, 19u, 23u, 29u, 31u, 37u}) {
        if (v % q == 0) return v == q;
    }
    uint32_t d = v - 1; int s = 0;
    while ((d & 1) == 0) { d >>= 1; s++; }
    for (uint32_t a : {2u, 7u, 61u}) {
        uint32_t x = powmod(a, d, v);
        if (x == 1 || x == v - 1) continue;
        bool comp = true;
        for (int r = 1; r < s; r++) {
            x = mulmod(x, x, v);
            if (x == v - 1) { comp = false; break; }
        }
        if (comp) return false;
    }
    return true;
}

static uint32_t invmod(uint32_t a, uint32_t p) { return powmod(a, (uint64_t)p - 2, p); }  // p prime

// ------------------------------------------------------------------------------------------------
// unsigned multi-limb integer (little endian 32-bit limbs), just what CRT needs
// ------------------------------------------------------------------------------------------------
struct Nat {
    std::vector<uint32_t> w;
    void trim() { while (!w.empty() && w.back() == 0) w.pop_back(); }
    bool zero() const { return w.empty(); }
};

static Nat nat_from(uint64_t v) { Nat a; while (v) { a.w.push_back((uint32_t)v); v >>= 32; } return a; }

static void nat_mul_small(Nat& a, uint32_t m) {
    uint64_t carry = 0;
    for (size_t i = 0; i < a.w.size(); i++) { uint64_t t = (uint64_t)a.w[i] * m + carry; a.w[i] = (uint32_t)t; carry = t >> 32; }
    if (carry) a.w.push_back((uint32_t)carry);
    a.trim();
}

static void nat_add(Nat& a, const Nat& b) {
    if (a.w.size() < b.w.size()) a.w.resize(b.w.size(), 0);
    uint64_t carry = 0;
    for (size_t i = 0; i < a.w.size(); i++) {
        uint64_t t = (uint64_t)a.w[i] + (i < b.w.size() ? b.w[i] : 0) + carry;
        a.w[i] = (uint32_t)t; carry = t >> 32;
    }
    if (carry) a.w.push_back((uint32_t)carry);
}

static int nat_cmp(const Nat& a, const Nat& b) {
    if (a.w.size() != b.w.size()) return a.w.size() < b.w.size() ? -1 : 1;
    for (size_t i = a.w.size(); i-- > 0;) if (a.w[i] != b.w[i]) return a.w[i] < b.w[i] ? -1 : 1;
    return 0;
}

// a -= b, requires a >= b
static void nat_sub(Nat& a, const Nat& b) {
    int64_t borrow = 0;
    for (size_t i = 0; i < a.w.size(); i++) {
        int64_t t = (int64_t)a.w[i] - (i < b.w.size() ? b.w[i] : 0) - borrow;
        if (t < 0) { t += (int64_t)1 << 32; borrow = 1; } else borrow = 0;
        a.w[i] = (uint32_t)t;
    }
    a.trim();
}

static uint32_t nat_mod_small(const Nat& a, uint32_t p) {
    uint64_t r = 0;
    for (size_t i = a.w.size(); i-- > 0;) r = ((r << 32) | a.w[i]) % p;
    return (uint32_t)r;
}

static uint32_t nat_divmod_small(Nat& a, uint32_t d) {
    uint64_t r = 0;
    for (size_t i = a.w.size(); i-- > 0;) { uint64_t cur = (r << 32) | a.w[i]; a.w[i] = (uint32_t)(cur / d); r = cur % d; }
    a.trim();
    return (uint32_t)r;
}

static bool nat_low_bits_zero(const Nat& a, int bits) {
    for (int i = 0; i < bits; i++) {
        size_t limb = (size_t)i / 32;
        if (limb < a.w.size() && ((a.w[limb] >> (i % 32)) & 1u)) return false;
    }
    return true;
}

static void nat_shr(Nat& a, int bits) {
    size_t limbs = (size_t)bits / 32; int r = bits % 32;
    if (limbs >= a.w.size()) { a.w.clear(); return; }
    a.w.erase(a.w.begin(), a.w.begin() + (long)limbs);
    if (r) {
        for (size_t i = 0; i < a.w.size(); i++) {
            uint32_t hi = (i + 1 < a.w.size()) ? a.w[i + 1] : 0;
            a.w[i] = (a.w[i] >> r) | (hi << (32 - r));
        }
    }
    a.trim();
}

static std::string nat_dec(Nat a) {
    if (a.zero()) return "0";
    std::vector<uint32_t> groups;                      // base 10^9 digits, least significant first
    while (!a.zero()) groups.push_back(nat_divmod_small(a, 1000000000u));
    std::string s = std::to_string(groups.back());
    for (size_t i = groups.size() - 1; i-- > 0;) {
        char buf[16]; std::snprintf(buf, sizeof buf, "%09u", groups[i]); s += buf;
    }
    return s;
}

// Garner's mixed-radix CRT: returns X in [0, prod p_i) with X = r_i mod p_i; *Mout = prod p_i.
static Nat garner(const uint32_t* p, const uint32_t* r, int m, Nat* Mout) {
    // mixed radix digits a_i:  X = a_0 + a_1 p_0 + a_2 p_0 p_1 + ...
    std::vector<uint32_t> a((size_t)m);
    for (int i = 0; i < m; i++) {
        // value of the already known part modulo p_i, Horner from the top digit
        uint64_t acc = 0;
        for (int j = i; j-- > 0;) acc = (acc * (p[j] % p[i]) + a[(size_t)j] % p[i]) % p[i];
        uint32_t diff = (uint32_t)(((uint64_t)(r[i] % p[i]) + p[i] - acc) % p[i]);
        uint32_t prodinv = 1;
        for (int j = 0; j < i; j++) prodinv = mulmod(prodinv, invmod(p[j] % p[i], p[i]), p[i]);
        a[(size_t)i] = mulmod(diff, prodinv, p[i]);
    }
    Nat X, M = nat_from(1);
    for (int i = 0; i < m; i++) {
        Nat t = M; nat_mul_small(t, a[(size_t)i]); nat_add(X, t); X.trim();
        nat_mul_small(M, p[i]);
    }
    if (Mout) *Mout = M;
    return X;
}

// 2 * 2^{2n-1} * prod_k (2n - d_k)  >= 2 |H|   (each |P_k| <= its number of summands)
static Nat twice_bound(int kind, int n) {
    Nat b = nat_from(1);
    for (int k = 1; k <= n; k++) nat_mul_small(b, (uint32_t)(2 * n - dist(kind, k)));
    for (int i = 0; i < 2 * n; i++) nat_mul_small(b, 2);
    return b;
}

static int put(const std::string& s, char* out, size_t cap) {
    if (!out) return PAIRINGS_ENULL;
    if (s.size() + 1 > cap) return PAIRINGS_ERANGE;
    std::memcpy(out, s.c_str(), s.size() + 1);
    return PAIRINGS_OK;
}

static void default_moduli(uint32_t* out, int count) {
    uint32_t v = 0x7fffffffu; int got = 0;
    while (got < count) { if (is_prime32(v)) out[got++] = v; v -= 2; }
}

}  // namespace pairings

using namespace pairings;

extern "C" {

int pairings_default_moduli(uint32_t* out, int count) {
    if (!out) return PAIRINGS_ENULL;
    if (count < 0 || count > PAIRINGS_MAX_MODULI) return PAIRINGS_EINVAL_MODULUS;
    default_moduli(out, count);
    return PAIRINGS_OK;
}

int pairings_min_moduli(int kind, int n) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    uint32_t p[PAIRINGS_MAX_MODULI]; default_moduli(p, PAIRINGS_MAX_MODULI);
    Nat bound = twice_bound(kind, n), M = nat_from(1);
    for (int m = 1; m <= PAIRINGS_MAX_MODULI; m++) {
        nat_mul_small(M, p[m - 1]);
        if (nat_cmp(M, bound) > 0) return m;
    }
    return PAIRINGS_ERANGE;
}

int pairings_bound_moduli(int kind, int n) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    uint32_t p[PAIRINGS_MAX_MODULI]; default_moduli(p, PAIRINGS_MAX_MODULI);
    Nat bound = nat_from(1);                                   // (2n)^n * 2^{2n}
    for (int k = 0; k < n; k++) nat_mul_small(bound, (uint32_t)(2 * n));
    for (int i = 0; i < 2 * n; i++) nat_mul_small(bound, 2);
    Nat M = nat_from(1);
    for (int m = 1; m <= PAIRINGS_MAX_MODULI; m++) {
        nat_mul_small(M, p[m - 1]);
        if (nat_cmp(M, bound) > 0) return m;
    }
    return PAIRINGS_ERANGE;
}

int pairings_lemma24(int kind, int n) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    // x^ = (x_1, -x_2, x_3, -x_4, ...): P_d(x^) = (-1)^d P_d(x) and prod_i x^_i = (-1)^n prod_i x_i, so
    // term(x^) = (-1)^{n + sum_k d_k} term(x)   (Lemma 2.4, written out for both kinds).
    long e = n;
    for (int k = 1; k <= n; k++) e += dist(kind, k);
    return (e % 2 == 0) ? 1 : 0;
}

int pairings_mode_chunks(int kind, int n, int chunk_bits, unsigned flags, uint64_t* needed_out) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, 0, 0); if (rc) return rc;
    if (!needed_out) return PAIRINGS_ENULL;
    if (flags & ~(unsigned)(PAIRINGS_RUN_LEMMA24 | PAIRINGS_RUN_DUPLICATE | PAIRINGS_RUN_AUDIT)) return PAIRINGS_EINVAL_OPTS;
    uint64_t needed = 1ULL << chunk_bits;
    int factor = 1;
    // Lemma 2.4: the most significant chunk bit is x_2, so the x_2 = +1 half of the sum is the chunk
    // range [0, 2^{C-1}); the other half equals it (factor 2) or cancels it (nothing to evaluate, H = 0).
    if ((flags & PAIRINGS_RUN_LEMMA24) && chunk_bits >= 1) {
        if (pairings_lemma24(kind, n) == 1) { needed >>= 1; factor = 2; }
        else { needed = 0; factor = 0; }
    }
    *needed_out = needed;
    return factor;
}

int pairings_finish_total(int kind, int n, int chunk_bits, unsigned flags, uint64_t chunks_covered,
                          const uint32_t* moduli, int n_moduli, uint32_t* total_inout) {
    uint64_t needed = 0;
    const int factor = pairings_mode_chunks(kind, n, chunk_bits, flags, &needed); if (factor < 0) return factor;
    int rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    if (!total_inout) return PAIRINGS_ENULL;
    if (chunks_covered > needed) return PAIRINGS_EINVAL_CHUNK;     // more than the mode evaluates: rows of the other half
    if (chunks_covered < needed) return 0;                         // incomplete: the raw partial sum stays as it is
    for (int i = 0; i < n_moduli; i++) if (total_inout[i] >= moduli[i]) return PAIRINGS_EINVAL_MODULUS;
    if (factor == 0) { for (int i = 0; i < n_moduli; i++) total_inout[i] = 0; }
    else if (factor == 2) { rc = pairings_sum_rows(total_inout, 1, moduli, n_moduli, total_inout); if (rc) return rc; }
    return 1;
}

int64_t pairings_partition(int chunk_bits, uint64_t max_chunks, const uint64_t* done, int n_done,
                           uint64_t* out_ranges, int64_t cap_ranges) {
    if (chunk_bits < 0 || chunk_bits > 63 || max_chunks == 0 || n_done < 0) return PAIRINGS_EINVAL_CHUNK;
    if (n_done > 0 && !done) return PAIRINGS_ENULL;
    if (cap_ranges > 0 && !out_ranges) return PAIRINGS_ENULL;
    const uint64_t total = 1ULL << chunk_bits;
    std::vector<std::pair<uint64_t, uint64_t>> d;
    for (int j = 0; j < n_done; j++) {
        uint64_t b = done[2 * j], e = done[2 * j + 1];
        if (b > e || e > total) return PAIRINGS_EINVAL_CHUNK;
        if (b < e) d.emplace_back(b, e);
    }
    std::sort(d.begin(), d.end());
    int64_t count = 0;
    auto emit = [&](uint64_t b, uint64_t e) {
        while (b < e) {
            uint64_t len = std::min<uint64_t>(max_chunks, e - b);
            if (count < cap_ranges) { out_ranges[2 * count] = b; out_ranges[2 * count + 1] = b + len; }
            count++; b += len;
        }
    };
    uint64_t cur = 0;
    for (auto& r : d) {
        if (r.first > cur) emit(cur, r.first);
        cur = std::max(cur, r.second);
    }
    if (cur < total) emit(cur, total);
    return count;
}

int pairings_rank_range(int chunk_bits, int rank, int world, uint64_t* out_begin, uint64_t* out_end) {
    if (!out_begin || !out_end) return PAIRINGS_ENULL;
    if (chunk_bits < 0 || chunk_bits > 63 || world < 1 || rank < 0 || rank >= world) return PAIRINGS_EINVAL_CHUNK;
    const uint64_t total = 1ULL << chunk_bits;
    const uint64_t q = total / (uint64_t)world, r = total % (uint64_t)world;
    const uint64_t rk = (uint64_t)rank;
    *out_begin = rk * q + std::min(rk, r);
    *out_end = *out_begin + q + (rk < r ? 1 : 0);
    return PAIRINGS_OK;
}

int pairings_sum_rows(const uint32_t* rows, uint64_t n_rows, const uint32_t* moduli, int n_moduli, uint32_t* total) {
    int rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    if (!total || (n_rows && !rows)) return PAIRINGS_ENULL;
    for (int i = 0; i < n_moduli; i++) {
        const uint32_t p = moduli[i];
        uint64_t acc = total[i] % p;
        for (uint64_t r = 0; r < n_rows; r++) {
            acc += rows[r * (uint64_t)n_moduli + (uint64_t)i] % p;
            if (acc >= (1ULL << 62)) acc %= p;
        }
        total[i] = (uint32_t)(acc % p);
    }
    return PAIRINGS_OK;
}

// ---- journal -------------------------------------------------------------------------------

static std::string journal_header(int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli) {
    std::string h = "pairings-journal v1 kind=" + std::to_string(kind) + " n=" + std::to_string(n) +
                    " chunk_bits=" + std::to_string(chunk_bits) + " moduli=";
    for (int i = 0; i < n_moduli; i++) { if (i) h += ","; h += std::to_string(moduli[i]); }
    return h;
}

// reads complete lines (a trailing line without '\n' is a torn write and is dropped); *complete_bytes = length of
// the file up to and including its last '\n'
static int read_lines(const char* path, std::vector<std::string>& lines, bool* exists, size_t* complete_bytes = nullptr,
                      size_t* file_bytes = nullptr) {
    FILE* f = std::fopen(path, "rb");
    if (complete_bytes) *complete_bytes = 0;
    if (file_bytes) *file_bytes = 0;
    if (!f) { *exists = false; return errno == ENOENT ? PAIRINGS_OK : PAIRINGS_EJOURNAL; }
    *exists = true;
    std::string data; char buf[65536]; size_t got;
    while ((got = std::fread(buf, 1, sizeof buf, f)) > 0) data.append(buf, got);
    const bool bad = std::ferror(f) != 0;
    std::fclose(f);
    if (bad) return PAIRINGS_EJOURNAL;
    size_t pos = 0;
    while (true) {
        size_t nl = data.find('\n', pos);
        if (nl == std::string::npos) break;
        lines.emplace_back(data.substr(pos, nl - pos));
        pos = nl + 1;
    }
    if (complete_bytes) *complete_bytes = pos;
    if (file_bytes) *file_bytes = data.size();
    return PAIRINGS_OK;
}

// one unsigned decimal token (digits only: no sign, no 0x) followed by a blank or the end of the line
static bool next_u64(const char*& s, unsigned long long* out) {
    while (*s == ' ') s++;
    if (*s < '0' || *s > '9') return false;
    unsigned long long v = 0;
    int digits = 0;
    while (*s >= '0' && *s <= '9') {
        if (++digits > 20 || v > (~0ULL - (unsigned)(*s - '0')) / 10ULL) return false;   // would not fit 64 bits
        v = v * 10ULL + (unsigned)(*s - '0');
        s++;
    }
    if (*s != ' ' && *s != '\0') return false;
    *out = v;
    return true;
}

struct JournalLine { uint64_t b, e; uint32_t row[PAIRINGS_MAX_MODULI]; };

// "begin end r_0 .. r_{m-1}", nothing else on the line
static bool parse_journal_line(const std::string& line, int n_moduli, const uint32_t* moduli, uint64_t total, JournalLine* out) {
    const char* s = line.c_str();
    unsigned long long b, e, v;
    if (!next_u64(s, &b) || !next_u64(s, &e)) return false;
    if (b >= e || e > total) return false;
    out->b = b; out->e = e;
    for (int i = 0; i < n_moduli; i++) {
        if (!next_u64(s, &v) || v >= moduli[i]) return false;
        out->row[i] = (uint32_t)v;
    }
    while (*s == ' ') s++;
    return *s == '\0';                     // trailing tokens: two lines glued together, or another file format
}

// all data lines of a journal, checked: header, syntax, ranges inside [0, 2^C), no two ranges overlap
static int load_journal(const char* path, int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli,
                        std::vector<JournalLine>& out, bool* exists_out = nullptr) {
    std::vector<std::string> lines; bool exists = false;
    int rc = read_lines(path, lines, &exists); if (rc) return rc;
    if (exists_out) *exists_out = exists;
    if (!exists || lines.empty()) return PAIRINGS_OK;
    if (lines[0] != journal_header(kind, n, chunk_bits, moduli, n_moduli)) return PAIRINGS_EJOURNAL;
    const uint64_t total = 1ULL << chunk_bits;
    out.reserve(lines.size());
    for (size_t li = 1; li < lines.size(); li++) {
        JournalLine jl;
        if (!parse_journal_line(lines[li], n_moduli, moduli, total, &jl)) return PAIRINGS_EJOURNAL;
        out.push_back(jl);
    }
    // overlap = double count: sort a copy of the ranges by begin, neighbours must not intersect
    std::vector<std::pair<uint64_t, uint64_t>> r; r.reserve(out.size());
    for (auto& jl : out) r.emplace_back(jl.b, jl.e);
    std::sort(r.begin(), r.end());
    for (size_t i = 1; i < r.size(); i++) if (r[i].first < r[i - 1].second) return PAIRINGS_EJOURNAL;
    return PAIRINGS_OK;
}

int64_t pairings_journal_load(const char* path, int kind, int n, int chunk_bits,
                              const uint32_t* moduli, int n_moduli,
                              uint64_t* out_ranges, int64_t cap_ranges, uint32_t* total_out) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, 0, 0); if (rc) return rc;
    if (!path || !total_out || (cap_ranges > 0 && !out_ranges)) return PAIRINGS_ENULL;
    for (int i = 0; i < n_moduli; i++) total_out[i] = 0;
    std::vector<JournalLine> lines;
    rc = load_journal(path, kind, n, chunk_bits, moduli, n_moduli, lines); if (rc) return rc;
    int64_t count = 0;
    for (auto& jl : lines) {
        pairings_sum_rows(jl.row, 1, moduli, n_moduli, total_out);
        if (count < cap_ranges) { out_ranges[2 * count] = jl.b; out_ranges[2 * count + 1] = jl.e; }
        count++;
    }
    return count;
}

static std::string format_journal_line(uint64_t b, uint64_t e, const uint32_t* row, int n_moduli) {
    std::string line = std::to_string(b) + " " + std::to_string(e);
    for (int i = 0; i < n_moduli; i++) line += " " + std::to_string(row[i]);
    line += "\n";
    return line;
}

// write + flush + fsync; the data must be on disk before the caller counts the range as done
static int write_all_sync(int fd, const std::string& data) {
    size_t off = 0;
    while (off < data.size()) {
        ssize_t w = ::write(fd, data.data() + off, data.size() - off);
        if (w < 0) { if (errno == EINTR) continue; return PAIRINGS_EJOURNAL; }
        off += (size_t)w;
    }
    return ::fsync(fd) == 0 ? PAIRINGS_OK : PAIRINGS_EJOURNAL;
}

int pairings_journal_append(const char* path, int kind, int n, int chunk_bits,
                            const uint32_t* moduli, int n_moduli,
                            uint64_t chunk_begin, uint64_t chunk_end, const uint32_t* row_sum) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, chunk_begin, chunk_end); if (rc) return rc;
    if (!path || !row_sum) return PAIRINGS_ENULL;
    if (chunk_begin == chunk_end) return PAIRINGS_EINVAL_CHUNK;
    for (int i = 0; i < n_moduli; i++) if (row_sum[i] >= moduli[i]) return PAIRINGS_EINVAL_MODULUS;
    std::vector<std::string> lines; bool exists = false; size_t complete = 0, size = 0;
    rc = read_lines(path, lines, &exists, &complete, &size); if (rc) return rc;
    const std::string header = journal_header(kind, n, chunk_bits, moduli, n_moduli);
    if (exists && !lines.empty() && lines[0] != header) return PAIRINGS_EJOURNAL;
    const bool need_header = !exists || lines.empty();
    // A torn last line (a crash in the middle of a write: bytes after the last '\n') is cut off first; appending
    // behind it would glue the new line onto the fragment.  A file with no complete line at all is started afresh.
    const int fd = ::open(path, O_WRONLY | O_CREAT, 0644);
    if (fd < 0) return PAIRINGS_EJOURNAL;
    const off_t keep = need_header ? 0 : (off_t)complete;
    if ((size != (size_t)keep && ::ftruncate(fd, keep) != 0) || ::lseek(fd, keep, SEEK_SET) != keep) { ::close(fd); return PAIRINGS_EJOURNAL; }
    std::string data;
    if (need_header) data += header + "\n";
    data += format_journal_line(chunk_begin, chunk_end, row_sum, n_moduli);
    rc = write_all_sync(fd, data);
    if (::close(fd) != 0 && rc == PAIRINGS_OK) rc = PAIRINGS_EJOURNAL;
    return rc;
}

int64_t pairings_journal_merge(const char* const* paths, int n_paths, const char* out_path, int kind, int n, int chunk_bits,
                               const uint32_t* moduli, int n_moduli, uint32_t* total_out, uint64_t* chunks_covered_out) {
    return pairings_journal_merge_mode(paths, n_paths, out_path, kind, n, chunk_bits, moduli, n_moduli, 0u,
                                       total_out, chunks_covered_out, nullptr);
}

int64_t pairings_journal_merge_mode(const char* const* paths, int n_paths, const char* out_path, int kind, int n, int chunk_bits,
                                    const uint32_t* moduli, int n_moduli, unsigned flags,
                                    uint32_t* total_out, uint64_t* chunks_covered_out, uint64_t* chunks_needed_out) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    rc = check_chunks(n, chunk_bits, 0, 0); if (rc) return rc;
    if (!paths || n_paths < 1 || !total_out) return PAIRINGS_ENULL;
    uint64_t needed = 0;
    rc = pairings_mode_chunks(kind, n, chunk_bits, flags, &needed); if (rc < 0) return rc;
    if (chunks_needed_out) *chunks_needed_out = needed;
    for (int i = 0; i < n_moduli; i++) total_out[i] = 0;
    std::vector<JournalLine> all;
    for (int j = 0; j < n_paths; j++) {
        if (!paths[j]) return PAIRINGS_ENULL;
        std::vector<JournalLine> part; bool exists = false;
        rc = load_journal(paths[j], kind, n, chunk_bits, moduli, n_moduli, part, &exists); if (rc) return rc;
        if (!exists) return PAIRINGS_EJOURNAL;                      // a rank's file is missing: not "nothing done"
        all.insert(all.end(), part.begin(), part.end());
    }
    std::sort(all.begin(), all.end(), [](const JournalLine& x, const JournalLine& y) { return x.b < y.b; });
    uint64_t covered = 0;
    for (size_t i = 0; i < all.size(); i++) {
        if (i && all[i].b < all[i - 1].e) return PAIRINGS_EJOURNAL;   // two journals hold the same chunk: double count
        // a range outside the half this mode evaluates (a journal of a job without the symmetry, or a mix of both
        // halves that happens to have the right length) would be doubled into a wrong count
        if (all[i].e > needed) return PAIRINGS_EJOURNAL;
        covered += all[i].e - all[i].b;
        pairings_sum_rows(all[i].row, 1, moduli, n_moduli, total_out);
    }
    if (chunks_covered_out) *chunks_covered_out = covered;
    if (out_path) {
        std::string data = journal_header(kind, n, chunk_bits, moduli, n_moduli) + "\n";
        for (auto& jl : all) data += format_journal_line(jl.b, jl.e, jl.row, n_moduli);
        const int fd = ::open(out_path, O_WRONLY | O_CREAT | O_TRUNC, 0644);
        if (fd < 0) return PAIRINGS_EJOURNAL;
        rc = write_all_sync(fd, data);
        if (::close(fd) != 0 && rc == PAIRINGS_OK) rc = PAIRINGS_EJOURNAL;
        if (rc) return rc;
    }
    return (int64_t)all.size();
}

int pairings_vote_rows(const uint32_t* a, const uint32_t* b, const uint32_t* c, uint64_t n_words) {
    if (!a || !b) return PAIRINGS_ENULL;
    const size_t bytes = (size_t)n_words * sizeof(uint32_t);
    if (std::memcmp(a, b, bytes) == 0) return 0;                  // the two runs agree: a stands
    if (!c) return 3;                                             // disagreement, a third run is needed
    if (std::memcmp(c, a, bytes) == 0) return 0;                  // third run confirms the first
    if (std::memcmp(c, b, bytes) == 0) return 1;                  // third run confirms the second
    return PAIRINGS_ECHECK;                                       // three runs, no two agree
}

int pairings_duplicate_vote(pairings_eval_fn eval, void* ctx, uint64_t n_words, uint32_t* rows_out, int* mismatch_out) {
    if (!eval || (n_words && !rows_out)) return PAIRINGS_ENULL;
    if (mismatch_out) *mismatch_out = 0;
    std::vector<uint32_t> second((size_t)n_words), third;
    int rc = eval(ctx, 0, rows_out); if (rc) return rc;
    rc = eval(ctx, 1, second.data()); if (rc) return rc;
    int v = pairings_vote_rows(rows_out, second.data(), nullptr, n_words);
    if (v == 0) return PAIRINGS_OK;
    if (v < 0) return v;
    if (mismatch_out) *mismatch_out = 1;                          // "ran a third time to establish a match"
    third.resize((size_t)n_words);
    rc = eval(ctx, 2, third.data()); if (rc) return rc;
    v = pairings_vote_rows(rows_out, second.data(), third.data(), n_words);
    if (v < 0) return v;
    if (v == 1) std::memcpy(rows_out, second.data(), (size_t)n_words * sizeof(uint32_t));
    return PAIRINGS_OK;
}

// ---- CRT -----------------------------------------------------------------------------------

int pairings_reconstruct(int kind, int n, const uint32_t* moduli, int n_moduli,
                         const uint32_t* total_residues,
                         char* out_distinct_dec, char* out_identified_dec, size_t cap) {
    int rc = check_kind_n(kind, n); if (rc) return rc;
    rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    if (n_moduli < 2) return PAIRINGS_EINVAL_MODULUS;  // at least one CRT prime + the check prime
    if (!total_residues || !out_distinct_dec || !out_identified_dec) return PAIRINGS_ENULL;
    for (int i = 0; i < n_moduli; i++) if (total_residues[i] >= moduli[i]) return PAIRINGS_EINVAL_MODULUS;
    const int m = n_moduli - 1;
    Nat M; Nat H = garner(moduli, total_residues, m, &M);
    if (nat_cmp(M, twice_bound(kind, n)) <= 0) return PAIRINGS_ERANGE;
    if (nat_mod_small(H, moduli[m]) != total_residues[m]) return PAIRINGS_ECHECK;
    if (!nat_low_bits_zero(H, 2 * n - 1)) return PAIRINGS_EINEXACT;
    Nat D = H; nat_shr(D, 2 * n - 1);
    if (!D.zero() && (D.w[0] & 1u)) return PAIRINGS_EINEXACT;   // n > 1: no palindromes
    Nat S = D; nat_shr(S, 1);
    rc = put(nat_dec(D), out_distinct_dec, cap); if (rc) return rc;
    return put(nat_dec(S), out_identified_dec, cap);
}

int pairings_crt_signed(const uint32_t* moduli, int n_moduli, const uint32_t* residues, char* out_dec, size_t cap) {
    int rc = check_moduli(moduli, n_moduli); if (rc) return rc;
    if (!residues || !out_dec) return PAIRINGS_ENULL;
    for (int i = 0; i < n_moduli; i++) if (residues[i] >= moduli[i]) return PAIRINGS_EINVAL_MODULUS;
    Nat M; Nat X = garner(moduli, residues, n_moduli, &M);
    Nat twoX = X; nat_mul_small(twoX, 2);
    if (nat_cmp(twoX, M) > 0) {            // X > M/2  ->  X - M (negative)
        Nat neg = M; nat_sub(neg, X);
        return put("-" + nat_dec(neg), out_dec, cap);
    }
    return put(nat_dec(X), out_dec, cap);
}

const char* pairings_strerror(int code) {
    switch (code) {
        case PAIRINGS_OK: return "ok";
        case PAIRINGS_EINVAL_KIND: return "invalid kind (0 = Skolem, 1 = Langford)";
        case PAIRINGS_EINVAL_N: return "n outside [2, 32]";
        case PAIRINGS_EINVAL_CHUNK: return "invalid chunk_bits or chunk range";
        case PAIRINGS_EINVAL_MODULUS: return "invalid modulus set (odd, distinct, in (2^30, 2^31), 1..16 of them)";
        case PAIRINGS_ENULL: return "required pointer is NULL";
        case PAIRINGS_ECUDA: return "CUDA runtime error";
        case PAIRINGS_ECHECK: return "CRT value disagrees with the check prime";
        case PAIRINGS_EINEXACT: return "sum not divisible by 2^(2n-1), or D odd";
        case PAIRINGS_ERANGE: return "modulus product too small for the bound, or output buffer too small";
        case PAIRINGS_EINVAL_OPTS: return "launch options not satisfiable";
        case PAIRINGS_EJOURNAL: return "journal unreadable or written for other parameters";
        case PAIRINGS_ETOOBIG: return "problem too large for the fixed scratch area of a no-allocation entry point";
        default: return "unknown error code";
    }
}

}  // extern "C"
