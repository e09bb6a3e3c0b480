// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU evaluator of Godfrey's algebraic sum for Skolem / Langford
// pairings, written from the paper text ("Counting Skolem Sequences", arxiv 1507.00315,
// /root/reference/PAPER.md).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this file.  It shares no code, header, table or helper with the
// CUDA path under paper_1507_00315_b200/ and neither includes the other.
//
// What is here, each with the passage it follows:
//   * godfrey_term / godfrey_range : Algorithm 1 "Godfrey()" (§2.1), i.e. Lemma 2.1
//      evaluated literally: for every X in {+1,-1}^{2n}: signX = prod X(i);
//     for i = 1..n: sum = sum_{k=1}^{2n-d_i} X(k) X(k+d_i); prod *= sum;  S += signX * prod.
//     No Gray code, no symmetry, no popcount tricks, no modular arithmetic; the running total and
//     the product are signed big integers (own fixed-width sign-magnitude type below, no GMP).
//     Readings: A2 multiply once per i after the k loop;
//     A3 the domain is {+1,-1}^{2n}; A4 Langford = distance d_i = i+1.
//   * brute_count / brute_list : Miller's backtracking (§2): place the pairs in
//     decreasing order, each at every position where both of its cells are free.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): the n=4 worked example (coefficient 6 and the six
// sequences), the example pairings, Tables 7/8 exact counts
// for n <= 13, existence conditions, the closed form
// F(n, all +1) = (2n-1)!/(n-1)!, Lemmas 2.2-2.4 as invariants,
// and formula == backtracking for every n it can reach.  Nothing here is "parity unpinned".
//
// Index convention of godfrey_range (chosen so that a contiguous index range is a power-of-two
// sub-cube): index X in [0, 2^{2n}); bit b of X (b = 0..2n-1) gives position 2n-b;
// bit = 1 means x = -1.  So X < 2^{2n-1} is exactly the half with x_1 = +1.
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#include <algorithm>

namespace {

// ---------------------------------------------------------------------------------------------
// Signed big integer, sign-magnitude, fixed 12 x 32-bit limbs (384 bits: |sum| <= 2^{64}*63!/31!
// < 2^{242} for n <= 32).  Overflow of the top limb sets `overflow` and is reported by callers.
// ---------------------------------------------------------------------------------------------
struct Big {
    static const int L = 12;
    uint32_t mag[L];
    int neg;        // 1 if negative (zero is never negative)
    int overflow;
    Big() { std::memset(mag, 0, sizeof mag); neg = 0; overflow = 0; }
    explicit Big(long long v) {
        std::memset(mag, 0, sizeof mag); overflow = 0;
        neg = v < 0;
        unsigned long long a = neg ? 0ULL - (unsigned long long)v : (unsigned long long)v;
        mag[0] = (uint32_t)a; mag[1] = (uint32_t)(a >> 32);
    }
    bool is_zero() const { for (int i = 0; i < L; i++) if (mag[i]) return false; return true; }
};

int cmp_mag(const Big& a, const Big& b) {
    for (int i = Big::L - 1; i >= 0; i--) {
        if (a.mag[i] != b.mag[i]) return a.mag[i] < b.mag[i] ? -1 : 1;
    }
    return 0;
}

// r = |a| + |b| (magnitudes)
void add_mag(const Big& a, const Big& b, Big& r) {
    uint64_t carry = 0;
    for (int i = 0; i < Big::L; i++) {
        uint64_t s = (uint64_t)a.mag[i] + b.mag[i] + carry;
        r.mag[i] = (uint32_t)s; carry = s >> 32;
    }
    if (carry) r.overflow = 1;
}

// r = |a| - |b|, requires |a| >= |b|
void sub_mag(const Big& a, const Big& b, Big& r) {
    int64_t borrow = 0;
    for (int i = 0; i < Big::L; i++) {
        int64_t s = (int64_t)a.mag[i] - b.mag[i] - borrow;
        if (s < 0) { s += ((int64_t)1 << 32); borrow = 1; } else borrow = 0;
        r.mag[i] = (uint32_t)s;
    }
}

Big add(const Big& a, const Big& b) {
    Big r; r.overflow = a.overflow | b.overflow;
    if (a.neg == b.neg) { add_mag(a, b, r); r.neg = a.neg; }
    else {
        int c = cmp_mag(a, b);
        if (c == 0) { r.neg = 0; }
        else if (c > 0) { sub_mag(a, b, r); r.neg = a.neg; }
        else { sub_mag(b, a, r); r.neg = b.neg; }
    }
    if (r.is_zero()) r.neg = 0;
    return r;
}

Big mul_small(const Big& a, long long s) {
    Big r; r.overflow = a.overflow;
    int sneg = s < 0;
    uint64_t m = sneg ? 0ULL - (uint64_t)s : (uint64_t)s;   // |s| < 2^31 in every use here
    uint64_t carry = 0;
    for (int i = 0; i < Big::L; i++) {
        uint64_t p = (uint64_t)a.mag[i] * m + carry;
        r.mag[i] = (uint32_t)p; carry = p >> 32;
    }
    if (carry) r.overflow = 1;
    r.neg = a.neg ^ sneg;
    if (r.is_zero()) r.neg = 0;
    return r;
}

// magnitude divided by small d in place, returns remainder
uint32_t divmod_small_mag(Big& a, uint32_t d) {
    uint64_t rem = 0;
    for (int i = Big::L - 1; i >= 0; i--) {
        uint64_t cur = (rem << 32) | a.mag[i];
        a.mag[i] = (uint32_t)(cur / d); rem = cur % d;
    }
    return (uint32_t)rem;
}

std::string to_dec(const Big& a) {
    Big t = a; std::string s;
    if (t.is_zero()) return "0";
    while (!t.is_zero()) { uint32_t r = divmod_small_mag(t, 10); s.push_back((char)('0' + r)); }
    if (a.neg) s.push_back('-');
    std::reverse(s.begin(), s.end());
    return s;
}

// mathematical (non-negative) residue of a modulo p   (reading A8: values in [0,p))
uint32_t mod_small(const Big& a, uint32_t p) {
    Big t = a; uint32_t r = divmod_small_mag(t, p);
    if (a.neg && r != 0) r = p - r;
    return r;
}

int put(const std::string& s, char* out, size_t cap) {
    if (!out || s.size() + 1 > cap) return -1;
    std::memcpy(out, s.c_str(), s.size() + 1);
    return 0;
}

// distance of pair i:  Skolem d_i = i, Langford d_i = i+1 (the two
// copies of k are "k units apart", i.e. their positions differ by k+1 — the n=4 example
// 2,3,4,2,1,3,1,4 has the 1s at positions 5 and 7).
inline int dist(int kind, int i) { return kind == 0 ? i : i + 1; }

// One evaluation: signX * prod_i sum_k X(k) X(k+d_i)  for the sign vector X[1..2n] (entries +-1).
// Algorithm 1's inner two loops, verbatim.  *nonzero is set to 1 if prod != 0.
Big evaluate(int kind, int n, const int* X, int* nonzero) {
    const int N = 2 * n;
    int signX = 1;
    for (int i = 1; i <= N; i++) signX = signX * X[i];
    Big prod(1);
    for (int i = 1; i <= n; i++) {
        int d = dist(kind, i);
        long long sum = 0;
        for (int k = 1; k <= N - d; k++) sum = sum + X[k] * X[k + d];
        prod = mul_small(prod, sum);
    }
    if (nonzero) *nonzero = prod.is_zero() ? 0 : 1;
    return mul_small(prod, signX);
}

void expand(int n, uint64_t index, int* X) {
    const int N = 2 * n;
    for (int b = 0; b < N; b++) X[N - b] = ((index >> b) & 1ULL) ? -1 : +1;
}

// ---------------------------------------------------------------------------------------------
// backtracking
// ---------------------------------------------------------------------------------------------
struct Brute {
    int kind, n, N;
    int seq[80];              // seq[p] = label at position p (1-based), 0 = free
    uint64_t count;
    int* out; int max_out; int n_out;
    void place(int k) {
        if (k == 0) {
            if (out && n_out < max_out) { for (int p = 1; p <= N; p++) out[n_out * N + (p - 1)] = seq[p]; }
            n_out++; count++; return;
        }
        int d = dist(kind, k);
        for (int a = 1; a + d <= N; a++) {
            if (seq[a] == 0 && seq[a + d] == 0) {
                seq[a] = k; seq[a + d] = k;
                place(k - 1);
                seq[a] = 0; seq[a + d] = 0;
            }
        }
    }
};

}  // namespace

extern "C" {

// Single term  signX * F(n, X)  as a decimal string.  xbits: bit (p-1) = 1 means x_p = -1 (p = 1..2n).
int godfrey_term(int kind, int n, uint64_t xbits, char* out_dec, size_t cap) {
    if (n < 1 || n > 32 || (kind != 0 && kind != 1)) return -2;
    int X[80];
    for (int p = 1; p <= 2 * n; p++) X[p] = ((xbits >> (p - 1)) & 1ULL) ? -1 : +1;
    Big t = evaluate(kind, n, X, nullptr);
    if (t.overflow) return -3;
    return put(to_dec(t), out_dec, cap);
}

// F(n, X) alone (without the sign factor), for Lemma 2.3 / closed-form pins.
int godfrey_F(int kind, int n, uint64_t xbits, char* out_dec, size_t cap) {
    if (n < 1 || n > 32 || (kind != 0 && kind != 1)) return -2;
    int X[80]; int signX = 1;
    for (int p = 1; p <= 2 * n; p++) { X[p] = ((xbits >> (p - 1)) & 1ULL) ? -1 : +1; signX *= X[p]; }
    Big t = evaluate(kind, n, X, nullptr);
    t = mul_small(t, signX);
    if (t.overflow) return -3;
    return put(to_dec(t), out_dec, cap);
}

// Sum of signX*prod over the index range [index_begin, index_end) of the 2^{2n} sign vectors
// (index convention in the header).  Outputs: the exact signed sum as a decimal string, the number
// of vectors whose product is non-zero, and (optionally) the sum's residues modulo moduli[0..m).
// index_end may be 2^{2n} only for n <= 31 (uint64_t); use two calls for n = 32.
int godfrey_range(int kind, int n, uint64_t index_begin, uint64_t index_end,
                  char* out_sum_dec, size_t cap, uint64_t* out_nonzero,
                  const uint32_t* moduli, int n_moduli, uint32_t* out_residues) {
    if (n < 1 || n > 32 || (kind != 0 && kind != 1)) return -2;
    if (index_end < index_begin) return -2;
    int X[80];
    Big S(0);
    uint64_t nz = 0;
    for (uint64_t idx = index_begin; idx < index_end; idx++) {
        expand(n, idx, X);
        int nonzero = 0;
        Big term = evaluate(kind, n, X, &nonzero);
        S = add(S, term);
        nz += (uint64_t)nonzero;
    }
    if (S.overflow) return -3;
    if (out_nonzero) *out_nonzero = nz;
    for (int i = 0; i < n_moduli; i++) out_residues[i] = mod_small(S, moduli[i]);
    return put(to_dec(S), out_sum_dec, cap);
}

// Number of pairings with reflections counted as distinct (A004075 / A176127).
uint64_t brute_count(int kind, int n) {
    if (n < 1 || n > 32 || (kind != 0 && kind != 1)) return 0;
    Brute b; b.kind = kind; b.n = n; b.N = 2 * n; b.count = 0; b.out = nullptr; b.max_out = 0; b.n_out = 0;
    std::memset(b.seq, 0, sizeof b.seq);
    b.place(n);
    return b.count;
}

// Lists up to max_solutions sequences (each 2n labels, position order) and returns the total count.
uint64_t brute_list(int kind, int n, int* out_seq, int max_solutions) {
    if (n < 1 || n > 32 || (kind != 0 && kind != 1)) return 0;
    Brute b; b.kind = kind; b.n = n; b.N = 2 * n; b.count = 0; b.out = out_seq; b.max_out = max_solutions; b.n_out = 0;
    std::memset(b.seq, 0, sizeof b.seq);
    b.place(n);
    return b.count;
}

}  // extern "C"
