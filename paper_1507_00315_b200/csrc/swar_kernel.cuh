// SWAR Gray-code kernel, specialised per (kind, n) — the fast path of count_pairings.
//
// What it computes is exactly §8(a) rows a2..a6 (PAPER.md:176 Gray-code ordering, PAPER.md:257
// residues modulo co-primes); how it computes it is designed for sm_100a's integer pipes:
//
//  * pair-sums live byte-packed, four per 32-bit register ("slots"): slot value = Q_k + 128 with
//    Q_k = P_k/2 for even d_k (P_k = N-d_k mod 2, so these are the only sums that can vanish) and
//    Q_k = P_k for odd d_k.  The factor 2^{#even} is restored once per thread at the end.
//    Even-d slots come first.  The zero test (row a4) is done for a whole inner block at once from
//    compile-time tables (see "zero-step tables" below): one 32-bit mask of the zero steps per block.
//  * the low H = 5 index bits are walked by ONE fully unrolled 32-step Gray block that always starts
//    in inner state 0.  For every inner position the packed vector C[b] of its neighbours that lie
//    OUTSIDE the inner bits is kept in registers; neighbours inside the inner bits are known at
//    compile time and folded into an immediate.  One Gray step (row a3) is therefore
//         Q[r] = Q[r] -/+ C[b][r] + K[r]          — one 3-input add per register, n/4 per step,
//    instead of n boundary-guarded updates.  (Deltas are added as whole 32-bit integers: bytes stay
//    in [65,191] after every step, so no carry ever crosses a slot.)
//  * between two blocks the inner state (only bit H-1 set) is flipped back to 0 together with the
//    outer flip (Gray order over index bits H..g-1), so every block runs the same compile-time
//    sequence; each sign vector is still visited exactly once.  The outer flip rebuilds the neighbour
//    vector of the flipped position from two de-interleaved copies (E: even index bits, O: odd) of
//    the sign word with a multiply-spread (4 bits -> 4 bytes), and patches one byte of each C[b].
//    Because g <= n-2, every left neighbour of a walked position exists: no boundary guards at all.
//  * non-zero terms are compacted (row a4's divergence problem).  The zero mask of a lane's whole block is known before
//    its first step, so the slots of all pushes are PLANNED at block start: nibble popcounts give the lane's number of
//    non-zero steps per quad (4 steps), one scan over the lanes in byte fields gives its first slot in every quad, REDUX
//    the warp totals.  Entries (the packed registers; the sign of the term is read off the distance-n sum) go to a
//    per-warp stack in shared memory with predicated stores; whenever 32 entries are stacked all lanes multiply one
//    entry each (any lane may process any term of its warp: the sum is commutative and a warp never spans two chunks).
//  * row a5: the product is formed from dp4a "pair factors" (two sums per LOP3 + IDP.4A), G exact
//    signed group products (< 2^31 each), a signed multi-word product, added into a W-word
//    two's-complement accumulator.  The reduction modulo the primes happens ONCE per thread (32-bit
//    Montgomery Horner), not per term — the residues written are identical, the per-term cost no
//    longer depends on the number of primes.
//  * row a6: shared with the generic kernel (block_reduce_write).
#pragma once

#include "internal.h"
#include "device_common.cuh"
#include "swar_list.h"

#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace pairings {
namespace swar {

constexpr int H = PAIRINGS_SWAR_H;              // unrolled inner Gray bits
constexpr int BLK = 1 << H;       // steps per unrolled block
#ifndef PAIRINGS_DRAIN2_MAXEW
#define PAIRINGS_DRAIN2_MAXEW 5   // larger entries have 8 drain sites per block: a second copy of the product there outgrows the instruction cache (S(24) -13 %)
#endif
constexpr int QUAD = 4;           // steps per slot allocation
static_assert(31 * QUAD + 32 * QUAD <= 255, "per-quad lane prefixes (<= 31 * QUAD) are scanned in byte fields, and a warp total (<= 32 * QUAD) may be added to one");

#define PAIRINGS_HD __host__ __device__ constexpr

// compile-time loop: f(std::integral_constant<int, I>) for I in [I0, I1)
template <int I0, int I1, class F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I0 < I1) {
        f(std::integral_constant<int, I0>{});
        static_for<I0 + 1, I1>(f);
    }
}
#define PAIRINGS_IC(name, ic) constexpr int name = decltype(ic)::value

PAIRINGS_HD int ctz_c(int v) { int c = 0; while (((v >> c) & 1) == 0) c++; return c; }
PAIRINGS_HD int gray_c(int s) { return s ^ (s >> 1); }
PAIRINGS_HD int bitlen_c(uint64_t v) { int c = 0; while (v) { c++; v >>= 1; } return c; }

// ------------------------------------------------------------------------------------------------
// compile-time layout of one (kind, n)
// ------------------------------------------------------------------------------------------------
template <int KIND, int NN>
struct Lay {
    static constexpr int N = 2 * NN;
    PAIRINGS_HD static int d_of_k(int k) { return KIND == PAIRINGS_SKOLEM ? k : k + 1; }
    PAIRINGS_HD static int n_even() { int c = 0; for (int k = 1; k <= NN; k++) c += (d_of_k(k) % 2 == 0); return c; }
    // slot order: even distances ascending, then odd distances ascending
    PAIRINGS_HD static int d_of_slot(int s) {
        int c = 0;
        for (int k = 1; k <= NN; k++) if (d_of_k(k) % 2 == 0) { if (c == s) return d_of_k(k); c++; }
        for (int k = 1; k <= NN; k++) if (d_of_k(k) % 2 == 1) { if (c == s) return d_of_k(k); c++; }
        return 0;
    }
    PAIRINGS_HD static int slot_of_d(int d) { for (int s = 0; s < NN; s++) if (d_of_slot(s) == d) return s; return -1; }
    PAIRINGS_HD static int unit(int s) { return d_of_slot(s) % 2 == 0 ? 1 : 2; }      // |dQ| per neighbour product
    PAIRINGS_HD static int cnt(int s) { return N - d_of_slot(s); }                     // number of summands of P
    PAIRINGS_HD static int bound(int s) { return d_of_slot(s) % 2 == 0 ? cnt(s) / 2 : cnt(s); }   // |Q| <= bound
    static constexpr int NR = (NN + 3) / 4;            // packed registers
    // ---- product plan (row a5).  The n factors are multiplied as "pair factors": byte i of register
    // 2p times byte i of register 2p+1 in ONE dp4a (the second operand masked to that byte), bytes
    // (0,1) and (2,3) of an unpaired last register likewise; a slot without a partner is a single
    // sign-extracted byte.  Pair factors are then packed (best fit, decreasing) into G groups whose
    // exact signed products stay below 2^31.
    static constexpr int NF_MAX = 4 * ((NR + 1) / 2) + 4;
    struct Plan {
        int nf;                    // number of factors
        int kind[NF_MAX];          // 1: registers (r, r+1) byte i;  2: register r bytes (i, i+1);  3: register r byte i alone
        int r[NF_MAX], i[NF_MAX];
        uint64_t bound[NF_MAX];    // |factor| <= bound
        int group[NF_MAX];
        int G;                     // number of groups
        int bits;                  // sum over groups of bitlen(bound of the group product)
        bool unbias[NR];           // register needs its own  ^ 0x80808080  (used as a dp4a first operand or for single bytes)
    };
    PAIRINGS_HD static uint64_t slot_bound(int s) { return s < NN ? (uint64_t)bound(s) : 0; }
    PAIRINGS_HD static Plan make_plan(bool last_as_singles) {
        Plan P{};
        int nf = 0;
        for (int r = 0; r < NR; r++) P.unbias[r] = false;
        for (int p = 0; 2 * p + 1 < NR; p++) {
            const int r = 2 * p;
            for (int i = 0; i < 4; i++) {
                const uint64_t b1 = slot_bound(4 * r + i), b2 = slot_bound(4 * (r + 1) + i);
                if (b1 && b2) { P.kind[nf] = 1; P.r[nf] = r; P.i[nf] = i; P.bound[nf] = b1 * b2; nf++; P.unbias[r] = true; }
                else if (b1) { P.kind[nf] = 3; P.r[nf] = r; P.i[nf] = i; P.bound[nf] = b1; nf++; P.unbias[r] = true; }
            }
        }
        if (NR % 2 == 1) {
            const int r = NR - 1;
            for (int i = 0; i < 4; i += (last_as_singles ? 1 : 2)) {
                const uint64_t b1 = slot_bound(4 * r + i), b2 = last_as_singles ? 0 : slot_bound(4 * r + i + 1);
                if (b1 && b2) { P.kind[nf] = 2; P.r[nf] = r; P.i[nf] = i; P.bound[nf] = b1 * b2; nf++; P.unbias[r] = true; }
                else if (b1) { P.kind[nf] = 3; P.r[nf] = r; P.i[nf] = i; P.bound[nf] = b1; nf++; P.unbias[r] = true; }
            }
        }
        P.nf = nf;
        // best-fit decreasing into the fewest groups with product < 2^31
        int order[NF_MAX] = {};
        for (int f = 0; f < nf; f++) order[f] = f;
        for (int a = 0; a < nf; a++)
            for (int c = a + 1; c < nf; c++)
                if (P.bound[order[c]] > P.bound[order[a]]) { const int t = order[a]; order[a] = order[c]; order[c] = t; }
        for (int G = 1; G <= 8; G++) {
            uint64_t prod[8] = {1, 1, 1, 1, 1, 1, 1, 1};
            bool ok = true;
            for (int a = 0; a < nf && ok; a++) {
                const int f = order[a];
                int best = -1;
                for (int g = 0; g < G; g++)
                    if (prod[g] * P.bound[f] < (1ULL << 31) && (best < 0 || prod[g] > prod[best])) best = g;
                if (best < 0) ok = false; else { prod[best] *= P.bound[f]; P.group[f] = best; }
            }
            if (ok) {
                P.G = G; P.bits = 0;
                for (int g = 0; g < G; g++) P.bits += bitlen_c(prod[g]);
                return P;
            }
        }
        P.G = 0;                                       // does not happen for n <= 32 (static_assert below)
        return P;
    }
    // finer factors for an unpaired last register only where that saves a group (n = 20: G = 3 instead of 4)
    static constexpr Plan plan = make_plan(true).G < make_plan(false).G ? make_plan(true) : make_plan(false);
    static constexpr int G = plan.G;
    // accumulator words: |sum| < 2^bits * 2^32 drained terms per thread (host enforces), + sign
    static constexpr int W = (plan.bits + 33 + 31) / 32;
    static_assert(G >= 1, "no grouping found");
    static_assert(W >= G && W <= 8, "accumulator must hold the multi-word product");
    // The sign of a term, prod_i x_i = (-1)^{#(x_i = -1)}, is not stored: for d = n the pairs (i, i+n) cover every
    // position exactly once, so #(x_i != x_{i+n}) = (n - P_n)/2 has the parity of #(x_i = -1).
    static constexpr int SIGN_SLOT = slot_of_d(NN);     // exists for both kinds (Skolem k = n, Langford k = n-1)
    static_assert(SIGN_SLOT >= 0, "distance n");
    static constexpr int EW = NR;                       // stack entry words (the packed sums)
    static constexpr int PLANES = (EW + 3) / 4;         // planes per entry: plane 0 holds words 0..3 at a 16-byte stride
    // Plane 1 (words 4..) of a 5- or 6-word entry is COMPACT: 4 or 8 bytes per entry at that stride, so that the
    // 32-/64-bit accesses of a warp fall into distinct banks (at a 16-byte stride they are 4-/2-way conflicts —
    // measured: the shared-memory pipe, not the issue port, bounded v11).  Its address is (slot >> P1SHIFT) + k1.
    // Drain checks: after every DQ quads.  Two quads per check (fewer checks, half the drain sites) where the stack of
    // 31 + 256 entries still lets 3 blocks of 8 warps share an SM: one plane, or the compact plane 1.
    static constexpr int DQ = (EW <= 5) ? 2 : 1;
    static constexpr int SCAP = 32 + 32 * QUAD * DQ;   // stack entries per warp: at most 31 left by the last drain + DQ quads
    static constexpr int PLANE_BYTES = SCAP * 16;      // plane 0 (and every non-compact plane): 16 bytes per entry
    static constexpr bool COMPACT1 = (EW == 5);        // EW == 6: measured slower (sparse 64-bit stores hardly conflict; the extra address costs an issue slot per step)
    static constexpr int P1SHIFT = EW == 5 ? 2 : 1;
    static constexpr int STACK_BYTES = COMPACT1 ? SCAP * 16 + SCAP * 4 * (EW - 4) : PLANES * SCAP * 16;   // per warp
    static_assert(STACK_BYTES % 16 == 0, "stacks stay 16-byte aligned");
    static constexpr uint32_t PAD = 0x40;               // value of unused slots (never reads as zero)
};

// ------------------------------------------------------------------------------------------------
// neighbour vectors
// ------------------------------------------------------------------------------------------------
// Byte-spread of the low L <= 4 bits of x: bit i -> bit 8i.
__device__ __forceinline__ uint32_t spread4(uint32_t x) { return (x * 0x00204081u) & 0x01010101u; }

// left_vec<b, INNER>: packed vector over slots of  unit(s) * x_{bit b + d_s}  (the LEFT neighbour of
// index bit b at distance d_s; it always exists for b <= n-3), as a 32-bit integer per register:
//     out[r] = sum_{s in r} unit(s) * x * 256^{s%4}      (signed bytes added as integers).
// INNER: only neighbours outside the inner bits (b + d_s >= H) are included.
// !INNER: the RIGHT neighbours (index bit b - d_s >= 0) are added too; at the moment outer bit b flips
//         the inner bits are all 0 (every block starts and ends there, see Walker::block_end), outer
//         bit b-1 is 1 (Gray order over the outer bits) and the outer bits below it are 0, so they
//         are compile-time constants.
template <int KIND, int NN, int b, bool INNER>
struct LeftVec {
    using L = Lay<KIND, NN>;
    // is slot s included, and does it start a run of slots whose neighbours are consecutive bits of E or O
    PAIRINGS_HD static bool included(int s) { return s < NN && !(INNER && b + L::d_of_slot(s) < H); }
    PAIRINGS_HD static bool run_start(int s) {
        if (!included(s)) return false;
        if (s % 4 == 0) return true;
        return !(included(s - 1) && L::d_of_slot(s - 1) == L::d_of_slot(s) - 2);
    }
    PAIRINGS_HD static int run_len(int s) {
        int len = 1;
        while ((s + len) % 4 != 0 && included(s + len) && L::d_of_slot(s + len) == L::d_of_slot(s) + 2 * len) len++;
        return len;
    }
    PAIRINGS_HD static uint32_t base(int r) {
        uint32_t v = 0;
        for (int o = 0; o < 4; o++) {
            const int s = 4 * r + o;
            if (s >= NN) continue;
            const int d = L::d_of_slot(s), u = L::unit(s);
            if (!INNER && d <= b) v += (uint32_t)((d == 1 && b > H) ? -u : u) << (8 * o);   // right neighbour, known
            if (included(s)) v += (uint32_t)u << (8 * o);                          // x = +1 part of the left neighbour
        }
        return v;
    }
    __device__ __forceinline__ static void eval(uint32_t E, uint32_t O, uint32_t (&out)[L::NR]) {
        static_for<0, L::NR>([&](auto rc) {
            PAIRINGS_IC(r, rc);
            uint32_t var = 0;
            static_for<0, 4>([&](auto oc) {
                PAIRINGS_IC(o, oc);
                constexpr int s = 4 * r + o;
                if constexpr (run_start(s)) {
                    constexpr int d = L::d_of_slot(s), u = L::unit(s), len = run_len(s);
                    const uint32_t word = ((b + d) & 1) ? O : E;
                    const uint32_t bits = (word >> ((b + d) >> 1)) & ((1u << len) - 1u);
                    var += spread4(bits) * (uint32_t)((2 * u) << (8 * o));       // a run shares the parity of d, hence the unit
                }
            });
            constexpr uint32_t bs = base(r);
            out[r] = bs - var;
        });
    }
};

// ------------------------------------------------------------------------------------------------
// compile-time constants of the unrolled inner blocks
// ------------------------------------------------------------------------------------------------
// inner state (bit set <-> x = -1) at inner step S of a block: every block starts at 0
PAIRINGS_HD int zbits(int s) { return gray_c(s); }

// K: contribution of the inner neighbours to dQ when inner bit bi flips in inner state zb
template <int KIND, int NN>
PAIRINGS_HD uint32_t kconst(int zb, int bi, int r) {
    using L = Lay<KIND, NN>;
    const int xo = 1 - 2 * ((zb >> bi) & 1);
    uint32_t K = 0;
    for (int o = 0; o < 4; o++) {
        const int s = 4 * r + o;
        if (s >= NN) continue;
        const int d = L::d_of_slot(s), u = L::unit(s);
        int nb = 0;
        if (bi + d < H) nb += 1 - 2 * ((zb >> (bi + d)) & 1);     // inner left neighbour
        if (bi - d >= 0) nb += 1 - 2 * ((zb >> (bi - d)) & 1);    // right neighbour (always inner)
        K += (uint32_t)(-u * xo * nb) << (8 * o);
    }
    return K;
}

// ------------------------------------------------------------------------------------------------
// zero-step tables (row a4 for a whole 32-step block at once)
// ------------------------------------------------------------------------------------------------
// Within one inner block only the H inner bits move, so an even-distance sum P_d takes the values
//     Q_d(S) = Q_d(0) + dQ_d(z(S), o),   z(S) = gray(S) the inner state, o = the signs of the (at most H)
// outer positions that are partners of an inner position for this d.  dQ_d is a fixed function: pairs
// (p, p+d) with p an inner index bit; the partner p+d is inner (p+d < H) or the outer index bit p+d.
// For d >= H all H partners are outer and the function is the same for every d ("generic" shape); d = 2
// and d = 4 have shapes of their own.  ztab[shape][Q_d(0) + ZR][o] is the 32-bit mask of the steps S at
// which P_d vanishes; OR-ing the masks of the even slots gives every zero term of the block with ~5
// instructions per slot and block instead of a 7-instruction test per step.
constexpr int ZR = 31;                                   // rows for Q_d(0) in [-ZR, ZR]  (n <= 32: |Q| <= 31)
constexpr int ZSHAPES = 3;                               // 0: d >= H, 1: d = 2, 2: d = 4
PAIRINGS_HD int zshape_of_d(int d) { return d >= H ? 0 : (d == 2 ? 1 : 2); }
PAIRINGS_HD int zshape_d(int shape) { return shape == 0 ? H : (shape == 1 ? 2 : 4); }   // a representative distance
struct alignas(128) ZeroTables { uint32_t t[ZSHAPES][2 * ZR + 1][32]; };
PAIRINGS_HD int zcontrib(int d, int z, int o) {          // sum over inner p of x_p * x_{p+d}
    int c = 0;
    for (int p = 0; p < H; p++) {
        const int xp = 1 - 2 * ((z >> p) & 1);
        const int q = p + d;
        // partner inside the inner bits, or pattern bit: outer index bit q, numbered from max(H, d)
        const int xq = q < H ? 1 - 2 * ((z >> q) & 1) : 1 - 2 * ((o >> (q - (d >= H ? d : H))) & 1);
        c += xp * xq;
    }
    return c;
}
PAIRINGS_HD ZeroTables make_zero_tables() {
    ZeroTables T{};
    for (int sh = 0; sh < ZSHAPES; sh++) {
        const int d = zshape_d(sh);
        for (int o = 0; o < 32; o++) {
            const int c0 = zcontrib(d, 0, o);
            for (int S = 0; S < BLK; S++) {                                  // Q(S) = q0 + dQ(S) = 0  <=>  q0 = -dQ(S)
                const int dq = (zcontrib(d, gray_c(S), o) - c0) / 2;
                T.t[sh][ZR - dq][o] |= 1u << S;
            }
        }
    }
    return T;
}
static_assert(H == 5 && BLK == 32, "the zero-step masks are 32-bit words indexed by 5 pattern bits");
static __device__ constexpr ZeroTables g_ztab = make_zero_tables();
// The same masks in the layout of the per-block copy in shared memory (long-lived blocks, KernelParams::ztab_shared):
// [shape][biased byte - ZB0][pattern 0..31] with rows of 33 words (132 bytes), so that the bank of a word is
// (byte + pattern) mod 32: lanes that share a pattern — every distance whose partners are walked bits — and differ in
// the byte, and lanes that share the byte and differ in the pattern, all hit different banks.  ONE dp4a forms
// 132 * byte + 4 * pattern.
constexpr int ZB0 = 128 - ZR - 1;                        // first biased byte value with a table row (64 rows)
constexpr int ZROW_BYTES = 132;                          // 32 patterns + one word of padding
constexpr int ZSH_BYTES = 64 * ZROW_BYTES;               // bytes per shape
constexpr int ZTAB_BYTES = ZSHAPES * ZSH_BYTES;
static_assert(2 * ZR + 1 <= 63 && ZB0 >= 0 && ZTAB_BYTES % 16 == 0 && ZROW_BYTES < 256, "64 rows hold every biased byte value [128 - ZR, 128 + ZR]");
struct alignas(16) ZeroTablesT { uint32_t t[ZSHAPES][64][ZROW_BYTES / 4]; };
PAIRINGS_HD ZeroTablesT make_zero_tables_t() {
    const ZeroTables T = make_zero_tables();
    ZeroTablesT U{};
    for (int sh = 0; sh < ZSHAPES; sh++)
        for (int pat = 0; pat < 32; pat++)
            for (int row = 0; row <= 2 * ZR; row++) U.t[sh][row + 1][pat] = T.t[sh][row][pat];   // row w <-> biased byte ZB0 + w
    return U;
}
static __device__ constexpr ZeroTablesT g_ztab_t = make_zero_tables_t();

// ------------------------------------------------------------------------------------------------
// stack entry -> signed multi-word term -> accumulator
// ------------------------------------------------------------------------------------------------
template <int W>
__device__ __forceinline__ void acc_add_signed(uint32_t (&acc)[W], const uint32_t* x /* W words, already ^mask */, uint32_t mask) {
    // acc += x + (mask & 1)  with carry propagation (two's complement add of +-T)
    uint32_t dummy;
    static_assert(W >= 2 && W <= 8, "accumulator width");
    if constexpr (W == 2) {
        asm volatile("add.cc.u32 %2, %5, 1;\n\taddc.cc.u32 %0, %0, %3;\n\taddc.u32 %1, %1, %4;"
                     : "+r"(acc[0]), "+r"(acc[1]), "=r"(dummy) : "r"(x[0]), "r"(x[1]), "r"(mask));
    } else if constexpr (W == 3) {
        asm volatile("add.cc.u32 %3, %7, 1;\n\taddc.cc.u32 %0, %0, %4;\n\taddc.cc.u32 %1, %1, %5;\n\taddc.u32 %2, %2, %6;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "=r"(dummy) : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(mask));
    } else if constexpr (W == 4) {
        asm volatile("add.cc.u32 %4, %9, 1;\n\taddc.cc.u32 %0, %0, %5;\n\taddc.cc.u32 %1, %1, %6;\n\taddc.cc.u32 %2, %2, %7;\n\taddc.u32 %3, %3, %8;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "=r"(dummy)
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(mask));
    } else if constexpr (W == 5) {
        asm volatile("add.cc.u32 %5, %11, 1;\n\taddc.cc.u32 %0, %0, %6;\n\taddc.cc.u32 %1, %1, %7;\n\taddc.cc.u32 %2, %2, %8;\n\t"
                     "addc.cc.u32 %3, %3, %9;\n\taddc.u32 %4, %4, %10;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "=r"(dummy)
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(mask));
    } else if constexpr (W == 6) {
        asm volatile("add.cc.u32 %6, %13, 1;\n\taddc.cc.u32 %0, %0, %7;\n\taddc.cc.u32 %1, %1, %8;\n\taddc.cc.u32 %2, %2, %9;\n\t"
                     "addc.cc.u32 %3, %3, %10;\n\taddc.cc.u32 %4, %4, %11;\n\taddc.u32 %5, %5, %12;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "+r"(acc[5]), "=r"(dummy)
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(mask));
    } else if constexpr (W == 7) {
        asm volatile("add.cc.u32 %7, %15, 1;\n\taddc.cc.u32 %0, %0, %8;\n\taddc.cc.u32 %1, %1, %9;\n\taddc.cc.u32 %2, %2, %10;\n\t"
                     "addc.cc.u32 %3, %3, %11;\n\taddc.cc.u32 %4, %4, %12;\n\taddc.cc.u32 %5, %5, %13;\n\taddc.u32 %6, %6, %14;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "+r"(acc[5]), "+r"(acc[6]), "=r"(dummy)
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(mask));
    } else {
        asm volatile("add.cc.u32 %8, %17, 1;\n\taddc.cc.u32 %0, %0, %9;\n\taddc.cc.u32 %1, %1, %10;\n\taddc.cc.u32 %2, %2, %11;\n\t"
                     "addc.cc.u32 %3, %3, %12;\n\taddc.cc.u32 %4, %4, %13;\n\taddc.cc.u32 %5, %5, %14;\n\taddc.cc.u32 %6, %6, %15;\n\t"
                     "addc.u32 %7, %7, %16;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "+r"(acc[5]), "+r"(acc[6]), "+r"(acc[7]), "=r"(dummy)
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(x[7]), "r"(mask));
    }
}

// acc += x  (W-word two's complement add with carry propagation)
template <int W>
__device__ __forceinline__ void acc_add(uint32_t (&acc)[W], const uint32_t (&x)[W]) {
    static_assert(W >= 2 && W <= 8, "accumulator width");
    if constexpr (W == 2) {
        asm volatile("add.cc.u32 %0, %0, %2;\n\taddc.u32 %1, %1, %3;"
                     : "+r"(acc[0]), "+r"(acc[1])
                     : "r"(x[0]), "r"(x[1]));
    }
    else if constexpr (W == 3) {
        asm volatile("add.cc.u32 %0, %0, %3;\n\taddc.cc.u32 %1, %1, %4;\n\taddc.u32 %2, %2, %5;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2])
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]));
    }
    else if constexpr (W == 4) {
        asm volatile("add.cc.u32 %0, %0, %4;\n\taddc.cc.u32 %1, %1, %5;\n\taddc.cc.u32 %2, %2, %6;\n\taddc.u32 %3, %3, %7;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3])
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]));
    }
    else if constexpr (W == 5) {
        asm volatile("add.cc.u32 %0, %0, %5;\n\taddc.cc.u32 %1, %1, %6;\n\taddc.cc.u32 %2, %2, %7;\n\taddc.cc.u32 %3, %3, %8;\n\taddc.u32 %4, %4, %9;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4])
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]));
    }
    else if constexpr (W == 6) {
        asm volatile("add.cc.u32 %0, %0, %6;\n\taddc.cc.u32 %1, %1, %7;\n\taddc.cc.u32 %2, %2, %8;\n\taddc.cc.u32 %3, %3, %9;\n\taddc.cc.u32 %4, %4, %10;\n\taddc.u32 %5, %5, %11;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "+r"(acc[5])
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]));
    }
    else if constexpr (W == 7) {
        asm volatile("add.cc.u32 %0, %0, %7;\n\taddc.cc.u32 %1, %1, %8;\n\taddc.cc.u32 %2, %2, %9;\n\taddc.cc.u32 %3, %3, %10;\n\taddc.cc.u32 %4, %4, %11;\n\taddc.cc.u32 %5, %5, %12;\n\taddc.u32 %6, %6, %13;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "+r"(acc[5]), "+r"(acc[6])
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]));
    }
    else if constexpr (W == 8) {
        asm volatile("add.cc.u32 %0, %0, %8;\n\taddc.cc.u32 %1, %1, %9;\n\taddc.cc.u32 %2, %2, %10;\n\taddc.cc.u32 %3, %3, %11;\n\taddc.cc.u32 %4, %4, %12;\n\taddc.cc.u32 %5, %5, %13;\n\taddc.cc.u32 %6, %6, %14;\n\taddc.u32 %7, %7, %15;"
                     : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(acc[4]), "+r"(acc[5]), "+r"(acc[6]), "+r"(acc[7])
                     : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(x[7]));
    }
}

// predicated on a CLEAR bit: store iff (word & bit) == 0 — the same test as the ballot's, so one predicate serves both
__device__ __forceinline__ void sts_v4_clr(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t word, uint32_t bit) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tand.b32 t, %5, %6;\n\tsetp.eq.u32 p, t, 0;\n\t@p st.shared.v4.u32 [%0], {%1, %2, %3, %4};\n\t}"
                 :: "r"(addr), "r"(a), "r"(b), "r"(c), "r"(d), "r"(word), "r"(bit) : "memory");
}
__device__ __forceinline__ void sts_v2_clr(uint32_t addr, uint32_t a, uint32_t b, uint32_t word, uint32_t bit) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tand.b32 t, %3, %4;\n\tsetp.eq.u32 p, t, 0;\n\t@p st.shared.v2.u32 [%0], {%1, %2};\n\t}"
                 :: "r"(addr), "r"(a), "r"(b), "r"(word), "r"(bit) : "memory");
}
__device__ __forceinline__ void sts_v1_clr(uint32_t addr, uint32_t a, uint32_t word, uint32_t bit) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tand.b32 t, %2, %3;\n\tsetp.eq.u32 p, t, 0;\n\t@p st.shared.u32 [%0], %1;\n\t}"
                 :: "r"(addr), "r"(a), "r"(word), "r"(bit) : "memory");
}
// slot += 16 iff (word & bit) == 0 — the same predicate as the stores of that step
__device__ __forceinline__ void add16_clr(uint32_t& slot, uint32_t word, uint32_t bit) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tand.b32 t, %1, %2;\n\tsetp.eq.u32 p, t, 0;\n\t@p add.u32 %0, %0, 16;\n\t}"
                 : "+r"(slot) : "r"(word), "r"(bit));
}
// one Kogge-Stone step of an inclusive scan over the lanes, two words at a time (byte fields that cannot overflow)
template <int D>
__device__ __forceinline__ void scan_up2(uint32_t& a, uint32_t& b) {
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t, u;\n\t"
                 "shfl.sync.up.b32 t|p, %0, %2, 0, 0xffffffff;\n\t"
                 "shfl.sync.up.b32 u, %1, %2, 0, 0xffffffff;\n\t"
                 "@p add.u32 %0, %0, t;\n\t@p add.u32 %1, %1, u;\n\t}" : "+r"(a), "+r"(b) : "n"(D));
}
__device__ __forceinline__ void lds_v2(uint32_t addr, uint32_t& a, uint32_t& b) {
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(addr) : "memory");
}
__device__ __forceinline__ void lds_v1(uint32_t addr, uint32_t& a) {
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a) : "r"(addr) : "memory");
}
__device__ __forceinline__ void lds_v4(uint32_t addr, uint32_t& a, uint32_t& b, uint32_t& c, uint32_t& d) {
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(addr) : "memory");
}

// sign-extended byte i of w (one PRMT: selector nibble i, then three times "replicate its sign")
template <int i>
__device__ __forceinline__ int sbyte(uint32_t w) {
    uint32_t r;   // (__byte_perm masks the selector's replicate-sign bits, prmt.b32 does not)
    asm("prmt.b32 %0, %1, 0, %2;" : "=r"(r) : "r"(w), "n"(0x8880 + 0x1111 * i));
    return (int)r;
}

// signed 32 x 32 -> 64 (+ 64) as ONE IMAD.WIDE each; hi / lo words of a 64-bit value
__device__ __forceinline__ long long mulw(int a, int b) { long long r; asm("mul.wide.s32 %0, %1, %2;" : "=l"(r) : "r"(a), "r"(b)); return r; }
__device__ __forceinline__ long long madw(int a, int b, long long c) { long long r; asm("mad.wide.s32 %0, %1, %2, %3;" : "=l"(r) : "r"(a), "r"(b), "l"(c)); return r; }
__device__ __forceinline__ void split64(long long v, uint32_t& lo, uint32_t& hi) { asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(v)); }
// signed digits of a 64-bit value: v = d1 * 2^32 + d0 with d0 = (int) low word
__device__ __forceinline__ void digits64(long long v, int& d0, int& d1) {
    uint32_t lo, hi; split64(v, lo, hi);
    d0 = (int)lo; d1 = (int)(hi + (lo >> 31));
}
// v >> 32 (arithmetic) as a 64-bit value: the sign-extended upper half
__device__ __forceinline__ long long upper64(long long v) {
    uint32_t lo, hi; split64(v, lo, hi);
    long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(hi), "r"((uint32_t)((int)hi >> 31)));
    return r;
}

// One stack entry (at shared byte address `addr` in plane 0) -> signed multi-word term -> acc.
template <int KIND, int NN>
__device__ __forceinline__ void drain_entry(uint32_t addr, uint32_t k1, uint32_t (&acc)[Lay<KIND, NN>::W], uint32_t c80) {
    using L = Lay<KIND, NN>;
    constexpr int NR = L::NR, G = L::G, W = L::W, PL = L::PLANES;
    uint32_t e[4 * PL];
    if constexpr (L::COMPACT1) {
        lds_v4(addr, e[0], e[1], e[2], e[3]);
        const uint32_t a1 = (addr >> L::P1SHIFT) + k1;
        if constexpr (L::EW == 5) lds_v1(a1, e[4]); else lds_v2(a1, e[4], e[5]);
    } else {
        static_for<0, PL>([&](auto pc) {
            PAIRINGS_IC(pl, pc);
            lds_v4(addr + pl * L::PLANE_BYTES, e[4 * pl], e[4 * pl + 1], e[4 * pl + 2], e[4 * pl + 3]);
        });
    }
    uint32_t w[NR];
    static_for<0, NR>([&](auto rc) {                                              // bytes -> two's complement Q
        PAIRINGS_IC(r, rc);
        constexpr bool ub = L::plan.unbias[r];
        w[r] = ub ? (e[r] ^ 0x80808080u) : 0u;
    });
    int gp[G];
#pragma unroll
    for (int g = 0; g < G; g++) gp[g] = 1;
    // sign of the term from the slot of distance n (biased byte u): n even: Q = P/2 = n/2 - pc, pc odd <=> (u ^ n/2) odd;
    // n odd: Q = P = n - 2 pc, pc odd <=> bit 1 of (u - n) set.  (Subtracting inside byte i never borrows from below.)
    {
        constexpr int r = L::SIGN_SLOT / 4, i = L::SIGN_SLOT % 4;
        bool negative;
        if constexpr (NN % 2 == 0) negative = (((e[r] >> (8 * i)) ^ (uint32_t)(NN / 2)) & 1u) != 0;
        else negative = (((e[r] - ((uint32_t)NN << (8 * i))) >> (8 * i + 1)) & 1u) != 0;
        gp[0] = negative ? -1 : 1;
    }
    static_for<0, L::NF_MAX>([&](auto fc) {
        PAIRINGS_IC(f, fc);
        if constexpr (f < L::plan.nf) {
            constexpr int kind = L::plan.kind[f], r = L::plan.r[f], i = L::plan.i[f], g = L::plan.group[f];
            int v;
            if constexpr (kind == 1) {          // Q[4r+i] * Q[4(r+1)+i]: second operand = ((e ^ 0x80..) & byte i)
                uint32_t b;
                asm("lop3.b32 %0, %1, %2, %3, 0x28;" : "=r"(b) : "r"(e[r + 1]), "r"(c80), "n"(0xFFu << (8 * i)));
                v = __dp4a((int)w[r], (int)b, 0);
            } else if constexpr (kind == 2) {   // Q[4r+i] * Q[4r+i+1]: second operand = byte i+1 moved to byte i
                const uint32_t b = __byte_perm(w[r], 0, i == 0 ? 0x4441 : 0x4344);
                v = __dp4a((int)w[r], (int)b, 0);
            } else {
                v = sbyte<i>(w[r]);
            }
            gp[g] *= v;                                                           // exact: |group| < 2^31
        }
    });
    if constexpr (G <= 4) {
        // signed multi-word product T = gp[0] * gp[1] * ... (two's complement, top word signed) from signed 64-bit
        // pieces only: a 64-bit product A = a1 * 2^32 + a0 is split with a SIGNED low digit a0 = (int) low word,
        // a1 = high word + bit 31 of the low word, so every partial product is one signed IMAD.WIDE whose 64-bit
        // addend carries the sign-extended upper half of the digit below — no unsigned-times-signed corrections.
        uint32_t T[W];
        if constexpr (G == 1) {
            T[0] = (uint32_t)gp[0];
        } else if constexpr (G == 2) {
            split64(mulw(gp[0], gp[1]), T[0], T[1]);
        } else if constexpr (G == 3) {
            int a0, a1; digits64(mulw(gp[0], gp[1]), a0, a1);                   // |A| < 2^62
            const long long X = mulw(a0, gp[2]);
            const long long Y = madw(a1, gp[2], upper64(X));
            uint32_t xh; split64(X, T[0], xh); split64(Y, T[1], T[2]);
        } else {
            int a0, a1, b0, b1;
            digits64(mulw(gp[0], gp[1]), a0, a1); digits64(mulw(gp[2], gp[3]), b0, b1);
            const long long X = mulw(a0, b0);
            const long long Y = madw(a0, b1, madw(a1, b0, upper64(X)));          // |a1 b0|, |a0 b1| <= 2^61
            const long long Z = madw(a1, b1, upper64(Y));
            uint32_t xh, yh; split64(X, T[0], xh); split64(Y, T[1], yh); split64(Z, T[2], T[3]);
        }
        const uint32_t sext = (uint32_t)((int)T[G - 1] >> 31);    // sign words above the G-word product
#pragma unroll
        for (int i = G; i < W; i++) T[i] = sext;
        acc_add<W>(acc, T);
    } else {
        // sign-magnitude: multi-word product of |gp[i]|
        uint32_t sx = 0;
#pragma unroll
        for (int g = 0; g < G; g++) sx ^= (uint32_t)gp[g];
        const uint32_t mask = (uint32_t)((int)sx >> 31);                              // all ones iff the term is negative
        uint32_t T[W];
#pragma unroll
        for (int i = 0; i < W; i++) T[i] = 0;
        T[0] = (uint32_t)abs(gp[0]);
#pragma unroll
        for (int g = 1; g < G; g++) {
            const uint32_t m = (uint32_t)abs(gp[g]);
            uint32_t carry = 0;
#pragma unroll
            for (int i = 0; i < g; i++) {
                const uint64_t p = (uint64_t)T[i] * m + carry;
                T[i] = (uint32_t)p; carry = (uint32_t)(p >> 32);
            }
            T[g] = carry;
        }
#pragma unroll
        for (int i = 0; i < W; i++) T[i] ^= mask;
        acc_add_signed<W>(acc, T, mask);
    }
}

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
template <int KIND, int NN>
struct Walker {
    using L = Lay<KIND, NN>;
    static constexpr int NR = L::NR, W = L::W, EW = L::EW;

    uint32_t Q[NR];
    uint32_t C[H][NR];
    uint32_t E, O;            // de-interleaved sign word: E bit i = index bit 2i, O bit i = index bit 2i+1
    uint32_t acc[W];
    // Non-zero terms go to a per-warp STACK in shared memory (the sum is commutative: any lane may multiply any
    // entry, in any order).  top = shared byte address (plane 0) of the first free entry, warp-uniform.
    uint32_t top;
    uint32_t lim;             // stack base + 32 entries: a full drain round is possible while top >= lim
    uint32_t k1;              // compact plane 1: address of an entry's words 4.. = (plane-0 address >> P1SHIFT) + k1
    uint32_t ztab;            // shared address of the block's zero-step tables, minus ZROW_BYTES * ZB0 (the dp4a offset starts at the
                              // byte value); 0 = no copy in shared memory: read the tables in global memory (short-lived blocks)
    uint32_t lane16;          // lane * 16
    uint32_t c80;             // 0x80808080 (KernelParams::c80)
    uint32_t Vo;              // outer sign word: bit i = index bit H + i (set <-> x = -1)
    uint32_t ZM;              // zero-step mask of the current block: bit S set <-> the term of step S has a zero factor
    // Slot plan of the current block, from ZM alone (known before the first step): byte j of ex[w] = number of
    // non-zero steps of quad 2j+w in the lanes below this one, byte j of tot[w] = that count over the whole warp.
    uint32_t ex[2], tot[2];
    uint32_t slot;            // this lane's next free entry of the current quad (lane-major inside a quad)
    uint32_t nzc;             // non-zero terms pushed by this lane (32-bit: reset per prefix)

    // Row a4 for the whole block: OR over the even-distance slots of the table masks (see ztab above).
    __device__ __forceinline__ void zero_mask() {
        uint32_t zm = 0;
        if (ztab != 0) {                              // warp-uniform (kernel parameter): the block's copy in shared memory
            static_for<0, L::n_even()>([&](auto sc) {
                PAIRINGS_IC(s, sc);
                constexpr int d = L::d_of_slot(s), sh = zshape_of_d(d);
                static_assert(L::bound(s) <= ZR, "table rows");
                uint32_t pat4;                                                              // 4 * pattern
                if constexpr (d >= H + 2) pat4 = (Vo >> (d - H - 2)) & 0x7Cu;
                else if constexpr (d >= H) pat4 = (Vo << (H + 2 - d)) & 0x7Cu;
                else pat4 = (Vo << 2) & (((1u << d) - 1u) << 2);
                // ONE dp4a: 132 * (biased byte of the slot) + 4 * pattern; the shape's base is an immediate of the load
                const uint32_t off = __dp4a(Q[s / 4], (uint32_t)ZROW_BYTES << (8 * (s % 4)), pat4);
                uint32_t mask;
                lds_v1(ztab + (uint32_t)(sh * ZSH_BYTES) + off, mask);
                zm |= mask;
            });
        } else {                                      // short-lived blocks: the tables in global memory (L1-resident)
            static_for<0, L::n_even()>([&](auto sc) {
                PAIRINGS_IC(s, sc);
                constexpr int d = L::d_of_slot(s), sh = zshape_of_d(d);
                const uint32_t u = __byte_perm(Q[s / 4], 0, 0x4440 + (s % 4));             // biased byte Q + 128
                uint32_t pat4;                                                              // 4 * pattern (byte offset in the row)
                if constexpr (d >= H + 2) pat4 = (Vo >> (d - H - 2)) & 0x7Cu;
                else if constexpr (d >= H) pat4 = (Vo << (H + 2 - d)) & 0x7Cu;
                else pat4 = (Vo << 2) & (((1u << d) - 1u) << 2);
                // address = table(shape) + (u - 128 + ZR) * 128 + pat4: the tables are 128-byte aligned, so pat4 is OR-ed
                // into the low word of the (biased) base and ONE wide multiply-add forms the 64-bit address
                const uint64_t base = (uint64_t)(uintptr_t)(&g_ztab.t[sh][0][0]) + (uint64_t)(int64_t)((ZR - 128) * 128);
                uint64_t addr;
                asm("{\n\t.reg .b32 lo, hi;\n\t.reg .b64 bp;\n\tmov.b64 {lo, hi}, %2;\n\tor.b32 lo, lo, %3;\n\tmov.b64 bp, {lo, hi};\n\t"
                    "mad.wide.u32 %0, %1, 128, bp;\n\t}" : "=l"(addr) : "r"(u), "l"(base), "r"(pat4));
                uint32_t mask;
                asm("ld.global.nc.u32 %0, [%1];" : "=r"(mask) : "l"(addr));
                zm |= mask;
            });
        }
        ZM = zm;
        // ---- slot plan: per-lane counts of the non-zero steps of each quad (nibble popcounts of ~ZM), then an
        // inclusive scan over the lanes in byte fields (a field is at most 4 * 32 = 128)
        const uint32_t nzm = ~zm;
        uint32_t x = nzm - ((nzm >> 1) & 0x55555555u);
        x = (x & 0x33333333u) + ((x >> 2) & 0x33333333u);                  // nibble q = steps 4q .. 4q+3
        const uint32_t c0 = x & 0x0F0F0F0Fu, c1 = (x >> 4) & 0x0F0F0F0Fu;   // byte j of c0: quad 2j, of c1: quad 2j+1
        uint32_t s0 = c0, s1 = c1;
        scan_up2<1>(s0, s1); scan_up2<2>(s0, s1); scan_up2<4>(s0, s1); scan_up2<8>(s0, s1); scan_up2<16>(s0, s1);
        ex[0] = s0 - c0; ex[1] = s1 - c1;                                  // no borrow: s >= c in every byte
        // warp totals by REDUX (a byte sum is at most 128: no carry between fields): provably warp-uniform, which the
        // stack pointer and every drain loop inherit — the compiler then knows the warp stays converged
        tot[0] = __reduce_add_sync(0xffffffffu, c0); tot[1] = __reduce_add_sync(0xffffffffu, c1);
        if constexpr (L::DQ == 2) ex[1] += tot[0];     // quads 2j and 2j+1 are pushed from the same stack pointer: 124 + 128 < 256
        nzc += (uint32_t)__popc(nzm);
    }

    template <int S>
    __device__ __forceinline__ void push_if_nonzero() {
        constexpr uint32_t bit = 1u << S;
        // entry words: Q[0..NR); plane p holds words 4p..4p+3 (predicated vector stores, no branch)
        if constexpr (L::COMPACT1) {
            sts_v4_clr(slot, Q[0], Q[1], Q[2], Q[3], ZM, bit);
            const uint32_t a1 = (slot >> L::P1SHIFT) + k1;
            if constexpr (EW == 5) sts_v1_clr(a1, Q[4], ZM, bit); else sts_v2_clr(a1, Q[4], Q[5], ZM, bit);
        } else {
            uint32_t e[4 * L::PLANES];
#pragma unroll
            for (int i = 0; i < 4 * L::PLANES; i++) e[i] = Q[i < NR ? i : 0];
            static_for<0, L::PLANES>([&](auto pc) {
                PAIRINGS_IC(pl, pc);
                constexpr int words = (EW - 4 * pl) >= 4 ? 4 : (EW - 4 * pl);
                if constexpr (words >= 3) sts_v4_clr(slot + pl * L::PLANE_BYTES, e[4 * pl], e[4 * pl + 1], e[4 * pl + 2], e[4 * pl + 3], ZM, bit);
                else if constexpr (words == 2) sts_v2_clr(slot + pl * L::PLANE_BYTES, e[4 * pl], e[4 * pl + 1], ZM, bit);
                else sts_v1_clr(slot + pl * L::PLANE_BYTES, e[4 * pl], ZM, bit);
            });
        }
        if constexpr (S % QUAD != QUAD - 1) add16_clr(slot, ZM, bit);
    }

    __device__ __forceinline__ void drain_full() {
        if constexpr (L::EW <= PAIRINGS_DRAIN2_MAXEW) {
            while (top >= lim + 32u * 16u) {                   // two rounds at once: half the loop overhead, the loads overlap
                top -= 64u * 16u;
                __syncwarp();
                drain_entry<KIND, NN>(top + lane16, k1, acc, c80);
                drain_entry<KIND, NN>(top + 32u * 16u + lane16, k1, acc, c80);
                __syncwarp();
            }
        }
        while (top >= lim) {                                   // warp-uniform
            top -= 32u * 16u;
            __syncwarp();
            drain_entry<KIND, NN>(top + lane16, k1, acc, c80);
            __syncwarp();
        }
    }

    __device__ __forceinline__ void drain_rest() {
        drain_full();
        const uint32_t base = lim - 32u * 16u;
        __syncwarp();
        if (lane16 < top - base) drain_entry<KIND, NN>(base + lane16, k1, acc, c80);
        top = base;
        __syncwarp();
    }

    // QUAD consecutive steps of the unrolled inner block, starting at step QUAD*QI: test + push the
    // current term, then flip inner bit ctz(S+1) (the block's last step is followed by block_end).
    template <int QI>
    __device__ __forceinline__ void quad() {
        constexpr uint32_t sel16 = 16u << (8 * (QI >> 1));                 // 16 * byte (QI >> 1) of word (QI & 1)
        slot = __dp4a(ex[QI & 1], sel16, 0u) + top;                        // top is warp-uniform (uniform datapath)
        static_for<QUAD * QI, QUAD * QI + QUAD>([&](auto sc) {
            PAIRINGS_IC(S, sc);
            push_if_nonzero<S>();
            if constexpr (S + 1 < BLK) inner_flip<zbits(S), ctz_c(S + 1)>();
        });
        constexpr int sh = 8 * (QI >> 1);                                  // uniform datapath: shift, mask, add
        if constexpr (L::DQ == 1) {
            if constexpr (sh >= 4) top += (tot[QI & 1] >> (sh - 4)) & 0xFF0u; else top += (tot[QI & 1] << 4) & 0xFF0u;
        } else if constexpr (QI & 1) {                                     // both quads of the pair at once
            if constexpr (sh >= 4) top += ((tot[0] >> (sh - 4)) & 0xFF0u) + ((tot[1] >> (sh - 4)) & 0xFF0u);
            else top += ((tot[0] << 4) & 0xFF0u) + ((tot[1] << 4) & 0xFF0u);
        }
    }

    // flip of inner bit bi in inner state ZB: dQ = -x_j * C[bi] + K  (row a3; K = inner neighbours, folded)
    template <int ZB, int bi>
    __device__ __forceinline__ void inner_flip() {
        constexpr int xo = 1 - 2 * ((ZB >> bi) & 1);                                 // old x_j
        static_for<0, NR>([&](auto rc) {
            PAIRINGS_IC(r, rc);
            constexpr uint32_t K = kconst<KIND, NN>(ZB, bi, r);
            if constexpr (xo > 0) Q[r] = Q[r] - C[bi][r] + K;
            else Q[r] = Q[r] + C[bi][r] + K;
        });
    }

    // Between two blocks: the inner walk ended in state 1 << (H-1); flip that bit back so that every
    // block runs the same compile-time sequence from inner state 0, then flip outer bit `bit`.
    __device__ __forceinline__ void block_end(int bit) {
        inner_flip<(1 << (H - 1)), H - 1>();
        outer_flip_dispatch<H>(bit);
    }

    // flip of index bit b >= H (between two inner blocks)
    template <int b>
    __device__ __forceinline__ void outer_flip() {
        const uint32_t word = (b & 1) ? O : E;
        const uint32_t sg = 1u - 2u * ((word >> (b >> 1)) & 1u);       // old x_j as +-1 (mod 2^32)
        uint32_t t[NR];
        LeftVec<KIND, NN, b, false>::eval(E, O, t);
        static_for<0, NR>([&](auto rc) { PAIRINGS_IC(r, rc); Q[r] -= sg * t[r]; });   // dQ = -x_j * (left + right neighbours)
        static_for<0, H>([&](auto bc) {
            PAIRINGS_IC(bi, bc);
            constexpr int s = L::slot_of_d(b - bi);
            if constexpr (s >= 0) {
                // byte s of C[bi] holds unit * x_j and x_j changes sign: delta = -2 * unit * old x_j
                constexpr uint32_t k = (uint32_t)((2 * L::unit(s)) << (8 * (s % 4)));
                C[bi][s / 4] -= sg * k;
            }
        });
        if (b & 1) O ^= 1u << (b >> 1); else E ^= 1u << (b >> 1);
        Vo ^= 1u << (b - H);
    }

    template <int b>
    __device__ __forceinline__ void outer_flip_dispatch(int bit) {
        if constexpr (b <= NN - 3) {
            if (bit == b) outer_flip<b>(); else outer_flip_dispatch<b + 1>(bit);
        }
    }

    // direct evaluation for the prefix V (low g bits zero): Q, C[0..H), E, O  (row a2)
    __device__ __forceinline__ void init_prefix(uint64_t V) {
        static_for<0, NR>([&](auto rc) {
            PAIRINGS_IC(r, rc);
            uint32_t q = 0;
            static_for<0, 4>([&](auto oc) {
                PAIRINGS_IC(o, oc);
                constexpr int s = 4 * r + o;
                if constexpr (s >= NN) { q |= L::PAD << (8 * o); }
                else {
                    constexpr int d = L::d_of_slot(s), c = L::cnt(s);
                    const int pc = __popcll((V ^ (V >> d)) & ((1ULL << c) - 1ULL));
                    const int qv = (L::unit(s) == 1) ? (c / 2 - pc) : (c - 2 * pc);
                    q |= (uint32_t)(qv + 128) << (8 * o);
                }
            });
            Q[r] = q;
        });
        uint32_t e = 0, o = 0;                                          // de-interleave
#pragma unroll
        for (int i = 0; i < 32; i++) {
            e |= (uint32_t)((V >> (2 * i)) & 1ULL) << i;
            o |= (uint32_t)((V >> (2 * i + 1)) & 1ULL) << i;
        }
        E = e; O = o;
        Vo = (uint32_t)(V >> H);
        static_for<0, H>([&](auto bc) { PAIRINGS_IC(bi, bc); LeftVec<KIND, NN, bi, true>::eval(E, O, C[bi]); });
    }
};

template <int KIND, int NN>
#ifndef PAIRINGS_SWAR_MINB
#define PAIRINGS_SWAR_MINB 3   // 3 blocks of 256 threads per SM : at most 85 registers; measured faster than 2 blocks without spills at n = 24
#endif
#ifndef PAIRINGS_SWAR_BIG_N
#define PAIRINGS_SWAR_BIG_N 25   // 7-8 packed registers, 35-40 neighbour registers: 2 blocks per SM without spills (measured: S(25) +4 %, L(27) +1.5 %, S(29) +7 % over 3 blocks with spills; n = 24 is 1 % faster with 3)
#endif
#ifndef PAIRINGS_SWAR_MAXT
#define PAIRINGS_SWAR_MAXT 256
#endif
__global__ void __launch_bounds__(PAIRINGS_SWAR_MAXT, (NN >= PAIRINGS_SWAR_BIG_N ? 2 : PAIRINGS_SWAR_MINB))
swar_kernel(const __grid_constant__ KernelParams kp) {
    using L = Lay<KIND, NN>;
    using Wk = Walker<KIND, NN>;
    constexpr int N = L::N, B = N - 1, W = L::W;
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // dynamic shared memory (16-byte aligned): [zero-step tables][stacks: warps x STACK_BYTES][reduction scratch]
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t ztab_bytes = kp.ztab_shared ? (uint32_t)ZTAB_BYTES : 0u;
    const uint32_t stacks = smem0 + ztab_bytes;
    if (kp.ztab_shared) {                                                        // 24 KB, coalesced 16-byte copies
        const uint4* src = reinterpret_cast<const uint4*>(&g_ztab_t.t[0][0][0]);
        uint4* dst = reinterpret_cast<uint4*>(smem);
        for (int i = threadIdx.x; i < ZTAB_BYTES / 16; i += blockDim.x) dst[i] = __ldg(src + i);
        __syncthreads();
    }
    const uint32_t stack_bytes = (blockDim.x >> 5) * (uint32_t)L::STACK_BYTES;
    unsigned long long* red = reinterpret_cast<unsigned long long*>(
        reinterpret_cast<unsigned char*>(smem) + ztab_bytes + stack_bytes);                       // 8 * 16 uint64

    const int C = kp.chunk_bits, g = kp.gray_bits;
    const uint64_t chunk_local = (uint64_t)blockIdx.x >> kp.log2_bpc;
    const uint64_t sub = (uint64_t)blockIdx.x & ((1ULL << kp.log2_bpc) - 1);
    const uint64_t chunk = kp.chunk_begin + chunk_local;
    const int tb = B - C;
    const uint64_t per_block = (1ULL << (tb - g)) >> kp.log2_bpc;     // multiple of blockDim (host)
    const uint64_t chunk_base = chunk << tb;                          // tb >= H > 0
    const uint32_t nblk = 1u << (g - H);

    Wk wk;
    wk.lane16 = (uint32_t)lane * 16u;
    wk.c80 = kp.c80;
    const uint32_t warp_u = __reduce_min_sync(0xffffffffu, (unsigned)warp);          // the same value, known to be warp-uniform
    wk.top = stacks + warp_u * (uint32_t)L::STACK_BYTES;
    wk.lim = wk.top + 32u * 16u;
    wk.ztab = kp.ztab_shared ? smem0 - (uint32_t)(ZROW_BYTES * ZB0) : 0u;
    wk.k1 = wk.top + (uint32_t)L::PLANE_BYTES - (wk.top >> L::P1SHIFT);     // plane 1 starts behind plane 0
#pragma unroll
    for (int i = 0; i < W; i++) wk.acc[i] = 0;
    unsigned long long nz = 0;

    // per_block is a multiple of blockDim (host): a block-uniform trip count keeps the warps provably converged
    const uint32_t rounds = (uint32_t)(per_block / blockDim.x);
#pragma unroll 1
    for (uint32_t rd = 0; rd < rounds; rd++) {
        const uint64_t q = sub * per_block + (uint64_t)rd * blockDim.x + threadIdx.x;
        wk.init_prefix(chunk_base | (q << g));
        wk.nzc = 0;
        // One inner block = BLK unrolled steps from inner state 0, a drain check every DQ quads.
#pragma unroll 1
        for (uint32_t u = 0; u < nblk; u++) {
            wk.zero_mask();
            static_for<0, BLK / QUAD>([&](auto qc) {
                PAIRINGS_IC(QI, qc);
                wk.template quad<QI>();
                if constexpr (QI % L::DQ == L::DQ - 1) wk.drain_full();
            });
            if (u + 1 < nblk) wk.block_end(H + (__ffs((int)(u + 1)) - 1));      // Gray order over the outer bits
        }
        nz += (unsigned long long)wk.nzc;
    }
    wk.drain_rest();

    // ---- once per thread: accumulator (W-word two's complement) -> residues, times 2^{#even}
    uint32_t vals[PAIRINGS_MAX_MODULI];
    const bool neg = (wk.acc[W - 1] >> 31) != 0;
#pragma unroll 1
    for (int i = 0; i < kp.n_moduli; i++) {
        const MontPrime mp = kp.primes[i];
        uint32_t r = 0;
        uint32_t pw = mp.r1;                                           // 2^{32 j} mod p
#pragma unroll
        for (int j = W - 1; j >= 0; j--) {
            r = montmul(r, mp.r2, mp.p, mp.pinv_neg) + montmul(wk.acc[j], mp.r1, mp.p, mp.pinv_neg);   // r*2^32 + acc[j]
            if (r >= mp.p) r -= mp.p;
        }
#pragma unroll
        for (int j = 1; j < W; j++) pw = montmul(pw, mp.r2, mp.p, mp.pinv_neg);                        // 2^{32 W} mod p
        if (neg) { r = (r >= pw) ? r - pw : r + mp.p - pw; }
        const uint32_t two_ne = montmul(1u << L::n_even(), mp.r2, mp.p, mp.pinv_neg);                  // 2^{#even} * 2^32
        vals[i] = montmul(r, two_ne, mp.p, mp.pinv_neg);
    }
    __syncthreads();
    block_reduce_write(kp, vals, nz, red, chunk_local);
}

template <int KIND, int NN>
int launch(const KernelParams& kp, int block_threads, unsigned grid, void* stream) {
    using L = Lay<KIND, NN>;
    const size_t smem = (size_t)(kp.ztab_shared ? ZTAB_BYTES : 0) + (size_t)(block_threads / 32) * L::STACK_BYTES
                      + (size_t)(8 * PAIRINGS_MAX_MODULI * 2) * sizeof(uint32_t);
    cudaError_t e = cudaFuncSetAttribute(swar_kernel<KIND, NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    swar_kernel<KIND, NN><<<grid, block_threads, smem, (cudaStream_t)stream>>>(kp);
    return (int)cudaGetLastError();
}

}  // namespace swar
}  // namespace pairings
