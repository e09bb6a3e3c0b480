/* pairings.h — C ABI of libpairings_b200.so
 *
 * Exact counting of Skolem pairings S(n) and Langford pairings L(n) by Godfrey's algebraic
 * sign-vector sum ("Counting Skolem Sequences", arxiv 1507.00315, §2.1, Lemma 2.1,
 * PAPER.md:166-168):
 *
 *      D(n) = 2^{-2n} * sum_{x in {+1,-1}^{2n}} (prod_i x_i) * prod_{k=1}^{n} P_k(x),
 *      P_k(x) = sum_{i=1}^{2n-d_k} x_i x_{i+d_k},   d_k = k (Skolem)  or  k+1 (Langford).
 *
 * D(n) counts reflected sequences as distinct (A004075 / A176127); the paper's headline numbers
 * S(n), L(n) identify reflections and are D(n)/2 for n > 1.  Lemma 2.2
 * lets x_1 be fixed to +1:  H = sum_{x: x_1=+1} term(x) = 2^{2n-1} D(n).
 *
 * The path:  host partitioner (pairings_partition / journal)  ->
 * count_pairings (one sm_100a kernel per chunk range: Gray-code walk, residues modulo
 * word-size primes)  ->  pairings_sum_rows  ->  pairings_reconstruct (CRT).
 *
 * Conventions common to all entry points
 *   - return 0 (PAIRINGS_OK) on success, a negative PAIRINGS_E* code on error; never throw, abort or print.
 *   - the caller owns every buffer; "HOST" / "DEVICE" says where a pointer must live.
 *   - thread-safe; no global mutable state.  There is no CPU fallback: without a CUDA device the
 *     compute entry points return PAIRINGS_ECUDA.
 *
 * Index <-> position contract (binding; it makes per-chunk rows and journals portable):
 *   N = 2n positions, x_1 = +1, B = 2n-1 index bits.  Index v in [0, 2^B); bit b of v (b = 0..B-1)
 *   is position N-b; bit = 1 means x = -1.  With C = chunk_bits, chunk c in [0, 2^C) is the set of
 *   all v with (v >> (B-C)) == c, i.e. x_2..x_{C+1} fixed, most significant chunk bit <-> x_2.
 *   Row value = T(c) mod p_i with T(c) = sum_{v in chunk c} term(x(v)) as an exact signed integer
 *   and the mathematical (non-negative) residue in [0, p_i).
 */
#ifndef PAIRINGS_B200_H
#define PAIRINGS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { PAIRINGS_SKOLEM = 0, PAIRINGS_LANGFORD = 1 };

enum {
    PAIRINGS_OK = 0,
    PAIRINGS_EINVAL_KIND = -1,    /* kind is not PAIRINGS_SKOLEM / PAIRINGS_LANGFORD */
    PAIRINGS_EINVAL_N = -2,       /* n outside [2, 32] */
    PAIRINGS_EINVAL_CHUNK = -3,   /* chunk_bits outside [0, 2n-1] or range outside [0, 2^chunk_bits] or begin > end */
    PAIRINGS_EINVAL_MODULUS = -4, /* a modulus is even, outside (2^30, 2^31), duplicated, or n_moduli outside [1, 16] */
    PAIRINGS_ENULL = -5,          /* a required pointer is NULL */
    PAIRINGS_ECUDA = -6,          /* CUDA runtime error (no device, launch failure, allocation failure) */
    PAIRINGS_ECHECK = -7,         /* CRT value disagrees with the redundant check prime */
    PAIRINGS_EINEXACT = -8,       /* H not divisible by 2^{2n-1}, or D odd (reading A16: never truncate) */
    PAIRINGS_ERANGE = -9,         /* product of the CRT moduli too small for the bound, or output buffer too small */
    PAIRINGS_EINVAL_OPTS = -10,   /* launch options not satisfiable for this (kind, n, chunk_bits) */
    PAIRINGS_EJOURNAL = -11,      /* journal file unreadable, or written for other parameters */
    PAIRINGS_ETOOBIG = -12        /* problem does not fit the fixed scratch area of a no-allocation entry point */
};

#define PAIRINGS_MAX_MODULI 16

/* ------------------------------------------------------------------------------------------------
 * count_pairings — §8(a) rows a2..a6: the Gray-code / residue kernel.
 *
 * Enqueues on `stream` the evaluation of chunks [chunk_begin, chunk_end) of the 2^chunk_bits chunks
 * and writes, for each chunk c and modulus i, T(c) mod moduli[i] to
 *      out_residues[(c - chunk_begin) * n_moduli + i]          (row-major, uint32, values in [0, p_i)).
 * This (chunk_end-chunk_begin) x n_moduli matrix is the only HBM traffic of the path.
 *
 *   kind, n        PAIRINGS_SKOLEM / PAIRINGS_LANGFORD, 2 <= n <= 32.  Values of n for which no
 *                  pairing exists are legal and yield rows that sum to zero.
 *   chunk_bits     C, 0 <= C <= 2n-1.
 *   moduli         HOST pointer, n_moduli distinct odd values in (2^30, 2^31), read at call time
 *                  (primality is the caller's responsibility; pairings_default_moduli supplies primes).
 *   out_residues   DEVICE pointer, (chunk_end - chunk_begin) * n_moduli uint32, fully overwritten.
 *   stream         cudaStream_t (NULL = default stream).  The call does not synchronise; invalid
 *                  arguments are reported before anything is enqueued; launch errors map to
 *                  PAIRINGS_ECUDA; asynchronous faults surface at the caller's next synchronise.
 *   An empty range (chunk_begin == chunk_end) is legal and enqueues nothing.
 */
int count_pairings(int kind, int n, int chunk_bits,
                   uint64_t chunk_begin, uint64_t chunk_end,
                   const uint32_t* moduli, int n_moduli,
                   uint32_t* out_residues, void* stream);

/* Launch options for count_pairings_ex.  Zero / NULL in a field means "library default".
 * The result never depends on these (tests check that); they only change the geometry. */
typedef struct pairings_launch_opts {
    int variant;          /* PAIRINGS_VARIANT_* */
    int gray_bits;        /* g: low index bits each thread walks in Gray-code order */
    int block_threads;    /* threads per block (multiple of 32) */
    int blocks_per_chunk; /* power of two; >1 splits one chunk's thread prefixes over several blocks */
    uint64_t* nonzero_terms; /* DEVICE, optional: one uint64 that receives += number of terms with a
                                non-zero product (the early-out statistic, §8(a) row a4) */
} pairings_launch_opts;

enum {
    PAIRINGS_VARIANT_AUTO = 0,
    PAIRINGS_VARIANT_GENERIC = 1, /* any (kind, n): int32 pair-sums, boundary-guarded delta rule, one
                                     Montgomery product chain per modulus and term */
    PAIRINGS_VARIANT_SWAR = 2     /* specialised (kind, n): byte-packed pair-sums, unrolled Gray blocks,
                                     warp-level compaction of non-zero terms, exact multi-word
                                     accumulation reduced modulo the primes once per thread */
};

int count_pairings_ex(int kind, int n, int chunk_bits,
                      uint64_t chunk_begin, uint64_t chunk_end,
                      const uint32_t* moduli, int n_moduli,
                      uint32_t* out_residues, void* stream,
                      const pairings_launch_opts* opts /* HOST, may be NULL */);

/* The launch geometry count_pairings_ex would use for a call over `n_chunks` chunks (chunk_end - chunk_begin) with
 * these options: kernel variant, Gray bits g per thread prefix, threads per block, blocks per chunk.
 * The geometry depends on n_chunks (few chunks are spread over several blocks each), so a test that wants the
 * geometry of a large launch on a small one asks here and pins the answer in `opts`.  Host only, launches
 * nothing.  Any *_out may be NULL.  Errors as count_pairings_ex (PAIRINGS_EINVAL_OPTS: options not satisfiable). */
int pairings_query_geometry(int kind, int n, int chunk_bits, uint64_t n_chunks,
                            const pairings_launch_opts* opts /* HOST, may be NULL */,
                            int* variant_out, int* gray_bits_out, int* block_threads_out, int* blocks_per_chunk_out);

/* 1 if PAIRINGS_VARIANT_SWAR is compiled for (kind, n), else 0. */
int pairings_has_swar(int kind, int n);

/* Same computation with a HOST output buffer: allocates the device rows on `stream` from a memory pool of the
 * library's own (one per device, created on first use, keeps at most 64 MiB between calls — the only device
 * memory the library ever retains), launches, copies the rows back and synchronises the stream.  This is the
 * end-to-end call bench.py times as "e2e".  out_residues_host: (chunk_end-chunk_begin)*n_moduli. */
int count_pairings_host(int kind, int n, int chunk_bits,
                        uint64_t chunk_begin, uint64_t chunk_end,
                        const uint32_t* moduli, int n_moduli,
                        uint32_t* out_residues_host, void* stream,
                        const pairings_launch_opts* opts /* HOST, may be NULL */);

/* ------------------------------------------------------------------------------------------------
 * Host side: moduli, partitioner, journal, row sums, CRT.
 */

/* The `count` largest primes below 2^31 in descending order (reading A7 of PAPER.md:257 "modulo
 * number of co-primes"): 2147483647, 2147483629, 2147483587, ...  out: HOST, count <= 16. */
int pairings_default_moduli(uint32_t* out, int count);

/* Smallest m such that the product of the first m default moduli exceeds 2 * 2^{2n-1} * prod_k (2n-d_k)
 * >= 2|H| (each |P_k| <= 2n-d_k).  Negative code on invalid (kind, n). */
int pairings_min_moduli(int kind, int n);

/* Number of CRT moduli the north_star bound (2n)^n * 2^{2n} asks for (>= pairings_min_moduli). */
int pairings_bound_moduli(int kind, int n);

/* §8(a) row a1 — host prefix partitioner ("split {1,-1}^{2n} sequences into several
 * independent sets and simply put the result together at the end"; splits are by fixed bits, so
 * every piece is a power-of-two sub-cube).  Cuts [0, 2^chunk_bits) minus the union of the `n_done`
 * half-open ranges done[2j], done[2j+1] into ranges of at most max_chunks chunks, in ascending order.
 * Writes up to cap_ranges pairs to out_ranges (HOST) and returns the number of pairs needed
 * (which may exceed cap_ranges), or a negative code. */
int64_t pairings_partition(int chunk_bits, uint64_t max_chunks,
                           const uint64_t* done, int n_done,
                           uint64_t* out_ranges, int64_t cap_ranges);

/* The slice of [0, 2^chunk_bits) owned by `rank` of `world` when chunks are dealt out as
 * contiguous, equal (+-1) ranges — replicas on disjoint ranges are the only multi-GPU mode (§8(e)). */
int pairings_rank_range(int chunk_bits, int rank, int world, uint64_t* out_begin, uint64_t* out_end);

/* Adds n_rows rows (HOST, row-major n_rows x n_moduli, values < p_i) into total[i] modulo moduli[i].
 * total (HOST, n_moduli values < p_i) is read and updated. */
int pairings_sum_rows(const uint32_t* rows, uint64_t n_rows,
                      const uint32_t* moduli, int n_moduli, uint32_t* total);

/* Resumable journal: an append-only text file.  Header line fixes (kind, n, chunk_bits, moduli);
 * every further line is "begin end r_0 .. r_{m-1}" = the summed rows of chunks [begin, end).
 * pairings_journal_append creates the file (with header) if absent and refuses (PAIRINGS_EJOURNAL)
 * a file written for other parameters.  pairings_journal_load returns the number of recorded
 * ranges (writing up to cap_ranges (begin,end) pairs) and the sum of their rows in total_out;
 * a missing file is 0 ranges.  A truncated last line (a crash mid-write: bytes behind the last newline) is ignored
 * by load and cut off by the next append; a line with missing, non-numeric or surplus tokens, a range outside
 * [0, 2^chunk_bits) or two overlapping ranges make the file PAIRINGS_EJOURNAL.  Every append is fsync-ed. */
int pairings_journal_append(const char* path, int kind, int n, int chunk_bits,
                            const uint32_t* moduli, int n_moduli,
                            uint64_t chunk_begin, uint64_t chunk_end, const uint32_t* row_sum);
int64_t pairings_journal_load(const char* path, int kind, int n, int chunk_bits,
                              const uint32_t* moduli, int n_moduli,
                              uint64_t* out_ranges, int64_t cap_ranges, uint32_t* total_out);

/* Puts the journals of several jobs together ("split ... into several independent sets and simply put
 * the result together at the end"; 4 / 64 / 256 / 1024 GPU jobs): every file of paths[0..n_paths) must
 * exist and carry the header of (kind, n, chunk_bits, moduli); their ranges must not overlap each other (a chunk
 * counted twice: PAIRINGS_EJOURNAL).  total_out (HOST, n_moduli) = sum of all rows; *chunks_covered_out (may be NULL) =
 * number of chunks they cover (the job is complete when it equals the number of chunks evaluated in that mode);
 * out_path (may be NULL) receives one merged journal, ranges ascending, written and fsync-ed.  Returns the number of
 * ranges or a negative code.  Host only. */
int64_t pairings_journal_merge(const char* const* paths, int n_paths, const char* out_path,
                               int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli,
                               uint32_t* total_out, uint64_t* chunks_covered_out);

/* The mode of a job, in one place (host only).  `flags` are the PAIRINGS_RUN_* bits of pairings_run_ex (declared
 * below; only PAIRINGS_RUN_LEMMA24 changes anything here).
 *
 * pairings_mode_chunks: *needed_out = the number of chunks a whole job evaluates in this mode, always the range
 * [0, needed): 2^chunk_bits without the symmetry; with PAIRINGS_RUN_LEMMA24 and chunk_bits >= 1 the x_2 = +1 half
 * [0, 2^(chunk_bits-1)) when the two halves are equal, 0 when they cancel (Lemma 2.4; the most
 * significant chunk bit is x_2).  Returns the factor that turns the sum over those chunks into H: 1, 2 or 0 (H = 0),
 * or a negative code.
 *
 * pairings_finish_total: the last step of a job whose rows were added up elsewhere (a slice run alone, merged
 * journals).  If chunks_covered equals the mode's chunk count, total_inout (HOST, n_moduli residues of the raw row
 * sum) is multiplied by that factor — the ONLY place outside pairings_run_ex where Lemma 2.4's doubling is applied —
 * and 1 is returned: total_inout is H mod p_i, ready for pairings_reconstruct.  Fewer chunks: returns 0, total
 * untouched.  More: PAIRINGS_EINVAL_CHUNK.
 *
 * pairings_journal_merge_mode: pairings_journal_merge for a given mode — additionally refuses (PAIRINGS_EJOURNAL) any
 * range that reaches outside [0, needed), so that journals of jobs run without the symmetry, or a mix of ranges from
 * both halves that merely adds up to the right length, cannot be doubled into a wrong count; *chunks_needed_out (may
 * be NULL) = needed.  The sum is NOT finished: pass it with *chunks_covered_out to pairings_finish_total. */
int pairings_mode_chunks(int kind, int n, int chunk_bits, unsigned flags, uint64_t* needed_out);
int pairings_finish_total(int kind, int n, int chunk_bits, unsigned flags, uint64_t chunks_covered,
                          const uint32_t* moduli, int n_moduli, uint32_t* total_inout);
int64_t pairings_journal_merge_mode(const char* const* paths, int n_paths, const char* out_path,
                                    int kind, int n, int chunk_bits, const uint32_t* moduli, int n_moduli, unsigned flags,
                                    uint32_t* total_out, uint64_t* chunks_covered_out, uint64_t* chunks_needed_out);

/* The duplicate-run protocol against silent GPU errors ("every GPU job was ran twice on separate GPUs.
 * The two results were then matched, if there was a mismatch the job was ran a third time to establish a match").
 * pairings_vote_rows compares n_words words (HOST): returns 0 if a == b, or if c (the third run, may be NULL) equals
 * a; 1 if c equals b (b stands); 3 if a != b and c is NULL (a third run is needed); PAIRINGS_ECHECK if no two of the
 * three agree.  pairings_duplicate_vote drives it: eval(ctx, attempt, rows) must fill n_words words for attempt 0 and
 * 1, and 2 only after a mismatch (attempts should differ in how they compute: other GPU, other launch geometry,
 * other kernel); rows_out receives the rows two runs agreed on, *mismatch_out (may be NULL) 1 if the first two
 * differed.  A non-zero return of eval is passed through.  Host only; pairings_run_ex uses it. */
typedef int (*pairings_eval_fn)(void* ctx, int attempt, uint32_t* rows_out);
int pairings_vote_rows(const uint32_t* a, const uint32_t* b, const uint32_t* c, uint64_t n_words);
int pairings_duplicate_vote(pairings_eval_fn eval, void* ctx, uint64_t n_words, uint32_t* rows_out, int* mismatch_out);

/* Whole-job host driver: partition -> count_pairings_host per range -> sum rows -> journal.
 * Skips ranges already in the journal (journal_path may be NULL = no journal).  Stops after
 * max_calls kernel calls if max_calls > 0 (so a run can be interrupted and resumed).
 * total_out (HOST, n_moduli) = summed residues of every chunk done so far (journal included);
 * *chunks_done_out = how many of the 2^chunk_bits chunks that covers. */
int pairings_run(int kind, int n, int chunk_bits,
                 const uint32_t* moduli, int n_moduli,
                 uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                 void* stream, const pairings_launch_opts* opts,
                 uint32_t* total_out, uint64_t* chunks_done_out);

/* §8(f) NEXT #1 — symmetry 3 (Lemma 2.4; the paper fixes a second variable with it,
 * PAPER.md:253).  With x^ = (x_1, -x_2, x_3, -x_4, ...):  term(x^) = (-1)^{n + sum_k d_k} term(x).
 * Returns 1 if the exponent is even (term(x^) = term(x): Skolem n = 0,1 mod 4, Langford n = 0,3 mod 4 —
 * exactly the n for which pairings exist), so the x_2 = +1 half of the sum is H/2;
 * 0 if it is odd (term(x^) = -term(x): the two halves cancel and H = 0); negative code on invalid (kind, n). */
int pairings_lemma24(int kind, int n);

/* pairings_run with flags.  PAIRINGS_RUN_LEMMA24: use symmetry 3 — x_2 is the most significant chunk
 * bit, so only chunks [0, 2^{chunk_bits-1}) are evaluated (none at all when pairings_lemma24 is 0) and
 * the sum is doubled at the end; needs chunk_bits >= 1, otherwise the flag is ignored.
 *   *chunks_needed_out (may be NULL) = number of chunks this mode evaluates in total.
 *   When *chunks_done_out == *chunks_needed_out, total_out holds H mod p_i (symmetry factor applied);
 *   before that it is the raw partial sum.  A journal that already holds chunks of the x_2 = -1 half
 *   (written by a run without the flag) is refused with PAIRINGS_EJOURNAL.
 *
 * PAIRINGS_RUN_DUPLICATE: the paper's protection against silent GPU errors (every job is run
 * twice, a third time on disagreement; §8(f) NEXT #3).  Every chunk range is evaluated twice — the second
 * time with another launch geometry (another Gray-bit count: another thread <-> term mapping and summation
 * order) — and the rows are compared word by word; on a mismatch a third run decides, and if no two runs
 * agree the call fails with PAIRINGS_ECHECK.  *duplicate_mismatches_out (may be NULL) counts the ranges
 * whose first two runs disagreed.  Costs twice the time.
 *
 * PAIRINGS_RUN_AUDIT: a cheap second opinion from an independent implementation — of every chunk range, the first
 * chunk and one seeded chunk are evaluated again by PAIRINGS_VARIANT_GENERIC (other kernel, other arithmetic: per-term
 * Montgomery residues instead of exact multi-word sums) and compared word by word; on a mismatch the auditor itself
 * runs that chunk once more at another Gray-bit count and decides: if this second generic run sides with the fast
 * row, the auditor's first run was a transient fault and the range stands (the mismatch is counted); if the generic
 * kernel reproduces its own row — so the fast kernel is wrong, however often it reproduces itself — or no two rows
 * agree, the call fails with PAIRINGS_ECHECK.  The audited kernel never votes on itself.  Costs a few per cent. */
enum { PAIRINGS_RUN_LEMMA24 = 1, PAIRINGS_RUN_DUPLICATE = 2, PAIRINGS_RUN_AUDIT = 4 };
int pairings_run_ex(int kind, int n, int chunk_bits,
                    const uint32_t* moduli, int n_moduli,
                    uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                    void* stream, const pairings_launch_opts* opts, unsigned flags,
                    uint32_t* total_out, uint64_t* chunks_done_out, uint64_t* chunks_needed_out,
                    uint64_t* duplicate_mismatches_out);

/* One job of a chunk farm ("split ... into several independent sets and simply put the result together
 * at the end"; S(25) as 4 GPU jobs, L(27) 64, n = 28 256, S(29) 1024): pairings_run_ex restricted to the
 * chunks of [slice_begin, slice_end) (within [0, 2^chunk_bits); with PAIRINGS_RUN_LEMMA24 only the part below
 * 2^{chunk_bits-1} is evaluated).  total_out = the summed rows of the slice (never doubled: the symmetry factor belongs
 * to the whole job and is applied by whoever adds the slices up), *chunks_needed_out = chunks of the slice this mode
 * evaluates.  A journal holding ranges outside the slice is refused (PAIRINGS_EJOURNAL).  The slices of the ranks come
 * from pairings_rank_range, their journals are put together by pairings_journal_merge. */
int pairings_run_slice(int kind, int n, int chunk_bits,
                       const uint32_t* moduli, int n_moduli,
                       uint64_t chunks_per_call, const char* journal_path, int64_t max_calls,
                       void* stream, const pairings_launch_opts* opts, unsigned flags,
                       uint64_t slice_begin, uint64_t slice_end,
                       uint32_t* total_out, uint64_t* chunks_done_out, uint64_t* chunks_needed_out,
                       uint64_t* duplicate_mismatches_out);

/* §8(a) row a7 — CRT reconstruction ("the actual value is obtained using the chinese
 * remainder theorem") and the exact division of Lemma 2.1.
 *   moduli[0..n_moduli-2] are the CRT primes, moduli[n_moduli-1] is the redundant check prime
 *   (n_moduli >= 2).  total_residues: HOST, H mod p_i summed over all 2^chunk_bits chunks.
 *   Garner CRT -> H in [0, prod p); H mod check prime must match (else PAIRINGS_ECHECK);
 *   2^{2n-1} must divide H and D = H / 2^{2n-1} must be even (else PAIRINGS_EINEXACT);
 *   the CRT product must exceed 2 * 2^{2n-1} * prod_k (2n-d_k) (else PAIRINGS_ERANGE).
 *   out_distinct_dec    D(n), reflections distinct, decimal, NUL-terminated
 *   out_identified_dec  D(n)/2, reflections identified (the paper's S(n) / L(n))
 *   cap                 size of each output buffer (PAIRINGS_ERANGE if too small) */
int pairings_reconstruct(int kind, int n,
                         const uint32_t* moduli, int n_moduli,
                         const uint32_t* total_residues,
                         char* out_distinct_dec, char* out_identified_dec, size_t cap);

/* Symmetric CRT lift of one row (no check prime, no division): the signed T(c) in (-M/2, M/2]
 * as a decimal string (reading A8).  For parity tests of single chunks. */
int pairings_crt_signed(const uint32_t* moduli, int n_moduli, const uint32_t* residues,
                        char* out_dec, size_t cap);

/* ------------------------------------------------------------------------------------------------
 * Approximate counting by parallel tempering — PAPER.md §3 (:259-325), Algorithm 2 (:291-319);
 * SURVEY.md §8(f) NEXT #4.  A second, statistical workload beside the exact count.
 *
 * The system: colour k occupies bins a_k and a_k + d_k, a_k in [1, 2n - d_k]; the energy of
 * a configuration is its number of empty bins; Z(0) = prod_k (2n - d_k) = (2n-1)!/(n-1)! for Skolem, and the
 * E = 0 configurations are the pairings (reflections distinct).  Levels: betas[0] = 0 < betas[1] < ... (HOST,
 * n_levels <= PAIRINGS_PT_MAX_LEVELS), the level above the last one is beta = infinity (reading C1).
 *
 * pairings_pt_run enqueues replicas [replica_begin, replica_end) of Algorithm 2, `iterations` iterations each
 * of which the first `burn_in` (< iterations) are run but not counted (0 = as printed; reading C4: many short
 * replicas need it, a replica started from a random configuration is biased by O(relaxation time / iterations)),
 * one thread per replica, and ADDS to the DEVICE counters (the caller zeroes them):
 *     hist_dev   n_levels x (2n+1) uint64: hist[j][E] = samples of level j with E empty bins
 *     moves_dev  n_levels uint64: accepted moves of level j         (column W1 of Table 6)
 *     swaps_dev  n_levels uint64: accepted exchanges j <-> j+1      (column W2)
 * Random numbers: draw(seed, ctr) = splitmix64_mix(seed + 0x9E3779B97F4A7C15 (ctr + 1)), counter layout and
 * the integer decision rule "u < floor(p 2^32)" as in DESIGN.md (readings C2, C3): the counters depend only on
 * (kind, n, betas, replica range, iterations, seed) — not on the launch — and add up over disjoint replica
 * ranges, which is how the work is sharded over calls or GPUs.  iterations <= 2^25, replica_end <= 2^30, and
 * replica_end * (iterations + 1) * n_levels * max(n, 3) < 2^64 (the draw counter must not wrap: PAIRINGS_EINVAL_OPTS).
 * Invalid arguments are reported before anything is enqueued; the call synchronises the stream once (the
 * threshold table is staged from host memory) and then returns with the kernel enqueued. */
#define PAIRINGS_PT_MAX_LEVELS 32
int pairings_pt_run(int kind, int n, const double* betas, int n_levels,
                    uint64_t replica_begin, uint64_t replica_end, uint64_t iterations, uint64_t burn_in, uint64_t seed,
                    uint64_t* hist_dev, uint64_t* moves_dev, uint64_t* swaps_dev, void* stream);

/* pairings_pt_run for callers that must not allocate device memory.
 *
 * Who needs this: pairings_pt_run takes its acceptance-threshold table (scratch the kernel reads, neither an input
 * nor an output of the caller) from cudaMallocAsync and gives it back with cudaFreeAsync on every call.  Some
 * programs cannot afford that.  A service that hands all of HBM to its own arena at start-up has nothing left for the
 * driver to give out, so the allocation fails.  A loop with a latency budget cannot take an allocator call whose cost
 * varies from microseconds to a device-wide synchronisation.  And code that runs where the CUDA allocator is simply
 * off limits (a plug-in inside a host application that owns the memory budget) may only launch work.  This entry
 * point runs the same kernel on the same arguments and produces the same counters, but its threshold table lives in
 * a fixed array compiled into the library (`static __device__`, PAIRINGS_PT_STATIC_WORDS 64-bit words = 16 KiB).
 * It calls neither cudaMalloc* nor cudaFree*, nor any library routine that allocates.  The price is 16 KiB of device
 * memory on every GPU that loads the library, held until the process exits, whether or not this is ever called.
 *
 * Limit: the table holds n_levels * (2n + 3) words, and that must not exceed PAIRINGS_PT_STATIC_WORDS (2048); a
 * larger request is refused with PAIRINGS_ETOOBIG before anything is enqueued (of the sizes pairings_pt_run takes,
 * only n >= 31 with 31 or 32 levels are that large).  Everything else — arguments, counters that are ADDED to the
 * caller's zeroed DEVICE arrays, the random streams, the other error codes, the one stream synchronisation while the
 * table is staged from the host — is as documented for pairings_pt_run.
 *
 * Set-up: the first call on each device looks up the device address of the array (cudaGetSymbolAddress, with that
 * device current) and remembers it per device; later calls on that device reuse it.  Make that first call before
 * any stream capture begins, with the device you mean to use current.
 *
 * Sharing: there is ONE array per device and every call overwrites it.  Each call rewrites every word its kernel
 * may read (including the never-accepted zero entries), so nothing left behind by an earlier call — a longer
 * ladder, a larger n — can leak into a later one.  Calls enqueued on the same stream are ordered by the stream
 * and are safe.  Two calls whose GPU work can overlap (different streams, or different host threads on different
 * streams) race on the table: the first kernel may read the second call's thresholds.  Serialise them, or use
 * pairings_pt_run for one of them. */
#define PAIRINGS_PT_STATIC_WORDS 2048
int pairings_pt_run_noalloc(int kind, int n, const double* betas, int n_levels,
                            uint64_t replica_begin, uint64_t replica_end, uint64_t iterations, uint64_t burn_in, uint64_t seed,
                            uint64_t* hist_dev, uint64_t* moves_dev, uint64_t* swaps_dev, void* stream);

/* Ladder choice (exchange acceptance "no smaller than one half", as few levels as that allows).
 * Builds betas_out[0] = 0 < betas_out[1] < ... level by level: a pilot run (pilot_replicas x pilot_iterations, half
 * of them burn-in) of the ladder so far gives the energy distribution of its last level, and the next beta is the
 * one whose predicted exchange acceptance with it (by reweighting) equals target_exchange (at most a doubling of
 * beta per level); stops when the last level is at E = 0 with probability >= 0.98 or beta >= 32.  Deterministic in (kind, n, target, pilot sizes, seed).  Synchronises
 * the stream.  Returns the number of levels (<= cap_levels, <= PAIRINGS_PT_MAX_LEVELS) or a negative code
 * (PAIRINGS_ERANGE: cap reached first).  betas_out: HOST, cap_levels doubles. */
int pairings_pt_ladder(int kind, int n, double target_exchange, uint64_t pilot_replicas, uint64_t pilot_iterations,
                       uint64_t seed, double* betas_out, int cap_levels, void* stream);

/* Host: Ratio(j)/iterations of Algorithm 2 from the histogram (HOST, n_levels x (2n+1)),
 *     ratios_out[j] = sum_E hist[j][E] exp(-(beta(j+1) - beta(j)) E) / sum_E hist[j][E]     (last level: [E = 0]),
 * and *log_distinct_out = log( Z(0) prod_j ratios[j] ), the natural logarithm of the estimated number of
 * pairings with reflections distinct (halve for the paper's S(n) / L(n), Table 6 caption).
 * PAIRINGS_ERANGE if a level has no samples or a ratio is estimated as zero. */
int pairings_pt_estimate(int kind, int n, const double* betas, int n_levels, const uint64_t* hist_host,
                         double* ratios_out, double* log_distinct_out);

/* Host: the two counting conventions from the estimate's logarithm (reflections distinct vs identified —
 * "the two different ways to count differ by exactly a factor of two" for n > 1; Table 6's caption and Tables 7/8 print
 * the identified count).  *distinct_out = exp(log_distinct), *identified_out = half of it (n > 1). */
int pairings_pt_counts(int n, double log_distinct, double* distinct_out, double* identified_out);

const char* pairings_strerror(int code);

/* Library build string: version, CUDA arch, compiled SWAR specialisations. */
const char* pairings_build_info(void);

#ifdef __cplusplus
}
#endif
#endif /* PAIRINGS_B200_H */
