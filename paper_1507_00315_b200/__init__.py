"""pairings-b200: exact counting of Skolem / Langford pairings by Godfrey's algebraic sum
(arxiv 1507.00315 §2) on one B200.  Thin ctypes binding over libpairings_b200.so (include/pairings.h);
every step of the path runs in the library's CUDA kernels / C++ host code.  There is no CPU
fallback: importing works without a GPU, compute calls raise PairingsError(PAIRINGS_ECUDA).
"""
from .api import (  # noqa: F401
    SKOLEM, LANGFORD, VARIANT_AUTO, VARIANT_GENERIC, VARIANT_SWAR,
    PairingsError, LaunchOpts, lib, library_path,
    count_pairings, count_pairings_ex, count_pairings_host, pairings_has_swar, pairings_query_geometry,
    pairings_default_moduli, pairings_min_moduli, pairings_bound_moduli,
    pairings_partition, pairings_rank_range, pairings_sum_rows,
    pairings_journal_append, pairings_journal_load, pairings_run, pairings_run_ex, pairings_run_slice, pairings_lemma24,
    RUN_LEMMA24, RUN_DUPLICATE, RUN_AUDIT, pairings_journal_merge, pairings_journal_merge_mode,
    pairings_mode_chunks, pairings_finish_total, pairings_vote_rows, pairings_duplicate_vote,
    default_chunk_bits, default_chunks_per_call,
    pairings_reconstruct, pairings_crt_signed, pairings_strerror, pairings_build_info,
    pairings_pt_run, pairings_pt_run_noalloc, pairings_pt_estimate, pairings_pt_counts, pairings_pt_ladder,
    count, approx_count,
)
