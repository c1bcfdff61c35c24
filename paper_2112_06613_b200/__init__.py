"""B200-native TCR-NET hot path (arXiv 2112.06613): all-pairs Levenshtein distance over CDR3-beta
sequences thresholded at l_max into CSR + degrees, as hand-written sm_100a CUDA behind the C ABI
of include/tcrnet.h.  This package is the thin Python binding; nothing here computes.
"""
from .binding import (ERR_ARG, ERR_CAPACITY, ERR_CUDA, ERR_EDGE_OVERFLOW, ERR_LENGTH, ERR_LMAX, ERR_NOMEM, ERR_RESIDUE,
                      ERR_STATE, EXPORTS, LIB_PATH, OK, OPT_COUNT_WORK, OPT_DEDUP, OPT_EARLY_EXIT, OPT_EDGE_CAPACITY,
                      OPT_EDGE_LIMIT, OPT_FAST_L1, OPT_TIMING, OPT_FIRST_CHECK, OPT_N_QUERY, OPT_PREFIX_TRIE, OPT_SEGMENT_JOIN, OPT_TEXT_CHUNK, OPT_TRIE_CHUNK, TcrNet, TcrNetError, build_network,
                      load_library, strerror, version, NOALLOC_MAX_ROWS, row_ptr_noalloc)

__all__ = [
    "TcrNet", "TcrNetError", "build_network", "load_library", "strerror", "version", "LIB_PATH", "EXPORTS",
    "OK", "ERR_ARG", "ERR_LENGTH", "ERR_RESIDUE", "ERR_LMAX", "ERR_STATE", "ERR_NOMEM", "ERR_EDGE_OVERFLOW",
    "ERR_CUDA", "ERR_CAPACITY", "NOALLOC_MAX_ROWS", "row_ptr_noalloc", "OPT_EARLY_EXIT", "OPT_FIRST_CHECK", "OPT_EDGE_CAPACITY", "OPT_EDGE_LIMIT", "OPT_COUNT_WORK",
    "OPT_TEXT_CHUNK", "OPT_PREFIX_TRIE", "OPT_TRIE_CHUNK", "OPT_N_QUERY", "OPT_DEDUP", "OPT_SEGMENT_JOIN", "OPT_FAST_L1", "OPT_TIMING",
]
