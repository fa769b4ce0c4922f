"""paper_1401_7457_b200 -- B200-native hot path of CX1 (arxiv 1401.7457): GPU suffix sorting of a
short-read collection and BWT emission, as hand-written sm_100a CUDA behind the C ABI of
include/cx_bwt.h.  This package is the thin Python binding (argument marshalling only)."""
from .binding import (CxError, Plan, bwt_of_collection, cx_bwt_workspace_bytes, cx_fasta_parse, bwt_of_fasta, cx_pack_reads, cx_sort_pairs, cx_sort_pairs_static, CX_SORT_STATIC_MAX_PAIRS, pack_reads_from_host, HostPipeline,  # noqa: F401
                      cx_strerror, lib, KERNEL_CLASSES)
from .shard import build_sharded, check_pieces, exchange_pieces  # noqa: F401,E402
