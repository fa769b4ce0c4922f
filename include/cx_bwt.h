/*
 * cx_bwt.h -- C ABI of the B200-native hot path of CX1 (arxiv 1401.7457, Liu, Luo, Lam):
 * "Input: a string collection R.  Parameters: l, m1, m2.  Output: the BWT of R"
 * (Figure 2).
 *
 * Everything behind these calls is hand-written sm_100a CUDA (libcxbwt.so).  There is no CPU
 * fallback: with no CUDA device every compute call returns CX_ERR_CUDA.
 *
 * Conventions (Section 2; pinned by Figure 1):
 *   alphabet  $ < A < C < G < T;  every read S_i is followed by its own end-marker $_i with
 *   $_i < $_j iff i < j;  the symbol preceding a suffix that starts at position 0 is '$'.
 *
 * Pointers are plain addresses; each argument says whether it is HOST or DEVICE memory.  The caller
 * owns every buffer, including the workspace; the library never allocates device memory on the
 * build path and keeps no reference to inputs after the work it enqueued has completed.
 * All functions return 0 (CX_OK) on success and a negative CX_ERR_* code otherwise; nothing aborts
 * or throws across this boundary.
 */
#ifndef CX_BWT_H
#define CX_BWT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* a cudaStream_t, spelled without pulling in cuda_runtime.h (NULL = the default stream) */
typedef struct CUstream_st *cx_stream_t;

typedef struct cx_bwt_plan_s cx_bwt_plan_t; /* opaque */

enum {
    CX_OK = 0,
    CX_ERR_ARG = -1,              /* null pointer, sizes above the plan's maxima, bad option, offsets not
                                     starting at 0 or decreasing */
    CX_ERR_BAD_BASE = -2,         /* cx_pack_reads saw a byte outside "ACGT" (reads are ACGT only) */
    CX_ERR_WORKSPACE = -3,        /* workspace too small for even one bucket-sized batch */
    CX_ERR_BUCKET_TOO_LARGE = -4, /* a partition still exceeds m1 after refining it by its next l characters down to
                                     2^20 bases (Fig. 2 step 1); not reachable with sane inputs */
    CX_ERR_CUDA = -5,             /* CUDA runtime error (or no device); text via cx_strerror */
    CX_ERR_NOMEM = -6             /* host allocation failed */
};

/* Parameters of Figure 2 plus the knobs of this implementation.  Zero = default. */
typedef struct cx_bwt_opts_s {
    uint32_t prefix_len;         /* l: partition prefix length in bases, 1..7; default 6        */
    uint32_t key_bases;          /* w: bases in the first-round sort key, l..29 ("stringword").  The key is
                                    the rank of the window's symbols among all strings of at most w bases plus one
                                    bit, about 2 w + 1.5 bits: w <= 15 packs into a 32-bit key (4 radix passes), larger
                                    w into a 64-bit key.  0 = 15 up to 2^30 suffixes in the collection, else what the
                                    radix passes that ceil(log4 N) bases need can carry (19 bases, 5 passes, at
                                    6e9 .. 1e11 suffixes)                                                       */
    uint64_t max_batch_suffixes; /* m1: most suffixes sorted in one GPU batch;
                                    0 = as many as the workspace allows                                       */
    uint32_t max_read_len;       /* longest read the plan must accept; 0 = unknown (forces 64-bit suffix ids
                                    unless n_reads and total_bases are tiny)                                  */
    int32_t  out_is_host_pinned; /* 1: out_bwt of cx_bwt_build is pinned HOST memory; batches are staged in
                                    the workspace and copied with cudaMemcpyAsync on a side stream           */
    uint32_t small_group_max;    /* tie refinement: groups up to this many suffixes are finished inside one
                                    thread block; 0 = default (256); 1 = use only the global re-key + sort   */
    uint32_t profile;            /* 1: bracket every kernel with CUDA events (see cx_bwt_kernel_time)         */
    uint32_t finish_slots;       /* tie refinement in registers: positions per warp window / 32.  0 = chosen per batch from a
                                    sample of its tie-group sizes; 2 = windows of 64 (groups up to 64, two-level keys);
                                    4 = windows of 128 (groups up to 128)                                       */
    uint32_t out_bits;           /* 0 or 8: out_bwt holds one ASCII byte per suffix.  4: NEXT-4, packed output,
                                    two symbols per byte, first symbol in the high nibble, codes $ A C G T = 0 1 2 3 4;
                                    out_bwt then has ceil(N / 2) bytes (the low nibble of the last byte is 0 if N is odd).
                                    Halves the device->host stream of an out-of-core build.  Not with shard_count > 1  */
    uint32_t shard_index;        /* with shard_count > 1: which contiguous range of partitions this plan sorts     */
    uint32_t shard_count;        /* 0 or 1: the whole collection.  W > 1: the paper's distributed scheme (PAPER.md:103,
                                    Section 3.3): every worker holds all reads and computes the same partition sizes;
                                    partition b belongs to worker floor(first_output_position(b) * W / N), so each
                                    worker gets consecutive partitions of about N / W suffixes, sorts only those, and
                                    writes them at their final positions of out_bwt; the pieces are disjoint and
                                    "can be simply concatenated".  W <= 65536                    */
} cx_bwt_opts_t;

/* What the last cx_bwt_build on a plan did (HOST struct, filled by cx_bwt_get_stats). */
typedef struct cx_bwt_stats_s {
    uint64_t n_suffixes;        /* N = total_bases + n_reads (n(m+1))                       */
    uint64_t max_batch;         /* m1 actually used                                                     */
    uint64_t largest_bucket;    /* largest l-prefix partition                                           */
    uint64_t refine_elements;   /* suffixes re-keyed, summed over refinement rounds and batches          */
    uint64_t small_group_elems; /* of those, finished by the in-block path                               */
    uint64_t kernel_launches;   /* kernels launched by the build                                        */
    uint64_t compare_ops;       /* rank-key comparisons of the in-block refinement (diagnostic)          */
    uint32_t n_batches;         /* GPU batches (the paper's "small rounds", Fig. 2 step 3(c))            */
    uint32_t id_bytes;          /* 4 or 8: width of a suffix id                                         */
    uint32_t sort_passes;       /* radix passes of the first sort of a batch                            */
    uint32_t refine_rounds;     /* global refinement rounds, max over batches                           */
    uint32_t max_read_len;      /* longest read seen                                                    */
    uint32_t uniform_len;       /* 1 if every read has the same length (the paper's setting)*/
    uint32_t refined_partitions;/* l-prefix partitions larger than m1 that were partitioned again */
    uint64_t shard_offset;      /* first position of out_bwt this build wrote (0 unless shard_count > 1)  */
    uint64_t shard_suffixes;    /* positions written from there: the shard's piece of the BWT (N if unsharded) */
    uint64_t finish_rounds;     /* refinement rounds of the in-block path, summed over its thread blocks (diagnostic) */
} cx_bwt_stats_t;

/* Kernel classes for cx_bwt_kernel_time; one per row of the hot path. */
enum {
    CX_K_PACK = 0,        /* a1 2-bit pack                                   */
    CX_K_PREP,            /* offsets check, max length, tile -> read table    */
    CX_K_HIST,            /* a2 bucket histogram                              */
    CX_K_LIST,            /* a4+a5 stable id listing fused with key build     */
    CX_K_SORT_HIST,       /* a6 upfront digit histograms                      */
    CX_K_SORT_SCAN,       /* a6 bin offsets                                   */
    CX_K_SORT_PASS,       /* a6 onesweep radix pass                           */
    CX_K_FINISH,          /* a7+a8 warp kernel: head flags, tie groups of <= 32 refined in registers, emit */
    CX_K_REFINE_SCAN,     /* a7 compaction scans of the global path           */
    CX_K_REFINE_KEY,      /* a7 re-key gather of the global path              */
    CX_K_REFINE_WRITE,    /* a7+a8 write-back, new flags, emit (global path)  */
    CX_K_REFINE_SORT,     /* a7 onesweep passes over the compacted members of oversize groups (global path) */
    CX_K_FINISH_BLOCK,    /* a7+a8 block kernel: tie groups of 33..256 suffixes refined in shared memory */
    CX_K_COUNT
};

/*
 * Bytes of DEVICE workspace cx_bwt_plan needs to sort a collection of up to n_reads reads and
 * total_bases bases in ONE batch (opts->max_batch_suffixes = 0) or in batches of at most
 * opts->max_batch_suffixes.  A smaller workspace is legal: the plan then lowers m1 (PAPER.md:97:
 * m1 "only depends on the GPU memory limit").  opts may be NULL.  bytes_out: HOST.
 */
int cx_bwt_workspace_bytes(uint64_t n_reads, uint64_t total_bases, const cx_bwt_opts_t *opts,
                           uint64_t *bytes_out);

/*
 * Create a plan.  workspace_dev: DEVICE, workspace_bytes long, 256-byte aligned, owned by the
 * caller and left untouched by others until cx_bwt_free.  The plan carves it into the partition-size
 * array, key/id double buffers, radix tile state, flags and (if asked) output staging, and derives
 * m1.  Small one-off initialisation runs on the default stream and is synchronised before return.
 * Errors: CX_ERR_ARG, CX_ERR_WORKSPACE, CX_ERR_CUDA, CX_ERR_NOMEM.
 */
int cx_bwt_plan(cx_bwt_plan_t **plan_out, uint64_t max_reads, uint64_t max_total_bases,
                const cx_bwt_opts_t *opts, void *workspace_dev, uint64_t workspace_bytes);

/*
 * Step a1: "standard 2-bit-per-character representation".  A,C,G,T -> 0,1,2,3;
 * base j of the concatenated reads lands in word j/32, bits 63-2(j%32) and 62-2(j%32) (first base in
 * the most significant bits).  ascii_dev: DEVICE, total_bases bytes.  packed_out_dev: DEVICE,
 * ceil(total_bases/32) words; the unused low bits of the last word are zero.
 * status_dev: DEVICE uint32, receives the number of bytes outside "ACGT" (0 = clean); the call is
 * then fully asynchronous and returns CX_OK.  If status_dev is NULL the call synchronises `stream`
 * and returns CX_ERR_BAD_BASE itself.
 */
int cx_pack_reads(const uint8_t *ascii_dev, uint64_t total_bases, uint64_t *packed_out_dev,
                  uint32_t *status_dev, cx_stream_t stream);

/*
 * NEXT-4, ingest: FASTA text -> the inputs of cx_pack_reads / cx_bwt_build, on the device.  "The input was in FASTA
 * format"; loading is "more than 16 minutes" of the paper's 6,886 s.  Grammar taken (the
 * paper gives none): lines end with '\n' (the last may lack it); a line whose first byte is '>' is a header and starts
 * a new read; every other line is a sequence line whose bytes, except '\r', are appended to the current read (a read
 * may span several lines, or none: length 0).  Bytes are copied as they are: cx_pack_reads rejects what is not ACGT.
 *   text_dev       : DEVICE, n_bytes of FASTA text
 *   bases_out_dev  : DEVICE, capacity n_bytes; receives the reads' bases, concatenated (the ascii_dev of cx_pack_reads)
 *   offsets_out_dev: DEVICE, max_reads + 1 entries; receives read_offsets (entries past max_reads are never written)
 *   counts_out_dev : DEVICE uint64[3]: reads found, bases found, sequence bytes met before the first header (these
 *                    belong to no read: non-zero means the text is not FASTA and the other outputs are meaningless).
 *                    The call is asynchronous; the caller reads counts after synchronising and must treat
 *                    counts[0] > max_reads or counts[2] != 0 as an error.
 *   workspace_dev  : DEVICE, cx_fasta_workspace_bytes(n_bytes) bytes, 256-byte aligned
 * Errors: CX_ERR_ARG (null pointers, workspace too small), CX_ERR_CUDA.
 */
int cx_fasta_workspace_bytes(uint64_t n_bytes, uint64_t *bytes_out);
int cx_fasta_parse(const uint8_t *text_dev, uint64_t n_bytes, uint8_t *bases_out_dev, uint64_t *offsets_out_dev,
                   uint64_t max_reads, uint64_t *counts_out_dev, void *workspace_dev, uint64_t workspace_bytes,
                   cx_stream_t stream);

/*
 * The whole of Figure 2 on the device: partition sizes, batch ranges, and per
 * batch: list suffix ids, build keys, radix sort, refine ties, emit preceding symbols.
 *   packed_reads: DEVICE, ceil(total_bases/32) words in the cx_pack_reads layout
 *   read_offsets: DEVICE, n_reads+1 base offsets, [0] = 0, non-decreasing; total_bases = [n_reads]
 *   out_bwt     : N = total_bases + n_reads bytes over "$ACGT" (ASCII), equal to B_R of
 *                 PAPER.md:55 (ceil(N / 2) bytes of 4-bit codes with opts.out_bits = 4).  DEVICE, or pinned HOST if the
 *                 plan was made with out_is_host_pinned.
 * With opts.shard_count = W > 1 only the bytes [stats.shard_offset, + stats.shard_suffixes) of out_bwt are
 * written (the piece of worker opts.shard_index); out_bwt is still addressed from position 0.
 * Reads may have different lengths, including 0 (one suffix, preceded by '$').  n_reads = 0 is a
 * successful no-op.  Work is enqueued on `stream` (and joined side streams); the call synchronises
 * `stream` to read the partition sizes and once per refinement round, and returns after the last
 * batch has been enqueued and -- for pinned-host output -- copied.
 * Errors: CX_ERR_ARG (also for sizes above the plan's, a read of 2^32 bases or more, or 2^40 bases or more in total:
 * the tie refinement keeps 32-bit lengths and 40-bit base indices), CX_ERR_BUCKET_TOO_LARGE, CX_ERR_CUDA.
 * The result is unique, so two runs on the same input are byte-identical.
 */
int cx_bwt_build(cx_bwt_plan_t *plan, const uint64_t *packed_reads, const uint64_t *read_offsets,
                 uint64_t n_reads, uint8_t *out_bwt, cx_stream_t stream);

/* Destroy a plan (HOST state, events, side streams).  The workspace stays the caller's. */
int cx_bwt_free(cx_bwt_plan_t *plan);

/* Statistics of the last build.  stats_out: HOST. */
int cx_bwt_get_stats(const cx_bwt_plan_t *plan, cx_bwt_stats_t *stats_out);

/*
 * Partition sizes of the last build (Fig. 2 step 1): hist_out[k*(l+1) + r] = number of
 * suffixes whose first l bases, A-padded, spell the base-4 number k and whose length min(m_i - p, l)
 * is r (r < l: the suffix ends inside the prefix -- the "special but easy handling" of PAPER.md:79).
 * hist_out: HOST, capacity entries; *n_out = 4^l * (l+1).
 */
int cx_bwt_get_histogram(const cx_bwt_plan_t *plan, uint64_t *hist_out, uint64_t capacity, uint64_t *n_out);

/*
 * With opts.profile = 1: device time (ms, from CUDA events on the build stream), launches and
 * algorithmic bytes of one kernel class, summed over the last build.  Outputs: HOST.
 */
int cx_bwt_kernel_time(const cx_bwt_plan_t *plan, int kernel_class, double *ms_out, uint64_t *launches_out,
                       uint64_t *bytes_out);

/*
 * Step a6 on its own: stable LSD radix sort ("onesweep": one read + one scatter-write per pass,
 * decoupled look-back between tiles) of n (key, value) pairs by key bits [begin_bit, end_bit).
 * keys/vals and keys_alt/vals_alt: DEVICE double buffers of n entries each; val_bytes is 4 or 8.
 * workspace_dev: DEVICE, at least cx_sort_pairs_workspace_bytes(n) bytes, zero-filled by the caller
 * before its first use.  *result_in_alt (HOST) = 1 if the sorted pairs ended up in the *_alt buffers.
 */
int cx_sort_pairs_workspace_bytes(uint64_t n, uint64_t *bytes_out);
int cx_sort_pairs(uint64_t *keys, void *vals, uint64_t *keys_alt, void *vals_alt, uint64_t n,
                  uint32_t val_bytes, uint32_t begin_bit, uint32_t end_bit, void *workspace_dev,
                  uint64_t workspace_bytes, int *result_in_alt, cx_stream_t stream);

/*
 * cx_sort_pairs for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same stable LSD radix sort (step a6), but its scratch (digit histograms, look-back tile states, ticket)
 * lives in a file-scope `static __device__` array of the library instead of a caller-supplied workspace.  The call makes no
 * cudaMalloc / cudaFree and uses no allocating library routine; the caller still passes inputs and outputs.
 *   n <= CX_SORT_STATIC_MAX_PAIRS (1,048,576 pairs; the array is cx_sort_pairs_workspace_bytes of that: about 0.86 MB, held
 *   by every GPU that loads the library until the process exits); larger n returns CX_ERR_ARG (text via cx_strerror_static).
 *   The array is resolved once per device on the first call there (cudaGetSymbolAddress with that device current), cleared
 *   on `stream` at the start of every call (it keeps the last call's contents) and SHARED by all calls: two calls whose GPU
 *   work overlaps (different streams, threads or processes on one context) race -- serialise them.
 * Other arguments and results as cx_sort_pairs.
 */
#define CX_SORT_STATIC_MAX_PAIRS 1048576ull
int cx_sort_pairs_static(uint64_t *keys, void *vals, uint64_t *keys_alt, void *vals_alt, uint64_t n, uint32_t val_bytes,
                         uint32_t begin_bit, uint32_t end_bit, int *result_in_alt, cx_stream_t stream);
/* Text of the last error cx_sort_pairs_static returned on this thread (which limit was exceeded, or the CUDA error). */
const char *cx_strerror_static(void);

/* Text for an error code; for CX_ERR_CUDA the text of the last CUDA error seen by this thread. */
const char *cx_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* CX_BWT_H */
