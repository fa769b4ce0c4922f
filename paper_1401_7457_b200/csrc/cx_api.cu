// cx_api.cu -- the C ABI of include/cx_bwt.h: plan (workspace carving, m1), build (Figure 2 of the
// paper, as a sequence of kernel launches), statistics and error text.
#include <stdio.h>
#include <string.h>

#include <functional>
#include <new>
#include <vector>

#include "cx_internal.cuh"
#include "cx_launch.h"

using namespace cx;

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    cudaGetLastError();   // clear the non-sticky state
    return CX_ERR_CUDA;
}
#define CX_CUDA(call)                                \
    do {                                             \
        cudaError_t e__ = (call);                    \
        if (e__ != cudaSuccess) return cuda_fail(e__); \
    } while (0)

uint32_t bit_width64(uint64_t v) {
    uint32_t b = 0;
    while (v) ++b, v >>= 1;
    return b;
}
uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

constexpr uint64_t kMaxBatch = 0xFFFF0000ull;   // positions inside a batch are 32-bit

// A region on the host: the partition prefix it stands for (an oversize partition is partitioned again by
// its next l characters, recursively).  Region 0 is the whole collection.
struct RegionHost {
    uint32_t depth = 0;
    std::vector<uint64_t> prefix;   // depth bases, 2 bit/base, MSB-first words
};

struct Batch {
    uint32_t bucket_lo, bucket_hi;   // partitions (codes at the region's depth) sorted together
    uint64_t count, out_offset;
    uint32_t region;                 // index into the plan's regions
    uint64_t ord_lo, ord_hi;         // slice of the listing order taken (a partition of identical suffixes cut into batches)
    uint32_t col;                    // column of the per-tile count table that holds this batch's counts
    bool count_here, scan_here;      // this batch launches the counting scan of its group / scans its column
    CountRanges ranges;              // the group counted when count_here
};

constexpr uint32_t kMaxRegionDepth = 1u << 20;   // bases; deeper refinement is reported as CX_ERR_BUCKET_TOO_LARGE

// Byte offsets of every region of the workspace for a given m1.
#ifndef CX_SPLIT_PAIRS
#define CX_SPLIT_PAIRS 1   // 12-byte (key, id) pairs through the first sort of batches with 64-bit keys and ids
#endif

struct Layout {
    uint64_t info, hist, tile_first, tile_count, tile_sums, scalars, prefix;
    uint64_t keys[2], ids[2], pos, heads[2], big_tiles, word_counts, word_sums, sort, stage[2], pstage[2];
    uint64_t total;
};

struct Shape {
    uint64_t max_reads, max_bases, max_suffixes, max_tiles;
    uint32_t ell, w, cap, id_bytes, pos_bits, prefix_words;
    uint64_t n_buckets;
    bool host_out, pack_out;   // pack_out: NEXT-4, 4-bit output codes
    uint32_t shard_index, shard_count;   // NEXT-2: this plan sorts one of shard_count contiguous partition ranges
    bool sharded() const { return shard_count > 1; }
};

Layout make_layout(const Shape& sh, uint64_t m1) {
    Layout L{};
    uint64_t at = 0;
    auto take = [&](uint64_t bytes) {
        uint64_t o = at;
        at = align_up(at + bytes, 256);
        return o;
    };
    L.info = take(sizeof(BuildInfo));
    L.hist = take(sh.n_buckets * 8);
    L.tile_first = take((sh.max_tiles + 1) * 4);
    // per-tile counts of up to kCountGroup batches at a time; a plan that always fits one batch never counts
    L.tile_count = take((sh.max_tiles + 1) * 8 * (sh.max_suffixes <= m1 && !sh.sharded() ? 1 : kCountGroup));
    L.tile_sums = take((scan_block_count(sh.max_tiles + 1) + 1) * 8);
    L.scalars = take(64);
    L.prefix = take((uint64_t)(sh.prefix_words) * 8);
    for (int i = 0; i < 2; ++i) L.keys[i] = take(m1 * 8);
    for (int i = 0; i < 2; ++i) L.ids[i] = take(m1 * sh.id_bytes + 16);   // (+16: the second position array starts 16-byte aligned)
    // the global path sorts (key, position) pairs: its two arrays of 32-bit positions share the spare id buffer when ids have
    // 8 bytes; with 4-byte ids the second one lives here
    L.pos = take(sh.id_bytes == 4 ? m1 * 4 : 0);
    uint64_t words = (m1 + 31) / 32 + 2;
    for (int i = 0; i < 2; ++i) L.heads[i] = take(words * 4);
    L.big_tiles = take(((m1 + kLocalTile - 1) / kLocalTile / 32 + 2) * 4);
    L.word_counts = take(words * 8);
    L.word_sums = take((scan_block_count(words) + 1) * 8);
    L.sort = take(sort_workspace_bytes(m1));
    // batches are emitted into a staging buffer when the output is pinned host memory (a9) or packed (NEXT-4: the pack
    // step reads it); a packed host output goes through a second, packed staging buffer
    for (int i = 0; i < 2; ++i) L.stage[i] = take(sh.host_out ? m1 : (sh.pack_out && i == 0 ? m1 : 0));
    for (int i = 0; i < 2; ++i) L.pstage[i] = take(sh.host_out && sh.pack_out ? m1 / 2 + 16 : 0);
    L.total = at;
    return L;
}

int make_shape(uint64_t max_reads, uint64_t max_bases, const cx_bwt_opts_t* o, Shape& sh) {
    cx_bwt_opts_t z;
    memset(&z, 0, sizeof(z));
    if (!o) o = &z;
    sh.ell = o->prefix_len ? o->prefix_len : 6;
    sh.w = o->key_bases;   // 0 = chosen in cx_bwt_plan from m1
    sh.cap = o->small_group_max ? o->small_group_max : (uint32_t)kLocalGroupCap;
    if (sh.ell < 1 || sh.ell > 7 || sh.w > 29 || (sh.w && sh.w < sh.ell)) return CX_ERR_ARG;
    if (o->finish_slots != 0 && o->finish_slots != 2 && o->finish_slots != 4) return CX_ERR_ARG;
    if (sh.cap > (uint32_t)kLocalGroupCap) sh.cap = kLocalGroupCap;
    if (max_reads >= 0xFFFFFFFFull) return CX_ERR_ARG;   // read indices travel as 32 bits in the tile table
    sh.max_reads = max_reads;
    sh.max_bases = max_bases;
    sh.max_suffixes = max_reads + max_bases;
    sh.max_tiles = (sh.max_suffixes + kListTile - 1) / kListTile;
    uint64_t max_len = o->max_read_len ? o->max_read_len : max_bases;
    if (max_len > max_bases) max_len = max_bases;
    sh.pos_bits = bit_width64(max_len);
    sh.prefix_words = (uint32_t)((max_len < kMaxRegionDepth ? max_len : kMaxRegionDepth) / 32 + 2);   // region prefix of a refined partition
    uint32_t read_bits = bit_width64(max_reads ? max_reads - 1 : 0);
    if (sh.pos_bits + read_bits > 64) return CX_ERR_ARG;
    sh.id_bytes = sh.pos_bits + read_bits <= 32 ? 4 : 8;
    sh.n_buckets = (1ull << (2 * sh.ell)) * (sh.ell + 1);
    sh.host_out = o->out_is_host_pinned != 0;
    if (o->out_bits != 0 && o->out_bits != 8 && o->out_bits != 4) return CX_ERR_ARG;
    sh.pack_out = o->out_bits == 4;
    sh.shard_count = o->shard_count ? o->shard_count : 1;
    sh.shard_index = o->shard_index;
    if (sh.shard_count > 65536 || sh.shard_index >= sh.shard_count) return CX_ERR_ARG;
    if (sh.pack_out && sh.shard_count > 1) return CX_ERR_ARG;   // pieces of a packed output would share bytes at their ends
    return CX_OK;
}

}  // namespace

struct cx_bwt_plan_s {
    Shape sh;
    cx_bwt_opts_t opts;
    Layout L;
    uint64_t m1;
    unsigned char* ws;
    int n_sms;
    SortWorkspace sort;
    // pinned host mirror: BuildInfo | scalars[8] | hist
    unsigned char* h_pinned;
    unsigned char* h_pinned_dev;   // the same memory as kernels address it
    BuildInfo* h_info;
    uint64_t* h_scalars;
    uint64_t* h_hist;
    std::vector<Batch> batches;
    std::vector<RegionHost> regions;
    uint64_t* h_hist2;   // pinned: sizes of the sub-partitions of the partition being refined
    Launch prof;
    cx_bwt_stats_t stats;
    cudaStream_t copy_stream;
    cudaEvent_t emit_done, stage_free[2];
    bool stage_busy[2];
    bool built;
};

// ---------------------------------------------------------------------------------------------
// plan
// ---------------------------------------------------------------------------------------------
extern "C" int cx_bwt_workspace_bytes(uint64_t n_reads, uint64_t total_bases, const cx_bwt_opts_t* opts, uint64_t* bytes_out) {
    if (!bytes_out) return CX_ERR_ARG;
    Shape sh;
    int rc = make_shape(n_reads, total_bases, opts, sh);
    if (rc) return rc;
    uint64_t m1 = sh.max_suffixes ? sh.max_suffixes : 1;
    if (opts && opts->max_batch_suffixes && opts->max_batch_suffixes < m1) m1 = opts->max_batch_suffixes;
    if (m1 > kMaxBatch) m1 = kMaxBatch;
    *bytes_out = make_layout(sh, m1).total;
    return CX_OK;
}

extern "C" int cx_bwt_plan(cx_bwt_plan_t** plan_out, uint64_t max_reads, uint64_t max_total_bases, const cx_bwt_opts_t* opts,
                           void* workspace_dev, uint64_t workspace_bytes) {
    if (!plan_out || !workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) & 255)) return CX_ERR_ARG;
    *plan_out = nullptr;
    Shape sh;
    int rc = make_shape(max_reads, max_total_bases, opts, sh);
    if (rc) return rc;
    // m1 = the largest batch whose layout fits (m1 depends only on the GPU memory limit)
    uint64_t hi = sh.max_suffixes ? sh.max_suffixes : 1;
    if (opts && opts->max_batch_suffixes && opts->max_batch_suffixes < hi) hi = opts->max_batch_suffixes;
    if (hi > kMaxBatch) hi = kMaxBatch;
    if (make_layout(sh, 1).total > workspace_bytes) return CX_ERR_WORKSPACE;
    uint64_t lo = 1;
    // the largest legal input in one batch needs a smaller count table than any split does, so test it first
    if (make_layout(sh, hi).total <= workspace_bytes) lo = hi;
    while (lo < hi) {
        uint64_t mid = lo + (hi - lo + 1) / 2;
        if (make_layout(sh, mid).total <= workspace_bytes) lo = mid; else hi = mid - 1;
    }
    int dev = 0, n_sms = 0;
    CX_CUDA(cudaGetDevice(&dev));
    CX_CUDA(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));

    // First-round window ("stringword"): wide enough that 4^w exceeds the number of suffixes of the
    // whole collection, so that random collisions are rare and tie groups are the genuinely shared substrings.  The key
    // (first_key: rank of the window's symbols + a "has w bases" bit) takes 32 bits at w = 15 -- half the bytes per
    // radix pass and 4 passes -- which is used up to 2^30 suffixes.  Beyond that the key is 64-bit with as many bases
    // as the passes that ceil(log4 N) bases need anyway can carry (19 bases in 40 bits, 5 passes, at 6e9 .. 1e11 suffixes).
    if (sh.w == 0) {
        if (sh.max_suffixes <= (1ull << 30)) {
            sh.w = 15;
        } else {
            const uint32_t log4 = (bit_width64(sh.max_suffixes - 1) + 1) / 2;
            const uint32_t passes = (first_key_bits(log4) + kRadixBits - 1) / kRadixBits;
            sh.w = log4;
            while (sh.w < 29 && (first_key_bits(sh.w + 1) + kRadixBits - 1) / kRadixBits == passes) ++sh.w;
        }
    }
    if (sh.w < sh.ell) sh.w = sh.ell;
    cx_bwt_plan_t* p = new (std::nothrow) cx_bwt_plan_t();
    if (!p) return CX_ERR_NOMEM;
    p->sh = sh;
    memset(&p->opts, 0, sizeof(p->opts));
    if (opts) p->opts = *opts;
    p->m1 = lo;
    p->L = make_layout(sh, lo);
    p->ws = static_cast<unsigned char*>(workspace_dev);
    p->n_sms = n_sms;
    p->prof.timing = p->opts.profile != 0;
    memset(&p->stats, 0, sizeof(p->stats));
    p->built = false;
    p->stage_busy[0] = p->stage_busy[1] = false;
    p->h_pinned = nullptr;
    p->h_pinned_dev = nullptr;
    p->copy_stream = nullptr;
    p->emit_done = p->stage_free[0] = p->stage_free[1] = nullptr;

    size_t host_bytes = sizeof(BuildInfo) + 64 + 2 * sh.n_buckets * 8;
    cudaError_t e = cudaHostAlloc((void**)&p->h_pinned, host_bytes, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&p->h_pinned_dev, p->h_pinned, 0);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->emit_done, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->stage_free[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->stage_free[1], cudaEventDisableTiming);
    // the tile-state array must start from epoch 0 everywhere
    if (e == cudaSuccess) e = cudaMemset(p->ws + p->L.sort, 0, sort_workspace_bytes(lo));
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        cx_bwt_free(p);
        return cuda_fail(e);
    }
    p->h_info = reinterpret_cast<BuildInfo*>(p->h_pinned);
    p->h_scalars = reinterpret_cast<uint64_t*>(p->h_pinned + sizeof(BuildInfo));
    p->h_hist = reinterpret_cast<uint64_t*>(p->h_pinned + sizeof(BuildInfo) + 64);
    p->h_hist2 = p->h_hist + sh.n_buckets;
    sort_workspace_carve(p->sort, p->ws + p->L.sort, lo);
    *plan_out = p;
    return CX_OK;
}

extern "C" int cx_bwt_free(cx_bwt_plan_t* p) {
    if (!p) return CX_OK;
    p->prof.destroy();
    if (p->h_pinned) cudaFreeHost(p->h_pinned);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    if (p->emit_done) cudaEventDestroy(p->emit_done);
    for (int i = 0; i < 2; ++i)
        if (p->stage_free[i]) cudaEventDestroy(p->stage_free[i]);
    delete p;
    return CX_OK;
}

// ---------------------------------------------------------------------------------------------
// small entry points
// ---------------------------------------------------------------------------------------------
extern "C" int cx_pack_reads(const uint8_t* ascii_dev, uint64_t total_bases, uint64_t* packed_out_dev, uint32_t* status_dev,
                             cx_stream_t stream) {
    if (total_bases == 0) {
        if (status_dev) CX_CUDA(cudaMemsetAsync(status_dev, 0, 4, stream));
        return CX_OK;
    }
    if (!ascii_dev || !packed_out_dev) return CX_ERR_ARG;
    uint32_t* st = status_dev ? status_dev : pack_fallback_status();
    if (!st) return cuda_fail(cudaGetLastError());
    CX_CUDA(cudaMemsetAsync(st, 0, 4, stream));
    CX_CUDA(launch_pack(ascii_dev, total_bases, packed_out_dev, st, stream));
    if (!status_dev) {
        uint32_t bad = 0;
        CX_CUDA(cudaMemcpyAsync(&bad, st, 4, cudaMemcpyDeviceToHost, stream));
        CX_CUDA(cudaStreamSynchronize(stream));
        if (bad) return CX_ERR_BAD_BASE;
    }
    return CX_OK;
}

extern "C" int cx_fasta_workspace_bytes(uint64_t n_bytes, uint64_t* bytes_out) {
    if (!bytes_out) return CX_ERR_ARG;
    *bytes_out = fasta_workspace_bytes(n_bytes);
    return CX_OK;
}

extern "C" int cx_fasta_parse(const uint8_t* text_dev, uint64_t n_bytes, uint8_t* bases_out_dev, uint64_t* offsets_out_dev, uint64_t max_reads,
                              uint64_t* counts_out_dev, void* workspace_dev, uint64_t workspace_bytes, cx_stream_t stream) {
    if (!offsets_out_dev || !counts_out_dev || (n_bytes && (!text_dev || !bases_out_dev || !workspace_dev))) return CX_ERR_ARG;
    if (n_bytes && (workspace_bytes < fasta_workspace_bytes(n_bytes) || (reinterpret_cast<uintptr_t>(workspace_dev) & 255))) return CX_ERR_ARG;
    if (n_bytes > (1ull << 43)) return CX_ERR_ARG;   // tiles are launched as one grid dimension
    CX_CUDA(launch_fasta_parse(text_dev, n_bytes, bases_out_dev, offsets_out_dev, max_reads, counts_out_dev,
                               static_cast<unsigned char*>(workspace_dev), stream));
    return CX_OK;
}

extern "C" const char* cx_strerror(int code) {
    switch (code) {
    case CX_OK: return "ok";
    case CX_ERR_ARG: return "invalid argument (null pointer, bad option, size above the plan's maximum, or bad offsets)";
    case CX_ERR_BAD_BASE: return "input contains a byte outside ACGT";
    case CX_ERR_WORKSPACE: return "workspace too small";
    case CX_ERR_BUCKET_TOO_LARGE: return "a partition still exceeds the batch limit m1 after refinement to the depth limit";
    case CX_ERR_CUDA: return g_cuda_msg;
    case CX_ERR_NOMEM: return "host allocation failed";
    default: return "unknown error code";
    }
}

extern "C" int cx_bwt_get_stats(const cx_bwt_plan_t* p, cx_bwt_stats_t* out) {
    if (!p || !out) return CX_ERR_ARG;
    *out = p->stats;
    return CX_OK;
}

extern "C" int cx_bwt_get_histogram(const cx_bwt_plan_t* p, uint64_t* hist_out, uint64_t capacity, uint64_t* n_out) {
    if (!p || !n_out) return CX_ERR_ARG;
    *n_out = p->sh.n_buckets;
    if (!p->built || !hist_out || capacity < p->sh.n_buckets) return CX_ERR_ARG;
    memcpy(hist_out, p->h_hist, p->sh.n_buckets * 8);
    return CX_OK;
}

extern "C" int cx_bwt_kernel_time(const cx_bwt_plan_t* p, int cls, double* ms_out, uint64_t* launches_out, uint64_t* bytes_out) {
    if (!p || cls < 0 || cls >= CX_K_COUNT) return CX_ERR_ARG;
    if (ms_out) *ms_out = p->prof.ms[cls];
    if (launches_out) *launches_out = p->prof.launches[cls];
    if (bytes_out) *bytes_out = p->prof.bytes[cls];
    return CX_OK;
}

// ---------------------------------------------------------------------------------------------
// build
// ---------------------------------------------------------------------------------------------
namespace {

// Fig. 2 steps 1, 2 and 3(b): consecutive partitions are merged into batches of total size
// <= m1; a partition larger than m1 is "further partition[ed] by looking at the next l characters ... recursively":
// its sub-partition sizes come from `sub_hist` (a device scan confined to the partition's region) and are planned the
// same way, in place, so that batches stay in BWT order.  A partition of suffixes that END inside the prefix holds
// identical strings, whose order is the listing order: it is simply cut into slices of that order.
struct Planner {
    cx_bwt_plan_t* p;
    std::function<int(uint32_t, uint64_t*)> sub_hist;   // sizes of the sub-partitions of region #i into p->h_hist2-sized array
    uint64_t out = 0;
    Batch cur{};
    bool open = false;
    uint64_t n_total = 0;                    // N, for the shard rule
    uint64_t shard_lo = ~0ull, shard_n = 0;  // output range of this plan's shard

    void flush() {
        if (!open) return;
        p->batches.push_back(cur);
        out += cur.count;
        open = false;
    }
    int region(uint32_t ri, const uint64_t* hist, bool top) {
        const Shape& sh = p->sh;
        const uint64_t nb = sh.n_buckets, m1 = p->m1;
        uint64_t seen = 0;   // suffixes in the partitions before b (top level: their first position in the BWT)
        for (uint64_t b = 0; b < nb; ++b) {
            const uint64_t c = hist[b];
            if (c == 0) continue;
            if (top && c > p->stats.largest_bucket) p->stats.largest_bucket = c;
            if (top && sh.sharded()) {
                // "a contiguous range of partitions of roughly equal total size" per worker: a partition
                // goes to the shard that its first output position falls in when [0, N) is cut into shard_count equal parts
                const uint64_t owner = (uint64_t)(((unsigned __int128)seen * sh.shard_count) / n_total);
                seen += c;
                if (owner != sh.shard_index) {
                    flush();
                    out += c;
                    continue;
                }
                if (shard_lo == ~0ull) shard_lo = seen - c;
                shard_n += c;
            }
            if (c > m1) {
                flush();
                const uint32_t r = (uint32_t)(b % (sh.ell + 1)), kmer = (uint32_t)(b / (sh.ell + 1));
                if (r < sh.ell) {   // identical suffixes: slices of the listing order
                    for (uint64_t k0 = 0; k0 < c; k0 += m1) {
                        const uint64_t n = c - k0 < m1 ? c - k0 : m1;
                        Batch s{};
                        s.bucket_lo = s.bucket_hi = (uint32_t)b;
                        s.count = n, s.out_offset = out, s.region = ri, s.ord_lo = k0, s.ord_hi = k0 + n;
                        p->batches.push_back(s);
                        out += n;
                    }
                } else {            // refine by the next l characters
                    const uint32_t depth = p->regions[ri].depth, child_depth = depth + sh.ell;
                    if (child_depth > kMaxRegionDepth || (child_depth + 31) / 32 + 1 > sh.prefix_words) return CX_ERR_BUCKET_TOO_LARGE;
                    RegionHost child;
                    child.depth = child_depth;
                    child.prefix = p->regions[ri].prefix;
                    child.prefix.resize((child_depth + 31) / 32 + 1, 0ull);
                    for (uint32_t i = 0; i < sh.ell; ++i) {
                        const uint64_t code = (kmer >> (2 * (sh.ell - 1 - i))) & 3u;
                        const uint32_t j = depth + i;
                        child.prefix[j / 32] |= code << (62 - 2 * (j % 32));
                    }
                    p->regions.push_back(child);
                    const uint32_t ci = (uint32_t)p->regions.size() - 1;
                    std::vector<uint64_t> h(nb);
                    int rc = sub_hist(ci, h.data());
                    if (rc) return rc;
                    uint64_t total = 0;
                    for (uint64_t q = 0; q < nb; ++q) total += h[q];
                    if (total != c) return CX_ERR_CUDA;   // the region scan and the partition scan disagree
                    p->stats.refined_partitions += 1;
                    rc = region(ci, h.data(), false);
                    if (rc) return rc;
                    flush();
                }
                continue;
            }
            if (open && cur.count + c > m1) flush();
            if (!open) {
                cur = Batch{};
                cur.bucket_lo = (uint32_t)b, cur.out_offset = out, cur.region = ri, cur.ord_lo = 0, cur.ord_hi = ~0ull;
                open = true;
            }
            cur.bucket_hi = (uint32_t)b;
            cur.count += c;
        }
        flush();
        return CX_OK;
    }
    // which batch launches the counting scan, which column of the count table each batch reads
    void assign_count_groups() {
        std::vector<Batch>& B = p->batches;
        for (size_t i = 0; i < B.size();) {
            if (B[i].ord_hi != ~0ull) {   // slices of one partition share one counted and scanned column
                size_t j = i;
                while (j < B.size() && B[j].ord_hi != ~0ull && B[j].region == B[i].region && B[j].bucket_lo == B[i].bucket_lo) {
                    B[j].col = 0, B[j].count_here = B[j].scan_here = (j == i);
                    ++j;
                }
                B[i].ranges.n = 1, B[i].ranges.first[0] = B[i].bucket_lo, B[i].ranges.first[1] = B[i].bucket_lo + 1;
                i = j;
                continue;
            }
            size_t j = i;
            CountRanges cr{};
            while (j < B.size() && cr.n < (uint32_t)kCountGroup && B[j].ord_hi == ~0ull && B[j].region == B[i].region) {
                B[j].col = cr.n, B[j].count_here = (j == i), B[j].scan_here = true;
                cr.first[cr.n++] = B[j].bucket_lo;
                ++j;
            }
            cr.first[cr.n] = B[j - 1].bucket_hi + 1;
            B[i].ranges = cr;
            i = j;
        }
    }
};

// Small results (sizes, counters, the partition histogram) come back through pinned host memory that a kernel writes itself.
// A cudaMemcpyAsync of a few bytes would queue behind whatever large copy the caller has in flight on the same copy engine
// (a pipelined caller's previous output on its way to the host) and stall the build for as long as that copy takes.
__global__ void readback_kernel(const uint64_t* __restrict__ src, uint64_t* __restrict__ dst_host, uint32_t n_words) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += gridDim.x * blockDim.x) dst_host[i] = src[i];
}
static_assert(sizeof(BuildInfo) % 8 == 0, "read back in 8-byte words");
// dst_host: an address inside the plan's pinned block (whole 8-byte words); visible to the host after the stream is synchronised
cudaError_t readback(cx_bwt_plan_t* p, void* dst_host, const void* src_dev, size_t bytes, cudaStream_t s) {
#if defined(CX_READBACK_MEMCPY) && CX_READBACK_MEMCPY   // the alternative it replaced, kept for the A/B in DESIGN.md section 16
    return cudaMemcpyAsync(dst_host, src_dev, bytes, cudaMemcpyDeviceToHost, s);
#endif
    const uint32_t n = (uint32_t)((bytes + 7) / 8);
    const uint32_t blocks = (n + 255) / 256;
    unsigned char* dst = p->h_pinned_dev + (static_cast<unsigned char*>(dst_host) - p->h_pinned);
    readback_kernel<<<blocks < 64 ? blocks : 64, 256, 0, s>>>(static_cast<const uint64_t*>(src_dev), reinterpret_cast<uint64_t*>(dst), n);
    p->prof.launches[CX_K_PREP] += 1;
    return cudaGetLastError();
}

template <typename KeyT, typename IdT>
int build_impl(cx_bwt_plan_t* p, const uint64_t* packed, const uint64_t* offsets, uint64_t n_reads, uint8_t* out, cudaStream_t s) {
    const Shape& sh = p->sh;
    const Layout& L = p->L;
    unsigned char* ws = p->ws;
    Launch* prof = &p->prof;
    BuildInfo* d_info = reinterpret_cast<BuildInfo*>(ws + L.info);
    uint64_t* d_hist = reinterpret_cast<uint64_t*>(ws + L.hist);
    uint32_t* d_tile_first = reinterpret_cast<uint32_t*>(ws + L.tile_first);
    uint64_t* d_tile_count = reinterpret_cast<uint64_t*>(ws + L.tile_count);
    uint64_t* d_tile_sums = reinterpret_cast<uint64_t*>(ws + L.tile_sums);
    uint64_t* d_scalars = reinterpret_cast<uint64_t*>(ws + L.scalars);   // [0] scan total, [1] elements finished locally
    uint64_t* d_keys[2] = {reinterpret_cast<uint64_t*>(ws + L.keys[0]), reinterpret_cast<uint64_t*>(ws + L.keys[1])};
    IdT* d_ids[2] = {reinterpret_cast<IdT*>(ws + L.ids[0]), reinterpret_cast<IdT*>(ws + L.ids[1])};
    uint32_t* d_pos = reinterpret_cast<uint32_t*>(ws + L.pos);
    uint32_t* d_heads[2] = {reinterpret_cast<uint32_t*>(ws + L.heads[0]), reinterpret_cast<uint32_t*>(ws + L.heads[1])};
    uint32_t* d_big_tiles = reinterpret_cast<uint32_t*>(ws + L.big_tiles);
    uint64_t* d_word_counts = reinterpret_cast<uint64_t*>(ws + L.word_counts);
    uint64_t* d_word_sums = reinterpret_cast<uint64_t*>(ws + L.word_sums);

    Reads R{};
    R.packed = packed;
    R.offsets = offsets;
    R.n_reads = n_reads;
    R.n_words = 0;   // set on the device from BuildInfo until the host knows total_bases
    R.pos_bits = sh.pos_bits;

    // ---- Fig. 2 step 1: scan all suffixes, partition sizes ------------------------------------
    {
        ScopedLaunch sl(prof, CX_K_PREP, (n_reads + 1) * 8, s);
        CX_CUDA(launch_prep(offsets, n_reads, sh.max_bases, d_info, s));
    }
    {
        ScopedLaunch sl(prof, CX_K_PREP, sh.max_tiles * 4, s);
        CX_CUDA(launch_tile_table(offsets, n_reads, d_info, d_tile_first, sh.max_tiles, s));
    }
    CX_CUDA(cudaMemsetAsync(d_hist, 0, sh.n_buckets * 8, s));
    CX_CUDA(cudaMemsetAsync(d_scalars, 0, 64, s));
    // A plan whose largest legal input fits one batch needs no partition sizes to list its suffixes: the listing
    // scan then counts them on the way (one read of the collection instead of two).
    const bool fused_scan = sh.max_suffixes <= p->m1 && !sh.sharded();
    const uint32_t w = sh.w;
    const uint32_t key_bits = first_key_bits(w);
    const uint32_t n_passes = (key_bits + kRadixBits - 1) / kRadixBits;
    KeyT* d_keys1[2] = {reinterpret_cast<KeyT*>(d_keys[0]), reinterpret_cast<KeyT*>(d_keys[1])};   // first-round keys
    // 32-bit key and 32-bit id: one 64-bit word per suffix (key << 32 | id), sorted keys-only over its upper half
    const bool pack_kv = sizeof(KeyT) == 4 && sizeof(IdT) == 4;
    if (fused_scan) {
        CX_CUDA(cudaMemsetAsync(p->sort.hist, 0, (size_t)n_passes * kRadix * sizeof(uint64_t), s));
        ScopedLaunch sl(prof, CX_K_LIST, 0, s);
        CX_CUDA((launch_list_write<KeyT, IdT>(R, d_info, d_tile_first, sh.ell, w, 0, 0, nullptr, d_keys1[0], d_ids[0], sh.max_tiles, n_passes,
                                              p->sort.hist, p->n_sms, pack_kv, d_hist, p->m1, Region{}, 0, ~0ull, s)));
    } else {
        ScopedLaunch sl(prof, CX_K_HIST, 0, s);
        CX_CUDA(launch_bucket_hist(R, d_info, d_tile_first, sh.ell, Region{}, d_hist, sh.max_tiles, p->n_sms, s));
    }
    CX_CUDA(readback(p, p->h_info, d_info, sizeof(BuildInfo), s));
    CX_CUDA(readback(p, p->h_hist, d_hist, sh.n_buckets * 8, s));
    CX_CUDA(cudaStreamSynchronize(s));
    const BuildInfo info = *p->h_info;
    if (info.bad_offsets || info.total_bases > sh.max_bases || (info.max_len >> sh.pos_bits) != 0) return CX_ERR_ARG;
    const uint64_t N = info.n_suffixes;
    // the in-block refinement keeps (first base of the window : 40 bits) and (bases left : 32 bits) per suffix
    if (info.max_len >= (1ull << 32) || info.total_bases >= (1ull << 40)) return CX_ERR_ARG;
    const uint32_t cap = sh.cap;
    if (fused_scan) prof->bytes[CX_K_LIST] += info.total_bases / 4 + (n_reads + 1) * 8 + N * (sizeof(KeyT) + sizeof(IdT));
    else prof->bytes[CX_K_HIST] += info.total_bases / 4 + (n_reads + 1) * 8;
    R.n_words = (info.total_bases + 31) >> 5;
    R.uniform = info.nonuniform ? 0u : 1u;
    R.uniform_len = info.first_len;
    p->stats.n_suffixes = N;
    p->stats.max_batch = p->m1;
    p->stats.id_bytes = sizeof(IdT);
    p->stats.max_read_len = (uint32_t)info.max_len;
    p->stats.uniform_len = R.uniform;
    p->built = true;

    // ---- steps 1-2, 3(b): batch ranges, oversize partitions refined by their next l characters ----------
    uint64_t* d_prefix = reinterpret_cast<uint64_t*>(ws + L.prefix);
    uint32_t region_on_device = 0;   // region 0 (depth 0) needs no prefix
    auto use_region = [&](uint32_t ri, Region& dev) -> cudaError_t {
        const RegionHost& rh = p->regions[ri];
        dev.prefix = d_prefix;
        dev.depth = rh.depth;
        if (rh.depth == 0 || ri == region_on_device) return cudaSuccess;
        region_on_device = ri;
        return cudaMemcpyAsync(d_prefix, rh.prefix.data(), rh.prefix.size() * 8, cudaMemcpyHostToDevice, s);   // pageable: staged at once
    };
    p->regions.clear();
    p->regions.push_back(RegionHost{});
    p->batches.clear();
    Planner planner{p, nullptr};
    planner.sub_hist = [&](uint32_t ri, uint64_t* hist_out) -> int {
        Region dev{};
        CX_CUDA(use_region(ri, dev));
        CX_CUDA(cudaMemsetAsync(d_hist, 0, sh.n_buckets * 8, s));
        {
            ScopedLaunch sl(prof, CX_K_HIST, info.total_bases / 4 + (n_reads + 1) * 8, s);
            CX_CUDA(launch_bucket_hist(R, d_info, d_tile_first, sh.ell, dev, d_hist, sh.max_tiles, p->n_sms, s));
        }
        CX_CUDA(readback(p, p->h_hist2, d_hist, sh.n_buckets * 8, s));
        CX_CUDA(cudaStreamSynchronize(s));
        memcpy(hist_out, p->h_hist2, sh.n_buckets * 8);
        return CX_OK;
    };
    planner.n_total = N;
    int rc = planner.region(0, p->h_hist, true);
    if (rc) return rc;
    if (planner.out != N) return CX_ERR_CUDA;   // a mismatch means the partition scan misbehaved
    planner.assign_count_groups();
    p->stats.n_batches = (uint32_t)p->batches.size();
    p->stats.shard_offset = sh.sharded() ? (planner.shard_n ? planner.shard_lo : N) : 0;
    p->stats.shard_suffixes = sh.sharded() ? planner.shard_n : N;
    const uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    const bool single = p->batches.size() == 1 && p->batches[0].ord_hi == ~0ull && p->batches[0].count == N;
    if (fused_scan && !single) return CX_ERR_CUDA;   // cannot happen: N <= max_suffixes <= m1
    p->stats.sort_passes = (key_bits + kRadixBits - 1) / kRadixBits;

    // Batches of a plan with 64-bit keys and ids travel through the sort as 12-byte pairs: the key above the id's high part in
    // the 64-bit word, the id's low word as a 32-bit value (cx_internal.cuh, launch_list_write).  0 = not used.
    uint32_t split = 0;
#if CX_SPLIT_PAIRS
    if (sizeof(KeyT) == 8 && sizeof(IdT) == 8 && !single && !fused_scan && key_bits < 64) {
        const uint32_t id_bits = R.pos_bits + (n_reads > 1 ? bit_width64(n_reads - 1) : 0u);
        if (id_bits <= 32 + (64 - key_bits)) split = 64 - key_bits;
    }
#endif

    for (size_t bi = 0; bi < p->batches.size(); ++bi) {
        const Batch& B = p->batches[bi];
        const uint64_t nb = B.count;
        Region region{};
        const uint32_t depth_base = p->regions[B.region].depth;   // symbols every suffix of the batch shares
        // ---- step 3(a) + 3(c)i: list the batch's suffixes with their first keys ----------------
        if (!fused_scan) CX_CUDA(cudaMemsetAsync(p->sort.hist, 0, (size_t)n_passes * kRadix * sizeof(uint64_t), s));
        if (fused_scan) {
            // listed before the partition sizes were read back
        } else if (single) {
            ScopedLaunch sl(prof, CX_K_LIST, info.total_bases / 4 + (n_reads + 1) * 8 + nb * (sizeof(KeyT) + sizeof(IdT)), s);
            CX_CUDA((launch_list_write<KeyT, IdT>(R, d_info, d_tile_first, sh.ell, w, B.bucket_lo, B.bucket_hi, nullptr, d_keys1[0],
                                                  d_ids[0], n_tiles, n_passes, p->sort.hist, p->n_sms, pack_kv, nullptr, ~0ull, Region{}, 0, ~0ull,
                                                  s)));
        } else {
            const uint64_t col_stride = sh.max_tiles + 1;
            CX_CUDA(use_region(B.region, region));
            const uint64_t n_tiles = list_scan_tiles(R, region, N);   // (shadows the whole-collection tile count)
            if (B.count_here) {   // one scan counts this batch and up to seven that follow it in the same region
                ScopedLaunch sl(prof, CX_K_LIST, info.total_bases / 4 + (n_reads + 1) * 8 + n_tiles * 8 * B.ranges.n, s);
                CX_CUDA(launch_list_count(R, d_info, d_tile_first, sh.ell, region, B.ranges, d_tile_count, col_stride, n_tiles, s));
            }
            uint64_t* d_col = d_tile_count + B.col * col_stride;
            if (B.scan_here) {
                ScopedLaunch sl(prof, CX_K_LIST, n_tiles * 16, s);
                CX_CUDA(launch_scan_u64(d_col, n_tiles, d_tile_sums, d_scalars + 2, s));
                prof->launches[CX_K_LIST] += 2;   // the scan is three kernels
            }
            ScopedLaunch sl(prof, CX_K_LIST, info.total_bases / 4 + (n_reads + 1) * 8 + nb * (split ? 12 : sizeof(KeyT) + sizeof(IdT)), s);
            CX_CUDA((launch_list_write<KeyT, IdT>(R, d_info, d_tile_first, sh.ell, w, B.bucket_lo, B.bucket_hi, d_col, d_keys1[0], d_ids[0],
                                                  n_tiles, n_passes, p->sort.hist, p->n_sms, pack_kv, nullptr, ~0ull, region, B.ord_lo, B.ord_hi,
                                                  s, split)));
        }
        // ---- step 3(c)ii: sort (first w symbols) ------------------------------------------------
        int in_alt = 0;
        if (pack_kv)
            CX_CUDA((sort_pairs<uint64_t, NoVal>(d_keys[0], nullptr, d_keys[1], nullptr, nb, 32, 32 + key_bits, p->sort, &in_alt, prof, s, true)));
        else if (split)
            CX_CUDA((sort_pairs<uint64_t, uint32_t>(d_keys[0], reinterpret_cast<uint32_t*>(d_ids[0]), d_keys[1], reinterpret_cast<uint32_t*>(d_ids[1]), nb, split,
                                                    64, p->sort, &in_alt, prof, s, true)));
        else
            CX_CUDA((sort_pairs<KeyT, IdT>(d_keys1[0], d_ids[0], d_keys1[1], d_ids[1], nb, 0, key_bits, p->sort, &in_alt, prof, s, true)));
        const int cur = in_alt;
        // `ids`: where the global path finds (and rearranges) the batch's ids.  Separate arrays: the sorted ids themselves.  Packed
        // or split pairs: a buffer that the warp kernel fills for the groups it leaves to that path.
        IdT* ids = pack_kv ? d_ids[0] : split ? d_ids[1 - cur] : d_ids[cur];
        IdT* spare_ids = pack_kv ? d_ids[1] : split ? d_ids[cur] : d_ids[1 - cur];   // free once the warp and block kernels are done
        // a9: with pinned-host output the batch is emitted into a staging buffer of the workspace
        const int st = sh.host_out ? (int)(bi & 1) : 0;
        uint8_t* dst = sh.host_out || sh.pack_out ? ws + L.stage[st] : out + B.out_offset;
        if (sh.host_out && p->stage_busy[st]) CX_CUDA(cudaStreamWaitEvent(s, p->stage_free[st], 0));
        // ---- steps 3(c)ii-iii fused: head flags, in-block tie refinement, emit ----------------------
        const uint64_t n_words = (nb + 31) >> 5;
        int hc = 0;
        unsigned long long* d_done = reinterpret_cast<unsigned long long*>(d_scalars + 1);
        // window width of the register refinement: from a sample of this batch's tie-group sizes unless the plan fixes it
        uint32_t slots = p->opts.finish_slots;
        if (slots == 0) {
            uint64_t sampled = 0;
            const uint64_t big_before = p->h_scalars[6];
            CX_CUDA((launch_group_probe<KeyT, IdT>(d_keys1[cur], w, nb, pack_kv, reinterpret_cast<unsigned long long*>(d_scalars + 6), &sampled, s, split)));
            if (sampled) {
                CX_CUDA(readback(p, p->h_scalars + 6, d_scalars + 6, 8, s));
                CX_CUDA(cudaStreamSynchronize(s));
            }
            slots = sampled && (p->h_scalars[6] - big_before) * 4 > sampled ? 4u : 2u;   // more than a quarter in groups above 64
        }
        CX_CUDA(cudaMemsetAsync(d_heads[0], 0xff, (n_words + 1) * 4, s));   // every position a group of one until the warp kernel says otherwise
        CX_CUDA((launch_finish_first<KeyT, IdT>(R, d_keys1[cur], w, depth_base + w, d_heads[0], split ? d_ids[cur] : ids, nb, cap, dst, d_done, d_big_tiles,
                                                p->n_sms, pack_kv, slots, prof, s, split, split ? ids : nullptr)));
        // groups of more than cap suffixes (counted by the warp kernel) go through global rounds; usually there are none
        const uint64_t over_before = p->h_scalars[5], local_before = p->h_scalars[1];
        CX_CUDA(readback(p, p->h_scalars, d_scalars, 48, s));
        CX_CUDA(cudaStreamSynchronize(s));
        const bool any_oversize = p->h_scalars[5] != over_before;
        // every suffix refined here also costs its id read, an 8-byte window gathered and its id written
        prof->bytes[CX_K_FINISH] += (p->h_scalars[1] - local_before) * (2 * sizeof(IdT) + 8);
        // ---- what is still tied goes through global rounds: re-key, sort, write back ------------------
        uint32_t depth = depth_base + w, rounds = 0;
        while (any_oversize) {
            {
                ScopedLaunch sl(prof, CX_K_REFINE_SCAN, n_words * 12, s);
                CX_CUDA(launch_active_count(d_heads[hc], nb, d_word_counts, s));
            }
            {
                ScopedLaunch sl(prof, CX_K_REFINE_SCAN, n_words * 16, s);
                CX_CUDA(launch_scan_u64(d_word_counts, n_words, d_word_sums, d_scalars, s));
            }
            prof->launches[CX_K_REFINE_SCAN] += 2;
            CX_CUDA(readback(p, p->h_scalars, d_scalars, 48, s));
            CX_CUDA(cudaStreamSynchronize(s));
            const uint64_t n_act = p->h_scalars[0] & 0xffffffffull;
            const uint64_t n_groups = p->h_scalars[0] >> 32;
            if (n_act == 0) break;
            // key = [group ordinal][w_r bases][length]: as deep a window as the ordinal leaves room for
            const uint32_t gbits = n_groups > 1 ? bit_width64(n_groups - 1) : 0;
            uint32_t w_r = (59 - gbits) / 2;
            if (w_r > 29) w_r = 29;
            // free at this point: both key buffers and the spare id buffer.  The sort ping-pongs (key, position) pairs between
            // them; whichever key buffer does not hold the sorted keys afterwards takes the gathered ids.
            uint64_t* kc = d_keys[1 - cur];
            uint32_t* pc = reinterpret_cast<uint32_t*>(spare_ids);
            uint32_t* pc_alt = sizeof(IdT) == 8 ? pc + ((p->m1 + 3) & ~3ull) : d_pos;
            {
                ScopedLaunch sl(prof, CX_K_REFINE_KEY, nb / 8 + n_act * (sizeof(IdT) + 8 + 8 + 4), s);
                CX_CUDA(launch_refine_rekey<IdT>(R, d_heads[hc], d_word_counts, ids, nb, depth, w_r, kc, pc, s));
            }
            int alt = 0;
            CX_CUDA((sort_pairs<uint64_t, uint32_t>(kc, pc, d_keys[cur], pc_alt, n_act, 0, 2 * w_r + 5 + gbits, p->sort, &alt, prof, s, false, CX_K_REFINE_SORT)));
            CX_CUDA(cudaMemcpyAsync(d_heads[1 - hc], d_heads[hc], (n_words + 1) * 4, cudaMemcpyDeviceToDevice, s));
            {
                ScopedLaunch sl(prof, CX_K_REFINE_WRITE, nb / 8 + n_act * (8 + 4 + 4 * sizeof(IdT) + 1), s);
                CX_CUDA(launch_refine_writeback<IdT>(R, alt ? d_keys[cur] : kc, alt ? pc_alt : pc, reinterpret_cast<IdT*>(alt ? kc : d_keys[cur]),
                                                     d_heads[hc], d_word_counts, nb, n_act, w_r, ids, d_heads[1 - hc], dst, s));
                prof->launches[CX_K_REFINE_WRITE] += 1;   // gather + write-back
            }
            hc = 1 - hc;                                  // the head bits with this round's new groups
            p->stats.refine_elements += n_act;
            depth += w_r;
            ++rounds;
            if (cap > 1) {
                CX_CUDA(cudaMemcpyAsync(d_heads[1 - hc], d_heads[hc], (n_words + 1) * 4, cudaMemcpyDeviceToDevice, s));
                ScopedLaunch sl(prof, CX_K_FINISH_BLOCK, nb / 4, s);
                CX_CUDA(launch_finish_later<IdT>(R, d_heads[hc], d_heads[1 - hc], ids, nb, depth, cap, dst, d_done, p->n_sms, s));
                hc = 1 - hc;
            }
        }
        p->stats.small_group_elems = p->h_scalars[1];
        p->stats.compare_ops = p->h_scalars[3];
        p->stats.finish_rounds = p->h_scalars[4];
        p->stats.refine_elements += p->h_scalars[1] - local_before;
        if (rounds > p->stats.refine_rounds) p->stats.refine_rounds = rounds;

        // NEXT-4: two symbols per byte.  Batches come in output order, so a byte shared by two batches is completed by the
        // later one (its high nibble is the earlier batch's last symbol, kept in a device word).
        const uint8_t* copy_src = dst;
        uint64_t copy_at = B.out_offset, copy_bytes = nb;
        if (sh.pack_out) {
            uint32_t* d_carry = reinterpret_cast<uint32_t*>(d_scalars + 7);
            uint8_t* packed = sh.host_out ? ws + L.pstage[st] : out + B.out_offset / 2;
            ScopedLaunch sl(prof, CX_K_PACK, nb + nb / 2, s);
            CX_CUDA(launch_pack_symbols(dst, nb, B.out_offset, packed, d_carry, s));
            prof->launches[CX_K_PACK] += 1;
            copy_src = packed, copy_at = B.out_offset / 2, copy_bytes = (nb + (B.out_offset & 1) + 1) / 2;
        }
        if (sh.host_out) {
            // a9: copy the staged batch on the side stream while the next batch computes
            CX_CUDA(cudaEventRecord(p->emit_done, s));
            CX_CUDA(cudaStreamWaitEvent(p->copy_stream, p->emit_done, 0));
            CX_CUDA(cudaMemcpyAsync(out + copy_at, copy_src, copy_bytes, cudaMemcpyDeviceToHost, p->copy_stream));
            CX_CUDA(cudaEventRecord(p->stage_free[st], p->copy_stream));
            p->stage_busy[st] = true;
        }
    }
    if (sh.host_out) {
        CX_CUDA(cudaStreamSynchronize(p->copy_stream));
        p->stage_busy[0] = p->stage_busy[1] = false;
    }
    if (prof->timing) {
        CX_CUDA(cudaStreamSynchronize(s));
        prof->resolve();
    }
    p->stats.kernel_launches = prof->total_launches();
    return CX_OK;
}

}  // namespace

extern "C" int cx_bwt_build(cx_bwt_plan_t* p, const uint64_t* packed_reads, const uint64_t* read_offsets, uint64_t n_reads,
                            uint8_t* out_bwt, cx_stream_t stream) {
    if (!p) return CX_ERR_ARG;
    p->prof.reset();
    memset(&p->stats, 0, sizeof(p->stats));
    p->h_scalars[0] = p->h_scalars[1] = p->h_scalars[3] = p->h_scalars[4] = p->h_scalars[5] = p->h_scalars[6] = 0;
    if (n_reads == 0) return CX_OK;
    if (!read_offsets || !out_bwt || n_reads > p->sh.max_reads) return CX_ERR_ARG;
    if (!packed_reads && p->sh.max_bases) return CX_ERR_ARG;
    const bool key32 = first_key_bits(p->sh.w) <= 32;
    if (p->sh.id_bytes == 4)
        return key32 ? build_impl<uint32_t, uint32_t>(p, packed_reads, read_offsets, n_reads, out_bwt, stream)
                     : build_impl<uint64_t, uint32_t>(p, packed_reads, read_offsets, n_reads, out_bwt, stream);
    return key32 ? build_impl<uint32_t, uint64_t>(p, packed_reads, read_offsets, n_reads, out_bwt, stream)
                 : build_impl<uint64_t, uint64_t>(p, packed_reads, read_offsets, n_reads, out_bwt, stream);
}

// ---------------------------------------------------------------------------------------------
// the sorter on its own
// ---------------------------------------------------------------------------------------------
extern "C" int cx_sort_pairs_workspace_bytes(uint64_t n, uint64_t* bytes_out) {
    if (!bytes_out) return CX_ERR_ARG;
    *bytes_out = sort_workspace_bytes(n);
    return CX_OK;
}

extern "C" int cx_sort_pairs(uint64_t* keys, void* vals, uint64_t* keys_alt, void* vals_alt, uint64_t n, uint32_t val_bytes,
                             uint32_t begin_bit, uint32_t end_bit, void* workspace_dev, uint64_t workspace_bytes, int* result_in_alt,
                             cx_stream_t stream) {
    if (!result_in_alt || (val_bytes != 4 && val_bytes != 8) || begin_bit > end_bit || end_bit > 64 || end_bit - begin_bit > 64)
        return CX_ERR_ARG;
    *result_in_alt = 0;
    if (n == 0) return CX_OK;
    if (!keys || !vals || !keys_alt || !vals_alt || !workspace_dev) return CX_ERR_ARG;
    if (workspace_bytes < sort_workspace_bytes(n)) return CX_ERR_WORKSPACE;
    // stateless call: start the tile state from scratch
    CX_CUDA(cudaMemsetAsync(workspace_dev, 0, sort_workspace_bytes(n), stream));
    SortWorkspace ws;
    sort_workspace_carve(ws, workspace_dev, n);
    if (val_bytes == 4)
        CX_CUDA((sort_pairs<uint64_t, uint32_t>(keys, (uint32_t*)vals, keys_alt, (uint32_t*)vals_alt, n, begin_bit, end_bit, ws,
                                                result_in_alt, nullptr, stream)));
    else
        CX_CUDA((sort_pairs<uint64_t, uint64_t>(keys, (uint64_t*)vals, keys_alt, (uint64_t*)vals_alt, n, begin_bit, end_bit, ws,
                                                result_in_alt, nullptr, stream)));
    return CX_OK;
}
