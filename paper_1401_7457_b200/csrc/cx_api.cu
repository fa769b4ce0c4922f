// cx_api.cu -- the C ABI of include/cx_bwt.h: plan (workspace carving, m1), build (Figure 2 of the
// paper, as a sequence of kernel launches), statistics and error text.
#include <stdio.h>
#include <string.h>

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

struct Batch {
    uint32_t bucket_lo, bucket_hi;
    uint64_t count, out_offset;
};

// Byte offsets of every region of the workspace for a given m1.
struct Layout {
    uint64_t info, hist, tile_first, tile_count, tile_sums, scalars;
    uint64_t keys[2], ids[3], pos, heads[2], word_counts, word_sums, sort, stage[2];
    uint64_t total;
};

struct Shape {
    uint64_t max_reads, max_bases, max_suffixes, max_tiles;
    uint32_t ell, w, cap, id_bytes, pos_bits;
    uint64_t n_buckets;
    bool host_out;
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
    L.tile_count = take((sh.max_tiles + 1) * 8 * (sh.max_suffixes <= m1 ? 1 : kCountGroup));
    L.tile_sums = take((scan_block_count(sh.max_tiles + 1) + 1) * 8);
    L.scalars = take(64);
    for (int i = 0; i < 2; ++i) L.keys[i] = take(m1 * 8);
    for (int i = 0; i < 3; ++i) L.ids[i] = take(m1 * sh.id_bytes);
    L.pos = take(m1 * 4);
    uint64_t words = (m1 + 31) / 32 + 2;
    for (int i = 0; i < 2; ++i) L.heads[i] = take(words * 4);
    L.word_counts = take(words * 8);
    L.word_sums = take((scan_block_count(words) + 1) * 8);
    L.sort = take(sort_workspace_bytes(m1));
    for (int i = 0; i < 2; ++i) L.stage[i] = take(sh.host_out ? m1 : 0);
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
    if (sh.cap > (uint32_t)kLocalGroupCap) sh.cap = kLocalGroupCap;
    if (max_reads >= 0xFFFFFFFFull) return CX_ERR_ARG;   // read indices travel as 32 bits in the tile table
    sh.max_reads = max_reads;
    sh.max_bases = max_bases;
    sh.max_suffixes = max_reads + max_bases;
    sh.max_tiles = (sh.max_suffixes + kListTile - 1) / kListTile;
    uint64_t max_len = o->max_read_len ? o->max_read_len : max_bases;
    if (max_len > max_bases) max_len = max_bases;
    sh.pos_bits = bit_width64(max_len);
    uint32_t read_bits = bit_width64(max_reads ? max_reads - 1 : 0);
    if (sh.pos_bits + read_bits > 64) return CX_ERR_ARG;
    sh.id_bytes = sh.pos_bits + read_bits <= 32 ? 4 : 8;
    sh.n_buckets = (1ull << (2 * sh.ell)) * (sh.ell + 1);
    sh.host_out = o->out_is_host_pinned != 0;
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
    BuildInfo* h_info;
    uint64_t* h_scalars;
    uint64_t* h_hist;
    std::vector<Batch> batches;
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
    // whole collection, so that random collisions are rare and tie groups are the genuinely shared substrings.
    // 14 bases + a 4-bit length is the most a 32-bit key holds: half the bytes per radix pass and 4 passes; it
    // still wins at 1e9 suffixes (C3: 86 ms against 115 ms with w = 29).  Beyond 2^30 suffixes the key is
    // 64-bit with w = ceil(log4 N) + 1 bases (6 passes at 6e9 .. 1e11 suffixes instead of 8).
    if (sh.w == 0) {
        if (sh.max_suffixes <= (1ull << 30)) {
            sh.w = 14;
        } else {
            uint32_t log4 = (bit_width64(sh.max_suffixes - 1) + 1) / 2;
            sh.w = log4 + 1 > 29 ? 29 : log4 + 1;
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
    p->copy_stream = nullptr;
    p->emit_done = p->stage_free[0] = p->stage_free[1] = nullptr;

    size_t host_bytes = sizeof(BuildInfo) + 64 + sh.n_buckets * 8;
    cudaError_t e = cudaMallocHost((void**)&p->h_pinned, host_bytes);
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

extern "C" const char* cx_strerror(int code) {
    switch (code) {
    case CX_OK: return "ok";
    case CX_ERR_ARG: return "invalid argument (null pointer, bad option, size above the plan's maximum, or bad offsets)";
    case CX_ERR_BAD_BASE: return "input contains a byte outside ACGT";
    case CX_ERR_WORKSPACE: return "workspace too small";
    case CX_ERR_BUCKET_TOO_LARGE: return "one prefix partition exceeds the batch limit m1 (recursive refinement not built)";
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

// Fig. 2 steps 2 and 3(b) ("merging a consecutive range of partitions"):
// greedy ranges of consecutive partitions with total size <= m1.
int plan_batches(cx_bwt_plan_t* p, uint64_t N) {
    p->batches.clear();
    const uint64_t nb = p->sh.n_buckets;
    uint64_t largest = 0, out = 0;
    Batch cur{0, 0, 0, 0};
    bool open = false;
    for (uint64_t b = 0; b < nb; ++b) {
        uint64_t c = p->h_hist[b];
        if (c == 0) continue;
        if (c > largest) largest = c;
        if (c > p->m1) {
            p->stats.largest_bucket = largest;
            return CX_ERR_BUCKET_TOO_LARGE;
        }
        if (open && cur.count + c > p->m1) {
            p->batches.push_back(cur);
            out += cur.count;
            open = false;
        }
        if (!open) {
            cur = Batch{(uint32_t)b, (uint32_t)b, 0, out};
            open = true;
        }
        cur.bucket_hi = (uint32_t)b;
        cur.count += c;
    }
    if (open) {
        p->batches.push_back(cur);
        out += cur.count;
    }
    p->stats.largest_bucket = largest;
    return out == N ? CX_OK : CX_ERR_CUDA;   // a mismatch means the histogram kernel misbehaved
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
    IdT* d_ids[3] = {reinterpret_cast<IdT*>(ws + L.ids[0]), reinterpret_cast<IdT*>(ws + L.ids[1]), reinterpret_cast<IdT*>(ws + L.ids[2])};
    uint32_t* d_pos = reinterpret_cast<uint32_t*>(ws + L.pos);
    uint32_t* d_heads[2] = {reinterpret_cast<uint32_t*>(ws + L.heads[0]), reinterpret_cast<uint32_t*>(ws + L.heads[1])};
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
    const bool fused_scan = sh.max_suffixes <= p->m1;
    const uint32_t w = sh.w;
    const uint32_t key_bits = 2 * w + key_len_bits(w);
    const uint32_t n_passes = (key_bits + kRadixBits - 1) / kRadixBits;
    KeyT* d_keys1[2] = {reinterpret_cast<KeyT*>(d_keys[0]), reinterpret_cast<KeyT*>(d_keys[1])};   // first-round keys
    // 32-bit key and 32-bit id: one 64-bit word per suffix (key << 32 | id), sorted keys-only over its upper half
    const bool pack_kv = sizeof(KeyT) == 4 && sizeof(IdT) == 4;
    if (fused_scan) {
        CX_CUDA(cudaMemsetAsync(p->sort.hist, 0, (size_t)n_passes * kRadix * sizeof(uint64_t), s));
        ScopedLaunch sl(prof, CX_K_LIST, 0, s);
        CX_CUDA((launch_list_write<KeyT, IdT>(R, d_info, d_tile_first, sh.ell, w, 0, 0, nullptr, d_keys1[0], d_ids[0], sh.max_tiles, n_passes,
                                              p->sort.hist, p->n_sms, pack_kv, d_hist, p->m1, s)));
    } else {
        ScopedLaunch sl(prof, CX_K_HIST, 0, s);
        CX_CUDA(launch_bucket_hist(R, d_info, d_tile_first, sh.ell, d_hist, sh.max_tiles, p->n_sms, s));
    }
    CX_CUDA(cudaMemcpyAsync(p->h_info, d_info, sizeof(BuildInfo), cudaMemcpyDeviceToHost, s));
    CX_CUDA(cudaMemcpyAsync(p->h_hist, d_hist, sh.n_buckets * 8, cudaMemcpyDeviceToHost, s));
    CX_CUDA(cudaStreamSynchronize(s));
    const BuildInfo info = *p->h_info;
    if (info.bad_offsets || info.total_bases > sh.max_bases || (info.max_len >> sh.pos_bits) != 0) return CX_ERR_ARG;
    const uint64_t N = info.n_suffixes;
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

    // ---- steps 2, 3(b): batch ranges -----------------------------------------------------------
    int rc = plan_batches(p, N);
    if (rc) return rc;
    p->stats.n_batches = (uint32_t)p->batches.size();
    const uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    const bool single = p->batches.size() == 1;
    if (fused_scan && !single) return CX_ERR_CUDA;   // cannot happen: N <= max_suffixes <= m1
    p->stats.sort_passes = (key_bits + kRadixBits - 1) / kRadixBits;

    for (size_t bi = 0; bi < p->batches.size(); ++bi) {
        const Batch& B = p->batches[bi];
        const uint64_t nb = B.count;
        // ---- step 3(a) + 3(c)i: list the batch's suffixes with their first keys ----------------
        if (!fused_scan) CX_CUDA(cudaMemsetAsync(p->sort.hist, 0, (size_t)n_passes * kRadix * sizeof(uint64_t), s));
        if (fused_scan) {
            // listed before the partition sizes were read back
        } else if (single) {
            ScopedLaunch sl(prof, CX_K_LIST, info.total_bases / 4 + (n_reads + 1) * 8 + nb * (sizeof(KeyT) + sizeof(IdT)), s);
            CX_CUDA((launch_list_write<KeyT, IdT>(R, d_info, d_tile_first, sh.ell, w, B.bucket_lo, B.bucket_hi, nullptr, d_keys1[0],
                                                  d_ids[0], n_tiles, n_passes, p->sort.hist, p->n_sms, pack_kv, nullptr, ~0ull, s)));
        } else {
            const uint64_t col_stride = sh.max_tiles + 1;
            if (bi % kCountGroup == 0) {   // one scan counts this batch and the next seven
                CountRanges cr{};
                for (size_t q = bi; q < p->batches.size() && cr.n < (uint32_t)kCountGroup; ++q) cr.first[cr.n++] = p->batches[q].bucket_lo;
                cr.first[cr.n] = p->batches[bi + cr.n - 1].bucket_hi + 1;
                ScopedLaunch sl(prof, CX_K_LIST, info.total_bases / 4 + (n_reads + 1) * 8 + n_tiles * 8 * cr.n, s);
                CX_CUDA(launch_list_count(R, d_info, d_tile_first, sh.ell, cr, d_tile_count, col_stride, n_tiles, s));
            }
            uint64_t* d_col = d_tile_count + (bi % kCountGroup) * col_stride;
            {
                ScopedLaunch sl(prof, CX_K_LIST, n_tiles * 16, s);
                CX_CUDA(launch_scan_u64(d_col, n_tiles, d_tile_sums, d_scalars + 2, s));
            }
            prof->launches[CX_K_LIST] += 2;   // the scan is three kernels
            ScopedLaunch sl(prof, CX_K_LIST, info.total_bases / 4 + (n_reads + 1) * 8 + nb * (sizeof(KeyT) + sizeof(IdT)), s);
            CX_CUDA((launch_list_write<KeyT, IdT>(R, d_info, d_tile_first, sh.ell, w, B.bucket_lo, B.bucket_hi, d_col,
                                                  d_keys1[0], d_ids[0], n_tiles, n_passes, p->sort.hist, p->n_sms, pack_kv, nullptr, ~0ull, s)));
        }
        // ---- step 3(c)ii: sort (first w symbols) ------------------------------------------------
        int in_alt = 0;
        if (pack_kv)
            CX_CUDA((sort_pairs<uint64_t, NoVal>(d_keys[0], nullptr, d_keys[1], nullptr, nb, 32, 32 + key_bits, p->sort, &in_alt, prof, s, true)));
        else
            CX_CUDA((sort_pairs<KeyT, IdT>(d_keys1[0], d_ids[0], d_keys1[1], d_ids[1], nb, 0, key_bits, p->sort, &in_alt, prof, s, true)));
        const int cur = in_alt;
        IdT* ids = pack_kv ? d_ids[0] : d_ids[cur];
        // a9: with pinned-host output the batch is emitted into a staging buffer of the workspace
        const int st = (int)(bi & 1);
        uint8_t* dst = sh.host_out ? ws + L.stage[st] : out + B.out_offset;
        if (sh.host_out && p->stage_busy[st]) CX_CUDA(cudaStreamWaitEvent(s, p->stage_free[st], 0));
        // ---- steps 3(c)ii-iii fused: head flags, in-block tie refinement, emit ----------------------
        const uint64_t n_words = (nb + 31) >> 5;
        int hc = 0;
        unsigned long long* d_done = reinterpret_cast<unsigned long long*>(d_scalars + 1);
        CX_CUDA(cudaMemsetAsync(d_heads[0], 0, (n_words + 1) * 4, s));
        {
            ScopedLaunch sl(prof, CX_K_FINISH, nb * (sizeof(KeyT) + sizeof(IdT) + 1) + nb / 8, s);
            CX_CUDA((launch_finish_first<KeyT, IdT>(R, d_keys1[cur], w, d_heads[0], ids, nb, sh.cap, dst, d_done, pack_kv, s)));
        }
        // ---- what is still tied goes through global rounds: re-key, sort, write back ------------------
        uint32_t depth = w, rounds = 0;
        uint64_t local_before = p->h_scalars[1];
        while (true) {
            {
                ScopedLaunch sl(prof, CX_K_REFINE_SCAN, n_words * 12, s);
                CX_CUDA(launch_active_count(d_heads[hc], nb, d_word_counts, s));
            }
            {
                ScopedLaunch sl(prof, CX_K_REFINE_SCAN, n_words * 16, s);
                CX_CUDA(launch_scan_u64(d_word_counts, n_words, d_word_sums, d_scalars, s));
            }
            prof->launches[CX_K_REFINE_SCAN] += 2;
            CX_CUDA(cudaMemcpyAsync(p->h_scalars, d_scalars, 32, cudaMemcpyDeviceToHost, s));
            CX_CUDA(cudaStreamSynchronize(s));
            const uint64_t n_act = p->h_scalars[0] & 0xffffffffull;
            const uint64_t n_groups = p->h_scalars[0] >> 32;
            if (n_act == 0) break;
            // key = [group ordinal][w_r bases][length]: as deep a window as the ordinal leaves room for
            const uint32_t gbits = n_groups > 1 ? bit_width64(n_groups - 1) : 0;
            uint32_t w_r = (59 - gbits) / 2;
            if (w_r > 29) w_r = 29;
            uint64_t* kc = d_keys[1 - cur];
            IdT* ic = pack_kv ? d_ids[1] : d_ids[1 - cur];
            {
                ScopedLaunch sl(prof, CX_K_REFINE_KEY, nb / 8 + n_act * (2 * sizeof(IdT) + 8 + 8 + 4), s);
                CX_CUDA(launch_refine_rekey<IdT>(R, d_heads[hc], d_word_counts, ids, nb, depth, w_r, kc, ic, d_pos, s));
            }
            int alt = 0;
            CX_CUDA((sort_pairs<uint64_t, IdT>(kc, ic, d_keys[cur], d_ids[2], n_act, 0, 2 * w_r + 5 + gbits, p->sort, &alt, prof, s)));
            {
                ScopedLaunch sl(prof, CX_K_REFINE_WRITE, n_act * (8 + 2 * sizeof(IdT) + 4 + 1), s);
                CX_CUDA(launch_refine_writeback<IdT>(R, alt ? d_keys[cur] : kc, alt ? d_ids[2] : ic, d_pos, n_act, w_r, ids, d_heads[hc],
                                                     dst, s));
            }
            p->stats.refine_elements += n_act;
            depth += w_r;
            ++rounds;
            if (sh.cap > 1) {
                CX_CUDA(cudaMemcpyAsync(d_heads[1 - hc], d_heads[hc], (n_words + 1) * 4, cudaMemcpyDeviceToDevice, s));
                ScopedLaunch sl(prof, CX_K_FINISH, nb / 4, s);
                CX_CUDA(launch_finish_later<IdT>(R, d_heads[hc], d_heads[1 - hc], ids, nb, depth, sh.cap, dst, d_done, s));
                hc = 1 - hc;
            }
        }
        p->stats.small_group_elems = p->h_scalars[1];
        p->stats.compare_ops = p->h_scalars[3];
        p->stats.refine_elements += p->h_scalars[1] - local_before;
        if (rounds > p->stats.refine_rounds) p->stats.refine_rounds = rounds;

        if (sh.host_out) {
            // a9: copy the staged batch on the side stream while the next batch computes
            CX_CUDA(cudaEventRecord(p->emit_done, s));
            CX_CUDA(cudaStreamWaitEvent(p->copy_stream, p->emit_done, 0));
            CX_CUDA(cudaMemcpyAsync(out + B.out_offset, dst, nb, cudaMemcpyDeviceToHost, p->copy_stream));
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
    p->h_scalars[0] = p->h_scalars[1] = p->h_scalars[3] = 0;
    if (n_reads == 0) return CX_OK;
    if (!read_offsets || !out_bwt || n_reads > p->sh.max_reads) return CX_ERR_ARG;
    if (!packed_reads && p->sh.max_bases) return CX_ERR_ARG;
    const bool key32 = 2 * p->sh.w + key_len_bits(p->sh.w) <= 32;
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
