// cx_internal.cuh -- shared declarations of libcxbwt (sm_100a only).  Not part of the C ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "cx_bwt.h"

namespace cx {

// ---------------------------------------------------------------------------------------------
// geometry shared by host and device
// ---------------------------------------------------------------------------------------------
constexpr int kListThreads = 256;
constexpr int kListItems = 8;
constexpr int kListTile = kListThreads * kListItems;   // suffix slots per listing / histogram tile

// scans with one read per thread (collections of equal-length reads): read lengths they take
constexpr int kReadMaxLen = 127;   // L + 1 <= 128 slots per read: a 128-bit mask per thread
constexpr int kReadMinLen = 16;    // (below, the tile tables sized per 2048 slots would be too small)

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

// onesweep tile shapes (threads x items); one per value width so that registers/smem stay balanced
constexpr int kSortThreads = 256;
struct NoVal {};   // value type of a keys-only sort (the 32-bit id rides in the low half of a 64-bit key word)
template <typename KeyT, typename ValT> struct SortShape {
    // pairs staged per tile: 8-byte pairs 8192 (64 KB), 12-byte pairs 6144 (72 KB), 16-byte pairs 5120 (80 KB); 2 blocks per SM
    static constexpr int pair_bytes = sizeof(KeyT) + (sizeof(ValT) >= 4 ? sizeof(ValT) : 0);
    static constexpr int items = pair_bytes >= 16 ? 10 : pair_bytes >= 12 ? 12 : 16;
};
constexpr int kSortTileMin = 2560;   // smallest tile: sizes the tile-state array

// tile-state word of the decoupled look-back: [epoch:8][flag:2][count:54]
constexpr uint64_t kStatusValueMask = (1ull << 54) - 1;
constexpr uint32_t kFlagAggregate = 1, kFlagInclusive = 2;

// in-block refinement
constexpr int kLocalThreads = 256;
// Sorted positions owned by one block.  The kernel is bound by random gathers, and what limits those is the L1 left
// beside the shared-memory carve-out: 512 + 256 positions x 5 blocks/SM fit the 164 KB carve-out (92 KB of L1);
// 768 + 256 needs 228 KB (28 KB of L1) and runs 1.5x slower on collections larger than L2.  Measured finish times,
// configs[1] / configs[2] / configs[3] x 0.25: 512 -> 5.38 / 35.7 / 116.6 ms; 768 -> 5.47 / 59.3 / 185.2 ms;
// 640 with 224 threads (196 KB carve-out) -> 5.31 / 39.8 / 130.6 ms.
constexpr int kLocalTile = 512;
constexpr int kLocalBlocksPerSM = 4;
constexpr int kLocalGroupCap = 256;      // largest tie group the in-block path accepts

// Facts about one build, produced by the prep kernel and read by later kernels and by the host.
struct BuildInfo {
    uint64_t total_bases;
    uint64_t n_suffixes;
    uint64_t max_len;
    uint64_t first_len;
    uint32_t bad_offsets;   // bit 0: offsets[0] != 0 or a decreasing pair; bit 1: more bases than the plan allows
    uint32_t nonuniform;    // some read differs in length from read 0
};

// The read collection as kernels see it.
struct Reads {
    const uint64_t* packed;    // 2 bit/base, MSB-first in each word
    const uint64_t* offsets;   // n_reads + 1
    uint64_t n_reads;
    uint64_t n_words;          // valid words of `packed`; loads at or past it read as zero
    uint64_t uniform_len;      // length of every read when `uniform`
    uint32_t pos_bits;         // id = (read << pos_bits) | pos
    uint32_t uniform;          // 1: all reads have the same length, offsets need not be gathered
};

// A region of the suffix space: the suffixes whose first `depth` bases spell `prefix`.  depth = 0 is the whole
// collection.  An l-prefix partition that is larger than a batch is partitioned again by its NEXT l characters,
// recursively (Fig. 2 step 1): the scans then work inside the region of that partition.
struct Region {
    const uint64_t* prefix;   // DEVICE: depth bases, 2 bit/base, MSB-first in each word
    uint32_t depth;
};

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31; }
__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}
__device__ __forceinline__ uint64_t ld_relaxed_u64(const uint64_t* p) {
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u64(uint64_t* p, uint64_t v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// 32 bases starting at base position b, first base in the two most significant bits.
// Words at or past n_words read as zero (A-padding; callers mask by the true remaining length).
__device__ __forceinline__ uint64_t load_window(const uint64_t* __restrict__ packed, uint64_t n_words, uint64_t b) {
    uint64_t wi = b >> 5;
    uint32_t sh = (uint32_t)(b & 31) * 2;
    uint64_t w0 = wi < n_words ? __ldg(packed + wi) : 0ull;
    if (sh == 0) return w0;
    uint64_t w1 = wi + 1 < n_words ? __ldg(packed + wi + 1) : 0ull;
    return (w0 << sh) | (w1 >> (64 - sh));
}

// Order-preserving keys of a window of w bases (reading A3 of PAPER.md:99).
//
// first_key (the first sort of a batch): the RANK of the suffix's first min(rem, w) symbols, end-marker included if it falls
// inside the window, among all strings of at most w bases over $ < A < C < G < T -- then one bit: 1 = the suffix has at least
// w bases.  With T(k) = (4^(w-k+1) - 1) / 3 strings below a node at depth k of that trie, the rank of c_0 .. c_(r-1) is
// sum_i (1 + c_i T(i+1)) = r + (4 B - S) / 3, B = the bases as a 2w-bit number (A-padded), S = the sum of their codes
// (4^k = 1 mod 3 makes the division exact).  Different strings get different keys in their true order; equal keys with the
// bit clear are IDENTICAL strings (final at once), equal keys with the bit set share their first w bases.
// The rank is below 4^(w+1) / 3: 15 bases and the bit fill a 32-bit key, 19 bases a 40-bit one (five 8-bit radix passes).
//
// make_key (the global path's re-keying): the bases, A-padded, then min(rem, w) in the low len_bits bits; a value < w in that
// field means the end-marker falls inside this window, and equal keys then mean identical strings.
__host__ __device__ __forceinline__ uint32_t first_key_bits(uint32_t w) {
    uint32_t bits = 0;
    for (uint64_t top = ((1ull << (2 * w + 2)) - 4) / 3; top; top >>= 1) ++bits;   // the largest rank, (4^(w+1) - 4) / 3
    return bits + 1;
}
__device__ __forceinline__ uint64_t first_key(uint64_t window, uint64_t rem, uint32_t w) {
    const uint32_t r = rem < (uint64_t)w ? (uint32_t)rem : w;
    const uint64_t B = r ? ((window >> (64 - 2 * r)) << (2 * (w - r))) : 0ull;
    const uint64_t S = (uint64_t)__popcll((long long)(B & 0x5555555555555555ull)) + 2ull * (uint64_t)__popcll((long long)(B & 0xAAAAAAAAAAAAAAAAull));
    const uint64_t rank = r + (4 * B - S) * 0xAAAAAAAAAAAAAAABull;   // exact division by 3 (the multiplier is 3^-1 mod 2^64)
    return (rank << 1) | (uint64_t)(r == w);
}
// the same for w <= 15 in 32-bit arithmetic (the listing scans are bound by instruction issue); window = the next 32 bases
__device__ __forceinline__ uint32_t first_key32(uint64_t window, uint32_t rem, uint32_t w) {
    const uint32_t r = rem < w ? rem : w;
    const uint32_t top = (uint32_t)(window >> 34);                       // the first 15 bases, right-aligned
    const uint32_t B = r ? (top >> (30 - 2 * r)) << (2 * (w - r)) : 0u;
    const uint32_t S = (uint32_t)__popc(B & 0x55555555u) + 2u * (uint32_t)__popc(B & 0xAAAAAAAAu);
    const uint32_t rank = r + (4u * B - S) * 0xAAAAAAABu;                // exact division by 3 (3^-1 mod 2^32); 4 B < 2^32 for w <= 15
    return (rank << 1) | (uint32_t)(r == w);
}
template <typename KeyT>
__device__ __forceinline__ KeyT first_key_as(uint64_t window, uint64_t rem, uint32_t w) {
    if constexpr (sizeof(KeyT) == 4) return first_key32(window, (uint32_t)(rem < 64 ? rem : 64), w);
    else return first_key(window, rem, w);
}
__host__ __device__ __forceinline__ uint32_t key_len_bits(uint32_t w) { return w >= 16 ? 5u : w >= 8 ? 4u : w >= 4 ? 3u : w >= 2 ? 2u : 1u; }
__device__ __forceinline__ uint64_t make_key(uint64_t window, uint64_t rem, uint32_t w, uint32_t len_bits = 5) {
    uint32_t r = rem < (uint64_t)w ? (uint32_t)rem : w;
    uint64_t bases = r ? ((window >> (64 - 2 * r)) << (2 * (w - r))) : 0ull;
    return (bases << len_bits) | r;
}

// Is the suffix that starts at base index b, with `rem` bases left and `window` = its next 32 bases, inside the region?
// If so, (window, rem) are advanced to describe the suffix at the region's depth.
__device__ __forceinline__ bool enter_region(const uint64_t* __restrict__ packed, uint64_t n_words, const Region& g, uint64_t b,
                                             uint64_t& window, uint32_t& rem) {
    if (g.depth == 0) return true;
    if (rem < g.depth) return false;
    for (uint32_t j = 0; j * 32 < g.depth; ++j) {
        const uint64_t wj = j == 0 ? window : load_window(packed, n_words, b + 32ull * j);
        const uint32_t nb = g.depth - j * 32 < 32 ? g.depth - j * 32 : 32;
        const uint64_t mask = nb == 32 ? ~0ull : ~0ull << (64 - 2 * nb);
        if ((wj ^ __ldg(g.prefix + j)) & mask) return false;
    }
    window = load_window(packed, n_words, b + g.depth);
    rem -= g.depth;
    return true;
}

template <typename IdT>
__device__ __forceinline__ IdT make_id(uint64_t read, uint64_t pos, uint32_t pos_bits) {
    return (IdT)((read << pos_bits) | pos);
}

#endif  // __CUDACC__

// ---------------------------------------------------------------------------------------------
// host-side launchers (one translation unit per group of kernels)
// ---------------------------------------------------------------------------------------------
struct Launch;   // profiling hook, defined in cx_api.cu

// SMs of the current device (grids of the persistent kernels are sized from it; nothing assumes 148)
inline int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 1;
    return n;
}

// cx_pack.cu
// NEXT-4: FASTA text -> bases + read offsets (cx_fasta.cu)
uint64_t fasta_workspace_bytes(uint64_t n_bytes);
cudaError_t launch_fasta_parse(const uint8_t* text, uint64_t n, uint8_t* bases_out, uint64_t* offsets_out, uint64_t max_reads, uint64_t* counts,
                               unsigned char* ws, cudaStream_t s);
cudaError_t launch_pack(const uint8_t* ascii, uint64_t total_bases, uint64_t* packed, uint32_t* status, cudaStream_t s);
uint32_t* pack_fallback_status();
// NEXT-4: n symbols of BWT positions [out_offset, out_offset + n) -> 4-bit codes; packed[0] = byte out_offset / 2 of the output;
// *carry holds the code of the symbol before the piece (and, afterwards, of the piece's last symbol)
cudaError_t launch_pack_symbols(const uint8_t* sym, uint64_t n, uint64_t out_offset, uint8_t* packed, uint32_t* carry, cudaStream_t s);

// cx_scan_reads.cu
cudaError_t launch_prep(const uint64_t* offsets, uint64_t n_reads, uint64_t max_bases, BuildInfo* info, cudaStream_t s);
cudaError_t launch_tile_table(const uint64_t* offsets, uint64_t n_reads, const BuildInfo* info, uint32_t* tile_first_read,
                              uint64_t max_tiles, cudaStream_t s);
cudaError_t launch_bucket_hist(const Reads& R, const BuildInfo* info, const uint32_t* tile_first_read, uint32_t ell, const Region& region,
                               uint64_t* hist, uint64_t max_tiles, int n_sms, cudaStream_t s);
// tiles of the multi-batch scans (count, scan of a column, select) of `region`: their size depends on the collection
// (reads of one length outside a region: 8192 slots; otherwise kListTile); all three steps must be given this count
uint64_t list_scan_tiles(const Reads& R, const Region& region, uint64_t n_suffixes);
// count, per tile, the suffixes of up to kCountGroup consecutive batches in one scan; batch j owns partitions
// [first[j], first[j + 1]); tile_count[j * col_stride + tile]
constexpr int kCountGroup = 8;
struct CountRanges {
    uint32_t n;
    uint32_t first[kCountGroup + 1];
};
cudaError_t launch_list_count(const Reads& R, const BuildInfo* info, const uint32_t* tile_first_read, uint32_t ell, const Region& region,
                              const CountRanges& ranges, uint64_t* tile_count, uint64_t col_stride, uint64_t n_tiles, cudaStream_t s);
// write (key, id) of those suffixes in (read, pos) order; tile_base == nullptr means "every suffix, index = slot".
// Also accumulates the digit counts of the n_passes radix passes over key bits [0, 8 * n_passes) into digit_hist
// (zeroed by the caller), which is what sort_pairs(..., hist_ready = true) expects.
template <typename KeyT, typename IdT>
cudaError_t launch_list_write(const Reads& R, const BuildInfo* info, const uint32_t* tile_first_read, uint32_t ell, uint32_t w,
                              uint32_t bucket_lo, uint32_t bucket_hi, const uint64_t* tile_base, KeyT* keys, IdT* ids,
                              uint64_t n_tiles, uint32_t n_passes, uint64_t* digit_hist, int n_sms, bool packed, uint64_t* bucket_hist,
                              uint64_t max_n, const Region& region, uint64_t ord_lo, uint64_t ord_hi, cudaStream_t s, uint32_t split = 0);
// split != 0 (select scans with 64-bit keys and ids only): a pair is (key << split | id >> 32) in `keys` and (uint32_t)id in a uint32 array at `ids`

// cx_onesweep.cu
struct SortWorkspace {
    uint64_t* hist = nullptr;     // [8][256] digit counts, then exclusive bin bases in place
    uint64_t* status = nullptr;   // [max_tiles][256] tile state
    uint32_t* ticket = nullptr;   // dynamic tile counter (monotone across launches)
    uint64_t max_tiles = 0;
    uint32_t epoch = 0;           // host-side: last epoch used (1..255)
    uint32_t ticket_base = 0;     // host-side: tickets handed out so far
};
size_t sort_workspace_bytes(uint64_t n);
// carve a zeroed region of sort_workspace_bytes(n) bytes
void sort_workspace_carve(SortWorkspace& ws, void* mem, uint64_t n);
// Sorts by key bits [begin_bit, end_bit).  *result_in_alt = 1 if the result is in the alt buffers.
// hist_ready: ws.hist already holds the digit counts of every pass (the list kernel built them); begin_bit must be 0.
template <typename KeyT, typename ValT>
cudaError_t sort_pairs(KeyT* keys, ValT* vals, KeyT* keys_alt, ValT* vals_alt, uint64_t n, uint32_t begin_bit,
                       uint32_t end_bit, SortWorkspace& ws, int* result_in_alt, Launch* prof, cudaStream_t s, bool hist_ready = false,
                       int pass_class = CX_K_SORT_PASS);

// cx_refine.cu
// word-level counts of active elements / active heads, packed (heads << 32 | elements)
cudaError_t launch_active_count(const uint32_t* heads, uint64_t n, uint64_t* word_counts, cudaStream_t s);
// exclusive scan in place; total written to *total; block_sums needs scan_block_count(n) entries
uint64_t scan_block_count(uint64_t n);
cudaError_t launch_scan_u64(uint64_t* data, uint64_t n, uint64_t* block_sums, uint64_t* total, cudaStream_t s);
// keys of the active elements (members of open groups, in position order) and, as the sort's values, their positions
template <typename IdT>
cudaError_t launch_refine_rekey(const Reads& R, const uint32_t* heads, const uint64_t* word_base, const IdT* ids, uint64_t n,
                                uint32_t depth, uint32_t w, uint64_t* keys_c, uint32_t* pos_c, cudaStream_t s);
// after the sort: fetches the sorted elements' ids through their old positions (into ids_tmp, n_c entries), writes them to
// the active positions in order, sets new head bits in heads_out (the caller's copy of `heads`, which is only read) and emits
// the BWT symbol of every suffix that became final
template <typename IdT>
cudaError_t launch_refine_writeback(const Reads& R, const uint64_t* keys_c, const uint32_t* pos_sorted, IdT* ids_tmp, const uint32_t* heads,
                                    const uint64_t* word_base, uint64_t n, uint64_t n_c, uint32_t w, IdT* ids, uint32_t* heads_out, uint8_t* out,
                                    cudaStream_t s);
// a7 + a8 over the freshly sorted first-round keys: the warp kernel finishes singletons and tie groups of at most 32
// suffixes, counts the groups it leaves to the global path (elems_done[4]) and clears all but their first bit in heads_out
// (the head bitmask of that path; filled with ones by the caller: every other position counts as a group of one); the block kernel then finishes the groups of 33..group_cap in the tiles the warp
// kernel flagged in big_tiles (n / kLocalTile / 32 + 2 words).  depth0: symbols the first-round sort has settled.
// packed: keys1 holds 64-bit words (32-bit key << 32 | 32-bit id); `ids` then receives the ids of the groups left to the
// global path (nothing else will need the others).
template <typename KeyT, typename IdT>
cudaError_t launch_finish_first(const Reads& R, const KeyT* keys1, uint32_t w1, uint32_t depth0, uint32_t* heads_out, IdT* ids, uint64_t n,
                                uint32_t group_cap, uint8_t* out, unsigned long long* elems_done, uint32_t* big_tiles, int n_sms, bool packed,
                                uint32_t slots, Launch* prof, cudaStream_t s, uint32_t split = 0, IdT* ids_out = nullptr);
// split != 0 (64-bit keys and ids): keys1 holds key << split | id >> 32 and `ids` is a uint32 array of the ids' low words (the
// sort's 12-byte pairs); the ids of the groups left to the global path are then assembled into ids_out (another buffer)
// a sample of the sorted first-round keys: *counter += sampled positions in tie groups of more than 64 suffixes, *sampled (HOST) =
// positions looked at (0: batch too small to sample).  slots of launch_finish_first: 4 if those are a large share, else 2
template <typename KeyT, typename IdT>
cudaError_t launch_group_probe(const KeyT* keys1, uint32_t w1, uint64_t n, bool packed, unsigned long long* counter, uint64_t* sampled, cudaStream_t s,
                               uint32_t split = 0);
// in-block refinement + emit of the groups a global round has split to at most group_cap members; heads_out = copy of heads_in
template <typename IdT>
cudaError_t launch_finish_later(const Reads& R, const uint32_t* heads_in, uint32_t* heads_out, const IdT* ids, uint64_t n, uint32_t depth,
                                uint32_t group_cap, uint8_t* out, unsigned long long* elems_done, int n_sms, cudaStream_t s);

}  // namespace cx
