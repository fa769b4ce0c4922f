// cx_refine.cu -- step a7: segmented tie refinement, and step a8: the BWT emit gather.
//
// After a sort by the first d symbols, suffixes with equal keys form a tie group.  A group whose key
// carries a length field < w saw its end-marker: its members are identical strings, already in
// read-index order because ids were listed in (read, pos) order and every reordering is stable
// -- it is final.  Every other group of two or more must be ordered by what follows
// (the first differing symbol decides).  The paper always runs all ceil(2(m+1)/32)
// iterations over all suffixes; here only the groups still tied are re-keyed:
//
//   local path : groups of at most kLocalGroupCap suffixes are finished inside one thread block --
//                one locator per member in shared memory (first base, bases left, preceding symbol: the
//                offsets table and the word before the suffix are gathered once), one 88-base gather per
//                member per round (192-bit key: bases, length, index in the group), stable rank by
//                counting inside sub-blocks and rank-merging them, looping over depth until every member
//                is placed; the BWT symbols then come straight from the locators;
//   global path: larger groups are compacted, re-keyed as (group ordinal | next w' bases | length)
//                in one 64-bit key, sorted by the onesweep sorter, and written back in place.
//
// Group heads live in a bitmask: bit j = 1 iff sorted position j starts a group.
#include "cx_internal.cuh"
#include "cx_launch.h"

namespace cx {
namespace {

constexpr uint32_t kFull = 0xffffffffu;

// (start, length) of read i
__device__ __forceinline__ void read_span(const Reads& R, uint64_t i, uint64_t& start, uint64_t& len) {
    if (R.uniform) {
        start = i * R.uniform_len;
        len = R.uniform_len;
    } else {
        start = __ldg(R.offsets + i);
        len = __ldg(R.offsets + i + 1) - start;
    }
}

// key of suffix `id` at depth d: the next w bases after the first d symbols (the next
// "stringword" permuted by the index already on the GPU -- here gathered from the resident reads)
template <typename IdT>
__device__ __forceinline__ uint64_t key_at_depth(const Reads& R, IdT id, uint32_t depth, uint32_t w) {
    uint64_t read = (uint64_t)id >> R.pos_bits;
    uint64_t pos = (uint64_t)id & ((1ull << R.pos_bits) - 1);
    uint64_t start, len;
    read_span(R, read, start, len);
    uint64_t at = pos + depth;
    uint64_t rem = at < len ? len - at : 0;
    uint64_t window = rem ? load_window(R.packed, R.n_words, start + at) : 0ull;
    return make_key(window, rem, w);
}

// per 32 positions: active elements (members of groups of >= 2) and active heads, packed hi|lo
__device__ __forceinline__ void active_masks(uint32_t H, uint32_t next_word, uint32_t& act, uint32_t& act_heads) {
    uint32_t Hn = (H >> 1) | (next_word << 31);   // bit j = head(j + 1)
    act = ~(H & Hn);
    act_heads = H & ~Hn;
}

__global__ void __launch_bounds__(256) active_count_kernel(const uint32_t* __restrict__ heads, uint64_t n_words,
                                                           uint64_t* __restrict__ word_counts) {
    uint64_t wi = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (wi >= n_words) return;
    uint32_t act, ah;
    active_masks(heads[wi], heads[wi + 1], act, ah);
    word_counts[wi] = ((uint64_t)__popc(ah) << 32) | (uint64_t)__popc(act);
}

// ---------------------------------------------------------------------------------------------
// exclusive scan of uint64 (reduce, scan of block sums, down-sweep)
// ---------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanChunk = kScanThreads * kScanItems;

__device__ __forceinline__ uint64_t block_exclusive_scan(uint64_t v, uint64_t* s_warp, uint64_t& total) {
    uint64_t incl = v;
    for (int o = 1; o < 32; o <<= 1) {
        uint64_t up = __shfl_up_sync(kFull, incl, o);
        if ((int)lane_id() >= o) incl += up;
    }
    uint32_t warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane_id() == 31) s_warp[warp] = incl;
    __syncthreads();
    uint64_t carry = 0, all = 0;
    for (uint32_t q = 0; q < kScanThreads / 32; ++q) {
        uint64_t t = s_warp[q];
        if (q < warp) carry += t;
        all += t;
    }
    total = all;
    return carry + incl - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_reduce_kernel(const uint64_t* __restrict__ data, uint64_t n,
                                                                   uint64_t* __restrict__ block_sums) {
    __shared__ uint64_t s_warp[kScanThreads / 32];
    uint64_t base = (uint64_t)blockIdx.x * kScanChunk;
    uint64_t sum = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        uint64_t idx = base + (uint64_t)i * kScanThreads + threadIdx.x;
        if (idx < n) sum += data[idx];
    }
    uint64_t total;
    block_exclusive_scan(sum, s_warp, total);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) scan_sums_kernel(uint64_t* __restrict__ block_sums, uint64_t n_blocks,
                                                                 uint64_t* __restrict__ total_out) {
    __shared__ uint64_t s_warp[kScanThreads / 32];
    uint64_t carry = 0;
    for (uint64_t base = 0; base < n_blocks; base += kScanThreads) {
        uint64_t idx = base + threadIdx.x;
        uint64_t v = idx < n_blocks ? block_sums[idx] : 0;
        uint64_t total;
        uint64_t excl = block_exclusive_scan(v, s_warp, total);
        if (idx < n_blocks) block_sums[idx] = carry + excl;
        carry += total;
    }
    if (threadIdx.x == 0) *total_out = carry;
}

__global__ void __launch_bounds__(kScanThreads) scan_down_kernel(uint64_t* __restrict__ data, uint64_t n,
                                                                 const uint64_t* __restrict__ block_sums) {
    __shared__ uint64_t s_warp[kScanThreads / 32];
    // blocked arrangement: thread t owns kScanItems consecutive entries
    uint64_t base = (uint64_t)blockIdx.x * kScanChunk + (uint64_t)threadIdx.x * kScanItems;
    uint64_t v[kScanItems];
    uint64_t sum = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = base + i < n ? data[base + i] : 0;
        sum += v[i];
    }
    uint64_t total;
    uint64_t run = block_exclusive_scan(sum, s_warp, total) + block_sums[blockIdx.x];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (base + i < n) data[base + i] = run;
        run += v[i];
    }
}

// ---------------------------------------------------------------------------------------------
// a8 helper: B[k] = '$' if the k-th suffix starts its read, else the base before it
// ---------------------------------------------------------------------------------------------
template <typename IdT>
__device__ __forceinline__ uint8_t preceding_symbol(const Reads& R, IdT id) {
    uint64_t read = (uint64_t)id >> R.pos_bits;
    uint64_t pos = (uint64_t)id & ((1ull << R.pos_bits) - 1);
    if (pos == 0) return (uint8_t)'$';
    uint64_t b = (R.uniform ? read * R.uniform_len : __ldg(R.offsets + read)) + pos - 1;
    uint32_t code = (uint32_t)(__ldg(R.packed + (b >> 5)) >> (62 - 2 * (b & 31))) & 3u;
    return (uint8_t)((0x54474341u >> (8 * code)) & 0xFFu);
}

// split != 0 (64-bit keys and ids, batches of a multi-batch plan): the word is key << split | id >> 32 and the id's low 32
// bits are a uint32 array where the ids would be
template <bool PACKED>
__device__ __forceinline__ uint64_t key_of(uint64_t word, uint32_t split) { return PACKED ? word >> 32 : word >> split; }
template <typename IdT>
__device__ __forceinline__ IdT split_id(uint64_t word, uint32_t split, const IdT* __restrict__ ids_lo, uint64_t j) {
    return (IdT)(((word & ((1ull << split) - 1)) << 32) | (uint64_t)__ldg(reinterpret_cast<const uint32_t*>(ids_lo) + j));
}

// ---------------------------------------------------------------------------------------------
// global path: compact + re-key, write back
// ---------------------------------------------------------------------------------------------
// One thread per 32 sorted positions looks for members still tied; the warp then handles every such word together,
// one lane per position (oversize groups are rare, so nearly all threads leave after one load).  f(j, c, g): position j is
// the c-th active one and belongs to the g-th open group.
template <typename F>
__device__ __forceinline__ void for_each_active(const uint32_t* __restrict__ heads, const uint64_t* __restrict__ word_base, uint64_t n, F&& f) {
    const uint64_t n_words = (n + 31) >> 5;
    const uint64_t wi = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t act = 0, ah = 0;
    if (wi < n_words) active_masks(heads[wi], heads[wi + 1], act, ah);
    uint64_t base = act ? word_base[wi] : 0ull;
    uint32_t todo = __ballot_sync(kFull, act != 0);
    const uint32_t bit = lane_id();
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const uint32_t wact = __shfl_sync(kFull, act, src), wah = __shfl_sync(kFull, ah, src);
        const uint64_t wbase = __shfl_sync(kFull, base, src);
        const uint64_t wwi = wi - bit + src;   // word index of lane `src` (lanes hold consecutive words)
        if ((wact >> bit) & 1u) {
            const uint32_t below = (1u << bit) - 1;
            f((wwi << 5) + bit, (wbase & 0xffffffffull) + __popc(wact & below), (wbase >> 32) + __popc(wah & (below | (1u << bit))) - 1);
        }
    }
}

// The sort of a global round carries, as its value, the POSITION of the element in the batch (32 bits: the ids stay where
// they are and are fetched through it afterwards), so it needs no buffer beyond the two key buffers and one id buffer that
// are free at this point.
template <typename IdT>
__global__ void __launch_bounds__(256) refine_rekey_kernel(Reads R, const uint32_t* __restrict__ heads,
                                                           const uint64_t* __restrict__ word_base, const IdT* __restrict__ ids,
                                                           uint64_t n, uint32_t depth, uint32_t w, uint64_t* __restrict__ keys_c,
                                                           uint32_t* __restrict__ pos_c) {
    for_each_active(heads, word_base, n, [&](uint64_t j, uint64_t c, uint64_t g) {
        keys_c[c] = (g << (2 * w + 5)) | key_at_depth(R, ids[j], depth, w);
        pos_c[c] = (uint32_t)j;
    });
}

// ids of the sorted elements, fetched through their old positions (into a buffer of their own: the write-back below moves
// them to positions that other threads still read from)
template <typename IdT>
__global__ void __launch_bounds__(256) refine_gather_kernel(const uint32_t* __restrict__ pos_sorted, uint64_t n_c, const IdT* __restrict__ ids,
                                                            IdT* __restrict__ ids_c) {
    const uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < n_c) ids_c[c] = ids[pos_sorted[c]];
}

// The c-th sorted element goes to the c-th active position.  `heads` is read (which positions are active), `heads_out` --
// a copy of it made by the caller -- receives the new head bits.
template <typename IdT>
__global__ void __launch_bounds__(256) refine_writeback_kernel(Reads R, const uint64_t* __restrict__ keys_c, const IdT* __restrict__ ids_c,
                                                               const uint32_t* __restrict__ heads, const uint64_t* __restrict__ word_base,
                                                               uint64_t n, uint64_t n_c, uint32_t w, IdT* __restrict__ ids,
                                                               uint32_t* __restrict__ heads_out, uint8_t* __restrict__ out) {
    for_each_active(heads, word_base, n, [&](uint64_t pos, uint64_t c, uint64_t) {
        const uint64_t k = keys_c[c];
        const IdT id = ids_c[c];
        ids[pos] = id;
        const bool head = c == 0 || k != keys_c[c - 1] || (uint32_t)(k & 31) < w;
        if (head) atomicOr(&heads_out[pos >> 5], 1u << (pos & 31));
        // alone in its group now (or its end-marker was inside the window): final, emit its BWT symbol
        bool next_is_head = true;
        if (c + 1 < n_c) {
            const uint64_t kn = keys_c[c + 1];
            next_is_head = kn != k || (uint32_t)(kn & 31) < w;
        }
        if (head && next_is_head) out[pos] = preceding_symbol(R, id);
    });
}

// ---------------------------------------------------------------------------------------------
// a7 + a8 fused, one block per tile of kLocalTile sorted positions ("finish" kernel):
//   FIRST : head flags from the freshly sorted first-round keys; every suffix that is alone in its
//           group is final and its BWT symbol is emitted at once; groups of 2..cap suffixes that start
//           in the tile are refined to the end in shared memory and emitted; larger groups are left
//           to the global path (their head bits go to `heads`).
//   !FIRST: after a global round; head flags come from `heads`; only groups of 2..cap are touched.
// A position is emitted exactly once, by whoever makes it final (here, or the global write-back).
//
// Refinement of one tie group (all members share their first D symbols):
//   * every member holds a WINDOW of the next kWin = 96 bases in shared memory (A-padded past the end of its read),
//     gathered ONCE -- a 100 bp read never needs a second gather after a 14-base first sort;
//   * the group's PIVOT is its member with the most bases in the window.  One XOR + count-leading-zeros of the
//     member's window against the pivot's gives where the member first differs from the pivot (a base, or the
//     end of one of the two), which is all that PAPER.md:55 needs to order it against everything else that was
//     compared with the same pivot:   below the pivot -- ascending depth of divergence, then the symbol there;
//     equal to the pivot through the window;   above the pivot -- descending depth, then the symbol.
//     That is an 11-bit key; with the member's index in the group below it a 32-bit unsigned compare ranks the
//     group stably -- the wide comparison is made once per member, not once per pair;
//   * members with equal keys form the next groups: those that ENDED at the divergence are identical strings and
//     final in their current (read index) order; the others go round again with their own pivot; a class that
//     equals the pivot through a full window gathers its next window first (reads longer than the window).
// ---------------------------------------------------------------------------------------------
constexpr int kLocalElems = kLocalTile + kLocalGroupCap;   // positions a block may touch
constexpr int kLocalWords = kLocalElems / 32 + 2;
constexpr int kLocalItems = kLocalElems / kLocalThreads;
static_assert(kLocalElems % kLocalThreads == 0 && kLocalThreads % 32 == 0, "tile shape");
static_assert(kLocalElems <= 1024 && kLocalGroupCap <= 256, "a position takes 10 bits and an index inside a group 8 bits of the rank key");
constexpr uint32_t kWin = 96;                         // bases per window (three packed words)
constexpr uint32_t kKeyEqual = kWin * 8;              // key of "equal to the pivot through the window"
constexpr uint32_t kKeyAbove = kKeyEqual + 8;         // first key of the members above the pivot
constexpr uint16_t kNone = 0xffff;

// Locator of a member: [code of the preceding symbol, 1 = $, 2..5 = A C G T : 3][window must be gathered : 1]
// [unused : 12][bases of the window that exist, <= kWin : 8][index of the window's first base in the packed text : 40]
constexpr uint32_t kLocBaseBits = 40, kLocTakeShift = 40, kLocCodeShift = 61;
constexpr uint64_t kLocBaseMask = (1ull << kLocBaseBits) - 1, kLocGather = 1ull << 60;
__device__ __forceinline__ uint8_t loc_symbol(uint64_t loc) { return (uint8_t)(0x544743412400ull >> (8 * (uint32_t)(loc >> kLocCodeShift))); }
__device__ __forceinline__ uint32_t loc_take(uint64_t loc) { return (uint32_t)(loc >> kLocTakeShift) & 255u; }

struct LocalSmem {
    uint64_t w0[kLocalElems], w1[kLocalElems], w2[kLocalElems];   // member's window: bases [0,32), [32,64), [64,96), A-padded
    uint64_t loc[kLocalElems];     // member's locator (holds the raw id between the head pass and the classify pass)
    uint32_t mrem[kLocalElems];    // member: bases of its read from the window's first base on
    uint32_t key[kLocalElems];     // position: rank key of the member now there; a position outside every open group holds
                                   // (position << 21), so that keys are comparable across a whole aligned 32-position window
    uint32_t sk[2][kLocalElems];   // position: keys of the sorted runs being merged, ping-pong
    uint16_t mem[2][kLocalElems];  // position -> member, ping-pong over rounds
    uint16_t gs[kLocalElems];      // position: first position of its open group (kNone: not ours / placed)
    uint16_t ge[kLocalElems];      // one past the last
    uint32_t gpiv[2][kLocalElems / 2];   // group (slot = first position / 2; a group has >= 2 members): max over members of
                                         // (bases in window << 10 | member); ping-pong over rounds
    uint32_t hw[kLocalWords];      // head bits of the window, updated as groups split
    uint32_t hw0[kLocalWords];     // as loaded
    uint8_t sym[kLocalElems];      // position: BWT symbol of the member placed there for good
};

// nearest set bit at or below position e, not lower than `lo`; -1 if none
__device__ __forceinline__ int prev_head(const uint32_t* hw, int e, int lo) {
    int wi = e >> 5;
    uint32_t bits = hw[wi] & (0xffffffffu >> (31 - (e & 31)));
    while (true) {
        if (bits) {
            int p = (wi << 5) + 31 - __clz(bits);
            return p >= lo ? p : -1;
        }
        if ((wi << 5) <= lo) return -1;
        --wi;
        bits = hw[wi];
    }
}
// nearest set bit above position e, not higher than `hi`; -1 if none
__device__ __forceinline__ int next_head(const uint32_t* hw, int e, int hi) {
    int wi = e >> 5;
    uint32_t bits = (e & 31) == 31 ? 0u : hw[wi] & (0xffffffffu << ((e & 31) + 1));
    while (true) {
        if (bits) {
            int p = (wi << 5) + __ffs(bits) - 1;
            return p <= hi ? p : -1;
        }
        ++wi;
        if ((wi << 5) > hi) return -1;
        bits = hw[wi];
    }
}

// x with only its first cnt bases kept (cnt may be <= 0 or >= 32)
__device__ __forceinline__ uint64_t keep_bases(uint64_t x, int cnt) {
    return cnt >= 32 ? x : (cnt <= 0 ? 0ull : x & (~0ull << (64 - 2 * cnt)));
}

// The window of `take` <= kWin bases that starts at base index b, into shared memory as three A-padded words.
struct Window {
    uint64_t x[4];     // the packed words from the one that holds base b (words the window does not touch are 0)
    uint32_t shift;    // bit offset of base b in x[0]
    uint32_t take;
};
__device__ __forceinline__ void window_load(const uint64_t* __restrict__ packed, uint64_t b, uint32_t take, bool want, Window& wd) {
    wd.shift = (uint32_t)(b & 31) * 2;
    wd.take = take;
    const uint32_t n_w = want && take ? (wd.shift + 2 * take + 63) >> 6 : 0u;   // words the window touches (<= 4)
    const uint64_t* p = packed + (b >> 5);
#pragma unroll
    for (int i = 0; i < 4; ++i) wd.x[i] = i < (int)n_w ? __ldg(p + i) : 0ull;
}
__device__ __forceinline__ void window_store(const Window& wd, LocalSmem& sm, int m) {
    uint64_t p0 = wd.x[0], p1 = wd.x[1], p2 = wd.x[2];
    if (wd.shift) {
        p0 = (wd.x[0] << wd.shift) | (wd.x[1] >> (64 - wd.shift));
        p1 = (wd.x[1] << wd.shift) | (wd.x[2] >> (64 - wd.shift));
        p2 = (wd.x[2] << wd.shift) | (wd.x[3] >> (64 - wd.shift));
    }
    sm.w0[m] = keep_bases(p0, (int)wd.take);
    sm.w1[m] = keep_bases(p1, (int)wd.take - 32);
    sm.w2[m] = keep_bases(p2, (int)wd.take - 64);
}

// Lanes hold consecutive positions; H = head bits of the warp's 32 positions.  The maximum of `val` over each run of lanes
// between heads is added to the slot of that run with ONE shared-memory atomic by the run's last lane (a group's members
// would otherwise all hit one address).  val = 0: nothing to publish (slot is then not read).
__device__ __forceinline__ void seg_max_publish(uint32_t val, uint32_t H, uint32_t* slots, uint32_t slot) {
    const uint32_t lane = lane_id();
    const uint32_t hb = H & (0xffffffffu >> (31 - lane));
    const uint32_t lo = hb ? 31u - (uint32_t)__clz(hb) : 0u;   // first lane of my run
#pragma unroll
    for (uint32_t o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(kFull, val, o);
        if (lane >= lo + o && v > val) val = v;
    }
    const bool last = lane == 31 || ((H >> (lane + 1)) & 1u);
    if (last && val) atomicMax(slots + slot, val);
}

// merge levels a group [s, t) needs after its aligned 32-position windows have been ranked: 0 if it lies in one window
__device__ __forceinline__ int merge_levels(int s, int t) {
    const uint32_t x = (uint32_t)(s ^ (t - 1)) >> 5;
    return x ? 32 - __clz(x) : 0;
}

template <typename KeyT, typename IdT, bool FIRST, bool PACKED>
__device__ __forceinline__ void finish_tile(LocalSmem& sm, uint64_t tile, const Reads& R, const KeyT* __restrict__ keys1,
                                            const uint32_t* __restrict__ heads_in, uint32_t* __restrict__ heads, const IdT* __restrict__ ids,
                                            uint64_t n, uint32_t depth0, uint32_t min_group, uint32_t cap, uint8_t* __restrict__ out,
                                            unsigned long long* elems_done, uint32_t split) {
    const uint64_t base = tile * kLocalTile;
    const uint64_t w0 = base >> 5;
    const uint64_t n_words = (n + 31) >> 5;   // heads[n_words] is the padding word ("the next position is a head")
    const int tid = threadIdx.x;

    for (int i = tid; i < kLocalElems / 2; i += kLocalThreads) sm.gpiv[0][i] = 0;
    // ---- head bits of the window ------------------------------------------------------------------
    if (FIRST) {
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            const uint64_t j = base + e;
            bool head = true;   // positions past n count as heads
            if (j < n) {
                if constexpr (PACKED) {
                    const uint64_t* pairs = reinterpret_cast<const uint64_t*>(keys1);
                    const uint64_t pc = __ldcs(pairs + j);
                    const uint32_t kc = (uint32_t)(pc >> 32);
                    head = j == 0 || kc != (uint32_t)(__ldg(pairs + j - 1) >> 32) || !(kc & 1u);
                    sm.loc[e] = (uint32_t)pc;
                } else {
                    const uint64_t wc = (uint64_t)__ldcs(keys1 + j);
                    const uint64_t kc = wc >> split;
                    head = j == 0 || kc != ((uint64_t)__ldg(keys1 + j - 1) >> split) || !((uint32_t)kc & 1u);
                    sm.loc[e] = split ? (uint64_t)split_id<IdT>(wc, split, ids, j) : (uint64_t)__ldcs(ids + j);
                }
            }
            const uint32_t word = __ballot_sync(kFull, head);
            if ((tid & 31) == 0) sm.hw[e >> 5] = word;
        }
        if (tid < kLocalWords - kLocalElems / 32) sm.hw[kLocalElems / 32 + tid] = kFull;
    } else {
        uint32_t incomplete = 0;
        for (int i = tid; i < kLocalWords; i += kLocalThreads) {
            const uint32_t v = w0 + i <= n_words ? heads_in[w0 + i] : kFull;
            sm.hw[i] = v;
            sm.hw0[i] = v;
            // positions 1 .. kLocalTile decide whether a group of >= 2 starts in this tile
            if (i <= kLocalTile / 32) {
                const uint32_t care = i == 0 ? ~1u : (i == kLocalTile / 32 ? 1u : kFull);
                incomplete |= (~v) & care;
            }
        }
        if (!__syncthreads_or(incomplete)) return;
    }
    __syncthreads();

    // ---- classify: groups that start in this tile and have at most cap members are ours -----------
    uint32_t n_active = 0, n_compares = 0;
    IdT idv[kLocalItems];
    uint32_t state = 0;   // 2 bits per position: 0 not ours, 1 alone in its group (final), 2 member of a group refined here
    uint16_t gsv[kLocalItems];
#pragma unroll
    for (int k = 0; k < kLocalItems; ++k) {
        const int e = k * kLocalThreads + tid;
        uint16_t s = kNone, t = kNone;
        uint32_t st = 0;
        idv[k] = 0;
        if (base + e < n) {
            const int lo = e - (int)cap + 1;
            const int ps = prev_head(sm.hw, e, lo < 0 ? 0 : lo);
            if (ps >= 0 && ps < kLocalTile) {
                const int ne = next_head(sm.hw, e, ps + (int)cap);
                if (ne > 0 && ne - ps >= (int)min_group) {   // FIRST: smaller groups were finished by the warp kernel
                    s = (uint16_t)ps;
                    t = (uint16_t)ne;
                    st = 2;
                    ++n_active;
                }
            }
            if (st) idv[k] = FIRST ? (IdT)sm.loc[e] : ids[base + e];
        }
        sm.gs[e] = s;
        sm.ge[e] = t;
        sm.mem[0][e] = (uint16_t)e;
        gsv[k] = s;
        state |= st << (2 * k);
    }
    // ---- locators, the base before every suffix of ours, and the window of every member: one batch of gathers --------
    // The kernel lives on these random reads; all of a thread's loads are issued before the first is used.
    {
        uint64_t first_base[kLocalItems];   // index of the suffix's first base in the packed text
        uint64_t left[kLocalItems];         // bases from there to the end of its read
        const uint64_t pos_mask = (1ull << R.pos_bits) - 1;
        if (R.uniform) {
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const uint64_t read = (uint64_t)idv[k] >> R.pos_bits, pos = (uint64_t)idv[k] & pos_mask;
                first_base[k] = read * R.uniform_len + pos;
                left[k] = R.uniform_len - pos;
            }
        } else {
            uint64_t lo[kLocalItems], hi[kLocalItems];
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const uint64_t* p = R.offsets + (((state >> (2 * k)) & 3u) ? (uint64_t)idv[k] >> R.pos_bits : 0ull);
                lo[k] = __ldg(p);
                hi[k] = __ldg(p + 1);
            }
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const uint64_t pos = (uint64_t)idv[k] & pos_mask;
                first_base[k] = lo[k] + pos;
                left[k] = hi[k] - lo[k] - pos;
            }
        }
        uint64_t before[kLocalItems];       // the word that holds the base before the suffix
        Window wd[kLocalItems];
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const uint32_t st = (state >> (2 * k)) & 3u;
            const bool want = st && ((uint64_t)idv[k] & pos_mask);
            before[k] = want ? __ldg(R.packed + ((first_base[k] - 1) >> 5)) : 0ull;   // no load for a read's first suffix
            const uint64_t rem = st == 2 ? left[k] - depth0 : 0ull;                    // a member of an open group has >= depth0 bases
            window_load(R.packed, first_base[k] + depth0, (uint32_t)(rem < kWin ? rem : kWin), st == 2, wd[k]);
        }
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            const uint32_t st = (state >> (2 * k)) & 3u;
            uint64_t code = 1;   // $: the suffix starts its read
            if ((uint64_t)idv[k] & pos_mask) code = 2 + ((before[k] >> (62 - 2 * ((first_base[k] - 1) & 31))) & 3u);
            uint32_t cand = 0;
            if (st == 2) {
                const uint64_t rem = left[k] - depth0;
                window_store(wd[k], sm, e);
                sm.loc[e] = (code << kLocCodeShift) | ((uint64_t)wd[k].take << kLocTakeShift) | (first_base[k] + depth0);
                sm.mrem[e] = (uint32_t)rem;   // reads are shorter than 2^32 bases (checked by the build)
                cand = (wd[k].take << 10) | (uint32_t)e;
            }
            // the pivot of every group: its member with the most bases in the window
            seg_max_publish(cand, sm.hw[e >> 5], sm.gpiv[0], (uint32_t)(gsv[k] >> 1));
        }
    }
    __syncthreads();

    // ---- rounds ----------------------------------------------------------------------------------------------------
    uint32_t n_rounds = 0;
    for (int pb = 0, mb = 0;; pb ^= 1, mb ^= 1, ++n_rounds) {
        // keys: where each member first differs from its group's pivot
        uint32_t mykey[kLocalItems];
        uint32_t any = 0;
        for (int i = tid; i < kLocalElems / 2; i += kLocalThreads) sm.gpiv[pb ^ 1][i] = 0;
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int q = k * kLocalThreads + tid;
            const int s = sm.gs[q];
            mykey[k] = (uint32_t)q << 21;
            if (s != kNone) {
                const int m = sm.mem[mb][q];
                const uint32_t pv = sm.gpiv[pb][s >> 1];
                const int pm = pv & 1023u;
                const uint32_t tb = pv >> 10, ta = loc_take(sm.loc[m]);
                const uint64_t a0 = sm.w0[m], a1 = sm.w1[m], a2 = sm.w2[m];
                const uint64_t x0 = a0 ^ sm.w0[pm], x1 = a1 ^ sm.w1[pm], x2 = a2 ^ sm.w2[pm];
                // first base at which the two windows differ (kWin: nowhere)
                const uint32_t d = x0 ? (uint32_t)__clzll((long long)x0) >> 1 : x1 ? 32u + ((uint32_t)__clzll((long long)x1) >> 1)
                                      : x2 ? 64u + ((uint32_t)__clzll((long long)x2) >> 1) : kWin;
                const uint32_t lim = ta < tb ? ta : tb;
                uint32_t K;
                if (d < lim || ta > tb) {
                    // a base of mine against a base of the pivot (d < lim), or against the pivot's end-marker (the pivot
                    // ended at tb and I go on: above it; cannot happen while the pivot is the longest member)
                    const uint32_t at = d < lim ? d : tb;
                    const uint64_t aw = at < 32 ? a0 : at < 64 ? a1 : a2;
                    const uint32_t sa = (uint32_t)(aw >> (62 - 2 * (at & 31))) & 3u;
                    bool below = false;
                    if (d < lim) {
                        const uint64_t bw = at < 32 ? sm.w0[pm] : at < 64 ? sm.w1[pm] : sm.w2[pm];
                        below = sa < ((uint32_t)(bw >> (62 - 2 * (at & 31))) & 3u);
                    }
                    K = below ? at * 8 + sa + 1 : kKeyAbove + (kWin - 1 - at) * 8 + sa + 1;
                } else if (ta < tb) {
                    K = ta * 8;          // my end-marker against a base of the pivot: below it ($ is the smallest symbol)
                } else {
                    K = kKeyEqual;       // equal to the pivot through the window (and of its length)
                }
                mykey[k] = ((uint32_t)s << 21) | (K << 8) | (uint32_t)(q - s);
                any = 1;
            }
            sm.key[q] = mykey[k];
        }
        if (!__syncthreads_or(any)) break;
        // Stable rank.  Keys are comparable across groups (the group's first position leads the key), so a member's place
        // inside its aligned window of 32 positions is the number of smaller keys among the 32, whoever owns them.
        int pos[kLocalItems];
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int q = k * kLocalThreads + tid;
            pos[k] = q;
            if (sm.gs[q] != kNone) {
                const uint4* wkeys = reinterpret_cast<const uint4*>(sm.key + (q & ~31));
                const uint32_t me = mykey[k];
                uint32_t below = 0;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const uint4 v = wkeys[i];
                    below += (uint32_t)(v.x < me) + (uint32_t)(v.y < me) + (uint32_t)(v.z < me) + (uint32_t)(v.w < me);
                }
                pos[k] = (q & ~31) + (int)below;
                sm.sk[0][pos[k]] = me;
                n_compares += 32;
            }
        }
        // groups that span several windows: sorted runs are merged pairwise, each member finding its rank in the
        // sibling run by binary search over the sorted keys (keys are distinct: the index in the group is part of them)
        for (int level = 0;; ++level) {
            uint32_t more = 0;
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const int q = k * kLocalThreads + tid;
                const int s = sm.gs[q];
                if (s != kNone) more |= (uint32_t)(merge_levels(s, sm.ge[q]) > level);
            }
            if (!__syncthreads_or(more)) break;
            const uint32_t* src = sm.sk[level & 1];
            uint32_t* dst = sm.sk[(level + 1) & 1];
            const int wd = 32 << level;
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const int q = k * kLocalThreads + tid;
                const int s = sm.gs[q];
                if (s == kNone) continue;
                const int t = sm.ge[q];
                if (merge_levels(s, t) <= level) continue;
                const int wbase = q & ~(wd - 1), sbase = wbase ^ wd;                  // my window and its sibling
                const int my_lo = max(s, wbase);
                const int sib_lo = max(s, sbase), sib_hi = min(t, sbase + wd);       // the group's part of the sibling run
                int lo = 0;
                if (sib_lo < sib_hi) {
                    int hi = sib_hi - sib_lo;
                    const uint32_t me = mykey[k];
                    n_compares += 32 - __clz(hi);
                    while (lo < hi) {                // lower bound: sibling members below me
                        const int mid = (lo + hi) >> 1;
                        if (src[sib_lo + mid] < me) lo = mid + 1; else hi = mid;
                    }
                }
                const int start = sib_lo < sib_hi && sbase < wbase ? sib_lo : my_lo;   // first position of the merged run
                pos[k] = start + (pos[k] - my_lo) + lo;
                dst[pos[k]] = mykey[k];
            }
        }
        // new head bits, position by position over the ranked keys; the member that ranked at a position moves there
        uint32_t info[kLocalItems];   // (key class << 16 | member now here), ~0u: position not in an open group
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int p = k * kLocalThreads + tid;
            const int s = sm.gs[p];
            bool head = false;
            info[k] = ~0u;
            if (s != kNone) {
                const uint32_t* fin = sm.sk[merge_levels(s, sm.ge[p]) & 1];
                const uint32_t kk = fin[p];
                const uint32_t K = (kk >> 8) & 0x7ffu;
                const uint32_t tb = sm.gpiv[pb][s >> 1] >> 10;
                // final classes: members that ended at their divergence, or equal the pivot and end with it -- identical
                // strings, already in read-index order; each becomes a group of one
                const bool final_class = (K < kKeyEqual && (K & 7u) == 0) || (K == kKeyEqual && tb < kWin);
                head = p == s || final_class || K != ((fin[p - 1] >> 8) & 0x7ffu);
                const uint32_t m = sm.mem[mb][s + (kk & 255u)];
                sm.mem[mb ^ 1][p] = (uint16_t)m;
                info[k] = (K << 16) | m;
            }
            const uint32_t word = __ballot_sync(kFull, head);
            if ((tid & 31) == 0 && word) sm.hw[p >> 5] |= word;
        }
        __syncthreads();
        // new group bounds; members alone in their group are placed for good; the others name their next pivot
        uint32_t regather = 0;
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int p = k * kLocalThreads + tid;
            uint32_t cand = 0, slot = 0;
            if (info[k] != ~0u) {
                const uint32_t m = info[k] & 0xffffu, K = info[k] >> 16;
                const uint32_t lo = sm.hw[p >> 5], hi = sm.hw[(p >> 5) + 1];
                uint64_t loc = sm.loc[m];
                if (((((uint64_t)hi << 32) | lo) >> (p & 31) & 3u) == 3u) {   // head bits of p and p + 1: alone, placed
                    sm.sym[p] = loc_symbol(loc);
                    sm.gs[p] = kNone;
                } else {
                    const int s2 = prev_head(sm.hw, p, sm.gs[p]);
                    const int t2 = next_head(sm.hw, p, sm.ge[p]);
                    sm.gs[p] = (uint16_t)s2;
                    sm.ge[p] = (uint16_t)t2;
                    uint32_t take = loc_take(loc);
                    if (K == kKeyEqual) {   // equal to the pivot through a full window: on to the next window of the read
                        const uint32_t rem = sm.mrem[m] - kWin;
                        sm.mrem[m] = rem;
                        take = rem < kWin ? rem : kWin;
                        loc = (loc & ~((0xffull << kLocTakeShift) | kLocBaseMask)) | ((uint64_t)take << kLocTakeShift) | ((loc & kLocBaseMask) + kWin) | kLocGather;
                        sm.loc[m] = loc;
                        regather = 1;
                    }
                    cand = (take << 10) | m;
                    slot = (uint32_t)s2 >> 1;
                }
            }
            seg_max_publish(cand, sm.hw[p >> 5], sm.gpiv[pb ^ 1], slot);
        }
        if (__syncthreads_or(regather)) {
            Window wd[kLocalItems];
            uint32_t mm[kLocalItems];
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const int p = k * kLocalThreads + tid;
                mm[k] = ~0u;
                uint64_t loc = 0;
                if (sm.gs[p] != kNone) {
                    const uint32_t m = sm.mem[mb ^ 1][p];
                    loc = sm.loc[m];
                    if (loc & kLocGather) mm[k] = m;
                }
                window_load(R.packed, loc & kLocBaseMask, loc_take(loc), mm[k] != ~0u, wd[k]);
            }
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                if (mm[k] == ~0u) continue;
                window_store(wd[k], sm, (int)mm[k]);
                sm.loc[mm[k]] &= ~kLocGather;
            }
            __syncthreads();
        }
    }

    // ---- emit what became final here; publish head bits for the global path ----------------------------
#pragma unroll
    for (int k = 0; k < kLocalItems; ++k) {
        const int e = k * kLocalThreads + tid;
        if (((state >> (2 * k)) & 3u) == 2) out[base + e] = sm.sym[e];
    }
    if (!FIRST) {   // FIRST: the warp kernel has published every position of a group of at most cap members as placed
        for (int i = tid; i < kLocalWords; i += kLocalThreads) {
            if (w0 + i > n_words) continue;
            const uint32_t add = sm.hw[i] & ~sm.hw0[i];
            if (add) atomicOr(&heads[w0 + i], add);
        }
    }
    // one statistics update per block (hundreds of thousands of atomics on one address would serialise in L2)
    __shared__ uint32_t s_done, s_cmp;
    if (tid == 0) s_done = 0, s_cmp = 0;
    __syncthreads();
    for (int o = 16; o; o >>= 1) {
        n_active += __shfl_xor_sync(kFull, n_active, o);
        n_compares += __shfl_xor_sync(kFull, n_compares, o);
    }
    if (lane_id() == 0 && n_active) atomicAdd(&s_done, n_active), atomicAdd(&s_cmp, n_compares);
    __syncthreads();
    if (tid == 0 && s_done) {
        atomicAdd(elems_done, (unsigned long long)s_done);
        atomicAdd(elems_done + 2, (unsigned long long)s_cmp);
        atomicAdd(elems_done + 3, (unsigned long long)n_rounds);   // refinement rounds (diagnostic)
    }
}

// Persistent blocks over the tiles.  FIRST: only tiles in which the warp kernel met a group of 33..cap members (big_tiles bit).
template <typename KeyT, typename IdT, bool FIRST, bool PACKED>
__global__ void __launch_bounds__(kLocalThreads, kLocalBlocksPerSM) finish_tile_kernel(Reads R, const KeyT* __restrict__ keys1,
                                                                    const uint32_t* __restrict__ heads_in, uint32_t* __restrict__ heads,
                                                                    const IdT* __restrict__ ids, uint64_t n, uint32_t depth0, uint32_t min_group,
                                                                    uint32_t cap, const uint32_t* __restrict__ big_tiles, uint8_t* __restrict__ out,
                                                                    unsigned long long* elems_done, uint32_t split) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    LocalSmem& sm = *reinterpret_cast<LocalSmem*>(smem_raw);
    const uint64_t n_tiles = (n + kLocalTile - 1) / kLocalTile;
    if constexpr (!FIRST) {
        // After a global round nearly every tile has nothing left to do, and finding that out inside finish_tile costs the whole
        // block a barrier per tile.  So the tiles go by in eights: each warp looks at the head words of one tile (the same test as
        // finish_tile's: does a group of two or more start at one of its positions?), and only the tiles that pass get the block.
        constexpr uint32_t kPer = kLocalThreads / 32;
        __shared__ uint32_t s_todo;
        const uint64_t n_words = (n + 31) >> 5;
        const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
        for (uint64_t t0 = (uint64_t)blockIdx.x * kPer; t0 < n_tiles; t0 += (uint64_t)gridDim.x * kPer) {
            if (threadIdx.x == 0) s_todo = 0;
            __syncthreads();
            const uint64_t tile = t0 + warp;
            uint32_t incomplete = 0;
            if (tile < n_tiles && lane <= (uint32_t)kLocalTile / 32) {
                const uint64_t wi = tile * (kLocalTile / 32) + lane;
                const uint32_t v = wi <= n_words ? heads_in[wi] : kFull;
                const uint32_t care = lane == 0 ? ~1u : (lane == (uint32_t)kLocalTile / 32 ? 1u : kFull);
                incomplete = (~v) & care;
            }
            if (__any_sync(kFull, incomplete != 0) && lane == 0) atomicOr(&s_todo, 1u << warp);
            __syncthreads();
            uint32_t todo = s_todo;
            while (todo) {
                const uint32_t w = (uint32_t)__ffs(todo) - 1;
                todo &= todo - 1;
                finish_tile<KeyT, IdT, FIRST, PACKED>(sm, t0 + w, R, keys1, heads_in, heads, ids, n, depth0, min_group, cap, out, elems_done, split);
                __syncthreads();   // the next tile reuses the shared memory
            }
        }
    } else {
        for (uint64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (!((__ldg(big_tiles + (tile >> 5)) >> (tile & 31)) & 1u)) continue;   // only the tiles the warp kernel flagged
            finish_tile<KeyT, IdT, FIRST, PACKED>(sm, tile, R, keys1, heads_in, heads, ids, n, depth0, min_group, cap, out, elems_done, split);
            __syncthreads();   // the next tile reuses the shared memory
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a7 + a8 for the common case, one WARP per chunk of sorted positions: tie groups of at most 32 S suffixes (coverage-sized
// groups of short-read collections; S = 2 slots per lane) never leave the registers of a warp.
//
// A warp walks its chunk in windows of 32 S positions that start at a group head; position p of the window lives in
// slot p / 32 of lane p % 32.  Groups that end inside the window are finished at once, the one cut by the window's end
// starts the next window.  Per window:
//   head flags from adjacent first-round keys (one shuffle); every position decodes its suffix id and gathers the base
//   before the suffix and -- members of a group of two or more -- its window of the next 96 bases, ONCE, as six 32-bit
//   words (bases past the end of the read are whatever follows in the packed text: they are never looked at);
//   the group's pivot is its member with the most bases (segmented max scan); its window reaches the others by shuffles;
//   one XOR + count-leading-zeros against the pivot gives where a member first differs from it, a second one where it
//   differs next (a pivot with a sequencing error sends its whole group to the same first divergence; the second level
//   orders them without another round): key = [group's first position : 6][level 1 : 10][level 2 : 10][index in group : 6];
//   a bitonic sort of the window's keys ranks every group stably and keeps groups in place;
//   classes that share a key and did not END there go round again (their data follows them by shuffles).
// Singletons and finished members are emitted as coalesced byte stores.
// Groups of more than 32 S and at most cap suffixes are left to the block kernel (their tile is flagged); larger ones to
// the global path (only their head bit is published, their ids handed over, and they are counted).
// ---------------------------------------------------------------------------------------------
#ifndef CX_WARP_MINB
#define CX_WARP_MINB 3
#endif
// sorted positions per warp (a chunk owns the groups that START in it): the larger one when the batch still fills the GPU
// several times over (fewer partly filled queue windows at the ends of chunks)
constexpr uint32_t kWarpChunkSmall = 2048, kWarpChunkLarge = 4096, kWarpChunkWaves = 8;
#ifndef CX_WARP_PREFETCH
#define CX_WARP_PREFETCH 8   // lanes that prefetch a 128-byte line of the following windows' keys (0: none)
#endif
#ifndef CX_WARP_QUEUE
#define CX_WARP_QUEUE 1
#endif
constexpr int kWarpThreads = 256;
// slots per lane: 2 (windows of 64 positions, two-level keys) unless the batch's tie groups are mostly larger, then 4
// (windows of 128 positions; the rank key has room for one level only)
constexpr int kWarpSlotsSmall = 2, kWarpSlotsLarge = 4;

// Event codes (the two levels of the rank key), order-preserving; 0 = no event:
//   1 + 5 d + s         below the pivot at base d: s = 0 my end-marker (FINAL: identical strings), 1..4 my base A..T
//   1 + kCodeEqual      equal to the pivot, which ends inside the window (FINAL);  + 1: equal through a full window, both go on
//   1 + kCodeAbove + 4 (95 - d) + b   above the pivot at base d, my base b = 0..3 there
constexpr uint32_t kCodeEqual = kWin * 5, kCodeAbove = kCodeEqual + 2;
// what a code says about the class of members that share it: 0 no event, 1 FINAL, 2 next window needed, 3 a base mismatch
__device__ __forceinline__ uint32_t code_type(uint32_t c) {
    const uint32_t k = c - 1;
    const uint32_t r = k - 5u * ((k * 13108u) >> 16);            // k % 5 for k < 2^13
    const bool fin = k == kCodeEqual || (k < kCodeEqual && r == 0);
    return c == 0 ? 0u : fin ? 1u : k == kCodeEqual + 1 ? 2u : 3u;
}

struct Win6 {
    uint32_t w[6];   // 16 bases per word, first base in the most significant bits
};
// Where window a (ta bases) differs from the pivot's window b (tb >= ta bases: the pivot is its group's longest member):
// the first two events (see the codes above).  Bases at or past ta are never looked at.
// (Every array index below is a compile-time constant: a data-dependent one would move the windows to local memory.)
__device__ __forceinline__ void diverge2(const Win6& a, const Win6& b, uint32_t ta, uint32_t tb, uint32_t& c1, uint32_t& c2) {
    uint32_t x[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) x[i] = a.w[i] ^ b.w[i];
    // first base at which the windows differ (kWin: none), the XOR word it is in and my word there
    uint32_t d = kWin, xw = 0, aw = 0;
#pragma unroll
    for (int i = 5; i >= 0; --i) {
        const bool hit = x[i] != 0;
        d = hit ? 16u * i + ((uint32_t)__clz(x[i]) >> 1) : d;
        xw = hit ? x[i] : xw;
        aw = hit ? a.w[i] : aw;
    }
    c2 = 0;
    if (d >= ta) {   // no base of mine differs: my end-marker against a base of the pivot ($ is the smallest symbol), or equal
        c1 = 1 + (ta < tb ? 5 * ta : (tb < kWin ? kCodeEqual : kCodeEqual + 1));
        return;
    }
    {
        const uint32_t sh = 30 - 2 * (d & 15);
        const uint32_t sa = (aw >> sh) & 3u, sb = sa ^ ((xw >> sh) & 3u);
        c1 = 1 + (sa < sb ? 5 * d + sa + 1 : kCodeAbove + 4 * (kWin - 1 - d) + sa);
        xw &= ~(3u << sh);   // forget this base: where do we differ next?
    }
    uint32_t d2 = kWin, xw2 = 0, aw2 = 0;
#pragma unroll
    for (int i = 5; i >= 0; --i) {
        const bool hit = x[i] != 0 && 16u * i > (d | 15u);   // words after the one of the first difference
        d2 = hit ? 16u * i + ((uint32_t)__clz(x[i]) >> 1) : d2;
        xw2 = hit ? x[i] : xw2;
        aw2 = hit ? a.w[i] : aw2;
    }
    if (xw) d2 = (d & ~15u) + ((uint32_t)__clz(xw) >> 1), xw2 = xw, aw2 = aw;   // the same word again
    if (d2 >= ta) {
        c2 = 1 + (ta < tb ? 5 * ta : (tb < kWin ? kCodeEqual : kCodeEqual + 1));
    } else {
        const uint32_t sh = 30 - 2 * (d2 & 15);
        const uint32_t sa = (aw2 >> sh) & 3u, sb = sa ^ ((xw2 >> sh) & 3u);
        c2 = 1 + (sa < sb ? 5 * d2 + sa + 1 : kCodeAbove + 4 * (kWin - 1 - d2) + sa);
    }
}

template <typename KeyT, bool PACKED>
__device__ __forceinline__ uint64_t load_keyword(const KeyT* __restrict__ keys1, uint64_t j) {
    if constexpr (PACKED) return __ldg(reinterpret_cast<const uint64_t*>(keys1) + j);   // key << 32 | id
    else return (uint64_t)__ldg(keys1 + j);
}

// first head at or after position p >= 1 (position n counts as one): a head starts a tie group
template <typename KeyT, bool PACKED>
__device__ __forceinline__ uint64_t scan_to_head(const KeyT* __restrict__ keys1, uint64_t p, uint64_t n, uint32_t split) {
    const uint32_t lane = lane_id();
    uint64_t carry = key_of<PACKED>(load_keyword<KeyT, PACKED>(keys1, p - 1), split);
    while (true) {
        const uint64_t j = p + lane;
        const uint64_t k = j < n ? key_of<PACKED>(load_keyword<KeyT, PACKED>(keys1, j), split) : 0ull;
        uint64_t kp = __shfl_up_sync(kFull, k, 1);
        if (lane == 0) kp = carry;
        const bool head = j >= n || k != kp || !((uint32_t)k & 1u);
        const uint32_t m = __ballot_sync(kFull, head);
        if (m) return p + (uint32_t)__ffs(m) - 1;
        carry = __shfl_sync(kFull, k, 31);
        p += 32;
    }
}

// The head bitmask of the global path starts as all ones (every position a group of one: placed); a group left to that
// path keeps only its first position's bit.  Clear the bits of positions [lo, hi); whole-warp call.
__device__ __forceinline__ void clear_heads(uint32_t* __restrict__ heads, uint64_t lo, uint64_t hi) {
    if (lo >= hi) return;
    const uint64_t w_lo = lo >> 5, w_hi = (hi - 1) >> 5;
    for (uint64_t w = w_lo + lane_id(); w <= w_hi; w += 32) {
        uint32_t m = kFull;
        if (w == w_lo) m &= kFull << (lo & 31);
        if (w == w_hi) m &= kFull >> (31 - ((hi - 1) & 31));
        if (m == kFull) heads[w] = 0u;          // a word inside one group has no other writer
        else atomicAnd(heads + w, ~m);
    }
}

// value of `v` at window position q (slot q / 32 of lane q % 32), for every lane its own q
// (written out per slot count: a loop over slots with a data-dependent pick ends up in local memory)
template <int S, typename T>
__device__ __forceinline__ T fetch_at(const T (&v)[S], uint32_t q) {
    static_assert(S == 1 || S == 2 || S == 4, "slots per lane");
    if constexpr (S == 1) {
        return __shfl_sync(kFull, v[0], q & 31);
    } else if constexpr (S == 2) {
        const T lo = __shfl_sync(kFull, v[0], q & 31), hi = __shfl_sync(kFull, v[1], q & 31);
        return (q & 32u) ? hi : lo;
    } else {
        const T a0 = __shfl_sync(kFull, v[0], q & 31), a1 = __shfl_sync(kFull, v[1], q & 31);
        const T a2 = __shfl_sync(kFull, v[2], q & 31), a3 = __shfl_sync(kFull, v[3], q & 31);
        const T lo = (q & 32u) ? a1 : a0, hi = (q & 32u) ? a3 : a2;
        return (q & 64u) ? hi : lo;
    }
}

// the packed bases from index b on, as six 32-bit words (16 bases each); loads only the words that `take` bases touch
__device__ __forceinline__ void window_words(const uint64_t* __restrict__ packed, uint64_t b, uint32_t take, bool want, Win6& out) {
    const uint32_t shift = (uint32_t)(b & 31) * 2;
    const uint32_t n_w = want && take ? (shift + 2 * take + 63) >> 6 : 0u;   // 64-bit words the window touches (<= 4)
    const uint64_t* p = packed + (b >> 5);
    uint32_t X[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint64_t v = i < (int)n_w ? __ldg(p + i) : 0ull;
        X[2 * i] = (uint32_t)(v >> 32);
        X[2 * i + 1] = (uint32_t)v;
    }
    const bool odd = shift >= 32;
    const uint32_t sh = shift & 31;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        const uint32_t hi = odd ? X[i + 1] : X[i], lo = odd ? X[i + 2] : X[i + 1];
        out.w[i] = __funnelshift_l(lo, hi, sh);
    }
}

// Group bounds of every window position from head bits (bit i of hb[s]: position 32 s + i starts a group; bit 0 of hb[S], the
// position after the window, is set): gs = the last head at or below the position, ge = the next head above it.
template <int S>
__device__ __forceinline__ void bounds_from_heads(const uint32_t (&hb)[S + 1], uint32_t lane, uint32_t (&gs)[S], uint32_t (&ge)[S]) {
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const uint32_t p = 32 * s + lane;
        uint32_t lo_bits = hb[s] & (0xffffffffu >> (31 - lane));
        gs[s] = 32 * s + 31 - (uint32_t)__clz(lo_bits);
#pragma unroll
        for (int t = s - 1; t >= 0; --t)
            if (!lo_bits && hb[t]) lo_bits = 1, gs[s] = 32 * t + 31 - (uint32_t)__clz(hb[t]);
        uint32_t hi_bits = lane == 31 ? 0u : hb[s] >> (lane + 1);
        ge[s] = p + (uint32_t)__ffs(hi_bits);
#pragma unroll
        for (int t = s + 1; t <= S; ++t)
            if (!hi_bits && hb[t]) hi_bits = 1, ge[s] = 32 * t + (uint32_t)__ffs(hb[t]) - 1;
    }
}

// Members whose class is still open after the first round of their window wait here, one queue per warp, and are refined
// again in dense windows of whole classes (a second round over the sparse leftovers of one window costs as much as a full
// one).  A ring of kQueueCap entries, structure of arrays; an entry is a member's state between two rounds.
constexpr uint32_t kQueueCap = 128, kQueueTake = 64;
struct WarpQueue {
    uint32_t win[6][kQueueCap];
    uint64_t wbase[kQueueCap];
    uint32_t mrem[kQueueCap];
    uint32_t meta[kQueueCap];   // symbol code | first of its class << 3 | (sorted position - start of the warp's chunk) << 4
};

template <typename KeyT, typename IdT, bool PACKED, int S>
__global__ void __launch_bounds__(kWarpThreads, S == 4 ? 2 : CX_WARP_MINB) finish_warp_kernel(Reads R, const KeyT* __restrict__ keys1, const IdT* __restrict__ ids_in,
                                                                   IdT* __restrict__ ids_out, uint64_t n, uint32_t depth0, uint32_t cap, uint32_t* __restrict__ heads,
                                                                   uint32_t* __restrict__ big_tiles, uint8_t* __restrict__ out,
                                                                   unsigned long long* counters, uint32_t chunk, uint32_t split) {
    constexpr uint32_t kSpan = 32 * S;                  // positions per window
    constexpr uint32_t kPosBits = S == 1 ? 5 : S == 2 ? 6 : 7;   // bits of a window position
    constexpr bool kTwoLevels = 2 * kPosBits + 20 <= 32;         // room for the second event in the 32-bit rank key
    constexpr uint32_t kClsBits = kTwoLevels ? 20 : 10;
    constexpr bool kQueue = CX_WARP_QUEUE && kSpan == kQueueTake;   // leftovers of a window's first round are queued
    constexpr bool kQueueAll = kQueue && CX_WARP_QUEUE >= 2;      // ... or every member, before its first round
    static_assert(S == 1 || S == 2 || S == 4, "slots per lane");
    static_assert(kWarpChunkLarge + kSpan < (1 << 28), "a queued position is kept in 28 bits");
    __shared__ WarpQueue s_queue[kQueue ? kWarpThreads / 32 : 1];
    WarpQueue& Q = s_queue[kQueue ? threadIdx.x >> 5 : 0];
    const uint32_t lane = lane_id();
    const uint64_t c0 = ((uint64_t)blockIdx.x * (kWarpThreads / 32) + (threadIdx.x >> 5)) * chunk;
    const uint64_t c1 = c0 + chunk < n ? c0 + chunk : n;
    const uint32_t cap_a = cap < kSpan ? cap : kSpan;   // largest group finished here
    const uint64_t pos_mask = (1ull << R.pos_bits) - 1;
    uint32_t n_members = 0, n_sorts = 0, n_over = 0;     // lane 0's tallies
    uint64_t a = c0;
    if (c0 < n && c0 > 0) a = scan_to_head<KeyT, PACKED>(keys1, c0, n, split);   // groups that began before the chunk are the previous warp's
    // ---- the work item: a window of the sorted order [a, a + n_comp), or a window of queued members ---------------------------
    uint32_t hw[S + 1];                                  // bit i of hw[s]: position a + 32 s + i is a head
    uint32_t n_comp = 0;
    uint32_t gs[S], ge[S], code[S], take[S], mrem[S];
    uint64_t wbase[S];
    Win6 win[S];
    bool mine[S], member[S];
    IdT idv[S];
    uint32_t open = 0;                                   // lanes with a member of a group that is not finished
    bool queued = false;                                 // the item came from the queue
    uint32_t q_head = 0, q_count = 0, q_take = 0;
#pragma unroll
    for (int s = 0; s < S; ++s) mine[s] = false, member[s] = false, idv[s] = 0, code[s] = 0;

    // emit the finished positions of a sorted-order window; publish head bits (everything finished here counts as a group of
    // one from now on)
    auto emit_window = [&]() {
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const uint32_t p = 32 * s + lane;
            const uint64_t j = a + p;
            if (mine[s] && !member[s]) out[j] = (uint8_t)(0x544743412400ull >> (8 * code[s]));
            const bool active = p < n_comp && j < n;
            const bool over = active && !mine[s];             // a complete group of more than cap members (cap < 32 S only)
            if (__any_sync(kFull, over)) {                    // the global path's: clear all but its first position's head bit
                const bool over_head = over && ((hw[s] >> lane) & 1u);
                if (PACKED || split) {
                    if (over) ids_out[j] = idv[s];
                }
                const uint32_t clear = __ballot_sync(kFull, over && !over_head), over_heads = __ballot_sync(kFull, over_head);
                const uint64_t at = a + 32 * s;
                const uint32_t sh = (uint32_t)(at & 31);
                if (lane == 0 && (clear << sh)) atomicAnd(heads + (at >> 5), ~(clear << sh));
                if (lane == 1 && sh && (clear >> (32 - sh))) atomicAnd(heads + (at >> 5) + 1, ~(clear >> (32 - sh)));
                if (lane == 0) n_over += (uint32_t)__popc(over_heads);
            }
        }
    };

    while (true) {
        if (!open) {
            if (kQueue && (q_count >= kQueueTake || (a >= c1 && q_count))) {
                // ---- a window of queued members: whole classes, at most 32 S of them ----------------------------------------
                uint32_t meta[S];
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    const uint32_t i = 32 * s + lane;
                    meta[s] = i < q_count ? Q.meta[(q_head + i) & (kQueueCap - 1)] : 8u;
                }
                q_take = q_count;
                if (q_count > kSpan) {
                    q_take = kSpan;
                    if (!((Q.meta[(q_head + kSpan) & (kQueueCap - 1)] >> 3) & 1u)) {   // a class would be cut: stop at its head
#pragma unroll
                        for (int s = 0; s < S; ++s) {
                            const uint32_t hd = __ballot_sync(kFull, (meta[s] >> 3) & 1u);
                            if (hd) q_take = 32 * s + 31 - (uint32_t)__clz(hd);
                        }
                    }
                }
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    const uint32_t i = 32 * s + lane;
                    const uint32_t slot = (q_head + i) & (kQueueCap - 1);
                    const bool in = i < q_take;
                    member[s] = in;
                    mine[s] = false;
                    code[s] = meta[s] & 7u;
                    hw[s] = __ballot_sync(kFull, !in || ((meta[s] >> 3) & 1u));
                    mrem[s] = in ? Q.mrem[slot] : 0u;
                    take[s] = mrem[s] < kWin ? mrem[s] : kWin;
                    wbase[s] = Q.wbase[slot];
#pragma unroll
                    for (int w = 0; w < 6; ++w) win[s].w[w] = Q.win[w][slot];
                }
                hw[S] = 1;
                bounds_from_heads<S>(hw, lane, gs, ge);
                queued = true;
                open = 1;
            } else if (a < c1) {
                // ---- the window [a, a + 32 S): a is a head --------------------------------------------------------------
#if CX_WARP_PREFETCH
                {   // ask L2 for the keys of the windows after this one (eight lanes, one 128-byte line each): their loads are
                    // the first link of the next window's chain of dependent loads
                    constexpr uint32_t kWordBytes = PACKED ? 8 : sizeof(KeyT);
                    const uint64_t pf = (a + kSpan) * kWordBytes + 128ull * lane;
                    if (lane < CX_WARP_PREFETCH && pf < n * kWordBytes) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(keys1) + pf));
                }
#endif
                uint64_t word[S];
                {
                    uint64_t k[S];
#pragma unroll
                    for (int s = 0; s < S; ++s) {
                        const uint64_t j = a + 32 * s + lane;
                        word[s] = j < n ? load_keyword<KeyT, PACKED>(keys1, j) : 0ull;
                        k[s] = key_of<PACKED>(word[s], split);
                    }
                    uint32_t carry_in = 1;                           // head bit of the slot's first position
#pragma unroll
                    for (int s = 0; s < S; ++s) {
                        const uint64_t j = a + 32 * s + lane;
                        uint64_t kn = __shfl_down_sync(kFull, k[s], 1);   // key of the next position
                        const bool valid_next = j + 1 < n;
                        if (s + 1 < S) {
                            const uint64_t first_of_next_slot = __shfl_sync(kFull, k[s + 1 < S ? s + 1 : s], 0);
                            if (lane == 31) kn = first_of_next_slot;
                        } else if (lane == 31) {
                            kn = valid_next ? key_of<PACKED>(load_keyword<KeyT, PACKED>(keys1, j + 1), split) : 0ull;
                        }
                        const bool head_next = !valid_next || kn != k[s] || !((uint32_t)kn & 1u);
                        const uint32_t HN = __ballot_sync(kFull, head_next);
                        hw[s] = (HN << 1) | carry_in;
                        carry_in = HN >> 31;
                    }
                    hw[S] = carry_in;
                }
                // complete groups: everything before the last head, or the whole window if position a + 32 S is a head; groups that
                // start at or after the end of the chunk are the next warp's
                n_comp = kSpan;
                if (!hw[S]) {
                    n_comp = 0;
#pragma unroll
                    for (int s = 0; s < S; ++s)
                        if (hw[s]) n_comp = 32 * s + 31 - (uint32_t)__clz(hw[s]);
                }
                if (a + n_comp > c1) {                               // c1 - a is 1 .. 32 S - 1 here
                    const uint32_t cut = (uint32_t)(c1 - a);
                    uint32_t first_later = n_comp;
#pragma unroll
                    for (int s = S - 1; s >= 0; --s) {
                        const uint32_t from = cut > 32u * s ? cut - 32u * s : 0u;
                        const uint32_t later = from >= 32 ? 0u : hw[s] & ~((1u << from) - 1);
                        if (later) first_later = 32 * s + (uint32_t)__ffs(later) - 1;
                    }
                    n_comp = min(n_comp, first_later);
                }
                if (n_comp == 0) {
                    // one group fills the window and goes on: more than 32 S members
                    const uint64_t e = scan_to_head<KeyT, PACKED>(keys1, a + kSpan, n, split);
                    const uint64_t g = e - a;
                    if (g <= cap) {          // the block kernel's: flag the tile it starts in
                        if (lane == 0) atomicOr(big_tiles + (a / kLocalTile >> 5), 1u << (a / kLocalTile & 31));
                    } else {                 // the global path's: only its first position stays a head; hand its ids over, count it
                        clear_heads(heads, a + 1, e);
                        if constexpr (PACKED) {
                            for (uint64_t q = a + lane; q < e; q += 32) ids_out[q] = (IdT)(uint32_t)load_keyword<KeyT, PACKED>(keys1, q);
                        } else if (split) {
                            for (uint64_t q = a + lane; q < e; q += 32) ids_out[q] = split_id<IdT>(load_keyword<KeyT, PACKED>(keys1, q), split, ids_in, q);
                        }
                        n_over += 1;
                    }
                    a = e;
                    continue;
                }
                // a head closes the complete part
#pragma unroll
                for (int s = 0; s <= S; ++s) {
                    const int lim = (int)n_comp - 32 * s;       // positions of this slot before the closing head
                    const uint32_t keep = lim >= 32 ? kFull : lim <= 0 ? 0u : (1u << lim) - 1;
                    const uint32_t close = lim >= 0 && lim < 32 ? 1u << lim : 0u;
                    hw[s] = (hw[s] & keep) | close;
                }
                // ---- my groups inside the window; locators, the base before every suffix, the members' windows: one batch of gathers -----
                bounds_from_heads<S>(hw, lane, gs, ge);
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    const uint32_t p = 32 * s + lane;
                    const uint64_t j = a + p;
                    const bool active = p < n_comp && j < n;
                    if (!active) gs[s] = p, ge[s] = p + 1;
                    const uint32_t size = ge[s] - gs[s];
                    mine[s] = active && size <= cap_a;              // (a complete group larger than cap_a exists only when cap < 32 S)
                    member[s] = mine[s] && size >= 2;
                    idv[s] = 0;
                    if (active) {
                        if constexpr (PACKED) idv[s] = (IdT)(uint32_t)word[s];
                        else idv[s] = split ? split_id<IdT>(word[s], split, ids_in, j) : __ldg(ids_in + j);
                    }
                }
                uint64_t before[S], first_base[S];
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    uint64_t left;
                    const uint64_t read = (uint64_t)idv[s] >> R.pos_bits, pos = (uint64_t)idv[s] & pos_mask;
                    if (R.uniform) {
                        first_base[s] = read * R.uniform_len + pos;
                        left = R.uniform_len - pos;
                    } else {
                        const uint64_t* q = R.offsets + (mine[s] ? read : 0ull);
                        const uint64_t lo = __ldg(q), hi = __ldg(q + 1);
                        first_base[s] = lo + pos;
                        left = hi - lo - pos;
                    }
                    const bool has_prev = mine[s] && pos;
                    before[s] = has_prev ? __ldg(R.packed + ((first_base[s] - 1) >> 5)) : 0ull;   // no load for a read's first suffix
                    wbase[s] = first_base[s] + depth0;                // index of the window's first base
                    mrem[s] = member[s] ? (uint32_t)(left - depth0) : 0u;   // a member of an open group has >= depth0 bases
                    take[s] = mrem[s] < kWin ? mrem[s] : kWin;
                    code[s] = has_prev ? 2u : 1u;                     // 1 = $: the suffix starts its read
                }
#pragma unroll
                for (int s = 0; s < S; ++s) window_words(R.packed, wbase[s], take[s], member[s], win[s]);
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    if (code[s] == 2u) code[s] = 2 + (uint32_t)((before[s] >> (62 - 2 * ((first_base[s] - 1) & 31))) & 3u);
                    const uint32_t mb = __ballot_sync(kFull, member[s]);
                    open |= mb;
                    if (lane == 0) n_members += (uint32_t)__popc(mb);
                }
                queued = false;
            } else {
                break;
            }
        }
        // ---- one round over the item's open groups -----------------------------------------------------------------------------
        uint32_t hb[S + 1];
#pragma unroll
        for (int s = 0; s <= S; ++s) hb[s] = hw[s];
        if (open && (queued || !kQueueAll)) {
            // pivot of every group: its member with the most bases in its window (segmented max scan, read at the group's last position)
            uint32_t best[S];
#pragma unroll
            for (int s = 0; s < S; ++s) best[s] = member[s] ? (take[s] << kPosBits) | (32 * s + lane) : 0u;
#pragma unroll
            for (uint32_t o = 1; o < 32; o <<= 1) {
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    const uint32_t v = __shfl_up_sync(kFull, best[s], o);
                    if (lane >= o && 32 * s + lane >= gs[s] + o && v > best[s]) best[s] = v;
                }
            }
#pragma unroll
            for (int s = 1; s < S; ++s) {                    // a group that began in the slot before
                const uint32_t carry = __shfl_sync(kFull, best[s - 1], 31);
                if (gs[s] < 32u * s && carry > best[s]) best[s] = carry;
            }
            uint32_t key[S];
            uint32_t c1v[S], tbv[S];
            Win6 piv[S];
#pragma unroll
            for (int s = 0; s < S; ++s) {
                const uint32_t tot = fetch_at<S>(best, ge[s] - 1);
                const uint32_t pp = tot & (kSpan - 1);
                tbv[s] = tot >> kPosBits;
#pragma unroll
                for (int i = 0; i < 6; ++i) {
                    uint32_t col[S];
#pragma unroll
                    for (int t = 0; t < S; ++t) col[t] = win[t].w[i];
                    piv[s].w[i] = fetch_at<S>(col, pp);
                }
            }
            uint32_t c2v[S];
#pragma unroll
            for (int s = 0; s < S; ++s) {
                c1v[s] = 0, c2v[s] = 0;
                if (member[s]) diverge2(win[s], piv[s], take[s], tbv[s], c1v[s], c2v[s]);
            }
#pragma unroll
            for (int s = 0; s < S; ++s) {
                const uint32_t p = 32 * s + lane;
                key[s] = member[s] ? (gs[s] << (32 - kPosBits)) | (c1v[s] << (kPosBits + kClsBits - 10)) | (kTwoLevels ? c2v[s] << kPosBits : 0u) | (p - gs[s])
                                   : p << (32 - kPosBits);   // a position outside every open group keeps its place
            }
            // bitonic sort of the window: groups stay in place (their first position leads the key), members are ranked inside
#pragma unroll
            for (uint32_t kk = 2; kk <= kSpan; kk <<= 1) {
#pragma unroll
                for (uint32_t jj = kk >> 1; jj > 0; jj >>= 1) {
                    if (jj >= 32) {                         // partner in the other slot of the same lane
#pragma unroll
                        for (int s = 0; s < S; ++s) {
                            const int t = s ^ (int)(jj >> 5);
                            if (t > s) {
                                const uint32_t lo = key[s] < key[t] ? key[s] : key[t], hi = key[s] < key[t] ? key[t] : key[s];
                                const bool up = ((32u * s) & kk) == 0;
                                key[s] = up ? lo : hi;
                                key[t] = up ? hi : lo;
                            }
                        }
                    } else {
#pragma unroll
                        for (int s = 0; s < S; ++s) {
                            const uint32_t p = 32 * s + lane;
                            const uint32_t other = __shfl_xor_sync(kFull, key[s], jj);
                            const bool keep_min = ((p & kk) == 0) == ((p & jj) == 0);
                            key[s] = keep_min ? (key[s] < other ? key[s] : other) : (key[s] > other ? key[s] : other);
                        }
                    }
                }
            }
            if (lane == 0) n_sorts += 1;
            // the member that ranked at each position; classes = runs of equal (level 1, level 2)
            uint32_t src[S], cls[S];
            bool head[S], was[S], nextwin[S];
#pragma unroll
            for (int s = 0; s < S; ++s) {
                src[s] = (key[s] >> (32 - kPosBits)) + (key[s] & (kSpan - 1));
                cls[s] = (key[s] >> kPosBits) & ((1u << kClsBits) - 1);
            }
#pragma unroll
            for (int s = 0; s < S; ++s) was[s] = cls[s] != 0;   // a member's level-1 code is never 0
#pragma unroll
            for (int s = 0; s < S; ++s) {
                const uint32_t p = 32 * s + lane;
                uint32_t prev = __shfl_up_sync(kFull, cls[s], 1);
                if (s > 0) {
                    const uint32_t last = __shfl_sync(kFull, cls[s > 0 ? s - 1 : 0], 31);
                    if (lane == 0) prev = last;
                }
                const uint32_t t1 = code_type(kTwoLevels ? cls[s] >> 10 : cls[s]);
                // the class's last event decides (with one level a base mismatch simply goes round again)
                const uint32_t ty = kTwoLevels && t1 == 3 && (cls[s] & 0x3ffu) ? code_type(cls[s] & 0x3ffu) : t1;
                nextwin[s] = ty == 2;
                head[s] = !was[s] || p == (key[s] >> (32 - kPosBits)) || ty == 1 || cls[s] != prev;
                hb[s] = __ballot_sync(kFull, head[s]);
            }
            hb[S] = 1;
            open = 0;
            bool still[S];
#pragma unroll
            for (int s = 0; s < S; ++s) {
                const uint32_t hn = lane == 31 ? hb[s + 1] & 1u : (hb[s] >> (lane + 1)) & 1u;
                still[s] = was[s] && !(head[s] && hn);      // not alone in my class yet
                open |= __ballot_sync(kFull, still[s]);
            }
            // my data follows me
            {
                uint32_t t32[S];
#pragma unroll
                for (int s = 0; s < S; ++s) t32[s] = code[s];
                uint32_t r[S];
#pragma unroll
                for (int s = 0; s < S; ++s) r[s] = fetch_at<S>(t32, src[s]);
#pragma unroll
                for (int s = 0; s < S; ++s) code[s] = r[s];
            }
            if (open) {
                uint32_t col[S], r[S];
#pragma unroll
                for (int i = 0; i < 6; ++i) {
#pragma unroll
                    for (int s = 0; s < S; ++s) col[s] = win[s].w[i];
#pragma unroll
                    for (int s = 0; s < S; ++s) r[s] = fetch_at<S>(col, src[s]);
#pragma unroll
                    for (int s = 0; s < S; ++s) win[s].w[i] = r[s];
                }
#pragma unroll
                for (int s = 0; s < S; ++s) col[s] = mrem[s];
#pragma unroll
                for (int s = 0; s < S; ++s) r[s] = fetch_at<S>(col, src[s]);
#pragma unroll
                for (int s = 0; s < S; ++s) mrem[s] = r[s], take[s] = r[s] < kWin ? r[s] : kWin;
                uint64_t r64[S];
#pragma unroll
                for (int s = 0; s < S; ++s) r64[s] = fetch_at<S>(wbase, src[s]);
#pragma unroll
                for (int s = 0; s < S; ++s) wbase[s] = r64[s];
            }
#pragma unroll
            for (int s = 0; s < S; ++s) member[s] = still[s];
            if (open) {
            bool any_next = false;
            bounds_from_heads<S>(hb, lane, gs, ge);
#pragma unroll
            for (int s = 0; s < S; ++s) any_next |= __any_sync(kFull, member[s] && nextwin[s]);
            if (any_next) {                                 // equal to the pivot through a full window: the next window of the read
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    const bool g = member[s] && nextwin[s];
                    if (g) {
                        wbase[s] += kWin;
                        mrem[s] -= kWin;
                        take[s] = mrem[s] < kWin ? mrem[s] : kWin;
                    }
                    Win6 nw;
                    window_words(R.packed, wbase[s], take[s], g, nw);
                    if (g) win[s] = nw;
                }
            }
            }
        }
        if (!queued) {
            if (kQueue) {
                // the window's finished positions are emitted now; the members of its open classes wait in the queue
                emit_window();
                if (open) {
                    uint32_t at = q_head + q_count;
#pragma unroll
                    for (int s = 0; s < S; ++s) {
                        const uint32_t mb = __ballot_sync(kFull, member[s]);
                        if (member[s]) {
                            const uint32_t slot = (at + (uint32_t)__popc(mb & ((1u << lane) - 1))) & (kQueueCap - 1);
#pragma unroll
                            for (int w = 0; w < 6; ++w) Q.win[w][slot] = win[s].w[w];
                            Q.wbase[slot] = wbase[s];
                            Q.mrem[slot] = mrem[s];
                            Q.meta[slot] = code[s] | (((hb[s] >> lane) & 1u) << 3) | ((uint32_t)(a + 32 * s + lane - c0) << 4);
                        }
                        at += (uint32_t)__popc(mb);
                    }
                    q_count = at - q_head;
                    __syncwarp();
                    open = 0;
                }
                a += n_comp;
            } else if (!open) {
                emit_window();
                a += n_comp;
            }
        } else if (!open) {
            // the queued window is finished: its symbols go to the positions its members were queued from
#pragma unroll
            for (int s = 0; s < S; ++s) {
                const uint32_t i = 32 * s + lane;
                if (i < q_take) out[c0 + (Q.meta[(q_head + i) & (kQueueCap - 1)] >> 4)] = (uint8_t)(0x544743412400ull >> (8 * code[s]));
            }
            __syncwarp();
            q_head += q_take;
            q_count -= q_take;
        }
    }
    // ---- tallies: one update per block ------------------------------------------------------------------------------------------
    __shared__ uint32_t s_tally[3];
    if (threadIdx.x < 3) s_tally[threadIdx.x] = 0;
    __syncthreads();
    if (lane == 0) {
        if (n_members) atomicAdd(&s_tally[0], n_members);
        if (n_sorts) atomicAdd(&s_tally[1], n_sorts);
        if (n_over) atomicAdd(&s_tally[2], n_over);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_tally[0]) atomicAdd(counters, (unsigned long long)s_tally[0]);                       // suffixes refined here
        if (s_tally[1]) atomicAdd(counters + 2, (unsigned long long)s_tally[1] * (S == 1 ? 80 : 192));   // rank-key comparisons of the sorts
        if (s_tally[1]) atomicAdd(counters + 3, (unsigned long long)s_tally[1]);                  // refinement rounds (warp windows)
        if (s_tally[2]) atomicAdd(counters + 4, (unsigned long long)s_tally[2]);                  // groups left to the global path
    }
}

// How large are the tie groups of this batch?  A sample of windows of 2048 sorted positions: positions that sit in a run of
// more than `limit` equal first-round keys (runs are cut at the window's ends, so this underestimates).  Decides the window
// width of the warp kernel.  counter[0] += such positions.
constexpr int kProbeSpan = 2048, kProbeBlocks = 128;
template <typename KeyT, bool PACKED>
__global__ void __launch_bounds__(256) group_probe_kernel(const KeyT* __restrict__ keys1, uint64_t n, uint32_t limit,
                                                          unsigned long long* counter, uint32_t split) {
    __shared__ uint32_t s_heads[kProbeSpan / 32 + 1];
    __shared__ uint32_t s_big;
    const uint64_t stride = n / gridDim.x;
    const uint64_t a = (uint64_t)blockIdx.x * stride;
    if (threadIdx.x == 0) s_big = 0, s_heads[kProbeSpan / 32] = 1u;
#pragma unroll
    for (int k = 0; k < kProbeSpan / 256; ++k) {
        const uint32_t e = k * 256 + threadIdx.x;
        const uint64_t j = a + e;
        bool head = true;
        if (j < n && e > 0) {
            const uint64_t kc = key_of<PACKED>(load_keyword<KeyT, PACKED>(keys1, j), split), kp = key_of<PACKED>(load_keyword<KeyT, PACKED>(keys1, j - 1), split);
            head = kc != kp || !((uint32_t)kc & 1u);
        }
        const uint32_t word = __ballot_sync(kFull, head);
        if ((threadIdx.x & 31) == 0) s_heads[e >> 5] = word;
    }
    __syncthreads();
    uint32_t big = 0;
#pragma unroll
    for (int k = 0; k < kProbeSpan / 256; ++k) {
        const int e = k * 256 + (int)threadIdx.x;
        if (a + e >= n) continue;
        const int ps = prev_head(s_heads, e, 0), ne = next_head(s_heads, e, kProbeSpan);
        big += (uint32_t)((ne < 0 ? kProbeSpan : ne) - ps > (int)limit);
    }
    for (int o = 16; o; o >>= 1) big += __shfl_xor_sync(kFull, big, o);
    if ((threadIdx.x & 31) == 0 && big) atomicAdd(&s_big, big);
    __syncthreads();
    if (threadIdx.x == 0 && s_big) atomicAdd(counter, (unsigned long long)s_big);
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
cudaError_t launch_active_count(const uint32_t* heads, uint64_t n, uint64_t* word_counts, cudaStream_t s) {
    uint64_t n_words = (n + 31) >> 5;
    if (n_words == 0) return cudaSuccess;
    active_count_kernel<<<(unsigned)((n_words + 255) / 256), 256, 0, s>>>(heads, n_words, word_counts);
    return cudaGetLastError();
}

uint64_t scan_block_count(uint64_t n) { return (n + kScanChunk - 1) / kScanChunk; }

cudaError_t launch_scan_u64(uint64_t* data, uint64_t n, uint64_t* block_sums, uint64_t* total, cudaStream_t s) {
    if (n == 0) return cudaMemsetAsync(total, 0, sizeof(uint64_t), s);
    uint64_t blocks = scan_block_count(n);
    scan_reduce_kernel<<<(unsigned)blocks, kScanThreads, 0, s>>>(data, n, block_sums);
    scan_sums_kernel<<<1, kScanThreads, 0, s>>>(block_sums, blocks, total);
    scan_down_kernel<<<(unsigned)blocks, kScanThreads, 0, s>>>(data, n, block_sums);
    return cudaGetLastError();
}

template <typename IdT>
cudaError_t launch_refine_rekey(const Reads& R, const uint32_t* heads, const uint64_t* word_base, const IdT* ids, uint64_t n,
                                uint32_t depth, uint32_t w, uint64_t* keys_c, uint32_t* pos_c, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    const uint64_t n_words = (n + 31) >> 5;
    refine_rekey_kernel<IdT><<<(unsigned)((n_words + 255) / 256), 256, 0, s>>>(R, heads, word_base, ids, n, depth, w, keys_c, pos_c);
    return cudaGetLastError();
}

template <typename IdT>
cudaError_t launch_refine_writeback(const Reads& R, const uint64_t* keys_c, const uint32_t* pos_sorted, IdT* ids_tmp, const uint32_t* heads,
                                    const uint64_t* word_base, uint64_t n, uint64_t n_c, uint32_t w, IdT* ids, uint32_t* heads_out, uint8_t* out,
                                    cudaStream_t s) {
    if (n_c == 0) return cudaSuccess;
    refine_gather_kernel<IdT><<<(unsigned)((n_c + 255) / 256), 256, 0, s>>>(pos_sorted, n_c, ids, ids_tmp);
    const uint64_t n_words = (n + 31) >> 5;
    refine_writeback_kernel<IdT><<<(unsigned)((n_words + 255) / 256), 256, 0, s>>>(R, keys_c, ids_tmp, heads, word_base, n, n_c, w, ids, heads_out, out);
    return cudaGetLastError();
}

template <typename KeyT, typename IdT>
cudaError_t launch_finish_first(const Reads& R, const KeyT* keys1, uint32_t w1, uint32_t depth0, uint32_t* heads_out, IdT* ids, uint64_t n,
                                uint32_t group_cap, uint8_t* out, unsigned long long* elems_done, uint32_t* big_tiles, int n_sms, bool packed,
                                uint32_t slots, Launch* prof, cudaStream_t s, uint32_t split, IdT* ids_out) {
    if (n == 0) return cudaSuccess;
    constexpr bool kCanPack = sizeof(KeyT) == 4 && sizeof(IdT) == 4;
    if (packed && !kCanPack) return cudaErrorInvalidValue;
    if (split && (packed || sizeof(KeyT) != 8 || sizeof(IdT) != 8 || !ids_out || ids_out == ids)) return cudaErrorInvalidValue;
    if (!split) ids_out = ids;   // (separate arrays: the ids stay where they are; packed: the oversize groups' ids go there)
    if (slots != (uint32_t)kWarpSlotsSmall && slots != (uint32_t)kWarpSlotsLarge) return cudaErrorInvalidValue;
    (void)w1;   // (a first-round key says in its lowest bit whether its suffix has w1 bases)
    if (group_cap > (uint32_t)kLocalGroupCap) group_cap = kLocalGroupCap;
    const uint64_t tiles = (n + kLocalTile - 1) / kLocalTile;
    cudaError_t e = cudaMemsetAsync(big_tiles, 0, ((tiles + 31) / 32 + 1) * sizeof(uint32_t), s);
    if (e != cudaSuccess) return e;
    {   // singletons and groups of at most 32: one warp per chunk, registers only
        // a7 flagging (key + 1) and a8 emit (id + base + byte) per suffix; the refined suffixes' term is added by the caller
        ScopedLaunch sl(prof, CX_K_FINISH, n * ((split ? 12 : sizeof(KeyT) + sizeof(IdT)) + 1 + 2), s);
        const uint64_t resident_warps = (uint64_t)n_sms * (slots == (uint32_t)kWarpSlotsLarge ? 2 : CX_WARP_MINB) * (kWarpThreads / 32);
        const uint32_t chunk = n >= resident_warps * kWarpChunkWaves * kWarpChunkLarge ? kWarpChunkLarge : kWarpChunkSmall;
        const uint64_t warps = (n + chunk - 1) / chunk;
        const unsigned grid = (unsigned)((warps + kWarpThreads / 32 - 1) / (kWarpThreads / 32));
        auto launch = [&](auto kernel) { kernel<<<grid, kWarpThreads, 0, s>>>(R, keys1, ids, ids_out, n, depth0, group_cap, heads_out, big_tiles, out, elems_done, chunk, split); };
        if (slots == (uint32_t)kWarpSlotsLarge) {
            if (packed) launch(finish_warp_kernel<KeyT, IdT, kCanPack, kWarpSlotsLarge>);
            else launch(finish_warp_kernel<KeyT, IdT, false, kWarpSlotsLarge>);
        } else {
            if (packed) launch(finish_warp_kernel<KeyT, IdT, kCanPack, kWarpSlotsSmall>);
            else launch(finish_warp_kernel<KeyT, IdT, false, kWarpSlotsSmall>);
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (group_cap <= 32 * slots) return cudaSuccess;
    // larger groups, up to cap: persistent blocks over the flagged tiles
    auto kernel = packed ? finish_tile_kernel<KeyT, IdT, true, kCanPack> : finish_tile_kernel<KeyT, IdT, true, false>;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LocalSmem));
    if (e != cudaSuccess) return e;
    const uint64_t resident = (uint64_t)n_sms * kLocalBlocksPerSM;
    ScopedLaunch sl(prof, CX_K_FINISH_BLOCK, 0, s);
    kernel<<<(unsigned)(tiles < resident ? tiles : resident), kLocalThreads, sizeof(LocalSmem), s>>>(R, keys1, nullptr, nullptr, ids, n, depth0, 32u * slots + 1,
                                                                                                   group_cap, big_tiles, out, elems_done, split);
    return cudaGetLastError();
}

template <typename KeyT, typename IdT>
cudaError_t launch_group_probe(const KeyT* keys1, uint32_t w1, uint64_t n, bool packed, unsigned long long* counter, uint64_t* sampled, cudaStream_t s,
                               uint32_t split) {
    constexpr bool kCanPack = sizeof(KeyT) == 4 && sizeof(IdT) == 4;
    *sampled = 0;
    if (n < (uint64_t)kProbeSpan * 2) return cudaSuccess;
    const unsigned blocks = (unsigned)(n / kProbeSpan < (uint64_t)kProbeBlocks ? n / kProbeSpan : (uint64_t)kProbeBlocks);
    *sampled = (uint64_t)blocks * kProbeSpan;
    (void)w1;
    if (packed) group_probe_kernel<KeyT, kCanPack><<<blocks, 256, 0, s>>>(keys1, n, 32u * kWarpSlotsSmall, counter, 0u);
    else group_probe_kernel<KeyT, false><<<blocks, 256, 0, s>>>(keys1, n, 32u * kWarpSlotsSmall, counter, split);
    return cudaGetLastError();
}

template <typename IdT>
cudaError_t launch_finish_later(const Reads& R, const uint32_t* heads_in, uint32_t* heads_out, const IdT* ids, uint64_t n, uint32_t depth,
                                uint32_t group_cap, uint8_t* out, unsigned long long* elems_done, int n_sms, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    auto kernel = finish_tile_kernel<uint64_t, IdT, false, false>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LocalSmem));
    if (e != cudaSuccess) return e;
    if (group_cap > (uint32_t)kLocalGroupCap) group_cap = kLocalGroupCap;
    const uint64_t tiles = (n + kLocalTile - 1) / kLocalTile;
    const uint64_t resident = (uint64_t)n_sms * kLocalBlocksPerSM;
    kernel<<<(unsigned)(tiles < resident ? tiles : resident), kLocalThreads, sizeof(LocalSmem), s>>>(R, nullptr, heads_in, heads_out, ids, n, depth, 2u, group_cap,
                                                                                                   nullptr, out, elems_done, 0u);
    return cudaGetLastError();
}

#define CX_INSTANTIATE(IdT)                                                                                                          \
    template cudaError_t launch_refine_rekey<IdT>(const Reads&, const uint32_t*, const uint64_t*, const IdT*, uint64_t, uint32_t,   \
                                                  uint32_t, uint64_t*, uint32_t*, cudaStream_t);                                     \
    template cudaError_t launch_refine_writeback<IdT>(const Reads&, const uint64_t*, const uint32_t*, IdT*, const uint32_t*,        \
                                                      const uint64_t*, uint64_t, uint64_t, uint32_t, IdT*, uint32_t*, uint8_t*,      \
                                                      cudaStream_t);                                                                 \
    template cudaError_t launch_finish_first<uint32_t, IdT>(const Reads&, const uint32_t*, uint32_t, uint32_t, uint32_t*, IdT*, uint64_t, \
                                                            uint32_t, uint8_t*, unsigned long long*, uint32_t*, int, bool, uint32_t, Launch*, cudaStream_t, uint32_t, IdT*); \
    template cudaError_t launch_finish_first<uint64_t, IdT>(const Reads&, const uint64_t*, uint32_t, uint32_t, uint32_t*, IdT*, uint64_t, \
                                                            uint32_t, uint8_t*, unsigned long long*, uint32_t*, int, bool, uint32_t, Launch*, cudaStream_t, uint32_t, IdT*); \
    template cudaError_t launch_group_probe<uint32_t, IdT>(const uint32_t*, uint32_t, uint64_t, bool, unsigned long long*, uint64_t*, cudaStream_t, uint32_t); \
    template cudaError_t launch_group_probe<uint64_t, IdT>(const uint64_t*, uint32_t, uint64_t, bool, unsigned long long*, uint64_t*, cudaStream_t, uint32_t); \
    template cudaError_t launch_finish_later<IdT>(const Reads&, const uint32_t*, uint32_t*, const IdT*, uint64_t, uint32_t,         \
                                                  uint32_t, uint8_t*, unsigned long long*, int, cudaStream_t);
CX_INSTANTIATE(uint32_t)
CX_INSTANTIATE(uint64_t)

}  // namespace cx
