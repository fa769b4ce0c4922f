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

// ---------------------------------------------------------------------------------------------
// global path: compact + re-key, write back
// ---------------------------------------------------------------------------------------------
// One thread per 32 sorted positions looks for members still tied; the warp then handles every such word together,
// one lane per position (oversize groups are rare, so nearly all threads leave after one load).
template <typename IdT>
__global__ void __launch_bounds__(256) refine_rekey_kernel(Reads R, const uint32_t* __restrict__ heads,
                                                           const uint64_t* __restrict__ word_base, const IdT* __restrict__ ids,
                                                           uint64_t n, uint32_t depth, uint32_t w, uint64_t* __restrict__ keys_c,
                                                           IdT* __restrict__ ids_c, uint32_t* __restrict__ pos_c) {
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
            const uint64_t j = (wwi << 5) + bit;
            const uint32_t below = (1u << bit) - 1;
            const uint64_t c = (wbase & 0xffffffffull) + __popc(wact & below);
            const uint64_t g = (wbase >> 32) + __popc(wah & (below | (1u << bit))) - 1;   // ordinal of this element's group
            const IdT id = ids[j];
            keys_c[c] = (g << (2 * w + 5)) | key_at_depth(R, id, depth, w);
            ids_c[c] = id;
            pos_c[c] = (uint32_t)j;
        }
    }
}

template <typename IdT>
__global__ void __launch_bounds__(256) refine_writeback_kernel(Reads R, const uint64_t* __restrict__ keys_c, const IdT* __restrict__ ids_c,
                                                               const uint32_t* __restrict__ pos_c, uint64_t n_c, uint32_t w,
                                                               IdT* __restrict__ ids, uint32_t* __restrict__ heads, uint8_t* __restrict__ out) {
    uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_c) return;
    uint64_t k = keys_c[c];
    uint32_t pos = pos_c[c];
    IdT id = ids_c[c];
    ids[pos] = id;
    bool head = c == 0 || k != keys_c[c - 1] || (uint32_t)(k & 31) < w;
    if (head) atomicOr(&heads[pos >> 5], 1u << (pos & 31));
    // alone in its group now (or its end-marker was inside the window): final, emit its BWT symbol
    bool next_is_head = true;
    if (c + 1 < n_c) {
        uint64_t kn = keys_c[c + 1];
        next_is_head = kn != k || (uint32_t)(kn & 31) < w;
    }
    if (head && next_is_head) out[pos] = preceding_symbol(R, id);
}

// ---------------------------------------------------------------------------------------------
// a7 + a8 fused, one block per tile of kLocalTile sorted positions ("finish" kernel):
//   FIRST : head flags from the freshly sorted first-round keys; every suffix that is alone in its
//           group is final and its BWT symbol is emitted at once; groups of 2..cap suffixes that start
//           in the tile are refined to the end in shared memory and emitted; larger groups are left
//           to the global path (their head bits go to `heads`).
//   !FIRST: after a global round; head flags come from `heads`; only groups of 2..cap are touched.
// A position is emitted exactly once, by whoever makes it final (here, or the global write-back).
// ---------------------------------------------------------------------------------------------
constexpr int kLocalElems = kLocalTile + kLocalGroupCap;   // positions a block may touch
constexpr int kLocalWords = kLocalElems / 32 + 2;
constexpr int kLocalItems = kLocalElems / kLocalThreads;
static_assert(kLocalElems % kLocalThreads == 0 && kLocalThreads % 32 == 0, "tile shape");
constexpr uint32_t kLocalW = 88;                            // bases per in-block round (192-bit round key)
constexpr uint16_t kNone = 0xffff;
constexpr int kSubBlock = 32;                               // members ranked by counting before runs are merged

template <typename IdT>
struct LocalSmem {
    // round key, 192 bits: [88 bases, A-padded : 176][0 : 1][min(remaining, 88) : 7][index inside the group : 8]
    uint4 key_lo[kLocalElems];  // bits 0..127, .x least significant
    uint2 key_hi[kLocalElems];  // bits 128..191 = the first 32 bases
    uint64_t loc[kLocalElems];  // locator of the suffix now at this position (layout above); 0: not ours.  Holds the raw
                                // id between the head pass and the classify pass
    uint16_t ord[2][kLocalElems];  // sorted order of the runs being merged, ping-pong; at the end of a round
                                   // ord[cur][p] = member that ranks at position p
    uint16_t gs[kLocalElems];   // first position of the element's current group (kNone: not ours / placed)
    uint16_t ge[kLocalElems];   // one past its last position
    uint32_t hw[kLocalWords];   // head bits of the window, updated as groups split
    uint32_t hw0[kLocalWords];  // as loaded
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

// Locator of a suffix this block owns: everything the rounds and the emit need, so that the offsets table and the
// word before the suffix are read once per suffix, not once per round and again at the emit (each such gather is a
// 64-byte DRAM fetch on a collection larger than L2):
//   [code of the preceding symbol, 1 = $, 2..5 = A C G T : 3][bases from its first base to the end of the read : 21]
//   [index of its first base in the packed text : 40]
constexpr uint32_t kLocBaseBits = 40, kLocRemBits = 21;
__device__ __forceinline__ uint8_t loc_symbol(uint64_t loc) {
    return (uint8_t)(0x544743412400ull >> (8 * (uint32_t)(loc >> (kLocBaseBits + kLocRemBits))));
}

// 192-bit round key of the suffix with locator `loc` at depth d: the next 88 bases (A-padded), then min(remaining, 88),
// then the member's index inside its tie group -- so that one unsigned compare orders the group stably.
// One round covers a 100 bp read after a 14-base first sort.
struct Key192 {
    uint4 lo;   // bits 0..127
    uint2 hi;   // bits 128..191
};
// x with only its first cnt bases kept (cnt may be <= 0 or >= 32)
__device__ __forceinline__ uint64_t keep_bases(uint64_t x, int cnt) {
    return cnt >= 32 ? x : (cnt <= 0 ? 0ull : x & (~0ull << (64 - 2 * cnt)));
}
// w: the four packed words from the one that holds the window's first base (words the window does not touch are 0);
// shift: bit offset of that base in w[0]; take: bases of the window that exist (<= 88)
__device__ __forceinline__ Key192 key192_of_words(const uint64_t (&w)[4], uint32_t shift, uint32_t take, uint32_t idx) {
    uint64_t p0 = w[0], p1 = w[1], p2 = w[2];   // bases [0,32), [32,64), [64,88) of the window
    if (shift) {
        p0 = (w[0] << shift) | (w[1] >> (64 - shift));
        p1 = (w[1] << shift) | (w[2] >> (64 - shift));
        p2 = (w[2] << shift) | (w[3] >> (64 - shift));
    }
    p0 = keep_bases(p0, (int)take);
    p1 = keep_bases(p1, (int)take - 32);
    p2 = keep_bases(p2, (int)take - 64);        // at most 24 bases: the low 16 bits are clear
    const uint64_t k0 = p2 | ((uint64_t)take << 8) | idx;
    Key192 k;
    k.lo = make_uint4((uint32_t)k0, (uint32_t)(k0 >> 32), (uint32_t)p1, (uint32_t)(p1 >> 32));
    k.hi = make_uint2((uint32_t)p0, (uint32_t)(p0 >> 32));
    return k;
}

// acc -= (a < b) for 192-bit unsigned a, b: the borrow of a - b, seven instructions
__device__ __forceinline__ void count_if_less(uint32_t& acc, const uint4& alo, const uint2& ahi, const uint4& blo, const uint2& bhi) {
    asm("{\n\t.reg .u32 t;\n\t"
        "sub.cc.u32 t, %1, %7;\n\tsubc.cc.u32 t, %2, %8;\n\tsubc.cc.u32 t, %3, %9;\n\tsubc.cc.u32 t, %4, %10;\n\t"
        "subc.cc.u32 t, %5, %11;\n\tsubc.cc.u32 t, %6, %12;\n\t"
        "subc.u32 %0, %0, 0;\n\t}"
        : "+r"(acc)
        : "r"(alo.x), "r"(alo.y), "r"(alo.z), "r"(alo.w), "r"(ahi.x), "r"(ahi.y), "r"(blo.x), "r"(blo.y), "r"(blo.z), "r"(blo.w), "r"(bhi.x),
          "r"(bhi.y));
}

template <typename KeyT, typename IdT, bool FIRST, bool PACKED>
__global__ void __launch_bounds__(kLocalThreads, kLocalBlocksPerSM) finish_tile_kernel(Reads R, const KeyT* __restrict__ keys1, uint32_t w1, uint32_t len_mask,
                                                                    const uint32_t* __restrict__ heads_in, uint32_t* __restrict__ heads,
                                                                    IdT* __restrict__ ids, uint64_t n,
                                                                    uint32_t depth0, uint32_t cap, uint8_t* __restrict__ out,
                                                                    unsigned long long* elems_done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    LocalSmem<IdT>& sm = *reinterpret_cast<LocalSmem<IdT>*>(smem_raw);
    const uint64_t base = (uint64_t)blockIdx.x * kLocalTile;
    const uint64_t w0 = base >> 5;
    const uint64_t n_words = (n + 31) >> 5;   // heads[n_words] is the padding word ("the next position is a head")
    const int tid = threadIdx.x;

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
                    head = j == 0 || kc != (uint32_t)(__ldg(pairs + j - 1) >> 32) || (kc & len_mask) < w1;
                    sm.loc[e] = (uint32_t)pc;
                } else {
                    const KeyT kc = __ldcs(keys1 + j);
                    head = j == 0 || kc != __ldg(keys1 + j - 1) || ((uint32_t)kc & len_mask) < w1;
                    sm.loc[e] = (uint64_t)__ldcs(ids + j);
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
    // The kernel lives on random gathers (the offsets table, the word before the suffix, the key words); every batch
    // of them is issued for all of a thread's positions before the first is used, so their latencies overlap.
    uint32_t n_active = 0, n_compares = 0;
    IdT idv[kLocalItems];
    uint32_t state = 0;   // 2 bits per position: 0 not ours, 1 alone in its group (final), 2 member of a group refined here
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
                if (ne > 0) {
                    if (ne - ps >= 2) {
                        s = (uint16_t)ps;
                        t = (uint16_t)ne;
                        st = 2;
                        ++n_active;
                    } else if (FIRST) {
                        st = 1;
                    }
                }
            }
            if (FIRST) {
                idv[k] = (IdT)sm.loc[e];
                // packed input carries the ids inside the key words: hand those of the suffixes left to the global path over
                if (PACKED && !st && e < kLocalTile) ids[base + e] = idv[k];
            } else if (st) {
                idv[k] = ids[base + e];
            }
        }
        sm.gs[e] = s;
        sm.ge[e] = t;
        state |= st << (2 * k);
    }
    {
        uint64_t first_base[kLocalItems];   // index of the suffix's first base in the packed text
        uint32_t left[kLocalItems];         // bases from there to the end of its read
        const uint64_t pos_mask = (1ull << R.pos_bits) - 1;
        if (R.uniform) {
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const uint64_t read = (uint64_t)idv[k] >> R.pos_bits, pos = (uint64_t)idv[k] & pos_mask;
                first_base[k] = read * R.uniform_len + pos;
                left[k] = (uint32_t)(R.uniform_len - pos);
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
                left[k] = (uint32_t)(hi[k] - lo[k] - pos);
            }
        }
        uint64_t before[kLocalItems];       // the word that holds the base before the suffix
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const bool want = ((state >> (2 * k)) & 3u) && ((uint64_t)idv[k] & pos_mask);
            before[k] = want ? __ldg(R.packed + ((first_base[k] - 1) >> 5)) : 0ull;   // no load at all for a read's first suffix (packed may hold no word)
        }
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            const uint32_t st = (state >> (2 * k)) & 3u;
            uint64_t code = 1;   // $: the suffix starts its read
            if ((uint64_t)idv[k] & pos_mask) code = 2 + ((before[k] >> (62 - 2 * ((first_base[k] - 1) & 31))) & 3u);
            const uint64_t loc = (code << (kLocBaseBits + kLocRemBits)) | ((uint64_t)left[k] << kLocBaseBits) | first_base[k];
            if (FIRST && st == 1) out[base + e] = loc_symbol(loc);   // alone in its group after the first sort: final
            sm.loc[e] = st == 2 ? loc : 0ull;
        }
    }
    __syncthreads();

    // ---- rounds: one 88-base gather per member still tied, stable rank (see below) ----------------------
    for (uint32_t depth = depth0;; depth += kLocalW) {
        uint32_t any = 0;
#pragma unroll
        for (int kk = 0; kk < kLocalItems; kk += 2) {
            uint64_t w[2][4];
            uint32_t take[2], shift[2];
            int start[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int e = (kk + j) * kLocalThreads + tid;
                const bool exists = kk + j < kLocalItems;
                start[j] = exists ? sm.gs[e] : kNone;
                const uint64_t loc = exists ? sm.loc[e] : 0ull;
                const uint32_t remaining = start[j] != kNone ? (uint32_t)(loc >> kLocBaseBits) & ((1u << kLocRemBits) - 1) : 0u;
                const uint32_t rem = remaining > depth ? remaining - depth : 0u;
                take[j] = rem < kLocalW ? rem : kLocalW;
                const uint64_t b = (loc & ((1ull << kLocBaseBits) - 1)) + depth;
                shift[j] = (uint32_t)(b & 31) * 2;
                const uint32_t n_w = take[j] ? (shift[j] + 2 * take[j] + 63) >> 6 : 0u;   // words the window touches
                const uint64_t* p = R.packed + (b >> 5);
#pragma unroll
                for (int i = 0; i < 4; ++i) w[j][i] = i < (int)n_w ? __ldg(p + i) : 0ull;
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (start[j] == kNone) continue;
                const int e = (kk + j) * kLocalThreads + tid;
                const Key192 key = key192_of_words(w[j], shift[j], take[j], (uint32_t)(e - start[j]));
                sm.key_lo[e] = key.lo;
                sm.key_hi[e] = key.hi;
                any = 1;
            }
        }
        if (!__syncthreads_or(any)) break;
        // Stable rank inside every group.  Members are first ranked by counting inside sub-blocks of kSubBlock
        // consecutive members (<= kSubBlock comparisons each); sorted runs are then merged pairwise, each member
        // finding its rank in the sibling run by binary search (keys are distinct: the group index is part of them),
        // so a group of g members costs ~kSubBlock + log2(g / kSubBlock) * log2(g) comparisons per member, not g.
        uint32_t myrank[kLocalItems];
        uint32_t more = 0;   // some group of mine is longer than one sub-block
        int cur = 0;
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            const int s = sm.gs[e];
            myrank[k] = 0;
            if (s != kNone) {
                const int t = sm.ge[e];
                const int b0 = s + ((e - s) / kSubBlock) * kSubBlock;
                const int b1 = min(b0 + kSubBlock, t);
                const uint4 my = sm.key_lo[e];
                const uint2 myh = sm.key_hi[e];
                n_compares += (uint32_t)(b1 - b0);
                uint32_t neg = 0;   // minus the number of sub-block members whose key is below mine
#pragma unroll 4
                for (int q = b0; q < b1; ++q) count_if_less(neg, sm.key_lo[q], sm.key_hi[q], my, myh);
                myrank[k] = 0u - neg;
                sm.ord[0][b0 + myrank[k]] = (uint16_t)e;
                more |= (uint32_t)(t - s > kSubBlock);
            }
        }
        static_assert((kSubBlock & (kSubBlock - 1)) == 0, "runs double from a power of two");
        for (int run = kSubBlock, sh = 31 - __clz(kSubBlock); __syncthreads_or(more); run *= 2, ++sh) {
            more = 0;
#pragma unroll
            for (int k = 0; k < kLocalItems; ++k) {
                const int e = k * kLocalThreads + tid;
                const int s = sm.gs[e];
                if (s == kNone) continue;
                const int t = sm.ge[e];
                const int r = (e - s) >> sh;             // my run, its sibling is r ^ 1
                uint32_t nr = myrank[k];
                if (t - s > run) {
                    const int sb = s + (r ^ 1) * run;    // sibling run [sb, sb + len)
                    if (sb < t) {
                        const uint4 my = sm.key_lo[e];
                        const uint2 myh = sm.key_hi[e];
                        int lo = 0, hi = min(run, t - sb);
                        n_compares += 32 - __clz(hi);
                        while (lo < hi) {                // lower bound: sibling members below me
                            const int mid = (lo + hi) >> 1;
                            uint32_t neg = 0;
                            const int qi = sm.ord[cur][sb + mid];
                            count_if_less(neg, sm.key_lo[qi], sm.key_hi[qi], my, myh);
                            if (neg) lo = mid + 1; else hi = mid;
                        }
                        nr += (uint32_t)lo;
                    }
                    myrank[k] = nr;
                    sm.ord[cur ^ 1][s + (r >> 1) * 2 * run + nr] = (uint16_t)e;
                    more |= (uint32_t)(t - s > 2 * run);
                } else {
                    sm.ord[cur ^ 1][s + nr] = (uint16_t)e;   // already one run: carried over
                }
            }
            cur ^= 1;
        }
        const uint16_t* src = sm.ord[cur];
        uint64_t locn[kLocalItems];
        uint32_t headbit = 0;
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            if (sm.gs[e] != kNone) {
                const int se = src[e];
                const uint4 kk = sm.key_lo[se];
                locn[k] = sm.loc[se];
                bool head = e == sm.gs[e] || ((kk.x >> 8) & 127u) < kLocalW;
                if (!head) {   // same bases and length as the member ranked just before?  (the low 8 bits are the group index)
                    const int sp = src[e - 1];
                    const uint4 kp = sm.key_lo[sp];
                    const uint2 hk = sm.key_hi[se], hp = sm.key_hi[sp];
                    head = (((((kk.x ^ kp.x) >> 8) | (kk.y ^ kp.y)) | ((kk.z ^ kp.z) | (kk.w ^ kp.w))) | ((hk.x ^ hp.x) | (hk.y ^ hp.y))) != 0;
                }
                headbit |= (uint32_t)head << k;
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            if (sm.gs[e] != kNone) sm.loc[e] = locn[k];
            // a warp's 32 positions share one head word and no other warp touches it in this phase: one ballot and one
            // plain update instead of up to 32 serialised shared-memory atomics (12 % of the kernel's shared wavefronts)
            const uint32_t word = __ballot_sync(kFull, (headbit >> k) & 1u);
            if ((tid & 31) == 0 && word) sm.hw[e >> 5] |= word;
        }
        __syncthreads();
        // new group bounds; members alone in their group are placed for good
#pragma unroll
        for (int k = 0; k < kLocalItems; ++k) {
            const int e = k * kLocalThreads + tid;
            const int s = sm.gs[e];
            if (s != kNone) {
                // head bits of e and e + 1 both set: alone in its group, placed for good
                const uint32_t lo = sm.hw[e >> 5], hi = sm.hw[(e >> 5) + 1];
                if (((((uint64_t)hi << 32) | lo) >> (e & 31) & 3u) == 3u) {
                    sm.gs[e] = kNone;
                } else {
                    const int t = sm.ge[e];
                    sm.gs[e] = (uint16_t)prev_head(sm.hw, e, s);
                    sm.ge[e] = (uint16_t)next_head(sm.hw, e, t);
                }
            }
        }
    }

    // ---- emit what became final here; publish head bits for the global path ----------------------------
#pragma unroll
    for (int k = 0; k < kLocalItems; ++k) {
        const int e = k * kLocalThreads + tid;
        const uint64_t loc = sm.loc[e];
        if (loc) out[base + e] = loc_symbol(loc);
    }
    for (int i = tid; i < kLocalWords; i += kLocalThreads) {
        if (w0 + i > n_words) continue;
        const uint32_t add = FIRST ? (i < kLocalElems / 32 ? sm.hw[i] : 0u) : (sm.hw[i] & ~sm.hw0[i]);
        if (add) atomicOr(&heads[w0 + i], add);
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
        atomicAdd(elems_done + 2, (unsigned long long)s_cmp);   // 128-bit key comparisons done (the ALU work of this kernel)
    }
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
                                uint32_t depth, uint32_t w, uint64_t* keys_c, IdT* ids_c, uint32_t* pos_c, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    const uint64_t n_words = (n + 31) >> 5;
    refine_rekey_kernel<IdT><<<(unsigned)((n_words + 255) / 256), 256, 0, s>>>(R, heads, word_base, ids, n, depth, w, keys_c, ids_c, pos_c);
    return cudaGetLastError();
}

template <typename IdT>
cudaError_t launch_refine_writeback(const Reads& R, const uint64_t* keys_c, const IdT* ids_c, const uint32_t* pos_c, uint64_t n_c,
                                    uint32_t w, IdT* ids, uint32_t* heads, uint8_t* out, cudaStream_t s) {
    if (n_c == 0) return cudaSuccess;
    refine_writeback_kernel<IdT><<<(unsigned)((n_c + 255) / 256), 256, 0, s>>>(R, keys_c, ids_c, pos_c, n_c, w, ids, heads, out);
    return cudaGetLastError();
}

template <typename KeyT, typename IdT>
cudaError_t launch_finish_first(const Reads& R, const KeyT* keys1, uint32_t w1, uint32_t depth0, uint32_t* heads_out, IdT* ids, uint64_t n,
                                uint32_t group_cap, uint8_t* out, unsigned long long* elems_done, bool packed, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    constexpr bool kCanPack = sizeof(KeyT) == 4 && sizeof(IdT) == 4;
    if (packed && !kCanPack) return cudaErrorInvalidValue;
    auto kernel = packed ? finish_tile_kernel<KeyT, IdT, true, kCanPack> : finish_tile_kernel<KeyT, IdT, true, false>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LocalSmem<IdT>));
    if (e != cudaSuccess) return e;
    if (group_cap > (uint32_t)kLocalGroupCap) group_cap = kLocalGroupCap;
    uint64_t blocks = (n + kLocalTile - 1) / kLocalTile;
    kernel<<<(unsigned)blocks, kLocalThreads, sizeof(LocalSmem<IdT>), s>>>(R, keys1, w1, (1u << key_len_bits(w1)) - 1, nullptr, heads_out, ids, n,
                                                                          depth0, group_cap, out, elems_done);
    return cudaGetLastError();
}

template <typename IdT>
cudaError_t launch_finish_later(const Reads& R, const uint32_t* heads_in, uint32_t* heads_out, const IdT* ids, uint64_t n, uint32_t depth,
                                uint32_t group_cap, uint8_t* out, unsigned long long* elems_done, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    auto kernel = finish_tile_kernel<uint64_t, IdT, false, false>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LocalSmem<IdT>));
    if (e != cudaSuccess) return e;
    if (group_cap > (uint32_t)kLocalGroupCap) group_cap = kLocalGroupCap;
    uint64_t blocks = (n + kLocalTile - 1) / kLocalTile;
    kernel<<<(unsigned)blocks, kLocalThreads, sizeof(LocalSmem<IdT>), s>>>(R, nullptr, 0, 0, heads_in, heads_out, const_cast<IdT*>(ids), n, depth, group_cap, out,
                                                                          elems_done);
    return cudaGetLastError();
}

#define CX_INSTANTIATE(IdT)                                                                                                          \
    template cudaError_t launch_refine_rekey<IdT>(const Reads&, const uint32_t*, const uint64_t*, const IdT*, uint64_t, uint32_t,   \
                                                  uint32_t, uint64_t*, IdT*, uint32_t*, cudaStream_t);                               \
    template cudaError_t launch_refine_writeback<IdT>(const Reads&, const uint64_t*, const IdT*, const uint32_t*, uint64_t,         \
                                                      uint32_t, IdT*, uint32_t*, uint8_t*, cudaStream_t);                            \
    template cudaError_t launch_finish_first<uint32_t, IdT>(const Reads&, const uint32_t*, uint32_t, uint32_t, uint32_t*, IdT*, uint64_t, \
                                                            uint32_t, uint8_t*, unsigned long long*, bool, cudaStream_t);            \
    template cudaError_t launch_finish_first<uint64_t, IdT>(const Reads&, const uint64_t*, uint32_t, uint32_t, uint32_t*, IdT*, uint64_t, \
                                                            uint32_t, uint8_t*, unsigned long long*, bool, cudaStream_t);            \
    template cudaError_t launch_finish_later<IdT>(const Reads&, const uint32_t*, uint32_t*, const IdT*, uint64_t, uint32_t,         \
                                                  uint32_t, uint8_t*, unsigned long long*, cudaStream_t);
CX_INSTANTIATE(uint32_t)
CX_INSTANTIATE(uint64_t)

}  // namespace cx
