// cx_scan_reads.cu -- the kernels that walk every suffix of R in (read, position) order:
//   prep        offsets sanity, longest read, uniform-length test
//   tile table  first read of every tile of kListTile consecutive suffix slots
//   a2 bucket histogram   (Fig. 2 step 1: "Scan all suffixes ... Store the size of each partition")
//   a4+a5 list + key build (Fig. 2 steps 3(a), 3(c)i; key = the paper's "stringword"):
//         list_write   the whole collection as one batch (also counts the partition sizes on the way)
//         list_count   per tile, the suffixes of eight consecutive batches in one scan (fewer scans)
//         list_select  one batch of several: the suffixes whose partition lies in the batch's range
//
// A suffix slot g in [0, N) is suffix (i, p) with g = offsets[i] + i + p: reads laid end to end, each
// followed by one slot for its end-marker.  Slots ascend in (read, position) order, which is the
// listing order PAPER.md:99 requires for the stable sort to realise $_i < $_j.
#include "cx_internal.cuh"

#ifndef CX_READ_TILE_PREFETCH
#define CX_READ_TILE_PREFETCH 1   // L2 prefetch of the read tile a grid-width ahead in the one-read-per-thread scans
#endif

namespace cx {
namespace {

// ---------------------------------------------------------------------------------------------
// prep
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prep_kernel(const uint64_t* __restrict__ offsets, uint64_t n_reads, uint64_t max_bases, BuildInfo* info) {
    uint64_t first_len = offsets[1] - offsets[0];
    uint64_t local_max = 0;
    uint32_t bad = 0, nonuni = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_reads; i += (uint64_t)gridDim.x * blockDim.x) {
        uint64_t a = offsets[i], b = offsets[i + 1];
        if (b < a) {
            bad = 1;
        } else {
            uint64_t len = b - a;
            local_max = len > local_max ? len : local_max;
            nonuni |= len != first_len;
        }
    }
    for (int o = 16; o; o >>= 1) {
        uint64_t other = __shfl_xor_sync(0xffffffffu, local_max, o);
        local_max = other > local_max ? other : local_max;
    }
    bad = __any_sync(0xffffffffu, bad);
    nonuni = __any_sync(0xffffffffu, nonuni);
    if (lane_id() == 0) {
        if (local_max) atomicMax((unsigned long long*)&info->max_len, (unsigned long long)local_max);
        if (bad) atomicOr(&info->bad_offsets, 1u);
        if (nonuni) atomicOr(&info->nonuniform, 1u);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (offsets[0] != 0) atomicOr(&info->bad_offsets, 1u);
        if (offsets[n_reads] > max_bases) atomicOr(&info->bad_offsets, 2u);   // more bases than the plan was made for
        info->total_bases = offsets[n_reads];
        info->n_suffixes = offsets[n_reads] + n_reads;
        info->first_len = first_len;
    }
}

// tile_first_read[t] = the read that owns slot t * kListTile (largest i with offsets[i] + i <= slot)
__global__ void __launch_bounds__(256) tile_table_kernel(const uint64_t* __restrict__ offsets, uint64_t n_reads,
                                                         const BuildInfo* __restrict__ info, uint32_t* __restrict__ tile_first_read,
                                                         uint64_t max_tiles) {
    uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint64_t N = info->n_suffixes;
    uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    if (t >= n_tiles || t >= max_tiles) return;
    uint64_t g = t * kListTile;
    uint64_t lo = 0, hi = n_reads - 1;   // invariant: offsets[lo] + lo <= g
    while (lo < hi) {
        uint64_t mid = (lo + hi + 1) >> 1;
        if (offsets[mid] + mid <= g) lo = mid; else hi = mid - 1;
    }
    tile_first_read[t] = (uint32_t)lo;
}

// ---------------------------------------------------------------------------------------------
// tile decode: the reads and packed bases that the slots [g0, g0 + kListTile) touch
// ---------------------------------------------------------------------------------------------
struct TileSmem {
    uint64_t off[kListTile + 2];           // offsets of the reads that intersect the tile
    uint64_t packed[kListTile / 32 + 4];   // the bases of the tile plus one window of look-ahead
};

struct TileCtx {
    uint64_t g0;        // first slot
    uint32_t n_slots;   // slots in this tile
    uint64_t r0;        // first read
    uint32_t n_tile_reads;
    uint64_t word0;     // first packed word staged
    uint32_t uniform;   // every read has length L: slot -> (read, pos) by division, no offsets needed
    uint32_t L1;        // L + 1
    uint32_t pos0;      // position of slot g0 inside read r0 (uniform only)
    float inv_L1;       // 1 / L1: slot -> read by a multiply and a one-step correction instead of an integer division
};

__device__ __forceinline__ TileCtx load_tile(const Reads& R, const BuildInfo* __restrict__ info,
                                             const uint32_t* __restrict__ tile_first_read, uint64_t t, uint64_t n_tiles, uint64_t N,
                                             TileSmem& sm) {
    TileCtx c;
    c.g0 = t * kListTile;
    c.n_slots = (uint32_t)min((uint64_t)kListTile, N - c.g0);
    c.uniform = info->nonuniform ? 0u : 1u;
    c.L1 = (uint32_t)info->first_len + 1u;
    c.inv_L1 = 1.0f / (float)c.L1;
    c.r0 = tile_first_read[t];
    c.pos0 = 0;
    c.n_tile_reads = 0;
    if (c.uniform) {
        c.pos0 = (uint32_t)(c.g0 - c.r0 * c.L1);
    } else {
        uint64_t r_last = (t + 1 < n_tiles) ? (uint64_t)tile_first_read[t + 1] : R.n_reads - 1;
        c.n_tile_reads = (uint32_t)(r_last - c.r0 + 1);                       // <= kListTile + 1
        for (uint32_t j = threadIdx.x; j <= c.n_tile_reads; j += blockDim.x) sm.off[j] = R.offsets[c.r0 + j];
    }
    // base position of slot g is g - (its read index); it grows by 0 or 1 per slot
    uint64_t b0 = c.g0 - c.r0;
    c.word0 = b0 >> 5;
    for (uint32_t j = threadIdx.x; j < kListTile / 32 + 4; j += blockDim.x) {
        uint64_t wi = c.word0 + j;
        sm.packed[j] = wi < R.n_words ? __ldg(R.packed + wi) : 0ull;
    }
    __syncthreads();
    return c;
}

struct Slot {
    uint64_t read, pos, rem;   // suffix (read, pos); rem = bases left = m_i - pos
    uint64_t window;           // the next 32 bases, MSB-first, junk past rem
    uint64_t b;                // index of its first base in the concatenation
    uint32_t lo;               // read - r0 (index into the staged offsets of a ragged collection)
};

__device__ __forceinline__ Slot decode_slot(const TileCtx& c, const TileSmem& sm, uint32_t s) {
    Slot sl;
    uint64_t b;
    if (c.uniform) {
        const uint32_t x = c.pos0 + s;
        // x < L1 + kListTile, so x / L1 <= kListTile + 1: the float estimate is within one of it (the integer division
        // this replaces was 8 % of the multi-batch listing's instructions)
        uint32_t rr = (uint32_t)((float)x * c.inv_L1);
        if ((uint64_t)rr * c.L1 > x) --rr;
        else if ((uint64_t)(rr + 1) * c.L1 <= x) ++rr;
        sl.read = c.r0 + rr;
        sl.pos = x - rr * c.L1;
        sl.rem = (c.L1 - 1) - sl.pos;
        sl.lo = rr;
        b = sl.read * (c.L1 - 1) + sl.pos;
    } else {
        uint64_t g = c.g0 + s;
        // largest j with off[j] + r0 + j <= g
        uint32_t lo = 0, hi = c.n_tile_reads - 1;
        while (lo < hi) {
            uint32_t mid = (lo + hi + 1) >> 1;
            if (sm.off[mid] + c.r0 + mid <= g) lo = mid; else hi = mid - 1;
        }
        sl.read = c.r0 + lo;
        sl.lo = lo;
        uint64_t start = sm.off[lo];
        sl.pos = g - (start + sl.read);
        sl.rem = sm.off[lo + 1] - start - sl.pos;
        b = start + sl.pos;
    }
    uint32_t wi = (uint32_t)((b >> 5) - c.word0);
    uint32_t sh = (uint32_t)(b & 31) * 2;
    uint64_t w0 = sm.packed[wi], w1 = sm.packed[wi + 1];
    sl.window = sh ? (w0 << sh) | (w1 >> (64 - sh)) : w0;
    sl.b = b;
    return sl;
}

// Partition code of a suffix (reading A4 of PAPER.md:79 "suffixes shorter than l require special
// but easy handling"): (first l bases, A-padded) * (l + 1) + min(rem, l).  Order-preserving.
__device__ __forceinline__ uint32_t bucket_of(const Slot& sl, uint32_t ell, uint32_t& kmer, uint32_t& r) {
    r = sl.rem < ell ? (uint32_t)sl.rem : ell;
    kmer = r ? (uint32_t)((sl.window >> (64 - 2 * r)) << (2 * (ell - r))) : 0u;
    return kmer * (ell + 1) + r;
}

// Lean state for scans that only need the partition code of most slots (the multi-batch listing): stepping from a
// suffix slot to the next one in (read, position) order needs no decoding from scratch -- inside a read the 32-base
// window shifts by one base taken from the 32 bases after it (both in registers: four shifts, no shared-memory
// access); after a read's end-marker slot the next read starts at the same base index, so the window stays.
struct Walk {
    uint64_t window, ahead;   // bases [b, b + 32) and [b + 32, b + 64), MSB-first
    uint64_t b;               // base index of the slot's first base
    uint32_t rem;             // bases left in the read from this slot
    uint32_t lo;              // read - r0
};
__device__ __forceinline__ Walk walk_init(const TileCtx& c, const TileSmem& sm, uint32_t s) {
    const Slot sl = decode_slot(c, sm, s);
    Walk wk;
    wk.window = sl.window;
    wk.b = sl.b;
    wk.rem = (uint32_t)sl.rem;
    wk.lo = sl.lo;
    const uint64_t nb = sl.b + 32;
    const uint32_t wi = (uint32_t)((nb >> 5) - c.word0);
    const uint32_t sh = (uint32_t)(nb & 31) * 2;
    const uint64_t w0 = sm.packed[wi], w1 = sm.packed[wi + 1];
    wk.ahead = sh ? (w0 << sh) | (w1 >> (64 - sh)) : w0;
    return wk;
}
// valid for at most 32 steps after walk_init (the scans take kListItems = 8)
__device__ __forceinline__ void walk_next(const TileCtx& c, const TileSmem& sm, Walk& wk) {
    if (wk.rem) {
        wk.window = (wk.window << 2) | (wk.ahead >> 62);
        wk.ahead <<= 2;
        wk.b += 1;
        wk.rem -= 1;
    } else {   // end-marker slot: the next read starts at the same base index
        wk.lo += 1;
        wk.rem = c.uniform ? c.L1 - 1 : (uint32_t)(sm.off[wk.lo + 1] - sm.off[wk.lo]);
    }
}
// hi: the next 16 bases of the suffix (the high word of its window)
__device__ __forceinline__ uint32_t window_bucket32(uint32_t hi, uint32_t rem, uint32_t ell) {
    const uint32_t r = rem < ell ? rem : ell;
    // the first l bases with those past the end of the read cleared (A-padded); no branch, valid for r = 0
    const uint32_t kmer = (hi >> (32 - 2 * ell)) & (0xffffffffu << (2 * (ell - r)));
    return kmer * (ell + 1) + r;
}
__device__ __forceinline__ uint32_t window_bucket(uint64_t window, uint32_t rem, uint32_t ell) {
    return window_bucket32((uint32_t)(window >> 32), rem, ell);
}
// Outside a region the partition code needs only the first l <= 7 bases of a suffix, and a thread walks kListItems = 8
// consecutive slots: the 16 bases in the high word of the first slot's window serve all of them (7 shifts of one base
// leave 9 >= l), so the walk is one 32-bit shift per slot instead of two 64-bit funnel shifts.
struct Walk32 {
    uint32_t top, rem, lo;
};
static_assert(16 - (kListItems - 1) >= 7, "the high word must still hold l bases at the last slot of a thread");
__device__ __forceinline__ Walk32 walk32_of(const Walk& wk) { return Walk32{(uint32_t)(wk.window >> 32), wk.rem, wk.lo}; }
// step to the next slot; `more`: that slot is still inside the tile (its read's length is staged)
__device__ __forceinline__ void walk32_next(const TileCtx& c, const TileSmem& sm, Walk32& w, bool more) {
    if (w.rem) {
        w.top <<= 2;
        w.rem -= 1;
    } else if (more) {   // end-marker slot: the next read starts at the same base index
        w.lo += 1;
        w.rem = c.uniform ? c.L1 - 1 : (uint32_t)(sm.off[w.lo + 1] - sm.off[w.lo]);
    }
}
// partition code of the walker's slot inside `region` (at the region's depth); false if the slot is outside it
template <bool REGION>
__device__ __forceinline__ bool walk_bucket(const Reads& R, const Region& region, const Walk& wk, uint32_t ell, uint32_t& code) {
    uint64_t window = wk.window;
    uint32_t rem = wk.rem;
    if (REGION && !enter_region(R.packed, R.n_words, region, wk.b, window, rem)) return false;
    code = window_bucket(window, rem, ell);
    return true;
}

// digit histograms of the sort that follows (one shared-memory counter per pass and digit): constant shifts, so a
// pass costs an extract and an atomic instead of a variable 64-bit shift inside a counted loop
template <typename KeyT>
__device__ __forceinline__ void digit_counts(uint32_t (*s_dh)[kRadix], KeyT key, uint32_t n_passes) {
#pragma unroll
    for (uint32_t p = 0; p < sizeof(KeyT); ++p)
        if (p < n_passes) atomicAdd(&s_dh[p][(uint32_t)(key >> (p * kRadixBits)) & (kRadix - 1)], 1u);
}

// ---------------------------------------------------------------------------------------------
// a2: bucket histogram.  Persistent blocks; full-length partitions (the bulk) are counted in a
// shared-memory histogram with warp-aggregated updates, the few short ones go straight to global.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kListThreads) bucket_hist_kernel(Reads R, const BuildInfo* __restrict__ info,
                                                                   const uint32_t* __restrict__ tile_first_read, uint32_t ell, Region region,
                                                                   unsigned long long* __restrict__ hist, uint32_t skip_if_uniform) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem& sm = *reinterpret_cast<TileSmem*>(smem_raw);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem_raw + sizeof(TileSmem));
    const uint32_t n_kmers = 1u << (2 * ell);
    // suffixes that end inside the prefix: (4^r - 1) / 3 + (their r bases) indexes the 4^r partitions of length r
    uint32_t* s_short = s_hist + n_kmers;
    const uint32_t n_short = (n_kmers - 1) / 3;
    for (uint32_t k = threadIdx.x; k < n_kmers + n_short; k += blockDim.x) s_hist[k] = 0;
    if (info->bad_offsets) return;   // reported by the host after it reads `info`
    if (skip_if_uniform && !info->nonuniform) return;   // bucket_hist_uniform_kernel has it
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm (and s_hist zeroed on the first trip)
        TileCtx c = load_tile(R, info, tile_first_read, t, n_tiles, N, sm);
#pragma unroll
        for (int k = 0; k < kListItems; ++k) {
            uint32_t s = k * kListThreads + threadIdx.x;
            bool valid = s < c.n_slots;
            if (valid) {
                uint32_t kmer = 0, r = 0;
                Slot sl = decode_slot(c, sm, s);
                if (region.depth) {   // sizes of the sub-partitions of an oversize partition
                    uint32_t rem = (uint32_t)sl.rem;
                    if (!enter_region(R.packed, R.n_words, region, sl.b, sl.window, rem)) continue;
                    sl.rem = rem;
                }
                uint32_t b = bucket_of(sl, ell, kmer, r);
                // consecutive suffixes rarely share an l-mer, so one shared-memory atomic per suffix beats warp
                // aggregation here (match.any costs ~25 cycles per distinct value on sm_100a)
                (void)b;
                if (r == ell) atomicAdd(&s_hist[kmer], 1u);
                else atomicAdd(&s_short[(((1u << (2 * r)) - 1) / 3) + (kmer >> (2 * (ell - r)))], 1u);
            }
        }
    }
    __syncthreads();
    for (uint32_t k = threadIdx.x; k < n_kmers; k += blockDim.x) {
        uint32_t v = s_hist[k];
        if (v) atomicAdd(hist + (uint64_t)k * (ell + 1) + ell, (unsigned long long)v);
    }
    for (uint32_t r = 0; r < ell; ++r) {
        const uint32_t first = ((1u << (2 * r)) - 1) / 3, count = 1u << (2 * r);
        for (uint32_t k = threadIdx.x; k < count; k += blockDim.x) {
            uint32_t v = s_short[first + k];
            if (v) atomicAdd(hist + ((uint64_t)k << (2 * (ell - r))) * (ell + 1) + r, (unsigned long long)v);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a4 (count half): suffixes per tile that fall in each of up to kCountGroup consecutive batches, in ONE scan of the
// collection (fewer scans).  Batch j owns the partitions [first[j], first[j + 1]).
// tile_count is laid out [batch][tile] so that each batch's column can be scanned in place.
// ---------------------------------------------------------------------------------------------
template <bool REGION>   // REGION = false: the whole collection, no region code in the loop
__global__ void __launch_bounds__(kListThreads) list_count_kernel(Reads R, const BuildInfo* __restrict__ info,
                                                                  const uint32_t* __restrict__ tile_first_read, uint32_t ell, Region region,
                                                                  CountRanges ranges, uint64_t* __restrict__ tile_count, uint64_t col_stride) {
    __shared__ TileSmem sm;
    __shared__ uint32_t s_total[kCountGroup];
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    if (info->bad_offsets) return;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm and s_total
        if (threadIdx.x < kCountGroup) s_total[threadIdx.x] = 0;
        TileCtx c = load_tile(R, info, tile_first_read, t, n_tiles, N, sm);
        // thread t walks the kListItems consecutive slots [t * kListItems, ...)
        uint64_t mine = 0;   // eight 8-bit counters
        const uint32_t s0 = threadIdx.x * kListItems;
        if (s0 < c.n_slots) {
            Walk wk = walk_init(c, sm, s0);
            Walk32 w32 = walk32_of(wk);
            const uint32_t n_here = min((uint32_t)kListItems, c.n_slots - s0);
#pragma unroll
            for (int i = 0; i < kListItems; ++i) {
                if ((uint32_t)i < n_here) {
                    uint32_t b = 0;
                    bool in;
                    if constexpr (REGION) in = walk_bucket<true>(R, region, wk, ell, b);
                    else in = true, b = window_bucket32(w32.top, w32.rem, ell);
                    if (in && b >= ranges.first[0] && b < ranges.first[ranges.n]) {
                        uint32_t j = 0;
#pragma unroll
                        for (int q = 1; q < kCountGroup; ++q) j += (q < (int)ranges.n && b >= ranges.first[q]);
                        mine += 1ull << (8 * j);
                    }
                    if constexpr (REGION) {
                        if ((uint32_t)i + 1 < n_here) walk_next(c, sm, wk);
                    } else {
                        walk32_next(c, sm, w32, (uint32_t)i + 1 < n_here);
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < kCountGroup; ++j) {
            uint32_t v = (uint32_t)(mine >> (8 * j)) & 255u;
            for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane_id() == 0 && v) atomicAdd(&s_total[j], v);
        }
        __syncthreads();
        if (threadIdx.x < ranges.n) tile_count[(uint64_t)threadIdx.x * col_stride + t] = s_total[threadIdx.x];
    }
}

// ---------------------------------------------------------------------------------------------
// a4 (write half) + a5 for one batch of a multi-batch build: the suffixes whose partition lies in
// [bucket_lo, bucket_hi], in (read, pos) order, each with its first key.  Most slots belong to other
// batches, so the scan walks the slots with next_slot() and decodes in full only what it takes.
// ---------------------------------------------------------------------------------------------
// One (first-round key, id) pair of a batch's listing.  Three layouts: packed 32 + 32 in one word; separate arrays; or -- split != 0,
// 64-bit keys and ids only -- the key shifted up by `split` bits above the id's high part in the word, and the id's low 32 bits in
// a uint32 array at `ids`: 12 bytes per pair through the sort instead of 16 (the sort then runs over bits split .. 64).
template <typename KeyT, typename IdT, bool PACKED>
__device__ __forceinline__ void store_pair(KeyT* __restrict__ keys, IdT* __restrict__ ids, uint64_t at, KeyT key, IdT id, uint32_t split) {
    if constexpr (PACKED) {
        reinterpret_cast<uint64_t*>(keys)[at] = ((uint64_t)key << 32) | (uint64_t)id;
    } else {
        if constexpr (sizeof(KeyT) == 8 && sizeof(IdT) == 8) {
            if (split) {
                keys[at] = (key << split) | (id >> 32);
                reinterpret_cast<uint32_t*>(ids)[at] = (uint32_t)id;
                return;
            }
        }
        keys[at] = key;
        ids[at] = id;
    }
}

template <typename KeyT, typename IdT, bool PACKED, bool REGION>
__global__ void __launch_bounds__(kListThreads) list_select_kernel(Reads R, const BuildInfo* __restrict__ info,
                                                                   const uint32_t* __restrict__ tile_first_read, uint32_t ell, uint32_t w,
                                                                   uint32_t bucket_lo, uint32_t bucket_hi,
                                                                   const uint64_t* __restrict__ tile_base, KeyT* __restrict__ keys,
                                                                   IdT* __restrict__ ids, uint32_t n_passes,
                                                                   unsigned long long* __restrict__ digit_hist, Region region,
                                                                   uint64_t ord_lo, uint64_t ord_hi, uint32_t split) {
    // region: the scan is confined to the suffixes of an oversize partition and keys start at its depth.
    // [ord_lo, ord_hi): of the selected suffixes, in listing order, only these ordinals are written (at ordinal - ord_lo):
    // a partition of IDENTICAL suffixes larger than a batch is cut this way, its order being the listing order anyway.
    __shared__ TileSmem sm;
    __shared__ uint32_t s_dh[8][kRadix];
    __shared__ uint32_t s_warp[kListThreads / 32];
    __shared__ uint16_t s_taken[kListTile];   // slots of the tile that belong to the batch, in slot order
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    const uint32_t warp = threadIdx.x >> 5;
    if (info->bad_offsets) return;
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) (&s_dh[0][0])[i] = 0;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm and s_warp
        TileCtx c = load_tile(R, info, tile_first_read, t, n_tiles, N, sm);
        const uint32_t s0 = threadIdx.x * kListItems;
        uint32_t mask = 0;   // which of my kListItems consecutive slots belong to this batch
        if (s0 < c.n_slots) {
            Walk wk = walk_init(c, sm, s0);
            Walk32 w32 = walk32_of(wk);
            const uint32_t n_here = min((uint32_t)kListItems, c.n_slots - s0);
#pragma unroll
            for (int i = 0; i < kListItems; ++i) {
                if ((uint32_t)i < n_here) {
                    if constexpr (REGION) {
                        uint32_t b = 0;
                        mask |= (uint32_t)(walk_bucket<true>(R, region, wk, ell, b) && b - bucket_lo <= bucket_hi - bucket_lo) << i;
                        if ((uint32_t)i + 1 < n_here) walk_next(c, sm, wk);
                    } else {
                        mask |= (uint32_t)(window_bucket32(w32.top, w32.rem, ell) - bucket_lo <= bucket_hi - bucket_lo) << i;
                        walk32_next(c, sm, w32, (uint32_t)i + 1 < n_here);
                    }
                }
            }
        }
        // exclusive scan of the per-thread counts: slot order = thread order
        const uint32_t cnt = __popc(mask);
        uint32_t incl = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t up = __shfl_up_sync(0xffffffffu, incl, o);
            if ((int)lane_id() >= o) incl += up;
        }
        if (lane_id() == 31) s_warp[warp] = incl;
        __syncthreads();
        uint32_t before = incl - cnt, total = 0;
        for (uint32_t q = 0; q < kListThreads / 32; ++q) {
            const uint32_t v = s_warp[q];
            if (q < warp) before += v;
            total += v;
        }
        // The taken slots are few and scattered over the threads: decoding them where they were found runs every warp
        // for as many rounds as its busiest lane has slots, one or two lanes at a time.  They are compacted first (slot
        // order = thread order) and then decoded one per thread: full warps, consecutive output addresses.
        while (mask) {
            const int i = __ffs(mask) - 1;
            mask &= mask - 1;
            s_taken[before++] = (uint16_t)(s0 + i);
        }
        __syncthreads();
        const uint64_t tile_dst = tile_base[t];
        for (uint32_t j = threadIdx.x; j < total; j += kListThreads) {
            const uint64_t dst = tile_dst + j;
            if (dst >= ord_lo && dst < ord_hi) {
                Slot sl = decode_slot(c, sm, s_taken[j]);
                if (REGION) {
                    sl.window = load_window(R.packed, R.n_words, sl.b + region.depth);
                    sl.rem -= region.depth;
                }
                const KeyT key = first_key_as<KeyT>(sl.window, sl.rem, w);
                const IdT id = make_id<IdT>(sl.read, sl.pos, R.pos_bits);
                digit_counts(s_dh, key, n_passes);
                store_pair<KeyT, IdT, PACKED>(keys, ids, dst - ord_lo, key, id, split);
            }
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) {
        uint32_t v = (&s_dh[0][0])[i];
        if (v) atomicAdd(digit_hist + i, (unsigned long long)v);
    }
}

// ---------------------------------------------------------------------------------------------
// a4 + a5 (+ a2) for a build that takes the whole collection in one batch: every suffix in (read, pos)
// order, index = slot, each with its first key.  The read is in shared memory already, so the round-1
// key costs no gather.  The same scan builds the digit histograms of the sort that follows and, when
// bucket_hist != nullptr, the partition sizes (as bucket_hist_kernel does): the collection is read once.
// PACKED (32-bit key and id only): one 64-bit word (key << 32 | id) per suffix goes to `keys`, nothing to
// `ids`; the sort is then keys-only over bits [32, 64) and the id travels with its key for free.
// ---------------------------------------------------------------------------------------------
template <typename KeyT, typename IdT, bool PACKED>
__global__ void __launch_bounds__(kListThreads) list_write_kernel(Reads R, const BuildInfo* __restrict__ info,
                                                                  const uint32_t* __restrict__ tile_first_read, uint32_t ell, uint32_t w,
                                                                  KeyT* __restrict__ keys, IdT* __restrict__ ids, uint32_t n_passes,
                                                                  unsigned long long* __restrict__ digit_hist,
                                                                  unsigned long long* __restrict__ bucket_hist, uint64_t max_n, uint32_t skip_if_reads) {
    __shared__ TileSmem sm;
    __shared__ uint32_t s_dh[8][kRadix];   // digit counts of every radix pass of the sort that follows (a6's upfront histogram)
    extern __shared__ uint32_t s_bh[];     // partition counters, laid out as in bucket_hist_kernel
    const uint32_t n_kmers = 1u << (2 * ell), n_short = (n_kmers - 1) / 3;
    if (bucket_hist)
        for (uint32_t k = threadIdx.x; k < n_kmers + n_short; k += blockDim.x) s_bh[k] = 0;
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    if (N > max_n || info->bad_offsets) return;   // the host reports both after reading `info`
    if (skip_if_reads && !info->nonuniform && info->first_len >= (uint64_t)kReadMinLen && info->first_len <= (uint64_t)kReadMaxLen) return;   // list_write_reads_kernel has it
    const uint64_t n_tiles = (N + kListTile - 1) / kListTile;
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) (&s_dh[0][0])[i] = 0;

    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm
        TileCtx c = load_tile(R, info, tile_first_read, t, n_tiles, N, sm);
#pragma unroll
        for (int k = 0; k < kListItems; ++k) {
            const uint32_t s = k * kListThreads + threadIdx.x;
            if (s >= c.n_slots) continue;
            const Slot sl = decode_slot(c, sm, s);
            if (bucket_hist) {
                uint32_t kmer, r;
                bucket_of(sl, ell, kmer, r);
                if (r == ell) atomicAdd(&s_bh[kmer], 1u);
                else atomicAdd(&s_bh[n_kmers + (((1u << (2 * r)) - 1) / 3) + (kmer >> (2 * (ell - r)))], 1u);
            }
            const KeyT key = first_key_as<KeyT>(sl.window, sl.rem, w);
            const IdT id = make_id<IdT>(sl.read, sl.pos, R.pos_bits);
            digit_counts(s_dh, key, n_passes);
            if constexpr (PACKED) {
                reinterpret_cast<uint64_t*>(keys)[c.g0 + s] = ((uint64_t)key << 32) | (uint64_t)id;
            } else {
                keys[c.g0 + s] = key;
                ids[c.g0 + s] = id;
            }
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) {
        uint32_t v = (&s_dh[0][0])[i];
        if (v) atomicAdd(digit_hist + i, (unsigned long long)v);
    }
    if (bucket_hist) {
        for (uint32_t k = threadIdx.x; k < n_kmers; k += blockDim.x) {
            uint32_t v = s_bh[k];
            if (v) atomicAdd(bucket_hist + (uint64_t)k * (ell + 1) + ell, (unsigned long long)v);
        }
        for (uint32_t r = 0; r < ell; ++r) {
            const uint32_t first = n_kmers + ((1u << (2 * r)) - 1) / 3, count = 1u << (2 * r);
            for (uint32_t k = threadIdx.x; k < count; k += blockDim.x) {
                uint32_t v = s_bh[first + k];
                if (v) atomicAdd(bucket_hist + ((uint64_t)k << (2 * (ell - r))) * (ell + 1) + r, (unsigned long long)v);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The multi-batch scans for collections of reads of ONE length (the paper's setting; configs[1], [2], [4]),
// outside any refined region.  Every batch of a collection larger than the workspace walks all N slots again
// (one listing scan per round), so the walk itself is what counts: tiles of 8192 slots, 32 consecutive slots
// per thread (the per-thread set-up is paid once per 32 slots), no offsets table (a slot is decoded by one division), a
// 16-base window in one register refilled every 8 slots, and a branch-free partition code per slot.
// ---------------------------------------------------------------------------------------------
constexpr int kBigItems = 32;
constexpr int kBigTile = kListThreads * kBigItems;
static_assert(kBigTile <= 65536, "taken slots are kept as 16-bit indices");

struct BigSmem {
    uint64_t packed[kBigTile / 32 + 4];   // the bases of the tile plus two windows of look-ahead
};
struct BigCtx {
    uint64_t g0, r0;        // first slot, the read that owns it
    uint32_t n_slots, pos0; // slots in this tile; position of slot g0 inside read r0
    uint32_t L1;            // read length + 1
    uint32_t brel0;         // base index of slot g0 relative to the first staged base
    float inv_L1;
};
__device__ __forceinline__ BigCtx load_big_tile(const Reads& R, const BuildInfo* __restrict__ info, uint64_t t, uint64_t N, BigSmem& sm) {
    BigCtx c;
    c.g0 = t * kBigTile;
    c.n_slots = (uint32_t)min((uint64_t)kBigTile, N - c.g0);
    c.L1 = (uint32_t)info->first_len + 1u;
    c.inv_L1 = 1.0f / (float)c.L1;
    c.r0 = c.g0 / c.L1;
    c.pos0 = (uint32_t)(c.g0 - c.r0 * c.L1);
    const uint64_t b0 = c.g0 - c.r0;                 // base index of slot g = g - (its read)
    const uint64_t word0 = b0 >> 5;
    c.brel0 = (uint32_t)(b0 & 31);
    for (uint32_t j = threadIdx.x; j < kBigTile / 32 + 4; j += blockDim.x) {
        const uint64_t wi = word0 + j;
        sm.packed[j] = wi < R.n_words ? __ldg(R.packed + wi) : 0ull;
    }
    __syncthreads();
    return c;
}
// slot s of the tile -> reads passed since r0 (rr), position in its read, staged base index
__device__ __forceinline__ void big_decode(const BigCtx& c, uint32_t s, uint32_t& rr, uint32_t& pos, uint32_t& brel) {
    const uint32_t x = c.pos0 + s;                   // < L1 + kBigTile: the float estimate of x / L1 is within one of it
    rr = (uint32_t)((float)x * c.inv_L1);
    if ((uint64_t)rr * c.L1 > x) --rr;
    else if ((uint64_t)(rr + 1) * c.L1 <= x) ++rr;
    pos = x - rr * c.L1;
    brel = c.brel0 + s - rr;
}
__device__ __forceinline__ uint64_t big_window(const BigSmem& sm, uint32_t brel) {
    const uint32_t wi = brel >> 5, sh = (brel & 31) * 2;
    const uint64_t w0 = sm.packed[wi], w1 = sm.packed[wi + 1];
    return sh ? (w0 << sh) | (w1 >> (64 - sh)) : w0;
}
// the 16 bases from staged base index brel on (first base in the most significant bits): the staged words seen as
// 32-bit halves, high half first
__device__ __forceinline__ uint32_t big_top16(const BigSmem& sm, uint32_t brel) {
    const uint32_t* half = reinterpret_cast<const uint32_t*>(sm.packed);
    const uint32_t q = brel >> 4, sh = (brel & 15) * 2;
    return __funnelshift_l(half[(q + 1) ^ 1], half[q ^ 1], sh);
}
// Walk of one thread over its kBigItems consecutive slots: f(i, l-mer A-padded, min(rem, l)) for each; branch-free per slot (a warp's lanes
// are at different phases of their reads, so a 'suffix ends inside the prefix' branch would be taken by some lane nearly always).
// GUARD: the tile is ragged (only the collection's last tile), slots at or past n_here do not exist.
template <bool GUARD, typename F>
__device__ __forceinline__ void big_walk(const BigCtx& c, const BigSmem& sm, uint32_t s0, uint32_t ell, F&& f) {
    uint32_t rr, pos, brel;
    big_decode(c, s0, rr, pos, brel);
    uint32_t rem = c.L1 - 1 - pos;
    const uint32_t n_here = GUARD ? min((uint32_t)kBigItems, c.n_slots - s0) : (uint32_t)kBigItems;
    uint32_t top = 0;
#pragma unroll
    for (int i = 0; i < kBigItems; ++i) {
        if ((i & 7) == 0) top = big_top16(sm, brel);     // at most 7 bases are consumed before the next refill: l <= 7 stay valid
        if (!GUARD || (uint32_t)i < n_here) {
            const uint32_t r = rem < ell ? rem : ell;
            // the first l bases with those past the end of the read cleared (A-padded), then the length: reading A4 of PAPER.md:79
            const uint32_t kmer = (top >> (32 - 2 * ell)) & (0xffffffffu << (2 * (ell - r)));
            f(i, kmer, r);   // partition code = kmer * (ell + 1) + r
            const bool adv = rem != 0;                    // at an end-marker slot the next read starts at the same base index
            top = adv ? top << 2 : top;
            brel += adv;
            rem = adv ? rem - 1 : c.L1 - 1;
        }
    }
}
__global__ void __launch_bounds__(kListThreads) list_count_uniform_kernel(Reads R, const BuildInfo* __restrict__ info, uint32_t ell, CountRanges ranges,
                                                                          uint64_t* __restrict__ tile_count, uint64_t col_stride) {
    __shared__ BigSmem sm;
    __shared__ uint32_t s_total[kCountGroup];
    __shared__ uint32_t s_first[kCountGroup + 1];    // first partition of every batch of the group; unused ones = one past the last
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t n_tiles = (N + kBigTile - 1) / kBigTile;
    if (info->bad_offsets) return;
    if (threadIdx.x <= kCountGroup) s_first[threadIdx.x] = ranges.first[threadIdx.x < ranges.n ? threadIdx.x : ranges.n];
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm and s_total (and the table filled on the first trip)
        if (threadIdx.x < kCountGroup) s_total[threadIdx.x] = 0;
        const BigCtx c = load_big_tile(R, info, t, N, sm);
        uint64_t mine = 0;   // eight 8-bit counters (at most 32 slots per thread)
        const uint32_t s0 = threadIdx.x * kBigItems;
        if (s0 < c.n_slots) {
            auto tally = [&](int, uint32_t kmer, uint32_t r) {
                const uint32_t code = kmer * (ell + 1) + r;
                // which of the group's batches owns the partition: a three-step search of the (at most eight) range starts
                uint32_t j = code >= s_first[4] ? 4u : 0u;
                j += code >= s_first[j + 2] ? 2u : 0u;
                j += code >= s_first[j + 1] ? 1u : 0u;
                if (code >= s_first[0] && code < s_first[kCountGroup]) mine += 1ull << (8 * j);
            };
            if (c.n_slots == (uint32_t)kBigTile) big_walk<false>(c, sm, s0, ell, tally);
            else big_walk<true>(c, sm, s0, ell, tally);
        }
#pragma unroll
        for (int j = 0; j < kCountGroup; ++j) {
            uint32_t v = (uint32_t)(mine >> (8 * j)) & 255u;
            for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane_id() == 0 && v) atomicAdd(&s_total[j], v);
        }
        __syncthreads();
        if (threadIdx.x < ranges.n) tile_count[(uint64_t)threadIdx.x * col_stride + t] = s_total[threadIdx.x];
    }
}

// a2 on the same walk: partition sizes of a collection of equal-length reads (the whole collection, no region).  Counters as in
// bucket_hist_kernel: full-length partitions by l-mer, the short ones behind them.
__global__ void __launch_bounds__(kListThreads) bucket_hist_uniform_kernel(Reads R, const BuildInfo* __restrict__ info, uint32_t ell,
                                                                           unsigned long long* __restrict__ hist) {
    __shared__ BigSmem sm;
    extern __shared__ uint32_t s_hist_u[];
    const uint32_t n_kmers = 1u << (2 * ell), n_short = (n_kmers - 1) / 3;
    for (uint32_t k = threadIdx.x; k < n_kmers + n_short; k += blockDim.x) s_hist_u[k] = 0;
    if (info->bad_offsets || info->nonuniform) return;   // (reads of different lengths: bucket_hist_kernel has it)
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t n_tiles = (N + kBigTile - 1) / kBigTile;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm (and the counters zeroed on the first trip)
        const BigCtx c = load_big_tile(R, info, t, N, sm);
        const uint32_t s0 = threadIdx.x * kBigItems;
        if (s0 < c.n_slots) {
            auto count = [&](int, uint32_t kmer, uint32_t r) {
                const uint32_t at = r == ell ? kmer : n_kmers + (((1u << (2 * r)) - 1) / 3) + (kmer >> (2 * (ell - r)));
                atomicAdd(&s_hist_u[at], 1u);
            };
            if (c.n_slots == (uint32_t)kBigTile) big_walk<false>(c, sm, s0, ell, count);
            else big_walk<true>(c, sm, s0, ell, count);
        }
    }
    __syncthreads();
    for (uint32_t k = threadIdx.x; k < n_kmers; k += blockDim.x) {
        const uint32_t v = s_hist_u[k];
        if (v) atomicAdd(hist + (uint64_t)k * (ell + 1) + ell, (unsigned long long)v);
    }
    for (uint32_t r = 0; r < ell; ++r) {
        const uint32_t first = n_kmers + ((1u << (2 * r)) - 1) / 3, count = 1u << (2 * r);
        for (uint32_t k = threadIdx.x; k < count; k += blockDim.x) {
            const uint32_t v = s_hist_u[first + k];
            if (v) atomicAdd(hist + ((uint64_t)k << (2 * (ell - r))) * (ell + 1) + r, (unsigned long long)v);
        }
    }
}

template <typename KeyT, typename IdT, bool PACKED>
__global__ void __launch_bounds__(kListThreads) list_select_uniform_kernel(Reads R, const BuildInfo* __restrict__ info, uint32_t ell, uint32_t w,
                                                                           uint32_t bucket_lo, uint32_t bucket_hi,
                                                                           const uint64_t* __restrict__ tile_base, KeyT* __restrict__ keys,
                                                                           IdT* __restrict__ ids, uint32_t n_passes,
                                                                           unsigned long long* __restrict__ digit_hist, uint64_t ord_lo, uint64_t ord_hi, uint32_t split) {
    __shared__ BigSmem sm;
    __shared__ uint32_t s_dh[8][kRadix];
    __shared__ uint32_t s_warp[kListThreads / 32];
    __shared__ uint16_t s_taken[kBigTile];   // slots of the tile that belong to the batch, in slot order
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t n_tiles = (N + kBigTile - 1) / kBigTile;
    const uint32_t warp = threadIdx.x >> 5;
    if (info->bad_offsets) return;
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) (&s_dh[0][0])[i] = 0;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with sm, s_warp and s_taken
        const BigCtx c = load_big_tile(R, info, t, N, sm);
        const uint32_t s0 = threadIdx.x * kBigItems;
        uint32_t mask = 0;   // which of my 32 consecutive slots belong to this batch
        if (s0 < c.n_slots) {
            auto mark = [&](int i, uint32_t kmer, uint32_t r) { mask |= (uint32_t)(kmer * (ell + 1) + r - bucket_lo <= bucket_hi - bucket_lo) << i; };
            if (c.n_slots == (uint32_t)kBigTile) big_walk<false>(c, sm, s0, ell, mark);
            else big_walk<true>(c, sm, s0, ell, mark);
        }
        // exclusive scan of the per-thread counts: slot order = thread order
        const uint32_t cnt = __popc(mask);
        uint32_t incl = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t up = __shfl_up_sync(0xffffffffu, incl, o);
            if ((int)lane_id() >= o) incl += up;
        }
        if (lane_id() == 31) s_warp[warp] = incl;
        __syncthreads();
        uint32_t before = incl - cnt, total = 0;
        for (uint32_t q = 0; q < kListThreads / 32; ++q) {
            const uint32_t v = s_warp[q];
            if (q < warp) before += v;
            total += v;
        }
        while (mask) {   // taken slots compacted first, decoded one per thread below (full warps, consecutive output addresses)
            const int i = __ffs(mask) - 1;
            mask &= mask - 1;
            s_taken[before++] = (uint16_t)(s0 + i);
        }
        __syncthreads();
        const uint64_t tile_dst = tile_base[t];
        for (uint32_t j = threadIdx.x; j < total; j += kListThreads) {
            const uint64_t dst = tile_dst + j;
            if (dst >= ord_lo && dst < ord_hi) {
                uint32_t rr, pos, brel;
                big_decode(c, s_taken[j], rr, pos, brel);
                const KeyT key = first_key_as<KeyT>(big_window(sm, brel), (uint64_t)(c.L1 - 1 - pos), w);
                const IdT id = make_id<IdT>(c.r0 + rr, pos, R.pos_bits);
                digit_counts(s_dh, key, n_passes);
                store_pair<KeyT, IdT, PACKED>(keys, ids, dst - ord_lo, key, id, split);
            }
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) {
        uint32_t v = (&s_dh[0][0])[i];
        if (v) atomicAdd(digit_hist + i, (unsigned long long)v);
    }
}

// ---------------------------------------------------------------------------------------------
// The multi-batch scans for reads of ONE length L <= 127 (the paper's 100 bp reads; configs[1], [2], [4]), outside any region:
// ONE READ PER THREAD.  Position p of the read has the same `bases left` in every lane, so the walk has no divergence, no
// per-slot decode and no end-marker bookkeeping: per slot a shift, the partition code and the range test.  A tile is 256
// consecutive reads (256 (L + 1) slots); a thread's slots are consecutive in listing order, so thread order = slot order
// (PAPER.md:99).  Every batch of a collection larger than the workspace walks all slots again, so this walk is
// what the out-of-core build spends its listing time on.
// ---------------------------------------------------------------------------------------------
constexpr int kReadTileWords = kListThreads * kReadMaxLen / 32 + 6;
constexpr int kTakenCap = 8192;                       // taken slots decoded per round

struct ReadTileCtx {
    uint64_t r0;        // first read of the tile
    uint32_t n;         // reads in the tile
    uint32_t L;         // read length
    uint32_t brel0;     // index of read r0's first base among the staged bases
};
__device__ __forceinline__ ReadTileCtx load_read_tile(const Reads& R, const BuildInfo* __restrict__ info, uint64_t t, uint64_t* packed_sm) {
    ReadTileCtx c;
    c.r0 = t * kListThreads;
    c.n = (uint32_t)min((uint64_t)kListThreads, R.n_reads - c.r0);
    c.L = (uint32_t)info->first_len;
    const uint64_t b0 = c.r0 * c.L;
    const uint64_t word0 = b0 >> 5;
    c.brel0 = (uint32_t)(b0 & 31);
    const uint32_t words = (c.brel0 + c.n * c.L + 31) / 32 + 3;   // + the look-ahead of the last read's last windows
    for (uint32_t j = threadIdx.x; j < words; j += blockDim.x) {
        const uint64_t wi = word0 + j;
        packed_sm[j] = wi < R.n_words ? __ldg(R.packed + wi) : 0ull;
    }
#if CX_READ_TILE_PREFETCH
    {   // the tile this block takes next (a grid-width on): ask L2 for its lines now
        const uint64_t next0 = ((t + gridDim.x) * kListThreads * c.L) >> 5;
        const uint64_t wi = next0 + 16ull * threadIdx.x;                    // one 128-byte line per thread
        if (16u * threadIdx.x < words && wi < R.n_words) asm volatile("prefetch.global.L2 [%0];" ::"l"(R.packed + wi));
    }
#endif
    __syncthreads();
    return c;
}
__device__ __forceinline__ uint32_t top16_at(const uint64_t* packed_sm, uint32_t brel) {
    const uint32_t* half = reinterpret_cast<const uint32_t*>(packed_sm);   // 32-bit halves, high half first
    const uint32_t q = brel >> 4, sh = (brel & 15) * 2;
    return __funnelshift_l(half[(q + 1) ^ 1], half[q ^ 1], sh);
}
__device__ __forceinline__ uint64_t window_at(const uint64_t* packed_sm, uint32_t brel) {
    const uint32_t wi = brel >> 5, sh = (brel & 31) * 2;
    const uint64_t w0 = packed_sm[wi], w1 = packed_sm[wi + 1];
    return sh ? (w0 << sh) | (w1 >> (64 - sh)) : w0;
}
// f(partition code) for every position p = 0 .. L of the thread's read (p = L: the end-marker suffix).  Positions with at least
// l bases left (all but the last l of a read) go in blocks of eight without length arithmetic; every branch depends on p, L and
// l only: the same in every lane.
template <typename F>
__device__ __forceinline__ void read_walk(const uint64_t* packed_sm, uint32_t brel, uint32_t L, uint32_t ell, F&& f) {
    const uint32_t e1 = ell + 1, sh = 32 - 2 * ell;
    const uint32_t n_full = L + 1 - ell;              // positions 0 .. n_full - 1 have at least l bases left (L >= kReadMinLen > l)
    uint32_t p = 0;
    for (; p + 8 <= n_full; p += 8) {
        uint32_t top = top16_at(packed_sm, brel + p);   // 16 bases; 8 are consumed: l <= 7 stay valid
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            f((top >> sh) * e1 + ell);
            top <<= 2;
        }
    }
    for (; p <= L; p += 8) {
        uint32_t top = top16_at(packed_sm, brel + p);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const uint32_t q = p + i;
            if (q <= L) {
                const uint32_t left = L - q, r = left < ell ? left : ell;
                // the first l bases with those past the end of the read cleared (A-padded), then the length: reading A4 of PAPER.md:79
                const uint32_t kmer = (top >> sh) & (0xffffffffu << (2 * (ell - r)));
                f(kmer * e1 + r);
            }
            top <<= 2;
        }
    }
}

// The same walk for the select scan: which positions of the read belong to the partition range [lo, hi]?  Bit p of (mhi:mlo).
// Positions with at least l bases left (all but the last l of a read) are taken in blocks of eight with a range test on the raw
// l-mer: code = kmer (l + 1) + l in [lo, hi]  <=>  kmer - klo <= kspan; only the blocks that reach the read's end pay for the
// length arithmetic.  Every branch depends on p, L and l only: the same in every lane.
__device__ __forceinline__ void read_select_walk(const uint64_t* packed_sm, uint32_t brel, uint32_t L, uint32_t ell, uint32_t lo, uint32_t hi,
                                                 uint64_t& mlo, uint64_t& mhi) {
    const uint32_t e1 = ell + 1, sh = 32 - 2 * ell;
    uint32_t klo = lo / e1, kspan = 0;
    if (hi >= ell && (hi - ell) / e1 >= klo) kspan = (hi - ell) / e1 - klo;
    else klo = 0xffffffffu;                           // no full-length partition in the range: kmer - klo <= 0 never holds
    const uint32_t n_full = L + 1 - ell;              // positions 0 .. n_full - 1 have at least l bases left (L >= kReadMinLen > l)
    mlo = 0, mhi = 0;
    uint32_t p = 0;
    for (; p + 8 <= n_full; p += 8) {
        uint32_t top = top16_at(packed_sm, brel + p);
        uint32_t acc = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            acc |= (uint32_t)((top >> sh) - klo <= kspan) << i;
            top <<= 2;
        }
        if (p < 64) mlo |= (uint64_t)acc << p;
        else mhi |= (uint64_t)acc << (p - 64);
    }
    for (; p <= L; p += 8) {                          // the rest: up to 7 full-length positions and the l + 1 that end inside the prefix
        uint32_t top = top16_at(packed_sm, brel + p);
        uint32_t acc = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const uint32_t q = p + i;
            if (q <= L) {
                const uint32_t left = L - q, r = left < ell ? left : ell;
                const uint32_t kmer = (top >> sh) & (0xffffffffu << (2 * (ell - r)));   // bases past the end of the read cleared (A4)
                acc |= (uint32_t)(kmer * e1 + r - lo <= hi - lo) << i;
            }
            top <<= 2;
        }
        if (p < 64) mlo |= (uint64_t)acc << p;
        else mhi |= (uint64_t)acc << (p - 64);
    }
}

__global__ void __launch_bounds__(kListThreads) list_count_reads_kernel(Reads R, const BuildInfo* __restrict__ info, uint32_t ell, CountRanges ranges,
                                                                        uint64_t* __restrict__ tile_count, uint64_t col_stride) {
    __shared__ uint64_t s_packed[kReadTileWords];
    __shared__ uint32_t s_total[kCountGroup];
    __shared__ uint32_t s_first[kCountGroup + 1];    // first partition of every batch of the group; unused ones = one past the last
    R.n_words = (info->total_bases + 31) >> 5;
    if (info->bad_offsets) return;
    const uint64_t n_tiles = (R.n_reads + kListThreads - 1) / kListThreads;
    if (threadIdx.x <= kCountGroup) s_first[threadIdx.x] = ranges.first[threadIdx.x < ranges.n ? threadIdx.x : ranges.n];
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with s_packed and s_total
        if (threadIdx.x < kCountGroup) s_total[threadIdx.x] = 0;
        const ReadTileCtx c = load_read_tile(R, info, t, s_packed);
        uint64_t mine = 0;   // eight 8-bit counters (at most 128 slots per thread)
        if (threadIdx.x < c.n) {
            read_walk(s_packed, c.brel0 + threadIdx.x * c.L, c.L, ell, [&](uint32_t code) {
                uint32_t j = code >= s_first[4] ? 4u : 0u;   // which of the group's batches owns the partition
                j += code >= s_first[j + 2] ? 2u : 0u;
                j += code >= s_first[j + 1] ? 1u : 0u;
                if (code >= s_first[0] && code < s_first[kCountGroup]) mine += 1ull << (8 * j);
            });
        }
#pragma unroll
        for (int j = 0; j < kCountGroup; ++j) {
            uint32_t v = (uint32_t)(mine >> (8 * j)) & 255u;
            for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane_id() == 0 && v) atomicAdd(&s_total[j], v);
        }
        __syncthreads();
        if (threadIdx.x < ranges.n) tile_count[(uint64_t)threadIdx.x * col_stride + t] = s_total[threadIdx.x];
    }
}

template <typename KeyT, typename IdT, bool PACKED>
__global__ void __launch_bounds__(kListThreads) list_select_reads_kernel(Reads R, const BuildInfo* __restrict__ info, uint32_t ell, uint32_t w,
                                                                         uint32_t bucket_lo, uint32_t bucket_hi,
                                                                         const uint64_t* __restrict__ tile_base, KeyT* __restrict__ keys,
                                                                         IdT* __restrict__ ids, uint32_t n_passes,
                                                                         unsigned long long* __restrict__ digit_hist, uint64_t ord_lo, uint64_t ord_hi, uint32_t split) {
    __shared__ uint64_t s_packed[kReadTileWords];
    __shared__ uint32_t s_dh[8][kRadix];
    __shared__ uint32_t s_warp[kListThreads / 32];
    __shared__ uint16_t s_taken[kTakenCap];   // slots of the tile that belong to the batch, in slot order, one round's worth
    R.n_words = (info->total_bases + 31) >> 5;
    if (info->bad_offsets) return;
    const uint64_t n_tiles = (R.n_reads + kListThreads - 1) / kListThreads;
    const uint32_t warp = threadIdx.x >> 5;
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) (&s_dh[0][0])[i] = 0;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        __syncthreads();   // previous tile done with s_packed, s_warp and s_taken
        const ReadTileCtx c = load_read_tile(R, info, t, s_packed);
        uint64_t mlo = 0, mhi = 0;   // which of my read's slots belong to this batch (position p -> bit p)
        if (threadIdx.x < c.n) read_select_walk(s_packed, c.brel0 + threadIdx.x * c.L, c.L, ell, bucket_lo, bucket_hi, mlo, mhi);
        // exclusive scan of the per-thread counts: slot order = thread order
        const uint32_t cnt = (uint32_t)__popcll(mlo) + (uint32_t)__popcll(mhi);
        uint32_t incl = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t up = __shfl_up_sync(0xffffffffu, incl, o);
            if ((int)lane_id() >= o) incl += up;
        }
        if (lane_id() == 31) s_warp[warp] = incl;
        __syncthreads();
        uint32_t before = incl - cnt, total = 0;
        for (uint32_t q = 0; q < kListThreads / 32; ++q) {
            const uint32_t v = s_warp[q];
            if (q < warp) before += v;
            total += v;
        }
        const uint64_t tile_dst = tile_base[t];
        // taken slots are compacted (slot order) and then decoded one per thread: full warps, consecutive output addresses;
        // kTakenCap of them per round (one round unless the batch takes a large share of the collection)
        for (uint32_t round0 = 0; round0 < total; round0 += kTakenCap) {
            if (round0) __syncthreads();   // the previous round's decode is done with s_taken
            uint32_t at = before;
            auto put = [&](uint64_t m, uint32_t p0) {
                while (m) {
                    const uint32_t i = (uint32_t)__ffsll((long long)m) - 1;
                    m &= m - 1;
                    if (at - round0 < (uint32_t)kTakenCap) s_taken[at - round0] = (uint16_t)((threadIdx.x << 7) | (p0 + i));   // (unsigned: below round0 wraps high)
                    ++at;
                }
            };
            put(mlo, 0), put(mhi, 64);
            __syncthreads();
            const uint32_t here = min((uint32_t)kTakenCap, total - round0);
            for (uint32_t j = threadIdx.x; j < here; j += kListThreads) {
                const uint64_t dst = tile_dst + round0 + j;
                if (dst >= ord_lo && dst < ord_hi) {
                    const uint32_t sl = s_taken[j];
                    const uint32_t rr = sl >> 7, pos = sl & 127u;   // (thread = read of the tile, position)
                    const KeyT key = first_key_as<KeyT>(window_at(s_packed, c.brel0 + rr * c.L + pos), (uint64_t)(c.L - pos), w);
                    const IdT id = make_id<IdT>(c.r0 + rr, pos, R.pos_bits);
                    digit_counts(s_dh, key, n_passes);
                    store_pair<KeyT, IdT, PACKED>(keys, ids, dst - ord_lo, key, id, split);
                }
            }
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) {
        uint32_t v = (&s_dh[0][0])[i];
        if (v) atomicAdd(digit_hist + i, (unsigned long long)v);
    }
}

// ---------------------------------------------------------------------------------------------
// a4 + a5 (+ a2) for a collection of equal-length reads (16..127 bases) that is sorted as ONE batch (configs[0..2]):
// list_write_kernel's work with one read per thread.  Everything that depends on the position p is the same in every lane:
// positions with at least w bases left take a key without masking, those with at least l a partition counter without length
// arithmetic.  A thread's (key, id) words are consecutive in the output, so they are staged in shared memory eight positions
// at a time (rows padded to nine words: conflict-free) and leave as runs of 64 bytes.
// ---------------------------------------------------------------------------------------------
constexpr int kStageCols = 8, kStagePitch = kStageCols + 1;
template <typename KeyT, typename IdT, bool PACKED>
__global__ void __launch_bounds__(kListThreads) list_write_reads_kernel(Reads R, const BuildInfo* __restrict__ info, uint32_t ell, uint32_t w,
                                                                        KeyT* __restrict__ keys, IdT* __restrict__ ids, uint32_t n_passes,
                                                                        unsigned long long* __restrict__ digit_hist,
                                                                        unsigned long long* __restrict__ bucket_hist, uint64_t max_n) {
    __shared__ uint64_t s_packed[kReadTileWords];
    // digit counts of every radix pass of the sort that follows (a6's upfront histogram), one 16-bit counter per (pass, digit,
    // lane): lanes 2k and 2k + 1 share a word, every lane pair has a bank of its own -- at most a 2-way bank conflict where
    // counters indexed by the digit alone see 3.4 lanes per bank with random digits.  Flushed before a counter can overflow.
    __shared__ uint64_t s_stage[kListThreads * kStagePitch];   // PACKED: key << 32 | id; else keys, and ids in s_stage_id
    extern __shared__ __align__(8) unsigned char s_dyn[];      // [!PACKED: id staging rows][partition counters, laid out as in bucket_hist_kernel]
    uint64_t* s_stage_id = reinterpret_cast<uint64_t*>(s_dyn);
    uint32_t* s_dl = reinterpret_cast<uint32_t*>(s_dyn + (PACKED ? 0 : sizeof(uint64_t) * kListThreads * kStagePitch));   // [pass][digit][16]
    uint32_t* s_bh = s_dl + n_passes * kRadix * 16;
    const uint32_t n_kmers = 1u << (2 * ell), n_short = (n_kmers - 1) / 3;
    if (bucket_hist)
        for (uint32_t k = threadIdx.x; k < n_kmers + n_short; k += blockDim.x) s_bh[k] = 0;
    R.n_words = (info->total_bases + 31) >> 5;
    const uint64_t N = info->n_suffixes;
    const uint64_t L64 = info->first_len;
    if (N > max_n || info->bad_offsets || info->nonuniform || L64 < (uint64_t)kReadMinLen || L64 > (uint64_t)kReadMaxLen) return;   // list_write_kernel has it
    const uint64_t n_tiles = (R.n_reads + kListThreads - 1) / kListThreads;
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix * 16; i += kListThreads) s_dl[i] = 0;
    const uint32_t tid = threadIdx.x;
    const uint32_t my_word = (tid & 31) >> 1, my_inc = (tid & 1) ? 0x10000u : 1u;
    auto flush_digits = [&]() {   // all threads; the counters are zero afterwards
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kListThreads) {
            uint32_t sum = 0;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const uint32_t v = s_dl[i * 16 + q];
                sum += (v & 0xffffu) + (v >> 16);
                s_dl[i * 16 + q] = 0;
            }
            if (sum) atomicAdd(digit_hist + i, (unsigned long long)sum);
        }
        __syncthreads();
    };
    uint32_t tiles_since_flush = 0;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        // a counter takes at most 8 warps x 128 positions per tile: flush before 65535
        if (++tiles_since_flush > 60) flush_digits(), tiles_since_flush = 1;
        __syncthreads();   // previous tile done with s_packed and the staging rows (and the counters zeroed on the first trip)
        const ReadTileCtx c = load_read_tile(R, info, t, s_packed);
        const uint32_t L = c.L, L1 = L + 1;
        const bool have = tid < c.n;
        const uint32_t brel = c.brel0 + tid * L;
        const uint64_t id_hi = (c.r0 + tid) << R.pos_bits;
        uint64_t win = 0;
        for (uint32_t p0 = 0; p0 <= L; p0 += kStageCols) {
            if ((p0 & 15) == 0 && have) win = window_at(s_packed, brel + p0);   // 32 bases; 16 are consumed before the next refill: w <= 16 stay valid
#pragma unroll
            for (int i = 0; i < kStageCols; ++i) {
                const uint32_t p = p0 + i;
                if (p <= L && have) {                         // (p <= L: the same in every lane)
                    const uint32_t left = L - p;
                    if (bucket_hist) {
                        if (left >= ell) {
                            atomicAdd(&s_bh[(uint32_t)(win >> (64 - 2 * ell))], 1u);
                        } else {
                            const uint32_t kmer = (uint32_t)(win >> (64 - 2 * ell)) & (0xffffffffu << (2 * (ell - left)));
                            atomicAdd(&s_bh[n_kmers + (((1u << (2 * left)) - 1) / 3) + (kmer >> (2 * (ell - left)))], 1u);
                        }
                    }
                    const KeyT key = first_key_as<KeyT>(win, (uint64_t)left, w);
#pragma unroll
                    for (uint32_t q = 0; q < sizeof(KeyT); ++q)
                        if (q < n_passes) atomicAdd(&s_dl[((q * kRadix + ((uint32_t)(key >> (q * kRadixBits)) & (kRadix - 1))) << 4) + my_word], my_inc);
                    if constexpr (PACKED) {
                        s_stage[tid * kStagePitch + i] = ((uint64_t)key << 32) | id_hi | p;
                    } else {
                        s_stage[tid * kStagePitch + i] = (uint64_t)key;
                        s_stage_id[tid * kStagePitch + i] = id_hi | p;
                    }
                    win <<= 2;
                }
            }
            __syncthreads();
            // the block's rows of eight words leave in slot order: word q of the block = (read q / 8, position p0 + q % 8)
            const uint32_t cols = min((uint32_t)kStageCols, L1 - p0);
            for (uint32_t q = tid; q < c.n * kStageCols; q += kListThreads) {
                const uint32_t rr = q / kStageCols, k = q % kStageCols;
                if (k < cols) {
                    const uint64_t at = (c.r0 + rr) * L1 + p0 + k;
                    if constexpr (PACKED) {
                        reinterpret_cast<uint64_t*>(keys)[at] = s_stage[rr * kStagePitch + k];
                    } else {
                        keys[at] = (KeyT)s_stage[rr * kStagePitch + k];
                        ids[at] = (IdT)s_stage_id[rr * kStagePitch + k];
                    }
                }
            }
            __syncthreads();
        }
    }
    flush_digits();
    if (bucket_hist) {
        for (uint32_t k = threadIdx.x; k < n_kmers; k += blockDim.x) {
            uint32_t v = s_bh[k];
            if (v) atomicAdd(bucket_hist + (uint64_t)k * (ell + 1) + ell, (unsigned long long)v);
        }
        for (uint32_t r = 0; r < ell; ++r) {
            const uint32_t first = n_kmers + ((1u << (2 * r)) - 1) / 3, count = 1u << (2 * r);
            for (uint32_t k = threadIdx.x; k < count; k += blockDim.x) {
                uint32_t v = s_bh[first + k];
                if (v) atomicAdd(bucket_hist + ((uint64_t)k << (2 * (ell - r))) * (ell + 1) + r, (unsigned long long)v);
            }
        }
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
// the multi-batch scans of a collection of equal-length reads outside a refined region run on tiles of kBigTile slots
static bool big_tiles(const Reads& R, const Region& region) { return R.uniform && region.depth == 0; }
// ... and one read per thread when that length is 16 .. 127 bases (tiles of 256 reads)
static bool read_tiles(const Reads& R, const Region& region) {
    return big_tiles(R, region) && R.uniform_len >= (uint64_t)kReadMinLen && R.uniform_len <= (uint64_t)kReadMaxLen;
}
uint64_t list_scan_tiles(const Reads& R, const Region& region, uint64_t n_suffixes) {
    if (read_tiles(R, region)) return (R.n_reads + kListThreads - 1) / kListThreads;
    const uint64_t tile = big_tiles(R, region) ? (uint64_t)kBigTile : (uint64_t)kListTile;
    return (n_suffixes + tile - 1) / tile;
}

cudaError_t launch_prep(const uint64_t* offsets, uint64_t n_reads, uint64_t max_bases, BuildInfo* info, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(info, 0, sizeof(BuildInfo), s);
    if (e != cudaSuccess) return e;
    uint64_t blocks = (n_reads + 255) / 256;
    const uint64_t want = (uint64_t)sm_count() * 8;
    unsigned grid = (unsigned)(blocks < want ? (blocks ? blocks : 1) : want);
    prep_kernel<<<grid, 256, 0, s>>>(offsets, n_reads, max_bases, info);
    return cudaGetLastError();
}

cudaError_t launch_tile_table(const uint64_t* offsets, uint64_t n_reads, const BuildInfo* info, uint32_t* tile_first_read,
                              uint64_t max_tiles, cudaStream_t s) {
    if (max_tiles == 0) return cudaSuccess;
    unsigned grid = (unsigned)((max_tiles + 255) / 256);
    tile_table_kernel<<<grid, 256, 0, s>>>(offsets, n_reads, info, tile_first_read, max_tiles);
    return cudaGetLastError();
}

size_t bucket_hist_smem(uint32_t ell) { return sizeof(TileSmem) + (sizeof(uint32_t) << (2 * ell)) + sizeof(uint32_t) * (((1u << (2 * ell)) - 1) / 3); }

cudaError_t launch_bucket_hist(const Reads& R, const BuildInfo* info, const uint32_t* tile_first_read, uint32_t ell, const Region& region,
                               uint64_t* hist, uint64_t max_tiles, int n_sms, cudaStream_t s) {
    if (max_tiles == 0) return cudaSuccess;
    size_t smem = bucket_hist_smem(ell);
    cudaError_t e = cudaFuncSetAttribute(bucket_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bucket_hist_smem(7));
    if (e != cudaSuccess) return e;
    int per_sm = ell <= 6 ? 4 : 2;
    uint64_t want = (uint64_t)n_sms * per_sm;
    unsigned grid = (unsigned)(max_tiles < want ? max_tiles : want);
    // Reads of one length outside a region (the DEVICE knows; the host may not have read BuildInfo yet) are counted on the
    // 8192-slot walk, anything else by the general kernel: both are launched, the one that does not apply returns at once.
    const uint32_t skip_uniform = region.depth == 0;
    if (skip_uniform) {
        const size_t smem_u = smem - sizeof(TileSmem);
        e = cudaFuncSetAttribute(bucket_hist_uniform_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bucket_hist_smem(7) - sizeof(TileSmem)));
        if (e != cudaSuccess) return e;
        const uint64_t big = (max_tiles * kListTile + kBigTile - 1) / kBigTile;
        bucket_hist_uniform_kernel<<<(unsigned)(big < want ? big : want), kListThreads, smem_u, s>>>(R, info, ell, (unsigned long long*)hist);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    bucket_hist_kernel<<<grid, kListThreads, smem, s>>>(R, info, tile_first_read, ell, region, (unsigned long long*)hist, skip_uniform);
    return cudaGetLastError();
}

cudaError_t launch_list_count(const Reads& R, const BuildInfo* info, const uint32_t* tile_first_read, uint32_t ell, const Region& region,
                              const CountRanges& ranges, uint64_t* tile_count, uint64_t col_stride, uint64_t n_tiles, cudaStream_t s) {
    if (n_tiles == 0 || ranges.n == 0) return cudaSuccess;
    uint64_t want = (uint64_t)sm_count() * 8;
    const unsigned grid = (unsigned)(n_tiles < want ? n_tiles : want);
    if (read_tiles(R, region)) {  // n_tiles counts tiles of 256 reads here (list_scan_tiles)
        list_count_reads_kernel<<<grid, kListThreads, 0, s>>>(R, info, ell, ranges, tile_count, col_stride);
        return cudaGetLastError();
    }
    if (big_tiles(R, region)) {   // n_tiles counts tiles of kBigTile slots here (list_scan_tiles)
        list_count_uniform_kernel<<<grid, kListThreads, 0, s>>>(R, info, ell, ranges, tile_count, col_stride);
        return cudaGetLastError();
    }
    if (region.depth)
        list_count_kernel<true><<<grid, kListThreads, 0, s>>>(R, info, tile_first_read, ell, region, ranges, tile_count, col_stride);
    else
        list_count_kernel<false><<<grid, kListThreads, 0, s>>>(R, info, tile_first_read, ell, region, ranges, tile_count, col_stride);
    return cudaGetLastError();
}

template <typename KeyT, typename IdT>
cudaError_t launch_list_write(const Reads& R, const BuildInfo* info, const uint32_t* tile_first_read, uint32_t ell, uint32_t w,
                              uint32_t bucket_lo, uint32_t bucket_hi, const uint64_t* tile_base, KeyT* keys, IdT* ids,
                              uint64_t n_tiles, uint32_t n_passes, uint64_t* digit_hist, int n_sms, bool packed, uint64_t* bucket_hist,
                              uint64_t max_n, const Region& region, uint64_t ord_lo, uint64_t ord_hi, cudaStream_t s, uint32_t split) {
    if (n_tiles == 0) return cudaSuccess;
    uint64_t want = (uint64_t)n_sms * (bucket_hist ? 4 : 6);
    unsigned grid = (unsigned)(n_tiles < want ? n_tiles : want);
    unsigned long long* dh = (unsigned long long*)digit_hist;
    unsigned long long* bh = (unsigned long long*)bucket_hist;
    constexpr bool kCanPack = sizeof(KeyT) == 4 && sizeof(IdT) == 4;
    if ((packed && !kCanPack) || (bucket_hist && tile_base)) return cudaErrorInvalidValue;
    if (split && (tile_base == nullptr || packed || sizeof(KeyT) != 8 || sizeof(IdT) != 8)) return cudaErrorInvalidValue;   // select scans only
    const size_t smem = bucket_hist ? bucket_hist_smem(ell) - sizeof(TileSmem) : 0;
    const uint32_t skip_reads = tile_base == nullptr && w <= 16 && !region.depth && R.n_reads > 0;   // (a register pair holds the 16 bases a key may need)
    auto launch = [&](auto kernel) {
        if (smem) {
            cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bucket_hist_smem(7) - sizeof(TileSmem)));
            if (e != cudaSuccess) return e;
        }
        kernel<<<grid, kListThreads, smem, s>>>(R, info, tile_first_read, ell, w, keys, ids, n_passes, dh, bh, max_n, skip_reads);
        return cudaGetLastError();
    };
    if (tile_base == nullptr) {
        // Reads of one length of 16..127 bases (the paper's setting; the DEVICE knows, the host may not have read BuildInfo yet) are
        // listed one read per thread, any other collection by the general kernel: both are launched, the one that does not apply
        // returns at once.
        if (skip_reads) {
            auto kernel = packed ? list_write_reads_kernel<KeyT, IdT, kCanPack> : list_write_reads_kernel<KeyT, IdT, false>;
            const size_t stage_id = (packed ? 0 : sizeof(uint64_t) * kListThreads * kStagePitch) + (size_t)n_passes * kRadix * 16 * sizeof(uint32_t);
            const size_t smem_r = smem + stage_id;
            cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r);
            if (e != cudaSuccess) return e;
            int per_sm = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kListThreads, smem_r);
            if (e != cudaSuccess) return e;
            const uint64_t resident = (uint64_t)n_sms * (per_sm > 0 ? per_sm : 1);
            const uint64_t tiles = (R.n_reads + kListThreads - 1) / kListThreads;
            kernel<<<(unsigned)(tiles < resident ? tiles : resident), kListThreads, smem_r, s>>>(R, info, ell, w, keys, ids, n_passes, dh, bh, max_n);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
        return packed ? launch(list_write_kernel<KeyT, IdT, kCanPack>) : launch(list_write_kernel<KeyT, IdT, false>);
    }
    auto select = [&](auto kernel) {
        // persistent blocks: exactly as many as are resident at once (48 registers: five per SM); a sixth per SM would
        // run as a second wave on an almost empty machine
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kListThreads, 0);
        if (e != cudaSuccess) return e;
        const uint64_t resident = (uint64_t)n_sms * (per_sm > 0 ? per_sm : 1);
        const unsigned grid = (unsigned)(n_tiles < resident ? n_tiles : resident);
        kernel<<<grid, kListThreads, 0, s>>>(R, info, tile_first_read, ell, w, bucket_lo, bucket_hi, tile_base, keys, ids, n_passes, dh, region, ord_lo,
                                             ord_hi, split);
        return cudaGetLastError();
    };
    if (read_tiles(R, region)) {
        auto kernel = packed ? list_select_reads_kernel<KeyT, IdT, kCanPack> : list_select_reads_kernel<KeyT, IdT, false>;
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kListThreads, 0);
        if (e != cudaSuccess) return e;
        const uint64_t resident = (uint64_t)n_sms * (per_sm > 0 ? per_sm : 1);
        kernel<<<(unsigned)(n_tiles < resident ? n_tiles : resident), kListThreads, 0, s>>>(R, info, ell, w, bucket_lo, bucket_hi, tile_base, keys, ids, n_passes, dh,
                                                                                          ord_lo, ord_hi, split);
        return cudaGetLastError();
    }
    if (big_tiles(R, region)) {
        auto kernel = packed ? list_select_uniform_kernel<KeyT, IdT, kCanPack> : list_select_uniform_kernel<KeyT, IdT, false>;
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kListThreads, 0);
        if (e != cudaSuccess) return e;
        const uint64_t resident = (uint64_t)n_sms * (per_sm > 0 ? per_sm : 1);
        kernel<<<(unsigned)(n_tiles < resident ? n_tiles : resident), kListThreads, 0, s>>>(R, info, ell, w, bucket_lo, bucket_hi, tile_base, keys, ids, n_passes, dh,
                                                                                          ord_lo, ord_hi, split);
        return cudaGetLastError();
    }
    if (region.depth) return packed ? select(list_select_kernel<KeyT, IdT, kCanPack, true>) : select(list_select_kernel<KeyT, IdT, false, true>);
    return packed ? select(list_select_kernel<KeyT, IdT, kCanPack, false>) : select(list_select_kernel<KeyT, IdT, false, false>);
}

#define CX_LIST_INST(K, I)                                                                                                        \
    template cudaError_t launch_list_write<K, I>(const Reads&, const BuildInfo*, const uint32_t*, uint32_t, uint32_t, uint32_t,  \
                                                 uint32_t, const uint64_t*, K*, I*, uint64_t, uint32_t, uint64_t*, int, bool, uint64_t*, uint64_t, const Region&,     \
                                                 uint64_t, uint64_t, cudaStream_t, uint32_t);
CX_LIST_INST(uint32_t, uint32_t)
CX_LIST_INST(uint32_t, uint64_t)
CX_LIST_INST(uint64_t, uint32_t)
CX_LIST_INST(uint64_t, uint64_t)

}  // namespace cx
