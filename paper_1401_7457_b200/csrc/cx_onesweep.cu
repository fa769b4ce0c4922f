// cx_onesweep.cu -- step a6: stable LSD radix sort of (64-bit key, suffix id) pairs
// (PAPER.md:91 LSD radix sort over several characters per iteration; "sorting by
// index"; PAPER.md:99 the sort must be stable).
//
// "Onesweep" structure: one upfront kernel builds the digit histograms of every pass; then each
// pass reads every pair once and scatter-writes it once.  A tile learns how many equal-digit pairs
// precede it from the tile-state words of earlier tiles (decoupled look-back), so there is no
// separate scan between passes.  Within a tile, ranks come from warp match + popc (multi-split),
// pairs are staged in shared memory in digit order and leave as runs of consecutive addresses.
//
// Algorithmic traffic per pass: 2 * (8 + sizeof(id)) bytes per pair; histogram kernel: 8 bytes per pair.
#include <stdio.h>

#include "cx_internal.cuh"
#include "cx_launch.h"

namespace cx {
namespace {

constexpr uint32_t kFull = 0xffffffffu;
constexpr int kLookWindow = 4;   // tile states fetched per look-back round trip

__device__ __forceinline__ uint64_t pack_status(uint32_t epoch, uint32_t flag, uint64_t value) {
    return ((uint64_t)epoch << 56) | ((uint64_t)flag << 54) | value;
}

// ---------------------------------------------------------------------------------------------
// upfront histograms: hist[p][d] = number of keys whose p-th digit is d
// ---------------------------------------------------------------------------------------------
constexpr int kHistThreads = 512;
constexpr int kHistItems = 8;

template <typename KeyT>
__global__ void __launch_bounds__(kHistThreads) digit_hist_kernel(const KeyT* __restrict__ keys, uint64_t n, uint32_t begin_bit,
                                                                 uint32_t end_bit, uint32_t n_passes,
                                                                 unsigned long long* __restrict__ hist) {
    __shared__ uint32_t s_hist[8][kRadix];
    for (uint32_t i = threadIdx.x; i < 8 * kRadix; i += kHistThreads) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const uint64_t chunk = (uint64_t)kHistThreads * kHistItems;
    for (uint64_t base = (uint64_t)blockIdx.x * chunk; base < n; base += (uint64_t)gridDim.x * chunk) {
        KeyT k[kHistItems];
#pragma unroll
        for (int i = 0; i < kHistItems; ++i) {
            uint64_t idx = base + (uint64_t)i * kHistThreads + threadIdx.x;
            k[i] = idx < n ? __ldcs(keys + idx) : (KeyT)0;
        }
#pragma unroll
        for (int i = 0; i < kHistItems; ++i) {
            uint64_t idx = base + (uint64_t)i * kHistThreads + threadIdx.x;
            if (idx < n) {
                for (uint32_t p = 0; p < n_passes; ++p) {
                    uint32_t lo = begin_bit + p * kRadixBits;
                    uint32_t bits = min((uint32_t)kRadixBits, end_bit - lo);
                    uint32_t d = (uint32_t)(k[i] >> lo) & ((1u << bits) - 1);
                    atomicAdd(&s_hist[p][d], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n_passes * kRadix; i += kHistThreads) {
        uint32_t v = (&s_hist[0][0])[i];
        if (v) atomicAdd(hist + i, (unsigned long long)v);
    }
}

// exclusive scan of each pass's 256 counts, in place: hist[p][d] becomes the first output index of digit d
__global__ void __launch_bounds__(kRadix) bin_scan_kernel(unsigned long long* __restrict__ hist) {
    __shared__ unsigned long long s_warp[kRadix / 32];
    unsigned long long* h = hist + (uint64_t)blockIdx.x * kRadix;
    unsigned long long v = h[threadIdx.x];
    unsigned long long incl = v;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long up = __shfl_up_sync(kFull, incl, o);
        if ((int)lane_id() >= o) incl += up;
    }
    if (lane_id() == 31) s_warp[threadIdx.x >> 5] = incl;
    __syncthreads();
    unsigned long long carry = 0;
    for (uint32_t wq = 0; wq < (threadIdx.x >> 5); ++wq) carry += s_warp[wq];
    h[threadIdx.x] = carry + incl - v;
}

// ---------------------------------------------------------------------------------------------
// one onesweep pass
// ---------------------------------------------------------------------------------------------
template <typename KeyT, typename ValT, int THREADS, int ITEMS>
struct PassSmem {
    static constexpr int kTile = THREADS * ITEMS;
    static constexpr int kWarps = THREADS / 32;
    static constexpr bool kHasVals = sizeof(ValT) >= 4;
    KeyT keys[kTile];
    ValT vals[kHasVals ? kTile : 1];
    alignas(16) uint32_t warp_count[kWarps][kRadix];  // per-warp digit counts, then the staged slot of the warp's first pair of that digit
    uint32_t gofs[kRadix];                // output index of staged slot e with digit d = gofs[d] + e (mod 2^32; batches are < 2^32)
    uint32_t warp_total[kRadix / 32];
    uint32_t tile;
};

// p &= (my bit B set) ? ballot : ~ballot, as LOP3.P, VOTE, SEL, LOP3 (nvcc's own code for the C++ form takes six)
template <int B>
__device__ __forceinline__ void ballot_step(uint32_t& p, uint32_t d) {
    asm("{\n\t.reg .pred q;\n\t.reg .b32 t, v, m;\n\t"
        "and.b32 t, %1, %2;\n\tsetp.ne.u32 q, t, 0;\n\t"
        "vote.sync.ballot.b32 v, q, 0xffffffff;\n\t"
        "selp.b32 m, 0, 0xffffffff, q;\n\t"
        "lop3.b32 %0, %0, v, m, 0x60;\n\t}"
        : "+r"(p)
        : "r"(d), "n"(1u << B));
}
template <int B, int END>
__device__ __forceinline__ void ballot_steps(uint32_t& p, uint32_t d) {
    if constexpr (B < END) {
        ballot_step<B>(p, d);
        ballot_steps<B + 1, END>(p, d);
    }
}

// Lanes of the warp whose 8-bit digit equals mine: eight ballot steps.
__device__ __forceinline__ uint32_t digit_peers(uint32_t d) {
    uint32_t p = kFull;
    ballot_steps<0, kRadixBits>(p, d);
    return p;
}

template <typename KeyT, typename ValT, int THREADS, int ITEMS, int MIN_BLOCKS>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
onesweep_pass_kernel(const KeyT* __restrict__ keys_in, const ValT* __restrict__ vals_in, KeyT* __restrict__ keys_out,
                     ValT* __restrict__ vals_out, uint64_t n, uint32_t shift, uint32_t digit_mask,
                     const uint64_t* __restrict__ bin_base, uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                     uint32_t ticket_base, uint32_t epoch, uint32_t prefetch_tiles) {
    using Smem = PassSmem<KeyT, ValT, THREADS, ITEMS>;
    constexpr int kTile = Smem::kTile;
    constexpr int kWarps = Smem::kWarps;
    constexpr bool kHasVals = Smem::kHasVals;
    static_assert(THREADS >= kRadix && THREADS % 32 == 0, "one thread per digit is required");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // Tiles are claimed in launch order of the blocks, so every earlier tile is owned by a block that
    // is already running: the look-back below can never wait on a block that has not started.
    if (tid == 0) sm.tile = atomicAdd(ticket, 1u) - ticket_base;
    {
        uint4* wc = reinterpret_cast<uint4*>(&sm.warp_count[0][0]);
        for (uint32_t i = tid; i < kWarps * kRadix / 4; i += THREADS) wc[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    const uint32_t tile = sm.tile;
    const uint32_t tile_off = tile * (uint32_t)kTile;
    // The tile that a block started now will claim in about one grid-width of tickets: ask L2 for it (one bulk prefetch per
    // array), so that its loads find their lines there instead of paying the HBM round trip at the head of the tile.
    if (tid == 0) {
        const uint64_t ahead = (uint64_t)tile_off + (uint64_t)prefetch_tiles * kTile;
        if (ahead + kTile <= n) {
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(keys_in + ahead), "r"((uint32_t)(kTile * sizeof(KeyT))) : "memory");
            if constexpr (kHasVals)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(vals_in + ahead), "r"((uint32_t)(kTile * sizeof(ValT))) : "memory");
        }
    }
    const uint32_t tile_n = (uint32_t)min((uint64_t)kTile, n - tile_off);
    const bool full = tile_n == (uint32_t)kTile;
    const uint32_t warp_base = warp * (32 * ITEMS);

    // warp-striped loads: element order inside the tile = (warp, item, lane); fully coalesced.
    // Slots past the end of the input get the all-ones key: they rank last in the last digit and are
    // never written out.
    KeyT key[ITEMS];
    ValT val[ITEMS];
    {
        const KeyT* kp = keys_in + tile_off + warp_base + lane;
        const ValT* vp = vals_in + tile_off + warp_base + lane;
        if (full) {
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) key[k] = __ldcs(kp + k * 32);
            if constexpr (kHasVals) {
#pragma unroll
                for (int k = 0; k < ITEMS; ++k) val[k] = __ldcs(vp + k * 32);
            }
        } else {
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) key[k] = warp_base + k * 32 + lane < tile_n ? __ldcs(kp + k * 32) : (KeyT)~(KeyT)0;
            if constexpr (kHasVals) {
#pragma unroll
                for (int k = 0; k < ITEMS; ++k) val[k] = warp_base + k * 32 + lane < tile_n ? __ldcs(vp + k * 32) : ValT{};
            }
        }
    }

    // per-(warp, digit) counts first ("early counts"): the tile's digit totals can then be published before the
    // ranking work, so that by the time a successor looks back they are visible and it does not spin
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) atomicAdd(&sm.warp_count[warp][(uint32_t)(key[k] >> shift) & digit_mask], 1u);
    __syncthreads();

    // per digit: tile count, tile-state publication, staged slot of every (warp, digit)
    uint32_t count = 0, excl = 0;
    if (tid < kRadix) {
#pragma unroll
        for (int wq = 0; wq < kWarps; ++wq) count += sm.warp_count[wq][tid];
        // the padding slots of a ragged last tile were counted in the top digit
        const uint32_t real = count - ((tid == digit_mask) ? (uint32_t)kTile - tile_n : 0u);
        st_relaxed_u64(status + (uint64_t)tile * kRadix + tid, pack_status(epoch, tile == 0 ? kFlagInclusive : kFlagAggregate, real));
        // exclusive scan of the 256 counts -> first staged slot of each digit
        uint32_t incl = count;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t up = __shfl_up_sync(kFull, incl, o);
            if ((int)lane >= o) incl += up;
        }
        if (lane == 31) sm.warp_total[warp] = incl;
        asm volatile("bar.sync 1, %0;" ::"n"(kRadix));   // only the 256 digit threads
        uint32_t carry = 0;
        for (uint32_t wq = 0; wq < warp; ++wq) carry += sm.warp_total[wq];
        excl = carry + incl - count;
        uint32_t run = excl;
#pragma unroll
        for (int wq = 0; wq < kWarps; ++wq) {
            uint32_t c = sm.warp_count[wq][tid];
            sm.warp_count[wq][tid] = run;
            run += c;
        }
        count = real;
    }
    __syncthreads();

    // rank inside the warp, row by row (keeps element order, hence stability: PAPER.md:99), and stage each pair
    // at once: the lowest lane of every group of equal digits advances the (warp, digit) slot counter
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t d = (uint32_t)(key[k] >> shift) & digit_mask;
        const uint32_t peers = digit_peers(d);
        const uint32_t below = __popc(peers & lt);
        // every lane of a digit reads the warp's slot counter of that digit; the lowest one moves it past the group
        // (plain load + predicated store: only this warp touches warp_count[warp][*] in this phase)
        uint32_t* counter = &sm.warp_count[warp][d];
        const uint32_t old = *counter;
        __syncwarp();
        if (below == 0) *counter = old + (uint32_t)__popc(peers);
        const uint32_t slot = old + below;
        sm.keys[slot] = key[k];
        if constexpr (kHasVals) sm.vals[slot] = val[k];
        __syncwarp();
    }

    // decoupled look-back, kLookWindow predecessors per round trip
    if (tid < kRadix) {
        uint32_t before = 0;   // equal-digit pairs in earlier tiles
        if (tile > 0) {
            int64_t t = (int64_t)tile - 1;
            bool done = false;
            while (!done) {
                uint64_t st[kLookWindow];
#pragma unroll
                for (int j = 0; j < kLookWindow; ++j) {
                    int64_t tj = t - j;
                    st[j] = tj >= 0 ? ld_relaxed_u64(status + (uint64_t)tj * kRadix + tid) : 0ull;
                }
#pragma unroll
                for (int j = 0; j < kLookWindow; ++j) {
                    if (done) break;
                    uint64_t v = st[j];
                    while ((uint32_t)(v >> 56) != epoch || ((uint32_t)(v >> 54) & 3u) == 0)   // not published yet
                        v = ld_relaxed_u64(status + (uint64_t)(t - j) * kRadix + tid);
                    before += (uint32_t)(v & kStatusValueMask);
                    done = ((uint32_t)(v >> 54) & 3u) == kFlagInclusive;
                }
                t -= kLookWindow;
            }
            st_relaxed_u64(status + (uint64_t)tile * kRadix + tid, pack_status(epoch, kFlagInclusive, (uint64_t)before + count));
        }
        sm.gofs[tid] = (uint32_t)bin_base[tid] + before - excl;
    }
    __syncthreads();

    // runs of equal digit leave as consecutive addresses
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t e = k * THREADS + tid;
        if (full || e < tile_n) {
            const KeyT kk = sm.keys[e];
            const uint32_t dst = sm.gofs[(uint32_t)(kk >> shift) & digit_mask] + e;
            // streaming stores: a pass's output is next read by the following launch, long after it has left L2
            __stcs(keys_out + dst, kk);
            if constexpr (kHasVals) __stcs(vals_out + dst, sm.vals[e]);
        }
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host driver
// ---------------------------------------------------------------------------------------------
size_t sort_workspace_bytes(uint64_t n) {
    uint64_t tiles = (n + kSortTileMin - 1) / kSortTileMin + 1;
    return 8 * kRadix * sizeof(uint64_t) + tiles * kRadix * sizeof(uint64_t) + 256;
}

void sort_workspace_carve(SortWorkspace& ws, void* mem, uint64_t n) {
    unsigned char* p = static_cast<unsigned char*>(mem);
    ws.hist = reinterpret_cast<uint64_t*>(p);
    p += 8 * kRadix * sizeof(uint64_t);
    ws.max_tiles = (n + kSortTileMin - 1) / kSortTileMin + 1;
    ws.status = reinterpret_cast<uint64_t*>(p);
    p += ws.max_tiles * kRadix * sizeof(uint64_t);
    ws.ticket = reinterpret_cast<uint32_t*>(p);
    ws.epoch = 0;
    ws.ticket_base = 0;
}

template <typename KeyT, typename ValT, int THREADS, int ITEMS, int kMinBlocks>
cudaError_t sort_pairs_shape(KeyT* keys, ValT* vals, KeyT* keys_alt, ValT* vals_alt, uint64_t n, uint32_t begin_bit,
                             uint32_t end_bit, SortWorkspace& ws, int* result_in_alt, Launch* prof, cudaStream_t s, bool hist_ready, int pass_class) {
    constexpr int kSortThreads = THREADS;
    constexpr int kTile = kSortThreads * ITEMS;
    static_assert(kTile >= kSortTileMin, "the tile-state array is sized for tiles of at least kSortTileMin pairs");
    using Smem = PassSmem<KeyT, ValT, kSortThreads, ITEMS>;
    auto kernel = onesweep_pass_kernel<KeyT, ValT, kSortThreads, ITEMS, kMinBlocks>;
    // per device and context, and cheap: set on every call (a cached flag would be wrong on a second GPU)
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem));
    if (e != cudaSuccess) return e;
    const uint32_t n_passes = (end_bit - begin_bit + kRadixBits - 1) / kRadixBits;
    const uint64_t n_tiles = (n + kTile - 1) / kTile;
    if (n_tiles > ws.max_tiles || n_passes > 8 || n > 0xFFFF0000ull) return cudaErrorInvalidValue;

    if (!hist_ready) {
        e = cudaMemsetAsync(ws.hist, 0, (size_t)n_passes * kRadix * sizeof(uint64_t), s);
        if (e != cudaSuccess) return e;
        uint64_t chunk = (uint64_t)kHistThreads * kHistItems;
        uint64_t blocks = (n + chunk - 1) / chunk;
        const uint64_t want = (uint64_t)sm_count() * 4;
        unsigned grid = (unsigned)(blocks < want ? blocks : want);
        ScopedLaunch sl(prof, CX_K_SORT_HIST, n * sizeof(KeyT), s);
        digit_hist_kernel<KeyT><<<grid, kHistThreads, 0, s>>>(keys, n, begin_bit, end_bit, n_passes, (unsigned long long*)ws.hist);
    }
    {
        ScopedLaunch sl(prof, CX_K_SORT_SCAN, (uint64_t)n_passes * kRadix * 16, s);
        bin_scan_kernel<<<n_passes, kRadix, 0, s>>>((unsigned long long*)ws.hist);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;

    KeyT* kin = keys;
    ValT* vin = vals;
    KeyT* kout = keys_alt;
    ValT* vout = vals_alt;
    for (uint32_t p = 0; p < n_passes; ++p) {
        uint32_t lo = begin_bit + p * kRadixBits;
        uint32_t bits = end_bit - lo < (uint32_t)kRadixBits ? end_bit - lo : (uint32_t)kRadixBits;
        if (ws.epoch == 255) {   // epoch wrap: forget every old tile state
            e = cudaMemsetAsync(ws.status, 0, ws.max_tiles * kRadix * sizeof(uint64_t), s);
            if (e != cudaSuccess) return e;
            ws.epoch = 0;
        }
        ws.epoch += 1;
        {
            ScopedLaunch sl(prof, pass_class, n * 2 * SortShape<KeyT, ValT>::pair_bytes, s);
            kernel<<<(unsigned)n_tiles, kSortThreads, sizeof(Smem), s>>>(kin, vin, kout, vout, n, lo, (1u << bits) - 1,
                                                                        ws.hist + (uint64_t)p * kRadix, ws.status, ws.ticket,
                                                                        ws.ticket_base, ws.epoch, (uint32_t)(sm_count() * kMinBlocks));
        }
        ws.ticket_base += (uint32_t)n_tiles;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        KeyT* tk = kin; kin = kout; kout = tk;
        ValT* tv = vin; vin = vout; vout = tv;
    }
    *result_in_alt = (int)(n_passes & 1);
    return cudaSuccess;
}

template <typename KeyT, typename ValT>
cudaError_t sort_pairs(KeyT* keys, ValT* vals, KeyT* keys_alt, ValT* vals_alt, uint64_t n, uint32_t begin_bit,
                       uint32_t end_bit, SortWorkspace& ws, int* result_in_alt, Launch* prof, cudaStream_t s, bool hist_ready, int pass_class) {
    *result_in_alt = 0;
    if (n <= 1 || end_bit <= begin_bit) return cudaSuccess;
    constexpr int ITEMS = SortShape<KeyT, ValT>::items;
    // keys-only (packed 32-bit key | id): 384 threads x 16 = 6144 words per tile, 3 blocks per SM, 56 registers.  Measured
    // at C2 (4 passes, ms): 384x16x3 1.91, 512x16x2 1.96, 256x24x3 2.00, 256x16x4 2.03; shapes that need register caps
    // to fit more blocks (256x16x5/6, 512x16x3) spill and lose: 2.29-2.52.
    if constexpr (sizeof(ValT) < 4)
        return sort_pairs_shape<KeyT, ValT, 384, 16, 3>(keys, vals, keys_alt, vals_alt, n, begin_bit, end_bit, ws, result_in_alt, prof, s, hist_ready, pass_class);
    return sort_pairs_shape<KeyT, ValT, kSortThreads, ITEMS, 4>(keys, vals, keys_alt, vals_alt, n, begin_bit, end_bit, ws, result_in_alt, prof, s, hist_ready, pass_class);
}

// ---------------------------------------------------------------------------------------------
// cx_sort_pairs_static: the sorter with its scratch in a file-scope device array (no allocation anywhere on the call)
// ---------------------------------------------------------------------------------------------
namespace {

constexpr uint64_t kStaticMaxPairs = CX_SORT_STATIC_MAX_PAIRS;
constexpr size_t kStaticTiles = (size_t)((kStaticMaxPairs + kSortTileMin - 1) / kSortTileMin + 1);
constexpr size_t kStaticBytes = 8 * kRadix * sizeof(uint64_t) + kStaticTiles * kRadix * sizeof(uint64_t) + 256;   // = sort_workspace_bytes(max)

// Digit histograms, tile states and the ticket of one sort of up to kStaticMaxPairs pairs.  In HOST code this name is a
// host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress (static_scratch below).
static __device__ __align__(256) unsigned char g_sort_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
void* g_scratch_of_device[kMaxDevices] = {};   // resolved once per device, with that device current
thread_local char g_static_msg[192] = "no error";

// device address of the array on the CURRENT device (nullptr + message on failure)
void* static_scratch() {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        snprintf(g_static_msg, sizeof(g_static_msg), "cx_sort_pairs_static: no current CUDA device (%s)", e != cudaSuccess ? cudaGetErrorString(e) : "index out of range");
        return nullptr;
    }
    void* p = __atomic_load_n(&g_scratch_of_device[dev], __ATOMIC_ACQUIRE);
    if (p) return p;
    e = cudaGetSymbolAddress(&p, g_sort_scratch);
    if (e != cudaSuccess || !p) {
        snprintf(g_static_msg, sizeof(g_static_msg), "cx_sort_pairs_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
        cudaGetLastError();
        return nullptr;
    }
    __atomic_store_n(&g_scratch_of_device[dev], p, __ATOMIC_RELEASE);   // (two threads may both resolve it: same value)
    return p;
}

}  // namespace
}  // namespace cx

extern "C" const char* cx_strerror_static(void) { return cx::g_static_msg; }

extern "C" int cx_sort_pairs_static(uint64_t* keys, void* vals, uint64_t* keys_alt, void* vals_alt, uint64_t n, uint32_t val_bytes,
                                    uint32_t begin_bit, uint32_t end_bit, int* result_in_alt, cx_stream_t stream) {
    using namespace cx;
    if (!result_in_alt || (val_bytes != 4 && val_bytes != 8) || begin_bit > end_bit || end_bit > 64) {
        snprintf(g_static_msg, sizeof(g_static_msg), "cx_sort_pairs_static: bad argument (result_in_alt, val_bytes 4 or 8, begin_bit <= end_bit <= 64)");
        return CX_ERR_ARG;
    }
    *result_in_alt = 0;
    if (n > kStaticMaxPairs) {
        snprintf(g_static_msg, sizeof(g_static_msg), "cx_sort_pairs_static: n = %llu exceeds CX_SORT_STATIC_MAX_PAIRS = %llu (the static scratch is sized for that; use cx_sort_pairs)",
                 (unsigned long long)n, (unsigned long long)kStaticMaxPairs);
        return CX_ERR_ARG;
    }
    if (n == 0) return CX_OK;
    if (!keys || !vals || !keys_alt || !vals_alt) {
        snprintf(g_static_msg, sizeof(g_static_msg), "cx_sort_pairs_static: null buffer");
        return CX_ERR_ARG;
    }
    void* scratch = static_scratch();
    if (!scratch) return CX_ERR_CUDA;
    // the array keeps the last call's contents: tile states and the ticket must start from zero
    const size_t bytes = sort_workspace_bytes(n);   // <= kStaticBytes
    cudaError_t e = cudaMemsetAsync(scratch, 0, bytes, stream);
    SortWorkspace ws;
    sort_workspace_carve(ws, scratch, n);
    if (e == cudaSuccess) {
        if (val_bytes == 4)
            e = sort_pairs<uint64_t, uint32_t>(keys, (uint32_t*)vals, keys_alt, (uint32_t*)vals_alt, n, begin_bit, end_bit, ws, result_in_alt, nullptr, stream);
        else
            e = sort_pairs<uint64_t, uint64_t>(keys, (uint64_t*)vals, keys_alt, (uint64_t*)vals_alt, n, begin_bit, end_bit, ws, result_in_alt, nullptr, stream);
    }
    if (e != cudaSuccess) {
        snprintf(g_static_msg, sizeof(g_static_msg), "cx_sort_pairs_static: CUDA error %d: %s", (int)e, cudaGetErrorString(e));
        cudaGetLastError();
        return CX_ERR_CUDA;
    }
    return CX_OK;
}

namespace cx {

#define CX_SORT_INST(K, V)                                                                                               \
    template cudaError_t sort_pairs<K, V>(K*, V*, K*, V*, uint64_t, uint32_t, uint32_t, SortWorkspace&, int*, Launch*, cudaStream_t, bool, int);
CX_SORT_INST(uint32_t, uint32_t)
CX_SORT_INST(uint32_t, uint64_t)
CX_SORT_INST(uint64_t, uint32_t)
CX_SORT_INST(uint64_t, uint64_t)
CX_SORT_INST(uint64_t, NoVal)

}  // namespace cx
