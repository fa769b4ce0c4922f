// cx_fasta.cu -- NEXT-4: FASTA text on the device -> concatenated bases + read offsets,
// the inputs of cx_pack_reads / cx_bwt_build.  "The input was in FASTA format"; reading it takes
// "more than 16 minutes" of the 6,886 s run and Section 5 names I/O as the next bottleneck.
//
// Grammar taken (the paper gives none): the text is a sequence of lines ended by '\n' (the last
// one may lack it).  A line whose first byte is '>' is a header: it starts a new read and contributes nothing else.
// Every other line is a sequence line: its bytes, except '\r', are appended to the current read.  Sequence bytes
// before the first header belong to no read ("orphans"): they are counted and the caller treats that as an error.
//
// Three steps, each a streaming pass over tiles of 16 KB (thread t owns 64 consecutive bytes):
//   summarise : per tile, the kind of its last line start, its header count, and its base count split into the part
//               whose kind is known inside the tile and the part that continues a line begun in an earlier tile;
//   resolve   : per tile, the kind of the line it starts in (walk back over the tile kinds: one step unless a line
//               spans many tiles), hence its base count; exclusive scans of bases and headers over the tiles;
//   write     : per tile, the same decode again; every base goes to its final index, every header writes the
//               base index at which its read starts.
// Algorithmic traffic: 2 reads of the text + 1 write of the bases (+ 8 B per read).
#include "cx_internal.cuh"

namespace cx {
namespace {

__host__ __device__ constexpr uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

constexpr int kFaThreads = 256;
constexpr int kFaVec = 4;                          // 16-byte loads per thread
constexpr int kFaBytes = 16 * kFaVec;              // consecutive bytes owned by a thread
constexpr int kFaTile = kFaThreads * kFaBytes;     // 16384
constexpr uint32_t kNone = 0, kHeader = 1, kSeq = 2;

struct ThreadDecode {
    uint32_t last_kind;   // kind of the last line start among my bytes (kNone if I hold none)
    uint32_t pre_cnt;     // bytes other than \n, \r before my first line start (all of mine if I hold none)
    uint32_t post_bases;  // bases of sequence lines that start among my bytes
    uint32_t n_headers;   // header lines that start among my bytes
};

struct Chunk {
    uint4 v[kFaVec];
};
__device__ __forceinline__ uint8_t byte_of(const Chunk& c, int i) {
    const uint4& v = c.v[i >> 4];
    const int j = i & 15;
    const uint32_t w = j < 4 ? v.x : j < 8 ? v.y : j < 12 ? v.z : v.w;
    return (uint8_t)(w >> (8 * (j & 3)));
}

// my bytes (zero-filled past the end) and the byte before them ('\n' before the text: byte 0 starts a line)
__device__ __forceinline__ void load_chunk(const uint8_t* __restrict__ text, uint64_t n, uint64_t at, Chunk& c, uint8_t& prev, uint32_t& cnt) {
#pragma unroll
    for (int q = 0; q < kFaVec; ++q) c.v[q] = make_uint4(0, 0, 0, 0);
    cnt = 0;
    prev = '\n';
    if (at >= n) return;
    cnt = (uint32_t)min((uint64_t)kFaBytes, n - at);
    if (at) prev = text[at - 1];
    if (cnt == kFaBytes && ((reinterpret_cast<uintptr_t>(text) + at) & 15) == 0) {
#pragma unroll
        for (int q = 0; q < kFaVec; ++q) c.v[q] = __ldg(reinterpret_cast<const uint4*>(text + at) + q);
    } else {
        uint32_t w[4 * kFaVec];
#pragma unroll
        for (int q = 0; q < 4 * kFaVec; ++q) w[q] = 0;
#pragma unroll
        for (int i = 0; i < kFaBytes; ++i)
            if ((uint32_t)i < cnt) w[i >> 2] |= (uint32_t)text[at + i] << (8 * (i & 3));
#pragma unroll
        for (int q = 0; q < kFaVec; ++q) c.v[q] = make_uint4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
    }
}

__device__ __forceinline__ ThreadDecode decode(const Chunk& v, uint8_t prev, uint32_t cnt) {
    ThreadDecode d{kNone, 0, 0, 0};
    uint32_t kind = kNone;
#pragma unroll
    for (int i = 0; i < kFaBytes; ++i) {
        if ((uint32_t)i < cnt) {
            const uint8_t c = byte_of(v, i);
            if (prev == '\n') {
                kind = c == '>' ? kHeader : kSeq;
                d.n_headers += kind == kHeader;
            }
            const bool payload = c != '\n' && c != '\r';
            if (kind == kNone) d.pre_cnt += payload;
            else if (kind == kSeq) d.post_bases += payload;
            prev = c;
        }
    }
    d.last_kind = kind;
    return d;
}

// kind of the line my first byte lies in, as far as the tile knows: the last line start held by an earlier thread of
// the block (kNone: the line began before the tile)
__device__ __forceinline__ uint32_t incoming_kind(uint32_t my_last, uint32_t* s_warp_last) {
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    const uint32_t have = __ballot_sync(0xffffffffu, my_last != kNone);
    const uint32_t below = have & ((1u << lane) - 1);
    const int src = below ? 31 - __clz(below) : 0;
    const uint32_t from_lane = __shfl_sync(0xffffffffu, my_last, src);
    const uint32_t warp_last = __shfl_sync(0xffffffffu, my_last, have ? 31 - __clz(have) : 0);
    if (lane == 0) s_warp_last[warp] = have ? warp_last : kNone;
    __syncthreads();
    if (below) return from_lane;
    uint32_t k = kNone;
    for (uint32_t q = 0; q < warp; ++q)
        if (s_warp_last[q] != kNone) k = s_warp_last[q];
    return k;
}

__device__ __forceinline__ uint64_t block_sum(uint64_t v, uint64_t* s_part) {
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane_id() == 0) s_part[threadIdx.x >> 5] = v;
    __syncthreads();
    uint64_t t = 0;
    for (int q = 0; q < kFaThreads / 32; ++q) t += s_part[q];
    return t;
}

// exclusive prefix of v over the block's threads
__device__ __forceinline__ uint64_t block_excl(uint64_t v, uint64_t* s_part) {
    uint64_t incl = v;
    for (int o = 1; o < 32; o <<= 1) {
        const uint64_t up = __shfl_up_sync(0xffffffffu, incl, o);
        if ((int)lane_id() >= o) incl += up;
    }
    __syncthreads();
    if (lane_id() == 31) s_part[threadIdx.x >> 5] = incl;
    __syncthreads();
    uint64_t carry = 0;
    for (uint32_t q = 0; q < (threadIdx.x >> 5); ++q) carry += s_part[q];
    return carry + incl - v;
}

struct TileSummary {
    uint32_t pre_cnt;     // payload bytes that continue a line begun before the tile
    uint32_t post_bases;  // bases whose line kind the tile knows
    uint32_t n_headers;
    uint32_t last_kind;   // kind of the tile's last line start, kNone if it holds none
};

__global__ void __launch_bounds__(kFaThreads) fasta_summarise_kernel(const uint8_t* __restrict__ text, uint64_t n, TileSummary* __restrict__ sums,
                                                                     uint8_t* __restrict__ tile_kind) {
    __shared__ uint32_t s_last[kFaThreads / 32];
    __shared__ uint64_t s_part[kFaThreads / 32];
    const uint64_t at = (uint64_t)blockIdx.x * kFaTile + (uint64_t)threadIdx.x * kFaBytes;
    Chunk v;
    uint8_t prev;
    uint32_t cnt;
    load_chunk(text, n, at, v, prev, cnt);
    const ThreadDecode d = decode(v, prev, cnt);
    const uint32_t inc = incoming_kind(d.last_kind, s_last);
    // three sums in one: each is at most kFaTile < 2^20
    const uint64_t all = block_sum((uint64_t)(inc == kNone ? d.pre_cnt : 0u) | ((uint64_t)(d.post_bases + (inc == kSeq ? d.pre_cnt : 0u)) << 20) |
                                   ((uint64_t)d.n_headers << 40), s_part);
    const uint32_t pre = (uint32_t)all & 0xfffffu, post = (uint32_t)(all >> 20) & 0xfffffu, heads = (uint32_t)(all >> 40);
    if (threadIdx.x == kFaThreads - 1) {
        const uint32_t last = d.last_kind != kNone ? d.last_kind : inc;
        sums[blockIdx.x] = TileSummary{pre, post, heads, last};
        tile_kind[blockIdx.x] = (uint8_t)last;
    }
}

// one thread per tile: the kind of the line the tile starts in, then its base and header counts
__global__ void __launch_bounds__(256) fasta_resolve_kernel(const TileSummary* __restrict__ sums, const uint8_t* __restrict__ tile_kind, uint64_t n_tiles,
                                                            uint8_t* __restrict__ tile_in, uint64_t* __restrict__ bases, uint64_t* __restrict__ heads) {
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_tiles) return;
    uint32_t in = kNone;
    for (uint64_t q = t; q-- > 0;) {   // one step unless a single line covers whole tiles
        const uint32_t k = tile_kind[q];
        if (k != kNone) {
            in = k;
            break;
        }
    }
    const TileSummary s = sums[t];
    tile_in[t] = (uint8_t)in;
    bases[t] = (uint64_t)s.post_bases + (in == kSeq ? s.pre_cnt : 0u);
    heads[t] = s.n_headers;
}

__global__ void __launch_bounds__(kFaThreads) fasta_write_kernel(const uint8_t* __restrict__ text, uint64_t n, const uint8_t* __restrict__ tile_in,
                                                                 const uint64_t* __restrict__ base_at, const uint64_t* __restrict__ head_at,
                                                                 uint8_t* __restrict__ bases_out, uint64_t* __restrict__ offsets_out, uint64_t max_reads,
                                                                 unsigned long long* __restrict__ orphans) {
    __shared__ uint32_t s_last[kFaThreads / 32];
    __shared__ uint64_t s_part[kFaThreads / 32];
    const uint64_t at = (uint64_t)blockIdx.x * kFaTile + (uint64_t)threadIdx.x * kFaBytes;
    Chunk v;
    uint8_t prev;
    uint32_t cnt;
    load_chunk(text, n, at, v, prev, cnt);
    const ThreadDecode d = decode(v, prev, cnt);
    uint32_t kind = incoming_kind(d.last_kind, s_last);
    if (kind == kNone) kind = tile_in[blockIdx.x];
    const uint32_t my_bases = d.post_bases + (kind == kSeq ? d.pre_cnt : 0u);
    // the tile's bases in order, staged so that they leave as aligned 16-byte stores: staged index i + skew holds the base
    // that goes to bases_out[tile_b + i], skew = the low four address bits of that destination
    __shared__ __align__(16) uint8_t s_bases[kFaTile + 16];
    __shared__ uint32_t s_total;
    const uint64_t both = block_excl((uint64_t)my_bases | ((uint64_t)d.n_headers << 32), s_part);   // two prefix sums in one
    uint32_t lb = (uint32_t)both;                                         // index of my first base among the tile's
    if (threadIdx.x == kFaThreads - 1) s_total = lb + my_bases;
    const uint64_t tile_b = base_at[blockIdx.x];                          // index of the tile's first base in the output
    uint64_t r = head_at[blockIdx.x] + (both >> 32);                      // reads started before my bytes
    const uint32_t skew = (uint32_t)(reinterpret_cast<uintptr_t>(bases_out + tile_b) & 15);
    uint32_t lost = 0;
#pragma unroll
    for (int i = 0; i < kFaBytes; ++i) {
        if ((uint32_t)i < cnt) {
            const uint8_t c = byte_of(v, i);
            if (prev == '\n') {
                kind = c == '>' ? kHeader : kSeq;
                if (kind == kHeader) {
                    if (r < max_reads) offsets_out[r] = tile_b + lb;
                    ++r;
                }
            }
            if (kind == kSeq && c != '\n' && c != '\r') {
                if (r == 0) ++lost;   // no header yet: the byte belongs to no read
                s_bases[skew + lb++] = c;
            }
            prev = c;
        }
    }
    __syncthreads();
    {
        const uint32_t end = skew + s_total;                 // staged bytes are [skew, end)
        uint8_t* dst = bases_out + tile_b - skew;            // 16-byte aligned; dst[j] <- s_bases[j]
        const uint32_t body_lo = skew ? 16u : 0u, body_hi = end & ~15u;
        for (uint32_t j = skew + threadIdx.x; j < min(end, body_lo); j += kFaThreads) dst[j] = s_bases[j];
        for (uint32_t j = body_lo + 16 * threadIdx.x; j + 16 <= body_hi; j += 16 * kFaThreads)
            *reinterpret_cast<uint4*>(dst + j) = *reinterpret_cast<const uint4*>(s_bases + j);
        for (uint32_t j = max(body_hi, body_lo) + threadIdx.x; j < end; j += kFaThreads) dst[j] = s_bases[j];
    }
    if (lost) atomicAdd(orphans, (unsigned long long)lost);
}

// counts[0] = reads, counts[1] = bases, counts[2] = orphan bytes (added by the write kernel); closes the offsets array
__global__ void fasta_finish_kernel(const uint64_t* __restrict__ totals, uint64_t* __restrict__ counts, uint64_t* __restrict__ offsets_out, uint64_t max_reads) {
    counts[0] = totals[1];
    counts[1] = totals[0];
    if (totals[1] <= max_reads) offsets_out[totals[1]] = totals[0];
}

}  // namespace

// workspace: per tile a summary (16 B), two kinds (2 B), two u64 scan arrays, their block sums, totals
uint64_t fasta_workspace_bytes(uint64_t n_bytes) {
    const uint64_t tiles = (n_bytes + kFaTile - 1) / kFaTile + 1;
    return align_up(tiles * sizeof(TileSummary), 256) + 2 * align_up(tiles, 256) + 2 * align_up(tiles * 8, 256) +
           2 * align_up((scan_block_count(tiles) + 1) * 8, 256) + 256;
}

cudaError_t launch_fasta_parse(const uint8_t* text, uint64_t n, uint8_t* bases_out, uint64_t* offsets_out, uint64_t max_reads, uint64_t* counts,
                               unsigned char* ws, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(counts, 0, 3 * sizeof(uint64_t), s);
    if (e != cudaSuccess) return e;
    if (n == 0) return cudaMemsetAsync(offsets_out, 0, sizeof(uint64_t), s);
    const uint64_t tiles = (n + kFaTile - 1) / kFaTile;
    unsigned char* p = ws;
    TileSummary* sums = reinterpret_cast<TileSummary*>(p);
    p += align_up((tiles + 1) * sizeof(TileSummary), 256);
    uint8_t* tile_kind = p;
    p += align_up(tiles + 1, 256);
    uint8_t* tile_in = p;
    p += align_up(tiles + 1, 256);
    uint64_t* bases = reinterpret_cast<uint64_t*>(p);
    p += align_up((tiles + 1) * 8, 256);
    uint64_t* heads = reinterpret_cast<uint64_t*>(p);
    p += align_up((tiles + 1) * 8, 256);
    uint64_t* sums_b = reinterpret_cast<uint64_t*>(p);
    p += align_up((scan_block_count(tiles + 1) + 1) * 8, 256);
    uint64_t* sums_h = reinterpret_cast<uint64_t*>(p);
    p += align_up((scan_block_count(tiles + 1) + 1) * 8, 256);
    uint64_t* totals = reinterpret_cast<uint64_t*>(p);   // [0] bases, [1] reads
    fasta_summarise_kernel<<<(unsigned)tiles, kFaThreads, 0, s>>>(text, n, sums, tile_kind);
    fasta_resolve_kernel<<<(unsigned)((tiles + 255) / 256), 256, 0, s>>>(sums, tile_kind, tiles, tile_in, bases, heads);
    e = launch_scan_u64(bases, tiles, sums_b, totals, s);
    if (e != cudaSuccess) return e;
    e = launch_scan_u64(heads, tiles, sums_h, totals + 1, s);
    if (e != cudaSuccess) return e;
    fasta_write_kernel<<<(unsigned)tiles, kFaThreads, 0, s>>>(text, n, tile_in, bases, heads, bases_out, offsets_out, max_reads,
                                                              reinterpret_cast<unsigned long long*>(counts + 2));
    fasta_finish_kernel<<<1, 1, 0, s>>>(totals, counts, offsets_out, max_reads);
    return cudaGetLastError();
}

}  // namespace cx
