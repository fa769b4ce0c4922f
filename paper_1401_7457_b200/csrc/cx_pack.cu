// cx_pack.cu -- step a1: ASCII bases -> 2 bit/base ("standard 2-bit-per-character representation",
// PAPER.md:71, 91).  Streaming kernel: 1 byte read + 0.25 byte written per base, HBM-bound.
#include "cx_internal.cuh"

namespace cx {
namespace {

// Four ASCII bytes (first base in the low byte) -> 8 bits, first base in the two MSBs.
// code(c) = ((c >> 1) ^ (c >> 2)) & 3 maps A,C,G,T -> 0,1,2,3.  *bad accumulates a non-zero value
// if any byte is not one of "ACGT" (checked by re-spelling the codes with a byte permute).
__device__ __forceinline__ uint32_t pack4(uint32_t x, uint32_t& bad) {
    uint32_t codes = ((x >> 1) ^ (x >> 2)) & 0x03030303u;
    uint32_t sel = (codes & 0xFu) | ((codes >> 4) & 0xF0u) | ((codes >> 8) & 0xF00u) | ((codes >> 12) & 0xF000u);
    bad |= __byte_perm(0x54474341u /* "ACGT" */, 0u, sel) ^ x;
    return (codes * 0x40100401u) >> 24;
}

__device__ __forceinline__ uint64_t pack32(const uint4& a, const uint4& b, uint32_t& bad) {
    uint32_t hi = (pack4(a.x, bad) << 24) | (pack4(a.y, bad) << 16) | (pack4(a.z, bad) << 8) | pack4(a.w, bad);
    uint32_t lo = (pack4(b.x, bad) << 24) | (pack4(b.y, bad) << 16) | (pack4(b.z, bad) << 8) | pack4(b.w, bad);
    return ((uint64_t)hi << 32) | lo;
}

__device__ __forceinline__ uint32_t code_or_bad(uint8_t c, uint32_t& bad) {
    uint32_t code = ((c >> 1) ^ (c >> 2)) & 3u;
    bad |= (uint32_t)((0x54474341u >> (8 * code)) & 0xFFu) ^ (uint32_t)c;
    return code;
}

// One thread per output word.  ALIGNED: ascii is 16-byte aligned, so full words use two 128-bit loads.
template <bool ALIGNED>
__global__ void __launch_bounds__(256) pack_kernel(const uint8_t* __restrict__ ascii, uint64_t total_bases,
                                                   uint64_t* __restrict__ packed, uint32_t* __restrict__ status) {
    uint64_t n_words = (total_bases + 31) >> 5;
    uint32_t bad = 0;
    for (uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += (uint64_t)gridDim.x * blockDim.x) {
        uint64_t b0 = w << 5;
        uint64_t word = 0;
        if (ALIGNED && b0 + 32 <= total_bases) {
            const uint4* p = reinterpret_cast<const uint4*>(ascii + b0);
            uint4 a = __ldcs(p), b = __ldcs(p + 1);
            word = pack32(a, b, bad);
        } else {
            uint32_t cnt = (uint32_t)min((uint64_t)32, total_bases - b0);
            for (uint32_t k = 0; k < cnt; ++k) word |= (uint64_t)code_or_bad(ascii[b0 + k], bad) << (62 - 2 * k);
        }
        packed[w] = word;
    }
    // one counter update per warp that saw a bad byte
    uint32_t any = __ballot_sync(0xffffffffu, bad != 0);
    if (any && lane_id() == 0) atomicAdd(status, __popc(any));
}

__device__ uint32_t g_pack_status;   // used when the caller passes no status word

// NEXT-4, packed output: n ASCII symbols over "$ACGT" that belong at positions [off, off + n) of the BWT -> 4-bit codes
// ($ A C G T = 0 1 2 3 4), two per byte, first symbol of a byte in its high nibble.  packed[0] is the byte that holds
// position off (byte off / 2 of the whole output).  If off is odd that byte's high nibble is the symbol before this
// piece: *carry (its code, written by the previous call on this stream).  Four output bytes per thread.
__device__ __forceinline__ uint32_t nibble_of(uint8_t c) { return (c & 0x40u) ? 1u + (((c >> 1) ^ (c >> 2)) & 3u) : 0u; }
__global__ void __launch_bounds__(256) pack_symbols_kernel(const uint8_t* __restrict__ sym, uint64_t n, uint32_t odd, uint8_t* __restrict__ packed,
                                                           uint32_t* __restrict__ carry) {
    const uint64_t n_bytes = (n + odd + 1) >> 1;
    const uint64_t b0 = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint64_t b = b0 + k;
        if (b >= n_bytes) break;
        const int64_t i = (int64_t)(2 * b) - (int64_t)odd;        // local index of the byte's first symbol
        const uint32_t hi = i >= 0 ? nibble_of(__ldg(sym + i)) : *carry;
        const uint32_t lo = (uint64_t)(i + 1) < n ? nibble_of(__ldg(sym + i + 1)) : 0u;
        packed[b] = (uint8_t)((hi << 4) | lo);
    }
}
__global__ void last_symbol_kernel(const uint8_t* __restrict__ sym, uint64_t n, uint32_t* __restrict__ carry) {
    if (n) *carry = nibble_of(sym[n - 1]);
}

}  // namespace

cudaError_t launch_pack(const uint8_t* ascii, uint64_t total_bases, uint64_t* packed, uint32_t* status, cudaStream_t s) {
    uint64_t n_words = (total_bases + 31) >> 5;
    if (n_words == 0) return cudaSuccess;
    uint64_t blocks = (n_words + 255) / 256;
    const uint64_t want = (uint64_t)sm_count() * 32;
    unsigned grid = (unsigned)(blocks < want ? blocks : want);
    if ((reinterpret_cast<uintptr_t>(ascii) & 15) == 0)
        pack_kernel<true><<<grid, 256, 0, s>>>(ascii, total_bases, packed, status);
    else
        pack_kernel<false><<<grid, 256, 0, s>>>(ascii, total_bases, packed, status);
    return cudaGetLastError();
}

cudaError_t launch_pack_symbols(const uint8_t* sym, uint64_t n, uint64_t out_offset, uint8_t* packed, uint32_t* carry, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    const uint32_t odd = (uint32_t)(out_offset & 1);
    const uint64_t n_bytes = (n + odd + 1) >> 1;
    pack_symbols_kernel<<<(unsigned)((n_bytes + 1023) / 1024), 256, 0, s>>>(sym, n, odd, packed, carry);
    last_symbol_kernel<<<1, 1, 0, s>>>(sym, n, carry);   // after the pack: it read the previous piece's last symbol
    return cudaGetLastError();
}

uint32_t* pack_fallback_status() {
    uint32_t* p = nullptr;
    cudaGetSymbolAddress((void**)&p, g_pack_status);
    return p;
}

}  // namespace cx
