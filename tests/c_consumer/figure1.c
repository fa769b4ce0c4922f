/* A C-language consumer of include/cx_bwt.h: builds the BWT of the paper's worked example
 * (Figure 1: {ACGT, TAGT, GGAA} -> TTAAG$TAG$CAGG$) through the C ABI only.
 * Compiled as C99 and linked against libcxbwt.so by tests/test_abi.py; device memory comes from the
 * CUDA runtime's C API (in the product it comes from PyTorch). */
#include <stdio.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "cx_bwt.h"

#define CHECK_CX(call)                                                        \
    do {                                                                      \
        int rc_ = (call);                                                     \
        if (rc_ != CX_OK) {                                                   \
            fprintf(stderr, "%s -> %d (%s)\n", #call, rc_, cx_strerror(rc_)); \
            return 2;                                                         \
        }                                                                     \
    } while (0)
#define CHECK_CUDA(call)                                                              \
    do {                                                                              \
        cudaError_t e_ = (call);                                                      \
        if (e_ != cudaSuccess) {                                                      \
            fprintf(stderr, "%s -> %s\n", #call, cudaGetErrorString(e_));             \
            return 3;                                                                 \
        }                                                                             \
    } while (0)

int main(void) {
    const char *bases = "ACGTTAGTGGAA";
    const uint64_t offsets[4] = {0, 4, 8, 12};
    const uint64_t n_reads = 3, total = 12, n_suffixes = 15;
    cx_bwt_opts_t opts;
    cx_bwt_plan_t *plan = NULL;
    cx_bwt_stats_t stats;
    uint64_t ws_bytes = 0;
    void *d_ws = NULL;
    uint8_t *d_ascii = NULL, *d_out = NULL;
    uint64_t *d_packed = NULL, *d_off = NULL;
    char out[16];

    memset(&opts, 0, sizeof(opts));
    opts.max_read_len = 4;
    CHECK_CX(cx_bwt_workspace_bytes(n_reads, total, &opts, &ws_bytes));
    CHECK_CUDA(cudaMalloc(&d_ws, ws_bytes));
    CHECK_CUDA(cudaMalloc((void **)&d_ascii, total));
    CHECK_CUDA(cudaMalloc((void **)&d_packed, 8));
    CHECK_CUDA(cudaMalloc((void **)&d_off, sizeof(offsets)));
    CHECK_CUDA(cudaMalloc((void **)&d_out, n_suffixes));
    CHECK_CUDA(cudaMemcpy(d_ascii, bases, total, cudaMemcpyHostToDevice));
    CHECK_CUDA(cudaMemcpy(d_off, offsets, sizeof(offsets), cudaMemcpyHostToDevice));
    CHECK_CX(cx_bwt_plan(&plan, n_reads, total, &opts, d_ws, ws_bytes));
    CHECK_CX(cx_pack_reads(d_ascii, total, d_packed, NULL, NULL));
    CHECK_CX(cx_bwt_build(plan, d_packed, d_off, n_reads, d_out, NULL));
    CHECK_CUDA(cudaDeviceSynchronize());
    CHECK_CUDA(cudaMemcpy(out, d_out, n_suffixes, cudaMemcpyDeviceToHost));
    out[n_suffixes] = 0;
    CHECK_CX(cx_bwt_get_stats(plan, &stats));
    CHECK_CX(cx_bwt_free(plan));
    printf("%s %llu\n", out, (unsigned long long)stats.n_suffixes);
    return strcmp(out, "TTAAG$TAG$CAGG$") == 0 && stats.n_suffixes == n_suffixes ? 0 : 1;
}
