// cx_launch.h -- launch accounting: counts kernels per class and, when profiling is on, brackets
// each launch with a pair of CUDA events on the launching stream (resolved after the build).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "cx_bwt.h"

namespace cx {

struct Launch {
    struct Rec {
        int cls;
        cudaEvent_t start, stop;
    };
    bool timing = false;
    uint64_t launches[CX_K_COUNT] = {};
    uint64_t bytes[CX_K_COUNT] = {};
    double ms[CX_K_COUNT] = {};
    std::vector<Rec> pending;
    std::vector<cudaEvent_t> pool;   // recycled events

    cudaEvent_t get_event() {
        if (!pool.empty()) {
            cudaEvent_t e = pool.back();
            pool.pop_back();
            return e;
        }
        cudaEvent_t e = nullptr;
        cudaEventCreate(&e);
        return e;
    }
    void reset() {
        for (int i = 0; i < CX_K_COUNT; ++i) launches[i] = 0, bytes[i] = 0, ms[i] = 0.0;
        for (auto& r : pending) pool.push_back(r.start), pool.push_back(r.stop);
        pending.clear();
    }
    // call after the stream has been synchronised
    void resolve() {
        for (auto& r : pending) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, r.start, r.stop) == cudaSuccess) ms[r.cls] += t;
            pool.push_back(r.start);
            pool.push_back(r.stop);
        }
        pending.clear();
    }
    void destroy() {
        reset();
        for (auto e : pool) cudaEventDestroy(e);
        pool.clear();
    }
    uint64_t total_launches() const {
        uint64_t t = 0;
        for (int i = 0; i < CX_K_COUNT; ++i) t += launches[i];
        return t;
    }
};

struct ScopedLaunch {
    Launch* p;
    cudaStream_t s;
    cudaEvent_t stop = nullptr;
    ScopedLaunch(Launch* prof, int cls, uint64_t algorithmic_bytes, cudaStream_t stream) : p(prof), s(stream) {
        if (!p) return;
        p->launches[cls] += 1;
        p->bytes[cls] += algorithmic_bytes;
        if (p->timing) {
            Launch::Rec r{cls, p->get_event(), p->get_event()};
            cudaEventRecord(r.start, s);
            stop = r.stop;
            p->pending.push_back(r);
        }
    }
    ~ScopedLaunch() {
        if (stop) cudaEventRecord(stop, s);
    }
};

}  // namespace cx
