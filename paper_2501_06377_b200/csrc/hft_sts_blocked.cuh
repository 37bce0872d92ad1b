// hft_sts_blocked.cuh -- temporally blocked STS stages (k stages per launch).  STUB: filled in next.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "hft_kernels.cuh"

namespace hft {

constexpr int STS_KMAX = 8;

template <typename real>
struct StsBlockedPlan {
    real* Y0;
    real* buf[5];
    const double *mu, *nu, *a, *g;
    int s, kb;
    cudaStream_t stream;
    double** part;
    double* zmean;
    double* capseq;
    void (*prof_begin)(void*, bool*);
    void (*prof_end)(void*, bool);
    void* user;
};

inline int sts_default_block(const Geom&, size_t) { return 1; }
inline bool sts_blocked_supported(const Geom&, size_t) { return false; }
inline size_t sts_zmean_bytes(const Geom&) { return 256; }
inline size_t sts_capseq_bytes(const Geom&) { return 256; }
inline int sts_blocked_init(const Geom&, bool) { return 0; }
template <typename real>
int sts_blocked_step(StsBlockedPlan<real>&, Tables<real>&, const Geom&, int64_t*) { return -1; }

}  // namespace hft
