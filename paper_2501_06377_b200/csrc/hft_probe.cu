// hft_probe.cu -- register-only FMA issue-rate probe behind the "alu" roofline of bench.py.
// Not part of the time-stepping path: it measures, on the device it runs on, how many FMA lane-operations per second the
// SMs sustain for three operand patterns, so that the denominators bench.py divides by can be re-measured by anyone:
//   pattern 0: x = fma(x, a, b)   two operands shared by every FMA of the thread        (the textbook peak loop)
//   pattern 1: x = fma(y, z, x)   three distinct register operands per FMA               (k_sts_pipe: coefficient in a register)
//   pattern 2: x = fma(y, c, x)   one operand from the constant bank / a uniform register (k_sts_upipe)
// 16 independent chains per thread, 128 threads per CTA, 4 CTAs per SM, no memory traffic inside the timed loop.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hft.h"

namespace {

constexpr int NCH = 16;        // independent accumulator chains per thread
constexpr int PROBE_TX = 128;
constexpr int PROBE_CTAS_PER_SM = 4;

__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }

template <typename real, int PATTERN>
__global__ void __launch_bounds__(PROBE_TX) k_probe_fma(real* out, const real* in, int iters, real ck) {
    real x[NCH], y[NCH], z[NCH];
#pragma unroll
    for (int i = 0; i < NCH; i++) {
        x[i] = in[threadIdx.x + i * PROBE_TX];
        y[i] = in[threadIdx.x + (NCH + i) * PROBE_TX];
        z[i] = in[threadIdx.x + (2 * NCH + i) * PROBE_TX];
    }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NCH; i++) {
            if (PATTERN == 0) x[i] = fma_t(x[i], y[0], z[0]);
            if (PATTERN == 1) x[i] = fma_t(y[i], z[i], x[i]);
            if (PATTERN == 2) x[i] = fma_t(y[i], ck, x[i]);
        }
    }
    real s = (real)0;
#pragma unroll
    for (int i = 0; i < NCH; i++) s += x[i] + y[i] + z[i];
    out[(size_t)blockIdx.x * PROBE_TX + threadIdx.x] = s;
}

template <typename real, int PATTERN>
int probe(double* h_rate) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HFT_ERR_DEVICE;
    const int ctas = sms * PROBE_CTAS_PER_SM, iters = 20000;
    real *in = nullptr, *out = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    int rc = HFT_ERR_CUDA;
    float ms = 0.f;
    if (cudaMalloc((void**)&in, 3 * NCH * PROBE_TX * sizeof(real)) != cudaSuccess) return HFT_ERR_NOMEM;
    if (cudaMalloc((void**)&out, (size_t)ctas * PROBE_TX * sizeof(real)) != cudaSuccess) { cudaFree(in); return HFT_ERR_NOMEM; }
    if (cudaMemset(in, 0, 3 * NCH * PROBE_TX * sizeof(real)) != cudaSuccess) goto done;   // zeros: every chain stays finite
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) goto done;
    k_probe_fma<real, PATTERN><<<ctas, PROBE_TX>>>(out, in, 200, (real)0.5);              // warm-up
    if (cudaEventRecord(a) != cudaSuccess) goto done;
    k_probe_fma<real, PATTERN><<<ctas, PROBE_TX>>>(out, in, iters, (real)0.5);
    if (cudaEventRecord(b) != cudaSuccess || cudaEventSynchronize(b) != cudaSuccess) goto done;
    if (cudaGetLastError() != cudaSuccess || cudaEventElapsedTime(&ms, a, b) != cudaSuccess || !(ms > 0.f)) goto done;
    *h_rate = (double)ctas * PROBE_TX * (double)iters * NCH / (ms * 1e-3);
    rc = HFT_OK;
done:
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(in); cudaFree(out);
    return rc;
}

}  // namespace

extern "C" int hft_probe_fma_rate(int32_t dtype, int32_t pattern, double* h_lane_fma_per_s) {
    if (!h_lane_fma_per_s || (dtype != 0 && dtype != 1) || pattern < 0 || pattern > 2) return HFT_ERR_ARG;
    if (dtype == 1) {
        if (pattern == 0) return probe<double, 0>(h_lane_fma_per_s);
        if (pattern == 1) return probe<double, 1>(h_lane_fma_per_s);
        return probe<double, 2>(h_lane_fma_per_s);
    }
    if (pattern == 0) return probe<float, 0>(h_lane_fma_per_s);
    if (pattern == 1) return probe<float, 1>(h_lane_fma_per_s);
    return probe<float, 2>(h_lane_fma_per_s);
}
