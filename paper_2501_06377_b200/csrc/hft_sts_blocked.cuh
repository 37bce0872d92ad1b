// hft_sts_blocked.cuh -- temporally blocked super-time-stepping: K STS stages per kernel launch.
//
// Why: one launch per stage moves 4 field passes per stage through HBM (read delta_{j-1}, delta_{j-2},
// L(Y0); write delta_j).  Blocking K stages on chip moves 3 reads + 2 writes per K stages instead.
//
// How: every WARP owns a strip of 32*C consecutive phi-columns (C columns
// per lane, one 16-byte vector) and streams down the theta-rows.  The K stage levels form a software
// pipeline skewed by one row per level: at row-step t the warp loads row t of the three inputs and
// computes row t-l of level l for l = 1..K.  Each level keeps a 3-row window in REGISTERS (theta
// neighbours), the phi neighbours come from the adjacent lanes by warp shuffle, so the stencil never
// touches shared memory and warps never synchronise with each other.  The price is a halo: the first and
// last K columns of a warp's strip become invalid (one column per level and side), so strips overlap by
// 2K columns and only 32*C - 2K columns are written.  Periodic phi is an index wrap of the strip origin.
//
// Polar caps: the cap update of level l needs the phi-sum of row 1 at level l-1 over ALL columns, a global
// dependency per stage.  Because every coefficient of L is phi-independent and phi is periodic, the
// phi-mean commutes with L: the zonal means m_j = mean_k u_jk obey the same recurrence with the phi-term
// dropped.  So the K cap values of a block follow from the zonal means of rows 1..K of the three input
// fields alone (a cone of K rows); k_sts_capseq computes them before the main kernel, which then treats
// rows 0 and nt+1 of every level as known boundary values.  (Exact in exact arithmetic; in floating
// point it differs from summing the actual stage rows by round-off only.  Valid because nu is constant in
// space -- SURVEY section 8 scope; a spatially varying nu would need the per-stage reduction instead.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <map>
#include <mutex>
#include <utility>

#include "hft_kernels.cuh"

namespace hft {

constexpr int STS_KMAX = 8;

template <typename real, int C> struct VecOf;
template <> struct VecOf<double, 2> { typedef double2 type; };
template <> struct VecOf<float, 4> { typedef float4 type; };
template <> struct VecOf<float, 2> { typedef float2 type; };

template <typename real, int C>
__device__ __forceinline__ void vload(real (&d)[C], const real* p) {
    typename VecOf<real, C>::type v = *reinterpret_cast<const typename VecOf<real, C>::type*>(p);
    const real* s = reinterpret_cast<const real*>(&v);
#pragma unroll
    for (int i = 0; i < C; i++) d[i] = s[i];
}
template <typename real, int C>
__device__ __forceinline__ void vstore(real* p, const real (&d)[C]) {
    typename VecOf<real, C>::type v;
    real* s = reinterpret_cast<real*>(&v);
#pragma unroll
    for (int i = 0; i < C; i++) s[i] = d[i];
    *reinterpret_cast<typename VecOf<real, C>::type*>(p) = v;
}

// ------------------------------------------------------------------ compute-type traits: a "group" is what one FMA handles
template <typename creal> struct UVec;
template <> struct UVec<double> {
    typedef double V;                       // one cell per FMA
    static constexpr int W = 1;
    static __device__ __forceinline__ V fma(V a, V b, V c) { return ::fma(a, b, c); }
    static __device__ __forceinline__ V mul(V a, V b) { return a * b; }
    static __device__ __forceinline__ V dup(double x) { return x; }
    static __device__ __forceinline__ double get(const V& v, int) { return v; }
    static __device__ __forceinline__ void set(V& v, int, double x) { v = x; }
    static __host__ V hdup(double x) { return x; }
};
template <> struct UVec<float> {
    typedef float2 V;                       // two cells per FFMA2
    static constexpr int W = 2;
    static __device__ __forceinline__ V fma(V a, V b, V c) { return __ffma2_rn(a, b, c); }
    static __device__ __forceinline__ V mul(V a, V b) { return __fmul2_rn(a, b); }
    static __device__ __forceinline__ V dup(float x) { return make_float2(x, x); }
    static __device__ __forceinline__ float get(const V& v, int i) { return i == 0 ? v.x : v.y; }
    static __device__ __forceinline__ void set(V& v, int i, float x) { if (i == 0) v.x = x; else v.y = x; }
    static __host__ V hdup(double x) { return make_float2((float)x, (float)x); }
};

template <typename real, int K>
struct BlkArgs {
    const real* cur;   // level 0  = delta_{j0}
    const real* prev;  // level -1 = delta_{j0-1} (not read if !has_prev: delta_0 = 0)
    const real* F;     // L(Y0)
    real* ocur;        // level K   = delta_{j0+K}
    real* oprev;       // level K-1 = delta_{j0+K-1}
    real* Y0;          // last block: Y0 += delta_s, ocur/oprev not written
    const double* capseq;  // [R][2][K] cap values of levels 1..K
    real mu[K], nu[K], a[K], g[K];  // scalars of stages j0+1 .. j0+K
    typename UVec<real>::V nu2[K], g2[K];   // nu, g once more as FMA operands: {x, x} pairs in fp32 (FFMA2)
    int has_prev, last;
    int rows_per_seg, nstrips;
};

// ------------------------------------------------------------------ cap sequence from zonal means
// grid (2 poles, R), block 32 * STS_KMAX.  i = distance from the pole in rows (i = 0 is the cap itself).  Warp i-1
// sums row i of the three inputs (16-byte loads, lane-strided partial sums, shuffle tree: a fixed order, so the
// result is deterministic); thread 0 then runs the K-stage recurrence on the K+1 zonal means.
template <typename real, int K>
__global__ void __launch_bounds__(32 * STS_KMAX) k_sts_capseq(BlkArgs<real, K> A, Tables<real> T, Geom G, double* capseq) {
    constexpr int C = 16 / (int)sizeof(real);
    __shared__ double m0[K + 1], mp[K + 1], mF[K + 1], s_out[K + 1], s_in[K + 1];
    const int pole = blockIdx.x, r = blockIdx.y;
    const int lane = threadIdx.x & 31, i = (threadIdx.x >> 5) + 1;
    const size_t base = (size_t)r * G.rstride;
    auto rowidx = [&](int d) { return pole == 0 ? d : G.nt + 1 - d; };
    if (i <= K) {
        const size_t off = base + (size_t)rowidx(i) * G.pitch;
        const bool lower = i < K;   // prev and F are needed on rows 1..K-1 only
        double a = 0.0, b = 0.0, c = 0.0;
        // whole 16-byte vectors, four iterations of independent loads in flight per lane (one dependent L2 round trip per
        // iteration made this kernel 10-16 us: a quarter of a step on a single 512x1024 realization)
        const int nvec = G.np / C;   // whole vectors in a row
#pragma unroll 4
        for (int iv = lane; iv < nvec; iv += 32) {
            const int k = iv * C;
            real v[C];
            vload<real, C>(v, A.cur + off + k);
#pragma unroll
            for (int q = 0; q < C; q++) a += (double)v[q];
            if (lower) {
                if (A.has_prev) {
                    vload<real, C>(v, A.prev + off + k);
#pragma unroll
                    for (int q = 0; q < C; q++) b += (double)v[q];
                }
                vload<real, C>(v, A.F + off + k);
#pragma unroll
                for (int q = 0; q < C; q++) c += (double)v[q];
            }
        }
        // n_phi not a multiple of C: the last columns of the row one by one
        for (int kk = nvec * C + lane; kk < G.np; kk += 32) {
            a += (double)A.cur[off + kk];
            if (lower) {
                if (A.has_prev) b += (double)A.prev[off + kk];
                c += (double)A.F[off + kk];
            }
        }
        a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
        if (lane == 0) { m0[i] = a / (double)G.np; mp[i] = b / (double)G.np; mF[i] = c / (double)G.np; }
    }
    const real* cp = T.cp + (size_t)r * (G.nt + 2);
    const real* cm = T.cm + (size_t)r * (G.nt + 2);
    if (lane == 1 && i <= K) {   // theta coefficients of row i: towards the equator / towards the pole
        const int j = rowidx(i);
        s_out[i] = (double)(pole == 0 ? cp[j] : cm[j]);
        s_in[i] = (double)(pole == 0 ? cm[j] : cp[j]);
    }
    if (threadIdx.x == 2) {      // the cap itself
        const size_t capoff = base + (size_t)rowidx(0) * G.pitch;
        m0[0] = (double)A.cur[capoff];
        mp[0] = A.has_prev ? (double)A.prev[capoff] : 0.0;
        mF[0] = (double)A.F[capoff];
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    const double capc = T.capc[2 * r + pole] * (double)G.np;
    double lc[K + 1], lp[K + 1], ln[K + 1];  // current level, previous level, new level
    for (int d = 0; d <= K; d++) { lc[d] = m0[d]; lp[d] = mp[d]; }
    for (int s = 1; s <= K; s++) {
        const double mu = (double)A.mu[s - 1], nu = (double)A.nu[s - 1], a = (double)A.a[s - 1], g = (double)A.g[s - 1];
        ln[0] = mu * lc[0] + nu * lp[0] + a * (capc * (lc[1] - lc[0])) + g * mF[0];
        for (int d = 1; d <= K - s; d++) {
            const double c_out = s_out[d], c_in = s_in[d];
            ln[d] = mu * lc[d] + nu * lp[d] + a * (c_out * (lc[d + 1] - lc[d]) - c_in * (lc[d] - lc[d - 1])) + g * mF[d];
        }
        capseq[((size_t)r * 2 + pole) * K + (s - 1)] = ln[0];
        for (int d = 0; d <= K - s; d++) { lp[d] = lc[d]; lc[d] = ln[d]; }
    }
}

// ------------------------------------------------------------------ host side

template <typename real> struct BlkCfg;
template <> struct BlkCfg<double> { static constexpr int C = 2; };
template <> struct BlkCfg<float> { static constexpr int C = 4; };

// the blocked kernels take any n_phi (lanes behind the seam move their columns one by one)
inline bool sts_blocked_supported(const Geom& G, size_t wbytes) {
    const int C = wbytes == 8 ? 2 : 4;
    return G.np >= 32 * C && G.nt >= 2 * STS_KMAX;
}
inline int sts_default_block(const Geom& G, size_t wbytes) { return sts_blocked_supported(G, wbytes) ? 8 : 1; }
inline size_t sts_zmean_bytes(const Geom&) { return 256; }
inline size_t sts_capseq_bytes(const Geom& G) { return (size_t)G.nr * 2 * STS_KMAX * sizeof(double) + 256; }
inline int sts_blocked_init(const Geom&, bool) { return 0; }

// CTAs of `kernel` resident on the current device (SMs x occupancy), cached per (device, kernel); the first call for a
// device also opts the kernel in to `smem` bytes of dynamic shared memory there.  < 1 on error.
template <typename KernelT>
int resident_ctas(KernelT kernel, int threads, int smem) {
    static std::mutex m;
    static std::map<std::pair<int, const void*>, int> cache;   // (kernels of one signature share this instantiation)
    int dev = 0, sms = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    std::lock_guard<std::mutex> lk(m);
    const auto key = std::make_pair(dev, (const void*)kernel);
    const auto it = cache.find(key);
    if (it != cache.end()) return it->second;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess || per_sm < 1)
        return -1;
    cache[key] = sms * per_sm;
    return sms * per_sm;
}

struct UPipePlan;   // hft_sts_upipe.cuh

template <typename real>
struct StsBlockedPlan {
    real* Y0;
    real* buf[5];
    const double *mu, *nu, *a, *g;  // per-stage scalars, index 1..s
    int s, kb;
    cudaStream_t stream;
    double** part;   // the two polar partial-sum buffers of the unblocked kernels
    double* zmean;
    double* capseq;
    void (*prof_begin)(void*, bool*);
    void (*prof_end)(void*, bool, int);
    void* user;
    const UPipePlan* up;   // uniform-coefficient kernel (hft_sts_upipe.cuh) if up && up->ok, else k_sts_pipe
};

}  // namespace hft
