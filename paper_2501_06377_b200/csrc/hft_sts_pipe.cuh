// hft_sts_pipe.cuh -- temporally blocked super-time-stepping, second generation: K STS stages per launch with
// (i) register windows that ROTATE by unrolling instead of moving, (ii) an asynchronous shared-memory ring
// (cp.async, several rows per warp in flight) for the three input streams, (iii) the per-(stage,row)
// coefficient products formed once per warp row-step by the 32 lanes together instead of by every lane.
//
// Decomposition (hft_sts_blocked.cuh): a WARP owns a strip of
// 32*C phi-columns (one 16-byte vector per lane) and streams down the theta-rows; level l (= stage j0+l) lags
// level l-1 by one row; phi-neighbours come from the adjacent lanes by shuffle; warps never synchronise with
// each other.  What changed is the instruction stream (profiles/r01_cfg3_f64_first_pass.md: 523 warp
// instructions per row-step of which 112 were the stencil's DFMAs):
//
//  * Row-step t keeps, for every level, rows t-l, t-l-1, t-l-2 in registers.  Row rho of level l lives in slot
//    rho mod 3, F row rho in slot rho mod (K+1).  The row loop is unrolled U = lcm(3, K+1) times, so every slot
//    index is a compile-time constant and no register is ever copied.
//  * Inputs (delta_{j0}, delta_{j0-1}, L(Y0)) arrive through a per-warp ring of D = K+1 rows in shared memory
//    filled by cp.async 16 B per lane, D-2 rows ahead: each lane copies and later reads only ITS OWN 16 bytes,
//    so no barrier of any kind is needed for the data, and ~10 KB per warp are in flight instead of one row.
//  * The products a_l*cm_j, a_l*cp_j, a_l*cf_j, mu_l - a_l*cd_j of level l at row j = t-l are warp-uniform.
//    Lane (l-1)*4+q forms product q of level l with ONE fma per row-step and publishes it in shared memory;
//    every lane then reads the 4 products of a level with one or two broadcast LDS.128.
//  * Two code paths per warp: the steady-state path (all K levels on interior rows) has no branch on the row
//    index; the generic path (first / last rows of the sphere) overrides the polar-cap rows with the values of
//    k_sts_capseq.
//
// Arithmetic per cell and level (Eq. 27-28 with constant nu; recurrence DESIGN.md U20):
//   delta_l[j,k] = g_l F + nu_l delta_{l-2} + Af (e + w) + Ac c + An n + As s      (7 flops as 1 add + 6 fma)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "hft_sts_blocked.cuh"
#include "hft_sts_map.cuh"

namespace hft {

__host__ __device__ constexpr int pmod(int a, int m) { return ((a % m) + m) % m; }

// CTA shape per precision: warps (= strips) per CTA -- warps never synchronise with each
// other -- and the resident CTAs per SM the register budget is set for.  fp64: 4 x 2 with the long body (206 registers);
// 12 warps per SM with the short body need 4 % fewer cycles but draw more power, and under the 1000 W cap the clock drops by
// more than that (122.5 against 120.7 ms per cfg 3 step).  fp32 (not power-limited): 4 x 3 with the short body at 168
// registers, 12 warps per SM: 59.7 -> 53.6 ms per step (3 x 3: 56.5, 2 x 5: 54.0, 2 x 6: 53.9, 3 x 4: 56.8).
template <typename real> struct PipeShape {
    static constexpr int WARPS = 4, MINB = sizeof(real) == 4 ? 3 : 2;
};

template <typename real, int K>
struct PipeCfg {
    static constexpr int C = 16 / (int)sizeof(real);          // columns per lane
    static constexpr int NF = K + 1;                          // F rows alive in registers
    // Two loop bodies.  SHIFTF = false (fp64): the F slots rotate by unrolling lcm(3, K+1) = 9 row-steps, no register is
    // ever moved.  SHIFTF = true (fp32): the body is 3 row-steps (the period of the level windows); the F rows live in a
    // sliding window of K+3 register rows that is shifted down by 3 rows after every body (K short register moves per 3
    // row-steps) and the slot of the shared-memory ring is a run-time offset -- a third of the straight-line code.  The
    // long body stalls on instruction fetch (0.31 per issue in fp32, 0.19 in fp64); measured on cfg 3 the short body is
    // 3 % faster in fp32 and 1.5 % slower in fp64 (where the extra moves and slot arithmetic cost more than the fetches).
    static constexpr bool SHIFTF = sizeof(real) == 4;
    static constexpr int U = SHIFTF ? 3 : ((NF % 3 == 0) ? NF : 3 * NF);   // row-steps per unrolled macro-iteration
    static constexpr int NFW = SHIFTF ? K + 3 : NF;
    static constexpr int D = NF;                              // ring depth in rows
    static constexpr int DP = D - 2;                          // prefetch distance in rows
    static constexpr int ROW = 32 * C;                        // reals per ring row (512 B)
    static constexpr int NCS = 3;                             // coefficient ring slots (divides U)
    static constexpr int W = UVec<real>::W, NG = C / W;       // cells per FMA (fp32: 2, FFMA2), groups per lane
    static constexpr int CS = K * 4 * W;                      // reals per coefficient slot: 4 products per level, fp32 as {p, p} pairs
    static constexpr int WARP_REALS = 3 * D * ROW + NCS * CS + D * 32;   // data rings, product ring, raw-coefficient ring
    static constexpr int WARP_BYTES = WARP_REALS * (int)sizeof(real);
    static constexpr int HALO = (K + C - 1) / C * C;          // invalid columns per strip side, whole 16-byte vectors
    static constexpr int WOUT = 32 * C - 2 * HALO;            // columns written per warp
    static_assert(DP >= 1, "K >= 2");
    static_assert(K * 4 <= 32, "one lane per (level, coefficient)");
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_small(uint32_t dst, const double* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_small(uint32_t dst, const float* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ double fma_r(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_r(float a, float b, float c) { return fmaf(a, b, c); }

// SPLIT = false: n_phi is a multiple of C, every lane moves its C columns as one 16-byte vector (the hot instantiation).
// SPLIT = true:  any n_phi; lanes that are misaligned or straddle the seam move their columns one by one.
template <typename real, int K, bool SPLIT>
struct PipeWarp {
    using P = PipeCfg<real, K>;
    static constexpr int C = P::C, U = P::U, D = P::D, DP = P::DP, NF = P::NF, ROW = P::ROW, NCS = P::NCS;
    static constexpr int W = P::W, NG = P::NG, CS = P::CS;
    static constexpr bool SHIFTF = P::SHIFTF;
    static constexpr bool HOIST_SHFL = true;
    using UV = UVec<real>;
    using V = typename UV::V;   // what one FMA handles: a double, or a float2 pair (packed FFMA2 / FMUL2 of sm_100)

    // registers
    V u[K][3][NG];     // level l (0..K-1), row rho in slot rho mod 3 (relative to the macro-iteration origin)
    V f[P::NFW][NG];   // F row rho in slot rho mod NF; SHIFTF: row tb + x of the current body in slot x + K, x = -K..2
    int rb;            // SHIFTF: shared-memory ring slot of row tb (0, 3, 6, .. < D)
    // per-warp constants
    const BlkArgs<real, K>& A;
    const real *gcur, *gprev, *gF;   // this lane's column of row 0 of the three inputs
    real *gocur, *goprev, *gY0;
    real *s_cur, *s_prev, *s_F, *s_coef;   // shared: this lane's 16 bytes of ring slot 0; coefficient ring
    real* s_raw;                     // shared: this lane's raw coefficient of ring slot 0 (one real per lane and slot)
    const real* c4;                  // raw row coefficients [nt+2][4] of this realization, offset by this lane's q
    const double *capN, *capS;
    real sa, sadd;                   // this lane's product: fma(sa, raw, sadd)
    int cl;                          // this lane's level - 1
    int nt, pitch, ja, jb, lane;
    // a lane whose C columns are 16-byte aligned and do not straddle the periodic seam moves them as one vector; with
    // n_phi not a multiple of C the lanes behind the seam of the first / last strip are misaligned and move their
    // columns one by one (dq = element offsets relative to the lane's first column, wmask = elements this lane writes)
    bool simple;
    int dq[C];
    int wmask;

    __device__ __forceinline__ PipeWarp(const BlkArgs<real, K>& A_) : A(A_) {}

    __device__ __forceinline__ void prefetch(int row, int slot) {
        if (row <= nt + 1) {
            const size_t o = (size_t)row * pitch;
            if (!SPLIT || simple) {
                cp_async16(smem_u32(s_cur + slot * ROW), gcur + o);
                cp_async16(smem_u32(s_prev + slot * ROW), gprev + o);
                cp_async16(smem_u32(s_F + slot * ROW), gF + o);
            } else {
#pragma unroll
                for (int q = 0; q < C; q++) {
                    cp_async_small(smem_u32(s_cur + slot * ROW + q), gcur + o + dq[q]);
                    cp_async_small(smem_u32(s_prev + slot * ROW + q), gprev + o + dq[q]);
                    cp_async_small(smem_u32(s_F + slot * ROW + q), gF + o + dq[q]);
                }
            }
        }
        // the raw row coefficient behind this lane's product of row-step row+1 rides in the same group, so it has
        // landed when the data of `row` has (an LDG issued three row-steps ahead still stalled 17 % of the warp
        // samples: profiles/r01_pipe_cfg3_gen2.md)
        if (cl < K) cp_async_small(smem_u32(s_raw + slot * 32), c4 + min(max(row - cl, 0), nt + 1) * 4);
        cp_async_commit();
    }

    // raw row coefficient behind this lane's product of row-step t: level cl+1 works on row t-(cl+1)
    __device__ __forceinline__ real raw_of(int t) const { return c4[min(max(t - (cl + 1), 0), nt + 1) * 4]; }

    // products used by row-step t
    __device__ __forceinline__ void gen_coef(int t, int slot) {
        if (cl < K) put_coef(slot, fma_r(sa, raw_of(t), sadd));
    }
    // this lane's product into its place of coefficient slot `slot` (fp32: both halves of the pair)
    __device__ __forceinline__ void put_coef(int slot, real p) {
        *reinterpret_cast<V*>(s_coef + slot * CS + lane * W) = UV::dup(p);
    }
    __device__ __forceinline__ static void vld(V (&d)[NG], const real* p) { vload<real, C>(*reinterpret_cast<real(*)[C]>(&d[0]), p); }

    template <int PH, bool GEN>
    __device__ __forceinline__ void rowstep(int t) {
        cp_async_wait<DP - 1>();   // this lane's copies of row t have landed
        __syncwarp();              // the products written during the previous row-step are visible
        int sl, slm1, slpf;        // ring slots of rows t, t-1 and t+DP
        if constexpr (SHIFTF) {
            sl = rb + PH; if (sl >= D) sl -= D;
            slm1 = sl - 1; if (slm1 < 0) slm1 += D;
            slpf = sl + DP; if (slpf >= D) slpf -= D;
        } else {
            sl = PH % D; slm1 = pmod(PH - 1, D); slpf = (PH + DP) % D;
        }
        constexpr int fnew = SHIFTF ? PH + K : PH % NF;
        vld(u[0][PH % 3], s_cur + sl * ROW);
        vld(f[fnew], s_F + sl * ROW);
        V pl1[NG];                 // delta_{j0-1} row t-1: the "two levels back" operand of level 1
        vld(pl1, s_prev + slm1 * ROW);
        prefetch(t + DP, slpf);    // overwrites the slot of row t-2, last read one row-step ago
        const real raw_next = s_raw[sl * 32];   // this lane's own copy, arrived with the group of row t
        const real* cfs = s_coef + (PH % NCS) * CS;
        V outK[NG];
        // phi-neighbours of every level first: level l reads row t-l of level l-1, which the PREVIOUS row-step produced, so
        // all 2K shuffles of a row-step are independent of its arithmetic (issued where they are used, their (e + w) adds
        // waited on the shuffle: 10 % of the warp samples, profiles/r02_blocked_kernels.md)
        real wv[K], ev[K];
        if constexpr (HOIST_SHFL) {
#pragma unroll
            for (int l = 1; l <= K; l++) {
                const int sC = pmod(PH - l, 3);
                wv[l - 1] = __shfl_up_sync(0xffffffffu, UV::get(u[l - 1][sC][NG - 1], W - 1), 1);
                ev[l - 1] = __shfl_down_sync(0xffffffffu, UV::get(u[l - 1][sC][0], 0), 1);
            }
        }
#pragma unroll
        for (int l = 1; l <= K; l++) {
            // level l-1: newest row t-l+1 (s), centre t-l (c), oldest t-l-1 (n)
            const int sN = pmod(PH - (l - 1), 3), sC = pmod(PH - l, 3), sO = pmod(PH - l - 1, 3);
            V cf4[4];              // An, As, Af, Ac of this level and row: two broadcast LDS.128
            vload<real, 2 * W>(*reinterpret_cast<real(*)[2 * W]>(&cf4[0]), cfs + (l - 1) * 4 * W);
            vload<real, 2 * W>(*reinterpret_cast<real(*)[2 * W]>(&cf4[2]), cfs + (l - 1) * 4 * W + 2 * W);
            const V An = cf4[0], As = cf4[1], Af = cf4[2], Ac = cf4[3];
            const V nuc = A.nu2[l - 1], gc = A.g2[l - 1];
            const real west = HOIST_SHFL ? wv[l - 1] : __shfl_up_sync(0xffffffffu, UV::get(u[l - 1][sC][NG - 1], W - 1), 1);
            const real east = HOIST_SHFL ? ev[l - 1] : __shfl_down_sync(0xffffffffu, UV::get(u[l - 1][sC][0], 0), 1);
            V res[NG];
#pragma unroll
            for (int gI = 0; gI < NG; gI++) {
                const V c = u[l - 1][sC][gI];
                V S;               // e + w of every cell of the group (scalar adds; the FMAs are packed in fp32)
#pragma unroll
                for (int i = 0; i < W; i++) {
                    const int q = gI * W + i;
                    const real w = (q == 0) ? west : UV::get(u[l - 1][sC][(q > 0 ? q - 1 : 0) / W], (q > 0 ? q - 1 : 0) % W);
                    const real e = (q == C - 1) ? east : UV::get(u[l - 1][sC][(q < C - 1 ? q + 1 : 0) / W], (q < C - 1 ? q + 1 : 0) % W);
                    UV::set(S, i, e + w);
                }
                const V p2 = (l == 1) ? pl1[gI] : u[l >= 2 ? l - 2 : 0][sC][gI];   // level l-2 row t-l is ITS oldest: slot (PH-(l-2)-2) mod 3 = sC
                V acc = UV::mul(gc, f[SHIFTF ? PH - l + K : pmod(PH - l, NF)][gI]);
                acc = UV::fma(nuc, p2, acc);
                acc = UV::fma(Af, S, acc);
                acc = UV::fma(Ac, c, acc);
                acc = UV::fma(An, u[l - 1][sO][gI], acc);
                acc = UV::fma(As, u[l - 1][sN][gI], acc);   // the only operand produced in this row-step
                res[gI] = acc;
            }
            if (GEN) {
                const int j = t - l;
                if (j == 0 || j == nt + 1) {
                    const real cv = (real)(j == 0 ? capN[l - 1] : capS[l - 1]);
#pragma unroll
                    for (int gI = 0; gI < NG; gI++) res[gI] = UV::dup(cv);
                }
            }
            if (l < K) {
#pragma unroll
                for (int gI = 0; gI < NG; gI++) u[l < K ? l : 0][sC][gI] = res[gI];   // level l newest = row t-l: slot (PH-l) mod 3 = sC
            } else {
#pragma unroll
                for (int gI = 0; gI < NG; gI++) outK[gI] = res[gI];
            }
        }
        // products for the next row-step (slot last read two row-steps ago)
        if (cl < K) put_coef((PH + 1) % NCS, fma_r(sa, raw_next, sadd));
        // row jo = t-K of levels K and K-1 (level K-1 row t-K is its centre: slot (PH-(K-1)-1) mod 3)
        const int jo = t - K;
        if (wmask && jo >= ja && jo < jb) {
            const size_t o = (size_t)jo * pitch;
            real oc[C], op[C];
#pragma unroll
            for (int q = 0; q < C; q++) {
                oc[q] = UV::get(outK[q / W], q % W);
                op[q] = UV::get(u[K - 1][pmod(PH - K, 3)][q / W], q % W);
            }
            if (!SPLIT || (simple && wmask == (1 << C) - 1)) {
                if (A.last) {
                    real y[C];
                    vload<real, C>(y, gY0 + o);
#pragma unroll
                    for (int q = 0; q < C; q++) y[q] += oc[q];
                    vstore<real, C>(gY0 + o, y);
                } else {
                    vstore<real, C>(gocur + o, oc);
                    vstore<real, C>(goprev + o, op);
                }
            } else {
#pragma unroll
                for (int q = 0; q < C; q++)
                    if (wmask >> q & 1) {
                        if (A.last) {
                            gY0[o + dq[q]] += oc[q];
                        } else {
                            gocur[o + dq[q]] = oc[q];
                            goprev[o + dq[q]] = op[q];
                        }
                    }
            }
        }
    }

    template <int PH, bool GEN>
    __device__ __forceinline__ void macro(int tb) {
        rowstep<PH, GEN>(tb + PH);
        if constexpr (PH + 1 < U) macro<PH + 1, GEN>(tb);
        else if constexpr (SHIFTF) {   // slide the F window down by the 3 rows of this body
#pragma unroll
            for (int i = 0; i < K; i++)
#pragma unroll
                for (int gI = 0; gI < NG; gI++) f[i][gI] = f[i + 3][gI];
            rb += 3;
            if (rb >= D) rb -= D;
        }
    }
};

template <typename real, int K, bool SPLIT = false>
__global__ void __launch_bounds__(PipeShape<real>::WARPS * 32, PipeShape<real>::MINB) k_sts_pipe(const __grid_constant__ BlkArgs<real, K> A, Tables<real> T, Geom G) {
    using P = PipeCfg<real, K>;
    constexpr int C = P::C, U = P::U, D = P::D, DP = P::DP, ROW = P::ROW;
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
    constexpr int PIPE_WARPS = PipeShape<real>::WARPS;
    // a warp's work item: (realization, strip) of theta segment blockIdx.y, strips fastest; the items of all realizations
    // are dealt to the CTAs as one list, so only the last CTA of a segment can have idle warps
    const int item = blockIdx.x * PIPE_WARPS + wrp;
    if (item >= A.nstrips * G.nr) return;   // warp-uniform; the kernel has no block-level barrier
    const int r = item / A.nstrips, strip = item - r * A.nstrips;
    const int nt = G.nt, np = G.np;
    PipeWarp<real, K, SPLIT> W(A);
    W.nt = nt; W.pitch = G.pitch; W.lane = lane;
    W.ja = blockIdx.y * A.rows_per_seg;
    W.jb = min(W.ja + A.rows_per_seg, nt + 2);
    const int t0 = max(W.ja - K, 0), tend = W.jb - 1 + K;
    const int uc = strip * P::WOUT - P::HALO + lane * C;   // unwrapped first column of this lane
    int col = uc % np;
    if (col < 0) col += np;
    W.simple = (col % C == 0) && (col + C <= np);
    W.wmask = 0;
#pragma unroll
    for (int q = 0; q < C; q++) {
        int cq = col + q;
        if (cq >= np) cq -= np;
        W.dq[q] = cq - col;
        if ((lane * C >= P::HALO) && (lane * C < P::HALO + P::WOUT) && (uc + q < np)) W.wmask |= 1 << q;
    }
    if (!SPLIT) W.wmask = ((lane * C >= P::HALO) && (lane * C < P::HALO + P::WOUT) && (uc < np)) ? (1 << C) - 1 : 0;
    const size_t base = (size_t)r * G.rstride + col;
    W.gcur = A.cur + base; W.gprev = A.prev + base; W.gF = A.F + base;
    W.gocur = A.ocur + base; W.goprev = A.oprev + base; W.gY0 = A.Y0 + base;
    real* ws = reinterpret_cast<real*>(pipe_smem) + (size_t)wrp * P::WARP_REALS;
    W.s_cur = ws + lane * C; W.s_prev = W.s_cur + D * ROW; W.s_F = W.s_prev + D * ROW;
    W.s_coef = ws + 3 * D * ROW;
    W.s_raw = W.s_coef + P::NCS * P::CS + lane;
    W.capN = A.capseq + ((size_t)r * 2 + 0) * K;
    W.capS = A.capseq + ((size_t)r * 2 + 1) * K;
    W.cl = lane >> 2;
    const int cq = lane & 3;
    W.c4 = T.c4 + (size_t)r * (nt + 2) * 4 + cq;
    W.sa = (real)0; W.sadd = (real)0;
    if (W.cl < K) {
        const real a = A.a[W.cl];
        W.sa = cq < 3 ? a : -a;
        W.sadd = cq < 3 ? (real)0 : A.mu[W.cl];
    }
#pragma unroll
    for (int l = 0; l < K; l++)
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int gI = 0; gI < P::NG; gI++) W.u[l][i][gI] = UVec<real>::dup((real)0);
#pragma unroll
    for (int i = 0; i < P::NFW; i++)
#pragma unroll
        for (int gI = 0; gI < P::NG; gI++) W.f[i][gI] = UVec<real>::dup((real)0);
    W.rb = 0;
    // clear this warp's shared memory (the ring slot of "row t0-1" is read before it is ever written)
    for (int i = lane; i < P::WARP_REALS; i += 32) ws[i] = (real)0;
    __syncwarp();
    for (int i = 0; i < DP; i++) W.prefetch(t0 + i, i);
    W.gen_coef(t0, 0);
    for (int tb = t0; tb <= tend; tb += U) {
        // steady state: every level of every row-step of this macro-iteration works on an interior row
        if (tb >= K + 1 && tb + U - 2 <= nt) W.template macro<0, false>(tb);
        else W.template macro<0, true>(tb);
    }
    cp_async_wait<0>();
}

// ------------------------------------------------------------------ host side

template <typename real, int K, bool SPLIT>
int sts_pipe_launch_impl(const StsBlockedPlan<real>& P, Tables<real>& T, const Geom& G, int j0, const real* cur, const real* prev,
                         real* ocur, real* oprev, bool last, int64_t* launches) {
    using PC = PipeCfg<real, K>;
    constexpr int PIPE_WARPS = PipeShape<real>::WARPS;
    const int smem = PIPE_WARPS * PC::WARP_BYTES;
    const int slots = resident_ctas(k_sts_pipe<real, K, SPLIT>, PIPE_WARPS * 32, smem);   // CTAs resident on this device
    if (slots < 1) return -1;
    BlkArgs<real, K> a;
    a.cur = cur; a.prev = prev; a.F = P.buf[0]; a.ocur = ocur; a.oprev = oprev; a.Y0 = P.Y0; a.capseq = P.capseq;
    for (int i = 0; i < K; i++) {
        a.mu[i] = (real)P.mu[j0 + 1 + i]; a.nu[i] = (real)P.nu[j0 + 1 + i];
        a.a[i] = (real)P.a[j0 + 1 + i]; a.g[i] = (real)P.g[j0 + 1 + i];
        a.nu2[i] = UVec<real>::hdup(P.nu[j0 + 1 + i]); a.g2[i] = UVec<real>::hdup(P.g[j0 + 1 + i]);
    }
    a.has_prev = 1; a.last = last;
    a.nstrips = (G.np + PC::WOUT - 1) / PC::WOUT;
    const long ctas_x = ((long)a.nstrips * G.nr + PIPE_WARPS - 1) / PIPE_WARPS;   // per theta segment
    // theta segments: every segment re-streams K rows above and below its own (the cone of K stages), and the grid
    // runs in waves of `slots` CTAs; take the count that minimises waves x row-steps per segment
    int nseg = 1;
    long best = -1;
    // (a small batch leaves most of the 148 SMs idle: short segments, down to K rows each, then cost nothing although
    // they re-stream more rows than they own -- cfg 1, one 512x1024 realization, runs 22 strips x 32 segments)
    for (int n = 1; n <= 64 && (G.nt + 2) / n >= K; n++) {
        const long rows = (G.nt + 2 + n - 1) / n + 2 * K;
        const long waves = (ctas_x * n + slots - 1) / slots;
        if (best < 0 || waves * rows < best) { best = waves * rows; nseg = n; }
    }
    if (ctas_x > 0x7fffffffL) return -1;
    a.rows_per_seg = (G.nt + 2 + nseg - 1) / nseg;
    nseg = (G.nt + 2 + a.rows_per_seg - 1) / a.rows_per_seg;   // no empty segment
    dim3 gc(2, G.nr), g((unsigned)ctas_x, nseg);
    k_sts_capseq<real, K><<<gc, 32 * STS_KMAX, 0, P.stream>>>(a, T, G, P.capseq);
    bool armed = false;
    P.prof_begin(P.user, &armed);
    k_sts_pipe<real, K, SPLIT><<<g, PIPE_WARPS * 32, smem, P.stream>>>(a, T, G);
    P.prof_end(P.user, armed, K);
    *launches += 2;
    return 0;
}

template <typename real, int K>
int sts_pipe_launch(const StsBlockedPlan<real>& P, Tables<real>& T, const Geom& G, int j0, const real* cur, const real* prev,
                    real* ocur, real* oprev, bool last, int64_t* launches) {
    if (G.np % PipeCfg<real, K>::C == 0) return sts_pipe_launch_impl<real, K, false>(P, T, G, j0, cur, prev, ocur, oprev, last, launches);
    return sts_pipe_launch_impl<real, K, true>(P, T, G, j0, cur, prev, ocur, oprev, last, launches);
}

}  // namespace hft
