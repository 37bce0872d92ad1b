// hft_sts_upipe.cuh -- temporally blocked super-time-stepping, third generation: the K-stage software pipeline of
// k_sts_pipe (hft_sts_pipe.cuh) with every coefficient delivered through the UNIFORM datapath instead of shared memory.
//
// What bound k_sts_pipe (profiles/r01_final_cfg3.md, r01d_pipe_f32_3rowstep.md): the products a_l*c_j of a stage scalar
// and a row coefficient are warp-uniform but differ for every (level, row), so each level of each row-step fetched four
// of them with broadcast LDS (fp64: a third of the shared-memory datapath, the binding limit) and the fp32 instantiation
// spent 226 of its 363 warp instructions per row-step on scalar FFMA/FMUL/FADD (issue-bound).
//
// Reformulation (exact in exact arithmetic; reading U32).  The STS recurrence in deviation form (U20) with the
// operator of Eq. 27-28 for a diffusivity nu_r * p(theta) (p common to the batch), L = nu_r Lh, and
// a_l = mu_l w1 dt (the definition of mu~_l, Sec. 3.7.2) is
//     delta_l = mu_l [delta_{l-1} + kappa_r Lh(delta_{l-1})] + nu_l delta_{l-2} + g_l F,        kappa_r = w1 dt nu_r.
// Inside a block the kernel carries zeta_l = delta_l / Pi_l with Pi_0 = 1, Pi_l = mu_l Pi_{l-1}:
//     zeta_l = zeta_{l-1} + kappa_r Lh(zeta_{l-1}) + N_l zeta_{l-2} + G_l F,   N_l = nu_l Pi_{l-2}/Pi_l,  G_l = g_l / Pi_l
// so the operator's row coefficients (cm_j, cp_j, cf_j, -cd_j)/nu_r no longer depend on the level or on the realization:
// ONE table of n_theta rows x 32 bytes serves the whole launch.  It lives in the constant bank; the row index is
// warp-uniform, so the compiler fetches a row with LDCU (uniform load) into uniform registers and DFMA / FFMA2 take the
// uniform register as an operand: no shared-memory traffic, no vector register, no instruction on the FMA pipe for any
// coefficient.  N_l, G_l, Pi_l are the same for every realization and ride in the kernel parameters (constant-bank
// operands at fixed offsets); kappa_r is the one per-realization scalar (two registers).  Pi_l <= 2^K: no range issue.
// Cost per cell and level: (e + w), four operations for Lh, three FMAs for the combination = 8 (k_sts_pipe: 7).
// The uniform path needs the compiler to PROVE the row index uniform: the row loop counts from 0 with a base that is
// block index x parameter + constant -- a min()/max() anywhere in that chain sends every load through vector registers
// (checked in the SASS: LDCU.64 UR, c[0x3][UR] feeding DFMA R, R, UR, R).
//
// fp32: a lane's four columns are two float2 pairs and every FMA is the packed FFMA2 of sm_100 (fma.rn.f32x2) with the
// coefficient pair {c, c} taken straight from the table (stored duplicated) -- half the FMA-pipe instructions.
// CREAL != REAL (fp32 storage, fp64 arithmetic; hft_options.f32_arith = 0): a lane owns two columns (8-byte vectors),
// converts on load, and rounds to fp32 only at the two stores per block (SURVEY.md section 7 hard part 3 fallback).
//
// Everything else is k_sts_pipe's design: a warp owns a strip of 32*C phi-columns and streams down the theta rows, level l
// lags level l-1 by one row, theta-neighbours live in rotating register slots, phi-neighbours come from the adjacent
// lanes by shuffle, inputs arrive through a per-warp cp.async ring, polar caps come from k_sts_capseq (reading U21).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <vector>

#include "hft_sts_pipe.cuh"

namespace hft {

constexpr int UTAB_BYTES = 65536;           // the whole user constant bank
constexpr int UTAB_ROW_BYTES = 32;          // 4 coefficients: 4 doubles, or 4 duplicated float pairs
constexpr int UTAB_MAX_ROWS = UTAB_BYTES / UTAB_ROW_BYTES;

// One instance per translation unit (= per arithmetic type; each has its own constant bank).
static __constant__ uint4 c_utab[UTAB_BYTES / 16];

template <typename real, typename creal, int K>
struct UArgs {
    const real *cur, *prev, *F;
    real *ocur, *oprev, *Y0;
    const double* capseq;                   // [R][2][K] cap values (delta units) of levels 1..K
    const double* kappa;                    // [R] w1 dt nu_r
    struct NG { typename UVec<creal>::V N, G; } ng[K];   // level scalars (see the header), duplicated pairs in fp32
    creal PiK, PiKm1;                       // delta_{j0+K} = PiK zeta_K, delta_{j0+K-1} = PiKm1 zeta_{K-1}
    creal iPi[K];                           // 1/Pi_l: cap values -> zeta units
    int last, rows_per_seg, nstrips, niter; // niter: macro-iterations of U row-steps per theta segment
    int rows_per_seg_u, ustep;              // == rows_per_seg, == U: the separately counted uniform row counter
    int zero;                               // 0, unknown to the compiler: see UPipeWarp::rowstep
};

template <typename real, typename creal, int K>
struct UCfg {
    static constexpr bool MIXED = sizeof(real) != sizeof(creal);
    static constexpr int C = MIXED ? 2 : 16 / (int)sizeof(real);   // columns per lane
    static constexpr int VB = C * (int)sizeof(real);               // bytes per lane and row (16, mixed: 8)
    static constexpr int W = UVec<creal>::W, NG = C / W;           // cells per group, groups per lane
    static constexpr int NF = K + 1;
    // loop body as in PipeCfg: fp64 arithmetic rotates the F slots by unrolling lcm(3, K+1) row-steps; fp32 runs a
    // 3-row-step body with a sliding F window
    static constexpr bool SHIFTF = true;
    static constexpr int U = SHIFTF ? 3 : ((NF % 3 == 0) ? NF : 3 * NF);
    static constexpr int NFW = SHIFTF ? K + 3 : NF;
    static constexpr int D = NF, DP = D - 2;
    static constexpr int ROW = 32 * C;                             // reals per ring row
    static constexpr int WARP_REALS = 3 * D * ROW;
    static constexpr int WARP_BYTES = WARP_REALS * (int)sizeof(real);
    static constexpr int HALO = (K + C - 1) / C * C;
    static constexpr int WOUT = 32 * C - 2 * HALO;
    static constexpr int WARPS = 4;
    static constexpr int MINB = sizeof(creal) == 4 ? 3 : 2;
    static_assert(DP >= 1, "K >= 2");
};

template <int BYTES> __device__ __forceinline__ void cp_async_vec(uint32_t dst, const void* src);
template <> __device__ __forceinline__ void cp_async_vec<16>(uint32_t dst, const void* src) { cp_async16(dst, src); }
template <> __device__ __forceinline__ void cp_async_vec<8>(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(dst), "l"(src) : "memory");
}

template <typename real, typename creal, int K, bool SPLIT>
struct UPipeWarp {
    using P = UCfg<real, creal, K>;
    using UV = UVec<creal>;
    using V = typename UV::V;
    static constexpr int C = P::C, W = P::W, NG = P::NG, U = P::U, D = P::D, DP = P::DP, NF = P::NF, ROW = P::ROW;
    static constexpr bool SHIFTF = P::SHIFTF;

    V u[K][3][NG];     // level l (0..K-1), row rho in slot rho mod 3
    V f[P::NFW][NG];   // F rows (slot rotation as in PipeWarp)
    int rb;
    const UArgs<real, creal, K>& A;
    V kap;             // {kappa_r, kappa_r}
    const real *gcur, *gprev, *gF;   // this lane's column of the NEXT row to prefetch (advance one row per prefetch)
    real *gocur, *goprev, *gY0;      // this lane's column of the row written by the CURRENT row-step (t - K)
    real *s_cur, *s_prev, *s_F;
    const double *capN, *capS;
    int nt, pitch, ja, jb;
    int zz;            // it * zero (see rowstep)
    bool simple;
    int dq[C];
    int wmask;

    __device__ __forceinline__ UPipeWarp(const UArgs<real, creal, K>& A_) : A(A_) {}

    __device__ __forceinline__ void prefetch(int row, int slot) {
        if (row >= 0 && row <= nt + 1) {
            if (!SPLIT || simple) {
                cp_async_vec<P::VB>(smem_u32(s_cur + slot * ROW), gcur);
                cp_async_vec<P::VB>(smem_u32(s_prev + slot * ROW), gprev);
                cp_async_vec<P::VB>(smem_u32(s_F + slot * ROW), gF);
            } else {
#pragma unroll
                for (int q = 0; q < C; q++) {
                    cp_async_small(smem_u32(s_cur + slot * ROW + q), gcur + dq[q]);
                    cp_async_small(smem_u32(s_prev + slot * ROW + q), gprev + dq[q]);
                    cp_async_small(smem_u32(s_F + slot * ROW + q), gF + dq[q]);
                }
            }
        }
        gcur += pitch; gprev += pitch; gF += pitch;
        cp_async_commit();
    }

    // this lane's C values of a ring row -> NG groups of the compute type
    __device__ __forceinline__ void ring_load(V (&d)[NG], const real* p) {
        real v[C];
        vload<real, C>(v, p);
#pragma unroll
        for (int q = 0; q < C; q++) UV::set(d[q / W], q % W, (creal)v[q]);
    }

    // t: this row-step, for predicates and the first / last rows of a segment.  tu: the same number, counted separately
    // (its own induction variable, advanced by a kernel parameter) and used for NOTHING but the table index of the steady
    // state.  The compiler promotes a value to the uniform datapath only if every use of it can run there; one clamp, one
    // conversion or one address computation on the row counter sends it -- and with it every table load -- to vector
    // registers and LDC (checked in the SASS; see the header).
    template <int PH, bool GEN>
    __device__ __forceinline__ void rowstep(int t, int tu) {
        cp_async_wait<DP - 1>();   // this lane's copies of row t have landed (each lane reads only its own bytes)
        int sl, slm1, slpf;        // ring slots of rows t, t-1 and t+DP
        if constexpr (SHIFTF) {
            sl = rb + PH; if (sl >= D) sl -= D;
            slm1 = sl - 1; if (slm1 < 0) slm1 += D;
            slpf = sl + DP; if (slpf >= D) slpf -= D;
        } else {
            sl = PH % D; slm1 = pmod(PH - 1, D); slpf = (PH + DP) % D;
        }
        constexpr int fnew = SHIFTF ? PH + K : PH % NF;
        ring_load(u[0][PH % 3], s_cur + sl * ROW);
        ring_load(f[fnew], s_F + sl * ROW);
        V pl1[NG];                 // delta_{j0-1} row t-1: the "two levels back" operand of level 1
        ring_load(pl1, s_prev + slm1 * ROW);
        prefetch(t + DP, slpf);    // overwrites the slot of row t-2, last read one row-step ago
        V outK[NG];
#pragma unroll
        for (int l = 1; l <= K; l++) {
            // level l-1: newest row t-l+1 (s), centre t-l (c), oldest t-l-1 (n)
            const int sN = pmod(PH - (l - 1), 3), sC = pmod(PH - l, 3), sO = pmod(PH - l - 1, 3);
            // the row of the table: warp-uniform index -> LDCU into uniform registers (GEN: clamped, the value of a row
            // outside 1..nt is never used -- caps are overridden below, rows beyond them feed nothing)
            int j = tu - l;
            if (GEN) j = min(max(t - l, 1), nt);   // (vector-register loads on this path: first / last rows of a segment only)
            // Every coefficient is loaded where it is used and dies there (4 + 2 uniform registers per level in flight).  Left
            // alone the compiler keeps them: a level reads table row j one row-step after the level below did, so the loads
            // of the unrolled body are common subexpressions with lifetimes of K row-steps, and the level scalars are loop
            // invariants -- together far more than the 63 uniform registers, so everything falls back to vector registers
            // and LDC.  The offsets l * zero (table) and zz = it * zero (level scalars) are 0 at run time and opaque at
            // compile time: loads of different levels / iterations are no longer provably equal.
            const V* row = reinterpret_cast<const V*>(c_utab) + 4 * (j - 1) + l * A.zero;
            const typename UArgs<real, creal, K>::NG& ng = A.ng[l - 1 + zz];
            const V An = row[0], As = row[1], Af = row[2], Ad = row[3];
            const creal west = __shfl_up_sync(0xffffffffu, UV::get(u[l - 1][sC][NG - 1], W - 1), 1);
            const creal east = __shfl_down_sync(0xffffffffu, UV::get(u[l - 1][sC][0], 0), 1);
            V res[NG];
#pragma unroll
            for (int gI = 0; gI < NG; gI++) {
                const V c = u[l - 1][sC][gI];
                V S;               // e + w of every cell of the group (scalar adds; the FMAs below are packed)
#pragma unroll
                for (int i = 0; i < W; i++) {
                    const int q = gI * W + i;
                    const creal w = (q == 0) ? west : UV::get(u[l - 1][sC][(q > 0 ? q - 1 : 0) / W], (q > 0 ? q - 1 : 0) % W);
                    const creal e = (q == C - 1) ? east : UV::get(u[l - 1][sC][(q < C - 1 ? q + 1 : 0) / W], (q < C - 1 ? q + 1 : 0) % W);
                    UV::set(S, i, e + w);
                }
                const V p2 = (l == 1) ? pl1[gI] : u[l >= 2 ? l - 2 : 0][sC][gI];
                V L = UV::mul(Ad, c);
                L = UV::fma(Af, S, L);
                L = UV::fma(An, u[l - 1][sO][gI], L);
                V acc = UV::fma(ng.N, p2, c);
                acc = UV::fma(ng.G, f[SHIFTF ? PH - l + K : pmod(PH - l, NF)][gI], acc);
                L = UV::fma(As, u[l - 1][sN][gI], L);       // the only operand produced in this row-step
                acc = UV::fma(kap, L, acc);
                res[gI] = acc;
            }
            if (GEN) {
                const int jj = t - l;
                if (jj == 0 || jj == nt + 1) {
                    const creal cv = (creal)((jj == 0 ? capN[l - 1] : capS[l - 1]) * (double)A.iPi[l - 1]);
#pragma unroll
                    for (int gI = 0; gI < NG; gI++) res[gI] = UV::dup(cv);
                }
            }
            if (l < K) {
#pragma unroll
                for (int gI = 0; gI < NG; gI++) u[l < K ? l : 0][sC][gI] = res[gI];
            } else {
#pragma unroll
                for (int gI = 0; gI < NG; gI++) outK[gI] = res[gI];
            }
        }
        // row jo = t-K of levels K and K-1, back in delta units
        const int jo = t - K;
        if (wmask && jo >= ja && jo < jb) {
            constexpr size_t o = 0;
            real oc[C], op[C];
#pragma unroll
            for (int q = 0; q < C; q++) {
                oc[q] = (real)(A.PiK * UV::get(outK[q / W], q % W));
                op[q] = (real)(A.PiKm1 * UV::get(u[K - 1][pmod(PH - K, 3)][q / W], q % W));
            }
            if (!SPLIT || (simple && wmask == (1 << C) - 1)) {
                if (A.last) {
                    real y[C];
                    vload<real, C>(y, gY0 + o);
#pragma unroll
                    for (int q = 0; q < C; q++) y[q] = (real)((creal)y[q] + A.PiK * UV::get(outK[q / W], q % W));
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
                            gY0[o + dq[q]] = (real)((creal)gY0[o + dq[q]] + A.PiK * UV::get(outK[q / W], q % W));
                        } else {
                            gocur[o + dq[q]] = oc[q];
                            goprev[o + dq[q]] = op[q];
                        }
                    }
            }
        }
        gocur += pitch; goprev += pitch; gY0 += pitch;
    }

    template <int PH, bool GEN>
    __device__ __forceinline__ void macro(int tb, int tbu) {
        rowstep<PH, GEN>(tb + PH, tbu + PH);
        if constexpr (PH + 1 < U) macro<PH + 1, GEN>(tb, tbu);
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

template <typename real, typename creal, int K, bool SPLIT>
__global__ void __launch_bounds__(UCfg<real, creal, K>::WARPS * 32, UCfg<real, creal, K>::MINB)
k_sts_upipe(const __grid_constant__ UArgs<real, creal, K> A, const __grid_constant__ Geom G) {
    using P = UCfg<real, creal, K>;
    using UV = UVec<creal>;
    constexpr int C = P::C, U = P::U, D = P::D, DP = P::DP, ROW = P::ROW;
    extern __shared__ __align__(128) unsigned char upipe_smem[];
    const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
    const int item = blockIdx.x * P::WARPS + wrp;   // (realization, strip) of theta segment blockIdx.y, as in k_sts_pipe
    if (item >= A.nstrips * G.nr) return;           // warp-uniform; the kernel has no block-level barrier
    const int r = item / A.nstrips, strip = item - r * A.nstrips;
    const int nt = G.nt, np = G.np;
    UPipeWarp<real, creal, K, SPLIT> Wp(A);
    Wp.nt = nt; Wp.pitch = G.pitch;
    Wp.kap = UV::dup((creal)A.kappa[r]);
    Wp.ja = blockIdx.y * A.rows_per_seg;
    Wp.jb = min(Wp.ja + A.rows_per_seg, nt + 2);
    // first row-step of this segment: the cone of its first output row.  NO max(.., 0) here: segment 0 starts K rows above
    // the sphere (rows < 0 are not loaded and feed nothing), so that the row counter stays block index x parameter +
    // constant and the table loads stay on the uniform datapath (see the header).
    const int t0 = Wp.ja - K;
    const int uc = strip * P::WOUT - P::HALO + lane * C;   // unwrapped first column of this lane
    int col = uc % np;
    if (col < 0) col += np;
    Wp.simple = (col % C == 0) && (col + C <= np);
    Wp.wmask = 0;
#pragma unroll
    for (int q = 0; q < C; q++) {
        int cq = col + q;
        if (cq >= np) cq -= np;
        Wp.dq[q] = cq - col;
        if ((lane * C >= P::HALO) && (lane * C < P::HALO + P::WOUT) && (uc + q < np)) Wp.wmask |= 1 << q;
    }
    if (!SPLIT) Wp.wmask = ((lane * C >= P::HALO) && (lane * C < P::HALO + P::WOUT) && (uc < np)) ? (1 << C) - 1 : 0;
    // row t0 (first prefetch) and row t0 - K (written by the first row-step); rows outside the sphere are never dereferenced
    const ptrdiff_t base = (ptrdiff_t)r * (ptrdiff_t)G.rstride + col + (ptrdiff_t)t0 * G.pitch;
    const ptrdiff_t obase = base - (ptrdiff_t)K * G.pitch;
    Wp.gcur = A.cur + base; Wp.gprev = A.prev + base; Wp.gF = A.F + base;
    Wp.gocur = A.ocur + obase; Wp.goprev = A.oprev + obase; Wp.gY0 = A.Y0 + obase;
    real* ws = reinterpret_cast<real*>(upipe_smem) + (size_t)wrp * P::WARP_REALS;
    Wp.s_cur = ws + lane * C; Wp.s_prev = Wp.s_cur + D * ROW; Wp.s_F = Wp.s_prev + D * ROW;
    Wp.capN = A.capseq + ((size_t)r * 2 + 0) * K;
    Wp.capS = A.capseq + ((size_t)r * 2 + 1) * K;
#pragma unroll
    for (int l = 0; l < K; l++)
#pragma unroll
        for (int i = 0; i < 3; i++)
#pragma unroll
            for (int gI = 0; gI < P::NG; gI++) Wp.u[l][i][gI] = UV::dup((creal)0);
#pragma unroll
    for (int i = 0; i < P::NFW; i++)
#pragma unroll
        for (int gI = 0; gI < P::NG; gI++) Wp.f[i][gI] = UV::dup((creal)0);
    Wp.rb = 0;
    // clear this warp's shared memory (ring slots of rows that do not exist are read before they are ever written)
    for (int i = lane; i < P::WARP_REALS; i += 32) ws[i] = (real)0;
    __syncwarp();
    for (int i = 0; i < DP; i++) Wp.prefetch(t0 + i, i);
    int tbu = (int)blockIdx.y * A.rows_per_seg_u - K;   // == tb, the uniform copy (UPipeWarp::rowstep)
    for (int it = 0; it < A.niter; it++) {
        const int tb = t0 + it * U;
        Wp.zz = tbu * A.zero;
        // steady state: every level of every row-step of this macro-iteration works on an interior row
        if (tb >= K + 1 && tb + U - 2 <= nt) Wp.template macro<0, false>(tb, tbu);
        else Wp.template macro<0, true>(tb, tbu);
        tbu += A.ustep;
    }
    cp_async_wait<0>();
}

// ------------------------------------------------------------------ host side

// The constant-bank table is per device and per translation unit; contexts take turns.  `key` identifies the content
// (context id, table version).  A change of owner waits for the device first: kernels of the previous owner may still read it.
struct UTabOwner {
    std::mutex m;
    uint64_t key[64] = {0};
};
static UTabOwner g_utab_owner;

inline int upipe_bind_table(const void* h_table, size_t bytes, uint64_t key, cudaStream_t stream) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return -1;
    std::lock_guard<std::mutex> lk(g_utab_owner.m);
    if (g_utab_owner.key[dev] == key) return 0;
    if (g_utab_owner.key[dev] != 0 && cudaDeviceSynchronize() != cudaSuccess) return -1;
    if (cudaMemcpyToSymbolAsync(c_utab, h_table, bytes, 0, cudaMemcpyHostToDevice, stream) != cudaSuccess) return -1;
    if (cudaStreamSynchronize(stream) != cudaSuccess) return -1;   // the host buffer may change after this call
    g_utab_owner.key[dev] = key;
    return 0;
}

// per-context description of the uniform-coefficient path, filled by hft_api.cu
struct UPipePlan {
    bool ok = false;              // the batch shares one coefficient table up to the factor nu_r, and it fits the bank
    bool mixed = false;           // fp32 storage, fp64 arithmetic
    const void* h_table = nullptr;   // [nt][4] of V (32 bytes per row), rows 1..nt: (cm, cp, cf, -cd) / nu_r
    uint64_t key = 0;
    const double* d_kappa = nullptr;   // [R] w1 dt nu_r (device)
    double w1dt = 0.0;
};

template <typename real, typename creal, int K, bool SPLIT>
int sts_upipe_launch_impl(const StsBlockedPlan<real>& P, const UPipePlan& UP, Tables<real>& T, const Geom& G, int j0, const real* cur,
                          const real* prev, real* ocur, real* oprev, bool last, int64_t* launches) {
    using PC = UCfg<real, creal, K>;
    using UV = UVec<creal>;
    const int smem = PC::WARPS * PC::WARP_BYTES;
    const int slots = resident_ctas(k_sts_upipe<real, creal, K, SPLIT>, PC::WARPS * 32, smem);
    if (slots < 1) return -1;
    if (upipe_bind_table(UP.h_table, (size_t)G.nt * UTAB_ROW_BYTES, UP.key, P.stream) != 0) return -1;
    // cap values of the block from the zonal means, as for k_sts_pipe
    BlkArgs<real, K> b;
    b.cur = cur; b.prev = prev; b.F = P.buf[0]; b.ocur = ocur; b.oprev = oprev; b.Y0 = P.Y0; b.capseq = P.capseq;
    for (int i = 0; i < K; i++) {
        b.mu[i] = (real)P.mu[j0 + 1 + i]; b.nu[i] = (real)P.nu[j0 + 1 + i];
        b.a[i] = (real)P.a[j0 + 1 + i]; b.g[i] = (real)P.g[j0 + 1 + i];
    }
    b.has_prev = 1; b.last = last; b.rows_per_seg = 0; b.nstrips = 0;
    dim3 gc(2, G.nr);
    k_sts_capseq<real, K><<<gc, 32 * STS_KMAX, 0, P.stream>>>(b, T, G, P.capseq);
    UArgs<real, creal, K> a;
    a.cur = cur; a.prev = prev; a.F = P.buf[0]; a.ocur = ocur; a.oprev = oprev; a.Y0 = P.Y0; a.capseq = P.capseq;
    a.kappa = UP.d_kappa;
    double Pi = 1.0, Pim1 = 1.0, Pim2 = 1.0;   // Pi_l, Pi_{l-1}, Pi_{l-2} (Pi_0 = Pi_{-1} = 1: both inputs come in delta units)
    for (int l = 1; l <= K; l++) {
        const int j = j0 + l;
        Pim2 = Pim1; Pim1 = Pi; Pi = P.mu[j] * Pim1;
        a.ng[l - 1].N = UV::hdup(P.nu[j] * Pim2 / Pi);
        a.ng[l - 1].G = UV::hdup(P.g[j] / Pi);
        a.iPi[l - 1] = (creal)(1.0 / Pi);
    }
    a.zero = 0;
    a.ustep = PC::U;
    a.PiK = (creal)Pi; a.PiKm1 = (creal)Pim1;
    a.last = last;
    a.nstrips = (G.np + PC::WOUT - 1) / PC::WOUT;
    const long ctas_x = ((long)a.nstrips * G.nr + PC::WARPS - 1) / PC::WARPS;   // per theta segment
    // theta segments: minimise waves x row-steps per segment (see sts_pipe_launch_impl)
    int nseg = 1;
    long best = -1;
    for (int n = 1; n <= 64 && (G.nt + 2) / n >= K; n++) {
        const long rows = (G.nt + 2 + n - 1) / n + 2 * K;
        const long waves = (ctas_x * n + slots - 1) / slots;
        if (best < 0 || waves * rows < best) { best = waves * rows; nseg = n; }
    }
    if (ctas_x > 0x7fffffffL) return -1;
    a.rows_per_seg = (G.nt + 2 + nseg - 1) / nseg;
    nseg = (G.nt + 2 + a.rows_per_seg - 1) / a.rows_per_seg;
    a.rows_per_seg_u = a.rows_per_seg;
    a.niter = (a.rows_per_seg + 2 * K + PC::U - 1) / PC::U;   // row-steps t0 .. t0 + rows_per_seg + 2K - 1 of every segment
    dim3 g((unsigned)ctas_x, nseg);
    bool armed = false;
    P.prof_begin(P.user, &armed);
    k_sts_upipe<real, creal, K, SPLIT><<<g, PC::WARPS * 32, smem, P.stream>>>(a, G);
    P.prof_end(P.user, armed, K);
    *launches += 2;
    return 0;
}

template <typename real, typename creal, int K>
int sts_upipe_launch(const StsBlockedPlan<real>& P, const UPipePlan& UP, Tables<real>& T, const Geom& G, int j0, const real* cur,
                     const real* prev, real* ocur, real* oprev, bool last, int64_t* launches) {
    if (G.np % UCfg<real, creal, K>::C == 0)
        return sts_upipe_launch_impl<real, creal, K, false>(P, UP, T, G, j0, cur, prev, ocur, oprev, last, launches);
    return sts_upipe_launch_impl<real, creal, K, true>(P, UP, T, G, j0, cur, prev, ocur, oprev, last, launches);
}

}  // namespace hft
