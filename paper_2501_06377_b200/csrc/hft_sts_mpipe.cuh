// hft_sts_mpipe.cuh -- temporally blocked super-time-stepping for a spatially varying diffusivity nu(theta, phi)
// (Eq. 27-28; reading U31): K = 4 STS stages per launch.
//
// With phi-dependent coefficients neither of the two things k_sts_pipe rests on holds: the coefficients of L are per cell,
// not per row, and the zonal mean no longer commutes with L, so the polar-cap values of a block cannot come from the
// zonal-mean recurrence (reading U21).  What replaces them (hard part 1):
//
//  * k_sts_mcapseq advances the POLAR BAND -- rows 0..K next to each pole, full phi extent: the exact dependency cone of the
//    K cap values of a block, about 1 % of the cells -- stage by stage inside one CTA per (pole, realization), with the
//    nu-weighted phi-sum of App. A (:646) taken after every stage in a fixed order, and hands the K cap values to
//  * k_sts_mpipe, the same pipeline as k_sts_pipe (a warp owns a strip of 32 C columns and streams down the rows, level l
//    lags level l-1 by one row, theta-neighbours in registers, phi-neighbours by shuffle, halo instead of exchange), which
//    treats rows 0 and nt+1 of every level as known.  The coefficients of Eq. 28 are carried as FACE CONDUCTANCES formed once
//    per row from the nu row that streams in beside the fields,
//        gt_{j+1/2,k} = (nu_{j+1/2,k+1/2} + nu_{j+1/2,k-1/2})/2 sin(theta_{j+1/2}) / dtheta_{j+1/2}     (theta-face below row j)
//        ge_{j,k+1/2} = (nu_{j+1/2,k+1/2} + nu_{j-1/2,k+1/2})/2                                        (phi-face east of cell j,k)
//    and kept in register windows of K+2 / K+1 rows, so that every level applies the operator in the difference form of Eq. 27
//        L = rt_j [gt_{j+1/2}(s - c) - gt_{j-1/2}(c - n)] + rp_j [ge_{k+1/2}(e - c) - ge_{k-1/2}(c - w)],
//        rt_j = 1/(sin(theta_j) dtheta_j), rp_j = 1/(sin^2(theta_j) dphi^2)
//    with 10 operations, and the recurrence delta_l = mu c + nu p2 + a L + g F with 4 more.
//
// Traffic per block: delta_{j0}, delta_{j0-1}, F, NU in, two levels out = 6 array passes per 4 stages, against 5 per stage for
// the one-launch-per-stage kernel (k_sts_stage_mapv<MAP = true>).  K = 4 is what the register file allows in fp64 with the
// two conductance windows beside the level windows.  Needs n_phi % C == 0.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "hft_sts_blocked.cuh"
#include "hft_sts_map.cuh"
#include "hft_sts_pipe.cuh"

namespace hft {

constexpr int MPIPE_K = 4;
constexpr int MPIPE_WARPS = 4;
constexpr int MCAP_THREADS = 1024;

template <typename real>
struct MPipeArgs {
    const real *cur, *prev, *F, *NU;   // level 0 = delta_{j0}, level -1 = delta_{j0-1}, L(Y0), nu on the half-half grid
    real *ocur, *oprev, *Y0;           // level K, level K-1; last block: Y0 += level K
    const double* capseq;              // [R][2][K] cap values of levels 1..K (k_sts_mcapseq)
    real mu[MPIPE_K], nu[MPIPE_K], a[MPIPE_K], g[MPIPE_K];
    int last, rows_per_seg, nstrips;
};

// ------------------------------------------------------------------ the polar band
// grid (2 poles, R), block MCAP_THREADS (the band is short and every stage ends in a CTA-wide barrier: the kernel is bound by
// the latency of its L2 round trips, so it takes the largest CTA).  Band row d = distance from the pole in rows (d = 0: the cap).  Three level buffers of
// (K+1) x n_phi doubles per (pole, realization) in global scratch (L2-resident: 120 KB at n_phi = 2048) rotate as
// level l-2 / l-1 / l; a CTA-wide barrier separates the stages (global writes of a CTA are visible to it after the barrier).
// All arithmetic in fp64 whatever the state type: the K values are boundary data for the main kernel.
template <typename real, int K>
__global__ void __launch_bounds__(MCAP_THREADS) k_sts_mcapseq(MPipeArgs<real> A, MapArgs<real> M, Tables<real> T, Geom G, double* scratch,
                                                     double* capseq) {
    __shared__ double red[32];
    __shared__ double s_cap[3];
    const int pole = blockIdx.x, r = blockIdx.y, nt = G.nt, np = G.np;
    const size_t base = (size_t)r * G.rstride;
    double* buf = scratch + ((size_t)r * 2 + pole) * 3 * (size_t)(K + 1) * np;
    auto lv = [&](int which) { return buf + (size_t)which * (K + 1) * np; };
    auto row_of = [&](int d) { return pole == 0 ? d : nt + 1 - d; };
    // level -1 -> buffer 0, level 0 -> buffer 1 (rows 0..K)
    for (int d = 0; d <= K; d++) {
        const size_t o = base + (size_t)row_of(d) * G.pitch;
        for (int k = threadIdx.x; k < np; k += blockDim.x) {
            lv(0)[(size_t)d * np + k] = (double)A.prev[o + k];
            lv(1)[(size_t)d * np + k] = (double)A.cur[o + k];
        }
    }
    __syncthreads();
    const real* nu = M.NU + base;
    const int face0 = pole == 0 ? 0 : nt;                 // the theta-face between the cap and its neighbour row
    for (int s = 1; s <= K; s++) {
        const double* p2 = lv((s - 1) % 3);               // level s-2
        const double* c1 = lv(s % 3);                     // level s-1
        double* out = lv((s + 1) % 3);                    // level s
        const double mu = (double)A.mu[s - 1], nuc = (double)A.nu[s - 1], a = (double)A.a[s - 1], g = (double)A.g[s - 1];
        // rows d = 1 .. K-s: Eq. 27 in difference form, the same expression as the main kernel
        for (int d = 1; d <= K - s; d++) {
            const int j = row_of(d);
            const int dn = pole == 0 ? d - 1 : d + 1, ds = pole == 0 ? d + 1 : d - 1;   // band rows of j-1 and j+1
            const double rt = (double)T.rdt[j], rp = (double)T.rdp[j] * (double)T.rdp[j];
            const double fs = (double)T.sth[j] * (double)T.rdf[j], fn = (double)T.sth[j - 1] * (double)T.rdf[j - 1];
            const real* nS = nu + (size_t)j * G.pitch;        // nu at face j+1/2
            const real* nN = nu + (size_t)(j - 1) * G.pitch;  // nu at face j-1/2
            const size_t oF = base + (size_t)j * G.pitch;
            for (int k = threadIdx.x; k < np; k += blockDim.x) {
                const int kw = k == 0 ? np - 1 : k - 1, ke = k == np - 1 ? 0 : k + 1;
                const double c = c1[(size_t)d * np + k];
                const double gts = 0.5 * ((double)nS[k] + (double)nS[kw]) * fs, gtn = 0.5 * ((double)nN[k] + (double)nN[kw]) * fn;
                const double gee = 0.5 * ((double)nS[k] + (double)nN[k]), gww = 0.5 * ((double)nS[kw] + (double)nN[kw]);
                const double L = rt * (gts * (c1[(size_t)ds * np + k] - c) - gtn * (c - c1[(size_t)dn * np + k])) +
                                 rp * (gee * (c1[(size_t)d * np + ke] - c) - gww * (c - c1[(size_t)d * np + kw]));
                out[(size_t)d * np + k] = mu * c + nuc * p2[(size_t)d * np + k] + a * L + g * (double)A.F[oF + k];
            }
        }
        // the cap (App. A :646 with the face-averaged nu): L_cap = capP (sum_k nu_k B[1,k] - (sum_k nu_k) B_cap)
        double part = 0.0;
        {
            const real* nf = nu + (size_t)face0 * G.pitch;
            for (int k = threadIdx.x; k < np; k += blockDim.x) {
                const int kw = k == 0 ? np - 1 : k - 1;
                part += 0.5 * ((double)nf[k] + (double)nf[kw]) * c1[(size_t)1 * np + k];
            }
        }
        const double S = block_sum(part, red);
        if (threadIdx.x == 0) {
            const double c0 = c1[0], Lc = M.capP[pole] * (S - M.capw[2 * r + pole] * c0);
            const double v = mu * c0 + nuc * p2[0] + a * Lc + g * (double)A.F[base + (size_t)row_of(0) * G.pitch];
            s_cap[0] = v;
            capseq[((size_t)r * 2 + pole) * K + (s - 1)] = v;
        }
        __syncthreads();
        const double capv = s_cap[0];
        for (int k = threadIdx.x; k < np; k += blockDim.x) out[k] = capv;   // band row 0, replicated like the field's cap row
        __syncthreads();
    }
}

// ------------------------------------------------------------------ the main kernel
template <typename real, int K>
struct MPipeCfg {
    static constexpr int C = 16 / (int)sizeof(real);
    static constexpr int HALO = (K + C - 1) / C * C;
    static constexpr int WOUT = 32 * C - 2 * HALO;
    // inputs arrive through a per-warp shared-memory ring filled by cp.async, DP rows ahead (as in k_sts_pipe: every lane
    // copies and later reads only its own 16 bytes); one row ahead in registers left the kernel waiting on DRAM latency
    static constexpr int DP = 6, D = DP + 1;
    static constexpr int WARP_BYTES = 4 * D * 32 * 16;     // cur, prev, F, NU
    // The row metric the operator needs -- 1/(sin(theta_j) dtheta_j), 1/(sin(theta_j) dphi)^2 per cell row, sin(theta) / dtheta per
    // theta-face -- for the rows of this CTA's theta segment sits in shared memory behind the rings, filled once per CTA.
    // (Fetched from the global tables where it is used -- 10 warp-uniform LDGs per row-step -- a quarter of all warp samples
    // were multiplies waiting for one of them: profiles/r02_blocked_kernels.md.)
    static constexpr int MTAB_ROWS = 1024;                 // >= rows per segment + 2 K + U + 1: the host picks the segments so
    static constexpr int MTAB_BYTES = MTAB_ROWS * 3 * (int)sizeof(real);
    static constexpr int SMEM_BYTES = MPIPE_WARPS * WARP_BYTES + MTAB_BYTES;
};

// Per-warp state.  Every register window ROTATES instead of moving (as in k_sts_pipe): the row loop is unrolled U = 6 times,
// row rho of a size-6 window (F, the two conductances) lives in slot rho mod 6, of a level window in slot rho mod 3, so all
// slot indices are compile-time constants of the phase PH = row-step mod 6.  (The first version shifted the windows: 96 register
// moves per row-step beside 112 floating-point operations.)
template <typename real, int K>
struct MPipeWarp {
    using P = MPipeCfg<real, K>;
    static constexpr int C = P::C, D = P::D, DP = P::DP, U = 6, SLOT = 32 * C, ARR = D * 32 * C;
    static_assert(K + 2 <= U, "window of K + 2 theta-face rows");
    real u[K][3][C];   // level l, row rho in slot rho mod 3
    real p[3][C];      // level -1 (delta_{j0-1})
    real f[U][C];      // F
    real gt[U][C];     // theta-face conductance of face rho + 1/2
    real ge[U][C];     // phi-face conductance east of cell (rho, q)
    real gw[U];        // ... and west of the lane's first column
    real nuN[C], nuNw; // nu at the previous row's south face, and its value west of the lane
    const MPipeArgs<real>& A;
    const Tables<real>& T;
    const real *gcur, *gprev, *gF, *gNU;    // this lane's columns of row 0
    real *gocur, *goprev, *gY0;
    real* ring;
    const real *mt2, *mtf;   // shared: {rdt_j, rdp_j^2} and sth rdf of row / face (index - first table row); mt2, mtf: row t
    const double *capN, *capS;
    int nt, pitch, ja, jb, slot;
    bool wr;

    __device__ __forceinline__ MPipeWarp(const MPipeArgs<real>& A_, const Tables<real>& T_) : A(A_), T(T_) {}

    __device__ __forceinline__ void prefetch(int row, int s) {
        if (row <= nt + 1) {
            const size_t off = (size_t)row * pitch;
            cp_async16(smem_u32(ring + s * SLOT), gcur + off);
            cp_async16(smem_u32(ring + ARR + s * SLOT), gprev + off);
            cp_async16(smem_u32(ring + 2 * ARR + s * SLOT), gF + off);
            if (row <= nt) cp_async16(smem_u32(ring + 3 * ARR + s * SLOT), gNU + off);
        }
        cp_async_commit();
    }

    // GEN = false: every level of this row-step works on an interior row (no branch on the row index: one basic block)
    template <int PH, bool GEN>
    __device__ __forceinline__ void rowstep(int t) {
        const unsigned full = 0xffffffffu;
        const real half = (real)0.5;
        cp_async_wait<DP - 1>();                              // this lane's copies of row t have landed
        __syncwarp();
        // row t arrives from the ring, row t + DP is requested into the slot of row t - 1
        real nuS[C];
        vload<real, C>(u[0][PH % 3], ring + slot * SLOT);
        vload<real, C>(p[PH % 3], ring + ARR + slot * SLOT);
        vload<real, C>(f[PH % U], ring + 2 * ARR + slot * SLOT);
        vload<real, C>(nuS, ring + 3 * ARR + slot * SLOT);
        {
            int ps = slot + DP;
            if (ps >= D) ps -= D;
            prefetch(t + DP, ps);
            if (++slot == D) slot = 0;
        }
        // conductances of row t: face t+1/2 (rows 0..nt) and the phi-faces of cell row t (rows 1..nt)
        const real nuSw = __shfl_up_sync(full, nuS[C - 1], 1);
        {
            const real fs = mtf[0];
#pragma unroll
            for (int q = 0; q < C; q++) {
                const real w = q == 0 ? nuSw : nuS[q > 0 ? q - 1 : 0];
                gt[PH % U][q] = half * (nuS[q] + w) * fs;
                ge[PH % U][q] = half * (nuS[q] + nuN[q]);
            }
            gw[PH % U] = half * (nuSw + nuNw);
        }
#pragma unroll
        for (int q = 0; q < C; q++) nuN[q] = nuS[q];
        nuNw = nuSw;

        real outK[C];
#pragma unroll
        for (int q = 0; q < C; q++) outK[q] = (real)0;
        // levels 1..K: level l computes its row j = t - l from level l-1 rows j-1, j, j+1
#pragma unroll
        for (int l = 1; l <= K; l++) {
            const int j = t - l;
            constexpr int dummy = 0; (void)dummy;
            const int sN = pmod(PH - (l - 1), 3), sC = pmod(PH - l, 3), sO = pmod(PH - l - 1, 3);   // level l-1: rows j+1, j, j-1
            const int wS = pmod(PH - l, U), wN = pmod(PH - l - 1, U);                               // size-6 windows: rows j, j-1
            real res[C];
            if (!GEN || (j >= 1 && j <= nt)) {
                real m2[2];
                vload<real, 2>(m2, mt2 - 2 * l);
                const real rt = m2[0], rp = m2[1];
                const real cmu = A.mu[l - 1], cnu = A.nu[l - 1], ca = A.a[l - 1], cg = A.g[l - 1];
                const real west = __shfl_up_sync(full, u[l - 1][sC][C - 1], 1);
                const real east = __shfl_down_sync(full, u[l - 1][sC][0], 1);
#pragma unroll
                for (int q = 0; q < C; q++) {
                    const real c = u[l - 1][sC][q];
                    const real w = (q == 0) ? west : u[l - 1][sC][q > 0 ? q - 1 : 0];
                    const real e = (q == C - 1) ? east : u[l - 1][sC][q < C - 1 ? q + 1 : 0];
                    const real gww = (q == 0) ? gw[wS] : ge[wS][q > 0 ? q - 1 : 0];
                    const real p2 = (l >= 2) ? u[(l >= 2) ? l - 2 : 0][sC][q] : p[pmod(PH - 1, 3)][q];   // level l-2 row j: ITS oldest
                    const real tth = gt[wS][q] * (u[l - 1][sN][q] - c) - gt[wN][q] * (c - u[l - 1][sO][q]);
                    const real tph = ge[wS][q] * (e - c) - gww * (c - w);
                    const real L = rt * tth + rp * tph;
                    res[q] = cmu * c + cnu * p2 + ca * L + cg * f[wS][q];
                }
            } else if (j == 0 || j == nt + 1) {
                const real cv = (real)(j == 0 ? capN[l - 1] : capS[l - 1]);
#pragma unroll
                for (int q = 0; q < C; q++) res[q] = cv;
            } else {
#pragma unroll
                for (int q = 0; q < C; q++) res[q] = (real)0;
            }
            if (l < K) {
#pragma unroll
                for (int q = 0; q < C; q++) u[(l < K) ? l : 0][sC][q] = res[q];   // level l row j: slot j mod 3 = sC
            } else {
#pragma unroll
                for (int q = 0; q < C; q++) outK[q] = res[q];
            }
        }
        // row jo = t - K of levels K and K-1 (level K-1 row t-K is its centre: slot (PH-(K-1)-1) mod 3)
        const int jo = t - K;
        if (wr && jo >= ja && jo < jb) {
            const size_t off = (size_t)jo * pitch;
            if (A.last) {
                real y[C];
                vload<real, C>(y, gY0 + off);
#pragma unroll
                for (int q = 0; q < C; q++) y[q] += outK[q];
                vstore<real, C>(gY0 + off, y);
            } else {
                vstore<real, C>(gocur + off, outK);
                vstore<real, C>(goprev + off, u[K - 1][pmod(PH - K, 3)]);
            }
        }
        mt2 += 2; mtf += 1;
    }

    template <int PH, bool GEN>
    __device__ __forceinline__ void macro(int tb) {
        rowstep<PH, GEN>(tb + PH);
        if constexpr (PH + 1 < U) macro<PH + 1, GEN>(tb);
    }
};

template <typename real, int K>
__global__ void __launch_bounds__(MPIPE_WARPS * 32, sizeof(real) == 8 ? 2 : 3)
k_sts_mpipe(const __grid_constant__ MPipeArgs<real> A, const __grid_constant__ Tables<real> T, Geom G) {
    using P = MPipeCfg<real, K>;
    constexpr int C = P::C, D = P::D, DP = P::DP;
    extern __shared__ __align__(128) unsigned char mpipe_smem[];
    const int lane = threadIdx.x & 31;
    const int nt = G.nt, np = G.np;
    MPipeWarp<real, K> W(A, T);
    W.nt = nt; W.pitch = G.pitch;
    W.ja = blockIdx.y * A.rows_per_seg; W.jb = min(W.ja + A.rows_per_seg, nt + 2);   // output rows [ja, jb)
    const int t0 = max(W.ja - K, 0), tend = W.jb - 1 + K;
    {   // metric table of rows t0 - K .. tend + 5 (the last row-step of the 6-fold unrolled loop), by the whole CTA
        real* mt = reinterpret_cast<real*>(mpipe_smem + MPIPE_WARPS * P::WARP_BYTES);
        const int jlo = t0 - K, n = tend + 6 - jlo;
        for (int i = threadIdx.x; i < n; i += blockDim.x) {
            const int j = jlo + i, tf = min(max(j, 0), nt);
            const bool in = j >= 1 && j <= nt;
            mt[2 * i] = in ? T.rdt[j] : (real)0;
            mt[2 * i + 1] = in ? T.rdp[j] * T.rdp[j] : (real)0;
            mt[2 * P::MTAB_ROWS + i] = T.sth[tf] * T.rdf[tf];
        }
        W.mt2 = mt + 2 * K; W.mtf = mt + 2 * P::MTAB_ROWS + K;   // row t0
    }
    __syncthreads();                                          // the only block-level barrier, before any warp leaves
    // a warp's work item: (realization, strip) of this CTA's theta segment, strips fastest -- the items of all realizations are
    // dealt to the CTAs as one list, so that only the last CTA of a segment can have idle warps (with one CTA row per
    // realization 2 of 20 (fp32) / 3 of 40 (fp64) warp slots of cfg 3 stayed empty)
    const int item = blockIdx.x * MPIPE_WARPS + (threadIdx.x >> 5);
    if (item >= A.nstrips * G.nr) return;                     // warp-uniform
    const int r = item / A.nstrips, strip = item - r * A.nstrips;
    const int uc = strip * P::WOUT - P::HALO + lane * C;      // unwrapped first column of this lane
    int col = uc % np;
    if (col < 0) col += np;                                   // n_phi % C == 0: the C columns never straddle the seam
    W.wr = (lane * C >= P::HALO) && (lane * C < P::HALO + P::WOUT) && (uc < np);
    const size_t base = (size_t)r * G.rstride + col;
    W.gcur = A.cur + base; W.gprev = A.prev + base; W.gF = A.F + base; W.gNU = A.NU + base;
    W.gocur = A.ocur + base; W.goprev = A.oprev + base; W.gY0 = A.Y0 + base;
    W.capN = A.capseq + ((size_t)r * 2 + 0) * K;
    W.capS = A.capseq + ((size_t)r * 2 + 1) * K;
#pragma unroll
    for (int q = 0; q < C; q++) {
#pragma unroll
        for (int l = 0; l < K; l++) { W.u[l][0][q] = W.u[l][1][q] = W.u[l][2][q] = (real)0; }
        W.p[0][q] = W.p[1][q] = W.p[2][q] = (real)0;
#pragma unroll
        for (int i = 0; i < 6; i++) { W.f[i][q] = (real)0; W.ge[i][q] = (real)0; W.gt[i][q] = (real)0; }
        W.nuN[q] = (real)0;
    }
#pragma unroll
    for (int i = 0; i < 6; i++) W.gw[i] = (real)0;
    W.nuNw = (real)0;
    if (t0 > 0) {   // nu at the face above the first streamed row
        vload<real, C>(W.nuN, W.gNU + (size_t)(t0 - 1) * G.pitch);
        W.nuNw = __shfl_up_sync(0xffffffffu, W.nuN[C - 1], 1);
    }
    W.ring = reinterpret_cast<real*>(mpipe_smem + (size_t)(threadIdx.x >> 5) * P::WARP_BYTES) + lane * C;   // this lane's 16 bytes
    for (int i = 0; i < 4 * D; i++) vstore<real, C>(W.ring + i * 32 * C, W.nuN);   // a defined ring (the NU slot of row nt+1 is read)
    __syncwarp();
    for (int i = 0; i < DP; i++) W.prefetch(t0 + i, i);
    W.slot = 0;                                               // ring slot of row t
    for (int tb = t0; tb <= tend; tb += 6) {                  // (row-steps past tend load and store nothing)
        if (tb - K >= 1 && tb + 5 - 1 <= nt) W.template macro<0, false>(tb);   // levels 1..K of row-steps tb..tb+5: rows tb-K .. tb+4
        else W.template macro<0, true>(tb);
    }
    cp_async_wait<0>();
}

// ------------------------------------------------------------------ host side

inline bool sts_mblocked_supported(const Geom& G, size_t wbytes) {
    const int C = wbytes == 8 ? 2 : 4;
    return G.np % C == 0 && G.np >= 32 * C && G.nt >= 4 * MPIPE_K;
}
inline size_t sts_mscratch_bytes(const Geom& G) { return (size_t)G.nr * 2 * 3 * (MPIPE_K + 1) * G.np * sizeof(double); }

template <typename real>
int sts_mpipe_launch(const StsBlockedPlan<real>& P, MapArgs<real>& M, Tables<real>& T, const Geom& G, double* scratch, int j0,
                     const real* cur, const real* prev, real* ocur, real* oprev, bool last, int64_t* launches) {
    constexpr int K = MPIPE_K;
    using PC = MPipeCfg<real, K>;
    const int smem = PC::SMEM_BYTES;
    const int slots = resident_ctas(k_sts_mpipe<real, K>, MPIPE_WARPS * 32, smem);
    if (slots < 1) return -1;
    MPipeArgs<real> a;
    a.cur = cur; a.prev = prev; a.F = P.buf[0]; a.NU = M.NU; a.ocur = ocur; a.oprev = oprev; a.Y0 = P.Y0; a.capseq = P.capseq;
    for (int i = 0; i < K; i++) {
        a.mu[i] = (real)P.mu[j0 + 1 + i]; a.nu[i] = (real)P.nu[j0 + 1 + i];
        a.a[i] = (real)P.a[j0 + 1 + i]; a.g[i] = (real)P.g[j0 + 1 + i];
    }
    a.last = last;
    a.nstrips = (G.np + PC::WOUT - 1) / PC::WOUT;
    const long ctas_x = ((long)a.nstrips * G.nr + MPIPE_WARPS - 1) / MPIPE_WARPS;   // per theta segment
    int nseg = 1;
    long best = -1;
    for (int n = 1; n <= 128 && (G.nt + 2) / n >= K; n++) {   // theta segments: minimise waves x row-steps per segment
        const long rows = (G.nt + 2 + n - 1) / n + 2 * K;
        if (rows + K + 8 > PC::MTAB_ROWS) continue;             // the segment's metric table has to fit its shared-memory slot
        const long waves = (ctas_x * n + slots - 1) / slots;
        if (best < 0 || waves * rows < best) { best = waves * rows; nseg = n; }
    }
    if (best < 0 || ctas_x > 0x7fffffffL) return -1;
    a.rows_per_seg = (G.nt + 2 + nseg - 1) / nseg;
    nseg = (G.nt + 2 + a.rows_per_seg - 1) / a.rows_per_seg;
    dim3 gc(2, G.nr), g((unsigned)ctas_x, nseg);
    k_sts_mcapseq<real, K><<<gc, MCAP_THREADS, 0, P.stream>>>(a, M, T, G, scratch, P.capseq);
    bool armed = false;
    P.prof_begin(P.user, &armed);
    k_sts_mpipe<real, K><<<g, MPIPE_WARPS * 32, smem, P.stream>>>(a, T, G);
    P.prof_end(P.user, armed, K);
    *launches += 2;
    return 0;
}

// One STS step with nu(theta, phi): stage 1 and the (s-1) mod K remainder stages one launch each (k_sts_stage_mapv<MAP = true>),
// then (s-1)/K blocks of K stages.  M.nparts_in / the polar partials are used by the un-blocked stages only.
template <typename real>
int sts_mblocked_step(StsBlockedPlan<real>& P, MapArgs<real>& M, Tables<real>& T, const Geom& G, double* scratch, int64_t* launches) {
    constexpr int K = MPIPE_K;
    constexpr int CV = 16 / (int)sizeof(real);
    const int s = P.s;
    real* b[4] = {P.buf[1], P.buf[2], P.buf[3], P.buf[4]};
    const int nbxv = (G.np / CV + TX - 1) / TX;
    dim3 g1(nbxv, (G.nt + 2 + MAPV_RPT - 1) / MAPV_RPT, G.nr), gs(G.nbx, 2, G.nr);
    k_polar_row_sums_map<real><<<gs, TX, 0, P.stream>>>(P.Y0, M.NU, P.part[0], G);
    M.nparts_in = G.nbx;
    StsArgs<real> a;
    a.F = P.buf[0]; a.Y0 = P.Y0; a.mu = 0; a.nu = 0; a.g = 0; a.use_d2 = 0;
    a.in = P.Y0; a.d2 = b[0]; a.part_in = P.part[0]; a.part_out = P.part[1]; a.a = (real)P.a[1];
    k_sts_stage_mapv<real, 0, true><<<g1, TX, 0, P.stream>>>(a, M, T, G);
    M.nparts_in = nbxv;
    *launches += 2;
    const int rem = (s - 1) % K;
    int icur = 0, iprev = 1, pin = 1;
    bool has_prev = false;
    for (int j = 2; j <= 1 + rem; j++) {
        a.in = b[icur]; a.d2 = b[iprev]; a.part_in = P.part[pin]; a.part_out = P.part[pin ^ 1];
        a.mu = (real)P.mu[j]; a.nu = (real)P.nu[j]; a.a = (real)P.a[j]; a.g = (real)P.g[j];
        a.use_d2 = has_prev;
        k_sts_stage_mapv<real, 1, true><<<g1, TX, 0, P.stream>>>(a, M, T, G);
        *launches += 1;
        int t = icur; icur = iprev; iprev = t;
        has_prev = true;
        pin ^= 1;
    }
    for (int j0 = 1 + rem; j0 < s; j0 += K) {
        int o1 = -1, o2 = -1;
        for (int q = 0; q < 4; q++)
            if (q != icur && q != iprev) { if (o1 < 0) o1 = q; else o2 = q; }
        if (!has_prev) {   // delta_0 = 0 is not stored: the blocked kernel reads it, so write it once
            if (cudaMemsetAsync(b[iprev], 0, (size_t)G.nr * G.rstride * sizeof(real), P.stream) != cudaSuccess) return -1;
            has_prev = true;
        }
        const int rc = sts_mpipe_launch<real>(P, M, T, G, scratch, j0, b[icur], b[iprev], b[o1], b[o2], j0 + K == s, launches);
        if (rc != 0) return rc;
        icur = o1; iprev = o2;
    }
    return 0;
}

}  // namespace hft
