// hft_kernels.cuh -- sm_100a kernels of the HipFT time-stepping hot path (baseline, one launch per stage).
//
// Layout: a field is [R][nt+2][pitch] of `real`; row 0 / row nt+1 are the north /
// south polar caps (one value each, stored replicated over the nphi columns so that the theta-stencil of
// rows 1 and nt is uniform); columns [nphi, pitch) are padding and are never read.  phi is contiguous:
// a warp reads 32 consecutive columns of one row (coalesced 128/256 B).  Periodic phi is an index wrap.
// All per-row coefficients are phi-independent and come from small tables (broadcast loads).
//
// Citations are to /root/reference/PAPER.md (the extracted paper text), as in include/hft.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace hft {

constexpr int TX = 128;  // threads per CTA = columns per CTA (one column per thread)
// Advection stage kernels: a warp owns 31 output columns; lane 31 computes only the phi-face flux of the column after them, so
// that every lane finds the flux of its EAST face in the lane to its right: each phi-face WENO value is evaluated once
// instead of twice (the kernels are bound by that arithmetic, not by memory)
constexpr int ADV_COLS = (TX / 32) * 31;
constexpr int RPT = 8;   // rows per thread (column strip streamed in registers)

template <typename real>
struct Tables {            // device pointers, all [R][nt+2] unless noted
    const real* cp;        // diffusion: nu sin(theta_{j+1/2}) / (sin(theta_j) dth^2)        Eq. 28 (:456)
    const real* cm;        //            nu sin(theta_{j-1/2}) / (sin(theta_j) dth^2)        Eq. 28 (:452)
    const real* cf;        //            nu / (sin^2(theta_j) dph^2)                         Eq. 28 (:450, :458)
    const real* cd;        //            cp + cm + 2 cf  (minus the diagonal a_{j,k} of Eq. 28, :454)
    const real* c4;        // [R][nt+2][4] = (cm, cp, cf, cd) interleaved, zero on the cap rows (k_sts_pipe)
    const double* capc;    // [R][2] P (nu_face/dth) dph, north / south polar cap diffusion prefactor   App. A (:646)
    const real* lm;        // advection LLF: (v_{j-1/2} + alpha_j)/2                         B2 (:684)
    const real* lp;        //                (v_{j+1/2} - alpha_j)/2
    const real* vtf;       // [R][nt+1] v_theta at theta-faces (upwind faces)                Eq. 4 (:84)
    const real* pm;        // phi LLF: (v_phi + |v_phi|)/2 per row                           B2 with alpha = |v_phi|
    const real* pp;        //          (v_phi - |v_phi|)/2 per row
    const real* sth;       // [nt+1] sin(theta_{j+1/2})                                      :354
    const real* rdt;       // [nt+2] 1/(sin(theta_j) dth)
    const real* rdp;       // [nt+2] 1/(sin(theta_j) dph)
    const double* dA;      // [nt+2] quadrature weights: sin(theta_j) dth_j dph; caps: A_pole   :225-230, App. A
    const real* rdf;       // [nt+1] 1 / (theta_{j+1} - theta_j): node spacing across theta-face j+1/2      Eq. 27
    const real* wmp;       // [nt+1][16] per theta-face: App. B D-factors of u^- (0..4), eps_w (5), of u^+ (8..12)   :662-680
    const double* th;      // [nt+2] theta_j
    double adv_capc[2];    // P dph, north / south cap                                       App. A (:646)
    int nonuniform;        // 0: uniform theta grid -- the WENO constants are 1/2, 1/3, 2/3 and eps_w = eps_t
    real eps_t, eps_p;     // WENO3-CS(h) eps_w = dth, dph                                    :670
};

struct Geom {
    int nt, np, pitch, nr;
    size_t rstride;  // (nt+2)*pitch
    int nbx;         // ceil(np / TX): CTAs along phi == number of polar partial sums per row
    int nbxa;        // ceil(np / ADV_COLS): the same for the advection stage kernels
};

// ------------------------------------------------------------------ reductions (fixed order => deterministic)

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the CTA (blockDim.x multiple of 32, <= 1024); result valid in thread 0.
__device__ __forceinline__ double block_sum(double v, double* smem /*[32]*/) {
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) smem[w] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < nw; i++) t += smem[i];
    return t;
}

// Sum of the nbx per-CTA partials of one polar row, in index order (every caller gets the same bits).
__device__ __forceinline__ double sum_partials(const double* p, int nbx) {
    double s = 0.0;
    for (int i = 0; i < nbx; i++) s += p[i];
    return s;
}

// ------------------------------------------------------------------ diffusion / STS (one stage per launch)

template <typename real>
struct StsArgs {
    const real* in;   // field whose L is taken: Y0 (MODE 0) or delta_{j-1}
    real* d2;         // MODE 0: out delta_1.  MODE 1/2: in delta_{j-2}, out delta_j (same element, same thread)
    real* F;          // L(Y0): written in MODE 0, read otherwise
    real* Y0;         // MODE 2: Y0 += delta_s
    const double* part_in;   // [R][2][nbx] phi-sums of rows 1 and nt of `in`
    double* part_out;        // same for the field written to d2
    real mu, nu, a, g;       // stage scalars: mu_j, nu_j, mut_j dt, mut_j b_{j-1} dt (MODE 0: a = mut_1 dt)
    int use_d2;              // 0 on stage 2 (delta_0 = 0 is not stored)
};

// MODE 0: F = L(Y0), delta_1 = a F.   MODE 1: delta_j = mu d1 + nu d2 + a L(d1) + g F.
// MODE 2: MODE 1, then Y0 += delta_j (last stage).  MODE 3: explicit Euler, Y0 += a L(Y0) (in = Y0, out d2 = new Y).
// Row A5/A6 of SURVEY.md section 8: Eq. 27-28 (:438-460) with constant nu; caps per App. A (:624-648):
// L_cap = P (nu/dth) dph sum_k (B[1,k] - B[0]).
template <typename real, int MODE>
__global__ void __launch_bounds__(TX) k_sts_stage(StsArgs<real> A, Tables<real> T, Geom G) {
    __shared__ double red[32];
    const int r = blockIdx.z;
    const int k = blockIdx.x * TX + threadIdx.x;
    const bool live = k < G.np;
    const int kk = live ? k : 0;
    const int kw = (kk == 0) ? G.np - 1 : kk - 1;
    const int ke = (kk == G.np - 1) ? 0 : kk + 1;
    const int j0 = blockIdx.y * RPT;
    const int j1 = min(j0 + RPT, G.nt + 2);
    const size_t base = (size_t)r * G.rstride;
    const real* in = A.in + base;
    const real* cp = T.cp + (size_t)r * (G.nt + 2);
    const real* cm = T.cm + (size_t)r * (G.nt + 2);
    const real* cf = T.cf + (size_t)r * (G.nt + 2);

    real n = (j0 > 0) ? in[(size_t)(j0 - 1) * G.pitch + kk] : (real)0;
    real c = in[(size_t)j0 * G.pitch + kk];
    double sumN = 0.0, sumS = 0.0;  // this thread's contribution to the phi-sums of output rows 1 and nt
    for (int j = j0; j < j1; j++) {
        const size_t off = base + (size_t)j * G.pitch + kk;
        real s = (j < G.nt + 1) ? in[(size_t)(j + 1) * G.pitch + kk] : (real)0;
        real L;
        if (j == 0 || j == G.nt + 1) {
            const int pole = (j == 0) ? 0 : 1;
            double S = sum_partials(A.part_in + ((size_t)r * 2 + pole) * G.nbx, G.nbx);
            L = (real)(T.capc[2 * r + pole] * (S - (double)G.np * (double)c));
        } else {
            real w = in[(size_t)j * G.pitch + kw], e = in[(size_t)j * G.pitch + ke];
            L = cp[j] * (s - c) - cm[j] * (c - n) + cf[j] * ((e - (real)2 * c) + w);
        }
        real out;
        if (MODE == 0) {
            out = A.a * L;
            if (live) A.F[off] = L;
        } else if (MODE == 3) {
            out = c + A.a * L;
        } else {
            real d2v = A.use_d2 ? A.d2[off] : (real)0;
            out = A.mu * c + A.nu * d2v + A.a * L + A.g * A.F[off];
        }
        if (live) {
            if (MODE == 2) A.Y0[off] += out;   // Y_s = Y_0 + delta_s; delta_s itself is not needed again
            else A.d2[off] = out;
        }
        if (j == 1) sumN = live ? (double)out : 0.0;
        if (j == G.nt) sumS = live ? (double)out : 0.0;
        n = c;
        c = s;
    }
    // phi-sums of the rows adjacent to the caps, for the next stage's cap update (block-uniform branches)
    if (j0 <= 1 && 1 < j1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part_out[((size_t)r * 2 + 0) * G.nbx + blockIdx.x] = t;
    }
    if (j0 <= G.nt && G.nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part_out[((size_t)r * 2 + 1) * G.nbx + blockIdx.x] = t;
    }
}

// phi-sums of rows 1 and nt of a field -> partials (same format as the stage kernels write).
template <typename real>
__global__ void __launch_bounds__(TX) k_polar_row_sums(const real* f, double* part, Geom G) {
    __shared__ double red[32];
    const int r = blockIdx.z, pole = blockIdx.y;
    const int k = blockIdx.x * TX + threadIdx.x;
    const int j = pole == 0 ? 1 : G.nt;
    double v = (k < G.np) ? (double)f[(size_t)r * G.rstride + (size_t)j * G.pitch + k] : 0.0;
    double t = block_sum(v, red);
    if (threadIdx.x == 0) part[((size_t)r * 2 + pole) * G.nbx + blockIdx.x] = t;
}

// ------------------------------------------------------------------ advection (one SSPRK stage per launch)

// WENO3-CS(h) one-sided face value (App. B :658-676, uniform grid: D = 1/2, 1/3, 2/3), written with one
// division: u = (d0 p0 (eps+b1)^2 + d1 p1 (eps+b0)^2) / (d0 (eps+b1)^2 + d1 (eps+b0)^2).
// num / den for den > 0 (a sum of squares here): hardware reciprocal seed (~20 bits), ONE Newton step (r = (1 + e) / den with
// |e| ~ 2^-40), the quotient q = num r, and one residual correction q + r (num - den q), whose error is e^2 ~ 2^-80 before the
// final rounding: within about an ulp of the IEEE quotient without the slow path of the correctly rounded division (the WENO
// weights need 3 to 4 of these per cell and stage; the division was the largest single cost of the stage kernel).  A second
// Newton step, as round 1 had it, changes nothing but the instruction count (measured on the B200: seed error 2^-19.9; 2e8
// random quotients over 200 binades all equal to the IEEE quotient).
__device__ __forceinline__ double pos_div(double num, double den) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(den));
    r = fma(fma(-den, r, 1.0), r, r);
    const double q = num * r;
    return fma(fma(-den, q, num), r, q);
}
__device__ __forceinline__ float pos_div(float num, float den) { return __fdividef(num, den); }

template <typename real>
__device__ __forceinline__ real weno3_side(real far, real near, real other, real eps) {
    real p0 = (real)1.5 * near - (real)0.5 * far;
    real p1 = (real)0.5 * (near + other);
    real q0 = near - far, q1 = other - near;
    real e0 = eps + q0 * q0, e1 = eps + q1 * q1;
    real a0 = e1 * e1;               // proportional to w0 = (1/3)/e0^2   (times e0^2 e1^2 * 3)
    real a1 = (real)2 * (e0 * e0);   // proportional to w1 = (2/3)/e1^2
    return pos_div(a0 * p0 + a1 * p1, a0 + a1);
}

// The same on a non-uniform grid, App. B (:662-680): D = (Dex, Da, Db, d0, d1) of this face and side (Tables::wmp).
//   p0 = (1 + Dex) near - Dex far, p1 = Da near + Db other, beta0 = 4 (Dex (near - far))^2, beta1 = 4 (Db (other - near))^2,
//   w0 = d0 / (eps + beta0)^2, w1 = d1 / (eps + beta1)^2; one division: multiply through by (eps+beta0)^2 (eps+beta1)^2.
template <typename real>
__device__ __forceinline__ real weno3_side_nu(real far, real near, real other, real eps, const real* D) {
    const real Dex = D[0], Da = D[1], Db = D[2], d0 = D[3], d1 = D[4];
    real p0 = near + Dex * (near - far);
    real p1 = Da * near + Db * other;
    real q0 = (real)2 * Dex * (near - far), q1 = (real)2 * Db * (other - near);
    real e0 = eps + q0 * q0, e1 = eps + q1 * q1;
    real a0 = d0 * (e1 * e1);
    real a1 = d1 * (e0 * e0);
    return pos_div(a0 * p0 + a1 * p1, a0 + a1);
}

template <typename real>
__device__ __forceinline__ real upwind(real v, real bm, real bp) {
    return v > (real)0 ? v * bm : (v < (real)0 ? v * bp : (real)0);
}

template <typename real>
struct AdvArgs {
    const real* in;   // f^(m-1)
    const real* fn;   // f^n (read only if ca != 0)
    real* out;        // f^(m) = ca f^n + cb f^(m-1) - cdt F_A(f^(m-1))      Eq. 25 (:418-424)
    double* part;     // [R][2][nbx] phi-sums of the theta-flux at the faces next to the caps
    real ca, cb, cdt;
    int upwind_only;  // adv_flux == 1
    // flow attenuation (Eq. 5 :100), k_adv_stage_att only: field-shaped arrays [R][nt+2][pitch]
    const real* VT;   // attenuated v_theta at face j+1/2 (row j = 0..nt)
    const real* VP;   // attenuated v_phi at face k-1/2 (rows 1..nt)
    const real *LMt, *LPt;   // theta LLF half-speeds of cell (j,k): (v_{j-1/2} + alpha)/2, (v_{j+1/2} - alpha)/2
    const real *LMp, *LPp;   // phi   LLF half-speeds of cell (j,k): (v_{k-1/2} + alpha)/2, (v_{k+1/2} - alpha)/2
    int nparts;              // CTAs along phi of the stage kernel = partial sums per (realization, pole) in `part`
    int rpt;                 // k_adv_stage_u / k_adv_stage_att_u: rows per thread, <= ADV_RPT (fewer on small batches: more CTAs)
};

// theta-face flux at face f (between rows f and f+1) from rows f-1, f, f+1, f+2 of one column.
// Faces 1/2, 3/2, nt-1/2, nt+1/2 (f <= 1 or f >= nt-1) are upwind (:388); the others WENO3-CS(h) with LLF (B2).
template <typename real>
__device__ __forceinline__ real theta_face_flux(int f, real bm1, real b0, real bp1, real bp2, const real* lm,
                                                const real* lp, const real* vtf, int nt, real eps, int upwind_only,
                                                const real* wmp /* null: uniform grid */) {
    if (upwind_only || f <= 1 || f >= nt - 1) return upwind(vtf[f], b0, bp1);
    if (wmp) {   // non-uniform theta grid: this face's D-factors and eps_w = its node spacing
        const real* D = wmp + 16 * (size_t)f;
        return weno3_side_nu(bp2 * lp[f + 2], bp1 * lp[f + 1], b0 * lp[f], D[5], D + 8) +
               weno3_side_nu(bm1 * lm[f - 1], b0 * lm[f], bp1 * lm[f + 1], D[5], D);
    }
    real um = weno3_side(bm1 * lm[f - 1], b0 * lm[f], bp1 * lm[f + 1], eps);   // right-moving part, from LM
    real up = weno3_side(bp2 * lp[f + 2], bp1 * lp[f + 1], b0 * lp[f], eps);   // left-moving part, from LP
    return up + um;
}

// phi-face flux at face k-1/2 of a row with uniform speed: LM = pm B, LP = pp B; one of pm, pp is exactly 0
// and its one-sided value is exactly 0 (reading U13), so only the live side is evaluated.
template <typename real>
__device__ __forceinline__ real phi_face_flux(real bm2, real bm1, real b0, real bp1, real pm, real pp, real eps,
                                              int upwind_only) {
    if (upwind_only) return pm * bm1 + pp * b0;   // v>0: v B_{k-1}; v<0: v B_k; v=0: 0
    if (pp == (real)0) return weno3_side(pm * bm2, pm * bm1, pm * b0, eps);
    return weno3_side(pp * bp1, pp * b0, pp * bm1, eps);
}

template <typename real>
__global__ void __launch_bounds__(TX) k_adv_stage(AdvArgs<real> A, Tables<real> T, Geom G) {
    __shared__ double red[32];
    const int r = blockIdx.z;
    const int lane = threadIdx.x & 31;
    const int k = (blockIdx.x * (TX / 32) + (threadIdx.x >> 5)) * 31 + lane;   // lane 31: the first column of the next warp
    const int np = G.np, nt = G.nt;
    const bool live = lane < 31 && k < np;          // this lane writes column k
    const int k0 = k % np;
    const int km1 = (k0 + np - 1) % np, km2 = (k0 + np - 2) % np, kp1 = (k0 + 1) % np;
    const int j0 = 1 + blockIdx.y * RPT;            // rows 1..nt only; caps are done by k_adv_caps
    const int j1 = min(j0 + RPT, nt + 1);
    const size_t base = (size_t)r * G.rstride;
    const real* in = A.in + base;
    const real* lm = T.lm + (size_t)r * (nt + 2);
    const real* lp = T.lp + (size_t)r * (nt + 2);
    const real* vtf = T.vtf + (size_t)r * (nt + 1);
    const real* pm = T.pm + (size_t)r * (nt + 2);
    const real* pp = T.pp + (size_t)r * (nt + 2);
    auto ld = [&](int j) -> real { return in[(size_t)min(max(j, 0), nt + 1) * G.pitch + k0]; };

    real w0 = ld(j0 - 2), w1 = ld(j0 - 1), w2 = ld(j0), w3 = ld(j0 + 1);
    const real* wmp = T.nonuniform ? T.wmp : nullptr;
    real Fn = theta_face_flux<real>(j0 - 1, w0, w1, w2, w3, lm, lp, vtf, nt, T.eps_t, A.upwind_only, wmp);
    double sumN = 0.0, sumS = 0.0;
    if (j0 == 1) sumN = live ? (double)Fn : 0.0;
    for (int j = j0; j < j1; j++) {
        real w4 = ld(j + 2);
        real Fs = theta_face_flux<real>(j, w1, w2, w3, w4, lm, lp, vtf, nt, T.eps_t, A.upwind_only, wmp);
        const real* row = in + (size_t)j * G.pitch;
        real bm2 = row[km2], bm1 = row[km1], bp1 = row[kp1];
        real Fw = phi_face_flux<real>(bm2, bm1, w2, bp1, pm[j], pp[j], T.eps_p, A.upwind_only);
        real Fe = __shfl_down_sync(0xffffffffu, Fw, 1);   // face k+1/2 = the west face of column k+1 (same operands, same bits)
        real tend = (T.sth[j] * Fs - T.sth[j - 1] * Fn) * T.rdt[j] + (Fe - Fw) * T.rdp[j];
        const size_t off = base + (size_t)j * G.pitch + k0;
        real o = A.cb * w2 - A.cdt * tend;
        if (A.ca != (real)0) o = A.ca * A.fn[off] + o;
        if (live) A.out[off] = o;
        if (j == nt) sumS = live ? (double)Fs : 0.0;
        Fn = Fs;
        w0 = w1; w1 = w2; w2 = w3; w3 = w4;
    }
    if (j0 == 1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 0) * A.nparts + blockIdx.x] = t;
    }
    if (j0 <= nt && nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 1) * A.nparts + blockIdx.x] = t;
    }
}

// k_adv_stage on a uniform theta grid with WENO3 fluxes, every shared quantity of the theta sweep evaluated once per row: the
// LLF products A_j = B_j lm_j, P_j = B_j lp_j, their row differences and the smoothness terms (eps + d^2)^2 are each used
// by two neighbouring faces, so they move through register windows (k_adv_stage forms three products, two differences and
// two smoothness terms per face and side).  Row pointers advance by the pitch; the per-row tables are read one new entry
// per row.  ADV_RPT rows per thread: the first face of a thread's strip is the one face it evaluates without writing a row.
// Face f (between rows f and f+1), App. B with D = 1/2, 1/3, 2/3 (weno3_side):
//   right-moving part from (A_{f-1}, A_f, A_{f+1}), left-moving part from (P_{f+2}, P_{f+1}, P_f); upwind at f <= 1, f >= nt-1.
constexpr int ADV_RPT = 32;

template <typename real>
__device__ __forceinline__ real weno3_shared(real near, real p0, real other, real s_q0, real s_q1) {
    // weno3_side with q0^2, q1^2 already turned into s = (eps + q^2)^2 and p0 = 1.5 near - 0.5 far given
    const real p1 = (real)0.5 * (near + other);
    const real a0 = s_q1, a1 = (real)2 * s_q0;
    return pos_div(a0 * p0 + a1 * p1, a0 + a1);
}

constexpr int ATT_COLS = (TX / 32) * 28;   // columns written per CTA by the kernels that take phi-neighbours by shuffle

// Third pass (ncu: 80 registers, 5.9 warps per scheduler, long_scoreboard 6.3 per issue -- the arithmetic waited for L1: three
// re-reads of the neighbouring columns and seven warp-uniform table loads per row): a warp covers 32 consecutive columns and
// writes the 28 in the middle, so B at k-2, k-1, k+1 comes from the neighbouring lanes by shuffle and every global load is
// this lane's own column; the per-row tables of the CTA's 32 + 4 rows sit in shared memory.
template <typename real>
__global__ void __launch_bounds__(TX) k_adv_stage_u(AdvArgs<real> A, Tables<real> T, Geom G) {
    __shared__ double red[32];
    constexpr int NTAB = ADV_RPT + 5;
    __shared__ real s_lm[NTAB], s_lp[NTAB], s_pm[NTAB], s_pp[NTAB], s_sth[NTAB], s_rdt[NTAB], s_rdp[NTAB];
    const int r = blockIdx.z;
    const int lane = threadIdx.x & 31;
    const int np = G.np, nt = G.nt;
    const int k = (blockIdx.x * (TX / 32) + (threadIdx.x >> 5)) * 28 + lane - 2;   // lanes 0, 1, 30, 31: neighbours only
    const bool live = lane >= 2 && lane < 30 && k < np;
    int k0 = k % np;
    if (k0 < 0) k0 += np;
    const int j0 = 1 + blockIdx.y * A.rpt;          // rows 1..nt only; caps are done by k_adv_caps
    const int j1 = min(j0 + A.rpt, nt + 1);
    auto cl = [&](int j) -> int { return min(max(j, 0), nt + 1); };
    const int jt = j0 - 2;                          // first table row (index i <-> row jt + i, clamped to 0..nt+1)
    if (threadIdx.x < NTAB) {
        const int row = cl(jt + threadIdx.x);
        const size_t o = (size_t)r * (nt + 2) + row;
        s_lm[threadIdx.x] = T.lm[o]; s_lp[threadIdx.x] = T.lp[o]; s_pm[threadIdx.x] = T.pm[o]; s_pp[threadIdx.x] = T.pp[o];
        s_sth[threadIdx.x] = T.sth[min(row, nt)]; s_rdt[threadIdx.x] = T.rdt[row]; s_rdp[threadIdx.x] = T.rdp[row];
    }
    __syncthreads();
    const size_t base = (size_t)r * G.rstride + k0;
    const real* __restrict__ in = A.in + base;      // (in, fn and out never alias: the SSPRK stages ping-pong between arrays)
    const real* vtf = T.vtf + (size_t)r * (nt + 1);
    const real eps = T.eps_t;
    auto ld = [&](int j) -> real { return in[(size_t)cl(j) * G.pitch]; };
    auto sm = [&](real q) -> real { const real e = eps + q * q; return e * e; };

    // rows f-1 .. f+2 around the first face f = j0 - 1
    real w1 = ld(j0 - 1), w2 = ld(j0), w3 = ld(j0 + 1);
    // windows at face f: A_{f-1}, A_f, A_{f+1};  P_f, P_{f+1}, P_{f+2}   (table rows outside 0..nt+1 feed upwind faces only)
    real Am = ld(j0 - 2) * s_lm[0], Ac = w1 * s_lm[1], Ap = w2 * s_lm[2];
    real Pc = w1 * s_lp[1], Pp = w2 * s_lp[2], Pq = w3 * s_lp[3];
    real qa1 = Ap - Ac, qp0 = Pp - Pq;              // right-moving: q1 = other - near; left-moving: q0 = near - far
    real sa0 = sm(Ac - Am), sa1 = sm(qa1), sp0 = sm(qp0), sp1 = sm(Pc - Pp);
    auto face = [&](int f, real b0, real bp1) -> real {
        if (f <= 1 || f >= nt - 1) return upwind(vtf[f], b0, bp1);
        const real um = weno3_shared(Ac, (real)1.5 * Ac - (real)0.5 * Am, Ap, sa0, sa1);
        const real up = weno3_shared(Pp, (real)1.5 * Pp - (real)0.5 * Pq, Pc, sp0, sp1);
        return up + um;
    };
    real Fn = face(j0 - 1, w1, w2);
    double sumN = 0.0, sumS = 0.0;
    if (j0 == 1) sumN = live ? (double)Fn : 0.0;
    const real* __restrict__ nxt = in + (size_t)cl(j0 + 2) * G.pitch;        // row j + 2, this column
    const real* __restrict__ fnp = A.fn + base + (size_t)j0 * G.pitch;
    real* __restrict__ outp = A.out + base + (size_t)j0 * G.pitch;
    const bool blend = A.ca != (real)0;
    const unsigned full = 0xffffffffu;
    // unrolled: the window shifts become register renaming, and the loads of the next rows move above this row's arithmetic
#pragma unroll 4
    for (int j = j0; j < j1; j++) {
        const int i = j - jt;                       // table index of row j
        const real w4 = *nxt;
        const real fnv = blend ? *fnp : (real)0;
        // slide the windows to face j: one new product, difference and smoothness term per side
        Am = Ac; Ac = Ap; Ap = w3 * s_lm[i + 1];
        Pc = Pp; Pp = Pq; Pq = w4 * s_lp[i + 2];
        sa0 = sa1; qa1 = Ap - Ac; sa1 = sm(qa1);
        sp1 = sp0; qp0 = Pp - Pq; sp0 = sm(qp0);
        const real Fs = face(j, w2, w3);
        const real bm1 = __shfl_up_sync(full, w2, 1), bm2 = __shfl_up_sync(full, w2, 2), bp1 = __shfl_down_sync(full, w2, 1);
        const real Fw = phi_face_flux<real>(bm2, bm1, w2, bp1, s_pm[i], s_pp[i], T.eps_p, 0);   // valid on lanes 2..30
        const real Fe = __shfl_down_sync(full, Fw, 1);   // face k+1/2 = the west face of column k+1 (same operands, same bits)
        const real tend = (s_sth[i] * Fs - s_sth[i - 1] * Fn) * s_rdt[i] + (Fe - Fw) * s_rdp[i];
        real o = A.cb * w2 - A.cdt * tend;
        if (blend) o = A.ca * fnv + o;
        if (live) *outp = o;
        if (j == nt) sumS = live ? (double)Fs : 0.0;
        Fn = Fs;
        w1 = w2; w2 = w3; w3 = w4;
        fnp += G.pitch; outp += G.pitch;
        if (j + 3 <= nt + 1) nxt += G.pitch;                    // row j + 3 of the next iteration, clamped to the south cap
    }
    if (j0 == 1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 0) * A.nparts + blockIdx.x] = t;
    }
    if (j0 <= nt && nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 1) * A.nparts + blockIdx.x] = t;
    }
}

// The same stage with flow attenuation (Eq. 5): per-cell LLF half-speeds (k_att_halfspeeds) instead of per-row tables,
// both LLF parts live in phi.  A thread streams RPT rows of its column; B and the theta half-speeds move through
// register windows (one new row of each per row-step), and ALL operands of a row are requested before its arithmetic
// starts, so that the ~16 independent loads of a row overlap (the first version interleaved them with the WENO
// arithmetic and stalled 9 issue slots per instruction on the scoreboard: profiles/r01_final_cfg3.md).
template <typename real>
__global__ void __launch_bounds__(TX) k_adv_stage_att(AdvArgs<real> A, Tables<real> T, Geom G) {
    __shared__ double red[32];
    const int r = blockIdx.z;
    const int lane = threadIdx.x & 31;
    const int k = (blockIdx.x * (TX / 32) + (threadIdx.x >> 5)) * 31 + lane;   // lane 31: the first column of the next warp
    const int np = G.np, nt = G.nt;
    const bool live = lane < 31 && k < np;
    const int k0 = k % np;
    const int km1 = (k0 + np - 1) % np, km2 = (k0 + np - 2) % np, kp1 = (k0 + 1) % np;
    const int j0 = 1 + blockIdx.y * RPT;
    const int j1 = min(j0 + RPT, nt + 1);
    const size_t base = (size_t)r * G.rstride;
    const real* in = A.in + base;
    auto col = [&](const real* p, int j) -> real { return p[base + (size_t)min(max(j, 0), nt + 1) * G.pitch + k0]; };
    const bool uw = A.upwind_only != 0;

    // theta-face flux at face f from B rows f-1..f+2 and the half-speeds LMt rows f-1..f+1, LPt rows f..f+2
    auto theta_flux = [&](int f, real bm1, real b0, real bp1, real bp2, real m0, real m1, real m2, real p0, real p1, real p2) -> real {
        if (uw || f <= 1 || f >= nt - 1) return upwind(col(A.VT, f), b0, bp1);
        if (T.nonuniform) {
            const real* D = T.wmp + 16 * (size_t)f;
            return weno3_side_nu(bp2 * p2, bp1 * p1, b0 * p0, D[5], D + 8) + weno3_side_nu(bm1 * m0, b0 * m1, bp1 * m2, D[5], D);
        }
        real um = weno3_side(bm1 * m0, b0 * m1, bp1 * m2, T.eps_t);
        real up = weno3_side(bp2 * p2, bp1 * p1, b0 * p0, T.eps_t);
        return up + um;
    };
    real w0 = col(A.in, j0 - 2), w1 = col(A.in, j0 - 1), w2 = col(A.in, j0), w3 = col(A.in, j0 + 1);
    // windows for face f = j0 - 1: LMt rows f-1, f, f+1; LPt rows f, f+1, f+2
    real m0 = col(A.LMt, j0 - 2), m1 = col(A.LMt, j0 - 1), m2 = col(A.LMt, j0);
    real p0 = col(A.LPt, j0 - 1), p1 = col(A.LPt, j0), p2 = col(A.LPt, j0 + 1);
    real Fn = theta_flux(j0 - 1, w0, w1, w2, w3, m0, m1, m2, p0, p1, p2);
    double sumN = 0.0, sumS = 0.0;
    if (j0 == 1) sumN = live ? (double)Fn : 0.0;
    for (int j = j0; j < j1; j++) {
        // ---- every load of this row first
        const size_t ro = base + (size_t)j * G.pitch;
        const real w4 = col(A.in, j + 2);
        const real m3 = col(A.LMt, j + 1), p3 = col(A.LPt, j + 2);
        const real* row = in + (size_t)j * G.pitch;
        const real bm2 = row[km2], bm1 = row[km1], bp1 = row[kp1];
        real a_m2 = 0, a_m1 = 0, a_0 = 0, b_m1 = 0, b_0 = 0, b_p1 = 0, vw = 0;
        if (uw) {
            vw = A.VP[ro + k0];
        } else {
            a_m2 = A.LMp[ro + km2]; a_m1 = A.LMp[ro + km1]; a_0 = A.LMp[ro + k0];
            b_m1 = A.LPp[ro + km1]; b_0 = A.LPp[ro + k0]; b_p1 = A.LPp[ro + kp1];
        }
        const real fnv = (A.ca != (real)0) ? A.fn[ro + k0] : (real)0;
        // ---- then the arithmetic.  Face j (between rows j, j+1): LMt rows j-1..j+1 = (m1, m2, m3), LPt rows j..j+2 = (p1, p2, p3)
        const real Fs = theta_flux(j, w1, w2, w3, w4, m1, m2, m3, p1, p2, p3);
        real Fw;
        if (uw) {
            Fw = upwind(vw, bm1, w2);
        } else {
            // face k-1/2: LM of cells k-2, k-1, k; LP of cells k+1, k, k-1
            Fw = weno3_side(bp1 * b_p1, w2 * b_0, bm1 * b_m1, T.eps_p) + weno3_side(bm2 * a_m2, bm1 * a_m1, w2 * a_0, T.eps_p);
        }
        const real Fe = __shfl_down_sync(0xffffffffu, Fw, 1);   // face k+1/2 = the west face of column k+1
        const real tend = (T.sth[j] * Fs - T.sth[j - 1] * Fn) * T.rdt[j] + (Fe - Fw) * T.rdp[j];
        real o = A.cb * w2 - A.cdt * tend;
        if (A.ca != (real)0) o = A.ca * fnv + o;
        if (live) A.out[ro + k0] = o;
        if (j == nt) sumS = live ? (double)Fs : 0.0;
        Fn = Fs;
        w0 = w1; w1 = w2; w2 = w3; w3 = w4;
        m0 = m1; m1 = m2; m2 = m3;
        p0 = p1; p1 = p2; p2 = p3;
    }
    if (j0 == 1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 0) * A.nparts + blockIdx.x] = t;
    }
    if (j0 <= nt && nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 1) * A.nparts + blockIdx.x] = t;
    }
}

// k_adv_stage_att on a uniform theta grid with WENO3 fluxes, own-column loads only.  A warp covers 32 consecutive columns and
// writes the 28 in the middle (lanes 2..29): the phi stencil of a face reaches two columns west and one east, and every
// neighbour value -- the LLF products B LMp, B LPp of the cells next door -- comes from the neighbouring lanes by shuffle
// instead of nine more loads per row (k_adv_stage_att: 13 loads per row and thread, 7 of them re-reads of other columns'
// operands).  The theta sweep shares its products, differences and smoothness terms between faces as k_adv_stage_u does.
template <typename real>
__global__ void __launch_bounds__(TX) k_adv_stage_att_u(AdvArgs<real> A, Tables<real> T, Geom G) {
    __shared__ double red[32];
    const int r = blockIdx.z;
    const int lane = threadIdx.x & 31;
    const int np = G.np, nt = G.nt;
    const int k = (blockIdx.x * (TX / 32) + (threadIdx.x >> 5)) * 28 + lane - 2;   // lanes 0, 1, 30, 31: neighbours only
    const bool live = lane >= 2 && lane < 30 && k < np;
    int k0 = k % np;
    if (k0 < 0) k0 += np;
    const int j0 = 1 + blockIdx.y * A.rpt;
    const int j1 = min(j0 + A.rpt, nt + 1);
    const size_t base = (size_t)r * G.rstride + k0;
    const real eps = T.eps_t;
    auto cl = [&](int j) -> int { return min(max(j, 0), nt + 1); };
    auto at = [&](const real* p, int j) -> real { return p[base + (size_t)cl(j) * G.pitch]; };
    auto sm = [&](real q) -> real { const real e = eps + q * q; return e * e; };

    real w1 = at(A.in, j0 - 1), w2 = at(A.in, j0), w3 = at(A.in, j0 + 1);
    // windows at face f = j0 - 1: A_{f-1}, A_f, A_{f+1} (B LMt) and P_f, P_{f+1}, P_{f+2} (B LPt)
    real Am = at(A.in, j0 - 2) * at(A.LMt, j0 - 2), Ac = w1 * at(A.LMt, j0 - 1), Ap = w2 * at(A.LMt, j0);
    real Pc = w1 * at(A.LPt, j0 - 1), Pp = w2 * at(A.LPt, j0), Pq = w3 * at(A.LPt, j0 + 1);
    real qa1 = Ap - Ac, qp0 = Pp - Pq;
    real sa0 = sm(Ac - Am), sa1 = sm(qa1), sp0 = sm(qp0), sp1 = sm(Pc - Pp);
    auto face = [&](int f, real b0, real bp1) -> real {
        if (f <= 1 || f >= nt - 1) return upwind(A.VT[base + (size_t)f * G.pitch], b0, bp1);
        const real um = weno3_shared(Ac, (real)1.5 * Ac - (real)0.5 * Am, Ap, sa0, sa1);
        const real up = weno3_shared(Pp, (real)1.5 * Pp - (real)0.5 * Pq, Pc, sp0, sp1);
        return up + um;
    };
    real Fn = face(j0 - 1, w1, w2);
    double sumN = 0.0, sumS = 0.0;
    if (j0 == 1) sumN = live ? (double)Fn : 0.0;
    const size_t p = G.pitch;
    const real* __restrict__ inn = A.in + base + (size_t)cl(j0 + 2) * p;     // B row j + 2
    const real* __restrict__ lmt = A.LMt + base + (size_t)(j0 + 1) * p;      // LMt row j + 1
    const real* __restrict__ lpt = A.LPt + base + (size_t)cl(j0 + 2) * p;    // LPt row j + 2
    const real* __restrict__ lmp = A.LMp + base + (size_t)j0 * p;            // row j
    const real* __restrict__ lpp = A.LPp + base + (size_t)j0 * p;
    const real* __restrict__ fnp = A.fn + base + (size_t)j0 * p;
    real* __restrict__ outp = A.out + base + (size_t)j0 * p;
    real sthn = T.sth[j0 - 1];
    const bool blend = A.ca != (real)0;
    const unsigned full = 0xffffffffu;
#pragma unroll 2
    for (int j = j0; j < j1; j++) {
        // ---- every load of this row first: six streams, this lane's column only
        const real w4 = *inn, m3 = *lmt, p3 = *lpt, am = *lmp, ap = *lpp;
        const real fnv = blend ? *fnp : (real)0;
        // ---- theta: slide the windows to face j
        Am = Ac; Ac = Ap; Ap = w3 * m3;
        Pc = Pp; Pp = Pq; Pq = w4 * p3;
        sa0 = sa1; qa1 = Ap - Ac; sa1 = sm(qa1);
        sp1 = sp0; qp0 = Pp - Pq; sp0 = sm(qp0);
        const real Fs = face(j, w2, w3);
        // ---- phi: this cell's LLF products, the neighbours' by shuffle.  Face k-1/2: LM of cells k-2, k-1, k; LP of k+1, k, k-1
        const real a0 = w2 * am, b0 = w2 * ap;
        const real a1 = __shfl_up_sync(full, a0, 1), a2 = __shfl_up_sync(full, a0, 2);
        const real b1 = __shfl_up_sync(full, b0, 1), bp = __shfl_down_sync(full, b0, 1);
        const real Fw = weno3_side(bp, b0, b1, T.eps_p) + weno3_side(a2, a1, a0, T.eps_p);   // valid on lanes 2..30
        const real Fe = __shfl_down_sync(full, Fw, 1);
        const real sths = T.sth[j];
        const real tend = (sths * Fs - sthn * Fn) * T.rdt[j] + (Fe - Fw) * T.rdp[j];
        real o = A.cb * w2 - A.cdt * tend;
        if (blend) o = A.ca * fnv + o;
        if (live) *outp = o;
        if (j == nt) sumS = live ? (double)Fs : 0.0;
        Fn = Fs; sthn = sths;
        w1 = w2; w2 = w3; w3 = w4;
        lmp += p; lpp += p; fnp += p; outp += p;
        if (j + 2 <= nt + 1) lmt += p;                       // LMt row j + 2 next (unused beyond the south cap)
        if (j + 3 <= nt + 1) { inn += p; lpt += p; }
    }
    if (j0 == 1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 0) * A.nparts + blockIdx.x] = t;
    }
    if (j0 <= nt && nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part[((size_t)r * 2 + 1) * A.nparts + blockIdx.x] = t;
    }
}

// Polar caps of one SSPRK stage (App. A :646): north +P sum_k F_theta[1/2,k] dph, south -P sum_k F_theta[nt+1/2,k] dph.
// grid (nbx, 2, R): every CTA re-sums the partials in index order and writes its TX columns of the cap row.
template <typename real>
__global__ void __launch_bounds__(TX) k_adv_caps(AdvArgs<real> A, Tables<real> T, Geom G) {
    const int r = blockIdx.z, pole = blockIdx.y;
    const int k = blockIdx.x * TX + threadIdx.x;
    if (k >= G.np) return;
    const int j = pole == 0 ? 0 : G.nt + 1;
    const size_t off = (size_t)r * G.rstride + (size_t)j * G.pitch;
    double S = sum_partials(A.part + ((size_t)r * 2 + pole) * A.nparts, A.nparts);
    real tend = (real)((pole == 0 ? 1.0 : -1.0) * (T.adv_capc[pole] * S));
    real o = A.cb * A.in[off] - A.cdt * tend;
    if (A.ca != (real)0) o = A.ca * A.fn[off] + o;
    A.out[off + k] = o;
}

// ------------------------------------------------------------------ flow attenuation, Eq. 5 (:100-103)

__device__ __forceinline__ double tanh_r(double x) { return tanh(x); }
__device__ __forceinline__ float tanh_r(float x) { return tanhf(x); }

// Face speeds v [1 - tanh(|B| / B0)] with |B| at a face = |mean of the two cells it separates| (U22), from the
// field at the start of the step (U23).  grid (nbx, nt+2, R): thread (j, k) writes VT[j][k] (face j+1/2, j <= nt) and
// VP[j][k] (face k-1/2, rows 1..nt).  B0[r] <= 0: no attenuation for that realization (factor exactly 1).
template <typename real>
__global__ void __launch_bounds__(TX) k_att_faces(const real* state, const real* B0, Tables<real> T, Geom G, real* VT, real* VP) {
    const int k = blockIdx.x * TX + threadIdx.x, j = blockIdx.y, r = blockIdx.z;
    if (k >= G.np) return;
    const int nt = G.nt, km1 = (k + G.np - 1) % G.np;
    const size_t ro = (size_t)r * G.rstride + (size_t)j * G.pitch;
    const real b0 = B0[r], b = state[ro + k];
    const bool on = b0 > (real)0;
    if (j <= nt) {
        const real bf = (real)0.5 * (b + state[ro + G.pitch + k]);
        const real g = on ? (real)1 - tanh_r(fabs(bf) / b0) : (real)1;
        VT[ro + k] = T.vtf[(size_t)r * (nt + 1) + j] * g;
    }
    if (j >= 1 && j <= nt) {
        const real bf = (real)0.5 * (state[ro + km1] + b);
        const real g = on ? (real)1 - tanh_r(fabs(bf) / b0) : (real)1;
        const size_t i = (size_t)r * (nt + 2) + j;
        VP[ro + k] = (T.pm[i] + T.pp[i]) * g;   // one of pm, pp is 0: the sum is the row speed v_phi exactly
    }
}

// LLF half-speeds of every cell (B2 :684) with alpha = max |v| over the six faces c-5/2 .. c+5/2 along the sweep
// (:689): clipped to existing faces in theta, periodic in phi.  grid (nbx, nt+2, R).
template <typename real>
__global__ void __launch_bounds__(TX) k_att_halfspeeds(const real* VT, const real* VP, Geom G, real* LMt, real* LPt, real* LMp,
                                                       real* LPp) {
    const int k = blockIdx.x * TX + threadIdx.x, j = blockIdx.y, r = blockIdx.z;
    if (k >= G.np) return;
    const int nt = G.nt, np = G.np;
    const size_t fo = (size_t)r * G.rstride, ro = fo + (size_t)j * G.pitch;
    real a = (real)0;
    for (int q = j - 3; q <= j + 2; q++)
        if (q >= 0 && q <= nt) a = fmax(a, fabs(VT[fo + (size_t)q * G.pitch + k]));
    LMt[ro + k] = (real)0.5 * ((j >= 1 ? VT[ro - G.pitch + k] : (real)0) + a);
    LPt[ro + k] = (real)0.5 * ((j <= nt ? VT[ro + k] : (real)0) - a);
    if (j >= 1 && j <= nt) {
        real ap = (real)0;
        for (int q = k - 2; q <= k + 3; q++) ap = fmax(ap, fabs(VP[ro + (q + np) % np]));
        LMp[ro + k] = (real)0.5 * (VP[ro + k] + ap);
        LPp[ro + k] = (real)0.5 * (VP[ro + (k + 1) % np] - ap);
    }
}

// ------------------------------------------------------------------ maps in / out, caps by row means

// rows 1..nt of the state <- user map [nt][np] (dir 0) or the reverse (dir 1). grid (nbx, nt, nz):
// state realization = r0 + blockIdx.z, map index = bcast ? 0 : blockIdx.z.
template <typename real>
__global__ void k_copy_map(real* state, real* map, Geom G, int r0, int bcast, int dir) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y;  // 0..nt-1
    if (k >= G.np) return;
    real* s = state + (size_t)(r0 + blockIdx.z) * G.rstride + (size_t)(i + 1) * G.pitch + k;
    real* m = map + ((size_t)(bcast ? 0 : blockIdx.z) * G.nt + i) * G.np + k;
    if (dir == 0) *s = *m; else *m = *s;
}

// full field incl. cap rows <-> dense [nt+2][np]
template <typename real>
__global__ void k_copy_full(real* state, real* dense, Geom G, int r, int dir) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    if (k >= G.np) return;
    real* s = state + (size_t)r * G.rstride + (size_t)j * G.pitch + k;
    real* m = dense + (size_t)j * G.np + k;
    if (dir == 0) *s = *m; else *m = *s;
}

// cap rows <- dph-weighted mean of the adjacent row (uniform grid: arithmetic mean). grid (2, R), block 256.
template <typename real>
__global__ void __launch_bounds__(256) k_caps_from_row_mean(real* state, Geom G, int r0) {
    __shared__ double red[32];
    __shared__ double mean;
    const int pole = blockIdx.x, r = r0 + blockIdx.y;
    real* f = state + (size_t)r * G.rstride;
    const real* row = f + (size_t)(pole == 0 ? 1 : G.nt) * G.pitch;
    double v = 0.0;
    for (int k = threadIdx.x; k < G.np; k += blockDim.x) v += (double)row[k];
    double t = block_sum(v, red);
    if (threadIdx.x == 0) mean = t / (double)G.np;
    __syncthreads();
    real* cap = f + (size_t)(pole == 0 ? 0 : G.nt + 1) * G.pitch;
    for (int k = threadIdx.x; k < G.np; k += blockDim.x) cap[k] = (real)mean;
}

// ------------------------------------------------------------------ assimilation + diagnostics

constexpr int RED_CTAS = 64;  // CTAs per realization for the flux integrals

// Flux integrals over rows 1..nt (:225-230): part[r][cta][2] = {sum_{v>0} v dA, sum_{v<=0 or <0} v dA}.
// WHAT 0: v = B (diagnostics; v == 0 contributes 0 either way).  WHAT 1: v = w (obs - B) (Eq. 10 increment, :146).
template <typename real, int WHAT>
__global__ void __launch_bounds__(256) k_flux_partials(const real* state, const real* obs, const real* wgt, int shared,
                                                       Tables<real> T, Geom G, double* part) {
    __shared__ double red[32];
    const int r = blockIdx.y;
    const real* f = state + (size_t)r * G.rstride;
    const size_t mapoff = shared ? 0 : (size_t)r * G.nt * G.np;
    double pp = 0.0, pm = 0.0;
    for (int j = 1 + blockIdx.x; j <= G.nt; j += gridDim.x) {
        double dA = T.dA[j], rp = 0.0, rm = 0.0;
        for (int k = threadIdx.x; k < G.np; k += blockDim.x) {
            real v = f[(size_t)j * G.pitch + k];
            if (WHAT == 1) {
                size_t m = mapoff + (size_t)(j - 1) * G.np + k;
                v = wgt[m] * (obs[m] - v);
            }
            if (v > (real)0) rp += (double)v; else rm += (double)v;
        }
        pp += rp * dA;
        pm += rm * dA;
    }
    double tp = block_sum(pp, red);
    double tm = block_sum(pm, red);
    if (threadIdx.x == 0) {
        part[((size_t)r * gridDim.x + blockIdx.x) * 2 + 0] = tp;
        part[((size_t)r * gridDim.x + blockIdx.x) * 2 + 1] = tm;
    }
}

// Cap obs / weight = row means of the adjacent row (reading U18); capinfo[r][pole] = {obs_mean, w_mean}. grid (2, R or 1)
template <typename real>
__global__ void __launch_bounds__(256) k_assim_cap_means(const real* obs, const real* wgt, Geom G, double* capinfo) {
    __shared__ double red[32];
    const int pole = blockIdx.x, r = blockIdx.y;
    const size_t rowoff = (size_t)r * G.nt * G.np + (size_t)(pole == 0 ? 0 : G.nt - 1) * G.np;
    double a = 0.0, b = 0.0;
    for (int k = threadIdx.x; k < G.np; k += blockDim.x) { a += (double)obs[rowoff + k]; b += (double)wgt[rowoff + k]; }
    double ta = block_sum(a, red);
    double tb = block_sum(b, red);
    if (threadIdx.x == 0) {
        capinfo[((size_t)r * 2 + pole) * 2 + 0] = ta / (double)G.np;
        capinfo[((size_t)r * 2 + pole) * 2 + 1] = tb / (double)G.np;
    }
}

// Finalize flux integrals: add the caps (areas dA[0], dA[nt+1]), sum the CTA partials in index order.
// WHAT 0: out[r][4] = {signed, unsigned, Phi+, Phi-} * scale.   WHAT 1: out[r] = sqrt|Phi+/Phi-| (1 if either is 0).
template <typename real, int WHAT>
__global__ void k_flux_finalize(const real* state, const double* part, int nparts, const double* capinfo, int shared,
                                Tables<real> T, Geom G, double scale, double* out) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= G.nr) return;
    double pp = 0.0, pm = 0.0;
    for (int i = 0; i < nparts; i++) { pp += part[((size_t)r * nparts + i) * 2]; pm += part[((size_t)r * nparts + i) * 2 + 1]; }
    for (int pole = 0; pole < 2; pole++) {
        real v = state[(size_t)r * G.rstride + (size_t)(pole == 0 ? 0 : G.nt + 1) * G.pitch];
        if (WHAT == 1) {
            const double* ci = capinfo + ((size_t)(shared ? 0 : r) * 2 + pole) * 2;
            v = (real)ci[1] * ((real)ci[0] - v);
        }
        double c = (double)v * T.dA[pole == 0 ? 0 : G.nt + 1];
        if (v > (real)0) pp += c; else pm += c;
    }
    if (WHAT == 0) {
        out[4 * r + 0] = (pp + pm) * scale;
        out[4 * r + 1] = (pp - pm) * scale;
        out[4 * r + 2] = pp * scale;
        out[4 * r + 3] = pm * scale;
    } else {
        out[r] = (pp != 0.0 && pm != 0.0) ? sqrt(fabs(pp / pm)) : 1.0;
    }
}

// Blend (Eq. 8 :131) or flux-balanced blend (Eq. 10-11 :144-153) on rows 0..nt+1; grid (nbx, nt+2, R).
template <typename real>
__global__ void __launch_bounds__(TX) k_assim_blend(real* state, const real* obs, const real* wgt, int shared,
                                                    const double* capinfo, const double* scale, int balanced, Geom G) {
    const int k = blockIdx.x * TX + threadIdx.x, j = blockIdx.y, r = blockIdx.z;
    if (k >= G.np) return;
    real* p = state + (size_t)r * G.rstride + (size_t)j * G.pitch + k;
    real F, Bd;
    if (j == 0 || j == G.nt + 1) {
        const double* ci = capinfo + ((size_t)(shared ? 0 : r) * 2 + (j == 0 ? 0 : 1)) * 2;
        Bd = (real)ci[0];
        F = (real)ci[1];
    } else {
        size_t m = (shared ? 0 : (size_t)r * G.nt * G.np) + (size_t)(j - 1) * G.np + k;
        Bd = obs[m];
        F = wgt[m];
    }
    real B = *p;
    if (!balanced) {
        *p = F * Bd + ((real)1 - F) * B;
    } else {
        real sc = (real)scale[r];
        real d = F * (Bd - B);
        d = (d > (real)0) ? d / sc : d * sc;
        *p = B + d;
    }
}

// The blend and the flux integrals of the blended state in ONE pass (north_star's "fused assimilation/diagnostics kernel";
// "fused into A7 when called together").  grid (RED_CTAS, R), block 256: a CTA owns the rows
// blockIdx.x, blockIdx.x + RED_CTAS, ... of 0..nt+1, blends them exactly as k_assim_blend does and accumulates Phi+ / Phi- of
// the NEW values of rows 1..nt (row sums in fp64, then x dA_j) into part[r][cta][2]; k_flux_finalize<WHAT = 0> adds the caps
// from the blended state.  The balanced form still needs its scale factor first (Eq. 11 needs Phi+- of the whole increment).
template <typename real>
__global__ void __launch_bounds__(256) k_assim_blend_diag(real* state, const real* obs, const real* wgt, int shared,
                                                          const double* capinfo, const double* scale, int balanced,
                                                          Tables<real> T, Geom G, double* part) {
    __shared__ double red[32];
    const int r = blockIdx.y;
    real* f = state + (size_t)r * G.rstride;
    const size_t mapoff = shared ? 0 : (size_t)r * G.nt * G.np;
    const real sc = balanced ? (real)scale[r] : (real)1;
    double pp = 0.0, pm = 0.0;
    for (int j = blockIdx.x; j <= G.nt + 1; j += gridDim.x) {
        const bool cap = j == 0 || j == G.nt + 1;
        const double* ci = capinfo + ((size_t)(shared ? 0 : r) * 2 + (j == 0 ? 0 : 1)) * 2;
        double rp = 0.0, rm = 0.0;
        for (int k = threadIdx.x; k < G.np; k += blockDim.x) {
            real Bd, F;
            if (cap) { Bd = (real)ci[0]; F = (real)ci[1]; }
            else { const size_t m = mapoff + (size_t)(j - 1) * G.np + k; Bd = obs[m]; F = wgt[m]; }
            const real B = f[(size_t)j * G.pitch + k];
            real v;
            if (!balanced) {
                v = F * Bd + ((real)1 - F) * B;
            } else {
                real d = F * (Bd - B);
                d = (d > (real)0) ? d / sc : d * sc;
                v = B + d;
            }
            f[(size_t)j * G.pitch + k] = v;
            if (!cap) { if (v > (real)0) rp += (double)v; else rm += (double)v; }
        }
        if (!cap) { pp += rp * T.dA[j]; pm += rm * T.dA[j]; }
    }
    const double tp = block_sum(pp, red);
    const double tm = block_sum(pm, red);
    if (threadIdx.x == 0) {
        part[((size_t)r * gridDim.x + blockIdx.x) * 2 + 0] = tp;
        part[((size_t)r * gridDim.x + blockIdx.x) * 2 + 1] = tm;
    }
}

// ------------------------------------------------------------------ remaining run-history diagnostics (:230-242)

constexpr int EXT_NPART = 10;  // per-CTA partials: Phi+N, Phi-N, Phi+S, Phi-S, h1, h2, d, min, max, min|B|
constexpr int EXT_NOUT = 13;   // see include/hft.h hft_diagnostics_ext

__device__ __forceinline__ double block_min(double v, double* smem /*[32]*/) {
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if (lane == 0) smem[w] = v;
    __syncthreads();
    double t = smem[0];
    for (int i = 1; i < nw; i++) t = fmin(t, smem[i]);
    return t;
}

// Rows 1..nt: polar-region fluxes (cells with theta_j <= thc or >= pi - thc), the dipole integrands of Eq. 16-17 and
// min / max / min|B|.  part[r][cta][EXT_NPART]; grid (RED_CTAS, R), block 256.  Row sums in fp64, weights per row.
template <typename real>
__global__ void __launch_bounds__(256) k_diag_ext_partials(const real* state, Tables<real> T, Geom G, double dph,
                                                           double thc, double* part) {
    __shared__ double red[32];
    const int r = blockIdx.y;
    const real* f = state + (size_t)r * G.rstride;
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    double vmin = 1.0e300, vmax = -1.0e300, amin = 1.0e300;
    for (int j = 1 + blockIdx.x; j <= G.nt; j += gridDim.x) {
        const double th = T.th[j], dA = T.dA[j];
        const int region = th <= thc ? 0 : (th >= 3.14159265358979323846264338327950288 - thc ? 1 : -1);
        double rp = 0.0, rm = 0.0, rc = 0.0, rs = 0.0;
        for (int k = threadIdx.x; k < G.np; k += blockDim.x) {
            const double v = (double)f[(size_t)j * G.pitch + k];
            double sn, cs;
            sincos((double)k * dph, &sn, &cs);
            if (v > 0.0) rp += v; else rm += v;
            rc += v * cs;
            rs += v * sn;
            vmin = fmin(vmin, v); vmax = fmax(vmax, v); amin = fmin(amin, fabs(v));
        }
        if (region >= 0) { acc[2 * region] += rp * dA; acc[2 * region + 1] += rm * dA; }
        const double st = sin(th), ct = cos(th);
        acc[4] += rc * st * dA;
        acc[5] += rs * st * dA;
        acc[6] += (rp + rm) * ct * dA;
    }
    double* out = part + ((size_t)r * gridDim.x + blockIdx.x) * EXT_NPART;
    for (int i = 0; i < 7; i++) {
        const double t = block_sum(acc[i], red);
        if (threadIdx.x == 0) out[i] = t;
    }
    const double tmin = block_min(vmin, red), tmax = -block_min(-vmax, red), tamin = block_min(amin, red);
    if (threadIdx.x == 0) { out[7] = tmin; out[8] = tmax; out[9] = tamin; }
}

// One thread per realization: partials in index order, then the two caps (one cell each: sin(theta) = 0, so they
// enter D, the polar fluxes / areas and the extrema only) and the region areas.
template <typename real>
__global__ void k_diag_ext_finalize(const real* state, const double* part, int nparts, Tables<real> T, Geom G,
                                    double thc, double scale, double* out) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= G.nr) return;
    const double PI_ = 3.14159265358979323846264338327950288;
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    double vmin = 1.0e300, vmax = -1.0e300, amin = 1.0e300;
    for (int i = 0; i < nparts; i++) {
        const double* p = part + ((size_t)r * nparts + i) * EXT_NPART;
        for (int q = 0; q < 7; q++) acc[q] += p[q];
        vmin = fmin(vmin, p[7]); vmax = fmax(vmax, p[8]); amin = fmin(amin, p[9]);
    }
    double area[2] = {0.0, 0.0};
    for (int j = 1; j <= G.nt; j++) {
        const double th = T.th[j];
        if (th <= thc) area[0] += T.dA[j] * (double)G.np;
        else if (th >= PI_ - thc) area[1] += T.dA[j] * (double)G.np;
    }
    for (int pole = 0; pole < 2; pole++) {
        const double v = (double)state[(size_t)r * G.rstride + (size_t)(pole == 0 ? 0 : G.nt + 1) * G.pitch];
        const double th = pole == 0 ? 0.0 : PI_, dA = T.dA[pole == 0 ? 0 : G.nt + 1];
        const int region = th <= thc ? 0 : (th >= PI_ - thc ? 1 : -1);
        if (region >= 0) {
            if (v > 0.0) acc[2 * region] += v * dA; else if (v < 0.0) acc[2 * region + 1] += v * dA;
            area[region] += dA;
        }
        acc[6] += v * (pole == 0 ? 1.0 : -1.0) * dA;
        vmin = fmin(vmin, v); vmax = fmax(vmax, v); amin = fmin(amin, fabs(v));
    }
    double* q = out + (size_t)r * EXT_NOUT;
    const double c = 3.0 / (4.0 * PI_);
    for (int i = 0; i < 4; i++) q[i] = acc[i] * scale;
    q[4] = area[0] * scale; q[5] = area[1] * scale;
    q[6] = vmin; q[7] = vmax; q[8] = amin;
    q[11] = c * acc[4]; q[12] = c * acc[5]; q[10] = c * acc[6];
    q[9] = sqrt(q[11] * q[11] + q[12] * q[12]);
}

// ------------------------------------------------------------------ random flux emergence, Sec. 2.4 (:155-209)

// Philox4x32-10 (Salmon et al. 2011): the counter-based generator both sides implement (reading U27).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t& o0, uint32_t& o1) {
#pragma unroll
    for (int round = 0; round < 10; round++) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1;
}

// One raw (unbalanced) source map, Eq. 13 (model 1) or Eq. 14 (model 2): S[j][k] = amp_j Y, Y the standard normal of
// cell i = (j-1) np + k of map `map` of realization r (counter (i, map, r, 0), key = seed; Box-Muller in fp64).
// Caps 0 (reading U28).  grid (nbx, nt+2, R).
template <typename real>
__global__ void __launch_bounds__(TX) k_rfe_generate(real* S, Tables<real> T, Geom G, int model, double flux_per_hr, double r2,
                                                     uint32_t seed_lo, uint32_t seed_hi, uint32_t map) {
    const int k = blockIdx.x * TX + threadIdx.x, j = blockIdx.y, r = blockIdx.z;
    if (k >= G.np) return;
    real v = (real)0;
    if (j >= 1 && j <= G.nt) {
        const double PI_ = 3.14159265358979323846264338327950288;
        const double dA = T.dA[j] * r2, ncells = (double)G.nt * (double)G.np;
        const double amp = model == 1 ? flux_per_hr / (dA * ncells) * sqrt(PI_ / 2.0) : flux_per_hr / (4.0 * PI_ * r2) * sqrt(PI_ / 2.0);
        uint32_t x0, x1;
        philox4x32_10((uint32_t)((j - 1) * G.np + k), map, (uint32_t)r, 0u, seed_lo, seed_hi, x0, x1);
        const double u1 = ((double)x0 + 0.5) * (1.0 / 4294967296.0), u2 = ((double)x1 + 0.5) * (1.0 / 4294967296.0);
        v = (real)(amp * (sqrt(-2.0 * log(u1)) * cos(2.0 * PI_ * u2)));
    }
    S[(size_t)r * G.rstride + (size_t)j * G.pitch + k] = v;
}

// Balance a source map "in the same manner as Eq. 11" (:207): flux[r][4] = {.., .., Phi+, Phi-} of the map (k_flux_*).
template <typename real>
__global__ void __launch_bounds__(TX) k_rfe_balance(real* S, const double* flux, Geom G) {
    const int k = blockIdx.x * TX + threadIdx.x, j = blockIdx.y, r = blockIdx.z;
    if (k >= G.np) return;
    const double pp = flux[4 * r + 2], pm = flux[4 * r + 3];
    if (pp == 0.0 || pm == 0.0) return;
    const real sc = (real)sqrt(fabs(pp / pm));
    real* p = S + (size_t)r * G.rstride + (size_t)j * G.pitch + k;
    const real v = *p;
    *p = v > (real)0 ? v / sc : v * sc;
}

// The source advance (Eq. 15 :203, forward Euler): B <- B + h [(1 - alpha) S1 + alpha S2].  grid (nbx, nt+2, R).
template <typename real>
__global__ void __launch_bounds__(TX) k_rfe_apply(real* B, const real* S1, const real* S2, real alpha, real h, Geom G) {
    const int k = blockIdx.x * TX + threadIdx.x, j = blockIdx.y, r = blockIdx.z;
    if (k >= G.np) return;
    const size_t i = (size_t)r * G.rstride + (size_t)j * G.pitch + k;
    B[i] = B[i] + h * (((real)1 - alpha) * S1[i] + alpha * S2[i]);
}

}  // namespace hft
