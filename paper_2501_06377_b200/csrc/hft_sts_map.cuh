// hft_sts_map.cuh -- diffusion / STS stage kernels for a spatially varying diffusivity nu(theta, phi).
//
// Eq. 27: "nu is located on a staggered grid in both the theta and phi direction".  NU is one more
// field-shaped array, NU[r][f][k] = nu at theta-face f+1/2 and phi-face k+1/2 (between columns k and k+1, periodic),
// f = 0..nt.  The four off-diagonal coefficients of Eq. 28 (:450-458) are formed in-kernel from the two NU rows a cell
// touches (the row above stays in registers while the thread streams down its columns), so a stage moves 3 + 1 + 1 array
// passes instead of the 3 + 1 + 4 a stored DIA matrix would:
//   L = a_s (s - c) - a_n (c - n) + a_e (e - c) - a_w (c - w)
//   a_s = (NU[j][k] + NU[j][k-1])/2 sin(theta_{j+1/2}) / (sin(theta_j) dth^2),  a_n likewise from NU row j-1
//   a_e = (NU[j][k] + NU[j-1][k])/2 / (sin^2(theta_j) dph^2),                   a_w likewise from column k-1
// Caps (App. A :624-648 with the face-averaged nu): L_cap = P dph/dth [sum_k nu_k B[1,k] - (sum_k nu_k) B_cap], nu_k =
// (NU[0][k] + NU[0][k-1])/2: the polar partial sums are nu-weighted, sum_k nu_k comes from the host (capw).
// With nu(theta, phi) the coefficients of L depend on phi, so neither the per-row tables nor the zonal-mean cap recurrence
// of the blocked kernel (U21) apply: this path is one launch per stage, bounded by HBM at 5 array passes.
//
// k_sts_stage_mapv: a thread owns C = 16 / sizeof(real) adjacent columns (one 16-byte vector per array and row), phi
//                   neighbours of the vector's end columns come from the adjacent lanes by shuffle, the two columns beyond
//                   a warp's strip from scalar loads of lanes 0 and 31.  Needs n_phi % C == 0.
// k_sts_stage_map:  one column per thread, any n_phi (fallback for odd n_phi).
// MODEs as k_sts_stage (hft_kernels.cuh).
#pragma once
#include "hft_sts_blocked.cuh"

namespace hft {

template <typename real>
struct MapArgs {
    const real* NU;       // [R][nt+2][pitch], rows 0..nt used
    const double* capw;   // [R][2] sum_k (NU[f][k] + NU[f][k-1])/2 for f = 0 and f = nt, in fp64 from the stored values
    double capP[2];       // P dph / (theta_1 - theta_0), north / south cap
    int nparts_in;        // polar partial sums per row in part_in (the writer's CTAs along phi)
};

// One output value: L -> the stage's result (MODE 0: F = L, delta_1 = a L; 1/2: recurrence; 3: Euler).
template <typename real, int MODE>
__device__ __forceinline__ real map_combine(const StsArgs<real>& A, real L, real c, real d2v, real Fv) {
    if (MODE == 0) return A.a * L;
    if (MODE == 3) return c + A.a * L;
    return A.mu * c + A.nu * d2v + A.a * L + A.g * Fv;
}

template <typename real, int MODE>
__global__ void __launch_bounds__(TX) k_sts_stage_map(StsArgs<real> A, MapArgs<real> M, Tables<real> T, Geom G) {
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
    const real* nu = M.NU + base;
    const real half = (real)0.5;

    real n = (j0 > 0) ? in[(size_t)(j0 - 1) * G.pitch + kk] : (real)0;
    real c = in[(size_t)j0 * G.pitch + kk];
    // nu at face j0 - 1/2 (north face of the first row of this thread), columns k+1/2 and k-1/2
    real nNk = (j0 > 0) ? nu[(size_t)(j0 - 1) * G.pitch + kk] : (real)0;
    real nNw = (j0 > 0) ? nu[(size_t)(j0 - 1) * G.pitch + kw] : (real)0;
    double sumN = 0.0, sumS = 0.0;
    for (int j = j0; j < j1; j++) {
        const size_t off = base + (size_t)j * G.pitch + kk;
        real s = (j < G.nt + 1) ? in[(size_t)(j + 1) * G.pitch + kk] : (real)0;
        real nSk = (j < G.nt + 1) ? nu[(size_t)j * G.pitch + kk] : (real)0;   // face j + 1/2
        real nSw = (j < G.nt + 1) ? nu[(size_t)j * G.pitch + kw] : (real)0;
        real L;
        if (j == 0 || j == G.nt + 1) {
            const int pole = (j == 0) ? 0 : 1;
            double S = sum_partials(A.part_in + ((size_t)r * 2 + pole) * G.nbx, M.nparts_in);
            L = (real)(M.capP[pole] * (S - M.capw[2 * r + pole] * (double)c));
        } else {
            real w = in[(size_t)j * G.pitch + kw], e = in[(size_t)j * G.pitch + ke];
            const real gp = T.rdp[j] * T.rdp[j];
            const real as = half * (nSk + nSw) * (T.sth[j] * (T.rdt[j] * T.rdf[j]));
            const real an = half * (nNk + nNw) * (T.sth[j - 1] * (T.rdt[j] * T.rdf[j - 1]));
            const real ae = half * (nSk + nNk) * gp;
            const real aw = half * (nSw + nNw) * gp;
            L = (as * (s - c) - an * (c - n)) + (ae * (e - c) - aw * (c - w));
        }
        const real d2v = (MODE == 1 || MODE == 2) && A.use_d2 ? A.d2[off] : (real)0;
        const real Fv = (MODE == 1 || MODE == 2) ? A.F[off] : (real)0;
        const real out = map_combine<real, MODE>(A, L, c, d2v, Fv);
        if (live) {
            if (MODE == 0) A.F[off] = L;
            if (MODE == 2) A.Y0[off] += out;   // Y_s = Y_0 + delta_s
            else A.d2[off] = out;
        }
        // nu-weighted phi-sums of the rows adjacent to the caps (weights: face 1/2 = NU row 0, face nt+1/2 = NU row nt)
        if (j == 1) sumN = live ? 0.5 * ((double)nNk + (double)nNw) * (double)out : 0.0;
        if (j == G.nt) sumS = live ? 0.5 * ((double)nSk + (double)nSw) * (double)out : 0.0;
        n = c;
        c = s;
        nNk = nSk;
        nNw = nSw;
    }
    if (j0 <= 1 && 1 < j1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part_out[((size_t)r * 2 + 0) * G.nbx + blockIdx.x] = t;
    }
    if (j0 <= G.nt && G.nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part_out[((size_t)r * 2 + 1) * G.nbx + blockIdx.x] = t;
    }
}

constexpr int MAPV_RPT = 16;   // rows streamed per thread of the vector kernel

// MAP = false: the same 16-byte-vector stage kernel with the per-row coefficient tables of k_sts_stage (scalar nu or
// nu(theta)), identical arithmetic to k_sts_stage; NU / capw are not read, the polar sums are unweighted.
template <typename real, int MODE, bool MAP = true>
__global__ void __launch_bounds__(TX) k_sts_stage_mapv(StsArgs<real> A, MapArgs<real> M, Tables<real> T, Geom G) {
    constexpr int C = 16 / (int)sizeof(real);
    __shared__ double red[32];
    const int r = blockIdx.z, lane = threadIdx.x & 31;
    const int col = (blockIdx.x * TX + threadIdx.x) * C;   // first of this thread's C columns
    const bool live = col < G.np;                           // n_phi % C == 0: a live thread owns C valid columns
    const int cc = live ? col : 0;
    const int cw = (cc == 0) ? G.np - 1 : cc - 1;           // column west of the vector, periodic
    const int ce = (cc + C >= G.np) ? 0 : cc + C;           // column east of the vector, periodic
    const bool edgeW = lane == 0, edgeE = lane == 31 || cc + C >= G.np;   // neighbour not held by an adjacent lane
    const int j0 = blockIdx.y * MAPV_RPT;
    const int j1 = min(j0 + MAPV_RPT, G.nt + 2);
    const size_t base = (size_t)r * G.rstride;
    const real* in = A.in + base;
    const real* nu = M.NU + base;
    const real half = (real)0.5;
    const unsigned full = 0xffffffffu;

    real n[C], c[C], nN[C], nNw = (real)0;
#pragma unroll
    for (int q = 0; q < C; q++) { n[q] = (real)0; nN[q] = (real)0; }
    if (j0 > 0) {
        vload<real, C>(n, in + (size_t)(j0 - 1) * G.pitch + cc);
        if (MAP) vload<real, C>(nN, nu + (size_t)(j0 - 1) * G.pitch + cc);   // face j0 - 1/2
    }
    vload<real, C>(c, in + (size_t)j0 * G.pitch + cc);
    if (MAP) {
        nNw = __shfl_up_sync(full, nN[C - 1], 1);
        if (edgeW && j0 > 0) nNw = nu[(size_t)(j0 - 1) * G.pitch + cw];
    }
    const real* cpt = T.cp + (size_t)r * (G.nt + 2);
    const real* cmt = T.cm + (size_t)r * (G.nt + 2);
    const real* cft = T.cf + (size_t)r * (G.nt + 2);
    double sumN = 0.0, sumS = 0.0;
    for (int j = j0; j < j1; j++) {
        const size_t off = base + (size_t)j * G.pitch + cc;
        real s[C], nS[C], nSw = (real)0, out[C], Lv[C];
#pragma unroll
        for (int q = 0; q < C; q++) { s[q] = (real)0; nS[q] = (real)0; }
        if (j < G.nt + 1) {
            vload<real, C>(s, in + (size_t)(j + 1) * G.pitch + cc);
            if (MAP) vload<real, C>(nS, nu + (size_t)j * G.pitch + cc);   // face j + 1/2
        }
        real d2v[C], Fv[C];
#pragma unroll
        for (int q = 0; q < C; q++) { d2v[q] = (real)0; Fv[q] = (real)0; }
        if (MODE == 1 || MODE == 2) {
            if (A.use_d2) vload<real, C>(d2v, A.d2 + off);
            vload<real, C>(Fv, A.F + off);
        }
        if (MAP) {
            nSw = __shfl_up_sync(full, nS[C - 1], 1);
            if (edgeW && j < G.nt + 1) nSw = nu[(size_t)j * G.pitch + cw];
        }
        if (j == 0 || j == G.nt + 1) {
            const int pole = (j == 0) ? 0 : 1;
            double S = sum_partials(A.part_in + ((size_t)r * 2 + pole) * G.nbx, M.nparts_in);
            const real L = MAP ? (real)(M.capP[pole] * (S - M.capw[2 * r + pole] * (double)c[0]))
                               : (real)(T.capc[2 * r + pole] * (S - (double)G.np * (double)c[0]));
#pragma unroll
            for (int q = 0; q < C; q++) Lv[q] = L;
        } else {
            real w0 = __shfl_up_sync(full, c[C - 1], 1), e0 = __shfl_down_sync(full, c[0], 1);
            if (edgeW) w0 = in[(size_t)j * G.pitch + cw];
            if (edgeE) e0 = in[(size_t)j * G.pitch + ce];
            if (!MAP) {
                const real cp = cpt[j], cm = cmt[j], cf = cft[j];
#pragma unroll
                for (int q = 0; q < C; q++) {
                    const real w = q == 0 ? w0 : c[q > 0 ? q - 1 : 0];
                    const real e = q == C - 1 ? e0 : c[q < C - 1 ? q + 1 : 0];
                    Lv[q] = cp * (s[q] - c[q]) - cm * (c[q] - n[q]) + cf * ((e - (real)2 * c[q]) + w);
                }
            }
            if (MAP) {
            const real gp = T.rdp[j] * T.rdp[j];
            const real gs = T.sth[j] * (T.rdt[j] * T.rdf[j]), gn = T.sth[j - 1] * (T.rdt[j] * T.rdf[j - 1]);
#pragma unroll
            for (int q = 0; q < C; q++) {
                const real nSq_w = q == 0 ? nSw : nS[q > 0 ? q - 1 : 0];
                const real nNq_w = q == 0 ? nNw : nN[q > 0 ? q - 1 : 0];
                const real w = q == 0 ? w0 : c[q > 0 ? q - 1 : 0];
                const real e = q == C - 1 ? e0 : c[q < C - 1 ? q + 1 : 0];
                const real as = half * (nS[q] + nSq_w) * gs;
                const real an = half * (nN[q] + nNq_w) * gn;
                const real ae = half * (nS[q] + nN[q]) * gp;
                const real aw = half * (nSq_w + nNq_w) * gp;
                Lv[q] = (as * (s[q] - c[q]) - an * (c[q] - n[q])) + (ae * (e - c[q]) - aw * (c[q] - w));
            }
            }
        }
#pragma unroll
        for (int q = 0; q < C; q++) out[q] = map_combine<real, MODE>(A, Lv[q], c[q], d2v[q], Fv[q]);
        if (live) {
            if (MODE == 0) vstore<real, C>(A.F + off, Lv);
            if (MODE == 2) {
                real y[C];
                vload<real, C>(y, A.Y0 + off);
#pragma unroll
                for (int q = 0; q < C; q++) y[q] += out[q];
                vstore<real, C>(A.Y0 + off, y);
            } else {
                vstore<real, C>(A.d2 + off, out);
            }
        }
        if (j == 1 || j == G.nt) {   // nu-weighted phi-sums of the rows adjacent to the caps
            double t = 0.0;
#pragma unroll
            for (int q = 0; q < C; q++) {
                const real a = (j == 1) ? nN[q] : nS[q];
                const real b = (j == 1) ? (q == 0 ? nNw : nN[q > 0 ? q - 1 : 0]) : (q == 0 ? nSw : nS[q > 0 ? q - 1 : 0]);
                t += MAP ? 0.5 * ((double)a + (double)b) * (double)out[q] : (double)out[q];
            }
            if (!live) t = 0.0;
            if (j == 1) sumN = t;
            if (j == G.nt) sumS = t;   // nt == 1 is excluded by the API (n_theta >= 8)
        }
#pragma unroll
        for (int q = 0; q < C; q++) { n[q] = c[q]; c[q] = s[q]; nN[q] = nS[q]; }
        nNw = nSw;
    }
    if (j0 <= 1 && 1 < j1) {
        double t = block_sum(sumN, red);
        if (threadIdx.x == 0) A.part_out[((size_t)r * 2 + 0) * G.nbx + blockIdx.x] = t;
    }
    if (j0 <= G.nt && G.nt < j1) {
        double t = block_sum(sumS, red);
        if (threadIdx.x == 0) A.part_out[((size_t)r * 2 + 1) * G.nbx + blockIdx.x] = t;
    }
}

// nu-weighted phi-sums of rows 1 and nt of a field -> partials (the format the stage kernels above read and write).
template <typename real>
__global__ void __launch_bounds__(TX) k_polar_row_sums_map(const real* f, const real* NU, double* part, Geom G) {
    __shared__ double red[32];
    const int r = blockIdx.z, pole = blockIdx.y;
    const int k = blockIdx.x * TX + threadIdx.x;
    const int j = pole == 0 ? 1 : G.nt, face = pole == 0 ? 0 : G.nt;
    double v = 0.0;
    if (k < G.np) {
        const int kw = (k == 0) ? G.np - 1 : k - 1;
        const real* nu = NU + (size_t)r * G.rstride + (size_t)face * G.pitch;
        v = 0.5 * ((double)nu[k] + (double)nu[kw]) * (double)f[(size_t)r * G.rstride + (size_t)j * G.pitch + k];
    }
    double t = block_sum(v, red);
    if (threadIdx.x == 0) part[((size_t)r * 2 + pole) * G.nbx + blockIdx.x] = t;
}

}  // namespace hft
