// hft_sts_step.cuh -- host schedule of one temporally blocked STS step (Sec. 3.7.2):
// stage 1, an odd remainder stage, one shorter block for the rest of the remainder, then (s-1)/K blocks of K stages.
// A block runs in k_sts_upipe (coefficients through the uniform datapath, hft_sts_upipe.cuh) when the batch shares one
// coefficient table up to the factor nu_r, else in k_sts_pipe (per-realization tables through shared memory).
#pragma once
#include "hft_sts_pipe.cuh"
#include "hft_sts_upipe.cuh"

namespace hft {

// fp32 storage / fp64 arithmetic: compiled in hft_sts_mixed.cu
#define HFT_EXT(K)                                                                                                                      \
    extern template int sts_upipe_launch<float, double, K>(const StsBlockedPlan<float>&, const UPipePlan&, Tables<float>&, const Geom&, \
                                                           int, const float*, const float*, float*, float*, bool, int64_t*);
HFT_EXT(2) HFT_EXT(4) HFT_EXT(6) HFT_EXT(8)
#undef HFT_EXT

template <typename real, int K>
int sts_block_launch(const StsBlockedPlan<real>& P, Tables<real>& T, const Geom& G, int j0, const real* cur, const real* prev,
                     real* ocur, real* oprev, bool last, int64_t* launches) {
    if (P.up && P.up->ok) {
        if constexpr (sizeof(real) == 4) {
            if (P.up->mixed) return sts_upipe_launch<real, double, K>(P, *P.up, T, G, j0, cur, prev, ocur, oprev, last, launches);
        }
        return sts_upipe_launch<real, real, K>(P, *P.up, T, G, j0, cur, prev, ocur, oprev, last, launches);
    }
    return sts_pipe_launch<real, K>(P, T, G, j0, cur, prev, ocur, oprev, last, launches);
}

template <typename real>
int sts_blocked_step(StsBlockedPlan<real>& P, Tables<real>& T, const Geom& G, int64_t* launches) {
    const int K = P.kb, s = P.s;
    real* F = P.buf[0];
    real* b[4] = {P.buf[1], P.buf[2], P.buf[3], P.buf[4]};
    // stage 1 and an odd remainder stage run one stage per launch, in the 16-byte-vector kernel when n_phi is a multiple of
    // the vector width (its polar partials come in nbxv pieces per row), else in the one-column-per-thread kernel
    constexpr int CV = 16 / (int)sizeof(real);
    const int nbxv = (G.np / CV + TX - 1) / TX;
    dim3 g1(nbxv, (G.nt + 2 + MAPV_RPT - 1) / MAPV_RPT, G.nr), gs(G.nbx, 2, G.nr);
    k_polar_row_sums<real><<<gs, TX, 0, P.stream>>>(P.Y0, P.part[0], G);
    MapArgs<real> M;
    M.NU = nullptr; M.capw = nullptr; M.capP[0] = M.capP[1] = 0.0; M.nparts_in = G.nbx;
    StsArgs<real> a;
    a.F = F; a.Y0 = P.Y0; a.mu = 0; a.nu = 0; a.g = 0; a.use_d2 = 0;
    a.in = P.Y0; a.d2 = b[0]; a.part_in = P.part[0]; a.part_out = P.part[1]; a.a = (real)P.a[1];
    const bool vec = G.np % CV == 0;
    dim3 g1s(G.nbx, (G.nt + 2 + RPT - 1) / RPT, G.nr);
    if (vec) k_sts_stage_mapv<real, 0, false><<<g1, TX, 0, P.stream>>>(a, M, T, G);
    else k_sts_stage<real, 0><<<g1s, TX, 0, P.stream>>>(a, T, G);
    M.nparts_in = nbxv;
    *launches += 2;
    const int rem = (s - 1) % K;
    // the remainder: one un-blocked stage if it is odd, then ONE shorter block of rem - (rem & 1) stages
    const int rem_single = rem & 1;
    int icur = 0, iprev = 1, pin = 1;
    bool has_prev = false;
    for (int j = 2; j <= 1 + rem_single; j++) {
        a.in = b[icur]; a.d2 = b[iprev]; a.part_in = P.part[pin]; a.part_out = P.part[pin ^ 1];
        a.mu = (real)P.mu[j]; a.nu = (real)P.nu[j]; a.a = (real)P.a[j]; a.g = (real)P.g[j];
        a.use_d2 = has_prev;
        if (vec) k_sts_stage_mapv<real, 1, false><<<g1, TX, 0, P.stream>>>(a, M, T, G);
        else k_sts_stage<real, 1><<<g1s, TX, 0, P.stream>>>(a, T, G);
        *launches += 1;
        int t = icur; icur = iprev; iprev = t;
        has_prev = true;
        pin ^= 1;
    }
    int j0 = 1 + rem_single;  // stages done so far
    while (j0 < s) {
        const int kb = (rem - rem_single > 0 && j0 == 1 + rem_single) ? rem - rem_single : K;   // stages in this block
        // outputs go to the two buffers that are not inputs
        int o1 = -1, o2 = -1;
        for (int q = 0; q < 4; q++)
            if (q != icur && q != iprev) { if (o1 < 0) o1 = q; else o2 = q; }
        const bool last = (j0 + kb == s);
        if (!has_prev) {  // delta_0 = 0 is not stored: the blocked kernels read it, so write it once
            if (cudaMemsetAsync(b[iprev], 0, (size_t)G.nr * G.rstride * sizeof(real), P.stream) != cudaSuccess) return -1;
            has_prev = true;
        }
        int rc = 0;
        switch (kb) {
            case 2: rc = sts_block_launch<real, 2>(P, T, G, j0, b[icur], b[iprev], b[o1], b[o2], last, launches); break;
            case 4: rc = sts_block_launch<real, 4>(P, T, G, j0, b[icur], b[iprev], b[o1], b[o2], last, launches); break;
            case 6: rc = sts_block_launch<real, 6>(P, T, G, j0, b[icur], b[iprev], b[o1], b[o2], last, launches); break;
            default: rc = sts_block_launch<real, 8>(P, T, G, j0, b[icur], b[iprev], b[o1], b[o2], last, launches); break;
        }
        if (rc != 0) return rc;
        icur = o1; iprev = o2;
        j0 += kb;
    }
    return 0;
}

}  // namespace hft
