// hft_api.cu -- C ABI (include/hft.h), context, host-side tables and the per-step launch schedule.
//
// Host work per hft_step: look up (or build) the STS stage scalars for (dt, s), then enqueue kernels on
// the caller's stream; nothing synchronises.  All floating-point work on the fields happens in the
// kernels of hft_kernels.cuh / hft_sts_blocked.cuh.  Tables are formed in fp64 and rounded once to the
// state precision.  Citations: /root/reference/PAPER.md.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <cmath>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/hft.h"
#include "hft_kernels.cuh"
#include "hft_sts_blocked.cuh"
#include "hft_sts_map.cuh"
#include "hft_sts_step.cuh"
#include "hft_sts_mpipe.cuh"

// The temporally blocked STS step (all k_sts_pipe / k_sts_upipe / k_sts_capseq instantiations) is compiled in its own
// translation units (hft_sts_f64.cu, hft_sts_f32.cu, hft_sts_mixed.cu), so that the units build in parallel.
extern template int hft::sts_blocked_step<double>(hft::StsBlockedPlan<double>&, hft::Tables<double>&, const hft::Geom&, int64_t*);
extern template int hft::sts_blocked_step<float>(hft::StsBlockedPlan<float>&, hft::Tables<float>&, const hft::Geom&, int64_t*);

using namespace hft;

namespace {

constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kMsToRsHr = 5.172413793103448e-6;    // PAPER.md:298  m/s -> R_sun/hr
constexpr double kKm2sToRs2Hr = 7.43162901307967e-9;  // PAPER.md:298  km^2/s -> R_sun^2/hr
constexpr int kNumArrays = 6;                         // state + 5 stage arrays
constexpr int kNumRfeArrays = 2;                      // random flux emergence: the two current source maps (hft_options.rfe)
constexpr int kNumAttArrays = 6;                      // flow attenuation: VT, VP, LMt, LPt, LMp, LPp (hft_options.flow_attenuation)
constexpr int kNumMapArrays = 1;                      // nu(theta, phi) on the half-half grid (hft_options.diffusivity_map)
constexpr int kProfEvents = 256;

struct StsCoef {  // per-stage scalars of Sec. 3.7.2 schemes, index 0..s
    int scheme = 0, s = 0;
    double dt = 0.0, w1 = 0.0;
    std::vector<double> mu, nu, a, g;  // mu_j, nu_j, mut_j*dt, mut_j*b_{j-1}*dt ; a[1] = mut_1*dt
};

}  // namespace

struct hft_ctx {
    hft_grid grid;
    hft_options opt;
    int nr = 0, dev = 0;
    cudaStream_t stream = nullptr;
    Geom G;
    size_t arr_bytes = 0;
    char* arr[kNumArrays] = {nullptr};
    int i_state = 0;  // index of the array that currently holds the state
    // flow attenuation (Eq. 5): field-shaped speed arrays behind the ring, B0 per realization, "speeds are current" flag
    char* att[kNumAttArrays] = {nullptr};
    std::vector<double> B0;
    void* d_B0 = nullptr;
    bool att_any = false, att_ready = false;
    // random flux emergence (Sec. 2.4): the two source maps behind the ring, the run clock and the map schedule
    char* rfe_map[kNumRfeArrays] = {nullptr};
    int rfe_model = 0;
    double rfe_flux = 0.0, rfe_tau = 0.0, rfe_t1 = 0.0, time = 0.0;
    uint64_t rfe_seed = 0;
    uint32_t rfe_next = 2;
    // nu(theta, phi) (Eq. 27-28): the NU array behind the ring; per realization: "a map was set", the Gershgorin diagonal
    // maximum of its matrix, and the two polar weight sums (device copy d_capw)
    char* numap = nullptr;
    bool map_any = false;
    std::vector<char> map_set;
    std::vector<double> map_diag, capw;
    double* d_capw = nullptr;
    // host tables (fp64)
    double dth = 0, dph = 0, P = 0, Apole = 0;   // uniform spacings; P, Apole: north cap (uniform grid: both)
    std::vector<double> st, sth;      // sin(theta_j) [nt+2], sin(theta_{j+1/2}) [nt+1]
    // theta grid (reading U33): nodes, half grid, cell widths (caps: half width), node spacing across the faces;
    // on the default uniform grid dthc / dthf hold the one value dth
    std::vector<double> th, thf, dthc, dthf;
    double PN = 0, PS = 0, ApoleN = 0, ApoleS = 0;
    std::vector<double> wm, wp;       // [nt+1][5] App. B D-factors per theta-face (oracle make_grid has the same list)
    bool uniform = true;
    std::vector<hft_params> params;   // as given to hft_create (the analytic flow tables follow the grid)
    std::vector<double> nu;           // [R] R_sun^2/hr
    std::vector<double> nuf;          // [R][nt+1] nu at the theta-faces (= nu unless a latitude profile was set; Eq. 6-7)
    std::vector<double> vt, om;       // [R][nt+1] R_sun/hr at faces, [R][nt+2] rad/hr at rows
    // device tables
    char* d_tab = nullptr;
    size_t tab_bytes = 0;
    Tables<float> Tf;
    Tables<double> Td;
    double* d_part[2] = {nullptr, nullptr};  // polar phi-sum partials, double-buffered [R][2][nbx]
    double* d_fluxpart = nullptr;            // [R][RED_CTAS][2]
    double* d_capinfo = nullptr;             // [R][2][2]
    double* d_scale = nullptr;               // [R]
    double* d_diag = nullptr;                // [R][4]
    double* d_zmean = nullptr;               // blocked STS: zonal partial sums (see hft_sts_blocked.cuh)
    double* d_capseq = nullptr;              // blocked STS: cap values per stage
    double* d_kappa = nullptr;               // k_sts_upipe: w1 dt nu_r per realization
    double* d_mscratch = nullptr;            // k_sts_mcapseq: polar-band level buffers, allocated on first use
    double* h_diag = nullptr;                // pinned
    double *d_extpart = nullptr, *d_ext = nullptr, *h_ext = nullptr;   // hft_diagnostics_ext, allocated on first use
    int64_t launches = 0;
    StsCoef coef;
    // uniform-coefficient blocked kernel (hft_sts_upipe.cuh): the shared table sigma*(cm, cp, cf, -cd)/nu_r, its owner key
    UPipePlan up;
    std::vector<unsigned char> utab;   // [nt][32 bytes]
    std::vector<double> nu_scale;      // [R]: nuf[r][f] = nu_scale[r] * nu_shape[f] when shape_common
    std::vector<double> nu_shape;      // [nt+1]
    bool shape_common = true;
    uint64_t id = 0, tab_version = 1;  // tab_version: bumped whenever the diffusion tables change
    uint64_t up_version = 0;           // tab_version/scheme/s/dt the table in `utab` was built for
    int up_scheme = 0, up_s = 0;
    double up_dt = 0.0;
    // sampled kernel timing
    int prof_which = 0;
    int prof_n = 0;
    int64_t prof_stages = 0;
    int64_t prof_seen = 0;
    cudaEvent_t prof_ev[2 * kProfEvents];
    bool prof_ev_made = false;
    std::string cuda_err;
    bool fp64() const { return grid.dtype == 1; }
};

namespace {

// every entry point runs on the device the context was created on, whatever device is current in the calling thread
struct DevGuard {
    int prev = -1;
    bool sw = false;
    explicit DevGuard(const hft_ctx* c) {
        if (!c) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != c->dev) sw = cudaSetDevice(c->dev) == cudaSuccess;
    }
    ~DevGuard() { if (sw) cudaSetDevice(prev); }
};

int cuda_fail(hft_ctx* c, cudaError_t e, const char* what) {
    if (c) c->cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    return HFT_ERR_CUDA;
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);    \
    } while (0)

int check_launch(hft_ctx* c) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "kernel launch");
    return HFT_OK;
}

size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int pitch_for(int np, int dtype) {
    size_t w = dtype == 1 ? 8 : 4;
    return (int)(round_up((size_t)np * w, 128) / w);  // rows start on 128-byte lines
}

bool valid_grid(const hft_grid* g) {
    return g && g->n_theta >= 8 && g->n_phi >= 8 && (g->dtype == 0 || g->dtype == 1) && g->reserved == 0 &&
           g->n_theta + 2 <= 65535 && g->n_phi <= (1 << 20) && g->radius_cm > 0.0;   // rows ride in gridDim.y (16 bits)
}

bool valid_params(const hft_params* p, int n) {
    for (int r = 0; r < n; r++) {
        const double v[7] = {p[r].eta_km2_s, p[r].d0, p[r].d2, p[r].d4, p[r].m1, p[r].m3, p[r].m5};
        for (double x : v)
            if (!std::isfinite(x)) return false;
        if (p[r].eta_km2_s < 0.0) return false;
    }
    return true;
}

hft_options default_options() {
    hft_options o;
    memset(&o, 0, sizeof(o));
    o.adv_flux = 2; o.adv_time = 4; o.diff_time = 3; o.sts_stages = 0; o.sts_block = 0;
    return o;
}

int extra_arrays(const hft_options* o) {
    return o ? (o->flow_attenuation ? kNumAttArrays : 0) + (o->rfe ? kNumRfeArrays : 0) + (o->diffusivity_map ? kNumMapArrays : 0) : 0;
}

bool valid_options(const hft_options* o) {
    if (o->adv_flux < 0 || o->adv_flux > 2) return false;
    if (o->adv_time != 1 && o->adv_time != 3 && o->adv_time != 4) return false;
    if (o->diff_time < 0 || o->diff_time > 3) return false;
    if (o->sts_stages != 0 && o->sts_stages < 2) return false;
    if (o->strang != 0 && o->strang != 1) return false;
    if (o->flow_attenuation != 0 && o->flow_attenuation != 1) return false;
    if (o->rfe != 0 && o->rfe != 1) return false;
    if (o->diffusivity_map != 0 && o->diffusivity_map != 1) return false;
    if (o->sts_block < 0 || o->sts_block > STS_KMAX || (o->sts_block > 1 && (o->sts_block & 1))) return false;
    if (o->f32_arith != 0 && o->f32_arith != 1) return false;
    if (o->sts_kernel < 0 || o->sts_kernel > 2) return false;
    return true;
}

// ---------------------------------------------------------------- host tables (fp64)

// Grid metric (App. A :642-646).  1 - cos(x) is formed as 2 sin^2(x/2).
void build_metric(hft_ctx* c, const double* theta_nodes) {
    const int nt = c->G.nt;
    c->dth = kPi / (double)(nt + 1);
    c->dph = 2.0 * kPi / (double)c->G.np;
    c->uniform = theta_nodes == nullptr;
    c->st.resize(nt + 2); c->sth.resize(nt + 1);
    c->th.resize(nt + 2); c->thf.resize(nt + 1); c->dthc.resize(nt + 2); c->dthf.resize(nt + 1);
    if (c->uniform) {
        for (int j = 0; j <= nt + 1; j++) { c->th[j] = c->dth * (double)j; c->dthc[j] = c->dth; }
        for (int j = 0; j <= nt; j++) { c->thf[j] = c->dth * ((double)j + 0.5); c->dthf[j] = c->dth; }
        c->dthc[0] = c->dthc[nt + 1] = 0.5 * c->dth;
    } else {
        for (int j = 0; j <= nt + 1; j++) c->th[j] = theta_nodes[j];
        for (int j = 0; j <= nt; j++) { c->thf[j] = 0.5 * (c->th[j] + c->th[j + 1]); c->dthf[j] = c->th[j + 1] - c->th[j]; }
        for (int j = 1; j <= nt; j++) c->dthc[j] = c->thf[j] - c->thf[j - 1];
        c->dthc[0] = c->thf[0] - c->th[0];
        c->dthc[nt + 1] = c->th[nt + 1] - c->thf[nt];
    }
    for (int j = 0; j <= nt + 1; j++) c->st[j] = sin(c->th[j]);
    for (int j = 0; j <= nt; j++) c->sth[j] = sin(c->thf[j]);
    for (int pole = 0; pole < 2; pole++) {   // App. A (:642-646) with the cap's own half width x
        const double x = c->dthc[pole ? nt + 1 : 0], q = sin(0.5 * x);
        const double A = 2.0 * kPi * (2.0 * q * q), P = sin(x) / A;
        if (pole) { c->ApoleS = A; c->PS = P; } else { c->ApoleN = A; c->PN = P; }
    }
    c->Apole = c->ApoleN; c->P = c->PN;
    // App. B (:662-680) D-factors per theta-face f (cell i = f+1, face i-1/2), Delta x = the cell widths; uniform: 1/2, 1/3, 2/3
    c->wm.assign(5 * (size_t)(nt + 1), 0.5); c->wp.assign(5 * (size_t)(nt + 1), 0.5);
    for (int f = 0; f <= nt; f++) {
        double *m = &c->wm[5 * (size_t)f], *q = &c->wp[5 * (size_t)f];
        m[3] = q[3] = 1.0 / 3.0; m[4] = q[4] = 2.0 / 3.0;
        if (c->uniform || f < 2 || f > nt - 2) continue;
        const int i = f + 1;
        const double xm2 = c->dthc[i - 2], xm1 = c->dthc[i - 1], x0 = c->dthc[i], xp1 = c->dthc[i + 1];
        m[0] = xm1 / (xm1 + xm2); m[1] = x0 / (x0 + xm1); m[2] = xm1 / (xm1 + x0);
        m[3] = x0 / (xm2 + xm1 + x0); m[4] = (xm1 + xm2) / (xm2 + xm1 + x0);
        q[0] = x0 / (x0 + xp1); q[1] = xm1 / (xm1 + x0); q[2] = x0 / (x0 + xm1);
        q[3] = xm1 / (xm1 + x0 + xp1); q[4] = (x0 + xp1) / (xm1 + x0 + xp1);
    }
}

// Analytic flows, Eq. 3-4 (:78-86), converted with :298.
void build_flow(hft_ctx* c, int r, const hft_params& p) {
    const int nt = c->G.nt;
    c->nu[r] = p.eta_km2_s * kKm2sToRs2Hr;
    for (int f = 0; f <= nt; f++) {
        const double th = c->thf[f], x = cos(th);
        c->vt[(size_t)r * (nt + 1) + f] = -(p.m1 * x + p.m3 * x * x * x + p.m5 * x * x * x * x * x) * sin(th) * kMsToRsHr;
    }
    for (int j = 0; j <= nt + 1; j++) {
        const double x = cos(c->th[j]), x2 = x * x;
        c->om[(size_t)r * (nt + 2) + j] = (p.d0 + p.d2 * x2 + p.d4 * x2 * x2) * kMsToRsHr;
    }
}

template <typename real>
struct HostTab {
    std::vector<real> cp, cm, cf, cd, c4, lm, lp, vtf, pm, pp, sth, rdt, rdp, rdf, wmp;
    std::vector<double> capc, dA;
};

template <typename real>
void fill_tables(const hft_ctx* c, HostTab<real>& H) {
    const int nt = c->G.nt, R = c->nr;
    const size_t n2 = (size_t)R * (nt + 2);
    H.cp.assign(n2, 0); H.cm.assign(n2, 0); H.cf.assign(n2, 0); H.cd.assign(n2, 0); H.lm.assign(n2, 0); H.lp.assign(n2, 0);
    H.pm.assign(n2, 0); H.pp.assign(n2, 0); H.c4.assign(4 * n2, 0);
    H.vtf.assign((size_t)R * (nt + 1), 0);
    H.sth.resize(nt + 1); H.rdt.assign(nt + 2, 0); H.rdp.assign(nt + 2, 0);
    H.capc.resize(2 * R); H.dA.resize(nt + 2);
    for (int f = 0; f <= nt; f++) H.sth[f] = (real)c->sth[f];
    for (int j = 1; j <= nt; j++) {
        H.rdt[j] = (real)(1.0 / (c->st[j] * c->dthc[j]));
        H.rdp[j] = (real)(1.0 / (c->st[j] * c->dph));
        H.dA[j] = c->st[j] * c->dthc[j] * c->dph;
    }
    H.dA[0] = c->ApoleN; H.dA[nt + 1] = c->ApoleS;
    H.rdf.resize(nt + 1);
    H.wmp.assign(16 * (size_t)(nt + 1), 0);   // per face: wm[0..4], eps_w, 2 pad, wp[0..4], 3 pad
    for (int f = 0; f <= nt; f++) {
        H.rdf[f] = (real)(1.0 / c->dthf[f]);
        for (int q = 0; q < 5; q++) { H.wmp[16 * (size_t)f + q] = (real)c->wm[5 * (size_t)f + q]; H.wmp[16 * (size_t)f + 8 + q] = (real)c->wp[5 * (size_t)f + q]; }
        H.wmp[16 * (size_t)f + 5] = (real)c->dthf[f];   // eps_w = h, the local spacing (:670)
    }
    for (int r = 0; r < R; r++) {
        const double* nuf = &c->nuf[(size_t)r * (nt + 1)];
        const double* vt = &c->vt[(size_t)r * (nt + 1)];
        const double* om = &c->om[(size_t)r * (nt + 2)];
        H.capc[2 * r] = c->PN * (nuf[0] / c->dthf[0]) * c->dph;        // north: nu at face 1/2
        H.capc[2 * r + 1] = c->PS * (nuf[nt] / c->dthf[nt]) * c->dph;   // south: nu at face nt+1/2
        for (int f = 0; f <= nt; f++) H.vtf[(size_t)r * (nt + 1) + f] = (real)vt[f];
        for (int j = 0; j <= nt + 1; j++) {
            const size_t i = (size_t)r * (nt + 2) + j;
            if (j >= 1 && j <= nt) {  // Eq. 28, uniform spacing, nu = nu(theta) on the half grid (:288)
                H.cp[i] = (real)(nuf[j] * c->sth[j] / (c->st[j] * c->dthc[j] * c->dthf[j]));
                H.cm[i] = (real)(nuf[j - 1] * c->sth[j - 1] / (c->st[j] * c->dthc[j] * c->dthf[j - 1]));
                H.cf[i] = (real)(0.5 * (nuf[j] + nuf[j - 1]) / (c->st[j] * c->st[j] * c->dph * c->dph));
                H.cd[i] = (real)((double)H.cp[i] + (double)H.cm[i] + 2.0 * (double)H.cf[i]);
                H.c4[4 * i + 0] = H.cm[i]; H.c4[4 * i + 1] = H.cp[i]; H.c4[4 * i + 2] = H.cf[i]; H.c4[4 * i + 3] = H.cd[i];
            }
            // LLF (B2 :684) with alpha_j = max |v| over faces j-5/2 .. j+5/2 that exist (:689)
            double al = 0.0;
            for (int f = j - 3; f <= j + 2; f++)
                if (f >= 0 && f <= nt) al = fmax(al, fabs(vt[f]));
            const real alr = (real)al;
            const real vm = (j >= 1) ? (real)vt[j - 1] : (real)0;  // v_{j-1/2}
            const real vp = (j <= nt) ? (real)vt[j] : (real)0;     // v_{j+1/2}
            H.lm[i] = (real)0.5 * (vm + alr);
            H.lp[i] = (real)0.5 * (vp - alr);
            const real vphi = (real)(om[j] * c->st[j]);
            const real aphi = (real)fabs(om[j] * c->st[j]);
            H.pm[i] = (real)0.5 * (vphi + aphi);
            H.pp[i] = (real)0.5 * (vphi - aphi);
        }
    }
}

template <typename real>
int upload_tables(hft_ctx* c, Tables<real>& T) {
    HostTab<real> H;
    fill_tables<real>(c, H);
    const int nt = c->G.nt, R = c->nr;
    const size_t n2 = (size_t)R * (nt + 2) * sizeof(real), n1 = (size_t)R * (nt + 1) * sizeof(real);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = round_up(off + bytes, 256); return o; };
    size_t o_cp = take(n2), o_cm = take(n2), o_cf = take(n2), o_cd = take(n2), o_c4 = take(4 * n2), o_lm = take(n2), o_lp = take(n2), o_pm = take(n2), o_pp = take(n2);
    size_t o_vtf = take(n1), o_sth = take((nt + 1) * sizeof(real)), o_rdt = take((nt + 2) * sizeof(real)), o_rdp = take((nt + 2) * sizeof(real));
    size_t o_capc = take(2 * R * sizeof(double)), o_dA = take((nt + 2) * sizeof(double));
    size_t o_rdf = take((nt + 1) * sizeof(real)), o_wmp = take(16 * (size_t)(nt + 1) * sizeof(real)), o_th = take((nt + 2) * sizeof(double));
    if (!c->d_tab) {
        c->tab_bytes = off;
        CK(cudaMalloc((void**)&c->d_tab, c->tab_bytes));
    }
    char* d = c->d_tab;
    auto up = [&](size_t o, const void* src, size_t bytes) { return cudaMemcpyAsync(d + o, src, bytes, cudaMemcpyHostToDevice, c->stream); };
    CK(up(o_cp, H.cp.data(), n2)); CK(up(o_cm, H.cm.data(), n2)); CK(up(o_cf, H.cf.data(), n2)); CK(up(o_cd, H.cd.data(), n2)); CK(up(o_c4, H.c4.data(), 4 * n2));
    CK(up(o_lm, H.lm.data(), n2)); CK(up(o_lp, H.lp.data(), n2)); CK(up(o_pm, H.pm.data(), n2)); CK(up(o_pp, H.pp.data(), n2));
    CK(up(o_vtf, H.vtf.data(), n1)); CK(up(o_sth, H.sth.data(), (nt + 1) * sizeof(real)));
    CK(up(o_rdt, H.rdt.data(), (nt + 2) * sizeof(real))); CK(up(o_rdp, H.rdp.data(), (nt + 2) * sizeof(real)));
    CK(up(o_capc, H.capc.data(), 2 * R * sizeof(double))); CK(up(o_dA, H.dA.data(), (nt + 2) * sizeof(double)));
    CK(up(o_rdf, H.rdf.data(), (nt + 1) * sizeof(real))); CK(up(o_wmp, H.wmp.data(), 16 * (size_t)(nt + 1) * sizeof(real)));
    CK(up(o_th, c->th.data(), (nt + 2) * sizeof(double)));
    CK(cudaStreamSynchronize(c->stream));  // H goes out of scope
    T.cp = (const real*)(d + o_cp); T.cm = (const real*)(d + o_cm); T.cf = (const real*)(d + o_cf); T.cd = (const real*)(d + o_cd); T.c4 = (const real*)(d + o_c4);
    T.lm = (const real*)(d + o_lm); T.lp = (const real*)(d + o_lp); T.pm = (const real*)(d + o_pm); T.pp = (const real*)(d + o_pp);
    T.vtf = (const real*)(d + o_vtf); T.sth = (const real*)(d + o_sth); T.rdt = (const real*)(d + o_rdt); T.rdp = (const real*)(d + o_rdp);
    T.capc = (const double*)(d + o_capc); T.dA = (const double*)(d + o_dA);
    T.rdf = (const real*)(d + o_rdf); T.wmp = (const real*)(d + o_wmp); T.th = (const double*)(d + o_th);
    T.adv_capc[0] = c->PN * c->dph; T.adv_capc[1] = c->PS * c->dph;
    T.nonuniform = c->uniform ? 0 : 1;
    T.eps_t = (real)c->dth;
    T.eps_p = (real)c->dph;
    return HFT_OK;
}

int upload_all_tables(hft_ctx* c) { return c->fp64() ? upload_tables<double>(c, c->Td) : upload_tables<float>(c, c->Tf); }

// ---------------------------------------------------------------- step-size helpers (row A9)

// Eq. 26 (:430) with flanking-face maxima (:406); |v_phi| / (sin(theta) dph) = |Omega| / dph.
double adv_dt_limit(const hft_ctx* c) {
    const int nt = c->G.nt;
    double best = INFINITY;
    for (int r = 0; r < c->nr; r++)
        for (int j = 1; j <= nt; j++) {
            const double a = fmax(fabs(c->vt[(size_t)r * (nt + 1) + j - 1]), fabs(c->vt[(size_t)r * (nt + 1) + j]));
            const double rate = a / c->dthc[j] + fabs(c->om[(size_t)r * (nt + 2) + j]) / c->dph;
            if (rate > 0.0) best = fmin(best, 1.0 / rate);
        }
    return best;
}

// Gershgorin bound: rho <= 2 max|diag|; explicit Euler limit 2/rho, with nu = max_r nu_r (:448).
double diff_dt_expl(const hft_ctx* c) {
    const int nt = c->G.nt;
    double d = 0.0;
    for (int r = 0; r < c->nr; r++) {
        if (c->map_set[r]) {   // nu(theta, phi): max |a_{j,k}| over every cell and both caps, found when the map was set
            d = fmax(d, c->map_diag[r]);
            continue;
        }
        const double* nuf = &c->nuf[(size_t)r * (nt + 1)];
        d = fmax(d, fmax(2.0 * kPi * c->PN * nuf[0] / c->dthf[0], 2.0 * kPi * c->PS * nuf[nt] / c->dthf[nt]));  // cap row diagonals
        for (int j = 1; j <= nt; j++) {
            const double t = (nuf[j] * c->sth[j] / c->dthf[j] + nuf[j - 1] * c->sth[j - 1] / c->dthf[j - 1]) / (c->st[j] * c->dthc[j]) +
                             (nuf[j] + nuf[j - 1]) / (c->st[j] * c->st[j] * c->dph * c->dph);
            d = fmax(d, t);
        }
    }
    return d > 0.0 ? 1.0 / d : INFINITY;
}

double sts_span(int scheme, int s) {  // dt / dt_expl reachable with s stages
    const double x = (double)s;
    return scheme == 2 ? (x * x + x - 2.0) / 4.0 : (x * x + 3.0 * x - 4.0) / 6.0;
}

int sts_stages_for(const hft_ctx* c, int scheme, double dt) {
    const double lim = diff_dt_expl(c);
    int s = 2;
    while (dt > lim * sts_span(scheme, s)) {
        if (++s > 10000000) return -1;
    }
    return s;
}

// Stage scalars.  RKL2: shifted Legendre (Meyer et al. 2014); RKG2(3/2): shifted Gegenbauer lambda = 3/2
// (Skaras et al. 2021); both named in PAPER.md:470-474, coefficients per DESIGN.md reading U7.
void build_sts_coef(StsCoef& K, int scheme, int s, double dt) {
    if (K.scheme == scheme && K.s == s && K.dt == dt) return;
    K.scheme = scheme; K.s = s; K.dt = dt;
    K.mu.assign(s + 1, 0); K.nu.assign(s + 1, 0); K.a.assign(s + 1, 0); K.g.assign(s + 1, 0);
    auto b = [&](int j) {
        const double x = (double)(j < 2 ? 2 : j);
        return scheme == 2 ? (x * x + x - 2.0) / (2.0 * x * (x + 1.0)) : 2.0 * (x - 1.0) * (x + 4.0) / (3.0 * x * (x + 3.0));
    };
    const double S = (double)s;
    const double w1 = scheme == 2 ? 4.0 / (S * S + S - 2.0) : 6.0 / ((S - 1.0) * (S + 4.0));
    K.w1 = w1;
    K.a[1] = b(1) * w1 * dt;
    for (int j = 2; j <= s; j++) {
        const double x = (double)j;
        const double Aj = scheme == 2 ? (2.0 * x - 1.0) / x : (2.0 * x + 1.0) / (x + 2.0);
        const double Bj = scheme == 2 ? (x - 1.0) / x : (x - 1.0) / (x + 2.0);
        K.mu[j] = Aj * b(j) / b(j - 1);
        K.nu[j] = -Bj * b(j) / b(j - 2);
        const double mut = K.mu[j] * w1;
        K.a[j] = mut * dt;
        K.g[j] = mut * b(j - 1) * dt;
    }
}

// The shared coefficient table of k_sts_upipe (hft_sts_upipe.cuh): (cm, cp, cf, -cd)_j / nu_r for rows 1..nt, in the
// arithmetic type of the kernel (fp64, or duplicated fp32 pairs), and kappa_r = w1 dt nu_r.  Usable when every
// realization's diffusivity is nu_scale[r] * nu_shape(theta) and the table fits the constant bank; rebuilt when
// (tables, scheme, s, dt) change.
std::atomic<uint64_t> g_utab_key{1};

int prepare_upipe(hft_ctx* c, int scheme, int s, double dt) {
    UPipePlan& up = c->up;
    if (c->up_version == c->tab_version && c->up_scheme == scheme && c->up_s == s && c->up_dt == dt) return HFT_OK;
    c->up_version = c->tab_version; c->up_scheme = scheme; c->up_s = s; c->up_dt = dt;
    up.ok = false;
    const int nt = c->G.nt;
    // default (0): k_sts_upipe wherever the block arithmetic is fp64 -- fp64 states, and fp32 storage with fp64 block
    // arithmetic (f32_arith = 0), where it is the only kernel; fp32 arithmetic stays with k_sts_pipe (FFMA2), measured equal
    const bool want_mixed = !c->fp64() && c->opt.f32_arith == 0;
    const bool want = c->opt.sts_kernel == 2 || (c->opt.sts_kernel == 0 && (want_mixed || c->fp64()));
    if (!want || !c->shape_common || nt > UTAB_MAX_ROWS) return HFT_OK;
    for (int r = 0; r < c->nr; r++)
        if (!(c->nu_scale[r] >= 0.0) || !std::isfinite(c->nu_scale[r])) return HFT_OK;
    const bool dbl = c->fp64() || want_mixed;
    up.mixed = want_mixed;
    c->utab.assign((size_t)nt * UTAB_ROW_BYTES, 0);
    for (int j = 1; j <= nt; j++) {
        const double cm = c->nu_shape[j - 1] * c->sth[j - 1] / (c->st[j] * c->dthc[j] * c->dthf[j - 1]);
        const double cp = c->nu_shape[j] * c->sth[j] / (c->st[j] * c->dthc[j] * c->dthf[j]);
        const double cf = 0.5 * (c->nu_shape[j] + c->nu_shape[j - 1]) / (c->st[j] * c->st[j] * c->dph * c->dph);
        unsigned char* row = &c->utab[(size_t)(j - 1) * UTAB_ROW_BYTES];
        if (dbl) {
            double v[4] = {cm, cp, cf, 0.0};
            v[3] = -(v[0] + v[1] + 2.0 * v[2]);
            memcpy(row, v, sizeof(v));
        } else {
            const float a = (float)cm, b = (float)cp, f = (float)cf;
            const float d = -(float)((double)a + (double)b + 2.0 * (double)f);
            const float v[8] = {a, a, b, b, f, f, d, d};
            memcpy(row, v, sizeof(v));
        }
    }
    std::vector<double> kap(c->nr);
    for (int r = 0; r < c->nr; r++) kap[r] = c->coef.w1 * dt * c->nu_scale[r];
    CK(cudaStreamSynchronize(c->stream));   // d_kappa may still be read by enqueued work
    CK(cudaMemcpy(c->d_kappa, kap.data(), (size_t)c->nr * sizeof(double), cudaMemcpyHostToDevice));
    up.h_table = c->utab.data();
    up.d_kappa = c->d_kappa;
    up.key = g_utab_key.fetch_add(1);
    up.ok = true;
    return HFT_OK;
}

// ---------------------------------------------------------------- launch helpers

template <typename real> Tables<real>& tables_of(hft_ctx* c);
template <> Tables<float>& tables_of<float>(hft_ctx* c) { return c->Tf; }
template <> Tables<double>& tables_of<double>(hft_ctx* c) { return c->Td; }

template <typename real> real* arr_of(hft_ctx* c, int i) { return (real*)c->arr[i]; }

void prof_begin(hft_ctx* c, int cls, bool& armed) {
    armed = false;
    if (c->prof_which != cls || c->prof_n >= kProfEvents) return;
    if ((c->prof_seen++ & 15) != 0) return;  // sample every 16th launch of the class
    cudaEventRecord(c->prof_ev[2 * c->prof_n], c->stream);
    armed = true;
}
void prof_end(hft_ctx* c, bool armed, int stages) {
    if (!armed) return;
    c->prof_stages += stages;
    cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], c->stream);
    c->prof_n++;
}

// one advection step (A of Eq. 21): SSPRK stages, each = stage kernel + cap kernel
template <typename real>
int advect(hft_ctx* c, double dt) {
    const Geom& G = c->G;
    Tables<real>& T = tables_of<real>(c);
    // scratch: the two arrays after the state in ring order
    const int is = c->i_state, ia = (is + 1) % kNumArrays, ib = (is + 2) % kNumArrays;
    real *S = arr_of<real>(c, is), *A = arr_of<real>(c, ia), *B = arr_of<real>(c, ib);
    struct St { const real* in; const real* fn; real* out; double ca, cb, cc; };
    std::vector<St> sts;
    if (c->opt.adv_time == 1) {
        sts.push_back({S, nullptr, A, 0.0, 1.0, 1.0});
    } else if (c->opt.adv_time == 3) {  // SSPRK(3,3) :412-416
        sts.push_back({S, nullptr, A, 0.0, 1.0, 1.0});
        sts.push_back({A, S, B, 0.75, 0.25, 0.25});
        sts.push_back({B, S, A, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0});
    } else {  // SSPRK(4,3) Eq. 25 :418-424
        sts.push_back({S, nullptr, A, 0.0, 1.0, 0.5});
        sts.push_back({A, nullptr, B, 0.0, 1.0, 0.5});
        sts.push_back({B, S, A, 2.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0});
        sts.push_back({A, nullptr, B, 0.0, 1.0, 0.5});
    }
    dim3 g(G.nbxa, (G.nt + RPT - 1) / RPT, c->nr), gc(G.nbx, 2, c->nr);
    const int nbxt = (G.np + ATT_COLS - 1) / ATT_COLS;   // k_adv_stage_u / k_adv_stage_att_u: 28 columns per warp
    // rows per thread: 32 on a full batch (the first face of a strip is evaluated without writing a row); on a small batch
    // shorter strips, so that every SM still gets several CTAs (one 510 x 1023 realization: 160 CTAs at 32 rows, 640 at 8)
    int rpt = ADV_RPT;
    while (rpt > 8 && (long)nbxt * ((G.nt + rpt - 1) / rpt) * c->nr < 148L * 8) rpt /= 2;
    dim3 gt(nbxt, (G.nt + rpt - 1) / rpt, c->nr);
    real* att[kNumAttArrays] = {nullptr};
    if (c->att_any) {
        for (int i = 0; i < kNumAttArrays; i++) att[i] = (real*)c->att[i];
        if (!c->att_ready) {   // once per time step, from the field at its start (reading U23)
            dim3 ga(G.nbx, G.nt + 2, c->nr);
            k_att_faces<real><<<ga, TX, 0, c->stream>>>(S, (const real*)c->d_B0, T, G, att[0], att[1]);
            k_att_halfspeeds<real><<<ga, TX, 0, c->stream>>>(att[0], att[1], G, att[2], att[3], att[4], att[5]);
            c->launches += 2;
            c->att_ready = true;
        }
    }
    for (const St& s : sts) {
        AdvArgs<real> a;
        a.in = s.in; a.fn = s.fn ? s.fn : s.in; a.out = s.out; a.part = c->d_part[0];
        a.ca = (real)s.ca; a.cb = (real)s.cb; a.cdt = (real)s.cc * (real)dt;
        a.upwind_only = c->opt.adv_flux == 1;
        a.VT = att[0]; a.VP = att[1]; a.LMt = att[2]; a.LPt = att[3]; a.LMp = att[4]; a.LPp = att[5];
        bool armed;
        prof_begin(c, 2, armed);
        const bool fast = !T.nonuniform && !a.upwind_only;   // uniform theta grid, WENO3: the kernels with shared theta-sweep terms
        a.nparts = fast ? nbxt : G.nbxa;
        a.rpt = rpt;
        if (c->att_any && fast) k_adv_stage_att_u<real><<<gt, TX, 0, c->stream>>>(a, T, G);
        else if (c->att_any) k_adv_stage_att<real><<<g, TX, 0, c->stream>>>(a, T, G);
        else if (!T.nonuniform && !a.upwind_only) k_adv_stage_u<real><<<gt, TX, 0, c->stream>>>(a, T, G);   // uniform theta grid, WENO3
        else k_adv_stage<real><<<g, TX, 0, c->stream>>>(a, T, G);
        prof_end(c, armed, 1);
        k_adv_caps<real><<<gc, TX, 0, c->stream>>>(a, T, G);
        c->launches += 2;
    }
    // the last stage's output array becomes the state
    const real* last = sts.back().out;
    c->i_state = (last == A) ? ia : ib;
    return HFT_OK;
}

// one diffusion step, one launch per stage.  MAP: nu(theta, phi) (Eq. 27-28; hft_set_diffusivity_map), else the per-row
// coefficient tables.  k_sts_stage_mapv (16-byte vectors) when n_phi is a multiple of the vector width, else the
// one-column-per-thread kernels k_sts_stage_map / k_sts_stage
template <typename real, int MODE, bool MAP = true>
void launch_map_stage(hft_ctx* c, const StsArgs<real>& a, MapArgs<real>& M, bool vec, int* nparts) {
    const Geom& G = c->G;
    Tables<real>& T = tables_of<real>(c);
    if (vec) {
        constexpr int C = 16 / (int)sizeof(real);
        const int nbxv = (G.np / C + TX - 1) / TX;
        dim3 g(nbxv, (G.nt + 2 + MAPV_RPT - 1) / MAPV_RPT, c->nr);
        k_sts_stage_mapv<real, MODE, MAP><<<g, TX, 0, c->stream>>>(a, M, T, G);
        *nparts = nbxv;
    } else if (!MAP) {
        dim3 g(G.nbx, (G.nt + 2 + RPT - 1) / RPT, c->nr);
        k_sts_stage<real, MODE><<<g, TX, 0, c->stream>>>(a, T, G);
        *nparts = G.nbx;
    } else {
        dim3 g(G.nbx, (G.nt + 2 + RPT - 1) / RPT, c->nr);
        k_sts_stage_map<real, MODE><<<g, TX, 0, c->stream>>>(a, M, T, G);
        *nparts = G.nbx;
    }
    c->launches++;
}

template <typename real, bool MAP>
int diffuse_stagewise(hft_ctx* c, double dt, int s) {
    const Geom& G = c->G;
    const int is = c->i_state;
    real* Y0 = arr_of<real>(c, is);
    real* F = arr_of<real>(c, (is + 1) % kNumArrays);
    real* da = arr_of<real>(c, (is + 2) % kNumArrays);
    real* db = arr_of<real>(c, (is + 3) % kNumArrays);
    const bool vec = G.np % (16 / (int)sizeof(real)) == 0;
    MapArgs<real> M;
    M.NU = (const real*)c->numap; M.capw = c->d_capw; M.capP[0] = c->PN * c->dph / c->dthf[0]; M.capP[1] = c->PS * c->dph / c->dthf[c->G.nt];
    M.nparts_in = G.nbx;
    dim3 gs(G.nbx, 2, c->nr);
    if (MAP) k_polar_row_sums_map<real><<<gs, TX, 0, c->stream>>>(Y0, M.NU, c->d_part[0], G);
    else k_polar_row_sums<real><<<gs, TX, 0, c->stream>>>(Y0, c->d_part[0], G);
    c->launches++;
    StsArgs<real> a;
    a.F = F; a.Y0 = Y0; a.mu = 0; a.nu = 0; a.g = 0; a.use_d2 = 0;
    int np_out = 0;
    if (c->opt.diff_time == 1) {  // explicit Euler (:474), new state written to `da`
        a.in = Y0; a.d2 = da; a.part_in = c->d_part[0]; a.part_out = c->d_part[1]; a.a = (real)dt;
        launch_map_stage<real, 3, MAP>(c, a, M, vec, &np_out);
        c->i_state = (is + 2) % kNumArrays;
        return HFT_OK;
    }
    const StsCoef& K = c->coef;
    a.in = Y0; a.d2 = da; a.part_in = c->d_part[0]; a.part_out = c->d_part[1]; a.a = (real)K.a[1];
    bool armed;
    prof_begin(c, 1, armed);
    launch_map_stage<real, 0, MAP>(c, a, M, vec, &np_out);
    prof_end(c, armed, 1);
    real *d1 = da, *d2 = db;
    int pin = 1;
    for (int j = 2; j <= s; j++) {
        a.in = d1; a.d2 = d2; a.part_in = c->d_part[pin]; a.part_out = c->d_part[pin ^ 1];
        a.mu = (real)K.mu[j]; a.nu = (real)K.nu[j]; a.a = (real)K.a[j]; a.g = (real)K.g[j];
        a.use_d2 = j > 2;
        M.nparts_in = np_out;
        prof_begin(c, 1, armed);
        if (j < s) launch_map_stage<real, 1, MAP>(c, a, M, vec, &np_out);
        else launch_map_stage<real, 2, MAP>(c, a, M, vec, &np_out);
        prof_end(c, armed, 1);
        real* t = d1; d1 = d2; d2 = t;
        pin ^= 1;
    }
    return HFT_OK;
}

// one diffusion step (D of Eq. 21), one launch per stage
template <typename real>
int diffuse_unblocked(hft_ctx* c, double dt, int s) {
    return c->map_any ? diffuse_stagewise<real, true>(c, dt, s) : diffuse_stagewise<real, false>(c, dt, s);
}

// ---------------------------------------------------------------- random flux emergence (Sec. 2.4)

// One flux-balanced source map `map` of every realization into S (Eq. 13 / 14, balanced like Eq. 11, :207).
template <typename real>
int rfe_make_map(hft_ctx* c, real* S, uint32_t map) {
    const Geom& G = c->G;
    Tables<real>& T = tables_of<real>(c);
    dim3 ga(G.nbx, G.nt + 2, c->nr), gp(RED_CTAS, c->nr);
    const double r2 = c->grid.radius_cm * c->grid.radius_cm;
    k_rfe_generate<real><<<ga, TX, 0, c->stream>>>(S, T, G, c->rfe_model, c->rfe_flux, r2, (uint32_t)c->rfe_seed,
                                                   (uint32_t)(c->rfe_seed >> 32), map);
    k_flux_partials<real, 0><<<gp, 256, 0, c->stream>>>(S, nullptr, nullptr, 0, T, G, c->d_fluxpart);
    k_flux_finalize<real, 0><<<(c->nr + 63) / 64, 64, 0, c->stream>>>(S, c->d_fluxpart, RED_CTAS, nullptr, 0, T, G, 1.0, c->d_diag);
    k_rfe_balance<real><<<ga, TX, 0, c->stream>>>(S, c->d_diag, G);
    c->launches += 4;
    return check_launch(c);
}

// S(B, h) at time t (reading U29): rotate the maps while t has reached the time of map 2, then forward Euler
// with the Eq. 15 interpolation frozen at t.
template <typename real>
int rfe_advance(hft_ctx* c, double t, double h) {
    const Geom& G = c->G;
    while (t >= c->rfe_t1 + c->rfe_tau) {
        char* tmp = c->rfe_map[0]; c->rfe_map[0] = c->rfe_map[1]; c->rfe_map[1] = tmp;   // map 2 becomes map 1
        const int rc = rfe_make_map<real>(c, (real*)c->rfe_map[1], c->rfe_next++);
        if (rc != HFT_OK) return rc;
        c->rfe_t1 += c->rfe_tau;
    }
    const real a = (real)((t - c->rfe_t1) / c->rfe_tau);
    dim3 ga(G.nbx, G.nt + 2, c->nr);
    k_rfe_apply<real><<<ga, TX, 0, c->stream>>>(arr_of<real>(c, c->i_state), (const real*)c->rfe_map[0], (const real*)c->rfe_map[1], a,
                                                (real)h, G);
    c->launches++;
    return check_launch(c);
}

template <typename real>
int step_once(hft_ctx* c, double dt, int s) {
    int rc = HFT_OK;
    c->att_ready = false;
    // Eq. 21 (:308-313): A(dt) then D(dt).  Strang, Eq. 22 (:317-326) with S omitted: A(dt/2), D(dt), A(dt/2).
    const bool strang = c->opt.strang != 0;
    if (c->rfe_model && strang) rc = rfe_advance<real>(c, c->time, 0.5 * dt);   // Eq. 22: S(dt/2) first
    if (rc == HFT_OK && c->opt.adv_flux != 0) rc = advect<real>(c, strang ? 0.5 * dt : dt);
    if (rc != HFT_OK) return rc;
    if (c->opt.diff_time != 0) {
        const int kb = c->opt.sts_block == 0 ? sts_default_block(c->G, sizeof(real)) : c->opt.sts_block;
        if (!c->map_any && c->opt.diff_time >= 2 && kb > 1 && s > 2 * kb && sts_blocked_supported(c->G, sizeof(real))) {
            StsBlockedPlan<real> P;
            P.Y0 = arr_of<real>(c, c->i_state);
            for (int i = 0; i < 5; i++) P.buf[i] = arr_of<real>(c, (c->i_state + 1 + i) % kNumArrays);
            P.mu = c->coef.mu.data(); P.nu = c->coef.nu.data(); P.a = c->coef.a.data(); P.g = c->coef.g.data();
            P.s = s; P.kb = kb; P.stream = c->stream;
            P.part = c->d_part; P.zmean = c->d_zmean; P.capseq = c->d_capseq;
            P.prof_begin = [](void* u, bool* armed) { prof_begin((hft_ctx*)u, 1, *armed); };
            P.prof_end = [](void* u, bool armed, int stages) { prof_end((hft_ctx*)u, armed, stages); };
            P.user = c;
            P.up = &c->up;
            int64_t n = 0;
            rc = sts_blocked_step<real>(P, tables_of<real>(c), c->G, &n) == 0 ? HFT_OK : HFT_ERR_CUDA;
            c->launches += n;
        } else if (c->map_any && c->opt.diff_time >= 2 && c->opt.sts_block != 1 && s > 2 * MPIPE_K &&
                   sts_mblocked_supported(c->G, sizeof(real))) {
            // nu(theta, phi): K = 4 stages per launch, cap values from the polar band (hft_sts_mpipe.cuh)
            if (!c->d_mscratch) {
                const cudaError_t e = cudaMalloc((void**)&c->d_mscratch, sts_mscratch_bytes(c->G));
                if (e != cudaSuccess) { cuda_fail(c, e, "cudaMalloc(polar band scratch)"); return HFT_ERR_NOMEM; }
            }
            StsBlockedPlan<real> P;
            P.Y0 = arr_of<real>(c, c->i_state);
            for (int i = 0; i < 5; i++) P.buf[i] = arr_of<real>(c, (c->i_state + 1 + i) % kNumArrays);
            P.mu = c->coef.mu.data(); P.nu = c->coef.nu.data(); P.a = c->coef.a.data(); P.g = c->coef.g.data();
            P.s = s; P.kb = MPIPE_K; P.stream = c->stream;
            P.part = c->d_part; P.zmean = c->d_zmean; P.capseq = c->d_capseq;
            P.prof_begin = [](void* u, bool* armed) { prof_begin((hft_ctx*)u, 1, *armed); };
            P.prof_end = [](void* u, bool armed, int stages) { prof_end((hft_ctx*)u, armed, stages); };
            P.user = c;
            P.up = nullptr;
            MapArgs<real> M;
            M.NU = (const real*)c->numap; M.capw = c->d_capw;
            M.capP[0] = c->PN * c->dph / c->dthf[0]; M.capP[1] = c->PS * c->dph / c->dthf[c->G.nt];
            M.nparts_in = c->G.nbx;
            int64_t n = 0;
            rc = sts_mblocked_step<real>(P, M, tables_of<real>(c), c->G, c->d_mscratch, &n) == 0 ? HFT_OK : HFT_ERR_CUDA;
            c->launches += n;
        } else {
            rc = diffuse_unblocked<real>(c, dt, s);
        }
    }
    if (rc == HFT_OK && strang && c->opt.adv_flux != 0) rc = advect<real>(c, 0.5 * dt);
    if (rc == HFT_OK && c->rfe_model) {   // Eq. 21: S after D; Eq. 22: the second S(dt/2)
        if (strang) rc = rfe_advance<real>(c, c->time + 0.5 * dt, 0.5 * dt);
        else rc = rfe_advance<real>(c, c->time, dt);
    }
    c->time += dt;
    return rc;
}

// nu(theta, phi) of realization q into the NU array: from h_map ([nt+1][np], R_sun^2/hr) or, if null, from the realization's
// theta-face profile nuf (constant along phi).  Also the Gershgorin diagonal maximum of Eq. 28 (:454) over every cell and
// both caps (fp64, from the given values) and the two polar weight sums (fp64, from the values as stored).
template <typename real>
int map_upload(hft_ctx* c, int q, const double* h_map) {
    const int nt = c->G.nt, np = c->G.np;
    std::vector<real> h((size_t)(nt + 1) * np);
    const double* nuf = &c->nuf[(size_t)q * (nt + 1)];
    for (int f = 0; f <= nt; f++)
        for (int k = 0; k < np; k++) h[(size_t)f * np + k] = (real)(h_map ? h_map[(size_t)f * np + k] : nuf[f]);
    double wN = 0.0, wS = 0.0;
    for (int k = 0; k < np; k++) {
        const int kw = (k + np - 1) % np;
        wN += 0.5 * ((double)h[k] + (double)h[kw]);
        wS += 0.5 * ((double)h[(size_t)nt * np + k] + (double)h[(size_t)nt * np + kw]);
    }
    c->capw[2 * q] = wN; c->capw[2 * q + 1] = wS;
    c->map_set[q] = h_map != nullptr;
    if (h_map) {
        double wn = 0.0, ws = 0.0;
        for (int k = 0; k < np; k++) {
            const int kw = (k + np - 1) % np;
            wn += 0.5 * (h_map[k] + h_map[kw]);
            ws += 0.5 * (h_map[(size_t)nt * np + k] + h_map[(size_t)nt * np + kw]);
        }
        double d = fmax(c->PN * wn * c->dph / c->dthf[0], c->PS * ws * c->dph / c->dthf[nt]);
        for (int j = 1; j <= nt; j++) {
            const double *nS = h_map + (size_t)j * np, *nN = h_map + (size_t)(j - 1) * np;
            const double gtc = 1.0 / (c->st[j] * c->dthc[j]), gp = 1.0 / (c->st[j] * c->st[j] * c->dph * c->dph);
            for (int k = 0; k < np; k++) {
                const int kw = (k + np - 1) % np;
                d = fmax(d, 0.5 * (nS[k] + nS[kw]) * c->sth[j] * gtc / c->dthf[j] + 0.5 * (nN[k] + nN[kw]) * c->sth[j - 1] * gtc / c->dthf[j - 1] +
                                0.5 * (nS[k] + nN[k]) * gp + 0.5 * (nS[kw] + nN[kw]) * gp);
            }
        }
        c->map_diag[q] = d;
    }
    CK(cudaMemcpy2DAsync(c->numap + (size_t)q * c->G.rstride * sizeof(real), (size_t)c->G.pitch * sizeof(real), h.data(),
                         (size_t)np * sizeof(real), (size_t)np * sizeof(real), nt + 1, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_capw + 2 * q, &c->capw[2 * q], 2 * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));   // h goes out of scope
    return HFT_OK;
}

int map_upload_any(hft_ctx* c, int q, const double* h_map) {
    return c->fp64() ? map_upload<double>(c, q, h_map) : map_upload<float>(c, q, h_map);
}

}  // namespace

// ===================================================================== C ABI

extern "C" {

const char* hft_error_string(int code) {
    switch (code) {
        case HFT_OK: return "ok";
        case HFT_ERR_ARG: return "invalid argument";
        case HFT_ERR_WORKSPACE: return "workspace too small or misaligned";
        case HFT_ERR_CUDA: return "CUDA runtime error";
        case HFT_ERR_UNSTABLE: return "unstable request (dt <= 0 or forced sts_stages below the stable count)";
        case HFT_ERR_NOMEM: return "out of memory";
        case HFT_ERR_DEVICE: return "no usable sm_100 device";
        default: return "unknown hft_status";
    }
}

const char* hft_last_cuda_error(hft_ctx* ctx) { return ctx ? ctx->cuda_err.c_str() : ""; }

int hft_workspace_bytes(const hft_grid* grid, int32_t n_real, const hft_options* opt, size_t* h_bytes) {
    if (!valid_grid(grid) || n_real < 1 || n_real > 65535 || !h_bytes) return HFT_ERR_ARG;   // realizations ride in gridDim.z
    if (opt && !valid_options(opt)) return HFT_ERR_ARG;
    const size_t w = grid->dtype == 1 ? 8 : 4;
    const size_t one = round_up((size_t)n_real * (grid->n_theta + 2) * pitch_for(grid->n_phi, grid->dtype) * w, 256);
    *h_bytes = one * (kNumArrays + extra_arrays(opt));
    return HFT_OK;
}

int hft_create(const hft_grid* grid, int32_t n_real, const hft_params* h_params, const hft_options* opt,
               void* d_workspace, size_t workspace_bytes, void* cuda_stream, hft_ctx** out) {
    if (!out) return HFT_ERR_ARG;
    *out = nullptr;
    if (!valid_grid(grid) || n_real < 1 || n_real > 65535 || !h_params || !d_workspace) return HFT_ERR_ARG;
    if (!valid_params(h_params, n_real)) return HFT_ERR_ARG;
    hft_options o = opt ? *opt : default_options();
    if (!valid_options(&o)) return HFT_ERR_ARG;
    size_t need = 0;
    hft_workspace_bytes(grid, n_real, &o, &need);
    if (workspace_bytes < need || ((uintptr_t)d_workspace & 255) != 0) return HFT_ERR_WORKSPACE;
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HFT_ERR_DEVICE;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) return HFT_ERR_DEVICE;
    hft_ctx* c = new (std::nothrow) hft_ctx();
    if (!c) return HFT_ERR_NOMEM;
    c->grid = *grid; c->opt = o; c->nr = n_real; c->dev = dev; c->stream = (cudaStream_t)cuda_stream;
    c->G.nt = grid->n_theta; c->G.np = grid->n_phi; c->G.pitch = pitch_for(grid->n_phi, grid->dtype); c->G.nr = n_real;
    c->G.rstride = (size_t)(grid->n_theta + 2) * c->G.pitch;
    c->G.nbx = (grid->n_phi + TX - 1) / TX;
    c->G.nbxa = (grid->n_phi + ADV_COLS - 1) / ADV_COLS;
    c->arr_bytes = need / (kNumArrays + extra_arrays(&o));
    for (int i = 0; i < kNumArrays; i++) c->arr[i] = (char*)d_workspace + (size_t)i * c->arr_bytes;
    if (o.flow_attenuation)
        for (int i = 0; i < kNumAttArrays; i++) c->att[i] = (char*)d_workspace + (size_t)(kNumArrays + i) * c->arr_bytes;
    if (o.rfe)
        for (int i = 0; i < kNumRfeArrays; i++)
            c->rfe_map[i] = (char*)d_workspace + (size_t)(kNumArrays + (o.flow_attenuation ? kNumAttArrays : 0) + i) * c->arr_bytes;
    if (o.diffusivity_map)
        c->numap = (char*)d_workspace + (size_t)(kNumArrays + (o.flow_attenuation ? kNumAttArrays : 0) + (o.rfe ? kNumRfeArrays : 0)) * c->arr_bytes;
    c->map_set.assign(n_real, 0); c->map_diag.assign(n_real, 0.0); c->capw.assign(2 * (size_t)n_real, 0.0);
    c->B0.assign(n_real, 0.0);
    c->nu.resize(n_real); c->nuf.resize((size_t)n_real * (c->G.nt + 1)); c->vt.resize((size_t)n_real * (c->G.nt + 1)); c->om.resize((size_t)n_real * (c->G.nt + 2));
    build_metric(c, nullptr);
    c->params.assign(h_params, h_params + n_real);
    c->nu_scale.resize(n_real); c->nu_shape.assign(c->G.nt + 1, 1.0);
    for (int r = 0; r < n_real; r++) {
        build_flow(c, r, h_params[r]);
        for (int f = 0; f <= c->G.nt; f++) c->nuf[(size_t)r * (c->G.nt + 1) + f] = c->nu[r];
        c->nu_scale[r] = c->nu[r];
    }
    int rc = HFT_OK;
    auto fail = [&](int code) { hft_destroy(c); return code; };
    cudaError_t e;
    const size_t partb = (size_t)n_real * 2 * ((grid->n_phi + ATT_COLS - 1) / ATT_COLS) * sizeof(double);   // the most CTAs along phi any stage kernel uses
    if ((e = cudaMalloc((void**)&c->d_part[0], partb)) != cudaSuccess || (e = cudaMalloc((void**)&c->d_part[1], partb)) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_fluxpart, (size_t)n_real * RED_CTAS * 2 * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_capinfo, (size_t)n_real * 4 * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_scale, (size_t)n_real * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_diag, (size_t)n_real * 4 * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_zmean, sts_zmean_bytes(c->G))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_capseq, sts_capseq_bytes(c->G))) != cudaSuccess ||
        (e = cudaMalloc(&c->d_B0, (size_t)n_real * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_kappa, (size_t)n_real * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc((void**)&c->d_capw, (size_t)n_real * 2 * sizeof(double))) != cudaSuccess ||
        (e = cudaMallocHost((void**)&c->h_diag, (size_t)n_real * 4 * sizeof(double))) != cudaSuccess) {
        cuda_fail(c, e, "cudaMalloc");
        return fail(HFT_ERR_NOMEM);
    }
    if ((e = cudaMemsetAsync(d_workspace, 0, need, c->stream)) != cudaSuccess) { cuda_fail(c, e, "memset"); return fail(HFT_ERR_CUDA); }
    if ((rc = upload_all_tables(c)) != HFT_OK) return fail(rc);
    if ((rc = sts_blocked_init(c->G, c->fp64())) != HFT_OK) return fail(HFT_ERR_CUDA);
    *out = c;
    return HFT_OK;
}

void hft_destroy(hft_ctx* c) {
    DevGuard dg_(c);
    if (!c) return;
    if (c->prof_ev_made)
        for (int i = 0; i < 2 * kProfEvents; i++) cudaEventDestroy(c->prof_ev[i]);
    cudaFree(c->d_tab); cudaFree(c->d_part[0]); cudaFree(c->d_part[1]); cudaFree(c->d_fluxpart);
    cudaFree(c->d_capinfo); cudaFree(c->d_scale); cudaFree(c->d_diag); cudaFree(c->d_zmean); cudaFree(c->d_capseq); cudaFree(c->d_kappa); cudaFree(c->d_mscratch); cudaFree(c->d_B0); cudaFree(c->d_capw);
    if (c->h_diag) cudaFreeHost(c->h_diag);
    cudaFree(c->d_extpart); cudaFree(c->d_ext);
    if (c->h_ext) cudaFreeHost(c->h_ext);
    delete c;
}

int hft_set_theta_nodes(hft_ctx* c, const double* h_theta) {
    DevGuard dg_(c);
    if (!c || !h_theta || c->map_any) return HFT_ERR_ARG;
    const int nt = c->G.nt;
    if (h_theta[0] != 0.0 || fabs(h_theta[nt + 1] - kPi) > 1e-14) return HFT_ERR_ARG;
    for (int j = 0; j <= nt; j++)
        if (!(h_theta[j + 1] > h_theta[j])) return HFT_ERR_ARG;
    CK(cudaStreamSynchronize(c->stream));   // the tables may still be read by enqueued work
    build_metric(c, h_theta);
    for (int r = 0; r < c->nr; r++) {
        const double nu = c->nu[r];
        build_flow(c, r, c->params[r]);      // Eq. 3-4 at the new angles (custom flow tables are set after this call)
        c->nu[r] = nu;
    }
    c->tab_version++;
    return upload_all_tables(c);
}

int hft_set_flow_tables(hft_ctx* c, int32_t r, const double* h_vtheta, const double* h_omega) {
    DevGuard dg_(c);
    if (!c || !h_vtheta || !h_omega || r < -1 || r >= c->nr) return HFT_ERR_ARG;
    const int nt = c->G.nt;
    for (int q = 0; q < c->nr; q++) {
        if (r >= 0 && q != r) continue;
        for (int f = 0; f <= nt; f++) c->vt[(size_t)q * (nt + 1) + f] = h_vtheta[f] * kMsToRsHr;
        for (int j = 0; j <= nt + 1; j++) c->om[(size_t)q * (nt + 2) + j] = h_omega[j] * kMsToRsHr;
    }
    return upload_all_tables(c);
}

int hft_set_diffusivity_profile(hft_ctx* c, int32_t r, const double* h_nu_face) {
    DevGuard dg_(c);
    if (!c || !h_nu_face || r < -1 || r >= c->nr) return HFT_ERR_ARG;
    const int nt = c->G.nt;
    for (int f = 0; f <= nt; f++)
        if (!(h_nu_face[f] >= 0.0)) return HFT_ERR_ARG;
    for (int q = 0; q < c->nr; q++)
        if (r < 0 || q == r)
            for (int f = 0; f <= nt; f++) c->nuf[(size_t)q * (nt + 1) + f] = h_nu_face[f] * kKm2sToRs2Hr;
    if (r < 0 || c->nr == 1) {   // one profile for the whole batch: nu_r(theta) = 1 * shape(theta)
        for (int f = 0; f <= nt; f++) c->nu_shape[f] = h_nu_face[f] * kKm2sToRs2Hr;
        for (int q = 0; q < c->nr; q++) c->nu_scale[q] = 1.0;
        c->shape_common = true;
    } else {
        c->shape_common = false;   // per-realization profiles: per-realization tables (k_sts_pipe)
    }
    c->tab_version++;
    CK(cudaStreamSynchronize(c->stream));   // the tables may still be read by enqueued work
    if (c->map_any)   // the realizations given a profile leave map mode's per-cell values for the profile's
        for (int q = 0; q < c->nr; q++)
            if (r < 0 || q == r) {
                const int rc = map_upload_any(c, q, nullptr);
                if (rc != HFT_OK) return rc;
            }
    return upload_all_tables(c);
}

int hft_set_diffusivity_map(hft_ctx* c, int32_t r, const double* h_nu_hh) {
    DevGuard dg_(c);
    if (!c || !h_nu_hh || r < -1 || r >= c->nr || !c->opt.diffusivity_map) return HFT_ERR_ARG;
    const int nt = c->G.nt, np = c->G.np;
    const size_t n = (size_t)(nt + 1) * np;
    std::vector<double> m(n);
    for (size_t i = 0; i < n; i++) {
        if (!(h_nu_hh[i] >= 0.0)) return HFT_ERR_ARG;
        m[i] = h_nu_hh[i] * kKm2sToRs2Hr;
    }
    CK(cudaStreamSynchronize(c->stream));   // NU may still be read by enqueued work
    for (int q = 0; q < c->nr; q++) {
        const bool mine = r < 0 || q == r;
        if (!mine && c->map_any) continue;   // already holds its own map or profile
        const int rc = map_upload_any(c, q, mine ? m.data() : nullptr);
        if (rc != HFT_OK) return rc;
    }
    c->map_any = true;
    return HFT_OK;
}

int hft_set_grid_diffusivity(hft_ctx* c, int32_t r, double alpha_nu) {
    DevGuard dg_(c);
    if (!c || r < -1 || r >= c->nr || !(alpha_nu >= 0.0)) return HFT_ERR_ARG;
    const int nt = c->G.nt;
    std::vector<double> p(nt + 1);
    for (int f = 0; f <= nt; f++) {   // Eq. 7 (:121) where nu lives: at the theta-faces
        const double dps = c->dph * c->sth[f];
        p[f] = alpha_nu * (c->dthf[f] * c->dthf[f] + dps * dps);
    }
    return hft_set_diffusivity_profile(c, r, p.data());
}

int hft_set_attenuation(hft_ctx* c, int32_t r, double b0_gauss) {
    DevGuard dg_(c);
    if (!c || r < -1 || r >= c->nr || !c->opt.flow_attenuation || b0_gauss != b0_gauss) return HFT_ERR_ARG;
    for (int q = 0; q < c->nr; q++)
        if (r < 0 || q == r) c->B0[q] = b0_gauss > 0.0 ? b0_gauss : 0.0;
    c->att_any = false;
    for (double b : c->B0) c->att_any = c->att_any || b > 0.0;
    CK(cudaStreamSynchronize(c->stream));   // the previous table may still be read by enqueued work
    if (c->fp64()) {
        CK(cudaMemcpy(c->d_B0, c->B0.data(), (size_t)c->nr * sizeof(double), cudaMemcpyHostToDevice));
    } else {
        std::vector<float> f(c->B0.begin(), c->B0.end());
        CK(cudaMemcpy(c->d_B0, f.data(), (size_t)c->nr * sizeof(float), cudaMemcpyHostToDevice));
    }
    return HFT_OK;
}

int hft_set_rfe(hft_ctx* c, int32_t model, double flux_per_hr, double tau_hours, uint64_t seed) {
    DevGuard dg_(c);
    if (!c || model < 0 || model > 2) return HFT_ERR_ARG;
    if (model != 0 && (!c->opt.rfe || !(flux_per_hr >= 0.0) || !(tau_hours > 0.0))) return HFT_ERR_ARG;
    c->rfe_model = model; c->rfe_flux = flux_per_hr; c->rfe_tau = tau_hours; c->rfe_seed = seed;
    c->time = 0.0; c->rfe_t1 = 0.0; c->rfe_next = 2;
    if (model == 0) return HFT_OK;
    for (uint32_t m = 0; m < 2; m++) {
        const int rc = c->fp64() ? rfe_make_map<double>(c, (double*)c->rfe_map[m], m) : rfe_make_map<float>(c, (float*)c->rfe_map[m], m);
        if (rc != HFT_OK) return rc;
    }
    return HFT_OK;
}

int hft_get_rfe_map(hft_ctx* c, int32_t r, int32_t which, void* d_out) {
    DevGuard dg_(c);
    if (!c || !d_out || r < 0 || r >= c->nr || which < 0 || which > 1 || !c->rfe_model) return HFT_ERR_ARG;
    const Geom& G = c->G;
    dim3 g((G.np + 255) / 256, G.nt, 1);
    if (c->fp64()) k_copy_map<double><<<g, 256, 0, c->stream>>>((double*)c->rfe_map[which], (double*)d_out, G, r, 0, 1);
    else k_copy_map<float><<<g, 256, 0, c->stream>>>((float*)c->rfe_map[which], (float*)d_out, G, r, 0, 1);
    c->launches++;
    return check_launch(c);
}

int hft_set_map(hft_ctx* c, int32_t r, const void* d_map) {
    DevGuard dg_(c);
    if (!c || !d_map || r < -1 || r >= c->nr) return HFT_ERR_ARG;
    const Geom& G = c->G;
    const int nz = r < 0 ? c->nr : 1, r0 = r < 0 ? 0 : r;
    dim3 g((G.np + 255) / 256, G.nt, nz), gm(2, nz);
    if (c->fp64()) {
        k_copy_map<double><<<g, 256, 0, c->stream>>>((double*)c->arr[c->i_state], (double*)d_map, G, r0, 1, 0);
        k_caps_from_row_mean<double><<<gm, 256, 0, c->stream>>>((double*)c->arr[c->i_state], G, r0);
    } else {
        k_copy_map<float><<<g, 256, 0, c->stream>>>((float*)c->arr[c->i_state], (float*)d_map, G, r0, 1, 0);
        k_caps_from_row_mean<float><<<gm, 256, 0, c->stream>>>((float*)c->arr[c->i_state], G, r0);
    }
    c->launches += 2;
    return check_launch(c);
}

int hft_get_map(hft_ctx* c, int32_t r, void* d_out) {
    DevGuard dg_(c);
    if (!c || !d_out || r < -1 || r >= c->nr) return HFT_ERR_ARG;
    const Geom& G = c->G;
    const int nz = r < 0 ? c->nr : 1, r0 = r < 0 ? 0 : r;
    dim3 g((G.np + 255) / 256, G.nt, nz);
    if (c->fp64()) k_copy_map<double><<<g, 256, 0, c->stream>>>((double*)c->arr[c->i_state], (double*)d_out, G, r0, 0, 1);
    else k_copy_map<float><<<g, 256, 0, c->stream>>>((float*)c->arr[c->i_state], (float*)d_out, G, r0, 0, 1);
    c->launches++;
    return check_launch(c);
}

static int copy_full(hft_ctx* c, int32_t r, void* d, int dir) {
    DevGuard dg_(c);
    if (!c || !d || r < 0 || r >= c->nr) return HFT_ERR_ARG;
    const Geom& G = c->G;
    dim3 g((G.np + 255) / 256, G.nt + 2);
    if (c->fp64()) k_copy_full<double><<<g, 256, 0, c->stream>>>((double*)c->arr[c->i_state], (double*)d, G, r, dir);
    else k_copy_full<float><<<g, 256, 0, c->stream>>>((float*)c->arr[c->i_state], (float*)d, G, r, dir);
    c->launches++;
    return check_launch(c);
}
int hft_get_full(hft_ctx* c, int32_t r, void* d_out) {
    DevGuard dg_(c); return copy_full(c, r, d_out, 1); }
int hft_set_full(hft_ctx* c, int32_t r, const void* d_in) {
    DevGuard dg_(c); return copy_full(c, r, (void*)d_in, 0); }

int hft_stable_dt(hft_ctx* c, double* h_adv, double* h_diff) {
    DevGuard dg_(c);
    if (!c || !h_adv || !h_diff) return HFT_ERR_ARG;
    *h_adv = adv_dt_limit(c);
    *h_diff = diff_dt_expl(c);
    return HFT_OK;
}

int hft_sts_stage_count(hft_ctx* c, double dt_hours, int32_t* h_stages) {
    DevGuard dg_(c);
    if (!c || !h_stages || !(dt_hours > 0.0)) return HFT_ERR_ARG;
    const int scheme = c->opt.diff_time == 2 ? 2 : 3;
    const int s = sts_stages_for(c, scheme, dt_hours);
    if (s < 0) return HFT_ERR_UNSTABLE;
    *h_stages = s;
    return HFT_OK;
}

int hft_step(hft_ctx* c, int32_t n_steps, double dt) {
    DevGuard dg_(c);
    if (!c || n_steps < 0) return HFT_ERR_ARG;
    if (!(dt > 0.0)) return HFT_ERR_UNSTABLE;
    int s = 0;
    if (c->opt.diff_time >= 2) {
        const int need = sts_stages_for(c, c->opt.diff_time, dt);
        if (need < 0) return HFT_ERR_UNSTABLE;
        s = c->opt.sts_stages ? c->opt.sts_stages : need;
        if (s < need) return HFT_ERR_UNSTABLE;
        build_sts_coef(c->coef, c->opt.diff_time, s, dt);
        const int rc = prepare_upipe(c, c->opt.diff_time, s, dt);
        if (rc != HFT_OK) return rc;
    }
    for (int n = 0; n < n_steps; n++) {
        int rc = c->fp64() ? step_once<double>(c, dt, s) : step_once<float>(c, dt, s);
        if (rc != HFT_OK) return rc;
    }
    return check_launch(c);
}

}  // extern "C"

// Eq. 8 / Eq. 10-11 blend; with h_diag the flux integrals of the blended state come out of the same pass (k_assim_blend_diag)
template <typename real>
static int assimilate_impl(hft_ctx* c, const real* obs, const real* w, int32_t shared, int32_t flags, double* h_diag) {
    const Geom& G = c->G;
    Tables<real>& T = tables_of<real>(c);
    const int balanced = flags & 1, nmaps = shared ? 1 : c->nr;
    dim3 gm(2, nmaps), gb(G.nbx, G.nt + 2, c->nr), gp(RED_CTAS, c->nr);
    const int fin_blocks = (c->nr + 63) / 64;
    real* S = (real*)c->arr[c->i_state];
    k_assim_cap_means<real><<<gm, 256, 0, c->stream>>>(obs, w, G, c->d_capinfo);
    if (balanced) {
        k_flux_partials<real, 1><<<gp, 256, 0, c->stream>>>(S, obs, w, shared, T, G, c->d_fluxpart);
        k_flux_finalize<real, 1><<<fin_blocks, 64, 0, c->stream>>>(S, c->d_fluxpart, RED_CTAS, c->d_capinfo, shared, T, G, 1.0, c->d_scale);
        c->launches += 2;
    }
    if (!h_diag) {
        k_assim_blend<real><<<gb, TX, 0, c->stream>>>(S, obs, w, shared, c->d_capinfo, c->d_scale, balanced, G);
        c->launches += 2;
        return check_launch(c);
    }
    const double scale = c->grid.radius_cm * c->grid.radius_cm;
    k_assim_blend_diag<real><<<gp, 256, 0, c->stream>>>(S, obs, w, shared, c->d_capinfo, c->d_scale, balanced, T, G, c->d_fluxpart);
    k_flux_finalize<real, 0><<<fin_blocks, 64, 0, c->stream>>>(S, c->d_fluxpart, RED_CTAS, nullptr, 0, T, G, scale, c->d_diag);
    c->launches += 3;
    CK(cudaMemcpyAsync(c->h_diag, c->d_diag, (size_t)c->nr * 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    memcpy(h_diag, c->h_diag, (size_t)c->nr * 4 * sizeof(double));
    return HFT_OK;
}

extern "C" {

int hft_assimilate(hft_ctx* c, const void* d_obs, const void* d_w, int32_t shared, int32_t flags) {
    DevGuard dg_(c);
    if (!c || !d_obs || !d_w) return HFT_ERR_ARG;
    return c->fp64() ? assimilate_impl<double>(c, (const double*)d_obs, (const double*)d_w, shared, flags, nullptr)
                     : assimilate_impl<float>(c, (const float*)d_obs, (const float*)d_w, shared, flags, nullptr);
}

int hft_assimilate_diagnostics(hft_ctx* c, const void* d_obs, const void* d_w, int32_t shared, int32_t flags, double* h_out) {
    DevGuard dg_(c);
    if (!c || !d_obs || !d_w || !h_out) return HFT_ERR_ARG;
    return c->fp64() ? assimilate_impl<double>(c, (const double*)d_obs, (const double*)d_w, shared, flags, h_out)
                     : assimilate_impl<float>(c, (const float*)d_obs, (const float*)d_w, shared, flags, h_out);
}

int hft_diagnostics(hft_ctx* c, double* h_out) {
    DevGuard dg_(c);
    if (!c || !h_out) return HFT_ERR_ARG;
    const Geom& G = c->G;
    dim3 gp(RED_CTAS, c->nr);
    const int fin_blocks = (c->nr + 63) / 64;
    const double scale = c->grid.radius_cm * c->grid.radius_cm;
    if (c->fp64()) {
        double* S = (double*)c->arr[c->i_state];
        k_flux_partials<double, 0><<<gp, 256, 0, c->stream>>>(S, nullptr, nullptr, 0, c->Td, G, c->d_fluxpart);
        k_flux_finalize<double, 0><<<fin_blocks, 64, 0, c->stream>>>(S, c->d_fluxpart, RED_CTAS, nullptr, 0, c->Td, G, scale, c->d_diag);
    } else {
        float* S = (float*)c->arr[c->i_state];
        k_flux_partials<float, 0><<<gp, 256, 0, c->stream>>>(S, nullptr, nullptr, 0, c->Tf, G, c->d_fluxpart);
        k_flux_finalize<float, 0><<<fin_blocks, 64, 0, c->stream>>>(S, c->d_fluxpart, RED_CTAS, nullptr, 0, c->Tf, G, scale, c->d_diag);
    }
    c->launches += 2;
    CK(cudaMemcpyAsync(c->h_diag, c->d_diag, (size_t)c->nr * 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    memcpy(h_out, c->h_diag, (size_t)c->nr * 4 * sizeof(double));
    return HFT_OK;
}

int hft_diagnostics_ext(hft_ctx* c, double polar_lat_deg, double* h_out) {
    DevGuard dg_(c);
    if (!c || !h_out || !(polar_lat_deg >= 0.0 && polar_lat_deg <= 90.0)) return HFT_ERR_ARG;
    const Geom& G = c->G;
    if (!c->d_extpart) {
        cudaError_t e;
        if ((e = cudaMalloc((void**)&c->d_extpart, (size_t)c->nr * RED_CTAS * EXT_NPART * sizeof(double))) != cudaSuccess ||
            (e = cudaMalloc((void**)&c->d_ext, (size_t)c->nr * EXT_NOUT * sizeof(double))) != cudaSuccess ||
            (e = cudaMallocHost((void**)&c->h_ext, (size_t)c->nr * EXT_NOUT * sizeof(double))) != cudaSuccess) {
            cuda_fail(c, e, "cudaMalloc");
            return HFT_ERR_NOMEM;
        }
    }
    dim3 gp(RED_CTAS, c->nr);
    const int fin_blocks = (c->nr + 63) / 64;
    const double scale = c->grid.radius_cm * c->grid.radius_cm;
    const double thc = (90.0 - polar_lat_deg) * kPi / 180.0;
    if (c->fp64()) {
        double* S = (double*)c->arr[c->i_state];
        k_diag_ext_partials<double><<<gp, 256, 0, c->stream>>>(S, c->Td, G, c->dph, thc, c->d_extpart);
        k_diag_ext_finalize<double><<<fin_blocks, 64, 0, c->stream>>>(S, c->d_extpart, RED_CTAS, c->Td, G, thc, scale, c->d_ext);
    } else {
        float* S = (float*)c->arr[c->i_state];
        k_diag_ext_partials<float><<<gp, 256, 0, c->stream>>>(S, c->Tf, G, c->dph, thc, c->d_extpart);
        k_diag_ext_finalize<float><<<fin_blocks, 64, 0, c->stream>>>(S, c->d_extpart, RED_CTAS, c->Tf, G, thc, scale, c->d_ext);
    }
    c->launches += 2;
    CK(cudaMemcpyAsync(c->h_ext, c->d_ext, (size_t)c->nr * EXT_NOUT * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    memcpy(h_out, c->h_ext, (size_t)c->nr * EXT_NOUT * sizeof(double));
    return HFT_OK;
}

int hft_synchronize(hft_ctx* c) {
    DevGuard dg_(c);
    if (!c) return HFT_ERR_ARG;
    CK(cudaStreamSynchronize(c->stream));   // an asynchronous fault of the kernels enqueued so far surfaces here
    return check_launch(c);
}

int hft_launch_count(hft_ctx* c, int64_t* h_count) {
    DevGuard dg_(c);
    if (!c || !h_count) return HFT_ERR_ARG;
    *h_count = c->launches;
    return HFT_OK;
}

int hft_profile_kernels(hft_ctx* c, int32_t which) {
    DevGuard dg_(c);
    if (!c || which < 0 || which > 2) return HFT_ERR_ARG;
    if (!c->prof_ev_made) {
        for (int i = 0; i < 2 * kProfEvents; i++) CK(cudaEventCreate(&c->prof_ev[i]));
        c->prof_ev_made = true;
    }
    c->prof_which = which; c->prof_n = 0; c->prof_seen = 0; c->prof_stages = 0;
    return HFT_OK;
}

int hft_kernel_time(hft_ctx* c, double* h_ms, int64_t* h_launches, int64_t* h_stages) {
    DevGuard dg_(c);
    if (!c || !h_ms || !h_launches || !h_stages) return HFT_ERR_ARG;
    CK(cudaStreamSynchronize(c->stream));
    double ms = 0.0;
    for (int i = 0; i < c->prof_n; i++) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
        ms += t;
    }
    *h_ms = ms; *h_launches = c->prof_n; *h_stages = c->prof_stages;
    c->prof_n = 0; c->prof_seen = 0; c->prof_stages = 0;
    return HFT_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ hft_diagnostics_noalloc
// The flux diagnostics for callers that may not allocate: the CTA partials of k_flux_partials, which
// hft_diagnostics keeps in a cudaMalloc'ed buffer of the context, go to a file-scope device array instead.  Every GPU that
// loads the library holds the array (HFT_NOALLOC_MAX_REAL x RED_CTAS x 2 doubles = 1 MiB) until the process exits.
static __device__ __align__(256) double g_noalloc_fluxpart[(size_t)HFT_NOALLOC_MAX_REAL * RED_CTAS * 2];

namespace {

// In host code g_noalloc_fluxpart names a host-side stand-in, not device memory: the kernels get the device address,
// resolved once per device with that device current.
std::mutex g_noalloc_mutex;
double* g_noalloc_ptr[64] = {nullptr};

int noalloc_scratch(hft_ctx* c, double** out) {
    if (c->dev < 0 || c->dev >= 64) return HFT_ERR_DEVICE;
    std::lock_guard<std::mutex> lk(g_noalloc_mutex);
    if (!g_noalloc_ptr[c->dev]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_fluxpart);   // the calling entry point made c->dev current
        if (e != cudaSuccess || !p) return cuda_fail(c, e, "cudaGetSymbolAddress(g_noalloc_fluxpart)");
        g_noalloc_ptr[c->dev] = p;
    }
    *out = g_noalloc_ptr[c->dev];
    return HFT_OK;
}

template <typename real>
int diagnostics_noalloc_impl(hft_ctx* c, const real* d_field, double* d_out, double* part) {
    Geom G = c->G;                      // the caller's array is dense: [n_real][n_theta + 2][n_phi]
    G.pitch = G.np;
    G.rstride = (size_t)(G.nt + 2) * G.np;
    dim3 gp(RED_CTAS, c->nr);
    const double scale = c->grid.radius_cm * c->grid.radius_cm;
    // every element of part[r][0..RED_CTAS-1][0..1] is written by k_flux_partials before k_flux_finalize reads it: what an
    // earlier call left in the array is never read, nothing has to be cleared
    k_flux_partials<real, 0><<<gp, 256, 0, c->stream>>>(d_field, nullptr, nullptr, 0, tables_of<real>(c), G, part);
    k_flux_finalize<real, 0><<<(c->nr + 63) / 64, 64, 0, c->stream>>>(d_field, part, RED_CTAS, nullptr, 0, tables_of<real>(c), G, scale, d_out);
    c->launches += 2;
    return check_launch(c);
}

}  // namespace

extern "C" int hft_diagnostics_noalloc(hft_ctx* c, const void* d_field, double* d_out) {
    DevGuard dg_(c);
    if (!c || !d_field || !d_out) return HFT_ERR_ARG;
    if (c->nr > HFT_NOALLOC_MAX_REAL) {
        c->cuda_err = "hft_diagnostics_noalloc: n_real = " + std::to_string(c->nr) + " exceeds HFT_NOALLOC_MAX_REAL = " +
                      std::to_string(HFT_NOALLOC_MAX_REAL) + " (the size of the static scratch array)";
        return HFT_ERR_ARG;
    }
    double* part = nullptr;
    const int rc = noalloc_scratch(c, &part);
    if (rc != HFT_OK) return rc;
    return c->fp64() ? diagnostics_noalloc_impl<double>(c, (const double*)d_field, d_out, part)
                     : diagnostics_noalloc_impl<float>(c, (const float*)d_field, d_out, part);
}
