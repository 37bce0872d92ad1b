/*
 * sft_oracle.c -- CPU oracle for the HipFT surface-flux-transport time step.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct
 * restatement of what the hot path computes, written from the paper
 * (arxiv 2501.06377, /root/reference/PAPER.md; cited below as PAPER.md:<line>)
 * and the readings listed in DESIGN.md ("Readings of the paper").  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares no code, header, table or constant generator with the
 * CUDA path under paper_2501_06377_b200/csrc/, and neither imports the other.
 *
 * Compiled twice: -DORACLE_FP32 -> symbols *_f32 (state and arithmetic in float),
 * otherwise *_f64 (double).  Tables are always formed in fp64 and rounded once to
 * the state precision; phi-sums (polar caps, diagnostics) are accumulated in fp64
 * with compensated (Kahan) summation in index order.  Build with
 *     gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC
 * so that no FMA contraction happens: every expression is evaluated left to
 * right exactly as written here.  OpenMP is used only as `parallel for` over rows
 * (each row's result is independent of the thread count).
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   units            PAPER.md:298 printed constants, :257 rigid-rotation speed
 *   diffusion L      Y_l^m eigenfunction decay exp(-l(l+1) nu t) (Eq. 19, :261), 2nd order;
 *                    dA-weighted symmetry (:448); constants in the null space; flux conservation
 *   STS              scalar stability polynomial: order conditions, |R|<=1 on the stated interval,
 *                    time ratio sqrt(6/4) (:476); dense-matrix polynomial on 8x16 (brute force)
 *   advection        upwind+Euler at Courant 1 = exact one-cell shift; phi-flux == textbook WENO3 (JS
 *                    weights 1/3,2/3) for uniform speed; 3rd-order convergence with eps=h and loss of
 *                    order with eps=1e-12 (:670, Fig. 15); App. C analytic theta solution (:697-731);
 *                    flux conservation incl. polar caps (App. A :622-648)
 *   assimilation     Eq. 8 (:131) closed form, Eq. 10-11 (:144-153) flux balance => net flux of dB is 0
 *   splitting        Strang (Eq. 22) reduces exactly to its parts; error order 1 (Eq. 21) vs 2 (Eq. 22)
 *   diagnostics      Eq. 16-17 dipoles of cos(theta), sin(theta)cos(phi - phi0): D = 1, H = 1 (2nd order); brute force
 *                    of all 13 run-history numbers on 8x16
 *   attenuation      Eq. 5: with B0 = inf the variable-speed rule equals the table rule bit for bit; uniform field =>
 *                    flow scaled by 1 - tanh(|c|/B0); |B| >> B0 => nothing moves; flux conserved; strong spot drifts less
 *   general rule     (tests/test_oracle_general_rule.py) sweep with speeds varying along the sweep: phi-mirror symmetry bit for
 *                    bit (swaps LP <-> LM); brute force on 8x16 with faces keyed by half-integers, written from B2 (:684) and
 *                    :689; alpha window: a speed spike at one face changes exactly the faces within 4 of it, a dip exactly
 *                    LM_q / LP_{q-1}'s readers -- for the phi sweep and for the theta table rule
 *   rotation         rows under differential rotation (Eq. 3) arrive with phase m Omega_j t, each row its own; error order >= 3
 *   PARITY UNPINNED against HipFT itself (no HipFT output in the container): which faces use upwind
 *   next to the poles (reading U6), the stage-count rule (U9), eps_w = coordinate spacing (U11), where |Br| is taken
 *   for a face speed and when the attenuated speeds are formed (U22, U23).
 *   They are pinned oracle<->GPU by definition only; see DESIGN.md.
 *
 * Index convention: rows j = 0..nt+1, row 0 = north polar cap, row nt+1 = south
 * polar cap, theta_j = j*dth, dth = pi/(nt+1); theta-faces j+1/2 (index j = 0..nt) at (j+1/2)*dth;
 * columns k = 0..np-1, phi_k = k*dph, dph = 2*pi/np, periodic.  A full field is (nt+2)*np values,
 * the two cap rows hold one value each, stored replicated.  (App. A :628.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_FP32
typedef float real;
#define SUF(n) n##_f32
#else
typedef double real;
#define SUF(n) n##_f64
#endif

#define PI 3.14159265358979323846264338327950288

/* unit conversions to R_sun and hours (R_sun = 6.96e10 cm, :292). */
#define M_S_TO_RS_HR 5.172413793103448e-6
#define KM2_S_TO_RS2_HR 7.43162901307967e-9

typedef struct {
    int nt, np, nr;
    double dth, dph;
    double radius_cm;
    double *st;   /* sin(theta_j),        j = 0..nt+1 */
    double *sth;  /* sin(theta_{j+1/2}),  j = 0..nt   */
    double P;     /* polar prefactor, App. A :646 (exact form); north cap (uniform grid: both) */
    double Apole; /* polar cap area 2*pi*(1-cos(dth/2)), App. A :642; north cap (uniform grid: both) */
    /* non-uniform theta grid ("logically-rectangular non-uniform"; reading U33).  On the default
       uniform grid every entry of dthc / dthf holds the SAME double dth, so all expressions below evaluate as before. */
    double *th;   /* theta_j,       j = 0..nt+1: the nodes where B_r lives; th[0] = 0, th[nt+1] = pi */
    double *thf;  /* theta_{j+1/2}, j = 0..nt: the half grid, midway between the nodes */
    double *dthc; /* Delta theta_j = theta_{j+1/2} - theta_{j-1/2}: width of cell j (Eq. 27, :354); caps: their half width */
    double *dthf; /* Delta theta_{j+1/2} = theta_{j+1} - theta_j: node spacing across face j+1/2 (Eq. 27) */
    double PN, PS, ApoleN, ApoleS;   /* per cap: P = sin(x)/(2 pi (1 - cos x)), A = 2 pi (1 - cos x), x = the cap's half width */
    /* WENO3-CS(h) constants of App. B (:662-680) per theta-face f (cell i = f+1, face i-1/2), reading U12:
       wm[f][0..4] = D^{c/cm}_{i-3/2}, D^{c/cm}_{i-1/2}, D^{c/cp}_{i-3/2}, D^{p/t}_{i-3/2}, D^{cm/t}_{i-3/2}   (u^-, from LM)
       wp[f][0..4] = D^{c/cp}_{i-1/2}, D^{c/cp}_{i-3/2}, D^{c/cm}_{i-1/2}, D^{m/t}_{i-1/2}, D^{cp/t}_{i-1/2}   (u^+, from LP) */
    double *wm, *wp;
    double *params; /* [nr][7] as given to create (the flow tables are re-made when the grid changes) */
    int uniform;
    double *nu;   /* [nr] diffusivity in R_sun^2/hr */
    double *nuf;  /* [nr][nt+1] diffusivity at the theta-faces j+1/2 (the half grid of :288), R_sun^2/hr; = nu unless a
                     latitude profile was set (nu(theta), grid-based nu_g of Eq. 7) */
    double **nuhh; /* [nr] -> NULL, or [nt+1][np] diffusivity nu(theta, phi) on the half-half grid (Eq. 27 :438-446: "nu is located
                     on a staggered grid in both the theta and phi direction"): nuhh[f][k] at theta-face f+1/2, phi-face k+1/2
                     (between columns k and k+1, periodic), R_sun^2/hr.  SURVEY 8(f)-4, reading U31 */
    double *vt;   /* [nr][nt+1] v_theta at theta-faces, R_sun/hr (Eq. 4 :84) */
    double *om;   /* [nr][nt+2] Omega = v_phi/sin(theta) at rows, rad/hr (Eq. 3 :78) */
    real *B;      /* [nr][nt+2][np] state */
    const real *att_src; /* Strang step with attenuation: the field at the start of the step (else NULL) */
    /* random flux emergence (Sec. 2.4): 0 = off, 1 = Eq. 13 (per cell), 2 = Eq. 14 (per unit area) */
    int rfe_model;
    double rfe_flux_per_hr, rfe_tau, rfe_t1;   /* Phi/hr in G radius_cm^2 / hr; lifetime tau in hr (inf allowed); time of map 1 */
    uint64_t rfe_seed;
    uint32_t rfe_next;                        /* index of the next source map to generate */
    real *S1, *S2;                            /* [nr][nt+2][np] the two current source maps, G/hr */
    double time;                              /* simulated hours since create / the last set_rfe */
    double *B0;   /* [nr] flow-attenuation saturation field of Eq. 5 (:100) in Gauss; <= 0: attenuation off */
} oracle_t;

/* ------------------------------------------------------------------ tables */

/* Step 0 of DESIGN.md: grid metric.  1-cos(x) is evaluated as 2 sin^2(x/2) (identical function,
 * no cancellation); P*Apole == sin(dth/2) to round-off, which is what makes the cap update
 * cancel the theta-face term of row 1 (flux conservation). */
static void make_grid(oracle_t *o, const double *theta_nodes) {
    int nt = o->nt;
    o->dth = PI / (double)(nt + 1);
    o->dph = 2.0 * PI / (double)o->np;
    o->uniform = theta_nodes == NULL;
    if (o->uniform) {
        for (int j = 0; j <= nt + 1; j++) { o->th[j] = (double)j * o->dth; o->dthc[j] = o->dth; }
        for (int j = 0; j <= nt; j++) { o->thf[j] = ((double)j + 0.5) * o->dth; o->dthf[j] = o->dth; }
        o->dthc[0] = o->dthc[nt + 1] = 0.5 * o->dth;
    } else {
        for (int j = 0; j <= nt + 1; j++) o->th[j] = theta_nodes[j];
        for (int j = 0; j <= nt; j++) { o->thf[j] = 0.5 * (o->th[j] + o->th[j + 1]); o->dthf[j] = o->th[j + 1] - o->th[j]; }
        for (int j = 1; j <= nt; j++) o->dthc[j] = o->thf[j] - o->thf[j - 1];
        o->dthc[0] = o->thf[0] - o->th[0];
        o->dthc[nt + 1] = o->th[nt + 1] - o->thf[nt];
    }
    for (int j = 0; j <= nt + 1; j++) o->st[j] = sin(o->th[j]);
    for (int j = 0; j <= nt; j++) o->sth[j] = sin(o->thf[j]);
    for (int pole = 0; pole < 2; pole++) {
        double x = o->dthc[pole ? nt + 1 : 0];          /* half width of the cap */
        double s4 = sin(0.5 * x);
        double one_minus_cos = 2.0 * s4 * s4;
        double A = 2.0 * PI * one_minus_cos, P = sin(x) / (2.0 * PI * one_minus_cos);
        if (pole) { o->ApoleS = A; o->PS = P; } else { o->ApoleN = A; o->PN = P; }
    }
    o->Apole = o->ApoleN; o->P = o->PN;
    /* App. B D-factors (Smit et al. 2005, :680) with Delta x_j = the cell widths dthc[j]; faces 2..nt-2 are WENO faces
       (cells i-2..i+1 = f-1..f+2 are regular cells); on the uniform grid the textbook constants exactly */
    for (int f = 0; f <= nt; f++) {
        double *m = o->wm + 5 * f, *q = o->wp + 5 * f;
        m[0] = m[1] = m[2] = q[0] = q[1] = q[2] = 0.5;
        m[3] = q[3] = 1.0 / 3.0; m[4] = q[4] = 2.0 / 3.0;
        if (o->uniform || f < 2 || f > nt - 2) continue;
        int i = f + 1;
        double xm2 = o->dthc[i - 2], xm1 = o->dthc[i - 1], x0 = o->dthc[i], xp1 = o->dthc[i + 1];
        m[0] = xm1 / (xm1 + xm2);            /* D^{c/cm}_{i-3/2}: centre i-1 over (i-1, i-2) */
        m[1] = x0 / (x0 + xm1);              /* D^{c/cm}_{i-1/2}: centre i   over (i, i-1)   */
        m[2] = xm1 / (xm1 + x0);             /* D^{c/cp}_{i-3/2}: centre i-1 over (i-1, i)   */
        m[3] = x0 / (xm2 + xm1 + x0);        /* D^{p/t}_{i-3/2}  */
        m[4] = (xm1 + xm2) / (xm2 + xm1 + x0);   /* D^{cm/t}_{i-3/2} */
        q[0] = x0 / (x0 + xp1);              /* D^{c/cp}_{i-1/2} */
        q[1] = xm1 / (xm1 + x0);             /* D^{c/cp}_{i-3/2} */
        q[2] = x0 / (x0 + xm1);              /* D^{c/cm}_{i-1/2} */
        q[3] = xm1 / (xm1 + x0 + xp1);       /* D^{m/t}_{i-1/2}  */
        q[4] = (x0 + xp1) / (xm1 + x0 + xp1);    /* D^{cp/t}_{i-1/2} */
    }
}

/* params per realization: eta_km2_s, d0, d2, d4, m1, m3, m5 (Eq. 3, 4, 6; units m/s, km^2/s). */
static void make_flow(oracle_t *o, int r, const double *p) {
    int nt = o->nt;
    o->nu[r] = p[0] * KM2_S_TO_RS2_HR;
    double d0 = p[1], d2 = p[2], d4 = p[3], m1 = p[4], m3 = p[5], m5 = p[6];
    for (int j = 0; j <= nt; j++) { /* Eq. 4 at the face angle */
        double th = o->thf[j];
        double c = cos(th), s = sin(th);
        o->vt[(size_t)r * (nt + 1) + j] = -(m1 * c + m3 * c * c * c + m5 * c * c * c * c * c) * s * M_S_TO_RS_HR;
    }
    for (int j = 0; j <= nt + 1; j++) { /* Eq. 3 divided by sin(theta) */
        double c = cos(o->th[j]);
        o->om[(size_t)r * (nt + 2) + j] = (d0 + d2 * c * c + d4 * c * c * c * c) * M_S_TO_RS_HR;
    }
}

void *SUF(sft_oracle_create)(int nt, int np, int nr, const double *params /*[nr][7]*/, double radius_cm) {
    oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
    o->nt = nt; o->np = np; o->nr = nr; o->radius_cm = radius_cm;
    o->st = (double *)calloc(nt + 2, sizeof(double));
    o->sth = (double *)calloc(nt + 1, sizeof(double));
    o->nu = (double *)calloc(nr, sizeof(double));
    o->nuf = (double *)calloc((size_t)nr * (nt + 1), sizeof(double));
    o->nuhh = (double **)calloc(nr, sizeof(double *));
    o->vt = (double *)calloc((size_t)nr * (nt + 1), sizeof(double));
    o->om = (double *)calloc((size_t)nr * (nt + 2), sizeof(double));
    o->B = (real *)calloc((size_t)nr * (nt + 2) * np, sizeof(real));
    o->B0 = (double *)calloc(nr, sizeof(double));
    o->th = (double *)calloc(nt + 2, sizeof(double)); o->thf = (double *)calloc(nt + 1, sizeof(double));
    o->dthc = (double *)calloc(nt + 2, sizeof(double)); o->dthf = (double *)calloc(nt + 1, sizeof(double));
    o->wm = (double *)calloc(5 * (size_t)(nt + 1), sizeof(double)); o->wp = (double *)calloc(5 * (size_t)(nt + 1), sizeof(double));
    o->params = (double *)malloc(7 * (size_t)nr * sizeof(double));
    memcpy(o->params, params, 7 * (size_t)nr * sizeof(double));
    make_grid(o, NULL);
    for (int r = 0; r < nr; r++) {
        make_flow(o, r, params + 7 * r);
        for (int f = 0; f <= nt; f++) o->nuf[(size_t)r * (nt + 1) + f] = o->nu[r];
    }
    return o;
}

void SUF(sft_oracle_destroy)(void *h) {
    oracle_t *o = (oracle_t *)h;
    for (int r = 0; r < o->nr; r++) free(o->nuhh[r]);
    free(o->nuhh);
    free(o->th); free(o->thf); free(o->dthc); free(o->dthf); free(o->wm); free(o->wp); free(o->params);
    free(o->st); free(o->sth); free(o->nu); free(o->nuf); free(o->vt); free(o->om); free(o->B); free(o->B0); free(o->S1); free(o->S2); free(o);
}

/* Non-uniform theta grid (reading U33): theta[nt+2] = the nodes where B_r lives, theta[0] = 0, theta[nt+1] = pi,
 * strictly increasing.  Re-makes the metric, the App. B constants and the analytic flow tables (custom flow tables and
 * diffusivity profiles set before this call are kept as given: they are per face / per row, not functions of theta). */
void SUF(sft_oracle_set_theta_nodes)(void *h, const double *theta) {
    oracle_t *o = (oracle_t *)h;
    make_grid(o, theta);
    for (int r = 0; r < o->nr; r++) {
        double nu_keep = o->nu[r];
        make_flow(o, r, o->params + 7 * r);
        o->nu[r] = nu_keep;
    }
}

void SUF(sft_oracle_get_grid)(void *h, double *th /*[nt+2]*/, double *thf /*[nt+1]*/, double *dthc /*[nt+2]*/, double *dthf /*[nt+1]*/,
                              double *caps /*[4]: PN, PS, ApoleN, ApoleS*/) {
    oracle_t *o = (oracle_t *)h;
    memcpy(th, o->th, sizeof(double) * (o->nt + 2)); memcpy(thf, o->thf, sizeof(double) * (o->nt + 1));
    memcpy(dthc, o->dthc, sizeof(double) * (o->nt + 2)); memcpy(dthf, o->dthf, sizeof(double) * (o->nt + 1));
    caps[0] = o->PN; caps[1] = o->PS; caps[2] = o->ApoleN; caps[3] = o->ApoleS;
}

/* Latitude-dependent diffusivity (Eq. 6 :109 with nu = nu(theta)): nu_face[f] in km^2/s at the theta-face f+1/2,
 * f = 0..nt, for realization r (r < 0: all). */
void SUF(sft_oracle_set_diffusivity_profile)(void *h, int r, const double *nu_face) {
    oracle_t *o = (oracle_t *)h;
    for (int q = 0; q < o->nr; q++)
        if (r < 0 || q == r)
            for (int f = 0; f <= o->nt; f++) o->nuf[(size_t)q * (o->nt + 1) + f] = nu_face[f] * KM2_S_TO_RS2_HR;
}

/* Spatially varying diffusivity nu(theta, phi) (Eq. 6 :109, Eq. 27-28 :438-460): nu_hh[f][k] in km^2/s on the half-half
 * grid, f = 0..nt (theta-face f+1/2), k = 0..np-1 (phi-face k+1/2, between columns k and k+1), for realization r (r < 0:
 * all).  NULL returns realization r to its latitude profile / scalar value. */
void SUF(sft_oracle_set_diffusivity_map)(void *h, int r, const double *nu_hh) {
    oracle_t *o = (oracle_t *)h;
    size_t n = (size_t)(o->nt + 1) * o->np;
    for (int q = 0; q < o->nr; q++)
        if (r < 0 || q == r) {
            free(o->nuhh[q]);
            o->nuhh[q] = NULL;
            if (nu_hh) {
                o->nuhh[q] = (double *)malloc(n * sizeof(double));
                for (size_t i = 0; i < n; i++) o->nuhh[q][i] = nu_hh[i] * KM2_S_TO_RS2_HR;
            }
        }
}

/* Grid-based diffusivity of the map smoother, Eq. 7 (:121): nu_g = alpha_nu [dtheta^2 + (dphi sin(theta))^2], evaluated
 * where nu lives, at the theta-faces; alpha_nu in km^2/s per rad^2 (dtheta, dphi in radians). */
void SUF(sft_oracle_set_grid_diffusivity)(void *h, int r, double alpha_nu) {
    oracle_t *o = (oracle_t *)h;
    for (int q = 0; q < o->nr; q++)
        if (r < 0 || q == r)
            for (int f = 0; f <= o->nt; f++) {
                double dps = o->dph * o->sth[f];
                o->nuf[(size_t)q * (o->nt + 1) + f] = alpha_nu * (o->dthf[f] * o->dthf[f] + dps * dps) * KM2_S_TO_RS2_HR;
            }
}

/* Flow attenuation (Sec. 2.1.3, Eq. 5 :100): B0 in Gauss for realization r (r < 0: all); B0 <= 0 switches it off. */
void SUF(sft_oracle_set_attenuation)(void *h, int r, double B0) {
    oracle_t *o = (oracle_t *)h;
    for (int q = 0; q < o->nr; q++) if (r < 0 || q == r) o->B0[q] = B0;
}

/* Custom per-row flow tables (needed for the App. C constant-v_theta test, :703): vt in R_sun/hr at
 * the nt+1 theta-faces, om in rad/hr at the nt+2 rows. */
void SUF(sft_oracle_set_flow_tables)(void *h, int r, const double *vt, const double *om) {
    oracle_t *o = (oracle_t *)h;
    memcpy(o->vt + (size_t)r * (o->nt + 1), vt, sizeof(double) * (o->nt + 1));
    memcpy(o->om + (size_t)r * (o->nt + 2), om, sizeof(double) * (o->nt + 2));
}

void SUF(sft_oracle_get_tables)(void *h, int r, double *st, double *sth, double *vt, double *om, double *scal /*[5]: dth,dph,P,Apole,nu*/) {
    oracle_t *o = (oracle_t *)h;
    memcpy(st, o->st, sizeof(double) * (o->nt + 2));
    memcpy(sth, o->sth, sizeof(double) * (o->nt + 1));
    memcpy(vt, o->vt + (size_t)r * (o->nt + 1), sizeof(double) * (o->nt + 1));
    memcpy(om, o->om + (size_t)r * (o->nt + 2), sizeof(double) * (o->nt + 2));
    scal[0] = o->dth; scal[1] = o->dph; scal[2] = o->P; scal[3] = o->Apole; scal[4] = o->nu[r];
}

/* ------------------------------------------------------------ small helpers */

static real *field(oracle_t *o, int r) { return o->B + (size_t)r * (o->nt + 2) * o->np; }
static size_t fsize(const oracle_t *o) { return (size_t)(o->nt + 2) * o->np; }

/* Kahan-compensated sum in index order, fp64 accumulator. */
typedef struct { double s, c; } kahan_t;
static void kadd(kahan_t *k, double x) {
    double y = x - k->c;
    double t = k->s + y;
    k->c = (t - k->s) - y;
    k->s = t;
}

static void fill_row(real *row, int np, real v) { for (int k = 0; k < np; k++) row[k] = v; }

/* mean of a row over phi (dph-weighted mean on a uniform grid = arithmetic mean) */
static double row_mean(const real *row, int np) {
    kahan_t a = {0.0, 0.0};
    for (int k = 0; k < np; k++) kadd(&a, (double)row[k]);
    return a.s / (double)np;
}

/* ----------------------------------------------------------------- set/get */

/* User maps are [nt][np] (rows 1..nt).  Caps := dph-weighted mean of the adjacent row
 * (reading U18: "pole-cell averaging"). r = -1 broadcasts to all realizations. */
void SUF(sft_oracle_set_map)(void *h, int r, const real *map) {
    oracle_t *o = (oracle_t *)h;
    int nt = o->nt, np = o->np;
    for (int q = 0; q < o->nr; q++) {
        if (r >= 0 && q != r) continue;
        real *B = field(o, q);
        memcpy(B + np, map, sizeof(real) * (size_t)nt * np);
        fill_row(B, np, (real)row_mean(B + np, np));
        fill_row(B + (size_t)(nt + 1) * np, np, (real)row_mean(B + (size_t)nt * np, np));
    }
}

void SUF(sft_oracle_get_map)(void *h, int r, real *out) {
    oracle_t *o = (oracle_t *)h;
    memcpy(out, field(o, r) + o->np, sizeof(real) * (size_t)o->nt * o->np);
}

/* full (nt+2)*np field incl. replicated cap rows -- for tests */
void SUF(sft_oracle_get_full)(void *h, int r, real *out) {
    oracle_t *o = (oracle_t *)h;
    memcpy(out, field(o, r), sizeof(real) * fsize(o));
}
void SUF(sft_oracle_set_full)(void *h, int r, const real *in) {
    oracle_t *o = (oracle_t *)h;
    memcpy(field(o, r), in, sizeof(real) * fsize(o));
}

/* ------------------------------------------------------ diffusion operator */

/* Step 4: L(B) = discrete div(nu grad B), Eq. 27/28 (:438-460) with spatially constant nu and
 * uniform spacing:
 *   rows 1..nt:  c+_j (B[j+1,k]-B[j,k]) - c-_j (B[j,k]-B[j-1,k]) + cphi_j (B[j,k+1] - 2 B[j,k] + B[j,k-1])
 *   c+-_j = nu sin(theta_{j+-1/2}) / (sin(theta_j) dth^2),  cphi_j = nu / (sin^2(theta_j) dph^2)
 *   caps (App. A :624-648, F = nu dB/dtheta by central differences at the first half-mesh point):
 *     north: P (nu/dth) sum_k (B[1,k]-B[0]) dph ;  south: P (nu/dth) sum_k (B[nt,k]-B[nt+1]) dph
 * Row coefficients are formed in fp64 and rounded once to `real`. */
/* Eq. 27 (:438-446) written out with nu(theta, phi) on the half-half grid and uniform spacing; the four off-diagonal
 * coefficients are those of Eq. 28 (:450-458), the diagonal is minus their sum, i.e. the difference form below:
 *   a_{j+1,k} = (nu_{j+1/2,k+1/2} + nu_{j+1/2,k-1/2}) sin(theta_{j+1/2}) / (2 dth^2 sin(theta_j))
 *   a_{j-1,k} = (nu_{j-1/2,k+1/2} + nu_{j-1/2,k-1/2}) sin(theta_{j-1/2}) / (2 dth^2 sin(theta_j))
 *   a_{j,k+1} = (nu_{j+1/2,k+1/2} + nu_{j-1/2,k+1/2}) / (2 dph^2 sin^2(theta_j))
 *   a_{j,k-1} = (nu_{j+1/2,k-1/2} + nu_{j-1/2,k-1/2}) / (2 dph^2 sin^2(theta_j))
 *   L(B)_{j,k} = a_{j+1,k} (B[j+1,k]-B[j,k]) - a_{j-1,k} (B[j,k]-B[j-1,k]) + a_{j,k+1} (B[j,k+1]-B[j,k]) - a_{j,k-1} (B[j,k]-B[j,k-1])
 * Caps (App. A :624-648 with F = nu dB/dtheta at the first half-mesh point, nu averaged to the theta-face like a_{j+-1,k}):
 *   north: P sum_k nu_{1/2,k} (B[1,k]-B[0]) / dth dph,  nu_{1/2,k} = (nu_{1/2,k+1/2} + nu_{1/2,k-1/2})/2;  south likewise.
 * Coefficients are formed in fp64 and rounded once to `real` (reading U31). */
static void diffusion_op_map(const oracle_t *o, int r, const real *B, real *out) {
    int nt = o->nt, np = o->np;
    const double *nu = o->nuhh[r];
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        const double *nS = nu + (size_t)j * np, *nN = nu + (size_t)(j - 1) * np; /* faces j+1/2 and j-1/2 */
        const real *Bc = B + (size_t)j * np, *Bn = Bc - np, *Bs = Bc + np;
        real *oc = out + (size_t)j * np;
        for (int k = 0; k < np; k++) {
            int kw = (k + np - 1) % np, ke = (k + 1) % np;
            real as = (real)(0.5 * (nS[k] + nS[kw]) * o->sth[j] / (o->st[j] * o->dthc[j] * o->dthf[j]));
            real an = (real)(0.5 * (nN[k] + nN[kw]) * o->sth[j - 1] / (o->st[j] * o->dthc[j] * o->dthf[j - 1]));
            real ae = (real)(0.5 * (nS[k] + nN[k]) / (o->st[j] * o->st[j] * o->dph * o->dph));
            real aw = (real)(0.5 * (nS[kw] + nN[kw]) / (o->st[j] * o->st[j] * o->dph * o->dph));
            real tth = as * (Bs[k] - Bc[k]) - an * (Bc[k] - Bn[k]);
            real tph = ae * (Bc[ke] - Bc[k]) - aw * (Bc[k] - Bc[kw]);
            oc[k] = tth + tph;
        }
    }
    const double *n0 = nu, *n1 = nu + (size_t)nt * np;
    kahan_t a = {0, 0}, b = {0, 0};
    for (int k = 0; k < np; k++) {
        int kw = (k + np - 1) % np;
        kadd(&a, 0.5 * (n0[k] + n0[kw]) * (double)(B[np + k] - B[0]));
        kadd(&b, 0.5 * (n1[k] + n1[kw]) * (double)(B[(size_t)nt * np + k] - B[(size_t)(nt + 1) * np]));
    }
    fill_row(out, np, (real)(o->PN / o->dthf[0] * o->dph * a.s));
    fill_row(out + (size_t)(nt + 1) * np, np, (real)(o->PS / o->dthf[nt] * o->dph * b.s));
}

static void diffusion_op(const oracle_t *o, int r, const real *B, real *out) {
    int nt = o->nt, np = o->np;
    if (o->nuhh[r]) { diffusion_op_map(o, r, B, out); return; }
    /* Eq. 28 (:450-458) with nu on the half grid and independent of phi: the theta-fluxes take nu at their face, the
     * phi-term the mean of the two faces of the row, (nu_{j+1/2} + nu_{j-1/2})/2 */
    const double *nuf = o->nuf + (size_t)r * (nt + 1);
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        real cp = (real)(nuf[j] * o->sth[j] / (o->st[j] * o->dthc[j] * o->dthf[j]));
        real cm = (real)(nuf[j - 1] * o->sth[j - 1] / (o->st[j] * o->dthc[j] * o->dthf[j - 1]));
        real cf = (real)(0.5 * (nuf[j] + nuf[j - 1]) / (o->st[j] * o->st[j] * o->dph * o->dph));
        const real *Bc = B + (size_t)j * np, *Bn = Bc - np, *Bs = Bc + np; /* Bn = row j-1 (towards north), Bs = row j+1 */
        real *oc = out + (size_t)j * np;
        for (int k = 0; k < np; k++) {
            int kw = (k + np - 1) % np, ke = (k + 1) % np;
            real tth = cp * (Bs[k] - Bc[k]) - cm * (Bc[k] - Bn[k]);
            real tph = cf * (Bc[ke] - (real)2 * Bc[k] + Bc[kw]);
            oc[k] = tth + tph;
        }
    }
    double capN = o->PN * (nuf[0] / o->dthf[0]) * o->dph, capS = o->PS * (nuf[nt] / o->dthf[nt]) * o->dph;
    kahan_t a = {0, 0}, b = {0, 0};
    for (int k = 0; k < np; k++) {
        kadd(&a, (double)(B[np + k] - B[0]));
        kadd(&b, (double)(B[(size_t)nt * np + k] - B[(size_t)(nt + 1) * np]));
    }
    fill_row(out, np, (real)(capN * a.s));
    fill_row(out + (size_t)(nt + 1) * np, np, (real)(capS * b.s));
}

void SUF(sft_oracle_diffusion_op)(void *h, int r, const real *in, real *out) {
    diffusion_op((oracle_t *)h, r, in, out);
}

/* Step 5: Euler limit.  Gershgorin: spectral radius <= 2 max|diag|, dt_expl = 2/rho =
 * 1 / max( max_j (c+_j + c-_j + 2 cphi_j), 2 pi P nu / dth ), with nu = max_r nu_r (reading U8). */
static double diffusion_dt_expl(const oracle_t *o) {
    double dmax = 0.0;
    for (int r = 0; r < o->nr; r++) {
        if (o->nuhh[r]) { /* nu(theta, phi): the same Gershgorin bound, max over every cell of -a_{j,k} of Eq. 28 (:454) */
            int nt = o->nt, np = o->np;
            const double *nu = o->nuhh[r];
            double wN = 0.0, wS = 0.0;
            for (int k = 0; k < np; k++) {
                int kw = (k + np - 1) % np;
                wN += 0.5 * (nu[k] + nu[kw]);
                wS += 0.5 * (nu[(size_t)nt * np + k] + nu[(size_t)nt * np + kw]);
            }
            if (o->PN * wN * o->dph / o->dthf[0] > dmax) dmax = o->PN * wN * o->dph / o->dthf[0];
            if (o->PS * wS * o->dph / o->dthf[o->nt] > dmax) dmax = o->PS * wS * o->dph / o->dthf[o->nt];
            for (int j = 1; j <= nt; j++) {
                const double *nS = nu + (size_t)j * np, *nN = nu + (size_t)(j - 1) * np;
                for (int k = 0; k < np; k++) {
                    int kw = (k + np - 1) % np;
                    double d = 0.5 * (nS[k] + nS[kw]) * o->sth[j] / (o->st[j] * o->dthc[j] * o->dthf[j])
                             + 0.5 * (nN[k] + nN[kw]) * o->sth[j - 1] / (o->st[j] * o->dthc[j] * o->dthf[j - 1])
                             + 0.5 * (nS[k] + nN[k]) / (o->st[j] * o->st[j] * o->dph * o->dph)
                             + 0.5 * (nS[kw] + nN[kw]) / (o->st[j] * o->st[j] * o->dph * o->dph);
                    if (d > dmax) dmax = d;
                }
            }
            continue;
        }
        const double *nuf = o->nuf + (size_t)r * (o->nt + 1);
        double dN = 2.0 * PI * o->PN * nuf[0] / o->dthf[0], dS = 2.0 * PI * o->PS * nuf[o->nt] / o->dthf[o->nt];
        if (dN > dmax) dmax = dN;
        if (dS > dmax) dmax = dS;
        for (int j = 1; j <= o->nt; j++) {
            double cp = nuf[j] * o->sth[j] / (o->st[j] * o->dthc[j] * o->dthf[j]);
            double cm = nuf[j - 1] * o->sth[j - 1] / (o->st[j] * o->dthc[j] * o->dthf[j - 1]);
            double cf = 0.5 * (nuf[j] + nuf[j - 1]) / (o->st[j] * o->st[j] * o->dph * o->dph);
            double d = cp + cm + 2.0 * cf;
            if (d > dmax) dmax = d;
        }
    }
    return dmax > 0.0 ? 1.0 / dmax : INFINITY;
}

/* ------------------------------------------------------------ STS schemes */

/* Step 7 coefficient families (reading U7).  scheme 2 = RKL2 (Legendre; Meyer et al. 2014 via
 * PAPER.md:470-474), scheme 3 = RKG2(3/2) (Gegenbauer lambda = 3/2, normalised G_j(1) = 1; Skaras et
 * al. 2021 via :472).  Arrays are indexed 0..s.  mu[j], nu[j], mut[j] (mu-tilde), gt[j] (gamma-tilde)
 * for j >= 2; mut[1] = b_1 w_1.  b_0 = b_1 = b_2.  a_j = 1 - b_j. */
static double sts_b(int scheme, int j) {
    if (j < 2) j = 2;
    double dj = (double)j;
    if (scheme == 2) return (dj * dj + dj - 2.0) / (2.0 * dj * (dj + 1.0));
    return 2.0 * (dj - 1.0) * (dj + 4.0) / (3.0 * dj * (dj + 3.0));
}
static double sts_w1(int scheme, int s) {
    double ds = (double)s;
    if (scheme == 2) return 4.0 / (ds * ds + ds - 2.0);
    return 6.0 / ((ds - 1.0) * (ds + 4.0));
}
void SUF(sft_oracle_sts_coeffs)(int scheme, int s, double *mu, double *nu, double *mut, double *gt, double *b) {
    double w1 = sts_w1(scheme, s);
    for (int j = 0; j <= s; j++) { b[j] = sts_b(scheme, j); mu[j] = nu[j] = mut[j] = gt[j] = 0.0; }
    mut[1] = b[1] * w1;
    for (int j = 2; j <= s; j++) {
        double dj = (double)j, A, Bc;
        if (scheme == 2) { A = (2.0 * dj - 1.0) / dj; Bc = (dj - 1.0) / dj; }
        else             { A = (2.0 * dj + 1.0) / (dj + 2.0); Bc = (dj - 1.0) / (dj + 2.0); }
        mu[j] = A * b[j] / b[j - 1];
        nu[j] = -Bc * b[j] / b[j - 2];
        mut[j] = mu[j] * w1;
        gt[j] = -(1.0 - b[j - 1]) * mut[j];
    }
}

/* Step 6 (reading U9): smallest s >= 2 with dt <= dt_expl * C(s); RKL2: C = (s^2+s-2)/4;
 * RKG2(3/2): C = (s^2+3s-4)/6.  One s for all realizations. */
static int sts_stage_count(int scheme, double dt, double dt_expl) {
    int s = 2;
    for (;;) {
        double ds = (double)s;
        double C = (scheme == 2) ? (ds * ds + ds - 2.0) / 4.0 : (ds * ds + 3.0 * ds - 4.0) / 6.0;
        if (dt <= dt_expl * C) return s;
        s++;
        if (s > 10000000) return -1;
    }
}

int SUF(sft_oracle_sts_stage_count)(void *h, double dt, int scheme) {
    return sts_stage_count(scheme, dt, diffusion_dt_expl((oracle_t *)h));
}

/* One STS step of size dt with s stages, in the deviation form:
 *   delta_j = Y_j - Y_0 ;  delta_0 = 0 ;  delta_1 = mut_1 dt L(Y_0)
 *   delta_j = mu_j delta_{j-1} + nu_j delta_{j-2} + mut_j dt L(delta_{j-1}) + mut_j b_{j-1} dt L(Y_0)
 *   Y_s = Y_0 + delta_s
 * which is the textbook recurrence
 *   Y_j = mu_j Y_{j-1} + nu_j Y_{j-2} + (1-mu_j-nu_j) Y_0 + mut_j dt L(Y_{j-1}) + gt_j dt L(Y_0)
 * rewritten using the linearity of L (caps included) and mut_j + gt_j = mut_j b_{j-1}.
 * Per-stage scalars are formed in fp64 and rounded once to `real`. */
static void sts_step(oracle_t *o, int r, int scheme, int s, double dt) {
    size_t n = fsize(o);
    real *Y = field(o, r);
    real *LY0 = (real *)malloc(n * sizeof(real)), *d1 = (real *)malloc(n * sizeof(real));
    real *d2 = (real *)calloc(n, sizeof(real)), *Ld = (real *)malloc(n * sizeof(real));
    double *mu = (double *)malloc((s + 1) * sizeof(double)), *nu = (double *)malloc((s + 1) * sizeof(double));
    double *mut = (double *)malloc((s + 1) * sizeof(double)), *gt = (double *)malloc((s + 1) * sizeof(double));
    double *b = (double *)malloc((s + 1) * sizeof(double));
    SUF(sft_oracle_sts_coeffs)(scheme, s, mu, nu, mut, gt, b);
    diffusion_op(o, r, Y, LY0);
    real a1 = (real)(mut[1] * dt);
    for (size_t i = 0; i < n; i++) d1[i] = a1 * LY0[i];
    for (int j = 2; j <= s; j++) {
        diffusion_op(o, r, d1, Ld);
        real mj = (real)mu[j], nj = (real)nu[j], aj = (real)(mut[j] * dt), gj = (real)(mut[j] * b[j - 1] * dt);
        #pragma omp parallel for schedule(static)
        for (size_t i = 0; i < n; i++) {
            real dn = mj * d1[i] + nj * d2[i] + aj * Ld[i] + gj * LY0[i];
            d2[i] = d1[i];
            d1[i] = dn;
        }
    }
    for (size_t i = 0; i < n; i++) Y[i] = Y[i] + d1[i];
    free(LY0); free(d1); free(d2); free(Ld); free(mu); free(nu); free(mut); free(gt); free(b);
}

/* The same step in the textbook form (used only by tests to pin the deviation form). */
static void sts_step_textbook(oracle_t *o, int r, int scheme, int s, double dt) {
    size_t n = fsize(o);
    real *Y0 = field(o, r);
    real *LY0 = (real *)malloc(n * sizeof(real)), *y1 = (real *)malloc(n * sizeof(real));
    real *y2 = (real *)malloc(n * sizeof(real)), *Ly = (real *)malloc(n * sizeof(real));
    double *mu = (double *)malloc((s + 1) * sizeof(double)), *nu = (double *)malloc((s + 1) * sizeof(double));
    double *mut = (double *)malloc((s + 1) * sizeof(double)), *gt = (double *)malloc((s + 1) * sizeof(double));
    double *b = (double *)malloc((s + 1) * sizeof(double));
    SUF(sft_oracle_sts_coeffs)(scheme, s, mu, nu, mut, gt, b);
    diffusion_op(o, r, Y0, LY0);
    real a1 = (real)(mut[1] * dt);
    for (size_t i = 0; i < n; i++) { y2[i] = Y0[i]; y1[i] = Y0[i] + a1 * LY0[i]; }
    for (int j = 2; j <= s; j++) {
        diffusion_op(o, r, y1, Ly);
        real mj = (real)mu[j], nj = (real)nu[j], cj = (real)(1.0 - mu[j] - nu[j]);
        real aj = (real)(mut[j] * dt), gj = (real)(gt[j] * dt);
        for (size_t i = 0; i < n; i++) {
            real yn = mj * y1[i] + nj * y2[i] + cj * Y0[i] + aj * Ly[i] + gj * LY0[i];
            y2[i] = y1[i];
            y1[i] = yn;
        }
    }
    memcpy(Y0, y1, n * sizeof(real));
    free(LY0); free(y1); free(y2); free(Ly); free(mu); free(nu); free(mut); free(gt); free(b);
}

/* explicit Euler diffusion step (reference scheme, :474) */
static void diffusion_euler_step(oracle_t *o, int r, double dt) {
    size_t n = fsize(o);
    real *Y = field(o, r), *LY = (real *)malloc(n * sizeof(real));
    diffusion_op(o, r, Y, LY);
    real a = (real)dt;
    for (size_t i = 0; i < n; i++) Y[i] = Y[i] + a * LY[i];
    free(LY);
}

/* --------------------------------------------------------------- advection */

/* Upwind flux (:362-366 with alpha_uw = 1): F_{i-1/2} = v B_{i-1} if v > 0, v B_i if v < 0, 0 if v = 0. */
static real upwind_flux(real v, real Bm, real Bp) {
    if (v > (real)0) return v * Bm;
    if (v < (real)0) return v * Bp;
    return (real)0;
}

/* WENO3-CS(h) face value from three split fluxes (App. B :658-676 on a uniform grid: D^{c/cm} =
 * D^{c/cp} = 1/2, D^{p/t} = D^{m/t} = 1/3, D^{cp/t} = D^{cm/t} = 2/3, reading U12):
 *   p0 = 3/2 f_near - 1/2 f_far ; p1 = 1/2 f_near + 1/2 f_other
 *   beta0 = (f_near - f_far)^2 ; beta1 = (f_other - f_near)^2
 *   w0 = (1/3)/(eps+beta0)^2 ; w1 = (2/3)/(eps+beta1)^2 ; u = (w0 p0 + w1 p1)/(w0 + w1)
 * For u^- (right-moving, from LM): far = LM_{i-2}, near = LM_{i-1}, other = LM_i.
 * For u^+ (left-moving, from LP):  far = LP_{i+1}, near = LP_i,     other = LP_{i-1}. */
static real weno3_side(real far, real near, real other, real eps) {
    real p0 = (real)1.5 * near - (real)0.5 * far;
    real p1 = (real)0.5 * near + (real)0.5 * other;
    real b0 = (near - far) * (near - far);
    real b1 = (other - near) * (other - near);
    real w0 = (real)(1.0 / 3.0) / ((eps + b0) * (eps + b0));
    real w1 = (real)(2.0 / 3.0) / ((eps + b1) * (eps + b1));
    return (w0 * p0 + w1 * p1) / (w0 + w1);
}

/* The same face value on a non-uniform grid, App. B (:662-680) with the D-factors of Smit et al. (reading U12):
 *   p0 = (1 + Dex) f_near - Dex f_far ; p1 = Da f_near + Db f_other
 *   beta0 = 4 (Dex (f_near - f_far))^2 ; beta1 = 4 (Db (f_other - f_near))^2
 *   w0 = d0/(eps+beta0)^2 ; w1 = d1/(eps+beta1)^2
 * D = (Dex, Da, Db, d0, d1): for u^- the row wm[f] of make_grid, for u^+ the row wp[f].  With (1/2, 1/2, 1/2, 1/3, 2/3) every
 * intermediate equals weno3_side's (scalings by powers of two are exact). */
static real weno3_side_nu(real far, real near, real other, real eps, const double *D) {
    real Dex = (real)D[0], Da = (real)D[1], Db = (real)D[2], d0 = (real)D[3], d1 = (real)D[4];
    real p0 = ((real)1 + Dex) * near - Dex * far;
    real p1 = Da * near + Db * other;
    real t0 = Dex * (near - far), t1 = Db * (other - near);
    real b0 = (real)4 * (t0 * t0);
    real b1 = (real)4 * (t1 * t1);
    real w0 = d0 / ((eps + b0) * (eps + b0));
    real w1 = d1 / ((eps + b1) * (eps + b1));
    return (w0 * p0 + w1 * p1) / (w0 + w1);
}

/* Steps 1-2: advection tendency F_A(B) = div_s(B v), :354, with
 *   theta-faces 1/2, 3/2, nt-1/2, nt+1/2 upwind (:388, reading U6), all others WENO3-CS(h) with
 *   LLF splitting (B2 :684): LP_i = B_i (v_{i+1/2} - alpha_i)/2, LM_i = B_i (v_{i-1/2} + alpha_i)/2,
 *   alpha_i = max|v| over faces i-5/2..i+5/2 clipped to existing faces (:689);
 *   phi-faces of rows 1..nt: WENO with the row speed v_phi = Omega_j sin(theta_j) at every face;
 *   eps_w = dth for theta-faces, dph for phi-faces (:670, reading U11);
 *   caps: north +P sum_k F_theta[1/2,k] dph, south -P sum_k F_theta[nt+1/2,k] dph (App. A :646, U5).
 * flux_mode 1 = upwind everywhere, 2 = WENO3-CS(h), 3 = WENO3 with eps_w = 1e-12 (test only, Fig. 15).
 * Ft: (nt+1)*np theta-face fluxes, Fp: (nt+2)*np phi-face fluxes, Fp[j][k] = flux at face k-1/2. */
static void advection_tendency(const oracle_t *o, int r, const real *B, real *out, int flux_mode, real *Ft, real *Fp) {
    int nt = o->nt, np = o->np;
    const double *vtd = o->vt + (size_t)r * (nt + 1);
    const double *omd = o->om + (size_t)r * (nt + 2);
    real eps_t = (real)o->dth, eps_p = (real)o->dph;
    if (flux_mode == 3) { eps_t = (real)1e-12; eps_p = (real)1e-12; }
    real *vt = (real *)malloc((nt + 1) * sizeof(real));
    real *al = (real *)malloc((nt + 2) * sizeof(real)); /* alpha_i for theta direction at rows */
    for (int j = 0; j <= nt; j++) vt[j] = (real)vtd[j];
    for (int i = 0; i <= nt + 1; i++) {
        double a = 0.0;
        for (int q = i - 3; q <= i + 2; q++) if (q >= 0 && q <= nt && fabs(vtd[q]) > a) a = fabs(vtd[q]);
        al[i] = (real)a;
    }
    /* theta-face fluxes: face f lies between rows f and f+1 (cell i = f+1, face i-1/2) */
    #pragma omp parallel for schedule(static)
    for (int f = 0; f <= nt; f++) {
        int use_upwind = (flux_mode == 1) || f <= 1 || f >= nt - 1;
        for (int k = 0; k < np; k++) {
            real F;
            if (use_upwind) {
                F = upwind_flux(vt[f], B[(size_t)f * np + k], B[(size_t)(f + 1) * np + k]);
            } else {
                int i = f + 1;
                real LMm2 = (real)0.5 * B[(size_t)(i - 2) * np + k] * (vt[i - 3] + al[i - 2]);
                real LMm1 = (real)0.5 * B[(size_t)(i - 1) * np + k] * (vt[i - 2] + al[i - 1]);
                real LM0  = (real)0.5 * B[(size_t)(i    ) * np + k] * (vt[i - 1] + al[i    ]);
                real LPp1 = (real)0.5 * B[(size_t)(i + 1) * np + k] * (vt[i + 1] - al[i + 1]);
                real LP0  = (real)0.5 * B[(size_t)(i    ) * np + k] * (vt[i    ] - al[i    ]);
                real LPm1 = (real)0.5 * B[(size_t)(i - 1) * np + k] * (vt[i - 1] - al[i - 1]);
                real ef = (flux_mode == 3) ? eps_t : (real)o->dthf[f];   /* eps_w = h, the local spacing (:670) */
                real um = weno3_side_nu(LMm2, LMm1, LM0, ef, o->wm + 5 * f);
                real up = weno3_side_nu(LPp1, LP0, LPm1, ef, o->wp + 5 * f);
                F = up + um;
            }
            Ft[(size_t)f * np + k] = F;
        }
    }
    /* phi-face fluxes for rows 1..nt: face k-1/2 lies between columns k-1 and k */
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        real v = (real)(omd[j] * o->st[j]);
        real a = (real)fabs(omd[j] * o->st[j]);
        const real *Bc = B + (size_t)j * np;
        for (int k = 0; k < np; k++) {
            int km2 = (k + np - 2) % np, km1 = (k + np - 1) % np, kp1 = (k + 1) % np;
            real F;
            if (flux_mode == 1) {
                F = upwind_flux(v, Bc[km1], Bc[k]);
            } else {
                real LMm2 = (real)0.5 * Bc[km2] * (v + a), LMm1 = (real)0.5 * Bc[km1] * (v + a), LM0 = (real)0.5 * Bc[k] * (v + a);
                real LPp1 = (real)0.5 * Bc[kp1] * (v - a), LP0 = (real)0.5 * Bc[k] * (v - a), LPm1 = (real)0.5 * Bc[km1] * (v - a);
                real um = weno3_side(LMm2, LMm1, LM0, eps_p);
                real up = weno3_side(LPp1, LP0, LPm1, eps_p);
                F = up + um;
            }
            Fp[(size_t)j * np + k] = F;
        }
    }
    /* divergence, rows 1..nt (:354) */
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        real sp = (real)o->sth[j], sm = (real)o->sth[j - 1];
        real dt_den = (real)(o->st[j] * o->dthc[j]), dp_den = (real)(o->st[j] * o->dph);
        for (int k = 0; k < np; k++) {
            int kp1 = (k + 1) % np;
            real tth = (sp * Ft[(size_t)j * np + k] - sm * Ft[(size_t)(j - 1) * np + k]) / dt_den;
            real tph = (Fp[(size_t)j * np + kp1] - Fp[(size_t)j * np + k]) / dp_den;
            out[(size_t)j * np + k] = tth + tph;
        }
    }
    kahan_t a = {0, 0}, b = {0, 0};
    for (int k = 0; k < np; k++) { kadd(&a, (double)Ft[k]); kadd(&b, (double)Ft[(size_t)nt * np + k]); }
    fill_row(out, np, (real)(o->PN * o->dph * a.s));
    fill_row(out + (size_t)(nt + 1) * np, np, (real)(-(o->PS * o->dph * b.s)));
    free(vt); free(al);
}

/* Flow attenuation, Eq. 5 (:100-103): v -> v [1 - tanh(|B_r| / B0)].  The velocities live on the faces (:284-288), B_r at
 * the cell centres; readings (U22, U23; the paper is silent on both):
 *   - |B_r| at a face is the magnitude of the mean of the two cells the face separates (for theta-faces 1/2 and
 *     nt+1/2 one of them is the polar cap);
 *   - the attenuated velocities are formed ONCE per time step from the field at the start of the step and kept fixed
 *     through the SSPRK stages (and through both half steps of a Strang step).
 * VT: (nt+1)*np theta-face speeds, VT[f][k] at face f+1/2 (between rows f, f+1) of column k;
 * VP: (nt+2)*np phi-face speeds, VP[j][k] at face k-1/2 (between columns k-1 and k) of row j (rows 1..nt). */
static void attenuated_velocities(const oracle_t *o, int r, const real *B, real *VT, real *VP) {
    int nt = o->nt, np = o->np;
    const double *vtd = o->vt + (size_t)r * (nt + 1);
    const double *omd = o->om + (size_t)r * (nt + 2);
    real B0 = (real)o->B0[r];
    #pragma omp parallel for schedule(static)
    for (int f = 0; f <= nt; f++) {
        real v = (real)vtd[f];
        for (int k = 0; k < np; k++) {
            real bf = (real)0.5 * (B[(size_t)f * np + k] + B[(size_t)(f + 1) * np + k]);
            VT[(size_t)f * np + k] = v * ((real)1 - (real)tanh((double)((real)fabs((double)bf) / B0)));
        }
    }
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        real v = (real)(omd[j] * o->st[j]);
        for (int k = 0; k < np; k++) {
            int km1 = (k + np - 1) % np;
            real bf = (real)0.5 * (B[(size_t)j * np + km1] + B[(size_t)j * np + k]);
            VP[(size_t)j * np + k] = v * ((real)1 - (real)tanh((double)((real)fabs((double)bf) / B0)));
        }
    }
}

/* Steps 1-2 with face speeds that vary along both directions (flow attenuation): the same rules as
 * advection_tendency -- upwind at theta-faces 1/2, 3/2, nt-1/2, nt+1/2, WENO3-CS(h) with LLF elsewhere -- with
 * alpha_i = max |v| over the six faces i-5/2..i+5/2 ALONG THE SWEEP DIRECTION (:689), clipped to existing faces in
 * theta and periodic in phi; now both LP and LM are live in phi. */
static void advection_tendency_general(const oracle_t *o, const real *B, real *out, int flux_mode, const real *VT, const real *VP,
                                       real *Ft, real *Fp) {
    int nt = o->nt, np = o->np;
    real eps_t = (real)o->dth, eps_p = (real)o->dph;
    if (flux_mode == 3) { eps_t = (real)1e-12; eps_p = (real)1e-12; }
    #pragma omp parallel for schedule(static)
    for (int f = 0; f <= nt; f++) {
        int use_upwind = (flux_mode == 1) || f <= 1 || f >= nt - 1;
        for (int k = 0; k < np; k++) {
            real F;
            if (use_upwind) {
                F = upwind_flux(VT[(size_t)f * np + k], B[(size_t)f * np + k], B[(size_t)(f + 1) * np + k]);
            } else {
                int i = f + 1;
                real al[4];   /* alpha of cells i-2, i-1, i, i+1 */
                for (int c = 0; c < 4; c++) {
                    int ci = i - 2 + c;
                    real a = (real)0;
                    for (int q = ci - 3; q <= ci + 2; q++)
                        if (q >= 0 && q <= nt) { real t = (real)fabs((double)VT[(size_t)q * np + k]); if (t > a) a = t; }
                    al[c] = a;
                }
                #define VTF(q) VT[(size_t)(q) * np + k]
                real LMm2 = (real)0.5 * B[(size_t)(i - 2) * np + k] * (VTF(i - 3) + al[0]);
                real LMm1 = (real)0.5 * B[(size_t)(i - 1) * np + k] * (VTF(i - 2) + al[1]);
                real LM0  = (real)0.5 * B[(size_t)(i    ) * np + k] * (VTF(i - 1) + al[2]);
                real LPp1 = (real)0.5 * B[(size_t)(i + 1) * np + k] * (VTF(i + 1) - al[3]);
                real LP0  = (real)0.5 * B[(size_t)(i    ) * np + k] * (VTF(i    ) - al[2]);
                real LPm1 = (real)0.5 * B[(size_t)(i - 1) * np + k] * (VTF(i - 1) - al[1]);
                #undef VTF
                real ef = (flux_mode == 3) ? eps_t : (real)o->dthf[f];
                F = weno3_side_nu(LPp1, LP0, LPm1, ef, o->wp + 5 * f) + weno3_side_nu(LMm2, LMm1, LM0, ef, o->wm + 5 * f);
            }
            Ft[(size_t)f * np + k] = F;
        }
    }
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        const real *Bc = B + (size_t)j * np, *V = VP + (size_t)j * np;
        for (int k = 0; k < np; k++) {
            #define W(q) (((q) % np + np) % np)
            real F;
            if (flux_mode == 1) {
                F = upwind_flux(V[k], Bc[W(k - 1)], Bc[k]);
            } else {
                real al[4];   /* alpha of cells k-2, k-1, k, k+1: faces c-5/2..c+5/2 = face indices c-2..c+3 */
                for (int c = 0; c < 4; c++) {
                    int ci = k - 2 + c;
                    real a = (real)0;
                    for (int q = ci - 2; q <= ci + 3; q++) { real t = (real)fabs((double)V[W(q)]); if (t > a) a = t; }
                    al[c] = a;
                }
                real LMm2 = (real)0.5 * Bc[W(k - 2)] * (V[W(k - 2)] + al[0]);
                real LMm1 = (real)0.5 * Bc[W(k - 1)] * (V[W(k - 1)] + al[1]);
                real LM0  = (real)0.5 * Bc[k]        * (V[k]        + al[2]);
                real LPp1 = (real)0.5 * Bc[W(k + 1)] * (V[W(k + 2)] - al[3]);
                real LP0  = (real)0.5 * Bc[k]        * (V[W(k + 1)] - al[2]);
                real LPm1 = (real)0.5 * Bc[W(k - 1)] * (V[k]        - al[1]);
                F = weno3_side(LPp1, LP0, LPm1, eps_p) + weno3_side(LMm2, LMm1, LM0, eps_p);
            }
            #undef W
            Fp[(size_t)j * np + k] = F;
        }
    }
    #pragma omp parallel for schedule(static)
    for (int j = 1; j <= nt; j++) {
        real sp = (real)o->sth[j], sm = (real)o->sth[j - 1];
        real dt_den = (real)(o->st[j] * o->dthc[j]), dp_den = (real)(o->st[j] * o->dph);
        for (int k = 0; k < np; k++) {
            int kp1 = (k + 1) % np;
            real tth = (sp * Ft[(size_t)j * np + k] - sm * Ft[(size_t)(j - 1) * np + k]) / dt_den;
            real tph = (Fp[(size_t)j * np + kp1] - Fp[(size_t)j * np + k]) / dp_den;
            out[(size_t)j * np + k] = tth + tph;
        }
    }
    kahan_t a = {0, 0}, b = {0, 0};
    for (int k = 0; k < np; k++) { kadd(&a, (double)Ft[k]); kadd(&b, (double)Ft[(size_t)nt * np + k]); }
    fill_row(out, np, (real)(o->PN * o->dph * a.s));
    fill_row(out + (size_t)(nt + 1) * np, np, (real)(-(o->PS * o->dph * b.s)));
}

/* test hook: the general rule with the un-attenuated table speeds copied to every face must reproduce
 * advection_tendency bit for bit (factor 1 - tanh(0) = 1) */
void SUF(sft_oracle_advection_tendency_general)(void *h, int r, const real *in, real *out, int flux_mode, double B0) {
    oracle_t *o = (oracle_t *)h;
    int nt = o->nt, np = o->np;
    real *Ft = (real *)malloc((size_t)(nt + 1) * np * sizeof(real)), *Fp = (real *)calloc(fsize(o), sizeof(real));
    real *VT = (real *)malloc((size_t)(nt + 1) * np * sizeof(real)), *VP = (real *)calloc(fsize(o), sizeof(real));
    double keep = o->B0[r];
    o->B0[r] = B0;
    attenuated_velocities(o, r, in, VT, VP);
    o->B0[r] = keep;
    advection_tendency_general(o, in, out, flux_mode, VT, VP, Ft, Fp);
    free(Ft); free(Fp); free(VT); free(VP);
}

/* test hook: the general rule with ARBITRARY face speeds (pins of the phi sweep with phi-varying speeds and of the alpha
 * window, tests/test_oracle_general_rule.py).  VT: [nt+1][np], VT[f][k] at theta-face f+1/2 of column k; VP: [nt+2][np],
 * VP[j][k] at phi-face k-1/2 of row j (rows 1..nt used). */
void SUF(sft_oracle_advection_tendency_faces)(void *h, const real *in, real *out, int flux_mode, const real *VT, const real *VP) {
    oracle_t *o = (oracle_t *)h;
    real *Ft = (real *)malloc((size_t)(o->nt + 1) * o->np * sizeof(real)), *Fp = (real *)calloc(fsize(o), sizeof(real));
    advection_tendency_general(o, in, out, flux_mode, VT, VP, Ft, Fp);
    free(Ft); free(Fp);
}

void SUF(sft_oracle_advection_tendency)(void *h, int r, const real *in, real *out, int flux_mode) {
    oracle_t *o = (oracle_t *)h;
    real *Ft = (real *)malloc((size_t)(o->nt + 1) * o->np * sizeof(real));
    real *Fp = (real *)calloc(fsize(o), sizeof(real));
    advection_tendency(o, r, in, out, flux_mode, Ft, Fp);
    free(Ft); free(Fp);
}

/* Step 3: advection time integrators.  adv_time 1 = forward Euler (Eq. 23 :396),
 * 3 = SSPRK(3,3) (:412-416), 4 = SSPRK(4,3) (Eq. 25 :418-424). */
/* F_A with the table speeds, or with the attenuated face speeds VT, VP when flow attenuation is on */
static void tendency(const oracle_t *o, int r, const real *in, real *out, int flux_mode, const real *VT, const real *VP, real *Ft, real *Fp) {
    if (VT) advection_tendency_general(o, in, out, flux_mode, VT, VP, Ft, Fp);
    else advection_tendency(o, r, in, out, flux_mode, Ft, Fp);
}

static void advection_step(oracle_t *o, int r, int flux_mode, int adv_time, double dt) {
    size_t n = fsize(o);
    real *f = field(o, r);
    real *T = (real *)malloc(n * sizeof(real)), *f1 = (real *)malloc(n * sizeof(real)), *f2 = (real *)malloc(n * sizeof(real));
    real *Ft = (real *)malloc((size_t)(o->nt + 1) * o->np * sizeof(real)), *Fp = (real *)calloc(n, sizeof(real));
    real h = (real)dt;
    real *VT = NULL, *VP = NULL;
    if (o->B0[r] > 0.0) {   /* Eq. 5: speeds from the field at the start of the step (reading U23) */
        VT = (real *)malloc((size_t)(o->nt + 1) * o->np * sizeof(real));
        VP = (real *)calloc(n, sizeof(real));
        attenuated_velocities(o, r, o->att_src ? o->att_src : f, VT, VP);
    }
    if (adv_time == 1) {
        tendency(o, r, f, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f[i] = f[i] - h * T[i];
    } else if (adv_time == 3) {
        tendency(o, r, f, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f1[i] = f[i] - h * T[i];
        tendency(o, r, f1, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f2[i] = (real)0.75 * f[i] + (real)0.25 * f1[i] - (real)0.25 * h * T[i];
        tendency(o, r, f2, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f[i] = (real)(1.0 / 3.0) * f[i] + (real)(2.0 / 3.0) * f2[i] - (real)(2.0 / 3.0) * h * T[i];
    } else {
        tendency(o, r, f, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f1[i] = f[i] - (real)0.5 * h * T[i];
        tendency(o, r, f1, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f2[i] = f1[i] - (real)0.5 * h * T[i];
        tendency(o, r, f2, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f1[i] = (real)(2.0 / 3.0) * f[i] + (real)(1.0 / 3.0) * f2[i] - (real)(1.0 / 6.0) * h * T[i];
        tendency(o, r, f1, T, flux_mode, VT, VP, Ft, Fp);
        for (size_t i = 0; i < n; i++) f[i] = f1[i] - (real)0.5 * h * T[i];
    }
    free(T); free(f1); free(f2); free(Ft); free(Fp); free(VT); free(VP);
}

/* Advective limit, Eq. 26 form (:430) with the velocities taken as the maximum of the flanking
 * staggered values (:406): min over rows 1..nt and realizations of
 *   [ max(|v_theta,j-1/2|, |v_theta,j+1/2|)/dth + |Omega_j|/dph ]^-1      (|v_phi|/(sin(theta) dph) = |Omega|/dph)
 * No safety factor is applied here (reading U15: the caller multiplies by its CFL number). */
static double advection_dt_limit(const oracle_t *o) {
    double best = INFINITY;
    for (int r = 0; r < o->nr; r++) {
        const double *vt = o->vt + (size_t)r * (o->nt + 1), *om = o->om + (size_t)r * (o->nt + 2);
        for (int j = 1; j <= o->nt; j++) {
            double a = fabs(vt[j - 1]) > fabs(vt[j]) ? fabs(vt[j - 1]) : fabs(vt[j]);
            double rate = a / o->dthc[j] + fabs(om[j]) / o->dph;
            if (rate > 0.0 && 1.0 / rate < best) best = 1.0 / rate;
        }
    }
    return best;
}

void SUF(sft_oracle_stable_dt)(void *h, double *dt_adv, double *dt_diff) {
    *dt_adv = advection_dt_limit((oracle_t *)h);
    *dt_diff = diffusion_dt_expl((oracle_t *)h);
}


/* ------------------------------------------------ random flux emergence, Sec. 2.4 (:155-209) */

/* Counter-based generator Philox4x32-10 (Salmon et al. 2011, "Parallel random numbers: as easy as 1, 2, 3"): ten
 * rounds of  (c0,c1,c2,c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)),  keys bumped by the
 * Weyl constants after every round.  The CUDA path implements the same published algorithm on its own (ground rule:
 * each side implements the same counter-based generator); pinned by the published known-answer vectors. */
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; round++) {
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void SUF(sft_oracle_philox)(const uint32_t *ctr, const uint32_t *key, uint32_t *out) { philox4x32_10(ctr, key, out); }

/* Standard normal Y_i of cell i = (j-1) np + k of source map m of realization r (reading U27): Philox counter
 * (i, m, r, 0), key = the two halves of the seed; u1 = (x0 + 1/2) 2^-32, u2 = (x1 + 1/2) 2^-32 in (0,1);
 * Box-Muller Y = sqrt(-2 ln u1) cos(2 pi u2), always in fp64. */
static double rfe_normal(uint64_t seed, uint32_t cell, uint32_t map, uint32_t r) {
    uint32_t ctr[4] = {cell, map, r, 0u}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, x[4];
    philox4x32_10(ctr, key, x);
    double u1 = ((double)x[0] + 0.5) * (1.0 / 4294967296.0), u2 = ((double)x[1] + 0.5) * (1.0 / 4294967296.0);
    return sqrt(-2.0 * log(u1)) * cos(2.0 * PI * u2);
}

/* One flux-balanced source map (G/hr) for realization r: Eq. 13 (model 1) or Eq. 14 (model 2) on rows 1..nt, polar
 * caps 0 (reading U28), then balanced "in the same manner as Eq. 11" (:207): with Phi+- = sum of S dA over S > 0 /
 * S < 0, positive values are divided and the others multiplied by sqrt|Phi+/Phi-| (no scaling if either is 0). */
static void rfe_make_map(const oracle_t *o, int r, uint32_t map, real *S) {
    int nt = o->nt, np = o->np;
    double r2 = o->radius_cm * o->radius_cm, ncells = (double)nt * (double)np;
    memset(S, 0, fsize(o) * sizeof(real));
    for (int j = 1; j <= nt; j++) {
        double dA = o->st[j] * o->dthc[j] * o->dph * r2;
        double amp = o->rfe_model == 1 ? o->rfe_flux_per_hr / (dA * ncells) * sqrt(PI / 2.0)
                                       : o->rfe_flux_per_hr / (4.0 * PI * r2) * sqrt(PI / 2.0);
        for (int k = 0; k < np; k++)
            S[(size_t)j * np + k] = (real)(amp * rfe_normal(o->rfe_seed, (uint32_t)((j - 1) * np + k), map, (uint32_t)r));
    }
    kahan_t pp = {0, 0}, pm = {0, 0};
    for (int j = 1; j <= nt; j++) {
        double dA = o->st[j] * o->dthc[j] * o->dph;
        for (int k = 0; k < np; k++) {
            double v = (double)S[(size_t)j * np + k];
            if (v > 0) kadd(&pp, v * dA); else kadd(&pm, v * dA);
        }
    }
    if (pp.s != 0.0 && pm.s != 0.0) {
        real sc = (real)sqrt(fabs(pp.s / pm.s));
        for (int j = 1; j <= nt; j++)
            for (int k = 0; k < np; k++) {
                real v = S[(size_t)j * np + k];
                S[(size_t)j * np + k] = v > (real)0 ? v / sc : v * sc;
            }
    }
}

/* model 0 switches the source off.  flux_per_hr in G radius_cm^2 per hour (Mx/hr for radius_cm = 6.96e10); tau = the
 * lifetime tau_RFE in hours (INFINITY: the first map stays for ever).  Resets the clock to 0 and draws maps 0 and 1. */
void SUF(sft_oracle_set_rfe)(void *h, int model, double flux_per_hr, double tau, uint64_t seed) {
    oracle_t *o = (oracle_t *)h;
    o->rfe_model = model; o->rfe_flux_per_hr = flux_per_hr; o->rfe_tau = tau; o->rfe_seed = seed;
    o->time = 0.0; o->rfe_t1 = 0.0; o->rfe_next = 2;
    if (!model) return;
    if (!o->S1) { o->S1 = (real *)calloc((size_t)o->nr * fsize(o), sizeof(real)); o->S2 = (real *)calloc((size_t)o->nr * fsize(o), sizeof(real)); }
    for (int r = 0; r < o->nr; r++) {
        rfe_make_map(o, r, 0, o->S1 + (size_t)r * fsize(o));
        rfe_make_map(o, r, 1, o->S2 + (size_t)r * fsize(o));
    }
}

void SUF(sft_oracle_get_rfe_maps)(void *h, int r, real *s1, real *s2) {
    oracle_t *o = (oracle_t *)h;
    memcpy(s1, o->S1 + (size_t)r * fsize(o), fsize(o) * sizeof(real));
    memcpy(s2, o->S2 + (size_t)r * fsize(o), fsize(o) * sizeof(real));
}

/* The source advance S(B, h) at time t (reading U29): when t has reached the time of the second map, map 2 becomes map
 * 1 and a new map 2 is drawn (:207); then B <- B + h [(1 - alpha) S1 + alpha S2], alpha = (t - t1)/tau (Eq. 15),
 * i.e. forward Euler with the source frozen at the start of the advance. */
static void rfe_advance(oracle_t *o, double t, double h) {
    size_t n = fsize(o);
    while (t >= o->rfe_t1 + o->rfe_tau) {
        for (int r = 0; r < o->nr; r++) {
            memcpy(o->S1 + r * n, o->S2 + r * n, n * sizeof(real));
            rfe_make_map(o, r, o->rfe_next, o->S2 + r * n);
        }
        o->rfe_next++;
        o->rfe_t1 += o->rfe_tau;
    }
    real a = (real)((t - o->rfe_t1) / o->rfe_tau), hh = (real)h;   /* tau = inf: alpha = 0 */
    for (int r = 0; r < o->nr; r++) {
        real *B = field(o, r);
        const real *s1 = o->S1 + r * n, *s2 = o->S2 + r * n;
        for (size_t i = 0; i < n; i++) B[i] = B[i] + hh * (((real)1 - a) * s1[i] + a * s2[i]);
    }
}

/* ------------------------------------------------------------------- step */

/* Step 8: n_steps of B^{n+1} = D(A(B^n)) (Eq. 21 :308-313, S omitted).
 * adv_flux 0 off / 1 upwind / 2 WENO3-CS(h) / 3 WENO3 eps=1e-12 (test only);
 * adv_time 1 / 3 / 4; diff_time 0 off / 1 Euler / 2 RKL2 / 3 RKG2(3/2) / 12, 13 = textbook-form
 * RKL2 / RKG2 (test only); sts_stages 0 = auto (Step 6) else forced.  Returns the stage count used. */
int SUF(sft_oracle_step_ex)(void *h, int n_steps, double dt, int adv_flux, int adv_time, int diff_time, int sts_stages, int split) {
    oracle_t *o = (oracle_t *)h;
    int s = 0;
    if (diff_time == 2 || diff_time == 3 || diff_time == 12 || diff_time == 13) {
        int scheme = diff_time % 10;
        s = sts_stages > 0 ? sts_stages : sts_stage_count(scheme, dt, diffusion_dt_expl(o));
        if (s < 2) return -1;
    }
    for (int n = 0; n < n_steps; n++) {
        /* Eq. 21: A, D, S.  Eq. 22 (Strang): S(dt/2), A(dt/2), D(dt), A(dt/2), S(dt/2). */
        if (o->rfe_model && split) rfe_advance(o, o->time, 0.5 * dt);
        for (int r = 0; r < o->nr; r++) {
            real *start = NULL;
            if (split && adv_flux != 0 && o->B0[r] > 0.0) {   /* reading U23: one set of attenuated speeds per step */
                start = (real *)malloc(fsize(o) * sizeof(real));
                memcpy(start, field(o, r), fsize(o) * sizeof(real));
                o->att_src = start;
            }
            if (adv_flux != 0) advection_step(o, r, adv_flux, adv_time, split ? 0.5 * dt : dt);
            if (diff_time == 1) diffusion_euler_step(o, r, dt);
            else if (diff_time == 2 || diff_time == 3) sts_step(o, r, diff_time, s, dt);
            else if (diff_time == 12 || diff_time == 13) sts_step_textbook(o, r, diff_time % 10, s, dt);
            if (split && adv_flux != 0) advection_step(o, r, adv_flux, adv_time, 0.5 * dt);
            o->att_src = NULL;
            free(start);
        }
        if (o->rfe_model) {
            if (split) rfe_advance(o, o->time + 0.5 * dt, 0.5 * dt);
            else rfe_advance(o, o->time, dt);
        }
        o->time += dt;
    }
    return s;
}

int SUF(sft_oracle_step)(void *h, int n_steps, double dt, int adv_flux, int adv_time, int diff_time, int sts_stages) {
    return SUF(sft_oracle_step_ex)(h, n_steps, dt, adv_flux, adv_time, diff_time, sts_stages, 0);
}

/* ----------------------------------------------------- assimilation, Step 9 */

/* Eq. 8 (:131): B <- F B_d + (1-F) B on rows 1..nt; flags bit0: flux-balanced form Eq. 10-11
 * (:144-153): dB = F (B_d - B); Phi+ / Phi- = surface integrals of dB over dB > 0 / dB <= 0;
 * dB > 0 is divided by sqrt|Phi+/Phi-|, dB <= 0 multiplied by it; if either is 0, no scaling.
 * Caps (reading U18): cap obs and cap weight are the dph-weighted means of the adjacent row's obs and
 * weight, the cap is blended with them like any cell (one value, stored replicated).
 * obs, w: [nr or 1][nt][np] (`shared` != 0: one map for all realizations). Quadrature (reading U19):
 * dA_j = sin(theta_j) dth dph, cap area Apole. */
void SUF(sft_oracle_assimilate)(void *h, const real *obs, const real *w, int shared, int flags) {
    oracle_t *o = (oracle_t *)h;
    int nt = o->nt, np = o->np;
    size_t mapn = (size_t)nt * np;
    for (int r = 0; r < o->nr; r++) {
        const real *ob = obs + (shared ? 0 : (size_t)r * mapn);
        const real *wt = w + (shared ? 0 : (size_t)r * mapn);
        real *B = field(o, r);
        real obN = (real)row_mean(ob, np), obS = (real)row_mean(ob + (size_t)(nt - 1) * np, np);
        real wN = (real)row_mean(wt, np), wS = (real)row_mean(wt + (size_t)(nt - 1) * np, np);
        if (!(flags & 1)) {
            for (int j = 1; j <= nt; j++)
                for (int k = 0; k < np; k++) {
                    real F = wt[(size_t)(j - 1) * np + k], Bd = ob[(size_t)(j - 1) * np + k];
                    B[(size_t)j * np + k] = F * Bd + ((real)1 - F) * B[(size_t)j * np + k];
                }
            fill_row(B, np, wN * obN + ((real)1 - wN) * B[0]);
            fill_row(B + (size_t)(nt + 1) * np, np, wS * obS + ((real)1 - wS) * B[(size_t)(nt + 1) * np]);
        } else {
            kahan_t pp = {0, 0}, pm = {0, 0};
            real dN = wN * (obN - B[0]), dS = wS * (obS - B[(size_t)(nt + 1) * np]);
            if (dN > (real)0) kadd(&pp, (double)dN * o->ApoleN); else kadd(&pm, (double)dN * o->ApoleN);
            for (int j = 1; j <= nt; j++) {
                double dA = o->st[j] * o->dthc[j] * o->dph;
                for (int k = 0; k < np; k++) {
                    real d = wt[(size_t)(j - 1) * np + k] * (ob[(size_t)(j - 1) * np + k] - B[(size_t)j * np + k]);
                    if (d > (real)0) kadd(&pp, (double)d * dA); else kadd(&pm, (double)d * dA);
                }
            }
            if (dS > (real)0) kadd(&pp, (double)dS * o->ApoleS); else kadd(&pm, (double)dS * o->ApoleS);
            real sc = (real)1;
            if (pp.s != 0.0 && pm.s != 0.0) sc = (real)sqrt(fabs(pp.s / pm.s));
            for (int j = 1; j <= nt; j++)
                for (int k = 0; k < np; k++) {
                    real d = wt[(size_t)(j - 1) * np + k] * (ob[(size_t)(j - 1) * np + k] - B[(size_t)j * np + k]);
                    d = (d > (real)0) ? d / sc : d * sc;
                    B[(size_t)j * np + k] = B[(size_t)j * np + k] + d;
                }
            dN = (dN > (real)0) ? dN / sc : dN * sc;
            dS = (dS > (real)0) ? dS / sc : dS * sc;
            fill_row(B, np, B[0] + dN);
            fill_row(B + (size_t)(nt + 1) * np, np, B[(size_t)(nt + 1) * np] + dS);
        }
    }
}

/* ------------------------------------------------------ diagnostics, Step 10 */

/* :225-230: Phi+ = int_{B>0} B dOmega, Phi- = int_{B<0} B dOmega; out[r] = {signed = Phi+ + Phi-,
 * unsigned = Phi+ - Phi-, Phi+, Phi-}, midpoint quadrature dA_j = sin(theta_j) dth dph plus the two
 * caps with area Apole (reading U19), times radius_cm^2 (Mx if B is in Gauss; 1 = unit sphere). */
void SUF(sft_oracle_diagnostics)(void *h, double *out /*[nr][4]*/) {
    oracle_t *o = (oracle_t *)h;
    int nt = o->nt, np = o->np;
    double r2 = o->radius_cm * o->radius_cm;
    for (int r = 0; r < o->nr; r++) {
        const real *B = field(o, r);
        kahan_t pp = {0, 0}, pm = {0, 0};
        double c0 = (double)B[0];
        if (c0 > 0) kadd(&pp, c0 * o->ApoleN); else if (c0 < 0) kadd(&pm, c0 * o->ApoleN);
        for (int j = 1; j <= nt; j++) {
            double dA = o->st[j] * o->dthc[j] * o->dph;
            for (int k = 0; k < np; k++) {
                double v = (double)B[(size_t)j * np + k];
                if (v > 0) kadd(&pp, v * dA); else if (v < 0) kadd(&pm, v * dA);
            }
        }
        double c1 = (double)B[(size_t)(nt + 1) * np];
        if (c1 > 0) kadd(&pp, c1 * o->ApoleS); else if (c1 < 0) kadd(&pm, c1 * o->ApoleS);
        out[4 * r + 0] = (pp.s + pm.s) * r2;
        out[4 * r + 1] = (pp.s - pm.s) * r2;
        out[4 * r + 2] = pp.s * r2;
        out[4 * r + 3] = pm.s * r2;
    }
}

/* Remaining run-history quantities (:230-242): out[r][13] =
 *   0..3  Phi+ and Phi- limited to the north polar region, then to the south polar region: the cells whose centre has
 *         |latitude| >= lat_cut_deg, i.e. theta_j <= thc or theta_j >= pi - thc with thc = (90 - lat_cut_deg) pi/180,
 *         caps included (x radius_cm^2);
 *   4, 5  area of the two regions (x radius_cm^2);
 *   6..8  min, max and min |B_r| over the whole map (caps included);
 *   9     H = sqrt(h1^2 + h2^2) (Eq. 16), 10  D (Eq. 17), 11 h1 (Eq. 16a), 12 h2 (Eq. 16b), with
 *         dOmega = sin(theta) dtheta dphi on the unit sphere and the quadrature weights of reading U19;
 *         a cap sits at sin(theta) = 0, cos(theta) = +-1: it contributes to D only. */
void SUF(sft_oracle_diagnostics_ext)(void *h, double lat_cut_deg, double *out /*[nr][13]*/) {
    oracle_t *o = (oracle_t *)h;
    int nt = o->nt, np = o->np;
    double r2 = o->radius_cm * o->radius_cm;
    double thc = (90.0 - lat_cut_deg) * PI / 180.0;
    for (int r = 0; r < o->nr; r++) {
        const real *B = field(o, r);
        kahan_t f[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}}, area[2] = {{0, 0}, {0, 0}}, h1 = {0, 0}, h2 = {0, 0}, d = {0, 0};
        double bmin = (double)B[0], bmax = (double)B[0], amin = fabs((double)B[0]);
        for (int j = 0; j <= nt + 1; j++) {
            int cap = (j == 0 || j == nt + 1);
            double th = o->th[j];
            double dA = cap ? (j == 0 ? o->ApoleN : o->ApoleS) : o->st[j] * o->dthc[j] * o->dph;
            int region = (th <= thc) ? 0 : (th >= PI - thc ? 1 : -1);
            int ncol = cap ? 1 : np;   /* a cap is one cell (stored replicated) */
            for (int k = 0; k < ncol; k++) {
                double v = (double)B[(size_t)j * np + k];
                if (v < bmin) bmin = v;
                if (v > bmax) bmax = v;
                if (fabs(v) < amin) amin = fabs(v);
                if (region >= 0) {
                    if (v > 0) kadd(&f[2 * region], v * dA); else if (v < 0) kadd(&f[2 * region + 1], v * dA);
                    kadd(&area[region], dA);
                }
                if (cap) {
                    kadd(&d, v * (j == 0 ? 1.0 : -1.0) * dA);
                } else {
                    double ph = (double)k * o->dph;
                    kadd(&h1, v * o->st[j] * cos(ph) * dA);
                    kadd(&h2, v * o->st[j] * sin(ph) * dA);
                    kadd(&d, v * cos(th) * dA);
                }
            }
        }
        double *q = out + 13 * r, c = 3.0 / (4.0 * PI);
        for (int i = 0; i < 4; i++) q[i] = f[i].s * r2;
        q[4] = area[0].s * r2; q[5] = area[1].s * r2;
        q[6] = bmin; q[7] = bmax; q[8] = amin;
        q[11] = c * h1.s; q[12] = c * h2.s; q[10] = c * d.s;
        q[9] = sqrt(q[11] * q[11] + q[12] * q[12]);
    }
}
