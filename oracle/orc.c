/*
 * orc.c -- fp64 CPU ORACLE (test infrastructure, NOT the product; see orc.h).
 *
 * Plain, slow, step-by-step restatement of the particle hot path of arXiv 2511.17710 in the
 * paper's order and notation.  P:nnn = line nnn of PAPER.md.  No tiling, no sorting, no fusion,
 * absolute coordinates, OpenMP over particles only.  Shares nothing with the CUDA path.
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NG ORC_NGHOST
static const double PI = 3.14159265358979323846264338327950288;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_set_num_threads(int n) {
    int prev = orc_num_threads();
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#endif
    return prev;
}

/* ------------------------------------------------------------------------------------------
 * array geometry: planar padded arrays, x1 fastest, N_GHOST = 2 each side.
 * element (i,j,k) of the active grid sits at padded index (i+2, j+2, k+2).
 * ------------------------------------------------------------------------------------------ */
static inline int64_t pext(const orc_grid *g, int d) { return d < g->D ? (int64_t)g->N[d] + 2 * NG : 1; }
int64_t orc_padded_size(const orc_grid *g) { return pext(g, 0) * pext(g, 1) * pext(g, 2); }
static inline int64_t pidx(const orc_grid *g, int i, int j, int k) {
    int64_t P0 = pext(g, 0), P1 = pext(g, 1);
    if (g->D == 2) return (int64_t)(i + NG) + P0 * (int64_t)(j + NG);
    return (int64_t)(i + NG) + P0 * ((int64_t)(j + NG) + P1 * (int64_t)(k + NG));
}

/* ------------------------------------------------------------------------------------------
 * O1  metric
 * ------------------------------------------------------------------------------------------ */
static inline double cell_size(const orc_grid *g, int d) { return (g->xmax[d] - g->xmin[d]) / (double)g->N[d]; }

double orc_theta_of_T(double vt, double T) {
    return T + 2.0 * vt * T * (1.0 - 2.0 * T / PI) * (1.0 - T / PI);
}
double orc_dtheta_dT(double vt, double T) {
    return 1.0 + 2.0 * vt + 12.0 * vt * (T / PI) * (T / PI - 1.0);
}

/* quasi-spherical helpers */
static inline double qs_Rmin(const orc_grid *g) { return log(g->xmin[0] - g->r0); }
static inline double qs_dR(const orc_grid *g) { return (log(g->xmax[0] - g->r0) - log(g->xmin[0] - g->r0)) / (double)g->N[0]; }
static inline double qs_dT(const orc_grid *g) { return PI / (double)g->N[1]; }

/* (r, theta) of a code position for the two axisymmetric metrics */
static void r_theta_of_code(const orc_grid *g, double x1, double x2, double *r, double *th) {
    if (g->kind == ORC_SPH) {
        *r = g->xmin[0] + x1 * cell_size(g, 0);
        *th = x2 * (PI / (double)g->N[1]);
    } else {
        double R = qs_Rmin(g) + x1 * qs_dR(g);
        double T = x2 * qs_dT(g);
        *r = g->r0 + exp(R);
        *th = orc_theta_of_T(g->vartheta, T);
    }
}

void orc_metric_h(const orc_grid *g, const double x[3], double h[3]) {
    if (g->kind == ORC_CART) {
        for (int d = 0; d < 3; ++d) {
            if (d < g->D) { double dx = cell_size(g, d); h[d] = dx * dx; }
            else h[d] = 1.0;
        }
    } else if (g->kind == ORC_SPH) {
        double dr = cell_size(g, 0), dth = PI / (double)g->N[1];
        double r = g->xmin[0] + x[0] * dr, th = x[1] * dth;
        h[0] = dr * dr;
        h[1] = (r * dth) * (r * dth);
        h[2] = (r * sin(th)) * (r * sin(th));
    } else {
        double dR = qs_dR(g), dT = qs_dT(g);
        double R = qs_Rmin(g) + x[0] * dR, T = x[1] * dT;
        double eR = exp(R), r = g->r0 + eR;
        double th = orc_theta_of_T(g->vartheta, T), dthdT = orc_dtheta_dT(g->vartheta, T);
        h[0] = (dR * eR) * (dR * eR);
        h[1] = (dT * dthdT * r) * (dT * dthdT * r);
        h[2] = (r * sin(th)) * (r * sin(th));
    }
}

/* the same at n positions (x1[k], x2[k], 0): h[3*k + d]; a loop over orc_metric_h, for the test helpers */
void orc_metric_h_many(const orc_grid *g, int64_t n, const double *x1, const double *x2, double *h) {
    for (int64_t k = 0; k < n; ++k) { double x[3] = { x1[k], x2[k], 0.0 }; orc_metric_h(g, x, h + 3 * k); }
}

/* Eq. 8: min over cell centres of (sum_d 1/h_dd)^(-1/2), d < D */
double orc_dx_min(const orc_grid *g) {
    double best = INFINITY;
    int K = g->D == 3 ? g->N[2] : 1;
    for (int k = 0; k < K; ++k)
        for (int j = 0; j < g->N[1]; ++j)
            for (int i = 0; i < g->N[0]; ++i) {
                double x[3] = { i + 0.5, j + 0.5, k + 0.5 }, h[3];
                orc_metric_h(g, x, h);
                double s = 0.0;
                for (int d = 0; d < g->D; ++d) s += 1.0 / h[d];
                double v = 1.0 / sqrt(s);
                if (v < best) best = v;
            }
    return best;
}

/* App. B: inverse of theta(T).  With s = T/pi the cubic is
 *   4 vt s^3 - 6 vt s^2 + (1 + 2 vt) s - theta/pi = 0,
 * depressed with u = s - 1/2:  4 vt u^3 + (1 - vt) u + (1/2 - theta/pi) = 0  (one real root for 0 < vt < 1).
 * Cardano on the depressed form, then two Newton steps on theta(T) - theta. */
double orc_T_of_theta(double vt, double theta) {
    if (vt == 0.0) return theta;                        /* "only performed when vartheta != 0" */
    double p = (1.0 - vt) / (4.0 * vt);
    double q = (0.5 - theta / PI) / (4.0 * vt);
    double disc = sqrt(q * q / 4.0 + p * p * p / 27.0);
    double u = cbrt(-q / 2.0 + disc) + cbrt(-q / 2.0 - disc);
    double T = PI * (u + 0.5);
    for (int it = 0; it < 2; ++it) T -= (orc_theta_of_T(vt, T) - theta) / orc_dtheta_dT(vt, T);
    return T;
}

/* Eq. (B3) evaluated literally; `theta` and `vt` as printed.  The extracted text has the radicand
 * pi^2 (4 - vt)(1 + 2 vt); the algebra requires (1 + 2 vt)^2.  The sign of vt selects:
 * vt > 0 -> corrected radicand, vt < 0 -> |vt| with the radicand exactly as printed (for the pin test). */
double orc_T_of_theta_printed_B3(double vt_signed, double theta) {
    int printed = vt_signed < 0.0;
    double vt = fabs(vt_signed);
    double f = printed ? (1.0 + 2.0 * vt) : (1.0 + 2.0 * vt) * (1.0 + 2.0 * vt);
    double rad = 108.0 * vt * theta * theta - 108.0 * vt * PI * theta + PI * PI * (4.0 - vt) * f;
    double Theta = cbrt(sqrt(3.0 * vt * vt * vt) * sqrt(rad) - 9.0 * vt * vt * (PI - 2.0 * theta));
    return pow(PI, 2.0 / 3.0) / 12.0 *
           (6.0 * cbrt(PI) - pow(2.0, 4.0 / 3.0) * pow(3.0 * PI, 2.0 / 3.0) * (1.0 - vt) / Theta +
            pow(2.0, 2.0 / 3.0) * cbrt(3.0) * Theta / vt);
}

/* ------------------------------------------------------------------------------------------
 * O5 / O6  coordinate maps
 * ------------------------------------------------------------------------------------------ */
void orc_code_to_cart(const orc_grid *g, const double x[3], double X[3]) {
    if (g->kind == ORC_CART) {
        for (int d = 0; d < 3; ++d) X[d] = d < g->D ? g->xmin[d] + x[d] * cell_size(g, d) : x[d];
        return;
    }
    double r, th, phi = x[2];
    r_theta_of_code(g, x[0], x[1], &r, &th);            /* P:285 / P:305-310 */
    X[0] = r * sin(th) * cos(phi);                      /* P:287-289 / P:311-315 */
    X[1] = r * sin(th) * sin(phi);
    X[2] = r * cos(th);
}

void orc_cart_to_code(const orc_grid *g, const double X[3], double x[3]) {
    if (g->kind == ORC_CART) {
        for (int d = 0; d < 3; ++d) x[d] = d < g->D ? (X[d] - g->xmin[d]) / cell_size(g, d) : X[d];
        return;
    }
    double r = sqrt(X[0] * X[0] + X[1] * X[1] + X[2] * X[2]);          /* P:294 / P:320 */
    double th = PI / 2.0 - atan2(X[2], sqrt(X[0] * X[0] + X[1] * X[1])); /* P:296 / P:322 */
    double phi = PI - atan2(X[1], -X[0]);                                /* P:297 / P:323 */
    if (phi >= 2.0 * PI) phi -= 2.0 * PI;               /* atan2 = -pi exactly (y = -0) would give 2 pi */
    if (g->kind == ORC_SPH) {
        x[0] = (r - g->xmin[0]) / cell_size(g, 0);
        x[1] = th / (PI / (double)g->N[1]);
    } else {
        x[0] = (log(r - g->r0) - qs_Rmin(g)) / qs_dR(g);
        x[1] = orc_T_of_theta(g->vartheta, th) / qs_dT(g);
    }
    x[2] = phi;
}

/* ------------------------------------------------------------------------------------------
 * O2  gather, P:131-133 with the first-order (cloud-in-cell) shape, reading G1:
 * direct multilinear interpolation of each component on its own staggered lattice.
 * Yee staggering:  E1(i+1/2,j,k) E2(i,j+1/2,k) E3(i,j,k+1/2)
 *                                      B1(i,j+1/2,k+1/2) B2(i+1/2,j,k+1/2) B3(i+1/2,j+1/2,k)
 * ------------------------------------------------------------------------------------------ */
static const int STAG[6][3] = { {1,0,0}, {0,1,0}, {0,0,1}, {0,1,1}, {1,0,1}, {1,1,0} };  /* 1 = half-cell shift */

void orc_gather(const orc_grid *g, const float *const F[6], const int32_t i[3], const double d[3], double out[6]) {
    for (int c = 0; c < 6; ++c) {
        int b[3] = {0, 0, 0};
        double f[3] = {0, 0, 0};
        for (int a = 0; a < g->D; ++a) {
            if (!STAG[c][a]) { b[a] = i[a]; f[a] = d[a]; }
            else if (d[a] < 0.5) { b[a] = i[a] - 1; f[a] = d[a] + 0.5; }
            else { b[a] = i[a]; f[a] = d[a] - 0.5; }
        }
        double acc = 0.0;
        int nk = g->D == 3 ? 2 : 1;
        for (int ck = 0; ck < nk; ++ck)
            for (int cj = 0; cj < 2; ++cj)
                for (int ci = 0; ci < 2; ++ci) {
                    double wgt = (ci ? f[0] : 1.0 - f[0]) * (cj ? f[1] : 1.0 - f[1]);
                    if (g->D == 3) wgt *= (ck ? f[2] : 1.0 - f[2]);
                    acc += wgt * (double)F[c][pidx(g, b[0] + ci, b[1] + cj, g->D == 3 ? b[2] + ck : 0)];
                }
        out[c] = acc;
    }
}

/* ------------------------------------------------------------------------------------------
 * O3  basis change: tetrad A^hat{i} = sqrt(h_ii) A^i at the particle (G2, G5), then for the
 * axisymmetric metrics the rotation (r,theta,phi)-hat -> (x,y,z)-hat, i.e. the normalised Jacobian
 * of P:287-289.  x = (x1, x2, x3) code position, with x3 = phi for the axisymmetric metrics.
 * ------------------------------------------------------------------------------------------ */
void orc_to_cartesian_basis(const orc_grid *g, const double x[3], const double A[3], double out[3]) {
    double h[3];
    orc_metric_h(g, x, h);
    double Ar = sqrt(h[0]) * A[0], At = sqrt(h[1]) * A[1], Ap = sqrt(h[2]) * A[2];
    if (g->kind == ORC_CART) { out[0] = Ar; out[1] = At; out[2] = Ap; return; }
    double r, th, phi = x[2];
    r_theta_of_code(g, x[0], x[1], &r, &th);
    double st = sin(th), ct = cos(th), sp = sin(phi), cp = cos(phi);
    out[0] = Ar * st * cp + At * ct * cp - Ap * sp;
    out[1] = Ar * st * sp + At * ct * sp + Ap * cp;
    out[2] = Ar * ct - At * st;
}

/* ------------------------------------------------------------------------------------------
 * O4  relativistic Boris (Eq. 3, reading G3): half electric kick, rotation, half kick.
 * ------------------------------------------------------------------------------------------ */
void orc_boris(double u[3], const double E[3], const double B[3], double qm, double dt) {
    double eps = qm * dt / 2.0;
    double um[3], t[3], s[3], up[3], uplus[3];
    for (int a = 0; a < 3; ++a) um[a] = u[a] + eps * E[a];
    double gm = sqrt(1.0 + um[0] * um[0] + um[1] * um[1] + um[2] * um[2]);
    for (int a = 0; a < 3; ++a) t[a] = eps * B[a] / gm;
    double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
    for (int a = 0; a < 3; ++a) s[a] = 2.0 * t[a] / (1.0 + t2);
    up[0] = um[0] + (um[1] * t[2] - um[2] * t[1]);
    up[1] = um[1] + (um[2] * t[0] - um[0] * t[2]);
    up[2] = um[2] + (um[0] * t[1] - um[1] * t[0]);
    uplus[0] = um[0] + (up[1] * s[2] - up[2] * s[1]);
    uplus[1] = um[1] + (up[2] * s[0] - up[0] * s[2]);
    uplus[2] = um[2] + (up[0] * s[1] - up[1] * s[0]);
    for (int a = 0; a < 3; ++a) u[a] = uplus[a] + eps * E[a];
}

/* ------------------------------------------------------------------------------------------
 * N3  the other "conventional particle pusher" P:95 names: J.-L. Vay, Phys. Plasmas 15, 056701 (2008).  Same interface and time
 * levels as orc_boris (u^(n-1/2) -> u^(n+1/2), fields at n).  Written out from the published scheme:
 *   u'   = u + eps (E + v x B) + eps E,  v = u / gamma(u),  eps = (q/m) dt / 2         (half step with the old velocity, then half E kick)
 *   tau  = eps B,  u* = u'.tau,  sigma = gamma'^2 - tau^2,  gamma'^2 = 1 + u'^2
 *   gamma_new^2 = [ sigma + sqrt(sigma^2 + 4 (tau^2 + u*^2)) ] / 2
 *   t = tau / gamma_new,  u_new = [ u' + (u'.t) t + u' x t ] / (1 + t^2)
 * ------------------------------------------------------------------------------------------ */
void orc_vay(double u[3], const double E[3], const double B[3], double qm, double dt) {
    double eps = qm * dt / 2.0;
    double g0 = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    double v[3] = { u[0] / g0, u[1] / g0, u[2] / g0 };
    double up[3], tau[3], t[3];
    up[0] = u[0] + eps * (2.0 * E[0] + (v[1] * B[2] - v[2] * B[1]));
    up[1] = u[1] + eps * (2.0 * E[1] + (v[2] * B[0] - v[0] * B[2]));
    up[2] = u[2] + eps * (2.0 * E[2] + (v[0] * B[1] - v[1] * B[0]));
    for (int a = 0; a < 3; ++a) tau[a] = eps * B[a];
    double tau2 = tau[0] * tau[0] + tau[1] * tau[1] + tau[2] * tau[2];
    double ustar = up[0] * tau[0] + up[1] * tau[1] + up[2] * tau[2];
    double gp2 = 1.0 + up[0] * up[0] + up[1] * up[1] + up[2] * up[2];
    double sigma = gp2 - tau2;
    double gnew = sqrt(0.5 * (sigma + sqrt(sigma * sigma + 4.0 * (tau2 + ustar * ustar))));
    for (int a = 0; a < 3; ++a) t[a] = tau[a] / gnew;
    double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
    double udt = up[0] * t[0] + up[1] * t[1] + up[2] * t[2];
    double sfac = 1.0 / (1.0 + t2);
    u[0] = sfac * (up[0] + udt * t[0] + (up[1] * t[2] - up[2] * t[1]));
    u[1] = sfac * (up[1] + udt * t[1] + (up[2] * t[0] - up[0] * t[2]));
    u[2] = sfac * (up[2] + udt * t[2] + (up[0] * t[1] - up[1] * t[0]));
}

static int orc_pusher_kind = 0;           /* 0 = Boris (default), 1 = Vay, 2 = Boris,GCA, 3 = Vay,GCA; read by orc_gather_push */
int orc_set_pusher(int kind) { int prev = orc_pusher_kind; if (kind >= 0 && kind <= 3) orc_pusher_kind = kind; return prev; }

/* N3, the hybrid pusher of P:976-980 ("Boris,GCA" / "Vay,GCA", fn. 21).  The paper gives two sentences: the pusher "switches between
 * the conventional algorithm ... and the guiding center approximation ... depending on the ratio of |E|/|B| and the particle's
 * nominal gyroradius at a given timestep, rho_L ~ gamma beta m c^2 / q|B|", with "the critical Larmor radius for the transition" an
 * input, and "in the guiding center regime, the particle's momentum perpendicular to the local magnetic field is set to zero,
 * effectively reducing its motion to that of its guiding center".  Reading (G26; parity unpinned beyond those sentences,
 * the cited scheme of Bacchini et al. 2020 is not in the paper): with E, B the fields at the particle in the orthonormal basis and
 * u the momentum BEFORE the push (the "given timestep"), the guiding-centre regime holds when
 *     |B| > 0,   |E| < eovb |B|,   rho_L = |u| m / (|q| |B|) < rho_crit            (c = 1; eovb, rho_crit: inputs)
 * and then the conventional push is followed by u <- (u . b) b, b = B/|B|: the rotation about B leaves u.b alone, so this is
 * u_par + (q/m) E_par dt along b with u_perp = 0; the move of sub-step 6 is unchanged (the particle slides along the field line). */
static double orc_gca_rho = 0.0, orc_gca_eovb = 0.0;
void orc_set_gca(double rho_crit, double eovb) { orc_gca_rho = rho_crit; orc_gca_eovb = eovb; }
int orc_gca_project(double u[3], const double u_before[3], const double E[3], const double B[3], double qm) {
    double B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2], E2 = E[0] * E[0] + E[1] * E[1] + E[2] * E[2];
    double U2 = u_before[0] * u_before[0] + u_before[1] * u_before[1] + u_before[2] * u_before[2];
    double k = orc_gca_rho * fabs(qm);                                   /* rho_L < rho_crit  <=>  |u|^2 < (rho_crit |q|/m)^2 |B|^2 */
    if (!(B2 > 0.0) || !(E2 < orc_gca_eovb * orc_gca_eovb * B2) || !(U2 < k * k * B2)) return 0;
    double up = (u[0] * B[0] + u[1] * B[1] + u[2] * B[2]) / B2;
    for (int a = 0; a < 3; ++a) u[a] = up * B[a];
    return 1;
}

/* ------------------------------------------------------------------------------------------
 * steps 3-7 + O7 crossing bookkeeping (readings G9, G11)
 * ------------------------------------------------------------------------------------------ */
static inline int floor_mod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

int orc_gather_push(const orc_grid *g, const float *const F[6], const orc_particles *in, orc_particles *out,
                    double qm, double dt) {
    const int D = g->D, axisym = g->kind != ORC_CART;
    if (axisym && D != 2) return -1;
    int64_t n = in->n;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        int alive = in->tag ? in->tag[p] != 0 : 1;
        int32_t ic[3] = {0, 0, 0};
        double dc[3] = {0, 0, 0}, u[3];
        for (int a = 0; a < D; ++a) { ic[a] = in->i[a][p]; dc[a] = in->d[a][p]; }
        for (int a = 0; a < 3; ++a) u[a] = in->u[a][p];
        double phi = axisym ? in->phi[p] : 0.0;
        int tag = alive;
        if (alive) {
            /* step 3: interpolate */
            double EB[6];
            orc_gather(g, F, ic, dc, EB);
            /* step 4: to the global Cartesian basis, at the particle position */
            double x[3] = { ic[0] + dc[0], ic[1] + dc[1], axisym ? phi : (D == 3 ? ic[2] + dc[2] : 0.0) };
            double E[3], B[3];
            orc_to_cartesian_basis(g, x, EB, E);
            orc_to_cartesian_basis(g, x, EB + 3, B);
            /* step 5: u^(n-1/2) -> u^(n+1/2) */
            double u_before[3] = { u[0], u[1], u[2] };
            if (orc_pusher_kind & 1) orc_vay(u, E, B, qm, dt); else orc_boris(u, E, B, qm, dt);
            if (orc_pusher_kind & 2) orc_gca_project(u, u_before, E, B, qm);
            /* step 6: x^(n) -> x^(n+1) with u^(n+1/2) / gamma^(n+1/2), in the global Cartesian frame */
            double gam = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
            double X[3], xn[3];
            orc_code_to_cart(g, x, X);
            if (g->kind == ORC_CART) { for (int a = 0; a < D; ++a) X[a] += u[a] / gam * dt; }
            else { for (int a = 0; a < 3; ++a) X[a] += u[a] / gam * dt; }
            /* step 7: back to code coordinates */
            orc_cart_to_code(g, X, xn);
            if (axisym) phi = xn[2];
            /* O7: split into cell index and offset, apply the boundary rule of each dimension */
            for (int a = 0; a < D; ++a) {
                double fl = floor(xn[a]);
                int inew = (int)fl;
                double dnew = xn[a] - fl;
                if (g->bc[a] == ORC_PERIODIC) inew = floor_mod(inew, g->N[a]);
                else if (g->bc[a] == ORC_AXIS) {
                    if (inew >= g->N[a]) { inew = g->N[a] - 1; dnew = nextafter(1.0, 0.0); }   /* theta = pi exactly, G11 */
                    if (inew < 0) { inew = 0; dnew = 0.0; }
                } else if (inew < 0 || inew >= g->N[a]) tag = 0;                               /* ABSORB, G9 */
                ic[a] = inew; dc[a] = dnew;
            }
        }
        for (int a = 0; a < D; ++a) { out->i[a][p] = ic[a]; out->d[a][p] = dc[a]; }
        for (int a = 0; a < 3; ++a) out->u[a][p] = u[a];
        if (axisym) out->phi[p] = phi;
        if (out->w && in->w && out->w != in->w) out->w[p] = in->w[p];
        if (out->tag) out->tag[p] = (int8_t)tag;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O8  deposit (Eq. 6, P:155-157 step 8, "modified zig-zag"; readings G6-G8)
 * ------------------------------------------------------------------------------------------ */
static inline double omega(double W, int s) { return s ? W : 1.0 - W; }

static inline void jadd(double *J, int64_t idx, double v) {
#pragma omp atomic
    J[idx] += v;
}

/* one straight segment inside cell c: displacement Dv, midpoint offset W (cell-local), Q = q w / dt */
static void deposit_segment_3d(const orc_grid *g, double *const J[3], const int c[3], const double Dv[3], const double W[3], double Q) {
    for (int comp = 0; comp < 3; ++comp) {
        int a = (comp + 1) % 3, b = (comp + 2) % 3;       /* cyclic transverse pair */
        for (int sb = 0; sb < 2; ++sb)
            for (int sa = 0; sa < 2; ++sa) {
                double sigma = (sa == sb) ? 1.0 : -1.0;
                double wgt = omega(W[a], sa) * omega(W[b], sb) + sigma * Dv[a] * Dv[b] / 12.0;   /* F2 / G7 */
                int n[3] = { c[0], c[1], c[2] };
                n[a] += sa; n[b] += sb;
                jadd(J[comp], pidx(g, n[0], n[1], n[2]), Q * Dv[comp] * wgt);
            }
    }
}

static void deposit_segment_2d(const orc_grid *g, double *const J[3], const int c[3], const double Dv[3], const double W[3],
                               double Q, double half_qw_v3) {
    for (int s = 0; s < 2; ++s) {
        jadd(J[0], pidx(g, c[0], c[1] + s, 0), Q * Dv[0] * omega(W[1], s));       /* J1[c + (0,s2)] */
        jadd(J[1], pidx(g, c[0] + s, c[1], 0), Q * Dv[1] * omega(W[0], s));       /* J2[c + (s1,0)] */
    }
    for (int s2 = 0; s2 < 2; ++s2)                                                  /* G8: out-of-plane, velocity form */
        for (int s1 = 0; s1 < 2; ++s1)
            jadd(J[2], pidx(g, c[0] + s1, c[1] + s2, 0), half_qw_v3 * omega(W[0], s1) * omega(W[1], s2));
}

int orc_deposit(const orc_grid *g, const orc_particles *po, const orc_particles *pn, double *const J[3], double q, double dt) {
    const int D = g->D, axisym = g->kind != ORC_CART;
    int64_t n = po->n;
    int err = 0;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        int alive = (po->tag ? po->tag[p] != 0 : 1) && (pn->tag ? pn->tag[p] != 0 : 1);
        if (!alive) continue;                              /* G9: absorbed particles deposit nothing */
        int c1[3] = {0, 0, 0}, c2[3] = {0, 0, 0}, di[3] = {0, 0, 0};
        double a[3] = {0, 0, 0}, b[3] = {0, 0, 0}, r[3] = {0, 0, 0};
        for (int k = 0; k < D; ++k) {
            int dd = pn->i[k][p] - po->i[k][p];
            if (g->bc[k] == ORC_PERIODIC) dd -= g->N[k] * (int)lround((double)dd / (double)g->N[k]);
            if (dd < -1 || dd > 1) {
#pragma omp atomic write
                err = -2;
                dd = 0;
            }
            di[k] = dd;
            a[k] = po->d[k][p];
            b[k] = dd + pn->d[k][p];                       /* new position in the OLD cell's frame */
            r[k] = dd == 0 ? 0.5 * (a[k] + b[k]) : (dd > 0 ? 1.0 : 0.0);   /* relay point, small numbers only */
            c1[k] = po->i[k][p];
            c2[k] = po->i[k][p] + dd;                      /* un-wrapped: may be -1 or N -> ghosts, folded later */
        }
        double D1[3] = {0, 0, 0}, W1[3] = {0, 0, 0}, D2[3] = {0, 0, 0}, W2[3] = {0, 0, 0};
        for (int k = 0; k < D; ++k) {
            D1[k] = r[k] - a[k];  W1[k] = 0.5 * (a[k] + r[k]);
            D2[k] = b[k] - r[k];  W2[k] = 0.5 * (r[k] + b[k]) - di[k];
        }
        double Q = q * po->w[p] / dt;
        if (D == 3) {
            deposit_segment_3d(g, J, c1, D1, W1, Q);
            deposit_segment_3d(g, J, c2, D2, W2, Q);
        } else {
            /* out-of-plane rate q w v3_code, half per segment (G8); v3_code = v^hat3 / sqrt(h33(x_mid)) */
            double ux = pn->u[0][p], uy = pn->u[1][p], uz = pn->u[2][p];
            double gam = sqrt(1.0 + ux * ux + uy * uy + uz * uz);
            double v3;
            if (!axisym) v3 = uz / gam;                    /* h33 = 1 */
            else {
                double dphi = pn->phi[p] - po->phi[p];
                dphi -= 2.0 * PI * floor((dphi + PI) / (2.0 * PI));      /* shorter arc, (-pi, pi] up to rounding */
                double phm = po->phi[p] + 0.5 * dphi;
                double xm[3] = { c1[0] + 0.5 * (a[0] + b[0]), c1[1] + 0.5 * (a[1] + b[1]), phm }, h[3];
                orc_metric_h(g, xm, h);
                double sh = sqrt(h[2]);
                v3 = sh < 1e-12 ? 0.0 : ((-ux * sin(phm) + uy * cos(phm)) / gam) / sh;
            }
            double hv = 0.5 * q * po->w[p] * v3;
            deposit_segment_2d(g, J, c1, D1, W1, Q, hv);
            deposit_segment_2d(g, J, c2, D2, W2, Q, hv);
        }
    }
    return err;
}

/* "currents synchronization" for a single periodic box: add what landed in the ghost layers of a
 * periodic dimension onto the opposite active layers, then refill those ghosts with the periodic image. */
static void fold_one(const orc_grid *g, double *A) {
    int64_t P[3] = { pext(g, 0), pext(g, 1), pext(g, 2) };
    int64_t stride[3] = { 1, P[0], P[0] * P[1] };
    for (int d = 0; d < g->D; ++d) {
        if (g->bc[d] != ORC_PERIODIC) continue;
        int N = g->N[d];
        int a = (d + 1) % 3, b = (d + 2) % 3;
        for (int64_t ib = 0; ib < P[b]; ++ib)
            for (int64_t ia = 0; ia < P[a]; ++ia) {
                double *line = A + ia * stride[a] + ib * stride[b];
                for (int gi = 0; gi < NG; ++gi) {
                    int lo = gi, hi = NG + N + gi;          /* padded indices of ghost layers */
                    line[(int64_t)(lo + N) * stride[d]] += line[(int64_t)lo * stride[d]];
                    line[(int64_t)(hi - N) * stride[d]] += line[(int64_t)hi * stride[d]];
                    line[(int64_t)lo * stride[d]] = 0.0;
                    line[(int64_t)hi * stride[d]] = 0.0;
                }
            }
    }
    for (int d = 0; d < g->D; ++d) {
        if (g->bc[d] != ORC_PERIODIC) continue;
        int N = g->N[d];
        int a = (d + 1) % 3, b = (d + 2) % 3;
        for (int64_t ib = 0; ib < P[b]; ++ib)
            for (int64_t ia = 0; ia < P[a]; ++ia) {
                double *line = A + ia * stride[a] + ib * stride[b];
                for (int gi = 0; gi < NG; ++gi) {
                    int lo = gi, hi = NG + N + gi;
                    line[(int64_t)lo * stride[d]] = line[(int64_t)(lo + N) * stride[d]];
                    line[(int64_t)hi * stride[d]] = line[(int64_t)(hi - N) * stride[d]];
                }
            }
    }
}
void orc_fold_current(const orc_grid *g, double *const J[3]) { for (int c = 0; c < 3; ++c) fold_one(g, J[c]); }
void orc_fold_scalar(const orc_grid *g, double *rho) { fold_one(g, rho); }

int orc_step(const orc_grid *g, const float *const F[6], orc_particles *p, double *const J[3], double q, double m, double dt) {
    const int D = g->D, axisym = g->kind != ORC_CART;
    int64_t n = p->n;
    orc_particles old = *p;
    for (int a = 0; a < D; ++a) {
        old.i[a] = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n ? n : 1));
        old.d[a] = (double *)malloc(sizeof(double) * (size_t)(n ? n : 1));
        memcpy(old.i[a], p->i[a], sizeof(int32_t) * (size_t)n);
        memcpy(old.d[a], p->d[a], sizeof(double) * (size_t)n);
    }
    old.phi = NULL; old.tag = NULL;
    if (axisym) { old.phi = (double *)malloc(sizeof(double) * (size_t)(n ? n : 1)); memcpy(old.phi, p->phi, sizeof(double) * (size_t)n); }
    if (p->tag) { old.tag = (int8_t *)malloc((size_t)(n ? n : 1)); memcpy(old.tag, p->tag, (size_t)n); }
    int rc = orc_gather_push(g, F, p, p, q / m, dt);
    if (rc == 0) rc = orc_deposit(g, &old, p, J, q, dt);
    for (int a = 0; a < D; ++a) { free(old.i[a]); free(old.d[a]); }
    free(old.phi); free(old.tag);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * N1  step 9 of the loop: digital filter passes on the conformal currents, Eqs. 9-11, then the
 * recovery of the current density J^i = conformal J^i / sqrt(h).
 * One pass = the (1/4, 1/2, 1/4) convolution along every dimension of the grid, f = (1/2)^(D + |di| + |dj| + |dk|), applied to
 * each component on its OWN staggered lattice ("we disregard the staggering ... when denoting the indices").
 * Values beyond the lattice of a component (readings):
 *   PERIODIC dimension: the periodic image;
 *   AXIS (theta) dimension: J^1(i+1/2, -1) = J^1(i+1/2, +1), J^2(i, -1/2) = -J^2(i, +1/2), J^3(i, 0) = 0, and the
 *     mirror image of the same at theta = pi (j = N_2);
 *   ABSORB dimension: zero (the paper is silent; what leaves through an absorbing side is discarded, G20).
 * Lattice of component c along dimension d: N_d points (0 .. N_d - 1) if d is periodic; otherwise the half-integer lattice of a
 * component staggered along d has N_d points (i + 1/2, i = 0 .. N_d - 1) and the integer lattice N_d + 1 (0 .. N_d).
 * J staggering = E staggering: J^1 (1,0,0), J^2 (0,1,0), J^3 (0,0,1); in 2D J^3 sits on the nodes.
 * divide != 0: afterwards J^c /= sqrt(h) at the component's own position, except on the polar axis itself (sqrt(h) = 0 there:
 * J^3 = 0 by Eq. 12 and E^1 is advanced with the conformal J^1 through Eq. 13, so those nodes keep the conformal value).
 * ------------------------------------------------------------------------------------------ */
static int lattice_extent(const orc_grid *g, int comp, int d) {
    if (d >= g->D) return 1;
    if (g->bc[d] == ORC_PERIODIC) return g->N[d];
    int stag = (comp == d);                                   /* J^c is staggered along its own direction only */
    return stag ? g->N[d] : g->N[d] + 1;
}
/* value of component comp at lattice index (i0,i1,i2), with the boundary rules above; *sign receives the parity factor */
static double filt_fetch(const orc_grid *g, const double *A, int comp, int i[3]) {
    double sign = 1.0;
    int q[3] = { i[0], i[1], i[2] };
    for (int d = 0; d < g->D; ++d) {
        int n = lattice_extent(g, comp, d);
        if (q[d] >= 0 && q[d] < n) continue;
        if (g->bc[d] == ORC_PERIODIC) { q[d] = ((q[d] % n) + n) % n; continue; }
        if (g->bc[d] == ORC_AXIS) {
            int stag = (comp == d);
            if (stag) { q[d] = q[d] < 0 ? -1 - q[d] : 2 * n - 1 - q[d]; sign = -sign; }      /* (j + 1/2) -> -(j + 1/2): odd */
            else { q[d] = q[d] < 0 ? -q[d] : 2 * (n - 1) - q[d]; }                            /* node j -> -j: even */
            continue;
        }
        return 0.0;                                            /* ABSORB */
    }
    return sign * A[pidx(g, q[0], q[1], g->D == 3 ? q[2] : 0)];
}
static int on_axis_node(const orc_grid *g, int comp, const int i[3]) {
    for (int d = 0; d < g->D; ++d)
        if (g->bc[d] == ORC_AXIS && comp != d && (i[d] == 0 || i[d] == g->N[d])) return 1;
    return 0;
}
void orc_filter_current(const orc_grid *g, double *const J[3], int npasses, int divide) {
    int64_t total = orc_padded_size(g);
    double *tmp = (double *)malloc(sizeof(double) * (size_t)total);
    for (int comp = 0; comp < 3; ++comp) {
        int n[3] = { lattice_extent(g, comp, 0), lattice_extent(g, comp, 1), lattice_extent(g, comp, 2) };
        for (int pass = 0; pass < npasses; ++pass) {
            memcpy(tmp, J[comp], sizeof(double) * (size_t)total);
            if (comp == 2 && g->D == 2)                        /* J^3(i, 0) = 0 is a condition on the INPUT of the convolution */
                for (int j = 0; j < n[1]; ++j)
                    for (int i = 0; i < n[0]; ++i) { int c[3] = { i, j, 0 }; if (on_axis_node(g, comp, c)) tmp[pidx(g, i, j, 0)] = 0.0; }
            for (int k = 0; k < n[2]; ++k)
                for (int j = 0; j < n[1]; ++j)
                    for (int i = 0; i < n[0]; ++i) {
                        int c[3] = { i, j, k };
                        double acc = 0.0;
                        if (comp == 2 && g->D == 2 && on_axis_node(g, comp, c)) { J[comp][pidx(g, i, j, 0)] = 0.0; continue; }   /* J^3(i, 0) = 0 */
                        for (int dk = (g->D == 3 ? -1 : 0); dk <= (g->D == 3 ? 1 : 0); ++dk)
                            for (int dj = -1; dj <= 1; ++dj)
                                for (int di = -1; di <= 1; ++di) {
                                    int q[3] = { i + di, j + dj, k + dk };
                                    double f = pow(0.5, g->D + abs(di) + abs(dj) + abs(dk));     /* Eqs. 9-11 */
                                    acc += f * filt_fetch(g, tmp, comp, q);
                                }
                        J[comp][pidx(g, i, j, g->D == 3 ? k : 0)] = acc;
                    }
        }
        if (divide)
            for (int k = 0; k < n[2]; ++k)
                for (int j = 0; j < n[1]; ++j)
                    for (int i = 0; i < n[0]; ++i) {
                        int c[3] = { i, j, k };
                        if (on_axis_node(g, comp, c)) continue;
                        double x[3] = { i + (comp == 0 ? 0.5 : 0.0), j + (comp == 1 ? 0.5 : 0.0), g->D == 3 ? k + (comp == 2 ? 0.5 : 0.0) : 0.0 }, h[3];
                        orc_metric_h(g, x, h);
                        J[comp][pidx(g, i, j, g->D == 3 ? k : 0)] /= sqrt(h[0] * h[1] * h[2]);
                    }
    }
    free(tmp);
}

/* ------------------------------------------------------------------------------------------
 * N2  field solver, sub-steps 2, 10, 11 of the loop: discretized Faraday (Eq. A1) and Ampere (Eq. A2) laws
 * on the Yee lattice in a diagonal metric (App. A), with the polar-axis treatment of Sec. 2.6.
 * Arrays: six (three) padded planar DOUBLE arrays, contravariant components E^i, B^i at the positions of ent.h / P:1044-1053:
 *   E^1 (i+1/2,j,k)  E^2 (i,j+1/2,k)  E^3 (i,j,k+1/2)   B^1 (i,j+1/2,k+1/2)  B^2 (i+1/2,j,k+1/2)  B^3 (i+1/2,j+1/2,k).
 * Code coordinates are counted in cells, so Delta x^i = 1 in the difference operators of P:1060-1064 and the cell sizes live in
 * h_ii.  Covariant components F_i = h_ii F^i, with h_ii and sqrt(h) evaluated at the component's own position.
 * With (c, a, b) a cyclic permutation of (1, 2, 3):
 *   A1:  B^c -= dt / sqrt(h) * { [E_b]_(+a) - [E_b] - ( [E_a]_(+b) - [E_a] ) }      at B^c's position (forward differences)
 *   A2:  E^c += dt / sqrt(h) * { [B_b] - [B_b]_(-a) - ( [B_a] - [B_a]_(-b) ) - jc * conformal J^c }   (backward differences)
 * (jc = 4 pi in Eq. A2; a parameter here because code units absorb it.)  A difference along a dimension the grid does not have
 * (x3 in 2D) is zero.  Lattice of a component along dimension d: N_d points if d is PERIODIC (index wraps); otherwise N_d points
 * for a component staggered along d and N_d + 1 (nodes 0 .. N_d) for one that is not.
 * Readings: the left side of A2 is garbled in the source ("Delta_{n+1}^{n+1}"): it is (E^(n+1) - E^(n)) / dt.
 * Faraday never reaches beyond the E lattices.  Ampere does, on a non-periodic side: there the E components tangential to that
 * face (the ones whose stencil needs a B value outside the lattice) are NOT advanced -- they are the caller's boundary condition
 * (the paper's conductor / absorbing layers are problem-generator code).  Polar axis (AXIS in x2, j = 0 and j = N_2):
 *   Eq. 12:  E^3(i, j) = 0 and B^2(i+1/2, j) = 0 are imposed and their update skipped;
 *   Eq. 13:  E^1(i+1/2, 0) += dt * { B_3(i+1/2, 1/2) - (jc/2) conformal J^1(i+1/2, 0) } / A(i+1/2), and the mirror image at
 *            j = N_2: E^1(i+1/2, N_2) += dt * { -B_3(i+1/2, N_2 - 1/2) - (jc/2) J^1(i+1/2, N_2) } / A(i+1/2)  (integral of A2 over
 *            the half cell next to the axis, where B_3 = h_33 B^3 vanishes on the axis);
 *   A(x1) = integral_0^(1/2) sqrt(h) dx2, in the closed forms the paper prints:
 *            SPH r^2 dr (1 - cos(dtheta/2));  QSPH (r0 + e^R)^2 e^R dR (1 - cos(theta(dT/2))).  (The line that defines A carries a
 *            factor 2 pi that its own closed forms do not have; the closed forms are the ones consistent with the B_3 term.)
 * ------------------------------------------------------------------------------------------ */
static int fld_stag(int comp6, int d) { int c = comp6 % 3; return comp6 < 3 ? (d == c) : (d != c); }
static int fld_extent(const orc_grid *g, int comp6, int d) {
    if (d >= g->D) return 1;
    if (g->bc[d] == ORC_PERIODIC) return g->N[d];
    return fld_stag(comp6, d) ? g->N[d] : g->N[d] + 1;
}
/* covariant component h_cc F^c of field component comp6 at lattice index q (periodic wrap); *ok = 0 if q lies outside the lattice */
static double fld_cov(const orc_grid *g, const double *A, int comp6, const int qin[3], int *ok) {
    int q[3] = { qin[0], qin[1], qin[2] };
    for (int d = 0; d < g->D; ++d) {
        int n = fld_extent(g, comp6, d);
        if (q[d] >= 0 && q[d] < n) continue;
        if (g->bc[d] == ORC_PERIODIC) { q[d] = ((q[d] % n) + n) % n; continue; }
        *ok = 0;
        return 0.0;
    }
    double x[3], h[3];
    for (int d = 0; d < 3; ++d) x[d] = d < g->D ? q[d] + (fld_stag(comp6, d) ? 0.5 : 0.0) : 0.0;
    orc_metric_h(g, x, h);
    return h[comp6 % 3] * A[pidx(g, q[0], q[1], g->D == 3 ? q[2] : 0)];
}
static double sqrt_h_at(const orc_grid *g, int comp6, const int q[3]) {
    double x[3], h[3];
    for (int d = 0; d < 3; ++d) x[d] = d < g->D ? q[d] + (fld_stag(comp6, d) ? 0.5 : 0.0) : 0.0;
    orc_metric_h(g, x, h);
    return sqrt(h[0] * h[1] * h[2]);
}
static int axis_dim(const orc_grid *g) { for (int d = 0; d < g->D; ++d) if (g->bc[d] == ORC_AXIS) return d; return -1; }

/* A(x1) of Eq. 13, closed forms of P:372-382 */
double orc_axis_area(const orc_grid *g, double x1) {
    if (g->kind == ORC_SPH) {
        double dr = cell_size(g, 0), dth = PI / (double)g->N[1], r = g->xmin[0] + x1 * dr;
        return r * r * dr * (1.0 - cos(0.5 * dth));
    }
    double dR = qs_dR(g), dT = qs_dT(g), eR = exp(qs_Rmin(g) + x1 * dR), vt = g->vartheta;
    double dtt = 0.5 * dT + vt * dT * (1.0 - dT / PI) * (1.0 - dT / (2.0 * PI));              /* = theta(dT / 2) */
    return (g->r0 + eR) * (g->r0 + eR) * eR * dR * (1.0 - cos(dtt));
}

void orc_faraday(const orc_grid *g, const double *const E[3], double *const B[3], double dt) {
    const int ax = axis_dim(g);
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3, cB = 3 + c;
        const int n[3] = { fld_extent(g, cB, 0), fld_extent(g, cB, 1), fld_extent(g, cB, 2) };
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    const int q[3] = { i, j, k };
                    const int64_t at = pidx(g, i, j, g->D == 3 ? k : 0);
                    if (ax >= 0 && c == 1 && (q[ax] == 0 || q[ax] == g->N[ax])) { B[c][at] = 0.0; continue; }     /* Eq. 12 */
                    int ok = 1;
                    double curl = 0.0;
                    if (a < g->D) { int qp[3] = { i, j, k }; qp[a] += 1; curl += fld_cov(g, E[b], b, qp, &ok) - fld_cov(g, E[b], b, q, &ok); }
                    if (b < g->D) { int qp[3] = { i, j, k }; qp[b] += 1; curl -= fld_cov(g, E[a], a, qp, &ok) - fld_cov(g, E[a], a, q, &ok); }
                    if (!ok) continue;                                    /* cannot happen: A1 stays inside the E lattices */
                    B[c][at] -= dt * curl / sqrt_h_at(g, cB, q);          /* Eq. A1 */
                }
    }
}

void orc_ampere(const orc_grid *g, double *const E[3], const double *const B[3], const double *const J[3], double dt, double jc) {
    const int ax = axis_dim(g);
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const int n[3] = { fld_extent(g, c, 0), fld_extent(g, c, 1), fld_extent(g, c, 2) };
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    const int q[3] = { i, j, k };
                    const int64_t at = pidx(g, i, j, g->D == 3 ? k : 0);
                    const double Jc = J ? J[c][at] : 0.0;
                    if (ax >= 0 && c != ax && (q[ax] == 0 || q[ax] == g->N[ax])) {          /* a point on the polar axis */
                        if (c == 2) { E[c][at] = 0.0; continue; }                           /* Eq. 12 */
                        /* c == 0: Eq. 13 */
                        int ok = 1, qb[3] = { i, j, k };
                        double sgn = 1.0;
                        if (q[ax] != 0) { qb[ax] = g->N[ax] - 1; sgn = -1.0; }              /* B^3 at (i+1/2, N_2 - 1/2) */
                        double B3 = fld_cov(g, B[2], 5, qb, &ok);
                        E[c][at] += dt * (sgn * B3 - 0.5 * jc * Jc) / orc_axis_area(g, i + 0.5);
                        continue;
                    }
                    int ok = 1;
                    double curl = 0.0;
                    if (a < g->D) { int qm[3] = { i, j, k }; qm[a] -= 1; curl += fld_cov(g, B[b], 3 + b, q, &ok) - fld_cov(g, B[b], 3 + b, qm, &ok); }
                    if (b < g->D) { int qm[3] = { i, j, k }; qm[b] -= 1; curl -= fld_cov(g, B[a], 3 + a, q, &ok) - fld_cov(g, B[a], 3 + a, qm, &ok); }
                    if (!ok) continue;                                    /* tangential E on a non-periodic face: the caller's boundary condition */
                    E[c][at] += dt * (curl - jc * Jc) / sqrt_h_at(g, c, q);                 /* Eq. A2 */
                }
    }
}

/* Ghost layers of the six field arrays, as the gather expects them (harness convention, reading G10): PERIODIC dimension: the
 * periodic image; AXIS: mirror image about the axis, E^1 / B^1 even, the theta- and phi-components odd; ABSORB: left alone. */
void orc_fill_field_ghosts(const orc_grid *g, double *const F[6]) {
    for (int c6 = 0; c6 < 6; ++c6)
        for (int d = 0; d < g->D; ++d) {
            if (g->bc[d] == ORC_ABSORB) continue;
            const int n = fld_extent(g, c6, d), a = (d + 1) % 3, b = (d + 2) % 3;
            const int lo_a = a < g->D ? -NG : 0, hi_a = a < g->D ? g->N[a] + NG : 1, lo_b = b < g->D ? -NG : 0, hi_b = b < g->D ? g->N[b] + NG : 1;
            for (int ib = lo_b; ib < hi_b; ++ib)
                for (int ia = lo_a; ia < hi_a; ++ia)
                    for (int gi = -NG; gi < g->N[d] + NG; ++gi) {
                        if (gi >= 0 && gi < n) continue;
                        int src; double sign = 1.0;
                        if (g->bc[d] == ORC_PERIODIC) src = ((gi % n) + n) % n;
                        else {                                          /* AXIS */
                            if (fld_stag(c6, d)) src = gi < 0 ? -1 - gi : 2 * n - 1 - gi;
                            else src = gi < 0 ? -gi : 2 * (n - 1) - gi;
                            if (c6 % 3 != 0) sign = -1.0;
                        }
                        int q[3], s[3];
                        q[d] = gi; q[a] = ia; q[b] = ib; s[d] = src; s[a] = ia; s[b] = ib;
                        F[c6][pidx(g, q[0], q[1], g->D == 3 ? q[2] : 0)] = sign * F[c6][pidx(g, s[0], s[1], g->D == 3 ? s[2] : 0)];
                    }
        }
}

/* ------------------------------------------------------------------------------------------
 * Eq. 6 checker.  Conformal nodal charge (no 1/sqrt(h)):  rho[n] = sum_p q w prod_d omega(delta_d, s_d)
 * ------------------------------------------------------------------------------------------ */
void orc_charge_density(const orc_grid *g, const orc_particles *p, const int8_t *mask, double q, double *rho) {
    const int D = g->D;
    for (int64_t k = 0; k < p->n; ++k) {
        if (mask && !mask[k]) continue;
        int nk = D == 3 ? 2 : 1;
        for (int s3 = 0; s3 < nk; ++s3)
            for (int s2 = 0; s2 < 2; ++s2)
                for (int s1 = 0; s1 < 2; ++s1) {
                    double wgt = omega(p->d[0][k], s1) * omega(p->d[1][k], s2);
                    if (D == 3) wgt *= omega(p->d[2][k], s3);
                    rho[pidx(g, p->i[0][k] + s1, p->i[1][k] + s2, D == 3 ? p->i[2][k] + s3 : 0)] += q * p->w[k] * wgt;
                }
    }
}

/* R[n] = sum_d (J^d[n] - J^d[n - e_d]) + (rho_new[n] - rho_old[n]) / dt over the valid nodes:
 * periodic dimension 0..N-1 (ghosts hold the periodic image after the fold), otherwise 0..N. */
double orc_continuity_residual(const orc_grid *g, double *const J[3], const double *rho_old, const double *rho_new,
                               double dt, double *R_out) {
    const int D = g->D;
    int hi[3];
    for (int d = 0; d < 3; ++d) hi[d] = d < D ? (g->bc[d] == ORC_PERIODIC ? g->N[d] - 1 : g->N[d]) : 0;
    double worst = 0.0;
    for (int k = 0; k <= hi[2]; ++k)
        for (int j = 0; j <= hi[1]; ++j)
            for (int i = 0; i <= hi[0]; ++i) {
                int64_t n = pidx(g, i, j, k);
                double R = (rho_new[n] - rho_old[n]) / dt;
                R += J[0][n] - J[0][pidx(g, i - 1, j, k)];
                R += J[1][n] - J[1][pidx(g, i, j - 1, k)];
                if (D == 3) R += J[2][n] - J[2][pidx(g, i, j, k - 1)];
                if (R_out) R_out[n] = R;
                if (fabs(R) > worst) worst = fabs(R);
            }
    return worst;
}

/* N4  tag sort: "sorts all the particle quantities based on their tag, after which npart always indicates the number
 * of alive particles, while the dead ones are shuffled to the end".  Stable: alive particles keep their order, so do the dead.
 * Returns the number of alive particles; out must not alias in. */
int64_t orc_compact(int D, int axisym, const orc_particles *in, orc_particles *out) {
    int64_t n = in->n, k = 0;
    for (int pass = 0; pass < 2; ++pass)                    /* pass 0: alive, pass 1: dead */
        for (int64_t p = 0; p < n; ++p) {
            int alive = in->tag ? in->tag[p] != 0 : 1;
            if (alive == pass) continue;
            for (int a = 0; a < D; ++a) { out->i[a][k] = in->i[a][p]; out->d[a][k] = in->d[a][p]; }
            for (int a = 0; a < 3; ++a) out->u[a][k] = in->u[a][p];
            out->w[k] = in->w[p];
            if (axisym) out->phi[k] = in->phi[p];
            if (out->tag) out->tag[k] = (int8_t)alive;
            ++k;
        }
    int64_t na = 0;
    for (int64_t p = 0; p < n; ++p) na += in->tag ? in->tag[p] != 0 : 1;
    return na;
}

/* S10 checker: keys non-decreasing; offsets[c] = number of keys < c (exclusive scan of the histogram) */
int orc_sort_check(const int64_t n, const int32_t *keys, int64_t ncell, const int32_t *offsets) {
    for (int64_t p = 1; p < n; ++p) if (keys[p] < keys[p - 1]) return 1;
    for (int64_t p = 0; p < n; ++p) if (keys[p] < 0 || keys[p] >= ncell) return 2;
    if (offsets) {
        int64_t p = 0;
        for (int64_t c = 0; c <= ncell; ++c) {
            while (p < n && keys[p] < c) ++p;
            if (offsets[c] != p) return 3;
        }
    }
    return 0;
}
