/*
 * orc.h -- fp64 CPU ORACLE for the particle hot path of arXiv 2511.17710
 *          ("Entity", curvilinear special-relativistic PIC module).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * source, header, table or helper with the CUDA path under paper_2511_17710_b200/.
 *
 * It follows the paper's algorithm step by step (PAPER.md = P:line):
 *   step 3  gather        P:131-133          -> orc_gather
 *   step 4  basis change  P:76-81, P:135-139 -> orc_to_cartesian_basis
 *   step 5  Boris push    P:89-95, P:141-143 -> orc_boris
 *   step 6  move          P:147-149          -> orc_gather_push (absolute coordinates, textbook way)
 *   step 7  back-map      P:151-153, App. B -> orc_cart_to_code
 *   step 8  deposit       P:105-109, P:155-157, P:575 -> orc_deposit (+ orc_fold_current)
 *   steps 2, 10, 11  field solver  P:127-129, App. A, Sec. 2.6 -> orc_faraday, orc_ampere
 * plus the discrete continuity checker of Eq. 6 and a sort checker.
 * Readings of silent / garbled passages are those of SURVEY.md section 8(c) (G1..G19), listed in DESIGN.md.
 *
 * Parity pins: tests/test_oracle_pins_*.py; tests/oracle_mutants.py lists the one-line misreadings those pins kill
 * (gamma^- in the Boris rotation, gamma^(n+1/2) in the move, time level / azimuth midpoint / evaluation point of the
 * out-of-plane current, the theta = pi clamp, the D_a D_b / 12 term, ...).  One choice stays a READING the paper does
 * not fix: the FORM of the 2D out-of-plane current J^3 (velocity form, half per segment, bilinear weights at the
 * segment midpoints, reading G8) -- "parity unpinned" by the paper beyond its nodal sum, time level and evaluation
 * point, which are pinned; see DESIGN.md.  A second one: the hybrid pusher (orc_gca_project, reading G26) -- the paper gives two
 * sentences and cites a scheme that is not in it; the switch and the zeroing of u_perp are pinned as stated, the rest
 * (no drift terms, the move unchanged) is "parity unpinned".
 *
 * All arithmetic is double.  Field arrays are the fp32 arrays handed to the GPU (up-cast on load).
 */
#ifndef ORC_H
#define ORC_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_NGHOST 2

enum { ORC_CART = 0, ORC_SPH = 1, ORC_QSPH = 2 };
enum { ORC_PERIODIC = 0, ORC_ABSORB = 1, ORC_AXIS = 2 };   /* boundary kind per dimension */

typedef struct {
    int32_t D;              /* 2 or 3 spatial dimensions of the grid                          */
    int32_t N[3];           /* active cells per dimension (N[2] = 1 when D == 2)              */
    int32_t bc[3];          /* ORC_PERIODIC / ORC_ABSORB / ORC_AXIS per dimension             */
    int32_t kind;           /* ORC_CART / ORC_SPH / ORC_QSPH                                  */
    double  xmin[3], xmax[3]; /* physical extent, Eq. 7 (SPH/QSPH: r range in [0], theta = [0,pi]) */
    double  r0, vartheta;   /* QSPH stretch parameters                             */
} orc_grid;

/* particle block: unpacked cell indices, everything else double */
typedef struct {
    int64_t  n;
    int32_t *i[3];          /* cell index per dimension (i[2] may be NULL in 2D)              */
    double  *d[3];          /* in-cell offset in [0,1)                                 */
    double  *phi;           /* azimuth (axisymmetric grids only, else NULL)            */
    double  *u[3];          /* four-velocity, global Cartesian basis                   */
    double  *w;             /* weight                                                         */
    int8_t  *tag;           /* 1 alive, 0 dead; may be NULL = all alive        */
} orc_particles;

/* ---- O1 metric ---- */
void   orc_metric_h(const orc_grid *g, const double x[3], double h[3]);   /* h11,h22,h33 at code coords */
double orc_theta_of_T(double vartheta, double T);
void   orc_metric_h_many(const orc_grid *g, int64_t n, const double *x1, const double *x2, double *h /* [n][3] */);
double orc_dtheta_dT(double vartheta, double T);
double orc_T_of_theta(double vartheta, double theta);                      /* App. B, corrected (F1) */
double orc_T_of_theta_printed_B3(double vartheta, double theta);           /* App. B exactly as printed + F1 fix flag; for the pin */
double orc_dx_min(const orc_grid *g);                                      /* Eq. 8 */

/* ---- O5/O6 coordinate maps ---- */
void orc_code_to_cart(const orc_grid *g, const double x[3] /* x1,x2,(x3 or phi) */, double X[3]);
void orc_cart_to_code(const orc_grid *g, const double X[3], double x[3]);

/* ---- O2 gather (reading G1) ---- */
void orc_gather(const orc_grid *g, const float *const F[6], const int32_t i[3], const double d[3], double out[6]);

/* ---- O3 basis change ---- */
void orc_to_cartesian_basis(const orc_grid *g, const double x[3], const double A_code[3], double A_cart[3]);

/* ---- O4 Boris ---- */
void orc_boris(double u[3], const double E[3], const double B[3], double q_over_m, double dt);

/* ---- N3: Vay (2008) pusher, same interface; orc_set_pusher selects the one orc_gather_push / orc_step use (0 Boris, 1 Vay) ---- */
void orc_vay(double u[3], const double E[3], const double B[3], double q_over_m, double dt);
int  orc_set_pusher(int kind);                                            /* 0 Boris, 1 Vay, 2 Boris,GCA, 3 Vay,GCA; returns the previous kind */
/* hybrid pusher of P:976-980 (reading G26): thresholds, and the guiding-centre step u <- (u.b) b when |E| < eovb |B| and
 * |u_before| m / (|q||B|) < rho_crit (returns 1 if applied) */
void orc_set_gca(double rho_crit, double eovb);
int  orc_gca_project(double u[3], const double u_before[3], const double E[3], const double B[3], double q_over_m);

/* ---- steps 3-7 for a particle block; out may alias in (arrays are overwritten element-wise) ---- */
int orc_gather_push(const orc_grid *g, const float *const F[6], const orc_particles *in, orc_particles *out,
                    double q_over_m, double dt);

/* ---- step 8: deposit conformal currents; ACCUMULATES into J (padded planar, double).
 *      pnew carries u at n+1/2 (needed for the 2D out-of-plane component). ---- */
int orc_deposit(const orc_grid *g, const orc_particles *pold, const orc_particles *pnew, double *const J[3],
                double q, double dt);
/* periodic ghost fold ("currents synchronization") + ghost refill in periodic dims */
void orc_fold_current(const orc_grid *g, double *const J[3]);
void orc_fold_scalar(const orc_grid *g, double *rho);

/* ---- step 9: npasses digital filter passes (Eqs. 9-11) with the periodic / axis / absorbing rules,
 *      then (divide != 0) J^i = conformal J^i / sqrt(h) at each component's own position.  In place; J must already be
 *      folded (orc_fold_current).  Ghost layers of the arrays are not touched. ---- */
void orc_filter_current(const orc_grid *g, double *const J[3], int npasses, int divide);

/* ---- N2 field solver (sub-steps 2, 10, 11; Eqs. A1, A2, 12, 13) on padded planar DOUBLE
 *      arrays of contravariant components.  orc_faraday: B -= dt curl(h E) / sqrt(h) (the loop calls it twice with dt/2);
 *      orc_ampere: E += dt (curl(h B) - jc conformal J) / sqrt(h), jc = 4 pi in Eq. A2, J may be NULL; axis rules inside.
 *      orc_fill_field_ghosts: periodic / axis-mirror ghost layers as the gather wants them (reading G10). ---- */
void   orc_faraday(const orc_grid *g, const double *const E[3], double *const B[3], double dt);
void   orc_ampere(const orc_grid *g, double *const E[3], const double *const B[3], const double *const J[3], double dt, double jc);
double orc_axis_area(const orc_grid *g, double x1);                        /* A(x1) of Eq. 13 */
void   orc_fill_field_ghosts(const orc_grid *g, double *const F[6]);

/* fused: gather_push then deposit (no fold) */
int orc_step(const orc_grid *g, const float *const F[6], orc_particles *p, double *const J[3],
             double q, double m, double dt);

/* ---- Eq. 6 checker: conformal nodal charge and the continuity residual ---- */
void   orc_charge_density(const orc_grid *g, const orc_particles *p, const int8_t *alive_mask, double q, double *rho /* padded, accumulates */);
/* residual R[n] over valid nodes, J folded, rho arrays folded; returns max|R|; writes the normaliser */
double orc_continuity_residual(const orc_grid *g, double *const J[3], const double *rho_old, const double *rho_new,
                               double dt, double *R_out /* padded or NULL */);

/* ---- N4 tag sort: alive particles first (stable), dead ones after; returns the number of alive particles ---- */
int64_t orc_compact(int D, int axisym, const orc_particles *in, orc_particles *out);

/* ---- sort checker: keys non-decreasing, offsets = exclusive scan of histogram; returns 0 if ok ---- */
int orc_sort_check(const int64_t n, const int32_t *keys_sorted, int64_t ncell, const int32_t *offsets /* ncell+1 or NULL */);

int64_t orc_padded_size(const orc_grid *g);
int     orc_num_threads(void);
int     orc_set_num_threads(int n);                                         /* returns the previous count */

#ifdef __cplusplus
}
#endif
#endif
