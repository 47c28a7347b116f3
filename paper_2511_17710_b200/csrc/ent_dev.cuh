// ent_dev.cuh -- device-side building blocks of the particle hot path (arXiv 2511.17710; P:nnn = PAPER.md line).
// Everything here is fp32 except the curvilinear coordinate maps, which are evaluated in fp64 (DESIGN.md
// "precision of the curvilinear round trip": the fp32 code->xyz->code round trip loses the displacement).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/ent.h"

namespace ent {

constexpr int NG = ENT_NGHOST;
constexpr double PI_D = 3.14159265358979323846264338327950288;
constexpr float TWO_PI_F = 6.28318548202514648f;   // float nearest to 2*pi (slightly above it)
constexpr float TWO_PI_LO = 1.74845553e-7f;         // TWO_PI_F - 2*pi
// sin and cos of an azimuth in [-pi, 3 pi] (phi or a midpoint of two phis): the argument is shifted by pi into the range where
// MUFU.SIN / MUFU.COS (__sincosf) are good to 2^-21.4 absolute, sin(x) = -sin(x - pi).  5e-7 on a rotation of the field basis and of
// the displacement is 2.5e-7 cells and 5e-7 of |E|, |B| at most: inside the 1e-5 bars with the margin the parity tests print.
__device__ __forceinline__ void sincos_azimuth(float phi, float &s, float &c) {
    float x = phi - 3.14159274101257324f;
    if (x > 3.14159274101257324f) x -= TWO_PI_F;
    __sincosf(x, &s, &c);
    s = -s; c = -c;
}

// Grid + metric constants, passed to kernels by value (the paper passes its metric object by value too).
struct GridDev {
    int D, kind;
    int N[3];          // active cells (N[2] = 1 in 2D)
    int P[3];          // padded extents N + 2*NG (P[2] = 1 in 2D)
    int bc[3];
    int T[3];          // tile extents in cells (T[2] = 1 in 2D)
    int nt[3];         // tiles per dimension
    int tcells;        // T0*T1*T2
    float dx[3];       // CART: sqrt(h_dd) = cell size (1 for dimensions >= D)
    float inv_dx[3];
    // SPH:  r = rmin + x1*dr, theta = x2*dth
    // QSPH: r = r0 + exp(Rmin + x1*dR), theta = theta(T), T = x2*dT
    double rmin, dr, dth;
    double Rmin, dR, dT, r0, vt;
    // fp32 copies for the displacement form of the curvilinear move (ent_particle.cuh) and its switch
    float rminf, drf, dthf, Rminf, dRf, dTf, r0f, vtf;
    int pusher;        // ENT_OPT_PUSHER: 0 Boris, 1 Vay, 2 Boris,GCA, 3 Vay,GCA
    float gca_c;       // hybrid pusher: 2 rho_crit / dt of the current call (x eps = rho_crit q/m), and (max |E|/|B|)^2
    float gca_eovb2;
    int curv_f64;      // 1: coordinate maps of the axisymmetric grids in fp64 through the global Cartesian frame (round-1 form)
};

__host__ __device__ inline long long padded_size(const GridDev &g) { return (long long)g.P[0] * g.P[1] * g.P[2]; }

template <int D>
__device__ __forceinline__ void unpack_cell(const GridDev &g, int cell, int i[3]) {
    if (D == 2) {
        i[1] = cell / g.N[0]; i[0] = cell - i[1] * g.N[0]; i[2] = 0;
    } else {
        int n01 = g.N[0] * g.N[1];
        i[2] = cell / n01; int r = cell - i[2] * n01;
        i[1] = r / g.N[0]; i[0] = r - i[1] * g.N[0];
    }
}
template <int D>
__device__ __forceinline__ int pack_cell(const GridDev &g, const int i[3]) {
    return D == 2 ? i[0] + g.N[0] * i[1] : i[0] + g.N[0] * (i[1] + g.N[1] * i[2]);
}
// padded linear index of active cell (i,j,k)
template <int D>
__device__ __forceinline__ long long pidx(const GridDev &g, int i, int j, int k) {
    return D == 2 ? (long long)(i + NG) + (long long)g.P[0] * (j + NG)
                  : (long long)(i + NG) + (long long)g.P[0] * ((long long)(j + NG) + (long long)g.P[1] * (k + NG));
}
// sort key of a cell (ent.h, ent_sort): tile-major
template <int D>
__device__ __forceinline__ int sort_key(const GridDev &g, const int i[3]) {
    int t0 = i[0] / g.T[0], t1 = i[1] / g.T[1];
    int l0 = i[0] - t0 * g.T[0], l1 = i[1] - t1 * g.T[1];
    if (D == 2) return (t0 + g.nt[0] * t1) * g.tcells + (l0 + g.T[0] * l1);
    int t2 = i[2] / g.T[2], l2 = i[2] - t2 * g.T[2];
    return (t0 + g.nt[0] * (t1 + g.nt[1] * t2)) * g.tcells + (l0 + g.T[0] * (l1 + g.T[1] * l2));
}

// ---------------------------------------------------------------------------------------------------------
// S1 gather (first-order shape, direct multilinear interpolation on each component's own staggered
// lattice; Yee staggering P:181).  F[c] = padded planar arrays.  Loader abstracts where the
// values come from (global memory here, a shared-memory tile in the tiled kernel).
// ---------------------------------------------------------------------------------------------------------
struct GlobalFieldLoader {
    const float *const *F;   // 6 pointers (kernel-parameter copy)
    __device__ __forceinline__ float operator()(int c, long long idx) const { return __ldg(F[c] + idx); }
};

template <int D, class Loader>
__device__ __forceinline__ void gather(const GridDev &g, const Loader &ld, const int i[3], const float d[3], float EB[6]) {
    // per dimension: node-centred (b0,f0) and half-shifted (bs,fs) base index and fraction
    int bs[3]; float fs[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (a < D) {
            bool lo = d[a] < 0.5f;
            bs[a] = lo ? i[a] - 1 : i[a];
            fs[a] = lo ? d[a] + 0.5f : d[a] - 0.5f;
        } else { bs[a] = 0; fs[a] = 0.f; }
    }
    const long long s1 = g.P[0], s2 = (long long)g.P[0] * g.P[1];
    // stagger pattern per component (1 = half-cell shift): E1 100, E2 010, E3 001, B1 011, B2 101, B3 110
    const int ST[6][3] = { {1,0,0}, {0,1,0}, {0,0,1}, {0,1,1}, {1,0,1}, {1,1,0} };
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        int b0 = ST[c][0] ? bs[0] : i[0];
        int b1 = ST[c][1] ? bs[1] : i[1];
        int b2 = (D == 3) ? (ST[c][2] ? bs[2] : i[2]) : 0;
        float f0 = ST[c][0] ? fs[0] : d[0];
        float f1 = ST[c][1] ? fs[1] : d[1];
        long long base = pidx<D>(g, b0, b1, b2);
        float v00 = ld(c, base), v10 = ld(c, base + 1), v01 = ld(c, base + s1), v11 = ld(c, base + s1 + 1);
        float lo = (v00 + f0 * (v10 - v00)) + f1 * ((v01 + f0 * (v11 - v01)) - (v00 + f0 * (v10 - v00)));
        if (D == 3) {
            float f2 = ST[c][2] ? fs[2] : d[2];
            float w00 = ld(c, base + s2), w10 = ld(c, base + s2 + 1), w01 = ld(c, base + s2 + s1), w11 = ld(c, base + s2 + s1 + 1);
            float hi = (w00 + f0 * (w10 - w00)) + f1 * ((w01 + f0 * (w11 - w01)) - (w00 + f0 * (w10 - w00)));
            lo = lo + f2 * (hi - lo);
        }
        EB[c] = lo;
    }
}

// ---------------------------------------------------------------------------------------------------------
// O1 metric pieces for the axisymmetric grids, fp64
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double theta_of_T(double vt, double T) {
    return T + 2.0 * vt * T * (1.0 - 2.0 * T / PI_D) * (1.0 - T / PI_D);
}
__device__ __forceinline__ double dtheta_dT(double vt, double T) {
    double s = T / PI_D;
    return 1.0 + 2.0 * vt + 12.0 * vt * s * (s - 1.0);
}
// inverse of theta(T) (App. B): theta(T) is a monotone cubic for 0 <= vartheta < 1, so Newton from
// T = theta converges quadratically; no cube root on the device (differs from Eq. B3).
// T0 = starting point: the particle's previous T plus the linearised change is within a fraction of a cell of the root,
// so two or three steps reach 1e-15.
__device__ __forceinline__ double T_of_theta(double vt, double th, double T0) {
    if (vt == 0.0) return th;
    double T = T0;
#pragma unroll 1
    for (int it = 0; it < 8; ++it) {
        double f = theta_of_T(vt, T) - th;
        T -= f / dtheta_dT(vt, T);
        if (fabs(f) < 1e-15) break;
    }
    return T;
}

// ---------------------------------------------------------------------------------------------------------
// fp32 description of a code position on the axisymmetric grids, for the DISPLACEMENT form of the move.
// The transcendental part of the metric lives at the grid NODES: exp(R_i) (or r_i) per x1 node, sin/cos(theta_j), d theta/dT and
// half the second derivative of theta(T) per x2 node, evaluated in fp64 and rounded once ("metric factors", BASELINE.json
// north_star (b)).  The tiled kernel stages them per tile in shared memory (TileGeo, ent_tiled_axisym.cuh); the untiled kernels
// evaluate them per particle (GlobalGeo) -- the same function, hence the same values.  At the particle only short polynomials in
// the in-cell offset remain: exp(x), x < dR, and sin/cos of the angle to the NEARER node, so sin(theta) keeps its relative
// accuracy next to either pole and (i + d) is never formed (the offset would lose its low bits).
// ---------------------------------------------------------------------------------------------------------
struct NodeY { float st, ct, th1, c2; };   // sin, cos of theta_j; d theta / dT and (d2 theta / dT2) / 2 at T_j (SPH: 1, 0)
template <int KIND>
__device__ __forceinline__ float node_x(const GridDev &g, int i) {            // P:243 / P:261: r_i (SPH) or exp(R_i) (QSPH)
    return KIND == ENT_SPH ? (float)(g.rmin + (double)i * g.dr) : (float)exp(g.Rmin + (double)i * g.dR);
}
template <int KIND>
__device__ __forceinline__ NodeY node_y(const GridDev &g, int j) {            // P:243 / P:265-267
    NodeY y;
    double th, s_, c_;
    if (KIND == ENT_SPH) { th = (double)j * g.dth; y.th1 = 1.f; y.c2 = 0.f; }
    else {
        const double T = (double)j * g.dT, s = T / PI_D;
        th = T + 2.0 * g.vt * T * (1.0 - 2.0 * s) * (1.0 - s);
        y.th1 = (float)(1.0 + 2.0 * g.vt + 12.0 * g.vt * s * (s - 1.0));
        y.c2 = (float)(6.0 * g.vt * (2.0 * s - 1.0) / PI_D);
    }
    sincos(th, &s_, &c_);
    y.st = (float)s_; y.ct = (float)c_;
    return y;
}
template <int KIND>
struct GlobalGeo {                       // node factors evaluated on the spot (untiled kernels, stray path)
    const GridDev &g;
    __device__ __forceinline__ float x(int i) const { return node_x<KIND>(g, i); }
    __device__ __forceinline__ NodeY y(int j) const { return node_y<KIND>(g, j); }
};

struct SphF {
    float r, rr0;           // r and r - r0
    float st, ct;           // sin(theta), cos(theta)
    float sh1, sh2, sh3;    // sqrt(h11), sqrt(h22), sqrt(h33)
    float th1, c2;          // QSPH: d theta / dT and (d2 theta / dT2) / 2 at the particle
};
// d1, d2 may lie a little outside [0, 1) (midpoint of a move)
template <int KIND, class GEO>
__device__ __forceinline__ SphF sphf_of_code(const GridDev &g, const GEO &geo, int i1, float d1, int i2, float d2) {
    SphF s;
    const int rnd = (int)floorf(d2 + 0.5f);                    // nearer x2 node
    const NodeY y = geo.y(i2 + rnd);
    float eps;                                                 // theta - theta_node
    if (KIND == ENT_SPH) {
        s.r = fmaf(d1, g.drf, geo.x(i1));
        s.rr0 = s.r;
        eps = (d2 - (float)rnd) * g.dthf;
        s.th1 = 1.f; s.c2 = 0.f;
        s.sh1 = g.drf; s.sh2 = s.r * g.dthf;
    } else {
        const float x = d1 * g.dRf;                            // exp(R_i + x) = exp(R_i) (1 + x + x^2/2 + x^3/6 + x^4/24), x < 2 dR
        const float eR = geo.x(i1) * fmaf(x, fmaf(x, fmaf(x, fmaf(x, 1.0f / 24.0f, 1.0f / 6.0f), 0.5f), 1.0f), 1.0f);
        s.r = g.r0f + eR; s.rr0 = eR;
        const float eT = (d2 - (float)rnd) * g.dTf;
        const float c3 = 4.0f * g.vtf * 0.101321183642337771f;                 // third derivative / 6 = 4 vt / pi^2: theta(T) is a cubic
        eps = ((c3 * eT + y.c2) * eT + y.th1) * eT;
        s.th1 = (3.0f * c3 * eT + 2.0f * y.c2) * eT + y.th1;
        s.c2 = y.c2 + 3.0f * c3 * eT;
        s.sh1 = g.dRf * eR; s.sh2 = g.dTf * s.th1 * s.r;
    }
    const float e2 = eps * eps;                                // |eps| <= half a cell
    const float se = eps * fmaf(e2, fmaf(e2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    const float ce = fmaf(e2, fmaf(e2, fmaf(e2, -1.0f / 720.0f, 1.0f / 24.0f), -0.5f), 1.0f);
    s.st = y.st * ce + y.ct * se;
    s.ct = y.ct * ce - y.st * se;
    s.sh3 = s.r * s.st;
    return s;
}

struct Sph {            // spherical-polar description of a code position + sqrt(h_ii) there
    double r, th;
    double sh1, sh2, sh3;   // sqrt(h11), sqrt(h22), sqrt(h33)
};
template <int KIND>
__device__ __forceinline__ Sph sph_of_code(const GridDev &g, double x1, double x2) {
    Sph s;
    if (KIND == ENT_SPH) {
        s.r = g.rmin + x1 * g.dr;
        s.th = x2 * g.dth;
        s.sh1 = g.dr; s.sh2 = s.r * g.dth;
    } else {
        double eR = exp(g.Rmin + x1 * g.dR);
        double T = x2 * g.dT;
        s.r = g.r0 + eR;
        s.th = theta_of_T(g.vt, T);
        s.sh1 = g.dR * eR; s.sh2 = g.dT * dtheta_dT(g.vt, T) * s.r;
    }
    s.sh3 = s.r * sin(s.th);
    return s;
}

// ---------------------------------------------------------------------------------------------------------
// S3 relativistic Boris (Eq. 3): half electric kick, rotation about B, half kick.  eps = (q/m) dt / 2
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void boris(float u[3], const float E[3], const float B[3], float eps) {
    float um0 = u[0] + eps * E[0], um1 = u[1] + eps * E[1], um2 = u[2] + eps * E[2];
    // 1 / gamma^- from MUFU.RSQ (2 ulp) scales the rotation angle only; the rotation itself conserves |u| for any t as long as
    // s = 2 t / (1 + t^2), whose division by MUFU.RCP (2 ulp) changes |u| by 2 ulp * |t|^2 at most
    const float ig = rsqrtf(1.0f + um0 * um0 + um1 * um1 + um2 * um2);
    float t0 = eps * B[0] * ig, t1 = eps * B[1] * ig, t2 = eps * B[2] * ig;
    float sc = __fdividef(2.0f, 1.0f + t0 * t0 + t1 * t1 + t2 * t2);
    float p0 = um0 + (um1 * t2 - um2 * t1);
    float p1 = um1 + (um2 * t0 - um0 * t2);
    float p2 = um2 + (um0 * t1 - um1 * t0);
    float s0 = sc * t0, s1 = sc * t1, s2 = sc * t2;
    u[0] = um0 + (p1 * s2 - p2 * s1) + eps * E[0];
    u[1] = um1 + (p2 * s0 - p0 * s2) + eps * E[1];
    u[2] = um2 + (p0 * s1 - p1 * s0) + eps * E[2];
}
// the other conventional pusher P:95 names: J.-L. Vay, Phys. Plasmas 15, 056701 (2008); same interface and time levels
__device__ __forceinline__ void vay(float u[3], const float E[3], const float B[3], float eps) {
    float g2 = 1.0f + u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    float ig = rsqrtf(g2);
    ig = ig * (1.5f - 0.5f * g2 * ig * ig);
    const float v0 = u[0] * ig, v1 = u[1] * ig, v2 = u[2] * ig;
    const float p0 = u[0] + eps * (2.0f * E[0] + (v1 * B[2] - v2 * B[1]));        // half step with the old velocity + half E kick
    const float p1 = u[1] + eps * (2.0f * E[1] + (v2 * B[0] - v0 * B[2]));
    const float p2 = u[2] + eps * (2.0f * E[2] + (v0 * B[1] - v1 * B[0]));
    const float a0 = eps * B[0], a1 = eps * B[1], a2 = eps * B[2];                // tau
    const float tau2 = a0 * a0 + a1 * a1 + a2 * a2;
    const float us = p0 * a0 + p1 * a1 + p2 * a2;
    const float sigma = 1.0f + p0 * p0 + p1 * p1 + p2 * p2 - tau2;
    const float gn2 = 0.5f * (sigma + sqrtf(sigma * sigma + 4.0f * (tau2 + us * us)));
    float ign = rsqrtf(gn2);
    ign = ign * (1.5f - 0.5f * gn2 * ign * ign);
    const float t0 = a0 * ign, t1 = a1 * ign, t2 = a2 * ign;
    const float sf = 1.0f / (1.0f + t0 * t0 + t1 * t1 + t2 * t2);
    const float ut = p0 * t0 + p1 * t1 + p2 * t2;
    u[0] = sf * (p0 + ut * t0 + (p1 * t2 - p2 * t1));
    u[1] = sf * (p1 + ut * t1 + (p2 * t0 - p0 * t2));
    u[2] = sf * (p2 + ut * t2 + (p0 * t1 - p1 * t0));
}
// step 5 with the pusher the grid struct selects (ENT_OPT_PUSHER): 0 Boris, 1 Vay
// bit 1 of the pusher: the hybrid pusher of P:976-980 (reading G26): in the guiding-centre regime -- |E| < eovb |B| and the nominal
// gyroradius of the momentum the particle has BEFORE the push, |u| m / (|q||B|), below rho_crit -- the conventional push is followed by
// u <- (u.b) b (momentum perpendicular to the local B set to zero; u.b has received (q/m) E_par dt)
__device__ __forceinline__ void push_momentum(const GridDev &g, float u[3], const float E[3], const float B[3], float eps) {
    float U2 = 0.f;
    if (g.pusher & 2) U2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];     // uniform branch: nothing extra for the conventional pushers
    if (g.pusher & 1) vay(u, E, B, eps); else boris(u, E, B, eps);
    if (g.pusher & 2) {
        const float B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2], E2 = E[0] * E[0] + E[1] * E[1] + E[2] * E[2];
        const float k = g.gca_c * eps;
        if (B2 > 0.f && E2 < g.gca_eovb2 * B2 && U2 < k * k * B2) {
            const float up = (u[0] * B[0] + u[1] * B[1] + u[2] * B[2]) / B2;
            u[0] = up * B[0]; u[1] = up * B[1]; u[2] = up * B[2];
        }
    }
}
__device__ __forceinline__ float inv_gamma(const float u[3]) {
    return rsqrtf(1.0f + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);      // MUFU.RSQ, 2 ulp: 1e-7 cells on a move of 0.45 cells
}

// split x = (old offset + displacement) into a cell shift and an offset in [0,1) (G11)
__device__ __forceinline__ void split_offset(float x, int &di, float &dn) {
    float fl = floorf(x);
    di = (int)fl;
    dn = x - fl;
    if (dn >= 1.0f) { dn = 0.0f; di += 1; }          // tiny negative x: x - floor(x) rounds to 1
}

}  // namespace ent
