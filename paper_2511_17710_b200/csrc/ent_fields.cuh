// ent_fields.cuh -- N2: field solver on the Yee lattice, sub-steps 2, 10, 11 of the loop: the discretized
// Faraday (Eq. A1) and Ampere (Eq. A2) laws of App. A in a diagonal metric, the polar-axis rules of Sec. 2.6
// (Eqs. 12-13), and the ghost-layer fill the gather of ent_step expects.  sm_100a.
//
// Arrays: six padded planar fp32 arrays of contravariant components (ent.h).  Code coordinates are counted in cells, so the
// difference operators of P:1060-1064 have Delta x = 1; covariant components F_i = h_ii F^i and sqrt(h) are taken at the
// component's own position.  With (c, a, b) cyclic:
//   A1:  B^c -= dt / sqrt(h) { E_b(+a) - E_b - (E_a(+b) - E_a) }                      forward differences, at B^c's position
//   A2:  E^c += dt / sqrt(h) { B_b - B_b(-a) - (B_a - B_a(-b)) - jc conformal J^c }   backward differences, at E^c's position
// One thread per lattice point of the updated component, x1 fastest (coalesced rows; the neighbours in x2, x3 come through L1/L2):
// the kernels move 36 B (Faraday) / 48 B (Ampere with currents) per cell and are bound by HBM.  Cartesian grids use constant
// fp32 factors h_b / sqrt(h); the axisymmetric grids evaluate the metric in fp64 per point (2D grids, a few million points).
#pragma once
#include "ent_kernels.cuh"

namespace ent {

struct FieldRW { float *c[6]; };
struct SolverGeom {
    int n[6][3];       // lattice extent of field component c6 (E1,E2,E3,B1,B2,B3) along dimension d
    int nmax[3];
    int axis;          // the AXIS dimension (1) or -1
    float cov[3];      // CART: h_cc (covariant factor of component c)
    float inv_sqrt_h;  // CART: 1 / sqrt(h)
};

__host__ __device__ inline bool fld_stag(int c6, int d) { const int c = c6 % 3; return c6 < 3 ? (d == c) : (d != c); }

// h11, h22, h33 at code position (x1, x2) of an axisymmetric grid, fp64
__device__ __forceinline__ void metric_h_axisym(const GridDev &g, double x1, double x2, double h[3]) {
    if (g.kind == ENT_SPH) {
        const double r = g.rmin + x1 * g.dr, th = x2 * g.dth, s = r * sin(th);
        h[0] = g.dr * g.dr; h[1] = (r * g.dth) * (r * g.dth); h[2] = s * s;
    } else {
        const double eR = exp(g.Rmin + x1 * g.dR), T = x2 * g.dT, r = g.r0 + eR;
        const double a = g.dR * eR, b = g.dT * dtheta_dT(g.vt, T) * r, s = r * sin(theta_of_T(g.vt, T));
        h[0] = a * a; h[1] = b * b; h[2] = s * s;
    }
}
// A(x1) of Eq. 13: integral of sqrt(h) over the half cell next to the axis, closed forms of P:372-382
__device__ __forceinline__ double axis_area(const GridDev &g, double x1) {
    if (g.kind == ENT_SPH) { const double r = g.rmin + x1 * g.dr; return r * r * g.dr * (1.0 - cos(0.5 * g.dth)); }
    const double eR = exp(g.Rmin + x1 * g.dR), r = g.r0 + eR;
    return r * r * eR * g.dR * (1.0 - cos(theta_of_T(g.vt, 0.5 * g.dT)));
}

// covariant component h_cc F^c of component c6 at lattice index q (periodic wrap); ok = false if q is outside the lattice
template <bool CARTESIAN>
__device__ __forceinline__ float fld_cov(const GridDev &g, const SolverGeom &L, const float *A, int c6, int q0, int q1, int q2, bool &ok) {
    int q[3] = { q0, q1, q2 };
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int n = L.n[c6][d];
        if ((unsigned)q[d] < (unsigned)n) continue;
        if (d < g.D && g.bc[d] == ENT_PERIODIC) q[d] += q[d] < 0 ? n : -n;
        else { ok = false; return 0.f; }
    }
    const float v = A[(long long)(q[0] + NG) + (long long)g.P[0] * ((long long)(q[1] + NG) + (g.D == 3 ? (long long)g.P[1] * (q[2] + NG) : 0))];
    if (CARTESIAN) return L.cov[c6 % 3] * v;
    double h[3];
    metric_h_axisym(g, q[0] + (fld_stag(c6, 0) ? 0.5 : 0.0), q[1] + (fld_stag(c6, 1) ? 0.5 : 0.0), h);
    return (float)(h[c6 % 3] * (double)v);
}
template <bool CARTESIAN>
__device__ __forceinline__ float inv_sqrt_h_of(const GridDev &g, const SolverGeom &L, int c6, int i, int j) {
    if (CARTESIAN) return L.inv_sqrt_h;
    double h[3];
    metric_h_axisym(g, i + (fld_stag(c6, 0) ? 0.5 : 0.0), j + (fld_stag(c6, 1) ? 0.5 : 0.0), h);
    return (float)(1.0 / sqrt(h[0] * h[1] * h[2]));
}

// blockIdx.x: chunk of x1, blockIdx.y: x2 index, blockIdx.z = component * nmax[2] + x3 index
template <bool CARTESIAN>
__global__ void __launch_bounds__(TPB) faraday_kernel(GridDev g, SolverGeom L, FieldRW F, float dt) {
    const int c = blockIdx.z / L.nmax[2], k = blockIdx.z - c * L.nmax[2], j = blockIdx.y, i = blockIdx.x * TPB + threadIdx.x;
    const int cB = 3 + c, a = (c + 1) % 3, b = (c + 2) % 3;
    if (i >= L.n[cB][0] || j >= L.n[cB][1] || k >= L.n[cB][2]) return;
    float *Bc = F.c[cB] + ((long long)(i + NG) + (long long)g.P[0] * ((long long)(j + NG) + (g.D == 3 ? (long long)g.P[1] * (k + NG) : 0)));
    if (!CARTESIAN && c == 1 && (j == 0 || j == g.N[1])) { *Bc = 0.f; return; }                 // Eq. 12: B^2 = 0 on the axis
    bool ok = true;
    float curl = 0.f;
    const int e[3][3] = { {1, 0, 0}, {0, 1, 0}, {0, 0, 1} };
    if (a < g.D) curl += fld_cov<CARTESIAN>(g, L, F.c[b], b, i + e[a][0], j + e[a][1], k + e[a][2], ok) - fld_cov<CARTESIAN>(g, L, F.c[b], b, i, j, k, ok);
    if (b < g.D) curl -= fld_cov<CARTESIAN>(g, L, F.c[a], a, i + e[b][0], j + e[b][1], k + e[b][2], ok) - fld_cov<CARTESIAN>(g, L, F.c[a], a, i, j, k, ok);
    if (!ok) return;                                                                           // cannot happen: A1 stays inside the E lattices
    *Bc -= dt * curl * inv_sqrt_h_of<CARTESIAN>(g, L, cB, i, j);                                // Eq. A1
}

template <bool CARTESIAN>
__global__ void __launch_bounds__(TPB) ampere_kernel(GridDev g, SolverGeom L, FieldRW F, CurrentPtrs J, int haveJ, float dt, float jc) {
    const int c = blockIdx.z / L.nmax[2], k = blockIdx.z - c * L.nmax[2], j = blockIdx.y, i = blockIdx.x * TPB + threadIdx.x;
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    if (i >= L.n[c][0] || j >= L.n[c][1] || k >= L.n[c][2]) return;
    const long long at = (long long)(i + NG) + (long long)g.P[0] * ((long long)(j + NG) + (g.D == 3 ? (long long)g.P[1] * (k + NG) : 0));
    float *Ec = F.c[c] + at;
    const float Jc = haveJ ? J.c[c][at] : 0.f;
    bool ok = true;
    if (!CARTESIAN && c != 1 && (j == 0 || j == g.N[1])) {                                       // a point on the polar axis
        if (c == 2) { *Ec = 0.f; return; }                                                      // Eq. 12: E^3 = 0
        const bool north = j == 0;                                                              // Eq. 13 and its mirror image at theta = pi
        const float B3 = fld_cov<CARTESIAN>(g, L, F.c[5], 5, i, north ? 0 : g.N[1] - 1, 0, ok);
        *Ec += (float)((double)dt * ((north ? B3 : -B3) - 0.5f * jc * Jc) / axis_area(g, i + 0.5));
        return;
    }
    float curl = 0.f;
    const int e[3][3] = { {1, 0, 0}, {0, 1, 0}, {0, 0, 1} };
    if (a < g.D) curl += fld_cov<CARTESIAN>(g, L, F.c[3 + b], 3 + b, i, j, k, ok) - fld_cov<CARTESIAN>(g, L, F.c[3 + b], 3 + b, i - e[a][0], j - e[a][1], k - e[a][2], ok);
    if (b < g.D) curl -= fld_cov<CARTESIAN>(g, L, F.c[3 + a], 3 + a, i, j, k, ok) - fld_cov<CARTESIAN>(g, L, F.c[3 + a], 3 + a, i - e[b][0], j - e[b][1], k - e[b][2], ok);
    if (!ok) return;                                   // tangential E on a non-periodic face: the caller's boundary condition
    *Ec += dt * (curl - jc * Jc) * inv_sqrt_h_of<CARTESIAN>(g, L, c, i, j);                      // Eq. A2
}

// ghost layers of the six arrays along dimension `dim` (the transverse range is the whole padded extent, so edges and corners
// are completed dimension after dimension): PERIODIC: periodic image; AXIS: mirror image, E^1 / B^1 even, the others odd
// (reading G10); ABSORB: not touched.  blockIdx.y = component.
__global__ void __launch_bounds__(TPB) field_ghost_kernel(GridDev g, SolverGeom L, FieldRW F, int dim) {
    const int c6 = blockIdx.y;
    const int a = (dim + 1) % 3, b = (dim + 2) % 3;
    const long long na = g.P[a], nb = g.P[b];
    long long t = (long long)blockIdx.x * TPB + threadIdx.x;
    if (t >= na * nb * 2 * NG) return;
    const int slot = (int)(t % (2 * NG)); t /= 2 * NG;
    const long long ia = t % na, ib = t / na;
    const int n = L.n[c6][dim];
    const int gi = slot < NG ? slot - NG : g.N[dim] + (slot - NG);        // -2, -1, N, N + 1 (active index of the layer)
    if (gi >= 0 && gi < n) return;                                        // node lattice of a non-periodic dimension: layer N is a lattice point
    int src; float sign = 1.f;
    if (g.bc[dim] == ENT_PERIODIC) src = gi < 0 ? gi + n : gi - n;
    else {
        src = fld_stag(c6, dim) ? (gi < 0 ? -1 - gi : 2 * n - 1 - gi) : (gi < 0 ? -gi : 2 * (n - 1) - gi);
        if (c6 % 3 != 0) sign = -1.f;
    }
    const long long stride[3] = { 1, g.P[0], (long long)g.P[0] * g.P[1] };
    float *line = F.c[c6] + ia * stride[a] + ib * stride[b];
    line[(long long)(gi + NG) * stride[dim]] = sign * line[(long long)(src + NG) * stride[dim]];
}

}  // namespace ent
