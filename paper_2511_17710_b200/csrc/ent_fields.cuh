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

// padded linear index of lattice index (i, j, k)
__device__ __forceinline__ long long fld_at(const GridDev &g, int i, int j, int k) {
    return (long long)(i + NG) + (long long)g.P[0] * ((long long)(j + NG) + (g.D == 3 ? (long long)g.P[1] * (k + NG) : 0));
}
// index of the neighbour of q along dimension A (compile time) at distance S = +1 / -1 on the lattice of component C6, periodic
// wrap; ok = false if it lies outside a non-periodic lattice
template <int C6, int A, int S>
__device__ __forceinline__ void fld_shift(const GridDev &g, const SolverGeom &L, int &i, int &j, int &k, bool &ok) {
    int &q = A == 0 ? i : (A == 1 ? j : k);
    const int n = L.n[C6][A];
    q += S;
    if (q < 0 || q >= n) { if (g.bc[A] == ENT_PERIODIC) q += q < 0 ? n : -n; else ok = false; }
}
// covariant component h_cc F^c of component C6 at lattice index (i, j, k) of its own lattice
template <bool CARTESIAN, int C6>
__device__ __forceinline__ float fld_cov(const GridDev &g, const SolverGeom &L, const float *A, int i, int j, int k) {
    const float v = A[fld_at(g, i, j, k)];
    if (CARTESIAN) return L.cov[C6 % 3] * v;
    double h[3];
    metric_h_axisym(g, i + (fld_stag(C6, 0) ? 0.5 : 0.0), j + (fld_stag(C6, 1) ? 0.5 : 0.0), h);
    return (float)(h[C6 % 3] * (double)v);
}
// F_C6(q + S e_A) - F_C6(q) (S = +1) or F_C6(q) - F_C6(q - e_A) (S = -1), covariant
template <bool CARTESIAN, int C6, int A, int S>
__device__ __forceinline__ float fld_diff(const GridDev &g, const SolverGeom &L, const float *F, int i, int j, int k, bool &ok) {
    int i2 = i, j2 = j, k2 = k;
    // the lattices of the updated component and of C6 differ along A only (node against half-integer points): on a non-periodic
    // dimension the last node has no C6 value "here" either
    if ((A == 0 ? i : (A == 1 ? j : k)) >= L.n[C6][A]) ok = false;
    fld_shift<C6, A, S>(g, L, i2, j2, k2, ok);
    if (!ok) return 0.f;
    const float here = fld_cov<CARTESIAN, C6>(g, L, F, i, j, k), there = fld_cov<CARTESIAN, C6>(g, L, F, i2, j2, k2);
    return S > 0 ? there - here : here - there;
}
template <bool CARTESIAN>
__device__ __forceinline__ float inv_sqrt_h_of(const GridDev &g, const SolverGeom &L, int c6, int i, int j) {
    if (CARTESIAN) return L.inv_sqrt_h;
    double h[3];
    metric_h_axisym(g, i + (fld_stag(c6, 0) ? 0.5 : 0.0), j + (fld_stag(c6, 1) ? 0.5 : 0.0), h);
    return (float)(1.0 / sqrt(h[0] * h[1] * h[2]));
}

// one lattice point of B^C (Eq. A1); C, and with it the stencil, is a compile-time constant
template <bool CARTESIAN, int C>
__device__ __forceinline__ void faraday_point(const GridDev &g, const SolverGeom &L, const FieldRW &F, float dt, int i, int j, int k) {
    constexpr int CB = 3 + C, A = (C + 1) % 3, B = (C + 2) % 3;
    if (i >= L.n[CB][0] || j >= L.n[CB][1] || k >= L.n[CB][2]) return;
    float *Bc = F.c[CB] + fld_at(g, i, j, k);
    if (!CARTESIAN && C == 1 && (j == 0 || j == g.N[1])) { *Bc = 0.f; return; }                 // Eq. 12: B^2 = 0 on the axis
    bool ok = true;
    float curl = 0.f;
    if (A < 2 || g.D == 3) curl += fld_diff<CARTESIAN, B, A, +1>(g, L, F.c[B], i, j, k, ok);     // E_b(+a) - E_b
    if (B < 2 || g.D == 3) curl -= fld_diff<CARTESIAN, A, B, +1>(g, L, F.c[A], i, j, k, ok);     // E_a(+b) - E_a
    if (!ok) return;                                                                           // cannot happen: A1 stays inside the E lattices
    *Bc -= dt * curl * inv_sqrt_h_of<CARTESIAN>(g, L, CB, i, j);                                // Eq. A1
}
// one lattice point of E^C (Eq. A2, Eqs. 12-13 on the axis)
template <bool CARTESIAN, int C>
__device__ __forceinline__ void ampere_point(const GridDev &g, const SolverGeom &L, const FieldRW &F, const CurrentPtrs &J, int haveJ, float dt,
                                             float jc, int i, int j, int k) {
    constexpr int A = (C + 1) % 3, B = (C + 2) % 3;
    if (i >= L.n[C][0] || j >= L.n[C][1] || k >= L.n[C][2]) return;
    const long long at = fld_at(g, i, j, k);
    float *Ec = F.c[C] + at;
    const float Jc = haveJ ? J.c[C][at] : 0.f;
    if (!CARTESIAN && C != 1 && (j == 0 || j == g.N[1])) {                                       // a point on the polar axis
        if (C == 2) { *Ec = 0.f; return; }                                                      // Eq. 12: E^3 = 0
        const bool north = j == 0;                                                              // Eq. 13 and its mirror image at theta = pi
        const float B3 = fld_cov<CARTESIAN, 5>(g, L, F.c[5], i, north ? 0 : g.N[1] - 1, 0);
        *Ec += (float)((double)dt * ((north ? B3 : -B3) - 0.5f * jc * Jc) / axis_area(g, i + 0.5));
        return;
    }
    bool ok = true;
    float curl = 0.f;
    if (A < 2 || g.D == 3) curl += fld_diff<CARTESIAN, 3 + B, A, -1>(g, L, F.c[3 + B], i, j, k, ok);   // B_b - B_b(-a)
    if (B < 2 || g.D == 3) curl -= fld_diff<CARTESIAN, 3 + A, B, -1>(g, L, F.c[3 + A], i, j, k, ok);   // B_a - B_a(-b)
    if (!ok) return;                                   // tangential E on a non-periodic face: the caller's boundary condition
    *Ec += dt * (curl - jc * Jc) * inv_sqrt_h_of<CARTESIAN>(g, L, C, i, j);                      // Eq. A2
}

// blockIdx.x: chunk of x1, blockIdx.y: x2 index, blockIdx.z = component * nmax[2] + x3 index
template <bool CARTESIAN>
__global__ void __launch_bounds__(TPB) faraday_kernel(GridDev g, SolverGeom L, FieldRW F, float dt) {
    const int c = blockIdx.z / L.nmax[2], k = blockIdx.z - c * L.nmax[2], j = blockIdx.y, i = blockIdx.x * TPB + threadIdx.x;
    if (c == 0) faraday_point<CARTESIAN, 0>(g, L, F, dt, i, j, k);
    else if (c == 1) faraday_point<CARTESIAN, 1>(g, L, F, dt, i, j, k);
    else faraday_point<CARTESIAN, 2>(g, L, F, dt, i, j, k);
}
template <bool CARTESIAN>
__global__ void __launch_bounds__(TPB) ampere_kernel(GridDev g, SolverGeom L, FieldRW F, CurrentPtrs J, int haveJ, float dt, float jc) {
    const int c = blockIdx.z / L.nmax[2], k = blockIdx.z - c * L.nmax[2], j = blockIdx.y, i = blockIdx.x * TPB + threadIdx.x;
    if (c == 0) ampere_point<CARTESIAN, 0>(g, L, F, J, haveJ, dt, jc, i, j, k);
    else if (c == 1) ampere_point<CARTESIAN, 1>(g, L, F, J, haveJ, dt, jc, i, j, k);
    else ampere_point<CARTESIAN, 2>(g, L, F, J, haveJ, dt, jc, i, j, k);
}

// All-periodic Cartesian grids (every lattice is N1 x N2 x N3): one thread per CELL advances the three components at once, so that
// every array is read from DRAM once per call (the per-component kernels read each source array twice) and the neighbours come from
// L1/L2; cells whose stencil wraps around the box (the last / first layer of a dimension) take the per-component code.
// Same arithmetic as faraday_point / ampere_point.  blockIdx.y = x2 index, blockIdx.z = x3 index.
__global__ void __launch_bounds__(TPB) faraday_cart_kernel(GridDev g, SolverGeom L, FieldRW F, float dt) {
    const int i = blockIdx.x * TPB + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= g.N[0]) return;
    const bool d3 = g.D == 3;
    if (i + 1 < g.N[0] && j + 1 < g.N[1] && (!d3 || k + 1 < g.N[2])) {
        const long long at = fld_at(g, i, j, k), sy = g.P[0], sz = d3 ? (long long)g.P[0] * g.P[1] : 0;
        const float *E1 = F.c[0] + at, *E2 = F.c[1] + at, *E3 = F.c[2] + at;
        const float e1 = E1[0], e2 = E2[0], e3 = E3[0];
        const float c1 = L.cov[0], c2 = L.cov[1], c3 = L.cov[2], f = dt * L.inv_sqrt_h;
        float curl1 = c3 * E3[sy] - c3 * e3, curl2 = -(c3 * E3[1] - c3 * e3), curl3 = (c2 * E2[1] - c2 * e2) - (c1 * E1[sy] - c1 * e1);
        if (d3) { curl1 -= c2 * E2[sz] - c2 * e2; curl2 += c1 * E1[sz] - c1 * e1; }
        F.c[3][at] -= curl1 * f; F.c[4][at] -= curl2 * f; F.c[5][at] -= curl3 * f;
        return;
    }
    faraday_point<true, 0>(g, L, F, dt, i, j, k);
    faraday_point<true, 1>(g, L, F, dt, i, j, k);
    faraday_point<true, 2>(g, L, F, dt, i, j, k);
}
__global__ void __launch_bounds__(TPB) ampere_cart_kernel(GridDev g, SolverGeom L, FieldRW F, CurrentPtrs J, int haveJ, float dt, float jc) {
    const int i = blockIdx.x * TPB + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= g.N[0]) return;
    const bool d3 = g.D == 3;
    if (i >= 1 && j >= 1 && (!d3 || k >= 1)) {
        const long long at = fld_at(g, i, j, k), sy = g.P[0], sz = d3 ? (long long)g.P[0] * g.P[1] : 0;
        const float *B1 = F.c[3] + at, *B2 = F.c[4] + at, *B3 = F.c[5] + at;
        const float b1 = B1[0], b2 = B2[0], b3 = B3[0];
        const float c1 = L.cov[0], c2 = L.cov[1], c3 = L.cov[2], f = dt * L.inv_sqrt_h;
        float curl1 = c3 * b3 - c3 * B3[-sy], curl2 = -(c3 * b3 - c3 * B3[-1]), curl3 = (c2 * b2 - c2 * B2[-1]) - (c1 * b1 - c1 * B1[-sy]);
        if (d3) { curl1 -= c2 * b2 - c2 * B2[-sz]; curl2 += c1 * b1 - c1 * B1[-sz]; }
        const float j1 = haveJ ? J.c[0][at] : 0.f, j2 = haveJ ? J.c[1][at] : 0.f, j3 = haveJ ? J.c[2][at] : 0.f;
        F.c[0][at] += (curl1 - jc * j1) * f; F.c[1][at] += (curl2 - jc * j2) * f; F.c[2][at] += (curl3 - jc * j3) * f;
        return;
    }
    ampere_point<true, 0>(g, L, F, J, haveJ, dt, jc, i, j, k);
    ampere_point<true, 1>(g, L, F, J, haveJ, dt, jc, i, j, k);
    ampere_point<true, 2>(g, L, F, J, haveJ, dt, jc, i, j, k);
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
