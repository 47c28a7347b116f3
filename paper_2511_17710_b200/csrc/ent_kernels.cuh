// ent_kernels.cuh -- untiled kernels: one thread per particle, global gathers, global atomics.
// This is the structure of the paper's own pusher and deposit functors and serves as the in-repo
// baseline for the tiled kernel (ent_tiled.cuh) as well as the path for unsorted particle blocks.
#pragma once
#include "ent_particle.cuh"

namespace ent {

struct FieldPtrs { const float *c[6]; };
struct CurrentPtrs { float *c[3]; };
struct PartPtrs {
    int32_t *cell; float *d[3]; float *phi; float *u[3]; float *w; uint8_t *tag;
};

constexpr int TPB = 256;

struct MagicDiv {                 // n / d for 0 <= n < 2^31, d >= 1 (multiply-high + shift)
    uint32_t mul, shr, d;
    __device__ __forceinline__ int div(int n) const { return d == 1 ? n : (int)(__umulhi((uint32_t)n, mul) >> shr); }
};
inline MagicDiv make_magicdiv(uint32_t d) {
    MagicDiv f{0, 0, d};
    if (d <= 1) return f;
    uint32_t lg = 0; while ((1ull << lg) < d) ++lg;
    uint32_t p = 31 + lg;
    f.mul = (uint32_t)(((1ull << p) + d - 1) / d);
    f.shr = p - 32;
    return f;
}


// ---- S0-S5: ent_gather_push ----
template <int D, int KIND>
__global__ void __launch_bounds__(TPB) gather_push_kernel(GridDev g, FieldPtrs F, PartPtrs in, PartPtrs out, long long n,
                                                          float eps, float dt) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    bool alive = in.tag ? in.tag[p] != 0 : true;
    int i[3], di[3]; float d[3] = {0.f, 0.f, 0.f}, u[3], phi = 0.f;
    int cell = in.cell[p];
#pragma unroll
    for (int a = 0; a < D; ++a) d[a] = in.d[a][p];
#pragma unroll
    for (int a = 0; a < 3; ++a) u[a] = in.u[a][p];
    if (KIND != ENT_CART) phi = in.phi[p];
    if (alive) {
        unpack_cell<D>(g, cell, i);
        const float *const Fp[6] = { F.c[0], F.c[1], F.c[2], F.c[3], F.c[4], F.c[5] };
        GlobalFieldLoader ld{Fp};
        push_particle<D, KIND>(g, ld, i, d, phi, u, eps, dt, di, alive);
        cell = pack_cell<D>(g, i);
    }
    out.cell[p] = cell;
#pragma unroll
    for (int a = 0; a < D; ++a) out.d[a][p] = d[a];
#pragma unroll
    for (int a = 0; a < 3; ++a) out.u[a][p] = u[a];
    if (KIND != ENT_CART) out.phi[p] = phi;
    if (out.tag) out.tag[p] = alive ? 1 : 0;
}

// ---- S7: ent_deposit (old and new blocks in memory, the paper's i_prev/dx_prev structure) ----
template <int D, int KIND>
__global__ void __launch_bounds__(TPB) deposit_kernel(GridDev g, PartPtrs po, PartPtrs pn, CurrentPtrs J, long long n,
                                                      float q, float inv_dt, unsigned long long *bad_moves) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    bool alive = (po.tag ? po.tag[p] != 0 : true) && (pn.tag ? pn.tag[p] != 0 : true);
    if (!alive) return;                                                        // G9
    int i0[3], i1[3], di[3] = {0, 0, 0};
    unpack_cell<D>(g, po.cell[p], i0);
    unpack_cell<D>(g, pn.cell[p], i1);
    float a[3] = {0.f, 0.f, 0.f}, dn[3] = {0.f, 0.f, 0.f}, u[3];
    bool bad = false;
#pragma unroll
    for (int k = 0; k < D; ++k) {
        int dd = i1[k] - i0[k];
        if (g.bc[k] == ENT_PERIODIC) {                                         // recover the un-wrapped shift
            if (2 * dd > g.N[k]) dd -= g.N[k];
            else if (2 * dd < -g.N[k]) dd += g.N[k];
        }
        if (dd < -1 || dd > 1) bad = true;
        di[k] = dd;
        a[k] = po.d[k][p];
        dn[k] = pn.d[k][p];
    }
    if (bad) { atomicAdd(bad_moves, 1ULL); return; }
#pragma unroll
    for (int k = 0; k < 3; ++k) u[k] = pn.u[k][p];
    float phi0 = 0.f, phi1 = 0.f;
    if (KIND != ENT_CART) { phi0 = po.phi[p]; phi1 = pn.phi[p]; }
    float *const Jp[3] = { J.c[0], J.c[1], J.c[2] };
    GlobalAcc acc{Jp};
    deposit_particle<D, KIND>(g, acc, i0, a, di, dn, phi0, phi1, u, q * po.w[p], inv_dt);
}

// ---- fused S0-S7, in place, untiled ----
template <int D, int KIND>
__global__ void __launch_bounds__(TPB) step_untiled_kernel(GridDev g, FieldPtrs F, PartPtrs P, CurrentPtrs J, long long n,
                                                           float eps, float dt, float q, float inv_dt,
                                                           unsigned long long *bad_moves) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    bool alive = P.tag ? P.tag[p] != 0 : true;
    if (!alive) return;                                                        // dead particles are left untouched
    int i[3], i0[3], di[3]; float d[3] = {0.f, 0.f, 0.f}, a[3], u[3], phi = 0.f;
    unpack_cell<D>(g, P.cell[p], i);
#pragma unroll
    for (int k = 0; k < D; ++k) d[k] = P.d[k][p];
#pragma unroll
    for (int k = 0; k < 3; ++k) { u[k] = P.u[k][p]; a[k] = d[k]; i0[k] = i[k]; }
    if (KIND != ENT_CART) phi = P.phi[p];
    float phi0 = phi;
    const float *const Fp[6] = { F.c[0], F.c[1], F.c[2], F.c[3], F.c[4], F.c[5] };
    GlobalFieldLoader ld{Fp};
    push_particle<D, KIND>(g, ld, i, d, phi, u, eps, dt, di, alive);
    P.cell[p] = pack_cell<D>(g, i);
#pragma unroll
    for (int k = 0; k < D; ++k) P.d[k][p] = d[k];
#pragma unroll
    for (int k = 0; k < 3; ++k) P.u[k][p] = u[k];
    if (KIND != ENT_CART) P.phi[p] = phi;
    if (!alive) { P.tag[p] = 0; return; }
    bool bad = false;
#pragma unroll
    for (int k = 0; k < D; ++k) bad |= (di[k] < -1 || di[k] > 1);
    if (bad) { atomicAdd(bad_moves, 1ULL); return; }
    float *const Jp[3] = { J.c[0], J.c[1], J.c[2] };
    GlobalAcc acc{Jp};
    deposit_particle<D, KIND>(g, acc, i0, a, di, d, phi0, phi, u, q * P.w[p], inv_dt);
}

// ---- S9: periodic ghost fold of one padded array along dimension dim ----
// pass 0: active += ghost on the opposite side, ghost = 0;  pass 1: ghost = periodic image.
// One thread per (ghost layer gi, transverse point); the transverse range covers the whole padded extent so that
// edges and corners are folded dimension after dimension.
__global__ void fold_kernel(GridDev g, CurrentPtrs J, int dim, int pass) {      // blockIdx.y = component
    float *A = J.c[blockIdx.y];
    int a = (dim + 1) % 3, b = (dim + 2) % 3;
    long long na = g.P[a], nb = g.P[b];
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= na * nb * NG) return;
    int gi = (int)(t % NG); t /= NG;
    long long ia = t % na, ib = t / na;
    long long stride[3] = { 1, g.P[0], (long long)g.P[0] * g.P[1] };
    float *line = A + ia * stride[a] + ib * stride[b];
    int N = g.N[dim];
    long long lo = gi, hi = NG + N + gi;
    long long sd = stride[dim];
    if (pass == 0) {
        atomicAdd(&line[(lo + N) * sd], line[lo * sd]);      // atomics: for N < 4 two ghost layers fold onto one cell
        atomicAdd(&line[(hi - N) * sd], line[hi * sd]);
        line[lo * sd] = 0.f;
        line[hi * sd] = 0.f;
    } else {
        line[lo * sd] = line[(lo + N) * sd];
        line[hi * sd] = line[(hi - N) * sd];
    }
}

// ---- N1, step 9 of the loop: one digital filter pass on the conformal currents, Eqs. 9-11 ----
// Each component is convolved with (1/4, 1/2, 1/4) along every grid dimension on its own staggered lattice.  Values beyond the
// lattice: periodic image; polar axis: J^1 even, J^2 odd about the axis, J^3 = 0 on it; ABSORB side: zero.
// `divide`: the pass also turns its result into J^i = conformal J^i / sqrt(h) at the component's own position, except on
// the axis itself (sqrt(h) = 0: Eq. 12-13 use the conformal value there).  `identity`: no convolution (scaling pass only).
// One thread per lattice point, blockIdx.y = component; src and dst are different arrays.
struct FilterGeom {
    int n[3][3];       // lattice extent of component c along dimension d
    int rule[3];       // boundary rule of dimension d (ENT_PERIODIC / ENT_ABSORB / ENT_AXIS); unused dimensions: ENT_PERIODIC, n = 1
};
__device__ __forceinline__ bool filter_on_axis(const GridDev &g, const FilterGeom &L, int comp, int q1) {
    return g.kind != ENT_CART && comp != 1 && (q1 == 0 || q1 == L.n[comp][1] - 1);      // theta lattice of J^1, J^3: nodes 0 .. N_2
}
__device__ __forceinline__ float filter_fetch(const GridDev &g, const FilterGeom &L, const float *A, int comp, int q0, int q1, int q2) {
    int q[3] = { q0, q1, q2 };
    float sign = 1.f;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int n = L.n[comp][d];
        if ((unsigned)q[d] < (unsigned)n) continue;
        if (L.rule[d] == ENT_PERIODIC) q[d] += q[d] < 0 ? n : -n;
        else if (L.rule[d] == ENT_AXIS) {
            if (comp == d) { q[d] = q[d] < 0 ? -1 - q[d] : 2 * n - 1 - q[d]; sign = -sign; }      // (j + 1/2) -> -(j + 1/2): odd
            else q[d] = q[d] < 0 ? -q[d] : 2 * (n - 1) - q[d];                                    // node j -> -j: even
        } else return 0.f;
    }
    if (comp == 2 && filter_on_axis(g, L, comp, q[1])) return 0.f;              // J^3(i, 0) = 0: a condition on the INPUT of the stencil
    const long long idx = (long long)(q[0] + NG) + (long long)g.P[0] * ((long long)(q[1] + NG) + (g.D == 3 ? (long long)g.P[1] * (q[2] + NG) : 0));
    return sign * A[idx];
}
__device__ __forceinline__ float sqrt_h_at(const GridDev &g, double x1, double x2) {          // sqrt(h11 h22 h33)
    if (g.kind == ENT_CART) return g.dx[0] * g.dx[1] * g.dx[2];
    if (g.kind == ENT_SPH) { const double r = g.rmin + x1 * g.dr, th = x2 * g.dth; return (float)(g.dr * (r * g.dth) * (r * sin(th))); }
    const double eR = exp(g.Rmin + x1 * g.dR), T = x2 * g.dT, r = g.r0 + eR;
    return (float)((g.dR * eR) * (g.dT * dtheta_dT(g.vt, T) * r) * (r * sin(theta_of_T(g.vt, T))));
}
// One pass, no shared memory and no barriers: a warp owns FT_W = 30 consecutive points of FT_R consecutive lattice rows (its 32
// lanes sit on x = i0 - 1 .. i0 + 30, the two outer lanes are halo) and marches along x3.  Per plane a lane loads the FT_R + 2
// values J(x, j - 1 .. j + FT_R, k) (coalesced rows, all in flight together; the two rows shared with the neighbouring warps of the
// CTA come from L1), filters them along x2 in registers, gets its x1 neighbours by two shuffles per row, and keeps the in-plane sums
// P_{k-1}, P_k, P_{k+1} of its rows in registers: out_k = P_{k-1}/4 + P_k/2 + P_{k+1}/4 (f = (1/2)^(D + |di| + |dj| + |dk|) =
// w(di) w(dj) w(dk), Eqs. 9-11); in 2D out = P.  The boundary rules are applied once per lane column, warp row and plane (MAPPED,
// see filter_load_rows), not per load.
// mode 0: filter; 1: no convolution (scaling pass only); 2: copy.  blockIdx.z = component * nkc + chunk of FT_K planes.
constexpr int FT_W = 30, FT_R = 3, FT_J = 4, FT_ROWS = FT_R * FT_J, FT_K = 16, FT_TPB = 32 * FT_J;   // measured: (R, warps, planes) = (3, 4, 16) .. (4, 4, 64) within 5 %
struct FilterRow { const float *A; int comp, x, j, k0, k1, n0, n1, n2; long long P0, P01;
                   int xo, ro[FT_R + 2], P01i; float xf, rf[FT_R + 2]; };     // MAPPED path: element offsets (a padded array has < 2^31 elements) and factors of the lane's column and the warp's rows
// the boundary rule of one dimension as (mapped index, factor): periodic image, mirror image about the polar axis (odd for the
// component along the dimension, even otherwise), zero beyond an ABSORB side.  An index more than one image away is not needed by
// any lattice point and maps to (0, 0).
__device__ __forceinline__ void filter_map1(const FilterGeom &L, int comp, int d, int q, int &qq, float &f) {
    const int n = L.n[comp][d];
    qq = q; f = 1.f;
    if ((unsigned)q < (unsigned)n) return;
    if (L.rule[d] == ENT_PERIODIC) qq = q + (q < 0 ? n : -n);
    else if (L.rule[d] == ENT_AXIS) {
        if (comp == d) { qq = q < 0 ? -1 - q : 2 * n - 1 - q; f = -1.f; }
        else qq = q < 0 ? -q : 2 * (n - 1) - q;
    } else { qq = 0; f = 0.f; }
    if ((unsigned)qq >= (unsigned)n) { qq = 0; f = 0.f; }
}
// MAPPED: the rules of filter_fetch are separable, so the lane's column, the warp's rows and the plane are mapped once each and a
// load is one address and (SIGNED: grids with a side that is not periodic) one multiplication.  !MAPPED: filter_fetch per load
// (lattices too small for the one-image mapping).
template <bool MAPPED, bool SIGNED>
__device__ __forceinline__ void filter_load_rows(const GridDev &g, const FilterGeom &L, const FilterRow &t, int k, float v[FT_R + 2]) {
    if (MAPPED) {
        int kk = k; float kf = 1.f;                                                          // warp-uniform
        if (SIGNED) filter_map1(L, t.comp, 2, k, kk, kf);
        else { kk += kk < 0 ? t.n2 : 0; kk -= kk >= t.n2 ? t.n2 : 0; }                       // every side periodic
        const float *p = t.A + (t.xo + t.P01i * (kk + NG));
#pragma unroll
        for (int r = 0; r < FT_R + 2; ++r) { v[r] = __ldg(p + t.ro[r]); if (SIGNED) v[r] *= t.xf * t.rf[r] * kf; }
    } else {
#pragma unroll
        for (int r = 0; r < FT_R + 2; ++r) v[r] = (t.x <= t.n0 && t.j - 1 + r <= t.n1) ? filter_fetch(g, L, t.A, t.comp, t.x, t.j - 1 + r, k) : 0.f;
    }
}
__device__ __forceinline__ void filter_in_plane(const float v[FT_R + 2], float P[FT_R]) {
#pragma unroll
    for (int r = 0; r < FT_R; ++r) {
        const float c = 0.25f * v[r] + 0.5f * v[r + 1] + 0.25f * v[r + 2];      // along x2, in the lane
        const float l = __shfl_up_sync(0xffffffffu, c, 1), rr = __shfl_down_sync(0xffffffffu, c, 1);
        P[r] = 0.25f * l + 0.5f * c + 0.25f * rr;                               // along x1, across lanes (valid on lanes 1 .. 30)
    }
}
template <bool MAPPED, bool SIGNED, class EMIT>
__device__ __forceinline__ void filter_march(const GridDev &g, const FilterGeom &L, const FilterRow &t, bool d3, EMIT &&emit) {
    float v[FT_R + 2], Pm[FT_R], Pc[FT_R], Pn[FT_R];
    if (!d3) {
        filter_load_rows<MAPPED, SIGNED>(g, L, t, 0, v); filter_in_plane(v, Pc);
#pragma unroll
        for (int r = 0; r < FT_R; ++r) emit(0, r, Pc[r]);
        return;
    }
    filter_load_rows<MAPPED, SIGNED>(g, L, t, t.k0 - 1, v); filter_in_plane(v, Pm);
    filter_load_rows<MAPPED, SIGNED>(g, L, t, t.k0, v); filter_in_plane(v, Pc);
    for (int k = t.k0; k < t.k1; ++k) {
        filter_load_rows<MAPPED, SIGNED>(g, L, t, k + 1, v); filter_in_plane(v, Pn);
#pragma unroll
        for (int r = 0; r < FT_R; ++r) { emit(k, r, 0.25f * Pm[r] + 0.5f * Pc[r] + 0.25f * Pn[r]); Pm[r] = Pc[r]; Pc[r] = Pn[r]; }
    }
}
__global__ void __launch_bounds__(FT_TPB) filter_pass_kernel(GridDev g, FilterGeom L, CurrentPtrs src, CurrentPtrs dst, int mode, int divide, int nkc) {
    FilterRow t;
    t.comp = blockIdx.z / nkc;
    const int kc = blockIdx.z - t.comp * nkc;
    const int n2 = L.n[t.comp][2];
    t.n0 = L.n[t.comp][0]; t.n1 = L.n[t.comp][1];
    const int lane = threadIdx.x & 31, i0 = blockIdx.x * FT_W, j0 = blockIdx.y * FT_ROWS;
    t.k0 = kc * FT_K;
    if (i0 >= t.n0 || j0 >= t.n1 || t.k0 >= n2) return;              // the grid is sized for the largest lattice
    t.k1 = min(t.k0 + FT_K, n2);
    t.x = i0 - 1 + lane; t.j = j0 + (threadIdx.x >> 5) * FT_R;       // first of the warp's rows
    if (t.j >= t.n1) return;                                         // whole warp: none of its rows exists (no barriers in this kernel)
    t.A = src.c[t.comp];
    float *O = dst.c[t.comp];
    t.P0 = g.P[0]; t.P01 = g.D == 3 ? (long long)g.P[0] * g.P[1] : 0;
    const bool mine_x = lane >= 1 && lane <= FT_W && t.x < t.n0;     // this lane owns the lattice points (x, j .. j + FT_R - 1)
    const long long at = (long long)(t.x + NG) + t.P0 * (t.j + NG) + (g.D == 3 ? t.P01 * NG : 0);     // (x, j, k = 0)
    float sh[FT_R]; bool axis_node[FT_R];
#pragma unroll
    for (int r = 0; r < FT_R; ++r) {
        axis_node[r] = filter_on_axis(g, L, t.comp, t.j + r);
        sh[r] = (divide && mine_x && t.j + r < t.n1 && !axis_node[r]) ? sqrt_h_at(g, t.x + (t.comp == 0 ? 0.5 : 0.0), t.j + r + (t.comp == 1 ? 0.5 : 0.0)) : 1.f;
    }
    auto emit = [&](int k, int r, float a) {
        if (!mine_x || t.j + r >= t.n1) return;
        if (mode == 0 && t.comp == 2 && axis_node[r]) a = 0.f;                  // J^3(i, 0) = 0
        if (divide && !axis_node[r]) a /= sh[r];
        O[at + t.P0 * r + t.P01 * k] = a;
    };
    if (mode != 0) {
        if (mine_x)
            for (int k = t.k0; k < t.k1; ++k)
#pragma unroll
                for (int r = 0; r < FT_R; ++r) if (t.j + r < t.n1) emit(k, r, t.A[at + t.P0 * r + t.P01 * k]);
        return;
    }
    const bool d3 = g.D == 3;
    const bool mapped = t.n0 >= 2 && t.n1 >= FT_R + 2 && (!d3 || n2 >= 3);
    if (mapped) {
        bool sgn = false;
        for (int d = 0; d < g.D; ++d) sgn = sgn || L.rule[d] != ENT_PERIODIC;
        int xx; float f; filter_map1(L, t.comp, 0, t.x, xx, f);
        if (sgn) t.xf = f;                                            // every side periodic: the factors are 1 and are not kept
        t.xo = xx + NG; t.P01i = (int)t.P01; t.n2 = n2;
#pragma unroll
        for (int r = 0; r < FT_R + 2; ++r) {
            int jj; filter_map1(L, t.comp, 1, t.j - 1 + r, jj, f);
            if (t.comp == 2 && filter_on_axis(g, L, t.comp, jj)) f = 0.f;                       // J^3(i, 0) = 0: a condition on the INPUT of the stencil
            if (sgn) t.rf[r] = f;
            t.ro[r] = (int)t.P0 * (jj + NG);
        }
        if (sgn) filter_march<true, true>(g, L, t, d3, emit); else filter_march<true, false>(g, L, t, d3, emit);
    } else filter_march<false, false>(g, L, t, d3, emit);
}

// ---- N4: tag sort: stable partition, alive particles first ----
__global__ void __launch_bounds__(TPB) compact_flag_kernel(const uint8_t *tag, long long n, int32_t *flag) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p < n) flag[p] = tag[p] != 0;
}
// pos[p] = number of alive particles before p (exclusive scan of the flags); pos[n] = number alive
__global__ void __launch_bounds__(TPB) compact_scatter_kernel(const int32_t *pos, PartPtrs in, PartPtrs out, long long n, int D, int axisym,
                                                              long long *n_alive) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    const long long na = pos[n];
    if (p == 0 && n_alive) *n_alive = na;
    const bool alive = in.tag[p] != 0;
    const long long dst = alive ? (long long)pos[p] : na + (p - pos[p]);
    out.cell[dst] = in.cell[p];
    for (int a = 0; a < D; ++a) out.d[a][dst] = in.d[a][p];
    for (int a = 0; a < 3; ++a) out.u[a][dst] = in.u[a][p];
    out.w[dst] = in.w[p];
    if (axisym) out.phi[dst] = in.phi[p];
    out.tag[dst] = alive ? 1 : 0;
}

// ---- S10: counting sort by tile-major key ----
template <int D>
__global__ void __launch_bounds__(TPB) sort_hist_kernel(GridDev g, const int32_t *cell, long long n, int32_t *keys, int32_t *count) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    int i[3];
    unpack_cell<D>(g, cell[p], i);
    int k = sort_key<D>(g, i);
    keys[p] = k;
    atomicAdd(count + k, 1);
}

constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_CHUNK = TPB * SCAN_ITEMS;

__device__ __forceinline__ int block_exclusive_scan(int v, int &total) {      // TPB threads
    __shared__ int wsum[TPB / 32];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int s = lane < TPB / 32 ? wsum[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        if (lane < TPB / 32) wsum[lane] = s;
    }
    __syncthreads();
    int base = wid ? wsum[wid - 1] : 0;
    total = wsum[TPB / 32 - 1];
    __syncthreads();
    return base + x - v;
}

// pass 1: per-chunk totals
__global__ void __launch_bounds__(TPB) scan_reduce_kernel(const int32_t *in, long long m, int32_t *chunk_sum) {
    long long base = (long long)blockIdx.x * SCAN_CHUNK + (long long)threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < m) s += in[base + k];
    int total;
    block_exclusive_scan(s, total);
    if (threadIdx.x == 0) chunk_sum[blockIdx.x] = total;
}
// pass 2: exclusive scan of the chunk totals, one block
__global__ void __launch_bounds__(TPB) scan_chunks_kernel(int32_t *chunk_sum, int nchunks) {
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nchunks; b0 += TPB) {
        int idx = b0 + threadIdx.x;
        int v = idx < nchunks ? chunk_sum[idx] : 0;
        int total;
        int ex = block_exclusive_scan(v, total);
        int c = carry;
        if (idx < nchunks) chunk_sum[idx] = c + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + total;
        __syncthreads();
    }
}
// pass 3: exclusive scan inside each chunk + chunk offset; out[m] = grand total is written by the last chunk.
// `cursor` (may alias nothing) receives a second copy used as the scatter cursor.
__global__ void __launch_bounds__(TPB) scan_apply_kernel(const int32_t *in, long long m, const int32_t *chunk_off,
                                                         int32_t *out, int32_t *cursor) {
    long long base = (long long)blockIdx.x * SCAN_CHUNK + (long long)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS]; int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = base + k < m ? in[base + k] : 0; s += v[k]; }
    int total;
    int ex = block_exclusive_scan(s, total) + chunk_off[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < m) { out[base + k] = ex; cursor[base + k] = ex; }
        ex += v[k];
        if (base + k == m - 1) out[m] = ex;
    }
}

// tile_off[t] = key_offsets[t * tcells], t = 0..ntiles; tile_count[t] = population of tile t
__global__ void tile_offsets_kernel(const int32_t *key_off, int tcells, long long ntiles, int32_t *tile_off, int32_t *tile_count) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t <= ntiles) tile_off[t] = key_off[t * tcells];
    if (t < ntiles) tile_count[t] = key_off[(t + 1) * tcells] - key_off[t * tcells];
}

// chunks[t] = ceil(count of tile t / chunk): the number of CTAs the tiled step gives to tile t
__global__ void tile_chunks_kernel(const int32_t *tile_off, long long ntiles, int chunk, int32_t *chunks) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < ntiles) chunks[t] = (tile_off[t + 1] - tile_off[t] + chunk - 1) / chunk;
}

// tile_wmax[t] = max |w| over the particles of tile t (scale of the tile's fixed-point J accumulation)
__global__ void __launch_bounds__(128) tile_wmax_kernel(const int32_t *tile_off, const float *w, float *tile_wmax) {
    __shared__ float red[4];
    const long long p0 = tile_off[blockIdx.x], p1 = tile_off[blockIdx.x + 1];
    float m = 0.f;
    for (long long p = p0 + threadIdx.x; p < p1; p += 128) m = fmaxf(m, fabsf(w[p]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) tile_wmax[blockIdx.x] = fmaxf(fmaxf(red[0], red[1]), fmaxf(red[2], red[3]));
}

__global__ void __launch_bounds__(TPB) sort_scatter_kernel(const int32_t *keys, int32_t *cursor, PartPtrs in, PartPtrs out,
                                                           long long n, int D, int axisym) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    long long dst = atomicAdd(cursor + keys[p], 1);
    out.cell[dst] = in.cell[p];
    for (int a = 0; a < D; ++a) out.d[a][dst] = in.d[a][p];
    for (int a = 0; a < 3; ++a) out.u[a][dst] = in.u[a][p];
    out.w[dst] = in.w[p];
    if (axisym) out.phi[dst] = in.phi[p];
    if (in.tag) out.tag[dst] = in.tag[p];
}


// Staged form of the scatter for blocks that arrive in an unrelated order (ENT_OPT_SORT_STAGING): scattering eight 4-byte arrays
// to random slots writes one word of every 32-byte DRAM sector it touches (a read-modify-write of the sector per word: measured
// 131 ms per species on the shuffled C4 block).  Here the record is packed to 32 bytes and written to its slot of an
// array-of-structures side buffer as ONE full sector (two 16-byte stores), and a second, fully coalesced pass unpacks the side
// buffer into the caller's arrays.  Record: cell, d0, d1, (d2 | phi | 0), u0, u1, u2, w.
__global__ void __launch_bounds__(TPB) sort_scatter_aos_kernel(const int32_t *keys, int32_t *cursor, PartPtrs in, float4 *aos, uint8_t *tag_out,
                                                               long long n, int D, int axisym) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    const long long dst = atomicAdd(cursor + keys[p], 1);
    const float third = D == 3 ? in.d[2][p] : (axisym ? in.phi[p] : 0.f);
    aos[2 * dst] = make_float4(__int_as_float(in.cell[p]), in.d[0][p], in.d[1][p], third);
    aos[2 * dst + 1] = make_float4(in.u[0][p], in.u[1][p], in.u[2][p], in.w[p]);
    if (in.tag) tag_out[dst] = in.tag[p];
}
__global__ void __launch_bounds__(TPB) sort_unpack_aos_kernel(const float4 *aos, PartPtrs out, long long n, int D, int axisym) {
    long long p = (long long)blockIdx.x * TPB + threadIdx.x;
    if (p >= n) return;
    const float4 a = aos[2 * p], b = aos[2 * p + 1];
    out.cell[p] = __float_as_int(a.x);
    out.d[0][p] = a.y; out.d[1][p] = a.z;
    if (D == 3) out.d[2][p] = a.w; else if (axisym) out.phi[p] = a.w;
    out.u[0][p] = b.x; out.u[1][p] = b.y; out.u[2][p] = b.z; out.w[p] = b.w;
}

// ---------------------------------------------------------------------------------------------------------
// S10, incremental form ("re-bin"): the input block is tile-contiguous already (a previous ent_sort produced it) and its
// particles have drifted a few cells, so almost all of them stay in their tile and the rest go to one of the 3^D - 1
// neighbouring tiles.  One CTA per SOURCE tile: class counts per destination in shared memory, one global reservation per
// (source tile, destination), particles of a warp that share a destination get consecutive slots in lane order (so the
// ~90 % that stay are written fully coalesced).  Order inside a destination tile: unspecified.
// ---------------------------------------------------------------------------------------------------------
constexpr int REBIN_TPB = 256;
constexpr int REBIN_CLASSES = 28;            // 27 neighbours (3^D used) + "far"

struct RebinGeom {
    int D, N[3], T[3], nt[3], per[3];
    int mext[3];                 // smallest tile extent of a dimension (the last tile may be partial)
    MagicDiv dN0, dN01, dT[3], dnt0, dnt01;
    __device__ __forceinline__ void tile_coords(int tile, int s[3]) const {
        s[2] = dnt01.div(tile); const int r = tile - s[2] * nt[0] * nt[1]; s[1] = dnt0.div(r); s[0] = r - s[1] * nt[0];
    }
    __device__ __forceinline__ void tile_of_cell(int cell, int t[3]) const {
        int i0, i1, i2 = 0;
        if (D == 2) { i1 = dN0.div(cell); i0 = cell - i1 * N[0]; }
        else { int n01 = N[0] * N[1]; i2 = dN01.div(cell); int r = cell - i2 * n01; i1 = dN0.div(r); i0 = r - i1 * N[0]; }
        t[0] = dT[0].div(i0); t[1] = dT[1].div(i1); t[2] = (D == 3) ? dT[2].div(i2) : 0;
    }
    // Destination class of a particle of source tile s (origin o, extent te: the last tile of a dimension may be partial), its
    // destination tile td and, for a particle that stays (class 13), the index lc of its cell inside the tile.  The ~87 % that
    // stay need the two divisions of the cell decode only; one that lands within one (smallest) tile extent of the source tile's
    // box, the shorter way round on a periodic axis, is in the neighbour tile that three comparisons name (td is not set: only
    // class 27 uses it); the rest take the tile divisions and the wrap logic of classify.
    __device__ __forceinline__ int classify_cell(int cell, int src, const int s[3], const int o[3], const int te[3], int &td, int &lc) const {
        int i0, i1, i2 = 0;
        if (D == 2) { i1 = dN0.div(cell); i0 = cell - i1 * N[0]; }
        else { int n01 = N[0] * N[1]; i2 = dN01.div(cell); int r = cell - i2 * n01; i1 = dN0.div(r); i0 = r - i1 * N[0]; }
        const int u0 = i0 - o[0], u1 = i1 - o[1], u2 = i2 - o[2];
        if ((unsigned)u0 < (unsigned)te[0] && (unsigned)u1 < (unsigned)te[1] && (unsigned)u2 < (unsigned)te[2]) {
            td = src; lc = u0 + T[0] * (u1 + T[1] * u2);
            return 13;
        }
        {
            int v[3] = { u0, u1, u2 }, rel = 0, mul = 1;
            bool near = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (per[a]) { if (2 * v[a] > N[a]) v[a] -= N[a]; else if (2 * v[a] < -N[a]) v[a] += N[a]; }
                near = near && v[a] >= -mext[a] && v[a] < te[a] + mext[a];
                rel += (v[a] < 0 ? 0 : v[a] >= te[a] ? 2 : 1) * mul; mul *= 3;
            }
            if (near) { td = -1; lc = 0; return rel; }
        }
        int t[3] = { dT[0].div(i0), dT[1].div(i1), (D == 3) ? dT[2].div(i2) : 0 };
        td = t[0] + nt[0] * (t[1] + nt[1] * t[2]); lc = 0;
        return classify(s, t);
    }
    // class of destination tile t seen from source tile s: 0..26 = neighbour (dz+1)*9 + (dy+1)*3 + (dx+1), 27 = far
    __device__ __forceinline__ int classify(const int s[3], const int t[3]) const {
        int rel = 0, mul = 1;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int dlt = t[a] - s[a];
            if (per[a]) { if (2 * dlt > nt[a]) dlt -= nt[a]; else if (2 * dlt < -nt[a]) dlt += nt[a]; }
            if (dlt < -1 || dlt > 1) return 27;
            rel += (dlt + 1) * mul; mul *= 3;
        }
        return rel;
    }
    __device__ __forceinline__ int dest_tile(const int s[3], int rel) const {      // -1 if the neighbour does not exist
        int t[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int dlt = rel % 3 - 1; rel /= 3;
            int v = s[a] + dlt;
            if (per[a]) { if (v < 0) v += nt[a]; if (v >= nt[a]) v -= nt[a]; }
            if (v < 0 || v >= nt[a]) return -1;
            t[a] = v;
        }
        return t[0] + nt[0] * (t[1] + nt[1] * t[2]);
    }
};

__global__ void __launch_bounds__(REBIN_TPB) rebin_count_kernel(RebinGeom G, const int32_t *cell, const int32_t *tile_off,
                                                                int32_t *class_count /* [ntiles][28] */, int32_t *tile_count) {
    __shared__ int cnt[REBIN_CLASSES];
    const int src = blockIdx.x;
    int s[3]; G.tile_coords(src, s);
    const int o[3] = { s[0] * G.T[0], s[1] * G.T[1], s[2] * G.T[2] };
    const int te[3] = { min(G.T[0], G.N[0] - o[0]), min(G.T[1], G.N[1] - o[1]), G.D == 3 ? min(G.T[2], G.N[2] - o[2]) : 1 };
    if (threadIdx.x < REBIN_CLASSES) cnt[threadIdx.x] = 0;
    __syncthreads();
    const long long p0 = tile_off[src], p1 = tile_off[src + 1];
    // only the particles that LEAVE are counted (one shared atomic each, ~13 %); those that stay are the rest of the range.  Four
    // independent loads per thread and trip.
    for (long long base = p0; base < p1; base += 4 * REBIN_TPB) {
        int c4[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) { const long long p = base + r * REBIN_TPB + threadIdx.x; c4[r] = p < p1 ? cell[p] : -1; }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            if (c4[r] < 0) continue;
            int td, lc;
            const int rel = G.classify_cell(c4[r], src, s, o, te, td, lc);
            if (rel == 13) continue;
            atomicAdd(&cnt[rel], 1);
            if (rel == 27) atomicAdd(tile_count + td, 1);
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int others = 0;
        for (int r = 0; r < REBIN_CLASSES; ++r) if (r != 13) others += cnt[r];
        cnt[13] = (int)(p1 - p0) - others;
    }
    __syncthreads();
    if (threadIdx.x < REBIN_CLASSES) {
        int c = cnt[threadIdx.x];
        class_count[(long long)src * REBIN_CLASSES + threadIdx.x] = c;
        if (threadIdx.x < 27 && c > 0) { int d = G.dest_tile(s, threadIdx.x); atomicAdd(tile_count + d, c); }
    }
}

__global__ void __launch_bounds__(REBIN_TPB) rebin_scatter_kernel(RebinGeom G, const int32_t *tile_off, const int32_t *class_count,
                                                                  int32_t *cursor, PartPtrs in, PartPtrs out, int axisym,
                                                                  unsigned *tile_wmax_bits) {
    __shared__ int base_s[REBIN_CLASSES], fill[REBIN_CLASSES], dest_s[REBIN_CLASSES];
    __shared__ unsigned wmx[REBIN_CLASSES];
    const int src = blockIdx.x;
    int s[3]; G.tile_coords(src, s);
    const int o[3] = { s[0] * G.T[0], s[1] * G.T[1], s[2] * G.T[2] };
    const int te[3] = { min(G.T[0], G.N[0] - o[0]), min(G.T[1], G.N[1] - o[1]), G.D == 3 ? min(G.T[2], G.N[2] - o[2]) : 1 };
    if (threadIdx.x < REBIN_CLASSES) {
        int c = class_count[(long long)src * REBIN_CLASSES + threadIdx.x];
        int d = threadIdx.x < 27 ? G.dest_tile(s, threadIdx.x) : -1;
        dest_s[threadIdx.x] = d;
        base_s[threadIdx.x] = (threadIdx.x < 27 && c > 0) ? atomicAdd(cursor + d, c) : 0;
        fill[threadIdx.x] = 0; wmx[threadIdx.x] = 0u;
    }
    __syncthreads();
    const long long p0 = tile_off[src], p1 = tile_off[src + 1];
    const int lane = threadIdx.x & 31;
    for (long long base = p0; base < p1; base += REBIN_TPB) {
        long long p = base + threadIdx.x;
        int rel = -1, td = 0, c = 0;
        // the whole record is loaded before the destination is known (the loads do not depend on it): one round trip
        float rd[3] = {0.f, 0.f, 0.f}, ru[3] = {0.f, 0.f, 0.f}, w = 0.f, rphi = 0.f; uint8_t rtag = 1;
        if (p < p1) {
            c = in.cell[p];
            for (int a = 0; a < 3; ++a) { if (a < G.D) rd[a] = in.d[a][p]; ru[a] = in.u[a][p]; }
            w = in.w[p];
            if (axisym) rphi = in.phi[p];
            if (in.tag) rtag = in.tag[p];
            int lc; rel = G.classify_cell(c, src, s, o, te, td, lc);
        }
        // stayers (class 13): one ballot, one reservation per warp, slots in lane order; the few others one by one
        const unsigned stay = __ballot_sync(0xffffffffu, rel == 13);
        const unsigned wbits = __float_as_uint(fabsf(w));
        const unsigned wstay = __reduce_max_sync(0xffffffffu, rel == 13 ? wbits : 0u);
        int r0 = 0;
        const int leader = __ffs(stay) - 1;
        if (stay && lane == leader) { r0 = atomicAdd(&fill[13], __popc(stay)); atomicMax(&wmx[13], wstay); }
        r0 = __shfl_sync(0xffffffffu, r0, leader < 0 ? 0 : leader);
        if (rel < 0) continue;
        long long dst;
        if (rel == 13) dst = (long long)base_s[13] + r0 + __popc(stay & ((1u << lane) - 1u));
        else if (rel == 27) {
            dst = atomicAdd(cursor + td, 1);
            atomicMax(tile_wmax_bits + td, wbits);
        } else {
            dst = (long long)base_s[rel] + atomicAdd(&fill[rel], 1);
            atomicMax(&wmx[rel], wbits);
        }
        out.cell[dst] = c;
        for (int a = 0; a < 3; ++a) { if (a < G.D) out.d[a][dst] = rd[a]; out.u[a][dst] = ru[a]; }
        out.w[dst] = w;
        if (axisym) out.phi[dst] = rphi;
        if (in.tag) out.tag[dst] = rtag;
    }
    __syncthreads();
    if (threadIdx.x < 27 && dest_s[threadIdx.x] >= 0 && wmx[threadIdx.x]) atomicMax(tile_wmax_bits + dest_s[threadIdx.x], wmx[threadIdx.x]);
}


// ---------------------------------------------------------------------------------------------------------
// Re-bin with the particles that stay ORDERED BY CELL (Cartesian grids).  The tiled step's shared-memory accesses are
// conflict-free when the lanes of a warp sit in the same or neighbouring cells and cost 3-4 wavefronts each when they sit in
// unrelated cells, and writing particles straight to cell-ordered global slots costs 8x the L2 write transactions (that is
// what makes the full counting sort slow).  So the stayers of a tile (~90 %) are counting-sorted by local cell INTO SHARED
// MEMORY (staged in arrival order, then a cell histogram, a scan and a permutation, all on chip) and copied out coalesced;
// the few that leave are written one by one as in rebin_scatter_kernel.  A tile with more than `cap` stayers is placed unordered.
// ---------------------------------------------------------------------------------------------------------
constexpr int ORD_TPB = 512;
constexpr int ORD_CAP_MAX = 2560;        // staged records per CTA at most: 8 arrays x 4 B + tag + local cell + permutation = 37 B each
constexpr int ORD_REC_BYTES = 37;
constexpr int ORD_BINS = 1024;           // cells per tile, at most

__global__ void __launch_bounds__(ORD_TPB) rebin_scatter_ordered_kernel(RebinGeom G, int tcells, int cap /* staged records, multiple of 4 */,
                                                                        const int32_t *tile_off, const int32_t *class_count, int32_t *cursor,
                                                                        PartPtrs in, PartPtrs out, unsigned *tile_wmax_bits) {
    extern __shared__ __align__(16) unsigned char ord_smem[];
    int *st_cell = reinterpret_cast<int *>(ord_smem);
    float *st_f = reinterpret_cast<float *>(ord_smem) + cap;                   // [7][cap]: d0,d1,d2,u0,u1,u2,w
    unsigned short *st_lc = reinterpret_cast<unsigned short *>(ord_smem + (size_t)cap * 32);   // local cell of every staged record
    unsigned short *perm = st_lc + cap;                                         // staged slot of the k-th record in cell order
    uint8_t *st_tag = ord_smem + (size_t)cap * 36;
    __shared__ int hist[ORD_BINS], wsum[ORD_TPB / 32];
    __shared__ int base_s[REBIN_CLASSES], fill[REBIN_CLASSES], dest_s[REBIN_CLASSES];
    __shared__ unsigned wmx[REBIN_CLASSES];
    const int src = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    int s[3]; G.tile_coords(src, s);
    const int o[3] = { s[0] * G.T[0], s[1] * G.T[1], s[2] * G.T[2] };
    const int te[3] = { min(G.T[0], G.N[0] - o[0]), min(G.T[1], G.N[1] - o[1]), G.D == 3 ? min(G.T[2], G.N[2] - o[2]) : 1 };
    if (tid < REBIN_CLASSES) {
        int c = class_count[(long long)src * REBIN_CLASSES + tid];
        int d = tid < 27 ? G.dest_tile(s, tid) : -1;
        dest_s[tid] = d;
        base_s[tid] = (tid < 27 && c > 0) ? atomicAdd(cursor + d, c) : 0;
        fill[tid] = 0; wmx[tid] = 0u;
    }
    for (int k = tid; k < ORD_BINS; k += ORD_TPB) hist[k] = 0;
    __syncthreads();
    const long long p0 = tile_off[src], p1 = tile_off[src + 1];
    const int nstay = class_count[(long long)src * REBIN_CLASSES + 13];
    const bool ordered = nstay <= cap;                                          // uniform over the CTA
    // every record is read once; a stayer is staged in arrival order (ordered tile) or placed at once (too full a tile)
    for (long long base = p0; base < p1; base += ORD_TPB) {
        const long long p = base + tid;
        int rel = -1, td = 0, c = 0, lc = 0;
        float rd[3] = {0.f, 0.f, 0.f}, ru[3] = {0.f, 0.f, 0.f}, w = 0.f; uint8_t rtag = 1;
        if (p < p1) {
            c = in.cell[p];
            for (int a = 0; a < 3; ++a) { if (a < G.D) rd[a] = in.d[a][p]; ru[a] = in.u[a][p]; }
            w = in.w[p];
            if (in.tag) rtag = in.tag[p];
            rel = G.classify_cell(c, src, s, o, te, td, lc);
        }
        const unsigned wbits = __float_as_uint(fabsf(w));
        const unsigned stay = __ballot_sync(0xffffffffu, rel == 13);
        const unsigned wstay = __reduce_max_sync(0xffffffffu, rel == 13 ? wbits : 0u);
        int r0 = 0;
        const int leader = __ffs(stay) - 1;
        if (stay && lane == leader) { r0 = atomicAdd(&fill[13], __popc(stay)); atomicMax(&wmx[13], wstay); }
        r0 = __shfl_sync(0xffffffffu, r0, leader < 0 ? 0 : leader);
        if (rel < 0) continue;
        const int mine = r0 + __popc(stay & ((1u << lane) - 1u));              // stayers: slot in arrival order
        if (rel == 13 && ordered) {
            st_cell[mine] = c;
            for (int a = 0; a < 3; ++a) { st_f[a * cap + mine] = rd[a]; st_f[(3 + a) * cap + mine] = ru[a]; }
            st_f[6 * cap + mine] = w;
            st_tag[mine] = rtag;
            st_lc[mine] = (unsigned short)lc;
            atomicAdd(&hist[lc], 1);
            continue;
        }
        long long dst;
        if (rel == 13) dst = (long long)base_s[13] + mine;
        else if (rel == 27) { dst = atomicAdd(cursor + td, 1); atomicMax(tile_wmax_bits + td, wbits); }
        else { dst = (long long)base_s[rel] + atomicAdd(&fill[rel], 1); atomicMax(&wmx[rel], wbits); }
        out.cell[dst] = c;
        for (int a = 0; a < 3; ++a) { if (a < G.D) out.d[a][dst] = rd[a]; out.u[a][dst] = ru[a]; }
        out.w[dst] = w;
        if (in.tag) out.tag[dst] = rtag;
    }
    __syncthreads();
    if (ordered) {
        // exclusive scan of the cell histogram (ORD_BINS / ORD_TPB consecutive bins per thread), permutation, coalesced
        // copy-out in cell order
        constexpr int BPT = ORD_BINS / ORD_TPB;
        int hb[BPT], x = 0;
#pragma unroll
        for (int j = 0; j < BPT; ++j) { int b = BPT * tid + j; hb[j] = b < tcells ? hist[b] : 0; x += hb[j]; }
        const int mysum = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) wsum[tid >> 5] = x;
        __syncthreads();
        if (tid < 32) {
            int v = tid < ORD_TPB / 32 ? wsum[tid] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += y; }
            if (tid < ORD_TPB / 32) wsum[tid] = v;
        }
        __syncthreads();
        int excl = x - mysum + ((tid >> 5) ? wsum[(tid >> 5) - 1] : 0);
#pragma unroll
        for (int j = 0; j < BPT; ++j) { int b = BPT * tid + j; if (b < tcells) hist[b] = excl; excl += hb[j]; }
        __syncthreads();
        for (int k = tid; k < nstay; k += ORD_TPB) perm[atomicAdd(&hist[st_lc[k]], 1)] = (unsigned short)k;
        __syncthreads();
        const long long b13 = base_s[13];
        for (int k = tid; k < nstay; k += ORD_TPB) {
            const int q = perm[k];
            out.cell[b13 + k] = st_cell[q];
            for (int a = 0; a < 3; ++a) { if (a < G.D) out.d[a][b13 + k] = st_f[a * cap + q]; out.u[a][b13 + k] = st_f[(3 + a) * cap + q]; }
            out.w[b13 + k] = st_f[6 * cap + q];
            if (in.tag) out.tag[b13 + k] = st_tag[q];
        }
    }
    if (tid < 27 && dest_s[tid] >= 0 && wmx[tid]) atomicMax(tile_wmax_bits + dest_s[tid], wmx[tid]);
}

}  // namespace ent
