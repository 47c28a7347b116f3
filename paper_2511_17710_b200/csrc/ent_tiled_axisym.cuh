// ent_tiled_axisym.cuh -- tiled fused step for the axisymmetric grids (SPH, QSPH), sm_100a.
// Same structure as ent_tiled.cuh (TMA-staged E,B box, fixed-point shared-memory J tile, TMA reduce-add flush, one particle
// per thread and iteration); the per-particle arithmetic is the one of ent_particle.cuh (fp64 coordinate maps, fp32 fields,
// Boris and deposit), with the gather reading the box and the deposit writing the tile.  Boundaries: ABSORB in x1, AXIS in x2
// (no periodic wrap), so a particle is local iff its cell lies within one cell of the tile.
#pragma once
#include "ent_tiled.cuh"

namespace ent {

// a contribution that does not fit the tile's fixed-point range goes straight to the global array (J^3 = q w v^phi / (r sin theta)
// is unbounded towards the axis, reading G8)
__device__ __noinline__ void global_add(const CarryCtx &c, int comp, int off, float v) {
    int bx = off % c.JX, r = off / c.JX, by = r % c.JY, bz = r / c.JY;
    long long idx = c.gbase + bx + (long long)c.P0 * by + (long long)c.P01 * bz;
    red_global_f32(c.J[comp] + idx, v);
    atomicAdd(c.carries + 1, 1ULL);                          // counters[5]: contributions too large for the tile's fixed-point range
}
// node factors of the metric staged per tile in shared memory (ent_dev.cuh sphf_of_code): x1 nodes o1 - 1 .. o1 + TX + 2,
// x2 nodes o2 - 1 .. o2 + TY + 2
struct TileGeo {
    const float *gx; const NodeY *gy; int o1, o2;
    __device__ __forceinline__ float x(int i) const { return gx[i - o1 + 1]; }
    __device__ __forceinline__ NodeY y(int j) const { return gy[j - o2 + 1]; }
};
struct TileAcc {                         // Acc of deposit_particle_at: fixed-point add into the shared J tile
    int *sJ; const CarryCtx *cc; float Sc;
    __device__ __forceinline__ void add(int comp, long long idx, float v) const {
        float sv = v * Sc;
        if (fabsf(sv) < 1.0e9f) acc_fixed(sJ, *cc, comp, (int)idx, sv);
        else if (sv == sv) global_add(*cc, comp, (int)idx, v);
    }
    // four contributions: if all fit the fixed-point range (the rule), the four atomics are issued together and one conservative
    // test covers their carries (|old| >= 2^30 somewhere; a contribution is below 2^30 in magnitude); else one by one
    __device__ __forceinline__ void add4(int c0, long long i0, float v0, int c1, long long i1, float v1,
                                         int c2, long long i2, float v2, int c3, long long i3, float v3) const {
        const float s0 = v0 * Sc, s1 = v1 * Sc, s2 = v2 * Sc, s3 = v3 * Sc;
        if (fmaxf(fmaxf(fabsf(s0), fabsf(s1)), fmaxf(fabsf(s2), fabsf(s3))) < 1.0e9f) {       // false for NaN as well
            const int JNP = cc->JNP;
            const int w0 = fixed_rn(s0), w1 = fixed_rn(s1), w2 = fixed_rn(s2), w3 = fixed_rn(s3);
            const int a0 = atomicAdd(sJ + c0 * JNP + (int)i0, w0), a1 = atomicAdd(sJ + c1 * JNP + (int)i1, w1),
                      a2 = atomicAdd(sJ + c2 * JNP + (int)i2, w2), a3 = atomicAdd(sJ + c3 * JNP + (int)i3, w3);
            if ((int)((((unsigned)a0 + 0x40000000u) | ((unsigned)a1 + 0x40000000u)) | (((unsigned)a2 + 0x40000000u) | ((unsigned)a3 + 0x40000000u))) < 0) {
                const int n0 = a0 + w0, n1 = a1 + w1, n2 = a2 + w2, n3 = a3 + w3;
                if (((a0 ^ n0) & (w0 ^ n0)) < 0) carry_fix(*cc, c0, (int)i0, w0 > 0);
                if (((a1 ^ n1) & (w1 ^ n1)) < 0) carry_fix(*cc, c1, (int)i1, w1 > 0);
                if (((a2 ^ n2) & (w2 ^ n2)) < 0) carry_fix(*cc, c2, (int)i2, w2 > 0);
                if (((a3 ^ n3) & (w3 ^ n3)) < 0) carry_fix(*cc, c3, (int)i3, w3 > 0);
            }
        } else { add(c0, i0, v0); add(c1, i1, v1); add(c2, i2, v2); add(c3, i3, v3); }
    }
};

template <int KIND>
__device__ __noinline__ void stray_step_axisym(const TiledArgs &A, long long p) {
    const GridDev &g = A.g;
    int i[3], i0[3], di[3]; float d[3] = {0.f, 0.f, 0.f}, a[3], u[3];
    unpack_cell<2>(g, A.P.cell[p], i);
    d[0] = A.P.d[0][p]; d[1] = A.P.d[1][p];
#pragma unroll
    for (int k = 0; k < 3; ++k) { u[k] = A.P.u[k][p]; a[k] = d[k]; i0[k] = i[k]; }
    float phi = A.P.phi[p];
    const float phi0 = phi;
    GlobalFieldLoader ld{A.F.c};
    bool alive = true;
    push_particle<2, KIND>(g, ld, i, d, phi, u, A.eps, A.dt, di, alive);
    A.P.cell[p] = pack_cell<2>(g, i);
    A.P.d[0][p] = d[0]; A.P.d[1][p] = d[1];
#pragma unroll
    for (int k = 0; k < 3; ++k) A.P.u[k][p] = u[k];
    A.P.phi[p] = phi;
    atomicAdd(A.counters + 1, 1ULL);
    if (!alive) { A.P.tag[p] = 0; return; }
    if (di[0] < -1 || di[0] > 1 || di[1] < -1 || di[1] > 1) { atomicAdd(A.counters + 0, 1ULL); return; }
    GlobalAcc acc{A.J.c};
    deposit_particle<2, KIND>(g, acc, i0, a, di, d, phi0, phi, u, A.q * A.P.w[p], A.inv_dt);
}

#ifndef ENT_AXISYM_MINB
#define ENT_AXISYM_MINB 4
#endif
// On these grids the inner cells hold hundreds of particles (density ~ r^-2), so the 32 lanes of a warp usually sit in ONE cell and
// every shared atomic serialises 32 ways on one address (measured on C5: 16 wavefronts per ATOMS, 84 % of all shared-memory
// wavefronts).  The J tile is therefore kept in AXI_NCOPY copies, lane L adding into copy L mod AXI_NCOPY; the copies are one word
// apart modulo the 32 banks, so the same node in different copies sits in different banks: a one-cell warp costs
// 32 / AXI_NCOPY wavefronts per ATOMS.  The copies are summed in the flush pass.  Measured on C5 (ms per species; copies x CTAs/SM):
// 1x4 6.30, 2x4 6.21, 4x4 6.07, 4x3 6.65, 8x3 6.84 -- shared-memory wavefronts fall 1295 M -> 553 M with 8 copies, but the kernel is
// then bound by instruction issue, so the fourth resident CTA is worth more than the last copies.  (Grouping equal-cell lanes with
// __match_any_sync + __reduce_add_sync was measured 1.6 x SLOWER than no grouping at all: the per-group masks serialise.)
#ifndef ENT_AXI_NCOPY
#define ENT_AXI_NCOPY 4
#endif
constexpr int AXI_NCOPY = ENT_AXI_NCOPY;
template <int TX, int TY> struct AxiGeom {
    using G = TileGeom<2, TX, TY, 1>;
    static constexpr int CSTRIDE = 3 * G::JNP + 1;                        // words between copies: 1 modulo 32
    static constexpr int JWORDS = ((AXI_NCOPY * CSTRIDE + 3) / 4) * 4;
    static constexpr int SMEM_BYTES = (6 * G::FNP + JWORDS) * 4;
};
template <int KIND, int TX, int TY>
__global__ void __launch_bounds__(TILED_TPB, ENT_AXISYM_MINB)
step_tiled_axisym_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ TiledArgs A) {
    using G = TileGeom<2, TX, TY, 1>;
    using X = AxiGeom<TX, TY>;
    extern __shared__ __align__(128) float smem[];
    float *sF = smem;
    int *sJ = reinterpret_cast<int *>(smem + 6 * G::FNP);          // AXI_NCOPY copies of [3][JNP], X::CSTRIDE words apart
    __shared__ uint64_t bar;
    __shared__ CarryCtx s_cc;
    __shared__ float s_gx[TX + 4];
    __shared__ NodeY s_gy[TY + 4];
    __shared__ float s_h[6];
    const GridDev &g = A.g;
    const int tid = threadIdx.x;
    const int tile = find_tile(A.chunk_off, A.ntiles, blockIdx.x);
    if (tile < 0) return;
    const int o0 = (tile % g.nt[0]) * TX, o1 = (tile / g.nt[0]) * TY;
    if (tid < TX + 4) s_gx[tid] = node_x<KIND>(g, o0 - 1 + tid);                 // metric factors at the nodes of this tile, fp64 -> fp32
    else if (tid >= 32 && tid < 32 + TY + 4) s_gy[tid - 32] = node_y<KIND>(g, o1 - 1 + tid - 32);

    if (tid == 0) {
        mbar_init(&bar, 1);
        fence_mbar_init();
        mbar_expect_tx(&bar, 6u * G::FN * 4u);
#pragma unroll
        for (int c = 0; c < 6; ++c) tma_load_box<2>(sF + c * G::FNP, &maps.F[c], &bar, o0, o1, 0);
    }
    for (int k = tid; k < X::JWORDS / 4; k += TILED_TPB) reinterpret_cast<int4 *>(sJ)[k] = make_int4(0, 0, 0, 0);

    long long p0 = A.key_off[tile], p1 = A.key_off[tile + 1];
    p0 += (long long)(blockIdx.x - A.chunk_off[tile]) * A.chunk;
    if (p1 > p0 + A.chunk) p1 = p0 + A.chunk;
    float Sc, invSc;
    {   // fixed-point scale of this CTA's J tile.  A contribution is q w / dt * D * weight with |D_a| <= dt / sqrt(h_aa) (|v| < 1), i.e.
        // at most |q| wmax / min sqrt(h_aa) over the tile (x 13/12); bounding |D| by 1 instead would waste ~10 bits on the
        // log-r grids, where a particle moves ~1e-3 cells per step.  J^3 = q w v^phi / sqrt(h33) is of the same size except next
        // to the axis, where the contributions that do not fit go to the global array (TileAcc).
        const float wm = A.tile_wmax[tile];
        if (tid >= 64 && tid < 70) {                                     // six sample points of the tile, one thread each (fp64 maps)
            const int c = tid - 64;
            const double x1a = fmax(0.0, (double)o0 - 1.0), x1b = fmin((double)g.N[0], (double)(o0 + TX) + 1.0);
            const double x2a = fmax(0.0, (double)o1 - 1.0), x2b = fmin((double)g.N[1], (double)(o1 + TY) + 1.0);
            Sph sp = sph_of_code<KIND>(g, (c & 1) ? x1b : x1a, c < 2 ? x2a : (c < 4 ? x2b : 0.5 * (x2a + x2b)));
            s_h[c] = (float)fmin(sp.sh1, sp.sh2);
        }
        __syncthreads();
        const float hmin = fminf(fminf(fminf(s_h[0], s_h[1]), fminf(s_h[2], s_h[3])), fminf(s_h[4], s_h[5]));
        float rate = fminf(A.inv_dt, 1.25f / hmin);                      // 1/dt: |D| <= 1 always
        float qmax = fabsf(A.q) * wm * fmaxf(rate, 1e-30f) * 1.0834f;
        Sc = (qmax > 0.f && qmax < 1e37f) ? 67100000.0f / qmax : 0.f;       // 26 bits: weights vary strongly inside a tile of a coarse grid
        if (!(Sc > 1e-30f && Sc < 1e30f)) Sc = 0.f;
        invSc = Sc > 0.f ? 1.0f / Sc : 0.f;
    }
    if (tid == 0) {
        s_cc.J = A.J.c; s_cc.P0 = g.P[0]; s_cc.P01 = g.P[0] * g.P[1]; s_cc.unit = 4294967296.0f * invSc;
        s_cc.JX = G::JX; s_cc.JY = G::JY; s_cc.JNP = G::JNP; s_cc.carries = A.counters + 4;
        s_cc.gbase = (long long)o0 + (long long)g.P[0] * o1;
    }
    __syncthreads();
    const TileAcc acc{sJ + (tid & (AXI_NCOPY - 1)) * X::CSTRIDE, &s_cc, Sc};
    const TileGeo geo{s_gx, s_gy, o0, o1};
    const float wguard = Sc > 0.f ? 60.0f * A.tile_wmax[tile] : -1.0f;
    bool waited = false;

    for (long long p = p0 + tid; p < p1; p += TILED_TPB) {
        const int cell = A.P.cell[p];
        float d[3] = { A.P.d[0][p], A.P.d[1][p], 0.f };
        float u[3] = { A.P.u[0][p], A.P.u[1][p], A.P.u[2][p] };
        float phi = A.P.phi[p];
        const float wgt = A.P.w[p];
        const bool live = A.P.tag[p] != 0;
        if (!waited) { mbar_wait(&bar, 0); waited = true; }
        if (!live) continue;
        int i[3];
        i[1] = A.divN0.div(cell); i[0] = cell - i[1] * g.N[0]; i[2] = 0;
        const int b0 = i[0] - o0 + 2, b1 = i[1] - o1 + 2;
        const bool local = ((unsigned)(b0 - 1) < (unsigned)(TX + 2)) & ((unsigned)(b1 - 1) < (unsigned)(TY + 2)) & (fabsf(wgt) <= wguard);
        if (!local) { defer_stray(A, p, [&] { stray_step_axisym<KIND>(A, p); }); continue; }
        // gather from the box: the box is addressed like a padded array of extents FX x FY whose "active" origin is the tile
        // origin, so the cell's coordinates in it are (b - 2)
        const int ib[3] = { b0 - NG, b1 - NG, 0 }, bb[3] = { b0, b1, 0 };
        float EB[6];
        gather_box<2, G::FX, G::FY, G::FNP>(sF, bb, d, EB);        // the gather of ent_tiled.cuh (packed pairs), same arithmetic as ent_dev.cuh
        const int i0[3] = { i[0], i[1], 0 };
        const float a[3] = { d[0], d[1], 0.f };
        const float phi0 = phi;
        int di[3]; bool alive = true;
        push_from_fields_geo<2, KIND>(g, geo, EB, i, d, phi, u, A.eps, A.dt, di, alive);
        A.P.cell[p] = i[0] + g.N[0] * i[1];
        A.P.d[0][p] = d[0]; A.P.d[1][p] = d[1];
        A.P.u[0][p] = u[0]; A.P.u[1][p] = u[1]; A.P.u[2][p] = u[2];
        A.P.phi[p] = phi;
        if (!alive) { A.P.tag[p] = 0; continue; }
        if (di[0] < -1 || di[0] > 1 || di[1] < -1 || di[1] > 1) { atomicAdd(A.counters + 0, 1ULL); continue; }
        GridDev gj = g; gj.P[0] = G::JX; gj.P[1] = G::JY; gj.P[2] = 1;
        deposit_particle_at<2, KIND>(g, geo, acc, i0, a, di, d, phi0, phi, u, A.q * wgt, A.inv_dt, gj, ib);
    }
    if (!waited) mbar_wait(&bar, 0);
    __syncthreads();
    for (int k = tid; k < 3 * G::JNP; k += TILED_TPB) {            // sum of the copies, fixed point -> fp32, into copy 0 (dense: the TMA box)
        long long v = sJ[k];                                       // each copy may hold up to +-2^31: the sum needs more than 32 bits
#pragma unroll
        for (int c = 1; c < AXI_NCOPY; ++c) v += sJ[k + c * X::CSTRIDE];
        reinterpret_cast<float *>(sJ)[k] = (float)v * invSc;
    }
    fence_proxy_async_smem();
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) tma_reduce_add_box<2>(&maps.J[c], sJ + c * G::JNP, o0, o1, 0);
        tma_commit();
        tma_wait_read0();
    }
}

template <int KIND>
__global__ void __launch_bounds__(256) stray_axisym_kernel(const __grid_constant__ TiledArgs A) {
    const unsigned long long cnt = A.counters[2];
    const long long m = (long long)cnt < A.stray_cap ? (long long)cnt : A.stray_cap;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (long long)gridDim.x * blockDim.x)
        stray_step_axisym<KIND>(A, A.stray_list[k]);
}

template <int D> inline void launch_strays(const TiledArgs &A, cudaStream_t stream) {
    const int grid = 148 * 4;
    if (A.g.kind == ENT_CART) stray_kernel<D><<<grid, 256, 0, stream>>>(A);
    else if (A.g.kind == ENT_SPH) stray_axisym_kernel<ENT_SPH><<<grid, 256, 0, stream>>>(A);
    else stray_axisym_kernel<ENT_QSPH><<<grid, 256, 0, stream>>>(A);
}

}  // namespace ent
