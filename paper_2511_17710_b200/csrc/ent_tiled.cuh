// ent_tiled.cuh -- tiled fused step for the Cartesian grids (sub-steps 3-8), sm_100a.
//
// A CTA works on one tile of TX x TY x TZ cells (a tile with more than tile_chunk_for(n) particles is shared by several CTAs: work
// list built by ent_sort).  The block handed to ent_step is the one ent_sort produced, so the particles of a tile are one
// contiguous range of the SoA arrays (tile-major key, ent.h).
//   * E,B: the tile's box of the six padded planar arrays, [o-2, o+T+2) per dimension, lands in shared memory by
//     TMA (cp.async.bulk.tensor, one box per component, one mbarrier);
//   * particles: one per thread and iteration, consecutive lanes on consecutive particles (fully coalesced lines), the
//     next record requested before the current one is advanced;
//   * deposit: fixed-point adds into a shared-memory tile of J covering nodes [o-2, o+T+3), then ONE flush per CTA with
//     the TMA reduce-add (cp.reduce.async.bulk.tensor .add.f32) into the un-wrapped padded J arrays;
//   * a particle whose cell has drifted more than one cell out of the tile since the sort goes to a list for stray_kernel
//     (global gathers, global atomics); one whose deposit could leave the padded array deposits through global atomics.
// Arithmetic per particle is the same as ent_particle.cuh (same Boris, same split_offset, same segment weights); a
// particle that crosses no face deposits its straight move as one segment (the two half segments of P:575 are
// collinear then, and the weights (1-W_a)(1-W_b) + D_a D_b/12 are the exact line integral, so the sum is identical).
#pragma once
#include <cuda.h>
#include "ent_kernels.cuh"

namespace ent {

// ---------------------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier + TMA (cp.async.bulk.tensor), sm_90+/sm_100a
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
template <int D>
__device__ __forceinline__ void tma_load_box(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2) {
    if (D == 3)
        asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                     ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
    else
        asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                     ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
template <int D>
__device__ __forceinline__ void tma_reduce_add_box(const CUtensorMap *map, const void *src, int c0, int c1, int c2) {
    if (D == 3)
        asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4}], [%1];"
                     ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2) : "memory");
    else
        asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3}], [%1];"
                     ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// ---- packed fp32 pairs (FFMA2 / FADD2 on sm_100a): two independent lerps per instruction ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
// a + f * (b - a), per half (the same FADD, FFMA sequence as the scalar gather of ent_dev.cuh: identical results)
__device__ __forceinline__ f32x2 lerp2(f32x2 a, f32x2 b, f32x2 f) {
    f32x2 d, r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(b), "l"(a));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f), "l"(d), "l"(a));
    return r;
}

// S1 gather of the six components from a shared-memory box (stencil and arithmetic of ent_dev.cuh gather): b = cell in
// box coordinates, d = in-cell offsets.  The seven lerps of a component run as packed pairs (z and z+1 planes together in 3D).
template <int D, int FX, int FY, int FNP>
__device__ __forceinline__ void gather_box(const float *sF, const int b[3], const float d[3], float EBv[6]) {
    int xs[2], ys[2], zs[2]; float fx[2], fy[2], fz[2];              // [0] node-centred, [1] half-shifted
    { bool lo = d[0] < 0.5f; xs[0] = b[0]; xs[1] = lo ? b[0] - 1 : b[0]; fx[0] = d[0]; fx[1] = lo ? d[0] + 0.5f : d[0] - 0.5f; }
    { bool lo = d[1] < 0.5f; ys[0] = b[1] * FX; ys[1] = lo ? ys[0] - FX : ys[0]; fy[0] = d[1]; fy[1] = lo ? d[1] + 0.5f : d[1] - 0.5f; }
    if (D == 3) { bool lo = d[2] < 0.5f; zs[0] = b[2] * (FX * FY); zs[1] = lo ? zs[0] - FX * FY : zs[0]; fz[0] = d[2]; fz[1] = lo ? d[2] + 0.5f : d[2] - 0.5f; }
    else { zs[0] = zs[1] = 0; fz[0] = fz[1] = 0.f; }
    const f32x2 FX2[2] = { pk2(fx[0], fx[0]), pk2(fx[1], fx[1]) }, FY2[2] = { pk2(fy[0], fy[0]), pk2(fy[1], fy[1]) };
    const int ST[6][3] = { {1,0,0}, {0,1,0}, {0,0,1}, {0,1,1}, {1,0,1}, {1,1,0} };
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float *Fc = sF + c * FNP + (xs[ST[c][0]] + ys[ST[c][1]] + zs[ST[c][2]]);
        if (D == 3) {
            const float *Fh = Fc + FX * FY;
            const f32x2 P00 = pk2(Fc[0], Fh[0]), P10 = pk2(Fc[1], Fh[1]), P01 = pk2(Fc[FX], Fh[FX]), P11 = pk2(Fc[FX + 1], Fh[FX + 1]);
            const f32x2 L0 = lerp2(P00, P10, FX2[ST[c][0]]), L1 = lerp2(P01, P11, FX2[ST[c][0]]);
            float lo, hi;
            upk2(lerp2(L0, L1, FY2[ST[c][1]]), lo, hi);
            EBv[c] = lo + fz[ST[c][2]] * (hi - lo);
        } else {
            const f32x2 P0 = pk2(Fc[0], Fc[FX]), P1 = pk2(Fc[1], Fc[FX + 1]);
            float l0, l1;
            upk2(lerp2(P0, P1, FX2[ST[c][0]]), l0, l1);
            EBv[c] = l0 + fy[ST[c][1]] * (l1 - l0);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// geometry of a tile in shared memory (compile time)
// ---------------------------------------------------------------------------------------------------------
template <int D, int TX, int TY, int TZ>
struct TileGeom {
    static constexpr int FX = TX + 4, FY = TY + 4, FZ = (D == 3) ? TZ + 4 : 1;                 // E,B box: cells [o-2, o+T+2)
    static constexpr int JX = ((TX + 5 + 3) / 4) * 4, JY = TY + 5, JZ = (D == 3) ? TZ + 5 : 1; // J box: nodes [o-2, o+T+3), x padded to 16 B
    static constexpr int FN = FX * FY * FZ, JN = JX * JY * JZ;
    static constexpr int FNP = ((FN + 31) / 32) * 32, JNP = ((JN + 31) / 32) * 32;              // 128-byte aligned component slabs
    static constexpr int SMEM_BYTES = (6 * FNP + 3 * JNP) * 4;
    static constexpr int TCELLS = TX * TY * TZ;
};

struct TileMaps { CUtensorMap F[6]; CUtensorMap J[3]; };

struct TiledArgs {
    GridDev g;
    FieldPtrs F;
    CurrentPtrs J;
    PartPtrs P;
    const int32_t *key_off;       // tile offsets: tile t owns particles [key_off[t], key_off[t+1]) (ent_sort)
    const float *tile_wmax;       // max |w| over the particles of each tile (ent_sort)
    const int32_t *chunk_off;     // work list: tile t is processed by CTAs [chunk_off[t], chunk_off[t+1]), tile_chunk_for(n) particles each
    int ntiles;
    long long n;
    float eps, dt, q, inv_dt;
    float cdt[3];                 // dt / dx_d
    // second species of a pair launch (ent_step_pair): same tile geometry, its own block, layout, charge and q/m
    int chunk;                    // particles per CTA of the work list (tile_chunk_for(n))
    int nsp;                      // 1, or 2: one CTA per tile advances both blocks through one E,B box and one J tile
    PartPtrs P2; const int32_t *key_off2; const float *tile_wmax2; float eps2, q2;
    unsigned long long *counters; // [0] bad moves, [1] strays, [2] length of stray_list, [4] carries of the fixed-point J tile
    int32_t *stray_list; long long stray_cap;   // particles left to stray_kernel (all lanes busy there instead of one per warp here)
    MagicDiv divN0, divN01;
};

// the global path for one particle (same code as step_untiled_kernel); kept out of line so that the tile loop stays lean
template <int D>
__device__ __noinline__ void stray_step(const TiledArgs &A, long long p, int sp = 0) {
    const GridDev &g = A.g;
    const PartPtrs &P = sp ? A.P2 : A.P;
    const float q = sp ? A.q2 : A.q, eps = sp ? A.eps2 : A.eps;
    int i[3], i0[3], di[3]; float d[3] = {0.f, 0.f, 0.f}, a[3], u[3], phi = 0.f;
    unpack_cell<D>(g, P.cell[p], i);
#pragma unroll
    for (int k = 0; k < D; ++k) d[k] = P.d[k][p];
#pragma unroll
    for (int k = 0; k < 3; ++k) { u[k] = P.u[k][p]; a[k] = d[k]; i0[k] = i[k]; }
    GlobalFieldLoader ld{A.F.c};
    bool alive = true;
    push_particle<D, ENT_CART>(g, ld, i, d, phi, u, eps, A.dt, di, alive);
    P.cell[p] = pack_cell<D>(g, i);
#pragma unroll
    for (int k = 0; k < D; ++k) P.d[k][p] = d[k];
#pragma unroll
    for (int k = 0; k < 3; ++k) P.u[k][p] = u[k];
    atomicAdd(A.counters + 1, 1ULL);
    if (!alive) { P.tag[p] = 0; return; }
    bool bad = false;
#pragma unroll
    for (int k = 0; k < D; ++k) bad |= (di[k] < -1 || di[k] > 1);
    if (bad) { atomicAdd(A.counters + 0, 1ULL); return; }
    GlobalAcc acc{A.J.c};
    deposit_particle<D, ENT_CART>(g, acc, i0, a, di, d, 0.f, 0.f, u, q * P.w[p], A.inv_dt);
}

// ---------------------------------------------------------------------------------------------------------
// Shared-memory accumulation of J.  fp32 atomicAdd on shared memory is a compare-and-swap loop on sm_100a
// (SASS: LDS + FADD + ATOMS.CAST.SPIN + branch, several passes under contention); 32-bit integer add is native
// (ATOMS.ADD).  The J tile is therefore accumulated in fixed point: value * 2^k rounded to nearest, k chosen per tile
// from the largest |q w|/dt of the tile's particles so that one contribution uses at most 24 bits.  Integer sums are
// exact and order-independent.  A signed wrap of the 32-bit accumulator (|J_node| * 2^k >= 2^31: hundreds of
// particles' worth of current on one node) is detected from the value the atomic returns and carried straight into
// the global array as +-2^32 / 2^k, so the sum stays exact for any input.
// ---------------------------------------------------------------------------------------------------------
constexpr float FIXED_ONE = 16777000.0f;     // the largest contribution of a tile in fixed-point units (just below 2^24)
__device__ __forceinline__ int fixed_rn(float v) { return __float2int_rn(v); }
struct CarryCtx { float *const *J; long long gbase; int P0, P01; float unit; int JX, JY, JNP; unsigned long long *carries; };

__device__ __noinline__ void carry_fix(const CarryCtx &c, int comp, int off, int positive) {
    int bx = off % c.JX, r = off / c.JX, by = r % c.JY, bz = r / c.JY;
    long long idx = c.gbase + bx + (long long)c.P0 * by + (long long)c.P01 * bz;
    red_global_f32(c.J[comp] + idx, positive ? c.unit : -c.unit);
    atomicAdd(c.carries, 1ULL);
}
__device__ __forceinline__ void acc_fixed(int *sJ, const CarryCtx &cc, int comp, int off, float scaled) {
    int v = fixed_rn(scaled);
    int old = atomicAdd(sJ + comp * cc.JNP + off, v);
    if ((int)((unsigned)old + 0x40000000u) < 0) {     // |old| >= 2^30: only then can |v| < 2^30 wrap the accumulator (conservative, cheap;
                                                      // unsigned: a signed overflow here would be undefined and was optimised away)
        int nw = old + v;
        if (((old ^ nw) & (v ^ nw)) < 0) carry_fix(cc, comp, off, v > 0);
    }
}
// four contributions of one component: all four atomics are issued before the first returned value is looked at.  One cheap,
// conservative test covers the four carries: a contribution is below 2^25 in magnitude, so an accumulator can only wrap if its
// old value is outside [-2^30, 2^30); only then the exact per-add test runs.
__device__ __forceinline__ void acc_fixed4(int *sJ, const CarryCtx &cc, int comp, int o0, int o1, int o2, int o3,
                                           float s0, float s1, float s2, float s3) {
    int *Jc = sJ + comp * cc.JNP;
    int v0 = fixed_rn(s0), v1 = fixed_rn(s1), v2 = fixed_rn(s2), v3 = fixed_rn(s3);
    int a0 = atomicAdd(Jc + o0, v0), a1 = atomicAdd(Jc + o1, v1), a2 = atomicAdd(Jc + o2, v2), a3 = atomicAdd(Jc + o3, v3);
    if ((int)((((unsigned)a0 + 0x40000000u) | ((unsigned)a1 + 0x40000000u)) | (((unsigned)a2 + 0x40000000u) | ((unsigned)a3 + 0x40000000u))) < 0) {
        int n0 = a0 + v0, n1 = a1 + v1, n2 = a2 + v2, n3 = a3 + v3;
        if (((a0 ^ n0) & (v0 ^ n0)) < 0) carry_fix(cc, comp, o0, v0 > 0);
        if (((a1 ^ n1) & (v1 ^ n1)) < 0) carry_fix(cc, comp, o1, v1 > 0);
        if (((a2 ^ n2) & (v2 ^ n2)) < 0) carry_fix(cc, comp, o2, v2 > 0);
        if (((a3 ^ n3) & (v3 ^ n3)) < 0) carry_fix(cc, comp, o3, v3 > 0);
    }
}
// One straight segment s -> e (cell-local coordinates) of the zig-zag deposit into the fixed-point J tile, element `base` = the
// segment's cell (Eq. 6).  3D: per component the four products Q D_c [w(W_a) w(W_b) +- D_a D_b / 12] (reading G7), written
// as v11 = QD (W_a W_b + D_a D_b / 12), v10 = QD W_a - v11, v01 = QD W_b - v11, v00 = QD - QD W_a - v01.  2D: in-plane components
// with linear weights and the out-of-plane rate hv (G8) with bilinear weights.
template <int D, class G>
__device__ __forceinline__ void tile_segment(int *sJ, const CarryCtx &cc, int base, const float s[3], const float e[3], float Q, float hv) {
    float Dv[3], W[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { Dv[a] = e[a] - s[a]; W[a] = 0.5f * (e[a] + s[a]); }
    if (D == 3) {
        // the twelve adds of the segment are all issued before the first returned value is looked at; one conservative test
        // (|old| >= 2^30 somewhere) covers the twelve carries, the exact per-add test runs only then
        constexpr int st[3] = { 1, G::JX, G::JX * G::JY };
        int v[12], old[12];
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            const int a = (comp + 1) % 3, bb = (comp + 2) % 3;
            const float QD = Q * Dv[comp];
            const float ta = QD * W[a], tb = QD * W[bb];
            const float v11 = fmaf(ta, W[bb], QD * (Dv[a] * Dv[bb] * (1.0f / 12.0f)));
            const float v10 = ta - v11, v01 = tb - v11, v00 = (QD - ta) - v01;
            v[4 * comp] = fixed_rn(v00); v[4 * comp + 1] = fixed_rn(v10); v[4 * comp + 2] = fixed_rn(v01); v[4 * comp + 3] = fixed_rn(v11);
            int *Jc = sJ + comp * cc.JNP + base;
            old[4 * comp] = atomicAdd(Jc, v[4 * comp]); old[4 * comp + 1] = atomicAdd(Jc + st[a], v[4 * comp + 1]);
            old[4 * comp + 2] = atomicAdd(Jc + st[bb], v[4 * comp + 2]); old[4 * comp + 3] = atomicAdd(Jc + st[a] + st[bb], v[4 * comp + 3]);
        }
        int mx = __vimax3_s32(old[0], old[1], old[2]), mn = __vimin3_s32(old[0], old[1], old[2]);     // VIMNMX3
#pragma unroll
        for (int k = 3; k < 11; k += 2) { mx = __vimax3_s32(mx, old[k], old[k + 1]); mn = __vimin3_s32(mn, old[k], old[k + 1]); }
        mx = max(mx, old[11]); mn = min(mn, old[11]);
        if (mx >= 0x40000000 || mn < -0x40000000) {
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                const int comp = k / 4, a = (comp + 1) % 3, bb = (comp + 2) % 3;
                const int off = base + ((k & 1) ? st[a] : 0) + ((k & 2) ? st[bb] : 0);
                const int nw = old[k] + v[k];
                if (((old[k] ^ nw) & (v[k] ^ nw)) < 0) carry_fix(cc, comp, off, v[k] > 0);
            }
        }
    } else {
        const float q0 = Q * Dv[0], q1 = Q * Dv[1];
        const float h1 = hv * W[1], h0 = hv - h1;
        acc_fixed4(sJ, cc, 0, base, base + G::JX, base, base + G::JX, q0 * (1.0f - W[1]), q0 * W[1], 0.f, 0.f);
        acc_fixed4(sJ, cc, 1, base, base + 1, base, base + 1, q1 * (1.0f - W[0]), q1 * W[0], 0.f, 0.f);
        acc_fixed4(sJ, cc, 2, base, base + 1, base + G::JX, base + G::JX + 1, h0 * (1.0f - W[0]), h0 * W[0], h1 * (1.0f - W[0]), h1 * W[0]);
    }
}
// S7 for one particle: old offsets a0 in cell b (box coordinates), new offsets d in cell b + di.  The relay point of P:575 per
// dimension, r = min(min(0, di) + 1, max(max(0, di), (a0 + di + d) / 2)) in the old cell's frame (Umeda's form: the midpoint if no
// face is crossed, else the face), without branches.  3D: a particle that crosses no face deposits its move as ONE segment (the two
// half segments are collinear and the weights above are the exact line integral).  2D: always two segments (the bilinear
// out-of-plane weights of two half segments do not sum to those of the whole one).
template <int D, class G>
__device__ __forceinline__ void tile_deposit(int *sJ, const CarryCtx &cc, const int b[3], const float a0[3], const float d[3], const int di[3],
                                             float Q, float hv) {
    const bool cross = (D == 2) || (di[0] | di[1] | di[2]) != 0;
    float r[3], s2[3], e2[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (a < D) {
            const float fdi = (float)di[a], bn = fdi + d[a];
            const float rr = fminf(fminf(fdi, 0.f) + 1.0f, fmaxf(fmaxf(fdi, 0.f), 0.5f * (a0[a] + bn)));
            r[a] = cross ? rr : bn;
            s2[a] = rr - fdi; e2[a] = d[a];
        } else { r[a] = 0.f; s2[a] = 0.f; e2[a] = 0.f; }
    }
    const int base = b[0] + G::JX * (b[1] + G::JY * b[2]);
    tile_segment<D, G>(sJ, cc, base, a0, r, Q, hv);
    if (cross) tile_segment<D, G>(sJ, cc, base + di[0] + G::JX * (di[1] + G::JY * di[2]), s2, e2, Q, hv);
}

#ifndef ENT_TILED_MINB
#define ENT_TILED_MINB 3
#endif

#ifndef ENT_TILED_TPB
#define ENT_TILED_TPB 256
#endif
constexpr int TILED_TPB = ENT_TILED_TPB;
constexpr int TILE_CHUNK_MAX = 4096;          // particles per CTA: a heavy tile is shared by several CTAs, each with its own J tile
// The chunk of a block of n particles: 4096 for the large blocks (per-tile prologue and flush amortised over 16 particles per thread),
// smaller for small blocks so that the launch still fills the 148 SMs a few times over (a 64^2 grid has 16 tiles).  A function of n
// alone: the work list (ent_sort) and the launches that use it agree without carrying the value.
inline int tile_chunk_for(long long n) {
    long long c = (n / (148LL * 3 * 4) + 255) / 256 * 256;
    return (int)(c < 512 ? 512 : c > TILE_CHUNK_MAX ? TILE_CHUNK_MAX : c);
}

// work-list lookup: the tile whose chunk range contains CTA `vb` (binary search in the exclusive scan), or -1
__device__ __forceinline__ int find_tile(const int32_t *chunk_off, int ntiles, int vb) {
    if (vb < ntiles) {                        // uniform plasma: one chunk per tile, chunk_off[t] == t (two independent loads)
        int a = chunk_off[vb], b = chunk_off[vb + 1];
        if (a == vb && b == vb + 1) return vb;
    }
    if (vb >= chunk_off[ntiles]) return -1;
    int lo = 0, hi = ntiles;                  // invariant: chunk_off[lo] <= vb < chunk_off[hi]
    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (chunk_off[mid] <= vb) lo = mid; else hi = mid; }
    return lo;
}

// deposit of one particle through global atomics (ent_particle.cuh), out of line: used by the few particles of a tile that
// cannot deposit into its shared-memory J tile
template <int D, class ARGS>
__device__ __noinline__ void edge_deposit(const ARGS &A, int i0, int i1, int i2, float a0, float a1, float a2, int di0, int di1, int di2,
                                          float d0, float d1, float d2, float u0, float u1, float u2, float qw) {
    const int i[3] = { i0, i1, i2 }, di[3] = { di0, di1, di2 };
    const float a[3] = { a0, a1, a2 }, dn[3] = { d0, d1, d2 }, u[3] = { u0, u1, u2 };
    GlobalAcc acc{A.J.c};
    deposit_particle<D, ENT_CART>(A.g, acc, i, a, di, dn, 0.f, 0.f, u, qw, A.inv_dt);
}

// a particle the tile cannot take: hand it to stray_kernel through the list, or advance it right here if the list is full
template <class F>
__device__ __forceinline__ void defer_stray(const TiledArgs &A, long long p, F &&fallback) {
    unsigned long long k = atomicAdd(A.counters + 2, 1ULL);
    if ((long long)k < A.stray_cap) A.stray_list[k] = (int32_t)p; else fallback();
}

// per-CTA constants of the tile loop
template <int D>
struct TileCtx {
    const float *sF;      // [6][FNP] E,B box
    int *sJ;              // [3][JNP] fixed-point J tile
    int o[3];             // tile origin (active cell coordinates)
    float sx[3];          // sqrt(h_ii) = cell sizes
    float Sc;             // fixed-point scale of this tile
    float wguard;         // weights above this deposit through the global path (contribution would not fit 2^30)
    CarryCtx cc;
};

// One particle through sub-steps 3-8 inside a tile.  cell, d[], u[] are updated in place.
// Returns 0: advanced (write the record back), 1: taken by the global path (already written), 2: advanced and left
// through an ABSORB side (write back, tag = 0), 3: dead or not ours (untouched).
template <int D, int TX, int TY, int TZ, bool ALLPER, bool PAIR>
__device__ __forceinline__ int tile_particle(const TiledArgs &A, const TileCtx<D> &T, long long p, int &cell, float d[3], float u[3],
                                             float wgt, float q, float eps, int sp) {
    using G = TileGeom<D, TX, TY, TZ>;
    const GridDev &g = A.g;
    // ---- where is the cell relative to the tile box?  b = cell index in box coordinates (box origin = o-2)
    int i[3] = { 0, 0, 0 }, b[3];
    const int TT[3] = { TX, TY, TZ };
    bool local = true, edge = false;
    {
        if (D == 2) { i[1] = A.divN0.div(cell); i[0] = cell - i[1] * g.N[0]; i[2] = 0; }
        else { i[2] = A.divN01.div(cell); int r = cell - i[2] * (g.N[0] * g.N[1]); i[1] = A.divN0.div(r); i[0] = r - i[1] * g.N[0]; }
        b[0] = i[0] - T.o[0] + 2; b[1] = i[1] - T.o[1] + 2; b[2] = (D == 3) ? i[2] - T.o[2] + 2 : 0;
#pragma unroll
        for (int a = 0; a < D; ++a) {
            const int wrapN = (ALLPER || g.bc[a] == ENT_PERIODIC) ? g.N[a] : 0;
            b[a] += (b[a] < 1) ? wrapN : 0;
            b[a] -= (b[a] > g.N[a]) ? wrapN : 0;
            local &= (unsigned)(b[a] - 1) < (unsigned)(TT[a] + 2);           // inside the box with one cell of margin
            // un-wrapped cell N (a particle that crossed the upper periodic face since the sort): its +1 crossing would deposit
            // at node N+2, outside the padded array -> it gathers from the box but deposits through the global path
            edge |= (T.o[a] - 2 + b[a] > g.N[a] - 1);
        }
    }
    // the true old cell (needed by the global-path deposit only)
    const int iold[3] = { i[0], i[1], i[2] };
    if (!local) {
        if (PAIR) stray_step<D>(A, p, sp);         // pair launch: the stray list does not record the species
        else defer_stray(A, p, [&] { stray_step<D>(A, p); });
        return 1;
    }
    // ---- S1 gather from the shared-memory box (same stencil as ent_dev.cuh gather)
    float EBv[6];
    gather_box<D, G::FX, G::FY, G::FNP>(T.sF, b, d, EBv);
    // ---- S2 tetrad (A^hat = sqrt(h_ii) A^i), S3 Boris (Eq. 3), S4-S5 move + crossing
    float E[3] = { T.sx[0] * EBv[0], T.sx[1] * EBv[1], T.sx[2] * EBv[2] }, B[3] = { T.sx[0] * EBv[3], T.sx[1] * EBv[4], T.sx[2] * EBv[5] };
    push_momentum(g, u, E, B, eps);
    const float ig = inv_gamma(u);
    const float a0[3] = { d[0], d[1], d[2] };
    int di[3] = {0, 0, 0};
    bool alive = true;
#pragma unroll
    for (int a = 0; a < D; ++a) {
        float x = d[a] + (u[a] * ig) * A.cdt[a];
        split_offset(x, di[a], d[a]);
        int in = i[a] + di[a];
        const int wrapN = (ALLPER || g.bc[a] == ENT_PERIODIC) ? g.N[a] : 0;
        in += (in < 0) ? wrapN : 0;
        in -= (in >= g.N[a]) ? wrapN : 0;
        if (!ALLPER) { if (in < 0) { alive = false; in = 0; } if (in >= g.N[a]) { alive = false; in = g.N[a] - 1; } }
        i[a] = in;
    }
    cell = (D == 2) ? i[0] + g.N[0] * i[1] : i[0] + g.N[0] * (i[1] + g.N[1] * i[2]);
    if (!alive) return 2;
    bool bad = false;
#pragma unroll
    for (int a = 0; a < D; ++a) bad |= (di[a] < -1) | (di[a] > 1);
    if (bad) { atomicAdd(A.counters + 0, 1ULL); return 0; }
    const float qw = q * wgt;
    edge |= !(fabsf(wgt) <= T.wguard);        // a weight far above the tile's recorded maximum (changed since the sort) cannot use the tile's scale
    if (edge) { edge_deposit<D, TiledArgs>(A, iold[0], iold[1], iold[2], a0[0], a0[1], a0[2], di[0], di[1], di[2], d[0], d[1], d[2], u[0], u[1], u[2], qw); return 0; }     // rare: global atomics, un-wrapped from the true cell
    // ---- S7 deposit into the shared-memory J tile (Eq. 6); node (b) of the box = element b of the J tile
    {
        const float a3[3] = { a0[0], a0[1], (D == 3) ? a0[2] : 0.f };
        const float hv = (D == 2) ? 0.5f * qw * T.Sc * (u[2] * ig) : 0.f;       // out-of-plane rate per segment (G8), h33 = 1
        tile_deposit<D, G>(T.sJ, T.cc, b, a3, d, di, qw * A.inv_dt * T.Sc, hv);   // Q in fixed-point units
    }
    return 0;
}

template <int D, int TX, int TY, int TZ, bool ALLPER, bool PAIR>     // ALLPER: every dimension periodic (no ABSORB bookkeeping); PAIR: two blocks
__global__ void __launch_bounds__(TILED_TPB, ENT_TILED_MINB)
step_tiled_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ TiledArgs A) {
    using G = TileGeom<D, TX, TY, TZ>;
    extern __shared__ __align__(128) float smem[];
    float *sF = smem;                                            // [6][FNP]
    int *sJ = reinterpret_cast<int *>(smem + 6 * G::FNP);        // [3][JNP], fixed point (see acc_fixed)
    __shared__ uint64_t bar;
    const GridDev &g = A.g;
    const int tid = threadIdx.x;

    // pair launch: one CTA per tile, whole ranges of both blocks; otherwise the work list (chunks of tile_chunk_for(n) particles)
    const int tile = PAIR ? (int)blockIdx.x : find_tile(A.chunk_off, A.ntiles, blockIdx.x);
    if (tile < 0) return;                                        // the grid is an upper bound of the work list
    const int t0 = tile % g.nt[0], t12 = tile / g.nt[0];
    const int t1 = (D == 3) ? t12 % g.nt[1] : t12, t2 = (D == 3) ? t12 / g.nt[1] : 0;
    TileCtx<D> T;
    T.sF = sF; T.sJ = sJ;
    T.o[0] = t0 * TX; T.o[1] = t1 * TY; T.o[2] = t2 * TZ;
    T.sx[0] = g.dx[0]; T.sx[1] = g.dx[1]; T.sx[2] = g.dx[2];

    if (tid == 0) {
        mbar_init(&bar, 1);
        fence_mbar_init();
        mbar_expect_tx(&bar, 6u * G::FN * 4u);
#pragma unroll
        for (int c = 0; c < 6; ++c) tma_load_box<D>(sF + c * G::FNP, &maps.F[c], &bar, T.o[0], T.o[1], T.o[2]);   // padded coords of active o-2
    }
    for (int k = tid; k < 3 * G::JNP / 4; k += TILED_TPB) reinterpret_cast<int4 *>(sJ)[k] = make_int4(0, 0, 0, 0);

    float invSc, wguard2 = -1.0f;
    {
        // fixed-point scale of this tile.  Largest contribution: |q| wmax / dt * |D| * weight with |D| <= 1, weight <= 13/12
        // (2D: J^3 = q w v^3 has no 1/dt); wmax = max |w| over the tile's particles (ent_sort).  It gets 24 bits; a nodal sum
        // beyond 2^31 (128 such contributions adding coherently) wraps and is carried exactly (carry_fix).
        float wm = A.tile_wmax[tile];
        // |D_a| <= min(1, dt / dx_a): the rate q w D / dt is at most q w / min dx (2D: J^3 = q w v^3, |v^3| < 1, h33 = 1)
        float rate = fminf(A.inv_dt, 1.02f * fmaxf(g.inv_dx[0], fmaxf(g.inv_dx[1], (D == 3) ? g.inv_dx[2] : 0.f)));
        if (D == 2) rate = fmaxf(rate, 0.5f);
        float qw1 = fabsf(A.q) * wm;
        if (PAIR) {                                              // one scale for both species: the larger |q| wmax
            const float wm2 = A.tile_wmax2[tile], qw2 = fabsf(A.q2) * wm2;
            const float qwm = fmaxf(qw1, qw2);
            wguard2 = 60.0f * (fabsf(A.q2) > 0.f ? qwm / fabsf(A.q2) : 0.f);
            wm = fabsf(A.q) > 0.f ? qwm / fabsf(A.q) : 0.f;
            qw1 = qwm;
        }
        float qmax = qw1 * rate * 1.0834f;
        float Sc = (qmax > 0.f && qmax < 1e37f) ? FIXED_ONE / qmax : 0.f;
        if (!(Sc > 1e-30f && Sc < 1e30f)) Sc = 0.f;
        invSc = Sc > 0.f ? 1.0f / Sc : 0.f;
        T.Sc = Sc; T.wguard = Sc > 0.f ? 60.0f * wm : -1.0f;
        if (!(Sc > 0.f)) wguard2 = -1.0f;
    }
    T.cc.J = A.J.c; T.cc.P0 = g.P[0]; T.cc.P01 = g.P[0] * g.P[1]; T.cc.unit = 4294967296.0f * invSc;
    T.cc.JX = G::JX; T.cc.JY = G::JY; T.cc.JNP = G::JNP; T.cc.carries = A.counters + 4;
    T.cc.gbase = (long long)T.o[0] + (long long)g.P[0] * T.o[1] + (D == 3 ? (long long)g.P[0] * g.P[1] * T.o[2] : 0);
    __syncthreads();                                             // sJ zeroed, mbarrier initialised
    bool waited = false;

    // ---- one particle per thread and iteration, consecutive lanes on consecutive particles: every access is a fully
    // coalesced 128-byte line per warp, the work of a tile is balanced to within one particle per thread, and the order of the
    // particles inside the tile's range does not matter (the incremental ent_sort does not keep one)
    // software pipeline: the record of the thread's next particle is requested before the current one is advanced
#pragma unroll 1
  for (int sp = 0; sp < (PAIR ? 2 : 1); ++sp) {
    const PartPtrs &P = (PAIR && sp) ? A.P2 : A.P;
    const float q = (PAIR && sp) ? A.q2 : A.q, eps = (PAIR && sp) ? A.eps2 : A.eps;
    if (PAIR && sp) T.wguard = wguard2;
    const int32_t *koff = (PAIR && sp) ? A.key_off2 : A.key_off;
    long long p0 = koff[tile], p1 = koff[tile + 1];
    if (!PAIR) {
        p0 += (long long)(blockIdx.x - A.chunk_off[tile]) * A.chunk;
        if (p1 > p0 + A.chunk) p1 = p0 + A.chunk;
    }
    long long p = p0 + tid;
    int ncell = 0; float nd0 = 0.f, nd1 = 0.f, nd2 = 0.f, nu0 = 0.f, nu1 = 0.f, nu2 = 0.f, nw = 0.f; bool nlive = true;
    if (p < p1) {
        ncell = P.cell[p]; nd0 = P.d[0][p]; nd1 = P.d[1][p]; if (D == 3) nd2 = P.d[2][p];
        nu0 = P.u[0][p]; nu1 = P.u[1][p]; nu2 = P.u[2][p]; nw = P.w[p];
        if (P.tag) nlive = P.tag[p] != 0;
    }
    for (; p < p1; p += TILED_TPB) {
        int cell = ncell;
        float d[3] = { nd0, nd1, nd2 }, u[3] = { nu0, nu1, nu2 };
        const float wgt = nw; const bool live = nlive;
        const long long pn = p + TILED_TPB;
        if (pn < p1) {
            ncell = P.cell[pn]; nd0 = P.d[0][pn]; nd1 = P.d[1][pn]; if (D == 3) nd2 = P.d[2][pn];
            nu0 = P.u[0][pn]; nu1 = P.u[1][pn]; nu2 = P.u[2][pn]; nw = P.w[pn];
            if (P.tag) nlive = P.tag[pn] != 0;
        }
        if (!waited) { mbar_wait(&bar, 0); waited = true; }
        if (!live) continue;
        const int code = tile_particle<D, TX, TY, TZ, ALLPER, PAIR>(A, T, p, cell, d, u, wgt, q, eps, sp);
        if (code & 1) continue;
        P.cell[p] = cell;
        P.d[0][p] = d[0]; P.d[1][p] = d[1]; if (D == 3) P.d[2][p] = d[2];
        P.u[0][p] = u[0]; P.u[1][p] = u[1]; P.u[2][p] = u[2];
        if (!ALLPER && code == 2) P.tag[p] = 0;
    }
  }
    if (!waited) mbar_wait(&bar, 0);          // never leave with a TMA load still in flight into this CTA's shared memory
    // ---- S8 flush: one TMA reduce-add per component into the un-wrapped padded J (ghost fold = ent_fold_current)
    __syncthreads();
    for (int k = tid; k < 3 * G::JNP / 4; k += TILED_TPB) {      // fixed point -> fp32, in place
        int4 v = reinterpret_cast<int4 *>(sJ)[k];
        reinterpret_cast<float4 *>(sJ)[k] = make_float4((float)v.x * invSc, (float)v.y * invSc, (float)v.z * invSc, (float)v.w * invSc);
    }
    fence_proxy_async_smem();
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) tma_reduce_add_box<D>(&maps.J[c], sJ + c * G::JNP, T.o[0], T.o[1], T.o[2]);
        tma_commit();
        tma_wait_read0();
    }
}

// the strays of the last tiled launch, one per thread (global gathers, global atomics)
template <int D>
__global__ void __launch_bounds__(256) stray_kernel(const __grid_constant__ TiledArgs A) {
    const unsigned long long cnt = A.counters[2];
    const long long m = (long long)cnt < A.stray_cap ? (long long)cnt : A.stray_cap;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (long long)gridDim.x * blockDim.x)
        stray_step<D>(A, A.stray_list[k]);
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TiledState {
    size_t scratch = 0;
    EncodeTiledFn encode = nullptr;
    bool tried_encode = false;
    int shape = -1;                         // index into the instantiated tile shapes, -1 = none fits
    int32_t *stray_list = nullptr; long long stray_cap = 0;     // ctx scratch (ent_reserve)
    const void *ptrF[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    const void *ptrJ[3] = {nullptr, nullptr, nullptr};
    TileMaps maps;
    bool attr_set[32] = {};
};


// instantiated tile shapes: index -> (D, TX, TY, TZ)
#define ENT_TILE_SHAPES(X) X(0, 3, 8, 8, 4) X(1, 3, 8, 8, 8) X(2, 2, 16, 16, 1)

inline int tiled_find_shape(const GridDev &g) {
#define X(IDX, DD, A, B, C) if (g.D == DD && g.T[0] == A && g.T[1] == B && g.T[2] == C) return IDX;
    ENT_TILE_SHAPES(X)
#undef X
    return -1;
}

inline int tiled_set_grid(TiledState &t, const GridDev &g, char *, size_t) {
    t.shape = -1;
    for (int c = 0; c < 6; ++c) t.ptrF[c] = nullptr;
    for (int c = 0; c < 3; ++c) t.ptrJ[c] = nullptr;
    if (!t.tried_encode) {
        t.tried_encode = true;
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess && qres == cudaDriverEntryPointSuccess)
            t.encode = (EncodeTiledFn)fn;
        else cudaGetLastError();
    }
    // TMA needs 16-byte global strides: padded row length (N0 + 4) * 4 bytes, i.e. N0 % 4 == 0.
    if (!t.encode || (g.P[0] % 4) != 0) return ENT_OK;
    t.shape = tiled_find_shape(g);
    return ENT_OK;
}
inline bool tiled_supported(const TiledState &t, const GridDev &) { return t.shape >= 0; }

template <int D, int TX, int TY, int TZ>
inline int tiled_encode(TiledState &t, const GridDev &g, const FieldPtrs &F, const CurrentPtrs &J, char *err, size_t errn) {
    using G = TileGeom<D, TX, TY, TZ>;
    cuuint64_t dims[3] = { (cuuint64_t)g.P[0], (cuuint64_t)g.P[1], (cuuint64_t)g.P[2] };
    cuuint64_t strides[2] = { (cuuint64_t)g.P[0] * 4, (cuuint64_t)g.P[0] * g.P[1] * 4 };
    cuuint32_t estr[3] = { 1, 1, 1 };
    for (int c = 0; c < 6; ++c) {
        if (t.ptrF[c] == F.c[c]) continue;
        cuuint32_t box[3] = { G::FX, G::FY, G::FZ };
        CUresult r = t.encode(&t.maps.F[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, D, (void *)F.c[c], dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { snprintf(err, errn, "cuTensorMapEncodeTiled(field %d) failed: %d", c, (int)r); return ENT_ECUDA; }
        t.ptrF[c] = F.c[c];
    }
    for (int c = 0; c < 3; ++c) {
        if (t.ptrJ[c] == J.c[c]) continue;
        cuuint32_t box[3] = { G::JX, G::JY, G::JZ };
        CUresult r = t.encode(&t.maps.J[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, D, (void *)J.c[c], dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { snprintf(err, errn, "cuTensorMapEncodeTiled(current %d) failed: %d", c, (int)r); return ENT_ECUDA; }
        t.ptrJ[c] = J.c[c];
    }
    return ENT_OK;
}

template <int KIND, int TX, int TY>
__global__ void step_tiled_axisym_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ TiledArgs A);   // ent_tiled_axisym.cuh
template <int TX, int TY> struct AxiGeom;

template <int D> inline void launch_strays(const TiledArgs &A, cudaStream_t stream);      // after the axisymmetric kernels are known

template <int IDX, int D, int TX, int TY, int TZ>
inline int tiled_launch(TiledState &t, const TiledArgs &A, cudaStream_t stream, char *err, size_t errn) {
    using G = TileGeom<D, TX, TY, TZ>;
    int rc = tiled_encode<D, TX, TY, TZ>(t, A.g, A.F, A.J, err, errn);
    if (rc) return rc;
    bool allper = true;
    for (int a = 0; a < D; ++a) allper &= A.g.bc[a] == ENT_PERIODIC;
    const bool pair = A.nsp == 2;
    void (*kern)(const TileMaps, const TiledArgs) =
        pair ? (allper ? step_tiled_kernel<D, TX, TY, TZ, true, true> : step_tiled_kernel<D, TX, TY, TZ, false, true>)
             : (allper ? step_tiled_kernel<D, TX, TY, TZ, true, false> : step_tiled_kernel<D, TX, TY, TZ, false, false>);
    int slot = 2 * IDX + (allper ? 1 : 0) + (pair ? 16 : 0);
    int smem_bytes = G::SMEM_BYTES;
    if constexpr (D == 2) {
        if (A.g.kind == ENT_SPH) { kern = step_tiled_axisym_kernel<ENT_SPH, TX, TY>; slot = 6; }
        else if (A.g.kind == ENT_QSPH) { kern = step_tiled_axisym_kernel<ENT_QSPH, TX, TY>; slot = 7; }
        if (A.g.kind != ENT_CART) smem_bytes = AxiGeom<TX, TY>::SMEM_BYTES;
    } else if (A.g.kind != ENT_CART) { snprintf(err, errn, "no 3D tiled kernel for this metric"); return ENT_EUNSUPPORTED; }
    if (!t.attr_set[slot]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
        if (e != cudaSuccess) { snprintf(err, errn, "cudaFuncSetAttribute(smem %d) failed: %s", smem_bytes, cudaGetErrorString(e)); return ENT_ECUDA; }
        t.attr_set[slot] = true;
    }
    const int ntiles = A.g.nt[0] * A.g.nt[1] * A.g.nt[2];
    const long long grid = A.nsp == 2 ? (long long)ntiles : (long long)ntiles + A.n / A.chunk + 1;        // upper bound of the number of chunks
    kern<<<(unsigned)grid, TILED_TPB, smem_bytes, stream>>>(t.maps, A);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { snprintf(err, errn, "launch of step_tiled_kernel failed: %s", cudaGetErrorString(e)); return ENT_ECUDA; }
    launch_strays<D>(A, stream);
    e = cudaGetLastError();
    if (e != cudaSuccess) { snprintf(err, errn, "launch of stray_kernel failed: %s", cudaGetErrorString(e)); return ENT_ECUDA; }
    return ENT_OK;
}

struct PairSpecies { PartPtrs P; const int32_t *key_off; const float *tile_wmax; float eps, q; };   // second block of ent_step_pair

inline int tiled_step(TiledState &t, const GridDev &g, cudaStream_t stream, FieldPtrs F, PartPtrs P, CurrentPtrs J, long long n,
                      const int32_t *key_off, const float *tile_wmax, const int32_t *chunk_off, float eps, float dt, float q, float inv_dt, unsigned long long *counters,
                      long long *launches, char *err, size_t errn, const PairSpecies *pair = nullptr) {
    TiledArgs A;
    A.g = g; A.F = F; A.J = J; A.P = P; A.key_off = key_off; A.tile_wmax = tile_wmax; A.chunk_off = chunk_off; A.ntiles = g.nt[0] * g.nt[1] * g.nt[2]; A.n = n; A.chunk = tile_chunk_for(n);
    A.eps = eps; A.dt = dt; A.q = q; A.inv_dt = inv_dt; A.counters = counters;
    A.nsp = 1; A.P2 = P; A.key_off2 = key_off; A.tile_wmax2 = tile_wmax; A.eps2 = eps; A.q2 = q;
    if (pair) { A.nsp = 2; A.P2 = pair->P; A.key_off2 = pair->key_off; A.tile_wmax2 = pair->tile_wmax; A.eps2 = pair->eps; A.q2 = pair->q; }
    A.stray_list = t.stray_list; A.stray_cap = t.stray_cap;
    for (int a = 0; a < 3; ++a) A.cdt[a] = dt * g.inv_dx[a];
    A.divN0 = make_magicdiv((uint32_t)g.N[0]);
    A.divN01 = make_magicdiv((uint32_t)(g.N[0] * g.N[1]));
    int rc = ENT_EUNSUPPORTED;
    switch (t.shape) {
#define X(IDX, DD, A_, B_, C_) case IDX: rc = tiled_launch<IDX, DD, A_, B_, C_>(t, A, stream, err, errn); break;
        ENT_TILE_SHAPES(X)
#undef X
        default: snprintf(err, errn, "no tiled kernel for this tile shape"); break;
    }
    if (rc == ENT_OK) *launches += 2;
    return rc;
}

}  // namespace ent
