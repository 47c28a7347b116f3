// ent_sorted.cuh -- fused step + re-bin for the Cartesian grids (sub-steps 3-8, and the tile sort S10), sm_100a.
//
// ent_step_sorted(in, out): ONE pass over a tile-contiguous block `in` advances every particle (gather, tetrad, Boris, move,
// crossing, deposit: the arithmetic of ent_tiled.cuh) and writes it to `out` in the range of the tile its INPUT cell lies
// in.  `out` is therefore tile-contiguous by the positions BEFORE the step: one step stale, i.e. every particle of a tile's
// range sits within one cell of the tile, which is exactly the halo the E,B box and the J tile of a CTA cover.  The
// populations per tile of the NEW positions are counted on the way (next_count), so the next call knows its output layout
// before it starts, and the per-tile max |w| of the output ranges is maintained.  No sort pass ever runs between steps.
//
// A CTA works on one chunk (<= tile_chunk_for(n) particles) of one tile, streaming: one particle per thread and iteration straight
// from global memory (consecutive lanes on consecutive particles, next record requested before the current one is advanced).
//   * slot in `out`: particles that stay in the tile (~87 %) take consecutive slots from ONE global reservation per warp and
//     iteration (ballot), the others one reservation each; the atomics are issued right after the cell index is decoded and
//     their results are used ~700 instructions later, so their latency is covered;
//   * the first version of this kernel staged the chunk in shared memory and processed it in rank-major cell order (consecutive
//     lanes on different, consecutive cells).  Measured on C3: 3.8 ms against 2.2 ms -- 305 of 1185 warp instructions per 32
//     particles went into staging and ordering, the phases serialised on barriers, and the bank conflicts stayed (gather 2.5,
//     ATOMS 2.7 wavefronts per instruction): lanes 30 keys apart alias because the rows of the E,B box are two cells wider than
//     the rows of cells that hold particles.  Dropped for this streaming form.
//   * the gather uses packed fp32 pairs (FFMA2 / FADD2): two of the seven lerps of a component per instruction.
#pragma once
#include "ent_tiled.cuh"

namespace ent {

constexpr int FUSED_TPB = 256;
#ifndef ENT_FUSED_MINB
#define ENT_FUSED_MINB 3
#endif

struct SortedArgs {
    GridDev g;
    FieldPtrs F;
    CurrentPtrs J;
    PartPtrs in, out;
    const int32_t *tile_off;      // layout of `in`: tile t owns particles [tile_off[t], tile_off[t+1])
    const int32_t *chunk_off;     // work list of `in` (chunks of tile_chunk_for(n) particles)
    int chunk;
    const float *tile_wmax;       // max |w| per range of `in`
    int32_t *cursor;              // per tile: next free slot of its range in `out` (starts at the out layout's offsets)
    int32_t *next_count;          // per tile: particles whose cell AFTER this step lies in it (layout of the next step's output)
    unsigned *wmax_out;           // per tile: max |w| (float bits) over the particles written to its range of `out`
    int ntiles;
    long long n;
    float eps, dt, q, inv_dt;
    float cdt[3];                 // dt / dx_d
    unsigned long long *counters; // [0] bad moves, [1] strays, [3] slot errors
    MagicDiv divN0, divN01, divnt0, divnt1;
};

// global 32-bit atomic add with return, as inline PTX: nvcc turns atomicAdd on a warp-uniform address into its own aggregate
// (one lane adds, SHFL broadcasts the result) and waits for the result on the spot; here the result must stay untouched until
// the particle has been advanced, so that the ~1 us round trip is covered by that work
__device__ __forceinline__ int atom_add_global(int32_t *p, int v) {
    int r;
    asm volatile("atom.global.add.u32 %0, [%1], %2;" : "=r"(r) : "l"(__cvta_generic_to_global(p)), "r"(v) : "memory");
    return r;
}

// tile of an active cell (rare paths only: plain divisions)
template <int D>
__device__ __forceinline__ int tile_of_cell_slow(const GridDev &g, int cell) {
    int i[3];
    unpack_cell<D>(g, cell, i);
    int t0 = i[0] / g.T[0], t1 = i[1] / g.T[1], t2 = (D == 3) ? i[2] / g.T[2] : 0;
    return t0 + g.nt[0] * (t1 + g.nt[1] * t2);
}

// a particle of the range that is NOT within one cell of its tile (the caller moved it, or the block is not the one the ctx
// believes it is): advanced with global gathers and global atomics, written to the range of its true tile
template <int D>
__device__ __noinline__ void stray_sorted(const SortedArgs &A, long long p) {
    const GridDev &g = A.g;
    int i[3], i0[3], di[3]; float d[3] = {0.f, 0.f, 0.f}, a[3], u[3], phi = 0.f;
    const int cell0 = A.in.cell[p];
    unpack_cell<D>(g, cell0, i);
#pragma unroll
    for (int k = 0; k < D; ++k) d[k] = A.in.d[k][p];
#pragma unroll
    for (int k = 0; k < 3; ++k) { u[k] = A.in.u[k][p]; a[k] = d[k]; i0[k] = i[k]; }
    const float w = A.in.w[p];
    bool live = A.in.tag ? A.in.tag[p] != 0 : true, alive = true;
    if (live) {
        GlobalFieldLoader ld{A.F.c};
        push_particle<D, ENT_CART>(g, ld, i, d, phi, u, A.eps, A.dt, di, alive);
    }
    const int cell1 = pack_cell<D>(g, i);
    const int tdst = tile_of_cell_slow<D>(g, cell0);
    const long long slot = atomicAdd(A.cursor + tdst, 1);
    atomicAdd(A.next_count + tile_of_cell_slow<D>(g, cell1), 1);
    atomicMax(A.wmax_out + tdst, __float_as_uint(fabsf(w)));
    atomicAdd(A.counters + 1, 1ULL);
    if (slot < 0 || slot >= A.n) { atomicAdd(A.counters + 3, 1ULL); return; }
    A.out.cell[slot] = cell1;
#pragma unroll
    for (int k = 0; k < D; ++k) A.out.d[k][slot] = d[k];
#pragma unroll
    for (int k = 0; k < 3; ++k) A.out.u[k][slot] = u[k];
    A.out.w[slot] = w;
    if (A.out.tag) A.out.tag[slot] = (live && alive) ? 1 : 0;
    if (!live || !alive) return;
    bool bad = false;
#pragma unroll
    for (int k = 0; k < D; ++k) bad |= (di[k] < -1 || di[k] > 1);
    if (bad) { atomicAdd(A.counters + 0, 1ULL); return; }
    GlobalAcc acc{A.J.c};
    deposit_particle<D, ENT_CART>(g, acc, i0, a, di, d, 0.f, 0.f, u, A.q * w, A.inv_dt);
}

template <int D, int TX, int TY, int TZ, bool ALLPER>     // ALLPER: every dimension periodic (no ABSORB bookkeeping)
__global__ void __launch_bounds__(FUSED_TPB, ENT_FUSED_MINB)
step_fused_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ SortedArgs A) {
    using G = TileGeom<D, TX, TY, TZ>;
    extern __shared__ __align__(128) float smem[];
    float *sF = smem;                                            // [6][FNP]
    int *sJ = reinterpret_cast<int *>(smem + 6 * G::FNP);        // [3][JNP], fixed point (ent_tiled.cuh acc_fixed)
    __shared__ uint64_t bar;
    __shared__ int dest_s[28], cnt2[28];
    __shared__ unsigned wmx[28];
    const GridDev &g = A.g;
    const int tid = threadIdx.x, lane = tid & 31;

    const int tile = find_tile(A.chunk_off, A.ntiles, blockIdx.x);
    if (tile < 0) return;                                        // the grid is an upper bound of the work list
    const int t12 = A.divnt0.div(tile), t0 = tile - t12 * g.nt[0];
    const int t2 = (D == 3) ? A.divnt1.div(t12) : 0, t1 = (D == 3) ? t12 - t2 * g.nt[1] : t12;
    const int o[3] = { t0 * TX, t1 * TY, t2 * TZ };
    // extent of THIS tile: the last tile of a dimension is partial when N is not a multiple of T
    const int te[3] = { min(TX, g.N[0] - o[0]), min(TY, g.N[1] - o[1]), (D == 3) ? min(TZ, g.N[2] - o[2]) : 1 };

    if (tid == 0) {
        mbar_init(&bar, 1);
        fence_mbar_init();
        mbar_expect_tx(&bar, 6u * G::FN * 4u);
#pragma unroll
        for (int c = 0; c < 6; ++c) tma_load_box<D>(sF + c * G::FNP, &maps.F[c], &bar, o[0], o[1], o[2]);   // padded coords of active o-2
    }
    for (int k = tid; k < 3 * G::JNP / 4; k += FUSED_TPB) reinterpret_cast<int4 *>(sJ)[k] = make_int4(0, 0, 0, 0);
    if (tid < 28) {
        cnt2[tid] = 0; wmx[tid] = 0u;
        int d = -1;
        if (tid < 27) {                                          // destination tile of class (c0, c1, c2), -1 if it does not exist
            int rel = tid, tt[3] = { t0, t1, t2 }; bool ok = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int c = rel % 3; rel /= 3;
                int v = tt[a] + c - 1;
                if (ALLPER || g.bc[a] == ENT_PERIODIC) { if (v < 0) v += g.nt[a]; if (v >= g.nt[a]) v -= g.nt[a]; }
                ok &= (v >= 0 && v < g.nt[a]);
                tt[a] = v;
            }
            if (ok) d = tt[0] + g.nt[0] * (tt[1] + g.nt[1] * tt[2]);
        }
        dest_s[tid] = d;
    }

    long long p0 = A.tile_off[tile], p1 = A.tile_off[tile + 1];
    p0 += (long long)(blockIdx.x - A.chunk_off[tile]) * A.chunk;
    if (p1 > p0 + A.chunk) p1 = p0 + A.chunk;
    TileCtx<D> T;
    T.sF = sF; T.sJ = sJ;
    T.o[0] = o[0]; T.o[1] = o[1]; T.o[2] = o[2];
    T.sx[0] = g.dx[0]; T.sx[1] = g.dx[1]; T.sx[2] = g.dx[2];
    float invSc;
    {   // fixed-point scale of this tile's J tile (ent_tiled.cuh): largest contribution |q| wmax rate (13/12) gets 24 bits
        const float wm = A.tile_wmax[tile];
        float rate = fminf(A.inv_dt, 1.02f * fmaxf(g.inv_dx[0], fmaxf(g.inv_dx[1], (D == 3) ? g.inv_dx[2] : 0.f)));
        if (D == 2) rate = fmaxf(rate, 0.5f);
        const float qmax = fabsf(A.q) * wm * rate * 1.0834f;
        float Sc = (qmax > 0.f && qmax < 1e37f) ? FIXED_ONE / qmax : 0.f;
        if (!(Sc > 1e-30f && Sc < 1e30f)) Sc = 0.f;
        invSc = Sc > 0.f ? 1.0f / Sc : 0.f;
        T.Sc = Sc; T.wguard = Sc > 0.f ? 60.0f * wm : -1.0f;
    }
    T.cc.J = A.J.c; T.cc.P0 = g.P[0]; T.cc.P01 = g.P[0] * g.P[1]; T.cc.unit = 4294967296.0f * invSc;
    T.cc.JX = G::JX; T.cc.JY = G::JY; T.cc.JNP = G::JNP; T.cc.carries = A.counters + 4;
    T.cc.gbase = (long long)o[0] + (long long)g.P[0] * o[1] + (D == 3 ? (long long)g.P[0] * g.P[1] * o[2] : 0);
    __syncthreads();                                             // sJ zeroed, mbarrier initialised, dest_s ready
    bool waited = false;

    // ---- one particle per thread and iteration, consecutive lanes on consecutive particles; the trip count is uniform over a
    // warp (ballots inside), the record of the thread's next particle is requested before the current one is advanced
    long long p = p0 + tid;
    int ncell = 0; float nd0 = 0.f, nd1 = 0.f, nd2 = 0.f, nu0 = 0.f, nu1 = 0.f, nu2 = 0.f, nw = 0.f; bool nlive = true;
    if (p < p1) {
        ncell = A.in.cell[p]; nd0 = A.in.d[0][p]; nd1 = A.in.d[1][p]; if (D == 3) nd2 = A.in.d[2][p];
        nu0 = A.in.u[0][p]; nu1 = A.in.u[1][p]; nu2 = A.in.u[2][p]; nw = A.in.w[p];
        if (A.in.tag) nlive = A.in.tag[p] != 0;
    }
    for (long long pb = p0 + (tid & ~31); pb < p1; pb += FUSED_TPB, p += FUSED_TPB) {
        const bool have = p < p1;
        int cell = ncell;
        float d[3] = { nd0, nd1, nd2 }, u[3] = { nu0, nu1, nu2 };
        const float wgt = nw; const bool live = nlive;
        const long long pn = p + FUSED_TPB;
        if (pn < p1) {
            ncell = A.in.cell[pn]; nd0 = A.in.d[0][pn]; nd1 = A.in.d[1][pn]; if (D == 3) nd2 = A.in.d[2][pn];
            nu0 = A.in.u[0][pn]; nu1 = A.in.u[1][pn]; nu2 = A.in.u[2][pn]; nw = A.in.w[pn];
            if (A.in.tag) nlive = A.in.tag[pn] != 0;
        }
        // ---- where is the cell relative to the tile box?  b = cell index in box coordinates (box origin = o - 2); class =
        // which of the 27 neighbouring tiles (13 = this one) the cell belongs to
        int i[3];
        if (D == 2) { i[1] = A.divN0.div(cell); i[0] = cell - i[1] * g.N[0]; i[2] = 0; }
        else { i[2] = A.divN01.div(cell); int r = cell - i[2] * (g.N[0] * g.N[1]); i[1] = A.divN0.div(r); i[0] = r - i[1] * g.N[0]; }
        const int iold[3] = { i[0], i[1], i[2] };
        int b[3] = { i[0] - o[0] + 2, i[1] - o[1] + 2, (D == 3) ? i[2] - o[2] + 2 : 0 };
        bool local = have, edge = false;
        int cls = 0;
        {
            int cmul = 1;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (a < D) {
                    const int wrapN = (ALLPER || g.bc[a] == ENT_PERIODIC) ? g.N[a] : 0;
                    b[a] += (b[a] < 1) ? wrapN : 0;
                    b[a] -= (b[a] > g.N[a]) ? wrapN : 0;
                    local &= (unsigned)(b[a] - 1) < (unsigned)(te[a] + 2);       // within one cell of the tile
                    cls += ((b[a] >= 2) + (b[a] >= te[a] + 2)) * cmul;
                    // un-wrapped cell N of a periodic dimension: its +1 crossing would deposit at node N + 2, outside the padded array
                    edge |= (o[a] - 2 + b[a] > g.N[a] - 1);
                } else cls += cmul;
                cmul *= 3;
            }
        }
        if (!local) cls = -1;
        // ---- slot in `out` (the range of the tile of the INPUT cell): reserved now, used after the particle is advanced
        const unsigned m13 = __ballot_sync(0xffffffffu, cls == 13);
        const unsigned wbits = __float_as_uint(fabsf(wgt));
        const unsigned w13 = __reduce_max_sync(0xffffffffu, cls == 13 ? wbits : 0u);
        int slot = 0;                                           // the reservation's result is not touched before the write-back
        const int leader = __ffs(m13) - 1;
        if (m13 && lane == leader) { slot = atom_add_global(A.cursor + tile, __popc(m13)); atomicMax(&wmx[13], w13); }
        if (cls >= 0 && cls != 13) {
            const int dt_ = dest_s[cls];
            slot = dt_ >= 0 ? atom_add_global(A.cursor + dt_, 1) : -1;
            atomicMax(&wmx[cls], wbits);
        }
        if (!waited) { mbar_wait(&bar, 0); waited = true; }
        if (have && !local) stray_sorted<D>(A, p);
        int cls2 = cls;                                          // a dead particle stays where it is
        bool alive = live;
        if (local && live) {
            // ---- S1 gather from the shared-memory box (same stencil and arithmetic as ent_dev.cuh gather)
            float EBv[6];
            gather_box<D, G::FX, G::FY, G::FNP>(sF, b, d, EBv);
            // ---- S2 tetrad, S3 Boris (Eq. 3), S4-S5 move + crossing
            float E[3] = { T.sx[0] * EBv[0], T.sx[1] * EBv[1], T.sx[2] * EBv[2] }, B[3] = { T.sx[0] * EBv[3], T.sx[1] * EBv[4], T.sx[2] * EBv[5] };
            push_momentum(g, u, E, B, A.eps);
            const float ig = inv_gamma(u);
            const float a0[3] = { d[0], d[1], d[2] };
            int di[3] = {0, 0, 0}, bn[3] = { b[0], b[1], b[2] };
#pragma unroll
            for (int a = 0; a < D; ++a) {
                float x = d[a] + (u[a] * ig) * A.cdt[a];
                split_offset(x, di[a], d[a]);
                int in = i[a] + di[a];
                if (ALLPER || g.bc[a] == ENT_PERIODIC) {
                    in += (in < 0) ? g.N[a] : 0;
                    in -= (in >= g.N[a]) ? g.N[a] : 0;
                    bn[a] = b[a] + di[a];
                } else {
                    if (in < 0) { alive = false; in = 0; }
                    if (in >= g.N[a]) { alive = false; in = g.N[a] - 1; }
                    bn[a] = b[a] + (in - iold[a]);
                }
                i[a] = in;
            }
            cell = (D == 2) ? i[0] + g.N[0] * i[1] : i[0] + g.N[0] * (i[1] + g.N[1] * i[2]);
            {   // class of the new cell (the next step's layout)
                bool near = true; int c2 = 0, cmul = 1;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    if (a < D) { near &= (unsigned)bn[a] < (unsigned)(te[a] + 4); c2 += ((bn[a] >= 2) + (bn[a] >= te[a] + 2)) * cmul; }
                    else c2 += cmul;
                    cmul *= 3;
                }
                cls2 = near ? c2 : 27;
            }
            bool bad = false;
#pragma unroll
            for (int a = 0; a < D; ++a) bad |= (di[a] < -1) | (di[a] > 1);
            if (bad) atomicAdd(A.counters + 0, 1ULL);
            else if (alive) {
                const float qw = A.q * wgt;
                edge |= !(fabsf(wgt) <= T.wguard);           // a weight far above the range's recorded maximum cannot use the tile's scale
                if (edge) edge_deposit<D, SortedArgs>(A, iold[0], iold[1], iold[2], a0[0], a0[1], a0[2], di[0], di[1], di[2], d[0], d[1], d[2], u[0], u[1], u[2], qw);
                else {
                    // ---- S7 deposit into the shared-memory J tile (Eq. 6); node (b) of the box = element b of the J tile
                    const float a3[3] = { a0[0], a0[1], (D == 3) ? a0[2] : 0.f };
                    const float hv = (D == 2) ? 0.5f * qw * T.Sc * (u[2] * ig) : 0.f;   // out-of-plane rate per segment (G8), h33 = 1
                    tile_deposit<D, G>(T.sJ, T.cc, b, a3, d, di, qw * A.inv_dt * T.Sc, hv);
                }
            }
        }
        // ---- populations of the NEW tiles (layout of the next step's output)
        const unsigned n13 = __ballot_sync(0xffffffffu, cls2 == 13);
        if (cls2 == 13) { if ((int)(__ffs(n13) - 1) == lane) atomicAdd(&cnt2[13], __popc(n13)); }
        else if (cls2 >= 0 && cls2 < 27) atomicAdd(&cnt2[cls2], 1);
        else if (cls2 == 27) atomicAdd(A.next_count + tile_of_cell_slow<D>(g, cell), 1);
        {   // particles that stay: consecutive slots after the leader's reservation.  The empty asm pins the first use of the
            // reservation's result here (the compiler would hoist the shuffle to right after the atomic and wait there)
            asm volatile("" : "+r"(slot) :: "memory");
            const int s13 = __shfl_sync(0xffffffffu, slot, leader < 0 ? 0 : leader) + __popc(m13 & ((1u << lane) - 1u));
            if (cls == 13) slot = s13;
        }
        if (cls < 0) continue;                                   // not ours (beyond the range) or taken by the stray path
        if (slot < 0 || slot >= A.n) { atomicAdd(A.counters + 3, 1ULL); continue; }
        A.out.cell[slot] = cell;
        A.out.d[0][slot] = d[0]; A.out.d[1][slot] = d[1]; if (D == 3) A.out.d[2][slot] = d[2];
        A.out.u[0][slot] = u[0]; A.out.u[1][slot] = u[1]; A.out.u[2][slot] = u[2];
        A.out.w[slot] = wgt;
        if (A.out.tag) A.out.tag[slot] = alive ? 1 : 0;
    }
    if (!waited) mbar_wait(&bar, 0);          // never leave with a TMA load still in flight into this CTA's shared memory
    // ---- populations and max |w| of the destination ranges; S8 flush: one TMA reduce-add per component (fold: P:642)
    __syncthreads();
    if (tid < 27 && dest_s[tid] >= 0) {
        if (cnt2[tid] > 0) atomicAdd(A.next_count + dest_s[tid], cnt2[tid]);
        if (wmx[tid]) atomicMax(A.wmax_out + dest_s[tid], wmx[tid]);
    }
    for (int k = tid; k < 3 * G::JNP / 4; k += FUSED_TPB) {      // fixed point -> fp32, in place
        int4 v = reinterpret_cast<int4 *>(sJ)[k];
        reinterpret_cast<float4 *>(sJ)[k] = make_float4((float)v.x * invSc, (float)v.y * invSc, (float)v.z * invSc, (float)v.w * invSc);
    }
    fence_proxy_async_smem();
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) tma_reduce_add_box<D>(&maps.J[c], sJ + c * G::JNP, o[0], o[1], o[2]);
        tma_commit();
        tma_wait_read0();
    }
}

// ---------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------
inline bool sorted_supported(const TiledState &t, const GridDev &g) { return g.kind == ENT_CART && t.shape >= 0; }

template <int D, int TX, int TY, int TZ>
inline int sorted_launch(TiledState &t, int attr_slot, const SortedArgs &A, cudaStream_t stream, char *err, size_t errn) {
    using G = TileGeom<D, TX, TY, TZ>;
    int rc = tiled_encode<D, TX, TY, TZ>(t, A.g, A.F, A.J, err, errn);
    if (rc) return rc;
    bool allper = true;
    for (int a = 0; a < D; ++a) allper &= A.g.bc[a] == ENT_PERIODIC;
    void (*kern)(const TileMaps, const SortedArgs) = allper ? step_fused_kernel<D, TX, TY, TZ, true> : step_fused_kernel<D, TX, TY, TZ, false>;
    const int slot = attr_slot + (allper ? 1 : 0);
    if (!t.attr_set[slot]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM_BYTES);
        if (e != cudaSuccess) { snprintf(err, errn, "cudaFuncSetAttribute(smem %d) failed: %s", G::SMEM_BYTES, cudaGetErrorString(e)); return ENT_ECUDA; }
        t.attr_set[slot] = true;
    }
    const long long grid = (long long)A.ntiles + A.n / A.chunk + 1;        // upper bound of the number of chunks
    kern<<<(unsigned)grid, FUSED_TPB, G::SMEM_BYTES, stream>>>(t.maps, A);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { snprintf(err, errn, "launch of step_fused_kernel failed: %s", cudaGetErrorString(e)); return ENT_ECUDA; }
    return ENT_OK;
}

inline int sorted_step(TiledState &t, SortedArgs &A, float dt, cudaStream_t stream, char *err, size_t errn) {
    for (int a = 0; a < 3; ++a) A.cdt[a] = dt * A.g.inv_dx[a];
    A.divN0 = make_magicdiv((uint32_t)A.g.N[0]);
    A.divN01 = make_magicdiv((uint32_t)(A.g.N[0] * A.g.N[1]));
    A.divnt0 = make_magicdiv((uint32_t)A.g.nt[0]);
    A.divnt1 = make_magicdiv((uint32_t)A.g.nt[1]);
    A.ntiles = A.g.nt[0] * A.g.nt[1] * A.g.nt[2];
    switch (t.shape) {
        case 0: return sorted_launch<3, 8, 8, 4>(t, 8, A, stream, err, errn);
        case 1: return sorted_launch<3, 8, 8, 8>(t, 10, A, stream, err, errn);
        case 2: return sorted_launch<2, 16, 16, 1>(t, 12, A, stream, err, errn);
        default: break;
    }
    snprintf(err, errn, "no fused step + re-bin kernel for this tile shape");
    return ENT_EUNSUPPORTED;
}

}  // namespace ent
