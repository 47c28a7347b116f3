// ent_sorted.cuh -- fused step + re-bin for the Cartesian grids (sub-steps 3-8, and the tile sort S10), sm_100a.
//
// ent_step_sorted(in, out): one pass over a tile-contiguous block `in` advances every particle (gather, tetrad, Boris, move,
// crossing, deposit) and writes it to `out` in the range of the tile its INPUT cell lies in, so `out` is tile-contiguous by
// the positions BEFORE the step: one step stale, i.e. every particle of a tile's range sits within one cell of the tile,
// which is exactly the halo the E,B box and the J tile of a CTA cover.  The counts per tile of the NEW positions are
// accumulated on the way (next_count), so that the next call knows its output layout before it starts.  No separate sort
// pass ever runs between steps.
//
// A CTA works on one chunk (<= SORTED_CAP particles) of one tile:
//   P0  TMA: the six E,B boxes (cp.async.bulk.tensor) AND the chunk's particle arrays (cp.async.bulk, 1D) land in shared
//       memory on one mbarrier; the J tile and the cell histogram are zeroed meanwhile.
//   P1  every particle: box coordinates of its cell, key = cell inside the (T+2)^D halo box, rank inside its cell from a
//       shared-memory histogram (ATOMS with return), class of its destination tile (27 neighbours), max |w|.
//   P2  rank-major order: position = (rank r, cells with more than r particles in cell order), built from ballots of the
//       histogram and one block scan.  Consecutive lanes then hold DIFFERENT, consecutive cells: gathers and shared atomics
//       of a warp hit distinct banks (measured: 1.27 SM-cycles per conflict-free LDS / ATOMS against 2.8 random, 4.1 with four
//       lanes per address).  The 27 destination ranges are reserved with one global atomic each.
//   P3  particles are read from shared memory in that order, advanced, deposited into the fixed-point J tile (no return
//       value, no carry test: see "scale" below), and written coalesced to their slot of `out`.
//   P4  next_count flush, J tile -> fp32, one TMA reduce-add per component.
// Scale of the fixed-point J tile: a node receives at most Nb contributions of at most A = |q| wmax rate (13/12) each from
// this CTA, Nb = min(chunk population, largest population of a 4^D cell neighbourhood), so with S = min(2^24, 0.98 2^31 / Nb) / A
// the true nodal sum fits int32.  32-bit addition is modular, so intermediate wraps are harmless and the result is exact:
// no per-add overflow test, no carries.
#pragma once
#include "ent_tiled.cuh"

namespace ent {

constexpr int SORTED_TPB = 384;
constexpr int SORTED_CAP = 1280;                 // particles per CTA (chunk)
constexpr int SORTED_CAPP = SORTED_CAP + 8;      // staged records: the chunk + alignment slack of the 16-byte bulk copies
constexpr int SORTED_RMAX = 16;                  // ranks placed rank-major; deeper ones go to the tail in arrival order
constexpr int SORTED_ITEMS = (SORTED_CAP + SORTED_TPB - 1) / SORTED_TPB;

struct SortedArgs {
    GridDev g;
    FieldPtrs F;
    CurrentPtrs J;
    PartPtrs in, out;
    const int32_t *tile_off;      // layout of `in`: tile t owns particles [tile_off[t], tile_off[t+1])
    const int32_t *chunk_off;     // work list of `in` (chunks of SORTED_CAP particles)
    int32_t *cursor;              // per tile: next free slot of its range in `out` (starts at the out layout's offsets)
    int32_t *next_count;          // per tile: particles whose cell AFTER this step lies in it (layout of the next step's output)
    int ntiles;
    long long n;
    float eps, dt, q, inv_dt;
    float cdt[3];                 // dt / dx_d
    unsigned long long *counters; // [0] bad moves, [1] strays, [3] slot errors
    MagicDiv divN0, divN01;
};

template <int D, int TX, int TY, int TZ>
struct SortedGeom {
    using G = TileGeom<D, TX, TY, TZ>;
    static constexpr int HX = TX + 2, HY = TY + 2, HZ = (D == 3) ? TZ + 2 : 1;      // cells a particle of the range can sit in
    static constexpr int NKEY = HX * HY * HZ, NW = (NKEY + 31) / 32, NKEYP = NW * 32;
    static constexpr int NROW = HY * HZ, NROWP = ((NROW + 31) / 32) * 32;
    static constexpr int NARR = (D == 3) ? 8 : 7;
    static constexpr int OFF_F = 0;
    static constexpr int OFF_J = OFF_F + 6 * G::FNP * 4;
    static constexpr int OFF_P = OFF_J + 3 * G::JNP * 4;
    static constexpr int OFF_PERM = OFF_P + 8 * SORTED_CAPP * 4;
    static constexpr int OFF_HIST = (OFF_PERM + SORTED_CAPP * 2 + 15) & ~15;
    static constexpr int OFF_WP = OFF_HIST + NKEYP * 4;
    static constexpr int OFF_ROW = OFF_WP + SORTED_RMAX * NW * 8;
    static constexpr int OFF_MISC = OFF_ROW + NROWP * 4;
    static constexpr int SMEM_BYTES = OFF_MISC + 1024;
};

struct SortedMisc {
    int cnt_in[28], base_s[28], fill[28], cnt2[28], dest_s[28];
    int wsum[32];
    unsigned wmaxbits;
    int ovf_cnt, nranked, maxN;
    uint64_t bar;
};
static_assert(sizeof(SortedMisc) <= 1024, "SortedMisc must fit its shared-memory slot");

__device__ __forceinline__ void tma_bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---- packed fp32 pairs (FFMA2 / FADD2 on sm_100a): two independent lerps per instruction ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
// a + f * (b - a), per half (the same FADD, FFMA sequence as the scalar gather of ent_dev.cuh)
__device__ __forceinline__ f32x2 lerp2(f32x2 a, f32x2 b, f32x2 f) {
    f32x2 d, r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(b), "l"(a));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f), "l"(d), "l"(a));
    return r;
}

template <int NT>
__device__ __forceinline__ int block_scan_excl(int v, int *wsum, int &total) {      // NT threads, all call it
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int s = lane < NT / 32 ? wsum[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        if (lane < NT / 32) wsum[lane] = s;
    }
    __syncthreads();
    const int base = wid ? wsum[wid - 1] : 0;
    total = wsum[NT / 32 - 1];
    __syncthreads();
    return base + x - v;
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
    const long long slot = atomicAdd(A.cursor + tile_of_cell_slow<D>(g, cell0), 1);
    atomicAdd(A.next_count + tile_of_cell_slow<D>(g, cell1), 1);
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

// deposit through global atomics for the few particles whose move could leave the padded array (un-wrapped cell N of a periodic
// dimension), out of line
template <int D>
__device__ __noinline__ void edge_deposit_sorted(const SortedArgs &A, int i0, int i1, int i2, float a0, float a1, float a2, int di0, int di1,
                                                 int di2, float d0, float d1, float d2, float u0, float u1, float u2, float qw) {
    const int i[3] = { i0, i1, i2 }, di[3] = { di0, di1, di2 };
    const float a[3] = { a0, a1, a2 }, dn[3] = { d0, d1, d2 }, u[3] = { u0, u1, u2 };
    GlobalAcc acc{A.J.c};
    deposit_particle<D, ENT_CART>(A.g, acc, i, a, di, dn, 0.f, 0.f, u, qw, A.inv_dt);
}

__device__ __forceinline__ void red_fixed(int *p, float scaled) { atomicAdd(p, __float2int_rn(scaled)); }   // result unused: ATOMS.ADD RZ

#ifndef ENT_SORTED_MINB
#define ENT_SORTED_MINB 2
#endif

template <int D, int TX, int TY, int TZ, bool ALLPER>
__global__ void __launch_bounds__(SORTED_TPB, ENT_SORTED_MINB)
step_sorted_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ SortedArgs A) {
    using S = SortedGeom<D, TX, TY, TZ>;
    using G = typename S::G;
    constexpr int TPB_ = SORTED_TPB, CAPP = SORTED_CAPP, NWARP = SORTED_TPB / 32;
    extern __shared__ __align__(128) unsigned char smraw[];
    float *sF = reinterpret_cast<float *>(smraw + S::OFF_F);
    int *sJ = reinterpret_cast<int *>(smraw + S::OFF_J);
    float *sP = reinterpret_cast<float *>(smraw + S::OFF_P);             // [8][CAPP]: cell, d0, d1, d2, u0, u1, u2, w
    unsigned short *perm = reinterpret_cast<unsigned short *>(smraw + S::OFF_PERM);
    int *hist = reinterpret_cast<int *>(smraw + S::OFF_HIST);
    uint2 *wp = reinterpret_cast<uint2 *>(smraw + S::OFF_WP);            // [RMAX][NW]: x = cells with count > r (bit per cell), y = position of the word's first cell
    int *rowv = reinterpret_cast<int *>(smraw + S::OFF_ROW);
    SortedMisc &M = *reinterpret_cast<SortedMisc *>(smraw + S::OFF_MISC);
    const GridDev &g = A.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int TT[3] = { TX, TY, TZ };

    const int tile = find_tile(A.chunk_off, A.ntiles, blockIdx.x);
    if (tile < 0) return;                                                // the grid is an upper bound of the work list
    const int t0 = tile % g.nt[0], t12 = tile / g.nt[0];
    const int t1 = (D == 3) ? t12 % g.nt[1] : t12, t2 = (D == 3) ? t12 / g.nt[1] : 0;
    const int o[3] = { t0 * TX, t1 * TY, t2 * TZ };
    // extent of THIS tile: the last tile of a dimension is partial when N is not a multiple of T
    const int te[3] = { min(TX, g.N[0] - o[0]), min(TY, g.N[1] - o[1]), (D == 3) ? min(TZ, g.N[2] - o[2]) : 1 };
    long long p0 = A.tile_off[tile], p1 = A.tile_off[tile + 1];
    p0 += (long long)(blockIdx.x - A.chunk_off[tile]) * SORTED_CAP;
    if (p1 > p0 + SORTED_CAP) p1 = p0 + SORTED_CAP;
    const int np = (int)(p1 - p0);
    const long long pa = p0 & ~3LL;                                      // 16-byte aligned start of the bulk copies
    long long bulk_end = (p1 + 3) & ~3LL;
    if (bulk_end > (A.n & ~3LL)) bulk_end = A.n & ~3LL;                  // never read past the arrays
    const int ioff = (int)(p0 - pa);                                     // staged index of particle p0 + k is ioff + k

    // ---- P0: TMA loads (fields + particle arrays) on one mbarrier; zero J tile, histogram, counters
    if (tid == 0) {
        mbar_init(&M.bar, 1);
        fence_mbar_init();
        const uint32_t nb = bulk_end > pa ? (uint32_t)(bulk_end - pa) * 4u : 0u;
        mbar_expect_tx(&M.bar, 6u * G::FN * 4u + (uint32_t)S::NARR * nb);
#pragma unroll
        for (int c = 0; c < 6; ++c) tma_load_box<D>(sF + c * G::FNP, &maps.F[c], &M.bar, o[0], o[1], o[2]);
        if (nb) {
            tma_bulk_load(sP + 0 * CAPP, A.in.cell + pa, nb, &M.bar);
#pragma unroll
            for (int a = 0; a < D; ++a) tma_bulk_load(sP + (1 + a) * CAPP, A.in.d[a] + pa, nb, &M.bar);
#pragma unroll
            for (int a = 0; a < 3; ++a) tma_bulk_load(sP + (4 + a) * CAPP, A.in.u[a] + pa, nb, &M.bar);
            tma_bulk_load(sP + 7 * CAPP, A.in.w + pa, nb, &M.bar);
        }
    }
    for (int k = tid; k < 3 * G::JNP / 4; k += TPB_) reinterpret_cast<int4 *>(sJ)[k] = make_int4(0, 0, 0, 0);
    for (int k = tid; k < S::NKEYP; k += TPB_) hist[k] = 0;
    if (tid < 28) {
        M.cnt_in[tid] = 0; M.fill[tid] = 0; M.cnt2[tid] = 0; M.base_s[tid] = 0;
        int d = -1;
        if (tid < 27) {                                                  // destination tile of class (c0, c1, c2), -1 if it does not exist
            int rel = tid, tt[3] = { t0, t1, t2 }; bool ok = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                int v = tt[a] + rel % 3 - 1; rel /= 3;
                if (ALLPER || g.bc[a] == ENT_PERIODIC) { if (v < 0) v += g.nt[a]; if (v >= g.nt[a]) v -= g.nt[a]; }
                ok &= (v >= 0 && v < g.nt[a]);
                tt[a] = v;
            }
            if (ok) d = tt[0] + g.nt[0] * (tt[1] + g.nt[1] * tt[2]);
        }
        M.dest_s[tid] = d;
    }
    if (tid == 32) { M.wmaxbits = 0u; M.ovf_cnt = 0; M.nranked = 0; M.maxN = 0; }
    {   // the records the 16-byte aligned bulk copies cannot reach: the last (n mod 4) particles of the block
        long long ps = bulk_end > p0 ? bulk_end : p0;
        if (bulk_end <= pa) ps = p0;
        const long long p = ps + tid;
        if (tid < 8 && p < p1) {
            const int idx = (int)(p - pa);
            sP[0 * CAPP + idx] = __int_as_float(A.in.cell[p]);
#pragma unroll
            for (int a = 0; a < D; ++a) sP[(1 + a) * CAPP + idx] = A.in.d[a][p];
#pragma unroll
            for (int a = 0; a < 3; ++a) sP[(4 + a) * CAPP + idx] = A.in.u[a][p];
            sP[7 * CAPP + idx] = A.in.w[p];
        }
    }
    __syncthreads();
    mbar_wait(&M.bar, 0);

    // ---- P1: key, rank, destination class of every particle of the chunk
    unsigned kr[SORTED_ITEMS];                                            // bit 31 valid, bit 30 live, bits 10..29 rank, bits 0..9 key
    float wm = 0.f;
#pragma unroll
    for (int it = 0; it < SORTED_ITEMS; ++it) {
        const int k = tid + it * TPB_;
        kr[it] = 0u;
        int cls = -1;
        if (k < np) {
            const int idx = ioff + k;
            const int cell = __float_as_int(sP[idx]);
            int i[3];
            if (D == 2) { i[1] = A.divN0.div(cell); i[0] = cell - i[1] * g.N[0]; i[2] = 0; }
            else { i[2] = A.divN01.div(cell); int r = cell - i[2] * (g.N[0] * g.N[1]); i[1] = A.divN0.div(r); i[0] = r - i[1] * g.N[0]; }
            int b[3] = { i[0] - o[0] + 2, i[1] - o[1] + 2, (D == 3) ? i[2] - o[2] + 2 : 2 };
            bool local = true;
            int key = 0, kmul = 1;
            cls = 0;
            int cmul = 1;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (a < D) {
                    const int wrapN = (ALLPER || g.bc[a] == ENT_PERIODIC) ? g.N[a] : 0;
                    b[a] += (b[a] < 1) ? wrapN : 0;
                    b[a] -= (b[a] > g.N[a]) ? wrapN : 0;
                    local &= (unsigned)(b[a] - 1) < (unsigned)(te[a] + 2);
                    key += (b[a] - 1) * kmul; kmul *= TT[a] + 2;
                    cls += ((b[a] >= 2) + (b[a] >= te[a] + 2)) * cmul;
                } else cls += cmul;
                cmul *= 3;
            }
            const bool live = A.in.tag ? A.in.tag[p0 + k] != 0 : true;
            if (!local) { cls = -1; stray_sorted<D>(A, p0 + k); }
            else {
                const int rank = atomicAdd(&hist[key], 1);
                kr[it] = 0x80000000u | (live ? 0x40000000u : 0u) | ((unsigned)rank << 10) | (unsigned)key;
                if (live) wm = fmaxf(wm, fabsf(sP[7 * CAPP + idx]));
            }
        }
        const unsigned m13 = __ballot_sync(0xffffffffu, cls == 13);
        if (cls == 13) { if ((int)(__ffs(m13) - 1) == lane) atomicAdd(&M.cnt_in[13], __popc(m13)); }
        else if (cls >= 0) atomicAdd(&M.cnt_in[cls], 1);
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) wm = fmaxf(wm, __shfl_xor_sync(0xffffffffu, wm, s));
    if (lane == 0 && wm > 0.f) atomicMax(&M.wmaxbits, __float_as_uint(wm));
    __syncthreads();

    // ---- P2: rank-major order
    for (int chunk = warp; chunk < S::NW; chunk += NWARP) {
        const int cnt = hist[chunk * 32 + lane];
        unsigned mine = 0u;
#pragma unroll
        for (int r = 0; r < SORTED_RMAX; ++r) { const unsigned bb = __ballot_sync(0xffffffffu, cnt > r); if (lane == r) mine = bb; }
        if (lane < SORTED_RMAX) wp[lane * S::NW + chunk].x = mine;
    }
    if (tid < S::NROW) {                                                 // largest population of 4 consecutive cells of each x-row
        const int *h = hist + tid * S::HX;
        int best = 0, run = 0;
#pragma unroll
        for (int x = 0; x < S::HX; ++x) { run += h[x]; if (x >= 4) run -= h[x - 4]; best = max(best, run); }
        rowv[tid] = best;
    }
    if (tid < 27) { const int c = M.cnt_in[tid]; if (c > 0 && M.dest_s[tid] >= 0) M.base_s[tid] = atomicAdd(A.cursor + M.dest_s[tid], c); }
    __syncthreads();
    {
        constexpr int NENT = SORTED_RMAX * S::NW;
        int carry = 0;
        for (int b0 = 0; b0 < NENT; b0 += TPB_) {
            const int e = b0 + tid;
            const int v = e < NENT ? __popc(wp[e].x) : 0;
            int total;
            const int ex = block_scan_excl<TPB_>(v, M.wsum, total);
            if (e < NENT) wp[e].y = (unsigned)(carry + ex);
            carry += total;
        }
        if (tid == 0) M.nranked = carry;
        if (tid < S::NROW) {                                             // bound of the contributions one node can receive: 4^D cells
            const int y = tid % S::HY, z = tid / S::HY;
            int s = 0;
#pragma unroll
            for (int dz = -2; dz <= 1; ++dz)
#pragma unroll
                for (int dy = -2; dy <= 1; ++dy) {
                    if (D == 2 && dz != 0) continue;
                    const int yy = y + dy, zz = z + dz;
                    if (yy >= 0 && yy < S::HY && zz >= 0 && zz < S::HZ) s += rowv[yy + S::HY * zz];
                }
            atomicMax(&M.maxN, s);
        }
    }
    __syncthreads();
    const int nranked = M.nranked;
#pragma unroll
    for (int it = 0; it < SORTED_ITEMS; ++it) {
        if (!(kr[it] & 0x80000000u)) continue;
        const int key = kr[it] & 1023, rank = (kr[it] >> 10) & 0xFFFFF;
        int pos;
        if (rank < SORTED_RMAX) { const uint2 e = wp[rank * S::NW + (key >> 5)]; pos = (int)e.y + __popc(e.x & ((1u << (key & 31)) - 1u)); }
        else pos = nranked + atomicAdd(&M.ovf_cnt, 1);
        perm[pos] = (unsigned short)((ioff + tid + it * TPB_) | ((kr[it] & 0x40000000u) ? 0x8000 : 0));
    }
    // fixed-point scale of this CTA's J tile (header comment)
    float Sc, invSc;
    {
        const float wmx = __uint_as_float(M.wmaxbits);
        float rate = fminf(A.inv_dt, 1.02f * fmaxf(g.inv_dx[0], fmaxf(g.inv_dx[1], (D == 3) ? g.inv_dx[2] : 0.f)));   // |D_a| <= min(1, dt / dx_a)
        if (D == 2) rate = fmaxf(rate, 1.0f);                            // J^3 = q w v^3 (no 1/dt), both segments on one node
        const float amax = fabsf(A.q) * wmx * rate * 1.0834f;
        const int nb = max(1, min(np, M.maxN));
        const float cap = fminf(16777000.0f, 2.1e9f / (float)nb);
        Sc = (amax > 0.f && amax < 1e37f) ? cap / amax : 0.f;
        if (!(Sc > 1e-30f && Sc < 1e30f)) Sc = 0.f;
        invSc = Sc > 0.f ? 1.0f / Sc : 0.f;
    }
    __syncthreads();
    const int nvalid = nranked + M.ovf_cnt;

    // ---- P3: the particles in rank-major order
    const float sx[3] = { g.dx[0], g.dx[1], g.dx[2] };
    for (int j0 = warp * 32; j0 < nvalid; j0 += TPB_) {
        const int j = j0 + lane;
        const bool have = j < nvalid;
        int cls = -1, cls2 = -1, cell = 0;
        float d[3] = {0.f, 0.f, 0.f}, u[3] = {0.f, 0.f, 0.f}, wgt = 0.f;
        bool alive = false;
        if (have) {
            const unsigned pe = perm[j];
            const int idx = pe & 0x7FFF;
            const bool live = (pe & 0x8000u) != 0;
            cell = __float_as_int(sP[idx]);
            d[0] = sP[1 * CAPP + idx]; d[1] = sP[2 * CAPP + idx]; if (D == 3) d[2] = sP[3 * CAPP + idx];
            u[0] = sP[4 * CAPP + idx]; u[1] = sP[5 * CAPP + idx]; u[2] = sP[6 * CAPP + idx];
            wgt = sP[7 * CAPP + idx];
            // ---- where is the cell relative to the tile box?  b = cell index in box coordinates (box origin = o - 2)
            int i[3];
            if (D == 2) { i[1] = A.divN0.div(cell); i[0] = cell - i[1] * g.N[0]; i[2] = 0; }
            else { i[2] = A.divN01.div(cell); int r = cell - i[2] * (g.N[0] * g.N[1]); i[1] = A.divN0.div(r); i[0] = r - i[1] * g.N[0]; }
            const int iold[3] = { i[0], i[1], i[2] };
            int b[3] = { i[0] - o[0] + 2, i[1] - o[1] + 2, (D == 3) ? i[2] - o[2] + 2 : 0 };
            bool edge = false;
            cls = 0;
            {
                int cmul = 1;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    if (a < D) {
                        const int wrapN = (ALLPER || g.bc[a] == ENT_PERIODIC) ? g.N[a] : 0;
                        b[a] += (b[a] < 1) ? wrapN : 0;
                        b[a] -= (b[a] > g.N[a]) ? wrapN : 0;
                        cls += ((b[a] >= 2) + (b[a] >= te[a] + 2)) * cmul;
                        // un-wrapped cell N of a periodic dimension: a +1 crossing would deposit at node N + 2, outside the padded array
                        edge |= (o[a] - 2 + b[a] > g.N[a] - 1);
                    } else cls += cmul;
                    cmul *= 3;
                }
            }
            cls2 = cls;                                                   // a dead particle stays where it is
            alive = live;
            if (live) {
                // ---- S1 gather from the shared-memory box (same stencil and arithmetic as ent_dev.cuh gather)
                float EBv[6];
                {
                    int xs[2], ys[2], zs[2]; float fx[2], fy[2], fz[2];    // [0] node-centred, [1] half-shifted
                    { bool lo = d[0] < 0.5f; xs[0] = b[0]; xs[1] = lo ? b[0] - 1 : b[0]; fx[0] = d[0]; fx[1] = lo ? d[0] + 0.5f : d[0] - 0.5f; }
                    { bool lo = d[1] < 0.5f; ys[0] = b[1] * G::FX; ys[1] = lo ? ys[0] - G::FX : ys[0]; fy[0] = d[1]; fy[1] = lo ? d[1] + 0.5f : d[1] - 0.5f; }
                    if (D == 3) { bool lo = d[2] < 0.5f; zs[0] = b[2] * (G::FX * G::FY); zs[1] = lo ? zs[0] - G::FX * G::FY : zs[0]; fz[0] = d[2]; fz[1] = lo ? d[2] + 0.5f : d[2] - 0.5f; }
                    else { zs[0] = zs[1] = 0; fz[0] = fz[1] = 0.f; }
                    const f32x2 FX2[2] = { pk2(fx[0], fx[0]), pk2(fx[1], fx[1]) }, FY2[2] = { pk2(fy[0], fy[0]), pk2(fy[1], fy[1]) };
                    const int ST[6][3] = { {1,0,0}, {0,1,0}, {0,0,1}, {0,1,1}, {1,0,1}, {1,1,0} };
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        const float *Fc = sF + c * G::FNP + (xs[ST[c][0]] + ys[ST[c][1]] + zs[ST[c][2]]);
                        if (D == 3) {
                            const float *Fh = Fc + G::FX * G::FY;
                            const f32x2 P00 = pk2(Fc[0], Fh[0]), P10 = pk2(Fc[1], Fh[1]), P01 = pk2(Fc[G::FX], Fh[G::FX]), P11 = pk2(Fc[G::FX + 1], Fh[G::FX + 1]);
                            const f32x2 L0 = lerp2(P00, P10, FX2[ST[c][0]]), L1 = lerp2(P01, P11, FX2[ST[c][0]]);
                            float lo, hi;
                            upk2(lerp2(L0, L1, FY2[ST[c][1]]), lo, hi);
                            EBv[c] = lo + fz[ST[c][2]] * (hi - lo);
                        } else {
                            const f32x2 P0 = pk2(Fc[0], Fc[G::FX]), P1 = pk2(Fc[1], Fc[G::FX + 1]);
                            float l0, l1;
                            upk2(lerp2(P0, P1, FX2[ST[c][0]]), l0, l1);
                            EBv[c] = l0 + fy[ST[c][1]] * (l1 - l0);
                        }
                    }
                }
                // ---- S2 tetrad, S3 Boris (Eq. 3), S4-S5 move + crossing
                float E[3] = { sx[0] * EBv[0], sx[1] * EBv[1], sx[2] * EBv[2] }, B[3] = { sx[0] * EBv[3], sx[1] * EBv[4], sx[2] * EBv[5] };
                boris(u, E, B, A.eps);
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
                {   // class of the new cell (next step's layout)
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
                    if (edge) edge_deposit_sorted<D>(A, iold[0], iold[1], iold[2], a0[0], a0[1], a0[2], di[0], di[1], di[2], d[0], d[1], d[2], u[0], u[1], u[2], qw);
                    else {
                        // ---- S7 deposit into the shared-memory J tile (Eq. 6); node (b) of the box = element b of the J tile
                        const float Q = qw * A.inv_dt * Sc;                                  // in fixed-point units
                        // 3D: one straight segment unless a face is crossed.  2D: always the two segments of P:575 (the out-of-plane
                        // weights of two half segments do not sum to those of the whole one)
                        const bool cross = (D == 2) || (di[0] | di[1] | di[2]) != 0;
                        float s[3], e[3], r[3];
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            if (a < D) {
                                const float bnew = (float)di[a] + d[a];                      // new position in the old cell's frame
                                r[a] = di[a] == 0 ? (cross ? 0.5f * (a0[a] + bnew) : bnew) : (di[a] > 0 ? 1.0f : 0.0f);
                                s[a] = a0[a]; e[a] = r[a];
                            } else { r[a] = s[a] = e[a] = 0.f; }
                        }
                        int base = b[0] + G::JX * (b[1] + G::JY * b[2]);
                        const int dbase = di[0] + G::JX * (di[1] + G::JY * di[2]);
                        float hv = 0.f;
                        if (D == 2) hv = 0.5f * qw * Sc * (u[2] * ig);                       // out-of-plane rate per segment (G8), h33 = 1
                        const int nseg = cross ? 2 : 1;
#pragma unroll 1
                        for (int seg = 0; seg < nseg; ++seg) {
                            float Dv[3], W[3];
#pragma unroll
                            for (int a = 0; a < 3; ++a) { Dv[a] = e[a] - s[a]; W[a] = 0.5f * (e[a] + s[a]); }
                            if (D == 3) {
                                const int st[3] = { 1, G::JX, G::JX * G::JY };
#pragma unroll
                                for (int comp = 0; comp < 3; ++comp) {
                                    const int a = (comp + 1) % 3, bb = (comp + 2) % 3;
                                    const float c = Dv[a] * Dv[bb] * (1.0f / 12.0f);
                                    const float QD = Q * Dv[comp];
                                    const float w11 = W[a] * W[bb] + c, w10 = W[a] - w11, w01 = W[bb] - w11, w00 = 1.0f - W[a] - w01;
                                    int *Jc = sJ + comp * G::JNP + base;
                                    red_fixed(Jc, QD * w00); red_fixed(Jc + st[a], QD * w10);
                                    red_fixed(Jc + st[bb], QD * w01); red_fixed(Jc + st[a] + st[bb], QD * w11);
                                }
                            } else {
                                const float q0 = Q * Dv[0], q1 = Q * Dv[1];
                                const float h1 = hv * W[1], h0 = hv - h1;
                                int *J0 = sJ + base, *J1 = sJ + G::JNP + base, *J2 = sJ + 2 * G::JNP + base;
                                red_fixed(J0, q0 * (1.0f - W[1])); red_fixed(J0 + G::JX, q0 * W[1]);
                                red_fixed(J1, q1 * (1.0f - W[0])); red_fixed(J1 + 1, q1 * W[0]);
                                red_fixed(J2, h0 * (1.0f - W[0])); red_fixed(J2 + 1, h0 * W[0]);
                                red_fixed(J2 + G::JX, h1 * (1.0f - W[0])); red_fixed(J2 + G::JX + 1, h1 * W[0]);
                            }
#pragma unroll
                            for (int a = 0; a < 3; ++a) { s[a] = r[a] - (float)di[a]; e[a] = d[a]; }
                            base += dbase;
                        }
                    }
                }
            }
        }
        // ---- slot in `out`: the range of the tile of the INPUT cell (reserved in P2); particles that stay get consecutive slots
        const unsigned m13 = __ballot_sync(0xffffffffu, cls == 13);
        int r0 = 0;
        const int leader = __ffs(m13) - 1;
        if (m13 && lane == leader) r0 = atomicAdd(&M.fill[13], __popc(m13));
        r0 = __shfl_sync(0xffffffffu, r0, leader < 0 ? 0 : leader);
        // counts of the NEW tiles
        const unsigned n13 = __ballot_sync(0xffffffffu, cls2 == 13);
        if (cls2 == 13) { if ((int)(__ffs(n13) - 1) == lane) atomicAdd(&M.cnt2[13], __popc(n13)); }
        else if (cls2 >= 0 && cls2 < 27) atomicAdd(&M.cnt2[cls2], 1);
        else if (cls2 == 27) atomicAdd(A.next_count + tile_of_cell_slow<D>(g, cell), 1);
        if (!have) continue;
        long long slot;
        if (cls == 13) slot = (long long)M.base_s[13] + r0 + __popc(m13 & ((1u << lane) - 1u));
        else slot = (long long)M.base_s[cls] + atomicAdd(&M.fill[cls], 1);
        if (slot < 0 || slot >= A.n || M.dest_s[cls] < 0) { atomicAdd(A.counters + 3, 1ULL); continue; }
        A.out.cell[slot] = cell;
        A.out.d[0][slot] = d[0]; A.out.d[1][slot] = d[1]; if (D == 3) A.out.d[2][slot] = d[2];
        A.out.u[0][slot] = u[0]; A.out.u[1][slot] = u[1]; A.out.u[2][slot] = u[2];
        A.out.w[slot] = wgt;
        if (A.out.tag) A.out.tag[slot] = alive ? 1 : 0;
    }

    // ---- P4: counts of the next layout; S8 flush: one TMA reduce-add per component into the un-wrapped padded J (fold: P:642)
    __syncthreads();
    if (tid < 27 && M.cnt2[tid] > 0 && M.dest_s[tid] >= 0) atomicAdd(A.next_count + M.dest_s[tid], M.cnt2[tid]);
    for (int k = tid; k < 3 * G::JNP / 4; k += TPB_) {                    // fixed point -> fp32, in place
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
inline bool sorted_supported(const TiledState &t, const GridDev &g) { return g.kind == ENT_CART && (t.shape == 0 || t.shape == 2); }

template <int D, int TX, int TY, int TZ>
inline int sorted_launch(TiledState &t, int attr_slot, const SortedArgs &A, cudaStream_t stream, char *err, size_t errn) {
    using S = SortedGeom<D, TX, TY, TZ>;
    int rc = tiled_encode<D, TX, TY, TZ>(t, A.g, A.F, A.J, err, errn);
    if (rc) return rc;
    bool allper = true;
    for (int a = 0; a < D; ++a) allper &= A.g.bc[a] == ENT_PERIODIC;
    void (*kern)(const TileMaps, const SortedArgs) = allper ? step_sorted_kernel<D, TX, TY, TZ, true> : step_sorted_kernel<D, TX, TY, TZ, false>;
    const int slot = attr_slot + (allper ? 1 : 0);
    if (!t.attr_set[slot]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_BYTES);
        if (e != cudaSuccess) { snprintf(err, errn, "cudaFuncSetAttribute(smem %d) failed: %s", S::SMEM_BYTES, cudaGetErrorString(e)); return ENT_ECUDA; }
        t.attr_set[slot] = true;
    }
    const long long grid = (long long)A.ntiles + A.n / SORTED_CAP + 1;        // upper bound of the number of chunks
    kern<<<(unsigned)grid, SORTED_TPB, S::SMEM_BYTES, stream>>>(t.maps, A);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { snprintf(err, errn, "launch of step_sorted_kernel failed: %s", cudaGetErrorString(e)); return ENT_ECUDA; }
    return ENT_OK;
}

inline int sorted_step(TiledState &t, SortedArgs &A, float dt, cudaStream_t stream, char *err, size_t errn) {
    for (int a = 0; a < 3; ++a) A.cdt[a] = dt * A.g.inv_dx[a];
    A.divN0 = make_magicdiv((uint32_t)A.g.N[0]);
    A.divN01 = make_magicdiv((uint32_t)(A.g.N[0] * A.g.N[1]));
    A.ntiles = A.g.nt[0] * A.g.nt[1] * A.g.nt[2];
    if (t.shape == 0) return sorted_launch<3, 8, 8, 4>(t, 8, A, stream, err, errn);
    if (t.shape == 2) return sorted_launch<2, 16, 16, 1>(t, 10, A, stream, err, errn);
    snprintf(err, errn, "no fused step + re-bin kernel for this tile shape");
    return ENT_EUNSUPPORTED;
}

}  // namespace ent
