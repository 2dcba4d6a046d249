// em_fused.cuh -- the fused sweep (EM_KERNEL_FUSED): ONE kernel per time step does
//   a1 H update, a2 E update, a3 source injection, a4 Joule accumulation, a5 PEC masks
// (eq. (2)-(3) L69-L76 in leapfrog form, L86 for the Joule heat) and moves
// each field value through HBM once per step: reads E^n, H^{n-1/2}, ids, q; writes E^{n+1},
// H^{n+1/2}, q  ->  12 words + 1 B + 2 words = 57 B (fp32) / 113 B (fp64) per cell-update.
//
// Decomposition:
//  * E and H are ping-ponged (read buffer / write buffer), so tiles never race on halos.
//  * A CTA owns TXo x TY columns (x,y) and marches all z planes k = 0..nz.  Warp w handles the
//    row cy = w-1 in [-1, TY]; a lane handles V = 16 B / sizeof(R) consecutive x columns with
//    128-bit accesses.  Lanes 0 and 31 and the rows -1 and TY are the recompute halo (H' is needed
//    at -1 for E', E' at +1 for the Joule cell sum), so TXo = 30 V and the CTA has TY+2 warps.
//  * x neighbours come from warp shuffles, y neighbours from shared-memory rows (128-bit,
//    conflict-free), z neighbours are carried in registers or in a private shared-memory spill.
//  * The next plane's inputs are prefetched with cp.async (LDGSTS, L2-only) into private
//    shared-memory slots one iteration ahead; stores are plain 128-bit STG of fully written sectors.
//  * Coefficients are rebuilt from the uint8 material ids through the shared-memory table every
//    step (bilinear = area-weighted mean, one reciprocal per edge), never stored per edge.
#pragma once
#include "em_aux.cuh"
#include "em_common.cuh"
#include <algorithm>
#include <type_traits>

namespace em {

#define EM_ST(ptr, val) (*reinterpret_cast<VecR *>(ptr) = (val))     // output stores of the phase-B includes

#ifndef EM_FUSED_TY
#define EM_FUSED_TY 14
#endif
#ifndef EM_FUSED_OCC
#define EM_FUSED_OCC 1
#endif
#ifndef EM_FUSED_TY64
#define EM_FUSED_TY64 10
#endif
constexpr int kFusedOcc = EM_FUSED_OCC;             // resident CTAs per SM
// Tile rows per working precision.  fp32: 14 owned rows = 16 warps x 128 registers.  fp64 needs ~170 registers per
// thread to stay spill-free (a spill is very expensive here: the 227 KB carve-out leaves almost no L1), so its tiles
// own 10 rows = 12 warps (measured on config 3 fp64: 1.22 -> 0.87 ms/step).
// TH = the thermally coupled sweep (em_sweep.cuh, sigma(T) planes + theta in the sweep): it also takes the 10-row tile
// (room in registers and shared memory for the extra state).
template <int SZ, bool TH = false> struct Tile {
    static constexpr int TY = (SZ == 8 || TH) ? EM_FUSED_TY64 : EM_FUSED_TY;   // owned rows per tile
    static constexpr int warps = TY + 2;                                // rows -1 .. TY
    static constexpr int threads = warps * 32;
    static constexpr int rows = TY + 4;                                 // exchange rows, r = cy + 2 (row 0 and last: dummies)
};
inline int tile_rows(int sizeof_real, bool thermal = false) { return (sizeof_real == 8 || thermal) ? Tile<8>::TY : Tile<4>::TY; }
constexpr int kFusedSlots = 21;                    // private 16-B slots per thread (see enum below)

constexpr int kFusedMaxZSplit = 8;                // z chunks per tile column (work items = tiles x chunks)

struct FusedPlan {
    int V, TXo, TY, ntx, nty, n_tiles;
    int nzs;                         // z chunks; chunk c owns the planes kb[c] <= k < kb[c+1], kb[nzs] = nz+1
    int kb[kFusedMaxZSplit + 1];
    size_t smem_bytes;
    int chunk_of(int k) const { int c = 0; while (c + 1 < nzs && k >= kb[c + 1]) ++c; return c; }
};

// Number of z chunks.  Work items are scheduled dynamically onto the SMs, so the step takes about
//   total work / n_sm  +  one item (the tail),   work of an item = its planes + ~4 planes of overhead
// (the re-run warm-up and closing planes of a chunk plus the prologue and the pipeline fill).  Fitted on B200:
// config 4 (666 tiles x 193 planes) -> 3, config 5 (385 x 257) -> 5, config 3 (185 x 129) -> 5, which are the
// measured optima (profiles/r1_configs.md).  n_sm = 0 (no device known yet: workspace sizing) returns the maximum.
inline int choose_zsplit(int n_tiles, int nz, int n_sm, int forced) {
    const int cap = std::max(1, std::min(kFusedMaxZSplit, (nz + 1) / 4));
    if (forced > 0) return std::min(forced, cap);
    if (n_sm <= 0) return kFusedMaxZSplit;
    int best = 1; double best_cost = 1e300;
    for (int s = 1; s <= cap; ++s) {
        const double over = s > 1 ? 4.0 : 0.0;
        const double item = (double)(nz + 1) / s + over;
        const double cost = (double)n_tiles * s * item / n_sm + item;
        if (cost < best_cost * 0.999) { best_cost = cost; best = s; }
    }
    return best;
}

inline FusedPlan make_fused_plan(int nx, int ny, int nz, int sizeof_real, int n_sm = 0, int forced_zsplit = 0,
                                 bool thermal = false) {
    FusedPlan f;
    f.V = 16 / sizeof_real;
    f.TXo = 30 * f.V;
    f.ntx = (nx + 1 + f.TXo - 1) / f.TXo;
    f.TY = tile_rows(sizeof_real, thermal);
    const int kFusedRows = f.TY + 4, kFusedThreads = (f.TY + 2) * 32;
    f.nty = (ny + 1 + f.TY - 1) / f.TY;
    f.n_tiles = f.ntx * f.nty;
    f.nzs = choose_zsplit(f.n_tiles, nz, n_sm * kFusedOcc, forced_zsplit);
    for (int c = 0; c <= kFusedMaxZSplit; ++c) f.kb[c] = nz + 1;
    for (int c = 0; c < f.nzs; ++c) f.kb[c] = (int)(((long long)(nz + 1) * c) / f.nzs);
    const size_t table = (size_t)kMaxTable * 4 * sizeof_real;
    const size_t rows = (size_t)4 * kFusedRows * 32 * 16;                 // H'x, H'z, Bx, Bz exchange rows
    const size_t slots = (size_t)kFusedSlots * kFusedThreads * 16;        // private slots
    const size_t extra = (size_t)(4 + 3) * 32 * 16 + 64 + (size_t)2 * kFusedRows * 32 * 4;   // top row (2 parities), x geometry, ids (2 parities)
    f.smem_bytes = table + rows + slots + extra;
    return f;
}

// Tiles that compute E' at node (i,j): the owner and, for nodes on a tile's low border, the
// neighbour(s) that recompute it as their +1 halo.  Returns the count (<= 4).
inline int tiles_of_node(const FusedPlan &f, int i, int j, int out[4]) {
    int txs[2], tys[2], nxs = 0, nys = 0;
    txs[nxs++] = i / f.TXo;
    if (i % f.TXo == 0 && i > 0) txs[nxs++] = i / f.TXo - 1;
    tys[nys++] = j / f.TY;
    if (j % f.TY == 0 && j > 0) tys[nys++] = j / f.TY - 1;
    int n = 0;
    for (int a = 0; a < nys; ++a)
        for (int b = 0; b < nxs; ++b)
            if (txs[b] < f.ntx && tys[a] < f.nty) out[n++] = tys[a] * f.ntx + txs[b];
    return n;
}

template <typename R> struct alignas(16) Vec { R v[16 / sizeof(R)]; };

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename R> __device__ __forceinline__ R shfl_up1(R v)   { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename R> __device__ __forceinline__ R shfl_down1(R v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// Fused-sweep source index (built by em_set_source): entries of tile t are
// tile_ent[tile_sbeg[t] .. tile_sbeg[t+1]) sorted by (k, j, i); ent = {i, j, k, u*4 + comp}.
struct FusedSources {
    const int *tile_sbeg;     // indexed by work item = tile * nzs + chunk (entries of a tile are sorted by k)
    const int4 *tile_ent;
};

// z chunks of the sweep (FusedPlan::kb), passed by value
struct FusedChunks {
    int nzs;
    int kb[kFusedMaxZSplit + 1];
};

// Private shared-memory slots of a thread (16 B each, [slot][tid], so slot rows of the neighbouring
// warps are directly readable as the y-neighbours of the staged inputs).
enum : int {
    kSlotEx = 0,    // ring of 3: Ex planes k, k+1, k+2
    kSlotEy = 3,    // ring of 3
    kSlotEz = 6,    // ring of 2: Ez layers k, k+1
    kSlotH = 8,     // Hx, Hy, Hz of layer k (old)
    kSlotQ = 11,    // q of layer k-1
    kSlotL = 12,    // Ly(a,b,m), Lx(a,b,m) of plane k-1 (coefficient partial means)
    kSlotHp = 18,   // Hx', Hy' of layer k-1
    kSlotPend = 20, // Joule partial sum of layer k-1
    kNumSlots = 21
};

template <typename R, int LOSS, bool UMU>
__global__ void __launch_bounds__(Tile<sizeof(R)>::threads, kFusedOcc)
k_fused_sweep(DevParams<R> p, DevSources<R> src, FusedSources fs, FusedChunks zc, int ntx, long long step) {
    constexpr int V = 16 / sizeof(R);
    constexpr int TXo = 30 * V;
    constexpr int kFusedTY = Tile<sizeof(R)>::TY, kFusedRows = Tile<sizeof(R)>::rows;
    constexpr int NT = Tile<sizeof(R)>::threads;
    using VecR = Vec<R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    MatEntry<R> *s_tab = reinterpret_cast<MatEntry<R> *>(smem_raw);
    VecR *s_rows = reinterpret_cast<VecR *>(smem_raw + (size_t)kMaxTable * sizeof(MatEntry<R>));
    VecR(*smHx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 0 * kFusedRows * 32);
    VecR(*smHz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 1 * kFusedRows * 32);
    VecR(*smBx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 2 * kFusedRows * 32);
    VecR(*smBz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 3 * kFusedRows * 32);
    VecR *S = s_rows + 4 * kFusedRows * 32;                   // private slots [kNumSlots][NT]
    VecR *s_top = S + kNumSlots * NT;                         // [2 parity][2][32]: Ex(k), Ez(k) of row TY+1
    VecR *s_geo = s_top + 128;                                // [3][32]: 1/dx, 1/dx~, fx of the lanes' columns
    R *s_z = reinterpret_cast<R *>(s_geo + 96);               // [2 parity][4]: fz, 1/dz, 1/dz~ of plane k
    unsigned(*smId)[32] = reinterpret_cast<unsigned(*)[32]>(s_geo + 96 + 4);   // [2 parity][kFusedRows][32]

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    // work item = (tile, z chunk); chunk c stores the planes kz0 <= k < kz1 and the q layers of the same
    // range; it starts one plane lower (warm-up: H'(kz0-1), the coefficient means and the ids of plane
    // kz0-1, nothing stored) and ends on plane ke = kz1 (E'(kz1) closes the Joule sum of layer kz1-1).
    const int item = blockIdx.x, tile = item / zc.nzs, chunk = item - tile * zc.nzs;
    const int tx = tile % ntx, ty = tile / ntx;
    const int kz0 = zc.kb[chunk], kz1 = zc.kb[chunk + 1];
    const int ks = (kz0 > 0 || p.warm_lo) ? kz0 - 1 : 0, ke = kz1 <= p.nz ? kz1 : p.nz;   // PMC at -z: plane -1 warms up too
    const int cy = w - 1, r = cy + 2;
    const int j = ty * kFusedTY + cy;
    const int i0 = tx * TXo - V + V * lane;
    const int ny = p.ny, nz = p.nz;
    const long long PX = p.PX, PXY = p.PXY;
    const bool is_top = (cy == kFusedTY);
    const bool active = (j <= ny + 1) && (i0 + V <= p.PX);
    const bool top_row_ok = is_top && active && (j + 1 <= ny + 1);
    const bool own = active && lane >= 1 && lane <= 30 && cy >= 0 && cy < kFusedTY && j <= ny;
    const bool own_q = own && j < ny;
    const int out_id = p.n_table - 1;                 // the "outside" entry
    const unsigned out_pack = (unsigned)out_id * 0x01010101u;

    // ---- prologue: table, zeroed rows and slots, coefficient means of the (outside) plane k = -1 --
    for (int t = tid; t < p.n_table; t += NT) s_tab[t] = p.table[t];
    {
        VecR z, one;
#pragma unroll
        for (int c = 0; c < V; ++c) { z.v[c] = R(0); one.v[c] = R(1); }
        for (int t = tid; t < 4 * kFusedRows * 32; t += NT) s_rows[t] = z;
        for (int t = 0; t < kNumSlots; ++t) S[t * NT + tid] = z;
        S[(kSlotL + 0) * NT + tid] = one; S[(kSlotL + 3) * NT + tid] = one;
        if (tid < 128) s_top[tid] = z;
        if (tid < 96) s_geo[tid] = z;
        for (int t = tid; t < 2 * kFusedRows * 32; t += NT) (&smId[0][0])[t] = out_pack;
    }
    __syncthreads();

    const R fy = active ? p.fy[j] : R(0), rdy = active ? p.rdy[j] : R(0), rty = active ? p.rty[j] : R(0);
    const R gq = p.dt * R(0.0625);
    const long long off0 = (long long)j * PX + i0;    // this thread's vector at plane 0
    auto ldv = [&](const R *a, long long off) -> VecR { return *reinterpret_cast<const VecR *>(a + off); };
    // ids travel as one aligned 32-bit word per lane (V = 4: exactly the lane's ids; V = 2: the
    // lane's two ids are the low or high half, selected by id_shift)
    const int id_shift = (V == 4) ? 0 : (int)((off0 & 2) * 8);
    auto id_src = [&](long long off) -> const uint8_t * { return p.mat + ((off) & ~3LL); };
    auto id_unpack = [&](unsigned wv) -> unsigned { return (V == 4) ? wv : ((wv >> id_shift) & 0xffffu) | (out_pack & 0xffff0000u); };
    // all V cells of an unpacked id word hold the same material
    auto id_uniform = [&](unsigned wv) -> bool { return (V == 4) ? (wv == (wv & 0xffu) * 0x01010101u) : (((wv >> 8) & 0xffu) == (wv & 0xffu)); };
    VecR *mine = S + tid;
    // x geometry of the 32 lanes of this tile column (same for every row of the CTA)
    if (w == 0 && (i0 + V <= p.PX)) {
        s_geo[0 * 32 + lane] = ldv(p.rdx, i0); s_geo[1 * 32 + lane] = ldv(p.rtx, i0); s_geo[2 * 32 + lane] = ldv(p.fx, i0);
    }

    // cp.async groups (every thread commits the same sequence):
    //   G_E(k): inputs of iteration k that the neighbours also read: Ex(k+1), Ey(k+1) -> ring slot
    //           (k+1)%3, Ez(k) -> parity slot, row TY+1 for the top warp; issued in phase C(k-2)
    //   G_H(k): H(k), own use only; issued at the end of phase A(k-1)
    //   G_q(k): q(k) for phase C(k+1); issued in phase C(k)
    // issue order per iteration k: G_H(k+1) | G_q(k), G_E(k+2)
    auto issue_E = [&](int kk, int ring, int par) {
        if (active && kk <= ke) {
            const long long o = off0 + (long long)kk * PXY;
            cp_async16(mine + (kSlotEx + ring) * NT, p.E[0] + o + PXY);
            cp_async16(mine + (kSlotEy + ring) * NT, p.E[1] + o + PXY);
            cp_async16(mine + (kSlotEz + par) * NT, p.E[2] + o);
            cp_async4(&smId[par * kFusedRows + r][lane], id_src(o));
            if (top_row_ok) {
                cp_async16(s_top + par * 64 + lane, p.E[0] + o + PX);
                cp_async16(s_top + par * 64 + 32 + lane, p.E[2] + o + PX);
            }
        }
        if (tid < (int)sizeof(R) / 4 && kk <= ke)   // z geometry of plane kk: {fz, 1/dz, 1/dz~, 0}
            cp_async16(reinterpret_cast<unsigned char *>(&s_z[par * 4]) + 16 * tid,
                       reinterpret_cast<const unsigned char *>(p.zgeo + 4 * (long long)kk) + 16 * tid);
        cp_async_commit();
    };
    auto issue_H = [&](int kk) {
        if (active && kk <= ke) {
            const long long o = off0 + (long long)kk * PXY;
            cp_async16(mine + (kSlotH + 0) * NT, p.H[0] + o);
            cp_async16(mine + (kSlotH + 1) * NT, p.H[1] + o);
            cp_async16(mine + (kSlotH + 2) * NT, p.H[2] + o);
        }
        cp_async_commit();
    };
    unsigned idw_prev = out_pack;
    bool rowu_prev = false;      // plane k-1: rows j-1 and j of this lane held one material
    bool l_stale = false;        // warp-uniform: the L slots were skipped by the one-material path
    bool q_live = false;         // q of layer k-1 was fetched (some sigma != 0 among the lane's cells)
    int rk = (ks + 3) % 3;                            // k % 3
    if (active) {
        cp_async16(mine + (kSlotEx + rk) * NT, p.E[0] + off0 + (long long)ks * PXY);   // plane ks into ring slot ks%3
        cp_async16(mine + (kSlotEy + rk) * NT, p.E[1] + off0 + (long long)ks * PXY);
    }
    issue_E(ks, (rk + 1) % 3, ks & 1);            // G_E(ks)
    issue_H(ks);                                  // G_H(ks)
    cp_async_commit();                            // G_q(ks-1), empty
    issue_E(ks + 1, (rk + 2) % 3, (ks + 1) & 1);  // G_E(ks+1)
    cp_async_wait<3>();                           // G_E(0) has landed
    __syncthreads();

    // source cursor: starts at the tile's first entry with k >= kz0 and may run into the next chunk's
    // entries on the closing plane k = kz1 (E'(kz1) enters the Joule sum of layer kz1-1)
    int s_cur = fs.tile_sbeg[item];
    const int s_end = fs.tile_sbeg[(tile + 1) * zc.nzs];
    int s_next_k = (s_cur < s_end) ? fs.tile_ent[s_cur].z : 0x7fffffff;

    for (int k = ks; k <= ke; ++k) {
        const int rk1 = (rk == 2) ? 0 : rk + 1;
        const int par = k & 1;
        const long long o = off0 + (long long)k * PXY;
        const bool st = own && k >= kz0 && k < kz1;          // this chunk stores H'(k), E'(k)
        const R fz = s_z[par * 4 + 0], rdz = s_z[par * 4 + 1], rtz = s_z[par * 4 + 2];

        // ---- phase A: H' = H - nbar * curl E  (inner factor of S = curl mu^-1 curl) ----
        cp_async_wait<2>();                       // G_H(k) has landed
        const unsigned idw = id_unpack(smId[par * kFusedRows + r][lane]);
        const unsigned idj = id_unpack(smId[par * kFusedRows + r - 1][lane]);
        // one material over the warp's whole coefficient neighbourhood (rows j-1..j, planes k-1..k)?
        const bool rowu = (idw == idj) && id_uniform(idw);
        const unsigned idw_lane0 = __shfl_sync(0xffffffffu, idw, 0);     // (not inside the && chain: every lane must execute it)
        const bool hom = __all_sync(0xffffffffu, rowu && rowu_prev && idw == idw_prev && idw == idw_lane0);
        VecR hxn, hyn, hzn;
        const VecR ex0 = mine[(kSlotEx + rk) * NT], ey0 = mine[(kSlotEy + rk) * NT], ez = mine[(kSlotEz + par) * NT];
        {
            const VecR ex1 = mine[(kSlotEx + rk1) * NT], ey1 = mine[(kSlotEy + rk1) * NT];
            const VecR hx = mine[(kSlotH + 0) * NT], hy = mine[(kSlotH + 1) * NT], hz = mine[(kSlotH + 2) * NT];
            const VecR exn = is_top ? s_top[par * 64 + lane] : mine[(kSlotEx + rk) * NT + 32];
            const VecR ezn = is_top ? s_top[par * 64 + 32 + lane] : mine[(kSlotEz + par) * NT + 32];
            const R ey0_r = shfl_down1(ey0.v[0]), ez_r = shfl_down1(ez.v[0]);
            const VecR rdxv = s_geo[0 * 32 + lane];
            VecR nbx, nby, nbz;
            if (UMU) {
                const R n0 = s_tab[0].n;
#pragma unroll
                for (int c = 0; c < V; ++c) nbx.v[c] = nby.v[c] = nbz.v[c] = n0;
            } else {
                const VecR fxv = s_geo[2 * 32 + lane];
                R ncur[V];
#pragma unroll
                for (int c = 0; c < V; ++c) ncur[c] = s_tab[(idw >> (8 * c)) & 0xff].n;
                const R n_l = shfl_up1(ncur[V - 1]);
#pragma unroll
                for (int c = 0; c < V; ++c) {
                    const R nj = s_tab[(idj >> (8 * c)) & 0xff].n;
                    const R nk = s_tab[(idw_prev >> (8 * c)) & 0xff].n;
                    nbx.v[c] = lerp(c > 0 ? ncur[c > 0 ? c - 1 : 0] : n_l, ncur[c], fxv.v[c]);
                    nby.v[c] = lerp(nj, ncur[c], fy);
                    nbz.v[c] = lerp(nk, ncur[c], fz);
                }
            }
#pragma unroll
            for (int c = 0; c < V; ++c) {
                const R eyip = (c < V - 1) ? ey0.v[c < V - 1 ? c + 1 : c] : ey0_r;
                const R ezip = (c < V - 1) ? ez.v[c < V - 1 ? c + 1 : c] : ez_r;
                hxn.v[c] = hx.v[c] - nbx.v[c] * ((ezn.v[c] - ez.v[c]) * rdy - (ey1.v[c] - ey0.v[c]) * rdz);
                hyn.v[c] = hy.v[c] - nby.v[c] * ((ex1.v[c] - ex0.v[c]) * rdz - (ezip - ez.v[c]) * rdxv.v[c]);
                hzn.v[c] = hz.v[c] - nbz.v[c] * ((eyip - ey0.v[c]) * rdxv.v[c] - (exn.v[c] - ex0.v[c]) * rdy);
            }
        }
        if (!active) {
#pragma unroll
            for (int c = 0; c < V; ++c) hxn.v[c] = hyn.v[c] = hzn.v[c] = R(0);
        }
        if (st) {
            *reinterpret_cast<VecR *>(p.Hn[0] + o) = hxn;
            *reinterpret_cast<VecR *>(p.Hn[1] + o) = hyn;
            *reinterpret_cast<VecR *>(p.Hn[2] + o) = hzn;
        }
        smHx[r][lane] = hxn; smHz[r][lane] = hzn;
        issue_H(k + 1);                           // G_H(k+1): the H slots are free again
        __syncthreads();                          // B2: H' rows visible

        // ---- phase B: E' = E + r (curl H' - J - sigma E), Joule squares (eq. 2-3) -------
        // (warp 0 = halo row -1 only supplies H' to row 0: no E', no Joule)
        VecR bx, by, bz;         // (2 Ebar)^2
        if (w != 0) {
            if (hom && s_next_k > k) {
#include "em_fused_phaseb_hom.inc"
                l_stale = true;
            } else {
                if (l_stale) {   // plane k-1 took the one-material path: its coefficient means are the entry itself
                    const MatEntry<R> Ap = s_tab[idw_prev & 0xff];
                    VecR va, vb, vm;
#pragma unroll
                    for (int c = 0; c < V; ++c) { va.v[c] = Ap.a; vb.v[c] = Ap.b; vm.v[c] = Ap.m * Ap.m; }
                    mine[(kSlotL + 0) * NT] = va; mine[(kSlotL + 1) * NT] = vb; mine[(kSlotL + 2) * NT] = vm;
                    mine[(kSlotL + 3) * NT] = va; mine[(kSlotL + 4) * NT] = vb; mine[(kSlotL + 5) * NT] = vm;
                    l_stale = false;
                }
                if (s_next_k <= k) {
#define EM_HAS_J 1
#include "em_fused_phaseb.inc"
#undef EM_HAS_J
                    s_next_k = (s_cur < s_end) ? fs.tile_ent[s_cur].z : 0x7fffffff;
                } else {
#define EM_HAS_J 0
#include "em_fused_phaseb.inc"
#undef EM_HAS_J
                }
            }
            if (!active) {
#pragma unroll
                for (int c = 0; c < V; ++c) bx.v[c] = by.v[c] = bz.v[c] = R(0);
            }
            smBx[r][lane] = bx; smBz[r][lane] = bz;
            mine[(kSlotHp + 0) * NT] = hxn; mine[(kSlotHp + 1) * NT] = hyn;
        }
        cp_async_wait<1>();                       // G_E(k+1) (and G_q(k-1)) have landed
        __syncthreads();                          // B3: B rows, next inputs and ids visible

        // ---- phase C: q(k-1) += dt sigma/16 (pend + Sxy(k)); pend = Sxy(k) + Sz(k) ---------------------
        if (w != 0 && !is_top) {
            const VecR bxn = smBx[r + 1][lane], bzn = smBz[r + 1][lane];
            const R by_r = shfl_down1(by.v[0]), bz_r = shfl_down1(bz.v[0]), bzn_r = shfl_down1(bzn.v[0]);
            VecR qv = mine[kSlotQ * NT];
            VecR pend = mine[kSlotPend * NT];
#pragma unroll
            for (int c = 0; c < V; ++c) {
                const R byip = (c < V - 1) ? by.v[c < V - 1 ? c + 1 : c] : by_r;
                const R bzip = (c < V - 1) ? bz.v[c < V - 1 ? c + 1 : c] : bz_r;
                const R bznip = (c < V - 1) ? bzn.v[c < V - 1 ? c + 1 : c] : bzn_r;
                const R sxy = (bx.v[c] + bxn.v[c]) + (by.v[c] + byip);
                const R sz = (bz.v[c] + bzip) + (bzn.v[c] + bznip);
                const R sg = s_tab[(idw_prev >> (8 * (hom ? 0 : c))) & 0xff].b;     // sigma of the cell of layer k-1
                qv.v[c] = mad(gq * sg, pend.v[c] + sxy, qv.v[c]);
                pend.v[c] = sxy + sz;
            }
            mine[kSlotPend * NT] = pend;
            // q of a lane whose V cells are one lossless material never changes: neither fetched nor stored
            if (own_q && k > kz0 && q_live) *reinterpret_cast<VecR *>(p.q + o - PXY) = qv;   // layer k-1 in [kz0, kz1)
            q_live = !(id_uniform(idw) && s_tab[idw & 0xff].b == R(0));
            if (own_q && k >= kz0 && k < ke && q_live) cp_async16(mine + kSlotQ * NT, p.q + o);   // G_q(k)
        }
        cp_async_commit();
        issue_E(k + 2, rk, par);                  // G_E(k+2): ring slot k%3 and parity k&1 are dead now
        idw_prev = idw;
        rowu_prev = rowu;
        rk = rk1;
    }
    cp_async_wait<0>();
}

template <typename R>
cudaError_t launch_fused(const FusedPlan &plan, const DevParams<R> &p, const DevSources<R> &src,
                         const FusedSources &fs, int loss, bool uniform_mu, long long step, cudaStream_t stream) {
    using K = void (*)(DevParams<R>, DevSources<R>, FusedSources, FusedChunks, int, long long);
    FusedChunks zc;
    zc.nzs = plan.nzs;
    for (int c = 0; c <= kFusedMaxZSplit; ++c) zc.kb[c] = plan.kb[c];
    K kern;
    if (loss == 0) kern = uniform_mu ? (K)k_fused_sweep<R, 0, true> : (K)k_fused_sweep<R, 0, false>;
    else           kern = uniform_mu ? (K)k_fused_sweep<R, 1, true> : (K)k_fused_sweep<R, 1, false>;
    static thread_local const void *configured[8] = {};
    bool done = false;
    for (auto c : configured) if (c == (const void *)kern) done = true;
    if (!done) {
        cudaError_t e = cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes);
        if (e != cudaSuccess) return e;
        for (auto &c : configured) if (!c) { c = (const void *)kern; break; }
    }
    kern<<<plan.n_tiles * plan.nzs, Tile<sizeof(R)>::threads, plan.smem_bytes, stream>>>(p, src, fs, zc, plan.ntx, step);
    return cudaGetLastError();
}

}  // namespace em
