// em_tile.cuh -- tile geometry and work decomposition of the sweep kernels (em_sweep.cuh), shared by the host side
// (plan, per-tile source index) and the device side (small PTX helpers).
//
// Decomposition:
//  * E and H are ping-ponged (read buffer / write buffer), so tiles never race on halos.
//  * A CTA owns TXo x TY columns (x, y) and marches the z planes of its chunk.  Warp w handles the row cy = w-1 in
//    [-1, TY]; a lane handles V = 16 B / sizeof(R) consecutive x columns with 128-bit accesses.  Lanes 0 and 31 and the
//    rows -1 and TY are the recompute halo (H' is needed at -1 for E', E' at +1 for the Joule cell sum), so TXo = 30 V
//    and the CTA has TY+2 warps.
//  * x neighbours come from warp shuffles, y neighbours from shared-memory rows (128-bit, conflict-free), z neighbours
//    are carried in private shared-memory slots.
//  * Coefficients are rebuilt from the uint8 material ids through the shared-memory table every step (bilinear =
//    area-weighted mean, one reciprocal per edge), never stored per edge.
#pragma once
#include "em_aux.cuh"
#include "em_common.cuh"
#include <algorithm>
#include <type_traits>

namespace em {

#ifndef EM_SWEEP_TY
#define EM_SWEEP_TY 14
#endif
#ifndef EM_SWEEP_OCC
#define EM_SWEEP_OCC 1
#endif
#ifndef EM_SWEEP_TY64
#define EM_SWEEP_TY64 10
#endif
constexpr int kSweepOcc = EM_SWEEP_OCC;             // resident CTAs per SM
// Tile rows per working precision.  fp32: 14 owned rows = 16 warps x 128 registers.  fp64 needs ~170 registers per
// thread to stay spill-free (a spill is very expensive here: the 227 KB carve-out leaves almost no L1), so its tiles
// own 10 rows = 12 warps (measured on config 3 fp64: 1.22 -> 0.87 ms/step).
// TH = the thermally coupled sweep (em_sweep.cuh, sigma(T) planes + theta in the sweep): it also takes the 10-row tile
// (room in registers and shared memory for the extra state).
template <int SZ, bool TH = false> struct Tile {
    static constexpr int TY = (SZ == 8 || TH) ? EM_SWEEP_TY64 : EM_SWEEP_TY;   // owned rows per tile
    static constexpr int warps = TY + 2;                                // rows -1 .. TY
    static constexpr int threads = warps * 32;
    static constexpr int rows = TY + 4;                                 // exchange rows, r = cy + 2 (row 0 and last: dummies)
};
inline int tile_rows(int sizeof_real, bool thermal = false) { return (sizeof_real == 8 || thermal) ? Tile<8>::TY : Tile<4>::TY; }

constexpr int kSweepMaxZSplit = 8;                // z chunks per tile column (work items = tiles x chunks)

struct SweepPlan {
    int V, TXo, TY, ntx, nty, n_tiles;
    int nzs;                         // z chunks; chunk c owns the planes kb[c] <= k < kb[c+1], kb[nzs] = nz+1
    int kb[kSweepMaxZSplit + 1];
    int chunk_of(int k) const { int c = 0; while (c + 1 < nzs && k >= kb[c + 1]) ++c; return c; }
};

// Number of z chunks.  Work items are scheduled dynamically onto the SMs, so the step takes about
//   total work / n_sm  +  one item (the tail),   work of an item = its planes + ~4 planes of overhead
// (the re-run warm-up and closing planes of a chunk plus the prologue and the pipeline fill).  Fitted on B200:
// config 4 (666 tiles x 193 planes) -> 3, config 5 (385 x 257) -> 5, config 3 (185 x 129) -> 5, which are the
// measured optima (profiles/r1_configs.md).  n_sm = 0 (no device known yet: workspace sizing) returns the maximum.
inline int choose_zsplit(int n_tiles, int nz, int n_sm, int forced) {
    const int cap = std::max(1, std::min(kSweepMaxZSplit, (nz + 1) / 4));
    if (forced > 0) return std::min(forced, cap);
    if (n_sm <= 0) return kSweepMaxZSplit;
    int best = 1; double best_cost = 1e300;
    for (int s = 1; s <= cap; ++s) {
        const double over = s > 1 ? 4.0 : 0.0;
        const double item = (double)(nz + 1) / s + over;
        const double cost = (double)n_tiles * s * item / n_sm + item;
        if (cost < best_cost * 0.999) { best_cost = cost; best = s; }
    }
    return best;
}

inline SweepPlan make_sweep_plan(int nx, int ny, int nz, int sizeof_real, int n_sm = 0, int forced_zsplit = 0,
                                 bool thermal = false) {
    SweepPlan f;
    f.V = 16 / sizeof_real;
    f.TXo = 30 * f.V;
    f.ntx = (nx + 1 + f.TXo - 1) / f.TXo;
    f.TY = tile_rows(sizeof_real, thermal);
    f.nty = (ny + 1 + f.TY - 1) / f.TY;
    f.n_tiles = f.ntx * f.nty;
    f.nzs = choose_zsplit(f.n_tiles, nz, n_sm * kSweepOcc, forced_zsplit);
    for (int c = 0; c <= kSweepMaxZSplit; ++c) f.kb[c] = nz + 1;
    for (int c = 0; c < f.nzs; ++c) f.kb[c] = (int)(((long long)(nz + 1) * c) / f.nzs);
    return f;
}

// Tiles that compute E' at node (i,j): the owner and, for nodes on a tile's low border, the
// neighbour(s) that recompute it as their +1 halo.  Returns the count (<= 4).
inline int tiles_of_node(const SweepPlan &f, int i, int j, int out[4]) {
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

// (cp_async16 / cp_async_commit / cp_async_wait: em_ptx.cuh)

template <typename R> __device__ __forceinline__ R shfl_up1(R v)   { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename R> __device__ __forceinline__ R shfl_down1(R v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// Sweep source index (built by em_set_source): entries of tile t are
// tile_ent[tile_sbeg[t] .. tile_sbeg[t+1]) sorted by (k, j, i); ent = {i, j, k, u*4 + comp}.
struct SweepSources {
    const int *tile_sbeg;     // indexed by work item = tile * nzs + chunk (entries of a tile are sorted by k)
    const int4 *tile_ent;
    const int *order;         // work item of CTA blockIdx.x (launch_order below)
};

// Launch order of the work items.  CTAs are handed to the SMs in blockIdx order, roughly one every (item time / n_sm),
// and a tile re-reads the halo rows / columns of its neighbours: those re-reads hit L2 only if the neighbour passes the
// same plane within a few plane-times, i.e. if it was launched within a few items (L2 holds ~9 plane-steps of the whole
// chip's traffic).  So: chunk-major (the chunks of one tile column share nothing), and inside a chunk the tiles in
// blocks of kOrderBY x kOrderBX tiles, y fastest -- x neighbours and most y neighbours are then a few items apart.
#ifndef EM_SWEEP_ORDER_BY
#define EM_SWEEP_ORDER_BY 1
#endif
#ifndef EM_SWEEP_ORDER_BX
#define EM_SWEEP_ORDER_BX (1 << 20)
#endif
inline void launch_order(const SweepPlan &f, int *order /* n_tiles * nzs */) {
    const int BY = EM_SWEEP_ORDER_BY, BX = EM_SWEEP_ORDER_BX;
    int n = 0;
    if (BY <= 0) {                                   // tile-major (the round-1 order)
        for (int t = 0; t < f.n_tiles; ++t) for (int c = 0; c < f.nzs; ++c) order[n++] = t * f.nzs + c;
    } else for (int c = 0; c < f.nzs; ++c)
        for (int by = 0; by < f.nty; by += BY)
            for (int bx = 0; bx < f.ntx; bx += BX)
                for (int x = bx; x < std::min(bx + BX, f.ntx); ++x)
                    for (int y = by; y < std::min(by + BY, f.nty); ++y) order[n++] = (y * f.ntx + x) * f.nzs + c;
}

// z chunks of the sweep (SweepPlan::kb), passed by value
struct SweepChunks {
    int nzs;
    int kb[kSweepMaxZSplit + 1];
};

}  // namespace em
