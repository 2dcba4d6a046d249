// em_sweep.cuh -- the TMA sweep (EM_KERNEL_TMA): ONE kernel per time step does
//   a0 coefficient gather, a1 H update, a2 E update, a3 source injection, a4 Joule accumulation, a5 PEC
// (eq. (2)-(3) L69-L76 in leapfrog form, L86 for the Joule heat) and moves each
// field value through HBM once per step: 57 B (fp32) / 113 B (fp64) per cell-update.
//
// Same decomposition and arithmetic as em_fused.cuh (tile = 30V x 14 columns marched in z, warp = one
// row, lane = V consecutive x, halo lanes/rows recompute), but the data movement and the
// synchronisation are Blackwell-native:
//  * every input plane (E, H, q, material ids) is staged into shared memory by TMA
//    (cp.async.bulk.tensor.3d, one box per array per plane, issued by one thread, completion counted
//    on an mbarrier): no per-thread address arithmetic, no LSU traffic for the loads, two planes in
//    flight per SM;
//  * there is NO CTA-wide barrier in the plane loop.  A warp waits only for what it consumes:
//      full[s]    : the TMA boxes of plane k have landed            (producer -> all warps)
//      flagH[w]   : warp w has published H'(k) of its row          (row w -> row w+1, E update)
//      flagB[w]   : warp w has published (2 Ebar)^2 of its row     (row w -> row w-1, Joule sum)
//      emptyA[s]  : every warp has finished reading stage s         (all warps -> producer)
//    so the warps of a CTA drift by up to a phase and the shared-memory-heavy and the FMA-heavy parts of
//    different rows overlap instead of running in lock step;
//  * the coefficient partial means of the previous plane are recomputed from the id ring instead of
//    being carried (frees 48 KB of shared memory for the second stage and the double-buffered rows).
// Warp 0 (halo row -1: only H') is also the TMA producer.
#pragma once
#include <cuda.h>

#include "em_fused.cuh"

namespace em {

constexpr int kSwTY = kFusedTY;                    // 14 owned rows
constexpr int kSwWarps = kSwTY + 2;                // rows -1 .. TY
constexpr int kSwThreads = kSwWarps * 32;          // 512
constexpr int kSwRow = 512;                        // bytes of one staged row (32 lanes x 16 B)
constexpr int kSwIdShift = 16;                     // the id map starts 16 B before the row (16-B aligned base)

struct alignas(64) SweepMaps { CUtensorMap E[3], H[3], q, mat; };

// Shared-memory layout (bytes; identical for fp32 and fp64 except the id rows; the table comes last
// because its size is only known at run time)
template <int SZ> struct SweepLayout {
    static constexpr int V = 16 / SZ;
    static constexpr int ex = 0;                                  // Ex ring of 3 planes, rows -1 .. TY+1
    static constexpr int ex_slot = 17 * kSwRow;
    static constexpr int ey = ex + 3 * ex_slot;                   // Ey ring of 3 planes, rows -1 .. TY
    static constexpr int ey_slot = 16 * kSwRow;
    static constexpr int ez = ey + 3 * ey_slot;                   // Ez, 2 stages, rows -1 .. TY+1
    static constexpr int ez_slot = 17 * kSwRow;
    static constexpr int h = ez + 2 * ez_slot;                    // [stage][Hx, Hy, Hz], rows -1 .. TY
    static constexpr int h_slot = 16 * kSwRow;
    static constexpr int q = h + 6 * h_slot;                      // q ring of 3 layers: TY rows x 30 lanes
    static constexpr int q_row = 30 * 16;
    static constexpr int q_slot = (kSwTY * q_row + 127) / 128 * 128;
    static constexpr int ids = q + 3 * q_slot;                    // id ring of 4 planes, rows -2 .. TY+1
    static constexpr int id_row = 32 * V + 16;                    // box starts on a 16-B boundary: up to 15 B of lead-in
    static constexpr int id_slot = (18 * id_row + 127) / 128 * 128;
    static constexpr int rows = ids + 4 * id_slot;                // [H'x, H'z, Bx, Bz][parity][16 rows]
    static constexpr int rows_slot = 16 * kSwRow;
    static constexpr int carry = rows + 8 * rows_slot;            // H'y of plane k-1
    static constexpr int geo = carry + 16 * kSwRow;               // 1/dx, 1/dx~, fx of the 32 lanes
    static constexpr int bar = geo + 3 * kSwRow;                  // full[2], emptyA[2], flagH[16], flagB[16]
    static constexpr int tab = bar + 8 * (4 + 2 * kSwWarps) + 64; // material table (n_table entries)
    static constexpr int stage_bytes = ex_slot + ey_slot + ez_slot + 3 * h_slot + 18 * id_row;
    static constexpr int q_bytes = kSwTY * q_row;
    static constexpr int first_extra_bytes = ex_slot + ey_slot + 18 * id_row;
};

inline size_t sweep_smem_bytes(int sizeof_real, int n_table) {
    const size_t tab = sizeof_real == 4 ? SweepLayout<4>::tab : SweepLayout<8>::tab;
    return tab + (size_t)n_table * 4 * sizeof_real;
}

// ---- mbarrier / TMA PTX wrappers ---------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "W_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra W_%=;\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap *map, unsigned bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar) : "memory");
}

// ---- the kernel ------------------------------------------------------------------------------------------
template <typename R, int LOSS, bool UMU>
__global__ void __launch_bounds__(kSwThreads, 1)
k_sweep_tma(const __grid_constant__ SweepMaps maps, DevParams<R> p, DevSources<R> src, FusedSources fs,
            FusedChunks zc, int ntx, long long step) {
    constexpr int V = 16 / sizeof(R);
    constexpr int TXo = 30 * V;
    using L = SweepLayout<(int)sizeof(R)>;
    using VecR = Vec<R>;
    using IdT = typename std::conditional<V == 4, unsigned, unsigned short>::type;
    extern __shared__ __align__(1024) unsigned char sm[];

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    // work item = (tile, z chunk), as in k_fused_sweep: the chunk stores planes kz0 <= k < kz1, starts one
    // plane lower (warm-up, nothing stored) and ends on plane ke (E'(ke) closes the Joule sum of layer ke-1)
    const int item = blockIdx.x, tile = item / zc.nzs, chunk = item - tile * zc.nzs;
    const int tx = tile % ntx, ty = tile / ntx;
    const int kz0 = zc.kb[chunk], kz1 = zc.kb[chunk + 1];
    const int ks = kz0 > 0 ? kz0 - 1 : 0, ke = kz1 <= p.nz ? kz1 : p.nz;
    const int cy = w - 1;
    const int j = ty * kSwTY + cy;
    const int i0 = tx * TXo - V + V * lane;
    const int ny = p.ny, nz = p.nz;
    const long long PX = p.PX, PXY = p.PXY;
    const bool is_top = (cy == kSwTY);
    const bool active = (j <= ny + 1) && (i0 + V <= p.PX);
    const bool own = active && lane >= 1 && lane <= 30 && cy >= 0 && cy < kSwTY && j <= ny;
    const bool own_q = own && j < ny;
    const unsigned out_pack = (unsigned)(p.n_table - 1) * 0x01010101u;

    // shared-memory views
    const int my = w * kSwRow + lane * 16;                    // this thread's vector inside a staged slot
    MatEntry<R> *s_tab = reinterpret_cast<MatEntry<R> *>(sm + L::tab);
    const VecR *s_geo = reinterpret_cast<const VecR *>(sm + L::geo);
    auto ldsv = [&](int byte_off) -> VecR { return *reinterpret_cast<const VecR *>(sm + byte_off); };
    auto stsv = [&](int byte_off, const VecR &v) { *reinterpret_cast<VecR *>(sm + byte_off) = v; };
    auto rows_off = [&](int arr, int par, int row) -> int { return L::rows + ((arr * 2 + par) * 16 + row) * kSwRow + lane * 16; };
    const int carry_hy = L::carry + my;
    const unsigned bar0 = smem_u32(sm + L::bar);
    auto bar_full = [&](int s) -> unsigned { return bar0 + 8 * s; };
    auto bar_empty = [&](int s) -> unsigned { return bar0 + 8 * (2 + s); };
    auto bar_H = [&](int ww) -> unsigned { return bar0 + 8 * (4 + ww); };
    auto bar_B = [&](int ww) -> unsigned { return bar0 + 8 * (4 + kSwWarps + ww); };

    // ---- prologue: barriers, table, x geometry, zeroed exchange rows and carries ----------------------------
    if (tid == 0) {
        for (int s = 0; s < 2; ++s) { mbar_init(bar_full(s), 1); mbar_init(bar_empty(s), kSwWarps); }
        for (int ww = 0; ww < kSwWarps; ++ww) { mbar_init(bar_H(ww), 1); mbar_init(bar_B(ww), 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int t = tid; t < p.n_table; t += kSwThreads) s_tab[t] = p.table[t];
    {
        VecR z;
#pragma unroll
        for (int c = 0; c < V; ++c) z.v[c] = R(0);
        for (int t = tid; t < 8 * 16 * 32; t += kSwThreads) reinterpret_cast<VecR *>(sm + L::rows)[t] = z;
        stsv(carry_hy, z);
        if (w == 0) {
            const bool in = (i0 + V <= p.PX);
            reinterpret_cast<VecR *>(sm + L::geo)[0 * 32 + lane] = in ? *reinterpret_cast<const VecR *>(p.rdx + i0) : z;
            reinterpret_cast<VecR *>(sm + L::geo)[1 * 32 + lane] = in ? *reinterpret_cast<const VecR *>(p.rtx + i0) : z;
            reinterpret_cast<VecR *>(sm + L::geo)[2 * 32 + lane] = in ? *reinterpret_cast<const VecR *>(p.fx + i0) : z;
        }
    }
    __syncthreads();

    // TMA coordinates of this tile (maps are based at logical (-V, -1, -1); ids at (-16 B, -1, -1))
    const int cx = tx * TXo, cyy = ty * kSwTY;
    // a box must start on a 16-B boundary: the id box starts at the boundary at or below the tile's first id
    const int id_x = (cx - V + kSwIdShift) & ~15, id_lead = (cx - V + kSwIdShift) & 15;
    // stage s = plane s: Ex(s+1), Ey(s+1), Ez(s), H(s), ids(s) and q(s-1) (consumed by phase C of plane s)
    auto issue_stage = [&](int s, bool first) {
        const bool with_q = (s - 1 >= kz0) && (s <= ke);
        const unsigned bar = bar_full(s & 1);
        const unsigned sb = smem_u32(sm);
        mbar_expect_tx(bar, (unsigned)(L::stage_bytes + (with_q ? L::q_bytes : 0) + (first ? L::first_extra_bytes : 0)));
        if (first) {
            tma_load_3d(sb + L::ex + (s % 3) * L::ex_slot, &maps.E[0], bar, cx, cyy, s + 1);
            tma_load_3d(sb + L::ey + (s % 3) * L::ey_slot, &maps.E[1], bar, cx, cyy, s + 1);
            tma_load_3d(sb + L::ids + ((s + 3) & 3) * L::id_slot, &maps.mat, bar, id_x, cyy - 1, s);
        }
        tma_load_3d(sb + L::ex + ((s + 1) % 3) * L::ex_slot, &maps.E[0], bar, cx, cyy, s + 2);
        tma_load_3d(sb + L::ey + ((s + 1) % 3) * L::ey_slot, &maps.E[1], bar, cx, cyy, s + 2);
        tma_load_3d(sb + L::ez + (s & 1) * L::ez_slot, &maps.E[2], bar, cx, cyy, s + 1);
        tma_load_3d(sb + L::h + ((s & 1) * 3 + 0) * L::h_slot, &maps.H[0], bar, cx, cyy, s + 1);
        tma_load_3d(sb + L::h + ((s & 1) * 3 + 1) * L::h_slot, &maps.H[1], bar, cx, cyy, s + 1);
        tma_load_3d(sb + L::h + ((s & 1) * 3 + 2) * L::h_slot, &maps.H[2], bar, cx, cyy, s + 1);
        tma_load_3d(sb + L::ids + (s & 3) * L::id_slot, &maps.mat, bar, id_x, cyy - 1, s + 1);
        if (with_q) tma_load_3d(sb + L::q + ((s + 2) % 3) * L::q_slot, &maps.q, bar, cx + V, cyy + 1, s);
    };
#if defined(EM_SW_STOP) && EM_SW_STOP == 1
    return;
#endif
    if (tid == 0) {
        issue_stage(ks, true);
        if (ks + 1 <= ke) issue_stage(ks + 1, false);
    }
#if defined(EM_SW_STOP) && EM_SW_STOP == 2
    mbar_wait(bar_full(ks & 1), 0);
    if (ks + 1 <= ke) mbar_wait(bar_full((ks + 1) & 1), 0);
    return;
#endif
#if defined(EM_SW_STOP) && EM_SW_STOP == 3
    if (tid == 0) { mbar_wait(bar_full(ks & 1), 0); if (ks + 1 <= ke) mbar_wait(bar_full((ks + 1) & 1), 0); }
    __syncthreads();
    return;
#endif

    const R fy = active ? p.fy[j] : R(0), rdy = active ? p.rdy[j] : R(0), rty = active ? p.rty[j] : R(0);
    const R gq = p.dt * R(0.0625);
    const long long off0 = (long long)j * PX + i0;    // this thread's vector at plane 0 (stores)
    auto id_uniform = [&](unsigned wv) -> bool { return (V == 4) ? (wv == (wv & 0xffu) * 0x01010101u) : (((wv >> 8) & 0xffu) == (wv & 0xffu)); };
    // ids of the lane's V cells of row `row` (0 = j-2 .. 17) of plane slot `slot`
    auto ld_ids = [&](int slot, int row) -> unsigned {
        const unsigned v = *reinterpret_cast<const IdT *>(sm + L::ids + slot * L::id_slot + row * L::id_row + id_lead + lane * V);
        return (V == 4) ? v : (v | (out_pack & 0xffff0000u));
    };

    unsigned idw_prev = out_pack;                     // set on the first plane from the staged ids of plane ks-1
    bool rowu_prev = false;      // plane k-1: rows j-1 and j of this lane held one material
    VecR pend;                   // Joule partial sum Sxy(k-1) + Sz(k-1) of layer k-1
#pragma unroll
    for (int c = 0; c < V; ++c) pend.v[c] = R(0);
    bool q_live = false;         // q of layer k-1 must be stored (some sigma != 0 among the lane's cells)
    int s_cur = fs.tile_sbeg[item];
    const int s_end = fs.tile_sbeg[(tile + 1) * zc.nzs];
    int s_next_k = (s_cur < s_end) ? fs.tile_ent[s_cur].z : 0x7fffffff;

    int rk = ks % 3;                                  // k % 3
    for (int k = ks; k <= ke; ++k) {
        const int it = k - ks;
        const int rk1 = (rk == 2) ? 0 : rk + 1;
        const int par = k & 1;
        const long long o = off0 + (long long)k * PXY;
        const bool st = own && k >= kz0 && k < kz1;          // this chunk stores H'(k), E'(k)
        const VecR zg = *reinterpret_cast<const VecR *>(p.zgeo + 4 * (long long)k);   // {fz, 1/dz, 1/dz~, 0} (V = 2: first two)
        const R fz = zg.v[0], rdz = zg.v[1];
        const R rtz = (V == 4) ? zg.v[V == 4 ? 2 : 0] : p.zgeo[4 * (long long)k + 2];

        mbar_wait(bar_full(par), (unsigned)(it >> 1) & 1u);  // the TMA boxes of plane k have landed
        const unsigned idw = ld_ids(k & 3, w + 1), idj = ld_ids(k & 3, w);
        if (it == 0) {
            idw_prev = ld_ids((k + 3) & 3, w + 1);
            rowu_prev = (idw_prev == ld_ids((k + 3) & 3, w)) && id_uniform(idw_prev);
        }
        // one material over the warp's whole coefficient neighbourhood (rows j-1..j, planes k-1..k)?
        const bool rowu = (idw == idj) && id_uniform(idw);
        const unsigned idw_lane0 = __shfl_sync(0xffffffffu, idw, 0);   // (every lane must execute it)
        const bool hom = __all_sync(0xffffffffu, rowu && rowu_prev && idw == idw_prev && idw == idw_lane0);

        // ---- phase A: H' = H - nbar * curl E  (inner factor of S = curl mu^-1 curl) ----------
        VecR hxn, hyn, hzn;
        const VecR ex0 = ldsv(L::ex + rk * L::ex_slot + my), ey0 = ldsv(L::ey + rk * L::ey_slot + my);
        const VecR ez = ldsv(L::ez + par * L::ez_slot + my);
        {
            const VecR ex1 = ldsv(L::ex + rk1 * L::ex_slot + my), ey1 = ldsv(L::ey + rk1 * L::ey_slot + my);
            const VecR hx = ldsv(L::h + (par * 3 + 0) * L::h_slot + my), hy = ldsv(L::h + (par * 3 + 1) * L::h_slot + my);
            const VecR hz = ldsv(L::h + (par * 3 + 2) * L::h_slot + my);
            const VecR exn = ldsv(L::ex + rk * L::ex_slot + my + kSwRow), ezn = ldsv(L::ez + par * L::ez_slot + my + kSwRow);
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
        stsv(rows_off(0, par, w), hxn); stsv(rows_off(1, par, w), hzn);
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(bar_H(w));                    // H'(k) of this row is visible
            mbar_arrive(bar_empty(par));              // this warp is done with the staged fields of plane k
            if (w == 0 && k + 2 <= ke) {              // producer: refill the stage once all 16 warps released it
                mbar_wait(bar_empty(par), (unsigned)(it >> 1) & 1u);
                issue_stage(k + 2, false);
            }
        }

        if (w != 0) {
            // ---- phase B: E' = E + r (curl H' - J - sigma E), Joule squares (eq. 2-3) --------
            mbar_wait(bar_H(w - 1), (unsigned)it & 1u);       // H'(k) of row j-1
            VecR bx, by, bz;         // (2 Ebar)^2
            if (hom && s_next_k > k) {
#include "em_sweep_phaseb_hom.inc"
            } else if (s_next_k <= k) {
#define EM_HAS_J 1
#include "em_sweep_phaseb.inc"
#undef EM_HAS_J
                s_next_k = (s_cur < s_end) ? fs.tile_ent[s_cur].z : 0x7fffffff;
            } else {
#define EM_HAS_J 0
#include "em_sweep_phaseb.inc"
#undef EM_HAS_J
            }
            if (!active) {
#pragma unroll
                for (int c = 0; c < V; ++c) bx.v[c] = by.v[c] = bz.v[c] = R(0);
            }
            stsv(rows_off(2, par, w), bx); stsv(rows_off(3, par, w), bz);
            stsv(carry_hy, hyn);
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_B(w));             // (2 Ebar)^2 of this row is visible

            // ---- phase C: q(k-1) += dt sigma/16 (pend + Sxy(k)); pend = Sxy(k) + Sz(k) ----------------------
            if (!is_top) {
                mbar_wait(bar_B(w + 1), (unsigned)it & 1u);   // row j+1
                const VecR bxn = ldsv(rows_off(2, par, w + 1)), bzn = ldsv(rows_off(3, par, w + 1));
                const R by_r = shfl_down1(by.v[0]), bz_r = shfl_down1(bz.v[0]), bzn_r = shfl_down1(bzn.v[0]);
                const bool have_q = own_q && k > kz0 && q_live;                      // layer k-1 in [kz0, kz1)
                VecR qv;
                if (have_q) qv = ldsv(L::q + ((k + 2) % 3) * L::q_slot + (w - 1) * L::q_row + (lane - 1) * 16);
#pragma unroll
                for (int c = 0; c < V; ++c) {
                    const R byip = (c < V - 1) ? by.v[c < V - 1 ? c + 1 : c] : by_r;
                    const R bzip = (c < V - 1) ? bz.v[c < V - 1 ? c + 1 : c] : bz_r;
                    const R bznip = (c < V - 1) ? bzn.v[c < V - 1 ? c + 1 : c] : bzn_r;
                    const R sxy = (bx.v[c] + bxn.v[c]) + (by.v[c] + byip);
                    const R sz = (bz.v[c] + bzip) + (bzn.v[c] + bznip);
                    const R sg = s_tab[(idw_prev >> (8 * (hom ? 0 : c))) & 0xff].b;     // sigma of the cell of layer k-1
                    if (have_q) qv.v[c] = mad(gq * sg, pend.v[c] + sxy, qv.v[c]);
                    pend.v[c] = sxy + sz;
                }
                // q of a lane whose V cells are one lossless material never changes: not stored
                if (have_q) *reinterpret_cast<VecR *>(p.q + o - PXY) = qv;
                q_live = !(id_uniform(idw) && s_tab[idw & 0xff].b == R(0));
            }
        } else {
            mbar_wait(bar_B(1), (unsigned)it & 1u);           // throttle: row -1 stays within one plane of row 0
        }
        idw_prev = idw;
        rowu_prev = rowu;
        rk = rk1;
    }
}

template <typename R>
cudaError_t launch_sweep_tma(const FusedPlan &plan, size_t smem_bytes, const SweepMaps &maps, const DevParams<R> &p,
                             const DevSources<R> &src, const FusedSources &fs, int loss, bool uniform_mu,
                             long long step, cudaStream_t stream) {
    using K = void (*)(const SweepMaps, DevParams<R>, DevSources<R>, FusedSources, FusedChunks, int, long long);
    FusedChunks zc;
    zc.nzs = plan.nzs;
    for (int c = 0; c <= kFusedMaxZSplit; ++c) zc.kb[c] = plan.kb[c];
    K kern;
    if (loss == 0) kern = uniform_mu ? (K)k_sweep_tma<R, 0, true> : (K)k_sweep_tma<R, 0, false>;
    else           kern = uniform_mu ? (K)k_sweep_tma<R, 1, true> : (K)k_sweep_tma<R, 1, false>;
    cudaError_t e = cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    kern<<<plan.n_tiles * plan.nzs, kSwThreads, smem_bytes, stream>>>(maps, p, src, fs, zc, plan.ntx, step);
    return cudaGetLastError();
}

}  // namespace em
