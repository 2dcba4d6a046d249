// em_sweep.cuh -- the TMA sweep (EM_KERNEL_TMA): ONE kernel per time step does
//   a0 coefficient gather, a1 H update, a2 E update, a3 source injection, a4 Joule accumulation, a5 PEC
// (eq. (2)-(3) L69-L76 in leapfrog form, L86 for the Joule heat) and moves each
// field value through HBM once per step: 57 B (fp32) / 113 B (fp64) per cell-update.
//
// Decomposition: em_tile.cuh (tile = 30V x TY columns marched in z, warp = one row, lane = V consecutive x, halo
// lanes / rows recompute).  Staging:
//  * every E, H and material-id plane of the tile is ONE cp.async.bulk.tensor.3d box per array, issued by
//    one thread and counted on an mbarrier: no per-thread address arithmetic, no LDGSTS instructions and
//    no LSU shared-memory write wavefronts for the loads;
//  * a box lands row-major, 512 B per row, i.e. exactly in the [row = warp][lane] x 16 B slot format the
//    threads read; the boxes of Ex and Ez carry a 17th row (the top warp's +1 neighbour);
//  * q (conditionally fetched: lossless lanes skip it) stays on cp.async; the per-plane z geometry is a bulk copy.
//
// EO = true: the paper's LITERAL E-only three-level recurrence (NEXT-4 of SURVEY.md 8(f); eq. (2)
// eq. (3)):  M e^{n+1} = N e^n - K e^{n-1} - dt^2 (dJ/dt)^n.  State e^n, e^{n-1}; no H array is read or written.  The same
// sweep: phase A forms g = dt D_nu C_e e^n of the plane on chip (what the leapfrog subtracts from H), phase B applies
// C_h to it and advances  e^{n+1} = e^n + d + r (-(C_h g) - dJ - sigma d),  d = e^n - e^{n-1},  which is eq. (2) divided by
// M (N - M - K = -dt^2 S).  The planes of e^{n-1} ride in the staging slots of H.  9 words + 1 B + 2 words per
// cell-update = 45 B (fp32) / 89 B (fp64) instead of 57 / 113.
#pragma once
#include "em_tile.cuh"

namespace em {

#define EM_ST(ptr, val) st_stream16((ptr), (val))     // output planes: streaming (evict-first) stores

constexpr int kSwRow = 512;                        // bytes of one staged row (32 lanes x 16 B)
constexpr int kSwIdShift = 16;                     // the id map starts 16 B before the row (16-B aligned base)
constexpr int kSwPriv = 8;                         // private 16-B slots per thread: q, L x 4, H' x 2, pend

struct alignas(64) SweepMaps { CUtensorMap E[3], H[3], q, mat, sig, th; };   // sig, th: sigma(T^n), theta^n (coupled sweep only)

// EXPERIMENTAL, OFF by default and NOT yet run on a GPU (the pool was closed for this repository when it was finished,
// profiles/r2_experiments.md): -DEM_SWEEP_FUSED_CONDUCTION=1 folds the conduction stencil of eq. (5) into the coupled
// sweep -- theta^n planes in a ring of 3 beside sigma(T), ids in a ring of 3, the stencil of layer k-1 in phase A of plane
// k with the lower-face flux carried -- so that a coupled step is ONE launch (no k_diffuse).  With the switch off the
// preprocessed kernel and its SASS are those of the verified build.
#ifndef EM_SWEEP_FUSED_CONDUCTION
#define EM_SWEEP_FUSED_CONDUCTION 0
#endif
constexpr bool kFusedConduction = EM_SWEEP_FUSED_CONDUCTION != 0;

// Shared-memory layout (bytes; identical for fp32 and fp64 except the id rows; the table comes last
// because its size is only known at run time)
template <int SZ, bool TH = false> struct SweepLayout {
    static constexpr int V = 16 / SZ;
    static constexpr int kSwWarps = Tile<SZ, TH>::warps, kSwRows = Tile<SZ, TH>::rows;
    static constexpr bool FC = TH && kFusedConduction;
    static constexpr int n_priv = kSwPriv + (TH ? (FC ? 2 : 1) : 0);   // coupled sweep: + theta of layer k-1 (FC: + the heat flux through its lower face)
    static constexpr int ex = 0;                                  // Ex ring of 3 planes, rows -1 .. TY+1
    static constexpr int ex_slot = (kSwWarps + 1) * kSwRow;
    static constexpr int ey = ex + 3 * ex_slot;                   // Ey ring of 3 planes, rows -1 .. TY
    static constexpr int ey_slot = kSwWarps * kSwRow;
    static constexpr int ez = ey + 3 * ey_slot;                   // Ez, 2 parities, rows -1 .. TY+1
    static constexpr int ez_slot = (kSwWarps + 1) * kSwRow;
    static constexpr int h = ez + 2 * ez_slot;                    // [2 parities][Hx, Hy, Hz], rows -1 .. TY
    static constexpr int h_slot = kSwWarps * kSwRow;
    static constexpr int ids = h + 6 * h_slot;                    // ids, 2 parities (coupled sweep: ring of 3), rows -2 .. TY+1
    static constexpr int n_ids = FC ? 3 : 2;
    static constexpr int id_row = 32 * V + 16;                    // box starts on a 16-B boundary: up to 15 B of lead-in
    static constexpr int id_slot = ((kSwWarps + 2) * id_row + 127) / 128 * 128;
    static constexpr int priv = ids + n_ids * id_slot;            // private slots [kSwPriv][512 threads]
    static constexpr int rows = priv + n_priv * kSwWarps * kSwRow;     // H'x, H'z, Bx, Bz exchange rows [kSwRows][32]
    static constexpr int geo = rows + 4 * kSwRows * kSwRow;    // 1/dx, 1/dx~, fx of the 32 lanes
    static constexpr int zg = geo + 3 * kSwRow;                   // [2 parity]{fz, 1/dz, 1/dz~, 0}
    static constexpr int sig = zg + 128;                          // coupled sweep: sigma(T^n), 2 parities, rows -2 .. TY (TMA: 128-B aligned)
    static constexpr int sig_slot = TH ? (kSwWarps + 1) * kSwRow : 0;
    static constexpr int tht = sig + 2 * sig_slot;                // coupled sweep: theta^n, ring of 3 planes, rows -1 .. TY
    static constexpr int th_slot = FC ? kSwWarps * kSwRow : 0;
    static constexpr int yg = tht + 3 * th_slot;                  // coupled sweep: {1/dy[j-1], 1/dy[j+1], 1/dy~[j+1], 0} per row
    static constexpr int yg_bytes = FC ? kSwWarps * 4 * SZ : 0;
    static constexpr int bar = FC ? (yg + yg_bytes + 63) / 64 * 64 : sig + 2 * sig_slot;   // fullE[2], fullH[2], empty[2], emptyH[2], rowH[kSwWarps]
    static constexpr int tab = (bar + 64 + 8 * kSwWarps + 31) / 32 * 32;         // material table (n_table entries of 4 reals)
    static constexpr int e_bytes = ex_slot + ey_slot + ez_slot + (kSwWarps + 2) * id_row + sig_slot + th_slot;
    static constexpr int first_extra_bytes = ex_slot + ey_slot;
    static constexpr int h_bytes = 3 * h_slot;
    // what the hardware requires of these offsets (the base is 1024-byte aligned): TMA box destinations 128 B, bulk-copy
    // destinations and 16-byte vector slots 16 B, mbarriers 8 B, table entries their own size -- for EVERY tile shape the
    // experiment switches can produce (a 5-row variant once faulted on a GPU with "misaligned address": its table sat
    // at 8 mod 16; tests/emu reproduces that on the host)
    static_assert(ex % 128 == 0 && ex_slot % 128 == 0 && ey % 128 == 0 && ey_slot % 128 == 0 && ez % 128 == 0 && ez_slot % 128 == 0,
                  "E plane slots: TMA destinations");
    static_assert(h % 128 == 0 && h_slot % 128 == 0 && ids % 128 == 0 && id_slot % 128 == 0, "H and id slots: TMA destinations");
    static_assert(sig % 128 == 0 && sig_slot % 128 == 0 && tht % 128 == 0 && th_slot % 128 == 0, "sigma(T) and theta slots: TMA destinations");
    static_assert(priv % 16 == 0 && rows % 16 == 0 && geo % 16 == 0 && zg % 16 == 0 && yg % 16 == 0, "16-byte vector regions");
    static_assert(bar % 8 == 0 && tab % (4 * SZ) == 0, "mbarriers and table entries");
};

// the material table, and for the coupled sweep the thermal table (ThEntry, same size) behind it
inline size_t sweep_smem_bytes(int sizeof_real, int n_table, bool thermal = false) {
    const size_t tab = thermal ? (sizeof_real == 4 ? SweepLayout<4, true>::tab : SweepLayout<8, true>::tab)
                               : (sizeof_real == 4 ? SweepLayout<4>::tab : SweepLayout<8>::tab);
    return tab + (size_t)n_table * 4 * sizeof_real * (thermal ? 2 : 1);
}

// ---- per-phase clock trace (experiment builds only: -DEM_SWEEP_TRACE) ----------------------------------------------------
#ifdef EM_SWEEP_TRACE
__device__ long long *g_em_trace = nullptr;      // [n_items][warps][planes<=80][8 stamps]
#define EM_TRACE(slot) do { if (g_em_trace && lane == 0 && (k - ks) < 80) \
    g_em_trace[(((long long)blockIdx.x * 16 + w) * 80 + (k - ks)) * 8 + (slot)] = clock64(); } while (0)
#else
#define EM_TRACE(slot) ((void)0)
#endif

// (mbarrier / TMA / named-barrier wrappers and the schedule-fuzzing hook EM_FUZZ: em_ptx.cuh)
// Every staged plane is loaded with the L2 evict_last policy (the output planes are written evict-first): the halo
// rows and columns of a box are re-read by the neighbouring tiles a few planes earlier or later, so input lines should
// outlive output lines in L2 (measured: -1 % step time on config 4; splitting each plane into halo boxes with evict_last
// and an interior box with evict_first was 3 % SLOWER).
#ifndef EM_SWEEP_LOADPOL
#define EM_SWEEP_LOADPOL 1
#endif
#ifndef EM_SWEEP_PFPOL
#define EM_SWEEP_PFPOL 0
#endif
// TMA prefetch of a box into L2 only (no shared memory, no barrier): the boxes of plane k + 2 + kSwL2Ahead can be requested
// from DRAM when the loads of plane k + 2 are issued.  OFF (0) by default: measured on config 4 it made the step SLOWER
// (2.30 -> 2.36 / 2.49 / 2.85 ms for 1 / 2 / 4 planes ahead, whatever the L2 policies): the later loads do hit L2 (read
// misses -37 %) but DRAM reads grow by 0.6 GB (prefetched lines are evicted before use) -- the waits for staged planes
// are bandwidth, not latency (profiles/r2_experiments.md).
#ifndef EM_SWEEP_L2AHEAD
#define EM_SWEEP_L2AHEAD 0
#endif
constexpr int kSwL2Ahead = EM_SWEEP_L2AHEAD;

// ---- the kernel ------------------------------------------------------------------------------------------
// TH = true: the thermally coupled sweep (eq. (4)-(6); DESIGN.md section 9 NEXT-1).  The per-cell sigma(T^n)
// is staged as one more TMA plane per step plane (rows -2 .. TY) and replaces the table's sigma in the coefficient
// gather; phase C adds the Joule heat of the step to theta (already advanced by the conduction kernel k_diffuse) and
// writes sigma(T^{n+1}) to the other sigma buffer.  The one-material path is taken only for materials with alpha = 0.
template <typename R, int LOSS, bool UMU, bool TH = false, bool EO = false>
__global__ void __launch_bounds__(Tile<sizeof(R), TH>::threads, kSweepOcc)
k_sweep_tma(const __grid_constant__ SweepMaps maps, DevParams<R> p, DevSources<R> src, SweepSources fs,
            SweepChunks zc, int ntx, long long step, ThermalSweep<R> th) {
    constexpr int V = 16 / sizeof(R);
    constexpr int TXo = 30 * V;
    constexpr int kSwTY = Tile<sizeof(R), TH>::TY, kSwWarps = Tile<sizeof(R), TH>::warps, kSwRows = Tile<sizeof(R), TH>::rows;
    constexpr int NT = Tile<sizeof(R), TH>::threads;
    using L = SweepLayout<(int)sizeof(R), TH>;
    constexpr bool FC = L::FC;        // conduction fused into the coupled sweep (experimental switch, see SweepLayout)
    using VecR = Vec<R>;
    using IdT = typename std::conditional<V == 4, unsigned, unsigned short>::type;
    // private 16-B slots of a thread
    constexpr int kSlotQ = 0, kSlotL = 1, kSlotHp = 5, kSlotPend = 7, kSlotTheta = 8, kSlotFz = 9;
    EM_DYN_SMEM(sm);

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    // work item = (tile, z chunk), as in k_fused_sweep: the chunk stores planes kz0 <= k < kz1, starts one
    // plane lower (warm-up, nothing stored) and ends on plane ke (E'(ke) closes the Joule sum of layer ke-1)
    const int item = fs.order[blockIdx.x], tile = item / zc.nzs, chunk = item - tile * zc.nzs;     // launch order: em_tile.cuh
    const int tx = tile % ntx, ty = tile / ntx;
    const int kz0 = zc.kb[chunk], kz1 = zc.kb[chunk + 1];
    const int ks = (kz0 > 0 || p.warm_lo) ? kz0 - 1 : 0, ke = kz1 <= p.nz ? kz1 : p.nz;   // PMC at -z: plane -1 warms up too
    const int cy = w - 1, r = cy + 2;
    const int j = ty * kSwTY + cy;
    const int i0 = tx * TXo - V + V * lane;
    const int ny = p.ny, nz = p.nz;
    const long long PX = p.PX, PXY = p.PXY;
    const bool is_top = (cy == kSwTY);
    const bool active = (j <= ny + 1) && (i0 + V <= p.PX);
    const bool own = active && lane >= 1 && lane <= 30 && cy >= 0 && cy < kSwTY && j <= ny;
    const bool own_q = own && j < ny;
    // the per-thread store predicates as plane thresholds held in two registers (opaque to the compiler, which otherwise
    // re-derives `own` from lane, row and grid size on every plane to stay inside the register cap)
    int st_lo = own ? kz0 : 0x7fffffff, q_lo = own_q ? kz0 : 0x7fffffff;
    opaque2(st_lo, q_lo);
    const unsigned out_pack = (unsigned)(p.n_table - 1) * 0x01010101u;
    const bool has_peer = p.peer_skip != 0;

    // shared-memory views
    MatEntry<R> *s_tab = reinterpret_cast<MatEntry<R> *>(sm + L::tab);
    VecR *s_rows = reinterpret_cast<VecR *>(sm + L::rows);
    VecR(*smHx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 0 * kSwRows * 32);
    VecR(*smHz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 1 * kSwRows * 32);
    VecR(*smBx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 2 * kSwRows * 32);
    VecR(*smBz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 3 * kSwRows * 32);
    VecR *mine = reinterpret_cast<VecR *>(sm + L::priv) + tid;    // private slots [kSwPriv][NT]
    VecR *s_geo = reinterpret_cast<VecR *>(sm + L::geo);
    R *s_z = reinterpret_cast<R *>(sm + L::zg);
    const VecR *stg = reinterpret_cast<const VecR *>(sm) + tid;   // this thread's vector inside a staged box
    auto staged = [&](int byte_off) -> VecR { return *reinterpret_cast<const VecR *>(reinterpret_cast<const unsigned char *>(stg) + byte_off); };
    const unsigned bar0 = smem_u32(sm + L::bar);
    auto bar_fullE = [&](int s) -> unsigned { return bar0 + 8 * s; };
    auto bar_fullH = [&](int s) -> unsigned { return bar0 + 16 + 8 * s; };
    auto bar_empty = [&](int s) -> unsigned { return bar0 + 32 + 8 * s; };     // every warp has consumed the staged plane
    auto bar_emptyH = [&](int s) -> unsigned { return bar0 + 48 + 8 * s; };    // EO: ... and its e^{n-1} planes (read in phase B)
    auto bar_rowH = [&](int ww) -> unsigned { return bar0 + 64 + 8 * ww; };    // H'(k) row of warp ww is published

    // ---- prologue: barriers, table, x geometry, zeroed exchange rows and private slots -------------------
    if (tid == 0) {
        mbar_init(bar_fullE(0), 1); mbar_init(bar_fullE(1), 1); mbar_init(bar_fullH(0), 1); mbar_init(bar_fullH(1), 1);
        mbar_init(bar_empty(0), kSwWarps); mbar_init(bar_empty(1), kSwWarps);
        mbar_init(bar_emptyH(0), kSwWarps); mbar_init(bar_emptyH(1), kSwWarps);
        for (int ww = 0; ww < kSwWarps; ++ww) mbar_init(bar_rowH(ww), 1);
        mbar_fence_init();
    }
    for (int t = tid; t < p.n_table; t += NT) s_tab[t] = p.table[t];
    ThEntry<R> *s_th = reinterpret_cast<ThEntry<R> *>(s_tab + p.n_table);     // coupled sweep only
    if (TH) for (int t = tid; t < p.n_table; t += NT) s_th[t] = th.ttable[t];
    {
        VecR z, mone;
#pragma unroll
        for (int c = 0; c < V; ++c) { z.v[c] = R(0); mone.v[c] = R(-1); }
        for (int t = tid; t < 4 * kSwRows * 32; t += NT) s_rows[t] = z;
        for (int t = 0; t < L::n_priv; ++t) mine[t * NT] = z;
        mine[(kSlotL + 0) * NT] = mone; mine[(kSlotL + 2) * NT] = mone;     // plane k = -1 is outside: eps/dt = 1, mask 0 (sign)
        if (w == 0) {
            const bool in = (i0 + V <= p.PX);
            s_geo[0 * 32 + lane] = in ? *reinterpret_cast<const VecR *>(p.rdx + i0) : z;
            s_geo[1 * 32 + lane] = in ? *reinterpret_cast<const VecR *>(p.rtx + i0) : z;
            s_geo[2 * 32 + lane] = in ? *reinterpret_cast<const VecR *>(p.fx + i0) : z;
        }
    }
    if (FC && lane == 0) {          // y geometry of the conduction stencil, per row: 1/dy[j-1], 1/dy[j+1], 1/dy~[j+1]
        R *yg = reinterpret_cast<R *>(sm + L::yg) + 4 * w;
        const bool in = (j <= ny + 1);
        yg[0] = in ? p.rdy[j - 1] : R(0); yg[1] = in ? p.rdy[j + 1] : R(0); yg[2] = in ? p.rty[j + 1] : R(0); yg[3] = R(0);
    }
    __syncthreads();

    // TMA coordinates of this tile (maps are based at logical (-V, -1, -1); ids at (-16 B, -1, -1))
    const int cx = tx * TXo, cyy = ty * kSwTY;
    // a box must start on a 16-B boundary: the id box starts at the boundary at or below the tile's first id
    const int id_x = (cx - V + kSwIdShift) & ~15, id_lead = (cx - V + kSwIdShift) & 15;
    // E group of plane kk: Ex(kk+1), Ey(kk+1) -> ring slot (kk+1)%3, Ez(kk) and ids(kk) -> parity kk&1
    auto issue_E = [&](int kk, bool first) {
        const unsigned bar = bar_fullE((kk - ks) & 1);
        const unsigned sb = smem_u32(sm);
        mbar_expect_tx(bar, (unsigned)(L::e_bytes + (first ? L::first_extra_bytes : 0) + 4 * sizeof(R)));
        bulk_load(smem_u32(&s_z[(kk & 1) * 4]), p.zgeo + 4 * (long long)kk, 4 * (unsigned)sizeof(R), bar);   // {fz, 1/dz, 1/dz~, 0}
        if (first) {
            tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::ex + ((kk + 3) % 3) * L::ex_slot, &maps.E[0], bar, cx, cyy, kk + 1);
            tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::ey + ((kk + 3) % 3) * L::ey_slot, &maps.E[1], bar, cx, cyy, kk + 1);
        }
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::ex + ((kk + 1) % 3) * L::ex_slot, &maps.E[0], bar, cx, cyy, kk + 2);
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::ey + ((kk + 1) % 3) * L::ey_slot, &maps.E[1], bar, cx, cyy, kk + 2);
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::ez + (kk & 1) * L::ez_slot, &maps.E[2], bar, cx, cyy, kk + 1);
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::ids + (FC ? (kk + 3) % 3 : (kk & 1)) * L::id_slot, &maps.mat, bar, id_x, cyy - 1, kk + 1);
        if (TH) {
            tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::sig + (kk & 1) * L::sig_slot, &maps.sig, bar, cx, cyy - 1, kk + 1);   // rows -2 .. TY
            if (FC) tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::tht + ((kk + 3) % 3) * L::th_slot, &maps.th, bar, cx, cyy, kk + 1);    // theta^n(kk), rows -1 .. TY
        }
        if (kSwL2Ahead > 0 && kk + kSwL2Ahead <= ke) {          // the same boxes of plane kk + kSwL2Ahead, into L2 only
            const int kp = kk + kSwL2Ahead;
            tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.E[0], cx, cyy, kp + 2); tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.E[1], cx, cyy, kp + 2);
            tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.E[2], cx, cyy, kp + 1); tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.mat, id_x, cyy - 1, kp + 1);
            if (TH) tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.sig, cx, cyy - 1, kp + 1);
        }
    };
    // H group of plane kk -> parity kk&1 (two planes in flight)
    auto issue_H = [&](int kk) {
        const unsigned sb = smem_u32(sm), bar = bar_fullH((kk - ks) & 1);
        mbar_expect_tx(bar, (unsigned)L::h_bytes);
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::h + ((kk & 1) * 3 + 0) * L::h_slot, &maps.H[0], bar, cx, cyy, kk + 1);
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::h + ((kk & 1) * 3 + 1) * L::h_slot, &maps.H[1], bar, cx, cyy, kk + 1);
        tma_load_3d<EM_SWEEP_LOADPOL>(sb + L::h + ((kk & 1) * 3 + 2) * L::h_slot, &maps.H[2], bar, cx, cyy, kk + 1);
        if (kSwL2Ahead > 0 && kk + kSwL2Ahead <= ke) {
            const int kp = kk + kSwL2Ahead;
            tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.H[0], cx, cyy, kp + 1); tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.H[1], cx, cyy, kp + 1);
            tma_prefetch_3d<EM_SWEEP_PFPOL>(&maps.H[2], cx, cyy, kp + 1);
        }
    };
    if (tid == 0) {
        issue_E(ks, true);
        issue_H(ks);
        if (ks + 1 <= ke) { issue_E(ks + 1, false); issue_H(ks + 1); }
    }

    const R fy = active ? p.fy[j] : R(0), rdy = active ? p.rdy[j] : R(0), rty = active ? p.rty[j] : R(0);
    const R gq = p.dt * R(0.0625);
    const long long off0 = (long long)j * PX + i0;    // this thread's vector at plane 0 (stores, q)
    // all V cells of an id word hold the same material
    auto id_uniform = [&](unsigned wv) -> bool { return (V == 4) ? (wv == (wv & 0xffu) * 0x01010101u) : (((wv >> 8) & 0xffu) == (wv & 0xffu)); };
    // ids of the lane's V cells of row `row` (0 = j0-2 .. 17) of parity slot `slot`
    auto ld_ids = [&](int slot, int row) -> unsigned {
        const unsigned v = *reinterpret_cast<const IdT *>(sm + L::ids + slot * L::id_slot + row * L::id_row + id_lead + lane * V);
        return (V == 4) ? v : (v | (out_pack & 0xffff0000u));
    };

    unsigned idw_prev = out_pack;
    bool rowu_prev = false;      // plane k-1: rows j-1 and j of this lane held one material
    bool l_stale = false;        // warp-uniform: the L slots were skipped by the one-material path
    bool q_live = false;         // q of layer k-1 was fetched (some sigma != 0 among the lane's cells)
    VecR sig_prev;               // coupled sweep: sigma(T^n) of the lane's cells of layer k-1 (Joule sum of phase C)
#pragma unroll
    for (int c = 0; c < V; ++c) sig_prev.v[c] = R(0);
    // source cursor: starts at the tile's first entry with k >= kz0 and may run into the next chunk's
    // entries on the closing plane k = kz1 (E'(kz1) enters the Joule sum of layer kz1-1)
    int s_cur = fs.tile_sbeg[item];
    const int s_end = fs.tile_sbeg[(tile + 1) * zc.nzs];
    int s_next_k = (s_cur < s_end) ? fs.tile_ent[s_cur].z : 0x7fffffff;

    int rk = (ks + 3) % 3;                                // k % 3
    long long o = off0 + (long long)ks * PXY;             // this thread's vector at plane k
    for (int k = ks; k <= ke; ++k, o += PXY) {
        const int it = k - ks;
        const int rk1 = (rk == 2) ? 0 : rk + 1;
        const int par = k & 1;
        const bool st = k >= st_lo && k < kz1;               // this chunk stores H'(k), E'(k)

        // ---- phase A: H' = H - nbar * curl E  (inner factor of S = curl mu^-1 curl) ----------
        EM_FUZZ();
        EM_TRACE(0);
        mbar_wait(bar_fullE(it & 1), (unsigned)(it >> 1) & 1u);   // E group of plane k has landed
        EM_TRACE(1);
        const R fz = s_z[par * 4 + 0], rdz = s_z[par * 4 + 1], rtz = s_z[par * 4 + 2];
        const int ids_k = FC ? rk : par;                          // slot of ids(k): ring of 3 in the coupled sweep
        const unsigned idw = ld_ids(ids_k, w + 1), idj = ld_ids(ids_k, w);
        // one material over the warp's whole coefficient neighbourhood (rows j-1..j, planes k-1..k)?
        const bool rowu = (idw == idj) && id_uniform(idw);
        const unsigned idw_lane0 = __shfl_sync(0xffffffffu, idw, 0);   // (every lane must execute it)
        bool hom = __all_sync(0xffffffffu, rowu && rowu_prev && idw == idw_prev && idw == idw_lane0);
        VecR sigw, sigj;             // coupled sweep: sigma(T^n) of rows j and j-1 of plane k (box rows start at j0-2)
        if (TH) {
            hom = hom && s_th[idw_lane0 & 0xff].alpha == R(0);     // sigma of the material does not depend on T
            sigw = staged(L::sig + par * L::sig_slot + kSwRow); sigj = staged(L::sig + par * L::sig_slot);
        }
        // ---- coupled sweep: conduction half of eq. (5) for cell layer k-1, theta_d = theta^n - dt/(rho c_p) (M_kk theta^n),
        // M_kk = V0a^T D_k V0 as the cell-centred -div k grad with the series conductivity of the two half cells on each
        // face (T3).  theta^n(k-1) with its x / y neighbours and theta^n(k) are resident (ring of 3 planes), and
        // so are the ids of plane k-1; the flux through the lower face was computed one plane ago.  Phase C adds the Joule
        // heat.  (k == ks: nothing below is resident yet; the layers concerned belong to the chunk below.)
        if (FC && w != 0 && !is_top) {
            VecR thd, fzo;
            if (k == ks) {
#pragma unroll
                for (int c = 0; c < V; ++c) thd.v[c] = fzo.v[c] = R(0);
            } else {
                const int rkm = (rk == 0) ? 2 : rk - 1;                       // (k - 1) % 3
                const unsigned char *tb = sm + L::tht + rkm * L::th_slot + tid * 16;
                const VecR t0 = *reinterpret_cast<const VecR *>(tb), tym = *reinterpret_cast<const VecR *>(tb - kSwRow);
                const VecR typ = *reinterpret_cast<const VecR *>(tb + kSwRow);
                const VecR tzp = *reinterpret_cast<const VecR *>(sm + L::tht + rk * L::th_slot + tid * 16);
                const VecR fzm = mine[kSlotFz * NT];
                const R tl_ = shfl_up1(t0.v[V - 1]), tr_ = shfl_down1(t0.v[0]);
                const unsigned idc = idw_prev, idym = ld_ids(rkm, w), idyp = ld_ids(rkm, w + 2);
                const unsigned idl = __shfl_up_sync(0xffffffffu, (idc >> (8 * (V - 1))) & 0xffu, 1);
                const unsigned idr = __shfl_down_sync(0xffffffffu, idc & 0xffu, 1);
                const VecR rdxv = s_geo[0 * 32 + lane], rtxv = s_geo[1 * 32 + lane];
                const R rdx_l = shfl_up1(rdxv.v[V - 1]), rdx_r = shfl_down1(rdxv.v[0]), rtx_r = shfl_down1(rtxv.v[0]);
                const R *yg = reinterpret_cast<const R *>(sm + L::yg) + 4 * w;
                const R rdym = yg[0], rdyp = yg[1], rtyp = yg[2];
                const R rdz1 = p.rdz[k - 1];                                   // 1/dz of layer k-1 (rdz, rtz: plane / layer k)
                const unsigned rep_id = (V == 4) ? (idc & 0xffu) * 0x01010101u : (((idc & 0xffu) * 0x0101u) | (out_pack & 0xffff0000u));
                const bool uni = idc == rep_id && idym == rep_id && idyp == rep_id && idw == rep_id &&
                                 idl == (idc & 0xffu) && idr == (idc & 0xffu);
                if (__all_sync(0xffffffffu, uni)) {
                    // one material over the whole neighbourhood: the series conductance of two equal half cells is k / d~
                    const ThEntry<R> me = s_th[idc & 0xffu];
                    const R cy0 = rdy * rty, cy1 = rdy * rtyp, cz1 = me.k * rtz, sc = p.dt * me.irc;
#pragma unroll
                    for (int c = 0; c < V; ++c) {
                        const R tc = t0.v[c];
                        const R tl = c > 0 ? t0.v[c > 0 ? c - 1 : 0] : tl_, tr = c < V - 1 ? t0.v[c < V - 1 ? c + 1 : c] : tr_;
                        const R rtx1 = c < V - 1 ? rtxv.v[c < V - 1 ? c + 1 : c] : rtx_r;
                        R lat = rdxv.v[c] * (rtxv.v[c] * (tc - tl) + rtx1 * (tc - tr));
                        lat = mad(cy0, tc - tym.v[c], lat); lat = mad(cy1, tc - typ.v[c], lat);
                        const R fz = cz1 * (tc - tzp.v[c]);
                        thd.v[c] = mad(-sc, mad(me.k, lat, rdz1 * (fz - fzm.v[c])), tc);
                        fzo.v[c] = fz;
                    }
                } else {
                    R kc[V + 2], rdxc[V + 2], gxf[V + 1];
                    kc[0] = s_th[idl].k; kc[V + 1] = s_th[idr].k; rdxc[0] = rdx_l; rdxc[V + 1] = rdx_r;
#pragma unroll
                    for (int c = 0; c < V; ++c) { kc[c + 1] = s_th[(idc >> (8 * c)) & 0xff].k; rdxc[c + 1] = rdxv.v[c]; }
#pragma unroll
                    for (int c = 0; c < V + 1; ++c) gxf[c] = half_cell_cond(rdxc[c] * kc[c], rdxc[c + 1] * kc[c + 1]);
#pragma unroll
                    for (int c = 0; c < V; ++c) {
                        const R tc = t0.v[c], kme = kc[c + 1], gy = rdy * kme, gz = rdz1 * kme;
                        const R tl = c > 0 ? t0.v[c > 0 ? c - 1 : 0] : tl_, tr = c < V - 1 ? t0.v[c < V - 1 ? c + 1 : c] : tr_;
                        R lat = rdxc[c + 1] * (gxf[c] * (tc - tl) + gxf[c + 1] * (tc - tr));
                        lat = mad(rdy, half_cell_cond(gy, rdym * s_th[(idym >> (8 * c)) & 0xff].k) * (tc - tym.v[c]), lat);
                        lat = mad(rdy, half_cell_cond(gy, rdyp * s_th[(idyp >> (8 * c)) & 0xff].k) * (tc - typ.v[c]), lat);
                        const R fz = half_cell_cond(gz, rdz * s_th[(idw >> (8 * c)) & 0xff].k) * (tc - tzp.v[c]);
                        thd.v[c] = mad(-p.dt * s_th[(idc >> (8 * c)) & 0xff].irc, lat + rdz1 * (fz - fzm.v[c]), tc);
                        fzo.v[c] = fz;
                    }
                }
            }
            mine[kSlotTheta * NT] = thd; mine[kSlotFz * NT] = fzo;
        }
        VecR hxn, hyn, hzn;
        const VecR ex0 = staged(L::ex + rk * L::ex_slot), ey0 = staged(L::ey + rk * L::ey_slot);
        const VecR ez = staged(L::ez + par * L::ez_slot);
        {
            const VecR ex1 = staged(L::ex + rk1 * L::ex_slot), ey1 = staged(L::ey + rk1 * L::ey_slot);
            const VecR exn = staged(L::ex + rk * L::ex_slot + kSwRow), ezn = staged(L::ez + par * L::ez_slot + kSwRow);
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
            VecR hx, hy, hz;
            if (EO) {               // no H state: H' stands for -g = -dt D_nu C_e e^n (eq. (3): the inner factor of S)
#pragma unroll
                for (int c = 0; c < V; ++c) hx.v[c] = hy.v[c] = hz.v[c] = R(0);
            } else {
                EM_TRACE(2);
                mbar_wait(bar_fullH(it & 1), (unsigned)(it >> 1) & 1u);   // H(k) has landed
                EM_TRACE(3);
                hx = staged(L::h + (par * 3 + 0) * L::h_slot); hy = staged(L::h + (par * 3 + 1) * L::h_slot);
                hz = staged(L::h + (par * 3 + 2) * L::h_slot);
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
        if (st && !EO) {
            EM_ST(p.Hn[0] + o, hxn);
            EM_ST(p.Hn[1] + o, hyn);
            EM_ST(p.Hn[2] + o, hzn);
        }
        EM_FUZZ();
        smHx[r][lane] = hxn; smHz[r][lane] = hzn;
        // No CTA barrier in the plane loop.  Row j+1 waits only for THIS row's H' (mbarrier rowH), and the producer
        // thread refills the staged slots once every warp has pulled plane k into registers (mbarrier empty).
        // WAR on the exchange rows is ordered by the chain  B(k) of row j+1 done -> pair barrier -> C(k), A(k+1) of row j.
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(bar_rowH(w)); mbar_arrive(bar_empty(it & 1));
            if (EO && w == 0) mbar_arrive(bar_emptyH(it & 1));         // (warp 0 has no phase B)
        }
        if (tid == 0 && k + 2 <= ke) {
            mbar_wait(bar_empty(it & 1), (unsigned)(it >> 1) & 1u);
            if (!EO) issue_H(k + 2);
            issue_E(k + 2, false);
            if (EO) {               // the e^{n-1} planes are read in phase B: their slots are released there
                mbar_wait(bar_emptyH(it & 1), (unsigned)(it >> 1) & 1u);
                issue_H(k + 2);
            }
        }
        EM_TRACE(4);
        if (w != 0) mbar_wait(bar_rowH(w - 1), (unsigned)it & 1u);   // H'(k) of row j-1 is visible
        EM_TRACE(5);

        // ---- phase B: E' = E + r (curl H' - J - sigma E), Joule squares (eq. 2-3) -------------
        // (warp 0 = halo row -1 only supplies H' to row 0: no E', no Joule)
        VecR bx, by, bz;         // (2 Ebar)^2
        // stores of E'x, E'y (comp 0, 1): own array unless the plane is a wall fed by the neighbouring slab, plus the
        // neighbour's wall plane when this is the plane it needs (DevParams::peer_*)
        auto store_exy = [&](int comp, const VecR &v) {
            if (!st) return;
            if (!has_peer) { EM_ST(p.En[comp] + o, v); return; }         // (kernel-uniform: no slab neighbour is wired)
            if (!((k == 0 && (p.peer_skip & 1)) || (k == nz && (p.peer_skip & 2)))) EM_ST(p.En[comp] + o, v);
            if (k == p.peer_k[0]) EM_ST(p.peer_e[0][comp] + (o - (long long)k * PXY), v);
            if (k == p.peer_k[1]) EM_ST(p.peer_e[1][comp] + (o - (long long)k * PXY), v);
        };
        if (w != 0) {
            // EO: d = e^n - e^{n-1} of the own edges is formed where it is used (em_sweep_phaseb*.inc) from the staged
            // e^{n-1} planes (the subtraction is exact in floating point when the two levels are within a factor 2)
            if (EO) mbar_wait(bar_fullH(it & 1), (unsigned)(it >> 1) & 1u);   // e^{n-1}(k) has landed
#define EM_PREV(comp) staged(L::h + (par * 3 + (comp)) * L::h_slot)
            if (hom && s_next_k > k) {
#include "em_sweep_phaseb_hom.inc"
                l_stale = true;
            } else {
                if (l_stale) {   // plane k-1 took the one-material path: its coefficient means are the entry itself
                    const MatEntry<R> Ap = s_tab[idw_prev & 0xff];
                    VecR va, vb;
#pragma unroll
                    for (int c = 0; c < V; ++c) { va.v[c] = Ap.m != R(0) ? Ap.a : -Ap.a; vb.v[c] = Ap.b; }
                    mine[(kSlotL + 0) * NT] = va; mine[(kSlotL + 1) * NT] = vb;
                    mine[(kSlotL + 2) * NT] = va; mine[(kSlotL + 3) * NT] = vb;
                    l_stale = false;
                }
                if (s_next_k <= k) {
#define EM_HAS_J 1
#include "em_sweep_phaseb.inc"
#undef EM_HAS_J
                    s_next_k = (s_cur < s_end) ? fs.tile_ent[s_cur].z : 0x7fffffff;
                } else {
#define EM_HAS_J 0
#include "em_sweep_phaseb.inc"
#undef EM_HAS_J
                }
            }
#undef EM_PREV
            if (EO) {               // the staged e^{n-1} planes have been read
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_emptyH(it & 1));
            }
            if (!active) {
#pragma unroll
                for (int c = 0; c < V; ++c) bx.v[c] = by.v[c] = bz.v[c] = R(0);
            }
            smBx[r][lane] = bx; smBz[r][lane] = bz;
            mine[(kSlotHp + 0) * NT] = hxn; mine[(kSlotHp + 1) * NT] = hyn;
        }
        // No CTA barrier here: row j needs only the (2 Ebar)^2 row of row j+1, so the two warps meet on a
        // producer/consumer named barrier of their own (id = the upper warp's index) and a warp on the one-material
        // path does not wait for a general-path warp elsewhere in the CTA.  Warp 0 (no phase C) still consumes, so
        // that it cannot overwrite its H' row (phase A of plane k+1) while warp 1 reads it in phase B.
        EM_TRACE(6);
        if (w != 0) pair_arrive(w);               // my B row is written (and I am done reading the H' row of row j-1)
        if (!is_top) pair_sync(w + 1);            // the B row of row j+1 is visible
        EM_TRACE(7);
        cp_async_wait<0>();                       // q(k-1) has landed (private slot: no barrier needed)

        // ---- phase C: q(k-1) += dt sigma/16 (pend + Sxy(k)); pend = Sxy(k) + Sz(k) ---------------------------
        EM_FUZZ();
        if (w != 0 && !is_top) {
            const VecR bxn = smBx[r + 1][lane], bzn = smBz[r + 1][lane];
            const R by_r = shfl_down1(by.v[0]), bz_r = shfl_down1(bz.v[0]), bzn_r = shfl_down1(bzn.v[0]);
            VecR qv = mine[kSlotQ * NT];
            VecR pend = mine[kSlotPend * NT];
            VecR thv, sgn;           // coupled sweep: theta and sigma(T^{n+1}) of the cells of layer k-1
            if (TH) thv = mine[kSlotTheta * NT];
#pragma unroll
            for (int c = 0; c < V; ++c) {
                const R byip = (c < V - 1) ? by.v[c < V - 1 ? c + 1 : c] : by_r;
                const R bzip = (c < V - 1) ? bz.v[c < V - 1 ? c + 1 : c] : bz_r;
                const R bznip = (c < V - 1) ? bzn.v[c < V - 1 ? c + 1 : c] : bzn_r;
                const R sxy = (bx.v[c] + bxn.v[c]) + (by.v[c] + byip);
                const R sz = (bz.v[c] + bzip) + (bzn.v[c] + bznip);
                if (TH) {            // eq. (5) source term and eq. (6), with sigma(T^n) as used by the E update
                    const ThEntry<R> te = s_th[(idw_prev >> (8 * c)) & 0xff];
                    const R dq = gq * sig_prev.v[c] * (pend.v[c] + sxy);
                    qv.v[c] += dq;
                    thv.v[c] = mad(dq, te.irc, thv.v[c]);
                    sgn.v[c] = te.sigma0 * rcp<R>(thermal_den(te.alpha, thv.v[c]));
                } else {
                    const R sg = s_tab[(idw_prev >> (8 * (hom ? 0 : c))) & 0xff].b;     // sigma of the cell of layer k-1
                    qv.v[c] = mad(gq * sg, pend.v[c] + sxy, qv.v[c]);
                }
                pend.v[c] = sxy + sz;
            }
            mine[kSlotPend * NT] = pend;
            // q of a lane whose V cells are one lossless material never changes: neither fetched nor stored
            // (coupled sweep: the same holds for theta -- only conduction moves it -- and for sigma = 0)
            if (!FC) {
                if (k > q_lo && q_live) {                                    // layer k-1 in [kz0, kz1)
                    EM_ST(p.q + o - PXY, qv);
                    if (TH) { EM_ST(th.theta + o - PXY, thv); EM_ST(th.sig_out + o - PXY, sgn); }
                }
            } else if (k > q_lo) {
                if (q_live) { EM_ST(p.q + o - PXY, qv); EM_ST(th.sig_out + o - PXY, sgn); }
                EM_ST(th.theta + o - PXY, thv);                          // fused conduction moves every cell's theta
            }
            q_live = !(id_uniform(idw) && s_tab[idw & 0xff].b == R(0));
            if (k >= q_lo && k < ke && q_live) {
                cp_async16(mine + kSlotQ * NT, p.q + o);                 // q(k)
                if (TH && !FC) cp_async16(mine + kSlotTheta * NT, th.theta + o);   // theta_d(k)
            }
        }
        cp_async_commit();
        idw_prev = idw;
        rowu_prev = rowu;
        if (TH) sig_prev = sigw;
        rk = rk1;
    }
    cp_async_wait<0>();
}

// The instantiation for a context: loss mode x uniform-mu fast path, or the coupled sweep (general mu path only), or the
// E-only recurrence.  select + configure once at em_create, launch per step.
template <typename R>
using SweepKernel = void (*)(const SweepMaps, DevParams<R>, DevSources<R>, SweepSources, SweepChunks, int, long long, ThermalSweep<R>);

template <typename R>
SweepKernel<R> select_sweep(int loss, bool uniform_mu, bool thermal, bool eonly) {
    using K = SweepKernel<R>;
    if (thermal) return loss == 0 ? (K)k_sweep_tma<R, 0, false, true> : (K)k_sweep_tma<R, 1, false, true>;
    if (eonly) {
        if (loss == 0) return uniform_mu ? (K)k_sweep_tma<R, 0, true, false, true> : (K)k_sweep_tma<R, 0, false, false, true>;
        return uniform_mu ? (K)k_sweep_tma<R, 1, true, false, true> : (K)k_sweep_tma<R, 1, false, false, true>;
    }
    if (loss == 0) return uniform_mu ? (K)k_sweep_tma<R, 0, true> : (K)k_sweep_tma<R, 0, false>;
    return uniform_mu ? (K)k_sweep_tma<R, 1, true> : (K)k_sweep_tma<R, 1, false>;
}

template <typename R>
cudaError_t configure_sweep(SweepKernel<R> kern, size_t smem_bytes) {
    return cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
}

template <typename R>
cudaError_t launch_sweep_tma(SweepKernel<R> kern, const SweepPlan &plan, size_t smem_bytes, const SweepMaps &maps,
                             const DevParams<R> &p, const DevSources<R> &src, const SweepSources &fs, long long step,
                             cudaStream_t stream, const ThermalSweep<R> *thermal = nullptr) {
    SweepChunks zc;
    zc.nzs = plan.nzs;
    for (int c = 0; c <= kSweepMaxZSplit; ++c) zc.kb[c] = plan.kb[c];
    ThermalSweep<R> th{};
    if (thermal) th = *thermal;
    const int threads = thermal ? Tile<sizeof(R), true>::threads : Tile<sizeof(R)>::threads;
    EM_LAUNCH(kern, plan.n_tiles * plan.nzs, threads, smem_bytes, stream)(maps, p, src, fs, zc, plan.ntx, step, th);
    return cudaGetLastError();
}

}  // namespace em
