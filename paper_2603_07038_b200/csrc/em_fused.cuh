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

namespace em {

constexpr int kFusedTY = 16;                       // owned rows per tile
constexpr int kFusedWarps = kFusedTY + 2;          // rows -1 .. TY
constexpr int kFusedThreads = kFusedWarps * 32;    // 576
constexpr int kFusedRows = kFusedTY + 4;           // exchange rows, r = cy + 2 (row 0 and last: dummies)
constexpr int kStageSlots = 7;                     // Ex1 Ey1 Ez Hx Hy Hz q

struct FusedPlan {
    int V, TXo, ntx, nty, n_tiles;
    size_t smem_bytes;
};

inline FusedPlan make_fused_plan(int nx, int ny, int nz, int sizeof_real) {
    (void)nz;
    FusedPlan f;
    f.V = 16 / sizeof_real;
    f.TXo = 30 * f.V;
    f.ntx = (nx + 1 + f.TXo - 1) / f.TXo;
    f.nty = (ny + 1 + kFusedTY - 1) / kFusedTY;
    f.n_tiles = f.ntx * f.nty;
    const size_t table = (size_t)kMaxTable * 4 * sizeof_real;
    const size_t rows = (size_t)6 * kFusedRows * 32 * 16 + (size_t)kFusedRows * 32 * 4;
    const size_t spill = (size_t)6 * kFusedThreads * 16;
    const size_t stage = (size_t)kStageSlots * kFusedThreads * 16 + (size_t)2 * 32 * 16;
    f.smem_bytes = table + rows + spill + stage;
    return f;
}

// Tiles that compute E' at node (i,j): the owner and, for nodes on a tile's low border, the
// neighbour(s) that recompute it as their +1 halo.  Returns the count (<= 4).
inline int tiles_of_node(const FusedPlan &f, int i, int j, int out[4]) {
    int txs[2], tys[2], nxs = 0, nys = 0;
    txs[nxs++] = i / f.TXo;
    if (i % f.TXo == 0 && i > 0) txs[nxs++] = i / f.TXo - 1;
    tys[nys++] = j / kFusedTY;
    if (j % kFusedTY == 0 && j > 0) tys[nys++] = j / kFusedTY - 1;
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
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename R> __device__ __forceinline__ R shfl_up1(R v)   { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename R> __device__ __forceinline__ R shfl_down1(R v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// Fused-sweep source index (built by em_set_source): entries of tile t are
// tile_ent[tile_sbeg[t] .. tile_sbeg[t+1]) sorted by (k, j, i); ent = {i, j, k, u*4 + comp}.
struct FusedSources {
    const int *tile_sbeg;
    const int4 *tile_ent;
};

template <typename R, int LOSS, bool UMU>
__global__ void __launch_bounds__(kFusedThreads, 1)
k_fused_sweep(DevParams<R> p, DevSources<R> src, FusedSources fs, int ntx, long long step) {
    constexpr int V = 16 / sizeof(R);
    constexpr int TXo = 30 * V;
    using VecR = Vec<R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    MatEntry<R> *s_tab = reinterpret_cast<MatEntry<R> *>(smem_raw);
    VecR *s_rows = reinterpret_cast<VecR *>(smem_raw + (size_t)kMaxTable * sizeof(MatEntry<R>));
    VecR(*smEx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 0 * kFusedRows * 32);
    VecR(*smEz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 1 * kFusedRows * 32);
    VecR(*smHx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 2 * kFusedRows * 32);
    VecR(*smHz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 3 * kFusedRows * 32);
    VecR(*smBx)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 4 * kFusedRows * 32);
    VecR(*smBz)[32] = reinterpret_cast<VecR(*)[32]>(s_rows + 5 * kFusedRows * 32);
    unsigned(*smId)[32] = reinterpret_cast<unsigned(*)[32]>(s_rows + 6 * kFusedRows * 32);
    VecR *s_spill = reinterpret_cast<VecR *>(reinterpret_cast<unsigned char *>(smId) + (size_t)kFusedRows * 32 * 4);
    VecR *s_stage = s_spill + 6 * kFusedThreads;
    VecR *s_top = s_stage + kStageSlots * kFusedThreads;      // [2][32]: Ex, Ez of row TY+1 (top warp only)

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int tile = blockIdx.x, tx = tile % ntx, ty = tile / ntx;
    const int cy = w - 1, r = cy + 2;
    const int j = ty * kFusedTY + cy;
    const int i0 = tx * TXo - V + V * lane;
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const long long PX = p.PX, PXY = p.PXY;
    const bool is_top = (cy == kFusedTY);
    const bool active = (j <= ny + 1) && (i0 + V <= p.PX);
    const bool top_row_ok = is_top && active && (j + 1 <= ny + 1);
    const bool own = active && lane >= 1 && lane <= 30 && cy >= 0 && cy < kFusedTY && j <= ny;
    const bool own_q = own && j < ny;

    // ---- prologue: table, zeroed exchange rows, spill of the (outside) plane k = -1 ---------------
    for (int t = tid; t < p.n_table; t += kFusedThreads) s_tab[t] = p.table[t];
    {
        VecR z;
#pragma unroll
        for (int c = 0; c < V; ++c) z.v[c] = R(0);
        for (int t = tid; t < 6 * kFusedRows * 32; t += kFusedThreads) s_rows[t] = z;
        for (int t = tid; t < kFusedRows * 32; t += kFusedThreads) (&smId[0][0])[t] = 0xffffffffu;
        VecR one;
#pragma unroll
        for (int c = 0; c < V; ++c) one.v[c] = R(1);
        s_spill[0 * kFusedThreads + tid] = one; s_spill[1 * kFusedThreads + tid] = z; s_spill[2 * kFusedThreads + tid] = z;
        s_spill[3 * kFusedThreads + tid] = one; s_spill[4 * kFusedThreads + tid] = z; s_spill[5 * kFusedThreads + tid] = z;
        for (int t = 0; t < kStageSlots; ++t) s_stage[t * kFusedThreads + tid] = z;
        if (tid < 64) s_top[tid] = z;
    }
    const int out_id = p.n_table - 1;                 // the "outside" entry
    // ids of the exchange rows default to "outside" (packed V ids per lane, one byte each)
    const unsigned out_pack = (unsigned)out_id * 0x01010101u;
    for (int t = tid; t < kFusedRows * 32; t += kFusedThreads) (&smId[0][0])[t] = out_pack;
    __syncthreads();

    // per-thread geometry
    R fxv[V], rdxv[V], rtxv[V];
#pragma unroll
    for (int c = 0; c < V; ++c) {
        const int i = i0 + c;
        const bool ok = active && i >= -1 && i <= p.PX;
        fxv[c] = ok ? p.fx[i] : R(0); rdxv[c] = ok ? p.rdx[i] : R(0); rtxv[c] = ok ? p.rtx[i] : R(0);
    }
    const R fy = active ? p.fy[j] : R(0), rdy = active ? p.rdy[j] : R(0), rty = active ? p.rty[j] : R(0);
    const R gq = p.dt * R(0.0625);

    // base offset of this thread's vector at plane 0
    const long long off0 = (long long)j * PX + i0;
    auto ldv = [&](const R *a, long long off) -> VecR { return *reinterpret_cast<const VecR *>(a + off); };
    auto ld_ids = [&](long long off) -> unsigned {
        if (V == 4) return *reinterpret_cast<const unsigned *>(p.mat + off);
        return (unsigned)*reinterpret_cast<const unsigned short *>(p.mat + off);
    };

    // carried state
    VecR ex0, ey0, hxp, hyp, pend, sgp, nzp;
#pragma unroll
    for (int c = 0; c < V; ++c) { ex0.v[c] = ey0.v[c] = hxp.v[c] = hyp.v[c] = pend.v[c] = sgp.v[c] = nzp.v[c] = R(0); }
    unsigned idw_next = out_pack;
    if (active) {
        ex0 = ldv(p.E[0], off0); ey0 = ldv(p.E[1], off0);
        idw_next = ld_ids(off0);
    }
    // stage(0): Ex(1), Ey(1), Ez(0), H(0)
    VecR *my_stage = s_stage + tid;
    auto issue_stage = [&](int k) {              // inputs of iteration k
        if (active) {
            const long long o = off0 + (long long)k * PXY;
            cp_async16(my_stage + 0 * kFusedThreads, p.E[0] + o + PXY);
            cp_async16(my_stage + 1 * kFusedThreads, p.E[1] + o + PXY);
            cp_async16(my_stage + 2 * kFusedThreads, p.E[2] + o);
            cp_async16(my_stage + 3 * kFusedThreads, p.H[0] + o);
            cp_async16(my_stage + 4 * kFusedThreads, p.H[1] + o);
            cp_async16(my_stage + 5 * kFusedThreads, p.H[2] + o);
            if (top_row_ok) {
                cp_async16(s_top + lane, p.E[0] + o + PX);
                cp_async16(s_top + 32 + lane, p.E[2] + o + PX);
            }
        }
        cp_async_commit();
    };
    issue_stage(0);
    cp_async_commit();                            // empty "q" group so the group arithmetic is uniform

    // source cursor of this tile
    int s_cur = fs.tile_sbeg[tile];
    const int s_end = fs.tile_sbeg[tile + 1];

    for (int k = 0; k <= nz; ++k) {
        const R fz = p.fz[k], rdz = p.rdz[k], rtz = p.rtz[k];
        const long long o = off0 + (long long)k * PXY;
        // ---- S1: stage plane-k values the neighbours need ----------------------------------------
        cp_async_wait<1>();                       // stage(k) has landed (the q group may still fly)
        const unsigned idw = idw_next;
        VecR ez = my_stage[2 * kFusedThreads];
        smEx[r][lane] = ex0; smEz[r][lane] = ez; smId[r][lane] = idw;
        if (active && k < nz) idw_next = ld_ids(o + PXY); else idw_next = out_pack;
        __syncthreads();                          // B1

        // ---- phase A: H' = H - nbar * curl E ------------------------------------------------------
        const VecR ex1 = my_stage[0 * kFusedThreads], ey1 = my_stage[1 * kFusedThreads];
        const VecR hx = my_stage[3 * kFusedThreads], hy = my_stage[4 * kFusedThreads], hz = my_stage[5 * kFusedThreads];
        const VecR exn = is_top ? s_top[lane] : smEx[r + 1][lane];
        const VecR ezn = is_top ? s_top[32 + lane] : smEz[r + 1][lane];
        const R ey0_r = shfl_down1(ey0.v[0]), ez_r = shfl_down1(ez.v[0]);
        int idc[V];
#pragma unroll
        for (int c = 0; c < V; ++c) idc[c] = (idw >> (8 * c)) & 0xff;
        const unsigned idj = smId[r - 1][lane];
        VecR nbx, nby, nbz, ncur;
        if (UMU) {
#pragma unroll
            for (int c = 0; c < V; ++c) nbx.v[c] = nby.v[c] = nbz.v[c] = ncur.v[c] = s_tab[0].n;
        } else {
#pragma unroll
            for (int c = 0; c < V; ++c) ncur.v[c] = s_tab[idc[c]].n;
            const R n_l = shfl_up1(ncur.v[V - 1]);
#pragma unroll
            for (int c = 0; c < V; ++c) {
                const R nj = s_tab[(idj >> (8 * c)) & 0xff].n;
                nbx.v[c] = lerp(c > 0 ? ncur.v[c > 0 ? c - 1 : 0] : n_l, ncur.v[c], fxv[c]);
                nby.v[c] = lerp(nj, ncur.v[c], fy);
                nbz.v[c] = lerp(nzp.v[c], ncur.v[c], fz);
            }
        }
        VecR hxn, hyn, hzn;
#pragma unroll
        for (int c = 0; c < V; ++c) {
            const R eyip = (c < V - 1) ? ey0.v[c < V - 1 ? c + 1 : c] : ey0_r;
            const R ezip = (c < V - 1) ? ez.v[c < V - 1 ? c + 1 : c] : ez_r;
            hxn.v[c] = hx.v[c] - nbx.v[c] * ((ezn.v[c] - ez.v[c]) * rdy - (ey1.v[c] - ey0.v[c]) * rdz);
            hyn.v[c] = hy.v[c] - nby.v[c] * ((ex1.v[c] - ex0.v[c]) * rdz - (ezip - ez.v[c]) * rdxv[c]);
            hzn.v[c] = hz.v[c] - nbz.v[c] * ((eyip - ey0.v[c]) * rdxv[c] - (exn.v[c] - ex0.v[c]) * rdy);
        }
        if (!active) {
#pragma unroll
            for (int c = 0; c < V; ++c) hxn.v[c] = hyn.v[c] = hzn.v[c] = R(0);
        }
        if (own) {
            *reinterpret_cast<VecR *>(p.Hn[0] + o) = hxn;
            *reinterpret_cast<VecR *>(p.Hn[1] + o) = hyn;
            *reinterpret_cast<VecR *>(p.Hn[2] + o) = hzn;
        }
        smHx[r][lane] = hxn; smHz[r][lane] = hzn;
        if (k < nz) issue_stage(k + 1); else cp_async_commit();   // slots 0..5 are free again
        __syncthreads();                          // B2

        // ---- phase B: E' = E + r (curl H' - J - sigma E), Joule squares ------------------------------
        const VecR hxj = smHx[r - 1][lane], hzj = smHz[r - 1][lane];
        const R hy_l = shfl_up1(hyn.v[V - 1]), hz_l = shfl_up1(hzn.v[V - 1]);
        MatEntry<R> A[V], Aj[V];
#pragma unroll
        for (int c = 0; c < V; ++c) { A[c] = s_tab[idc[c]]; Aj[c] = s_tab[(idj >> (8 * c)) & 0xff]; }
        MatEntry<R> A_l, Aj_l;
        A_l.a = shfl_up1(A[V - 1].a); A_l.b = shfl_up1(A[V - 1].b); A_l.m = shfl_up1(A[V - 1].m);
        Aj_l.a = shfl_up1(Aj[V - 1].a); Aj_l.b = shfl_up1(Aj[V - 1].b); Aj_l.m = shfl_up1(Aj[V - 1].m);
        // sources of this tile at plane k (rare): J per own edge
        R Jv[3][V];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int c = 0; c < V; ++c) Jv[a][c] = R(0);
        while (s_cur < s_end) {
            const int4 e = fs.tile_ent[s_cur];
            if (e.z > k) break;
            if (e.z == k && e.y == j) {
                const int ci = e.x - i0;
                if (ci >= 0 && ci < V) {
                    const int u = e.w >> 2, comp = e.w & 3;
                    R J = 0;
                    for (int q = src.cbeg[u]; q < src.cbeg[u + 1]; ++q) {
                        const int pt = src.con_port[q];
                        if (step < src.port_wlen[pt]) J = mad(src.con_scale[q], src.wave[src.port_woff[pt] + step], J);
                    }
#pragma unroll
                    for (int a = 0; a < 3; ++a)
#pragma unroll
                        for (int c = 0; c < V; ++c)
                            if (a == comp && c == ci) Jv[a][c] += J;
                }
            }
            ++s_cur;
        }
        const VecR lyPa = s_spill[0 * kFusedThreads + tid], lyPb = s_spill[1 * kFusedThreads + tid], lyPm = s_spill[2 * kFusedThreads + tid];
        const VecR lxPa = s_spill[3 * kFusedThreads + tid], lxPb = s_spill[4 * kFusedThreads + tid], lxPm = s_spill[5 * kFusedThreads + tid];
        VecR lya, lyb, lym, lxa, lxb, lxm;
        VecR exq, eyq, ezq;      // E^{n+1}
        VecR bx, by, bz;         // (2 Ebar)^2
#pragma unroll
        for (int c = 0; c < V; ++c) {
            const MatEntry<R> &Am = (c > 0) ? A[c > 0 ? c - 1 : 0] : A_l;
            const MatEntry<R> &Ajm = (c > 0) ? Aj[c > 0 ? c - 1 : 0] : Aj_l;
            lya.v[c] = lerp(Aj[c].a, A[c].a, fy); lyb.v[c] = lerp(Aj[c].b, A[c].b, fy); lym.v[c] = Aj[c].m * A[c].m;
            lxa.v[c] = lerp(Am.a, A[c].a, fxv[c]); lxb.v[c] = lerp(Am.b, A[c].b, fxv[c]); lxm.v[c] = Am.m * A[c].m;
            const R lxja = lerp(Ajm.a, Aj[c].a, fxv[c]), lxjb = lerp(Ajm.b, Aj[c].b, fxv[c]), lxjm = Ajm.m * Aj[c].m;
            const R hyim = (c > 0) ? hyn.v[c > 0 ? c - 1 : 0] : hy_l;
            const R hzim = (c > 0) ? hzn.v[c > 0 ? c - 1 : 0] : hz_l;
            // Ex(i,j,k): cells (j-1..j) x (k-1..k)
            {
                const R a = lerp(lyPa.v[c], lya.v[c], fz), b = lerp(lyPb.v[c], lyb.v[c], fz), m = lyPm.v[c] * lym.v[c];
                const R rr = loss_r<R, LOSS>(a, b), rm = m * rr;
                const R h2 = (LOSS == 0) ? R(2) * a * rr : R(2) - rr * b;
                const R X = ((hzn.v[c] - hzj.v[c]) * rty - (hyn.v[c] - hyp.v[c]) * rtz) - Jv[0][c];
                exq.v[c] = mad(rm, mad(-b, ex0.v[c], X), ex0.v[c]);
                const R t2 = mad(rm, X, h2 * ex0.v[c]);
                bx.v[c] = t2 * t2;
            }
            // Ey(i,j,k): cells (i-1..i) x (k-1..k)
            {
                const R a = lerp(lxPa.v[c], lxa.v[c], fz), b = lerp(lxPb.v[c], lxb.v[c], fz), m = lxPm.v[c] * lxm.v[c];
                const R rr = loss_r<R, LOSS>(a, b), rm = m * rr;
                const R h2 = (LOSS == 0) ? R(2) * a * rr : R(2) - rr * b;
                const R X = ((hxn.v[c] - hxp.v[c]) * rtz - (hzn.v[c] - hzim) * rtxv[c]) - Jv[1][c];
                eyq.v[c] = mad(rm, mad(-b, ey0.v[c], X), ey0.v[c]);
                const R t2 = mad(rm, X, h2 * ey0.v[c]);
                by.v[c] = t2 * t2;
            }
            // Ez(i,j,k): cells (i-1..i) x (j-1..j)
            {
                const R a = lerp(lxja, lxa.v[c], fy), b = lerp(lxjb, lxb.v[c], fy), m = lxjm * lxm.v[c];
                const R rr = loss_r<R, LOSS>(a, b), rm = m * rr;
                const R h2 = (LOSS == 0) ? R(2) * a * rr : R(2) - rr * b;
                const R X = ((hyn.v[c] - hyim) * rtxv[c] - (hxn.v[c] - hxj.v[c]) * rty) - Jv[2][c];
                ezq.v[c] = mad(rm, mad(-b, ez.v[c], X), ez.v[c]);
                const R t2 = mad(rm, X, h2 * ez.v[c]);
                bz.v[c] = t2 * t2;
            }
        }
        s_spill[0 * kFusedThreads + tid] = lya; s_spill[1 * kFusedThreads + tid] = lyb; s_spill[2 * kFusedThreads + tid] = lym;
        s_spill[3 * kFusedThreads + tid] = lxa; s_spill[4 * kFusedThreads + tid] = lxb; s_spill[5 * kFusedThreads + tid] = lxm;
        if (!active) {
#pragma unroll
            for (int c = 0; c < V; ++c) bx.v[c] = by.v[c] = bz.v[c] = R(0);
        }
        if (own) {
            *reinterpret_cast<VecR *>(p.En[0] + o) = exq;
            *reinterpret_cast<VecR *>(p.En[1] + o) = eyq;
            if (k < nz) *reinterpret_cast<VecR *>(p.En[2] + o) = ezq;
        }
        smBx[r][lane] = bx; smBz[r][lane] = bz;
        __syncthreads();                          // B3

        // ---- phase C: q(k-1) += dt sigma/16 (pend + Sxy(k)); pend = Sxy(k) + Sz(k) ---------------------
        cp_async_wait<1>();                       // q(k-1) has landed (stage(k+1) may still fly)
        {
            const VecR bxn = smBx[r + 1][lane], bzn = smBz[r + 1][lane];
            const R by_r = shfl_down1(by.v[0]), bz_r = shfl_down1(bz.v[0]), bzn_r = shfl_down1(bzn.v[0]);
            VecR qv = my_stage[6 * kFusedThreads];
#pragma unroll
            for (int c = 0; c < V; ++c) {
                const R byip = (c < V - 1) ? by.v[c < V - 1 ? c + 1 : c] : by_r;
                const R bzip = (c < V - 1) ? bz.v[c < V - 1 ? c + 1 : c] : bz_r;
                const R bznip = (c < V - 1) ? bzn.v[c < V - 1 ? c + 1 : c] : bzn_r;
                const R sxy = (bx.v[c] + bxn.v[c]) + (by.v[c] + byip);
                const R sz = (bz.v[c] + bzip) + (bzn.v[c] + bznip);
                qv.v[c] = mad(gq * sgp.v[c], pend.v[c] + sxy, qv.v[c]);
                pend.v[c] = sxy + sz;
            }
            if (own_q && k >= 1) *reinterpret_cast<VecR *>(p.q + o - PXY) = qv;
            // prefetch q(k) for the next iteration into the (now free) slot
            if (own_q && k < nz) cp_async16(my_stage + 6 * kFusedThreads, p.q + o);
            cp_async_commit();
        }
        // ---- advance ------------------------------------------------------------------------------------
        ex0 = ex1; ey0 = ey1; hxp = hxn; hyp = hyn; nzp = ncur;
#pragma unroll
        for (int c = 0; c < V; ++c) sgp.v[c] = A[c].b;
    }
    cp_async_wait<0>();
}

template <typename R>
cudaError_t launch_fused(const FusedPlan &plan, const DevParams<R> &p, const DevSources<R> &src,
                         const FusedSources &fs, int loss, bool uniform_mu, long long step, cudaStream_t stream) {
    using K = void (*)(DevParams<R>, DevSources<R>, FusedSources, int, long long);
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
    kern<<<plan.n_tiles, kFusedThreads, plan.smem_bytes, stream>>>(p, src, fs, plan.ntx, step);
    return cudaGetLastError();
}

}  // namespace em
