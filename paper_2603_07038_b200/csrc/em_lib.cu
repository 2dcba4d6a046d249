// em_lib.cu -- host side of libem.so: the C ABI declared in include/em.h.
// No torch types, no device allocation: the caller's workspace is carved here.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/em.h"
#include "em_aux.cuh"
#include "em_common.cuh"
#include "em_split.cuh"
#include "em_sweep.cuh"
#include "em_thermal.cuh"
#include "em_tile.cuh"

namespace {

thread_local std::string g_err;
int32_t fail(int32_t code, const std::string &msg) { g_err = msg; return code; }

#define CU(call)                                                                               \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(EM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));      \
    } while (0)

// Every entry point runs on the context's own device whatever the caller's current device is, and restores it.
struct DeviceGuard {
    int prev = -1; bool switched = false;
    explicit DeviceGuard(int dev) {
        if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

constexpr size_t kAlign = 256;
size_t align_up(size_t v, size_t a = kAlign) { return (v + a - 1) / a * a; }

struct Geometry {
    int nx, ny, nz, PX, PY, PZ;
    long long PXY, vol, origin;   // origin: elements from the allocation start to logical (0,0,0)
    long long alloc_elems;        // vol + guards
};

Geometry make_geometry(int nx, int ny, int nz) {
    Geometry g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    // nx + 2 for the i = -1 / nx + 1 pads; + 16 so that the id box of the TMA sweep (based 16 B before the
    // row) still holds the "outside" id of cell i = nx inside the row
    g.PX = (nx + 18 + 31) / 32 * 32;
    g.PY = ny + 3; g.PZ = nz + 3;
    g.PXY = (long long)g.PX * g.PY;
    g.vol = g.PXY * g.PZ;
    // one guard row in front (i = -1 of row j = -1, plane k = -1) and 2 behind (vector tails)
    g.origin = g.PX + g.PXY + g.PX;   // guard + plane k=-1 + row j=-1
    g.alloc_elems = g.vol + g.PX + std::max(2LL * g.PX, (long long)g.PX + 256);
    return g;
}

constexpr int kProbeChunk = 4096;
constexpr int kReduceBlocks = 1024;
constexpr int kTimingRing = 4096;

// Workspace carving: identical code computes sizes (base == nullptr) and pointers.
struct Carver {
    char *base; size_t off = 0;
    explicit Carver(void *b) : base(static_cast<char *>(b)) {}
    template <typename T> T *take(size_t n) {
        off = align_up(off);
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

template <typename R>
struct Carved {
    R *field[12];            // E[3], En[3], H[3], Hn[3] allocation starts
    R *q;
    uint8_t *mat;
    em::MatEntry<R> *table;
    R *zgeo;                 // {fz, rdz, rtz, 0} x (PZ + 8)
    R *axis[9];              // rdx, rtx, fx, rdy, rty, fy, rdz, rtz, fz (allocation starts; index -1 first)
    double *vx, *vy, *vz;    // cell sizes in fp64 for the Joule total
    double *partial, *scalar;
    long long *probe_off; int *probe_comp; double *probe_out;
    // sources
    long long *src_off; int *src_comp; R *src_r; int *src_cbeg; int *src_flags;
    int *con_port; R *con_scale; long long *port_woff, *port_wlen; R *wave;
    // fused-sweep tile source index
    int *tile_sbeg; int4 *tile_ent; int *order;
    // thermal coupling (only when em_grid.thermal != 0): theta ping-pong, sigma(T) per cell, thermal table
    R *theta[2]; R *sig, *sig2; em::ThEntry<R> *ttable;
};

template <typename R>
size_t carve(const Geometry &g, const em_grid &gr, void *base, Carved<R> *c, int n_items) {
    Carver w(base);
    Carved<R> tmp;
    Carved<R> &o = c ? *c : tmp;
    // leapfrog: E, En, H, Hn (12 arrays); E-only (eq. (2)): three rotating levels of e (9 arrays)
    const int n_field = gr.formulation == EM_FORM_EONLY ? 9 : 12;
    for (int a = 0; a < 12; ++a) o.field[a] = a < n_field ? w.take<R>(g.alloc_elems) : nullptr;
    o.q = w.take<R>(g.alloc_elems);
    o.mat = w.take<uint8_t>(g.alloc_elems);
    o.table = w.take<em::MatEntry<R>>(em::kMaxTable);
    const int len[3] = {g.PX + 8, g.PY + 8, g.PZ + 8};   // 4 leading + 4 trailing pads (aligned vector loads)
    for (int a = 0; a < 9; ++a) o.axis[a] = w.take<R>(len[a / 3]);
    o.zgeo = w.take<R>((size_t)4 * len[2]);
    o.vx = w.take<double>(g.nx); o.vy = w.take<double>(g.ny); o.vz = w.take<double>(g.nz);
    o.partial = w.take<double>(kReduceBlocks); o.scalar = w.take<double>(1);
    o.probe_off = w.take<long long>(kProbeChunk); o.probe_comp = w.take<int>(kProbeChunk);
    o.probe_out = w.take<double>(kProbeChunk);
    const size_t me = (size_t)std::max<int64_t>(gr.max_source_edges, 1), mp = (size_t)std::max(gr.max_ports, 1);
    o.src_off = w.take<long long>(me); o.src_comp = w.take<int>(me); o.src_r = w.take<R>(me);
    o.src_cbeg = w.take<int>(me + 1); o.src_flags = w.take<int>(me);
    o.con_port = w.take<int>(me); o.con_scale = w.take<R>(me);
    o.port_woff = w.take<long long>(mp); o.port_wlen = w.take<long long>(mp);
    o.wave = w.take<R>((size_t)std::max<int64_t>(gr.max_wave_samples, 1));
    o.tile_sbeg = w.take<int>((size_t)n_items + 1);
    o.order = w.take<int>((size_t)n_items);
    o.tile_ent = w.take<int4>(4 * me);
    o.theta[0] = o.theta[1] = o.sig = o.sig2 = nullptr; o.ttable = nullptr;
    if (gr.thermal) {
        o.theta[0] = w.take<R>(g.alloc_elems); o.theta[1] = w.take<R>(g.alloc_elems); o.sig = w.take<R>(g.alloc_elems);
        o.sig2 = w.take<R>(g.alloc_elems);
        o.ttable = w.take<em::ThEntry<R>>(em::kMaxTable);
    }
    return align_up(w.off);
}

struct Timing {
    bool enabled = false;
    std::vector<cudaEvent_t> beg, end;
    int head = 0, pending = 0;
    long long launches = 0; double ms = 0.0;
};

}  // namespace

// ------------------------------------------------------------------------------------------------
struct em_ctx {
    virtual ~em_ctx() {}
    virtual int32_t set_source(int32_t, const em_port *, const em_edge *, int64_t, const double *, int64_t) = 0;
    virtual int32_t set_field(int32_t, const void *, int32_t) = 0;
    virtual int32_t get_field(int32_t, void *, int32_t) = 0;
    virtual int32_t plane(int32_t comp, int32_t k, void *dst, const void *src, int32_t is_dev) = 0;
    virtual int32_t step(int64_t) = 0;
    virtual int32_t joule(void *, void *, double *, int32_t) = 0;
    virtual int32_t probe(int32_t, const em_probe_pt *, double *) = 0;
    virtual int32_t reset() = 0;
    virtual int32_t set_thermal(const em_thermal_material *, int32_t) = 0;
    virtual int32_t temperature_rise(void *, const void *, int32_t) = 0;
    virtual int32_t halo(int32_t kp, int32_t kl, void *dst, const void *src, void *stream) = 0;
    virtual int32_t halo_elems(int64_t *n) = 0;
    virtual int32_t joule_layers(int32_t k0, int32_t k1, double *total) = 0;
    virtual int32_t wall_offset(int32_t side, int32_t parity, int32_t comp, size_t *off) = 0;
    virtual int32_t set_peer_halo(int32_t side, int32_t k_send, void *const dst[4]) = 0;
    virtual int32_t set_joule_energy(const void *src, int32_t is_dev) = 0;
    virtual int32_t check_finite(int32_t *all_finite) = 0;
    int64_t step_index = 0, launches = 0;
    Timing timing;
    const char *main_kernel = "";
    cudaStream_t stream = nullptr;
    int device = -1;                    // the device that owns the workspace
    int32_t timing_flush();
};

int32_t em_ctx::timing_flush() {
    Timing &t = timing;
    while (t.pending > 0) {
        const int idx = (t.head - t.pending + kTimingRing) % kTimingRing;
        CU(cudaEventSynchronize(t.end[idx]));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, t.beg[idx], t.end[idx]));
        t.ms += ms; t.launches += 1; t.pending -= 1;
    }
    return EM_OK;
}

namespace {

template <typename R>
struct Ctx final : em_ctx {
    Geometry g;
    em_grid grid;
    int loss = 0, kernel = EM_KERNEL_SPLIT;
    double dt = 0;
    Carved<R> c;
    em::DevParams<R> p;
    std::vector<em_material> table;
    std::vector<uint8_t> fixed_cell;   // host copy of "mask == 0" per material (incl. outside)
    std::vector<uint8_t> host_mat;     // host copy of the ids (for argument checks of sources)
    int n_unique = 0, n_ports = 0;
    em::DevSources<R> src;
    em::SweepPlan plan;
    bool uniform_mu = true;
    bool eonly = false;                 // E-only three-level recurrence (em_grid.formulation = EM_FORM_EONLY)
    em::SweepKernel<R> sweep_kernel = nullptr;
    int n_field = 12;

    R *org(int a) const { return c.field[a] + g.origin; }

    // leapfrog: E / En ping-pong in arrays 0-5 (e_cur), H / Hn in 6-11 (h_cur).
    // E-only: the three levels rotate through the array triples 0-2, 3-5, 6-8: e^n = triple lvl, e^{n-1} = triple
    // (lvl + 2) % 3 (bound to p.H: the sweep stages it in the H slots), e^{n+1} is written to triple (lvl + 1) % 3.
    void bind() {
        for (int a = 0; a < 3; ++a) {
            if (eonly) {
                p.E[a] = org(lvl * 3 + a); p.En[a] = org(((lvl + 1) % 3) * 3 + a);
                p.H[a] = org(((lvl + 2) % 3) * 3 + a); p.Hn[a] = nullptr;
            } else {
                p.E[a] = org(e_cur * 3 + a); p.En[a] = org((1 - e_cur) * 3 + a);
                p.H[a] = org(6 + h_cur * 3 + a); p.Hn[a] = org(6 + (1 - h_cur) * 3 + a);
            }
        }
        // the neighbouring slabs step in lockstep: their E^{n+1} array has the parity of mine
        for (int sd = 0; sd < 2; ++sd) for (int cc = 0; cc < 2; ++cc) p.peer_e[sd][cc] = peer_dst[sd][1 - e_cur][cc];
    }
    int e_cur = 0, h_cur = 0, lvl = 0;

    int32_t init(const em_grid *gr, const uint8_t *mat_id, const em_material *tab, int32_t n_mat, double dt_,
                 void *workspace, size_t ws_bytes, void *stream_);
    int32_t zero_state();
    int32_t set_source(int32_t, const em_port *, const em_edge *, int64_t, const double *, int64_t) override;
    int32_t set_field(int32_t, const void *, int32_t) override;
    int32_t get_field(int32_t, void *, int32_t) override;
    int32_t plane(int32_t comp, int32_t k, void *dst, const void *src, int32_t is_dev) override;
    int32_t step(int64_t) override;
    int32_t joule(void *, void *, double *, int32_t) override;
    int32_t probe(int32_t, const em_probe_pt *, double *) override;
    int32_t reset() override { return zero_state(); }
    int32_t set_thermal(const em_thermal_material *, int32_t) override;
    int32_t temperature_rise(void *dst, const void *src, int32_t is_dev) override;
    int32_t halo(int32_t kp, int32_t kl, void *dst, const void *src, void *stream) override;
    int32_t halo_elems(int64_t *n) override {
        *n = (int64_t)(g.ny + 1) * g.nx + (int64_t)g.ny * (g.nx + 1) +
             (!thermal_on ? 0 : nodal ? (int64_t)(g.ny + 1) * (g.nx + 1) : (int64_t)g.ny * g.nx);
        return EM_OK;
    }
    int32_t joule_layers(int32_t k0, int32_t k1, double *total) override;
    int32_t wall_offset(int32_t side, int32_t parity, int32_t comp, size_t *off) override;
    int32_t set_peer_halo(int32_t side, int32_t k_send, void *const dst[4]) override;
    int32_t set_joule_energy(const void *src, int32_t is_dev) override;
    int32_t check_finite(int32_t *all_finite) override;
    void *ws_base = nullptr;
    R *peer_dst[2][2][2] = {};          // [side][parity of the neighbour's E array][comp]
    int32_t step_thermal();
    int32_t step_thermal_nodal();
    bool nodal = false;                 // em_grid.thermal = EM_THERMAL_NODE: theta on the mesh nodes (split kernels)
    int32_t step_thermal_sweep();
    int sg_cur = 0;                     // which sigma(T) buffer is current (the coupled sweep ping-pongs them)
    R *sig_buf(int which) const { return (which ? c.sig2 : c.sig) + g.origin; }
    CUtensorMap map_sig[2], map_theta[2];
    int32_t refresh_sigma();
    bool thermal_on = false;            // em_set_thermal was called
    int th_cur = 0;
    int n_mat_ = 0;
    em::ThermalParams<R> tp() const {
        em::ThermalParams<R> t;
        t.theta = c.theta[th_cur] + g.origin; t.theta_n = c.theta[1 - th_cur] + g.origin;
        t.sig = sig_buf(sg_cur); t.ttable = c.ttable;
        return t;
    }
    int32_t step_split();
    int32_t step_tma();
    int32_t make_maps();
    CUtensorMap map_field[12], map_q, map_mat;   // TMA descriptors of the padded arrays (sweep boxes)
    CUtensorMap map_prev[9];                     // E-only: the same arrays in the role of e^{n-1} (boxes of rows -1 .. TY)
    size_t sweep_smem = 0;
    void comp_dims(int comp, int *sx, int *sy, int *sz) const {
        const int nx = g.nx, ny = g.ny, nz = g.nz;
        switch (comp) {
        case 0: case 6: *sx = nx;     *sy = ny + 1; *sz = nz + 1; break;
        case 1: case 7: *sx = nx + 1; *sy = ny;     *sz = nz + 1; break;
        case 2: case 8: *sx = nx + 1; *sy = ny + 1; *sz = nz;     break;
        case 3: *sx = nx + 1; *sy = ny;     *sz = nz;     break;
        case 4: *sx = nx;     *sy = ny + 1; *sz = nz;     break;
        default:*sx = nx;     *sy = ny;     *sz = nz + 1; break;
        }
    }
    // components 0-2: E^n (e^n), 3-5: H^{n-1/2} (leapfrog only), 6-8: e^{n-1} (E-only only)
    R *comp_ptr(int comp) const { return comp < 3 ? p.E[comp] : comp < 6 ? p.H[comp - 3] : p.H[comp - 6]; }
    bool comp_ok(int comp) const { return comp >= 0 && (comp < 3 || (eonly ? (comp >= 6 && comp < 9) : comp < 6)); }
    dim3 node_grid(dim3 b, int ex) const { return dim3((g.nx + ex + b.x - 1) / b.x, (g.ny + ex + b.y - 1) / b.y, g.nz + ex); }
    int32_t record_begin();
    int32_t record_end();
};

int32_t validate_grid(const em_grid *g) {
    if (!g) return fail(EM_ERR_INVALID_ARG, "grid is null");
    if (g->nx < 1 || g->ny < 1 || g->nz < 1) return fail(EM_ERR_INVALID_ARG, "grid dims must be >= 1");
    if ((long long)g->nx + 34 > 2147483647LL / 4) return fail(EM_ERR_INVALID_ARG, "nx too large");
    if (g->ny > 8 * 65535 - 8 || g->nz > 65534)                     // (the light kernels run one 32 x 8 block column per z plane)
        return fail(EM_ERR_INVALID_ARG, "ny must be <= 524272 and nz <= 65534");
    if (g->precision != 32 && g->precision != 64) return fail(EM_ERR_INVALID_ARG, "precision must be 32 or 64");
    if (g->loss_mode != EM_LOSS_CD && g->loss_mode != EM_LOSS_EXP) return fail(EM_ERR_INVALID_ARG, "bad loss_mode");
    if (g->kernel < EM_KERNEL_AUTO || g->kernel > EM_KERNEL_TMA) return fail(EM_ERR_INVALID_ARG, "bad kernel strategy");
    if (g->thermal < 0 || g->thermal > EM_THERMAL_NODE) return fail(EM_ERR_INVALID_ARG, "thermal must be 0, 1 (per cell) or 2 (per node)");
    if (g->thermal == EM_THERMAL_NODE && g->kernel == EM_KERNEL_TMA)
        return fail(EM_ERR_UNSUPPORTED, "the nodal thermal stage runs on the split kernels");
    if (g->formulation != EM_FORM_LEAPFROG && g->formulation != EM_FORM_EONLY) return fail(EM_ERR_INVALID_ARG, "bad formulation");
    if (g->formulation == EM_FORM_EONLY && (g->thermal || g->kernel == EM_KERNEL_SPLIT))
        return fail(EM_ERR_UNSUPPORTED, "the E-only recurrence runs on the TMA sweep, without thermal coupling");
    if (g->z_chunks < 0 || g->z_chunks > em::kSweepMaxZSplit) return fail(EM_ERR_INVALID_ARG, "z_chunks must be 0 (auto) .. 8");
    if (g->max_ports < 0 || g->max_source_edges < 0 || g->max_wave_samples < 0)
        return fail(EM_ERR_INVALID_ARG, "negative source capacity");
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::zero_state() {
    for (int a = 0; a < n_field; ++a) CU(cudaMemsetAsync(c.field[a], 0, sizeof(R) * g.alloc_elems, stream));
    CU(cudaMemsetAsync(c.q, 0, sizeof(R) * g.alloc_elems, stream));
    e_cur = h_cur = lvl = 0; bind();
    step_index = 0;
    if (grid.thermal) {
        CU(cudaMemsetAsync(c.theta[0], 0, sizeof(R) * g.alloc_elems, stream));
        CU(cudaMemsetAsync(c.theta[1], 0, sizeof(R) * g.alloc_elems, stream));
        th_cur = 0;
        if (thermal_on) return refresh_sigma();
    }
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::init(const em_grid *gr, const uint8_t *mat_id, const em_material *tab, int32_t n_mat, double dt_,
                     void *workspace, size_t ws_bytes, void *stream_) {
    grid = *gr; grid.dx = grid.dy = grid.dz = nullptr;
    g = make_geometry(gr->nx, gr->ny, gr->nz);
    loss = gr->loss_mode; dt = dt_;
    stream = static_cast<cudaStream_t>(stream_);
    eonly = gr->formulation == EM_FORM_EONLY;
    n_field = eonly ? 9 : 12;
    {
        int n_sm = 0;
        CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device));
        plan = em::make_sweep_plan(g.nx, g.ny, g.nz, (int)sizeof(R), n_sm, gr->z_chunks, gr->thermal != 0);
    }
    kernel = gr->kernel;
    const int max_items = plan.n_tiles * em::kSweepMaxZSplit;
    const size_t need = carve<R>(g, *gr, nullptr, nullptr, max_items);
    if (ws_bytes < need) return fail(EM_ERR_WORKSPACE_TOO_SMALL, "workspace too small");
    carve<R>(g, *gr, workspace, &c, max_items);
    sweep_smem = em::sweep_smem_bytes((int)sizeof(R), n_mat + 2);
    n_mat_ = n_mat;
    // thermal coupling: the coupled TMA sweep (sigma(T) planes staged beside the ids) or, if its shared-memory layout
    // does not fit / on request, the split kernels (em_thermal.cuh)
    nodal = gr->thermal == EM_THERMAL_NODE;
    if (nodal) kernel = EM_KERNEL_SPLIT;                 // (theta on the mesh nodes: em_thermal.cuh k_thermal_nodal)
    if (gr->thermal && !nodal) {
        sweep_smem = em::sweep_smem_bytes((int)sizeof(R), n_mat + 2, true);
        if (kernel == EM_KERNEL_AUTO) kernel = EM_KERNEL_TMA;
    }
    if (kernel == EM_KERNEL_AUTO) kernel = EM_KERNEL_TMA;
    if (kernel == EM_KERNEL_TMA) {           // (the layout holds the largest table, 255 + 2 entries, in both precisions)
        int optin = 0;
        CU(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
        if (sweep_smem > (size_t)optin) {
            // (only the fp64 coupled sweep with > 250 materials: its two tables of 32-B entries exceed the layout by 160 B)
            if (gr->thermal && gr->kernel == EM_KERNEL_AUTO) kernel = EM_KERNEL_SPLIT;
            else return fail(EM_ERR_UNSUPPORTED, "the sweep's shared-memory layout does not fit this device");
        }
    }
    main_kernel = kernel == EM_KERNEL_TMA ? "k_sweep_tma" : "k_split_e";

    // ---- material table -> (eps/dt, sigma, mask, dt/mu), built in fp64, rounded once ----------
    table.assign(tab, tab + n_mat);
    // table = the materials, then (only with a PMC wall) the "outside, beyond PMC walls only" entry whose mask is 1,
    // then, always last, the "outside / PEC" entry whose mask is 0 (what fixes the tangential E of PEC walls)
    bool any_pmc = false;
    for (int b = 0; b < 6; ++b) any_pmc = any_pmc || gr->bc[b] == EM_BC_PMC;
    const int n_table = n_mat + (any_pmc ? 2 : 1);
    std::vector<em::MatEntry<R>> ht(n_table);
    fixed_cell.assign(n_table, 0);
    for (int m = 0; m < n_mat; ++m) {
        const bool pec = (tab[m].flags & EM_MAT_PEC) != 0;
        ht[m].a = (R)(tab[m].eps / dt); ht[m].b = (R)tab[m].sigma;
        ht[m].m = pec ? R(0) : R(1); ht[m].n = (R)(dt / tab[m].mu);
        fixed_cell[m] = pec;
    }
    if (any_pmc) { ht[n_mat].a = R(1); ht[n_mat].b = R(0); ht[n_mat].m = R(1); ht[n_mat].n = R(0); }
    ht[n_table - 1].a = R(1); ht[n_table - 1].b = R(0); ht[n_table - 1].m = R(0); ht[n_table - 1].n = R(0);
    fixed_cell[n_table - 1] = 1;
    CU(cudaMemcpyAsync(c.table, ht.data(), sizeof(em::MatEntry<R>) * n_table, cudaMemcpyHostToDevice, stream));

    // ---- per-axis arrays, index -1 .. n+1 (+ slack), fp64 then rounded once -------------------
    const double *d[3] = {gr->dx, gr->dy, gr->dz};
    const int n[3] = {g.nx, g.ny, g.nz};
    const int len[3] = {g.PX + 8, g.PY + 8, g.PZ + 8};
    std::vector<std::vector<R>> hax(9);
    for (int a = 0; a < 3; ++a) {
        auto dd = [&](int i) { return (i >= 0 && i < n[a]) ? d[a][i] : 0.0; };
        std::vector<R> rd(len[a], R(0)), rt(len[a], R(0)), f(len[a], R(0));
        for (int s = 0; s < len[a]; ++s) {
            const int i = s - 4;
            if (i >= 0 && i < n[a]) rd[s] = (R)(1.0 / d[a][i]);
            const double lo = dd(i - 1), hi = dd(i);
            if (lo + hi > 0.0) { rt[s] = (R)(2.0 / (lo + hi)); f[s] = (R)(hi / (lo + hi)); }
        }
        hax[a * 3 + 0] = rd; hax[a * 3 + 1] = rt; hax[a * 3 + 2] = f;
    }
    for (int a = 0; a < 9; ++a)
        CU(cudaMemcpyAsync(c.axis[a], hax[a].data(), sizeof(R) * hax[a].size(), cudaMemcpyHostToDevice, stream));
    {
        std::vector<R> zg((size_t)4 * len[2], R(0));
        for (int s = 0; s < len[2]; ++s) { zg[4 * s + 0] = hax[8][s]; zg[4 * s + 1] = hax[6][s]; zg[4 * s + 2] = hax[7][s]; }
        CU(cudaMemcpyAsync(c.zgeo, zg.data(), sizeof(R) * zg.size(), cudaMemcpyHostToDevice, stream));
        CU(cudaStreamSynchronize(stream));      // zg is a local
    }
    CU(cudaMemcpyAsync(c.vx, gr->dx, sizeof(double) * g.nx, cudaMemcpyHostToDevice, stream));
    CU(cudaMemcpyAsync(c.vy, gr->dy, sizeof(double) * g.ny, cudaMemcpyHostToDevice, stream));
    CU(cudaMemcpyAsync(c.vz, gr->dz, sizeof(double) * g.nz, cudaMemcpyHostToDevice, stream));

    // ---- material ids: halo = the "outside / PEC" id, interior copied with a pitched 3-D copy; pad cells that
    // lie beyond PMC walls only get the "outside / PMC" id (em_aux.cuh k_pad_pmc) -----------------------------
    CU(cudaMemsetAsync(c.mat, n_table - 1, g.alloc_elems, stream));
    if (any_pmc) {
        int pmc_mask = 0;
        for (int b = 0; b < 6; ++b) if (gr->bc[b] == EM_BC_PMC) pmc_mask |= 1 << b;
        const long long n = g.vol;
        EM_LAUNCH(em::k_pad_pmc, (unsigned)((n + 255) / 256), 256, 0, stream)(c.mat + g.origin - g.PXY - g.PX - 1, g.nx, g.ny, g.nz,
                                                                        g.PX, g.PY, n, pmc_mask, (uint8_t)n_mat);
        CU(cudaGetLastError());
    }
    {
        cudaMemcpy3DParms m = {};
        m.srcPtr = make_cudaPitchedPtr(const_cast<uint8_t *>(mat_id), g.nx, g.nx, g.ny);
        m.dstPtr = make_cudaPitchedPtr(c.mat + g.origin, g.PX, g.PX, g.PY);
        m.extent = make_cudaExtent(g.nx, g.ny, g.nz);
        m.kind = cudaMemcpyHostToDevice;
        CU(cudaMemcpy3DAsync(&m, stream));
    }
    host_mat.assign(mat_id, mat_id + (size_t)g.nx * g.ny * g.nz);
    uniform_mu = true;
    {
        std::vector<char> used(n_mat, 0);
        for (uint8_t v : host_mat) used[v] = 1;
        double mu0 = -1;
        for (int m = 0; m < n_mat; ++m) if (used[m]) { if (mu0 < 0) mu0 = tab[m].mu; else if (tab[m].mu != mu0) uniform_mu = false; }
        if (tab[0].mu != mu0) uniform_mu = false;     // the uniform-mu kernels read dt/mu from table entry 0
    }

    // ---- device parameter block -----------------------------------------------------------------
    p.nx = g.nx; p.ny = g.ny; p.nz = g.nz; p.PX = g.PX; p.PY = g.PY; p.PXY = g.PXY;
    p.q = c.q + g.origin; p.mat = c.mat + g.origin; p.table = c.table; p.n_table = n_table;
    p.warm_lo = gr->bc[4] == EM_BC_PMC ? 1 : 0;
    p.rdx = c.axis[0] + 4; p.rtx = c.axis[1] + 4; p.fx = c.axis[2] + 4;
    p.rdy = c.axis[3] + 4; p.rty = c.axis[4] + 4; p.fy = c.axis[5] + 4;
    p.rdz = c.axis[6] + 4; p.rtz = c.axis[7] + 4; p.fz = c.axis[8] + 4;
    p.zgeo = c.zgeo + 16;
    p.dt = (R)dt;
    p.peer_k[0] = p.peer_k[1] = -1000; p.peer_skip = 0;
    ws_base = workspace;
    src = em::DevSources<R>{};
    src.n_unique = 0;
    CU(cudaMemsetAsync(c.tile_sbeg, 0, sizeof(int) * (plan.n_tiles * plan.nzs + 1), stream));
    {
        std::vector<int> ord((size_t)plan.n_tiles * plan.nzs);
        em::launch_order(plan, ord.data());
        CU(cudaMemcpyAsync(c.order, ord.data(), sizeof(int) * ord.size(), cudaMemcpyHostToDevice, stream));
        CU(cudaStreamSynchronize(stream));              // ord is a local
    }
    int32_t rc = zero_state();
    if (rc) return rc;
    if (kernel == EM_KERNEL_TMA) {
        rc = make_maps(); if (rc) return rc;
        // one instantiation per context: selected and given its dynamic shared memory once, here
        sweep_kernel = em::select_sweep<R>(loss, uniform_mu, gr->thermal != 0, eonly);
        CU(em::configure_sweep<R>(sweep_kernel, sweep_smem));
    }
    CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

// ---- TMA descriptors of the sweep boxes (em_sweep.cuh) -----------------------------------------------
// Field-like arrays: 3-D map over the padded allocation based at logical (-V, -1, -1) (16-B aligned:
// V elements = 16 B), dims (PX, PY, PZ); box = 32 lanes x 16 (Ey, H) or 17 (Ex, Ez) rows x 1 plane;
// q: box 30 lanes x 14 rows; ids (uint8): based 16 B before the row, box 32 V bytes x 18 rows.
// Out-of-range box parts are zero-filled, which equals the pad content of the field arrays.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <typename R>
int32_t Ctx<R>::make_maps() {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CU(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return fail(EM_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(fn);
    const int V = 16 / (int)sizeof(R);
    const cuuint32_t ones[3] = {1, 1, 1};
#ifndef EM_SWEEP_PROMO
#define EM_SWEEP_PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_128B
#endif
    const CUtensorMapL2promotion promo = (CUtensorMapL2promotion)EM_SWEEP_PROMO;
    auto encode = [&](CUtensorMap *m, CUtensorMapDataType dt, size_t esz, void *base, int bx, int by) -> int32_t {
        const cuuint64_t dims[3] = {(cuuint64_t)g.PX, (cuuint64_t)g.PY, (cuuint64_t)g.PZ};
        const cuuint64_t strides[2] = {(cuuint64_t)g.PX * esz, (cuuint64_t)g.PXY * esz};
        const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
        CUresult r = enc(m, dt, 3, base, dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(EM_ERR_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
        return EM_OK;
    };
    const int sw_warps = grid.thermal ? em::Tile<sizeof(R), true>::warps : em::Tile<sizeof(R)>::warps;
    const CUtensorMapDataType fdt = sizeof(R) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    for (int a = 0; a < n_field; ++a) {
        const int comp = a % 3, is_e = eonly || a < 6;
        const int rows = (is_e && comp != 1) ? sw_warps + 1 : sw_warps;         // Ex, Ez carry row TY+1
        int32_t rc = encode(&map_field[a], fdt, sizeof(R), c.field[a] + g.PX - V, 32 * V, rows);
        if (rc) return rc;
        if (eonly) { rc = encode(&map_prev[a], fdt, sizeof(R), c.field[a] + g.PX - V, 32 * V, sw_warps); if (rc) return rc; }
    }
    int32_t rc = encode(&map_q, fdt, sizeof(R), c.q + g.PX - V, 30 * V, sw_warps - 2);
    if (rc) return rc;
    rc = encode(&map_mat, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, c.mat + g.PX - em::kSwIdShift, 32 * V + 16, sw_warps + 2);
    if (rc) return rc;
    if (grid.thermal) {                                   // sigma(T) planes of the coupled sweep: rows -2 .. TY
        rc = encode(&map_sig[0], fdt, sizeof(R), c.sig + g.PX - V, 32 * V, sw_warps + 1); if (rc) return rc;
        rc = encode(&map_sig[1], fdt, sizeof(R), c.sig2 + g.PX - V, 32 * V, sw_warps + 1); if (rc) return rc;
        for (int q = 0; q < 2 && em::kFusedConduction; ++q) {     // (experimental fused conduction) theta^n planes: rows -1 .. TY
            rc = encode(&map_theta[q], fdt, sizeof(R), c.theta[q] + g.PX - V, 32 * V, sw_warps); if (rc) return rc;
        }
    }
    return EM_OK;
}

// ---- sources ------------------------------------------------------------------------------------
template <typename R>
int32_t Ctx<R>::set_source(int32_t np, const em_port *ports, const em_edge *edges, int64_t ne,
                           const double *wave, int64_t ns) {
    if (np < 0 || ne < 0 || ns < 0) return fail(EM_ERR_INVALID_ARG, "negative count");
    if ((np && !ports) || (ne && !edges) || (ns && !wave)) return fail(EM_ERR_INVALID_ARG, "null source array");
    if (np > grid.max_ports || ne > grid.max_source_edges || ns > grid.max_wave_samples)
        return fail(EM_ERR_WORKSPACE_TOO_SMALL, "source set exceeds the capacities given to em_create");
    for (int64_t e = 0; e < ne; ++e) {
        if (edges[e].comp < 0 || edges[e].comp > 2) return fail(EM_ERR_INVALID_ARG, "edge comp must be 0..2");
        int sx, sy, sz; comp_dims(edges[e].comp, &sx, &sy, &sz);
        if (edges[e].i < 0 || edges[e].i >= sx || edges[e].j < 0 || edges[e].j >= sy || edges[e].k < 0 || edges[e].k >= sz)
            return fail(EM_ERR_INVALID_ARG, "source edge outside the grid");
    }
    for (int q = 0; q < np; ++q) {
        if (ports[q].edge_begin < 0 || ports[q].edge_end < ports[q].edge_begin || ports[q].edge_end > ne)
            return fail(EM_ERR_INVALID_ARG, "port edge range");
        if (ports[q].wave_offset < 0 || ports[q].wave_len < 0 || ports[q].wave_offset + ports[q].wave_len > ns)
            return fail(EM_ERR_INVALID_ARG, "port waveform range");
    }
    // contributions (edge, port) sorted by tile of the fused sweep, then by offset: unique edges own
    // their contributions in input order, so overlapping ports add deterministically
    struct Con { long long off; int comp, port, i, j, k; R scale; int64_t seq; };
    std::vector<Con> cons;
    for (int q = 0; q < np; ++q)
        for (int64_t e = ports[q].edge_begin; e < ports[q].edge_end; ++e) {
            Con cn;
            cn.off = ((long long)edges[e].k * g.PY + edges[e].j) * g.PX + edges[e].i;
            cn.comp = edges[e].comp; cn.port = q; cn.scale = (R)(ports[q].amplitude * edges[e].weight);
            cn.i = edges[e].i; cn.j = edges[e].j; cn.k = edges[e].k;
            cn.seq = (int64_t)cons.size();
            cons.push_back(cn);
        }
    if ((int64_t)cons.size() > grid.max_source_edges)
        return fail(EM_ERR_WORKSPACE_TOO_SMALL, "more (edge, port) pairs than max_source_edges");
    std::sort(cons.begin(), cons.end(), [](const Con &a, const Con &b) {
        if (a.off != b.off) return a.off < b.off;
        if (a.comp != b.comp) return a.comp < b.comp;
        return a.seq < b.seq;
    });
    std::vector<long long> u_off; std::vector<int> u_comp, u_cbeg, c_port; std::vector<R> c_scale;
    struct TE { int tile; int4 e; };
    std::vector<TE> tes;
    for (size_t s = 0; s < cons.size(); ++s) {
        if (s == 0 || cons[s].off != cons[s - 1].off || cons[s].comp != cons[s - 1].comp) {
            const int u = (int)u_off.size();
            u_off.push_back(cons[s].off); u_comp.push_back(cons[s].comp); u_cbeg.push_back((int)s);
            int tl[4];
            const int nt = em::tiles_of_node(plan, cons[s].i, cons[s].j, tl);
            for (int t = 0; t < nt; ++t) tes.push_back(TE{tl[t], make_int4(cons[s].i, cons[s].j, cons[s].k, u * 4 + cons[s].comp)});
        }
        c_port.push_back(cons[s].port); c_scale.push_back(cons[s].scale);
    }
    u_cbeg.push_back((int)cons.size());
    const int nu = (int)u_off.size();
    std::stable_sort(tes.begin(), tes.end(), [](const TE &a, const TE &b) {
        if (a.tile != b.tile) return a.tile < b.tile;
        if (a.e.z != b.e.z) return a.e.z < b.e.z;
        if (a.e.y != b.e.y) return a.e.y < b.e.y;
        return a.e.x < b.e.x;
    });
    // cursor per work item (tile, z chunk): the entries of a tile are sorted by k, so the items of a tile
    // are consecutive ranges
    const int n_items = plan.n_tiles * plan.nzs;
    std::vector<int> tile_beg(n_items + 1, 0);
    std::vector<int4> tile_ent(tes.size());
    for (size_t s = 0; s < tes.size(); ++s) {
        tile_beg[tes[s].tile * plan.nzs + plan.chunk_of(tes[s].e.z) + 1] += 1;
        tile_ent[s] = tes[s].e;
    }
    for (int t = 0; t < n_items; ++t) tile_beg[t + 1] += tile_beg[t];
    std::vector<long long> woff(std::max(np, 1)), wlen(std::max(np, 1));
    for (int q = 0; q < np; ++q) { woff[q] = ports[q].wave_offset; wlen[q] = ports[q].wave_len; }
    std::vector<R> hw((size_t)std::max<int64_t>(ns, 1));
    for (int64_t s = 0; s < ns; ++s) hw[s] = (R)wave[s];

    CU(cudaStreamSynchronize(stream));
    if (nu) {
        CU(cudaMemcpyAsync(c.src_off, u_off.data(), sizeof(long long) * nu, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(c.src_comp, u_comp.data(), sizeof(int) * nu, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(c.con_port, c_port.data(), sizeof(int) * c_port.size(), cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(c.con_scale, c_scale.data(), sizeof(R) * c_scale.size(), cudaMemcpyHostToDevice, stream));
    }
    CU(cudaMemcpyAsync(c.src_cbeg, u_cbeg.data(), sizeof(int) * (nu + 1), cudaMemcpyHostToDevice, stream));
    CU(cudaMemcpyAsync(c.tile_sbeg, tile_beg.data(), sizeof(int) * (n_items + 1), cudaMemcpyHostToDevice, stream));
    if (!tile_ent.empty())
        CU(cudaMemcpyAsync(c.tile_ent, tile_ent.data(), sizeof(int4) * tile_ent.size(), cudaMemcpyHostToDevice, stream));
    if (np) {
        CU(cudaMemcpyAsync(c.port_woff, woff.data(), sizeof(long long) * np, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(c.port_wlen, wlen.data(), sizeof(long long) * np, cudaMemcpyHostToDevice, stream));
    }
    if (ns) CU(cudaMemcpyAsync(c.wave, hw.data(), sizeof(R) * ns, cudaMemcpyHostToDevice, stream));
    src.n_unique = nu; src.off = c.src_off; src.comp = c.src_comp; src.r = c.src_r; src.cbeg = c.src_cbeg;
    src.con_port = c.con_port; src.con_scale = c.con_scale; src.port_woff = c.port_woff; src.port_wlen = c.port_wlen;
    src.wave = c.wave;
    n_unique = nu; n_ports = np;
    if (nu) {
        const int bs = 128, gs = (nu + bs - 1) / bs;
        if (loss == EM_LOSS_CD) EM_LAUNCH((em::k_source_coef<R, 0>), gs, bs, 0, stream)(p, src, c.src_flags);
        else                    EM_LAUNCH((em::k_source_coef<R, 1>), gs, bs, 0, stream)(p, src, c.src_flags);
        CU(cudaGetLastError());
        std::vector<int> flags(nu);
        CU(cudaMemcpyAsync(flags.data(), c.src_flags, sizeof(int) * nu, cudaMemcpyDeviceToHost, stream));
        CU(cudaStreamSynchronize(stream));
        for (int u = 0; u < nu; ++u)
            if (flags[u]) {
                src.n_unique = 0; n_unique = 0;
                cudaMemsetAsync(c.tile_sbeg, 0, sizeof(int) * (n_items + 1), stream);
                return fail(EM_ERR_INVALID_ARG, "a source edge is PEC-fixed");
            }
    }
    CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

// ---- dense <-> padded copies ----------------------------------------------------------------------
template <typename R>
int32_t Ctx<R>::set_field(int32_t comp, const void *srcp, int32_t is_dev) {
    if (!comp_ok(comp) || !srcp) return fail(EM_ERR_INVALID_ARG, "set_field arguments");
    int sx, sy, sz; comp_dims(comp, &sx, &sy, &sz);
    cudaMemcpy3DParms m = {};
    m.srcPtr = make_cudaPitchedPtr(const_cast<void *>(srcp), sizeof(R) * sx, sx, sy);
    m.dstPtr = make_cudaPitchedPtr(comp_ptr(comp), sizeof(R) * g.PX, g.PX, g.PY);
    m.extent = make_cudaExtent(sizeof(R) * sx, sy, sz);
    m.kind = is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpy3DAsync(&m, stream));
    if (comp < 3 || comp >= 6) {
        dim3 b(32, 8);
        EM_LAUNCH(em::k_mask_fixed<R>, node_grid(b, 1), b, 0, stream)(p, comp_ptr(comp), comp % 3, 0);
        CU(cudaGetLastError());
    }
    if (!is_dev) CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

// One z plane of a component out (dst) or in (src): the halo exchange of a z-slab decomposition.
template <typename R>
int32_t Ctx<R>::plane(int32_t comp, int32_t k, void *dst, const void *srcp, int32_t is_dev) {
    if (!comp_ok(comp)) return fail(EM_ERR_INVALID_ARG, "plane: bad component");
    int sx, sy, sz; comp_dims(comp, &sx, &sy, &sz);
    if (k < 0 || k >= sz) return fail(EM_ERR_INVALID_ARG, "plane: k out of range");
    R *base = comp_ptr(comp) + (long long)k * g.PXY;
    const size_t wbytes = sizeof(R) * sx;
    if (dst) {
        CU(cudaMemcpy2DAsync(dst, wbytes, base, sizeof(R) * g.PX, wbytes, sy,
                             is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, stream));
    } else {
        CU(cudaMemcpy2DAsync(base, sizeof(R) * g.PX, srcp, wbytes, wbytes, sy,
                             is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, stream));
        if (comp < 3 || comp >= 6) {                      // PEC-fixed edges of this plane stay 0
            dim3 b(32, 8);
            dim3 gr((g.nx + 1 + b.x - 1) / b.x, (g.ny + 1 + b.y - 1) / b.y, 1);
            EM_LAUNCH(em::k_mask_fixed<R>, gr, b, 0, stream)(p, comp_ptr(comp), comp % 3, k);
            CU(cudaGetLastError());
        }
    }
    if (!is_dev) CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::get_field(int32_t comp, void *dst, int32_t is_dev) {
    if (!comp_ok(comp) || !dst) return fail(EM_ERR_INVALID_ARG, "get_field arguments");
    int sx, sy, sz; comp_dims(comp, &sx, &sy, &sz);
    cudaMemcpy3DParms m = {};
    m.srcPtr = make_cudaPitchedPtr(comp_ptr(comp), sizeof(R) * g.PX, g.PX, g.PY);
    m.dstPtr = make_cudaPitchedPtr(dst, sizeof(R) * sx, sx, sy);
    m.extent = make_cudaExtent(sizeof(R) * sx, sy, sz);
    m.kind = is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    CU(cudaMemcpy3DAsync(&m, stream));
    if (!is_dev) CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

// ---- z-slab halo -------------------------------------------------------------------------
// dst: pack [Ex | Ey] of node plane kp (+ theta of cell layer kl in a coupled context); src: the reverse, PEC-fixed
// edges kept at 0 and sigma(T) of the layer refreshed.  One kernel, on `st` (null: the context's stream).
template <typename R>
int32_t Ctx<R>::halo(int32_t kp, int32_t kl, void *dst, const void *srcp, void *st) {
    if (eonly) return fail(EM_ERR_UNSUPPORTED, "the halo calls cover the leapfrog formulation");
    if (kp < 0 || kp > g.nz) return fail(EM_ERR_INVALID_ARG, "halo: node plane out of range");
    if (thermal_on && (kl < 0 || kl >= g.nz)) return fail(EM_ERR_INVALID_ARG, "halo: cell layer out of range");
    cudaStream_t s = st ? static_cast<cudaStream_t>(st) : stream;
    if (nodal && thermal_on) {
        // theta lives on the nodes: the message is [Ex | Ey | theta] of node plane kp; on the way in, sigma(T) of cell
        // layer kl (the ghost layer behind the wall plane, eq. (6) from its 8 node temperatures) is refreshed
        const long long n_e = (long long)(g.ny + 1) * g.nx + (long long)g.ny * (g.nx + 1), n_t = (long long)(g.ny + 1) * (g.nx + 1);
        const unsigned be = (unsigned)((n_e + 255) / 256), bt = (unsigned)((n_t + 255) / 256);
        R *th = c.theta[th_cur] + g.origin;
        if (dst) {
            EM_LAUNCH(em::k_pack_halo<R>, be, 256, 0, s)(p, p.E[0], p.E[1], nullptr, kp, kl, static_cast<R *>(dst));
            EM_LAUNCH(em::k_node_plane<R>, bt, 256, 0, s)(p, th, kp, static_cast<R *>(dst) + n_e, 0);
            launches += 2;
        } else {
            R *src = const_cast<R *>(static_cast<const R *>(srcp));
            EM_LAUNCH(em::k_unpack_halo<R>, be, 256, 0, s)(p, p.E[0], p.E[1], nullptr, nullptr, nullptr, c.ttable, kp, kl, src);
            EM_LAUNCH(em::k_node_plane<R>, bt, 256, 0, s)(p, th, kp, src + n_e, 1);
            dim3 b(32, 8), gr((g.nx + b.x - 1) / b.x, (g.ny + b.y - 1) / b.y, 1);
            em::ThermalParams<R> t = tp();
            EM_LAUNCH(em::k_sigma_nodal<R>, gr, b, 0, s)(p, t, kl);
            t.sig = sig_buf(1 - sg_cur);
            EM_LAUNCH(em::k_sigma_nodal<R>, gr, b, 0, s)(p, t, kl);
            launches += 4;
        }
        CU(cudaGetLastError());
        return EM_OK;
    }
    int64_t n = 0; halo_elems(&n);
    const unsigned blocks = (unsigned)((n + 255) / 256);
    R *th = thermal_on ? c.theta[th_cur] + g.origin : nullptr;
    if (dst) EM_LAUNCH(em::k_pack_halo<R>, blocks, 256, 0, s)(p, p.E[0], p.E[1], th, kp, kl, static_cast<R *>(dst));
    else     EM_LAUNCH(em::k_unpack_halo<R>, blocks, 256, 0, s)(p, p.E[0], p.E[1], th, thermal_on ? sig_buf(0) : nullptr,
                                                          thermal_on ? sig_buf(1) : nullptr, c.ttable, kp, kl, static_cast<const R *>(srcp));
    CU(cudaGetLastError());
    launches += 1;
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::joule_layers(int32_t k0, int32_t k1, double *total) {
    if (k0 < 0 || k1 < k0 || k1 > g.nz || !total) return fail(EM_ERR_INVALID_ARG, "joule_layers: need 0 <= k0 <= k1 <= nz");
    EM_LAUNCH(em::k_energy_partial<R>, kReduceBlocks, 256, 0, stream)(p, c.vx, c.vy, c.vz, k0, k1, c.partial);
    EM_LAUNCH(em::k_energy_final, 1, 256, 0, stream)(c.partial, kReduceBlocks, c.scalar);
    CU(cudaGetLastError()); launches += 2;
    CU(cudaMemcpyAsync(total, c.scalar, sizeof(double), cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

// Byte offset, from the workspace base, of element (0, 0) of the wall plane (side 0: plane 0, side 1: plane nz) of the E
// array with ping-pong parity `parity`, comp 0 = Ex, 1 = Ey: what a neighbouring slab adds to ITS mapping of this
// workspace to store into that plane (em_set_peer_halo).
template <typename R>
int32_t Ctx<R>::wall_offset(int32_t side, int32_t parity, int32_t comp, size_t *off) {
    if (side < 0 || side > 1 || parity < 0 || parity > 1 || comp < 0 || comp > 1 || !off) return fail(EM_ERR_INVALID_ARG, "wall_offset arguments");
    if (eonly) return fail(EM_ERR_UNSUPPORTED, "the halo calls cover the leapfrog formulation");
    const R *ptr = org(parity * 3 + comp) + (long long)(side ? g.nz : 0) * g.PXY;
    *off = (size_t)(reinterpret_cast<const char *>(ptr) - static_cast<const char *>(ws_base));
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::set_peer_halo(int32_t side, int32_t k_send, void *const dst[4]) {
    if (side < 0 || side > 1) return fail(EM_ERR_INVALID_ARG, "side must be 0 (-z) or 1 (+z)");
    if (eonly || kernel != EM_KERNEL_TMA || grid.thermal) return fail(EM_ERR_UNSUPPORTED, "peer halo stores run in the leapfrog TMA sweep (no thermal coupling)");
    if (!dst) {
        for (int q = 0; q < 2; ++q) for (int cc = 0; cc < 2; ++cc) peer_dst[side][q][cc] = nullptr;
        p.peer_k[side] = -1000; p.peer_skip &= ~(1 << side);
        bind();
        return EM_OK;
    }
    if (grid.bc[4 + side] != EM_BC_PMC) return fail(EM_ERR_STATE, "the wall on that side is not an artificial (PMC) slab wall");
    if (k_send < 0 || k_send > g.nz) return fail(EM_ERR_INVALID_ARG, "k_send out of range");
    for (int q = 0; q < 4; ++q) if (!dst[q]) return fail(EM_ERR_INVALID_ARG, "null peer address");
    for (int q = 0; q < 4; ++q)                                  // (the sweep writes them with 16-byte vector stores)
        if (reinterpret_cast<uintptr_t>(dst[q]) % 16) return fail(EM_ERR_INVALID_ARG, "peer addresses must be 16-byte aligned");
    for (int q = 0; q < 2; ++q) for (int cc = 0; cc < 2; ++cc) peer_dst[side][q][cc] = static_cast<R *>(dst[q * 2 + cc]);
    p.peer_k[side] = k_send; p.peer_skip |= 1 << side;
    bind();
    return EM_OK;
}

// ---- time stepping ----------------------------------------------------------------------------------
template <typename R>
int32_t Ctx<R>::record_begin() {
    if (!timing.enabled) return EM_OK;
    if (timing.pending == kTimingRing) { int32_t rc = timing_flush(); if (rc) return rc; }
    CU(cudaEventRecord(timing.beg[timing.head], stream));
    return EM_OK;
}
template <typename R>
int32_t Ctx<R>::record_end() {
    if (!timing.enabled) return EM_OK;
    CU(cudaEventRecord(timing.end[timing.head], stream));
    timing.head = (timing.head + 1) % kTimingRing; timing.pending += 1;
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::step_split() {
    dim3 b(32, 8);
    EM_LAUNCH(em::k_split_h<R>, node_grid(b, 1), b, 0, stream)(p);
    int32_t rc = record_begin(); if (rc) return rc;
    if (loss == EM_LOSS_CD) EM_LAUNCH((em::k_split_e<R, 0>), node_grid(b, 1), b, 0, stream)(p);
    else                    EM_LAUNCH((em::k_split_e<R, 1>), node_grid(b, 1), b, 0, stream)(p);
    rc = record_end(); if (rc) return rc;
    launches += 2;
    if (n_unique) {
        EM_LAUNCH(em::k_apply_source<R>, (n_unique + 127) / 128, 128, 0, stream)(p.En[0], p.En[1], p.En[2], p.Hn[0], p.Hn[1], p.Hn[2], src, (long long)step_index);
        launches += 1;
    }
    EM_LAUNCH(em::k_split_joule<R>, node_grid(b, 0), b, 0, stream)(p);
    launches += 1;
    CU(cudaGetLastError());
    e_cur ^= 1; bind();
    return EM_OK;
}

// ---- thermal coupling (NEXT-1; eq. (4)-(6); em_thermal.cuh) ---------------------------------------
template <typename R>
int32_t Ctx<R>::refresh_sigma() {
    dim3 b(32, 8);
    em::ThermalParams<R> t = tp();
    if (nodal) {
        EM_LAUNCH(em::k_sigma_nodal<R>, node_grid(b, 0), b, 0, stream)(p, t, 0);
        t.sig = sig_buf(1 - sg_cur);
        EM_LAUNCH(em::k_sigma_nodal<R>, node_grid(b, 0), b, 0, stream)(p, t, 0);
        CU(cudaGetLastError());
        return EM_OK;
    }
    EM_LAUNCH(em::k_sigma_refresh<R>, node_grid(b, 0), b, 0, stream)(p, t);
    t.sig = sig_buf(1 - sg_cur);                        // both buffers: the coupled sweep rewrites only the lossy lanes
    EM_LAUNCH(em::k_sigma_refresh<R>, node_grid(b, 0), b, 0, stream)(p, t);
    CU(cudaGetLastError());
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::set_thermal(const em_thermal_material *tt, int32_t n_mat) {
    if (!grid.thermal) return fail(EM_ERR_STATE, "the context was created with em_grid.thermal = 0");
    if (!tt || n_mat != n_mat_) return fail(EM_ERR_INVALID_ARG, "thermal table must have the n_mat entries of em_create");
    for (int m = 0; m < n_mat; ++m)
        if (!(tt[m].rho_cp > 0.0) || !(tt[m].k >= 0.0) || !std::isfinite(tt[m].rho_cp + tt[m].k + tt[m].alpha))
            return fail(EM_ERR_INVALID_ARG, "need finite rho_cp > 0, k >= 0 and alpha");
    std::vector<em::ThEntry<R>> ht(p.n_table);          // the outside entries stay 0: no heat, no conduction
    for (auto &e : ht) { e.irc = R(0); e.k = R(0); e.alpha = R(0); e.sigma0 = R(0); }
    for (int m = 0; m < n_mat; ++m) {
        ht[m].irc = (R)(1.0 / tt[m].rho_cp); ht[m].k = (R)tt[m].k; ht[m].alpha = (R)tt[m].alpha; ht[m].sigma0 = (R)table[m].sigma;
    }
    CU(cudaMemcpyAsync(c.ttable, ht.data(), sizeof(em::ThEntry<R>) * ht.size(), cudaMemcpyHostToDevice, stream));
    CU(cudaMemsetAsync(c.theta[0], 0, sizeof(R) * g.alloc_elems, stream));
    CU(cudaMemsetAsync(c.theta[1], 0, sizeof(R) * g.alloc_elems, stream));
    CU(cudaMemsetAsync(c.sig, 0, sizeof(R) * g.alloc_elems, stream));
    CU(cudaMemsetAsync(c.sig2, 0, sizeof(R) * g.alloc_elems, stream));
    sg_cur = 0;
    th_cur = 0;
    thermal_on = true;
    int32_t rc = refresh_sigma(); if (rc) return rc;
    CU(cudaStreamSynchronize(stream));                   // ht is a local
    return EM_OK;
}

// dst != null: copy theta out; src != null: copy theta in and refresh sigma(T).  Dense [nz][ny][nx] maps.
template <typename R>
int32_t Ctx<R>::temperature_rise(void *dst, const void *srcp, int32_t is_dev) {
    if (!thermal_on) return fail(EM_ERR_STATE, "thermal coupling is not switched on (em_set_thermal)");
    R *th = c.theta[th_cur] + g.origin;
    cudaMemcpy3DParms m = {};
    const int ex = nodal ? 1 : 0;                         // nodal: dense [nz+1][ny+1][nx+1] maps
    const size_t tx = (size_t)g.nx + ex, ty = (size_t)g.ny + ex, tz = (size_t)g.nz + ex;
    m.extent = make_cudaExtent(sizeof(R) * tx, ty, tz);
    if (dst) {
        m.srcPtr = make_cudaPitchedPtr(th, sizeof(R) * g.PX, g.PX, g.PY);
        m.dstPtr = make_cudaPitchedPtr(dst, sizeof(R) * tx, tx, ty);
        m.kind = is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
        CU(cudaMemcpy3DAsync(&m, stream));
    } else {
        m.srcPtr = make_cudaPitchedPtr(const_cast<void *>(srcp), sizeof(R) * tx, tx, ty);
        m.dstPtr = make_cudaPitchedPtr(th, sizeof(R) * g.PX, g.PX, g.PY);
        m.kind = is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        CU(cudaMemcpy3DAsync(&m, stream));
        int32_t rc = refresh_sigma(); if (rc) return rc;
    }
    if (!is_dev) CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

// One coupled step: a1, a2 with D_sigma(T^n), a3 with r_e(sigma(T^n)), then a4 + eq. (5) + eq. (6) in one kernel.
template <typename R>
int32_t Ctx<R>::step_thermal() {
    dim3 b(32, 8);
    const R *sig = sig_buf(sg_cur);
    EM_LAUNCH(em::k_split_h<R>, node_grid(b, 1), b, 0, stream)(p);
    int32_t rc = record_begin(); if (rc) return rc;
    if (loss == EM_LOSS_CD) EM_LAUNCH((em::k_split_e_sig<R, 0>), node_grid(b, 1), b, 0, stream)(p, sig);
    else                    EM_LAUNCH((em::k_split_e_sig<R, 1>), node_grid(b, 1), b, 0, stream)(p, sig);
    rc = record_end(); if (rc) return rc;
    launches += 2;
    if (n_unique) {
        const int gs = (n_unique + 127) / 128;
        if (loss == EM_LOSS_CD) EM_LAUNCH((em::k_source_coef_sig<R, 0>), gs, 128, 0, stream)(p, src, sig);
        else                    EM_LAUNCH((em::k_source_coef_sig<R, 1>), gs, 128, 0, stream)(p, src, sig);
        EM_LAUNCH(em::k_apply_source<R>, gs, 128, 0, stream)(p.En[0], p.En[1], p.En[2], p.Hn[0], p.Hn[1], p.Hn[2], src, (long long)step_index);
        launches += 2;
    }
    EM_LAUNCH(em::k_joule_thermal<R>, node_grid(b, 0), b, 0, stream)(p, tp());
    launches += 1;
    CU(cudaGetLastError());
    e_cur ^= 1; th_cur ^= 1; bind();
    return EM_OK;
}

// One coupled step with theta on the mesh NODES (em_grid.thermal = EM_THERMAL_NODE; readings N1-N4): a1, a2 with
// D_sigma(T^n), a3, a4 into the per-cell Joule map, then eq. (5) on the nodes (edge heat split between the end nodes, edge
// conductances, nodal capacities) and eq. (6) per cell from the mean of its 8 node temperatures.
template <typename R>
int32_t Ctx<R>::step_thermal_nodal() {
    dim3 b(32, 8);
    const R *sig = sig_buf(sg_cur);
    EM_LAUNCH(em::k_split_h<R>, node_grid(b, 1), b, 0, stream)(p);
    int32_t rc = record_begin(); if (rc) return rc;
    if (loss == EM_LOSS_CD) EM_LAUNCH((em::k_split_e_sig<R, 0>), node_grid(b, 1), b, 0, stream)(p, sig);
    else                    EM_LAUNCH((em::k_split_e_sig<R, 1>), node_grid(b, 1), b, 0, stream)(p, sig);
    rc = record_end(); if (rc) return rc;
    launches += 2;
    if (n_unique) {
        const int gs = (n_unique + 127) / 128;
        if (loss == EM_LOSS_CD) EM_LAUNCH((em::k_source_coef_sig<R, 0>), gs, 128, 0, stream)(p, src, sig);
        else                    EM_LAUNCH((em::k_source_coef_sig<R, 1>), gs, 128, 0, stream)(p, src, sig);
        EM_LAUNCH(em::k_apply_source<R>, gs, 128, 0, stream)(p.En[0], p.En[1], p.En[2], p.Hn[0], p.Hn[1], p.Hn[2], src, (long long)step_index);
        launches += 2;
    }
    EM_LAUNCH(em::k_joule_sig<R>, node_grid(b, 0), b, 0, stream)(p, sig);
    EM_LAUNCH(em::k_thermal_nodal<R>, node_grid(b, 1), b, 0, stream)(p, tp(), c.vx, c.vy, c.vz);
    th_cur ^= 1;
    EM_LAUNCH(em::k_sigma_nodal<R>, node_grid(b, 0), b, 0, stream)(p, tp(), 0);       // sigma(T^{n+1}) from the new theta
    launches += 3;
    CU(cudaGetLastError());
    e_cur ^= 1; bind();
    return EM_OK;
}

// One coupled step on the TMA sweep: conduction first (theta_d = theta^n - dt/(rho c_p) M_kk theta^n into the other theta
// buffer), then the sweep with D_sigma(T^n) from the current sigma buffer; its phase C adds the Joule heat of the step to
// theta_d in place and writes sigma(T^{n+1}) of the lossy lanes to the other sigma buffer.  Buffers are swapped.
// (-DEM_SWEEP_FUSED_CONDUCTION=1, experimental: the conduction stencil runs inside the sweep and k_diffuse is not launched.)
template <typename R>
int32_t Ctx<R>::step_thermal_sweep() {
    dim3 b(32, 8);
    R *th_in = c.theta[th_cur] + g.origin, *th_out = c.theta[1 - th_cur] + g.origin;
    if (!em::kFusedConduction) {
        constexpr int V = 16 / (int)sizeof(R);
        dim3 gd(((g.nx + V - 1) / V + b.x - 1) / b.x, (g.ny + b.y - 1) / b.y, g.nz);
        EM_LAUNCH(em::k_diffuse<R>, gd, b, 0, stream)(p, c.ttable, th_in, th_out);
        launches += 1;
    }
    int32_t rc = record_begin(); if (rc) return rc;
    em::SweepSources fsrc{c.tile_sbeg, c.tile_ent, c.order};
    em::SweepMaps maps;
    for (int a = 0; a < 3; ++a) { maps.E[a] = map_field[e_cur * 3 + a]; maps.H[a] = map_field[6 + h_cur * 3 + a]; }
    maps.q = map_q; maps.mat = map_mat; maps.sig = map_sig[sg_cur];
    if (em::kFusedConduction) maps.th = map_theta[th_cur];
    em::ThermalSweep<R> tsw{th_out, sig_buf(1 - sg_cur), c.ttable};
    cudaError_t e = em::launch_sweep_tma<R>(sweep_kernel, plan, sweep_smem, maps, p, src, fsrc, (long long)step_index, stream, &tsw);
    if (e != cudaSuccess) return fail(EM_ERR_CUDA, std::string("coupled TMA sweep launch: ") + cudaGetErrorString(e));
    rc = record_end(); if (rc) return rc;
    launches += 1;
    e_cur ^= 1; h_cur ^= 1; th_cur ^= 1; sg_cur ^= 1; bind();
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::step_tma() {
    int32_t rc = record_begin(); if (rc) return rc;
    em::SweepSources fsrc{c.tile_sbeg, c.tile_ent, c.order};
    em::SweepMaps maps;
    for (int a = 0; a < 3; ++a) {
        if (eonly) { maps.E[a] = map_field[lvl * 3 + a]; maps.H[a] = map_prev[((lvl + 2) % 3) * 3 + a]; }
        else       { maps.E[a] = map_field[e_cur * 3 + a]; maps.H[a] = map_field[6 + h_cur * 3 + a]; }
    }
    maps.q = map_q; maps.mat = map_mat;
    cudaError_t e = em::launch_sweep_tma<R>(sweep_kernel, plan, sweep_smem, maps, p, src, fsrc, (long long)step_index, stream);
    if (e != cudaSuccess) return fail(EM_ERR_CUDA, std::string("TMA sweep launch: ") + cudaGetErrorString(e));
    rc = record_end(); if (rc) return rc;
    launches += 1;
    if (eonly) lvl = (lvl + 1) % 3; else { e_cur ^= 1; h_cur ^= 1; }
    bind();
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::step(int64_t n) {
    if (n < 0) return fail(EM_ERR_INVALID_ARG, "n < 0");
    for (int64_t s = 0; s < n; ++s) {
        int32_t rc = thermal_on ? (nodal ? step_thermal_nodal() : kernel == EM_KERNEL_TMA ? step_thermal_sweep() : step_thermal())
                   : grid.thermal ? step_split()            // (tile geometry of the coupled sweep: EM-only steps run split)
                   : kernel == EM_KERNEL_TMA ? step_tma() : step_split();
        if (rc) return rc;
        step_index += 1;
    }
    return EM_OK;
}

// ---- outputs ----------------------------------------------------------------------------------------
template <typename R>
int32_t Ctx<R>::joule(void *power, void *energy, double *total, int32_t do_reset) {
    dim3 b(32, 8);
    if (power) {
        if (thermal_on) EM_LAUNCH(em::k_power_sig<R>, node_grid(b, 0), b, 0, stream)(p, sig_buf(sg_cur), static_cast<R *>(power));
        else            EM_LAUNCH(em::k_power<R>, node_grid(b, 0), b, 0, stream)(p, static_cast<R *>(power));
        CU(cudaGetLastError()); launches += 1;
    }
    if (energy) {
        cudaMemcpy3DParms m = {};
        m.srcPtr = make_cudaPitchedPtr(p.q, sizeof(R) * g.PX, g.PX, g.PY);
        m.dstPtr = make_cudaPitchedPtr(energy, sizeof(R) * g.nx, g.nx, g.ny);
        m.extent = make_cudaExtent(sizeof(R) * g.nx, g.ny, g.nz);
        m.kind = cudaMemcpyDeviceToDevice;
        CU(cudaMemcpy3DAsync(&m, stream));
    }
    if (total) {
        EM_LAUNCH(em::k_energy_partial<R>, kReduceBlocks, 256, 0, stream)(p, c.vx, c.vy, c.vz, 0, g.nz, c.partial);
        EM_LAUNCH(em::k_energy_final, 1, 256, 0, stream)(c.partial, kReduceBlocks, c.scalar);
        CU(cudaGetLastError()); launches += 2;
        CU(cudaMemcpyAsync(total, c.scalar, sizeof(double), cudaMemcpyDeviceToHost, stream));
        CU(cudaStreamSynchronize(stream));
    }
    if (do_reset) CU(cudaMemsetAsync(c.q, 0, sizeof(R) * g.alloc_elems, stream));
    return EM_OK;
}

// ---- checkpoint / resume, failure detection (em.h) ------------------------------------------------------------------
template <typename R>
int32_t Ctx<R>::set_joule_energy(const void *srcp, int32_t is_dev) {
    if (!srcp) return fail(EM_ERR_INVALID_ARG, "set_joule_energy: null");
    cudaMemcpy3DParms m = {};
    m.srcPtr = make_cudaPitchedPtr(const_cast<void *>(srcp), sizeof(R) * g.nx, g.nx, g.ny);
    m.dstPtr = make_cudaPitchedPtr(p.q, sizeof(R) * g.PX, g.PX, g.PY);
    m.extent = make_cudaExtent(sizeof(R) * g.nx, g.ny, g.nz);
    m.kind = is_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpy3DAsync(&m, stream));
    if (!is_dev) CU(cudaStreamSynchronize(stream));
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::check_finite(int32_t *all_finite) {
    if (!all_finite) return fail(EM_ERR_INVALID_ARG, "check_finite: null");
    int *flag = reinterpret_cast<int *>(c.partial);                      // (scratch of the Joule reduction)
    CU(cudaMemsetAsync(flag, 0, sizeof(int), stream));
    const long long n = g.alloc_elems;                                   // whole allocations: the pads hold zeros
    const unsigned blocks = (unsigned)std::min<long long>((n + 255) / 256, 4096);
    for (int a = 0; a < n_field; ++a) { EM_LAUNCH(em::k_check_finite<R>, blocks, 256, 0, stream)(c.field[a], n, flag); launches += 1; }
    EM_LAUNCH(em::k_check_finite<R>, blocks, 256, 0, stream)(c.q, n, flag); launches += 1;
    if (thermal_on) { EM_LAUNCH(em::k_check_finite<R>, blocks, 256, 0, stream)(c.theta[th_cur], n, flag); launches += 1; }
    CU(cudaGetLastError());
    int host_flag = 0;
    CU(cudaMemcpyAsync(&host_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    *all_finite = host_flag ? 0 : 1;
    return EM_OK;
}

template <typename R>
int32_t Ctx<R>::probe(int32_t n, const em_probe_pt *pts, double *out) {
    if (n < 0 || (n && (!pts || !out))) return fail(EM_ERR_INVALID_ARG, "probe arguments");
    for (int q = 0; q < n; ++q) {
        if (!comp_ok(pts[q].comp)) return fail(EM_ERR_INVALID_ARG, "probe comp must be 0..5 (E-only contexts: 0..2, 6..8)");
        int sx, sy, sz; comp_dims(pts[q].comp, &sx, &sy, &sz);
        if (pts[q].i < 0 || pts[q].i >= sx || pts[q].j < 0 || pts[q].j >= sy || pts[q].k < 0 || pts[q].k >= sz)
            return fail(EM_ERR_INVALID_ARG, "probe point outside the grid");
    }
    em::ProbeArrays<R> pa;
    for (int a = 0; a < 3; ++a) { pa.f[a] = p.E[a]; pa.f[3 + a] = p.H[a]; pa.f[6 + a] = p.H[a]; }
    std::vector<long long> off(kProbeChunk); std::vector<int> comp(kProbeChunk);
    for (int base = 0; base < n; base += kProbeChunk) {
        const int m = std::min(kProbeChunk, n - base);
        for (int q = 0; q < m; ++q) {
            const em_probe_pt &pt = pts[base + q];
            off[q] = ((long long)pt.k * g.PY + pt.j) * g.PX + pt.i; comp[q] = pt.comp;
        }
        CU(cudaMemcpyAsync(c.probe_off, off.data(), sizeof(long long) * m, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(c.probe_comp, comp.data(), sizeof(int) * m, cudaMemcpyHostToDevice, stream));
        EM_LAUNCH(em::k_probe<R>, (m + 127) / 128, 128, 0, stream)(pa, c.probe_off, c.probe_comp, m, c.probe_out);
        CU(cudaGetLastError()); launches += 1;
        CU(cudaMemcpyAsync(out + base, c.probe_out, sizeof(double) * m, cudaMemcpyDeviceToHost, stream));
        CU(cudaStreamSynchronize(stream));
    }
    return EM_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

const char *em_last_error(void) { return g_err.c_str(); }

int32_t em_workspace_bytes(const em_grid *gr, size_t *out) {
    if (!out) return fail(EM_ERR_INVALID_ARG, "out is null");
    int32_t rc = validate_grid(gr); if (rc) return rc;
    const Geometry g = make_geometry(gr->nx, gr->ny, gr->nz);
    const em::SweepPlan plan = em::make_sweep_plan(g.nx, g.ny, g.nz, gr->precision / 8, 0, 0, gr->thermal != 0);
    const int max_items = plan.n_tiles * em::kSweepMaxZSplit;
    *out = gr->precision == 32 ? carve<float>(g, *gr, nullptr, nullptr, max_items)
                               : carve<double>(g, *gr, nullptr, nullptr, max_items);
    return EM_OK;
}

int32_t em_cfl_dt(const em_grid *gr, const uint8_t *mat_id, const em_material *tab, int32_t n_mat, double *dt_max) {
    if (!gr || !mat_id || !tab || !dt_max || !gr->dx || !gr->dy || !gr->dz) return fail(EM_ERR_INVALID_ARG, "null argument");
    if (gr->nx < 1 || gr->ny < 1 || gr->nz < 1 || n_mat < 1 || n_mat > 255) return fail(EM_ERR_INVALID_ARG, "bad sizes");
    std::vector<double> slow(n_mat);
    for (int m = 0; m < n_mat; ++m) slow[m] = std::sqrt(tab[m].eps * tab[m].mu);
    double best = INFINITY;
    for (int k = 0; k < gr->nz; ++k) {
        const double gz = 1.0 / (gr->dz[k] * gr->dz[k]);
        for (int j = 0; j < gr->ny; ++j) {
            const double gyz = gz + 1.0 / (gr->dy[j] * gr->dy[j]);
            const uint8_t *row = mat_id + ((size_t)k * gr->ny + j) * gr->nx;
            for (int i = 0; i < gr->nx; ++i) {
                if (row[i] >= n_mat) return fail(EM_ERR_INVALID_ARG, "material id >= n_mat");
                const double v = slow[row[i]] / std::sqrt(gyz + 1.0 / (gr->dx[i] * gr->dx[i]));
                if (v < best) best = v;
            }
        }
    }
    *dt_max = best;
    return EM_OK;
}

int32_t em_create(const em_grid *gr, const uint8_t *mat_id, const em_material *tab, int32_t n_mat, double dt,
                  void *workspace, size_t ws_bytes, void *stream, em_ctx **out) {
    if (!out) return fail(EM_ERR_INVALID_ARG, "out is null");
    *out = nullptr;
    int32_t rc = validate_grid(gr); if (rc) return rc;
    if (!mat_id || !tab || !gr->dx || !gr->dy || !gr->dz) return fail(EM_ERR_INVALID_ARG, "null input array");
    if (n_mat < 1 || n_mat > 255) return fail(EM_ERR_INVALID_ARG, "n_mat must be 1..255");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(EM_ERR_INVALID_ARG, "dt must be > 0");
    for (int b = 0; b < 6; ++b) {
        if (gr->bc[b] != EM_BC_PEC && gr->bc[b] != EM_BC_PMC) return fail(EM_ERR_INVALID_ARG, "unknown boundary condition");
        if (gr->bc[b] == EM_BC_PMC && n_mat > 254) return fail(EM_ERR_INVALID_ARG, "n_mat must be <= 254 with a PMC wall");
    }
    for (int m = 0; m < n_mat; ++m)
        if (!(tab[m].eps > 0.0) || !(tab[m].mu > 0.0) || !(tab[m].sigma >= 0.0) || !std::isfinite(tab[m].eps + tab[m].mu + tab[m].sigma))
            return fail(EM_ERR_INVALID_ARG, "material table: need eps > 0, mu > 0, sigma >= 0");
    const double *d[3] = {gr->dx, gr->dy, gr->dz}; const int n[3] = {gr->nx, gr->ny, gr->nz};
    for (int a = 0; a < 3; ++a) for (int i = 0; i < n[a]; ++i)
        if (!(d[a][i] > 0.0) || !std::isfinite(d[a][i])) return fail(EM_ERR_INVALID_ARG, "cell sizes must be > 0");
    const size_t ncell = (size_t)gr->nx * gr->ny * gr->nz;
    for (size_t q = 0; q < ncell; ++q) if (mat_id[q] >= n_mat) return fail(EM_ERR_INVALID_ARG, "material id >= n_mat");
    if (!workspace) return fail(EM_ERR_INVALID_ARG, "workspace is null");
    if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return fail(EM_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return fail(EM_ERR_CUDA, "no CUDA device");
    // the context lives on the device that owns the workspace, whatever the caller's current device is
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return fail(EM_ERR_INVALID_ARG, "workspace is not a device pointer");
    }
    DeviceGuard guard(attr.device);
    em_ctx *ctx = nullptr;
    if (gr->precision == 32) {
        auto *c = new Ctx<float>(); ctx = c; c->device = attr.device;
        rc = c->init(gr, mat_id, tab, n_mat, dt, workspace, ws_bytes, stream);
    } else {
        auto *c = new Ctx<double>(); ctx = c; c->device = attr.device;
        rc = c->init(gr, mat_id, tab, n_mat, dt, workspace, ws_bytes, stream);
    }
    if (rc) { delete ctx; return rc; }
    *out = ctx;
    return EM_OK;
}

int32_t em_abi_version(void) { return EM_ABI_VERSION; }

#ifdef EM_SWEEP_TRACE
int32_t em_trace_buffer(long long *dev) {
    return cudaMemcpyToSymbol(em::g_em_trace, &dev, sizeof(dev)) == cudaSuccess ? EM_OK : EM_ERR_CUDA;
}
#endif

#ifdef EM_SWEEP_FUZZ
// test builds only (libem_fuzz.so; em_sweep.cuh "schedule fuzzing"): 0 switches the random delays off
int32_t em_fuzz_seed(uint32_t seed) {
    return cudaMemcpyToSymbol(em::g_em_fuzz_seed, &seed, sizeof(seed)) == cudaSuccess ? EM_OK : EM_ERR_CUDA;
}
#endif

int32_t em_destroy(em_ctx *ctx) {
    if (!ctx) return EM_OK;
    DeviceGuard guard(ctx->device);
    for (auto e : ctx->timing.beg) cudaEventDestroy(e);
    for (auto e : ctx->timing.end) cudaEventDestroy(e);
    delete ctx;
    return EM_OK;
}

#define EM_CHECK_CTX if (!ctx) return fail(EM_ERR_INVALID_ARG, "ctx is null"); DeviceGuard guard_(ctx->device)

int32_t em_set_source(em_ctx *ctx, int32_t n_ports, const em_port *ports, const em_edge *edges, int64_t n_edges,
                      const double *wave, int64_t n_samples) {
    EM_CHECK_CTX; return ctx->set_source(n_ports, ports, edges, n_edges, wave, n_samples);
}
int32_t em_set_field(em_ctx *ctx, int32_t comp, const void *src, int32_t is_dev) { EM_CHECK_CTX; return ctx->set_field(comp, src, is_dev); }
int32_t em_get_field(em_ctx *ctx, int32_t comp, void *dst, int32_t is_dev) { EM_CHECK_CTX; return ctx->get_field(comp, dst, is_dev); }
int32_t em_get_plane(em_ctx *ctx, int32_t comp, int32_t k, void *dst, int32_t is_dev) {
    EM_CHECK_CTX; if (!dst) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->plane(comp, k, dst, nullptr, is_dev);
}
int32_t em_set_plane(em_ctx *ctx, int32_t comp, int32_t k, const void *src, int32_t is_dev) {
    EM_CHECK_CTX; if (!src) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->plane(comp, k, nullptr, src, is_dev);
}
int32_t em_step(em_ctx *ctx, int64_t n) { EM_CHECK_CTX; return ctx->step(n); }
int32_t em_joule(em_ctx *ctx, void *p, void *q, double *t, int32_t reset) { EM_CHECK_CTX; return ctx->joule(p, q, t, reset); }
int32_t em_probe(em_ctx *ctx, int32_t n, const em_probe_pt *pts, double *out) { EM_CHECK_CTX; return ctx->probe(n, pts, out); }
int32_t em_reset(em_ctx *ctx) { EM_CHECK_CTX; return ctx->reset(); }

int32_t em_set_thermal(em_ctx *ctx, const em_thermal_material *table, int32_t n_mat) { EM_CHECK_CTX; return ctx->set_thermal(table, n_mat); }
int32_t em_get_temperature_rise(em_ctx *ctx, void *dst, int32_t dst_is_device) {
    EM_CHECK_CTX; if (!dst) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->temperature_rise(dst, nullptr, dst_is_device);
}
int32_t em_set_temperature_rise(em_ctx *ctx, const void *src, int32_t src_is_device) {
    EM_CHECK_CTX; if (!src) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->temperature_rise(nullptr, src, src_is_device);
}
int32_t em_halo_elems(em_ctx *ctx, int64_t *n) { EM_CHECK_CTX; if (!n) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->halo_elems(n); }
int32_t em_get_halo(em_ctx *ctx, int32_t k_plane, int32_t k_layer, void *dst, void *stream) {
    EM_CHECK_CTX; if (!dst) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->halo(k_plane, k_layer, dst, nullptr, stream);
}
int32_t em_set_halo(em_ctx *ctx, int32_t k_plane, int32_t k_layer, const void *src, void *stream) {
    EM_CHECK_CTX; if (!src) return fail(EM_ERR_INVALID_ARG, "null"); return ctx->halo(k_plane, k_layer, nullptr, src, stream);
}
int32_t em_joule_layers(em_ctx *ctx, int32_t k0, int32_t k1, double *total) { EM_CHECK_CTX; return ctx->joule_layers(k0, k1, total); }
int32_t em_wall_offset(em_ctx *ctx, int32_t side, int32_t parity, int32_t comp, size_t *off) { EM_CHECK_CTX; return ctx->wall_offset(side, parity, comp, off); }
int32_t em_set_peer_halo(em_ctx *ctx, int32_t side, int32_t k_send, void *const dst[4]) { EM_CHECK_CTX; return ctx->set_peer_halo(side, k_send, dst); }

int32_t em_set_joule_energy(em_ctx *ctx, const void *src, int32_t is_dev) { EM_CHECK_CTX; return ctx->set_joule_energy(src, is_dev); }
int32_t em_set_step_index(em_ctx *ctx, int64_t n) {
    EM_CHECK_CTX; if (n < 0) return fail(EM_ERR_INVALID_ARG, "step index must be >= 0"); ctx->step_index = n; return EM_OK;
}
int32_t em_check_finite(em_ctx *ctx, int32_t *all_finite) { EM_CHECK_CTX; return ctx->check_finite(all_finite); }
int32_t em_step_index(em_ctx *ctx, int64_t *n) { EM_CHECK_CTX; if (!n) return fail(EM_ERR_INVALID_ARG, "null"); *n = ctx->step_index; return EM_OK; }
int32_t em_launch_count(em_ctx *ctx, int64_t *n) { EM_CHECK_CTX; if (!n) return fail(EM_ERR_INVALID_ARG, "null"); *n = ctx->launches; return EM_OK; }

int32_t em_timing_enable(em_ctx *ctx, int32_t enable) {
    EM_CHECK_CTX;
    Timing &t = ctx->timing;
    if (enable && t.beg.empty()) {
        t.beg.resize(kTimingRing); t.end.resize(kTimingRing);
        for (int i = 0; i < kTimingRing; ++i) { CU(cudaEventCreate(&t.beg[i])); CU(cudaEventCreate(&t.end[i])); }
    }
    int32_t rc = ctx->timing_flush(); if (rc) return rc;
    t.enabled = enable != 0; t.launches = 0; t.ms = 0.0;
    return EM_OK;
}

int32_t em_timing_read(em_ctx *ctx, const char **name, int64_t *launches, double *ms) {
    EM_CHECK_CTX;
    int32_t rc = ctx->timing_flush(); if (rc) return rc;
    if (name) *name = ctx->main_kernel;
    if (launches) *launches = ctx->timing.launches;
    if (ms) *ms = ctx->timing.ms;
    return EM_OK;
}

}  // extern "C"
