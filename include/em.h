/*
 * em.h -- C ABI of the B200 (sm_100a) explicit EM time-marching + Joule-heat library (libem.so).
 *
 * The operation is the paper's explicit central-difference update of the edge-based vector wave
 * equation on a structured non-uniform grid,
 *     D_eps e'' + (D_sigma e)' + S e = -J'                       (eq. 1)
 *     M e^{n+1} = N e^n - K e^{n-1} - dt^2 (dJ/dt)^n             (eq. 2)
 *     M,K = D_eps +- dt/2 D_sigma,  N = 2 D_eps - dt^2 S,  S = curl mu^-1 curl   (L65, L73-L76, eq. 3)
 * marched as the algebraically identical material-weighted E/H leapfrog,
 * with external current-source injection (L63-L69, L144) and the per-cell Joule heat
 * P = D_sigma e^2 (L86) that drives the paper's thermal stage (L90).
 *
 * Conventions
 *  - Every call returns an int32 status (EM_OK = 0); it never throws, aborts or prints.
 *    em_last_error() returns a human-readable string for the last failure on this thread.
 *  - The library NEVER allocates device memory: the caller passes one device workspace
 *    (em_workspace_bytes) and every output buffer.  The context borrows the workspace and the
 *    CUDA stream until em_destroy.  All device work is enqueued on that stream; calls are
 *    asynchronous unless a host scalar / host array is returned (documented per call).
 *  - "host" / "device" is stated for every pointer.  Setup inputs are host pointers and are copied
 *    during the call.  SI units; material table entries are absolute eps [F/m], mu [H/m],
 *    sigma [S/m] as double whatever the working precision.
 *  - User-visible field arrays are dense, C order [k][j][i] (x fastest), in the WORKING precision
 *    (float for precision 32, double for 64):
 *        Ex (nz+1, ny+1, nx)   Ey (nz+1, ny, nx+1)   Ez (nz, ny+1, nx+1)     edge tangentials
 *        Hx (nz, ny, nx+1)     Hy (nz, ny+1, nx)     Hz (nz+1, ny, nx)       face normals
 *        mat_id, Joule maps (nz, ny, nx)
 *    Ex(i,j,k) is the edge from node (i,j,k) to (i+1,j,k); Hx(i,j,k) the x-normal face at node
 *    plane i over cell (j,k); cyclic for y, z.  (Placement pinned by the DOF count of PAPER.md L160.)
 *  - State after n steps: E at t = n dt, H at t = (n - 1/2) dt, Joule energy over [0, n dt].
 *  - One context = one host thread at a time.  Several contexts may coexist.
 */
#ifndef EM_H_
#define EM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EM_OK 0
#define EM_ERR_INVALID_ARG 1
#define EM_ERR_WORKSPACE_TOO_SMALL 2
#define EM_ERR_CUDA 3
#define EM_ERR_STATE 4
#define EM_ERR_UNSUPPORTED 5

#define EM_LOSS_CD 0  /* paper eq. (3): trapezoidal conduction term, M,K = D_eps +- dt/2 D_sigma */
#define EM_LOSS_EXP 1 /* exponential-loss update: ca = exp(-s dt/eps), cb = -expm1(-s dt/eps)/s  */

#define EM_BC_PEC 0 /* tangential E = 0 on the wall (north_star; ground plane PAPER.md L134)          */
#define EM_BC_PMC 1 /* the paper's EM truncation: tangential H = 0 on the wall.  The   */
                    /* wall's tangential E edges stay unknowns, updated with the half dual face inside */
                    /* the domain and H = 0 outside -- the symmetry plane of the   */
                    /* mirrored domain.  An edge shared with a PEC wall stays fixed.  Needs n_mat<=254. */

#define EM_MAT_PEC 1 /* em_material.flags bit0: every edge touching such a cell is held at 0      */

/* em_grid.kernel: kernel strategy.  AUTO = TMA: the sweep (one launch per step; E, H and id planes staged
 * by cp.async.bulk.tensor boxes counted on mbarriers; its shared-memory layout holds the largest material
 * table).  SPLIT runs the separate H / E / source / Joule kernels.  Both are CUDA paths of this library and
 * are cross-checked against each other and the oracle in the tests. */
#define EM_KERNEL_AUTO 0
#define EM_KERNEL_SPLIT 1
#define EM_KERNEL_TMA 2

/* em_grid.formulation.  LEAPFROG: the E/H leapfrog (state E^n, H^{n-1/2}).  EONLY: the paper's literal
 * three-level recurrence M e^{n+1} = N e^n - K e^{n-1} - dt^2 (dJ/dt)^n (eq. (2), L73-L76 eq. (3)):
 * state e^n and e^{n-1}, no H array; field components 0-2 are e^n and 6-8 are e^{n-1} (3-5 do not exist:
 * INVALID_ARG), (dJ/dt)^n dt = wave[n] - wave[n-1].  Algebraically identical to LEAPFROG from consistent
 * states; moves 9 instead of 12 field words per cell-update, but every rounding error of e enters the
 * difference e^n - e^{n-1} and is amplified by ~1/(omega dt): in fp32 it leaves the 2e-5 parity bound after a
 * few hundred steps, so LEAPFROG is the default.  TMA sweep only, no thermal coupling. */
#define EM_FORM_LEAPFROG 0
#define EM_FORM_EONLY 1

#define EM_ABI_VERSION 4 /* bumped whenever em_grid or a signature changes; em_abi_version() returns it */

typedef struct em_ctx em_ctx; /* opaque, host-side */

typedef struct em_grid {
    int32_t nx, ny, nz;          /* cells per axis, each >= 1; ny <= 524272, nz <= 65534 (launch grid) */
    const double *dx, *dy, *dz;  /* HOST: cell sizes [m], lengths nx, ny, nz, all > 0                */
    int32_t precision;           /* 32 or 64: working precision of fields, maps and arithmetic      */
    int32_t loss_mode;           /* EM_LOSS_CD or EM_LOSS_EXP                                        */
    int32_t bc[6];               /* -x,+x,-y,+y,-z,+z: EM_BC_PEC or EM_BC_PMC                          */
    int32_t kernel;              /* EM_KERNEL_*                                                      */
    int32_t max_ports;           /* capacity reserved in the workspace for em_set_source            */
    int64_t max_source_edges;
    int64_t max_wave_samples;
    int32_t thermal;             /* EM_THERMAL_CELL (1): reserve workspace for the thermal stage (em_set_thermal),  */
                                 /*    theta per cell: AUTO / TMA run the coupled TMA sweep, SPLIT the split kernels; */
                                 /* EM_THERMAL_NODE (2): theta on the mesh nodes, the paper's placement (split kernels) */
    int32_t formulation;         /* EM_FORM_LEAPFROG or EM_FORM_EONLY                                            */
    int32_t z_chunks;            /* 0: the library chooses how many z chunks a tile column is cut into (work     */
                                 /* items = tiles x chunks, from the SM count); 1..8 forces it (tests, tuning)   */
    int32_t pad_;
} em_grid;

typedef struct em_material { double eps, mu, sigma; int32_t flags; int32_t pad_; } em_material;

/* Port p drives edges[edge_begin .. edge_end) with
 *   J_e(t_{n+1/2}) = amplitude * edges[e].weight * wave[wave_offset + n]   for n < wave_len, else 0,
 * n = absolute step index since em_create / em_reset; wave[n] samples J [A/m^2] at t = (n+1/2) dt
 * so that (dJ/dt)^n of eq. (2) is the centred difference of two consecutive samples. */
typedef struct em_port { int64_t edge_begin, edge_end; double amplitude; int64_t wave_offset, wave_len; } em_port;
typedef struct em_edge { int32_t comp /*0=x,1=y,2=z*/, i, j, k; double weight; } em_edge;
typedef struct em_probe_pt { int32_t comp /*0..5 = Ex,Ey,Ez,Hx,Hy,Hz*/, i, j, k; } em_probe_pt;

/* Thread-local description of the last error returned by any call on this thread (thread-local rather than
 * per-context so that a failed em_create, which has no context, can be described too). */
const char *em_last_error(void);

/* EM_ABI_VERSION of the built library: a binding compares it with the header it was written against. */
int32_t em_abi_version(void);

/* Bytes of device workspace needed for this grid (fields with padding and their ping-pong copies,
 * material ids, Joule accumulator, coefficient tables, source lists up to the max_* capacities).
 * Host-only.  Errors: EM_ERR_INVALID_ARG (null, dims < 1, precision not 32/64). */
int32_t em_workspace_bytes(const em_grid *g, size_t *out_bytes);

/* Build a context.  mat_id: HOST uint8 [nz][ny][nx], every id < n_mat <= 255.  table: HOST,
 * n_mat entries, eps > 0, mu > 0, sigma >= 0.  dt > 0 (CFL is the caller's business: em_cfl_dt).
 * workspace: DEVICE, 256-byte aligned, >= em_workspace_bytes.  stream: cudaStream_t (may be 0).
 * Zeroes fields, Joule accumulator and the step counter.  Synchronises the stream before returning
 * (the host inputs may be freed on return).  The context belongs to the device that owns `workspace`: every
 * call switches to it and restores the caller's current device.
 * Errors: INVALID_ARG, WORKSPACE_TOO_SMALL, CUDA, UNSUPPORTED (INVALID_ARG also for an unknown bc, or a PMC wall
 * with n_mat > 254; UNSUPPORTED for EONLY with SPLIT or thermal). */
int32_t em_create(const em_grid *g, const uint8_t *mat_id, const em_material *table, int32_t n_mat,
                  double dt, void *workspace, size_t workspace_bytes, void *stream, em_ctx **out);

/* Frees the host-side context only; the workspace stays with the caller. */
int32_t em_destroy(em_ctx *ctx);

/* Host-only helper ("constrained by the CFL condition"):
 * *dt_max = min over cells of sqrt(eps mu) / sqrt(dx_i^-2 + dy_j^-2 + dz_k^-2).  The caller applies
 * its own safety factor (0.9 in the five configurations). */
int32_t em_cfl_dt(const em_grid *g, const uint8_t *mat_id, const em_material *table, int32_t n_mat,
                  double *dt_max);

/* Replace the source set.  All pointers HOST; copied.  Edges must be inside the grid and must not be
 * PEC-fixed (INVALID_ARG).  Ports that share an edge add.  n_ports = 0 removes all sources.
 * Errors: INVALID_ARG, WORKSPACE_TOO_SMALL (capacities of em_grid exceeded), CUDA. */
int32_t em_set_source(em_ctx *ctx, int32_t n_ports, const em_port *ports, const em_edge *edges,
                      int64_t n_edges, const double *wave, int64_t n_samples);

/* Copy one field component (0..5 = Ex,Ey,Ez,Hx,Hy,Hz; EONLY contexts: 0..2 = e^n, 6..8 = e^{n-1} with the
 * shapes of Ex,Ey,Ez) from/to a dense array in the working
 * precision.  src/dst may be a HOST (is_device = 0) or DEVICE (is_device != 0) pointer.  Tangential E
 * on PEC-fixed edges is forced to 0 on set.  Host transfers synchronise the stream. */
int32_t em_set_field(em_ctx *ctx, int32_t comp, const void *src, int32_t src_is_device);
int32_t em_get_field(em_ctx *ctx, int32_t comp, void *dst, int32_t dst_is_device);

/* One z plane k of a component (dense [sy][sx] of that component's logical shape, working precision) out of / into
 * the context: the halo exchange of a z-slab decomposition (paper_2603_07038_b200/slabs.py), where the
 * artificial slab walls are PMC walls whose tangential E is refreshed from the neighbouring slab after every step.
 * Errors: INVALID_ARG (component, k out of range, null), CUDA.  Host transfers synchronise the stream. */
int32_t em_get_plane(em_ctx *ctx, int32_t comp, int32_t k, void *dst, int32_t dst_is_device);
int32_t em_set_plane(em_ctx *ctx, int32_t comp, int32_t k, const void *src, int32_t src_is_device);

/* ---- z-slab halo in two calls (paper_2603_07038_b200/slabs.py) -------------------------------------
 * The halo of a slab after a step is the tangential E of ONE node plane per neighbour -- and, in a thermally coupled
 * context, the temperature rise of the cell layer behind it (the ghost layer's theta and sigma(T) feed the owned layer's
 * conduction and edge conductivities).  Packed DEVICE buffer of em_halo_elems values in the working precision:
 * [Ex plane (ny+1) x nx | Ey plane ny x (nx+1) | theta layer ny x nx (coupled contexts only)].
 * em_get_halo packs node plane k_plane (and cell layer k_layer) with one kernel; em_set_halo unpacks with one kernel,
 * keeping PEC-fixed edges at 0 and refreshing sigma(T) of the layer.  With theta on the NODES (EM_THERMAL_NODE) the
 * third part is instead the temperature rise of node plane k_plane itself, (ny+1) x (nx+1): the wall plane's nodes are
 * the only ones a slab cannot update itself; em_set_halo then refreshes sigma(T) of cell layer k_layer (the ghost layer
 * behind the wall plane) from its 8 node temperatures (two light kernels out, four in).  stream: cudaStream_t to
 * enqueue on (NULL: the context's stream); ordering between streams is the caller's.  Leapfrog contexts only
 * (UNSUPPORTED otherwise). */
int32_t em_halo_elems(em_ctx *ctx, int64_t *n);
int32_t em_get_halo(em_ctx *ctx, int32_t k_plane, int32_t k_layer, void *dst_device, void *stream);
int32_t em_set_halo(em_ctx *ctx, int32_t k_plane, int32_t k_layer, const void *src_device, void *stream);

/* The same halo FUSED into the sweep: direct stores into the neighbouring slab's memory (NVLink peer mapping, CUDA IPC
 * or the same device).  em_wall_offset: byte offset, from this context's workspace base, of element (0, 0) of its wall
 * plane (side 0: the -z wall, plane 0; side 1: the +z wall, plane nz) in the E array of ping-pong parity 0/1, comp
 * 0 = Ex, 1 = Ey.  The NEIGHBOUR adds that offset to its mapping of this workspace and passes the four addresses
 * (dst[parity * 2 + comp]) to em_set_peer_halo(side, k_send, dst) on ITS context: from then on its sweep also stores
 * E'x, E'y of its node plane k_send there, and no longer stores its own wall plane on that side (the neighbour feeds it).
 * Both contexts must step in lockstep (same number of steps since em_create / em_reset) with one cross-rank barrier
 * between steps; dst = NULL switches the side off.  Leapfrog TMA sweep only, no thermal coupling (UNSUPPORTED).
 * The four addresses must be 16-byte aligned (the sweep writes them with 16-byte vector stores; a workspace base from
 * cudaMalloc / cudaIpcOpenMemHandle plus em_wall_offset always is).
 * Errors: INVALID_ARG (side, k_send, a null or misaligned address), STATE (the wall on that side is not an artificial
 * PMC wall), UNSUPPORTED. */
int32_t em_wall_offset(em_ctx *ctx, int32_t side, int32_t parity, int32_t comp, size_t *byte_offset);
int32_t em_set_peer_halo(em_ctx *ctx, int32_t side, int32_t k_send, void *const dst[4]);

/* Joule energy of the cell layers k0 <= k < k1 only: sum q_c V_c [J] (HOST scalar; synchronises).  A slab reports its
 * OWNED layers with this and the ranks all-reduce the sum. */
int32_t em_joule_layers(em_ctx *ctx, int32_t k0, int32_t k1, double *total_energy);

/* Advance n >= 0 steps (n = 0 is a no-op).  Per step: H^{n+1/2} = H^{n-1/2} - dt nu (C_e E^n);
 * E^{n+1} = ca E^n + cb (C_h H^{n+1/2} - J^{n+1/2}) on non-fixed edges; Joule energy density
 * q_c += dt sigma_c 1/4 sum over the 12 edges of c of ((E^{n+1} + E^n)/2)^2.  Asynchronous. */
int32_t em_step(em_ctx *ctx, int64_t n);

/* Joule outputs.  power_density (DEVICE, nullable): p_c = sigma_c 1/4 sum_12 (E_e^n)^2 [W/m^3] from
 * the current field (literal).  energy_density (DEVICE, nullable): q_c [J/m^3].  Both
 * dense [nz][ny][nx] in the working precision.  total_energy (HOST, nullable): sum_c q_c V_c [J],
 * reduced in fp64 in a fixed order; requesting it synchronises the stream.  reset != 0 zeroes q
 * after the outputs are produced. */
int32_t em_joule(em_ctx *ctx, void *power_density, void *energy_density, double *total_energy,
                 int32_t reset);

/* Raw staggered samples (E at t_n, H at t_{n-1/2}) as double.  pts, out: HOST.  Synchronises. */
int32_t em_probe(em_ctx *ctx, int32_t n_pts, const em_probe_pt *pts, double *out);

/* Zero the six fields, q and the step counter; keep grid, materials and sources. */
int32_t em_reset(em_ctx *ctx);

/* ---- two-way thermal coupling (eq. (4)-(6), L84-L96; NEXT-1 of SURVEY.md 8(f)) ------------------------
 * State: the temperature RISE theta = T - T0 per cell [K] (eq. (4) and (6) see only T - T0), dense [nz][ny][nx] maps
 * in the working precision.  Per step, after a1-a4:
 *   eq. (5)  theta' = theta - dt/(rho c_p) (M_kk theta) + dq/(rho c_p),  dq = the Joule energy density of the step (a4)
 *   eq. (6)  sigma' = sigma_0 / (1 + alpha theta'), used by the next step's E update ("D_sigma(T^n)", L78)
 * M_kk = V0a^T D_k V0: cell-centred -div k grad with the series conductivity of the two half cells on each face,
 * adiabatic walls (L142).  NOTE -- a deviation from the paper's placement: the paper solves T on the mesh NODES
 * (7 092 878 unknowns on its 376x408x45 mesh) and does not print its edge-to-node map of D_sigma e^2;
 * here theta lives per CELL (6 903 360 unknowns on that mesh), where the Joule heat is defined (T1, T3), so
 * the coupled numbers quoted for this library are for that cell-centred variant of eq. (4)-(5); em_grid.thermal =
 * EM_THERMAL_NODE (below) selects the paper's nodal placement instead.
 * Valid range: 1 + alpha theta > 0 (copper: theta > -256 K); below it sigma(T) is clamped at sigma_0 / 1e-6.  sigma_0 = the em_material.sigma given to em_create.  em_joule's power density then uses
 * the current sigma(T).  em_reset also zeroes theta.  Per step: one conduction kernel (theta^n -> theta - dt/(rho c_p)
 * M_kk theta) and the coupled TMA sweep (sigma(T^n) staged as one more plane per step plane, Joule heat added to theta
 * and sigma(T^{n+1}) written in its Joule phase); kernel = SPLIT runs the same step on the split kernels.  Until
 * em_set_thermal is called such a context steps EM-only on the split kernels. */
/* em_grid.thermal = EM_THERMAL_NODE -- the paper's OWN placement: theta on the (nx+1)(ny+1)(nz+1) mesh nodes (7 092 878
 * on its mesh), dense [nz+1][ny+1][nx+1] maps in em_get / em_set_temperature_rise.  Readings N1-N4
 * (DESIGN.md section 9): M_kk = V0a^T D_k V0 literally -- per edge the conductance k_e A~_e / l_e with k_e A~_e = the sum over the
 * <= 4 cells round the edge of k_c A_{c,e} / 4 (the area-weighted mean of C5 times the dual face), nodal heat capacities C_n =
 * sum over the <= 8 cells of rho c_p V_c / 8, adiabatic walls; the EDGE vector P = D_sigma e^2 (L86), as energy of the step
 * dQ_e = dt Ebar_e^2 l_e sum_c sigma_c(T^n) A_{c,e} / 4, goes half to each end node (its total is the Joule map's, so EM
 * loss == heat gained exactly); eq. (6) per cell with the mean of its 8 node temperatures.  Runs on the split kernels
 * (kernel = AUTO or SPLIT; TMA: UNSUPPORTED); the z-slab halo calls cover the per-cell stage only. */
#define EM_THERMAL_CELL 1
#define EM_THERMAL_NODE 2
typedef struct em_thermal_material { double rho_cp /* J/(m^3 K) > 0 */, k /* W/(m K) >= 0 */, alpha /* 1/K */; } em_thermal_material;

/* Switches the coupling on (theta = 0).  table: HOST, n_mat entries (the n_mat of em_create).
 * Errors: STATE (ctx created with em_grid.thermal = 0), INVALID_ARG, CUDA. */
int32_t em_set_thermal(em_ctx *ctx, const em_thermal_material *table, int32_t n_mat);
/* theta out / in (in: also refreshes sigma(T)); device or host pointer; host copies synchronise.  Dense [nz][ny][nx]
 * (EM_THERMAL_CELL) or [nz+1][ny+1][nx+1] (EM_THERMAL_NODE) in the working precision.
 * Errors: STATE (coupling not switched on), INVALID_ARG, CUDA. */
int32_t em_get_temperature_rise(em_ctx *ctx, void *dst, int32_t dst_is_device);
int32_t em_set_temperature_rise(em_ctx *ctx, const void *src, int32_t src_is_device);

/* Absolute step index n (host bookkeeping). */
int32_t em_step_index(em_ctx *ctx, int64_t *n);

/* ---- checkpoint / resume and failure detection -----------------------------------------------
 * The state of a run is: the six field arrays (E-only contexts: e^n and e^{n-1}), the Joule accumulator q, the step
 * index n (it selects the waveform samples J((n + 1/2) dt), C3) and, in a coupled context, theta.  A checkpoint is
 * em_get_field x 6, em_joule(energy_density), em_step_index (, em_get_temperature_rise); a resume on a context created
 * with the same grid, materials, dt and sources is em_set_field x 6, em_set_joule_energy, em_set_step_index
 * (, em_set_temperature_rise) -- after which em_step continues BIT FOR BIT as the uninterrupted run would.
 *
 * em_set_joule_energy: q [J/m^3], dense [nz][ny][nx] in the working precision, device or host pointer (host copies
 * synchronise).  em_set_step_index: n >= 0.  Errors: INVALID_ARG, CUDA. */
int32_t em_set_joule_energy(em_ctx *ctx, const void *energy_density, int32_t src_is_device);
int32_t em_set_step_index(em_ctx *ctx, int64_t n);

/* *all_finite (HOST) = 1 if every value of the field arrays, q and (coupled contexts) theta is finite, else 0: an
 * unstable dt or a corrupted input shows as Inf / NaN within a few hundred steps.  One small kernel per array;
 * synchronises the stream.  Errors: INVALID_ARG, CUDA. */
int32_t em_check_finite(em_ctx *ctx, int32_t *all_finite);

/* Number of kernel launches enqueued by this context so far (for bench accounting). */
int32_t em_launch_count(em_ctx *ctx, int64_t *n);

/* Name, launch count and accumulated device time of the dominant kernel of em_step since the last
 * em_timing_reset, measured with CUDA events on the context's stream when timing is enabled
 * (enable != 0 adds one event pair per launch of that kernel).  ms may be read after a sync. */
int32_t em_timing_enable(em_ctx *ctx, int32_t enable);
int32_t em_timing_read(em_ctx *ctx, const char **kernel_name, int64_t *launches, double *ms);

#ifdef __cplusplus
}
#endif
#endif /* EM_H_ */
