/*
 * em_oracle_eonly.c -- plain, slow, obviously-correct CPU ORACLE of the paper's LITERAL E-only three-level
 * recurrence (NEXT-4 of SURVEY.md 8(f)).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may load it.  It shares no code, header, table or helper with the CUDA library
 * under paper_2603_07038_b200/csrc and include/em.h (nor with em_oracle.c: the file is self-contained so that it can
 * be read against the paper by eye).
 *
 * What it computes (fp64, dense logical arrays, triple loops), exactly as the paper writes it:
 *       M e^{n+1} = N e^n - K e^{n-1} - dt^2 (dJ/dt)^n                                   PAPER.md L69      eq. (2)
 *       M = D_eps + dt/2 D_sigma,   N = 2 D_eps - dt^2 S,   K = D_eps - dt/2 D_sigma     PAPER.md L73-L76  eq. (3)
 *       S = C_h D_nu C_e   ("curl mu^-1 curl")
 * State: e^n and e^{n-1} on all primal edges (no H array).  One step:
 *   1. g  = D_nu (C_e e^n)                     on the faces   (scratch)
 *   2. s  = C_h g                              on the edges   (= S e^n)
 *   3. e^{n+1} = ( 2 D_eps e^n - dt^2 s - K e^{n-1} - dt (J^{n+1/2} - J^{n-1/2}) ) / M     on every non-fixed edge
 *   4. Joule:  q_c += dt sigma_c 1/4 sum_{12 edges of c} ((e^{n+1} + e^n)/2)^2             (C7)
 * Readings: C1 unknown placement; C3 (dJ/dt)^n = (J^{n+1/2} - J^{n-1/2})/dt with
 * wave[n] = J((n+1/2) dt) and J^{-1/2} = 0; C4 start-up state (e^0, e^{-1}), default 0; C5 area-weighted D_eps, D_sigma,
 * length-weighted D_nu; C8 PMC walls (the wall's tangential edges stay unknowns, half dual face, no g outside);
 * C6: loss mode EXP is eq. (3) with D_eps replaced by the effective permittivity
 *       eps' = (sigma dt/2) coth(sigma dt / (2 eps))      (eps' = eps for sigma = 0)
 * for which M = sigma dt/(1 - exp(-sigma dt/eps)) and K = exp(-sigma dt/eps) M, i.e. the exponential-loss update.
 *
 * Pins (tests/test_oracle_eonly.py): the dense NumPy iteration of eq. (2)-(3) with incidence-assembled matrices
 * (tests/discrete.py) from random e^0, e^{-1}; equality with the leapfrog oracle em_oracle.c (itself pinned by P0-P10)
 * on heterogeneous non-uniform grids with sources, PMC walls, CD and EXP; the TE101 closed form (three-term ratio
 * cos(w~ dt)); r^n decay and the Joule geometric series in a uniform conductor.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define EMO_OK 0
#define EMO_ERR_INVALID_ARG 1
#define EMO_LOSS_CD 0
#define EMO_LOSS_EXP 1
#define EMO_BC_PEC 0
#define EMO_BC_PMC 1

typedef struct {
    int32_t nx, ny, nz;
    const double *dx, *dy, *dz;
    int32_t loss_mode;
    int32_t bc[6];                /* -x,+x,-y,+y,-z,+z */
} emo_grid;
typedef struct { double eps, mu, sigma; int32_t flags; } emo_material;
typedef struct { int64_t edge_begin, edge_end; double amplitude; int64_t wave_offset, wave_len; } emo_port;
typedef struct { int32_t comp, i, j, k; double weight; } emo_edge;
typedef struct { int32_t comp, i, j, k; } emo_probe_pt;

typedef struct emo2_ctx {
    int32_t nx, ny, nz, loss_mode;
    int32_t bc[6];
    double dt;
    double *dx, *dy, *dz, *tx, *ty, *tz;   /* primal and dual lengths */
    double *sigma_c;                       /* per-cell sigma (Joule heat) */
    double *Deps[3], *Dsig[3];             /* D_eps (EXP: the effective eps'), D_sigma on the edges */
    uint8_t *fixed[3];                     /* 1 = PEC-fixed edge */
    double *Dnu[3];                        /* D_nu = 1/mu on the faces */
    double *e[3], *em[3], *en[3];          /* e^n, e^{n-1}, e^{n+1} */
    double *g[3];                          /* D_nu C_e e^n (faces) */
    double *J[3], *Jm[3];                  /* J^{n+1/2}, J^{n-1/2} on the edges (scattered per step) */
    double *q;
    int64_t step;
    int32_t n_ports; emo_port *ports; int64_t n_edges; emo_edge *edges; int64_t n_wave; double *wave;
} emo2_ctx;

static void dims_of(const emo2_ctx *c, int comp, int *sx, int *sy, int *sz) {
    int nx = c->nx, ny = c->ny, nz = c->nz;
    switch (comp) {
    case 0: *sx = nx;     *sy = ny + 1; *sz = nz + 1; break;   /* Ex */
    case 1: *sx = nx + 1; *sy = ny;     *sz = nz + 1; break;   /* Ey */
    case 2: *sx = nx + 1; *sy = ny + 1; *sz = nz;     break;   /* Ez */
    case 3: *sx = nx + 1; *sy = ny;     *sz = nz;     break;   /* x-normal faces */
    case 4: *sx = nx;     *sy = ny + 1; *sz = nz;     break;   /* y-normal faces */
    default:*sx = nx;     *sy = ny;     *sz = nz + 1; break;   /* z-normal faces */
    }
}
static int64_t count_of(const emo2_ctx *c, int comp) {
    int sx, sy, sz; dims_of(c, comp, &sx, &sy, &sz); return (int64_t)sx * sy * sz;
}
#define IX(sx, sy, i, j, k) (((int64_t)(k) * (sy) + (j)) * (sx) + (i))
#define EX(i,j,k) IX(nx,     ny + 1, i, j, k)
#define EY(i,j,k) IX(nx + 1, ny,     i, j, k)
#define EZ(i,j,k) IX(nx + 1, ny + 1, i, j, k)
#define FX(i,j,k) IX(nx + 1, ny,     i, j, k)
#define FY(i,j,k) IX(nx,     ny + 1, i, j, k)
#define FZ(i,j,k) IX(nx,     ny,     i, j, k)
#define CELL(i,j,k) IX(nx, ny, i, j, k)

int32_t emo2_set_threads(int32_t n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n; return 1;
#endif
}

static void free_ctx(emo2_ctx *c) {
    if (!c) return;
    free(c->dx); free(c->dy); free(c->dz); free(c->tx); free(c->ty); free(c->tz); free(c->sigma_c); free(c->q);
    for (int a = 0; a < 3; ++a) {
        free(c->Deps[a]); free(c->Dsig[a]); free(c->fixed[a]); free(c->Dnu[a]); free(c->e[a]); free(c->em[a]);
        free(c->en[a]); free(c->g[a]); free(c->J[a]); free(c->Jm[a]);
    }
    free(c->ports); free(c->edges); free(c->wave);
    free(c);
}
int32_t emo2_destroy(emo2_ctx *c) { free_ctx(c); return EMO_OK; }

/* effective permittivity of the exponential-loss update (header, reading C6) */
static double eps_effective(int mode, double eps, double sig, double dt) {
    if (mode == EMO_LOSS_CD || !(sig > 0.0)) return eps;
    const double x = 0.5 * sig * dt / eps;
    return 0.5 * sig * dt / tanh(x);
}

int32_t emo2_create(const emo_grid *g, const uint8_t *mat_id, const emo_material *tab, int32_t n_mat, double dt,
                    emo2_ctx **out) {
    if (!g || !mat_id || !tab || !out) return EMO_ERR_INVALID_ARG;
    if (g->nx < 1 || g->ny < 1 || g->nz < 1 || n_mat < 1 || n_mat > 256 || !(dt > 0.0)) return EMO_ERR_INVALID_ARG;
    if (g->loss_mode != EMO_LOSS_CD && g->loss_mode != EMO_LOSS_EXP) return EMO_ERR_INVALID_ARG;
    for (int b = 0; b < 6; ++b) if (g->bc[b] != EMO_BC_PEC && g->bc[b] != EMO_BC_PMC) return EMO_ERR_INVALID_ARG;
    for (int m = 0; m < n_mat; ++m)
        if (!(tab[m].eps > 0.0) || !(tab[m].mu > 0.0) || !(tab[m].sigma >= 0.0)) return EMO_ERR_INVALID_ARG;
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const int64_t ncell = (int64_t)nx * ny * nz;
    for (int64_t q = 0; q < ncell; ++q) if (mat_id[q] >= n_mat) return EMO_ERR_INVALID_ARG;

    emo2_ctx *c = (emo2_ctx *)calloc(1, sizeof(emo2_ctx));
    c->nx = nx; c->ny = ny; c->nz = nz; c->loss_mode = g->loss_mode; c->dt = dt;
    for (int b = 0; b < 6; ++b) c->bc[b] = g->bc[b];
    c->dx = (double *)malloc(sizeof(double) * nx); memcpy(c->dx, g->dx, sizeof(double) * nx);
    c->dy = (double *)malloc(sizeof(double) * ny); memcpy(c->dy, g->dy, sizeof(double) * ny);
    c->dz = (double *)malloc(sizeof(double) * nz); memcpy(c->dz, g->dz, sizeof(double) * nz);
    c->tx = (double *)malloc(sizeof(double) * (nx + 1));
    c->ty = (double *)malloc(sizeof(double) * (ny + 1));
    c->tz = (double *)malloc(sizeof(double) * (nz + 1));
    for (int i = 0; i <= nx; ++i) c->tx[i] = 0.5 * ((i > 0 ? c->dx[i - 1] : 0.0) + (i < nx ? c->dx[i] : 0.0));
    for (int j = 0; j <= ny; ++j) c->ty[j] = 0.5 * ((j > 0 ? c->dy[j - 1] : 0.0) + (j < ny ? c->dy[j] : 0.0));
    for (int k = 0; k <= nz; ++k) c->tz[k] = 0.5 * ((k > 0 ? c->dz[k - 1] : 0.0) + (k < nz ? c->dz[k] : 0.0));
    c->sigma_c = (double *)malloc(sizeof(double) * ncell);
    for (int64_t q = 0; q < ncell; ++q) c->sigma_c[q] = tab[mat_id[q]].sigma;
    c->q = (double *)calloc(ncell, sizeof(double));
    for (int a = 0; a < 3; ++a) {
        const int64_t ne = count_of(c, a), nf = count_of(c, 3 + a);
        c->Deps[a] = (double *)calloc(ne, sizeof(double)); c->Dsig[a] = (double *)calloc(ne, sizeof(double));
        c->fixed[a] = (uint8_t *)calloc(ne, 1);
        c->e[a] = (double *)calloc(ne, sizeof(double)); c->em[a] = (double *)calloc(ne, sizeof(double));
        c->en[a] = (double *)calloc(ne, sizeof(double));
        c->J[a] = (double *)calloc(ne, sizeof(double)); c->Jm[a] = (double *)calloc(ne, sizeof(double));
        c->Dnu[a] = (double *)calloc(nf, sizeof(double)); c->g[a] = (double *)calloc(nf, sizeof(double));
    }
    const int wall[6] = {g->bc[0] == EMO_BC_PEC, g->bc[1] == EMO_BC_PEC, g->bc[2] == EMO_BC_PEC,
                         g->bc[3] == EMO_BC_PEC, g->bc[4] == EMO_BC_PEC, g->bc[5] == EMO_BC_PEC};
    const int n[3] = {nx, ny, nz};
    const double *d[3] = {c->dx, c->dy, c->dz};
    /* D_eps, D_sigma: area-weighted mean over the <= 4 cells round the edge (C5); an edge of direction a is round by
     * the cells that differ in the two other directions b, c2 */
    for (int a = 0; a < 3; ++a) {
        const int b = (a + 1) % 3, c2 = (a + 2) % 3;
        int sx, sy, sz; dims_of(c, a, &sx, &sy, &sz);
        for (int k = 0; k < sz; ++k) for (int j = 0; j < sy; ++j) for (int i = 0; i < sx; ++i) {
            const int p[3] = {i, j, k};
            double sw = 0, se = 0, ss = 0; int pec = 0;
            for (int ob = -1; ob <= 0; ++ob) for (int oc = -1; oc <= 0; ++oc) {
                int cc[3] = {p[0], p[1], p[2]};
                cc[b] += ob; cc[c2] += oc;
                if (cc[b] < 0 || cc[b] >= n[b] || cc[c2] < 0 || cc[c2] >= n[c2]) continue;
                const int64_t q = CELL(cc[0], cc[1], cc[2]);
                const double w = d[b][cc[b]] * d[c2][cc[c2]];
                sw += w; se += w * tab[mat_id[q]].eps; ss += w * tab[mat_id[q]].sigma; pec |= tab[mat_id[q]].flags & 1;
            }
            const int fx = (p[b] == 0 && wall[2 * b]) || (p[b] == n[b] && wall[2 * b + 1]) ||
                           (p[c2] == 0 && wall[2 * c2]) || (p[c2] == n[c2] && wall[2 * c2 + 1]) || pec;
            const int64_t e = IX(sx, sy, i, j, k);
            c->fixed[a][e] = (uint8_t)fx;
            c->Dsig[a][e] = ss / sw;
            c->Deps[a][e] = eps_effective(c->loss_mode, se / sw, ss / sw, dt);
        }
    }
    /* D_nu: length-weighted mean of 1/mu over the <= 2 cells across the face (C5) */
    for (int a = 0; a < 3; ++a) {
        int sx, sy, sz; dims_of(c, 3 + a, &sx, &sy, &sz);
        for (int k = 0; k < sz; ++k) for (int j = 0; j < sy; ++j) for (int i = 0; i < sx; ++i) {
            const int p[3] = {i, j, k};
            double sw = 0, sn = 0;
            for (int o = -1; o <= 0; ++o) {
                int cc[3] = {p[0], p[1], p[2]};
                cc[a] += o;
                if (cc[a] < 0 || cc[a] >= n[a]) continue;
                sw += d[a][cc[a]]; sn += d[a][cc[a]] / tab[mat_id[CELL(cc[0], cc[1], cc[2])]].mu;
            }
            c->Dnu[a][IX(sx, sy, i, j, k)] = sn / sw;
        }
    }
    *out = c;
    return EMO_OK;
}

int32_t emo2_set_source(emo2_ctx *c, int32_t n_ports, const emo_port *ports, const emo_edge *edges, int64_t n_edges,
                        const double *wave, int64_t n_samples) {
    if (!c || n_ports < 0 || n_edges < 0 || n_samples < 0) return EMO_ERR_INVALID_ARG;
    for (int64_t e = 0; e < n_edges; ++e) {
        if (edges[e].comp < 0 || edges[e].comp > 2) return EMO_ERR_INVALID_ARG;
        int sx, sy, sz; dims_of(c, edges[e].comp, &sx, &sy, &sz);
        if (edges[e].i < 0 || edges[e].i >= sx || edges[e].j < 0 || edges[e].j >= sy || edges[e].k < 0 || edges[e].k >= sz)
            return EMO_ERR_INVALID_ARG;
        if (c->fixed[edges[e].comp][IX(sx, sy, edges[e].i, edges[e].j, edges[e].k)]) return EMO_ERR_INVALID_ARG;
    }
    for (int p = 0; p < n_ports; ++p) {
        if (ports[p].edge_begin < 0 || ports[p].edge_end < ports[p].edge_begin || ports[p].edge_end > n_edges) return EMO_ERR_INVALID_ARG;
        if (ports[p].wave_offset < 0 || ports[p].wave_len < 0 || ports[p].wave_offset + ports[p].wave_len > n_samples) return EMO_ERR_INVALID_ARG;
    }
    free(c->ports); free(c->edges); free(c->wave);
    c->n_ports = n_ports; c->n_edges = n_edges; c->n_wave = n_samples;
    c->ports = (emo_port *)malloc(sizeof(emo_port) * (n_ports > 0 ? n_ports : 1));
    c->edges = (emo_edge *)malloc(sizeof(emo_edge) * (n_edges > 0 ? n_edges : 1));
    c->wave = (double *)malloc(sizeof(double) * (n_samples > 0 ? n_samples : 1));
    if (n_ports) memcpy(c->ports, ports, sizeof(emo_port) * n_ports);
    if (n_edges) memcpy(c->edges, edges, sizeof(emo_edge) * n_edges);
    if (n_samples) memcpy(c->wave, wave, sizeof(double) * n_samples);
    return EMO_OK;
}

/* level 0: e^n, level 1: e^{n-1}; comp 0..2.  PEC-fixed edges are forced to 0. */
int32_t emo2_set_field(emo2_ctx *c, int32_t level, int32_t comp, const double *src) {
    if (!c || comp < 0 || comp > 2 || level < 0 || level > 1 || !src) return EMO_ERR_INVALID_ARG;
    double *dst = level ? c->em[comp] : c->e[comp];
    const int64_t n = count_of(c, comp);
    for (int64_t e = 0; e < n; ++e) dst[e] = c->fixed[comp][e] ? 0.0 : src[e];
    return EMO_OK;
}
int32_t emo2_get_field(emo2_ctx *c, int32_t level, int32_t comp, double *dst) {
    if (!c || comp < 0 || comp > 2 || level < 0 || level > 1 || !dst) return EMO_ERR_INVALID_ARG;
    memcpy(dst, level ? c->em[comp] : c->e[comp], sizeof(double) * count_of(c, comp));
    return EMO_OK;
}
/* the absolute step index n of the state (e^n, e^{n-1}): selects the waveform samples of the next step */
int32_t emo2_set_step_index(emo2_ctx *c, int64_t n) { if (!c || n < 0) return EMO_ERR_INVALID_ARG; c->step = n; return EMO_OK; }
int64_t emo2_step_index(const emo2_ctx *c) { return c ? c->step : -1; }

/* J^{m+1/2} scattered on the edges (adds; pass sign = -1 with the same m to clear) */
static void scatter_J(emo2_ctx *c, double *J[3], int64_t m, double sign) {
    if (m < 0) return;                                            /* J^{-1/2} = 0 (C4) */
    for (int p = 0; p < c->n_ports; ++p) {
        const emo_port *pt = &c->ports[p];
        const double w = (m < pt->wave_len) ? c->wave[pt->wave_offset + m] : 0.0;
        for (int64_t e = pt->edge_begin; e < pt->edge_end; ++e) {
            const emo_edge *ed = &c->edges[e];
            int sx, sy, sz; dims_of(c, ed->comp, &sx, &sy, &sz);
            J[ed->comp][IX(sx, sy, ed->i, ed->j, ed->k)] += sign * pt->amplitude * ed->weight * w;
        }
    }
}
static void clear_J(emo2_ctx *c, double *J[3]) {
    for (int p = 0; p < c->n_ports; ++p) {
        const emo_port *pt = &c->ports[p];
        for (int64_t e = pt->edge_begin; e < pt->edge_end; ++e) {
            const emo_edge *ed = &c->edges[e];
            int sx, sy, sz; dims_of(c, ed->comp, &sx, &sy, &sz);
            J[ed->comp][IX(sx, sy, ed->i, ed->j, ed->k)] = 0.0;
        }
    }
}

static void one_step(emo2_ctx *c) {
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const double dt = c->dt;
    const double *dx = c->dx, *dy = c->dy, *dz = c->dz, *tx = c->tx, *ty = c->ty, *tz = c->tz;
    const double *ex = c->e[0], *ey = c->e[1], *ez = c->e[2];
    double *gx = c->g[0], *gy = c->g[1], *gz = c->g[2];
    int k;

    /* 1. g = D_nu (C_e e^n): the curl of e on every face, times 1/mu */
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i)
        gx[FX(i, j, k)] = c->Dnu[0][FX(i, j, k)] *
            ((ez[EZ(i, j + 1, k)] - ez[EZ(i, j, k)]) / dy[j] - (ey[EY(i, j, k + 1)] - ey[EY(i, j, k)]) / dz[k]);
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i)
        gy[FY(i, j, k)] = c->Dnu[1][FY(i, j, k)] *
            ((ex[EX(i, j, k + 1)] - ex[EX(i, j, k)]) / dz[k] - (ez[EZ(i + 1, j, k)] - ez[EZ(i, j, k)]) / dx[i]);
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i)
        gz[FZ(i, j, k)] = c->Dnu[2][FZ(i, j, k)] *
            ((ey[EY(i + 1, j, k)] - ey[EY(i, j, k)]) / dx[i] - (ex[EX(i, j + 1, k)] - ex[EX(i, j, k)]) / dy[j]);

    /* dt^2 (dJ/dt)^n = dt (J^{n+1/2} - J^{n-1/2})   (C3) */
    scatter_J(c, c->J, c->step, 1.0);
    scatter_J(c, c->Jm, c->step - 1, 1.0);

    /* 2.-3. s = C_h g, then eq. (2) solved for e^{n+1} (M is diagonal).  g with an out-of-range index does not exist
     * (only reachable from the non-fixed edges of a PMC wall, whose dual length is the half cell; C8). */
#define GX(i, j, k) (((j) >= 0 && (j) < ny && (k) >= 0 && (k) < nz) ? gx[FX(i, j, k)] : 0.0)
#define GY(i, j, k) (((i) >= 0 && (i) < nx && (k) >= 0 && (k) < nz) ? gy[FY(i, j, k)] : 0.0)
#define GZ(i, j, k) (((i) >= 0 && (i) < nx && (j) >= 0 && (j) < ny) ? gz[FZ(i, j, k)] : 0.0)
#define EQ2(a, idx, s) do {                                                                       \
        const double De_ = c->Deps[a][idx], Ds_ = c->Dsig[a][idx];                               \
        const double M_ = De_ + 0.5 * dt * Ds_, K_ = De_ - 0.5 * dt * Ds_;                       \
        const double Ne_ = 2.0 * De_ * c->e[a][idx] - dt * dt * (s);                             \
        c->en[a][idx] = (Ne_ - K_ * c->em[a][idx] - dt * (c->J[a][idx] - c->Jm[a][idx])) / M_;   \
    } while (0)
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) {
        const int64_t e = EX(i, j, k);
        if (c->fixed[0][e]) { c->en[0][e] = 0.0; continue; }
        const double s = (GZ(i, j, k) - GZ(i, j - 1, k)) / ty[j] - (GY(i, j, k) - GY(i, j, k - 1)) / tz[k];
        EQ2(0, e, s);
    }
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) {
        const int64_t e = EY(i, j, k);
        if (c->fixed[1][e]) { c->en[1][e] = 0.0; continue; }
        const double s = (GX(i, j, k) - GX(i, j, k - 1)) / tz[k] - (GZ(i, j, k) - GZ(i - 1, j, k)) / tx[i];
        EQ2(1, e, s);
    }
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        const int64_t e = EZ(i, j, k);
        if (c->fixed[2][e]) { c->en[2][e] = 0.0; continue; }
        const double s = (GY(i, j, k) - GY(i - 1, j, k)) / tx[i] - (GX(i, j, k) - GX(i, j - 1, k)) / ty[j];
        EQ2(2, e, s);
    }
#undef EQ2
#undef GX
#undef GY
#undef GZ

    /* 4. Joule heat of the step (C7): q_c += dt sigma_c 1/4 sum_12 ((e^{n+1} + e^n)/2)^2 */
    const double *exn = c->en[0], *eyn = c->en[1], *ezn = c->en[2];
#define B2(A, An, idx) ({ double b_ = 0.5 * ((An)[idx] + (A)[idx]); b_ * b_; })
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        const double s = 0.25 * (
            B2(ex, exn, EX(i, j, k)) + B2(ex, exn, EX(i, j + 1, k)) + B2(ex, exn, EX(i, j, k + 1)) + B2(ex, exn, EX(i, j + 1, k + 1)) +
            B2(ey, eyn, EY(i, j, k)) + B2(ey, eyn, EY(i + 1, j, k)) + B2(ey, eyn, EY(i, j, k + 1)) + B2(ey, eyn, EY(i + 1, j, k + 1)) +
            B2(ez, ezn, EZ(i, j, k)) + B2(ez, ezn, EZ(i + 1, j, k)) + B2(ez, ezn, EZ(i, j + 1, k)) + B2(ez, ezn, EZ(i + 1, j + 1, k)));
        c->q[CELL(i, j, k)] += dt * c->sigma_c[CELL(i, j, k)] * s;
    }
#undef B2

    /* (e^{n-1}, e^n, e^{n+1}) <- (e^n, e^{n+1}, scratch); clear the source scatter */
    for (int a = 0; a < 3; ++a) { double *t = c->em[a]; c->em[a] = c->e[a]; c->e[a] = c->en[a]; c->en[a] = t; }
    clear_J(c, c->J); clear_J(c, c->Jm);
    c->step += 1;
}

int32_t emo2_step(emo2_ctx *c, int64_t n) {
    if (!c || n < 0) return EMO_ERR_INVALID_ARG;
    for (int64_t s = 0; s < n; ++s) one_step(c);
    return EMO_OK;
}

/* p_c = sigma_c 1/4 sum_12 (e^n)^2, q_c, Q = sum_c q_c V_c (Kahan) */
int32_t emo2_joule(emo2_ctx *c, double *power_density, double *energy_density, double *total_energy, int32_t reset) {
    if (!c) return EMO_ERR_INVALID_ARG;
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const double *ex = c->e[0], *ey = c->e[1], *ez = c->e[2];
#define SQ(A, idx) ((A)[idx] * (A)[idx])
    if (power_density)
        for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
            const double s = 0.25 * (
                SQ(ex, EX(i, j, k)) + SQ(ex, EX(i, j + 1, k)) + SQ(ex, EX(i, j, k + 1)) + SQ(ex, EX(i, j + 1, k + 1)) +
                SQ(ey, EY(i, j, k)) + SQ(ey, EY(i + 1, j, k)) + SQ(ey, EY(i, j, k + 1)) + SQ(ey, EY(i + 1, j, k + 1)) +
                SQ(ez, EZ(i, j, k)) + SQ(ez, EZ(i + 1, j, k)) + SQ(ez, EZ(i, j + 1, k)) + SQ(ez, EZ(i + 1, j + 1, k)));
            power_density[CELL(i, j, k)] = c->sigma_c[CELL(i, j, k)] * s;
        }
#undef SQ
    const int64_t ncell = (int64_t)nx * ny * nz;
    if (energy_density) memcpy(energy_density, c->q, sizeof(double) * ncell);
    if (total_energy) {
        double sum = 0.0, comp = 0.0;
        for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
            const double v = c->q[CELL(i, j, k)] * (c->dx[i] * c->dy[j] * c->dz[k]);
            const double y = v - comp, t = sum + y;
            comp = (t - sum) - y; sum = t;
        }
        *total_energy = sum;
    }
    if (reset) memset(c->q, 0, sizeof(double) * ncell);
    return EMO_OK;
}

int32_t emo2_probe(emo2_ctx *c, int32_t n_pts, const emo_probe_pt *pts, double *out) {
    if (!c || n_pts < 0 || (n_pts && (!pts || !out))) return EMO_ERR_INVALID_ARG;
    for (int p = 0; p < n_pts; ++p) {
        const int comp = pts[p].comp;
        if (comp < 0 || comp > 2) return EMO_ERR_INVALID_ARG;
        int sx, sy, sz; dims_of(c, comp, &sx, &sy, &sz);
        if (pts[p].i < 0 || pts[p].i >= sx || pts[p].j < 0 || pts[p].j >= sy || pts[p].k < 0 || pts[p].k >= sz) return EMO_ERR_INVALID_ARG;
        out[p] = c->e[comp][IX(sx, sy, pts[p].i, pts[p].j, pts[p].k)];
    }
    return EMO_OK;
}

int32_t emo2_reset(emo2_ctx *c) {
    if (!c) return EMO_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) {
        memset(c->e[a], 0, sizeof(double) * count_of(c, a));
        memset(c->em[a], 0, sizeof(double) * count_of(c, a));
        memset(c->en[a], 0, sizeof(double) * count_of(c, a));
    }
    memset(c->q, 0, sizeof(double) * (int64_t)c->nx * c->ny * c->nz);
    c->step = 0;
    return EMO_OK;
}
