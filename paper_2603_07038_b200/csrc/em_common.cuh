// em_common.cuh -- device-side data layout and small helpers shared by every kernel of libem.so.
//
// Data layout in HBM: structure of arrays.  Every per-node/per-cell array
// (six field components and their ping-pong copies, the uint8 material ids, the Joule
// accumulator) uses ONE padded index geometry
//     off(i,j,k) = (k*PY + j)*PX + i,   i in [-1, PX-2], j in [-1, ny+1], k in [-1, nz+1]
// with PX = roundup(nx+2, 32), PY = ny+3, PZ = nz+3 and the array pointer already shifted to the
// logical origin, so that one offset serves all arrays and +-1 neighbours are +-1, +-PX, +-PX*PY.
// Entries outside a component's logical range are kept at 0 ("halo-free padded pitches": the pad
// plays the role of the halo, no special-casing at the walls); material ids outside the grid hold
// the extra table entry n_mat = "outside/PEC" whose mask is 0.
#pragma once
#include <cstdint>
#include "em_ptx.cuh"

namespace em {

constexpr int kMaxTable = 256;   // n_mat <= 255 plus the "outside" entry

template <typename R> struct Vec4;
template <> struct Vec4<float>  { using type = float4;  };
template <> struct Vec4<double> { using type = double4; };

// Per-material coefficient entry, built in fp64 on the host and rounded once:
//   a = eps/dt,  b = sigma,  m = 1 (ordinary) or 0 (PEC-flagged / outside),  n = dt/mu
template <typename R> struct alignas(4 * sizeof(R)) MatEntry { R a, b, m, n; };

template <typename R>
struct DevParams {
    int nx, ny, nz;
    int PX, PY;              // pitches (elements)
    long long PXY;           // plane stride
    R *E[3], *En[3];         // E^n and E^{n+1} (ping-pong)
    R *H[3], *Hn[3];         // H^{n-1/2} and H^{n+1/2} (ping-pong in the sweep; split: H in place, Hn carries E' + E to the Joule kernels)
    R *q;                    // Joule energy density accumulator
    const uint8_t *mat;      // material ids, same geometry
    const MatEntry<R> *table;// n_table entries in global memory
    int n_table;
    int warm_lo;             // 1: the -z wall is PMC, the sweeps also run plane k = -1 as a warm-up plane
    // per-axis arrays indexed [-1 .. n+1] (pointer shifted to index 0):
    //   rd = 1/d (0 outside), rt = 1/d~, f = d[i]/(d[i-1]+d[i]) with d[-1] = d[n] = 0
    const R *rdx, *rtx, *fx, *rdy, *rty, *fy, *rdz, *rtz, *fz;
    const R *zgeo;           // interleaved {fz, 1/dz, 1/dz~, 0} per plane (one bulk copy per plane in the sweep)
    R dt;
    // z-slab halo fused into the sweep (em_set_peer_halo; SURVEY.md 8(e) "direct peer stores over NVLink"): E'x, E'y of
    // node plane peer_k[s] are ALSO stored into the neighbouring slab's wall plane -- peer_e[s][comp] is the address of
    // element (0, 0) of that plane in the neighbour's E^{n+1} array, a peer-mapped pointer -- and the own wall planes
    // fed by a neighbour are not stored (peer_skip bit 0: plane 0, bit 1: plane nz).  peer_k = -1000: side unused.
    R *peer_e[2][2];
    int peer_k[2];
    int peer_skip;
};

// Thermal coupling (eq. (4)-(6)).  Per material: 1/(rho c_p), k, alpha, sigma_0; the "outside" entries are all
// 0 (no heat, no conduction).
template <typename R> struct alignas(4 * sizeof(R)) ThEntry { R irc, k, alpha, sigma0; };

// Denominator of eq. (6), sigma(T) = sigma_0 / (1 + alpha theta), floored at 1e-6: below 1 + alpha theta = 0 the
// formula has no meaning (include/em.h states the valid range); the floor keeps sigma finite and positive there.
template <typename R> __device__ __forceinline__ R thermal_den(R alpha, R theta) {
    const R d = alpha * theta + R(1);
    return d > R(1e-6) ? d : R(1e-6);
}

// Extra arguments of the thermally coupled sweep (em_sweep.cuh, TH = true); unused otherwise.
template <typename R>
struct ThermalSweep {
    R *theta;                    // temperature rise after the conduction kernel (theta_d); the sweep adds dq/(rho c_p) in place
    R *sig_out;                  // sigma(T^{n+1}) (the sigma(T^n) array is read through its tensor map)
    const ThEntry<R> *ttable;    // n_table entries
};

__device__ __forceinline__ float  mad(float a, float b, float c)    { return ::fmaf(a, b, c); }
__device__ __forceinline__ double mad(double a, double b, double c) { return ::fma(a, b, c); }
template <typename R> __device__ __forceinline__ R lerp(R lo, R hi, R f) { return mad(f, hi - lo, lo); }

// (st_stream16, the 16-byte streaming store of the output planes: em_ptx.cuh)

template <typename R> __device__ __forceinline__ R rcp(R x);
template <> __device__ __forceinline__ float  rcp<float>(float x) {
    // MUFU.RCP (<= 1 ulp) + one Newton step: no slow-path branch; x is a positive normal number here
    const float r = rcp_approx(x);
    return fmaf(r, fmaf(-x, r, 1.0f), r);
}
template <> __device__ __forceinline__ double rcp<double>(double x) { return 1.0 / x; }

// Loss coefficient r of the incremental form  E' = E + r (curlH - J - sigma E):
//   CD  (paper eq. 3): r = 1/(eps/dt + sigma/2)          == cb,  ca = 1 - sigma r
//   EXP               : r = -expm1(-sigma dt/eps)/sigma  == cb,  ca = 1 - sigma r = exp(-sigma dt/eps)
template <typename R, int LOSS>
__device__ __forceinline__ R loss_r(R A /*eps/dt*/, R B /*sigma*/) {
    if (LOSS == 0) {
        return rcp<R>(mad(R(0.5), B, A));
    } else {
        if (B > R(0)) {
            R u = B / A;
            return -::expm1(-u) / B;
        }
        return rcp<R>(A);
    }
}

// series conductance per unit face area of the two half cells: k_f / l~_f = 2 / (d_a/k_a + d_b/k_b) = 2 g_a g_b / (g_a + g_b)
// with the half-cell conductances g = k/d; 0 if either cell does not conduct (k = 0, or a pad cell: 1/d = 0)
template <typename R> __device__ __forceinline__ R half_cell_cond(R ga, R gb) {
    const R den = ga + gb;
    return den > R(0) ? R(2) * ga * gb * rcp<R>(den) : R(0);
}

}  // namespace em
