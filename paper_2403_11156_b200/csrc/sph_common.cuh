// sph_common.cuh -- shared device-side definitions of libsph_b200 (sm_100a).
//
// Product code: shares nothing with oracle/ (the CPU fp64 test oracle).  Citations are
// /root/reference/PAPER.md line numbers and the readings Rn of DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sph.h"

namespace sph {

constexpr int kBlock = 128;        // threads per CTA of the per-particle kernels
constexpr int kWarp = 32;
constexpr int kBigCell = 2048;     // cells above this size keep atomic order (R12 note in DESIGN.md)

// Uniform grid geometry (reading R11): cell edge c = h (1 + 2^-10) in fp32, origin = domain_min,
// n_a = floor((max_a - o_a) * inv_c) + 1, linear key x-fastest.
// Internally every R11 cell is split into kFineX slabs along x ("fine cells"): the store is sorted by
// fine key, and the x-run of a particle in fine cell f is the fine cells [f - kFineX, f + kFineX] =
// (2 + 1/kFineX) c wide instead of 3 c -- fewer candidates for the list builder.  Multiplying the
// fp32 cell coordinate t = (x - o) * inv_c by a power of two is exact, so floor(kFineX t) / kFineX =
// floor(t): the R11 cell of a particle is its fine cell / kFineX, and because the key is x-fastest
// the R11 cell_start is every kFineX-th entry of the fine one (what the ABI exports).
constexpr int kFineX = 2;          // power of two
struct Geom {
    float ox, oy, oz, inv_c;
    float inv_cx;                  // kFineX * inv_c
    int nx, ny, nz, ncells;        // FINE cell counts (nx = kFineX * R11 nx)
    int nxc, ncells_c;             // R11 (coarse) counts
};

// Per-simulation constants handed to kernels by value.
struct SimConst {
    Geom g;
    int nf, nb;          // fluid / boundary particle counts
    int nown;            // slab mode: particles whose original index is < nown are OWNED, the rest are ghosts
                         // of a neighbouring slab and stay out of the error sums; = nf otherwise
    int kf, kb;          // neighbour-list capacities (rows per warp tile)
    float h, h2, inv_h;  // support radius, h*h in fp32 (R10), 1/h
    float sigma;         // 8 / (pi h^3)           (R1)
    float grad_c;        // sigma / h
    float ga, gb;        // gradient factor of the inner branch: 6 (3q - 2) / h = ga r + gb, ga = 18 / h^2, gb = -12 / h
    float half_h;        // branch point q = 1/2 in terms of r
    float m;             // fluid particle mass     (R3)
    float rho0, dt;      // dt: the configured step (upper bound of the CFL rule, reading R26)
    const float *dt_dev; // the CURRENT step's dt (DevControl::dt), chosen on the device by k_step_begin
    float gx, gy, gz;
    float nu, mu;        // kinematic / dynamic viscosity (mu = nu rho0, R21)
    float visc_eps;      // 0.01 h^2                (Eq. 15 / 19, R4)
    float wc_k, wc_gamma;
    int has_dynamic;     // any dynamic rigid body
    int warm;            // warm start of both DFSPH solves (reading R27)
    float warm_w;        // omega
    float pci_k;         // PCISPH: delta dt^2 (reading R28)
};

// Loop-control block in device memory (one per simulation).  Written by the host only through
// cudaMemcpyAsync on the simulation's stream (sph_set_forced_iterations).
struct DevControl {
    int forced_v, forced_d, forced_cg;   // -1: tolerances decide
    int min_v, max_v, min_d, max_d, max_cg;
    int min_p, max_p;                    // PCISPH pressure loop (reading R28)
    int enable_div;
    float eta_v, eta_d, cg_tol;
    // running state of the current step
    int cont;                            // loop predicate as last evaluated (host-driven mode reads it)
    int it;                              // iteration counter of the running loop
    double cg_bb, cg_rr, cg_alpha, cg_beta;
    int cg_break;
    float dt;                            // time step of the running step (R26; = SphParams.dt when cfl_factor = 0)
    unsigned long long acc;              // running P-pass: CTA counter (top 20 bits) | fixed-point error sum (A12)
    unsigned long long last_total;       // fixed-point error sum of the last P-pass (slab mode: summed over the slabs by the host)
    int fold_end;                        // the P-pass that ends the step's last loop also closes the step's statistics (no k_step_end launch)
};

// Statistics block in device memory; sph_read_stats copies it out and converts to SphStats.
struct ListCounters {
    int max_f, max_b;            // read together (one 8-byte load) by the list builder's guard
    int overflow, pad;
    unsigned long long sum_f;
};
struct DevStats {
    long long steps_done, total_it_v, total_it_d, total_cg;
    int it_v, it_d, cg_iters, max_iter_hit;
    float err_v, err_rho, cg_residual;
    int oob, nan_count;
    unsigned vmax_bits;
    ListCounters lc;
    float dt_last;
    double sim_time;
};

// end of a step: running totals (k_step_end, or the last CTA of the P-pass that ends the step's last solver loop)
__device__ __forceinline__ void step_end_accumulate(DevStats *st, const DevControl *ctl)
{
    st->steps_done += 1;
    st->dt_last = ctl->dt; st->sim_time += (double)ctl->dt;
    st->total_it_v += st->it_v; st->total_it_d += st->it_d; st->total_cg += st->cg_iters;
}

// time step of the running step
__device__ __forceinline__ float step_dt(const SimConst &c) { return __ldg(c.dt_dev); }

// ---------------------------------------------------------------------------------------------
// Cell coordinate of one point: (int)floorf((x - o) * inv_c) with separate fp32 subtract and
// multiply (no contraction), clamped into [0, n-1]; NaN goes to cell 0 (R11).
__device__ __forceinline__ int cell_coord(float x, float o, float inv_c, int n, bool &clamped)
{
    float t = __fmul_rn(__fsub_rn(x, o), inv_c);
    if (!(t == t)) { clamped = true; return 0; }
    if (t < 0.0f) { clamped = true; return 0; }
    if (t >= (float)n) { clamped = true; return n - 1; }
    return (int)floorf(t);
}

// FINE key and coordinates (cx is the fine x coordinate)
__device__ __forceinline__ int cell_key(const Geom &g, float x, float y, float z, bool &clamped,
                                        int &cx, int &cy, int &cz)
{
    clamped = false;
    cx = cell_coord(x, g.ox, g.inv_cx, g.nx, clamped);
    cy = cell_coord(y, g.oy, g.inv_c, g.ny, clamped);
    cz = cell_coord(z, g.oz, g.inv_c, g.nz, clamped);
    return cx + g.nx * (cy + g.ny * cz);
}

// Squared distance of reading R10: d2 = fma(dz, dz, fma(dy, dy, dx*dx)), every operation in
// binary32 with round-to-nearest and exactly this association, so that the strict predicate
// d2 < h2 selects bit-identical neighbour sets on every implementation.
__device__ __forceinline__ float dist2_r10(float dx, float dy, float dz)
{
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// Cubic spline with support radius h (R1): W = sigma { 6(q^3 - q^2) + 1, q <= 1/2 ; 2(1-q)^3, q <= 1 }.
// Returns w(q) WITHOUT sigma (callers scale the finished sum once).
__device__ __forceinline__ float spline_w(float q)
{
    float t = 1.0f - q;
    float a = fmaf(6.0f * q * q, q - 1.0f, 1.0f);
    float b = 2.0f * t * t * t;
    return q <= 0.5f ? a : b;
}

// Gradient factor f with grad_i W(x_i - x_j) = sigma/h * f * (x_i - x_j):
//   q <= 1/2: w'(q)/r = 6 q (3q - 2) / r = 6 (3q - 2) / h      (no division, finite at r = 0)
//   q <= 1  : w'(q)/r = -6 (1 - q)^2 / r
// (R1, R2: the product with d = 0 vanishes at zero distance).  rinv = 1/r (unused when q <= 1/2).
__device__ __forceinline__ float spline_gradf(float q, float rinv, float inv_h)
{
    float t = 1.0f - q;
    float a = 6.0f * fmaf(3.0f, q, -2.0f) * inv_h;
    float b = -6.0f * t * t * rinv;
    return q <= 0.5f ? a : b;
}

// r and 1/r from d2 (d2 > 0 for the second branch; guarded for d2 == 0).  The argument of the
// reciprocal square root is never denormal (>= 1e-30), so the flush-to-zero MUFU form returns the
// same value as rsqrtf() without its denormal pre-/post-scaling instructions.
__device__ __forceinline__ void r_and_rinv(float d2, float &r, float &rinv)
{
    float a = fmaxf(d2, 1e-30f);
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(a));
    r = d2 * rinv;
}

// ---------------------------------------------------------------------------------------------
// Block-wide sums (warp shuffle, then one shared-memory hop).  Result valid in thread 0.
__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

template <typename T>
__device__ __forceinline__ T block_sum(T v, T *smem /* >= blockDim/32 */)
{
    v = warp_sum(v);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (lane == 0) smem[w] = v;
    __syncthreads();
    T r = T(0);
    if (w == 0) {
        r = lane < nw ? smem[lane] : T(0);
        r = warp_sum(r);
    }
    return r;
}

}  // namespace sph
