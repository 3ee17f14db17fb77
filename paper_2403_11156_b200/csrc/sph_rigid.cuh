// sph_rigid.cuh -- A8: Akinci boundary volumes, the reaction force of Eq. 14 and the rigid-body
// stand-in integrator (R9, R18), plus the loop-control kernels (A12) and the
// id-order import / export kernels of sph_read_state / sph_write_state.
#pragma once
#include "sph_passes.cuh"

namespace sph {

// ---------------------------------------------------------------------------------------------
// float[n*3] (caller order) -> float4[n]
__global__ void __launch_bounds__(256)
k_pack_vec3(const float *__restrict__ src, int n, float4 *__restrict__ dst, float w)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    dst[i] = make_float4(src[3 * i], src[3 * i + 1], src[3 * i + 2], w);
}
__global__ void __launch_bounds__(256) k_iota(int *a, int n)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = i;
}
// sorted float4 -> caller-order float[n*3]:  out[id[s]] = src[s].xyz
__global__ void __launch_bounds__(256)
k_export_vec3(const float4 *__restrict__ src, const int *__restrict__ id, int n, float *__restrict__ out)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    float4 v = src[s];
    int o = id != nullptr ? id[s] : s;
    out[3 * o] = v.x; out[3 * o + 1] = v.y; out[3 * o + 2] = v.z;
}
__global__ void __launch_bounds__(256)
k_export_w(const float4 *__restrict__ src, const int *__restrict__ id, int n, float *__restrict__ out,
           int stride /* float4 elements between consecutive particles */)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    out[id != nullptr ? id[s] : s] = src[(size_t)s * stride].w;
}
__global__ void __launch_bounds__(256)
k_export_scalar(const float *__restrict__ src, const int *__restrict__ id, int n, float *__restrict__ out)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    out[id[s]] = src[s];
}
// caller-order float[n*3] -> sorted float4 xyz (w kept): dst[s].xyz = src[id[s]]
__global__ void __launch_bounds__(256)
k_import_vec3(const float *__restrict__ src, const int *__restrict__ id, int n, float4 *__restrict__ dst)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int o = id != nullptr ? id[s] : s;
    float4 v = dst[s];
    v.x = src[3 * o]; v.y = src[3 * o + 1]; v.z = src[3 * o + 2];
    dst[s] = v;
}
// caller-order float[n] -> fourth lane of the sorted float4: dst[s].w = src[id[s]]
__global__ void __launch_bounds__(256)
k_import_w(const float *__restrict__ src, const int *__restrict__ id, int n, float4 *__restrict__ dst)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    dst[s].w = src[id[s]];
}
__global__ void __launch_bounds__(256)
k_export_counts(const int *__restrict__ ncount, const int *__restrict__ id, int n, int *__restrict__ out)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int p = ncount[s];
    out[2 * id[s]] = p & 0xffff;
    out[2 * id[s] + 1] = (p >> 16) & 0xffff;
}
// fluid neighbour rows in caller ids, -1 padded: 16-bit (run, offset) entries decoded through the
// particle's run starts (sph_passes.cuh)
__global__ void __launch_bounds__(256)
k_export_fluid_neighbors(const uint16_t *__restrict__ nl, const int *__restrict__ ncount,
                         const float4 *__restrict__ pos, Geom g, const int *__restrict__ fcs,
                         const int *__restrict__ id, int n, int K, int *__restrict__ out)
{
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * K) return;
    int s = (int)(t / K), k = (int)(t % K);
    int cnt = ncount[s] & 0xffff;
    int v = -1;
    if (k < cnt) {
        unsigned e = nl[list_tile(s, K) + (size_t)(k >> 1) * 64 + (s & 31) * 2 + (k & 1)];
        float4 x = pos[s];
        CellOf c = cell_of(g, x.x, x.y, x.z);
        int first;
        if (run_first_cell(g, c, (int)(e >> kOffBits), first)) v = id[fcs[first] + (int)(e & kOffMask)];
    }
    out[(size_t)id[s] * K + k] = v;
}

// boundary neighbour rows in caller ids, -1 padded: out[id[s]*K + k] = nid[list entry k of s]
__global__ void __launch_bounds__(256)
k_export_neighbors(const int *__restrict__ nl, const int *__restrict__ ncount, int shift,
                   const int *__restrict__ id, const int *__restrict__ nid, int n, int K,
                   int *__restrict__ out)
{
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * K) return;
    int s = (int)(t / K), k = (int)(t % K);
    int cnt = (ncount[s] >> shift) & 0xffff;
    int v = -1;
    if (k < cnt) v = nid[nl[(size_t)(s >> 5) * K * 32 + k * 32 + (s & 31)]];
    out[(size_t)id[s] * K + k] = v;
}

// ---------------------------------------------------------------------------------------------
// Slab mode: x-slab domain decomposition.  A slab's simulation holds its OWNED particles
// (original indices [0, nown)) followed by GHOSTS, copies of the neighbouring slabs' particles within h of the cut.
// Ghosts take part in every pass as neighbours; what a pass computes FOR them is wrong (their own neighbourhood is
// incomplete) and is overwritten with the owner's value before the next pass reads it (gather on the owner's side,
// scatter on the ghost's side, both addressed by original index through inv[]).
__global__ void __launch_bounds__(256) k_slab_inverse(const int *__restrict__ id, int n, int *__restrict__ inv)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) inv[id[s]] = s;
}
// out[k] = field[inv[idx[k]] * stride]   (float4 elements)
__global__ void __launch_bounds__(256)
k_slab_gather(const float4 *__restrict__ field, int stride, const int *__restrict__ inv, const int *__restrict__ idx, int n,
              float4 *__restrict__ out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = field[(size_t)inv[idx[k]] * stride];
}
// field[inv[first + k] * stride] = in[k]
__global__ void __launch_bounds__(256)
k_slab_scatter(float4 *__restrict__ field, int stride, const int *__restrict__ inv, int first, int n, const float4 *__restrict__ in)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) field[(size_t)inv[first + k] * stride] = in[k];
}
// loop state decided by the host from the error sums of ALL slabs (reading R14 evaluated once for the whole domain)
__global__ void k_slab_set_loop(DevControl *ctl, DevStats *st, int mode, int cont, int it, float err)
{
    ctl->cont = cont; ctl->it = it;
    if (mode == 0) { st->it_v = it; st->err_v = err; } else { st->it_d = it; st->err_rho = err; }
}
// selection of the particles with lo <= x < hi (and key[i] < key_lt when key != NULL) for migration / ghost layers:
// flag, exclusive scan (the grid builder's), compacting copy -- deterministic, input order kept
__global__ void __launch_bounds__(256)
k_select_flag(const float4 *__restrict__ pos, const int *__restrict__ key, int key_lt, int n, float lo, float hi, int *__restrict__ flag)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    int f = 0;
    if (i < n) {
        const float x = pos[i].x;
        f = (x >= lo && x < hi && (key == nullptr || key[i] < key_lt)) ? 1 : 0;
    }
    flag[i] = f;
}
__global__ void __launch_bounds__(256)
k_select_copy(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const int *__restrict__ gid, const int *__restrict__ key,
              const int *__restrict__ offset, int n, float4 *__restrict__ opos, float4 *__restrict__ ovel, int *__restrict__ ogid,
              int *__restrict__ oidx, int max_out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int o = offset[i];
    if (offset[i + 1] == o || o >= max_out) return;
    opos[o] = pos[i]; ovel[o] = vel[i];
    ogid[o] = gid[key != nullptr ? key[i] : i];        // gid is indexed by ORIGINAL index when a key (= original index of slot i) is given
    if (oidx != nullptr) oidx[o] = i;
}

// ---------------------------------------------------------------------------------------------
// Body-frame coordinates and initial sample velocities: xbar_k = R(q)^T (x_k - X),
// v_k = V + omega x (x_k - X) for dynamic bodies, 0 for static ones.
__device__ __forceinline__ void quat_to_R(const float q[4], double R[9])
{
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
    R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
    R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

// set_vel = 0 leaves the sample velocities alone (sph_write_state of positions only).
__global__ void __launch_bounds__(256)
k_body_rest(const float4 *__restrict__ bpos, const int *__restrict__ bbody,
            const SphRigidBody *__restrict__ bodies, int nb, float4 *__restrict__ brest,
            float4 *__restrict__ bvel, int set_vel)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nb) return;
    const SphRigidBody &B = bodies[bbody[k]];
    double R[9];
    quat_to_R(B.quat, R);
    float4 x = bpos[k];
    double d[3] = { (double)x.x - B.com[0], (double)x.y - B.com[1], (double)x.z - B.com[2] };
    brest[k] = make_float4((float)(R[0] * d[0] + R[3] * d[1] + R[6] * d[2]),
                           (float)(R[1] * d[0] + R[4] * d[1] + R[7] * d[2]),
                           (float)(R[2] * d[0] + R[5] * d[1] + R[8] * d[2]), 0.f);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (B.dynamic) {
        v.x = (float)(B.lin_vel[0] + (B.ang_vel[1] * d[2] - B.ang_vel[2] * d[1]));
        v.y = (float)(B.lin_vel[1] + (B.ang_vel[2] * d[0] - B.ang_vel[0] * d[2]));
        v.z = (float)(B.lin_vel[2] + (B.ang_vel[0] * d[1] - B.ang_vel[1] * d[0]));
    }
    if (set_vel) bvel[k] = v;
}

// Samples of DYNAMIC bodies re-posed from the body states (after sph_write_state of SPH_FIELD_RIGID_BODIES):
// x_k = X + R(q) xbar_k (set_pos), v_k = V + omega x (x_k - X) (set_vel); same arithmetic as the tail of k_rigid_step.
__global__ void __launch_bounds__(256)
k_body_pose(const float4 *__restrict__ brest, const int *__restrict__ bbody,
            const SphRigidBody *__restrict__ bodies, int nb, float4 *__restrict__ bpos,
            float4 *__restrict__ bvel, int set_pos, int set_vel)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nb) return;
    const SphRigidBody &B = bodies[bbody[k]];
    if (!B.dynamic) return;
    double R[9];
    quat_to_R(B.quat, R);
    float4 xb = brest[k];
    double r[3];
    for (int a = 0; a < 3; ++a) r[a] = R[3 * a] * xb.x + R[3 * a + 1] * xb.y + R[3 * a + 2] * xb.z;
    if (set_pos) {
        float4 x = bpos[k];
        x.x = (float)((double)B.com[0] + r[0]); x.y = (float)((double)B.com[1] + r[1]); x.z = (float)((double)B.com[2] + r[2]);
        bpos[k] = x;
    }
    if (set_vel)
        bvel[k] = make_float4((float)((double)B.lin_vel[0] + (double)B.ang_vel[1] * r[2] - (double)B.ang_vel[2] * r[1]),
                              (float)((double)B.lin_vel[1] + (double)B.ang_vel[2] * r[0] - (double)B.ang_vel[0] * r[2]),
                              (float)((double)B.lin_vel[2] + (double)B.ang_vel[0] * r[1] - (double)B.ang_vel[1] * r[0]), 0.f);
}

// Eq. 11 (R9): Psi_k = rho0 / sum_{k' in the same body, k included} W_kk'.
// One thread per SORTED boundary slot; writes Psi into the sorted store and the caller-order one.
__global__ void __launch_bounds__(kBlock)
k_boundary_psi(SimConst c, float4 *__restrict__ bpos_s, const int *__restrict__ bid_s,
               const int *__restrict__ bcs, const int *__restrict__ bbody,
               float4 *__restrict__ bpos_orig)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= c.nb) return;
    float4 x = bpos_s[s];
    int me = bid_s[s], body = bbody[me];
    const CellOf cell = cell_of(c.g, x.x, x.y, x.z);
    float sw = 0.f;
    for_each_candidate(c.g, bcs, cell, [&](int j, int, int) {
        if (j == s) return;
        float4 q = bpos_s[j];
        float dx = __fsub_rn(x.x, q.x), dy = __fsub_rn(x.y, q.y), dz = __fsub_rn(x.z, q.z);
        float d2 = dist2_r10(dx, dy, dz);
        if (d2 < c.h2 && bbody[bid_s[j]] == body) {
            float r, rinv;
            r_and_rinv(d2, r, rinv);
            sw += spline_w(r * c.inv_h);
        }
    });
    float psi = c.rho0 / (c.sigma * (1.0f + sw));
    bpos_s[s].w = psi;
    bpos_orig[me].w = psi;
}

// Eq. 14: reaction on boundary sample k of a dynamic body,
//   F_k += sum_{i in N(k)} m Psi_k (kappa_i / rho_i) gradW_ik,
// gathered on the boundary side (deterministic, no atomics): one thread per dynamic sample walks
// the FLUID grid around x_k.  Runs after every C-pass (the kappa/rho of that pass is in posk).
__global__ void __launch_bounds__(kBlock)
k_boundary_force(SimConst c, const int *__restrict__ dyn_idx, int ndyn,
                 const float4 *__restrict__ bpos_orig, const float4 *__restrict__ posk,
                 const int *__restrict__ fcs, float4 *__restrict__ bforce)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ndyn) return;
    int k = dyn_idx[t];
    float4 xk = bpos_orig[k];
    const CellOf cell = cell_of(c.g, xk.x, xk.y, xk.z);
    float fx = 0.f, fy = 0.f, fz = 0.f;
    for_each_candidate(c.g, fcs, cell, [&](int i, int, int) {
        float4 q = __ldg(posk + i);
        float dx = __fsub_rn(q.x, xk.x), dy = __fsub_rn(q.y, xk.y), dz = __fsub_rn(q.z, xk.z);  // x_i - x_k
        float d2 = dist2_r10(dx, dy, dz);
        if (d2 < c.h2) {
            float s = q.w * pair_gradf(c, d2);
            fx = fmaf(s, dx, fx); fy = fmaf(s, dy, fy); fz = fmaf(s, dz, fz);
        }
    });
    float s = c.m * xk.w * c.grad_c;
    float4 f = bforce[k];
    f.x = fmaf(s, fx, f.x); f.y = fmaf(s, fy, f.y); f.z = fmaf(s, fz, f.z);
    bforce[k] = f;
}

// Rigid stand-in (R18; PAPER.md:266 delegates this to an external engine): one CTA per body.
//   F = M g + sum F_k, tau = sum (x_k - X) x F_k; V += dt F / M;
//   omega += dt Iw^-1 (tau - omega x Iw omega), Iw = R Ib R^T; X += dt V;
//   q += dt/2 (0, omega) (x) q, normalised; frictionless inelastic contact sphere vs the tank AABB;
//   x_k = X + R xbar_k, v_k = V + omega x (x_k - X)  (constant during the next fluid solve: weak
//   coupling).  Body arithmetic in fp64 (one thread), samples in fp32.
__global__ void __launch_bounds__(256)
k_rigid_step(SimConst c, SphRigidBody *__restrict__ bodies, float tminx, float tminy, float tminz,
             float tmaxx, float tmaxy, float tmaxz, const float4 *__restrict__ brest,
             const float4 *__restrict__ bforce, float4 *__restrict__ bpos_orig,
             float4 *__restrict__ bvel_orig)
{
    __shared__ double red[8];
    __shared__ double sh[6];
    __shared__ double shR[9], shX[3], shV[3], shW[3];
    SphRigidBody &B = bodies[blockIdx.x];
    if (!B.dynamic) return;
    int k0 = B.first_particle, k1 = k0 + B.n_particles;
    double acc[6] = { 0, 0, 0, 0, 0, 0 };
    for (int k = k0 + threadIdx.x; k < k1; k += blockDim.x) {
        float4 f = bforce[k], x = bpos_orig[k];
        double r0 = (double)x.x - B.com[0], r1 = (double)x.y - B.com[1], r2 = (double)x.z - B.com[2];
        acc[0] += f.x; acc[1] += f.y; acc[2] += f.z;
        acc[3] += r1 * f.z - r2 * f.y; acc[4] += r2 * f.x - r0 * f.z; acc[5] += r0 * f.y - r1 * f.x;
    }
    for (int a = 0; a < 6; ++a) {
        double s = block_sum(acc[a], red);
        if (threadIdx.x == 0) sh[a] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double dt = step_dt(c), M = B.mass;
        double g[3] = { c.gx, c.gy, c.gz };
        double V[3], w[3], X[3], q[4], R[9];
        for (int a = 0; a < 3; ++a) { V[a] = B.lin_vel[a] + dt * (M * g[a] + sh[a]) / M; w[a] = B.ang_vel[a]; X[a] = B.com[a]; }
        quat_to_R(B.quat, R);
        double wb[3], Iw[3], gy[3], rhs[3], tb[3];
        for (int a = 0; a < 3; ++a) wb[a] = (R[0 + a] * w[0] + R[3 + a] * w[1] + R[6 + a] * w[2]) * B.inertia_body[a];
        for (int a = 0; a < 3; ++a) Iw[a] = R[3 * a] * wb[0] + R[3 * a + 1] * wb[1] + R[3 * a + 2] * wb[2];
        gy[0] = w[1] * Iw[2] - w[2] * Iw[1]; gy[1] = w[2] * Iw[0] - w[0] * Iw[2]; gy[2] = w[0] * Iw[1] - w[1] * Iw[0];
        for (int a = 0; a < 3; ++a) rhs[a] = sh[3 + a] - gy[a];
        for (int a = 0; a < 3; ++a) tb[a] = (R[0 + a] * rhs[0] + R[3 + a] * rhs[1] + R[6 + a] * rhs[2]) / B.inertia_body[a];
        for (int a = 0; a < 3; ++a) w[a] += dt * (R[3 * a] * tb[0] + R[3 * a + 1] * tb[1] + R[3 * a + 2] * tb[2]);
        for (int a = 0; a < 3; ++a) X[a] += dt * V[a];
        for (int a = 0; a < 4; ++a) q[a] = B.quat[a];
        double dq[4] = { -w[0] * q[1] - w[1] * q[2] - w[2] * q[3],
                          w[0] * q[0] + w[1] * q[3] - w[2] * q[2],
                          w[1] * q[0] + w[2] * q[1] - w[0] * q[3],
                          w[2] * q[0] + w[0] * q[2] - w[1] * q[1] };
        double nrm = 0.0;
        for (int a = 0; a < 4; ++a) { q[a] += 0.5 * dt * dq[a]; nrm += q[a] * q[a]; }
        nrm = sqrt(nrm);
        double lo[3] = { (double)tminx + B.contact_radius, (double)tminy + B.contact_radius, (double)tminz + B.contact_radius };
        double hi[3] = { (double)tmaxx - B.contact_radius, (double)tmaxy - B.contact_radius, (double)tmaxz - B.contact_radius };
        for (int a = 0; a < 3; ++a) {
            if (X[a] < lo[a]) { X[a] = lo[a]; if (V[a] < 0.0) V[a] = 0.0; }
            if (X[a] > hi[a]) { X[a] = hi[a]; if (V[a] > 0.0) V[a] = 0.0; }
        }
        for (int a = 0; a < 4; ++a) B.quat[a] = (float)(q[a] / nrm);
        for (int a = 0; a < 3; ++a) { B.com[a] = (float)X[a]; B.lin_vel[a] = (float)V[a]; B.ang_vel[a] = (float)w[a]; }
        quat_to_R(B.quat, R);
        for (int a = 0; a < 9; ++a) shR[a] = R[a];
        for (int a = 0; a < 3; ++a) { shX[a] = B.com[a]; shV[a] = B.lin_vel[a]; shW[a] = B.ang_vel[a]; }
    }
    __syncthreads();
    for (int k = k0 + threadIdx.x; k < k1; k += blockDim.x) {
        float4 xb = brest[k];
        double r[3];
        for (int a = 0; a < 3; ++a) r[a] = shR[3 * a] * xb.x + shR[3 * a + 1] * xb.y + shR[3 * a + 2] * xb.z;
        float4 x = bpos_orig[k];
        x.x = (float)(shX[0] + r[0]); x.y = (float)(shX[1] + r[1]); x.z = (float)(shX[2] + r[2]);
        bpos_orig[k] = x;
        bvel_orig[k] = make_float4((float)(shV[0] + shW[1] * r[2] - shW[2] * r[1]),
                                   (float)(shV[1] + shW[2] * r[0] - shW[0] * r[2]),
                                   (float)(shV[2] + shW[0] * r[1] - shW[1] * r[0]), 0.f);
    }
}

// ---------------------------------------------------------------------------------------------
// A12 loop control kernels (single CTA each).
enum { LOOP_DIV = 0, LOOP_DENS = 1, LOOP_CG = 2 };
constexpr int kCtrlThreads = 1024;   // one CTA sums the per-CTA partials: wide, so that the loads overlap

// Start of a step: choose its dt (reading R26: dt = clamp(lambda 2r / max|v|, dt_min, dt_max) with the
// velocities at the step's start -- st->vmax_bits holds their maximum, left there by the previous step's
// integration or by k_vmax; cfl2r = lambda 2r, 0 = fixed dt), then reset the per-step statistics.
__global__ void k_step_begin(DevStats *st, DevControl *ctl, float cfl2r, float dt_min, float dt_max, int fold_end)
{
    ctl->fold_end = fold_end;
    float dt = dt_max;
    if (cfl2r > 0.f) {
        float vmax = __uint_as_float(st->vmax_bits);
        dt = fminf(dt_max, cfl2r / fmaxf(vmax, 1e-30f));
        dt = fmaxf(dt, dt_min);
    }
    ctl->dt = dt;
    st->it_v = 0; st->it_d = 0; st->cg_iters = 0; st->max_iter_hit = 0;
    st->err_v = 0.f; st->err_rho = 0.f; st->cg_residual = 0.f;
    st->oob = 0; st->nan_count = 0; st->vmax_bits = 0u;
    st->lc.overflow = 0; st->lc.max_f = 0; st->lc.max_b = 0; st->lc.sum_f = 0ull;
    ctl->it = 0; ctl->cont = 0; ctl->cg_break = 0;
}
__global__ void k_list_counters_reset(DevStats *st)
{
    st->oob = 0;
    st->lc.overflow = 0; st->lc.max_f = 0; st->lc.max_b = 0; st->lc.sum_f = 0ull;
}
__global__ void k_step_end(DevStats *st, const DevControl *ctl)
{
    step_end_accumulate(st, ctl);
}

// CG start: |b|^2, |r0|^2, first predicate (R23: stop when |r| <= tol |b| or max iterations)
__global__ void __launch_bounds__(kCtrlThreads)
k_cg_ctrl0(const float *__restrict__ pbb, const float *__restrict__ prr, int nparts, DevControl *ctl,
           DevStats *st, cudaGraphConditionalHandle h, int use_handle)
{
    __shared__ double sm[kCtrlThreads / 32];
    double bb = reduce_partials(pbb, nparts, sm);
    double rr = reduce_partials(prr, nparts, sm);
    if (threadIdx.x != 0) return;
    ctl->cg_bb = bb; ctl->cg_rr = rr; ctl->it = 0; ctl->cg_break = 0;
    int maxit = ctl->forced_cg >= 0 ? ctl->forced_cg : ctl->max_cg;
    double tol2 = (double)ctl->cg_tol * (double)ctl->cg_tol * bb;
    int cont = 0 < maxit && (ctl->forced_cg >= 0 || rr > tol2);
    st->cg_iters = 0;
    st->cg_residual = bb > 0.0 ? (float)sqrt(rr / bb) : 0.f;
    set_loop_condition(h, use_handle, ctl, cont);
}
// alpha = rr / pAp
__global__ void __launch_bounds__(kCtrlThreads)
k_cg_ctrl1(const float *__restrict__ ppap, int nparts, DevControl *ctl)
{
    __shared__ double sm[kCtrlThreads / 32];
    double pAp = reduce_partials(ppap, nparts, sm);
    if (threadIdx.x != 0) return;
    if (!(pAp > 0.0)) { ctl->cg_alpha = 0.0; ctl->cg_break = 1; }
    else ctl->cg_alpha = ctl->cg_rr / pAp;
}
// beta = rr_new / rr, iteration count, predicate
__global__ void __launch_bounds__(kCtrlThreads)
k_cg_ctrl2(const float *__restrict__ prr, int nparts, DevControl *ctl, DevStats *st,
           cudaGraphConditionalHandle h, int use_handle)
{
    __shared__ double sm[kCtrlThreads / 32];
    double rr_new = reduce_partials(prr, nparts, sm);
    if (threadIdx.x != 0) return;
    int cont = 0;
    if (ctl->cg_break) { ctl->cg_beta = 0.0; }
    else {
        ctl->cg_beta = ctl->cg_rr > 0.0 ? rr_new / ctl->cg_rr : 0.0;
        ctl->cg_rr = rr_new;
        int it = ++ctl->it;
        int maxit = ctl->forced_cg >= 0 ? ctl->forced_cg : ctl->max_cg;
        double tol2 = (double)ctl->cg_tol * (double)ctl->cg_tol * ctl->cg_bb;
        cont = it < maxit && (ctl->forced_cg >= 0 || rr_new > tol2);
        st->cg_iters = it;
        st->cg_residual = ctl->cg_bb > 0.0 ? (float)sqrt(rr_new / ctl->cg_bb) : 0.f;
        if (ctl->forced_cg < 0 && !cont && rr_new > tol2) st->max_iter_hit |= 4;
    }
    set_loop_condition(h, use_handle, ctl, cont);
}

// max_i |v_i| of the persistent store into st->vmax_bits (same arithmetic as the integration tail): run
// before a step whose start velocities were not left by a previous step (first step, after sph_write_state)
__global__ void __launch_bounds__(256)
k_vmax(const float4 *__restrict__ vel, int n, unsigned *__restrict__ vmax_bits)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float v2 = 0.f;
    if (i < n) {
        float4 v = vel[i];
        v2 = fmaf(v.x, v.x, fmaf(v.y, v.y, v.z * v.z));
        if (!isfinite(v2)) v2 = 0.f;
    }
    v2 = warp_max(v2);
    if ((threadIdx.x & 31) == 0) {
        unsigned vb = __float_as_uint(sqrtf(v2));
        if (vb > *(volatile unsigned *)vmax_bits) atomicMax(vmax_bits, vb);
    }
}

}  // namespace sph
