// sph_passes.cuh -- A4-A7, A9-A12: the neighbour-sum kernels, their device-side reductions and
// loop control.
//
// Store layout (all fp32, sorted cell order, one thread per fluid particle):
//   pos [nf] float4  x, y, z, -
//   pv  [nf] PV      32-byte record { x, y, z, - | vx, vy, vz, rho }: the passes that need position
//                    AND velocity of a neighbour (A4 with the fused divergence P-pass, every P-pass,
//                    viscosity) fetch both with ONE 256-bit gather (LDG.E.256, sm_100) -- the list
//                    passes are bound by L1 gather wavefronts, and one 32-byte sector per neighbour
//                    costs fewer of them than two 16-byte gathers from two arrays.  rho_i rides in
//                    v.w (the viscosity sums need rho_j): k_density_alpha writes rho to its own array,
//                    the first C-pass (or k_wcsph_eos) copies it into the record it rewrites anyway.  pos stays as a packed copy: the list
//                    builder reads TWO candidates per 256-bit load from it.
//   posk[nf] float4  x, y, z, kappa_i/rho_i (written by every P-pass, gathered by the C-pass:
//                                            one 16-byte gather per neighbour instead of two)
//   bpos[nb] float4  x, y, z, Psi           bvel[nb] float4 vx, vy, vz, -
// Neighbour lists (built once per step by k_build_lists, consumed by every later pass): warp-tiled,
//   16-bit (x-run, offset) entries for fluid neighbours, 32-bit indices for boundary neighbours; see
//   list_tile() and for_each_neighbor() below.
#pragma once
#include "sph_common.cuh"

namespace sph {

enum { MODE_DIV = 0, MODE_DENS = 1, MODE_PCI = 2 };   // MODE_PCI: PCISPH pressure loop (reading R28)

struct __align__(32) PV { float4 x, v; };   // position (x, y, z, -) | velocity (vx, vy, vz, rho)

// list words are read once per pass: keep them out of L1, which the gathers need
__device__ __forceinline__ uint32_t ldg_stream(const uint32_t *p)
{
    uint32_t v;
    asm("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void ldg256_if(bool on, const float4 *p, float4 &a, float4 &b)
{
    asm("{\n\t.reg .pred pp;\n\tsetp.ne.u32 pp, %9, 0;\n\t"
        "@pp ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"
        : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
        : "l"(p), "r"((unsigned)on));
}
// 32 bytes (aligned) through the read-only path with one instruction
__device__ __forceinline__ void ldg256(const float4 *p, float4 &a, float4 &b)
{
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
        : "l"(p));
}


struct PassCtx {
    SimConst c;
    const float4 *pos;
    const float4 *bpos;
    const int *fcs;     // fluid cell_start [ncells + 1]
    const int *bcs;     // boundary cell_start
    uint16_t *nl_f;     // fluid neighbour list, 16-bit (x-run, offset) entries (see below)
    int *nl_b;          // boundary neighbour list, sorted boundary indices
    int *ncount;        // [nf] (#fluid) | (#boundary << 16)
    const int *id;      // [nf] original index of the particle in sorted slot s (slab mode: owned / ghost)
};

// ---------------------------------------------------------------------------------------------
// Candidate enumeration: the 27 cells around (cx, cy, cz) as 9 x-runs.  Cells are linearised
// x-fastest and the store is sorted by cell, so the three x-adjacent cells of one (y, z) row are
// ONE contiguous index range [cell_start[row + x0], cell_start[row + x1 + 1]).  The runs are
// numbered r = 3 (dz + 1) + (dy + 1); visiting them in this order visits the candidates in
// ascending sorted index.
constexpr int kRows = 9;
constexpr int kOffBits = 12;                 // fluid list entry = (r << 12) | (j - run start)
constexpr int kOffMask = (1 << kOffBits) - 1;

struct CellOf { int cx, cy, cz, x0, x1; };

__device__ __forceinline__ CellOf cell_of(const Geom &g, float x, float y, float z)
{
    CellOf c; bool cl;
    cell_key(g, x, y, z, cl, c.cx, c.cy, c.cz);
    c.x0 = max(c.cx - kFineX, 0); c.x1 = min(c.cx + kFineX, g.nx - 1);
    return c;
}

// first cell of x-run r (index into cell_start), false if the run lies outside the grid
__device__ __forceinline__ bool run_first_cell(const Geom &g, const CellOf &c, int r, int &first)
{
    int z = c.cz + r / 3 - 1, y = c.cy + r % 3 - 1;
    if ((unsigned)z >= (unsigned)g.nz || (unsigned)y >= (unsigned)g.ny) return false;
    first = g.nx * (y + g.ny * z) + c.x0;
    return true;
}

// f(j, r, s): candidate j of run r whose first index is s
template <class F>
__device__ __forceinline__ void for_each_candidate(const Geom &g, const int *__restrict__ cs,
                                                   const CellOf &c, F &&f)
{
#pragma unroll 1
    for (int r = 0; r < kRows; ++r) {
        int first;
        if (!run_first_cell(g, c, r, first)) continue;
        int s = __ldg(cs + first), e = __ldg(cs + first + (c.x1 - c.x0) + 1);
#pragma unroll 4
        for (int j = s; j < e; ++j) f(j, r, s);
    }
}

// Fluid neighbour list.  Warp tile w = i / 32 owns kf * 32 16-bit entries; entry k of particle i
// is at tile + (k >> 1) * 64 + (i & 31) * 2 + (k & 1): a warp reads entries 2p and 2p + 1 of all its
// lanes with ONE coalesced 128-byte load.  An entry names its neighbour by x-run and offset inside
// the run, decoded through the particle's table of 9 run starts (tbl, one shared-memory column per
// thread): j = tbl[r] + off.  Half the bytes of a 32-bit index list: the list is the dominant HBM
// stream of every solver pass.
__device__ __forceinline__ size_t list_tile(int i, int cap) { return (size_t)(i >> 5) * (size_t)cap * 32; }

__device__ __forceinline__ void fill_run_table(const Geom &g, const int *__restrict__ cs, const CellOf &c,
                                               int *tbl /* + threadIdx.x, stride kBlock */)
{
#pragma unroll
    for (int r = 0; r < kRows; ++r) {
        int first;
        tbl[r * kBlock] = run_first_cell(g, c, r, first) ? __ldg(cs + first) : 0;
    }
}

constexpr int kPairs1 = 4;    // entry pairs per software-pipeline stage when one array is gathered
constexpr int kPairs2 = 2;    // ... when two arrays (or 32-byte records) are gathered

// Visit every neighbour of fluid particle i (sorted index), fluid first then boundary, both in
// ascending sorted index:
//   ff(j, qj, q2j, dx, dy, dz, d2) for fluid j != i with d2 < h2,  fb(k, pk, dx, dy, dz, d2) for boundary k;
//   d = x_i - x_j in fp32, d2 as in reading R10; qj = src[j], q2j = src2[j] (NSRC == 2, else qj);
//   NSRC == 3: src points at PV records, (qj, q2j) = (pv[j].x, pv[j].v) from one 256-bit load.
// LIST = true : gather through the per-step list (predicate was evaluated when it was built).  The
//   list words of the next stage are requested before the gathers of the current one are consumed,
//   and all gathers of a stage are issued before their arithmetic: the pass is bound by memory
//   latency otherwise.
// LIST = false: walk the cells and evaluate the predicate (same visiting order, same arithmetic).
// `src` is the float4 array whose xyz are the neighbour positions (pos or posk);
// WITH_B = false skips the boundary part.  tbl: kRows * kBlock ints of shared memory (LIST only).
// PADSAFE (NSRC 1 or 2, LIST): ff is also called for the slots past the end of a lane's list, with the
//   lane's OWN record as the neighbour (d = 0 exactly): legal when every term ff accumulates carries a
//   factor d (or v_i - v_j), so that such a call adds exactly 0 -- it removes one branch per slot from
//   the issue-bound C-pass.
template <bool LIST, bool WITH_B, int NSRC, bool PADSAFE, class FF, class FB>
__device__ __forceinline__ void for_each_neighbor(const PassCtx &p, const float4 *__restrict__ src,
                                                  const float4 *__restrict__ src2, int *tbl_base,
                                                  int i, float xi, float yi, float zi, FF &&ff, FB &&fb)
{
    const CellOf cell = cell_of(p.c.g, xi, yi, zi);
    if (LIST) {
        constexpr int PB = NSRC >= 2 ? kPairs2 : kPairs1;
        const int packed = p.ncount[i];
        const int cf = packed & 0xffff, cb = (packed >> 16) & 0xffff;
        int *tbl = tbl_base + threadIdx.x;
        fill_run_table(p.c.g, p.fcs, cell, tbl);
        const uint32_t *lp = reinterpret_cast<const uint32_t *>(p.nl_f + list_tile(i, p.c.kf)) + (i & 31);
        const int npair = (cf + 1) >> 1;
        uint32_t cur[PB];
#pragma unroll
        for (int t = 0; t < PB; ++t) cur[t] = t < npair ? ldg_stream(lp + t * 32) : 0u;
#pragma unroll 1
        for (int pb = 0; pb < npair; pb += PB) {
            uint32_t nxt[PB];
#pragma unroll
            for (int t = 0; t < PB; ++t) nxt[t] = pb + PB + t < npair ? ldg_stream(lp + (pb + PB + t) * 32) : 0u;
            int jj[2 * PB];
            float4 q[2 * PB], q2[NSRC >= 2 ? 2 * PB : 1];
            const int rem = cf - 2 * pb;                  // entries left, this stage included
#pragma unroll
            for (int u = 0; u < 2 * PB; ++u) {
                const bool valid = u < rem;
                // (words past the list are 0 and the builder zeroes the unwritten half of an odd tail pair: every
                // slot decodes to a table entry, no guard needed before the look-up)
                const uint32_t e = (u & 1) ? (cur[u >> 1] >> 16) : (cur[u >> 1] & 0xffffu);
                int j = tbl[(e >> kOffBits) * kBlock] + (int)(e & kOffMask);
                jj[u] = valid ? j : i;
                // predicated record gather: a lane whose list has ended issues no memory access at all (its registers
                // stay undefined and are never read -- the arithmetic below is under the same predicate); the record
                // passes are bound by L1 wavefronts, and ended lanes would each touch their own record's line
                if (NSRC == 3) ldg256_if(valid, src + 2 * jj[u], q[u], q2[u]);
                else {
                    q[u] = __ldg(src + jj[u]);       // (measured: predication costs the issue-bound C-pass more than it saves)
                    if (NSRC == 2) q2[u] = __ldg(src2 + jj[u]);
                }
            }
#pragma unroll
            for (int u = 0; u < 2 * PB; ++u) {
                if ((PADSAFE && NSRC != 3) || u < rem) {
                    float dx = __fsub_rn(xi, q[u].x), dy = __fsub_rn(yi, q[u].y), dz = __fsub_rn(zi, q[u].z);
                    ff(jj[u], q[u], NSRC >= 2 ? q2[u] : q[u], dx, dy, dz, dist2_r10(dx, dy, dz));
                }
            }
#pragma unroll
            for (int t = 0; t < PB; ++t) cur[t] = nxt[t];
        }
        if (WITH_B && cb > 0) {
            const int *lb = p.nl_b + list_tile(i, p.c.kb) + (i & 31);
#pragma unroll 2
            for (int k = 0; k < cb; ++k) {
                int j = __ldg(lb + k * 32);
                float4 q = __ldg(p.bpos + j);
                float dx = __fsub_rn(xi, q.x), dy = __fsub_rn(yi, q.y), dz = __fsub_rn(zi, q.z);
                fb(j, q, dx, dy, dz, dist2_r10(dx, dy, dz));
            }
        }
    } else {
        const float h2 = p.c.h2;
        for_each_candidate(p.c.g, p.fcs, cell, [&](int j, int, int) {
            float4 q, q2;
            if (NSRC == 3) ldg256(src + 2 * j, q, q2); else q = __ldg(src + j);
            float dx = __fsub_rn(xi, q.x), dy = __fsub_rn(yi, q.y), dz = __fsub_rn(zi, q.z);
            float d2 = dist2_r10(dx, dy, dz);
            if (d2 < h2 && j != i) ff(j, q, NSRC == 3 ? q2 : (NSRC == 2 ? __ldg(src2 + j) : q), dx, dy, dz, d2);
        });
        if (WITH_B && p.c.nb > 0) {
            for_each_candidate(p.c.g, p.bcs, cell, [&](int j, int, int) {
                float4 q = __ldg(p.bpos + j);
                float dx = __fsub_rn(xi, q.x), dy = __fsub_rn(yi, q.y), dz = __fsub_rn(zi, q.z);
                float d2 = dist2_r10(dx, dy, dz);
                if (d2 < h2) fb(j, q, dx, dy, dz, d2);
            });
        }
    }
}

// gradient factor for a pair at squared distance d2: grad_i W_ij = grad_c * gf * d
__device__ __forceinline__ float pair_gradf(const SimConst &c, float d2)
{
    // spline_gradf(r / h, 1 / r, 1 / h) with the constants folded (R1): inner branch 6 (3q - 2) / h = ga r + gb,
    // outer branch -6 (1 - q)^2 / r
    float r, rinv;
    r_and_rinv(d2, r, rinv);
    float a = fmaf(r, c.ga, c.gb);
    float t = fmaf(r, -c.inv_h, 1.0f);
    float b = (t * t) * (-6.0f * rinv);
    return r <= c.half_h ? a : b;
}

// ---------------------------------------------------------------------------------------------
// A12: device-side reductions and loop control.  Every P-pass reduces its error term on the
// device; the LAST CTA of the launch to finish evaluates the loop predicate of Alg. 2
// (R14: the error measured by this iteration's P-pass decides whether another
// iteration follows its C-pass) and sets the CUDA-graph WHILE condition -- no host round trip and
// no separate control launch (solver_tail below).  reduce_partials serves the CG dot products.  The C-pass that follows reads ctl->cont: the last C-pass of
// a loop also does the work that follows the loop (gravity after the divergence solve,
// integration after the density solve).
__device__ __forceinline__ double reduce_partials(const float *__restrict__ partial, int n, double *sm)
{
    // fixed summation order (deterministic): float4 loads that bypass L1 (the partials were written
    // by other SMs, possibly during this very launch), four chains per thread
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    const int st = blockDim.x, n4 = n >> 2;
    const float4 *p4 = reinterpret_cast<const float4 *>(partial);
    int k = threadIdx.x;
    for (; k + 3 * st < n4; k += 4 * st) {
        float4 a = __ldcg(p4 + k), b = __ldcg(p4 + k + st), c = __ldcg(p4 + k + 2 * st), d = __ldcg(p4 + k + 3 * st);
        s0 += ((double)a.x + (double)a.y) + ((double)a.z + (double)a.w);
        s1 += ((double)b.x + (double)b.y) + ((double)b.z + (double)b.w);
        s2 += ((double)c.x + (double)c.y) + ((double)c.z + (double)c.w);
        s3 += ((double)d.x + (double)d.y) + ((double)d.z + (double)d.w);
    }
    for (; k < n4; k += st) {
        float4 a = __ldcg(p4 + k);
        s0 += ((double)a.x + (double)a.y) + ((double)a.z + (double)a.w);
    }
    for (k = (n4 << 2) + threadIdx.x; k < n; k += st) s1 += (double)__ldcg(partial + k);
    return block_sum((s0 + s1) + (s2 + s3), sm);
}

__device__ __forceinline__ void set_loop_condition(cudaGraphConditionalHandle h, int use_handle,
                                                   DevControl *ctl, int cont)
{
    ctl->cont = cont;
    if (use_handle) cudaGraphSetConditional(h, cont ? 1u : 0u);
}

struct LoopHandle { cudaGraphConditionalHandle h; int use_handle; };

// thread 0 of the last CTA: predicate of the divergence (MODE_DIV) / density (MODE_DENS) loop.
// err: the loop's error measure (R6); first: this P-pass opens the loop (iteration counter restarts at 1).
template <int MODE>
__device__ __forceinline__ void solver_ctrl_eval(double err, DevControl *ctl, DevStats *st, LoopHandle lh, bool first)
{
    const bool on = MODE == MODE_DIV ? (ctl->enable_div && ctl->forced_v != 0 && ctl->max_v > 0)
                  : MODE == MODE_DENS ? (ctl->forced_d != 0 && ctl->max_d > 0) : (ctl->forced_d != 0 && ctl->max_p > 0);
    if (!on) {
        // loop switched off: the peeled first iteration runs with kappa = 0 (a no-op on v)
        if (MODE == MODE_DIV) { st->it_v = 0; st->err_v = 0.f; } else { st->it_d = 0; st->err_rho = 0.f; }
        ctl->it = 0;
        set_loop_condition(lh.h, lh.use_handle, ctl, 0);
        if (MODE != MODE_DIV && ctl->fold_end) step_end_accumulate(st, ctl);
        return;
    }
    const int l = first ? 1 : ctl->it + 1;
    ctl->it = l;
    int cont;
    if (MODE == MODE_DIV) {
        int f = ctl->forced_v;
        cont = f > 0 ? (l < f) : ((err > (double)ctl->eta_v || l < ctl->min_v) && l < ctl->max_v);
        st->it_v = l; st->err_v = (float)err;
        if (f < 0 && !cont && err > (double)ctl->eta_v) st->max_iter_hit |= 1;
    } else {
        int f = ctl->forced_d;
        const int mn = MODE == MODE_PCI ? ctl->min_p : ctl->min_d, mx = MODE == MODE_PCI ? ctl->max_p : ctl->max_d;
        cont = f > 0 ? (l < f) : ((err > (double)ctl->eta_d || l < mn) && l < mx);
        st->it_d = l; st->err_rho = (float)err;
        if (f < 0 && !cont && err > (double)ctl->eta_d) st->max_iter_hit |= 2;
        // the density (or PCISPH pressure) loop is the step's last: its final P-pass closes the step's statistics
        if (!cont && ctl->fold_end) step_end_accumulate(st, ctl);
    }
    set_loop_condition(lh.h, lh.use_handle, ctl, cont);
}

// End of a P-pass kernel: `term` is this thread's error term (R_i or E_i >= 0).  All threads of the
// CTA call it.  The CTA's sum (fixed shuffle order, fp32) is made dimensionless -- dt/rho0 * sum R_i
// (R6: density change per step) or sum E_i / rho0 (R6) -- converted to 44-bit fixed point (2^-20
// resolution) and added, together with a 1 in the CTA counter held in the top 20 bits, by ONE 64-bit
// atomic: integer addition is associative, so the total is bit-identical whatever order the CTAs
// arrive in, and the atomic's return value tells the last CTA that it is the last and what the
// total is -- no fence, no partial array, no second pass.  Contributions are clamped so that the
// 44-bit field cannot carry into the counter (a mean error above ~13 at 1.2M particles saturates).
constexpr int kAccFracBits = 20, kAccSumBits = 44;

// slab mode: ghosts (copies of a neighbouring slab's particles) do not count in the error sums
__device__ __forceinline__ bool is_ghost(const PassCtx &p, int i) { return p.c.nown < p.c.nf && p.id[i] >= p.c.nown; }

template <int MODE>
__device__ __forceinline__ void solver_tail(const SimConst &c, float term, DevControl *ctl, DevStats *st,
                                            LoopHandle lh, bool first)
{
    __shared__ float red[kBlock / 32];
    float s = block_sum(term, red);
    if (threadIdx.x != 0) return;
    const double norm = MODE == MODE_DIV ? (double)step_dt(c) / (double)c.rho0 : 1.0 / (double)c.rho0;
    const unsigned long long cap = ((1ull << kAccSumBits) - 1ull) / (unsigned long long)gridDim.x;
    double d = (double)s * norm * (double)(1u << kAccFracBits) + 0.5;
    unsigned long long q = d > 0.0 ? (d < (double)cap ? (unsigned long long)d : cap) : 0ull;   // NaN -> 0
    unsigned long long old = atomicAdd(&ctl->acc, (1ull << kAccSumBits) | q);
    if ((old >> kAccSumBits) != (unsigned long long)(gridDim.x - 1)) return;
    ctl->acc = 0ull;                                            // every CTA has arrived: reset for the next pass
    unsigned long long total = (old & ((1ull << kAccSumBits) - 1ull)) + q;
    ctl->last_total = total;
    double err = c.nf > 0 ? (double)total / (double)(1u << kAccFracBits) / (double)c.nf : 0.0;
    solver_ctrl_eval<MODE>(err, ctl, st, lh, first);
}

// ---------------------------------------------------------------------------------------------
// A4 second half: density (Eq. 4 + Eq. 12; self term included, R2) and the
// DFSPH factor alpha_i = rho_i / (|S_i|^2 + T_i), S_i = sum_j m gradW_ij + sum_k Psi_k gradW_ik,
// T_i = sum_j |m gradW_ij|^2 (R5, R7).
// DIVP = true additionally runs the P-pass of the FIRST divergence-solve iteration in the same
// neighbour loop (A5): D_i needs only the velocities of the step's start, and kappa^v_i the
// alpha_i that this very loop produces -- one full neighbour pass less per step.  It writes
// posk[i] = (x_i, kappa^v_i / rho_i) (0 when the divergence solve is switched off) and the CTA
// error sum of R_i = max(D_i, 0) (solver_tail).
template <bool LIST, bool DIVP, bool DYN>
__global__ void __launch_bounds__(kBlock)
k_density_alpha(PassCtx p, const PV *__restrict__ pv, const float4 *__restrict__ bvel,
                float *__restrict__ alpha, float *__restrict__ rho_out, float4 *__restrict__ posk,
                DevControl *ctl, DevStats *st, LoopHandle lh)
{
    __shared__ int tbl[LIST ? kRows * kBlock : 1];
    const SimConst &c = p.c;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float term = 0.f;
    if (i < c.nf) {
        float4 xi = p.pos[i];
        float4 vi = pv[i].v;
        float sw = 0.f, sx = 0.f, sy = 0.f, sz = 0.f, t2 = 0.f;    // fluid: sum w, sum gf d, sum gf^2 d2
        float bw = 0.f, bx = 0.f, by = 0.f, bz = 0.f;              // boundary, Psi-weighted
        float df = 0.f, db = 0.f;                                  // density rate (DIVP)
        for_each_neighbor<LIST, true, DIVP ? 3 : 1, false>(p, DIVP ? reinterpret_cast<const float4 *>(pv) : p.pos, nullptr, tbl, i, xi.x, xi.y, xi.z,
            [&](int, float4, float4 vj, float dx, float dy, float dz, float d2) {
                float r, rinv;
                r_and_rinv(d2, r, rinv);
                float q = r * c.inv_h;
                sw += spline_w(q);
                float gf = spline_gradf(q, rinv, c.inv_h);
                sx = fmaf(gf, dx, sx); sy = fmaf(gf, dy, sy); sz = fmaf(gf, dz, sz);
                t2 = fmaf(gf * gf, d2, t2);
                if (DIVP) {
                    float dv = fmaf(vi.x - vj.x, dx, fmaf(vi.y - vj.y, dy, (vi.z - vj.z) * dz));
                    df = fmaf(gf, dv, df);
                }
            },
            [&](int k, float4 pk, float dx, float dy, float dz, float d2) {
                float r, rinv;
                r_and_rinv(d2, r, rinv);
                float q = r * c.inv_h;
                bw = fmaf(pk.w, spline_w(q), bw);
                float gf = pk.w * spline_gradf(q, rinv, c.inv_h);
                bx = fmaf(gf, dx, bx); by = fmaf(gf, dy, by); bz = fmaf(gf, dz, bz);
                if (DIVP) {
                    float dv;
                    if (DYN) {
                        float4 vk = __ldg(bvel + k);
                        dv = fmaf(vi.x - vk.x, dx, fmaf(vi.y - vk.y, dy, (vi.z - vk.z) * dz));
                    } else dv = fmaf(vi.x, dx, fmaf(vi.y, dy, vi.z * dz));
                    db = fmaf(gf, dv, db);
                }
            });
        float rho = c.sigma * fmaf(c.m, 1.0f + sw, bw);            // W(0) = sigma
        float Sx = c.grad_c * fmaf(c.m, sx, bx), Sy = c.grad_c * fmaf(c.m, sy, by),
              Sz = c.grad_c * fmaf(c.m, sz, bz);
        float T = (c.grad_c * c.m) * (c.grad_c * c.m) * t2;
        float den = fmaf(Sx, Sx, fmaf(Sy, Sy, fmaf(Sz, Sz, T)));
        float a = den > 1e-6f ? rho / den : 0.0f;
        alpha[i] = a;
        rho_out[i] = rho;                                          // the record's rho lane is filled by the pass that follows
                                                                   // (other CTAs of this launch gather whole records)
        if (DIVP) {
            // Eq. 10 source (R15): R_i = max(D_i, 0), kappa^v_i = alpha_i R_i / dt
            bool on = ctl->enable_div && ctl->forced_v != 0 && ctl->max_v > 0;
            float D = c.grad_c * fmaf(c.m, df, db);
            term = fmaxf(D, 0.f);
            float kappa = a * term / step_dt(c);
            posk[i] = make_float4(xi.x, xi.y, xi.z, on ? kappa / rho : 0.f);
            if (is_ghost(p, i)) term = 0.f;
        }
    }
    if (DIVP) solver_tail<MODE_DIV>(c, term, ctl, st, lh, true);
}

// ---------------------------------------------------------------------------------------------
// P-pass of both solvers (A5 / A7).  Density rate (Eq. 6 times rho):
//   D_i = sum_j m (v_i - v_j).gradW_ij + sum_k Psi_k (v_i - v_k).gradW_ik
// DIV  (Eq. 10 source; R15): R_i = max(D_i, 0), kappa^v_i = alpha_i R_i / dt, term = R_i
// DENS (Eq. 8-9; R15) : E_i = max(rho_i + dt D_i, rho0) - rho0,
//                                          kappa_i = alpha_i E_i / dt^2, term = E_i
// Writes posk[i] = (x_i, kappa_i / rho_i); the error term is reduced by solver_tail (A12).

template <bool LIST, int MODE, bool DYN>
__global__ void __launch_bounds__(kBlock)
k_solver_p(PassCtx p, const PV *__restrict__ pv, const float4 *__restrict__ bvel,
           const float *__restrict__ alpha, float4 *__restrict__ posk,
           DevControl *ctl, DevStats *st, LoopHandle lh, int first, float *__restrict__ ksum)
{
    __shared__ int tbl[LIST ? kRows * kBlock : 1];
    const SimConst &c = p.c;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float term = 0.f;
    if (i < c.nf) {
        float4 xi, vi;
        ldg256(reinterpret_cast<const float4 *>(pv + i), xi, vi);
        float df = 0.f, db = 0.f;
        for_each_neighbor<LIST, true, 3, false>(p, reinterpret_cast<const float4 *>(pv), nullptr, tbl, i, xi.x, xi.y, xi.z,
            [&](int, float4, float4 vj, float dx, float dy, float dz, float d2) {
                float gf = pair_gradf(c, d2);
                float dv = fmaf(vi.x - vj.x, dx, fmaf(vi.y - vj.y, dy, (vi.z - vj.z) * dz));
                df = fmaf(gf, dv, df);
            },
            [&](int k, float4 pk, float dx, float dy, float dz, float d2) {
                float gf = pk.w * pair_gradf(c, d2);
                float dv;
                if (DYN) {
                    float4 vk = __ldg(bvel + k);
                    dv = fmaf(vi.x - vk.x, dx, fmaf(vi.y - vk.y, dy, (vi.z - vk.z) * dz));
                } else dv = fmaf(vi.x, dx, fmaf(vi.y, dy, vi.z * dz));
                db = fmaf(gf, dv, db);
            });
        float D = c.grad_c * fmaf(c.m, df, db);
        const float dt = step_dt(c);
        float rho = vi.w, a = alpha[i], kappa;
        if (MODE == MODE_PCI) {
            // reading R28: rho* = rho + dt D (Eq. 9), p <- max(p + delta (rho* - rho0), 0), delta = pci_k / dt^2;
            // the C-pass applies the INCREMENT of p / rho^2 (the pressure force of Eq. 7 is linear in p)
            const float e = fmaf(dt, D, rho) - c.rho0;
            term = fmaxf(e, 0.f);
            const float pold = ksum[i];
            float pn = fmaxf(fmaf(c.pci_k / (dt * dt), e, pold), 0.f);
            if (first && !(ctl->forced_d != 0 && ctl->max_p > 0)) pn = pold;
            ksum[i] = pn;
            kappa = (pn - pold) / rho;                              // written below as kappa / rho = dp / rho^2
        } else if (MODE == MODE_DIV) {
            term = fmaxf(D, 0.f);
            kappa = a * term / dt;
            // (warm-start path only: there this launch opens the divergence loop, which may be switched off)
            if (first && !(ctl->enable_div && ctl->forced_v != 0 && ctl->max_v > 0)) kappa = 0.f;
        } else {
            term = fmaxf(fmaf(dt, D, rho), c.rho0) - c.rho0;
            kappa = a * term / (dt * dt);
            // the P-pass that opens the density loop runs even when the loop is switched off
            // (forced 0 iterations): kappa = 0 then, and its C-pass only integrates
            if (first && !(ctl->forced_d != 0 && ctl->max_d > 0)) kappa = 0.f;
        }
        posk[i] = make_float4(xi.x, xi.y, xi.z, kappa / rho);
        if (MODE != MODE_PCI && ksum != nullptr) ksum[i] += kappa; // running total of the solve (warm start, R27)
        if (is_ghost(p, i)) term = 0.f;
    }
    solver_tail<MODE>(c, term, ctl, st, lh, first != 0);
}

// Warm start (reading R27): before a solve's loop the total stiffness K_i that the
// same solve applied in the LAST step, scaled by omega, is applied once through an ordinary C-pass with the
// densities and gradients of the current step.  K_i travels with the particle in the fourth lane of the persistent
// position (density solve) / velocity (divergence solve) and has been permuted by the sort.  This kernel writes
// posk[i] = (x_i, omega K_i / rho_i) and starts the solve's running total at omega K_i (0 when the solve is off).
template <int MODE>
__global__ void __launch_bounds__(256)
k_warm_prepare(SimConst c, const float4 *__restrict__ pos, const PV *__restrict__ pv, const float *__restrict__ rho,
               const DevControl *__restrict__ ctl, float4 *__restrict__ posk, float *__restrict__ ksum)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.nf) return;
    const bool on = MODE == MODE_DIV ? (ctl->enable_div && ctl->forced_v != 0 && ctl->max_v > 0)
                                     : (ctl->forced_d != 0 && ctl->max_d > 0);
    const float4 x = pos[i];
    const float K = MODE == MODE_DIV ? pv[i].v.w : x.w;
    const float k = on ? c.warm_w * K : 0.f;
    posk[i] = make_float4(x.x, x.y, x.z, k / rho[i]);
    ksum[i] = k;
}

// C-pass (A5 / A7 / A10): pressure-like velocity update (Eq. 7 + Eq. 13 with p/rho^2 == kappa/rho,
// PAPER.md:123, 200):  v_i -= dt [ sum_j m (kr_i + kr_j) gradW_ij + sum_k Psi_k kr_i gradW_ik ].
// The LAST C-pass of a loop (ctl->cont == 0, set by the P-pass before it) also does what follows the
// loop, on the value it holds in registers:
//   TAIL_DIV : v += dt g              (A6 without viscosity, Alg. 1 l.1-2; add_gravity)
//   TAIL_DENS: x += dt v with the updated v (A9, symplectic Euler, Alg. 1 l.5-6); writes
//              the persistent store (pos_out, vel_out, id_out) that the next step's sort reads and
//              the step's v_max / non-finite counters
//   TAIL_WCSPH: as TAIL_DENS, unconditionally (the WCSPH step has one C-pass).
enum { TAIL_DIV = 0, TAIL_DENS = 1, TAIL_WCSPH = 2 };

struct CTail {
    const DevControl *ctl;
    const float *rho;         // TAIL_DIV: rho_i of this step, copied into the record's fourth velocity lane
    int add_gravity;
    const int *id;
    float4 *pos_out, *vel_out;
    int *id_out;
    unsigned *vmax_bits;
    int *nan_count;
    int force_mid;            // 1: this launch is never the loop's last one (the warm-start C-pass, reading R27)
    const float *ksum_v, *ksum_d;   // warm start: totals of this step's solves, stored with the persistent state (else NULL)
};

template <bool LIST, int TAIL>
__global__ void __launch_bounds__(kBlock)
k_solver_c(PassCtx p, const float4 *__restrict__ posk, PV *__restrict__ pv, CTail t)
{
    __shared__ int tbl[LIST ? kRows * kBlock : 1];
    const SimConst &c = p.c;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool last = !t.force_mid && (TAIL == TAIL_WCSPH || t.ctl->cont == 0);
    float v2 = 0.f;
    bool bad = false;
    if (i < c.nf) {
        float4 xi = posk[i];
        float kri = xi.w;
        float fx = 0.f, fy = 0.f, fz = 0.f, bx = 0.f, by = 0.f, bz = 0.f;
        for_each_neighbor<LIST, true, 1, true>(p, posk, posk, tbl, i, xi.x, xi.y, xi.z,
            [&](int, float4 pj, float4, float dx, float dy, float dz, float d2) {
                float s = (kri + pj.w) * pair_gradf(c, d2);
                fx = fmaf(s, dx, fx); fy = fmaf(s, dy, fy); fz = fmaf(s, dz, fz);
            },
            [&](int, float4 pk, float dx, float dy, float dz, float d2) {
                float s = pk.w * pair_gradf(c, d2);
                bx = fmaf(s, dx, bx); by = fmaf(s, dy, by); bz = fmaf(s, dz, bz);
            });
        float4 v = pv[i].v;
        const float dt = step_dt(c);
        if (TAIL == TAIL_WCSPH && t.add_gravity) {              // A10: v + dt g first, then the pressure term
            v.x = fmaf(dt, c.gx, v.x); v.y = fmaf(dt, c.gy, v.y); v.z = fmaf(dt, c.gz, v.z);
        }
        float k = dt * c.grad_c;
        v.x -= k * fmaf(c.m, fx, kri * bx);
        v.y -= k * fmaf(c.m, fy, kri * by);
        v.z -= k * fmaf(c.m, fz, kri * bz);
        if (TAIL == TAIL_DIV) {
            if (last && t.add_gravity) {
                v.x = fmaf(dt, c.gx, v.x); v.y = fmaf(dt, c.gy, v.y); v.z = fmaf(dt, c.gz, v.z);
            }
            v.w = t.rho[i];       // no other thread reads the records during a C-pass (it gathers posk)
            pv[i].v = v;
        } else {
            pv[i].v = v;
            if (last) {
                float4 x;
                x.x = fmaf(dt, v.x, xi.x); x.y = fmaf(dt, v.y, xi.y); x.z = fmaf(dt, v.z, xi.z);
                // the fourth lanes of the persistent store carry the warm-start totals through the next sort (R27)
                x.w = t.ksum_d != nullptr ? t.ksum_d[i] : 0.f;
                t.pos_out[i] = x;
                t.vel_out[i] = make_float4(v.x, v.y, v.z, t.ksum_v != nullptr ? t.ksum_v[i] : 0.f);
                t.id_out[i] = t.id[i];
                v2 = fmaf(v.x, v.x, fmaf(v.y, v.y, v.z * v.z));
                bad = !(isfinite(x.x) && isfinite(x.y) && isfinite(x.z) && isfinite(v2));
                if (bad) v2 = 0.f;
            }
        }
    }
    if (TAIL != TAIL_DIV && last) {
        v2 = warp_max(v2);
        unsigned b = __ballot_sync(0xffffffffu, bad);
        if ((threadIdx.x & 31) == 0) {
            unsigned vb = __float_as_uint(sqrtf(v2));           // non-negative floats order like their bits
            if (vb > *(volatile unsigned *)t.vmax_bits) atomicMax(t.vmax_bits, vb);   // guarded: same-address atomics serialise
            if (b) atomicAdd(t.nan_count, __popc(b));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// A6, Alg. 1 l.1-2: v* = v + dt (g + a_visc).
// mode 0 / 2: gravity only -- folded into the last C-pass of the divergence solve (TAIL_DIV above).

// mode 1: explicit viscosity, Eq. 15 (R4, R16, R22):
//   a_i = nu 2(d+2) sum_j (m / rho_j) (v_ij.x_ij) / (|x_ij|^2 + 0.01 h^2) gradW_ij, fluid-fluid only.
// rho_j is pv[j].v.w; CLAMP = true (WCSPH, R17) uses rho~_j = max(rho_j, rho0).  Reads the records vin,
// writes the records vout != vin (position copied).
template <bool LIST, bool CLAMP>
__global__ void __launch_bounds__(kBlock)
k_explicit_viscosity(PassCtx p, const PV *__restrict__ vin, PV *__restrict__ vout)
{
    __shared__ int tbl[LIST ? kRows * kBlock : 1];
    const SimConst &c = p.c;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.nf) return;
    float4 xi, vi;
    ldg256(reinterpret_cast<const float4 *>(vin + i), xi, vi);
    float ax = 0.f, ay = 0.f, az = 0.f;
    for_each_neighbor<LIST, false, 3, false>(p, reinterpret_cast<const float4 *>(vin), nullptr, tbl, i, xi.x, xi.y, xi.z,
        [&](int, float4, float4 vj, float dx, float dy, float dz, float d2) {
            float dv = fmaf(vi.x - vj.x, dx, fmaf(vi.y - vj.y, dy, (vi.z - vj.z) * dz));
            float rj = CLAMP ? fmaxf(vj.w, c.rho0) : vj.w;
            float s = pair_gradf(c, d2) * dv / ((d2 + c.visc_eps) * rj);
            ax = fmaf(s, dx, ax); ay = fmaf(s, dy, ay); az = fmaf(s, dz, az);
        },
        [&](int, float4, float, float, float, float) {});
    const float dt = step_dt(c);
    float k = dt * c.nu * 10.0f * c.m * c.grad_c;
    vi.x += fmaf(dt, c.gx, k * ax);
    vi.y += fmaf(dt, c.gy, k * ay);
    vi.z += fmaf(dt, c.gz, k * az);
    vout[i].x = xi;
    vout[i].v = vi;
}

// ---------------------------------------------------------------------------------------------
// A11: implicit viscosity (Eq. 16-19; R4, R21, R23), matrix-free CG on
// (I - dt A) v* = v~ with
//   (A u)_i = 2(d+2) sum_j mu m / (rho_i rho_j) (u_ij.x_ij) / (|x_ij|^2 + 0.01 h^2) gradW_ij.
// Vectors are float4 with rho in .w; the two that are gathered -- the start vector b = v~ and the search
// direction p -- live in 32-byte {x | vector} records (one 256-bit gather per neighbour).  out_i = u_i - dt (A u)_i when RESIDUAL0 = false;
// RESIDUAL0 = true is the start-up r0 = b - (I - dt A) b = dt A b (x0 = b = v~), which also seeds
// the search direction and reduces |b|^2, |r0|^2.
template <bool LIST, bool RESIDUAL0>
__global__ void __launch_bounds__(kBlock)
k_cg_apply(PassCtx p, const float4 *__restrict__ u /* PV records: velocities (RESIDUAL0) or search direction */,
           float4 *__restrict__ out, PV *__restrict__ out2, float *__restrict__ partial, float *__restrict__ partial2)
{
    __shared__ float red[kBlock / 32];
    __shared__ int tbl[LIST ? kRows * kBlock : 1];
    const SimConst &c = p.c;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float t1 = 0.f, t2 = 0.f;
    if (i < c.nf) {
        float4 xi = p.pos[i];
        float4 ui = u[2 * i + 1];
        float ax = 0.f, ay = 0.f, az = 0.f;
        for_each_neighbor<LIST, false, 3, false>(p, u, nullptr, tbl, i, xi.x, xi.y, xi.z,
            [&](int, float4, float4 uj, float dx, float dy, float dz, float d2) {
                float du = fmaf(ui.x - uj.x, dx, fmaf(ui.y - uj.y, dy, (ui.z - uj.z) * dz));
                float s = pair_gradf(c, d2) * du / ((d2 + c.visc_eps) * uj.w);
                ax = fmaf(s, dx, ax); ay = fmaf(s, dy, ay); az = fmaf(s, dz, az);
            },
            [&](int, float4, float, float, float, float) {});
        float k = step_dt(c) * 10.0f * c.mu * c.m * c.grad_c / ui.w;   // dt * 2(d+2) mu m / rho_i
        float Ax = k * ax, Ay = k * ay, Az = k * az;               // dt (A u)_i
        if (RESIDUAL0) {
            float4 r = make_float4(Ax, Ay, Az, ui.w);
            out[i] = r;                                            // r0
            out2[i].x = xi; out2[i].v = r;                         // p0 = r0 (a record: the next applies gather it)
            t1 = fmaf(ui.x, ui.x, fmaf(ui.y, ui.y, ui.z * ui.z));  // |b|^2
            t2 = fmaf(Ax, Ax, fmaf(Ay, Ay, Az * Az));              // |r0|^2
        } else {
            float ox = ui.x - Ax, oy = ui.y - Ay, oz = ui.z - Az;  // (I - dt A) p
            out[i] = make_float4(ox, oy, oz, ui.w);
            t1 = fmaf(ui.x, ox, fmaf(ui.y, oy, ui.z * oz));        // p.Ap
        }
    }
    float s1 = block_sum(t1, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = s1;
    if (RESIDUAL0) {
        float s2 = block_sum(t2, red);
        if (threadIdx.x == 0) partial2[blockIdx.x] = s2;
    }
}

// x += a p;  r -= a Ap;  partial |r|^2
__global__ void __launch_bounds__(256)
k_cg_update(int n, const DevControl *__restrict__ ctl, const PV *__restrict__ pd,
            const float4 *__restrict__ Ap, PV *__restrict__ x, float4 *__restrict__ r,
            float *__restrict__ partial)
{
    __shared__ float red[8];
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float t = 0.f;
    if (i < n) {
        float a = (float)ctl->cg_alpha;
        float4 pv = pd[i].v, av = Ap[i], xv = x[i].v, rv = r[i];
        xv.x = fmaf(a, pv.x, xv.x); xv.y = fmaf(a, pv.y, xv.y); xv.z = fmaf(a, pv.z, xv.z);
        rv.x = fmaf(-a, av.x, rv.x); rv.y = fmaf(-a, av.y, rv.y); rv.z = fmaf(-a, av.z, rv.z);
        x[i].v = xv; r[i] = rv;
        t = fmaf(rv.x, rv.x, fmaf(rv.y, rv.y, rv.z * rv.z));
    }
    float s = block_sum(t, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// p = r + beta p
__global__ void __launch_bounds__(256)
k_cg_direction(int n, const DevControl *__restrict__ ctl, const float4 *__restrict__ r,
               PV *__restrict__ pd)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float b = (float)ctl->cg_beta;
    float4 rv = r[i], pv = pd[i].v;
    pv.x = fmaf(b, pv.x, rv.x); pv.y = fmaf(b, pv.y, rv.y); pv.z = fmaf(b, pv.z, rv.z);
    pd[i].v = pv;
}

// ---------------------------------------------------------------------------------------------
// A10: WCSPH equation of state (R17): rho~ = max(rho, rho0),
// p = k((rho~/rho0)^gamma - 1), evaluated as k expm1(gamma log1p(delta)), delta = (rho~ - rho0)/rho0,
// which keeps the small excess accurate in fp32.  posk.w = p / rho~^2; the record's fourth velocity lane
// receives rho (the viscosity sums gather rho_j from it).
__global__ void __launch_bounds__(256)
k_wcsph_eos(SimConst c, const float4 *__restrict__ pos, const float *__restrict__ rho_in, PV *__restrict__ pv,
            float4 *__restrict__ posk)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.nf) return;
    float4 x = pos[i];
    float rho = rho_in[i];
    pv[i].v.w = rho;
    float rt = fmaxf(rho, c.rho0);
    float delta = (rt - c.rho0) / c.rho0;
    float pr = c.wc_k * expm1f(c.wc_gamma * log1pf(delta));
    posk[i] = make_float4(x.x, x.y, x.z, pr / (rt * rt));
}

// PCISPH (reading R28), start of the pressure stage: the record's fourth velocity lane receives rho (the viscosity
// sums gather rho_j from it, every P-pass reads rho_i from it), the accumulated pressure restarts at 0, and
// v* = v + dt g (Alg. 1 l.1-2) unless the explicit-viscosity kernel, which adds gravity itself, follows.
__global__ void __launch_bounds__(256)
k_pci_begin(SimConst c, const float *__restrict__ rho, PV *__restrict__ pv, float *__restrict__ pacc, int add_gravity)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.nf) return;
    float4 v = pv[i].v;
    if (add_gravity) {
        const float dt = step_dt(c);
        v.x = fmaf(dt, c.gx, v.x); v.y = fmaf(dt, c.gy, v.y); v.z = fmaf(dt, c.gz, v.z);
    }
    v.w = rho[i];
    pv[i].v = v;
    pacc[i] = 0.f;
}

// A9 (symplectic Euler) is the tail of the last C-pass: see k_solver_c, TAIL_DENS / TAIL_WCSPH.

}  // namespace sph
