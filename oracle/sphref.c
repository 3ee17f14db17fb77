/*
 * sphref.c -- fp64 CPU ORACLE for the DFSPH particle pipeline of arxiv 2403.11156.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code
 * with the CUDA path under paper_2403_11156_b200/csrc and neither includes the other.
 *
 * It is a plain, slow, obviously-correct restatement of what the hot path computes:
 * every function cites the passage of /root/reference/PAPER.md (or the DESIGN.md
 * reading Rn, mirrored from SURVEY.md section 8(c.3)) that it follows.  Arithmetic is
 * fp64 except where the method itself fixes fp32: the neighbour predicate and the cell
 * coordinate are evaluated in emulated fp32 (readings R10, R11) so that neighbour sets
 * and cell offsets can be compared bit-exactly with the GPU.  Compile with
 * -ffp-contract=off so that only the explicit fmaf() calls fuse.
 *
 * Particles stay in their ORIGINAL id order here (no reordering); a cell list
 * (indices sorted by cell key) is the only acceleration structure, and the tests pin it
 * against an O(N^2) numpy brute force.  OpenMP parallelises over particles only; no
 * blocking, fusion or reordering beyond the definitions.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): kernel normalisation / continuity /
 * antisymmetry; brute-force neighbour sets; lattice rest density and alpha; two-particle
 * closed form; planar Akinci volumes; free fall; momentum invariants of both solvers;
 * fluid + rigid momentum exchange (Eq. 14); implicit-viscosity operator symmetry and CG
 * vs dense solve; explicit Laplacian of a quadratic field; rigid stand-in closed forms;
 * scale of the implicit-viscosity operator (tied to the Eq. 15 lattice constant); boundary
 * terms of D and U against a moving one-sample body (closed form, incl. the Eq. 14 reaction);
 * torque / angular response through total angular momentum of fluid + body.
 * Multi-step GPU-vs-oracle trajectories beyond a few steps: "parity unpinned" (chaotic),
 * only statistics are compared.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846

typedef struct SphRefParams {
    double particle_radius;     /* r */
    double support_radius;      /* h   PAPER.md:100,282 (support radius of W) */
    double rest_density;        /* rho0 PAPER.md:282 */
    double particle_mass;       /* 0 => rho0 (2r)^3, reading R3 */
    double dt;
    double gravity[3];
    double domain_min[3], domain_max[3];
    double tank_min[3], tank_max[3];
    int viscosity_mode;         /* 0 none, 1 explicit Eq.15, 2 implicit Eq.17-19 */
    double kinematic_viscosity; /* nu = mu / rho0 */
    double cg_rel_tol;
    int cg_max_iter;
    double eta_density;
    int min_iter_density, max_iter_density;
    double eta_divergence;
    int min_iter_divergence, max_iter_divergence;
    int enable_divergence_solve;
    int force_iterations;
    double wcsph_stiffness, wcsph_exponent;
    double cfl_factor;          /* lambda of reading R26; 0 => fixed dt */
    double dt_min;
    int warm_start;             /* reading R27: 1 => both DFSPH solves start from the stiffness applied in the last step */
    double warm_start_factor;   /* omega of reading R27 (0.5 in the cited source's public implementation) */
    int pcisph_min_iter, pcisph_max_iter;   /* reading R28 */
} SphRefParams;

typedef struct SphRefBody {
    int first_particle, n_particles, dynamic;
    double mass, inertia_body[3];
    double com[3], quat[4], lin_vel[3], ang_vel[3];
    double contact_radius;
} SphRefBody;

typedef struct SphRefStats {
    int it_v, it_d, cg_iters, oob_count;
    double err_v, err_rho, cg_residual, v_max;
    double dt_last, sim_time;   /* time step of the last step, simulated time so far */
} SphRefStats;

/* cell list over an arbitrary point set (reading R11) */
typedef struct CellList {
    int n, nx, ny, nz, ncells, oob;
    float o[3], inv_c;
    int *key;        /* [n] linear cell key of every point */
    int *cell_start; /* [ncells+1] */
    int *order;      /* [n] point indices sorted by (key, index) */
} CellList;

typedef struct SphRef {
    SphRefParams p;
    int nf, nb, nbodies;
    double m;            /* fluid particle mass */
    double *x, *v;       /* [3 nf] fluid position / velocity (id order) */
    double *bx, *bv;     /* [3 nb] boundary sample position / velocity */
    double *brest;       /* [3 nb] body-frame coordinates */
    double *psi;         /* [nb] Akinci volume-mass Psi, Eq. 11 */
    double *bforce;      /* [3 nb] reaction force on boundary samples, Eq. 14 */
    int *bbody;
    SphRefBody *bodies;
    double *rho, *alpha, *kappa, *kr; /* [nf] */
    double *ksum_v, *ksum_d; /* [nf] total stiffness applied by the divergence / density solve of the last step (R27) */
    double *kacc;            /* [nf] scratch: running total of the solve in progress */
    double pci_delta;        /* PCISPH scaling factor (R28), computed at creation */
    double *vstar;       /* scratch */
    CellList gf, gb;     /* fluid grid, boundary grid */
    int *nf_start, *nf_idx; /* CSR fluid neighbours of fluid i */
    int *nb_start, *nb_idx; /* CSR boundary neighbours of fluid i */
    int lists_valid;
    SphRefStats stats;
    double dt_max, forced_dt;   /* configured dt (upper bound of the CFL rule); > 0: dt imposed by the caller */
    double *cg_hist; int cg_hist_n;
} SphRef;

/* ------------------------------------------------------------------ kernel (reading R1) */

/* Cubic spline with support radius h, sigma = 8 / (pi h^3) in 3-D (reading R1: the paper
 * never prints W; BASELINE.json says cubic spline; h is the SUPPORT radius). */
double sphref_W(double rlen, double h)
{
    double sigma = 8.0 / (PI * h * h * h);
    double q = rlen / h;
    if (q <= 0.5) return sigma * (6.0 * (q * q * q - q * q) + 1.0);
    if (q <= 1.0) { double t = 1.0 - q; return sigma * 2.0 * t * t * t; }
    return 0.0;
}

/* grad_i W(x_i - x_j) for d = x_i - x_j; zero at zero distance (reading R2). */
void sphref_gradW(const double d[3], double h, double out[3])
{
    double rlen = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    out[0] = out[1] = out[2] = 0.0;
    if (rlen < 1e-9 * h) return;
    double sigma = 8.0 / (PI * h * h * h);
    double q = rlen / h, wp;
    if (q <= 0.5) wp = 6.0 * q * (3.0 * q - 2.0);
    else if (q <= 1.0) { double t = 1.0 - q; wp = -6.0 * t * t; }
    else return;
    double f = sigma / h * wp / rlen;
    out[0] = f * d[0]; out[1] = f * d[1]; out[2] = f * d[2];
}

/* ------------------------------------------------------------------ grid (readings R10, R11) */

/* fp32-emulated neighbour predicate, reading R10: strict d2 < h2 with
 * d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx)), all operands and operations in binary32. */
static int is_neighbor32(const float a[3], const float b[3], float h2)
{
    float dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
    float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    return d2 < h2;
}

static void celllist_free(CellList *g)
{
    free(g->key); free(g->cell_start); free(g->order);
    memset(g, 0, sizeof(*g));
}

/* Geometry, reading R11: cell edge c = h (1 + 2^-10) in fp32, origin = domain_min,
 * n_a = floor((max_a - o_a) * inv_c) + 1, inv_c = 1/c in fp32. */
static void celllist_geometry(CellList *g, const SphRefParams *p)
{
    float h = (float)p->support_radius;
    float c = h * 1.0009765625f;
    g->inv_c = 1.0f / c;
    int n[3];
    for (int a = 0; a < 3; ++a) {
        g->o[a] = (float)p->domain_min[a];
        float ext = (float)p->domain_max[a] - g->o[a];
        n[a] = (int)floorf(ext * g->inv_c) + 1;
        if (n[a] < 1) n[a] = 1;
    }
    g->nx = n[0]; g->ny = n[1]; g->nz = n[2];
    g->ncells = n[0] * n[1] * n[2];
}

/* cell coordinate of one point: (int)floorf((x - o) * inv_c), clamped; *oob counts clamps */
static void cell_of(const CellList *g, const float x[3], int c[3], int *oob)
{
    int n[3] = { g->nx, g->ny, g->nz };
    int clamped = 0;
    for (int a = 0; a < 3; ++a) {
        float t = (x[a] - g->o[a]) * g->inv_c;
        int ci;
        if (!(t == t)) { ci = 0; clamped = 1; }           /* NaN */
        else if (t < 0.0f) { ci = 0; clamped = 1; }
        else if (t >= (float)n[a]) { ci = n[a] - 1; clamped = 1; }
        else ci = (int)floorf(t);
        c[a] = ci;
    }
    if (oob && clamped) ++*oob;
}

/* Build: key per point, cell_start[k] = #points with key < k, order = stable sort by key. */
static void celllist_build(CellList *g, const SphRefParams *p, const double *x, int n)
{
    celllist_free(g);
    celllist_geometry(g, p);
    g->n = n;
    g->key = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
    g->order = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
    g->cell_start = (int *)calloc((size_t)g->ncells + 1, sizeof(int));
    g->oob = 0;
    for (int i = 0; i < n; ++i) {
        float xf[3] = { (float)x[3 * i], (float)x[3 * i + 1], (float)x[3 * i + 2] };
        int c[3];
        cell_of(g, xf, c, &g->oob);
        g->key[i] = c[0] + g->nx * (c[1] + g->ny * c[2]);
    }
    for (int i = 0; i < n; ++i) g->cell_start[g->key[i] + 1]++;
    for (int k = 0; k < g->ncells; ++k) g->cell_start[k + 1] += g->cell_start[k];
    int *cursor = (int *)malloc(sizeof(int) * (size_t)g->ncells);
    memcpy(cursor, g->cell_start, sizeof(int) * (size_t)g->ncells);
    for (int i = 0; i < n; ++i) g->order[cursor[g->key[i]]++] = i; /* ascending index within a cell */
    free(cursor);
}

/* Visit every point j of grid g (coordinates px, fp64 rounded to fp32) with
 * is_neighbor32(xq, x_j); the 27 cells around xq's (clamped) cell are scanned. */
typedef void (*visit_fn)(int j, void *ctx);
static void celllist_query(const CellList *g, const double *px, const float xq[3], float h2,
                           int skip, visit_fn fn, void *ctx)
{
    if (g->n == 0) return;
    int c[3];
    cell_of(g, xq, c, NULL);
    for (int dz = -1; dz <= 1; ++dz) {
        int cz = c[2] + dz; if (cz < 0 || cz >= g->nz) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            int cy = c[1] + dy; if (cy < 0 || cy >= g->ny) continue;
            for (int dx = -1; dx <= 1; ++dx) {
                int cx = c[0] + dx; if (cx < 0 || cx >= g->nx) continue;
                int k = cx + g->nx * (cy + g->ny * cz);
                for (int s = g->cell_start[k]; s < g->cell_start[k + 1]; ++s) {
                    int j = g->order[s];
                    if (j == skip) continue;
                    float xj[3] = { (float)px[3 * j], (float)px[3 * j + 1], (float)px[3 * j + 2] };
                    if (is_neighbor32(xq, xj, h2)) fn(j, ctx);
                }
            }
        }
    }
}

typedef struct { int *buf; int n, cap; } IntVec;
static void ivec_push(int j, void *ctx)
{
    IntVec *v = (IntVec *)ctx;
    if (v->n == v->cap) { v->cap = v->cap ? 2 * v->cap : 64; v->buf = (int *)realloc(v->buf, sizeof(int) * (size_t)v->cap); }
    v->buf[v->n++] = j;
}
static int cmp_int(const void *a, const void *b) { int x = *(const int *)a, y = *(const int *)b; return (x > y) - (x < y); }

/* Neighbour sets N(i) of every fluid particle (definition in SURVEY 8(c.1)): fluid
 * neighbours j != i and boundary neighbours k, each as a CSR list of ascending ids. */
static void build_neighbor_lists(SphRef *s)
{
    int nf = s->nf;
    float hf = (float)s->p.support_radius;
    float h2 = hf * hf;
    IntVec *vf = (IntVec *)calloc((size_t)(nf > 0 ? nf : 1), sizeof(IntVec));
    IntVec *vb = (IntVec *)calloc((size_t)(nf > 0 ? nf : 1), sizeof(IntVec));
#pragma omp parallel for schedule(dynamic, 256)
    for (int i = 0; i < nf; ++i) {
        float xi[3] = { (float)s->x[3 * i], (float)s->x[3 * i + 1], (float)s->x[3 * i + 2] };
        celllist_query(&s->gf, s->x, xi, h2, i, ivec_push, &vf[i]);
        celllist_query(&s->gb, s->bx, xi, h2, -1, ivec_push, &vb[i]);
        qsort(vf[i].buf, (size_t)vf[i].n, sizeof(int), cmp_int);
        qsort(vb[i].buf, (size_t)vb[i].n, sizeof(int), cmp_int);
    }
    free(s->nf_start); free(s->nf_idx); free(s->nb_start); free(s->nb_idx);
    s->nf_start = (int *)calloc((size_t)nf + 1, sizeof(int));
    s->nb_start = (int *)calloc((size_t)nf + 1, sizeof(int));
    for (int i = 0; i < nf; ++i) { s->nf_start[i + 1] = s->nf_start[i] + vf[i].n; s->nb_start[i + 1] = s->nb_start[i] + vb[i].n; }
    s->nf_idx = (int *)malloc(sizeof(int) * (size_t)(s->nf_start[nf] + 1));
    s->nb_idx = (int *)malloc(sizeof(int) * (size_t)(s->nb_start[nf] + 1));
    for (int i = 0; i < nf; ++i) {
        memcpy(s->nf_idx + s->nf_start[i], vf[i].buf, sizeof(int) * (size_t)vf[i].n);
        memcpy(s->nb_idx + s->nb_start[i], vb[i].buf, sizeof(int) * (size_t)vb[i].n);
        free(vf[i].buf); free(vb[i].buf);
    }
    free(vf); free(vb);
    s->lists_valid = 1;
}

/* Step 1 of (c.2): grid on the current positions (fluid; boundary incl. dynamic samples). */
int sphref_build_grid(SphRef *s)
{
    celllist_build(&s->gf, &s->p, s->x, s->nf);
    celllist_build(&s->gb, &s->p, s->bx, s->nb);
    s->stats.oob_count = s->gf.oob;
    build_neighbor_lists(s);
    return 0;
}

/* ------------------------------------------------------------------ small vector helpers */
static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static void cross3(const double a[3], const double b[3], double o[3])
{
    o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}
static void quat_to_R(const double q[4], double R[9])
{
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
    R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
    R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

/* ------------------------------------------------------------------ Akinci volumes */

typedef struct { const SphRef *s; int k; double sum; } PsiCtx;
static void psi_visit(int j, void *ctx)
{
    PsiCtx *c = (PsiCtx *)ctx;
    const SphRef *s = c->s;
    if (s->bbody[j] != s->bbody[c->k]) return;           /* same body only, reading R9 */
    double d[3] = { s->bx[3 * c->k] - s->bx[3 * j], s->bx[3 * c->k + 1] - s->bx[3 * j + 1], s->bx[3 * c->k + 2] - s->bx[3 * j + 2] };
    c->sum += sphref_W(sqrt(dot3(d, d)), s->p.support_radius);
}

/* Eq. 11: Psi_k = rho0 / sum_k' W_kk', k' over boundary samples of the
 * same body INCLUDING k itself, once at creation (reading R9). */
static void compute_psi(SphRef *s)
{
    float hf = (float)s->p.support_radius, h2 = hf * hf;
    celllist_build(&s->gb, &s->p, s->bx, s->nb);
#pragma omp parallel for schedule(dynamic, 256)
    for (int k = 0; k < s->nb; ++k) {
        PsiCtx c = { s, k, sphref_W(0.0, s->p.support_radius) };
        float xk[3] = { (float)s->bx[3 * k], (float)s->bx[3 * k + 1], (float)s->bx[3 * k + 2] };
        celllist_query(&s->gb, s->bx, xk, h2, k, psi_visit, &c);
        s->psi[k] = s->p.rest_density / c.sum;
    }
}

/* ------------------------------------------------------------------ create / destroy */

SphRef *sphref_create(const SphRefParams *p, int nf, const float *fpos, const float *fvel,
                      int nb, const float *bpos, const int *bbody, int nbodies, const SphRefBody *bodies)
{
    SphRef *s = (SphRef *)calloc(1, sizeof(SphRef));
    s->p = *p;
    s->dt_max = p->dt; s->forced_dt = 0.0;
    s->nf = nf; s->nb = nb; s->nbodies = nbodies;
    double d = 2.0 * p->particle_radius;
    s->m = p->particle_mass > 0.0 ? p->particle_mass : p->rest_density * d * d * d; /* R3 */
    size_t f3 = (size_t)(nf > 0 ? nf : 1) * 3, b3 = (size_t)(nb > 0 ? nb : 1) * 3;
    s->x = (double *)calloc(f3, sizeof(double)); s->v = (double *)calloc(f3, sizeof(double));
    s->vstar = (double *)calloc(f3, sizeof(double));
    s->rho = (double *)calloc(f3, sizeof(double)); s->alpha = (double *)calloc(f3, sizeof(double));
    s->kappa = (double *)calloc(f3, sizeof(double)); s->kr = (double *)calloc(f3, sizeof(double));
    s->ksum_v = (double *)calloc(f3, sizeof(double)); s->ksum_d = (double *)calloc(f3, sizeof(double));
    s->kacc = (double *)calloc(f3, sizeof(double));
    s->bx = (double *)calloc(b3, sizeof(double)); s->bv = (double *)calloc(b3, sizeof(double));
    s->brest = (double *)calloc(b3, sizeof(double)); s->bforce = (double *)calloc(b3, sizeof(double));
    s->psi = (double *)calloc(b3, sizeof(double));
    s->bbody = (int *)calloc(b3, sizeof(int));
    s->bodies = (SphRefBody *)calloc((size_t)(nbodies > 0 ? nbodies : 1), sizeof(SphRefBody));
    s->cg_hist = (double *)calloc((size_t)(p->cg_max_iter > 0 ? p->cg_max_iter : 1) + 2, sizeof(double));
    for (int i = 0; i < 3 * nf; ++i) { s->x[i] = fpos[i]; s->v[i] = fvel[i]; }
    for (int i = 0; i < 3 * nb; ++i) s->bx[i] = bpos[i];
    for (int k = 0; k < nb; ++k) s->bbody[k] = bbody[k];
    for (int b = 0; b < nbodies; ++b) s->bodies[b] = bodies[b];
    /* body-frame coordinates and initial sample velocities of dynamic bodies */
    for (int k = 0; k < nb; ++k) {
        const SphRefBody *B = &s->bodies[s->bbody[k]];
        double R[9]; quat_to_R(B->quat, R);
        double dlt[3] = { s->bx[3 * k] - B->com[0], s->bx[3 * k + 1] - B->com[1], s->bx[3 * k + 2] - B->com[2] };
        for (int a = 0; a < 3; ++a) s->brest[3 * k + a] = R[0 + a] * dlt[0] + R[3 + a] * dlt[1] + R[6 + a] * dlt[2]; /* R^T d */
        if (B->dynamic) {
            double w[3]; cross3(B->ang_vel, dlt, w);
            for (int a = 0; a < 3; ++a) s->bv[3 * k + a] = B->lin_vel[a] + w[a];
        }
    }
    compute_psi(s);
    return s;
}

void sphref_destroy(SphRef *s)
{
    if (!s) return;
    free(s->x); free(s->v); free(s->vstar); free(s->rho); free(s->alpha); free(s->kappa); free(s->kr);
    free(s->ksum_v); free(s->ksum_d); free(s->kacc);
    free(s->bx); free(s->bv); free(s->brest); free(s->bforce); free(s->psi); free(s->bbody); free(s->bodies);
    free(s->nf_start); free(s->nf_idx); free(s->nb_start); free(s->nb_idx); free(s->cg_hist);
    celllist_free(&s->gf); celllist_free(&s->gb);
    free(s);
}

/* ------------------------------------------------------------------ sums of (c.1) */

/* Density, Eq. 4 + Eq. 12, self term included (R2):
 * rho_i = m W(0) + sum_j m W_ij + sum_k Psi_k W_ik.
 * Alpha (reading R5, from cited [5]): S_i = sum_j m gradW_ij + sum_k Psi_k gradW_ik,
 * T_i = sum_j |m gradW_ij|^2 (fluid only), alpha_i = rho_i / (|S_i|^2 + T_i), 0 if the
 * denominator is <= 1e-6 (R7). */
int sphref_compute_density_alpha(SphRef *s)
{
    if (!s->lists_valid) return -1;
    double h = s->p.support_radius, m = s->m;
#pragma omp parallel for schedule(dynamic, 256)
    for (int i = 0; i < s->nf; ++i) {
        const double *xi = s->x + 3 * i;
        double rho = m * sphref_W(0.0, h), S[3] = { 0, 0, 0 }, T = 0.0, g[3];
        for (int t = s->nf_start[i]; t < s->nf_start[i + 1]; ++t) {
            int j = s->nf_idx[t];
            double d[3] = { xi[0] - s->x[3 * j], xi[1] - s->x[3 * j + 1], xi[2] - s->x[3 * j + 2] };
            rho += m * sphref_W(sqrt(dot3(d, d)), h);
            sphref_gradW(d, h, g);
            for (int a = 0; a < 3; ++a) S[a] += m * g[a];
            T += m * m * dot3(g, g);
        }
        for (int t = s->nb_start[i]; t < s->nb_start[i + 1]; ++t) {
            int k = s->nb_idx[t];
            double d[3] = { xi[0] - s->bx[3 * k], xi[1] - s->bx[3 * k + 1], xi[2] - s->bx[3 * k + 2] };
            rho += s->psi[k] * sphref_W(sqrt(dot3(d, d)), h);
            sphref_gradW(d, h, g);
            for (int a = 0; a < 3; ++a) S[a] += s->psi[k] * g[a];
        }
        double den = dot3(S, S) + T;
        s->rho[i] = rho;
        s->alpha[i] = den > 1e-6 ? rho / den : 0.0;
    }
    return 0;
}

/* Density rate (Eq. 6 times rho):
 * D_i[v] = sum_j m (v_i - v_j).gradW_ij + sum_k Psi_k (v_i - v_k).gradW_ik. */
static double density_rate(const SphRef *s, const double *vel, int i)
{
    double h = s->p.support_radius, m = s->m, D = 0.0, g[3];
    const double *xi = s->x + 3 * i, *vi = vel + 3 * i;
    for (int t = s->nf_start[i]; t < s->nf_start[i + 1]; ++t) {
        int j = s->nf_idx[t];
        double d[3] = { xi[0] - s->x[3 * j], xi[1] - s->x[3 * j + 1], xi[2] - s->x[3 * j + 2] };
        double dv[3] = { vi[0] - vel[3 * j], vi[1] - vel[3 * j + 1], vi[2] - vel[3 * j + 2] };
        sphref_gradW(d, h, g);
        D += m * dot3(dv, g);
    }
    for (int t = s->nb_start[i]; t < s->nb_start[i + 1]; ++t) {
        int k = s->nb_idx[t];
        double d[3] = { xi[0] - s->bx[3 * k], xi[1] - s->bx[3 * k + 1], xi[2] - s->bx[3 * k + 2] };
        double dv[3] = { vi[0] - s->bv[3 * k], vi[1] - s->bv[3 * k + 1], vi[2] - s->bv[3 * k + 2] };
        sphref_gradW(d, h, g);
        D += s->psi[k] * dot3(dv, g);
    }
    return D;
}

/* Pressure-like velocity update (Eq. 7 + Eq. 13 with p/rho^2 == kappa/rho):
 * U_i = sum_j m (kr_i + kr_j) gradW_ij + sum_k Psi_k kr_i gradW_ik;  v_i <- v_i - dt U_i.
 * Reaction on boundary sample k (Eq. 14): F_k += m Psi_k kr_i gradW_ik. */
static void apply_pressure_update(SphRef *s, double *vel)
{
    double h = s->p.support_radius, m = s->m, dt = s->p.dt;
    const double *kr = s->kr;
#pragma omp parallel for schedule(dynamic, 256)
    for (int i = 0; i < s->nf; ++i) {
        const double *xi = s->x + 3 * i;
        double U[3] = { 0, 0, 0 }, g[3];
        for (int t = s->nf_start[i]; t < s->nf_start[i + 1]; ++t) {
            int j = s->nf_idx[t];
            double d[3] = { xi[0] - s->x[3 * j], xi[1] - s->x[3 * j + 1], xi[2] - s->x[3 * j + 2] };
            sphref_gradW(d, h, g);
            double c = m * (kr[i] + kr[j]);
            for (int a = 0; a < 3; ++a) U[a] += c * g[a];
        }
        for (int t = s->nb_start[i]; t < s->nb_start[i + 1]; ++t) {
            int k = s->nb_idx[t];
            double d[3] = { xi[0] - s->bx[3 * k], xi[1] - s->bx[3 * k + 1], xi[2] - s->bx[3 * k + 2] };
            sphref_gradW(d, h, g);
            double c = s->psi[k] * kr[i];
            for (int a = 0; a < 3; ++a) U[a] += c * g[a];
        }
        for (int a = 0; a < 3; ++a) s->vstar[3 * i + a] = vel[3 * i + a] - dt * U[a];
    }
    /* Eq. 14 reaction, serial scatter (only samples of dynamic bodies keep it) */
    for (int i = 0; i < s->nf; ++i) {
        if (kr[i] == 0.0) continue;
        const double *xi = s->x + 3 * i;
        double g[3];
        for (int t = s->nb_start[i]; t < s->nb_start[i + 1]; ++t) {
            int k = s->nb_idx[t];
            if (!s->bodies[s->bbody[k]].dynamic) continue;
            double d[3] = { xi[0] - s->bx[3 * k], xi[1] - s->bx[3 * k + 1], xi[2] - s->bx[3 * k + 2] };
            sphref_gradW(d, h, g);
            double c = m * s->psi[k] * kr[i];
            for (int a = 0; a < 3; ++a) s->bforce[3 * k + a] += c * g[a];
        }
    }
    memcpy(vel, s->vstar, sizeof(double) * 3 * (size_t)s->nf);
}

/* Warm start (reading R27; PAPER.md:49, 170 only say that the PPE solvers need fewer refinement rounds / allow larger
 * steps -- the technique is the one of the cited DFSPH source [5]): before a solve's loop, the total stiffness K_i that
 * the same solve applied in the LAST step, scaled by omega, is applied once through the ordinary pressure update,
 *   v <- v - dt U[omega K / rho]   (rho, gradW of the CURRENT step),
 * and the solve's running total starts from it: K_i(new) = omega K_i(old) + sum over this step's iterations of kappa_i.
 * Returns with s->kacc initialised (zeros when warm start is off). */
static void warm_start_apply(SphRef *s, double *vel, const double *ksum_prev)
{
    const SphRefParams *p = &s->p;
    for (int i = 0; i < s->nf; ++i) s->kacc[i] = 0.0;
    if (!p->warm_start) return;
    for (int i = 0; i < s->nf; ++i) {
        s->kappa[i] = p->warm_start_factor * ksum_prev[i];
        s->kr[i] = s->kappa[i] / s->rho[i];
        s->kacc[i] = s->kappa[i];
    }
    apply_pressure_update(s, vel);
}

/* Divergence-free solve, (c.2) step 3 (Eq. 10 source term PAPER.md:156; loop Alg. 2
 * PAPER.md:160-168; details from cited [5], readings R5, R14, R15):
 * do { P: R_i = max(D_i[v], 0); err_v = (dt/rho0) mean R_i; kappa^v_i = alpha_i R_i / dt;
 *      C: v <- v - dt U[kappa^v / rho]; l++ }
 * while ((err_v > eta_v || l < min_v) && l < max_v).  forced >= 0: exactly that many. */
int sphref_divergence_solve(SphRef *s, double *vel, int forced)
{
    const SphRefParams *p = &s->p;
    int l = 0;
    double err = 0.0;
    if (forced == 0) { s->stats.it_v = 0; s->stats.err_v = 0.0; for (int i = 0; i < s->nf; ++i) s->ksum_v[i] = 0.0; return 0; }
    warm_start_apply(s, vel, s->ksum_v);
    for (;;) {
        double sum = 0.0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : sum)
        for (int i = 0; i < s->nf; ++i) {
            double R = density_rate(s, vel, i);
            if (R < 0.0) R = 0.0;
            sum += R;
            s->kappa[i] = s->alpha[i] * R / p->dt;
            s->kr[i] = s->kappa[i] / s->rho[i];
            s->kacc[i] += s->kappa[i];
        }
        err = s->nf > 0 ? p->dt / p->rest_density * sum / s->nf : 0.0;
        apply_pressure_update(s, vel);
        ++l;
        if (forced > 0) { if (l >= forced) break; }
        else if (!((err > p->eta_divergence || l < p->min_iter_divergence) && l < p->max_iter_divergence)) break;
    }
    s->stats.it_v = l; s->stats.err_v = err;
    memcpy(s->ksum_v, s->kacc, sizeof(double) * (size_t)s->nf);
    return l;
}

/* Constant-density solve, (c.2) step 5 (Eq. 8-9; Alg. 2; [5]):
 * do { P: E_i = max(rho_i + dt D_i[v*], rho0) - rho0; err = mean E_i / rho0;
 *      kappa_i = alpha_i E_i / dt^2;  C: v* <- v* - dt U[kappa / rho]; l++ }
 * while ((err > eta || l < min) && l < max). */
int sphref_density_solve(SphRef *s, double *vel, int forced)
{
    const SphRefParams *p = &s->p;
    int l = 0;
    double err = 0.0;
    if (forced == 0) { s->stats.it_d = 0; s->stats.err_rho = 0.0; for (int i = 0; i < s->nf; ++i) s->ksum_d[i] = 0.0; return 0; }
    warm_start_apply(s, vel, s->ksum_d);
    for (;;) {
        double sum = 0.0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : sum)
        for (int i = 0; i < s->nf; ++i) {
            double rs = s->rho[i] + p->dt * density_rate(s, vel, i);
            double E = (rs > p->rest_density ? rs : p->rest_density) - p->rest_density;
            sum += E;
            s->kappa[i] = s->alpha[i] * E / (p->dt * p->dt);
            s->kr[i] = s->kappa[i] / s->rho[i];
            s->kacc[i] += s->kappa[i];
        }
        err = s->nf > 0 ? sum / s->nf / p->rest_density : 0.0;
        apply_pressure_update(s, vel);
        ++l;
        if (forced > 0) { if (l >= forced) break; }
        else if (!((err > p->eta_density || l < p->min_iter_density) && l < p->max_iter_density)) break;
    }
    s->stats.it_d = l; s->stats.err_rho = err;
    memcpy(s->ksum_d, s->kacc, sizeof(double) * (size_t)s->nf);
    return l;
}

/* ------------------------------------------------------------------ PCISPH (reading R28) */

/* PCISPH scaling factor of the cited source [25] (PAPER.md:158, 264 name the method; the paper prints none of its
 * equations -- reading R28):  delta = 1 / (beta (|sum_j gradW_ij|^2 + sum_j |gradW_ij|^2)),  beta = 2 (dt m / rho0)^2,
 * evaluated ONCE for a prototype particle with a filled neighbourhood: the sites of a simple-cubic lattice of spacing 2r
 * strictly inside the support radius h (the first sum vanishes there by symmetry, it is kept for the definition's sake).
 * Returned WITHOUT the dt^-2 factor:  k = rho0^2 / (2 m^2 (...)),  delta = k / dt^2  (dt may change per step, R26). */
double sphref_pcisph_k(const SphRef *s)
{
    double h = s->p.support_radius, sp = 2.0 * s->p.particle_radius, m = s->m;
    int n = (int)ceil(h / sp) + 1;
    double S[3] = { 0, 0, 0 }, T = 0.0, g[3];
    for (int a = -n; a <= n; ++a) for (int b = -n; b <= n; ++b) for (int c = -n; c <= n; ++c) {
        if (a == 0 && b == 0 && c == 0) continue;
        double d[3] = { -a * sp, -b * sp, -c * sp };            /* x_i - x_j, particle i at the origin */
        if (dot3(d, d) >= h * h) continue;
        sphref_gradW(d, h, g);
        for (int q = 0; q < 3; ++q) S[q] += g[q];
        T += dot3(g, g);
    }
    return s->p.rest_density * s->p.rest_density / (2.0 * m * m * (dot3(S, S) + T));
}

/* PCISPH pressure loop in the form of Alg. 2 with the density-based source term, Eq. 8, and the
 * prediction of Eq. 9: starting from p = 0 and the velocities v* after the non-pressure forces,
 *   do { P: rho*_i = rho_i + dt D_i[v*]                                (Eq. 9 times ... with D of (c.1))
 *           err = mean_i max(rho*_i - rho0, 0) / rho0                   (same measure as the DFSPH density solve, R6)
 *           p_i(new) = max(p_i + delta (rho*_i - rho0), 0)              ([25]: global delta, pressure clamped at zero)
 *        C: v* <- v* - dt U[(p_i(new) - p_i) / rho_i^2]                 (Eq. 7 + 13; the pressure force is linear in p,
 *                                                                        so applying the increment equals recomputing
 *                                                                        the force from the accumulated pressure)
 *           l++ }
 * while ((err > eta_density || l < pcisph_min_iter) && l < pcisph_max_iter)   ([25] asks for at least 3 iterations).
 * forced >= 0: exactly that many iterations.  s->kappa holds the accumulated pressure on return. */
int sphref_pcisph_solve(SphRef *s, double *vel, int forced)
{
    const SphRefParams *p = &s->p;
    int l = 0;
    double err = 0.0;
    double delta = sphref_pcisph_k(s) / (p->dt * p->dt);
    int mn = p->pcisph_min_iter > 0 ? p->pcisph_min_iter : 3, mx = p->pcisph_max_iter > 0 ? p->pcisph_max_iter : 100;
    for (int i = 0; i < s->nf; ++i) s->kappa[i] = 0.0;
    if (forced == 0) { s->stats.it_d = 0; s->stats.err_rho = 0.0; return 0; }
    for (;;) {
        double sum = 0.0;
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : sum)
        for (int i = 0; i < s->nf; ++i) {
            double rs = s->rho[i] + p->dt * density_rate(s, vel, i);
            double e = rs - p->rest_density;
            sum += e > 0.0 ? e : 0.0;
            double pn = s->kappa[i] + delta * e;
            if (pn < 0.0) pn = 0.0;
            s->kr[i] = (pn - s->kappa[i]) / (s->rho[i] * s->rho[i]);
            s->kappa[i] = pn;
        }
        err = s->nf > 0 ? sum / s->nf / p->rest_density : 0.0;
        apply_pressure_update(s, vel);
        ++l;
        if (forced > 0) { if (l >= forced) break; }
        else if (!((err > p->eta_density || l < mn) && l < mx)) break;
    }
    s->stats.it_d = l; s->stats.err_rho = err;
    return l;
}

/* ------------------------------------------------------------------ viscosity */

/* Shared pair factor of Eq. 15 / Eq. 19: (v_ij . x_ij) / (|x_ij|^2 + 0.01 h^2) gradW_ij
 * (denominator per reading R4). */
static void visc_pair(const double d[3], const double dv[3], double h, double out[3])
{
    double g[3];
    sphref_gradW(d, h, g);
    double f = dot3(dv, d) / (dot3(d, d) + 0.01 * h * h);
    out[0] = f * g[0]; out[1] = f * g[1]; out[2] = f * g[2];
}

/* Explicit viscosity, Eq. 15, reading R16: a_i = nu * 2(d+2) sum_j (m/rho_j)
 * (v_ij.x_ij)/(|x_ij|^2 + 0.01h^2) gradW_ij, fluid-fluid only (R22), d = 3.
 * rho_for_visc: the densities used for m/rho_j (rho for DFSPH, clamped rho~ for WCSPH). */
void sphref_explicit_viscosity_accel(const SphRef *s, const double *vel, const double *rho_for_visc, double *acc)
{
    double h = s->p.support_radius, m = s->m, nu = s->p.kinematic_viscosity;
#pragma omp parallel for schedule(dynamic, 256)
    for (int i = 0; i < s->nf; ++i) {
        double a[3] = { 0, 0, 0 }, t3[3];
        for (int t = s->nf_start[i]; t < s->nf_start[i + 1]; ++t) {
            int j = s->nf_idx[t];
            double d[3] = { s->x[3 * i] - s->x[3 * j], s->x[3 * i + 1] - s->x[3 * j + 1], s->x[3 * i + 2] - s->x[3 * j + 2] };
            double dv[3] = { vel[3 * i] - vel[3 * j], vel[3 * i + 1] - vel[3 * j + 1], vel[3 * i + 2] - vel[3 * j + 2] };
            visc_pair(d, dv, h, t3);
            double c = m / rho_for_visc[j];
            for (int q = 0; q < 3; ++q) a[q] += c * t3[q];
        }
        for (int q = 0; q < 3; ++q) acc[3 * i + q] = nu * 10.0 * a[q];
    }
}

/* Implicit-viscosity operator, Eq. 19 matrix-free (readings R4, R21):
 * (A u)_i = 2(d+2) sum_j mu mbar_ij / (rho_i rho_j) (u_ij.x_ij)/(|x_ij|^2 + 0.01h^2) gradW_ij,
 * mu = nu rho0, mbar_ij = m. */
void sphref_viscosity_operator(const SphRef *s, const double *u, double *Au)
{
    double h = s->p.support_radius, m = s->m, mu = s->p.kinematic_viscosity * s->p.rest_density;
#pragma omp parallel for schedule(dynamic, 256)
    for (int i = 0; i < s->nf; ++i) {
        double a[3] = { 0, 0, 0 }, t3[3];
        for (int t = s->nf_start[i]; t < s->nf_start[i + 1]; ++t) {
            int j = s->nf_idx[t];
            double d[3] = { s->x[3 * i] - s->x[3 * j], s->x[3 * i + 1] - s->x[3 * j + 1], s->x[3 * i + 2] - s->x[3 * j + 2] };
            double du[3] = { u[3 * i] - u[3 * j], u[3 * i + 1] - u[3 * j + 1], u[3 * i + 2] - u[3 * j + 2] };
            visc_pair(d, du, h, t3);
            double c = mu * m / (s->rho[i] * s->rho[j]);
            for (int q = 0; q < 3; ++q) a[q] += c * t3[q];
        }
        for (int q = 0; q < 3; ++q) Au[3 * i + q] = 10.0 * a[q];
    }
}

/* Solve (I - dt A) v* = v~ (Eq. 18) by plain CG (reading R23):
 * x0 = v~, stop when |r|_2 <= tol |v~|_2 or cg_max_iter; forced >= 0: exactly that many
 * iterations.  x holds v~ on entry and v* on exit.  Returns iterations done. */
int sphref_implicit_viscosity_solve(SphRef *s, double *xv, int forced)
{
    int n3 = 3 * s->nf;
    double dt = s->p.dt;
    double *b = (double *)malloc(sizeof(double) * (size_t)(n3 + 1));
    double *r = (double *)malloc(sizeof(double) * (size_t)(n3 + 1));
    double *pd = (double *)malloc(sizeof(double) * (size_t)(n3 + 1));
    double *Ap = (double *)malloc(sizeof(double) * (size_t)(n3 + 1));
    memcpy(b, xv, sizeof(double) * (size_t)n3);
    double bb = 0.0;
    for (int i = 0; i < n3; ++i) bb += b[i] * b[i];
    sphref_viscosity_operator(s, xv, Ap);
    double rr = 0.0;
    for (int i = 0; i < n3; ++i) { r[i] = b[i] - (xv[i] - dt * Ap[i]); pd[i] = r[i]; rr += r[i] * r[i]; }
    double tol2 = s->p.cg_rel_tol * s->p.cg_rel_tol * bb;
    int it = 0, maxit = forced >= 0 ? forced : s->p.cg_max_iter;
    s->cg_hist_n = 0;
    s->cg_hist[s->cg_hist_n++] = bb > 0 ? sqrt(rr / bb) : 0.0;
    while (it < maxit && (forced >= 0 || rr > tol2)) {
        sphref_viscosity_operator(s, pd, Ap);
        double pAp = 0.0;
        for (int i = 0; i < n3; ++i) { Ap[i] = pd[i] - dt * Ap[i]; pAp += pd[i] * Ap[i]; }
        if (!(pAp > 0.0)) break;
        double a = rr / pAp, rr_new = 0.0;
        for (int i = 0; i < n3; ++i) { xv[i] += a * pd[i]; r[i] -= a * Ap[i]; rr_new += r[i] * r[i]; }
        double beta = rr_new / rr;
        for (int i = 0; i < n3; ++i) pd[i] = r[i] + beta * pd[i];
        rr = rr_new;
        ++it;
        if (s->cg_hist_n < s->p.cg_max_iter + 1) s->cg_hist[s->cg_hist_n++] = bb > 0 ? sqrt(rr / bb) : 0.0;
    }
    s->stats.cg_iters = it;
    s->stats.cg_residual = bb > 0 ? sqrt(rr / bb) : 0.0;
    free(b); free(r); free(pd); free(Ap);
    return it;
}

/* ------------------------------------------------------------------ rigid stand-in (reading R18) */

/* (c.2) step 7.  PAPER.md:266 delegates rigid dynamics to PyBullet; this explicit
 * symplectic update with a frictionless, inelastic contact sphere against the tank AABB
 * (no rigid-rigid contact) stands in for it.  Weak coupling: sample velocities are only
 * refreshed here, i.e. constant during the fluid solve. */
void sphref_rigid_step(SphRef *s)
{
    double dt = s->p.dt;
    for (int b = 0; b < s->nbodies; ++b) {
        SphRefBody *B = &s->bodies[b];
        if (!B->dynamic) continue;
        double F[3] = { B->mass * s->p.gravity[0], B->mass * s->p.gravity[1], B->mass * s->p.gravity[2] };
        double tau[3] = { 0, 0, 0 };
        for (int k = B->first_particle; k < B->first_particle + B->n_particles; ++k) {
            double rk[3] = { s->bx[3 * k] - B->com[0], s->bx[3 * k + 1] - B->com[1], s->bx[3 * k + 2] - B->com[2] };
            double c[3]; cross3(rk, s->bforce + 3 * k, c);
            for (int a = 0; a < 3; ++a) { F[a] += s->bforce[3 * k + a]; tau[a] += c[a]; }
        }
        for (int a = 0; a < 3; ++a) B->lin_vel[a] += dt * F[a] / B->mass;
        /* omega += dt Iw^-1 (tau - omega x Iw omega), Iw = R Ib R^T */
        double R[9]; quat_to_R(B->quat, R);
        double wb[3], Iw_w[3], tb[3];
        for (int a = 0; a < 3; ++a) wb[a] = R[0 + a] * B->ang_vel[0] + R[3 + a] * B->ang_vel[1] + R[6 + a] * B->ang_vel[2]; /* R^T w */
        for (int a = 0; a < 3; ++a) wb[a] *= B->inertia_body[a];
        for (int a = 0; a < 3; ++a) Iw_w[a] = R[3 * a] * wb[0] + R[3 * a + 1] * wb[1] + R[3 * a + 2] * wb[2];
        double gyro[3]; cross3(B->ang_vel, Iw_w, gyro);
        double rhs[3] = { tau[0] - gyro[0], tau[1] - gyro[1], tau[2] - gyro[2] };
        for (int a = 0; a < 3; ++a) tb[a] = (R[0 + a] * rhs[0] + R[3 + a] * rhs[1] + R[6 + a] * rhs[2]) / B->inertia_body[a];
        for (int a = 0; a < 3; ++a) B->ang_vel[a] += dt * (R[3 * a] * tb[0] + R[3 * a + 1] * tb[1] + R[3 * a + 2] * tb[2]);
        for (int a = 0; a < 3; ++a) B->com[a] += dt * B->lin_vel[a];
        /* q += dt/2 (0, omega) (x) q, normalise */
        double w[3] = { B->ang_vel[0], B->ang_vel[1], B->ang_vel[2] }, q[4] = { B->quat[0], B->quat[1], B->quat[2], B->quat[3] };
        double dq[4] = { -w[0] * q[1] - w[1] * q[2] - w[2] * q[3],
                          w[0] * q[0] + w[1] * q[3] - w[2] * q[2],
                          w[1] * q[0] + w[2] * q[1] - w[0] * q[3],
                          w[2] * q[0] + w[0] * q[2] - w[1] * q[1] };
        double nrm = 0.0;
        for (int a = 0; a < 4; ++a) { q[a] += 0.5 * dt * dq[a]; nrm += q[a] * q[a]; }
        nrm = sqrt(nrm);
        for (int a = 0; a < 4; ++a) B->quat[a] = q[a] / nrm;
        /* wall stand-in */
        for (int a = 0; a < 3; ++a) {
            double lo = s->p.tank_min[a] + B->contact_radius, hi = s->p.tank_max[a] - B->contact_radius;
            if (B->com[a] < lo) { B->com[a] = lo; if (B->lin_vel[a] < 0.0) B->lin_vel[a] = 0.0; }
            if (B->com[a] > hi) { B->com[a] = hi; if (B->lin_vel[a] > 0.0) B->lin_vel[a] = 0.0; }
        }
        quat_to_R(B->quat, R);
        for (int k = B->first_particle; k < B->first_particle + B->n_particles; ++k) {
            double rk[3], wxr[3];
            for (int a = 0; a < 3; ++a) rk[a] = R[3 * a] * s->brest[3 * k] + R[3 * a + 1] * s->brest[3 * k + 1] + R[3 * a + 2] * s->brest[3 * k + 2];
            cross3(B->ang_vel, rk, wxr);
            for (int a = 0; a < 3; ++a) { s->bx[3 * k + a] = B->com[a] + rk[a]; s->bv[3 * k + a] = B->lin_vel[a] + wxr[a]; }
        }
    }
}

/* ------------------------------------------------------------------ steps */

static double max_speed(const SphRef *s)
{
    double vm = 0.0;
    for (int i = 0; i < s->nf; ++i) { double q = dot3(s->v + 3 * i, s->v + 3 * i); if (q > vm) vm = q; }
    return sqrt(vm);
}

/* Time step of the coming step (reading R26; PAPER.md:49 only says that implicit pressure solvers allow
 * "larger time steps", the rule is the usual CFL condition of the cited DFSPH source [5]):
 *   dt = clamp(lambda 2r / max_i |v_i|, dt_min, dt_max), dt_max = the configured dt, lambda = cfl_factor,
 * with the velocities at the START of the step; lambda = 0 keeps dt fixed.  forced_dt > 0 overrides
 * (parity runs hand the GPU's fp32 choice to the oracle, as they do with the iteration counts, R20). */
static double choose_dt(SphRef *s)
{
    const SphRefParams *p = &s->p;
    double dt = s->dt_max;
    if (s->forced_dt > 0.0) return s->forced_dt;
    if (p->cfl_factor > 0.0) {
        double vm = max_speed(s);
        double c = p->cfl_factor * 2.0 * p->particle_radius / (vm > 1e-30 ? vm : 1e-30);
        if (c < dt) dt = c;
        if (dt < p->dt_min) dt = p->dt_min;
    }
    return dt;
}
void sphref_set_forced_dt(SphRef *s, double dt) { s->forced_dt = dt; }

/* One DFSPH step, (c.2) steps 1-7 (Alg. 1 PAPER.md:127-134 with the pressure solve of
 * Alg. 2 realised by DFSPH [5]; order of stages per PAPER.md:262 and reading R13).
 * forced_*: -1 = free running (tolerances decide), >= 0 = exactly that many iterations. */
int sphref_step_dfsph(SphRef *s, int forced_v, int forced_d, int forced_cg)
{
    const SphRefParams *p = &s->p;
    int n3 = 3 * s->nf;
    s->p.dt = choose_dt(s);                                 /* every stage below reads p->dt */
    if (p->force_iterations) {
        if (forced_v < 0) forced_v = p->min_iter_divergence;
        if (forced_d < 0) forced_d = p->min_iter_density;
    }
    sphref_build_grid(s);                                   /* 1 */
    memset(s->bforce, 0, sizeof(double) * 3 * (size_t)(s->nb > 0 ? s->nb : 1));
    sphref_compute_density_alpha(s);                        /* 2 */
    if (p->enable_divergence_solve) sphref_divergence_solve(s, s->v, forced_v); /* 3 */
    else { s->stats.it_v = 0; s->stats.err_v = 0.0; }
    /* 4: non-pressure accelerations (Alg. 1 l.1-2) */
    s->stats.cg_iters = 0; s->stats.cg_residual = 0.0;
    if (p->viscosity_mode == 1) {
        double *acc = (double *)malloc(sizeof(double) * (size_t)(n3 + 1));
        sphref_explicit_viscosity_accel(s, s->v, s->rho, acc);
        for (int i = 0; i < n3; ++i) s->v[i] += p->dt * (p->gravity[i % 3] + acc[i]);
        free(acc);
    } else {
        for (int i = 0; i < n3; ++i) s->v[i] += p->dt * p->gravity[i % 3];
        if (p->viscosity_mode == 2) sphref_implicit_viscosity_solve(s, s->v, forced_cg);
    }
    sphref_density_solve(s, s->v, forced_d);                /* 5 */
    for (int i = 0; i < n3; ++i) s->x[i] += p->dt * s->v[i]; /* 6: symplectic Euler, Alg. 1 l.5-6 */
    sphref_rigid_step(s);                                   /* 7 */
    s->stats.v_max = max_speed(s);
    s->stats.dt_last = s->p.dt; s->stats.sim_time += s->p.dt;
    s->p.dt = s->dt_max;
    s->lists_valid = 0;
    return 0;
}

/* One WCSPH step, (c.2): grid -> rho (Eq. 12) -> rho~ = max(rho, rho0) (R17) ->
 * p = k((rho~/rho0)^gamma - 1) -> a_i = g + visc(Eq. 15 with rho~_j)
 * - sum_j m (p_i/rho~_i^2 + p_j/rho~_j^2) gradW_ij - sum_k Psi_k (p_i/rho~_i^2) gradW_ik
 * (Eq. 7, 13) -> v += dt a -> x += dt v -> rigid step. */
int sphref_step_wcsph(SphRef *s)
{
    const SphRefParams *p = &s->p;
    int n3 = 3 * s->nf;
    double h = p->support_radius, m = s->m;
    s->p.dt = choose_dt(s);
    sphref_build_grid(s);
    memset(s->bforce, 0, sizeof(double) * 3 * (size_t)(s->nb > 0 ? s->nb : 1));
    sphref_compute_density_alpha(s);
    double *rt = (double *)malloc(sizeof(double) * (size_t)(s->nf + 1));
    double *acc = (double *)calloc((size_t)(n3 + 1), sizeof(double));
    for (int i = 0; i < s->nf; ++i) {
        rt[i] = s->rho[i] > p->rest_density ? s->rho[i] : p->rest_density;
        double pr = p->wcsph_stiffness * (pow(rt[i] / p->rest_density, p->wcsph_exponent) - 1.0);
        s->kappa[i] = pr;
        s->kr[i] = pr / (rt[i] * rt[i]);
    }
    if (p->viscosity_mode == 1) sphref_explicit_viscosity_accel(s, s->v, rt, acc);
    for (int i = 0; i < n3; ++i) s->v[i] += p->dt * (p->gravity[i % 3] + acc[i]);
    apply_pressure_update(s, s->v);   /* v -= dt U[p/rho~^2], accumulates Eq. 14 reactions */
    (void)h; (void)m;
    for (int i = 0; i < n3; ++i) s->x[i] += p->dt * s->v[i];
    sphref_rigid_step(s);
    s->stats.it_v = 0; s->stats.it_d = 0; s->stats.v_max = max_speed(s);
    s->stats.dt_last = s->p.dt; s->stats.sim_time += s->p.dt;
    s->p.dt = s->dt_max;
    free(rt); free(acc);
    s->lists_valid = 0;
    return 0;
}

/* One PCISPH step (reading R28; Alg. 1 PAPER.md:127-134 with the pressure solve of Alg. 2 realised by [25]):
 * grid -> rho (Eq. 12) -> v* = v + dt (g + Eq. 15 if viscosity_mode 1) -> pressure loop above -> x += dt v* -> rigid step.
 * (viscosity_mode 2 is not combined with this solver.) */
int sphref_step_pcisph(SphRef *s, int forced)
{
    const SphRefParams *p = &s->p;
    int n3 = 3 * s->nf;
    s->p.dt = choose_dt(s);
    if (p->force_iterations && forced < 0) forced = p->pcisph_min_iter > 0 ? p->pcisph_min_iter : 3;
    sphref_build_grid(s);
    memset(s->bforce, 0, sizeof(double) * 3 * (size_t)(s->nb > 0 ? s->nb : 1));
    sphref_compute_density_alpha(s);
    if (p->viscosity_mode == 1) {
        double *acc = (double *)malloc(sizeof(double) * (size_t)(n3 + 1));
        sphref_explicit_viscosity_accel(s, s->v, s->rho, acc);
        for (int i = 0; i < n3; ++i) s->v[i] += p->dt * (p->gravity[i % 3] + acc[i]);
        free(acc);
    } else {
        for (int i = 0; i < n3; ++i) s->v[i] += p->dt * p->gravity[i % 3];
    }
    sphref_pcisph_solve(s, s->v, forced);
    for (int i = 0; i < n3; ++i) s->x[i] += p->dt * s->v[i];
    sphref_rigid_step(s);
    s->stats.it_v = 0; s->stats.cg_iters = 0; s->stats.v_max = max_speed(s);
    s->stats.dt_last = s->p.dt; s->stats.sim_time += s->p.dt;
    s->p.dt = s->dt_max;
    s->lists_valid = 0;
    return 0;
}

/* ------------------------------------------------------------------ state access */

void sphref_set_state(SphRef *s, const float *pos, const float *vel)
{
    for (int i = 0; i < 3 * s->nf; ++i) { s->x[i] = pos[i]; s->v[i] = vel[i]; }
    s->lists_valid = 0;
}
void sphref_set_state_f64(SphRef *s, const double *pos, const double *vel)
{
    memcpy(s->x, pos, sizeof(double) * 3 * (size_t)s->nf);
    memcpy(s->v, vel, sizeof(double) * 3 * (size_t)s->nf);
    s->lists_valid = 0;
}
/* boundary sample state (fp32 from the GPU at a resync point) and body state */
void sphref_set_boundary_state(SphRef *s, const float *bpos, const float *bvel)
{
    for (int i = 0; i < 3 * s->nb; ++i) { s->bx[i] = bpos[i]; s->bv[i] = bvel[i]; }
    s->lists_valid = 0;
}
void sphref_set_bodies(SphRef *s, const SphRefBody *b) { for (int i = 0; i < s->nbodies; ++i) s->bodies[i] = b[i]; }
void sphref_get_bodies(const SphRef *s, SphRefBody *b) { for (int i = 0; i < s->nbodies; ++i) b[i] = s->bodies[i]; }
void sphref_set_params(SphRef *s, const SphRefParams *p) { s->p = *p; s->dt_max = p->dt; }

double *sphref_pos(SphRef *s) { return s->x; }
double *sphref_vel(SphRef *s) { return s->v; }
double *sphref_density(SphRef *s) { return s->rho; }
double *sphref_alpha(SphRef *s) { return s->alpha; }
double *sphref_kappa(SphRef *s) { return s->kappa; }
double *sphref_kr(SphRef *s) { return s->kr; }
double *sphref_ksum_v(SphRef *s) { return s->ksum_v; }
double *sphref_ksum_d(SphRef *s) { return s->ksum_d; }
void sphref_set_warm_state(SphRef *s, const double *kv, const double *kd)
{
    memcpy(s->ksum_v, kv, sizeof(double) * (size_t)s->nf);
    memcpy(s->ksum_d, kd, sizeof(double) * (size_t)s->nf);
}
double *sphref_psi(SphRef *s) { return s->psi; }
double *sphref_boundary_pos(SphRef *s) { return s->bx; }
double *sphref_boundary_vel(SphRef *s) { return s->bv; }
double *sphref_boundary_force(SphRef *s) { return s->bforce; }
double *sphref_cg_history(SphRef *s, int *n) { *n = s->cg_hist_n; return s->cg_hist; }
double sphref_mass(const SphRef *s) { return s->m; }
void sphref_get_stats(const SphRef *s, SphRefStats *o) { *o = s->stats; }

/* grid: which = 0 fluid, 1 boundary */
void sphref_grid_dims(const SphRef *s, int which, int dims[4])
{
    const CellList *g = which ? &s->gb : &s->gf;
    dims[0] = g->nx; dims[1] = g->ny; dims[2] = g->nz; dims[3] = g->ncells;
}
int *sphref_cell_start(SphRef *s, int which) { return which ? s->gb.cell_start : s->gf.cell_start; }
int *sphref_cell_of_particle(SphRef *s, int which) { return which ? s->gb.key : s->gf.key; }
int *sphref_neighbor_start(SphRef *s, int which) { return which ? s->nb_start : s->nf_start; }
int *sphref_neighbor_idx(SphRef *s, int which) { return which ? s->nb_idx : s->nf_idx; }

int sphref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
