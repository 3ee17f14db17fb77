/*
 * sph.h -- C ABI of libsph_b200: the per-time-step DFSPH particle pipeline of
 * arxiv 2403.11156 ("Journey into SPH Simulation") as hand-written CUDA for sm_100a.
 *
 * Citations are /root/reference/PAPER.md line numbers (section / equation named) and the
 * readings Rn of DESIGN.md (the paper prints no DFSPH equations, no kernel function and no
 * neighbour-search description; every gap is an explicit reading there).
 *
 * Conventions
 *   - every function returns SPH_OK (0) or a negative SphError; nothing throws across the ABI;
 *     sph_last_error() gives the text of the last failure of that simulation (or of create).
 *   - the library NEVER allocates or frees device memory: the caller (PyTorch tensors in the
 *     Python binding) owns the inputs and one workspace of sph_workspace_bytes() bytes that
 *     must stay alive and untouched until sph_destroy().  It creates one helper stream (used
 *     only to capture CUDA-graph loop bodies, never to run work) and a few KB of pinned host
 *     memory.
 *   - all work is enqueued asynchronously on the cudaStream_t given to sph_create(); the only
 *     calls that synchronise that stream are sph_read_stats(), sph_launch_count(),
 *     sph_read_kernel_times(), sph_set_forced_iterations() (its three words travel through a
 *     pinned block that the next call reuses), host-buffer copies of
 *     sph_read_state()/sph_write_state(), sph_create() itself (it computes the Akinci
 *     volumes) and the step calls when SphParams.use_cuda_graph == 0 (debug mode: the
 *     solver loops are then driven from the host).
 *   - "device" pointers are CUDA device pointers on `cuda_device`; "host" pointers are
 *     ordinary (preferably pinned) host memory.
 *   - particles are handed over and read back in the caller's ORIGINAL id order; internally
 *     the store is kept sorted by grid cell (SoA float4, fp32) and re-sorted every step.
 *   - device-side conditions (particles clamped at the grid edge, neighbour-list overflow,
 *     NaN, max-iterations reached) are counters in SphStats, not return codes.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPH_ABI_VERSION 2

typedef enum SphError {
    SPH_OK = 0,
    SPH_EINVAL = -1,  /* bad argument / inconsistent parameters */
    SPH_ENOMEM = -2,  /* workspace too small */
    SPH_ECUDA = -3,   /* a CUDA runtime call failed (text in sph_last_error) */
    SPH_EDOMAIN = -4, /* grid would exceed 2^31 cells or domain is empty */
    SPH_ESTATE = -5   /* call not valid in this state (e.g. read of a field not yet computed) */
} SphError;

/* Problem statement ("domain boundary, simulation method, particle radius,
 * support radius, density, viscosity, initial position, velocity"; PAPER.md:140 k, gamma;
 * PAPER.md:170 "max error").  Plain C struct, passed by pointer, copied by sph_create. */
typedef struct SphParams {
    float particle_radius;     /* r */
    float support_radius;      /* h, support radius of W (= 4r) */
    float rest_density;        /* rho0 */
    float particle_mass;       /* 0 => rho0 (2r)^3                    reading R3 */
    float dt;                  /* time step; with cfl_factor > 0 its upper bound   readings R19, R26 */
    float gravity[3];
    float domain_min[3];       /* grid origin and extent; particles outside are clamped into */
    float domain_max[3];       /*   the edge cells and counted in SphStats.oob_count (R11)   */
    float tank_min[3];         /* AABB used only by the rigid-body wall-contact stand-in (R18) */
    float tank_max[3];
    int   viscosity_mode;      /* 0 none, 1 explicit Eq. 15, 2 implicit Eq. 16-19 (CG; DFSPH steps only:
                                  sph_step_wcsph returns SPH_ESTATE); anything else: SPH_EINVAL at create */
    float kinematic_viscosity; /* nu = mu / rho0 */
    float cg_rel_tol;          /* |r|_2 <= tol |b|_2                  reading R23 */
    int   cg_max_iter;
    float eta_density;         /* mean(rho* - rho0)/rho0 threshold    reading R6 */
    int   min_iter_density, max_iter_density;
    float eta_divergence;      /* dt mean(Drho/Dt)/rho0 threshold     reading R6 */
    int   min_iter_divergence, max_iter_divergence;
    int   enable_divergence_solve;
    int   force_iterations;    /* 1: run exactly min_iter_* iterations, ignore the errors */
    float wcsph_stiffness;     /* k */
    float wcsph_exponent;      /* gamma */
    int   max_fluid_neighbors;    /* capacity of the per-particle fluid neighbour list, 0 => 64;
                                     rounded up to a multiple of 4, at most 768 (the list builder
                                     stages a warp's lists in shared memory).  Overflow is counted in
                                     SphStats.overflow_count and the step's results are invalid */
    int   max_boundary_neighbors; /* same for boundary neighbours, 0 => 64 */
    int   use_cuda_graph;      /* 1: one CUDA graph per step with device-side WHILE loops (default
                                  path); 0: plain launches, loop predicates read by the host */
    int   use_neighbor_list;   /* 1: solver passes gather through the per-step neighbour list
                                  (default); 0: every pass re-walks the 27 cells */
    float cfl_factor;          /* lambda > 0: CFL-adaptive step, evaluated on the device before every step,
                                  dt = clamp(lambda 2r / max_i |v_i|, dt_min, dt) with the velocities at the
                                  step's start (reading R26); 0: fixed dt */
    float dt_min;
    int   warm_start;          /* 1: both DFSPH solves start from the stiffness applied in the last step (reading R27;
                                  SURVEY 8(f) NEXT-1): before each loop one C-pass applies
                                  omega K_i, K_i = total kappa_i of that solve in the previous step, carried with the
                                  particle through the sort.  Costs one C-pass per solve (and un-fuses the first
                                  divergence P-pass); pays when the loops run well above their minimum counts */
    float warm_start_factor;   /* omega in [0, 1]; 0.5 in the public implementation of the cited source [5] */
    int   pcisph_min_iter, pcisph_max_iter;   /* sph_step_pcisph (reading R28): 0 => 3 / 100 */
} SphParams;

/* Rigid body = contiguous range of boundary samples (Akinci [3]).  Dynamics are
 * a minimal stand-in for the external engine the paper delegates to (R18). */
typedef struct SphRigidBody {
    int   first_particle, n_particles; /* range in the boundary arrays (original order) */
    int   dynamic;                     /* 0: static (walls, obstacles) */
    float mass;
    float inertia_body[3];             /* principal moments, body frame */
    float com[3];
    float quat[4];                     /* w, x, y, z */
    float lin_vel[3];
    float ang_vel[3];
    float contact_radius;              /* wall-contact sphere radius of the stand-in */
} SphRigidBody;

/* Inputs of sph_create; all DEVICE pointers, owned by the caller, read during sph_create only
 * (copied into the workspace), except `workspace` which the simulation lives in. */
typedef struct SphBuffers {
    const float *fluid_pos;      /* [n_fluid * 3] xyz, original id order */
    const float *fluid_vel;      /* [n_fluid * 3] */
    const float *boundary_pos;   /* [n_boundary * 3] world coordinates at t = 0 (may be NULL if 0) */
    const int   *boundary_body;  /* [n_boundary] index into bodies[] */
    void        *workspace;      /* >= sph_workspace_bytes(...), 256-byte aligned */
    size_t       workspace_bytes;
} SphBuffers;

typedef struct SphStats {
    long long steps_done;        /* steps since create */
    long long total_it_v;        /* summed over steps_done (mean iterations = total / steps) */
    long long total_it_d;
    long long total_cg_iters;
    int   it_v, it_d, cg_iters;  /* last step */
    float err_v, err_rho;        /* last step: errors measured in the last P-pass (R14) */
    float cg_residual;           /* |r|/|b| at exit */
    int   oob_count;             /* fluid particles clamped into edge cells in the last grid build */
    int   overflow_count;        /* particles whose neighbour list overflowed (last step) */
    int   nan_count;             /* fluid particles with a non-finite position or velocity after the step */
    int   max_iter_hit;          /* bit 0: divergence, bit 1: density, bit 2: CG reached max iterations */
    float v_max;                 /* max |v| after the last step (CFL monitor) */
    int   max_fluid_neighbors;   /* largest fluid / boundary neighbour count seen in the last list build */
    int   max_boundary_neighbors;
    float mean_fluid_neighbors;
    float dt_last;               /* time step of the last step */
    double sim_time;             /* simulated time since create (sum of the steps' dt) */
} SphStats;

/* Fields of sph_read_state / sph_write_state.  Per-particle fields are in ORIGINAL id order. */
typedef enum SphField {
    SPH_FIELD_POS = 0,             /* float [n_fluid*3]                                  rw */
    SPH_FIELD_VEL = 1,             /* float [n_fluid*3]                                  rw */
    SPH_FIELD_DENSITY = 2,         /* float [n_fluid]   rho_i of the last density pass (Eq. 4 + 12) */
    SPH_FIELD_ALPHA = 3,           /* float [n_fluid]   DFSPH factor (R5) */
    SPH_FIELD_KAPPA_OVER_RHO = 4,  /* float [n_fluid]   kappa_i / rho_i of the last P-pass (WCSPH: p_i / rho~_i^2) */
    SPH_FIELD_CELL_START = 5,      /* int   [n_cells+1] fluid grid, linear x-fastest cell order (R11) */
    SPH_FIELD_CELL_OF_PARTICLE = 6,/* int   [n_fluid]   linear cell key of every fluid particle */
    SPH_FIELD_SORTED_ID = 7,       /* int   [n_fluid]   original id of the particle in sorted slot s */
    SPH_FIELD_NEIGHBOR_COUNT = 8,  /* int   [n_fluid*2] (#fluid, #boundary) neighbours */
    SPH_FIELD_FLUID_NEIGHBORS = 9, /* int   [n_fluid*Kf] original ids of fluid neighbours, -1 padded (Kf = fluid list capacity) */
    SPH_FIELD_BOUNDARY_NEIGHBORS = 10, /* int [n_fluid*Kb] original boundary ids, -1 padded */
    SPH_FIELD_BOUNDARY_POS = 11,   /* float [n_boundary*3] current world positions           rw */
    SPH_FIELD_BOUNDARY_VEL = 12,   /* float [n_boundary*3]                                   rw */
    SPH_FIELD_BOUNDARY_PSI = 13,   /* float [n_boundary]   Akinci Psi_k (Eq. 11) */
    SPH_FIELD_BOUNDARY_FORCE = 14, /* float [n_boundary*3] Eq. 14 reaction of the last step (dynamic samples only, else 0) */
    SPH_FIELD_RIGID_BODIES = 15,   /* SphRigidBody [n_bodies]                                rw */
    SPH_FIELD_BOUNDARY_CELL_START = 16, /* int [n_cells+1] boundary grid */
    SPH_FIELD_BOUNDARY_CELL_OF_PARTICLE = 17, /* int [n_boundary] */
    SPH_FIELD_KSUM_DIVERGENCE = 18,/* float [n_fluid]   total kappa^v_i the divergence solve applied in the last step (R27)  rw */
    SPH_FIELD_KSUM_DENSITY = 19    /* float [n_fluid]   total kappa_i the density solve applied in the last step (R27)      rw */
} SphField;

typedef struct SphSim SphSim;

/* Bytes of device workspace a simulation of this size needs (0 on invalid parameters). */
size_t sph_workspace_bytes(const SphParams *params, int n_fluid, int n_boundary, int n_bodies);

/* Grid geometry the library will use for these parameters (R11): dims[0..2] = n_x, n_y, n_z,
 * dims[3] = n_cells.  Also the neighbour-list capacities after rounding: caps[0] = Kf, caps[1] = Kb. */
int sph_grid_dims(const SphParams *params, int dims[4], int caps[2]);

/* Create: copies the inputs into the workspace, builds the boundary grid, computes the Akinci
 * volumes Psi_k = rho0 / sum_{k' in same body} W_kk' (Eq. 11, R9), builds the fluid
 * grid.  `bodies` is a HOST array.  `cuda_stream` is a cudaStream_t (NULL = legacy default
 * stream).  Synchronises the stream once.  On failure *out = NULL and the error text is
 * available from sph_last_error(NULL). */
int sph_create(const SphParams *params, const SphBuffers *buffers, int n_fluid, int n_boundary,
               const SphRigidBody *bodies, int n_bodies, int cuda_device, void *cuda_stream,
               SphSim **out);

/* A1-A3 only: cell keys, histogram + exclusive prefix scan, counting-sort scatter and reorder of
 * the particle store ("prefix sum"; R11, R12).  Leaves the store sorted.  Also
 * builds the per-particle neighbour lists and rho, alpha (A4) so that every read field is
 * consistent with the current positions. */
int sph_build_grid(SphSim *sim);

/* n_steps DFSPH steps (Alg. 1 PAPER.md:127-134 with the pressure solve of Alg. 2
 * realised by DFSPH [5] = Eq. 8 and Eq. 10 sources): grid -> rho, alpha ->
 * divergence-free solve -> non-pressure forces (gravity, Eq. 15 or Eq. 16-19) -> constant-density
 * solve -> symplectic Euler -> rigid bodies.  Asynchronous, one CUDA-graph launch per step. */
int sph_step_dfsph(SphSim *sim, int n_steps);

/* n_steps WCSPH steps (PAPER.md:140 EOS; Eq. 7, 12, 13; R17): fixed work per step. */
int sph_step_wcsph(SphSim *sim, int n_steps);

/* n_steps PCISPH steps (the paper's second PPE solver; cited source [25]; reading R28):
 * grid -> rho -> v* = v + dt (g [+ Eq. 15]) -> pressure loop of Alg. 2 with the density source term (Eq. 8) and the
 * prediction of Eq. 9: p_i <- max(p_i + delta (rho*_i - rho0), 0) with the global scaling factor delta of [25]
 * (prototype particle in a filled lattice neighbourhood), the increment applied through Eq. 7 + 13; at least
 * pcisph_min_iter iterations, until mean(max(rho* - rho0, 0)) / rho0 <= eta_density -> symplectic Euler -> rigid
 * bodies.  SphStats.it_d / err_rho report the loop; forced_d of sph_set_forced_iterations overrides its count.
 * viscosity_mode 2 is not combined with this solver (SPH_ESTATE). */
int sph_step_pcisph(SphSim *sim, int n_steps);

/* ---- Slab mode: x-slab domain decomposition across GPUs (the paper runs on one GPU,
 * this is the build's own extension for the 4M-8M sweep).  Every rank (or, for tests, every slab of one
 * device) owns the particles of an x-range and keeps copies ("ghosts") of the neighbouring slabs' particles within h of
 * the cuts.  A slab is an ordinary simulation created with n_fluid = its CAPACITY, use_cuda_graph = 0 and static
 * boundaries; per step the caller
 *   1. selects migrating particles and ghost layers (sph_select_range), exchanges them with the x-neighbours and hands
 *      the slab its new set (sph_slab_set_particles: owned first, then ghosts);
 *   2. runs the passes one by one (sph_slab_phase).  A pass computes garbage FOR ghosts (their neighbourhood is
 *      incomplete); before the next pass reads that field the owners' values replace it: sph_slab_gather on the owner
 *      (addressed by the ORIGINAL indices the ghost layer was selected with), transfer, sph_slab_scatter on the ghost
 *      side.  Fields: KR = kappa/rho (written by every P-pass, read by the C-pass), VEL = velocity + density lane
 *      (written by every C-pass and the viscosity kernel, read by the P-pass / viscosity);
 *   3. decides each solver loop ONCE for the whole domain: every P-pass leaves the slab's fixed-point error sum over its
 *      OWNED particles (sph_slab_read_error_sum: 2^-20 units of dt/rho0 * sum R_i or sum E_i / rho0; integer, so the sum
 *      over slabs does not depend on the partition), the caller adds them up (all-reduce), applies reading R14 and
 *      writes the result back (sph_slab_set_loop) before the C-pass, whose tail work depends on it.
 * paper_2403_11156_b200/slabs.py holds that schedule with two exchange back ends (slabs of one device; torch.distributed).
 * Not supported in slab mode: dynamic bodies, implicit viscosity, warm start, CUDA-graph launches. */
typedef enum SphSlabPhase {
    SPH_SLAB_BEGIN = 0,         /* time step, A1-A3, neighbour lists, original-index -> slot map */
    SPH_SLAB_DENSITY_DIVP = 1,  /* rho, alpha + first divergence P-pass          -> refresh KR, decide the divergence loop */
    SPH_SLAB_C_DIV = 2,         /* C-pass of the divergence solve (last: + dt g)  -> refresh VEL */
    SPH_SLAB_P_DIV = 3,         /* further divergence P-pass                      -> refresh KR, decide */
    SPH_SLAB_VISCOSITY = 4,     /* explicit viscosity, Eq. 15 (no-op otherwise)   -> refresh VEL */
    SPH_SLAB_P_DENS_FIRST = 5,  /* first density P-pass                           -> refresh KR, decide the density loop */
    SPH_SLAB_P_DENS = 6,        /* further density P-pass                         -> refresh KR, decide */
    SPH_SLAB_C_DENS = 7,        /* C-pass of the density solve (last: integrates) -> refresh VEL unless last */
    SPH_SLAB_END = 8            /* step statistics */
} SphSlabPhase;
typedef enum SphSlabField { SPH_SLAB_FIELD_KR = 0, SPH_SLAB_FIELD_VEL = 1 } SphSlabField;

/* pos4 / vel4: DEVICE, (n_owned + n_ghost) x 4 floats (x, y, z, -), owned particles first; <= the capacity of create. */
int sph_slab_set_particles(SphSim *sim, const float *pos4, const float *vel4, int n_owned, int n_ghost);
int sph_slab_phase(SphSim *sim, int phase);
/* out4[k] = field of the particle whose original index is orig_idx[k] (DEVICE arrays, 4 floats per entry). */
int sph_slab_gather(SphSim *sim, int field, const int *orig_idx, int n, float *out4);
/* field of the particles with original indices first_orig .. first_orig + n - 1 = in4[k]. */
int sph_slab_scatter(SphSim *sim, int field, int first_orig, int n, const float *in4);
int sph_slab_read_error_sum(SphSim *sim, unsigned long long *total_host);   /* synchronises */
/* mode 0: divergence loop, 1: density loop; cont = another iteration follows this C-pass; it, err: for SphStats. */
int sph_slab_set_loop(SphSim *sim, int mode, int cont, int it, float err);
/* Device pointers INTO the workspace: the persistent store after a step (sorted order; 4 floats per particle) and the
 * original index of every slot (< n_owned: owned).  Valid until the next sph_slab_set_particles. */
int sph_slab_store(SphSim *sim, const float **pos4, const float **vel4, const int **orig_idx, int *n, int *n_owned);
/* Deterministic selection (input order kept) of the entries i < n with x_lo <= pos4[i].x < x_hi and, when key != NULL,
 * key[i] < key_lt: copies pos4 / vel4, the id gid[key ? key[i] : i] and (optionally) i itself.  All arrays DEVICE except
 * count_host; scratch: 16-byte aligned, >= n + 8 + (n + 1) / 4096 ints.  Synchronises the stream.  Not tied to a simulation. */
int sph_select_range(void *cuda_stream, const float *pos4, const float *vel4, const int *gid, const int *key, int key_lt,
                     int n, float x_lo, float x_hi, float *out_pos4, float *out_vel4, int *out_gid, int *out_idx,
                     int max_out, int *scratch, size_t scratch_ints, int *count_host);

/* sph_select_range for callers that cannot allocate device memory (code under CUDA-graph capture, serving loops,
 * harnesses that forbid cudaMalloc): same selection, same arguments minus the scratch -- the flag / scan scratch is a
 * file-scope `static __device__` array inside the library, sized for n <= SPH_SELECT_STATIC_MAX entries
 * (SPH_SELECT_STATIC_MAX + 1024 ints = 4 MiB + 4 KiB, held by every GPU that loads the library until the process exits).
 * The call allocates nothing: no cudaMalloc / cudaFree and no allocating library routine; the array's device address is
 * looked up once per device (cudaGetSymbolAddress, with the CURRENT device -- the one the stream and all pointers belong
 * to -- which must be the same on every call that uses that device's array).
 *   n > SPH_SELECT_STATIC_MAX: SPH_EINVAL, *count_host = 0, text in sph_last_error(NULL); nothing is launched.
 *   Every call on a device shares that device's array, which keeps the last call's contents; nothing in it has to start
 *   at zero (every word a call reads it has written itself first).  Two calls whose kernels overlap on the GPU (different
 *   streams, or one graph launched twice concurrently) RACE on it: serialise them.  The call itself synchronises the
 *   stream, like sph_select_range. */
#define SPH_SELECT_STATIC_MAX (1 << 20)
int sph_select_range_static(void *cuda_stream, const float *pos4, const float *vel4, const int *gid, const int *key, int key_lt,
                            int n, float x_lo, float x_hi, float *out_pos4, float *out_vel4, int *out_gid, int *out_idx,
                            int max_out, int *count_host);

/* Override the iteration counts of the next steps: -1 = tolerances decide, >= 0 = exactly that
 * many iterations of the divergence solve / density solve / CG.  Takes effect without re-capture.
 * Synchronises the stream. */
int sph_set_forced_iterations(SphSim *sim, int forced_v, int forced_d, int forced_cg);

/* Copy one field out (un-permuted to original id order) / in.  `bytes` must equal the field's
 * size.  is_host = 0: dst/src is a device pointer, copy is asynchronous on the stream;
 * is_host = 1: host pointer, the call returns after the copy has completed;
 * is_host = 2: PINNED host pointer, asynchronous: the buffer must stay valid and untouched until sph_host_sync()
 *              returns.  Reads run on the simulation's stream.  Writes (fluid fields only) run on a second, internal
 *              stream: a write starts after everything enqueued before it (steps, and earlier asynchronous reads that
 *              may still be filling `src`) and overlaps what is enqueued after it, until a call needs the written array
 *              (a step, sph_build_grid, a read of the same array), which waits for it.  PCIe is full duplex: the upload of
 *              the next step's positions can run beside the download of this step's velocities.
 * sph_write_state (any writable field) invalidates grid-derived fields until the next
 * sph_build_grid / step.  Boundary fields take effect at that next sph_build_grid / step call (or at the next
 * sph_read_state of a boundary / body field, which then already shows the re-posed samples):
 *   SPH_FIELD_BOUNDARY_POS : the samples' world positions are replaced; their body-frame coordinates
 *                            (pose of their body as it is then) and the Akinci volumes Psi_k (Eq. 11,
 *                            PAPER.md:178) are recomputed; the sorted boundary store is rebuilt;
 *   SPH_FIELD_BOUNDARY_VEL : the samples' velocities are replaced (for a dynamic body until its next
 *                            rigid step derives them from the body state again);
 *   SPH_FIELD_RIGID_BODIES : the body states are replaced and the samples of DYNAMIC bodies re-posed,
 *                            x_k = X + R(q) xbar_k, v_k = V + omega x (x_k - X) -- except for what a
 *                            write of BOUNDARY_POS / BOUNDARY_VEL since the last refresh set directly.
 *                            first_particle / n_particles / dynamic must not change. */
int sph_read_state(SphSim *sim, int field, void *dst, size_t bytes, int is_host);
int sph_write_state(SphSim *sim, int field, const void *src, size_t bytes, int is_host);

/* Waits for everything enqueued for this simulation, asynchronous host copies included. */
int sph_host_sync(SphSim *sim);

/* The only call that always synchronises: copies the device statistics block to the host. */
int sph_read_stats(SphSim *sim, SphStats *dst_host);

/* Number of kernel launches (graph kernel nodes executed are counted per node per graph launch,
 * loop bodies once per executed iteration) issued for this simulation since create. */
long long sph_launch_count(SphSim *sim);

/* Per-kernel timing for roofline reports: with SphParams.use_cuda_graph == 0, every kernel
 * launch of the following steps is bracketed by a pair of CUDA events on the simulation's stream.
 * sph_read_kernel_times synchronises, then writes one text line per kernel,
 * "<kernel name> <launches> <total milliseconds>\n", NUL-terminated, into buf (SPH_ENOMEM if it
 * does not fit) and clears the record. */
int sph_enable_kernel_timing(SphSim *sim, int enable);
int sph_read_kernel_times(SphSim *sim, char *buf, size_t bytes);

/* Post-processing stage as CUDA kernels (section 4.3: surface reconstruction of the fluid particles;
 * the paper uses an external tool and prints no equations -- reading R29): the SPH colour field
 *   phi(g) = sum_i (m / rho_i) W(|g - x_i|, h)          (cubic spline of reading R1, strict support |g - x_i| < h)
 * on the nodes g = grid_min + (ix, iy, iz) * cube_size (fp32) of a regular grid of dims[0] x dims[1] x dims[2] nodes,
 * then marching cubes on its cells: a corner is inside when phi > iso, vertices by linear interpolation from the
 * edge's lower-index corner, triangles (outward normals) from a case table generated by face tracing.  Particles and
 * densities are those of the sorted store of the last sph_build_grid / start of the last step (SPH_ESTATE otherwise).
 *   workspace   DEVICE, >= sph_surface_workspace_bytes() bytes, 256-byte aligned; on return its first
 *               dims[0]*dims[1]*dims[2] floats hold phi (x fastest, then y, then z);
 *   triangles   DEVICE, max_triangles * 9 floats: triangle t = vertices (x, y, z) x 3, in cell order (cells x fastest),
 *               the triangles of a cell in table order; triangles beyond max_triangles are dropped;
 *   n_triangles HOST (may be NULL): total number of triangles of the surface; when given, the call synchronises.
 * Asynchronous on the simulation's stream otherwise.  Deterministic (no atomics). */
typedef struct SphSurfaceParams {
    float grid_min[3];
    int   dims[3];        /* nodes per axis, >= 2 each */
    float cube_size;
    float iso;            /* surface threshold on phi (the usual choice is ~0.6) */
} SphSurfaceParams;
size_t sph_surface_workspace_bytes(const SphSurfaceParams *params);
int sph_surface_extract(SphSim *sim, const SphSurfaceParams *params, void *workspace, size_t workspace_bytes,
                        float *triangles, long long max_triangles, long long *n_triangles);

/* ---- Particle image (optional part; reading R30).  The paper renders its results with a third-party
 * path tracer (Blender Cycles / OptiX -- unavailable here, and no equation is printed); the stand-in is
 * an orthographic sphere splat of the fluid particles into headless DEVICE buffers, no graphics API involved:
 *   camera   origin, orthonormal axes right / up (|right| = |up| = 1, right.up = 0 to 1e-4, else SPH_EINVAL), view direction
 *            w = right x up; pixel (px, py), 0 <= px < width, 0 <= py < height, looks along w through
 *            origin + (px + 1/2) pixel_size right + (py + 1/2) pixel_size up;
 *   particle a sphere of radius `radius` (0: the simulation's particle radius) at its CURRENT position (the persistent
 *            store: valid after sph_create, sph_write_state and every step): with (a, b, z) its camera coordinates it
 *            covers the pixel centre (X, Y) when q = R^2 - (X - a)^2 - (Y - b)^2 > 0, at depth t = z - sqrt(q);
 *   outputs  row-major [height][width], each may be NULL: depth = smallest t over the covering particles (+inf: empty),
 *            id = the particle that attains it in the caller's order, the smallest id among equal depths (-1: empty),
 *            shade = Lambert term max(0, -n.l) with the sphere normal n at the hit point and l = light / |light|, the
 *            direction the light travels (0: empty).
 * Deterministic: the depth / id race is decided by a 64-bit integer atomicMin.  workspace: DEVICE, 256-byte aligned,
 * >= sph_render_workspace_bytes (8 bytes per pixel + 4 per fluid particle; 0 for invalid parameters).  Asynchronous on the
 * simulation's stream. */
typedef struct SphRenderParams {
    float origin[3], right[3], up[3];
    float pixel_size;
    int   width, height;
    float radius;         /* 0: particle_radius */
    float light[3];       /* direction the light travels; the zero vector: the view direction w (a headlight) */
} SphRenderParams;
size_t sph_render_workspace_bytes(const SphRenderParams *params, int n_fluid);
int sph_render_particles(SphSim *sim, const SphRenderParams *params, void *workspace, size_t workspace_bytes,
                         float *depth, int *id, float *shade);

const char *sph_last_error(const SphSim *sim);
void sph_destroy(SphSim *sim);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
