// sph_api.cu -- host side of libsph_b200: workspace layout, step orchestration (one CUDA graph
// per step with device-side WHILE loops) and the C ABI of include/sph.h.
//
// Product code.  It never includes, links or calls anything under oracle/.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "sph_common.cuh"
#include "sph_grid.cuh"
#include "sph_passes.cuh"
#include "sph_lists.cuh"
#include "sph_rigid.cuh"
#include "sph_surface.cuh"
#include "sph_render.cuh"

using namespace sph;

namespace {

thread_local std::string g_create_error;

struct Carver {             // carves 256-byte aligned sub-buffers out of the workspace
    char *base;
    size_t off = 0;
    explicit Carver(void *b) : base(static_cast<char *>(b)) {}
    template <typename T> T *take(size_t n)
    {
        size_t bytes = (n * sizeof(T) + 255) & ~size_t(255);
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += bytes;
        return p;
    }
};

struct GridBufs {           // one uniform grid over one particle set
    int n = 0;
    int *key = nullptr, *off = nullptr, *slot = nullptr;
    int *cell_start = nullptr;      // [ncells + 1 (+ pad to 4)]
    int *tile_sum = nullptr;
    int ntiles = 0;
};

}  // namespace

struct SphSim {
    SphParams prm{};
    SimConst c{};
    int nbodies = 0, ndyn = 0;
    int device = 0;
    cudaStream_t stream = nullptr, cap_stream = nullptr;
    int nblocks = 0;                // CTAs of the per-particle kernels (= number of partials)
    size_t cs_len = 0;              // ncells + 1 rounded up to 4
    // fluid store
    float4 *posA = nullptr, *velA = nullptr, *posB = nullptr, *posk = nullptr;
    float *px = nullptr, *py = nullptr, *pz = nullptr;   // sorted positions, structure of arrays (+ 4 floats of padding)
    PV *pvB = nullptr, *pvC = nullptr;   // { pos | vel, rho } records of the passes; pvC: output of explicit viscosity
    int *idA = nullptr, *idB = nullptr;
    float *alpha = nullptr, *rho = nullptr;
    float *ksum_v = nullptr, *ksum_d = nullptr;   // warm start: running totals of the step's solves (sorted order)
    float *pacc = nullptr;          // PCISPH: accumulated pressure of the running step (sorted order)
    int cap = 0;                    // fluid capacity the workspace was laid out for (= n_fluid of sph_create)
    int *inv = nullptr;             // slab mode: original index -> sorted slot of the running step
    PV *slab_vcur = nullptr;        // slab mode: the records the density solve works on (pvB, or pvC after explicit viscosity)
    GridBufs gf, gb;
    uint16_t *nl_f = nullptr;       // 16-bit (run, offset) entries, warp-tiled (sph_passes.cuh)
    int *nl_b = nullptr, *ncount = nullptr;
    float *partial = nullptr, *partial2 = nullptr;
    float4 *cg_r = nullptr, *cg_Ap = nullptr;
    PV *cg_p = nullptr;             // search direction as {x | p, rho} records (gathered by k_cg_apply)
    // boundary store
    float4 *borig_pos = nullptr, *borig_vel = nullptr, *brest = nullptr, *bforce = nullptr;
    float4 *bpos_s = nullptr, *bvel_s = nullptr;
    int *bbody = nullptr, *bid_s = nullptr, *dyn_idx = nullptr;
    SphRigidBody *bodies = nullptr;
    DevControl *ctl = nullptr;
    DevStats *stats = nullptr;
    void *staging = nullptr, *staging_in = nullptr;   // device staging of host reads / of asynchronous host writes
    size_t staging_bytes = 0;
    cudaStream_t copy_stream = nullptr;   // asynchronous host writes (is_host = 2) run here, beside reads on the main stream
    cudaEvent_t ev_main = nullptr, ev_write = nullptr;
    // chunk-wise pipelining of an asynchronous host read with the asynchronous write that uploads the same buffer again
    static constexpr int kHostChunks = 4;
    cudaEvent_t ev_chunk[kHostChunks] = {};
    unsigned long long op_seq = 0;                 // bumped by every API call that may enqueue work on the main stream
    struct { const void *dst = nullptr; size_t bytes = 0; unsigned long long seq = 0; } last_read;   // last asynchronous host read
    unsigned pending_writes = 0;    // arrays with an asynchronous write in flight (WR_* bits)
    // host
    int *pinned = nullptr;          // small pinned block (loop predicate, stats)
    int boundary_dirty = 0;         // DIRTY_* bits: boundary fields written through sph_write_state since the last refresh
    bool pci_step = false;          // the step being enqueued is a PCISPH step
    bool vmax_valid = false;        // stats->vmax_bits = max |v| of the persistent store (needed by the CFL rule)
    bool derived_valid = false;     // B-order fields (rho, alpha, lists, cell_start) match the store
    cudaGraphExec_t exec[3] = { nullptr, nullptr, nullptr };   // 0 DFSPH, 1 WCSPH, 2 PCISPH
    long long fixed_nodes[3] = { 0, 0, 0 };
    long long body_nodes[3][3] = { { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
    long long graph_steps[3] = { 0, 0, 0 };           // graph launches per method (host view)
    long long misc_launches = 0;
    long long *cur_counter = nullptr;
    // optional per-kernel CUDA-event timing (host-driven launch mode only, see sph_enable_kernel_timing)
    bool timing = false;
    struct TimedLaunch { const char *name; cudaEvent_t a, b; };
    std::vector<TimedLaunch> timed;
    std::vector<cudaEvent_t> event_pool;
    std::string err;
};

namespace {

#define CUDA_TRY(sim, expr)                                                                     \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            char b_[512];                                                                       \
            snprintf(b_, sizeof b_, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
            (sim)->err = b_;                                                                    \
            return SPH_ECUDA;                                                                   \
        }                                                                                       \
    } while (0)

#define LAUNCH(sim, kern, grid, block, strm, ...)                                               \
    do {                                                                                        \
        cudaEvent_t ea_ = nullptr, eb_ = nullptr;                                               \
        if ((sim)->timing) {                                                                    \
            ea_ = take_event(sim); eb_ = take_event(sim);                                       \
            cudaEventRecord(ea_, (strm));                                                       \
        }                                                                                       \
        kern<<<(grid), (block), 0, (strm)>>>(__VA_ARGS__);                                      \
        if ((sim)->timing) {                                                                    \
            cudaEventRecord(eb_, (strm));                                                       \
            (sim)->timed.push_back({ #kern, ea_, eb_ });                                        \
        }                                                                                       \
        ++*(sim)->cur_counter;                                                                  \
        CUDA_TRY(sim, cudaGetLastError());                                                      \
    } while (0)

inline cudaEvent_t take_event(SphSim *s)
{
    cudaEvent_t e = nullptr;
    if (!s->event_pool.empty()) { e = s->event_pool.back(); s->event_pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}

// host (pageable) -> device through pinned memory, ordered on the simulation's stream; returns after the copy
// has completed (the stream given to sph_create may be non-blocking: nothing may go through the legacy stream)
int upload(SphSim *s, void *dst_dev, const void *src_host, size_t bytes)
{
    if (bytes == 0) return SPH_OK;
    void *tmp = nullptr;
    CUDA_TRY(s, cudaMallocHost(&tmp, bytes));
    memcpy(tmp, src_host, bytes);
    cudaError_t e = cudaMemcpyAsync(dst_dev, tmp, bytes, cudaMemcpyHostToDevice, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    cudaFreeHost(tmp);
    CUDA_TRY(s, e);
    return SPH_OK;
}

inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

// Asynchronous host writes (sph_write_state, is_host = 2) run on a second stream so that the upload of one field can
// overlap the download of another (PCIe is full duplex).  WR_*: which persistent arrays a pending write touches.
enum { WR_POS = 1, WR_VEL = 2, WR_BOUNDARY = 4 };
unsigned write_mask(int field)
{
    switch (field) {
    case SPH_FIELD_POS: case SPH_FIELD_KSUM_DENSITY: return WR_POS;
    case SPH_FIELD_VEL: case SPH_FIELD_KSUM_DIVERGENCE: return WR_VEL;
    default: return WR_BOUNDARY | WR_POS | WR_VEL;
    }
}
inline size_t host_chunk_bytes(size_t bytes)
{
    const size_t c = (bytes + SphSim::kHostChunks - 1) / SphSim::kHostChunks;
    return (c + 255) & ~size_t(255);
}
// everything enqueued on the main stream from now on sees the pending asynchronous writes
int join_writes(SphSim *s)
{
    if (s->pending_writes) {
        CUDA_TRY(s, cudaStreamWaitEvent(s->stream, s->ev_write, 0));
        s->pending_writes = 0;
    }
    return SPH_OK;
}

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    explicit DeviceGuard(SphSim *s) : DeviceGuard(s->device) { ++s->op_seq; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Grid geometry, reading R11 (restated here; the oracle has its own copy of this definition).
bool make_geom(const SphParams &p, Geom &g, std::string &why)
{
    float h = p.support_radius;
    if (!(h > 0.f)) { why = "support_radius must be > 0"; return false; }
    float cedge = h * 1.0009765625f;
    g.inv_c = 1.0f / cedge;
    g.ox = p.domain_min[0]; g.oy = p.domain_min[1]; g.oz = p.domain_min[2];
    long long n[3];
    for (int a = 0; a < 3; ++a) {
        float ext = p.domain_max[a] - p.domain_min[a];
        if (!(ext >= 0.f)) { why = "domain_max < domain_min"; return false; }
        float t = floorf(ext * g.inv_c);
        if (!(t < 2.0e9f)) { why = "grid too large"; return false; }
        n[a] = (long long)t + 1;
        if (n[a] < 1) n[a] = 1;
    }
    long long nc = n[0] * n[1] * n[2];
    if (nc > 2000000000LL) { why = "grid exceeds 2^31 cells"; return false; }
    if (nc * kFineX > 2000000000LL) { why = "grid exceeds 2^31 cells"; return false; }
    g.nxc = (int)n[0]; g.ncells_c = (int)nc;
    g.nx = (int)n[0] * kFineX; g.ny = (int)n[1]; g.nz = (int)n[2]; g.ncells = (int)nc * kFineX;
    g.inv_cx = g.inv_c * (float)kFineX;
    return true;
}

enum { DIRTY_BPOS = 1, DIRTY_BVEL = 2, DIRTY_BODIES = 4 };

int list_cap(int v, int vmax) { if (v <= 0) v = 64; v = (v + 3) & ~3; if (v > vmax) v = vmax; return v; }

bool make_const(const SphParams &p, int nf, int nb, SimConst &c, std::string &why)
{
    if (nf < 0 || nb < 0) { why = "negative particle count"; return false; }
    if (!(p.particle_radius > 0.f) || !(p.rest_density > 0.f) || !(p.dt > 0.f)) {
        why = "particle_radius, rest_density and dt must be > 0"; return false;
    }
    if (!(p.cfl_factor >= 0.f) || !(p.dt_min >= 0.f) || p.dt_min > p.dt) {
        why = "cfl_factor must be >= 0 and 0 <= dt_min <= dt"; return false;
    }
    if (p.viscosity_mode < 0 || p.viscosity_mode > 2) { why = "viscosity_mode must be 0 (none), 1 (explicit, Eq. 15) or 2 (implicit, Eq. 16-19)"; return false; }
    if (!make_geom(p, c.g, why)) return false;
    c.nf = nf; c.nb = nb; c.nown = nf;
    c.kf = list_cap(p.max_fluid_neighbors, kMaxListCap);
    c.kb = list_cap(p.max_boundary_neighbors, 65532);
    c.h = p.support_radius;
    c.h2 = c.h * c.h;                                   // fp32 product (R10)
    c.inv_h = 1.0f / c.h;
    double hd = (double)p.support_radius;
    double sigma = 8.0 / (3.14159265358979323846 * hd * hd * hd);   // R1
    c.sigma = (float)sigma;
    c.grad_c = (float)(sigma / hd);
    c.ga = (float)(18.0 / (hd * hd)); c.gb = (float)(-12.0 / hd); c.half_h = 0.5f * c.h;
    double d = 2.0 * (double)p.particle_radius;
    c.m = p.particle_mass > 0.f ? p.particle_mass : (float)((double)p.rest_density * d * d * d);   // R3
    c.rho0 = p.rest_density; c.dt = p.dt;
    c.gx = p.gravity[0]; c.gy = p.gravity[1]; c.gz = p.gravity[2];
    c.nu = p.kinematic_viscosity;
    c.mu = p.kinematic_viscosity * p.rest_density;      // R21
    c.visc_eps = (float)(0.01 * hd * hd);
    c.wc_k = p.wcsph_stiffness; c.wc_gamma = p.wcsph_exponent;
    {
        // PCISPH scaling factor (reading R28, cited source [25]): delta dt^2 = rho0^2 / (2 m^2 (|sum gradW|^2 + sum |gradW|^2))
        // for a prototype particle inside a simple-cubic lattice of spacing 2r, neighbours strictly inside h
        const double sp = d, h = hd;
        const int n = (int)std::ceil(h / sp) + 1;
        double S[3] = { 0, 0, 0 }, T = 0.0;
        for (int ia = -n; ia <= n; ++ia) for (int ib = -n; ib <= n; ++ib) for (int ic = -n; ic <= n; ++ic) {
            if (!ia && !ib && !ic) continue;
            const double dx = -ia * sp, dy = -ib * sp, dz = -ic * sp, r2 = dx * dx + dy * dy + dz * dz;
            if (r2 >= h * h) continue;
            const double r = std::sqrt(r2), q = r / h;
            const double wp = q <= 0.5 ? 6.0 * q * (3.0 * q - 2.0) : -6.0 * (1.0 - q) * (1.0 - q);
            const double f = sigma / h * wp / r;
            S[0] += f * dx; S[1] += f * dy; S[2] += f * dz;
            T += f * f * r2;
        }
        const double den = 2.0 * (double)c.m * (double)c.m * (S[0] * S[0] + S[1] * S[1] + S[2] * S[2] + T);
        c.pci_k = den > 0.0 ? (float)((double)p.rest_density * (double)p.rest_density / den) : 0.f;
    }
    c.has_dynamic = 0;
    c.warm = p.warm_start ? 1 : 0;
    c.warm_w = p.warm_start_factor;
    if (p.warm_start && !(p.warm_start_factor >= 0.f && p.warm_start_factor <= 1.f)) { why = "warm_start_factor must lie in [0, 1]"; return false; }
    return true;
}

// Workspace layout: fills the simulation's pointers when base != NULL, returns the bytes needed.
size_t layout(SphSim &s, void *base)
{
    Carver w(base);
    const size_t nf = (size_t)s.c.nf, nb = (size_t)s.c.nb;
    const size_t nf1 = nf ? nf : 1, nb1 = nb ? nb : 1;
    s.cs_len = ((size_t)s.c.g.ncells + 1 + 3) & ~size_t(3);
    s.nblocks = cdiv((long long)nf1, kBlock);
    const size_t nwarps = (nf1 + 31) / 32;
    s.ctl = w.take<DevControl>(1);
    s.stats = w.take<DevStats>(1);
    s.posA = w.take<float4>(nf1); s.velA = w.take<float4>(nf1); s.idA = w.take<int>(nf1);
    s.posB = w.take<float4>(nf1);
    s.px = w.take<float>(nf1 + 4); s.py = w.take<float>(nf1 + 4); s.pz = w.take<float>(nf1 + 4);
    s.pvB = w.take<PV>(nf1); s.idB = w.take<int>(nf1);
    s.pvC = s.prm.viscosity_mode == 1 ? w.take<PV>(nf1) : nullptr;
    s.posk = w.take<float4>(nf1);
    s.alpha = w.take<float>(nf1);
    s.rho = w.take<float>(nf1);
    if (s.prm.warm_start) { s.ksum_v = w.take<float>(nf1); s.ksum_d = w.take<float>(nf1); }
    s.pacc = w.take<float>(nf1);
    s.inv = w.take<int>(nf1);
    s.gf.n = (int)nf;
    s.gf.key = w.take<int>(nf1); s.gf.off = w.take<int>(nf1); s.gf.slot = w.take<int>(nf1);
    s.gf.cell_start = w.take<int>(s.cs_len);
    s.gf.ntiles = cdiv((long long)s.cs_len, kScanTile);
    s.gf.tile_sum = w.take<int>((size_t)s.gf.ntiles);
    s.nl_f = w.take<uint16_t>(nwarps * (size_t)s.c.kf * 32);
    s.nl_b = w.take<int>(nwarps * (size_t)s.c.kb * 32);
    s.ncount = w.take<int>(nf1);
    s.partial = w.take<float>((size_t)s.nblocks);
    s.partial2 = w.take<float>((size_t)s.nblocks);
    if (s.prm.viscosity_mode == 2) {
        s.cg_r = w.take<float4>(nf1); s.cg_p = w.take<PV>(nf1); s.cg_Ap = w.take<float4>(nf1);
    }
    s.borig_pos = w.take<float4>(nb1); s.borig_vel = w.take<float4>(nb1);
    s.brest = w.take<float4>(nb1); s.bforce = w.take<float4>(nb1);
    s.bpos_s = w.take<float4>(nb1); s.bvel_s = w.take<float4>(nb1);
    s.bbody = w.take<int>(nb1); s.bid_s = w.take<int>(nb1); s.dyn_idx = w.take<int>(nb1);
    s.gb.n = (int)nb;
    s.gb.key = w.take<int>(nb1); s.gb.off = w.take<int>(nb1); s.gb.slot = w.take<int>(nb1);
    s.gb.cell_start = w.take<int>(s.cs_len);
    s.gb.ntiles = s.gf.ntiles;
    s.gb.tile_sum = w.take<int>((size_t)s.gb.ntiles);
    s.bodies = w.take<SphRigidBody>((size_t)(s.nbodies > 0 ? s.nbodies : 1));
    size_t st = 16 * (nf1 > nb1 ? nf1 : nb1);
    if (st < 4 * s.cs_len) st = 4 * s.cs_len;
    if (st < sizeof(SphRigidBody) * (size_t)(s.nbodies + 1)) st = sizeof(SphRigidBody) * (size_t)(s.nbodies + 1);
    s.staging_bytes = st;
    s.staging = w.take<char>(st);
    s.staging_in = w.take<char>(st);
    return w.off;
}

// ------------------------------------------------------------------------------------------
// A1-A3 on one particle set: keys + histogram, scan, scatter, canonical reorder.
int enqueue_grid(SphSim *s, cudaStream_t st, GridBufs &g, const float4 *a_in, const float4 *b_in,
                 const int *id_in, float4 *a_out, float4 *b_out, int *id_out, int *oob, bool fluid)
{
    CUDA_TRY(s, cudaMemsetAsync(g.cell_start, 0, s->cs_len * sizeof(int), st));
    if (g.n > 0)
        LAUNCH(s, k_cell_key_hist, cdiv(g.n, 256), 256, st, a_in, g.n, s->c.g, g.key, g.off, g.cell_start, oob);
    const int nscan = s->c.g.ncells + 1;
    LAUNCH(s, k_scan_tile_sums, g.ntiles, kScanThreads, st, g.cell_start, nscan, g.tile_sum);
    LAUNCH(s, k_scan_apply, g.ntiles, kScanThreads, st, g.cell_start, nscan, g.tile_sum);
    if (g.n > 0) {
        LAUNCH(s, k_scatter_slots, cdiv(g.n, 256 * kScatterPer), 256, st, g.key, g.off, g.cell_start, g.n, g.slot);
        if (fluid) LAUNCH(s, k_reorder<true>, cdiv(g.n, 256 * kReorderPer), 256, st, g.slot, g.key, g.cell_start, g.n, a_in, b_in, id_in,
                          a_out, b_out, id_out, s->px, s->py, s->pz);
        else       LAUNCH(s, k_reorder<false>, cdiv(g.n, 256 * kReorderPer), 256, st, g.slot, g.key, g.cell_start, g.n, a_in, b_in, id_in,
                          a_out, b_out, id_out, (float *)nullptr, (float *)nullptr, (float *)nullptr);
    }
    return SPH_OK;
}

PassCtx make_ctx(const SphSim *s)
{
    PassCtx p;
    p.c = s->c;
    p.pos = s->posB; p.bpos = s->bpos_s;
    p.fcs = s->gf.cell_start; p.bcs = s->gb.cell_start;
    p.nl_f = s->nl_f; p.nl_b = s->nl_b; p.ncount = s->ncount; p.id = s->idB;
    return p;
}

int enqueue_boundary_grid(SphSim *s, cudaStream_t st)
{
    return enqueue_grid(s, st, s->gb, s->borig_pos, s->borig_vel, nullptr, s->bpos_s, s->bvel_s, s->bid_s, nullptr, false);
}

// Boundary fields written through sph_write_state take effect here (start of sph_build_grid / of a step call):
//  * body states written: the samples of dynamic bodies are re-posed from them (unless sample positions /
//    velocities were written as well: those win);
//  * sample positions written: body-frame coordinates and the Akinci volumes Psi (Eq. 11) are recomputed;
//  * in every case the sorted boundary store that the passes read is rebuilt.
int refresh_boundary(SphSim *s)
{
    const int dirty = s->boundary_dirty;
    if (!dirty) return SPH_OK;
    s->boundary_dirty = 0;
    const int nb = s->c.nb;
    if (nb <= 0) return SPH_OK;
    cudaStream_t st = s->stream;
    if (dirty & DIRTY_BODIES) {
        const int set_pos = !(dirty & DIRTY_BPOS), set_vel = !(dirty & DIRTY_BVEL);
        if (set_pos || set_vel)
            LAUNCH(s, k_body_pose, cdiv(nb, 256), 256, st, s->brest, s->bbody, s->bodies, nb, s->borig_pos, s->borig_vel, set_pos, set_vel);
    }
    if (dirty & DIRTY_BPOS)
        LAUNCH(s, k_body_rest, cdiv(nb, 256), 256, st, s->borig_pos, s->bbody, s->bodies, nb, s->brest, s->borig_vel, 0);
    int rc = enqueue_boundary_grid(s, st);
    if (rc) return rc;
    if (dirty & DIRTY_BPOS)
        LAUNCH(s, k_boundary_psi, cdiv(nb, kBlock), kBlock, st, s->c, s->bpos_s, s->bid_s, s->gb.cell_start, s->bbody, s->borig_pos);
    return SPH_OK;
}

// Solver loops.  graph mode: a conditional WHILE node whose body is captured on the helper
// stream; host mode: the host reads the predicate after every iteration.
struct LoopCtx {
    cudaStream_t st;
    cudaGraphConditionalHandle h;
    int use_handle;
};

// A1-A3 on the fluid, then the neighbour lists (A4 first half).
int enqueue_fluid_grid_and_lists(SphSim *s, cudaStream_t st)
{
    int rc = enqueue_grid(s, st, s->gf, s->posA, s->velA, s->idA, s->posB, reinterpret_cast<float4 *>(s->pvB), s->idB, &s->stats->oob, true);
    if (rc) return rc;
    if (s->c.nf > 0) {
        PassCtx p = make_ctx(s);
        const BuildShape bs = build_shape(s->c.kf);
        const int grid = cdiv(s->c.nf, 64 * bs.warps);
        cudaEvent_t ea_ = nullptr, eb_ = nullptr;
        if (s->timing) { ea_ = take_event(s); eb_ = take_event(s); cudaEventRecord(ea_, st); }
        k_build_lists<<<grid, 32 * bs.warps, bs.smem, st>>>(p, s->px, s->py, s->pz, &s->stats->lc, bs.rows);
        if (s->timing) { cudaEventRecord(eb_, st); s->timed.push_back({ "k_build_lists", ea_, eb_ }); }
        ++*s->cur_counter;
        CUDA_TRY(s, cudaGetLastError());
    }
    return SPH_OK;
}

// rho and alpha (A4 second half).  divp: also the P-pass of the first divergence-solve iteration
// and, in its last CTA, the loop predicate (DFSPH steps only).
int enqueue_density(SphSim *s, const LoopCtx &lc, bool divp)
{
    if (s->c.nf <= 0) return SPH_OK;
    PassCtx p = make_ctx(s);
    const bool dyn = s->c.has_dynamic != 0;
    LoopHandle lh{ lc.h, lc.use_handle };
#define DENS(LIST, DIVP, DYN) LAUNCH(s, (k_density_alpha<LIST, DIVP, DYN>), s->nblocks, kBlock, lc.st, p, s->pvB, s->bvel_s, s->alpha, s->rho, s->posk, s->ctl, s->stats, lh)
    if (s->prm.use_neighbor_list) {
        if (!divp) DENS(true, false, false); else if (dyn) DENS(true, true, true); else DENS(true, true, false);
    } else {
        if (!divp) DENS(false, false, false); else if (dyn) DENS(false, true, true); else DENS(false, true, false);
    }
#undef DENS
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------

int read_cont(SphSim *s, int *cont)
{
    CUDA_TRY(s, cudaMemcpyAsync(s->pinned, &s->ctl->cont, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    *cont = s->pinned[0];
    return SPH_OK;
}

template <class Init, class Body>
int run_loop(SphSim *s, bool graph_mode, long long *body_counter, Init init, Body body)
{
    if (!graph_mode) {
        LoopCtx lc{ s->stream, 0, 0 };
        int rc = init(lc);
        if (rc) return rc;
        int cont = 0;
        if ((rc = read_cont(s, &cont))) return rc;
        while (cont) {
            if ((rc = body(lc))) return rc;
            if ((rc = read_cont(s, &cont))) return rc;
        }
        return SPH_OK;
    }
    cudaStreamCaptureStatus status;
    cudaGraph_t graph = nullptr;
    const cudaGraphNode_t *deps = nullptr;
    size_t ndeps = 0;
    CUDA_TRY(s, cudaStreamGetCaptureInfo_v2(s->stream, &status, nullptr, &graph, &deps, &ndeps));
    if (status != cudaStreamCaptureStatusActive) { s->err = "run_loop: stream is not capturing"; return SPH_ESTATE; }
    cudaGraphConditionalHandle handle;
    CUDA_TRY(s, cudaGraphConditionalHandleCreate(&handle, graph, 0, 0));
    LoopCtx top{ s->stream, handle, 1 };
    int rc = init(top);                  // captured into the parent graph; sets the first predicate
    if (rc) return rc;
    CUDA_TRY(s, cudaStreamGetCaptureInfo_v2(s->stream, &status, nullptr, &graph, &deps, &ndeps));
    cudaGraphNodeParams np = { cudaGraphNodeTypeConditional };
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    CUDA_TRY(s, cudaGraphAddNode(&node, graph, deps, ndeps, &np));
    cudaGraph_t body_graph = np.conditional.phGraph_out[0];
    CUDA_TRY(s, cudaStreamUpdateCaptureDependencies(s->stream, &node, 1, cudaStreamSetCaptureDependencies));
    CUDA_TRY(s, cudaStreamBeginCaptureToGraph(s->cap_stream, body_graph, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    long long *saved = s->cur_counter;
    s->cur_counter = body_counter;
    LoopCtx in{ s->cap_stream, handle, 1 };
    rc = body(in);
    s->cur_counter = saved;
    cudaGraph_t dummy = nullptr;
    cudaError_t e = cudaStreamEndCapture(s->cap_stream, &dummy);
    if (rc) return rc;
    CUDA_TRY(s, e);
    return SPH_OK;
}

// P-pass of one solver iteration (its last CTA evaluates the loop predicate, A12)
template <bool LIST>
int enqueue_solver_p(SphSim *s, const LoopCtx &lc, int mode, PV *vel, int first)
{
    float *ksum = mode == MODE_PCI ? s->pacc : (mode == MODE_DIV ? s->ksum_v : s->ksum_d);   // warm start totals (NULL when off) / PCISPH pressure
    PassCtx p = make_ctx(s);
    const bool dyn = s->c.has_dynamic != 0;
    LoopHandle lh{ lc.h, lc.use_handle };
#define SOLP(MODE, DYN) LAUNCH(s, (k_solver_p<LIST, MODE, DYN>), s->nblocks, kBlock, lc.st, p, vel, s->bvel_s, s->alpha, s->posk, s->ctl, s->stats, lh, first, ksum)
    if (mode == MODE_DIV) { if (dyn) SOLP(MODE_DIV, true); else SOLP(MODE_DIV, false); }
    else if (mode == MODE_PCI) { if (dyn) SOLP(MODE_PCI, true); else SOLP(MODE_PCI, false); }
    else                  { if (dyn) SOLP(MODE_DENS, true); else SOLP(MODE_DENS, false); }
#undef SOLP
    return SPH_OK;
}

// C-pass (with the tail work of the loop's last iteration) and the Eq. 14 reactions
template <bool LIST>
int enqueue_solver_c(SphSim *s, cudaStream_t st, int tail, PV *vel, int force_mid = 0)
{
    PassCtx p = make_ctx(s);
    const bool dyn = s->c.has_dynamic != 0;
    CTail t;
    t.ctl = s->ctl;
    t.rho = s->rho;
    t.add_gravity = s->prm.viscosity_mode != 1;
    t.id = s->idB; t.pos_out = s->posA; t.vel_out = s->velA; t.id_out = s->idA;
    t.vmax_bits = &s->stats->vmax_bits; t.nan_count = &s->stats->nan_count;
    t.force_mid = force_mid;
    const bool keep_totals = tail != TAIL_WCSPH && !s->pci_step;   // only DFSPH steps maintain the warm-start totals
    t.ksum_v = keep_totals ? s->ksum_v : nullptr; t.ksum_d = keep_totals ? s->ksum_d : nullptr;
    if (tail == TAIL_DIV)       LAUNCH(s, (k_solver_c<LIST, TAIL_DIV>), s->nblocks, kBlock, st, p, s->posk, vel, t);
    else if (tail == TAIL_DENS) LAUNCH(s, (k_solver_c<LIST, TAIL_DENS>), s->nblocks, kBlock, st, p, s->posk, vel, t);
    else                        LAUNCH(s, (k_solver_c<LIST, TAIL_WCSPH>), s->nblocks, kBlock, st, p, s->posk, vel, t);
    if (dyn && s->ndyn > 0)
        LAUNCH(s, k_boundary_force, cdiv(s->ndyn, kBlock), kBlock, st, s->c, s->dyn_idx, s->ndyn, s->borig_pos,
               s->posk, s->gf.cell_start, s->bforce);
    return SPH_OK;
}

template <bool LIST>
int enqueue_solver_iteration(SphSim *s, const LoopCtx &lc, int mode, PV *vel, int first)
{
    int rc = enqueue_solver_p<LIST>(s, lc, mode, vel, first);
    if (rc) return rc;
    return enqueue_solver_c<LIST>(s, lc.st, mode == MODE_DIV ? TAIL_DIV : TAIL_DENS, vel);   // MODE_PCI: the density loop's tail
}

template <bool LIST>
int enqueue_step_t(SphSim *s, int method, bool graph_mode)
{
    cudaStream_t st = s->stream;
    const int nf = s->c.nf;
    const bool dyn = s->c.has_dynamic != 0;
    long long *bc = s->body_nodes[method];
    // DFSPH / PCISPH steps with particles end in a solver loop whose last P-pass also closes the step's statistics
    const bool fold_end = nf > 0 && method != 1;
    LAUNCH(s, k_step_begin, 1, 1, st, s->stats, s->ctl, s->prm.cfl_factor * 2.0f * s->prm.particle_radius, s->prm.dt_min, s->prm.dt, fold_end ? 1 : 0);
    if (dyn) {
        int rc = enqueue_boundary_grid(s, st);
        if (rc) return rc;
        CUDA_TRY(s, cudaMemsetAsync(s->bforce, 0, sizeof(float4) * (size_t)s->c.nb, st));
    }
    int rc = enqueue_fluid_grid_and_lists(s, st);
    if (rc) return rc;
    PV *vcur = s->pvB;
    if (nf > 0) {
        PassCtx p = make_ctx(s);
        if (method == 0) {
            // divergence-free solve (A5).  The loop is peeled: the P-pass of its first iteration runs
            // inside k_density_alpha (which also sets the predicate), the first C-pass follows,
            // further iterations (rare under the default tolerance) are the WHILE body.  The last
            // C-pass adds dt g (A6) unless a viscosity kernel follows.
            const bool warm = s->c.warm != 0;
            if (warm) {
                // reading R27: rho, alpha alone (the fused first P-pass would see the velocities BEFORE the warm start),
                // then the warm-start C-pass of the divergence solve; the loop's first P-pass is an ordinary launch
                LoopCtx plain{ st, 0, 0 };
                rc = enqueue_density(s, plain, false);
                if (rc) return rc;
                LAUNCH(s, k_warm_prepare<MODE_DIV>, cdiv(nf, 256), 256, st, s->c, s->posB, s->pvB, s->rho, s->ctl, s->posk, s->ksum_v);
                rc = enqueue_solver_c<LIST>(s, st, TAIL_DIV, s->pvB, 1);
                if (rc) return rc;
            }
            rc = run_loop(s, graph_mode, &bc[LOOP_DIV],
                [&](const LoopCtx &lc) -> int {
                    if (warm) return enqueue_solver_iteration<LIST>(s, lc, MODE_DIV, s->pvB, 1);
                    int r = enqueue_density(s, lc, true);
                    if (r) return r;
                    return enqueue_solver_c<LIST>(s, lc.st, TAIL_DIV, s->pvB);
                },
                [&](const LoopCtx &lc) -> int { return enqueue_solver_iteration<LIST>(s, lc, MODE_DIV, s->pvB, 0); });
            if (rc) return rc;
            // non-pressure accelerations (A6 / A11)
            if (s->prm.viscosity_mode == 1) {
                LAUNCH(s, (k_explicit_viscosity<LIST, false>), s->nblocks, kBlock, st, p, s->pvB, s->pvC);
                vcur = s->pvC;
            } else if (s->prm.viscosity_mode == 2) {
                rc = run_loop(s, graph_mode, &bc[LOOP_CG],
                    [&](const LoopCtx &lc) -> int {
                        LAUNCH(s, (k_cg_apply<LIST, true>), s->nblocks, kBlock, lc.st, p, reinterpret_cast<const float4 *>(s->pvB), s->cg_r, s->cg_p, s->partial, s->partial2);
                        LAUNCH(s, k_cg_ctrl0, 1, kCtrlThreads, lc.st, s->partial, s->partial2, s->nblocks, s->ctl, s->stats, lc.h, lc.use_handle);
                        return (int)SPH_OK;
                    },
                    [&](const LoopCtx &lc) -> int {
                        LAUNCH(s, (k_cg_apply<LIST, false>), s->nblocks, kBlock, lc.st, p, reinterpret_cast<const float4 *>(s->cg_p), s->cg_Ap, (PV *)nullptr, s->partial, (float *)nullptr);
                        LAUNCH(s, k_cg_ctrl1, 1, kCtrlThreads, lc.st, s->partial, s->nblocks, s->ctl);
                        LAUNCH(s, k_cg_update, cdiv(nf, 256), 256, lc.st, nf, s->ctl, s->cg_p, s->cg_Ap, s->pvB, s->cg_r, s->partial2);
                        LAUNCH(s, k_cg_ctrl2, 1, kCtrlThreads, lc.st, s->partial2, cdiv(nf, 256), s->ctl, s->stats, lc.h, lc.use_handle);
                        LAUNCH(s, k_cg_direction, cdiv(nf, 256), 256, lc.st, nf, s->ctl, s->cg_r, s->cg_p);
                        return (int)SPH_OK;
                    });
                if (rc) return rc;
            }
            // constant-density solve (A7), peeled the same way; its last C-pass integrates (A9)
            if (warm) {
                LAUNCH(s, k_warm_prepare<MODE_DENS>, cdiv(nf, 256), 256, st, s->c, s->posB, vcur, s->rho, s->ctl, s->posk, s->ksum_d);
                rc = enqueue_solver_c<LIST>(s, st, TAIL_DENS, vcur, 1);
                if (rc) return rc;
            }
            rc = run_loop(s, graph_mode, &bc[LOOP_DENS],
                [&](const LoopCtx &lc) -> int { return enqueue_solver_iteration<LIST>(s, lc, MODE_DENS, vcur, 1); },
                [&](const LoopCtx &lc) -> int { return enqueue_solver_iteration<LIST>(s, lc, MODE_DENS, vcur, 0); });
            if (rc) return rc;
        } else if (method == 2) {
            // PCISPH (reading R28): rho -> v* = v + dt (g [+ Eq. 15]) -> pressure loop (P-pass with the global delta,
            // ordinary C-pass; peeled like the density loop, the last C-pass integrates) -> rigid bodies
            LoopCtx plain{ st, 0, 0 };
            rc = enqueue_density(s, plain, false);
            if (rc) return rc;
            LAUNCH(s, k_pci_begin, cdiv(nf, 256), 256, st, s->c, s->rho, s->pvB, s->pacc, s->prm.viscosity_mode != 1);
            if (s->prm.viscosity_mode == 1) {
                LAUNCH(s, (k_explicit_viscosity<LIST, false>), s->nblocks, kBlock, st, p, s->pvB, s->pvC);
                vcur = s->pvC;
            }
            s->pci_step = true;
            rc = run_loop(s, graph_mode, &bc[LOOP_DENS],
                [&](const LoopCtx &lc) -> int { return enqueue_solver_iteration<LIST>(s, lc, MODE_PCI, vcur, 1); },
                [&](const LoopCtx &lc) -> int { return enqueue_solver_iteration<LIST>(s, lc, MODE_PCI, vcur, 0); });
            s->pci_step = false;
            if (rc) return rc;
        } else {
            // WCSPH (A10): rho, EOS, [viscosity], one C-pass that also adds dt g and integrates
            LoopCtx plain{ st, 0, 0 };
            rc = enqueue_density(s, plain, false);
            if (rc) return rc;
            LAUNCH(s, k_wcsph_eos, cdiv(nf, 256), 256, st, s->c, s->posB, s->rho, s->pvB, s->posk);
            if (s->prm.viscosity_mode == 1) {
                LAUNCH(s, (k_explicit_viscosity<LIST, true>), s->nblocks, kBlock, st, p, s->pvB, s->pvC);
                vcur = s->pvC;
            }
            rc = enqueue_solver_c<LIST>(s, st, TAIL_WCSPH, vcur);
            if (rc) return rc;
        }
    }
    if (dyn && s->nbodies > 0)
        LAUNCH(s, k_rigid_step, s->nbodies, 256, st, s->c, s->bodies, s->prm.tank_min[0], s->prm.tank_min[1],
               s->prm.tank_min[2], s->prm.tank_max[0], s->prm.tank_max[1], s->prm.tank_max[2], s->brest, s->bforce,
               s->borig_pos, s->borig_vel);
    if (!fold_end) LAUNCH(s, k_step_end, 1, 1, st, s->stats, s->ctl);
    return SPH_OK;
}

int enqueue_step(SphSim *s, int method, bool graph_mode)
{
    return s->prm.use_neighbor_list ? enqueue_step_t<true>(s, method, graph_mode)
                                    : enqueue_step_t<false>(s, method, graph_mode);
}

int build_graph(SphSim *s, int method)
{
    long long fixed = 0;
    s->cur_counter = &fixed;
    s->body_nodes[method][0] = s->body_nodes[method][1] = s->body_nodes[method][2] = 0;
    cudaError_t e = cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) { s->cur_counter = &s->misc_launches; CUDA_TRY(s, e); }
    int rc = enqueue_step(s, method, true);
    cudaGraph_t graph = nullptr;
    e = cudaStreamEndCapture(s->stream, &graph);
    s->cur_counter = &s->misc_launches;
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    CUDA_TRY(s, e);
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    CUDA_TRY(s, e);
    s->exec[method] = exec;
    s->fixed_nodes[method] = fixed;
    return SPH_OK;
}

int do_steps(SphSim *s, int method, int n_steps)
{
    if (!s) return SPH_EINVAL;
    if (n_steps < 0) { s->err = "n_steps < 0"; return SPH_EINVAL; }
    if (method == 2 && s->prm.viscosity_mode == 2) { s->err = "sph_step_pcisph has no implicit viscosity (viscosity_mode 2): use mode 0 or 1"; return SPH_ESTATE; }
    if (method == 1 && s->prm.viscosity_mode == 2) { s->err = "sph_step_wcsph has no implicit viscosity (viscosity_mode 2): use mode 0 or 1"; return SPH_ESTATE; }
    DeviceGuard dg(s);
    { int rc = join_writes(s); if (rc) return rc; }
    if (n_steps > 0) { int rc = refresh_boundary(s); if (rc) return rc; }
    if (s->prm.cfl_factor > 0.f && !s->vmax_valid && n_steps > 0 && s->c.nf > 0) {
        // the CFL rule needs max |v| at the start of the step; later steps get it from the integration tail
        CUDA_TRY(s, cudaMemsetAsync(&s->stats->vmax_bits, 0, sizeof(unsigned), s->stream));
        LAUNCH(s, k_vmax, cdiv(s->c.nf, 256), 256, s->stream, s->velA, s->c.nf, &s->stats->vmax_bits);
    }
    if (n_steps > 0) s->vmax_valid = true;
    if (s->prm.use_cuda_graph) {
        if (!s->exec[method]) {
            int rc = build_graph(s, method);
            if (rc) return rc;
        }
        for (int k = 0; k < n_steps; ++k) CUDA_TRY(s, cudaGraphLaunch(s->exec[method], s->stream));
        s->graph_steps[method] += n_steps;
    } else {
        for (int k = 0; k < n_steps; ++k) {
            int rc = enqueue_step(s, method, false);
            if (rc) return rc;
        }
    }
    if (n_steps > 0) s->derived_valid = true;
    return SPH_OK;
}

struct FieldInfo { size_t bytes; bool writable; bool derived; };

bool field_info(const SphSim *s, int field, FieldInfo &fi)
{
    const size_t nf = (size_t)s->c.nf, nb = (size_t)s->c.nb, nc1 = (size_t)s->c.g.ncells_c + 1;
    switch (field) {
    case SPH_FIELD_POS: case SPH_FIELD_VEL: fi = { nf * 12, true, false }; return true;
    case SPH_FIELD_DENSITY: case SPH_FIELD_ALPHA: case SPH_FIELD_KAPPA_OVER_RHO: fi = { nf * 4, false, true }; return true;
    case SPH_FIELD_KSUM_DIVERGENCE: case SPH_FIELD_KSUM_DENSITY: fi = { nf * 4, true, false }; return true;
    case SPH_FIELD_CELL_START: fi = { nc1 * 4, false, true }; return true;
    case SPH_FIELD_CELL_OF_PARTICLE: case SPH_FIELD_SORTED_ID: fi = { nf * 4, false, true }; return true;
    case SPH_FIELD_NEIGHBOR_COUNT: fi = { nf * 8, false, true }; return true;
    case SPH_FIELD_FLUID_NEIGHBORS: fi = { nf * (size_t)s->c.kf * 4, false, true }; return true;
    case SPH_FIELD_BOUNDARY_NEIGHBORS: fi = { nf * (size_t)s->c.kb * 4, false, true }; return true;
    case SPH_FIELD_BOUNDARY_POS: case SPH_FIELD_BOUNDARY_VEL: fi = { nb * 12, true, false }; return true;
    case SPH_FIELD_BOUNDARY_PSI: fi = { nb * 4, false, false }; return true;
    case SPH_FIELD_BOUNDARY_FORCE: fi = { nb * 12, false, false }; return true;
    case SPH_FIELD_RIGID_BODIES: fi = { sizeof(SphRigidBody) * (size_t)s->nbodies, true, false }; return true;
    case SPH_FIELD_BOUNDARY_CELL_START: fi = { nc1 * 4, false, false }; return true;
    case SPH_FIELD_BOUNDARY_CELL_OF_PARTICLE: fi = { nb * 4, false, false }; return true;
    default: return false;
    }
}

// writes the field into a DEVICE buffer `out` (asynchronously on the stream)
int export_field(SphSim *s, int field, void *out, size_t bytes)
{
    cudaStream_t st = s->stream;
    const int nf = s->c.nf, nb = s->c.nb;
    if (bytes == 0) return SPH_OK;
    switch (field) {
    case SPH_FIELD_POS: LAUNCH(s, k_export_vec3, cdiv(nf, 256), 256, st, s->posA, s->idA, nf, (float *)out); break;
    case SPH_FIELD_VEL: LAUNCH(s, k_export_vec3, cdiv(nf, 256), 256, st, s->velA, s->idA, nf, (float *)out); break;
    case SPH_FIELD_KSUM_DIVERGENCE: LAUNCH(s, k_export_w, cdiv(nf, 256), 256, st, s->velA, s->idA, nf, (float *)out, 1); break;
    case SPH_FIELD_KSUM_DENSITY: LAUNCH(s, k_export_w, cdiv(nf, 256), 256, st, s->posA, s->idA, nf, (float *)out, 1); break;
    case SPH_FIELD_DENSITY: LAUNCH(s, k_export_scalar, cdiv(nf, 256), 256, st, s->rho, s->idB, nf, (float *)out); break;
    case SPH_FIELD_ALPHA: LAUNCH(s, k_export_scalar, cdiv(nf, 256), 256, st, s->alpha, s->idB, nf, (float *)out); break;
    case SPH_FIELD_KAPPA_OVER_RHO: LAUNCH(s, k_export_w, cdiv(nf, 256), 256, st, s->posk, s->idB, nf, (float *)out, 1); break;
    case SPH_FIELD_CELL_START:
        LAUNCH(s, k_export_cell_start, cdiv(s->c.g.ncells_c + 1, 256), 256, st, s->gf.cell_start, s->c.g.ncells_c + 1, (int *)out); break;
    case SPH_FIELD_BOUNDARY_CELL_START:
        LAUNCH(s, k_export_cell_start, cdiv(s->c.g.ncells_c + 1, 256), 256, st, s->gb.cell_start, s->c.g.ncells_c + 1, (int *)out); break;
    case SPH_FIELD_CELL_OF_PARTICLE:
        LAUNCH(s, k_export_keys, cdiv(nf, 256), 256, st, s->posB, s->idB, nf, s->c.g, (int *)out); break;
    case SPH_FIELD_BOUNDARY_CELL_OF_PARTICLE:
        LAUNCH(s, k_export_keys, cdiv(nb, 256), 256, st, s->bpos_s, s->bid_s, nb, s->c.g, (int *)out); break;
    case SPH_FIELD_SORTED_ID:
        CUDA_TRY(s, cudaMemcpyAsync(out, s->idB, bytes, cudaMemcpyDeviceToDevice, st)); break;
    case SPH_FIELD_NEIGHBOR_COUNT: LAUNCH(s, k_export_counts, cdiv(nf, 256), 256, st, s->ncount, s->idB, nf, (int *)out); break;
    case SPH_FIELD_FLUID_NEIGHBORS:
        LAUNCH(s, k_export_fluid_neighbors, cdiv((long long)nf * s->c.kf, 256), 256, st, s->nl_f, s->ncount, s->posB, s->c.g, s->gf.cell_start, s->idB, nf, s->c.kf, (int *)out); break;
    case SPH_FIELD_BOUNDARY_NEIGHBORS:
        LAUNCH(s, k_export_neighbors, cdiv((long long)nf * s->c.kb, 256), 256, st, s->nl_b, s->ncount, 16, s->idB, s->bid_s, nf, s->c.kb, (int *)out); break;
    case SPH_FIELD_BOUNDARY_POS: LAUNCH(s, k_export_vec3, cdiv(nb, 256), 256, st, s->borig_pos, (const int *)nullptr, nb, (float *)out); break;
    case SPH_FIELD_BOUNDARY_VEL: LAUNCH(s, k_export_vec3, cdiv(nb, 256), 256, st, s->borig_vel, (const int *)nullptr, nb, (float *)out); break;
    case SPH_FIELD_BOUNDARY_PSI: LAUNCH(s, k_export_w, cdiv(nb, 256), 256, st, s->borig_pos, (const int *)nullptr, nb, (float *)out, 1); break;
    case SPH_FIELD_BOUNDARY_FORCE: LAUNCH(s, k_export_vec3, cdiv(nb, 256), 256, st, s->bforce, (const int *)nullptr, nb, (float *)out); break;
    case SPH_FIELD_RIGID_BODIES:
        CUDA_TRY(s, cudaMemcpyAsync(out, s->bodies, bytes, cudaMemcpyDeviceToDevice, st)); break;
    default: s->err = "unknown field"; return SPH_EINVAL;
    }
    return SPH_OK;
}

int import_field(SphSim *s, int field, const void *src, size_t bytes, cudaStream_t st)
{
    const int nf = s->c.nf, nb = s->c.nb;
    if (bytes == 0) return SPH_OK;
    switch (field) {
    case SPH_FIELD_POS: LAUNCH(s, k_import_vec3, cdiv(nf, 256), 256, st, (const float *)src, s->idA, nf, s->posA); break;
    case SPH_FIELD_VEL: LAUNCH(s, k_import_vec3, cdiv(nf, 256), 256, st, (const float *)src, s->idA, nf, s->velA); s->vmax_valid = false; break;
    case SPH_FIELD_KSUM_DIVERGENCE: LAUNCH(s, k_import_w, cdiv(nf, 256), 256, st, (const float *)src, s->idA, nf, s->velA); break;
    case SPH_FIELD_KSUM_DENSITY: LAUNCH(s, k_import_w, cdiv(nf, 256), 256, st, (const float *)src, s->idA, nf, s->posA); break;
    case SPH_FIELD_BOUNDARY_POS: LAUNCH(s, k_import_vec3, cdiv(nb, 256), 256, st, (const float *)src, (const int *)nullptr, nb, s->borig_pos); s->boundary_dirty |= DIRTY_BPOS; break;
    case SPH_FIELD_BOUNDARY_VEL: LAUNCH(s, k_import_vec3, cdiv(nb, 256), 256, st, (const float *)src, (const int *)nullptr, nb, s->borig_vel); s->boundary_dirty |= DIRTY_BVEL; break;
    case SPH_FIELD_RIGID_BODIES:
        CUDA_TRY(s, cudaMemcpyAsync(s->bodies, src, bytes, cudaMemcpyDeviceToDevice, st)); s->boundary_dirty |= DIRTY_BODIES; break;
    default: s->err = "field is not writable"; return SPH_EINVAL;
    }
    return SPH_OK;
}

}  // namespace

// ==============================================================================================
extern "C" {

size_t sph_workspace_bytes(const SphParams *params, int n_fluid, int n_boundary, int n_bodies)
{
    if (!params || n_bodies < 0) return 0;
    SphSim tmp;
    tmp.prm = *params;
    tmp.nbodies = n_bodies;
    std::string why;
    if (!make_const(*params, n_fluid, n_boundary, tmp.c, why)) return 0;
    return layout(tmp, nullptr);
}

int sph_grid_dims(const SphParams *params, int dims[4], int caps[2])
{
    if (!params) return SPH_EINVAL;
    Geom g;
    std::string why;
    if (!make_geom(*params, g, why)) return SPH_EDOMAIN;
    if (dims) { dims[0] = g.nxc; dims[1] = g.ny; dims[2] = g.nz; dims[3] = g.ncells_c; }
    if (caps) { caps[0] = list_cap(params->max_fluid_neighbors, kMaxListCap); caps[1] = list_cap(params->max_boundary_neighbors, 65532); }
    return SPH_OK;
}

int sph_create(const SphParams *params, const SphBuffers *buf, int n_fluid, int n_boundary,
               const SphRigidBody *bodies, int n_bodies, int cuda_device, void *cuda_stream, SphSim **out)
{
    if (out) *out = nullptr;
    if (!params || !buf || !out || n_bodies < 0 || (n_bodies > 0 && !bodies)) { g_create_error = "null argument"; return SPH_EINVAL; }
    SphSim *s = new SphSim;
    s->prm = *params;
    s->nbodies = n_bodies;
    s->device = cuda_device;
    s->cap = n_fluid;
    s->stream = static_cast<cudaStream_t>(cuda_stream);
    s->cur_counter = &s->misc_launches;
    auto fail = [&](int code) { g_create_error = s->err; if (s->cap_stream) cudaStreamDestroy(s->cap_stream); if (s->copy_stream) cudaStreamDestroy(s->copy_stream); if (s->ev_main) cudaEventDestroy(s->ev_main); if (s->ev_write) cudaEventDestroy(s->ev_write); if (s->pinned) cudaFreeHost(s->pinned); delete s; return code; };
    if (!make_const(*params, n_fluid, n_boundary, s->c, s->err)) return fail(s->err.find("grid") != std::string::npos ? SPH_EDOMAIN : SPH_EINVAL);
    if (n_fluid > 0 && (!buf->fluid_pos || !buf->fluid_vel)) { s->err = "fluid_pos / fluid_vel is NULL"; return fail(SPH_EINVAL); }
    if (n_boundary > 0 && (!buf->boundary_pos || !buf->boundary_body)) { s->err = "boundary_pos / boundary_body is NULL"; return fail(SPH_EINVAL); }
    if (params->use_cuda_graph && s->stream == nullptr) { s->err = "use_cuda_graph needs a created stream: CUDA graphs cannot be captured on the legacy default stream"; return fail(SPH_EINVAL); }
    if (n_boundary > 0 && n_bodies == 0) { s->err = "boundary particles need at least one body"; return fail(SPH_EINVAL); }
    std::vector<int> dyn;
    for (int b = 0; b < n_bodies; ++b) {
        const SphRigidBody &B = bodies[b];
        if (B.first_particle < 0 || B.n_particles < 0 || B.first_particle + B.n_particles > n_boundary) { s->err = "body particle range out of bounds"; return fail(SPH_EINVAL); }
        if (B.dynamic) {
            if (!(B.mass > 0.f) || !(B.inertia_body[0] > 0.f) || !(B.inertia_body[1] > 0.f) || !(B.inertia_body[2] > 0.f)) { s->err = "dynamic body needs positive mass and inertia"; return fail(SPH_EINVAL); }
            s->c.has_dynamic = 1;
            for (int k = 0; k < B.n_particles; ++k) dyn.push_back(B.first_particle + k);
        }
    }
    s->ndyn = (int)dyn.size();
    size_t need = layout(*s, nullptr);
    if (!buf->workspace || buf->workspace_bytes < need) {
        char b[160]; snprintf(b, sizeof b, "workspace too small: need %zu bytes, got %zu", need, buf->workspace_bytes);
        s->err = b; return fail(SPH_ENOMEM);
    }
    if ((reinterpret_cast<uintptr_t>(buf->workspace) & 255) != 0) { s->err = "workspace must be 256-byte aligned"; return fail(SPH_EINVAL); }
    layout(*s, buf->workspace);
    s->c.dt_dev = &s->ctl->dt;

    DeviceGuard dg(s);
    auto run = [&]() -> int {
        cudaStream_t st = s->stream;
        CUDA_TRY(s, cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
        CUDA_TRY(s, cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
        CUDA_TRY(s, cudaEventCreateWithFlags(&s->ev_main, cudaEventDisableTiming));
        CUDA_TRY(s, cudaEventCreateWithFlags(&s->ev_write, cudaEventDisableTiming));
        for (int k = 0; k < SphSim::kHostChunks; ++k) CUDA_TRY(s, cudaEventCreateWithFlags(&s->ev_chunk[k], cudaEventDisableTiming));
        CUDA_TRY(s, cudaMallocHost(&s->pinned, 4096));
        // The list passes keep only a 4.6 KB run table per CTA in shared memory and are bound by the L1
        // gather path: ask for a small shared-memory carveout so that most of the 256 KB of an SM is L1
        // (measured on config 4: P-pass 134.6 -> 126.8 us, step 0.887 -> 0.865 ms at 16-20 %; 12 % leaves
        // too little shared memory for the resident CTAs, the driver's default behaves like ~37 %).
        {
            const int carve = 20;
#define CARVE(k) CUDA_TRY(s, cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, carve))
            CARVE((k_solver_p<true, MODE_DENS, false>)); CARVE((k_solver_p<true, MODE_DENS, true>));
            CARVE((k_solver_p<true, MODE_DIV, false>)); CARVE((k_solver_p<true, MODE_DIV, true>));
            CARVE((k_solver_c<true, TAIL_DIV>)); CARVE((k_solver_c<true, TAIL_DENS>)); CARVE((k_solver_c<true, TAIL_WCSPH>));
            CARVE((k_density_alpha<true, true, false>)); CARVE((k_density_alpha<true, true, true>));
            CARVE((k_density_alpha<true, false, false>));
            CARVE((k_explicit_viscosity<true, false>)); CARVE((k_explicit_viscosity<true, true>));
            CARVE((k_cg_apply<true, true>)); CARVE((k_cg_apply<true, false>));
#undef CARVE
        }
        CUDA_TRY(s, cudaFuncSetAttribute(k_build_lists, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)build_shape(s->c.kf).smem));
        // the SoA arrays are read up to 3 elements past the last particle (16-byte granules of the bulk copies)
        CUDA_TRY(s, cudaMemsetAsync(s->px + s->c.nf, 0, 4 * sizeof(float), s->stream));
        CUDA_TRY(s, cudaMemsetAsync(s->py + s->c.nf, 0, 4 * sizeof(float), s->stream));
        CUDA_TRY(s, cudaMemsetAsync(s->pz + s->c.nf, 0, 4 * sizeof(float), s->stream));
        const int nf = s->c.nf, nb = s->c.nb;
        // control + statistics blocks
        DevControl hc;
        memset(&hc, 0, sizeof hc);
        const SphParams &p = s->prm;
        hc.forced_v = p.force_iterations ? p.min_iter_divergence : -1;
        hc.forced_d = p.force_iterations ? p.min_iter_density : -1;   // (PCISPH steps with force_iterations: set the count with sph_set_forced_iterations)
        hc.forced_cg = -1;
        hc.min_v = p.min_iter_divergence; hc.max_v = p.max_iter_divergence;
        hc.min_d = p.min_iter_density; hc.max_d = p.max_iter_density;
        hc.max_cg = p.cg_max_iter; hc.enable_div = p.enable_divergence_solve;
        hc.min_p = p.pcisph_min_iter > 0 ? p.pcisph_min_iter : 3; hc.max_p = p.pcisph_max_iter > 0 ? p.pcisph_max_iter : 100;
        hc.dt = p.dt;
        hc.eta_v = p.eta_divergence; hc.eta_d = p.eta_density; hc.cg_tol = p.cg_rel_tol;
        memcpy(s->pinned, &hc, sizeof hc);
        CUDA_TRY(s, cudaMemcpyAsync(s->ctl, s->pinned, sizeof hc, cudaMemcpyHostToDevice, st));
        CUDA_TRY(s, cudaMemsetAsync(s->stats, 0, sizeof(DevStats), st));
        // fluid store, original order; ids = identity
        if (nf > 0) {
            LAUNCH(s, k_pack_vec3, cdiv(nf, 256), 256, st, buf->fluid_pos, nf, s->posA, 0.f);
            LAUNCH(s, k_pack_vec3, cdiv(nf, 256), 256, st, buf->fluid_vel, nf, s->velA, 0.f);
            LAUNCH(s, k_iota, cdiv(nf, 256), 256, st, s->idA, nf);
        }
        // boundary store
        if (s->nbodies > 0) {
            CUDA_TRY(s, cudaStreamSynchronize(st));       // pinned block is reused below
            int rc = upload(s, s->bodies, bodies, sizeof(SphRigidBody) * (size_t)s->nbodies);
            if (rc) return rc;
        }
        CUDA_TRY(s, cudaMemsetAsync(s->gb.cell_start, 0, s->cs_len * sizeof(int), st));
        if (nb > 0) {
            LAUNCH(s, k_pack_vec3, cdiv(nb, 256), 256, st, buf->boundary_pos, nb, s->borig_pos, 0.f);
            CUDA_TRY(s, cudaMemcpyAsync(s->bbody, buf->boundary_body, sizeof(int) * (size_t)nb, cudaMemcpyDeviceToDevice, st));
            CUDA_TRY(s, cudaMemsetAsync(s->bforce, 0, sizeof(float4) * (size_t)nb, st));
            if (s->ndyn > 0) { int rc = upload(s, s->dyn_idx, dyn.data(), sizeof(int) * dyn.size()); if (rc) return rc; }
            LAUNCH(s, k_body_rest, cdiv(nb, 256), 256, st, s->borig_pos, s->bbody, s->bodies, nb, s->brest, s->borig_vel, 1);
            int rc = enqueue_boundary_grid(s, st);
            if (rc) return rc;
            LAUNCH(s, k_boundary_psi, cdiv(nb, kBlock), kBlock, st, s->c, s->bpos_s, s->bid_s, s->gb.cell_start, s->bbody, s->borig_pos);
        }
        CUDA_TRY(s, cudaStreamSynchronize(st));
        return SPH_OK;
    };
    int rc = run();
    if (rc) return fail(rc);
    rc = sph_build_grid(s);
    if (rc) return fail(rc);
    cudaError_t e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) { s->err = std::string("sph_create: ") + cudaGetErrorString(e); return fail(SPH_ECUDA); }
    *out = s;
    return SPH_OK;
}

int sph_build_grid(SphSim *s)
{
    if (!s) return SPH_EINVAL;
    DeviceGuard dg(s);
    cudaStream_t st = s->stream;
    { int rc = join_writes(s); if (rc) return rc; }
    { int rc = refresh_boundary(s); if (rc) return rc; }
    LAUNCH(s, k_list_counters_reset, 1, 1, st, s->stats);
    if (s->c.has_dynamic) {
        int rc = enqueue_boundary_grid(s, st);
        if (rc) return rc;
    }
    int rc = enqueue_fluid_grid_and_lists(s, st);
    if (!rc) { LoopCtx plain{ st, 0, 0 }; rc = enqueue_density(s, plain, false); }
    if (rc) return rc;
    // leave the persistent store sorted as well (the next step's sort is then the identity)
    const size_t nf = (size_t)s->c.nf;
    if (nf > 0) {
        CUDA_TRY(s, cudaMemcpyAsync(s->posA, s->posB, nf * sizeof(float4), cudaMemcpyDeviceToDevice, st));
        CUDA_TRY(s, cudaMemcpy2DAsync(s->velA, sizeof(float4), &s->pvB->v, sizeof(PV), sizeof(float4), nf, cudaMemcpyDeviceToDevice, st));
        CUDA_TRY(s, cudaMemcpyAsync(s->idA, s->idB, nf * sizeof(int), cudaMemcpyDeviceToDevice, st));
        // posk mirrors the positions with kappa/rho = 0 until a solver pass writes it
        CUDA_TRY(s, cudaMemcpyAsync(s->posk, s->posA, nf * sizeof(float4), cudaMemcpyDeviceToDevice, st));
    }
    s->derived_valid = true;
    return SPH_OK;
}

int sph_step_dfsph(SphSim *s, int n_steps) { return do_steps(s, 0, n_steps); }
int sph_step_wcsph(SphSim *s, int n_steps) { return do_steps(s, 1, n_steps); }
int sph_step_pcisph(SphSim *s, int n_steps) { return do_steps(s, 2, n_steps); }

// ---- slab mode: the pieces of a DFSPH step as separate calls, so that the caller can
// refresh the ghost particles between the passes and decide the loops from the error sums of ALL slabs
}  // extern "C"
namespace {
int slab_check(SphSim *s)
{
    if (!s) return SPH_EINVAL;
    if (s->prm.use_cuda_graph) { s->err = "slab mode drives the passes from the host: create the simulation with use_cuda_graph = 0"; return SPH_ESTATE; }
    if (s->c.has_dynamic) { s->err = "slab mode supports static boundaries only"; return SPH_ESTATE; }
    if (s->prm.viscosity_mode == 2 || s->prm.warm_start) { s->err = "slab mode: implicit viscosity and warm start are not supported"; return SPH_ESTATE; }
    if (s->prm.cfl_factor > 0.f) { s->err = "slab mode: the CFL-adaptive time step needs a global velocity maximum and is not supported"; return SPH_ESTATE; }
    return join_writes(s);
}
template <bool LIST>
int slab_phase_t(SphSim *s, int phase)
{
    cudaStream_t st = s->stream;
    LoopCtx plain{ st, 0, 0 };
    const int nf = s->c.nf;
    switch (phase) {
    case SPH_SLAB_BEGIN: {
        LAUNCH(s, k_step_begin, 1, 1, st, s->stats, s->ctl, s->prm.cfl_factor * 2.0f * s->prm.particle_radius, s->prm.dt_min, s->prm.dt, 0);
        int rc = enqueue_fluid_grid_and_lists(s, st);
        if (rc) return rc;
        if (nf > 0) LAUNCH(s, k_slab_inverse, cdiv(nf, 256), 256, st, s->idB, nf, s->inv);
        s->slab_vcur = s->pvB;
        return SPH_OK;
    }
    case SPH_SLAB_DENSITY_DIVP: return enqueue_density(s, plain, true);
    case SPH_SLAB_C_DIV: return nf > 0 ? enqueue_solver_c<LIST>(s, st, TAIL_DIV, s->pvB) : (int)SPH_OK;
    case SPH_SLAB_P_DIV: return nf > 0 ? enqueue_solver_p<LIST>(s, plain, MODE_DIV, s->pvB, 0) : (int)SPH_OK;
    case SPH_SLAB_VISCOSITY:
        if (s->prm.viscosity_mode == 1 && nf > 0) {
            PassCtx p = make_ctx(s);
            LAUNCH(s, (k_explicit_viscosity<LIST, false>), s->nblocks, kBlock, st, p, s->pvB, s->pvC);
            s->slab_vcur = s->pvC;
        }
        return SPH_OK;
    case SPH_SLAB_P_DENS_FIRST: return nf > 0 ? enqueue_solver_p<LIST>(s, plain, MODE_DENS, s->slab_vcur, 1) : (int)SPH_OK;
    case SPH_SLAB_P_DENS: return nf > 0 ? enqueue_solver_p<LIST>(s, plain, MODE_DENS, s->slab_vcur, 0) : (int)SPH_OK;
    case SPH_SLAB_C_DENS: return nf > 0 ? enqueue_solver_c<LIST>(s, st, TAIL_DENS, s->slab_vcur) : (int)SPH_OK;
    case SPH_SLAB_END:
        LAUNCH(s, k_step_end, 1, 1, st, s->stats, s->ctl);
        s->derived_valid = true; s->vmax_valid = true;
        return SPH_OK;
    default: s->err = "unknown slab phase"; return SPH_EINVAL;
    }
}
}  // namespace
extern "C" {

int sph_slab_set_particles(SphSim *s, const float *pos4, const float *vel4, int n_owned, int n_ghost)
{
    int rc = slab_check(s);
    if (rc) return rc;
    const long long n = (long long)n_owned + n_ghost;
    if (n_owned < 0 || n_ghost < 0 || n > s->cap) { char b[160]; snprintf(b, sizeof b, "slab particle count %lld exceeds the capacity %d the simulation was created with", n, s->cap); s->err = b; return SPH_ENOMEM; }
    if (n > 0 && (!pos4 || !vel4)) { s->err = "pos4 / vel4 is NULL"; return SPH_EINVAL; }
    DeviceGuard dg(s);
    cudaStream_t st = s->stream;
    s->c.nf = (int)n; s->c.nown = n_owned;
    s->gf.n = (int)n;
    s->nblocks = cdiv(n > 0 ? n : 1, kBlock);
    if (n > 0) {
        CUDA_TRY(s, cudaMemcpyAsync(s->posA, pos4, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToDevice, st));
        CUDA_TRY(s, cudaMemcpyAsync(s->velA, vel4, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToDevice, st));
        LAUNCH(s, k_iota, cdiv(n, 256), 256, st, s->idA, (int)n);
    }
    // the list builder reads the SoA positions up to 3 elements past the last particle
    CUDA_TRY(s, cudaMemsetAsync(s->px + n, 0, 4 * sizeof(float), st));
    CUDA_TRY(s, cudaMemsetAsync(s->py + n, 0, 4 * sizeof(float), st));
    CUDA_TRY(s, cudaMemsetAsync(s->pz + n, 0, 4 * sizeof(float), st));
    s->derived_valid = false; s->vmax_valid = false;
    return SPH_OK;
}

int sph_slab_phase(SphSim *s, int phase)
{
    int rc = slab_check(s);
    if (rc) return rc;
    DeviceGuard dg(s);
    return s->prm.use_neighbor_list ? slab_phase_t<true>(s, phase) : slab_phase_t<false>(s, phase);
}

int sph_slab_gather(SphSim *s, int what, const int *orig_idx, int n, float *out4)
{
    int rc = slab_check(s);
    if (rc) return rc;
    if (n < 0 || (n > 0 && (!orig_idx || !out4)) || (what != SPH_SLAB_FIELD_KR && what != SPH_SLAB_FIELD_VEL)) { s->err = "sph_slab_gather: bad argument"; return SPH_EINVAL; }
    if (n == 0) return SPH_OK;
    DeviceGuard dg(s);
    const float4 *f = what == SPH_SLAB_FIELD_KR ? s->posk : &s->slab_vcur->v;
    LAUNCH(s, k_slab_gather, cdiv(n, 256), 256, s->stream, f, what == SPH_SLAB_FIELD_KR ? 1 : 2, s->inv, orig_idx, n, reinterpret_cast<float4 *>(out4));
    return SPH_OK;
}

int sph_slab_scatter(SphSim *s, int what, int first_orig, int n, const float *in4)
{
    int rc = slab_check(s);
    if (rc) return rc;
    if (n < 0 || first_orig < 0 || (long long)first_orig + n > s->c.nf || (n > 0 && !in4) || (what != SPH_SLAB_FIELD_KR && what != SPH_SLAB_FIELD_VEL)) { s->err = "sph_slab_scatter: bad argument"; return SPH_EINVAL; }
    if (n == 0) return SPH_OK;
    DeviceGuard dg(s);
    float4 *f = what == SPH_SLAB_FIELD_KR ? s->posk : &s->slab_vcur->v;
    LAUNCH(s, k_slab_scatter, cdiv(n, 256), 256, s->stream, f, what == SPH_SLAB_FIELD_KR ? 1 : 2, s->inv, first_orig, n, reinterpret_cast<const float4 *>(in4));
    return SPH_OK;
}

int sph_slab_read_error_sum(SphSim *s, unsigned long long *total)
{
    int rc = slab_check(s);
    if (rc) return rc;
    if (!total) return SPH_EINVAL;
    DeviceGuard dg(s);
    unsigned long long *h = reinterpret_cast<unsigned long long *>(s->pinned + 8);
    *h = 0ull;
    if (s->c.nf > 0) {
        CUDA_TRY(s, cudaMemcpyAsync(h, &s->ctl->last_total, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    }
    *total = *h;
    return SPH_OK;
}

int sph_slab_set_loop(SphSim *s, int mode, int cont, int it, float err)
{
    int rc = slab_check(s);
    if (rc) return rc;
    DeviceGuard dg(s);
    LAUNCH(s, k_slab_set_loop, 1, 1, s->stream, s->ctl, s->stats, mode, cont, it, err);
    return SPH_OK;
}

int sph_slab_store(SphSim *s, const float **pos4, const float **vel4, const int **orig_idx, int *n, int *n_owned)
{
    if (!s) return SPH_EINVAL;
    if (pos4) *pos4 = reinterpret_cast<const float *>(s->posA);
    if (vel4) *vel4 = reinterpret_cast<const float *>(s->velA);
    if (orig_idx) *orig_idx = s->idA;
    if (n) *n = s->c.nf;
    if (n_owned) *n_owned = s->c.nown;
    return SPH_OK;
}

int sph_select_range(void *cuda_stream, const float *pos4, const float *vel4, const int *gid, const int *key, int key_lt,
                     int n, float x_lo, float x_hi, float *out_pos4, float *out_vel4, int *out_gid, int *out_idx,
                     int max_out, int *scratch, size_t scratch_ints, int *count_host)
{
    if (n < 0 || max_out < 0 || !scratch || !count_host || (reinterpret_cast<uintptr_t>(scratch) & 15) != 0) return SPH_EINVAL;
    *count_host = 0;
    if (n == 0) return SPH_OK;
    if (!pos4 || !vel4 || !gid || (max_out > 0 && (!out_pos4 || !out_vel4 || !out_gid))) return SPH_EINVAL;
    const int ntiles = cdiv((long long)n + 1, kScanTile);
    const size_t flag_len = ((size_t)n + 1 + 3) & ~size_t(3);
    if (scratch_ints < flag_len + (size_t)ntiles + 4) return SPH_ENOMEM;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int *flag = scratch, *tiles = scratch + flag_len;
    k_select_flag<<<cdiv((long long)n + 1, 256), 256, 0, st>>>(reinterpret_cast<const float4 *>(pos4), key, key_lt, n, x_lo, x_hi, flag);
    k_scan_tile_sums<<<ntiles, kScanThreads, 0, st>>>(flag, n + 1, tiles);
    k_scan_apply<<<ntiles, kScanThreads, 0, st>>>(flag, n + 1, tiles);
    if (max_out > 0)
        k_select_copy<<<cdiv(n, 256), 256, 0, st>>>(reinterpret_cast<const float4 *>(pos4), reinterpret_cast<const float4 *>(vel4), gid, key,
                                                  flag, n, reinterpret_cast<float4 *>(out_pos4), reinterpret_cast<float4 *>(out_vel4), out_gid, out_idx, max_out);
    if (cudaMemcpyAsync(count_host, flag + n, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess) return SPH_ECUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return SPH_ECUDA;
    return cudaGetLastError() == cudaSuccess ? SPH_OK : SPH_ECUDA;
}

}  // extern "C"

// ---- sph_select_range_static: the selection for callers that may not allocate.  Its flag / scan scratch lives in the
// library image: one copy per GPU that loads it, held until the process exits.  In HOST code `g_select_scratch` is only
// a stand-in for the symbol (not a device address): the per-device address comes from cudaGetSymbolAddress, looked up
// once per device with that device current, and is what the kernels get.
constexpr size_t kSelectStaticInts = (size_t)SPH_SELECT_STATIC_MAX + 1024;      // n + 1 flags (padded to 4) + tile sums + 4
static __device__ __align__(256) int g_select_scratch[kSelectStaticInts];
namespace {
constexpr int kMaxDevices = 64;
int *g_select_scratch_dev[kMaxDevices] = {};       // device address of g_select_scratch on device d (NULL: not looked up yet)
std::mutex g_select_scratch_mutex;

// address of the CURRENT device's copy of the array; no allocation (the array is part of the loaded module)
int select_scratch_address(int **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { g_create_error = std::string("sph_select_range_static: cudaGetDevice failed: ") + cudaGetErrorString(e); return SPH_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) { g_create_error = "sph_select_range_static: device ordinal beyond 63"; return SPH_EINVAL; }
    std::lock_guard<std::mutex> lock(g_select_scratch_mutex);
    if (!g_select_scratch_dev[dev]) {
        int *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_select_scratch);
        if (e != cudaSuccess || !ptr) {
            g_create_error = std::string("sph_select_range_static: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e);
            return SPH_ECUDA;
        }
        g_select_scratch_dev[dev] = ptr;
    }
    *out = g_select_scratch_dev[dev];
    return SPH_OK;
}
}  // namespace
extern "C" {

int sph_select_range_static(void *cuda_stream, const float *pos4, const float *vel4, const int *gid, const int *key, int key_lt,
                            int n, float x_lo, float x_hi, float *out_pos4, float *out_vel4, int *out_gid, int *out_idx,
                            int max_out, int *count_host)
{
    if (!count_host) return SPH_EINVAL;
    *count_host = 0;
    if (n > SPH_SELECT_STATIC_MAX) {
        char b[160];
        snprintf(b, sizeof b, "sph_select_range_static: n = %d exceeds SPH_SELECT_STATIC_MAX = %d (use sph_select_range with caller scratch)",
                 n, (int)SPH_SELECT_STATIC_MAX);
        g_create_error = b;
        return SPH_EINVAL;
    }
    int *scratch = nullptr;
    const int rc = select_scratch_address(&scratch);
    if (rc) return rc;
    // the existing path, unchanged, on the library's own scratch: flag[0 .. n] and the tile sums are written by this
    // call's first two kernels before anything reads them, so the array's stale contents never matter
    return sph_select_range(cuda_stream, pos4, vel4, gid, key, key_lt, n, x_lo, x_hi, out_pos4, out_vel4, out_gid, out_idx,
                            max_out, scratch, kSelectStaticInts, count_host);
}

int sph_set_forced_iterations(SphSim *s, int forced_v, int forced_d, int forced_cg)
{
    if (!s) return SPH_EINVAL;
    DeviceGuard dg(s);
    // the three ints are the first members of DevControl
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    s->pinned[0] = forced_v; s->pinned[1] = forced_d; s->pinned[2] = forced_cg;
    CUDA_TRY(s, cudaMemcpyAsync(s->ctl, s->pinned, 3 * sizeof(int), cudaMemcpyHostToDevice, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return SPH_OK;
}

int sph_read_state(SphSim *s, int field, void *dst, size_t bytes, int is_host)
{
    if (!s) return SPH_EINVAL;
    FieldInfo fi;
    if (!field_info(s, field, fi)) { s->err = "unknown field"; return SPH_EINVAL; }
    if (bytes != fi.bytes) { char b[128]; snprintf(b, sizeof b, "field %d is %zu bytes, caller passed %zu", field, fi.bytes, bytes); s->err = b; return SPH_EINVAL; }
    if (bytes > 0 && !dst) { s->err = "dst is NULL"; return SPH_EINVAL; }
    if (fi.derived && !s->derived_valid) { s->err = "field is stale: call sph_build_grid or a step first"; return SPH_ESTATE; }
    DeviceGuard dg(s);
    // pending boundary / body writes become visible to reads as well (samples re-posed, Psi recomputed)
    // a pending asynchronous write of an array this read touches has to land first (reads of other arrays overlap it)
    if (s->pending_writes & write_mask(field)) { int rc = join_writes(s); if (rc) return rc; }
    if (s->boundary_dirty && field >= SPH_FIELD_BOUNDARY_POS) { int rc = refresh_boundary(s); if (rc) return rc; }
    if (!is_host) return export_field(s, field, dst, bytes);
    if (bytes > s->staging_bytes) { s->err = "field too large for a host read; read it into a device buffer"; return SPH_EINVAL; }
    int rc = export_field(s, field, s->staging, bytes);
    if (rc) return rc;
    if (is_host == 2) {
        // asynchronous: the caller waits with sph_host_sync.  The copy goes out in chunks with an event behind each, so
        // that an asynchronous write of the same host buffer that follows directly can upload chunk k as soon as it has
        // arrived (both directions of the bus busy at once), instead of after the whole field
        CUDA_TRY(s, cudaEventRecord(s->ev_main, s->stream));           // the export kernel and all earlier work
        const size_t chunk = host_chunk_bytes(bytes);
        for (int k = 0; k < SphSim::kHostChunks; ++k) {
            const size_t off = (size_t)k * chunk, len = off < bytes ? (bytes - off < chunk ? bytes - off : chunk) : 0;
            if (len > 0) CUDA_TRY(s, cudaMemcpyAsync((char *)dst + off, (const char *)s->staging + off, len, cudaMemcpyDeviceToHost, s->stream));
            CUDA_TRY(s, cudaEventRecord(s->ev_chunk[k], s->stream));
        }
        s->last_read.dst = dst; s->last_read.bytes = bytes; s->last_read.seq = s->op_seq;
        return SPH_OK;
    }
    if (bytes > 0) CUDA_TRY(s, cudaMemcpyAsync(dst, s->staging, bytes, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return SPH_OK;
}

int sph_write_state(SphSim *s, int field, const void *src, size_t bytes, int is_host)
{
    if (!s) return SPH_EINVAL;
    FieldInfo fi;
    if (!field_info(s, field, fi) || !fi.writable) { s->err = "field is not writable"; return SPH_EINVAL; }
    if (bytes != fi.bytes) { char b[128]; snprintf(b, sizeof b, "field %d is %zu bytes, caller passed %zu", field, fi.bytes, bytes); s->err = b; return SPH_EINVAL; }
    if (bytes > 0 && !src) { s->err = "src is NULL"; return SPH_EINVAL; }
    DeviceGuard dg(s);
    int rc;
    if (is_host == 2) {
        // asynchronous host write on the copy stream: ordered after everything enqueued on the main stream so far
        // (earlier steps, and earlier asynchronous READS that may be filling `src`), beside what follows there
        if (bytes > s->staging_bytes) { s->err = "field too large for a host write"; return SPH_EINVAL; }
        if (field >= SPH_FIELD_BOUNDARY_POS && field != SPH_FIELD_KSUM_DIVERGENCE && field != SPH_FIELD_KSUM_DENSITY) { s->err = "asynchronous host writes are for the fluid fields"; return SPH_EINVAL; }
        if (bytes > 0 && src == s->last_read.dst && bytes == s->last_read.bytes && s->last_read.seq + 1 == s->op_seq) {
            // the buffer is the target of the asynchronous read enqueued by the previous call: upload chunk k behind
            // download chunk k (ev_main was recorded by that read, behind its export kernel and all earlier work)
            CUDA_TRY(s, cudaStreamWaitEvent(s->copy_stream, s->ev_main, 0));
            const size_t chunk = host_chunk_bytes(bytes);
            for (int k = 0; k < SphSim::kHostChunks; ++k) {
                const size_t off = (size_t)k * chunk, len = off < bytes ? (bytes - off < chunk ? bytes - off : chunk) : 0;
                CUDA_TRY(s, cudaStreamWaitEvent(s->copy_stream, s->ev_chunk[k], 0));
                if (len > 0) CUDA_TRY(s, cudaMemcpyAsync((char *)s->staging_in + off, (const char *)src + off, len, cudaMemcpyHostToDevice, s->copy_stream));
            }
        } else {
            CUDA_TRY(s, cudaEventRecord(s->ev_main, s->stream));
            CUDA_TRY(s, cudaStreamWaitEvent(s->copy_stream, s->ev_main, 0));
            if (bytes > 0) CUDA_TRY(s, cudaMemcpyAsync(s->staging_in, src, bytes, cudaMemcpyHostToDevice, s->copy_stream));
        }
        rc = import_field(s, field, s->staging_in, bytes, s->copy_stream);
        if (rc) return rc;
        CUDA_TRY(s, cudaEventRecord(s->ev_write, s->copy_stream));
        s->pending_writes |= write_mask(field);
        s->derived_valid = false;
        return SPH_OK;
    }
    if ((rc = join_writes(s))) return rc;
    if (is_host) {
        if (bytes > s->staging_bytes) { s->err = "field too large for a host write"; return SPH_EINVAL; }
        if (bytes > 0) CUDA_TRY(s, cudaMemcpyAsync(s->staging, src, bytes, cudaMemcpyHostToDevice, s->stream));
        rc = import_field(s, field, s->staging, bytes, s->stream);
        if (rc) return rc;
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    } else {
        rc = import_field(s, field, src, bytes, s->stream);
        if (rc) return rc;
    }
    s->derived_valid = false;
    return SPH_OK;
}

int sph_host_sync(SphSim *s)
{
    if (!s) return SPH_EINVAL;
    DeviceGuard dg(s);
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->copy_stream));
    return SPH_OK;
}

int sph_read_stats(SphSim *s, SphStats *o)
{
    if (!s || !o) return SPH_EINVAL;
    DeviceGuard dg(s);
    DevStats *h = reinterpret_cast<DevStats *>(s->pinned + 64);
    CUDA_TRY(s, cudaMemcpyAsync(h, s->stats, sizeof(DevStats), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    memset(o, 0, sizeof *o);
    o->steps_done = h->steps_done; o->total_it_v = h->total_it_v; o->total_it_d = h->total_it_d;
    o->total_cg_iters = h->total_cg;
    o->it_v = h->it_v; o->it_d = h->it_d; o->cg_iters = h->cg_iters;
    o->err_v = h->err_v; o->err_rho = h->err_rho; o->cg_residual = h->cg_residual;
    o->oob_count = h->oob; o->overflow_count = h->lc.overflow; o->nan_count = h->nan_count;
    o->max_iter_hit = h->max_iter_hit;
    o->dt_last = h->dt_last; o->sim_time = h->sim_time;
    unsigned vb = h->vmax_bits; float vm; memcpy(&vm, &vb, 4); o->v_max = vm;
    o->max_fluid_neighbors = h->lc.max_f; o->max_boundary_neighbors = h->lc.max_b;
    o->mean_fluid_neighbors = s->c.nf > 0 ? (float)((double)h->lc.sum_f / (double)s->c.nf) : 0.f;
    return SPH_OK;
}

long long sph_launch_count(SphSim *s)
{
    if (!s) return 0;
    long long n = s->misc_launches;
    if (s->prm.use_cuda_graph && (s->graph_steps[0] + s->graph_steps[1] + s->graph_steps[2]) > 0) {
        SphStats st;
        if (sph_read_stats(s, &st) != SPH_OK) return n;
        // loop bodies: iterations are only recorded per solver, not per method; a simulation
        // normally uses one method, so attribute them to the method that has run
        int m = s->graph_steps[0] > 0 ? 0 : (s->graph_steps[2] > 0 ? 2 : 1);
        n += s->graph_steps[0] * s->fixed_nodes[0] + s->graph_steps[1] * s->fixed_nodes[1] + s->graph_steps[2] * s->fixed_nodes[2];
        // the divergence and density loops are peeled: their WHILE bodies run (iterations - 1) times per step
        const long long steps = s->graph_steps[0] + s->graph_steps[1] + s->graph_steps[2];
        const long long body_v = st.total_it_v > steps ? st.total_it_v - steps : 0;
        const long long body_d = st.total_it_d > steps ? st.total_it_d - steps : 0;
        n += body_v * s->body_nodes[m][LOOP_DIV] + body_d * s->body_nodes[m][LOOP_DENS] +
             st.total_cg_iters * s->body_nodes[m][LOOP_CG];
    }
    return n;
}

int sph_enable_kernel_timing(SphSim *s, int enable)
{
    if (!s) return SPH_EINVAL;
    if (enable && s->prm.use_cuda_graph) { s->err = "kernel timing needs use_cuda_graph = 0 (events cannot bracket nodes of a loop body)"; return SPH_ESTATE; }
    s->timing = enable != 0;
    return SPH_OK;
}

int sph_read_kernel_times(SphSim *s, char *buf, size_t bytes)
{
    if (!s || !buf || bytes == 0) return SPH_EINVAL;
    DeviceGuard dg(s);
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    struct Acc { std::string name; long long n; double ms; };
    std::vector<Acc> acc;
    for (auto &t : s->timed) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t.a, t.b);
        std::string nm = t.name;
        // strip template arguments, parentheses and the namespace
        size_t lt = nm.find('<'); if (lt != std::string::npos) nm = nm.substr(0, lt);
        while (!nm.empty() && (nm[0] == '(' || nm[0] == ' ')) nm.erase(0, 1);
        bool found = false;
        for (auto &a : acc) if (a.name == nm) { a.n++; a.ms += ms; found = true; break; }
        if (!found) acc.push_back({ nm, 1, ms });
        s->event_pool.push_back(t.a); s->event_pool.push_back(t.b);
    }
    s->timed.clear();
    std::string out;
    for (auto &a : acc) { char line[160]; snprintf(line, sizeof line, "%s %lld %.6f\n", a.name.c_str(), a.n, a.ms); out += line; }
    if (out.size() + 1 > bytes) { s->err = "buffer too small"; return SPH_ENOMEM; }
    memcpy(buf, out.c_str(), out.size() + 1);
    return SPH_OK;
}

// ---- post-processing stage (sph_surface.cuh)
namespace {
struct SurfLayout { size_t field, count, tiles, total; long long nnodes, ncells; int ntiles; };
bool surf_layout(const SphSurfaceParams *p, SurfLayout &L)
{
    if (!p || p->dims[0] < 2 || p->dims[1] < 2 || p->dims[2] < 2 || !(p->cube_size > 0.f)) return false;
    L.nnodes = (long long)p->dims[0] * p->dims[1] * p->dims[2];
    L.ncells = (long long)(p->dims[0] - 1) * (p->dims[1] - 1) * (p->dims[2] - 1);
    if (L.nnodes > 2000000000LL) return false;
    L.ntiles = cdiv(L.ncells + 1, kScanTile);
    auto up = [](size_t b) { return (b + 255) & ~size_t(255); };
    L.field = 0;
    L.count = up((size_t)L.nnodes * sizeof(float));
    L.tiles = L.count + up(((size_t)L.ncells + 1 + 4) * sizeof(int));
    L.total = L.tiles + up((size_t)L.ntiles * sizeof(int));
    return true;
}
bool g_mc_table_ready[64] = { false };
}  // namespace

size_t sph_surface_workspace_bytes(const SphSurfaceParams *p)
{
    SurfLayout L;
    return surf_layout(p, L) ? L.total : 0;
}

int sph_surface_extract(SphSim *s, const SphSurfaceParams *sp, void *workspace, size_t workspace_bytes,
                        float *triangles, long long max_triangles, long long *n_triangles)
{
    if (!s) return SPH_EINVAL;
    SurfLayout L;
    if (!surf_layout(sp, L)) { s->err = "surface grid needs >= 2 nodes per axis, cube_size > 0 and < 2^31 nodes"; return SPH_EINVAL; }
    if (!workspace || workspace_bytes < L.total) { s->err = "surface workspace too small"; return SPH_ENOMEM; }
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) { s->err = "surface workspace must be 256-byte aligned"; return SPH_EINVAL; }
    if (max_triangles < 0 || (max_triangles > 0 && !triangles)) { s->err = "triangles is NULL"; return SPH_EINVAL; }
    if (!s->derived_valid) { s->err = "the surface is extracted from the sorted store of the last sph_build_grid / step: call sph_build_grid first"; return SPH_ESTATE; }
    DeviceGuard dg(s);
    cudaStream_t st = s->stream;
    { int rc = join_writes(s); if (rc) return rc; }
    if (s->device >= 0 && s->device < 64 && !g_mc_table_ready[s->device]) {
        unsigned char cnt[256], edg[256 * kMcMaxTris * 3];
        memset(edg, 0, sizeof edg);
        if (!mc_build_table(cnt, edg)) { s->err = "marching-cubes table generation failed"; return SPH_ESTATE; }
        CUDA_TRY(s, cudaMemcpyToSymbol(c_mc_count, cnt, sizeof cnt));
        CUDA_TRY(s, cudaMemcpyToSymbol(c_mc_edges, edg, sizeof edg));
        g_mc_table_ready[s->device] = true;
    }
    char *base = static_cast<char *>(workspace);
    float *phi = reinterpret_cast<float *>(base + L.field);
    int *count = reinterpret_cast<int *>(base + L.count);
    int *tiles = reinterpret_cast<int *>(base + L.tiles);
    SurfGrid sg;
    sg.gx = sp->grid_min[0]; sg.gy = sp->grid_min[1]; sg.gz = sp->grid_min[2]; sg.cs = sp->cube_size; sg.iso = sp->iso;
    sg.nx = sp->dims[0]; sg.ny = sp->dims[1]; sg.nz = sp->dims[2];
    LAUNCH(s, k_surface_field, cdiv(L.nnodes, kBlock), kBlock, st, s->c, sg, s->posB, s->rho, s->gf.cell_start, phi);
    LAUNCH(s, k_surface_classify, cdiv(L.ncells + 1, 256), 256, st, sg, phi, count, L.ncells);
    const int nscan = (int)(L.ncells + 1);
    LAUNCH(s, k_scan_tile_sums, L.ntiles, kScanThreads, st, count, nscan, tiles);
    LAUNCH(s, k_scan_apply, L.ntiles, kScanThreads, st, count, nscan, tiles);
    if (max_triangles > 0)
        LAUNCH(s, k_surface_emit, cdiv(L.ncells, 256), 256, st, sg, phi, count, L.ncells, triangles, max_triangles);
    if (n_triangles) {
        CUDA_TRY(s, cudaMemcpyAsync(s->pinned, count + L.ncells, sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(s, cudaStreamSynchronize(st));
        *n_triangles = s->pinned[0];
    }
    return SPH_OK;
}

}  // extern "C"
namespace {
// validates the camera and fills the kernel's view of it; false: invalid parameters
bool render_camera(const SphRenderParams *p, float default_radius, RenderCam &c)
{
    if (!p || p->width < 1 || p->height < 1 || !(p->pixel_size > 0.f) || (long long)p->width * p->height > 2000000000LL) return false;
    const double r[3] = { p->right[0], p->right[1], p->right[2] }, u[3] = { p->up[0], p->up[1], p->up[2] };
    const double rr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2], uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    const double ru = r[0] * u[0] + r[1] * u[1] + r[2] * u[2];
    if (!(std::fabs(rr - 1.0) <= 1e-4) || !(std::fabs(uu - 1.0) <= 1e-4) || !(std::fabs(ru) <= 1e-4)) return false;
    const double w[3] = { r[1] * u[2] - r[2] * u[1], r[2] * u[0] - r[0] * u[2], r[0] * u[1] - r[1] * u[0] };
    double l[3] = { p->light[0], p->light[1], p->light[2] };
    double ll = std::sqrt(l[0] * l[0] + l[1] * l[1] + l[2] * l[2]);
    if (!(ll == ll)) return false;
    if (ll == 0.0) { l[0] = w[0]; l[1] = w[1]; l[2] = w[2]; ll = std::sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]); }   // headlight
    const float R = p->radius > 0.f ? p->radius : default_radius;
    if (!(R > 0.f) || p->radius < 0.f) return false;
    c.ox = p->origin[0]; c.oy = p->origin[1]; c.oz = p->origin[2];
    c.rx = (float)r[0]; c.ry = (float)r[1]; c.rz = (float)r[2];
    c.ux = (float)u[0]; c.uy = (float)u[1]; c.uz = (float)u[2];
    c.wx = (float)w[0]; c.wy = (float)w[1]; c.wz = (float)w[2];
    c.lr = (float)((l[0] * r[0] + l[1] * r[1] + l[2] * r[2]) / ll);
    c.lu = (float)((l[0] * u[0] + l[1] * u[1] + l[2] * u[2]) / ll);
    c.lw = (float)((l[0] * w[0] + l[1] * w[1] + l[2] * w[2]) / ll);
    c.ps = p->pixel_size; c.inv_ps = 1.0f / p->pixel_size;
    c.R = R; c.R2 = R * R; c.inv_R = 1.0f / R;
    c.W = p->width; c.H = p->height;
    return true;
}
inline size_t render_keys_bytes(const SphRenderParams *p) { return (((size_t)p->width * (size_t)p->height * 8) + 255) & ~size_t(255); }
}  // namespace
extern "C" {

size_t sph_render_workspace_bytes(const SphRenderParams *p, int n_fluid)
{
    RenderCam c;
    if (n_fluid < 0 || !render_camera(p, 1.0f, c)) return 0;
    return render_keys_bytes(p) + ((((size_t)(n_fluid > 0 ? n_fluid : 1) * sizeof(int)) + 255) & ~size_t(255));
}

int sph_render_particles(SphSim *s, const SphRenderParams *p, void *workspace, size_t workspace_bytes,
                         float *depth, int *id, float *shade)
{
    if (!s) return SPH_EINVAL;
    RenderCam c;
    if (!render_camera(p, s->prm.particle_radius, c)) {
        s->err = "render: width, height, pixel_size must be positive, radius >= 0, right / up orthonormal (1e-4), light finite";
        return SPH_EINVAL;
    }
    const size_t need = sph_render_workspace_bytes(p, s->c.nf);
    if (!workspace || workspace_bytes < need) { s->err = "render workspace too small"; return SPH_ENOMEM; }
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) { s->err = "render workspace must be 256-byte aligned"; return SPH_EINVAL; }
    DeviceGuard dg(s);
    cudaStream_t st = s->stream;
    { int rc = join_writes(s); if (rc) return rc; }
    unsigned long long *keys = static_cast<unsigned long long *>(workspace);
    int *inv = reinterpret_cast<int *>(static_cast<char *>(workspace) + render_keys_bytes(p));
    const long long npix = (long long)c.W * c.H;
    const int nf = s->c.nf;
    const long long nclear = npix > nf ? npix : nf;
    LAUNCH(s, k_render_clear, cdiv(nclear, 256), 256, st, keys, npix, s->idA, nf, inv);
    if (nf > 0) LAUNCH(s, k_render_splat, cdiv(nf, 256), 256, st, c, s->posA, s->idA, nf, keys);
    LAUNCH(s, k_render_resolve, cdiv(npix, 256), 256, st, c, s->posA, inv, keys, depth, id, shade);
    return SPH_OK;
}

const char *sph_last_error(const SphSim *s) { return s ? s->err.c_str() : g_create_error.c_str(); }

void sph_destroy(SphSim *s)
{
    if (!s) return;
    DeviceGuard dg(s);
    cudaStreamSynchronize(s->stream);
    if (s->copy_stream) { cudaStreamSynchronize(s->copy_stream); cudaStreamDestroy(s->copy_stream); }
    if (s->ev_main) cudaEventDestroy(s->ev_main);
    if (s->ev_write) cudaEventDestroy(s->ev_write);
    for (int k = 0; k < SphSim::kHostChunks; ++k) if (s->ev_chunk[k]) cudaEventDestroy(s->ev_chunk[k]);
    for (int m = 0; m < 3; ++m) if (s->exec[m]) cudaGraphExecDestroy(s->exec[m]);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    if (s->pinned) cudaFreeHost(s->pinned);
    for (auto &t : s->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
    for (auto e : s->event_pool) cudaEventDestroy(e);
    delete s;
}

}  // extern "C"
