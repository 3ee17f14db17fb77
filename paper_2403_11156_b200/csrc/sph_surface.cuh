// sph_surface.cuh -- post-processing stage as CUDA kernels (section 4.3: the paper
// hands its particles to an external surface-reconstruction tool and prints no equations -- reading R29 of DESIGN.md):
//   field    phi(g) = sum_i V_i W(|g - x_i|, h), V_i = m / rho_i, on the nodes g = grid_min + (ix, iy, iz) * cube_size
//            (node coordinates in fp32: one multiply, one add), gathered per node through the simulation's sorted
//            particle store and cell grid -- deterministic, no atomics;
//   surface  marching cubes on the cells of that grid: corner c = dx + 2 dy + 4 dz is inside when phi > iso; vertices
//            by linear interpolation from the edge's lower-index corner; triangles from a 256-entry case table that
//            is GENERATED at start-up by tracing, on each cube face, the segments between its crossing edges (four
//            crossings: the two edges next to each inside corner are paired, a rule that depends on the face's corner
//            signs only, so neighbouring cells agree and the mesh is watertight), closing them into loops oriented with
//            the normals out of the fluid, and fan-triangulating every loop from its smallest edge id.
// Three launches + the grid builder's scan: classify + count, exclusive scan, emit (triangle soup in cell order).
// Product code: shares nothing with oracle/surface_ref.py.
#pragma once
#include "sph_passes.cuh"

namespace sph {

constexpr int kMcMaxTris = 5;
__constant__ unsigned char c_mc_count[256];
__constant__ unsigned char c_mc_edges[256 * kMcMaxTris * 3];
// edge e joins corners c_mc_ea[e] < c_mc_eb[e]: 4 edges along x, 4 along y, 4 along z
__constant__ unsigned char c_mc_ea[12] = { 0, 2, 4, 6, 0, 1, 4, 5, 0, 1, 2, 3 };
__constant__ unsigned char c_mc_eb[12] = { 1, 3, 5, 7, 2, 3, 6, 7, 4, 5, 6, 7 };

// Host: the case table.  Returns false if a case needs more than kMcMaxTris triangles (cannot happen with this rule).
inline bool mc_build_table(unsigned char count[256], unsigned char edges[256 * kMcMaxTris * 3])
{
    static const int ea[12] = { 0, 2, 4, 6, 0, 1, 4, 5, 0, 1, 2, 3 }, eb[12] = { 1, 3, 5, 7, 2, 3, 6, 7, 4, 5, 6, 7 };
    auto edge_of = [&](int a, int b) { if (a > b) { int t = a; a = b; b = t; } for (int e = 0; e < 12; ++e) if (ea[e] == a && eb[e] == b) return e; return -1; };
    // faces: corners counter-clockwise seen from outside
    int face[6][4];
    int nfc = 0;
    for (int axis = 0; axis < 3; ++axis) {
        const int u = (axis + 1) % 3, v = (axis + 2) % 3;
        for (int side = 0; side < 2; ++side) {
            static const int ab[4][2] = { { 0, 0 }, { 1, 0 }, { 1, 1 }, { 0, 1 } };
            int cyc[4];
            for (int k = 0; k < 4; ++k) {
                int d[3] = { 0, 0, 0 };
                d[axis] = side; d[u] = ab[k][0]; d[v] = ab[k][1];
                cyc[k] = d[0] + 2 * d[1] + 4 * d[2];
            }
            for (int k = 0; k < 4; ++k) face[nfc][k] = side ? cyc[k] : cyc[3 - k];
            ++nfc;
        }
    }
    for (int mask = 0; mask < 256; ++mask) {
        int next[12];
        for (int e = 0; e < 12; ++e) next[e] = -1;
        for (int f = 0; f < 6; ++f) {
            const int *cyc = face[f];
            for (int k = 0; k < 4; ++k) {
                const int c = cyc[k], cp = cyc[(k + 3) & 3];
                if (!((mask >> c) & 1) || ((mask >> cp) & 1)) continue;      // runs of inside corners start after an outside one
                int kk = k;
                while (((mask >> cyc[(kk + 1) & 3]) & 1) && ((kk + 1) & 3) != k) kk = (kk + 1) & 3;
                const int after = cyc[(kk + 1) & 3];
                if ((mask >> after) & 1) continue;
                next[edge_of(cp, c)] = edge_of(cyc[kk], after);              // around the inside corners, counter-clockwise
            }
        }
        bool seen[12] = { false };
        int n = 0;
        for (int s = 0; s < 12; ++s) {
            if (next[s] < 0 || seen[s]) continue;
            int loop[12], len = 0;
            for (int e = s; !seen[e]; e = next[e]) { seen[e] = true; loop[len++] = e; }
            for (int k = 1; k + 1 < len; ++k) {
                if (n >= kMcMaxTris) return false;
                edges[(mask * kMcMaxTris + n) * 3 + 0] = (unsigned char)loop[0];
                edges[(mask * kMcMaxTris + n) * 3 + 1] = (unsigned char)loop[k];
                edges[(mask * kMcMaxTris + n) * 3 + 2] = (unsigned char)loop[k + 1];
                ++n;
            }
        }
        count[mask] = (unsigned char)n;
    }
    return true;
}

struct SurfGrid {
    float gx, gy, gz, cs, iso;
    int nx, ny, nz;                 // nodes per axis
};
__device__ __forceinline__ float node_coord(float g0, int i, float cs) { return __fadd_rn(g0, __fmul_rn((float)i, cs)); }

// field on every node (x-fastest): one thread per node walks the 27 cells around it (the node is treated like a
// particle position: same cell arithmetic, same fp32 distance predicate, strict |g - x| < h)
__global__ void __launch_bounds__(kBlock)
k_surface_field(SimConst c, SurfGrid sg, const float4 *__restrict__ pos, const float *__restrict__ rho,
                const int *__restrict__ fcs, float *__restrict__ phi)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nn = (long long)sg.nx * sg.ny * sg.nz;
    if (t >= nn) return;
    const int ix = (int)(t % sg.nx), iy = (int)((t / sg.nx) % sg.ny), iz = (int)(t / ((long long)sg.nx * sg.ny));
    const float x = node_coord(sg.gx, ix, sg.cs), y = node_coord(sg.gy, iy, sg.cs), z = node_coord(sg.gz, iz, sg.cs);
    const CellOf cell = cell_of(c.g, x, y, z);
    float sum = 0.f;
    for_each_candidate(c.g, fcs, cell, [&](int j, int, int) {
        const float4 q = __ldg(pos + j);
        const float dx = __fsub_rn(x, q.x), dy = __fsub_rn(y, q.y), dz = __fsub_rn(z, q.z);
        const float d2 = dist2_r10(dx, dy, dz);
        if (d2 < c.h2) {
            float r, rinv;
            r_and_rinv(d2, r, rinv);
            sum = fmaf(c.m / __ldg(rho + j), spline_w(r * c.inv_h), sum);
        }
    });
    phi[t] = c.sigma * sum;
}

__device__ __forceinline__ int mc_case(const SurfGrid &sg, const float *__restrict__ phi, int ix, int iy, int iz, float f[8])
{
    int mask = 0;
#pragma unroll
    for (int cidx = 0; cidx < 8; ++cidx) {
        const size_t n = (size_t)(ix + (cidx & 1)) + (size_t)sg.nx * ((size_t)(iy + ((cidx >> 1) & 1)) + (size_t)sg.ny * (size_t)(iz + (cidx >> 2)));
        f[cidx] = __ldg(phi + n);
        mask |= (f[cidx] > sg.iso ? 1 : 0) << cidx;
    }
    return mask;
}

// triangles per cell (cells x-fastest over (nx-1)(ny-1)(nz-1)); count[ncells] = 0 so that the scan's last entry is the total
__global__ void __launch_bounds__(256)
k_surface_classify(SurfGrid sg, const float *__restrict__ phi, int *__restrict__ count, long long ncells)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t > ncells) return;
    if (t == ncells) { count[t] = 0; return; }
    const int cx = sg.nx - 1, cy = sg.ny - 1;
    const int ix = (int)(t % cx), iy = (int)((t / cx) % cy), iz = (int)(t / ((long long)cx * cy));
    float f[8];
    count[t] = c_mc_count[mc_case(sg, phi, ix, iy, iz, f)];
}

// triangle soup: 9 floats per triangle at offset[cell]; triangles past max_tris are dropped (the total is still reported)
__global__ void __launch_bounds__(256)
k_surface_emit(SurfGrid sg, const float *__restrict__ phi, const int *__restrict__ offset, long long ncells,
               float *__restrict__ tris, long long max_tris)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncells) return;
    const int first = offset[t], n = offset[t + 1] - first;
    if (n == 0) return;
    const int cx = sg.nx - 1, cy = sg.ny - 1;
    const int ix = (int)(t % cx), iy = (int)((t / cx) % cy), iz = (int)(t / ((long long)cx * cy));
    float f[8];
    const int mask = mc_case(sg, phi, ix, iy, iz, f);
    for (int k = 0; k < n; ++k) {
        if ((long long)first + k >= max_tris) return;
        float *o = tris + ((size_t)first + k) * 9;
#pragma unroll
        for (int v = 0; v < 3; ++v) {
            const int e = c_mc_edges[(mask * kMcMaxTris + k) * 3 + v];
            const int a = c_mc_ea[e], b = c_mc_eb[e];
            const float s = (sg.iso - f[a]) / (f[b] - f[a]);
            const float ax = node_coord(sg.gx, ix + (a & 1), sg.cs), ay = node_coord(sg.gy, iy + ((a >> 1) & 1), sg.cs),
                        az = node_coord(sg.gz, iz + (a >> 2), sg.cs);
            const float bx = node_coord(sg.gx, ix + (b & 1), sg.cs), by = node_coord(sg.gy, iy + ((b >> 1) & 1), sg.cs),
                        bz = node_coord(sg.gz, iz + (b >> 2), sg.cs);
            o[3 * v + 0] = __fmaf_rn(s, __fsub_rn(bx, ax), ax);
            o[3 * v + 1] = __fmaf_rn(s, __fsub_rn(by, ay), ay);
            o[3 * v + 2] = __fmaf_rn(s, __fsub_rn(bz, az), az);
        }
    }
}

}  // namespace sph
