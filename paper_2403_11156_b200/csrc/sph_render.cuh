// sph_render.cuh -- particle image stage (reading R30 of DESIGN.md, optional part).
//
// The paper renders with a third-party path tracer and prints no equation; the stand-in is an
// orthographic sphere splat of the fluid particles into headless device buffers: per pixel the smallest depth
// t = z - sqrt(R^2 - dx^2 - dy^2) over the covering particles, the particle that attains it (smallest original id among
// equal depths) and a Lambert term.  Three kernels:
//   k_render_clear    keys = all ones (empty), inverse map original id -> slot of the persistent store
//   k_render_splat    one thread per particle: every pixel centre inside its disc gets atomicMin of the 64-bit key
//                     (order-preserving bits of the fp32 depth << 32 | original id) -- integer minimum, so the image does
//                     not depend on the order in which particles arrive, and equal depths resolve to the smallest id
//   k_render_resolve  one thread per pixel: key -> depth, id; normal and Lambert term recomputed from the winner
// Product code: shares nothing with oracle/render_ref.py.
#pragma once
#include "sph_common.cuh"

namespace sph {

struct RenderCam {
    float ox, oy, oz;       // origin
    float rx, ry, rz;       // right
    float ux, uy, uz;       // up
    float wx, wy, wz;       // view direction = right x up
    float lr, lu, lw;       // unit light direction in camera coordinates (l.right, l.up, l.w)
    float ps, inv_ps, R, R2, inv_R;
    int W, H;
};

// fp32 <-> 32-bit keys whose unsigned order is the order of the floats (negative depths: camera inside the scene)
__device__ __forceinline__ unsigned depth_key(float t)
{
    const unsigned b = __float_as_uint(t);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key_depth(unsigned k)
{
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// camera coordinates of a point: separate subtractions, then fused dot products (fixed association)
__device__ __forceinline__ void cam_coords(const RenderCam &c, float x, float y, float z, float &a, float &b, float &d)
{
    const float px = x - c.ox, py = y - c.oy, pz = z - c.oz;
    a = fmaf(pz, c.rz, fmaf(py, c.ry, px * c.rx));
    b = fmaf(pz, c.uz, fmaf(py, c.uy, px * c.ux));
    d = fmaf(pz, c.wz, fmaf(py, c.wy, px * c.wx));
}

__global__ void __launch_bounds__(256)
k_render_clear(unsigned long long *__restrict__ keys, long long npix, const int *__restrict__ id, int n, int *__restrict__ inv)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < npix) keys[t] = ~0ull;
    if (t < n) inv[id[t]] = (int)t;
}

__global__ void __launch_bounds__(256)
k_render_splat(RenderCam c, const float4 *__restrict__ pos, const int *__restrict__ id, int n, unsigned long long *__restrict__ keys)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 x = pos[i];
    float a, b, z;
    cam_coords(c, x.x, x.y, x.z, a, b, z);
    if (!(a == a) || !(b == b) || !(z == z)) return;                    // NaN positions draw nothing
    // pixel centres (p + 1/2) ps within R of (a, b), one pixel of slack against rounding; the exact test is q > 0
    const float fx0 = floorf((a - c.R) * c.inv_ps - 0.5f) , fx1 = ceilf((a + c.R) * c.inv_ps - 0.5f);
    const float fy0 = floorf((b - c.R) * c.inv_ps - 0.5f) , fy1 = ceilf((b + c.R) * c.inv_ps - 0.5f);
    if (fx1 < 0.f || fy1 < 0.f || fx0 > (float)(c.W - 1) || fy0 > (float)(c.H - 1)) return;
    const int x0 = (int)fmaxf(fx0, 0.f), x1 = (int)fminf(fx1, (float)(c.W - 1));
    const int y0 = (int)fmaxf(fy0, 0.f), y1 = (int)fminf(fy1, (float)(c.H - 1));
    const unsigned long long low = (unsigned long long)(unsigned)id[i];
    for (int py = y0; py <= y1; ++py) {
        const float dy = ((float)py + 0.5f) * c.ps - b;
        const float qy = fmaf(-dy, dy, c.R2);
        if (!(qy > 0.f)) continue;
        for (int px = x0; px <= x1; ++px) {
            const float dx = ((float)px + 0.5f) * c.ps - a;
            const float q = fmaf(-dx, dx, qy);
            if (q > 0.f) {
                const float t = z - sqrtf(q);
                atomicMin(&keys[(size_t)py * c.W + px], ((unsigned long long)depth_key(t) << 32) | low);
            }
        }
    }
}

__global__ void __launch_bounds__(256)
k_render_resolve(RenderCam c, const float4 *__restrict__ pos, const int *__restrict__ inv,
                 const unsigned long long *__restrict__ keys, float *__restrict__ depth, int *__restrict__ id_out,
                 float *__restrict__ shade)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)c.W * c.H) return;
    const unsigned long long k = keys[t];
    float d = __uint_as_float(0x7f800000u), sh = 0.f;
    int pid = -1;
    if (k != ~0ull) {
        pid = (int)(unsigned)(k & 0xffffffffull);
        d = key_depth((unsigned)(k >> 32));
        const int px = (int)(t % c.W), py = (int)(t / c.W);
        const float4 x = pos[inv[pid]];
        float a, b, z;
        cam_coords(c, x.x, x.y, x.z, a, b, z);
        const float dx = ((float)px + 0.5f) * c.ps - a, dy = ((float)py + 0.5f) * c.ps - b;
        const float s = sqrtf(fmaxf(fmaf(-dx, dx, fmaf(-dy, dy, c.R2)), 0.f));
        sh = fmaxf(0.f, -(fmaf(dx, c.lr, fmaf(dy, c.lu, -s * c.lw)) * c.inv_R));
    }
    if (depth) depth[t] = d;
    if (id_out) id_out[t] = pid;
    if (shade) shade[t] = sh;
}

}  // namespace sph
