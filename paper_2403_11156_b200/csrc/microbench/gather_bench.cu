// gather_bench.cu -- stand-alone microbenchmark behind DESIGN.md section 6: what does the bare
// neighbour gather of a list pass cost on this GPU, and do the alternatives pay?
//
// Not part of libsph_b200 and not used by any test: it only measures memory-access patterns on
// synthetic index lists with the structure of the real ones (8 particles per cell, 9 x-runs of 3
// cells, ~29 neighbours per particle picked at random inside the runs, lists warp-tiled and padded
// to the warp maximum).  No SPH arithmetic.  Build and run:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o gather_bench gather_bench.cu && ./gather_bench
#include <cuda_runtime.h>
#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <random>
#include <vector>

constexpr int PPC = 8, NX = 100, NY = 75, NZ = 20, NC = NX * NY * NZ, N = NC * PPC;   // 1.2M particles
constexpr int B = 128;

struct __align__(32) Rec { float4 a, b; };

__device__ __forceinline__ void ldg256(const void *p, float4 &a, float4 &b)
{
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// MODE 0: one 16-byte array; 1: two 16-byte arrays; 2: one 32-byte record array, 256-bit load;
//      3: 16 bytes out of 32-byte records
template <int MODE>
__global__ void __launch_bounds__(B) k_global(const int *__restrict__ nl, const int *__restrict__ wslots,
        const size_t *__restrict__ woff, const float4 *__restrict__ pos, const float4 *__restrict__ vel,
        const Rec *__restrict__ rec, float4 *out, int n)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x; if (i >= n) return;
    int w = i >> 5, ns = wslots[w];
    const int *lp = nl + woff[w] + (i & 31);
    float sx = 0, sy = 0, sz = 0, sw = 0;
#pragma unroll 1
    for (int k0 = 0; k0 < ns; k0 += 4) {
        int j[4]; float4 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) j[u] = __ldg(lp + (k0 + u) * 32);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (MODE == 0) { a[u] = __ldg(pos + j[u]); b[u] = a[u]; }
            if (MODE == 1) { a[u] = __ldg(pos + j[u]); b[u] = __ldg(vel + j[u]); }
            if (MODE == 2) ldg256(rec + j[u], a[u], b[u]);
            if (MODE == 3) { a[u] = __ldg(&rec[j[u]].a); b[u] = a[u]; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) { sx += a[u].x * b[u].x; sy += a[u].y * b[u].y; sz += a[u].z * b[u].z; sw += a[u].w * b[u].w; }
    }
    out[i] = make_float4(sx, sy, sz, sw);
}

// candidate tile of the CTA (9 contiguous index ranges) bulk-copied to shared memory, gathers with LDS.128
// through 16-bit tile-relative entries
__global__ void __launch_bounds__(B) k_smem(const uint32_t *__restrict__ nl16, const int *__restrict__ cnt, int kf,
        const float4 *__restrict__ pos, float4 *out, int n, int skip_copy)
{
    extern __shared__ __align__(128) char sm[];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ int rs[9], rn[9];
    int i0 = blockIdx.x * B, i = i0 + threadIdx.x, ilast = min(i0 + B - 1, n - 1);
    if (threadIdx.x < 9) {
        int r = threadIdx.x, ca = i0 / PPC, cb = ilast / PPC, off = NX * ((r % 3 - 1) + NY * (r / 3 - 1));
        long lo = max((long)ca + off - 1, 0L), hi = min((long)cb + off + 1, (long)NC - 1);
        rs[r] = hi >= lo ? (int)lo * PPC : 0; rn[r] = hi >= lo ? ((int)hi + 1) * PPC - rs[r] : 0;
        if (skip_copy) rn[r] = r == 0 ? 16 : 0;
    }
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&bar)));
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0; for (int r = 0; r < 9; ++r) tot += rn[r];
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(&bar)), "r"(tot * 16));
        int o = 0;
        for (int r = 0; r < 9; ++r) if (rn[r] > 0) {
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                :: "r"(smem_u32(sm + (size_t)o * 16)), "l"(pos + rs[r]), "r"(rn[r] * 16), "r"(smem_u32(&bar)) : "memory");
            o += rn[r];
        }
    }
    int c = i < n ? cnt[i] : 0, npair = (c + 1) >> 1;
    const uint32_t *lp = nl16 + (size_t)(i >> 5) * (kf / 2) * 32 + (i & 31);
    uint32_t ok = 0;
    while (!ok) asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0,1,0,p; }" : "=r"(ok) : "r"(smem_u32(&bar)) : "memory");
    float sx = 0, sy = 0, sz = 0, sw = 0;
    // list words software-pipelined exactly like the library's list passes
    constexpr int PB = 4;
    uint32_t cur[PB];
#pragma unroll
    for (int t = 0; t < PB; ++t) cur[t] = t < npair ? __ldg(lp + t * 32) : 0u;
#pragma unroll 1
    for (int pb = 0; pb < npair; pb += PB) {
        uint32_t nxt[PB];
#pragma unroll
        for (int t = 0; t < PB; ++t) nxt[t] = pb + PB + t < npair ? __ldg(lp + (pb + PB + t) * 32) : 0u;
        float4 a[2 * PB];
#pragma unroll
        for (int u = 0; u < 2 * PB; ++u) {
            uint32_t e = (u & 1) ? (cur[u >> 1] >> 16) : (cur[u >> 1] & 0xffffu);
            a[u] = *reinterpret_cast<const float4 *>(sm + (size_t)e * 16);
        }
#pragma unroll
        for (int u = 0; u < 2 * PB; ++u) if (2 * pb + u < c) { sx += a[u].x; sy += a[u].y; sz += a[u].z; sw += a[u].w; }
#pragma unroll
        for (int t = 0; t < PB; ++t) cur[t] = nxt[t];
    }
    if (i < n) out[i] = make_float4(sx, sy, sz, sw);
}

template <class F> static float best_of(F &&launch)
{
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0); launch(); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    return best * 1e3f;
}

int main()
{
    const int NW = (N + 31) / 32, nb = (N + B - 1) / B, kf = 64;
    std::mt19937 rng(1);
    // neighbours of every particle, per x-run
    std::vector<std::vector<int>> nbr((size_t)N * 9);
    for (int i = 0; i < N; ++i) {
        int c = i / PPC, cx = c % NX, cy = (c / NX) % NY, cz = c / (NX * NY);
        for (int r = 0; r < 9; ++r) {
            int y = cy + r % 3 - 1, z = cz + r / 3 - 1; if (y < 0 || y >= NY || z < 0 || z >= NZ) continue;
            int x0 = std::max(cx - 1, 0), x1 = std::min(cx + 1, NX - 1);
            int s = ((z * NY + y) * NX + x0) * PPC, e = ((z * NY + y) * NX + x1 + 1) * PPC;
            float p = r == 4 ? 0.30f : ((r % 3 == 1 || r / 3 == 1) ? 0.16f : 0.07f);
            for (int j = s; j < e; ++j) if (j != i && (rng() & 0xffff) < p * 65536) nbr[(size_t)i * 9 + r].push_back(j);
        }
    }
    float4 *dpos, *dvel, *dout; Rec *drec; int *dws; size_t *dwo;
    cudaMalloc(&dpos, (size_t)N * 16); cudaMalloc(&dvel, (size_t)N * 16); cudaMalloc(&dout, (size_t)N * 16);
    cudaMalloc(&drec, (size_t)N * 32); cudaMalloc(&dws, NW * 4); cudaMalloc(&dwo, NW * 8);
    cudaMemset(dpos, 0, (size_t)N * 16); cudaMemset(dvel, 0, (size_t)N * 16); cudaMemset(drec, 0, (size_t)N * 32);
    // ---- global gathers: flat list (1 group) and per-run / per-layer padded lists (9 / 3 groups)
    for (int ng : { 1, 9, 3 }) {
        std::vector<int> ws(NW), nl; std::vector<size_t> wo(NW); size_t tot = 0; double slots = 0;
        for (int w = 0; w < NW; ++w) {
            std::vector<std::vector<int>> lane(32); int total = 0;
            for (int g = 0; g < ng; ++g) {
                int mx = 0; std::vector<std::vector<int>> seg(32);
                for (int l = 0; l < 32; ++l) { int i = w * 32 + l; if (i >= N) continue;
                    for (int r = 0; r < 9; ++r) { int gg = ng == 1 ? 0 : (ng == 9 ? r : r / 3); if (gg != g) continue;
                        for (int j : nbr[(size_t)i * 9 + r]) seg[l].push_back(j); }
                    mx = std::max(mx, (int)seg[l].size()); }
                for (int l = 0; l < 32; ++l) { int i = std::min(w * 32 + l, N - 1);
                    while ((int)seg[l].size() < mx) seg[l].push_back(i);
                    for (int j : seg[l]) lane[l].push_back(j); }
                total += mx;
            }
            int padded = (total + 3) / 4 * 4;
            for (int l = 0; l < 32; ++l) { int i = std::min(w * 32 + l, N - 1); while ((int)lane[l].size() < padded) lane[l].push_back(i); }
            ws[w] = padded; wo[w] = tot; nl.resize(tot + (size_t)padded * 32);
            for (int k = 0; k < padded; ++k) for (int l = 0; l < 32; ++l) nl[tot + (size_t)k * 32 + l] = lane[l][k];
            tot += (size_t)padded * 32; slots += padded;
        }
        int *dnl; cudaMalloc(&dnl, nl.size() * 4); cudaMemcpy(dnl, nl.data(), nl.size() * 4, cudaMemcpyHostToDevice);
        cudaMemcpy(dws, ws.data(), NW * 4, cudaMemcpyHostToDevice); cudaMemcpy(dwo, wo.data(), NW * 8, cudaMemcpyHostToDevice);
        printf("list padded in %d group(s): %.1f slots per warp\n", ng, slots / NW);
        printf("  one 16-byte array                 %7.1f us\n", best_of([&] { k_global<0><<<nb, B>>>(dnl, dws, dwo, dpos, dvel, drec, dout, N); }));
        if (ng == 1) {
            printf("  two 16-byte arrays                %7.1f us\n", best_of([&] { k_global<1><<<nb, B>>>(dnl, dws, dwo, dpos, dvel, drec, dout, N); }));
            printf("  one 32-byte record, 256-bit load  %7.1f us\n", best_of([&] { k_global<2><<<nb, B>>>(dnl, dws, dwo, dpos, dvel, drec, dout, N); }));
            printf("  16 bytes out of 32-byte records   %7.1f us\n", best_of([&] { k_global<3><<<nb, B>>>(dnl, dws, dwo, dpos, dvel, drec, dout, N); }));
        }
        cudaFree(dnl);
    }
    // ---- shared-memory staged tile, 16-bit tile-relative entries; cf = 1: entries nudged so that the 8 lanes
    // of a quarter-warp always hit 8 different 16-byte bank groups (what a conflict-free schedule would give)
    for (int cf = 0; cf < 2; ++cf) {
        std::vector<uint16_t> nl16((size_t)NW * kf * 32, 0); std::vector<int> cnt(N); double staged = 0;
        for (int b = 0; b < nb; ++b) {
            int i0 = b * B, il = std::min(i0 + B - 1, N - 1), ca = i0 / PPC, cb = il / PPC, rs[9], rn[9], pre[9], o = 0;
            for (int r = 0; r < 9; ++r) { int off = NX * ((r % 3 - 1) + NY * (r / 3 - 1));
                long lo = std::max((long)ca + off - 1, 0L), hi = std::min((long)cb + off + 1, (long)NC - 1);
                rs[r] = hi >= lo ? (int)lo * PPC : 0; rn[r] = hi >= lo ? ((int)hi + 1) * PPC - rs[r] : 0; pre[r] = o; o += rn[r]; }
            staged += o;
            for (int i = i0; i <= il; ++i) {
                uint16_t *lp = &nl16[(size_t)(i >> 5) * kf * 32 + (i & 31) * 2]; int k = 0;
                for (int r = 0; r < 9; ++r) for (int j : nbr[(size_t)i * 9 + r]) if (k < kf) { int e = pre[r] + j - rs[r]; if (cf) e = (e & ~7) | (((i & 31) + k) & 7); lp[(k >> 1) * 64 + (k & 1)] = (uint16_t)e; ++k; }
                if (k & 1) lp[(k >> 1) * 64 + 1] = lp[(k >> 1) * 64];
                cnt[i] = k;
            }
        }
        uint32_t *dnl; int *dcnt; cudaMalloc(&dnl, nl16.size() * 2); cudaMalloc(&dcnt, N * 4);
        cudaMemcpy(dnl, nl16.data(), nl16.size() * 2, cudaMemcpyHostToDevice); cudaMemcpy(dcnt, cnt.data(), N * 4, cudaMemcpyHostToDevice);
        printf("shared-memory staged tile (%s): %.0f records per CTA of %d particles\n", cf ? "conflict-free entries" : "real entries", staged / nb, B);
        for (int skip : { 0, 1 })
            printf("  LDS.128 gathers, %-28s %7.1f us\n", skip ? "tile copy skipped (gather only)" : "cp.async.bulk tile copy",
                   best_of([&] { k_smem<<<nb, B, 1536 * 16>>>(dnl, dcnt, kf, dpos, dout, N, skip); }));
        cudaFree(dnl); cudaFree(dcnt);
    }
    printf("%s\n", cudaGetErrorString(cudaDeviceSynchronize()));
    return 0;
}
