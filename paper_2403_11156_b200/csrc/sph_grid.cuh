// sph_grid.cuh -- A1-A3: cell keys + histogram, exclusive prefix scan, counting-sort scatter,
// canonical intra-cell order and reorder of the particle store.
//
// The paper only says that its neighbour structure is built with a prefix sum;
// geometry, linearisation and clamping are reading R11, the order inside a cell reading R12.
#pragma once
#include "sph_common.cuh"

namespace sph {

// A1 + first half of A2: key[i] = linear cell of pos[i]; off[i] = arrival rank inside the cell
// (atomic, NOT deterministic -- k_reorder canonicalises); count[key]++; clamps counted per warp.
// (Measured and rejected, round 2: accumulating the scan's tile sums here as well, to save k_scan_tile_sums --
// one atomic per warp, or per CTA, whose particles share a scan tile: 22-28 us instead of 13 + 8; several
// particles per thread: no gain either, the kernel is bound by the throughput of the returning atomics.)
constexpr int kScanThreads = 256;
constexpr int kScanRounds = 4;                                  // int4 per thread per round
constexpr int kScanTile = kScanThreads * 4 * kScanRounds;       // 4096 cells per CTA

__global__ void __launch_bounds__(256)
k_cell_key_hist(const float4 *__restrict__ pos, int n, Geom g, int *__restrict__ key,
                int *__restrict__ off, int *__restrict__ count, int *__restrict__ oob)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool clamped = false;
    if (i < n) {
        float4 p = pos[i];
        int cx, cy, cz;
        int k = cell_key(g, p.x, p.y, p.z, clamped, cx, cy, cz);
        key[i] = k;
        off[i] = atomicAdd(&count[k], 1);
    }
    unsigned b = __ballot_sync(0xffffffffu, clamped);
    if (oob != nullptr && b != 0u && (threadIdx.x & 31) == 0) atomicAdd(oob, __popc(b));
}

// keys only (SPH_FIELD_CELL_OF_PARTICLE export): out[id[s]] = key of sorted slot s.
__global__ void __launch_bounds__(256)
k_export_keys(const float4 *__restrict__ pos, const int *__restrict__ id, int n, Geom g,
              int *__restrict__ out)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    float4 p = pos[s];
    bool clamped; int cx, cy, cz;
    cell_key(g, p.x, p.y, p.z, clamped, cx, cy, cz);
    out[id[s]] = cx / kFineX + g.nxc * (cy + g.ny * cz);           // the R11 key
}

// ---------------------------------------------------------------------------------------------
// A2: exclusive prefix scan of count[0 .. n) in place (n = ncells + 1, count[ncells] = 0 so that
// the last entry becomes N).  Two launches: tile sums, tile rescan (which sums the preceding tiles' sums itself).

__device__ __forceinline__ int4 load_int4_guard(const int *a, int base, int n)
{
    if (base + 3 < n) return *reinterpret_cast<const int4 *>(a + base);
    int4 v = make_int4(0, 0, 0, 0);
    if (base < n) v.x = a[base];
    if (base + 1 < n) v.y = a[base + 1];
    if (base + 2 < n) v.z = a[base + 2];
    return v;
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_tile_sums(const int *__restrict__ a, int n, int *__restrict__ tile_sum)
{
    __shared__ int sm[kScanThreads / 32];
    int base = blockIdx.x * kScanTile;
    int s = 0;
#pragma unroll
    for (int r = 0; r < kScanRounds; ++r) {
        int4 v = load_int4_guard(a, base + r * kScanThreads * 4 + threadIdx.x * 4, n);
        s += v.x + v.y + v.z + v.w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) t += sm[w];
        tile_sum[blockIdx.x] = t;
    }
}

// tile_sum holds the raw tile sums: every CTA adds up the sums of the tiles before its own (a few hundred to a few
// thousand ints, L2-resident) -- cheaper than a separate one-CTA scan launch in between (7 us on 4.4 M cells).
// The tile's four rounds are loaded up front and scanned together: four interleaved warp scans, ONE barrier, then
// every warp scans the 32 (round, warp) totals for itself.
static_assert(kScanRounds * (kScanThreads / 32) == 32, "k_scan_apply scans the (round, warp) totals with one warp");
__global__ void __launch_bounds__(kScanThreads)
k_scan_apply(int *__restrict__ a, int n, const int *__restrict__ tile_sum)
{
    constexpr int NW = kScanThreads / 32;
    __shared__ int sm_tot[kScanRounds * NW];
    __shared__ int sm_carry[NW];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int base = blockIdx.x * kScanTile;
    int4 v[kScanRounds];
#pragma unroll
    for (int r = 0; r < kScanRounds; ++r) v[r] = load_int4_guard(a, base + r * kScanThreads * 4 + threadIdx.x * 4, n);
    int part = 0;
    for (int t = threadIdx.x; t < (int)blockIdx.x; t += kScanThreads) part += tile_sum[t];
    int tsum[kScanRounds], inc[kScanRounds];
#pragma unroll
    for (int r = 0; r < kScanRounds; ++r) inc[r] = tsum[r] = v[r].x + v[r].y + v[r].z + v[r].w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int r = 0; r < kScanRounds; ++r) {
            const int t = __shfl_up_sync(0xffffffffu, inc[r], o);
            if (lane >= o) inc[r] += t;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 31) {
#pragma unroll
        for (int r = 0; r < kScanRounds; ++r) sm_tot[r * NW + w] = inc[r];
    }
    if (lane == 0) sm_carry[w] = part;
    __syncthreads();
    const int x = sm_tot[lane];                 // entry (round lane / NW, warp lane % NW): the order of the elements
    int xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, xi, o);
        if (lane >= o) xi += t;
    }
    int carry = 0;
#pragma unroll
    for (int q = 0; q < NW; ++q) carry += sm_carry[q];
    const int excl = xi - x + carry;
#pragma unroll
    for (int r = 0; r < kScanRounds; ++r) {
        const int e = base + r * kScanThreads * 4 + threadIdx.x * 4;
        const int ex = __shfl_sync(0xffffffffu, excl, r * NW + w) + inc[r] - tsum[r];
        int4 o;
        o.x = ex; o.y = ex + v[r].x; o.z = o.y + v[r].y; o.w = o.z + v[r].z;
        if (e + 3 < n) *reinterpret_cast<int4 *>(a + e) = o;
        else {
            if (e < n) a[e] = o.x;
            if (e + 1 < n) a[e + 1] = o.y;
            if (e + 2 < n) a[e + 2] = o.z;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// A3 first half: slot[cell_start[key] + off] = source index (four particles per thread).
constexpr int kScatterPer = 4;
__global__ void __launch_bounds__(256)
k_scatter_slots(const int *__restrict__ key, const int *__restrict__ off,
                const int *__restrict__ cell_start, int n, int *__restrict__ slot_src)
{
    const int base = blockIdx.x * (256 * kScatterPer) + threadIdx.x;
    int k[kScatterPer], o[kScatterPer], cs[kScatterPer];
#pragma unroll
    for (int u = 0; u < kScatterPer; ++u) {
        const int i = base + u * 256;
        k[u] = i < n ? key[i] : 0;
        o[u] = i < n ? off[i] : 0;
    }
#pragma unroll
    for (int u = 0; u < kScatterPer; ++u) cs[u] = cell_start[k[u]];
#pragma unroll
    for (int u = 0; u < kScatterPer; ++u) {
        const int i = base + u * 256;
        if (i < n) slot_src[cs[u] + o[u]] = i;
    }
}

// A3 second half: canonical order inside a cell = ascending source index (= order of the
// previous sorted store, R12: makes the run bit-reproducible although the histogram atomics are
// not), then gather of every persistent field into sorted order.
// For the fluid store (FLUID): a = pos(x,y,z,-), b = vel(vx,vy,vz,-), ids carried; a_out = packed
// positions, b_out = { pos | vel } records, (sx, sy, sz) = structure-of-arrays positions.
// For the boundary store: a = (x,y,z,psi), b = (vx,vy,vz,-), ids = original boundary index.
// Two slots per thread; every load that depends on the source index alone is requested together with the key, so
// that the chain slot -> key -> cell_start -> cell mates is not followed by a fourth round trip for the payload.
constexpr int kReorderPer = 2;
template <bool FLUID>
__global__ void __launch_bounds__(256)
k_reorder(const int *__restrict__ slot_src, const int *__restrict__ key,
          const int *__restrict__ cell_start, int n,
          const float4 *__restrict__ a_in, const float4 *__restrict__ b_in,
          const int *__restrict__ id_in, float4 *__restrict__ a_out, float4 *__restrict__ b_out,
          int *__restrict__ id_out, float *__restrict__ sx, float *__restrict__ sy, float *__restrict__ sz)
{
    const int base = blockIdx.x * (256 * kReorderPer) + threadIdx.x;
    int src[kReorderPer];
#pragma unroll
    for (int u = 0; u < kReorderPer; ++u) {
        const int s = base + u * 256;
        src[u] = s < n ? slot_src[s] : 0;
    }
    int k[kReorderPer], id[kReorderPer];
    float4 a[kReorderPer], b[kReorderPer];
#pragma unroll
    for (int u = 0; u < kReorderPer; ++u) {
        k[u] = key[src[u]];
        a[u] = a_in[src[u]];
        b[u] = b_in != nullptr ? b_in[src[u]] : make_float4(0.f, 0.f, 0.f, 0.f);
        id[u] = id_in != nullptr ? id_in[src[u]] : src[u];
    }
    int cs[kReorderPer], ce[kReorderPer];
#pragma unroll
    for (int u = 0; u < kReorderPer; ++u) { cs[u] = cell_start[k[u]]; ce[u] = cell_start[k[u] + 1]; }
#pragma unroll
    for (int u = 0; u < kReorderPer; ++u) {
        const int s = base + u * 256;
        if (s >= n) continue;
        int rank;
        if (ce[u] - cs[u] > kBigCell) rank = s - cs[u];       // degenerate pile-up: keep arrival order
        else {
            rank = 0;
            for (int t = cs[u]; t < ce[u]; ++t) rank += (slot_src[t] < src[u]) ? 1 : 0;
        }
        const int dst = cs[u] + rank;
        a_out[dst] = a[u];
        if (FLUID) {
            // b_out is the 32-byte record array { pos | vel } of the passes (PV in sph_passes.cuh)
            b_out[2 * dst] = a[u];
            b_out[2 * dst + 1] = b[u];
            sx[dst] = a[u].x; sy[dst] = a[u].y; sz[dst] = a[u].z;     // SoA copy: what the list builder reads as 16-byte quads
        } else if (b_in != nullptr) b_out[dst] = b[u];
        id_out[dst] = id[u];
    }
}

// R11 cell_start = every kFineX-th entry of the fine one (n = coarse cells + 1 entries)
__global__ void __launch_bounds__(256)
k_export_cell_start(const int *__restrict__ fine, int n, int *__restrict__ out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = fine[(size_t)k * kFineX];
}

}  // namespace sph
