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
constexpr int kScanThreads = 256;
constexpr int kScanRounds = 4;                                  // int4 per thread per round
constexpr int kScanTile = kScanThreads * 4 * kScanRounds;       // 4096 cells per CTA

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

// block-wide exclusive scan of one int per thread; returns exclusive prefix, *total = block sum
__device__ __forceinline__ int block_excl_scan(int v, int *sm /* [blockDim/32 + 1] */, int *total)
{
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();
    if (lane == 31) sm[w] = inc;
    __syncthreads();
    if (w == 0) {
        int x = lane < nw ? sm[lane] : 0;
        int xi = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, xi, o);
            if (lane >= o) xi += t;
        }
        if (lane < nw) sm[lane] = xi - x;   // exclusive warp offsets
        if (lane == 31) sm[32] = xi;        // total (nw <= 32)
    }
    __syncthreads();
    *total = sm[32];
    return sm[w] + inc - v;
}

// tile_sum holds the raw tile sums: every CTA adds up the sums of the tiles before its own (a few hundred to a few
// thousand ints, L2-resident) -- cheaper than a separate one-CTA scan launch in between (7 us on 4.4 M cells).
__global__ void __launch_bounds__(kScanThreads)
k_scan_apply(int *__restrict__ a, int n, const int *__restrict__ tile_sum)
{
    __shared__ int sm[33];
    int base = blockIdx.x * kScanTile;
    int carry;
    {
        int part = 0;
        for (int t = threadIdx.x; t < (int)blockIdx.x; t += kScanThreads) part += tile_sum[t];
        block_excl_scan(part, sm, &carry);
        __syncthreads();
    }
#pragma unroll 1
    for (int r = 0; r < kScanRounds; ++r) {
        int e = base + r * kScanThreads * 4 + threadIdx.x * 4;
        int4 v = load_int4_guard(a, e, n);
        int t = v.x + v.y + v.z + v.w;
        int total;
        int ex = block_excl_scan(t, sm, &total) + carry;
        int4 o;
        o.x = ex; o.y = ex + v.x; o.z = o.y + v.y; o.w = o.z + v.z;
        if (e + 3 < n) *reinterpret_cast<int4 *>(a + e) = o;
        else {
            if (e < n) a[e] = o.x;
            if (e + 1 < n) a[e + 1] = o.y;
            if (e + 2 < n) a[e + 2] = o.z;
        }
        carry += total;
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// A3 first half: slot[cell_start[key] + off] = source index.
__global__ void __launch_bounds__(256)
k_scatter_slots(const int *__restrict__ key, const int *__restrict__ off,
                const int *__restrict__ cell_start, int n, int *__restrict__ slot_src)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    slot_src[cell_start[key[i]] + off[i]] = i;
}

// A3 second half: canonical order inside a cell = ascending source index (= order of the
// previous sorted store, R12: makes the run bit-reproducible although the histogram atomics are
// not), then gather of every persistent field into sorted order.
// For the fluid store (FLUID): a = pos(x,y,z,-), b = vel(vx,vy,vz,-), ids carried; a_out = packed
// positions, b_out = { pos | vel } records, (sx, sy, sz) = structure-of-arrays positions.
// For the boundary store: a = (x,y,z,psi), b = (vx,vy,vz,-), ids = original boundary index.
template <bool FLUID>
__global__ void __launch_bounds__(256)
k_reorder(const int *__restrict__ slot_src, const int *__restrict__ key,
          const int *__restrict__ cell_start, int n,
          const float4 *__restrict__ a_in, const float4 *__restrict__ b_in,
          const int *__restrict__ id_in, float4 *__restrict__ a_out, float4 *__restrict__ b_out,
          int *__restrict__ id_out, float *__restrict__ sx, float *__restrict__ sy, float *__restrict__ sz)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int src = slot_src[s];
    int k = key[src];
    int cs = cell_start[k], ce = cell_start[k + 1];
    int rank;
    if (ce - cs > kBigCell) rank = s - cs;       // degenerate pile-up: keep arrival order
    else {
        rank = 0;
        for (int t = cs; t < ce; ++t) rank += (slot_src[t] < src) ? 1 : 0;
    }
    int dst = cs + rank;
    float4 a = a_in[src];
    a_out[dst] = a;
    if (FLUID) {
        // b_out is the 32-byte record array { pos | vel } of the passes (PV in sph_passes.cuh)
        b_out[2 * dst] = a;
        b_out[2 * dst + 1] = b_in[src];
        sx[dst] = a.x; sy[dst] = a.y; sz[dst] = a.z;     // SoA copy: what the list builder bulk-copies into its tiles
    } else if (b_in != nullptr) b_out[dst] = b_in[src];
    id_out[dst] = id_in != nullptr ? id_in[src] : src;
}

// R11 cell_start = every kFineX-th entry of the fine one (n = coarse cells + 1 entries)
__global__ void __launch_bounds__(256)
k_export_cell_start(const int *__restrict__ fine, int n, int *__restrict__ out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = fine[(size_t)k * kFineX];
}

}  // namespace sph
