// sph_lists.cuh -- A4, first half: the per-step neighbour lists.
//
// ONE evaluation of the neighbour predicate (reading R10, bit-exact) per (particle, candidate) pair
// per step; every later pass gathers through the lists this kernel writes (format: list_tile() and
// for_each_neighbor() in sph_passes.cuh -- 16-bit (x-run, offset) entries in ascending sorted index).
//
// Design (round 2; the round-1 builder tested one candidate per thread with ~26 issued instructions
// per candidate and was 85 % issue-bound):
//  * Two targets per lane, packed fp32x2 arithmetic (sm_100 FADD2 / FMUL2 / FFMA2, IEEE round to
//    nearest per half, so the predicate stays bit-exact).  Lane l of a warp owns the sorted particles
//    2l and 2l + 1 of the warp's 64, which almost always lie in the same cell row and therefore share
//    a candidate window per x-run; one candidate is tested against both by 3 FADD2 + FMUL2 + 2 FFMA2
//    + 2 FSETP -- about 11 issued instructions per (target, candidate) pair including the stores.
//  * Candidates come from structure-of-arrays positions (px, py, pz, written by the reorder kernel):
//    one 16-byte read-only load per coordinate fetches FOUR consecutive candidates (runs are split into
//    an unaligned head, aligned quads and a tail).  Lanes of one cell read the same address, so a
//    warp-wide load touches a few consecutive 128-byte lines that L1 keeps resident across the
//    neighbouring warps.
//  * Entries are staged per target in shared memory (2-byte stores, one bank per lane) and written out
//    as coalesced 32-bit words.  The staging columns hold kStageRows entries; a target with more
//    neighbours (dense pile-ups only) gets the rest from a second, scalar walk (spill_walk).
//
// Measured and rejected: the same loops fed from a CTA tile of candidates staged
// in shared memory by 1-D bulk copies (cp.async.bulk + mbarrier; 9 merged index ranges per 256
// targets).  The tile plus the staging columns limit an SM to 4 CTAs = 16 warps, and the kernel then
// spends ~2/3 of its warp-time on exposed latencies outside the test loop (tile hand-shake,
// cell_start look-ups, epilogue): 185 us against 160 us for the L1-fed version at 32 warps per SM,
// although the loop itself needed 40 % fewer load wavefronts.
#pragma once
#include "sph_passes.cuh"

namespace sph {

constexpr int kMaxListCap = 768;
constexpr int kStageRows = 40;     // staging rows per target in shared memory (even)
constexpr int kBuildWarps = 4;     // 64 targets per warp

struct BuildShape { int warps, rows; size_t smem; };
inline BuildShape build_shape(int kf)
{
    BuildShape b;
    b.warps = kBuildWarps;
    b.rows = kf < kStageRows ? kf : kStageRows;
    b.smem = (size_t)(b.rows + 1) * 128 * b.warps;       // + one row that swallows the stores past a full column
    return b;
}

typedef unsigned long long u64;
__device__ __forceinline__ u64 pack2(float a, float b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpack2(u64 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 c; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b)); return c; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 c; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(c) : "l"(a), "l"(b)); return c; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 d) { u64 c; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(c) : "l"(a), "l"(b), "l"(d)); return c; }

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// staging store: volatile (ordered against the copy-out's volatile loads) but no memory clobber, so that the
// candidate loads of later iterations may be hoisted above it
__device__ __forceinline__ void sts_u16(uint32_t addr, int v)
{
    asm volatile("st.shared.u16 [%0], %1;" :: "r"(addr), "h"((unsigned short)v));
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr)
{
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr) : "memory");
    return v;
}

// staging cursor of one target: byte address of the slot of its next entry; `end` = the slot one row past its
// shared-memory column, a spare row that swallows the stores of a full column.  The cursor keeps advancing past
// `end` (it counts the hits); entries beyond the column are not staged.
struct StageCur { uint32_t w, end; };

struct PairCtx {                   // what the test loop needs, per lane
    const float *px, *py, *pz;
    u64 X, Y, Z;                   // the two targets, packed (a target that is switched off holds NaN and never hits)
    float h2;
};

// One candidate t tested against both targets; entry of a hit = t + cA (resp. cB) = run tag + offset inside the
// target's own run.  No capacity test in the loop: the store address is clamped to the spare row (one VIMNMX instead
// of a compare and a second predicate per target: quad loop 91 -> 78 instructions, builder 183 -> 170 us), the cursor
// still advances.  (Looked at and not kept: a saturating cursor -- the compiler emits add-and-min + select, same count;
// the same written as predicated PTX -- 96 instructions; saturating once per quad with four spare rows -- 75
// instructions, but the count then needs a second walk whenever a column fills exactly; an unguarded second loop for
// runs that certainly fit -- slower, the kernel is sensitive to code size.)
__device__ __forceinline__ void test_one(const PairCtx &q, u64 X, int t, float qx, float qy, float qz, int cA, int cB,
                                         StageCur &A, StageCur &B)
{
    const u64 dx = sub2(X, pack2(qx, qx)), dy = sub2(q.Y, pack2(qy, qy)), dz = sub2(q.Z, pack2(qz, qz));
    const u64 d2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));      // reading R10, both halves in binary32 RN
    float a, b;
    unpack2(d2, a, b);
    const bool ha = a < q.h2, hb = b < q.h2;
    if (ha) sts_u16(min(A.w, A.end), t + cA);
    if (hb) sts_u16(min(B.w, B.end), t + cB);
    if (ha) A.w += 128;
    if (hb) B.w += 128;
}

// candidates [t0, t1), t0 and t1 multiples of four: one 16-byte load per coordinate and trip.  (Requesting the next
// trip's loads before this trip's tests was measured too: slower, the extra registers and moves cost more than the
// 32 resident warps per SM fail to hide.)
__device__ __forceinline__ void test_quads(const PairCtx &q, int t0, int t1, int cA, int cB, StageCur &A, StageCur &B)
{
#pragma unroll 1
    for (int t = t0; t < t1; t += 4) {
        const float4 vx = __ldg(reinterpret_cast<const float4 *>(q.px + t)), vy = __ldg(reinterpret_cast<const float4 *>(q.py + t)),
                     vz = __ldg(reinterpret_cast<const float4 *>(q.pz + t));
        test_one(q, q.X, t, vx.x, vy.x, vz.x, cA, cB, A, B);
        test_one(q, q.X, t + 1, vx.y, vy.y, vz.y, cA, cB, A, B);
        test_one(q, q.X, t + 2, vx.z, vy.z, vz.z, cA, cB, A, B);
        test_one(q, q.X, t + 3, vx.w, vy.w, vz.w, cA, cB, A, B);
    }
}

// The 9 runs of the lane's pair of targets.  cell: cell of the first active target; cx_hi: fine x-coordinate of the
// second one when both share the cell row (else = cell.cx).  oA / oB: the targets are on.
__device__ __forceinline__ void build_pair(const PassCtx &p, const PairCtx &q, const CellOf &cell, int cx_hi,
                                           int iA, int iB, bool oA, bool oB, StageCur &A, StageCur &B, bool &ovf)
{
    const Geom &g = p.c.g;
    const int x0 = cell.x0, x1 = min(cx_hi + kFineX, g.nx - 1), xb0 = max(cx_hi - kFineX, 0);
    // the cell_start words of run r + 1 are requested before run r is walked (and only combined afterwards: no
    // instruction in between waits on them)
    auto run_range = [&](int r, int &s, int &e, int &sB) {
        s = 0; e = 0; sB = 0;
        if (r >= kRows) return;
        const int z = cell.cz + r / 3 - 1, y = cell.cy + r % 3 - 1;
        if ((unsigned)z >= (unsigned)g.nz || (unsigned)y >= (unsigned)g.ny) return;
        const int *row = p.fcs + g.nx * (y + g.ny * z);
        s = __ldg(row + x0); e = __ldg(row + x1 + 1); sB = __ldg(row + xb0);
    };
    int s_n, e_n, sB_n;
    run_range(0, s_n, e_n, sB_n);
#pragma unroll 1
    for (int r = 0; r < kRows; ++r) {
        const int s = s_n, sB = sB_n;
        int len = e_n - s_n;
        run_range(r + 1, s_n, e_n, sB_n);
        if (len <= 0) continue;
        if (len > kOffMask + 1) { ovf = true; len = kOffMask + 1; }     // offsets are 12-bit
        const int tag = r << kOffBits;
        const int cA = tag - s, cB = tag - sB;
        // [s, e) as: single candidates up to the first multiple of four, quads (one 16-byte load per coordinate),
        // single candidates after the last multiple of four.  (The window must not simply be widened to whole
        // quads: what follows a run in memory is the NEXT cell row, whose particles may well be neighbours and are
        // visited by their own run.)  The code between two runs is kept as short as it gets: a run is only ~5 quads
        // long, and every instruction of per-run overhead showed in the kernel's time (a generic piece loop here
        // cost 30 us of 180).
        const int e = s + len;
        const int h1 = min((s + 3) & ~3, e), h2 = max(e & ~3, h1);
        if (r != 4) {
#pragma unroll 1
            for (int t = s; t < h1; ++t) test_one(q, q.X, t, __ldg(q.px + t), __ldg(q.py + t), __ldg(q.pz + t), cA, cB, A, B);
            test_quads(q, h1, h2, cA, cB, A, B);
#pragma unroll 1
            for (int t = h2; t < e; ++t) test_one(q, q.X, t, __ldg(q.px + t), __ldg(q.py + t), __ldg(q.pz + t), cA, cB, A, B);
            continue;
        }
        // Run 4 is the targets' own run: the slots of the active targets (adjacent: iA, iB) are tested against the
        // OTHER target only (own half switched off), as single candidates -- the quads that hold them form a
        // third singles piece in the middle.
        const int f1 = oA ? iA : iB, f2 = (oB ? iB : iA) + 1;
        const int q1 = min(max(f1 & ~3, h1), h2), q2 = min(max((f2 + 3) & ~3, h1), h2);
#pragma unroll 1
        for (int pc = 0; pc < 5; ++pc) {
            // pieces: 0 singles [s, h1) . 1 quads [h1, q1) . 2 singles [q1, q2) . 3 quads [q2, h2) . 4 singles [h2, e)
            const int a = pc == 0 ? s : (pc == 1 ? h1 : (pc == 2 ? q1 : (pc == 3 ? q2 : h2)));
            const int b = pc == 0 ? h1 : (pc == 1 ? q1 : (pc == 2 ? q2 : (pc == 3 ? h2 : e)));
            if (pc & 1) test_quads(q, a, b, cA, cB, A, B);
            else {
#pragma unroll 1
                for (int t = a; t < b; ++t) {
                    u64 X = q.X;
                    if (t >= f1 && t < f2) {
                        const bool isA = oA && t == iA;
                        float xa, xb; unpack2(q.X, xa, xb);
                        X = pack2(isA ? __int_as_float(0x7fc00000) : xa, isA ? xb : __int_as_float(0x7fc00000));
                    }
                    test_one(q, X, t, __ldg(q.px + t), __ldg(q.py + t), __ldg(q.pz + t), cA, cB, A, B);
                }
            }
        }
    }
}

// Entries k >= rows of a target with more than `rows` neighbours (dense pile-ups only): a second, scalar walk of
// its 9 runs that stores entry k straight into the warp-tiled global list.
__device__ __noinline__ void spill_walk(const PassCtx &p, const float *__restrict__ px, const float *__restrict__ py,
                                        const float *__restrict__ pz, int i, float xi, float yi, float zi, int rows)
{
    const Geom &g = p.c.g;
    const CellOf cell = cell_of(g, xi, yi, zi);
    uint16_t *gl = p.nl_f + list_tile(i, p.c.kf) + (i & 31) * 2;
    int k = 0;
    for (int r = 0; r < kRows; ++r) {
        int first;
        if (!run_first_cell(g, cell, r, first)) continue;
        const int s = __ldg(p.fcs + first), e = min(__ldg(p.fcs + first + (cell.x1 - cell.x0) + 1), s + kOffMask + 1);
        for (int j = s; j < e; ++j) {
            const float dx = __fsub_rn(xi, __ldg(px + j)), dy = __fsub_rn(yi, __ldg(py + j)), dz = __fsub_rn(zi, __ldg(pz + j));
            if (dist2_r10(dx, dy, dz) < p.c.h2 && j != i) {
                if (k >= rows && k < p.c.kf) gl[(size_t)(k >> 1) * 64 + (k & 1)] = (uint16_t)((r << kOffBits) | (j - s));
                ++k;
            }
        }
    }
    // the passes decode both halves of a list word without a guard: the unwritten half of an odd tail pair must be a
    // decodable entry (the copy-out zeroes it for staged entries; here the pair may lie past the staged rows)
    if (k > rows && (k & 1) && k < p.c.kf) gl[(size_t)(k >> 1) * 64 + 1] = 0;
}

__global__ void __launch_bounds__(32 * kBuildWarps, 8)
k_build_lists(PassCtx p, const float *__restrict__ px, const float *__restrict__ py, const float *__restrict__ pz,
              ListCounters *__restrict__ lc, int rows)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const SimConst &c = p.c;
    const Geom &g = c.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int w0 = (blockIdx.x * kBuildWarps + warp) * 64;           // first target of the warp
    if (w0 >= c.nf) return;
    const uint32_t stage0 = smem_addr(smem_raw) + (uint32_t)warp * (uint32_t)(rows + 1) * 128u;
    // guard of the statistics atomics at the end, requested now (a stale value only costs an extra atomic)
    const unsigned long long seen = *reinterpret_cast<volatile unsigned long long *>(&lc->max_f);

    // ---- the lane's two targets
    const int iA = w0 + 2 * lane, iB = iA + 1;
    const bool vA = iA < c.nf, vB = iB < c.nf;
    const float nanf_ = __int_as_float(0x7fc00000);
    float ax = 0.f, ay = 0.f, az = 0.f, bx = 0.f, by = 0.f, bz = 0.f;
    if (vA) { ax = __ldg(px + iA); ay = __ldg(py + iA); az = __ldg(pz + iA); }
    if (vB) { bx = __ldg(px + iB); by = __ldg(py + iB); bz = __ldg(pz + iB); }
    const CellOf cellA = cell_of(g, ax, ay, az), cellB = cell_of(g, bx, by, bz);
    const bool same = vB && cellA.cy == cellB.cy && cellA.cz == cellB.cz && cellB.cx >= cellA.cx;

    // ---- is any boundary sample near the warp?  Lane r < 9 looks at the cell range of row offset r around the
    // warp's first and last target (cells are linearised x-fastest: one index range of the BOUNDARY grid per row
    // offset).  Most warps are far from every wall and skip the boundary part altogether.
    bool near_b = false;
    if (c.nb > 0) {
        const int last = min(w0 + 63, c.nf - 1);
        int ga = 0, gb = 0;
        if (lane < kRows) {
            bool cl; int tx, ty, tz;
            const int fa = cell_key(g, __ldg(px + w0), __ldg(py + w0), __ldg(pz + w0), cl, tx, ty, tz);
            const int fb = cell_key(g, __ldg(px + last), __ldg(py + last), __ldg(pz + last), cl, tx, ty, tz);
            const long long off = (long long)g.nx * ((lane % 3 - 1) + (long long)g.ny * (lane / 3 - 1));
            long long lo = (long long)fa + off - kFineX, hi = (long long)fb + off + kFineX;
            lo = lo < 0 ? 0 : lo;
            hi = hi > (long long)g.ncells - 1 ? (long long)g.ncells - 1 : hi;
            if (hi >= lo) { ga = __ldg(p.bcs + lo); gb = __ldg(p.bcs + hi + 1); }
        }
        near_b = __any_sync(0xffffffffu, gb > ga);
    }

    StageCur A, B;
    A.w = stage0 + (uint32_t)(2 * lane) * 2u; A.end = A.w + (uint32_t)rows * 128u;
    B.w = A.w + 2u; B.end = B.w + (uint32_t)rows * 128u;
    const uint32_t wA0 = A.w, wB0 = B.w;
    bool ovf = false;
    if (vA) {
        // pass 0: A, and B too when it shares A's cell row; pass 1 (rare: row change inside the pair): B alone
        const int npass = (vB && !same) ? 2 : 1;
#pragma unroll 1
        for (int pass = 0; pass < npass; ++pass) {
            const bool oA = pass == 0, oB = vB && (same ? pass == 0 : pass == 1);
            PairCtx q;
            q.px = px; q.py = py; q.pz = pz; q.h2 = c.h2;
            q.X = pack2(oA ? ax : nanf_, oB ? bx : nanf_); q.Y = pack2(oA ? ay : nanf_, oB ? by : nanf_);
            q.Z = pack2(oA ? az : nanf_, oB ? bz : nanf_);
            const CellOf &cell = pass == 0 ? cellA : cellB;
            const int cx_hi = (pass == 0 && same) ? cellB.cx : cell.cx;
            build_pair(p, q, cell, cx_hi, iA, iB, oA, oB, A, B, ovf);
        }
    }
    const int cfA = (int)((A.w - wA0) >> 7), cfB = (int)((B.w - wB0) >> 7);
    if (cfA > rows) spill_walk(p, px, py, pz, iA, ax, ay, az, rows);
    if (cfB > rows) spill_walk(p, px, py, pz, iB, bx, by, bz, rows);

    // ---- boundary neighbours of both targets (32-bit sorted boundary indices, written directly).  A lane first
    // requests the 18 cell_start words of a target together, then walks the non-empty runs
    int cbA = 0, cbB = 0;
    if (near_b) {
#pragma unroll 1
        for (int w = 0; w < 2; ++w) {
            const int i = w ? iB : iA;
            if (i >= c.nf) break;
            const float xi = w ? bx : ax, yi = w ? by : ay, zi = w ? bz : az;
            const CellOf &cell = w ? cellB : cellA;
            int bs[kRows], bl[kRows];
#pragma unroll
            for (int r = 0; r < kRows; ++r) {
                int first;
                bs[r] = 0; bl[r] = 0;
                if (run_first_cell(g, cell, r, first)) {
                    bs[r] = __ldg(p.bcs + first);
                    bl[r] = __ldg(p.bcs + first + (cell.x1 - cell.x0) + 1) - bs[r];
                }
            }
            int *lb = p.nl_b + list_tile(i, c.kb) + (i & 31);
            int cb = 0;
#pragma unroll
            for (int r = 0; r < kRows; ++r) {
                for (int k = bs[r]; k < bs[r] + bl[r]; ++k) {
                    float4 qb = __ldg(p.bpos + k);
                    float dx = __fsub_rn(xi, qb.x), dy = __fsub_rn(yi, qb.y), dz = __fsub_rn(zi, qb.z);
                    if (dist2_r10(dx, dy, dz) < c.h2) {
                        if (cb < c.kb) lb[cb * 32] = k;
                        ++cb;
                    }
                }
            }
            if (w) cbB = cb; else cbA = cb;
        }
    }
    if (vA) p.ncount[iA] = min(cfA, c.kf) | (min(cbA, c.kb) << 16);
    if (vB) p.ncount[iB] = min(cfB, c.kf) | (min(cbB, c.kb) << 16);
    const int novf = ((ovf || cfA > c.kf || cbA > c.kb) ? 1 : 0) + ((cfB > c.kf || cbB > c.kb) ? 1 : 0);

    // ---- copy-out: lane l writes the staged columns of targets l and l + 32 of its warp (one list tile each):
    // word k of the tile row = entries (2k, 2k + 1) (layout of list_tile); entries >= rows are in place already
    __syncwarp();
#pragma unroll 1
    for (int hlf = 0; hlf < 2; ++hlf) {
        const int tau = hlf * 32 + lane, i = w0 + tau;
        const int ca = __shfl_sync(0xffffffffu, cfA, tau >> 1), cb2 = __shfl_sync(0xffffffffu, cfB, tau >> 1);
        if (i >= c.nf) continue;
        const int n = min(min((tau & 1) ? cb2 : ca, c.kf), rows);
        const uint32_t col = stage0 + (uint32_t)tau * 2u;
        uint32_t *dst = reinterpret_cast<uint32_t *>(p.nl_f + list_tile(i, c.kf)) + lane;
        for (int k = 0; k < n; k += 2) {
            uint32_t lo = lds_u16(col + (uint32_t)k * 128u), hi = k + 1 < n ? lds_u16(col + (uint32_t)(k + 1) * 128u) : 0u;
            dst[(k >> 1) * 32] = lo | (hi << 16);
        }
    }

    // ---- statistics: overflow count, maxima, neighbour-count sum (one reduction atomic per warp for the sums; the
    // maxima only grow, so the value read at the start guards their atomics: same-address atomics serialise in L2)
    int mf = max(cfA, cfB), mb = max(cbA, cbB), sf = cfA + cfB, so = novf;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mf = max(mf, __shfl_xor_sync(0xffffffffu, mf, o));
        mb = max(mb, __shfl_xor_sync(0xffffffffu, mb, o));
        sf += __shfl_xor_sync(0xffffffffu, sf, o);
        so += __shfl_xor_sync(0xffffffffu, so, o);
    }
    if (lane == 0) {
        if (mf > (int)(unsigned)(seen & 0xffffffffull)) atomicMax(&lc->max_f, mf);
        if (mb > (int)(unsigned)(seen >> 32)) atomicMax(&lc->max_b, mb);
        atomicAdd(&lc->sum_f, (unsigned long long)sf);
        if (so) atomicAdd(&lc->overflow, so);
    }
}

}  // namespace sph
