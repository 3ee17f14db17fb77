"""fp64 CPU ORACLE of the post-processing stage: particles -> scalar field on a regular grid ->
marching-cubes iso-surface.  TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as sphref.c: only tests/ and bench.py's
cpu_baseline may import it; it shares no code, table or table generator with the CUDA path).

What the paper says (section 4.3): "Surface reconstruction of fluid particles is done using SplashSurf
[18]" -- no equations.  Reading R29: the usual SPH surface reconstruction that tool implements:

  field     phi(g) = sum_i V_i W(|g - x_i|, h),  V_i = m / rho_i  (the SPH colour field: ~1 inside the fluid, 0 outside),
            W the cubic spline of reading R1 with the simulation's support radius, on the nodes
            g = grid_min + (ix, iy, iz) * cube_size of a regular grid;
  surface   the iso-surface phi = iso by marching cubes (Lorensen and Cline 1987) on the cells of that grid:
            corner c = dx + 2 dy + 4 dz is INSIDE when phi > iso; a cell edge whose end points differ carries one vertex,
            linearly interpolated FROM ITS LOWER-INDEX CORNER (both cells that share the edge compute the same point);
            the vertices of a cell are joined by tracing, on every cube face, the segments between its crossing edges
            (a face with four crossings -- the ambiguous case -- pairs the two edges next to each INSIDE corner, a rule
            that depends on that face's corner signs only, so neighbouring cells agree and the mesh is watertight);
            the segments close into loops, every loop is oriented so that the triangle normals point out of the
            fluid (towards smaller phi) and fan-triangulated from its smallest-numbered edge.
            The 256-entry case table is GENERATED from this rule (case_table below), not copied from anywhere.

Plain numpy / Python loops; small inputs only.
"""
from __future__ import annotations

import numpy as np

# ---------------------------------------------------------------------------------------------- cube topology
# corner c = dx + 2 dy + 4 dz
CORNERS = np.array([[c & 1, (c >> 1) & 1, (c >> 2) & 1] for c in range(8)], dtype=np.int64)
# 12 edges as (lower corner, higher corner): 4 along x, 4 along y, 4 along z
EDGES = [(0, 1), (2, 3), (4, 5), (6, 7), (0, 2), (1, 3), (4, 6), (5, 7), (0, 4), (1, 5), (2, 6), (3, 7)]
_EDGE_OF = {frozenset(e): k for k, e in enumerate(EDGES)}


def _faces():
    """Six faces, each as its 4 corners in COUNTER-CLOCKWISE order seen from OUTSIDE the cube."""
    out = []
    for axis in range(3):
        u, v = (axis + 1) % 3, (axis + 2) % 3           # (axis, u, v) is a cyclic permutation of (x, y, z)
        for side in (0, 1):
            cyc = []
            for (a, b) in ((0, 0), (1, 0), (1, 1), (0, 1)):   # counter-clockwise seen from +axis
                d = [0, 0, 0]
                d[axis] = side; d[u] = a; d[v] = b
                cyc.append(d[0] + 2 * d[1] + 4 * d[2])
            if side == 0:
                cyc = cyc[::-1]                                # seen from -axis the same cycle runs clockwise
            out.append(cyc)
    return out


FACES = _faces()


def case_triangles(mask: int):
    """Triangles of one marching-cubes case as triples of EDGE ids, normals pointing out of the inside region.
    mask bit c = corner c is inside."""
    inside = [(mask >> c) & 1 for c in range(8)]
    nxt = {}                                            # directed segments: edge id -> next edge id
    for cyc in FACES:
        # walking the face counter-clockwise (seen from outside): corners k0 -> k1 -> k2 -> k3 -> k0
        for k in range(4):
            c = cyc[k]
            if not inside[c]:
                continue
            cp = cyc[(k - 1) % 4]                          # previous corner on the face
            # maximal run of inside corners that starts at c (going counter-clockwise) and whose predecessor is outside
            if inside[cp]:
                continue
            run_end = c
            kk = k
            while inside[cyc[(kk + 1) % 4]] and (kk + 1) % 4 != k:
                kk = (kk + 1) % 4
                run_end = cyc[kk]
            if inside[cyc[(kk + 1) % 4]]:
                continue                                   # all four corners inside: no crossing on this face
            e_in = _EDGE_OF[frozenset((cp, c))]            # crossing edge before the run
            e_out = _EDGE_OF[frozenset((run_end, cyc[(kk + 1) % 4]))]   # crossing edge after the run
            # the segment runs from the crossing edge BEFORE the run to the one AFTER it (counter-clockwise seen from
            # outside the cube, i.e. around the inside corners it cuts off): with this orientation the loops' normals point
            # away from the inside corners, out of the fluid (pinned: positive enclosed volume of a sphere)
            assert e_in not in nxt
            nxt[e_in] = e_out
    tris = []
    seen = set()
    for start in sorted(nxt):
        if start in seen:
            continue
        loop = [start]
        seen.add(start)
        e = nxt[start]
        while e != start:
            loop.append(e)
            seen.add(e)
            e = nxt[e]
        for k in range(1, len(loop) - 1):
            tris.append((loop[0], loop[k], loop[k + 1]))
    return tris


_TABLE = None


def case_table():
    """256 lists of edge-id triples."""
    global _TABLE
    if _TABLE is None:
        _TABLE = [case_triangles(m) for m in range(256)]
    return _TABLE


# ---------------------------------------------------------------------------------------------- field
def kernel_w(r: np.ndarray, h: float) -> np.ndarray:
    """Cubic spline with support radius h (reading R1), restated here (the surface oracle is self-contained)."""
    q = np.asarray(r, dtype=np.float64) / h
    sigma = 8.0 / (np.pi * h ** 3)
    w = np.where(q <= 0.5, 6.0 * (q ** 3 - q ** 2) + 1.0, np.where(q <= 1.0, 2.0 * (1.0 - np.minimum(q, 1.0)) ** 3, 0.0))
    return sigma * w


def grid_nodes(grid_min, dims, cube_size):
    """Node coordinates as the CUDA path defines them: fp32 grid_min + fp32(index) * fp32 cube_size, evaluated in fp32
    (so both sides sample the field at bit-identical points), returned as fp64, shape (nz, ny, nx, 3)."""
    gm = np.asarray(grid_min, dtype=np.float32)
    cs = np.float32(cube_size)
    ax = [gm[a] + np.arange(dims[a], dtype=np.float32) * cs for a in range(3)]
    z, y, x = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return np.stack([x, y, z], axis=-1).astype(np.float64)


def scalar_field(pos, vol, h, grid_min, dims, cube_size):
    """phi(g) = sum_i V_i W(|g - x_i|, h) on every node; shape (nz, ny, nx).  Strict support: |g - x_i| < h."""
    pos = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    vol = np.asarray(vol, dtype=np.float64).reshape(-1)
    g = grid_nodes(grid_min, dims, cube_size)
    phi = np.zeros(g.shape[:3])
    # plain loop over particles, vectorised over the nodes of the particle's bounding box
    gm = np.asarray(grid_min, dtype=np.float64)
    for x, v in zip(pos, vol):
        lo = np.maximum(np.floor((x - h - gm) / cube_size).astype(int) - 1, 0)
        hi = np.minimum(np.ceil((x + h - gm) / cube_size).astype(int) + 2, np.asarray(dims))
        if np.any(hi <= lo):
            continue
        sub = g[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]]
        r = np.linalg.norm(sub - x, axis=-1)
        phi[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] += np.where(r < h, v * kernel_w(r, h), 0.0)
    return phi


# ---------------------------------------------------------------------------------------------- marching cubes
def marching_cubes(phi, iso, grid_min, cube_size):
    """Triangle soup of the iso-surface: (ntri, 3, 3) float64 vertex coordinates and (ntri,) cell ids (x-fastest
    linear index over the (nx-1)(ny-1)(nz-1) cells), in cell order, triangles of a cell in table order.
    phi: (nz, ny, nx); it is used AS GIVEN (the parity tests hand the CUDA path's fp32 field over, so that the inside /
    outside decisions are taken on identical numbers)."""
    phi = np.asarray(phi)
    nz, ny, nx = phi.shape
    nodes = grid_nodes(grid_min, (nx, ny, nz), cube_size)
    table = case_table()
    tris, cells = [], []
    f64 = phi.astype(np.float64)
    for iz in range(nz - 1):
        for iy in range(ny - 1):
            for ix in range(nx - 1):
                vals = [f64[iz + d[2], iy + d[1], ix + d[0]] for d in CORNERS]
                mask = 0
                for c in range(8):
                    if vals[c] > iso:
                        mask |= 1 << c
                if mask == 0 or mask == 255:
                    continue
                pts = {}
                for t in table[mask]:
                    tri = []
                    for e in t:
                        if e not in pts:
                            a, b = EDGES[e]
                            pa = nodes[iz + CORNERS[a][2], iy + CORNERS[a][1], ix + CORNERS[a][0]]
                            pb = nodes[iz + CORNERS[b][2], iy + CORNERS[b][1], ix + CORNERS[b][0]]
                            s = (iso - vals[a]) / (vals[b] - vals[a])
                            pts[e] = pa + s * (pb - pa)
                        tri.append(pts[e])
                    tris.append(tri)
                    cells.append(ix + (nx - 1) * (iy + (ny - 1) * iz))
    if not tris:
        return np.zeros((0, 3, 3)), np.zeros((0,), dtype=np.int64)
    return np.asarray(tris, dtype=np.float64), np.asarray(cells, dtype=np.int64)


def mesh_volume_area(tris):
    """Enclosed volume (divergence theorem, positive for outward normals) and area of a triangle soup."""
    a, b, c = tris[:, 0], tris[:, 1], tris[:, 2]
    vol = np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0
    area = 0.5 * np.linalg.norm(np.cross(b - a, c - a), axis=1).sum()
    return float(vol), float(area)


def mesh_topology(tris, decimals=9):
    """(V, E, F, every directed edge is matched by exactly one opposite edge) of a triangle soup, vertices merged by
    rounded coordinates."""
    key = np.round(tris.reshape(-1, 3), decimals)
    uniq, inv = np.unique(key, axis=0, return_inverse=True)
    f = inv.reshape(-1, 3)
    directed = {}
    for t in f:
        for k in range(3):
            e = (int(t[k]), int(t[(k + 1) % 3]))
            directed[e] = directed.get(e, 0) + 1
    closed = all(n == 1 and directed.get((b, a), 0) == 1 for (a, b), n in directed.items())
    E = len({frozenset(e) for e in directed})
    return len(uniq), E, len(f), closed
