"""Pins of the post-processing oracle (oracle/surface_ref.py, reading R29).
CPU only.  The field is pinned by closed forms; the GENERATED marching-cubes case table and the mesh it produces are
pinned by what any correct iso-surface of a known field must satisfy: closed 2-manifold, Euler characteristic,
outward orientation, enclosed volume and area converging to the analytic values."""
import numpy as np
import pytest

from oracle import surface_ref as SR

R = 0.01
S = 2 * R
H = 4 * R


def test_case_table_structure():
    """All 256 cases: empty for 0 / 255; only crossing edges are used and every crossing edge is used; each case's
    triangles form closed, consistently oriented loops when the cube faces are added (every directed triangle edge that
    is not matched inside the cell lies on a cube face); at most 5 triangles per cell (the classic bound);
    single-corner cases give exactly one triangle on that corner's three edges."""
    tab = SR.case_table()
    assert tab[0] == [] and tab[255] == []
    assert max(len(t) for t in tab) <= 5
    for mask in range(256):
        inside = [(mask >> c) & 1 for c in range(8)]
        crossing = {k for k, (a, b) in enumerate(SR.EDGES) if inside[a] != inside[b]}
        used = {e for t in tab[mask] for e in t}
        assert used == crossing, mask
        # n-gon loops fan-triangulated: triangles = crossing edges - 2 * loops  => parity / bounds
        assert len(tab[mask]) >= (1 if crossing else 0)
        for t in tab[mask]:
            assert len(set(t)) == 3
    for c in range(8):
        t = tab[1 << c]
        assert len(t) == 1 and set(t[0]) == {k for k, e in enumerate(SR.EDGES) if c in e}
        # the complementary case cuts the same corner off with the opposite orientation
        tc = tab[255 ^ (1 << c)]
        assert len(tc) == 1 and set(tc[0]) == set(t[0])
        i = t[0].index(tc[0][0])
        assert (t[0][(i + 1) % 3], t[0][(i + 2) % 3]) == (tc[0][2], tc[0][1])


def test_ambiguous_faces_agree_between_neighbouring_cells():
    """The face rule depends on the face's corner signs only: for every pair of cases that share the face x = 1 / x = 0
    with identical corner signs, the segments on that face (pairs of face edges joined by a triangle side) coincide.
    Catches a table whose ambiguous cases tear the mesh."""
    tab = SR.case_table()
    face_hi = [k for k, (a, b) in enumerate(SR.EDGES) if (a & 1) and (b & 1)]     # edges on the face x = 1
    face_lo = [k for k, (a, b) in enumerate(SR.EDGES) if not (a & 1) and not (b & 1)]
    lo_of_hi = {}
    for k in face_hi:
        a, b = SR.EDGES[k]
        lo_of_hi[k] = SR._EDGE_OF[frozenset((a - 1, b - 1))]

    def segs(mask, face):
        out = set()
        for t in tab[mask]:
            for i in range(3):
                e0, e1 = t[i], t[(i + 1) % 3]
                if e0 in face and e1 in face:
                    out.add(frozenset((e0, e1)))
        return out

    rng = np.random.default_rng(0)
    for _ in range(400):
        left, right = int(rng.integers(256)), int(rng.integers(256))
        # make the shared face agree: corners with x = 1 of `left` == corners with x = 0 of `right`
        for c in range(8):
            if not (c & 1):
                right = (right & ~(1 << c)) | (((left >> (c + 1)) & 1) << c)
        sl = {frozenset(lo_of_hi[e] for e in s) for s in segs(left, set(face_hi))}
        sr = segs(right, set(face_lo))
        assert sl == sr, (left, right)


def test_field_closed_forms():
    """One particle: phi(g) = V W(|g - x|) at every node (strict support).  Uniform lattice with V = m / rho of that
    lattice: phi = 1 at a particle site (sum_j V W_ij = (m / rho) (rho / m))."""
    x = np.array([[0.1, 0.1, 0.1]])
    V = np.array([8e-6])
    gmin, dims, cs = (0.05, 0.05, 0.05), (11, 11, 11), 0.01
    phi = SR.scalar_field(x, V, H, gmin, dims, cs)
    g = SR.grid_nodes(gmin, dims, cs)
    r = np.linalg.norm(g - x[0], axis=-1)
    sigma = 8.0 / (np.pi * H ** 3)
    assert phi[5, 5, 5] == pytest.approx(V[0] * sigma, rel=1e-6)          # node ~ on the particle (fp32 node coordinates)
    q = r / H
    ref = V[0] * sigma * np.where(q <= 0.5, 6 * (q ** 3 - q ** 2) + 1, np.where(q < 1, 2 * (1 - q) ** 3, 0.0))
    assert np.allclose(phi, ref, rtol=1e-12, atol=0)
    assert (phi[r >= H] == 0).all() and (phi[r < 0.99 * H] > 0).all()
    # lattice: 7^3 particles, spacing S; node on the central particle
    gr = (np.arange(7) + 0.5) * S
    z, y, xx = np.meshgrid(gr, gr, gr, indexing="ij")
    pos = np.stack([xx.ravel(), y.ravel(), z.ravel()], 1)
    m = 1000.0 * S ** 3
    rho = 0.99997247 * 1000.0                                              # golden lattice density (closed_forms.txt)
    phi = SR.scalar_field(pos, np.full(len(pos), m / rho), H, tuple(pos[171] - 0.0), (2, 2, 2), S)
    assert phi[0, 0, 0] == pytest.approx(1.0, abs=2e-7)


def _sphere_field(n, radius, centre=(0.5, 0.5, 0.5)):
    cs = 1.0 / (n - 1)
    g = SR.grid_nodes((0.0, 0.0, 0.0), (n, n, n), cs)
    return radius - np.linalg.norm(g - np.asarray(centre), axis=-1), cs


@pytest.mark.parametrize("n", [13, 25])
def test_marching_cubes_sphere(n):
    """Iso-surface 0 of phi = R - |x - c|: closed 2-manifold (every directed edge matched by exactly one opposite one),
    Euler characteristic 2, OUTWARD normals (positive volume), volume and area within O(cube_size^2) of
    4/3 pi R^3 and 4 pi R^2, vertices ON the cell edges at the linear-interpolation point."""
    Rs = 0.31
    phi, cs = _sphere_field(n, Rs)
    tris, cells = SR.marching_cubes(phi, 0.0, (0.0, 0.0, 0.0), cs)
    V, E, F, closed = SR.mesh_topology(tris)
    assert closed and V - E + F == 2
    vol, area = SR.mesh_volume_area(tris)
    tol = 2.5 * (cs / Rs) ** 2
    assert vol > 0
    assert vol == pytest.approx(4 / 3 * np.pi * Rs ** 3, rel=tol)
    assert area == pytest.approx(4 * np.pi * Rs ** 2, rel=tol)
    # every vertex lies within the linear-interpolation error of the sphere: |r - R| <= cs^2 / (8 R) * 3 (3 axes)
    rad = np.linalg.norm(tris.reshape(-1, 3) - 0.5, axis=1)
    assert np.abs(rad - Rs).max() <= 0.5 * cs * cs / Rs
    assert np.all(np.diff(cells) >= 0)                                     # cell order


def test_marching_cubes_topology_of_torus_and_two_spheres():
    """Genus and components: a torus has Euler characteristic 0, two disjoint spheres 4 -- with many ambiguous faces on
    the way.  Both meshes closed and outward oriented."""
    n = 33
    cs = 1.0 / (n - 1)
    g = SR.grid_nodes((0.0, 0.0, 0.0), (n, n, n), cs) - 0.5
    rho = np.sqrt(g[..., 0] ** 2 + g[..., 1] ** 2)
    torus = 0.11 - np.sqrt((rho - 0.28) ** 2 + g[..., 2] ** 2)
    tris, _ = SR.marching_cubes(torus, 0.0, (0.0, 0.0, 0.0), cs)
    V, E, F, closed = SR.mesh_topology(tris)
    assert closed and V - E + F == 0
    vol, _ = SR.mesh_volume_area(tris)
    assert vol == pytest.approx(2 * np.pi ** 2 * 0.28 * 0.11 ** 2, rel=0.03)
    two = np.maximum(0.17 - np.linalg.norm(g - np.array([0.22, 0.0, 0.0]), axis=-1),
                     0.17 - np.linalg.norm(g + np.array([0.22, 0.0, 0.0]), axis=-1))
    tris, _ = SR.marching_cubes(two, 0.0, (0.0, 0.0, 0.0), cs)
    V, E, F, closed = SR.mesh_topology(tris)
    assert closed and V - E + F == 4


def test_marching_cubes_random_field_is_watertight():
    """A rough random field exercises every case incl. all ambiguous ones: the mesh is still closed away from the grid
    border (checked on a field forced negative on the border, so that the surface cannot leave the grid)."""
    rng = np.random.default_rng(5)
    phi = rng.uniform(-1, 1, size=(9, 10, 11))
    phi[0] = phi[-1] = -1; phi[:, 0] = phi[:, -1] = -1; phi[:, :, 0] = phi[:, :, -1] = -1
    tris, _ = SR.marching_cubes(phi, 0.0, (0.0, 0.0, 0.0), 0.1)
    V, E, F, closed = SR.mesh_topology(tris)
    assert F > 300 and closed
    assert SR.mesh_volume_area(tris)[0] > 0
    used = set()
    nz, ny, nx = phi.shape
    for iz in range(nz - 1):
        for iy in range(ny - 1):
            for ix in range(nx - 1):
                m = 0
                for c, d in enumerate(SR.CORNERS):
                    m |= int(phi[iz + d[2], iy + d[1], ix + d[0]] > 0) << c
                used.add(m)
    assert len(used) > 180                                                  # most of the 256 cases occurred
