"""Pins of the particle-image oracle (oracle/render_ref.py, reading R30): closed forms of one sphere, occlusion,
an independent 3-D ray / sphere brute force, invariance under a common rotation of camera and particles, empty pixels.
The paper prints nothing for this stage (PAPER.md:274, 282 name a third-party renderer), so mathematics is the pin."""
import numpy as np

from oracle import render_ref as R

EX, EY, EZ = np.eye(3)


def test_single_sphere_closed_forms():
    """Sphere of radius 0.5 whose centre lies on a pixel centre, camera looking along +z, light along the view:
    depth(dx) = z - sqrt(R^2 - dx^2), shade = sqrt(R^2 - dx^2) / R, covered pixels ~ pi R^2 / ps^2."""
    ps, rad = 0.01, 0.5
    n = 129                                        # centre of pixel 64 is at 0.645
    c = np.array([[0.645, 0.645, 3.0]])
    d, i, s, gap, edge = R.render(c, [7], (0, 0, 0), EX, EY, ps, n, n, rad, (0, 0, 1))
    assert abs(d[64, 64] - 2.5) < 1e-12 and i[64, 64] == 7 and abs(s[64, 64] - 1.0) < 1e-12
    for k in (1, 10, 30, 49):
        dx = k * ps
        want = 3.0 - np.sqrt(rad * rad - dx * dx)
        assert abs(d[64, 64 + k] - want) < 1e-12 and abs(d[64 - k, 64] - want) < 1e-12
        assert abs(s[64, 64 + k] - np.sqrt(rad * rad - dx * dx) / rad) < 1e-12
    assert np.isinf(d[64, 64 + 51]) and i[64, 64 + 51] == -1 and s[64, 64 + 51] == 0.0     # outside the silhouette
    covered = np.isfinite(d).sum()
    assert abs(covered - np.pi * rad * rad / (ps * ps)) < 2 * np.pi * rad / ps              # within one pixel ring
    assert np.array_equal(np.isfinite(d), i >= 0) and np.isinf(gap).all()
    # light from the side (+x travelling): the half facing -x is lit, the other is dark; symmetric in y
    d2, _, s2, _, _ = R.render(c, [7], (0, 0, 0), EX, EY, ps, n, n, rad, (1, 0, 0))
    assert np.array_equal(d2, d)
    assert abs(s2[64, 64 - 30] - 0.3 / 0.5) < 1e-12 and s2[64, 64 + 30] == 0.0
    assert np.allclose(s2[64 - 20, :], s2[64 + 20, :])


def test_occlusion_and_id_of_equal_depths():
    ps = 0.02
    pos = np.array([[0.5, 0.5, 2.0], [0.5, 0.5, 1.0], [0.52, 0.5, 1.0], [0.9, 0.9, 5.0]])
    d, i, s, gap, _ = R.render(pos, [10, 11, 12, 13], (0, 0, 0), EX, EY, ps, 60, 60, 0.1, (0, 0, 1))
    # the far sphere 10 is hidden completely by 11 (same axis, nearer)
    assert not (i == 10).any() and (i == 11).any() and (i == 12).any() and (i == 13).any()
    # on the symmetry plane x = 0.51 (a pixel centre: pixel 25) spheres 11 and 12 have EQUAL depth: smallest id wins, gap 0
    assert abs((25 + 0.5) * ps - 0.51) < 1e-12
    assert i[25, 25] == 11 and gap[25, 25] == 0.0
    assert i[25, 24] == 11 and i[25, 26] == 12 and gap[25, 24] > 0
    # order of the input must not matter
    p = [3, 1, 0, 2]
    d2, i2, s2, _, _ = R.render(pos[p], np.array([10, 11, 12, 13])[p], (0, 0, 0), EX, EY, ps, 60, 60, 0.1, (0, 0, 1))
    assert np.array_equal(d, d2) and np.array_equal(i, i2) and np.array_equal(s, s2)


def _brute_force(pos, ids, o, r, u, ps, W, H, rad, light):
    """Independent formulation: every pixel's ray P + t w against every sphere by the 3-D quadratic
    |P + t w - c|^2 = R^2, smaller root; normal from the 3-D hit point."""
    w = np.cross(r, u)
    l = np.asarray(light, float) / np.linalg.norm(light)
    depth = np.full((H, W), np.inf); win = np.full((H, W), -1); shade = np.zeros((H, W))
    for py in range(H):
        for px in range(W):
            P = np.asarray(o, float) + (px + 0.5) * ps * r + (py + 0.5) * ps * u
            best = (np.inf, -1, 0.0)
            for c, pid in zip(pos, ids):
                m = P - c
                bq = m @ w
                disc = bq * bq - (m @ m - rad * rad)
                if disc <= 0.0:
                    continue
                t = -bq - np.sqrt(disc)
                nrm = (P + t * w - c) / rad
                if (t, pid) < best[:2]:
                    best = (t, pid, max(0.0, -float(nrm @ l)))
            depth[py, px], win[py, px], shade[py, px] = best
    return depth, win, shade


def test_against_ray_sphere_brute_force_with_a_tilted_camera():
    rng = np.random.default_rng(5)
    pos = rng.uniform(0.0, 1.0, (40, 3))
    ids = rng.permutation(40)
    # an orthonormal camera frame that is not axis-aligned
    a = np.array([1.0, 0.3, -0.2]); a /= np.linalg.norm(a)
    b = np.cross(a, [0.1, 0.9, 0.4]); b /= np.linalg.norm(b)
    o = np.array([0.5, 0.5, 0.5]) - 0.7 * a - 0.7 * b - 2.0 * np.cross(a, b)
    args = (o, a, b, 0.05, 28, 28, 0.11, (0.3, -0.5, 0.8))
    d, i, s, gap, edge = R.render(pos, ids, *args)
    bd, bi, bs = _brute_force(pos, ids, *args)
    sure = edge > 1e-9
    assert np.isfinite(d).sum() > 150
    assert np.array_equal(np.isfinite(d)[sure], np.isfinite(bd)[sure])
    f = np.isfinite(d) & np.isfinite(bd)
    assert np.abs(d[f] - bd[f]).max() < 1e-12
    clear = f & (gap > 1e-9)
    assert np.array_equal(i[clear], bi[clear]) and np.abs(s[clear] - bs[clear]).max() < 1e-10
    # the sampled single-pixel form agrees with the image
    for (py, px) in [(3, 4), (14, 14), (20, 9), (27, 27), (0, 0)]:
        t, pid, sh, g, e = R.render_pixel(pos, ids, o, a, b, 0.05, 0.11, (0.3, -0.5, 0.8), px, py)
        assert (np.isinf(t) and np.isinf(d[py, px])) or abs(t - d[py, px]) < 1e-12
        assert pid == i[py, px] and abs(sh - s[py, px]) < 1e-12
        assert (np.isinf(g) and np.isinf(gap[py, px])) or abs(g - gap[py, px]) < 1e-12


def test_common_rotation_of_camera_and_particles_leaves_the_image_unchanged():
    rng = np.random.default_rng(6)
    pos = rng.uniform(0.2, 0.8, (60, 3))
    ids = np.arange(60)
    light = np.array([0.2, 0.1, 1.0])
    d, i, s, gap, _ = R.render(pos, ids, (0, 0, -1), EX, EY, 0.025, 40, 40, 0.06, light)
    # rotation about an arbitrary axis (Rodrigues)
    k = np.array([0.3, -0.7, 0.64]); k /= np.linalg.norm(k)
    th = 0.9
    K = np.array([[0, -k[2], k[1]], [k[2], 0, -k[0]], [-k[1], k[0], 0]])
    Q = np.eye(3) + np.sin(th) * K + (1 - np.cos(th)) * K @ K
    d2, i2, s2, _, _ = R.render(pos @ Q.T, ids, Q @ np.array([0, 0, -1.0]), Q @ EX, Q @ EY, 0.025, 40, 40, 0.06, Q @ light)
    f = np.isfinite(d)
    assert np.array_equal(f, np.isfinite(d2)) and np.abs(d[f] - d2[f]).max() < 1e-12
    clear = f & (gap > 1e-9)
    assert np.array_equal(i[clear], i2[clear]) and np.abs(s[clear] - s2[clear]).max() < 1e-10


def test_empty_image_and_particles_outside_the_view():
    d, i, s, gap, edge = R.render(np.zeros((0, 3)), [], (0, 0, 0), EX, EY, 0.1, 8, 6, 0.05, (0, 0, 1))
    assert d.shape == (6, 8) and np.isinf(d).all() and (i == -1).all() and (s == 0).all()
    d, i, s, _, _ = R.render([[-5.0, 0.2, 1.0], [0.4, 9.0, 1.0]], [0, 1], (0, 0, 0), EX, EY, 0.1, 8, 6, 0.05, (0, 0, 1))
    assert np.isinf(d).all() and (i == -1).all()
    # a sphere cut by the image border covers only the pixels inside
    d, i, _, _, _ = R.render([[0.0, 0.3, 1.0]], [4], (0, 0, 0), EX, EY, 0.1, 8, 6, 0.25, (0, 0, 1))
    assert (i[:, 0] == 4).sum() >= 3 and (i[:, 3:] == -1).all()
