"""GPU parity of the particle image stage (sph_render_particles, reading R30) against oracle/render_ref.py, through the
C ABI.  Depth is compared wherever both sides see a particle; the particle id and the Lambert term wherever the decision
is unique (the oracle's runner-up is farther than the fp32 noise, and no silhouette passes through the pixel centre)."""
import numpy as np
import pytest

from paper_2403_11156_b200 import scenes
from gpu_util import np_

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2403_11156_b200 import binding, build
    build.build()
    binding.load()
    return binding


def _camera(look, up_hint, centre, half_w, half_h, back):
    w = np.asarray(look, float); w /= np.linalg.norm(w)
    r = np.cross(np.asarray(up_hint, float), w); r /= np.linalg.norm(r)
    u = np.cross(w, r)                                   # right x up = w
    assert np.allclose(np.cross(r, u), w)
    o = np.asarray(centre, float) - half_w * r - half_h * u - back * w
    return o, r, u


def _compare(depth, pid, shade, ref, scale):
    rd, ri, rs, gap, edge = ref
    cov, rcov = np.isfinite(depth), np.isfinite(rd)
    sure = edge > 1e-4                                   # no silhouette through the pixel centre
    assert np.array_equal(cov[sure], rcov[sure])
    assert (~sure).sum() < 0.01 * sure.size
    both = cov & rcov & (edge > 1e-3)
    assert both.sum() > 0.2 * rcov.sum()
    assert np.abs(depth[both] - rd[both]).max() <= 1e-5 * scale
    clear = both & (gap > 1e-4 * scale)
    assert clear.sum() > 0.8 * both.sum()
    assert np.array_equal(pid[clear], ri[clear])
    assert np.abs(shade[clear] - rs[clear]).max() <= 1e-3
    inner = clear & (edge > 0.05)
    assert np.abs(shade[inner] - rs[inner]).max() <= 1e-4
    assert (pid[~cov] == -1).all() and (shade[~cov] == 0).all() and (shade >= 0).all() and (shade <= 1.0 + 1e-6).all()


def test_render_parity_config0_after_steps(B):
    from oracle import render_ref
    import torch
    sc = scenes.config(0)
    g = B.Sim.from_scene(sc)
    g.sph_step_dfsph(40)
    pos = np_(g.sph_read_state(B.POS)).astype(np.float64)
    ids = np.arange(g.nf)
    r0 = sc.params["particle_radius"]
    for look, up_hint, light, W, H, rad in (((0.0, 1.0, 0.0), (0, 0, 1), (0.2, 1.0, -0.3), 220, 200, 0.0),
                                            ((-0.5, 0.7, -0.45), (0, 0, 1), (0.0, 0.3, -1.0), 256, 192, 1.5 * r0)):
        ps = 0.6 / W
        o, r, u = _camera(look, up_hint, (0.25, 0.25, 0.2), 0.5 * W * ps, 0.5 * H * ps, 2.0)
        depth, pid, shade = g.sph_render_particles(o, r, u, ps, W, H, radius=rad, light=light)
        d2, p2, s2 = g.sph_render_particles(o, r, u, ps, W, H, radius=rad, light=light)
        assert torch.equal(depth, d2) and torch.equal(pid, p2) and torch.equal(shade, s2)      # deterministic
        # the oracle sees the same fp32 camera and radius the library was handed
        f32 = lambda v: np.asarray(v, dtype=np.float32).astype(np.float64)
        ref = render_ref.render(pos, ids, f32(o), f32(r), f32(u), float(np.float32(ps)), W, H,
                                float(np.float32(rad if rad > 0 else r0)), light)
        assert np.isfinite(ref[0]).sum() > 2000
        _compare(np_(depth).astype(np.float64), np_(pid), np_(shade).astype(np.float64), ref, 2.5)
    # rendering does not disturb the simulation: the next steps equal those of an undisturbed run
    g2 = B.Sim.from_scene(sc)
    g2.sph_step_dfsph(45); g.sph_step_dfsph(5)
    assert torch.equal(g.sph_read_state(B.POS), g2.sph_read_state(B.POS))
    g.close(); g2.close()


def test_render_edge_cases(B):
    import ctypes as C
    import torch
    sc = scenes.dam_break((6, 6, 6), (10, 10, 10))
    g = B.Sim.from_scene(sc)
    # nothing in view: camera looks at empty space
    d, i, s = g.sph_render_particles((50, 50, 50), (1, 0, 0), (0, 1, 0), 0.01, 33, 17)
    assert torch.isinf(d).all() and (i == -1).all() and (s == 0).all() and d.shape == (17, 33)
    # one pixel
    d, i, s = g.sph_render_particles((0, 0, -1), (1, 0, 0), (0, 1, 0), 1.0, 1, 1, radius=5.0)
    assert d.shape == (1, 1) and int(i[0, 0]) >= 0
    # the zero light vector is a headlight: the same image as light = view direction (here right x up = +z)
    a = g.sph_render_particles((0, 0, -1), (1, 0, 0), (0, 1, 0), 0.004, 64, 64)
    b = g.sph_render_particles((0, 0, -1), (1, 0, 0), (0, 1, 0), 0.004, 64, 64, light=(0, 0, 2.5))
    assert torch.equal(a[2], b[2]) and float(a[2].max()) > 0.9
    # invalid cameras / sizes are rejected, and the workspace size of an invalid camera is 0
    for kw in (dict(right=(1, 0, 0), up=(1, 0, 0)), dict(right=(2, 0, 0), up=(0, 1, 0)), dict(pixel_size=0.0),
               dict(width=0), dict(radius=-1.0), dict(light=(float("nan"), 0, 0))):
        a = dict(origin=(0, 0, 0), right=(1, 0, 0), up=(0, 1, 0), pixel_size=0.01, width=8, height=8, radius=0.0, light=(0, 0, 1))
        a.update(kw)
        with pytest.raises(B.SphError):
            g.sph_render_particles(**a)
    # outputs may be NULL; too small a workspace is SPH_ENOMEM
    rp = B.SphRenderParams()
    rp.origin = (C.c_float * 3)(0, 0, -1); rp.right = (C.c_float * 3)(1, 0, 0); rp.up = (C.c_float * 3)(0, 1, 0)
    rp.pixel_size = 0.01; rp.width = 16; rp.height = 16; rp.radius = 0.0; rp.light = (C.c_float * 3)(0, 0, 1)
    L = B.load()
    need = L.sph_render_workspace_bytes(C.byref(rp), g.nf)
    assert need >= 16 * 16 * 8 + 4 * g.nf
    ws = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    wptr = ws.data_ptr() + (-ws.data_ptr()) % 256
    ids = torch.full((16, 16), -5, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    assert L.sph_render_particles(g._h, C.byref(rp), C.c_void_p(wptr), need, None, C.c_void_p(ids.data_ptr()), None) == B.SPH_OK
    g.stream.synchronize()
    assert (ids >= -1).all() and (ids >= 0).any()
    assert L.sph_render_particles(g._h, C.byref(rp), C.c_void_p(wptr), need - 1, None, None, None) == B.SPH_ENOMEM
    assert L.sph_render_particles(g._h, C.byref(rp), C.c_void_p(wptr + 4), need, None, None, None) == B.SPH_EINVAL
    g.close()


def test_render_full_size_config4_sampled(B):
    """1.23M particles of the post-impact state, 1024 x 512 top view of the whole tank: sampled pixels against the
    oracle's one-pixel form over ALL particles; global properties of the image."""
    from oracle import render_ref
    sc = scenes.config(4)
    g = B.Sim.from_scene(sc)
    g.sph_step_dfsph(130)
    pos = np_(g.sph_read_state(B.POS)).astype(np.float64)
    ids = np.arange(g.nf)
    W, H = 1024, 512
    ps = 4.0 / W
    o, r, u = (0.0, 2.0, 3.0), (1.0, 0.0, 0.0), (0.0, -1.0, 0.0)          # looking down: w = right x up = (0, 0, -1)
    light = (0.3, 0.2, -1.0)
    depth, pid, shade = g.sph_render_particles(o, r, u, ps, W, H, light=light)
    depth, pid, shade = np_(depth).astype(np.float64), np_(pid), np_(shade).astype(np.float64)
    cov = np.isfinite(depth)
    assert 0.15 * W * H < cov.sum() < 0.4 * W * H                         # two blocks of 1.0 x 0.75 m seen from above (1.5 of 8 m^2) plus the splash
    assert (pid[cov] >= 0).all() and (pid[cov] < g.nf).all() and (pid[~cov] == -1).all()
    assert 3.0 - 2.0 - 0.01 <= depth[cov].min() and depth[cov].max() <= 3.0 + 0.01
    rng = np.random.default_rng(3)
    ys, xs = np.nonzero(cov)
    pick = rng.choice(len(ys), size=150, replace=False)
    samples = [(int(ys[k]), int(xs[k])) for k in pick] + [(int(rng.integers(H)), int(rng.integers(W))) for _ in range(50)]
    R = float(np.float32(sc.params["particle_radius"]))
    checked = 0
    for py, px in samples:
        t, wid, sh, gap, edge = render_ref.render_pixel(pos, ids, o, r, u, float(np.float32(ps)), R, light, px, py)
        if edge <= 1e-4:
            continue
        assert np.isfinite(t) == bool(cov[py, px])
        if not np.isfinite(t) or edge <= 1e-3:
            continue
        assert abs(depth[py, px] - t) <= 1e-5 * 3.0
        if gap > 1e-4 * 3.0:
            assert pid[py, px] == wid and abs(shade[py, px] - sh) <= 1e-3
            checked += 1
    assert checked >= 80
    g.close()
