"""fp64 CPU oracle of the particle image stage (reading R30 of DESIGN.md).  TEST INFRASTRUCTURE ONLY: imported by
tests/, never by the product (paper_2403_11156_b200/) -- it shares no code with the CUDA path.

The paper renders its results with a third-party path tracer (Blender Cycles, OptiX) and prints no
equation for it; SURVEY.md 8(f) NEXT-4 asks for "a CUDA sphere-splat / ray-march image of the particles" into a
headless buffer instead.  Reading R30 fixes what that image is:

  camera      orthographic: origin o, orthonormal image axes `right`, `up`, view direction w = right x up;
              pixel (px, py) looks along w through the point o + X right + Y up, X = (px + 1/2) ps, Y = (py + 1/2) ps
  particle    a sphere of radius R at c: in camera coordinates a = (c - o).right, b = (c - o).up, z = (c - o).w
  coverage    q = R^2 - (X - a)^2 - (Y - b)^2 > 0
  depth       t = z - sqrt(q)       (first intersection of the pixel's ray with the sphere)
  pixel       depth = min over the covering particles, id = the particle that attains it (smallest id among equals);
              empty pixels: depth = +inf, id = -1, shade = 0
  shade       Lambert term max(0, -n.l) with the unit normal n = ((X - a) right + (Y - b) up - sqrt(q) w) / R at the
              hit point and l = light / |light| (the direction the light travels)

Everything is written out particle by particle and pixel by pixel (numpy only vectorises the pixel block one sphere
covers).  `gap` (second smallest depth minus the smallest) and `edge` (min over particles of |q| / R^2) are returned for
the tests: they mark the pixels where a different rounding may legitimately pick another particle or flip coverage.
"""
from __future__ import annotations

import numpy as np


def camera_axes(right, up):
    r = np.asarray(right, dtype=np.float64)
    u = np.asarray(up, dtype=np.float64)
    return r, u, np.cross(r, u)


def render(pos, ids, origin, right, up, pixel_size, width, height, radius, light):
    """pos (n, 3), ids (n,) -> depth (H, W) f64, id (H, W) i64, shade (H, W) f64, gap (H, W) f64, edge (H, W) f64."""
    pos = np.asarray(pos, dtype=np.float64)
    ids = np.asarray(ids, dtype=np.int64)
    o = np.asarray(origin, dtype=np.float64)
    r, u, w = camera_axes(right, up)
    ps, R = float(pixel_size), float(radius)
    l = np.asarray(light, dtype=np.float64)
    l = l / np.linalg.norm(l)
    depth = np.full((height, width), np.inf)
    second = np.full((height, width), np.inf)
    win = np.full((height, width), -1, dtype=np.int64)
    shade = np.zeros((height, width))
    edge = np.full((height, width), np.inf)
    lr, lu, lw = float(l @ r), float(l @ u), float(l @ w)
    for c, pid in zip(pos, ids):
        a, b, z = float((c - o) @ r), float((c - o) @ u), float((c - o) @ w)
        # pixels whose centre can lie inside the disc (one pixel of margin: `edge` also wants the near misses)
        x0 = max(int(np.floor((a - R) / ps - 0.5)) - 1, 0); x1 = min(int(np.ceil((a + R) / ps - 0.5)) + 1, width - 1)
        y0 = max(int(np.floor((b - R) / ps - 0.5)) - 1, 0); y1 = min(int(np.ceil((b + R) / ps - 0.5)) + 1, height - 1)
        if x1 < x0 or y1 < y0:
            continue
        X = (np.arange(x0, x1 + 1) + 0.5) * ps
        Y = (np.arange(y0, y1 + 1) + 0.5) * ps
        dx = X[None, :] - a
        dy = Y[:, None] - b
        q = R * R - dx * dx - dy * dy
        blk = (slice(y0, y1 + 1), slice(x0, x1 + 1))
        edge[blk] = np.minimum(edge[blk], np.abs(q) / (R * R))
        s = np.sqrt(np.maximum(q, 0.0))
        t = np.where(q > 0.0, z - s, np.inf)
        d_old, w_old = depth[blk], win[blk]
        better = (t < d_old) | ((t == d_old) & np.isfinite(t) & (pid < w_old))
        # runner-up depth: the old best where it is beaten, else this one if it beats the old runner-up
        second[blk] = np.where(better, np.minimum(d_old, second[blk]), np.minimum(second[blk], t))
        sh = np.maximum(0.0, -((dx * lr + dy * lu - s * lw) / R))
        depth[blk] = np.where(better, t, d_old)
        win[blk] = np.where(better, pid, w_old)
        shade[blk] = np.where(better, sh, shade[blk])
    gap = np.full((height, width), np.inf)
    hit = np.isfinite(depth)
    gap[hit] = second[hit] - depth[hit]
    return depth, win, shade, gap, edge


def render_pixel(pos, ids, origin, right, up, pixel_size, radius, light, px, py):
    """One pixel against ALL particles (for sampled checks at full size): depth, id, shade, gap, edge."""
    pos = np.asarray(pos, dtype=np.float64)
    ids = np.asarray(ids, dtype=np.int64)
    o = np.asarray(origin, dtype=np.float64)
    r, u, w = camera_axes(right, up)
    ps, R = float(pixel_size), float(radius)
    l = np.asarray(light, dtype=np.float64)
    l = l / np.linalg.norm(l)
    X, Y = (px + 0.5) * ps, (py + 0.5) * ps
    rel = pos - o[None, :]
    dx = X - rel @ r
    dy = Y - rel @ u
    z = rel @ w
    q = R * R - dx * dx - dy * dy
    edge = float(np.min(np.abs(q)) / (R * R)) if len(q) else np.inf
    hit = np.nonzero(q > 0.0)[0]
    if hit.size == 0:
        return np.inf, -1, 0.0, np.inf, edge
    s = np.sqrt(q[hit])
    t = z[hit] - s
    order = np.lexsort((ids[hit], t))
    k = order[0]
    gap = float(t[order[1]] - t[k]) if hit.size > 1 else np.inf
    sh = max(0.0, -float((dx[hit][k] * (l @ r) + dy[hit][k] * (l @ u) - s[k] * (l @ w)) / R))
    return float(t[k]), int(ids[hit][k]), sh, gap, edge
