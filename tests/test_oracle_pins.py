"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each test names the oracle part it pins and the plausible mistake it would catch.
Citations: PAPER.md line numbers; Rn = readings listed in DESIGN.md.
"""
import numpy as np
import pytest

from paper_2403_11156_b200 import scenes

R = 0.01
S = 2 * R
H = 4 * R
RHO0 = 1000.0
SIGMA = 8.0 / (np.pi * H ** 3)


def make_sim(oracle, fpos, fvel=None, bpos=None, bbody=None, bodies=None, **prm):
    fpos = np.asarray(fpos, dtype=np.float64).reshape(-1, 3)
    fvel = np.zeros_like(fpos) if fvel is None else np.asarray(fvel, dtype=np.float64)
    bpos = np.zeros((0, 3)) if bpos is None else np.asarray(bpos, dtype=np.float64)
    if bbody is None:
        bbody = np.zeros(len(bpos), dtype=np.int32)
    if bodies is None:
        bodies = [scenes.Body(0, len(bpos), dynamic=0)] if len(bpos) else []
    p = scenes.default_params(R, 4e-4)
    allp = np.concatenate([fpos, bpos]) if len(bpos) else fpos
    p["domain_min"] = tuple(allp.min(axis=0) - 2 * H)
    p["domain_max"] = tuple(allp.max(axis=0) + 2 * H)
    p["tank_min"] = p["domain_min"]
    p["tank_max"] = p["domain_max"]
    p.update(prm)
    return oracle.Sim(fpos, fvel, bpos, bbody, bodies, p)


# ---------------------------------------------------------------- kernel (R1, R2)

def test_kernel_normalisation_quadrature(oracle):
    """4 pi int_0^h W r^2 dr = 1: catches a wrong sigma or a wrong branch polynomial."""
    n = 200000
    r = (np.arange(n) + 0.5) * (H / n)
    w = np.array([oracle.W(x, H) for x in r[::100]])  # coarse check of callable
    assert np.all(w >= 0)
    rr = (np.arange(20000) + 0.5) * (H / 20000)
    ww = np.array([oracle.W(x, H) for x in rr])
    integral = 4 * np.pi * np.sum(ww * rr ** 2) * (H / 20000)
    assert abs(integral - 1.0) < 1e-7


def test_kernel_branch_values(oracle):
    """sigma h^3 = 8/pi; W(h) = 0; both branches meet at q = 1/2 with value sigma/4 and
    slope -1.5 sigma/h (hand evaluation of the cubic spline)."""
    assert oracle.W(0.0, H) * H ** 3 == pytest.approx(8 / np.pi, rel=1e-14)
    assert oracle.W(H, H) == 0.0
    assert oracle.W(1.0001 * H, H) == 0.0
    e = 1e-9 * H
    assert oracle.W(0.5 * H - e, H) == pytest.approx(SIGMA / 4, rel=1e-7)
    assert oracle.W(0.5 * H + e, H) == pytest.approx(SIGMA / 4, rel=1e-7)
    # q = 1/4: 6 (1/64 - 1/16) + 1 = 23/32
    assert oracle.W(0.25 * H, H) == pytest.approx(SIGMA * 23 / 32, rel=1e-14)
    # q = 3/4: 2 (1/4)^3 = 1/32
    assert oracle.W(0.75 * H, H) == pytest.approx(SIGMA / 32, rel=1e-14)
    for q in (0.5 - 1e-9, 0.5 + 1e-9):
        g = oracle.gradW([q * H, 0, 0], H)
        assert g[0] == pytest.approx(-1.5 * SIGMA / H, rel=1e-6)


def test_kernel_gradient_is_derivative_and_antisymmetric(oracle):
    """gradW = dW/dx by central differences (ties gradW to W: catches a wrong w'(q) or a
    missing 1/h), gradW(-x) = -gradW(x), gradW(0) = 0 (R2), non-positive multiple of x."""
    rng = np.random.default_rng(0)
    for _ in range(50):
        d = rng.uniform(-1, 1, 3)
        d *= rng.uniform(0.02, 0.99) * H / np.linalg.norm(d)
        g = oracle.gradW(d, H)
        eps = 1e-7 * H
        fd = np.array([(oracle.W(np.linalg.norm(d + eps * e), H) - oracle.W(np.linalg.norm(d - eps * e), H)) / (2 * eps)
                       for e in np.eye(3)])
        assert np.allclose(g, fd, rtol=1e-5, atol=1e-6 * SIGMA / H)
        assert np.allclose(oracle.gradW(-d, H), -g, rtol=0, atol=0)
        assert np.dot(g, d) <= 0.0
        assert np.linalg.norm(np.cross(g, d)) < 1e-12 * np.linalg.norm(g) * np.linalg.norm(d) + 1e-300
    assert np.all(oracle.gradW([0, 0, 0], H) == 0)
    assert np.all(oracle.gradW([1.01 * H, 0, 0], H) == 0)


# ---------------------------------------------------------------- grid + neighbour sets (R10, R11)

def brute_force_sets(xq, xs, h, skip_self):
    """O(N^2) neighbour sets with the fp32 predicate of R10 written with numpy float32 ops:
    d2 = fma(dz, dz, fma(dy, dy, dx*dx)); fma emulated exactly in float64 then rounded
    (a product of two float32 is exact in float64; the sum of that and a float32 rounds once
    to float64 then once to float32 -- double rounding is possible in principle, so boundary
    cases are detected and resolved with exact rationals)."""
    from fractions import Fraction
    xq = xq.astype(np.float32); xs = xs.astype(np.float32)
    h2 = np.float32(h) * np.float32(h)
    out = []
    for i in range(len(xq)):
        d = (xq[i][None, :] - xs).astype(np.float32)        # fp32 subtraction
        dx, dy, dz = d[:, 0].astype(np.float64), d[:, 1].astype(np.float64), d[:, 2].astype(np.float64)
        t0 = (dx * dx).astype(np.float32).astype(np.float64)      # fp32 rounding of exact product
        t1 = (dy * dy + t0)                                      # may be inexact in f64
        t1f = t1.astype(np.float32)
        t2 = (dz * dz + t1f.astype(np.float64))
        d2 = t2.astype(np.float32)
        mask = d2 < h2
        # exact re-evaluation of anything within 2 ulp of the threshold
        near = np.abs(d2.astype(np.float64) - float(h2)) <= 4 * np.spacing(np.float32(h2))
        for j in np.nonzero(near)[0]:
            fx, fy, fz = Fraction(float(d[j, 0])), Fraction(float(d[j, 1])), Fraction(float(d[j, 2]))
            a = np.float32(float(fx * fx))                       # correctly rounded product
            b = _round32(fy * fy + Fraction(float(a)))
            c = _round32(fz * fz + Fraction(float(b)))
            mask[j] = c < h2
        if skip_self:
            mask[i] = False
        out.append(set(np.nonzero(mask)[0].tolist()))
    return out


def _round32(fr):
    """Correctly round an exact Fraction to float32 (via nearest of the two float32 neighbours)."""
    x = np.float32(float(fr))   # float(fr) is correctly rounded to f64; then to f32: may double round
    cands = [x, np.nextafter(x, np.float32(np.inf)), np.nextafter(x, np.float32(-np.inf))]
    from fractions import Fraction
    best = min(cands, key=lambda c: (abs(Fraction(float(c)) - fr), int(np.float32(c).view(np.uint32)) & 1))
    return np.float32(best)


def csr_sets(start, idx):
    return [set(idx[start[i]:start[i + 1]].tolist()) for i in range(len(start) - 1)]


def independent_cell_keys(pos, prm):
    """Reading R11 recomputed with numpy float32 ops."""
    h = np.float32(prm["support_radius"])
    c = h * np.float32(1.0009765625)
    inv_c = np.float32(1.0) / c
    o = np.asarray(prm["domain_min"], dtype=np.float32)
    mx = np.asarray(prm["domain_max"], dtype=np.float32)
    n = (np.floor((mx - o) * inv_c).astype(np.int64) + 1)
    t = ((pos.astype(np.float32) - o) * inv_c).astype(np.float32)
    ci = np.clip(np.floor(t).astype(np.int64), 0, n - 1)
    return (ci[:, 0] + n[0] * (ci[:, 1] + n[1] * ci[:, 2])).astype(np.int64), n


@pytest.mark.parametrize("kind", ["random", "lattice", "one_cell", "cell_faces"])
def test_neighbor_sets_match_brute_force(oracle, kind):
    """Cell-list neighbour sets (fluid and boundary) == O(N^2) brute force with the same fp32
    predicate; cell_start = cumulative histogram; keys match an independent recomputation.
    Catches: a missed adjacent cell, wrong clamping at the grid edge, wrong linearisation,
    <= instead of <, self-inclusion."""
    rng = np.random.default_rng(1)
    if kind == "random":
        sc = scenes.random_cloud(1500, (0.3, 0.25, 0.2), seed=3, n_boundary=400)
        fpos, bpos = sc.fluid_pos, sc.boundary_pos
    elif kind == "lattice":
        sc = scenes.dam_break((7, 6, 5), (9, 8, 7))
        fpos, bpos = sc.fluid_pos, sc.boundary_pos
    elif kind == "one_cell":
        fpos = (rng.uniform(0, 1, (300, 3)) * 0.9 * H + 5 * H).astype(np.float32)
        bpos = (rng.uniform(0, 1, (50, 3)) * 0.9 * H + 5 * H).astype(np.float32)
    else:  # particles exactly on cell faces / at exactly h distance
        c = np.float32(H) * np.float32(1.0009765625)
        g = np.arange(0, 6, dtype=np.float32) * c
        z, y, x = np.meshgrid(g, g, g, indexing="ij")
        fpos = np.stack([x.ravel(), y.ravel(), z.ravel()], 1).astype(np.float32)
        fpos = np.concatenate([fpos, fpos[:50] + np.float32(H) * np.array([1, 0, 0], dtype=np.float32)])
        bpos = fpos[::7] + np.float32(0.5 * H)
    prm = {}
    if kind == "cell_faces":
        prm = dict(domain_min=(0.0, 0.0, 0.0), domain_max=tuple(float(v) for v in fpos.max(0) + np.float32(H)))
    sim = make_sim(oracle, fpos, bpos=bpos, **prm)
    sim.build_grid()
    nf = len(fpos)
    st, idx = sim.neighbors(0)
    assert csr_sets(st, idx) == brute_force_sets(fpos, fpos, H, True)
    stb, idxb = sim.neighbors(1)
    assert csr_sets(stb, idxb) == brute_force_sets(fpos, bpos, H, False)
    # grid structure
    keys, n = independent_cell_keys(fpos, sim.params)
    assert sim.grid_dims(0)[:3] == tuple(int(v) for v in n)
    assert np.array_equal(sim.cell_of_particle(0), keys)
    cs = sim.cell_start(0)
    ncell = int(np.prod(n))
    assert cs[0] == 0 and cs[-1] == nf and len(cs) == ncell + 1
    assert np.array_equal(cs, np.concatenate([[0], np.cumsum(np.bincount(keys, minlength=ncell))]))
    assert sim.stats()["oob_count"] == 0


def test_out_of_domain_particles_are_clamped_and_counted(oracle):
    fpos = np.array([[0.1, 0.1, 0.1], [0.5, 0.1, 0.1], [-0.3, 0.1, 0.1]], dtype=np.float32)
    sim = make_sim(oracle, fpos, domain_min=(0.0, 0.0, 0.0), domain_max=(0.3, 0.3, 0.3))
    sim.build_grid()
    assert sim.stats()["oob_count"] == 2
    nx = sim.grid_dims(0)[0]
    keys = sim.cell_of_particle(0)
    assert keys[1] % nx == nx - 1 and keys[2] % nx == 0


# ---------------------------------------------------------------- density / alpha (Eq. 4, R3, R5)

def test_two_particle_closed_form(oracle):
    """rho = m (W(0) + W(delta)); S = m gradW, T = |m gradW|^2 => alpha = rho / (2 T).
    delta = h/2: W = sigma/4, |gradW| = 1.5 sigma/h (hand values).  Catches a dropped self
    term, a missing square, boundary/fluid term confusion."""
    x = np.array([[0.1, 0.1, 0.1], [0.1 + 0.5 * H, 0.1, 0.1]])
    sim = make_sim(oracle, x)
    sim.build_grid(); sim.compute_density_alpha()
    m = RHO0 * S ** 3
    assert sim.mass() == pytest.approx(m, rel=1e-14)
    rho = m * (SIGMA + SIGMA / 4)
    g = 1.5 * SIGMA / H
    assert np.allclose(sim.density(), rho, rtol=1e-6)
    assert np.allclose(sim.alpha(), rho / (2 * (m * g) ** 2), rtol=1e-5)


def test_isolated_particle_alpha_guard(oracle):
    """R7: denominator <= 1e-6 => alpha = 0; density = m W(0)."""
    sim = make_sim(oracle, np.array([[0.0, 0.0, 0.0], [1.0, 1.0, 1.0]]))
    sim.build_grid(); sim.compute_density_alpha()
    assert np.all(sim.alpha() == 0.0)
    assert np.allclose(sim.density(), RHO0 * S ** 3 * SIGMA, rtol=1e-14)


def test_lattice_rest_density_and_alpha(oracle):
    """Interior of a simple-cubic lattice (spacing 2r, h = 4r, m = rho0 (2r)^3): the density is
    a Riemann sum of rho0 * int W = rho0, so |rho/rho0 - 1| is small (BASELINE.json pin); by
    symmetry S = 0.  Values from the survey's independent prototype: 0.99997247 rho0 and
    alpha = 9.41505e-7, and an explicit lattice
    sum over the 26 + 6 shell offsets is evaluated here in numpy."""
    n = 9
    g = (np.arange(n) + 0.5) * S
    z, y, x = np.meshgrid(g, g, g, indexing="ij")
    pos = np.stack([x.ravel(), y.ravel(), z.ravel()], 1)
    sim = make_sim(oracle, np.zeros((n ** 3, 3), dtype=np.float32))
    sim.set_state(pos, np.zeros_like(pos))      # exact fp64 lattice
    sim.build_grid(); sim.compute_density_alpha()
    c = (n // 2) * (n * n + n + 1)
    rho_c, al_c = sim.density()[c], sim.alpha()[c]
    assert abs(rho_c / RHO0 - 1.0) < 1e-4
    assert rho_c / RHO0 == pytest.approx(0.99997247, abs=2e-8)
    assert al_c == pytest.approx(9.41505e-7, rel=2e-6)
    # explicit shell sum: offsets (a,b,c) in {-2..2}^3 with distance < h
    tot = 0.0
    T = 0.0
    m = RHO0 * S ** 3
    for a in range(-2, 3):
        for b in range(-2, 3):
            for cc in range(-2, 3):
                d = S * np.sqrt(a * a + b * b + cc * cc)
                q = d / H
                if q <= 0.5:
                    w = 6 * (q ** 3 - q ** 2) + 1; wp = 6 * q * (3 * q - 2)
                elif q <= 1:
                    w = 2 * (1 - q) ** 3; wp = -6 * (1 - q) ** 2
                else:
                    w = 0.0; wp = 0.0
                tot += m * SIGMA * w
                if d > 0:
                    T += (m * SIGMA / H * wp) ** 2
    assert rho_c == pytest.approx(tot, rel=1e-12)
    assert al_c == pytest.approx(tot / T, rel=1e-10)


# ---------------------------------------------------------------- Akinci volumes (Eq. 11, R9)

def test_akinci_planar_closed_forms(oracle):
    """Psi / rho0 for an infinite planar lattice of spacing s = h/2, by hand from W:
    one layer: sum_k' W = sigma (1 + 4/4 + 4*2(1-1/sqrt2)^3)        => V = pi/(2 + 8a^3) s^3
    two layers: + sigma (1/4 + 4*2 a^3 + 4*2 b^3), b = 1 - sqrt3/2   => V = pi/(2.25 + 16a^3 + 8b^3) s^3
    (= 1.427341 and 1.176072).  Catches: self term missing, wrong body
    filter, rho0 misplaced."""
    a = 1 - 1 / np.sqrt(2); b = 1 - np.sqrt(3) / 2
    v1 = np.pi / (2 + 8 * a ** 3)
    v2 = np.pi / (2.25 + 16 * a ** 3 + 8 * b ** 3)
    assert v1 == pytest.approx(1.427341, abs=1e-6) and v2 == pytest.approx(1.176072, abs=1e-6)
    n = 9
    g = (np.arange(n) + 0.5) * S
    y, x = np.meshgrid(g, g, indexing="ij")
    l0 = np.stack([x.ravel(), y.ravel(), np.full(n * n, 0.5 * S)], 1)
    l1 = l0 + np.array([0, 0, S])
    fl = np.array([[10.0, 10.0, 10.0]])
    c = (n // 2) * (n + 1)
    sim = make_sim(oracle, fl, bpos=l0)
    assert sim.psi()[c] / RHO0 / S ** 3 == pytest.approx(v1, rel=2e-6)
    sim = make_sim(oracle, fl, bpos=np.concatenate([l0, l1]))
    assert sim.psi()[c] / RHO0 / S ** 3 == pytest.approx(v2, rel=2e-6)
    assert sim.psi()[n * n + c] / RHO0 / S ** 3 == pytest.approx(v2, rel=2e-6)
    # the two layers as DIFFERENT bodies must not see each other (R9)
    bb = np.concatenate([np.zeros(n * n, np.int32), np.ones(n * n, np.int32)])
    bodies = [scenes.Body(0, n * n), scenes.Body(n * n, n * n)]
    sim = make_sim(oracle, fl, bpos=np.concatenate([l0, l1]), bbody=bb, bodies=bodies)
    assert sim.psi()[c] / RHO0 / S ** 3 == pytest.approx(v1, rel=2e-6)


def test_boundary_density_term(oracle):
    """Eq. 12: one fluid particle at distance h/2 from one boundary sample:
    rho = m W(0) + Psi W(h/2), Psi = rho0 / W(0) (single-sample body)."""
    sim = make_sim(oracle, np.array([[0.1, 0.1, 0.1]]), bpos=np.array([[0.1, 0.1, 0.1 + 0.5 * H]]))
    sim.build_grid(); sim.compute_density_alpha()
    psi = RHO0 / SIGMA
    assert sim.psi()[0] == pytest.approx(psi, rel=1e-12)
    assert sim.density()[0] == pytest.approx(RHO0 * S ** 3 * SIGMA + psi * SIGMA / 4, rel=1e-6)
    # alpha: S = Psi gradW (boundary in S only), T = 0 (R5)
    g = 1.5 * SIGMA / H
    assert sim.alpha()[0] == pytest.approx(sim.density()[0] / (psi * g) ** 2, rel=1e-5)


# ---------------------------------------------------------------- solvers (Eq. 8-10, Alg. 2, [5])

def test_density_solve_two_particle_closed_form(oracle):
    """Two particles, v = 0, heavy enough that rho > rho0.  One forced iteration gives
    dv_i = +(rho - rho0) / (m |gradW| dt) along x_ij (derivation in the docstring of the
    solver pins: kappa = alpha E/dt^2, alpha = rho/(2T), U_i = m 2 kr gradW).  Catches wrong
    dt powers, sign of the correction, kappa_i + kappa_j symmetrisation."""
    dt = 4e-4
    m = 4.0 * RHO0 * S ** 3
    x = np.array([[0.1, 0.1, 0.1], [0.1 + 0.5 * H, 0.1, 0.1]])
    sim = make_sim(oracle, x, particle_mass=m, dt=dt)
    sim.build_grid(); sim.compute_density_alpha()
    rho = m * 1.25 * SIGMA
    assert rho > RHO0
    v, it = sim.density_solve(np.zeros((2, 3)), forced=1)
    dv = (rho - RHO0) / (m * 1.5 * SIGMA / H * dt)
    assert it == 1
    assert np.allclose(v, [[-dv, 0, 0], [dv, 0, 0]], rtol=1e-5, atol=1e-12)
    assert sim.stats()["err_rho"] == pytest.approx((rho - RHO0) / RHO0, rel=1e-6)


def test_divergence_solve_two_particle_closed_form(oracle):
    """Two approaching particles: one iteration removes 2x the normal relative velocity of the
    pair (each particle's alpha assumes the whole correction): v_i' = v_i - (v_ij . n) n."""
    x = np.array([[0.1, 0.1, 0.1], [0.1 + 0.5 * H, 0.1, 0.1]])
    v0 = np.array([[0.3, 0.1, 0.0], [-0.2, 0.0, 0.05]])
    sim = make_sim(oracle, x)
    sim.build_grid(); sim.compute_density_alpha()
    v, it = sim.divergence_solve(v0, forced=1)
    vn = v0[0, 0] - v0[1, 0]   # approaching along x: D > 0
    exp = v0.copy(); exp[0, 0] -= vn; exp[1, 0] += vn
    assert np.allclose(v, exp, rtol=1e-6, atol=1e-12)
    m = RHO0 * S ** 3
    D = m * vn * 1.5 * SIGMA / H
    assert sim.stats()["err_v"] == pytest.approx(4e-4 / RHO0 * D, rel=1e-5)
    # separating pair: clamp R_i = max(D, 0) => untouched (R15)
    v, _ = sim.divergence_solve(-v0, forced=1)
    assert np.allclose(v, -v0, atol=0)


def _compressed_block(oracle, n=6, squeeze=0.93, seed=0, **prm):
    sc = scenes.free_block((n, n, n), jitter=0.05, vel_scale=0.5, seed=seed)
    pos = sc.fluid_pos.astype(np.float64) * squeeze
    sim = make_sim(oracle, pos.astype(np.float32), fvel=sc.fluid_vel, **prm)
    return sim, pos.astype(np.float32).astype(np.float64), sc.fluid_vel.astype(np.float64)


def test_solvers_conserve_linear_and_angular_momentum(oracle):
    """Fluid only, g = 0: pair terms are antisymmetric and central => sum m v and
    sum x cross m v unchanged by A5 and A7 (BASELINE.json pin).  Catches any asymmetry
    (kappa_i only, wrong sign on one side, non-central force)."""
    sim, pos, vel = _compressed_block(oracle)
    sim.build_grid(); sim.compute_density_alpha()
    P0 = vel.sum(0); L0 = np.cross(pos, vel).sum(0)
    v1, it1 = sim.divergence_solve(vel, forced=3)
    assert np.abs(v1 - vel).max() > 1e-3       # the solver did something
    v2, it2 = sim.density_solve(v1, forced=3)
    assert np.abs(v2 - v1).max() > 1e-3
    scale = np.abs(vel).sum()
    for v in (v1, v2):
        assert np.abs(v.sum(0) - P0).max() < 1e-12 * scale
        assert np.abs(np.cross(pos, v).sum(0) - L0).max() < 1e-12 * scale


def test_density_solve_converges_and_reduces_error(oracle):
    """Alg. 2 loop: free-running solve exits with err_rho <= eta after >= min iterations, and
    the error of a forced longer run is monotonically small (DFSPH converges,
    BASELINE.json: average density error < 0.1 %)."""
    sim, pos, vel = _compressed_block(oracle, squeeze=0.97)
    sim.build_grid(); sim.compute_density_alpha()
    v, it = sim.density_solve(np.zeros_like(vel))
    st = sim.stats()
    assert 2 <= it < 100 and st["err_rho"] <= 1e-3
    # after the solve, the predicted density error is indeed small
    _, _ = sim.density_solve(v, forced=1)
    assert sim.stats()["err_rho"] <= 1e-3


def test_free_fall_closed_form(oracle):
    """Block far from everything: rho* <= rho0 => kappa = 0 => v_n = n g dt,
    x_n = x_0 + g dt^2 n(n+1)/2 exactly (symplectic Euler, Alg. 1 l.5-6)."""
    sc = scenes.free_block((5, 5, 5), gravity=(0.0, 0.0, -9.81))
    sc.params["domain_min"] = tuple(np.array(sc.params["domain_min"]) - np.array([0, 0, 0.5]))
    sim = oracle.Sim.from_scene(sc)
    x0 = sc.fluid_pos.astype(np.float64)
    dt = sc.params["dt"]
    n = 7
    for _ in range(n):
        sim.step_dfsph()
    assert np.allclose(sim.vel(), [0, 0, -9.81 * n * dt], rtol=1e-13, atol=1e-15)
    assert np.allclose(sim.pos() - x0, [0, 0, -9.81 * dt * dt * n * (n + 1) / 2], rtol=1e-9, atol=1e-13)


def test_dam_break_config0_small_converges(oracle):
    """Scaled config 0 (10^3 block in a 14^3 tank): every step exits with err_rho < 0.1 %,
    mass (particle count) constant, density stays within ~0.5 % of rho0."""
    sc = scenes.dam_break((10, 10, 10), (14, 14, 14))
    sim = oracle.Sim.from_scene(sc)
    for _ in range(20):
        sim.step_dfsph()
        st = sim.stats()
        assert st["err_rho"] < 1e-3 and st["oob_count"] == 0
        assert st["it_d"] >= 2 and st["it_v"] >= 1
    assert sim.density().max() < 1005.0
    assert sim.vel()[:, 2].mean() < 0.0


# ---------------------------------------------------------------- rigid coupling (Eq. 13-14, R18)

def test_fluid_rigid_momentum_exchange(oracle):
    """g = 0: sum_fluid m v + M V is conserved by the pressure exchange (Eq. 14 is the exact
    negative of Eq. 13)."""
    sc = scenes.free_block((6, 6, 6), jitter=0.03, vel_scale=0.0, seed=1)
    pos = sc.fluid_pos.astype(np.float64)
    vel = np.zeros_like(pos); vel[:, 2] = -1.0      # fluid moving down onto the body
    ctr = pos.mean(0)
    pts, body = scenes.make_rigid_box((ctr[0], ctr[1], pos[:, 2].min() - 0.5 * 0.06 - 0.8 * S), (0.06, 0.06, 0.06), 800.0, S)
    body.first_particle = 0; body.n_particles = len(pts)
    sim = make_sim(oracle, pos.astype(np.float32), fvel=vel, bpos=pts, bodies=[body], gravity=(0.0, 0.0, 0.0))
    m = sim.mass()
    P0 = m * vel.sum(0) + body.mass * np.array(body.lin_vel)
    for _ in range(3):
        sim.step_dfsph()
    b = sim.bodies()[0]
    P1 = m * sim.vel().sum(0) + b["mass"] * b["lin_vel"]
    assert abs(b["lin_vel"][2]) > 1e-4          # the body was pushed
    assert np.abs(P1 - P0).max() < 1e-10 * m * len(pos)


def test_rigid_stand_in_closed_forms(oracle):
    """R18: free fall V_n = n g dt, X_n = X_0 + g dt^2 n(n+1)/2; torque-free spin keeps |L|
    to O(dt); samples follow x_k = X + R(q) xbar_k, v_k = V + omega x (x_k - X)."""
    pts, body = scenes.make_rigid_box((0.5, 0.5, 0.5), (0.3, 0.1, 0.1), 1000.0, S)
    body.first_particle = 0; body.n_particles = len(pts)
    body.ang_vel = (0.3, 2.0, 0.1)
    fl = np.array([[5.0, 5.0, 5.0]])
    sim = make_sim(oracle, fl, bpos=pts, bodies=[body], gravity=(0.0, 0.0, -9.81),
                   tank_min=(-10.0, -10.0, -10.0), tank_max=(10.0, 10.0, 10.0),
                   domain_min=(-1.0, -1.0, -1.0), domain_max=(6.0, 6.0, 6.0))
    dt = 4e-4
    I = np.array(body.inertia_body)

    def L_world(b):
        w, x, y, z = b["quat"]
        Rm = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                       [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                       [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
        return Rm @ (I * (Rm.T @ b["ang_vel"])), Rm
    L0, _ = L_world(sim.bodies()[0])
    n = 200
    for _ in range(n):
        sim.rigid_step()
    b = sim.bodies()[0]
    assert np.allclose(b["lin_vel"], [0, 0, -9.81 * n * dt], rtol=1e-12)
    assert np.allclose(b["com"], [0.5, 0.5, 0.5 - 9.81 * dt * dt * n * (n + 1) / 2], rtol=1e-12)
    L1, Rm = L_world(b)
    assert abs(np.linalg.norm(L1) / np.linalg.norm(L0) - 1) < 5e-3
    assert abs(np.linalg.norm(b["quat"]) - 1) < 1e-14
    rest = (pts - np.array([0.5, 0.5, 0.5]))
    assert np.allclose(sim.boundary_pos(), b["com"] + rest @ Rm.T, atol=1e-6)   # fp32 input rounding
    assert np.allclose(sim.boundary_vel(), b["lin_vel"] + np.cross(b["ang_vel"], sim.boundary_pos() - b["com"]), atol=1e-12)


def test_rigid_wall_contact_stand_in(oracle):
    """R18: contact sphere clamped to the tank AABB, outward normal velocity zeroed."""
    pts, body = scenes.make_rigid_sphere((0.5, 0.5, 0.101), 0.1, 1000.0, S)
    body.first_particle = 0; body.n_particles = len(pts)
    body.lin_vel = (0.2, 0.0, -1.0)
    sim = make_sim(oracle, np.array([[0.9, 0.9, 0.9]]), bpos=pts, bodies=[body], gravity=(0.0, 0.0, -9.81),
                   tank_min=(0.0, 0.0, 0.0), tank_max=(1.0, 1.0, 1.0),
                   domain_min=(-0.1, -0.1, -0.1), domain_max=(1.1, 1.1, 1.1))
    for _ in range(10):
        sim.rigid_step()
    b = sim.bodies()[0]
    assert b["com"][2] == pytest.approx(0.1, abs=1e-15) and b["lin_vel"][2] == 0.0
    assert b["lin_vel"][0] == pytest.approx(0.2)


# ---------------------------------------------------------------- viscosity (Eq. 15-19)

def _lattice(n, spacing):
    g = (np.arange(n) + 0.5) * spacing
    z, y, x = np.meshgrid(g, g, g, indexing="ij")
    return np.stack([x.ravel(), y.ravel(), z.ravel()], 1)


@pytest.mark.parametrize("ratio,expect", [(2, 1.396226), (4, 1.91156)])
def test_explicit_laplacian_of_quadratic_field(oracle, ratio, expect):
    """Eq. 15 on an interior simple-cubic lattice (rho = rho0, m/rho = s^3) with v = (y^2, 0, 0):
    exact Laplacian (2, 0, 0).  h = 2s (the paper's h = 4r) gives 1.396226 (coarse support:
    30 % low, this is what the formula yields); h = 4s gives 1.91156, i.e. the reading
    converges towards 2.  y, z components vanish; a linear field gives 0.
    Catches a wrong 2(d+2), a missing 0.01 h^2, x_ij/v_ij sign slips, m/rho_j misplacement."""
    sp = H / ratio
    n = 2 * ratio + 3
    pos = _lattice(n, sp)
    sim = make_sim(oracle, np.zeros((len(pos), 3), np.float32), particle_mass=RHO0 * sp ** 3,
                   kinematic_viscosity=1.0, viscosity_mode=1,
                   domain_min=(-H, -H, -H), domain_max=tuple([n * sp + H] * 3))
    sim.set_state(pos, np.zeros_like(pos))
    sim.build_grid(); sim.compute_density_alpha()
    c = (n // 2) * (n * n + n + 1)
    rho = np.full(len(pos), RHO0)
    v = np.zeros_like(pos); v[:, 0] = pos[:, 1] ** 2
    acc = sim.explicit_viscosity_accel(v, rho)
    assert acc[c, 0] == pytest.approx(expect, abs=2e-5)
    assert abs(acc[c, 1]) < 1e-9 and abs(acc[c, 2]) < 1e-9
    v = np.zeros_like(pos); v[:, 0] = 3.0 * pos[:, 1] + 0.5
    acc = sim.explicit_viscosity_accel(v, rho)
    assert np.abs(acc[c]).max() < 1e-9


def test_implicit_viscosity_operator_properties(oracle):
    """Eq. 19 (R4, R21): A symmetric (u'Aw = w'Au), negative semidefinite, annihilates rigid
    translations and rotations; the implicit solve conserves linear momentum
    (sum_i (v* - v~)_i = 0)."""
    sim, pos, vel = _compressed_block(oracle, n=5, squeeze=1.0, kinematic_viscosity=10.0, viscosity_mode=2, dt=1e-3)
    sim.build_grid(); sim.compute_density_alpha()
    rng = np.random.default_rng(5)
    u = rng.normal(size=pos.shape); w = rng.normal(size=pos.shape)
    Au, Aw = sim.viscosity_operator(u), sim.viscosity_operator(w)
    sc = abs(np.sum(u * Au))
    assert abs(np.sum(u * Aw) - np.sum(w * Au)) < 1e-12 * sc
    assert np.sum(u * Au) < 0 and np.sum(w * Aw) < 0
    assert np.abs(sim.viscosity_operator(np.ones_like(pos) * [1.0, -2.0, 0.5])).max() < 1e-9 * np.abs(Au).max()
    rot = np.cross([0.3, -1.0, 2.0], pos)
    assert np.abs(sim.viscosity_operator(rot)).max() < 1e-9 * np.abs(Au).max()
    vs, it = sim.implicit_viscosity_solve(vel)
    assert it > 3
    assert np.abs((vs - vel).sum(0)).max() < 1e-9 * np.abs(vel).sum()


def test_cg_matches_dense_solve(oracle):
    """Plain CG (R23) on N = 125 against numpy.linalg.solve of the densely assembled
    (I - dt A); residual history decreasing to <= tol."""
    sim, pos, vel = _compressed_block(oracle, n=5, squeeze=1.0, kinematic_viscosity=10.0, viscosity_mode=2,
                                      dt=1e-3, cg_rel_tol=1e-10, cg_max_iter=400)
    sim.build_grid(); sim.compute_density_alpha()
    n3 = pos.size
    A = np.zeros((n3, n3))
    for k in range(n3):
        e = np.zeros(n3); e[k] = 1.0
        A[:, k] = sim.viscosity_operator(e.reshape(-1, 3)).ravel()
    assert np.allclose(A, A.T, atol=1e-9 * np.abs(A).max())
    M = np.eye(n3) - 1e-3 * A
    ref = np.linalg.solve(M, vel.ravel()).reshape(-1, 3)
    vs, it = sim.implicit_viscosity_solve(vel)
    assert np.abs(vs - ref).max() < 1e-8 * np.abs(ref).max()
    hist = sim.cg_history()
    assert len(hist) == it + 1 and hist[-1] <= 1e-10 and hist[0] > hist[-1]
    assert np.linalg.cond(M) > 50          # the system is genuinely ill-conditioned at nu = 10
    # forced iteration count is honoured
    _, it2 = sim.implicit_viscosity_solve(vel, forced=5)
    assert it2 == 5 and len(sim.cg_history()) == 6


# ---------------------------------------------------------------- WCSPH (Eq. 7, 13)

def test_wcsph_eos_and_momentum(oracle):
    """EOS p = k((rho~/rho0)^gamma - 1) with rho~ = max(rho, rho0) (R17): a two-particle pair
    with rho > rho0 is accelerated apart by dt * m * 2 p/rho^2 |gradW| (Eq. 7); momentum is
    conserved (g = 0); a light pair (rho < rho0) feels no pressure."""
    dt = 1e-4
    m = 4.0 * RHO0 * S ** 3
    x = np.array([[0.1, 0.1, 0.1], [0.1 + 0.5 * H, 0.1, 0.1]])
    sim = make_sim(oracle, x, particle_mass=m, dt=dt, gravity=(0.0, 0.0, 0.0))
    sim.step_wcsph()
    rho = m * 1.25 * SIGMA
    p = 50000.0 * ((rho / RHO0) ** 7 - 1)
    dv = dt * m * 2 * p / rho ** 2 * 1.5 * SIGMA / H
    assert np.allclose(sim.vel(), [[-dv, 0, 0], [dv, 0, 0]], rtol=1e-5)
    assert np.allclose(sim.pos() - x.astype(np.float32), dt * sim.vel(), atol=1e-12)
    sim = make_sim(oracle, x, dt=dt, gravity=(0.0, 0.0, -9.81))
    sim.step_wcsph()
    assert np.allclose(sim.vel(), [0, 0, -9.81 * dt], rtol=1e-12)


def test_wcsph_vs_dfsph_centre_of_mass(oracle):
    """Cross-check of the two pressure solvers (BASELINE.json config 1): fluid centre of mass
    at equal physical time agrees to 0.25 * (2r) on a small dam break."""
    sc = scenes.dam_break((8, 8, 12), (14, 10, 14))
    a = oracle.Sim.from_scene(sc)
    b = oracle.Sim.from_scene(sc, dt=1e-4)
    for _ in range(60):
        a.step_dfsph()
    for _ in range(240):
        b.step_wcsph()
    ca, cb = a.pos().mean(0), b.pos().mean(0)
    c0 = sc.fluid_pos.astype(np.float64).mean(0)
    assert np.linalg.norm(ca - c0) > 0.25 * S * 0.2     # the fluid moved
    assert np.linalg.norm(ca - cb) <= 0.25 * S


# ---------------------------------------------------------------- tests/golden fixtures

def _golden():
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, val, _ = [t.strip() for t in line.split("|", 2)]
            out[name] = float(val)
    return out


def test_golden_closed_forms_are_what_the_formulas_give():
    """Every stored constant of tests/golden/closed_forms.txt is re-derived here in numpy from its
    definition (no oracle involved), so a typo in the fixture cannot silently weaken a pin."""
    g = _golden()
    assert g["kernel_sigma_h3"] == pytest.approx(8.0 / np.pi, rel=1e-15)
    assert g["psi_single_sample_over_rho0_h3"] == pytest.approx(np.pi / 8.0, rel=1e-15)
    assert g["gradw_at_half_h_times_h4"] == pytest.approx(12.0 / np.pi, rel=1e-15)
    a = 1 - 1 / np.sqrt(2); b = 1 - np.sqrt(3) / 2
    assert g["akinci_volume_one_layer"] == pytest.approx(np.pi / (2 + 8 * a ** 3), abs=1e-6)
    assert g["akinci_volume_two_layers"] == pytest.approx(np.pi / (2.25 + 16 * a ** 3 + 8 * b ** 3), abs=1e-6)

    def w_and_wp(q):
        if q <= 0.5:
            return 6 * (q ** 3 - q ** 2) + 1, 6 * q * (3 * q - 2)
        if q <= 1:
            return 2 * (1 - q) ** 3, -6 * (1 - q) ** 2
        return 0.0, 0.0

    # lattice sums with h = 2 s, in units s = 1, sigma = 8 / (pi h^3)
    h = 2.0
    sigma = 8.0 / (np.pi * h ** 3)
    rho = 0.0
    T = 0.0
    for i in range(-2, 3):
        for j in range(-2, 3):
            for k in range(-2, 3):
                d = np.sqrt(i * i + j * j + k * k)
                w, wp = w_and_wp(d / h)
                rho += sigma * w
                if d > 0:
                    T += (sigma / h * wp) ** 2
    assert g["lattice_density_over_rho0"] == pytest.approx(rho, abs=2e-8)
    assert g["lattice_alpha_times_rho0_over_s2"] == pytest.approx(rho / T, rel=2e-6)

    # Eq. 15 on v = (y^2, 0, 0), rho = rho0, m / rho = s^3 = 1
    for key, ratio in (("laplacian_h_2s", 2), ("laplacian_h_4s", 4)):
        h = float(ratio)
        sigma = 8.0 / (np.pi * h ** 3)
        n = ratio
        lap = 0.0
        for i in range(-n, n + 1):
            for j in range(-n, n + 1):
                for k in range(-n, n + 1):
                    d2 = float(i * i + j * j + k * k)
                    d = np.sqrt(d2)
                    if d == 0 or d >= h:
                        continue
                    _, wp = w_and_wp(d / h)
                    # particle i at the origin, neighbour at (i, j, k): x_ij = -(i, j, k), v_ij = (0 - j^2, 0, 0)
                    vij_dot_xij = (-(j * j)) * (-i)
                    gradx = sigma / h * wp * (-i) / d
                    lap += 10.0 * vij_dot_xij / (d2 + 0.01 * h * h) * gradx
        assert g[key] == pytest.approx(lap, abs=2e-6), (key, lap)


def test_oracle_matches_golden_lattice_constants(oracle):
    g = _golden()
    n = 9
    gr = (np.arange(n) + 0.5) * S
    z, y, x = np.meshgrid(gr, gr, gr, indexing="ij")
    pos = np.stack([x.ravel(), y.ravel(), z.ravel()], 1)
    sim = make_sim(oracle, np.zeros((n ** 3, 3), dtype=np.float32))
    sim.set_state(pos, np.zeros_like(pos))
    sim.build_grid(); sim.compute_density_alpha()
    c = (n // 2) * (n * n + n + 1)
    assert sim.density()[c] / RHO0 == pytest.approx(g["lattice_density_over_rho0"], abs=2e-8)
    assert sim.alpha()[c] * RHO0 / S ** 2 == pytest.approx(g["lattice_alpha_times_rho0_over_s2"], rel=2e-6)


# ---------------------------------------------------------------- CFL-adaptive time step (R26, NEXT-1)

def test_cfl_time_step_rule_and_free_fall_recurrence(oracle):
    """dt_n = clamp(lambda 2r / max|v|, dt_min, dt_max) with the velocities at the start of step n.
    A block in free fall far from everything feels no pressure (rho* <= rho0), so v and x follow
    the symplectic-Euler recurrence with the VARIABLE dt -- re-evaluated here in plain Python.
    Catches: v_max taken after instead of before the step, clamp order, dt not used consistently
    by gravity and integration."""
    lam, dt_max, dt_min = 0.4, 4e-4, 1e-5
    g = 9.81
    n = 4
    gr = (np.arange(n) + 0.5) * S
    z, y, x = np.meshgrid(gr, gr, gr, indexing="ij")
    pos = np.stack([x.ravel(), y.ravel(), z.ravel() + 5.0], 1)
    v0 = np.tile(np.array([[3.0, 0.0, -19.5]]), (len(pos), 1))    # |v| crosses lambda 2r / dt_max = 20 m/s on the way
    sim = make_sim(oracle, pos.astype(np.float32), v0.astype(np.float32), cfl_factor=lam, dt_min=dt_min,
                   domain_min=(-1.0, -1.0, 0.0), domain_max=(2.0, 1.0, 6.0))
    p0 = sim.pos().copy()
    v = np.array([3.0, 0.0, -19.5])
    xx = np.zeros(3)
    t = 0.0
    dts = []
    for k in range(200):
        dt = min(dt_max, max(dt_min, lam * 2 * R / np.linalg.norm(v)))
        dts.append(dt)
        sim.step_dfsph()
        st = sim.stats()
        assert st["dt_last"] == pytest.approx(dt, rel=1e-12), k
        v = v + dt * np.array([0.0, 0.0, -g])
        xx = xx + dt * v
        t += dt
        assert st["sim_time"] == pytest.approx(t, rel=1e-12)
    assert dts[0] == dt_max and dts[-1] < dt_max         # the rule switched on during the fall
    assert np.allclose(sim.vel(), v[None, :], rtol=1e-12, atol=1e-12)
    assert np.allclose(sim.pos() - p0, xx[None, :], rtol=1e-10, atol=1e-12)
    # clamps: slow fluid -> dt_max; forced dt overrides; lambda = 0 -> fixed dt
    sim.set_state(p0, np.full_like(p0, 1e-3)); sim.step_dfsph()
    assert sim.stats()["dt_last"] == dt_max
    sim.set_state(p0, np.tile(np.array([[1e4, 0.0, 0.0]]), (len(p0), 1))); sim.step_dfsph()
    assert sim.stats()["dt_last"] == dt_min
    sim.set_forced_dt(1.25e-4); sim.step_dfsph()
    assert sim.stats()["dt_last"] == 1.25e-4
    sim.set_forced_dt(0.0)
    fixed = make_sim(oracle, pos.astype(np.float32), (10 * v0).astype(np.float32),
                     domain_min=(-1.0, -1.0, 0.0), domain_max=(2.0, 1.0, 6.0))
    fixed.step_dfsph()
    assert fixed.stats()["dt_last"] == 4e-4


# ---------------------------------------------------------------- round-2 pins: operator scale, boundary terms, torque

@pytest.mark.parametrize("ratio,expect", [(2, 1.396226), (4, 1.91156)])
def test_implicit_viscosity_operator_scale(oracle, ratio, expect):
    """SCALE of Eq. 19 (R4, R21), tied to the pinned Eq. 15: on an interior
    simple-cubic lattice (rho_i = rho_j = rho_c, m = rho0 s^3) with u = (y^2, 0, 0)
        (A u)_c = 2(d+2) mu m / rho_c^2 sum_j (...) = nu L (rho0 / rho_c)^2,
    L = the discrete Laplacian constant of test_explicit_laplacian_of_quadratic_field (1.396226 at
    h = 2s, 1.91156 at h = 4s; tests/golden/closed_forms.txt), rho_c the oracle's own lattice density.
    Catches what the symmetry / null-space / CG-vs-dense pins cannot: a wrong 2(d+2) (8 for 10), mu m /
    (rho_i rho_j) off by a constant (rho0 missing in mu = nu rho0, m^2 for m, rho_i^2 only)."""
    sp = H / ratio
    n = 4 * ratio + 1                 # centre +- 2h: the centre's neighbours are interior particles too
    pos = _lattice(n, sp)
    nu = 3.0
    sim = make_sim(oracle, np.zeros((len(pos), 3), np.float32), particle_mass=RHO0 * sp ** 3,
                   kinematic_viscosity=nu, viscosity_mode=2,
                   domain_min=(-H, -H, -H), domain_max=tuple([n * sp + H] * 3))
    sim.set_state(pos, np.zeros_like(pos))
    sim.build_grid(); sim.compute_density_alpha()
    c = (n // 2) * (n * n + n + 1)
    rho = sim.density()
    st, idx = sim.neighbors(0)
    nb = idx[st[c]:st[c + 1]]
    assert len(nb) > 20 and np.abs(rho[nb] - rho[c]).max() < 1e-9 * rho[c]      # interior: one density
    assert abs(rho[c] / RHO0 - 1) < 0.01 and rho[c] != RHO0
    u = np.zeros_like(pos); u[:, 0] = pos[:, 1] ** 2
    Au = sim.viscosity_operator(u)
    want = nu * expect * (RHO0 / rho[c]) ** 2
    assert Au[c, 0] == pytest.approx(want, rel=2e-5)
    assert abs(Au[c, 1]) < 1e-9 * want and abs(Au[c, 2]) < 1e-9 * want
    # and it is the explicit formula with rho_j = rho_c, up to the extra rho0 / rho_c of mu m/(rho_i rho_j)
    acc = sim.explicit_viscosity_accel(u, np.full(len(pos), rho[c]))
    assert Au[c, 0] == pytest.approx(acc[c, 0] * RHO0 / rho[c], rel=1e-12)


def _one_fluid_one_dynamic_sample(oracle, vi, vk, **prm):
    """fluid particle i at the origin-ish point, ONE boundary sample k = a dynamic single-sample body at
    distance h/2 in +x, moving with v_k (its sample velocity is lin_vel: no rotation arm)."""
    xi = np.array([0.1, 0.1, 0.1]); xk = xi + np.array([0.5 * H, 0.0, 0.0])
    body = scenes.Body(0, 1, dynamic=1, mass=0.5, inertia_body=(1e-3, 1e-3, 1e-3), com=tuple(xk),
                       lin_vel=tuple(vk), contact_radius=0.0)
    far = 50.0
    sim = make_sim(oracle, xi[None, :], fvel=np.asarray(vi, dtype=np.float64)[None, :], bpos=xk[None, :],
                   bodies=[body], gravity=(0.0, 0.0, 0.0), tank_min=(-far,) * 3, tank_max=(far,) * 3, **prm)
    return sim, xi, xk


def test_boundary_terms_of_density_rate_and_pressure_update(oracle):
    """Boundary sums of D_i and U_i with a MOVING sample (Eq. 6 / 10 / 13 / 14, PAPER.md:110, 156, 200, 204;
    R8): one fluid particle at h/2 from a one-sample dynamic body.  By hand: Psi = rho0 / W(0) (Eq. 11),
    gradW_ik = -(1.5 sigma / h) n with n = (x_i - x_k)/|.| = -e_x, so
        D = Psi (v_i - v_k).gradW_ik,   err_v = dt D / rho0,
    and one forced divergence iteration (alpha = rho / |Psi gradW|^2, T = 0) removes exactly the approaching
    normal relative velocity, v_i' = v_i - ((v_i - v_k).n) n, with the Eq. 14 reaction F_k = -m (v_i' - v_i)/dt.
    A separating pair is untouched (R15).  Catches: v_k dropped or with the wrong sign in D, m in place of
    Psi_k, Psi_k^2, a wrong sign or missing m in the reaction."""
    dt = 4e-4
    gold = _golden()
    psi = gold["psi_single_sample_over_rho0_h3"] * RHO0 * H ** 3      # = rho0 / W(0)
    g = gold["gradw_at_half_h_times_h4"] / H ** 4                     # = 1.5 sigma / h
    assert psi == pytest.approx(RHO0 / SIGMA, rel=1e-14) and g == pytest.approx(1.5 * SIGMA / H, rel=1e-14)
    m = RHO0 * S ** 3
    vi = np.array([0.05, 0.2, -0.1]); vk = np.array([-0.35, 0.1, 0.3])
    sim, xi, xk = _one_fluid_one_dynamic_sample(oracle, vi, vk, dt=dt)
    assert sim.psi()[0] == pytest.approx(psi, rel=1e-12)
    assert np.allclose(sim.boundary_vel()[0], vk, atol=1e-7)
    sim.build_grid(); sim.compute_density_alpha()
    v1, it = sim.divergence_solve(vi[None, :], forced=1)
    n = np.array([-1.0, 0.0, 0.0])
    D = psi * np.dot(vi - vk, -g * n)                 # = psi * 0.4 * g > 0: approaching
    assert D > 0
    assert sim.stats()["err_v"] == pytest.approx(dt / RHO0 * D, rel=1e-6)
    want = vi - np.dot(vi - vk, n) * n
    assert np.allclose(v1[0], want, rtol=1e-6, atol=1e-9)
    assert abs(v1[0, 0] - vk[0]) < 1e-6               # normal velocities now equal
    F = sim.boundary_force()[0]
    assert np.allclose(F, -m * (v1[0] - vi) / dt, rtol=1e-6, atol=1e-9 * m / dt)
    assert F[0] > 0                                   # the fluid pushes the sample away from itself (+x)
    # v_k matters: the same fluid velocity against a sample at rest approaches 8x slower
    sim0, _, _ = _one_fluid_one_dynamic_sample(oracle, vi, np.zeros(3), dt=dt)
    sim0.build_grid(); sim0.compute_density_alpha()
    sim0.divergence_solve(vi[None, :], forced=1)
    assert sim0.stats()["err_v"] == pytest.approx(dt / RHO0 * psi * g * vi[0], rel=1e-6)
    # separating pair: D < 0 is clamped (R15), nothing moves, no reaction
    sims, _, _ = _one_fluid_one_dynamic_sample(oracle, vk, vi, dt=dt)
    sims.build_grid(); sims.compute_density_alpha()
    v2, _ = sims.divergence_solve(vk[None, :], forced=1)
    assert np.array_equal(v2[0], vk)
    assert np.all(sims.boundary_force()[0] == 0.0)
    # the density solve sees the same boundary term: rho* = rho + dt D, kappa = alpha (rho* - rho0)/dt^2
    simd, _, _ = _one_fluid_one_dynamic_sample(oracle, vi, vk, dt=dt, particle_mass=3.0 * m)
    simd.build_grid(); simd.compute_density_alpha()
    rho = 3.0 * m * SIGMA + psi * SIGMA / 4
    assert simd.density()[0] == pytest.approx(rho, rel=1e-6) and rho > RHO0
    v3, _ = simd.density_solve(vi[None, :], forced=1)
    E = rho + dt * D - RHO0
    assert simd.stats()["err_rho"] == pytest.approx(E / RHO0, rel=1e-6)
    # v' = v - dt Psi (kappa/rho) gradW = v + (E / (dt Psi g)) n
    assert np.allclose(v3[0], vi + E / (dt * psi * g) * n, rtol=1e-6, atol=1e-9)


def _angular_momentum_about_origin(sim, m):
    """sum x cross m v (fluid) + X cross M V + R I_b R^T omega (body 0), fp64."""
    b = sim.bodies()[0]
    w, x, y, z = b["quat"]
    Rm = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                   [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                   [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
    spin = Rm @ (b["inertia_body"] * (Rm.T @ b["ang_vel"]))
    orbital = np.cross(b["com"], b["mass"] * b["lin_vel"])
    fluid = m * np.cross(sim.pos(), sim.vel()).sum(0)
    return fluid + orbital + spin, spin, b


def test_torque_conserves_total_angular_momentum(oracle):
    """tau = sum_k (x_k - X) x F_k and the angular response of the rigid stand-in (Eq. 14, PAPER.md:204;
    R18): g = 0, a box with a small fluid block pressed against an OFF-CENTRE part of its top face.  Pair
    forces are central (along x_i - x_k), so the total angular momentum about a fixed point,
        sum_i x_i x m v_i + X x M V + I_w omega,
    is conserved by every C-pass exactly and by the explicit body integration to O(dt^2 omega^2); it must
    stay constant to a small fraction of the spin the body picks up.  A flipped cross product (F x r), a
    torque about the origin instead of X, a missing I^-1 or a transposed R fail it (error ~ 2x the spin);
    the linear-momentum pin cannot see any of them."""
    dt = 4e-4
    sc = scenes.free_block((3, 3, 2), jitter=0.0, vel_scale=0.0, seed=0)
    pos = sc.fluid_pos.astype(np.float64)
    pos += np.array([0.5, 0.5, 0.5]) - pos.min(0)
    vel = np.zeros_like(pos); vel[:, 2] = -1.0
    size = (0.16, 0.1, 0.06)
    # box top face 0.9 s below the lowest fluid layer; fluid over the +x end of the face, off-centre in y too
    ctr = (pos[:, 0].mean() - 0.05, pos[:, 1].mean() - 0.02, pos[:, 2].min() - 0.9 * S - 0.5 * size[2])
    pts, body = scenes.make_rigid_box(ctr, size, 600.0, S)
    body.first_particle = 0; body.n_particles = len(pts)
    far = 50.0
    sim = make_sim(oracle, pos.astype(np.float32), fvel=vel, bpos=pts, bodies=[body], gravity=(0.0, 0.0, 0.0),
                   dt=dt, tank_min=(-far,) * 3, tank_max=(far,) * 3)
    m = sim.mass()
    L0, spin0, _ = _angular_momentum_about_origin(sim, m)
    assert np.all(spin0 == 0)
    Ls = []
    for _ in range(3):
        sim.step_dfsph()
        Ls.append(_angular_momentum_about_origin(sim, m))
    L3, spin3, b = Ls[-1]
    I = np.asarray(b["inertia_body"])
    assert np.linalg.norm(b["ang_vel"]) > 1e-3                   # the body was set spinning ...
    assert abs(b["ang_vel"][1]) > 10 * abs(b["ang_vel"][2])      # ... mainly about y (fluid over the +x end)
    assert b["ang_vel"][1] > 0                                   # -z force at +x arm: tau_y = r_z F_x - r_x F_z > 0
    assert b["lin_vel"][2] < -1e-4                               # and pushed down
    # integrator error of the explicit body update: I_w is taken at the old orientation, so each step leaves
    # dt |omega x I_w omega| + O(dt^2) unaccounted; everything else is exact
    bound = 3 * 2.0 * dt * np.linalg.norm(np.cross(b["ang_vel"], spin3)) + 1e-9 * np.linalg.norm(spin3)
    assert bound < 2e-2 * np.linalg.norm(spin3)      # a flipped or mis-centred torque is off by ~2 |spin|
    for L, _, _ in Ls:
        assert np.abs(L - L0).max() < bound, (L - L0, spin3, bound)
    # magnitude of the response: omega = I_w^-1 L_spin with the body still (almost) axis-aligned
    assert np.allclose(b["ang_vel"][:2], (spin3 / I)[:2], rtol=2e-2)
