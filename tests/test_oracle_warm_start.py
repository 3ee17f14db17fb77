"""Pins of the oracle's warm start (reading R27; the technique is the
one of the cited DFSPH source [5]).  CPU only.  Each test names the mistake it would catch."""
import numpy as np
import pytest

from paper_2403_11156_b200 import scenes
from test_oracle_pins import make_sim, _compressed_block, H, S, RHO0, SIGMA


def test_warm_start_two_particle_closed_form(oracle):
    """Two particles at distance h/2, light enough that rho < rho0 (the iteration after the warm start adds kappa = 0
    because the warm start only pushes them apart).  With stored totals K_0, K_1 the warm start alone gives
        v_0 = -dt m omega (K_0 + K_1) / rho * gradW_01,   gradW_01 = +1.5 sigma / h  x^   (|w'(1/2)| = 1.5),
    v_1 = -v_0, and the new totals are omega K.  Catches a missing omega, K used without 1/rho, K_i only
    (no symmetrisation), the wrong sign, dt squared."""
    dt, om = 4e-4, 0.5
    x = np.array([[0.1, 0.1, 0.1], [0.1 + 0.5 * H, 0.1, 0.1]])
    m = RHO0 * S ** 3
    rho = m * 1.25 * SIGMA
    assert rho < RHO0
    g = 1.5 * SIGMA / H
    K = np.array([3.0e5, 1.0e5])
    for solve, setk in (("density_solve", lambda s: s.set_warm_state(np.zeros(2), K)),
                        ("divergence_solve", lambda s: s.set_warm_state(K, np.zeros(2)))):
        sim = make_sim(oracle, x, dt=dt, warm_start=1, warm_start_factor=om)
        sim.build_grid(); sim.compute_density_alpha()
        assert sim.density()[0] == pytest.approx(rho, rel=1e-6)     # positions are fp32 inputs
        setk(sim)
        v, it = getattr(sim, solve)(np.zeros((2, 3)), forced=1)
        dv = dt * m * om * (K[0] + K[1]) / rho * g
        assert it == 1
        assert np.allclose(v, [[-dv, 0, 0], [dv, 0, 0]], rtol=1e-5, atol=1e-15)
        tot = sim.ksum_d() if solve == "density_solve" else sim.ksum_v()
        assert np.allclose(tot, om * K, rtol=1e-14)
        st = sim.stats()
        assert (st["err_rho"] if solve == "density_solve" else st["err_v"]) == 0.0


def test_warm_start_off_and_zero_factor_equal_the_cold_solve(oracle):
    """warm_start = 0 ignores stored totals; warm_start = 1 with omega = 0 applies a zero update: both are
    bit-identical to the cold solve.  Catches a warm start that leaks into the default path."""
    outs = []
    for ws, om in ((0, 0.5), (1, 0.0), (0, 0.0)):
        sim, pos, vel = _compressed_block(oracle, warm_start=ws, warm_start_factor=om)
        sim.build_grid(); sim.compute_density_alpha()
        sim.set_warm_state(np.full(sim.nf, 1e5), np.full(sim.nf, 2e5))
        v1, _ = sim.divergence_solve(vel, forced=2)
        v2, _ = sim.density_solve(v1, forced=2)
        outs.append(v2)
    assert np.array_equal(outs[0], outs[2]) and np.array_equal(outs[1], outs[2])


def test_totals_are_the_sum_of_the_iterations_stiffness(oracle):
    """K_i(new) = omega K_i(old) + sum_l kappa_i^(l): three forced iterations in one call leave the same total as
    the kappa of three one-iteration calls summed (cold start), and a warm-started call adds omega K(old)."""
    sim, pos, vel = _compressed_block(oracle, squeeze=0.9)
    sim.build_grid(); sim.compute_density_alpha()
    v3, _ = sim.density_solve(np.zeros_like(vel), forced=3)
    total3 = sim.ksum_d()
    acc = np.zeros(sim.nf); v = np.zeros_like(vel)
    for _ in range(3):
        v, _ = sim.density_solve(v, forced=1)
        acc += sim.kappa()
    assert np.allclose(v, v3, rtol=1e-13, atol=1e-15)
    assert np.allclose(acc, total3, rtol=1e-12) and total3.max() > 0.0
    # same check for the divergence solve
    vd, _ = sim.divergence_solve(vel, forced=2)
    tv = sim.ksum_v()
    acc = np.zeros(sim.nf); v = vel.copy()
    for _ in range(2):
        v, _ = sim.divergence_solve(v, forced=1)
        acc += sim.kappa()
    assert np.allclose(acc, tv, rtol=1e-12) and tv.max() > 0.0


def test_warm_start_conserves_momentum(oracle):
    """The warm start is an ordinary symmetric pressure update: fluid only, g = 0 => sum m v and sum x cross m v
    unchanged.  Catches an asymmetric warm start (K_i only)."""
    sim, pos, vel = _compressed_block(oracle, warm_start=1, warm_start_factor=0.5)
    sim.build_grid(); sim.compute_density_alpha()
    rng = np.random.default_rng(3)
    sim.set_warm_state(rng.uniform(0, 2e5, sim.nf), rng.uniform(0, 2e5, sim.nf))
    P0 = vel.sum(0); L0 = np.cross(pos, vel).sum(0)
    v1, _ = sim.divergence_solve(vel, forced=1)
    v2, _ = sim.density_solve(v1, forced=1)
    scale = np.abs(vel).sum()
    assert np.abs(v2 - vel).max() > 1e-3
    assert np.abs(v2.sum(0) - P0).max() < 1e-12 * scale
    assert np.abs(np.cross(pos, v2).sum(0) - L0).max() < 1e-12 * scale


def test_warm_start_needs_fewer_iterations_on_a_resting_column(oracle):
    """What the technique is for (fewer refinement rounds): a hydrostatic column under a tight
    tolerance.  Cold: every step re-derives the whole hydrostatic stiffness; warm: it starts from half of it.
    Both converge to err_rho <= eta on every step; the warm-started run needs clearly fewer iterations."""
    tot = {}
    for ws in (0, 1):
        sc = scenes.dam_break((8, 8, 30), (8, 8, 34), dt=1e-3, eta_density=1e-4, min_iter_density=1,
                              warm_start=ws, warm_start_factor=0.5)
        o = oracle.Sim.from_scene(sc)
        n = 0
        for _ in range(60):           # the column needs ~30 steps to settle into hydrostatic compression
            o.step_dfsph()
            st = o.stats()
            assert st["err_rho"] <= 1e-4 and st["it_d"] < 100
            n += st["it_d"]
        tot[ws] = n
        o.close()
    assert tot[1] <= 0.75 * tot[0], tot
