"""Pins of the fp64 oracle on the paper's own velocity set, D3Q19 (Fig. 2 :107) -- CPU only.

The D3Q19 oracle is the second translation unit oracle/hhrr_oracle_q19.c (19 directions, weights 1/3, 1/18,
1/36, third-order basis of the paper's ref. [43], reading R23).  What is specific to the set is
pinned here against the mathematics; every lattice-generic pin of test_oracle_pins.py and
test_oracle_pins_coupling.py is run again on it (their module constant Q is switched to 19 for the call).
"""
import numpy as np
import pytest

import test_oracle_pins as P
import test_oracle_pins_coupling as PC


@pytest.fixture
def o19(oracle, monkeypatch):
    monkeypatch.setattr(P, "Q", 19)
    monkeypatch.setattr(PC, "Q", 19)
    return oracle.view(19)


def _c(O):
    cx, cy, cz, w = O.lattice_tables()
    return np.stack([cx, cy, cz]).astype(np.float64), w


def _H3(c, a, b, g):
    d = lambda p, q: 1.0 if p == q else 0.0
    return c[a] * c[b] * c[g] - (c[a] * d(b, g) + c[b] * d(a, g) + c[g] * d(a, b)) / 3


GROUPS = [((0, 0, 1), (1, 2, 2)), ((0, 2, 2), (0, 1, 1)), ((1, 1, 2), (0, 0, 2))]   # (xxy, yzz), (xzz, xyy), (yyz, xxz)


def test_q19_velocity_set(o19):
    """D3Q19 (Fig. 2): rest + 6 axis + 12 face-diagonal directions, no cube corners; weights 1/3, 1/18,
    1/36; sum w = 1, second moment c_s^2 delta with c_s^2 = 1/3, isotropic fourth moment, opposite = 18 - i."""
    c, w = _c(o19)
    assert c.shape == (3, 19)
    n2 = np.sum(c * c, axis=0)
    assert sorted(n2) == [0] + [1] * 6 + [2] * 12
    assert np.allclose(w[n2 == 0], 1 / 3) and np.allclose(w[n2 == 1], 1 / 18) and np.allclose(w[n2 == 2], 1 / 36)
    assert len({tuple(c[:, i]) for i in range(19)}) == 19
    P.test_lattice_isotropy(o19)


def test_q19_third_order_basis_is_orthogonal(o19):
    """Reading R23 (paper's ref. [43], named at PAPER.md:94): on D3Q19 the supported third-order polynomials are the
    sums H_xxy + H_yzz, H_xzz + H_xyy, H_yyz + H_xxz and the matching differences.  They are mutually orthogonal
    under the weights, orthogonal to orders 0-2, with squared norms 2 c_s^6 (the "2 c_s^6" of Eq. 11)
    and 6 c_s^6; H_xyz vanishes on every direction of the set."""
    c, w = _c(o19)
    basis = []
    for g1, g2 in GROUPS:
        basis += [_H3(c, *g1) + _H3(c, *g2), _H3(c, *g1) - _H3(c, *g2)]
    G = np.array([[np.sum(w * p * q) for q in basis] for p in basis])
    assert np.allclose(G, np.diag([2 / 27, 6 / 27] * 3), atol=1e-16)
    low = [np.ones(19), c[0], c[1], c[2]] + [c[a] * c[b] - (a == b) / 3 for a in range(3) for b in range(a, 3)]
    for p in basis:
        for q in low:
            assert abs(np.sum(w * p * q)) < 1e-16
    assert np.all(_H3(c, 0, 1, 2) == 0)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_q19_equilibrium_moments(o19, seed):
    """Eq. 11 on D3Q19: moments 0, 1, 2 exact; the six supported third-order moments equal those of
    rho u u u; and the velocity set cannot tell f_eq from its second-order truncation in the H_xyz direction."""
    rng = np.random.default_rng(seed)
    c, w = _c(o19)
    rho = 1 + 0.1 * rng.standard_normal()
    u = 0.1 * rng.standard_normal(3)
    f = o19.equilibrium(rho, u)
    assert abs(f.sum() - rho) < 1e-15
    assert np.allclose(c @ f, rho * u, atol=1e-16)
    Pm = np.einsum("i,ai,bi->ab", f, c, c)
    assert np.allclose(Pm, rho * np.outer(u, u) + rho / 3 * np.eye(3), atol=1e-16)
    a3 = rho * np.einsum("a,b,g->abg", u, u, u)
    for g1, g2 in GROUPS:
        for sgn in (1, -1):
            m = np.sum(f * (_H3(c, *g1) + sgn * _H3(c, *g2)))
            assert abs(m - (a3[g1] + sgn * a3[g2])) < 1e-16
    # and it differs from the plain second-order equilibrium by exactly that third-order part (not zero)
    f2 = w * (rho + 3 * (c.T @ (rho * u)) + 4.5 * np.einsum("ai,bi,a,b->i", c, c, u, u) * rho - 1.5 * rho * (u @ u))
    assert np.max(np.abs(f - f2)) > 1e-6


@pytest.mark.parametrize("seed", range(3))
def test_q19_collision_invariants(o19, seed):
    """Eq. 6 on D3Q19: mass, momentum rho*uhat, second moment rho uh uh + rho cs^2 I + (1 - 1/tau) a2_hyb; supported
    third-order moments = those of rho uh uh uh + (1 - 1/tau)(uh a2 recursion, R3)."""
    rng = np.random.default_rng(seed)
    c, w = _c(o19)
    f = w * (1 + 0.05 * rng.standard_normal(19))
    g = 1e-3 * rng.standard_normal(3)
    d = rng.random()
    uB = 0.05 * rng.standard_normal(3)
    S = 1e-3 * rng.standard_normal((3, 3)); S = 0.5 * (S + S.T)
    sigma, tau0, cs = 0.7, 0.6, 0.17
    out, diag = o19.collide_cell(f, g, d, uB, S, sigma, tau0, cs)
    rho = f.sum()
    uh = d * (c @ f + g) / rho + (1 - d) * uB
    assert abs(out.sum() - rho) < 1e-14 and np.allclose(c @ out, rho * uh, atol=1e-15)
    pi = np.einsum("i,ai,bi->ab", f, c, c) - rho / 3 * np.eye(3) - rho * np.outer(uh, uh)
    tau = diag[4]
    assert tau == pytest.approx(PC._tau_fixed_point(tau0, cs, rho, pi), rel=1e-13)
    a2 = sigma * pi - (1 - sigma) * 2 * rho / 3 * tau * S
    assert np.allclose(np.einsum("i,ai,bi->ab", out, c, c), rho * np.outer(uh, uh) + rho / 3 * np.eye(3) + (1 - 1 / tau) * a2,
                       atol=1e-15)
    a3 = rho * np.einsum("a,b,g->abg", uh, uh, uh) + (1 - 1 / tau) * (
        np.einsum("a,bg->abg", uh, a2) + np.einsum("b,ag->abg", uh, a2) + np.einsum("g,ab->abg", uh, a2))
    for g1, g2 in GROUPS:
        for sgn in (1, -1):
            m = np.sum(out * (_H3(c, *g1) + sgn * _H3(c, *g2)))
            assert abs(m - (a3[g1] + sgn * a3[g2])) < 1e-15


# ---- the lattice-generic pins, again on D3Q19 ---------------------------------------------------------------
def test_q19_hlbm_limits(o19):
    P.test_hlbm_porosity_one_ignores_solid_velocity(o19)
    P.test_hlbm_porosity_zero_imposes_solid_velocity(o19)


def test_q19_one_step_matches_numpy_assembly(o19):
    P.test_one_step_matches_numpy_assembly(o19)


def test_q19_mirror_axis_equals_even_extension(o19):
    P.test_mirror_axis_equals_even_extension(o19)


def test_q19_hybrid_fd_term_closed_form(o19):
    P.test_hybrid_fd_term_closed_form(o19)


@pytest.mark.parametrize("tau0,sigma,cs", [(0.55, 1.0, 0.0), (0.8, 0.0, 0.0), (0.55, 0.995, 0.1)])
def test_q19_taylor_green_decay_gives_viscosity(o19, tau0, sigma, cs):
    P.test_taylor_green_decay_gives_viscosity(o19, tau0, sigma, cs)


def test_q19_config1_tgv3d_decay(o19):
    P.test_config1_tgv3d_decay(o19)


def test_q19_force_and_torque_structure(o19):
    P.test_force_vanishes_for_comoving_solid(o19)
    P.test_torque_of_hydrostatic_load_closed_form(o19)
    PC.test_force_solid_velocity_term_is_minus_us_times_mass_inflow(o19)
    PC.test_rotor_coefficients_definition_3(o19)


def test_q19_half_channel_wall_drag_equals_body_force(o19):
    PC.test_half_channel_wall_drag_equals_body_force(o19)


def test_q19_wall_model_coupling_and_fringe(o19):
    P.test_wall_model_on_uniform_and_shear_flow(o19)
    PC.test_wall_model_state_is_consumed_by_the_collision(o19)
    PC.test_fringe_imposes_the_inflow_velocity(o19)
    PC.test_wall_model_across_a_mirror_plane_equals_even_extension(o19)
    PC.test_force_on_a_mirror_lattice_equals_even_extension(o19)


def test_q19_rigid_rotation_and_geometry(o19):
    P.test_rigid_rotation_has_zero_fd_strain(o19)
    PC.test_growth_layer_is_the_26_neighbourhood(o19, (0, 3, 6), (1, 1, 1))
