"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each test names the oracle part it pins and the PAPER.md passage / DESIGN.md reading.
None of them compares the oracle with itself or with the CUDA path.
"""
import itertools

import numpy as np
import pytest

Q = 27   # tests/test_oracle_pins_q19.py runs the lattice-generic tests of this module again with Q = 19


def _c(O):
    cx, cy, cz, w = O.lattice_tables()
    return np.stack([cx, cy, cz]).astype(np.float64), w


def _flip_y(c):
    """index of the direction with the y component reversed, for every direction of the set"""
    dirs = [tuple(int(v) for v in c[:, i]) for i in range(c.shape[1])]
    return np.array([dirs.index((d[0], -d[1], d[2])) for d in dirs])


# ------------------------------------------------------------------ P1 lattice tables
def test_lattice_isotropy(oracle):
    """D3Q27 weights/velocities: sum w = 1, second moment cs^2 delta, fourth moment isotropic,
    opposite = 26 - i (conventions)."""
    c, w = _c(oracle)
    assert abs(w.sum() - 1) < 1e-15
    assert np.allclose(c @ w, 0, atol=1e-16)
    m2 = np.einsum("i,ai,bi->ab", w, c, c)
    assert np.allclose(m2, np.eye(3) / 3, atol=1e-15)
    m4 = np.einsum("i,ai,bi,ci,di->abcd", w, c, c, c, c)
    I = np.eye(3)
    iso = (np.einsum("ab,cd->abcd", I, I) + np.einsum("ac,bd->abcd", I, I) + np.einsum("ad,bc->abcd", I, I)) / 9
    assert np.allclose(m4, iso, atol=1e-15)
    for i in range(Q):
        assert np.all(c[:, i] == -c[:, Q - 1 - i])
    assert np.all(c[:, (Q - 1) // 2] == 0)


# ------------------------------------------------------------------ P2 equilibrium moments
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_equilibrium_moments(oracle, seed):
    """Eq. 11 with reading R3: moments 0..2 exact, the 7 third moments that D3Q27
    supports equal rho u_a u_b u_g."""
    rng = np.random.default_rng(seed)
    c, w = _c(oracle)
    rho = 1 + 0.1 * rng.standard_normal()
    u = 0.1 * rng.standard_normal(3)
    f = oracle.equilibrium(rho, u)
    assert abs(f.sum() - rho) < 1e-15
    assert np.allclose(c @ f, rho * u, atol=1e-16)
    P = np.einsum("i,ai,bi->ab", f, c, c)
    assert np.allclose(P, rho * np.outer(u, u) + rho / 3 * np.eye(3), atol=1e-16)
    for a, b, g in [(0, 0, 1), (0, 0, 2), (0, 1, 1), (1, 1, 2), (0, 2, 2), (1, 2, 2), (0, 1, 2)]:
        m3 = np.sum(f * c[a] * c[b] * c[g])
        # central (Hermite) third moment: subtract the cs^2 (rho u) delta parts
        expect = rho * u[a] * u[b] * u[g] + rho / 3 * (u[a] * (b == g) + u[b] * (a == g) + u[g] * (a == b))
        assert abs(m3 - expect) < 1e-16


def _rand_cell(rng):
    c_w = rng.random(Q) * 0.02
    return c_w


# ------------------------------------------------------------------ P3 collision invariants
@pytest.mark.parametrize("seed", range(4))
def test_collision_invariants(oracle, seed):
    """Eq. 6: mass conserved; post-collision momentum = rho*uhat (R4); second moment =
    rho uhat uhat + rho cs^2 I + (1 - 1/tau_eff) a2_hyb with a2_hyb of Eq. 7+10 (R2)."""
    rng = np.random.default_rng(seed)
    c, w = _c(oracle)
    f = w * (1 + 0.05 * rng.standard_normal(Q))
    g = 1e-3 * rng.standard_normal(3)
    d = rng.random()
    uB = 0.05 * rng.standard_normal(3)
    S = 1e-3 * rng.standard_normal((3, 3)); S = 0.5 * (S + S.T)
    sigma, tau0, cs = 0.7, 0.6, 0.17
    out, diag = oracle.collide_cell(f, g, d, uB, S, sigma, tau0, cs)
    rho = f.sum()
    u = (c @ f + g) / rho
    uh = d * u + (1 - d) * uB
    assert abs(diag[0] - rho) < 1e-15 and np.allclose(diag[1:4], uh, atol=1e-16)
    assert abs(out.sum() - rho) < 1e-14
    assert np.allclose(c @ out, rho * uh, atol=1e-15)
    pi = np.einsum("i,ai,bi->ab", f, c, c) - rho / 3 * np.eye(3) - rho * np.outer(uh, uh)
    tau = diag[4]
    a2 = sigma * pi - (1 - sigma) * 2 * rho / 3 * tau * S
    P_out = np.einsum("i,ai,bi->ab", out, c, c)
    assert np.allclose(P_out, rho * np.outer(uh, uh) + rho / 3 * np.eye(3) + (1 - 1 / tau) * a2, atol=1e-15)
    # third-order part: supported third moments = rho uuu (+delta parts) + (1-1/tau) (u a2 recursion), R3
    a3 = (np.einsum("a,bg->abg", uh, a2) + np.einsum("b,ag->abg", uh, a2) + np.einsum("g,ab->abg", uh, a2))
    for a, b, g_ in [(0, 0, 1), (0, 1, 1), (1, 1, 2), (0, 1, 2)]:
        m3 = np.sum(out * c[a] * c[b] * c[g_])
        e = rho * uh[a] * uh[b] * uh[g_] + rho / 3 * (uh[a] * (b == g_) + uh[b] * (a == g_) + uh[g_] * (a == b))
        e += (1 - 1 / tau) * a3[a, b, g_]
        assert abs(m3 - e) < 1e-15


# ------------------------------------------------------------------ P4 / P5 HLBM limits
def test_hlbm_porosity_one_ignores_solid_velocity(oracle):
    """Eq. 12 (R1): d = 1 is plain HRR -- the result must not depend on u^B at all (bit-identical)."""
    rng = np.random.default_rng(5)
    _, w = _c(oracle)
    f = w * (1 + 0.05 * rng.standard_normal(Q))
    S = np.zeros((3, 3))
    a, _ = oracle.collide_cell(f, np.zeros(3), 1.0, np.zeros(3), S, 0.995, 0.55, 0.1)
    b, _ = oracle.collide_cell(f, np.zeros(3), 1.0, np.array([0.3, -0.2, 0.1]), S, 0.995, 0.55, 0.1)
    assert np.array_equal(a, b)


def test_hlbm_porosity_zero_imposes_solid_velocity(oracle):
    """d = 0: post-collision momentum is rho*u^B whatever the fluid momentum was (no-slip)."""
    rng = np.random.default_rng(6)
    c, w = _c(oracle)
    f = w * (1 + 0.05 * rng.standard_normal(Q))
    uB = np.array([0.03, -0.02, 0.01])
    out, _ = oracle.collide_cell(f, np.zeros(3), 0.0, uB, np.zeros((3, 3)), 0.995, 0.55, 0.1)
    assert np.allclose(c @ out, f.sum() * uB, atol=1e-16)


# ------------------------------------------------------------------ P8 Smagorinsky closed form
def test_smagorinsky_fixed_point(oracle):
    """Eq. 4 + Eq. 14: tau_eff = tau0 + nu_t/cs^2, nu_t = Cs^2 |S|, |S| = sqrt(2 S:S),
    S = -Pi/(2 rho cs^2 tau_eff)  (R6) -- the closed form must satisfy this implicit relation."""
    rng = np.random.default_rng(7)
    for _ in range(10):
        pi = 1e-3 * rng.standard_normal((3, 3)); pi = 0.5 * (pi + pi.T)
        rho, tau0, cs = 1.03, 0.5 + 0.1 * rng.random(), 0.05 + 0.2 * rng.random()
        tau = oracle.tau_eff(tau0, cs, rho, pi)
        S = -pi / (2 * rho / 3 * tau)
        nut = cs ** 2 * np.sqrt(2 * np.sum(S * S))
        assert abs(tau - (tau0 + 3 * nut)) < 1e-14
    assert oracle.tau_eff(0.6, 0.1, 1.0, np.zeros((3, 3))) == pytest.approx(0.6, abs=1e-16)


# ------------------------------------------------------------------ brute force: one step on a tiny lattice
def _numpy_step(O, f, shape, tau0, sigma, cs, g):
    """One periodic step assembled from numpy primitives: np.roll central differences for S^FD,
    the oracle's per-cell collision, np.roll for streaming (f_i(x+c_i) = f*_i(x))."""
    nz, ny, nx = shape
    c, w = _c(O)
    F = f.reshape(Q, nz, ny, nx)
    rho = F.sum(0)
    u = (np.einsum("ai,izyx->azyx", c, F) + np.asarray(g)[:, None, None, None]) / rho
    grad = np.zeros((3, 3) + rho.shape)  # grad[a][b] = d_b u_a; array axes (z,y,x) <-> b = (2,1,0)
    for b, ax in ((0, 2), (1, 1), (2, 0)):
        grad[:, b] = 0.5 * (np.roll(u, -1, axis=ax + 1) - np.roll(u, 1, axis=ax + 1))
    out = np.zeros_like(F)
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        G = grad[:, :, z, y, x]
        o, _ = O.collide_cell(F[:, z, y, x], g, 1.0, np.zeros(3), 0.5 * (G + G.T), sigma, tau0, cs)
        out[:, z, y, x] = o
    res = np.zeros_like(F)
    for i in range(Q):
        res[i] = np.roll(out[i], shift=(int(c[2, i]), int(c[1, i]), int(c[0, i])), axis=(0, 1, 2))
    return res.reshape(Q, -1)


def test_one_step_matches_numpy_assembly(oracle):
    """O2+O3 field assembly (neighbour indexing, FD stencil R5, streaming direction Eq. 6 lhs) on a
    6x5x4 periodic lattice against np.roll."""
    nx, ny, nz = 6, 5, 4
    rng = np.random.default_rng(11)
    _, w = _c(oracle)
    f0 = w[:, None] * (1 + 0.05 * rng.standard_normal((Q, nx * ny * nz)))
    g = (1e-4, -2e-4, 3e-4)
    p = oracle.make_params(nx, ny, nz, tau0=0.6, sigma=0.4, smagorinsky_cs=0.1, body_force=g)
    L = oracle.Lattice(p)
    L.set_populations(f0)
    L.step(1)
    ref = _numpy_step(oracle, f0, (nz, ny, nx), 0.6, 0.4, 0.1, g)
    assert np.allclose(L.populations(), ref, atol=1e-15)


def test_mirror_axis_equals_even_extension(oracle):
    """R12: a MIRROR y-axis of ny cells must evolve exactly like the lower half of a periodic lattice
    of 2*ny cells started from the mirror-symmetric state (c_y-flipped populations)."""
    nx, ny, nz = 4, 5, 3
    rng = np.random.default_rng(12)
    c, w = _c(oracle)
    f0 = (w[:, None] * (1 + 0.05 * rng.standard_normal((Q, nz * ny * nx)))).reshape(Q, nz, ny, nx)
    flip = _flip_y(c)
    big = np.zeros((Q, nz, 2 * ny, nx))
    big[:, :, :ny] = f0
    big[:, :, ny:] = f0[flip][:, :, ::-1]
    kw = dict(tau0=0.58, sigma=0.3, smagorinsky_cs=0.12, body_force=(1e-4, 0, 0))
    A = oracle.Lattice(oracle.make_params(nx, ny, nz, mode=(0, 1, 0), **kw))
    B = oracle.Lattice(oracle.make_params(nx, 2 * ny, nz, **kw))
    A.set_populations(f0.reshape(Q, -1)); B.set_populations(big.reshape(Q, -1))
    A.step(3); B.step(3)
    fa = A.populations().reshape(Q, nz, ny, nx)
    fb = B.populations().reshape(Q, nz, 2 * ny, nx)
    assert np.allclose(fa, fb[:, :, :ny], atol=1e-15)


# ------------------------------------------------------------------ FD strain: sign, factor, stencil
def test_hybrid_fd_term_closed_form(oracle):
    """sigma = 0: post-collision off-diagonal stress of an equilibrium shear wave u_x = A sin(k y) is
    rho u u - (1 - 1/tau) 2 rho cs^2 tau S_xy with S_xy = (A/2) sin(k) cos(k y)  (Eq. 7, Eq. 10 with R2,
    central differences R5)."""
    nx, ny, nz = 3, 16, 3
    A_, k = 0.02, 2 * np.pi / 16
    c, w = _c(oracle)
    y = np.tile(np.arange(ny)[None, :, None], (nz, 1, nx)).reshape(-1).astype(float)
    u = np.zeros((3, nx * ny * nz)); u[0] = A_ * np.sin(k * y)
    tau0 = 0.7
    L = oracle.Lattice(oracle.make_params(nx, ny, nz, tau0=tau0, sigma=0.0, smagorinsky_cs=0.0))
    L.init_equilibrium(np.ones(nx * ny * nz), u, False)
    f0 = L.populations()
    L.step(1)
    f1 = L.populations().reshape(Q, nz, ny, nx)
    # undo streaming with np.roll to get the post-collision state at the source cell
    post = np.stack([np.roll(f1[i], shift=(-int(c[2, i]), -int(c[1, i]), -int(c[0, i])), axis=(0, 1, 2))
                     for i in range(Q)]).reshape(Q, -1)
    Pxy = np.einsum("ic,i,i->c", post, c[0], c[1])
    Sxy = 0.5 * A_ * np.sin(k) * np.cos(k * y)
    expect = -(1 - 1 / tau0) * 2 * (1 / 3) * tau0 * Sxy      # rho = 1, u_x u_y = 0
    assert np.allclose(Pxy, expect, atol=1e-15)
    assert np.max(np.abs(expect)) > 1e-4


# ------------------------------------------------------------------ P6 / P16 viscosity from Taylor-Green decay
def _tgv2d_rate(O, n, tau0, sigma, cs, steps=(20, 60)):
    k = 2 * np.pi / n
    nz = 2
    z, y, x = np.meshgrid(np.arange(nz), np.arange(n), np.arange(n), indexing="ij")
    U0 = 0.01
    u = np.stack([U0 * np.sin(k * x) * np.cos(k * y), -U0 * np.cos(k * x) * np.sin(k * y), 0 * x * 1.0]).reshape(3, -1)
    rho = (1 + 3 * U0 ** 2 / 4 * (np.cos(2 * k * x) + np.cos(2 * k * y))).reshape(-1)
    L = O.Lattice(O.make_params(n, n, nz, tau0=tau0, sigma=sigma, smagorinsky_cs=cs))
    L.init_equilibrium(rho, u, True)
    L.step(steps[0])
    _, v0 = L.moments()
    L.step(steps[1] - steps[0])
    _, v1 = L.moments()
    rate = -np.log(np.sum(v1 ** 2) / np.sum(v0 ** 2)) / (steps[1] - steps[0])
    return rate / (4 * (tau0 - 0.5) / 3 * k * k)   # energy decays at 4 nu k^2


@pytest.mark.parametrize("tau0,sigma,cs", [(0.55, 1.0, 0.0), (0.8, 0.5, 0.0), (0.8, 0.0, 0.0), (0.55, 0.995, 0.1)])
def test_taylor_green_decay_gives_viscosity(oracle, tau0, sigma, cs):
    """nu = cs^2 (tau - 1/2) (Eq. 14): kinetic energy of the 2-D Taylor-Green vortex (exact NS solution)
    decays at 4 nu k^2.  Holds for the local (sigma=1), hybrid and pure-FD (sigma=0) reconstruction, which
    pins the sign and factor of Eq. 7/10 (R2) dynamically."""
    r = _tgv2d_rate(oracle, 32, tau0, sigma, cs)
    assert abs(r - 1) < 0.02, r


def test_second_order_convergence(oracle):
    """second-order in space -- the decay-rate error drops ~4x from N=16 to N=32."""
    e16 = abs(_tgv2d_rate(oracle, 16, 0.8, 0.5, 0.0, steps=(10, 30)) - 1)
    e32 = abs(_tgv2d_rate(oracle, 32, 0.8, 0.5, 0.0, steps=(40, 120)) - 1)
    assert e16 / e32 > 3.0, (e16, e32)


def test_config1_tgv3d_decay(oracle):
    """BASELINE config 1: 3-D TGV, d ln E/dt over steps 10..20 ~ -6 nu k^2 (early-time viscous decay)."""
    from paper_2510_13726_b200 import inputs
    case = inputs.case_tgv(32, 20)
    L = oracle.Lattice(oracle.make_params(32, 32, 32, **case.params))
    inputs.apply_case(case, L)
    E = []
    for s in range(21):
        _, v = L.moments()
        E.append(np.sum(v ** 2))
        L.step(1)
    rate = np.mean(np.diff(np.log(E))[10:20])
    k = 2 * np.pi / 32
    assert abs(rate / (-6 * (0.05 / 3) * k * k) - 1) < 0.03


# ------------------------------------------------------------------ P9 / P10 Poiseuille + force
@pytest.fixture(scope="module")
def poiseuille(oracle):
    nx, ny, nz = 3, 24, 3
    tau0, g = 0.8, 1e-6
    y = np.tile(np.arange(ny)[None, :, None], (nz, 1, nx)).reshape(-1).astype(float)
    phi = np.minimum(y - 1.5, (ny - 2.5) - y)          # solid for y<=0.5.. i.e. cells 0 and ny-1 (phi<=-1)
    L = oracle.Lattice(oracle.make_params(nx, ny, nz, tau0=tau0, sigma=1.0, smagorinsky_cs=0.0,
                                          body_force=(g, 0, 0), eps_cells=2.0))
    L.set_static_geometry(phi, np.ones(nx * ny * nz, np.uint8))
    L.init_equilibrium(np.ones(nx * ny * nz), np.zeros((3, nx * ny * nz)), False)
    L.step(9000)
    return L, (nx, ny, nz), tau0, g


def test_poiseuille_second_difference(poiseuille):
    """R11 body force + porosity-0 wall (P5): steady profile obeys u(y+1) - 2u(y) + u(y-1) = -g/nu."""
    L, (nx, ny, nz), tau0, g = poiseuille
    _, v = L.moments()
    ux = v[0].reshape(nz, ny, nx)[1, :, 1]
    nu = (tau0 - 0.5) / 3
    d2 = ux[5:ny - 3] - 2 * ux[4:ny - 4] + ux[3:ny - 5]     # centres whose stencil is plain fluid (d = 1)
    assert np.allclose(d2 / (-g / nu), 1.0, atol=1e-6), d2 / (-g / nu)
    assert ux[0] == pytest.approx(0, abs=1e-12) or abs(ux[0]) < 1e-3 * ux.max()


def test_momentum_exchange_equals_body_force(poiseuille):
    """Eq. 23 with R7: in steady state the force ON the walls equals the momentum the body
    force injects per step into the fluid (global momentum balance), sign positive along g."""
    L, (nx, ny, nz), tau0, g = poiseuille
    t, tag, d = L.cell_types()
    F = L.forces()[-1]
    rho, _ = L.moments()
    # Eq. 23's control volume is the set {d < 1}; in steady state the momentum flowing into it over its
    # links is what the body force injects per step into the cells outside it (rho u = j + g there).
    injected = g * np.sum(d == 1.0)
    assert F[1, 0] > 0
    assert F[1, 0] == pytest.approx(injected, rel=1e-8)
    assert abs(F[1, 1]) < 1e-12 and abs(F[1, 2]) < 1e-12


def test_force_vanishes_for_comoving_solid(oracle):
    """Eq. 23 structure (R7: second population is the opposite one): a solid translating with a uniform
    stream at the same velocity feels no force; with the printed f_i instead of f_ibar the sum would be
    2 rho U per cell."""
    from paper_2510_13726_b200 import inputs
    nx = ny = nz = 12
    U = np.array([0.03, -0.02, 0.01])
    phi = inputs.sphere_phi(nx, ny, nz, (5.5, 5.5, 5.5), 3.0)
    L = oracle.Lattice(oracle.make_params(nx, ny, nz))
    L.set_static_geometry(phi, np.ones(nx * ny * nz, np.uint8))
    L.set_body(1, vel=U)
    u = np.tile(U[:, None], (1, nx * ny * nz))
    L.init_equilibrium(np.ones(nx * ny * nz), u, False)
    F = L.force_only()
    assert np.max(np.abs(F)) < 1e-13


def _sphere_at_rest(oracle, rho, centre_body, n=16, R=3.6):
    from paper_2510_13726_b200 import inputs
    phi = inputs.sphere_phi(n, n, n, (7.3, 8.1, 7.6), R)
    L = oracle.Lattice(oracle.make_params(n, n, n))
    L.set_static_geometry(phi, np.ones(n ** 3, np.uint8))
    L.set_body(1, centre=centre_body)
    L.init_equilibrium(rho, np.zeros((3, n ** 3)), False)
    return L


def test_torque_of_hydrostatic_load_closed_form(oracle):
    """Torque output (moment of Eq. 23's per-cell forces): for a fluid
    at rest with a linear density rho = 1 + a.x every population is w_i rho, so a cell's momentum-exchange
    force is -sum_i c_i w_i (rho(x + c_i) + rho(x)) = -a cs^2 (the pressure gradient), and the torque on N
    such cells about x_c is N (xbar - x_c) x (-a/3), xbar their centroid.  Fails for F x r, a lever arm
    from the wrong origin, a transposed component."""
    n = 16
    a = np.array([2e-3, -1e-3, 3e-3])
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    rho = (1 + a[0] * x + a[1] * y + a[2] * z).ravel().astype(np.float64)
    xc = np.array([2.5, 11.0, 6.25])
    L = _sphere_at_rest(oracle, rho, xc)
    F = L.force_only()
    M = L.torque_only()
    t, tag, d = L.cell_types()
    cells = np.flatnonzero(d < 1.0)
    assert len(cells) > 100
    pos = np.stack([x.ravel()[cells], y.ravel()[cells], z.ravel()[cells]], axis=1).astype(np.float64)
    assert pos.min() >= 2 and pos.max() <= n - 3          # away from the periodic seam of rho
    assert np.allclose(F[1], -len(cells) * a / 3, rtol=1e-12, atol=1e-16)
    expect = np.cross(pos.sum(axis=0) - len(cells) * xc, -a / 3)
    assert np.max(np.abs(expect)) > 1e-2
    assert np.allclose(M[1], expect, rtol=1e-11, atol=1e-15)
    assert np.all(M[[0, 2, 3]] == 0)


def test_torque_shift_of_reference_point(oracle):
    """Moving the reference point by D changes the torque by -D x F (rigid-body statics): pins the cross
    product's orientation against the already pinned force sum, on a flow with non-trivial forces."""
    from paper_2510_13726_b200 import inputs
    n = 16
    rho, u = inputs.noisy_uniform(n, n, n, (0.04, 0.01, -0.02), 5e-3, 5)
    out = []
    for xc in [(7.3, 8.1, 7.6), (1.0, 12.5, -3.0)]:
        phi = inputs.sphere_phi(n, n, n, (7.3, 8.1, 7.6), 3.6)
        L = oracle.Lattice(oracle.make_params(n, n, n))
        L.set_static_geometry(phi, np.ones(n ** 3, np.uint8))
        L.set_body(1, centre=xc)
        L.init_equilibrium(rho, u, True)
        L.step(3)
        out.append((np.array(xc), L.forces()[-1, 1], L.torques()[-1, 1]))
    (c0, F0, M0), (c1, F1, M1) = out
    assert np.array_equal(F0, F1) and np.linalg.norm(F0) > 1e-3
    assert np.allclose(M1, M0 - np.cross(c1 - c0, F0), rtol=1e-10, atol=1e-14)


# ------------------------------------------------------------------ P11 wall function
@pytest.mark.parametrize("U,y,nu", [(0.05, 2.75, 3.156e-4), (0.04, 3.0, 6.25e-5), (1e-4, 2.2, 1e-2), (0.2, 2.9, 1.3e-4)])
def test_spalding_relation(oracle, U, y, nu):
    """Converged Newton (Eq. 19) root satisfies Eq. 18 to 1e-12; never below the laminar bound of Eq. 20."""
    u0 = np.sqrt(nu * U / y)
    ut, _ = oracle.newton_utau(u0, U, y, nu, max_iter=200, tol=0.0)
    yp = y * ut / nu
    assert abs(oracle.spalding_f(ut, U, y, nu)) < 1e-12 * max(yp, 1.0)
    assert ut >= u0 * (1 - 1e-12)
    # Eq. 17 written out independently
    up, k, E = U / ut, 0.41 * U / ut, 9.8
    assert yp == pytest.approx(up + (np.exp(k) - 1 - k - k * k / 2 - k ** 3 / 6) / E, rel=1e-11)


def test_spalding_asymptotes(oracle):
    """y+ -> 0: u+ = y+ (u_tau -> sqrt(nu U / y)); large y+: log law u+ ~ ln(E y+)/kappa."""
    U, y, nu = 1e-6, 1.0, 0.1
    ut, _ = oracle.newton_utau(np.sqrt(nu * U / y), U, y, nu, max_iter=100, tol=0.0)
    assert ut == pytest.approx(np.sqrt(nu * U / y), rel=1e-6)
    U, y, nu = 0.1, 50.0, 1e-5
    # the cold start of Eq. 20 sits at u+ = 707; Newton on the exponential sheds ~1/kappa per iteration
    ut, _ = oracle.newton_utau(np.sqrt(nu * U / y), U, y, nu, max_iter=3000, tol=0.0)
    yp, up = y * ut / nu, U / ut
    assert abs(oracle.spalding_f(ut, U, y, nu)) < 1e-12 * yp
    assert yp > 1e3
    assert up == pytest.approx(np.log(9.8 * yp) / 0.41, rel=0.02)


def test_newton_stop_rule(oracle):
    """at most 10 iterations; stops early once |f(u^{j+1}) - f(u^j)| < 1e-4."""
    U, y, nu = 0.05, 2.75, 3.156e-4
    root, _ = oracle.newton_utau(np.sqrt(nu * U / y), U, y, nu, max_iter=200, tol=0.0)
    _, it_cold = oracle.newton_utau(np.sqrt(nu * U / y), U, y, nu)
    assert 1 <= it_cold <= 10
    _, it_warm = oracle.newton_utau(root, U, y, nu)
    assert it_warm == 1


def test_wall_model_on_uniform_and_shear_flow(oracle):
    """WallModelO (R8, R10, R13, R15) on prescribed states over a flat wall phi = y - 1.25:
    uniform stream V: U = |V_t|, slip = u_tau V_t/|V_t| with u_tau solving Eq. 18 at y = y1 + h_s, S_wm = 0;
    linear shear v_x = gamma y: trilinear sampling is exact, S_xy = gamma/2 and U = gamma (y_w + h_s)."""
    from paper_2510_13726_b200 import inputs
    nx, ny, nz = 4, 12, 4
    n = nx * ny * nz
    phi = inputs.wall_phi(nx, ny, nz, 1.25)
    tau0 = 0.5 + 3 * 3.156e-4
    nu = (tau0 - 0.5) / 3
    mk = lambda: oracle.Lattice(oracle.make_params(nx, ny, nz, mode=(0, 1, 0), tau0=tau0, sampling_distance=2.0))
    # uniform stream with a wall-normal component that must be projected out
    V = np.array([0.03, 0.004, -0.02])
    L = mk(); L.set_static_geometry(phi, np.ones(n, np.uint8)); L.enable_wall_model(True)
    L.init_equilibrium(np.ones(n), np.tile(V[:, None], (1, n)), False)
    L.wall_model_only()
    idx, y1n, ut, valid = L.wall_list()
    assert len(idx) == nx * nz and np.all(valid == 1)
    assert np.allclose(y1n, [0, 0.75, 0], atol=1e-12)
    Vt = np.array([V[0], 0, V[2]]); U = np.linalg.norm(Vt)
    cell = int(idx[0])
    ok, utau, uwm, swm = L.wall_state(cell)
    assert ok == 1
    expect, _ = oracle.newton_utau(np.sqrt(nu * U / 2.75), U, 2.75, nu)
    assert utau == pytest.approx(expect, rel=1e-13)
    assert np.allclose(uwm, utau * Vt / U, atol=1e-15)
    assert np.allclose(swm, 0, atol=1e-14)
    # linear shear
    gamma = 0.004
    y = np.tile(np.arange(ny)[None, :, None], (nz, 1, nx)).reshape(-1).astype(float)
    u = np.zeros((3, n)); u[0] = gamma * y
    L = mk(); L.set_static_geometry(phi, np.ones(n, np.uint8)); L.enable_wall_model(True)
    L.init_equilibrium(np.ones(n), u, False)
    L.wall_model_only()
    ok, utau, uwm, swm = L.wall_state(cell)
    assert np.allclose(swm, [0, 0, 0, gamma / 2, 0, 0], atol=1e-14)
    U = gamma * 4.0                   # wall cell y=2, sampled at y=4
    expect, _ = oracle.newton_utau(np.sqrt(nu * U / 2.75), U, 2.75, nu)
    assert utau == pytest.approx(expect, rel=1e-12)


# ------------------------------------------------------------------ P12 geometry
def test_porosity_level_set_and_types(oracle):
    """Def. 1 / Eq. 21-22: d = 0 for phi <= -eps/2, 1 for phi >= eps/2, linear between,
    d = 1/2 on phi = 0; types of Fig. 4."""
    nx, ny, nz = 3, 9, 3
    y = np.tile(np.arange(ny)[None, :, None], (nz, 1, nx)).reshape(-1).astype(float)
    phi = y - 3.0
    L = oracle.Lattice(oracle.make_params(nx, ny, nz, mode=(0, 1, 0), eps_cells=2.0))
    L.set_static_geometry(phi, np.ones(nx * ny * nz, np.uint8))
    L.update_geometry()
    t, tag, d = L.cell_types()
    col = lambda a: a.reshape(nz, ny, nx)[1, :, 1]
    assert list(col(d)) == [0, 0, 0, 0.5, 1, 1, 1, 1, 1]
    S, Fr, G, Fl = oracle.T_SOLID, oracle.T_FRONTIER, oracle.T_GROWTH, oracle.T_FLUID
    assert list(col(t)) == [S, S, S, Fr, G, Fl, Fl, Fl, Fl]
    assert list(col(tag)) == [1, 1, 1, 1, 1, 0, 0, 0, 0]
    phi2 = y - 3.25
    L.set_static_geometry(phi2, np.ones(nx * ny * nz, np.uint8)); L.update_geometry()
    t, tag, d = L.cell_types()
    assert np.allclose(col(d), [0, 0, 0, 0.375, 0.875, 1, 1, 1, 1])
    assert list(col(t)) == [S, S, S, Fr, Fr, G, Fl, Fl, Fl]


def test_sphere_volume(oracle):
    """sum(1 - d) over a smoothed sphere -> 4/3 pi r^3 (the wall is the level set d = 1/2)."""
    from paper_2510_13726_b200 import inputs
    n, r = 40, 12.0
    phi = inputs.sphere_phi(n, n, n, (19.5, 19.5, 19.5), r)
    L = oracle.Lattice(oracle.make_params(n, n, n))
    L.set_static_geometry(phi, np.ones(n ** 3, np.uint8)); L.update_geometry()
    _, _, d = L.cell_types()
    # closed form of the radial integral of the linear ramp of width eps = 2: 4/3 pi r^3 (1 + eps^2/(4 r^2))
    assert np.sum(1 - d) == pytest.approx(4 / 3 * np.pi * r ** 3 * (1 + 4 / (4 * r * r)), rel=1e-3)


def test_rotor_sampling_rotates_rigidly(oracle):
    """Rotor embedding: with an analytic sphere-cap reference grid the embedded phi is
    rotation invariant; with an off-axis ball it moves on a circle: its centroid at step n sits at angle
    theta0 + n*Omega about the axis (O6), and u^B = Omega x r."""
    g = 41; sp = 0.5
    ax = -10 + sp * np.arange(g)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    sdf = np.clip(np.sqrt(X ** 2 + (Y - 5.0) ** 2 + Z ** 2) - 3.0, -4, 4).astype(np.float32)   # ball at y=+5
    tag = np.ones_like(sdf, dtype=np.uint8)
    n = 24
    L = oracle.Lattice(oracle.make_params(n, n, n))
    om = 0.05
    L.set_rotor(sdf, tag, sp, (-10, -10, -10), (11.5, 11.5, 11.5), (1, 0, 0), om, 0.3, 1)
    L.init_equilibrium(np.ones(n ** 3), np.zeros((3, n ** 3)), False)
    for steps in (0, 7):
        if steps:
            L.step(steps)
        L.update_geometry()
        _, _, d = L.cell_types()
        m = (1 - d).reshape(n, n, n)
        z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
        cy = np.sum(m * (y - 11.5)) / m.sum(); cz = np.sum(m * (z - 11.5)) / m.sum(); cxm = np.sum(m * (x - 11.5)) / m.sum()
        th = 0.3 + steps * om
        assert abs(cxm) < 0.02
        assert cy == pytest.approx(5 * np.cos(th), abs=0.03)
        assert cz == pytest.approx(5 * np.sin(th), abs=0.03)
        assert m.sum() == pytest.approx(4 / 3 * np.pi * 27 * (1 + 1 / 9), rel=0.02)   # ramp-widened volume


def test_rigid_rotation_has_zero_fd_strain(oracle):
    """P15: inside a rigidly rotating solid uhat = Omega x r is linear with antisymmetric gradient, so the
    FD strain vanishes and the post-collision state there is the pure equilibrium of (rho, u^B) when sigma=0."""
    from paper_2510_13726_b200 import inputs
    n = 16
    phi = inputs.sphere_phi(n, n, n, (7.5, 7.5, 7.5), 6.0)
    L = oracle.Lattice(oracle.make_params(n, n, n, sigma=0.0, tau0=0.6))
    L.set_static_geometry(phi, np.ones(n ** 3, np.uint8))
    om = np.array([0.002, -0.001, 0.003])
    L.set_body(1, centre=(7.5, 7.5, 7.5), omega=om)
    L.init_equilibrium(np.ones(n ** 3), np.zeros((3, n ** 3)), False)
    L.step(1)
    c, w = _c(oracle)
    f1 = L.populations().reshape(Q, n, n, n)
    post = np.stack([np.roll(f1[i], shift=(-int(c[2, i]), -int(c[1, i]), -int(c[0, i])), axis=(0, 1, 2)) for i in range(Q)])
    for (x, y, z) in [(7, 7, 7), (9, 6, 8), (5, 8, 7)]:
        r = np.array([x, y, z]) - 7.5
        feq = oracle.equilibrium(1.0, np.cross(om, r))
        assert np.allclose(post[:, z, y, x], feq, atol=1e-16)


# ------------------------------------------------------------------ region split: bulk RRLBM-LES (Listing 2)
def test_bulk_region_types_and_violation(oracle):
    """the simpler model runs where no wall-modelled structure can be.  Fluid cells outside
    every FSI box become BULK (type 5), everything inside keeps its type; a solid cell outside the boxes is
    reported, not silently re-typed."""
    from paper_2510_13726_b200 import inputs
    nx, ny, nz = 24, 16, 12
    phi = inputs.sphere_phi(nx, ny, nz, (8.0, 7.5, 5.5), 3.0)
    L = oracle.Lattice(oracle.make_params(nx, ny, nz, tau0=0.6))
    L.set_static_geometry(phi, np.ones(nx * ny * nz, np.uint8))
    L.update_geometry()
    t0, _, _ = L.cell_types()
    box = (2, 15, 1, 14, 0, 12)
    L.set_fsi_region([box]); L.update_geometry()
    t1, g1, d1 = L.cell_types()
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    inside = ((x >= 2) & (x < 15) & (y >= 1) & (y < 14)).reshape(-1)
    assert np.array_equal(t1[inside], t0[inside])
    assert np.all(t0[~inside] == 0) and np.all(t1[~inside] == 5)
    assert np.all(g1[~inside] == 0) and np.all(d1[~inside] == 1.0)
    assert not L.region_violation()
    L.set_fsi_region([(9, 15, 1, 14, 0, 12)]); L.update_geometry()     # cuts through the sphere
    assert L.region_violation()
    L.set_fsi_region([]); L.update_geometry()                            # back to HHRRLBM everywhere
    assert np.array_equal(L.cell_types()[0], t0) and not L.region_violation()


def test_bulk_region_is_the_sigma_one_scheme(oracle):
    """Listing 2: the bulk model is the third-order recursive-regularised collision with
    the Smagorinsky relaxation and no hybrid part, i.e. Eq. 7 at sigma = 1.  (i) A run whose cells are all
    BULK under sigma = 0.5 reproduces, to rounding, the run with sigma = 1 and no region split; (ii) with an
    all-bulk lattice the 2-D Taylor-Green energy decays at 4 nu k^2 whatever sigma says (a bulk cell that
    still took the sigma = 0.3 hybrid part on a tau0 = 0.8 lattice would show in the split run differing
    from the reference, which itself is pinned by test_taylor_green_decay_gives_viscosity)."""
    n, nz, U0, tau0 = 32, 2, 0.01, 0.8
    k = 2 * np.pi / n
    z, y, x = np.meshgrid(np.arange(nz), np.arange(n), np.arange(n), indexing="ij")
    u = np.stack([U0 * np.sin(k * x) * np.cos(k * y), -U0 * np.cos(k * x) * np.sin(k * y), 0 * x * 1.0]).reshape(3, -1)
    rho = (1 + 3 * U0 ** 2 / 4 * (np.cos(2 * k * x) + np.cos(2 * k * y))).reshape(-1)

    def run(sigma, boxes):
        L = oracle.Lattice(oracle.make_params(n, n, nz, tau0=tau0, sigma=sigma, smagorinsky_cs=0.1))
        L.set_fsi_region(boxes)
        L.init_equilibrium(rho, u, True)
        L.step(20); _, v0 = L.moments()
        L.step(40); _, v1 = L.moments()
        types = L.cell_types()[0]
        return v1, -np.log(np.sum(v1 ** 2) / np.sum(v0 ** 2)) / 40 / (4 * (tau0 - 0.5) / 3 * k * k), types

    v_ref, r_ref, t_ref = run(1.0, [])
    v_blk, r_blk, t_blk = run(0.3, [(0, 0, 0, 0, 0, 0)])       # one empty box: every cell is bulk
    assert np.all(t_ref == 0) and np.all(t_blk == 5)
    assert np.max(np.abs(v_blk - v_ref)) <= 1e-15
    assert abs(r_blk - 1) < 0.02, r_blk
    v_hyb, r_hyb, _ = run(0.3, [])                              # the hybrid scheme itself differs measurably
    assert np.max(np.abs(v_hyb - v_ref)) > 1e-9


def test_bulk_region_interface_is_seamless(oracle):
    """A fluid-only lattice split into an FSI half and a bulk half: cells in the FSI half keep the hybrid
    collision (they differ from the all-bulk run), cells deep in the bulk half follow the sigma = 1 run
    until the difference has travelled there (one cell per step)."""
    n, nz, U0, tau0 = 32, 2, 0.02, 0.7
    k = 2 * np.pi / n
    z, y, x = np.meshgrid(np.arange(nz), np.arange(n), np.arange(n), indexing="ij")
    u = np.stack([U0 * np.sin(k * x) * np.cos(k * y), -U0 * np.cos(k * x) * np.sin(k * y), 0 * x * 1.0]).reshape(3, -1)
    rho = np.ones(n * n * nz)

    def run(sigma, boxes, steps):
        L = oracle.Lattice(oracle.make_params(n, n, nz, tau0=tau0, sigma=sigma, smagorinsky_cs=0.0))
        L.set_fsi_region(boxes)
        L.init_equilibrium(rho, u, True)
        L.step(steps)
        return L.moments()[1].reshape(3, nz, n, n)

    steps = 3
    split = run(0.0, [(0, 8, 0, n, 0, nz)], steps)       # x in [0, 8) hybrid (pure FD), the rest bulk
    allb = run(1.0, [], steps)
    far = slice(8 + steps + 1, n - steps - 1)            # bulk cells no hybrid cell has reached yet
    assert np.max(np.abs(split[:, :, :, far] - allb[:, :, :, far])) <= 1e-16
    assert np.max(np.abs(split[:, :, :, 0:8] - allb[:, :, :, 0:8])) > 1e-9


# ------------------------------------------------------------------ Musker's wall function (BASELINE.json config 3)
def test_musker_profile_limits_and_ode(oracle):
    """Musker's explicit profile: no slip (u+ -> 0, du+/dy+ -> 1 at the wall), log law u+ -> ln(y+)/0.411 + 5.0 far
    from it, monotone, and its slope follows Musker's eddy-viscosity ODE du+/dy+ = (k + C y^2)/(k + C y^2 + C k y^3),
    k = 0.41, C = 0.001093 (the explicit form is that ODE integrated with rounded constants: 1 % agreement)."""
    M = oracle.musker_uplus
    assert abs(M(0.0)) < 0.02
    assert abs((M(1e-3) - M(0.0)) / 1e-3 - 1.0) < 2e-3
    for yp in (3e3, 1e4, 1e5):
        assert abs(M(yp) - (np.log(yp) / 0.4112 + 5.0)) < 0.03
    ys = np.logspace(-2, 5, 400)
    u = np.array([M(y) for y in ys])
    assert np.all(np.diff(u) > 0)
    for yp in (0.5, 2.0, 5.0, 11.0, 30.0, 100.0, 1000.0):
        h = 1e-4 * yp
        slope = (M(yp + h) - M(yp - h)) / (2 * h)
        ode = (0.41 + 0.001093 * yp ** 2) / (0.41 + 0.001093 * yp ** 2 + 0.001093 * 0.41 * yp ** 3)
        assert abs(slope / ode - 1) < 0.012, (yp, slope, ode)
    # between the two laws: the buffer layer value every law of the wall passes through (u+ ~ 13.2 at y+ = 30)
    assert 12.5 < M(30.0) < 14.0


@pytest.mark.parametrize("U,y,nu", [(0.05, 2.75, 3.156e-4), (0.04, 3.0, 6.25e-5), (1e-4, 2.2, 1e-2), (0.2, 2.9, 1.3e-4)])
def test_musker_newton_satisfies_its_relation(oracle, U, y, nu):
    """Converged Newton (Eq. 19 run long) on Musker's residual: U/u_tau = u+(y u_tau/nu) to 1e-12; close to Spalding's
    u_tau for the same sample (two fits of the same law of the wall)."""
    u0 = np.sqrt(nu * U / y)
    ut, it = oracle.newton_utau_musker(u0, U, y, nu, max_iter=200, tol=0.0)
    assert ut > 0
    assert abs(U / ut - oracle.musker_uplus(y * ut / nu)) <= 1e-12 * max(1.0, U / ut)
    us, _ = oracle.newton_utau(u0, U, y, nu, max_iter=200, tol=0.0)
    assert abs(ut / us - 1) < 0.08
    # the paper's stop rule applies unchanged
    ut10, it10 = oracle.newton_utau_musker(u0, U, y, nu, max_iter=10, tol=1e-4)
    assert 1 <= it10 <= 10


def test_wall_model_with_musker_profile_on_uniform_flow(oracle):
    """WallModelO with the wall function switched to Musker's profile: over a flat wall in a uniform stream the stored
    u_tau is the Newton solution of U/u_tau = u+_Musker((y1 + h_s) u_tau/nu), everything else (projection, slip
    direction, zero strain) as with Spalding's law."""
    from paper_2510_13726_b200 import inputs
    nx, ny, nz = 4, 12, 4
    n = nx * ny * nz
    phi = inputs.wall_phi(nx, ny, nz, 1.25)
    tau0 = 0.5 + 3 * 6.25e-5
    nu = (tau0 - 0.5) / 3
    V = np.array([0.05, 0.004, -0.02])
    L = oracle.Lattice(oracle.make_params(nx, ny, nz, mode=(0, 1, 0), tau0=tau0, sampling_distance=2.0))
    L.set_static_geometry(phi, np.ones(n, np.uint8)); L.enable_wall_model(True); L.set_wall_function(1)
    L.init_equilibrium(np.ones(n), np.tile(V[:, None], (1, n)), False)
    L.wall_model_only()
    idx, _, _, valid = L.wall_list()
    assert np.all(valid == 1)
    Vt = np.array([V[0], 0, V[2]]); U = np.linalg.norm(Vt)
    ok, utau, uwm, swm = L.wall_state(int(idx[0]))
    expect, _ = oracle.newton_utau_musker(np.sqrt(nu * U / 2.75), U, 2.75, nu)
    spal, _ = oracle.newton_utau(np.sqrt(nu * U / 2.75), U, 2.75, nu)
    assert utau == pytest.approx(expect, rel=1e-13) and abs(utau - spal) > 1e-6 * spal
    assert np.allclose(uwm, utau * Vt / U, atol=1e-15) and np.allclose(swm, 0, atol=1e-14)


# ------------------------------------------------------------------ second readings of the wall model (R22)
def test_spalding_inverse_satisfies_eq17_and_its_limits(oracle):
    """u+(y+) used by the 'velocity at Y1' reading: satisfies Eq. 17 (:166) to 1e-13, is the
    viscous sublayer u+ = y+ near the wall and the log law ln(E y+)/kappa far from it, increasing throughout."""
    kap, E = 0.41, 9.8
    ys = np.concatenate([[0.0], np.logspace(-3, 5, 300)])
    us = np.array([oracle.spalding_uplus(y) for y in ys])
    k = kap * us
    back = us + (np.exp(k) - 1 - k - k ** 2 / 2 - k ** 3 / 6) / E
    assert np.allclose(back, ys, rtol=1e-13, atol=1e-15)
    assert np.all(np.diff(us) > 0) and us[0] == 0.0
    assert oracle.spalding_uplus(1e-3) == pytest.approx(1e-3, rel=1e-9)
    assert oracle.spalding_uplus(1.0) == pytest.approx(1.0, rel=2e-3)
    for yp in (1e3, 1e4, 1e5):
        assert oracle.spalding_uplus(yp) == pytest.approx(np.log(E * yp) / kap, rel=0.05)
    assert 12.5 < oracle.spalding_uplus(30.0) < 14.5        # buffer-layer value every law of the wall passes through
    # the two wall functions are fits of the same profile
    for yp in (0.5, 5.0, 30.0, 100.0, 1000.0):
        assert oracle.wall_uplus(0, yp) == pytest.approx(oracle.wall_uplus(1, yp), rel=0.12)
        assert oracle.wall_uplus(1, yp) == oracle.musker_uplus(yp)


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("U,y,nu", [(0.05, 2.75, 3.156e-4), (0.04, 3.0, 6.25e-5), (1e-4, 2.2, 1e-2), (0.2, 2.9, 1.3e-4)])
def test_analytic_wall_shear_is_the_slope_of_the_profile(oracle, kind, U, y, nu):
    """'shear stress (cf. Eq. 17)' second reading: with u_tau converged for the sample (U, y), the
    analytic du/dy equals the centred difference of the profile u(y) = u_tau u+(y u_tau/nu) at y; in the viscous
    sublayer it is tau_w/(rho nu) = u_tau^2/nu (Eq. 15)."""
    u0 = np.sqrt(nu * U / y)
    newton = oracle.newton_utau_musker if kind else oracle.newton_utau
    ut, _ = newton(u0, U, y, nu, max_iter=200, tol=0.0)
    prof = lambda yy: ut * oracle.wall_uplus(kind, yy * ut / nu)
    assert prof(y) == pytest.approx(U, rel=1e-10)
    h = 1e-4 * y
    fd = (prof(y + h) - prof(y - h)) / (2 * h)
    assert oracle.wall_shear(kind, ut, U, y, nu) == pytest.approx(fd, rel=1e-6)
    # never steeper than the sublayer (Musker's closed form, with its rounded constants, has slope 1.0003 at the wall)
    assert 0 < oracle.wall_shear(kind, ut, U, y, nu) <= ut * ut / nu * (1 + (1e-3 if kind else 1e-12))
    # sublayer: a sample at y+ = 0.01
    ys, Us = 0.01 * nu / ut, 0.01 * ut
    assert oracle.wall_shear(kind, ut, Us, ys, nu) == pytest.approx(ut * ut / nu, rel=2e-3 if kind else 1e-6)


@pytest.mark.parametrize("kind", [0, 1])
def test_wall_model_second_readings_on_uniform_flow(oracle, kind):
    """WallModelO with slip = 'wall-function velocity at y1' and shear = 'analytic slope' (R22) over a flat wall
    in a uniform stream: u_tau unchanged (same sample, same Newton); |u_wm| = u_tau u+(y1 u_tau/nu) < U along the
    tangential sample; S_wm = sym(du/dy e_t n^T): trace 0, sqrt(2 S:S) = du/dy, and S n . e_t = du/dy / 2."""
    from paper_2510_13726_b200 import inputs
    nx, ny, nz = 4, 12, 4
    n = nx * ny * nz
    phi = inputs.wall_phi(nx, ny, nz, 1.25)
    tau0 = 0.5 + 3 * 6.25e-5
    nu = (tau0 - 0.5) / 3
    V = np.array([0.05, 0.004, -0.02])
    out = []
    for slip, shear in ((0, 0), (1, 1)):
        L = oracle.Lattice(oracle.make_params(nx, ny, nz, mode=(0, 1, 0), tau0=tau0, sampling_distance=2.0,
                                              newton_max_iter=200, newton_tol=0.0))
        L.set_static_geometry(phi, np.ones(n, np.uint8)); L.enable_wall_model(True); L.set_wall_function(kind)
        L.set_wall_model_variant(slip, shear)
        L.init_equilibrium(np.ones(n), np.tile(V[:, None], (1, n)), False)
        L.wall_model_only()
        idx, y1n, _, valid = L.wall_list()
        assert np.all(valid == 1)
        out.append(L.wall_state(int(idx[0])) + (y1n[0],))
    (_, ut0, uw0, sw0, _), (_, ut1, uw1, sw1, y1v) = out
    Vt = np.array([V[0], 0, V[2]]); U = np.linalg.norm(Vt); et = Vt / U
    y1 = np.linalg.norm(y1v); nrm = y1v / y1
    assert y1 == pytest.approx(0.75, abs=1e-6) and np.allclose(nrm, [0, 1, 0], atol=1e-9)
    assert ut1 == ut0 and np.allclose(sw0, 0, atol=1e-14)
    up1 = oracle.wall_uplus(kind, y1 * ut1 / nu)
    assert np.allclose(uw1, ut1 * up1 * et, rtol=1e-12, atol=1e-16)
    assert ut1 * up1 < U and np.linalg.norm(uw1) != pytest.approx(np.linalg.norm(uw0), rel=1e-3)
    dudy = oracle.wall_shear(kind, ut1, U, 2.75, nu)
    S = np.array([[sw1[0], sw1[3], sw1[4]], [sw1[3], sw1[1], sw1[5]], [sw1[4], sw1[5], sw1[2]]])
    assert abs(np.trace(S)) < 1e-15
    assert np.sqrt(2 * np.sum(S * S)) == pytest.approx(dudy, rel=1e-12)
    assert et @ S @ nrm == pytest.approx(0.5 * dudy, rel=1e-12)
