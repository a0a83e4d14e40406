"""GPU-vs-oracle parity on the paper's own velocity set, D3Q19 -- run with -m gpu.

libhhrr_q19.so is the same source built with HHRR_Q = 19 (19 TMA planes, 152 B per cell update); the oracle is
oracle/hhrr_oracle_q19.c.  Same bars as the D3Q27 tests: rel-Linf <= 1e-5 after 10 steps, <= 1e-3 at the end of
long runs, integer geometry bit-exact, forces at the same tolerances.
"""
import numpy as np
import pytest

from paper_2510_13726_b200 import inputs as I
from test_parity_gpu import TOL10, TOL_LONG, _gpu_lattice, run_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def o19(oracle):
    return oracle.view(19)


@pytest.mark.parametrize("variant", [0, 2, 5])
def test_q19_config1_tgv32(o19, variant):
    """BASELINE.json config 1 recipe on D3Q19 (32^3: variant 5 falls back to 2)."""
    run_parity(o19, I.baseline_config(1), 10, variant, TOL10)


@pytest.mark.parametrize("variant", [0, 2, 5])
def test_q19_ragged_mirror_and_tiny(o19, variant):
    rho, u = I.noisy_uniform(45, 19, 23, (0.03, -0.02, 0.01), 5e-3, 77)
    run_parity(o19, I.Case("ragged", 45, 19, 23, 10, params=dict(I.DEFAULTS, tau0=0.53), rho=rho, u=u, with_neq=True),
               10, variant, TOL10)
    rho, u = I.noisy_uniform(20, 12, 9, (0.0, 0.0, 0.0), 1e-2, 9)
    run_parity(o19, I.Case("mirror", 20, 12, 9, 10, mode=(I.MIRROR, I.MIRROR, I.MIRROR),
                           params=dict(I.DEFAULTS, tau0=0.56), rho=rho, u=u, with_neq=True), 10, variant, TOL10)
    for ext in [(1, 1, 1), (5, 1, 1), (2, 2, 2)]:
        rho, u = I.noisy_uniform(*ext, (0.02, 0.01, -0.01), 2e-3, 5)
        run_parity(o19, I.Case("tiny", *ext, 5, params=dict(I.DEFAULTS, tau0=0.6), rho=rho, u=u), 5, variant, TOL10)


@pytest.mark.parametrize("ext", [(192, 16, 11), (384, 12, 11)])
def test_q19_xpull_tiles_and_seams(o19, ext):
    """The default kernel on D3Q19 with both tile shapes: periodic x seam, tile seams, z-chunks; then mirror y / z."""
    rho, u = I.noisy_uniform(*ext, (0.03, -0.02, 0.01), 5e-3, 78)
    case = I.Case("xpull", *ext, 10, params=dict(I.DEFAULTS, tau0=0.53), rho=rho, u=u, with_neq=True)
    G = _gpu_lattice(case, 5, q=19)
    assert G.population_storage() == 1 and G.q == 19 and G.populations().shape[0] == 19
    G.close()
    run_parity(o19, case, 10, 5, TOL10)
    import dataclasses
    run_parity(o19, dataclasses.replace(case, mode=(I.PERIODIC, I.MIRROR, I.MIRROR)), 10, 5, TOL10)


@pytest.mark.parametrize("variant", [0, 5])
def test_q19_config2_sphere_full_size(o19, variant):
    """BASELINE.json config 2 recipe on D3Q19: smoothed-porosity sphere, inflow fringe, force on the sphere; small
    for 10 steps, then 128 x 64 x 64 for its 200 steps."""
    run_parity(o19, I.case_sphere(128, 32, 32, 5.0, 10), 10, variant, TOL10, check_every=5)
    e = run_parity(o19, I.baseline_config(2), 200, variant, TOL_LONG, check_every=100, force_tol=TOL_LONG)
    print("D3Q19 config2 200 steps rel-Linf", e)


def test_q19_channel_and_rotor(o19):
    """Config 3 and config 4 recipes on D3Q19 at extents the default kernel tiles: wall model (sampling gathers 19
    populations per stencil cell), moving porosity, per-blade forces and torques, region split."""
    case = I.case_channel(128, 48, 16, 30)
    run_parity(o19, case, 10, 5, TOL10, check_every=1)
    run_parity(o19, case, 30, 5, TOL_LONG, check_every=15, force_tol=TOL_LONG)
    case = I.case_rotor(128, 72, 72, 20.0, 12, omega=0.012)
    run_parity(o19, case, 12, 5, TOL10, check_every=1)
    run_parity(o19, I.with_region_split(case), 12, 5, TOL10, check_every=4)
    run_parity(o19, I.case_rotor(96, 72, 72, 20.0, 6, omega=0.012), 6, 2, TOL10, check_every=2)


def test_q19_deterministic_and_bytes(o19):
    """Bitwise determinism of the D3Q19 default kernel; the library reports its velocity set."""
    from paper_2510_13726_b200 import binding as B
    assert B.lib(19).hhrr_velocity_set() == 19 and B.lib(27).hhrr_velocity_set() == 27
    case = I.case_rotor(128, 72, 72, 20.0, 6, omega=0.012)
    A, Bv = _gpu_lattice(case, 5, q=19), _gpu_lattice(case, 5, q=19)
    A.step(6); Bv.step(6)
    assert np.array_equal(A.populations(), Bv.populations())
    A.close(); Bv.close()
