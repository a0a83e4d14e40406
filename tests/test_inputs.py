"""Host logic of the seeded input recipes (CPU only): the FSI boxes of with_region_split cover the structure."""
import numpy as np
import pytest

from paper_2510_13726_b200 import inputs as I


@pytest.mark.parametrize("make", [
    lambda: I.case_rotor(96, 72, 72, 20.0, 30, omega=0.05),
    lambda: I.case_sphere(64, 32, 32, 5.0, 2),
    lambda: I.case_channel(32, 24, 8, 2),
])
def test_region_split_boxes_cover_everything_that_is_not_plain_fluid(oracle, make):
    """the bulk model may only run where no wall-modelled structure can be.  Over a quarter turn of
    the rotor (0.05 rad per step) no solid, frontier, growth or fringe cell ever lies outside the boxes (the
    oracle reports it if one does), and a sizeable part of the lattice is bulk."""
    case = I.with_region_split(make())
    assert case.fsi_boxes and all(b[0] < b[1] and b[2] < b[3] and b[4] < b[5] for b in case.fsi_boxes)
    L = oracle.Lattice(oracle.make_params(case.nx, case.ny, case.nz, mode=case.mode, **case.params))
    I.apply_case(case, L)
    for _ in range(case.steps):
        L.update_geometry()
        assert not L.region_violation()
        L.step(1)
    types = L.cell_types()[0]
    z, y, x = np.meshgrid(np.arange(case.nz), np.arange(case.ny), np.arange(case.nx), indexing="ij")
    inside = np.zeros(case.n, bool)
    for (x0, x1, y0, y1, z0, z1) in case.fsi_boxes:
        inside |= ((x >= x0) & (x < x1) & (y >= y0) & (y < y1) & (z >= z0) & (z < z1)).reshape(-1)
    assert np.all(types[~inside] == 5) and np.all(types[inside] != 5)
    if case.rotor is not None:
        assert np.count_nonzero(types == 5) > 0.2 * case.n
    L.close()
