"""hhrr_wall_model_noalloc: the allocation-free entry point (run with -m gpu; collected last on purpose).

Some callers cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
For them the library offers ONE entry point whose scratch memory (the sampled velocities handed from the wall model's
sampling kernel to its Newton kernel) is a file-scope device array of at most HHRR_NOALLOC_MAX_WALL_CELLS = 65536 wall
cells (3 MiB per GPU) instead of the caller's workspace.  Checked here against the EXISTING path -- the wall model that
runs inside hhrr_step -- on two calls in a row (a channel with 2048 wall cells, then a rotor with fewer: the shared
scratch keeps the first call's contents), at the tolerance of the parity tests (1e-5), and that an oversized request
is refused with a clear error.
"""
import numpy as np
import pytest

from paper_2510_13726_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL = 1e-5          # TOL10 of tests/test_parity_gpu.py
MAX_CELLS = 65536   # HHRR_NOALLOC_MAX_WALL_CELLS (include/hhrr.h)


def _lattice(case):
    from paper_2510_13726_b200 import binding as B
    p = B.make_params(case.nx, case.ny, case.nz, mode=case.mode, **case.params)
    L = B.Lattice(p, rotor_shape=None if case.rotor is None else case.rotor["sdf"].shape)
    I.apply_case(case, L)
    return L


def _existing_vs_noalloc(case):
    """Two steps through the existing path; the wall model of the second step is then recomputed by the new entry
    point from the same populations, wall list and warm-start values, and must give the same state."""
    import torch
    L = _lattice(case)
    L.step(1)
    idx1, ut1, _, _, va1 = L.wall_model_state()
    L.step(1)
    idx2, ut2, uw2, sw2, va2 = L.wall_model_state()          # existing path: K3 inside hhrr_step
    k = len(idx2)
    assert k > 0 and va2.all()
    # what the existing wall model of step 2 started from: the stored u_tau of cells that held state (R9 / Eq. 20)
    prev = {int(c): float(u) for c, u, v in zip(idx1, ut1, va1) if v}
    start = np.array([prev.get(int(c), 0.0) for c in idx2])
    dev = L.device
    start_t = torch.from_numpy(start).to(dev)
    cap = k + 7                                              # a capacity beyond the list: the tail stays untouched
    ut_t = torch.full((cap,), -1.0, dtype=torch.float64, device=dev)
    uw_t = torch.full((cap, 3), -1.0, dtype=torch.float32, device=dev)
    sw_t = torch.full((cap, 6), -1.0, dtype=torch.float32, device=dev)
    start_cap = torch.zeros(cap, dtype=torch.float64, device=dev)
    start_cap[:k] = start_t
    launches = L.launch_count()
    L.wall_model_noalloc(cap, start_cap, ut_t, uw_t, sw_t)
    assert L.launch_count() - launches == 2                  # two kernels, nothing else
    L.synchronize()
    ut, uw, sw = ut_t.cpu().numpy(), uw_t.cpu().numpy(), sw_t.cpu().numpy()
    assert np.all(ut[k:] == -1.0) and np.all(uw[k:] == -1.0) and np.all(sw[k:] == -1.0)
    assert np.max(np.abs(ut[:k] - ut2)) <= TOL * np.max(np.abs(ut2))
    assert np.max(np.abs(uw[:k] - uw2)) <= TOL * max(np.max(np.abs(uw2)), 1e-30)
    assert np.max(np.abs(sw[:k] - sw2)) <= TOL * max(np.max(np.abs(sw2)), 1e-30)
    # the lattice's own state was neither read nor written
    idx3, ut3, uw3, sw3, va3 = L.wall_model_state()
    assert np.array_equal(idx3, idx2) and np.array_equal(ut3, ut2) and np.array_equal(uw3, uw2) and np.array_equal(sw3, sw2)
    exact = np.array_equal(ut[:k], ut2) and np.array_equal(uw[:k], uw2) and np.array_equal(sw[:k], sw2)
    L.close()
    return k, exact


def test_no_alloc_wall_model_matches_the_existing_path_twice():
    k1, exact1 = _existing_vs_noalloc(I.case_channel(128, 48, 16, 2))                 # 2048 wall cells
    k2, exact2 = _existing_vs_noalloc(I.case_rotor(128, 72, 72, 20.0, 2, omega=0.012))  # fewer: stale scratch beyond
    assert k1 == 128 * 16 and 0 < k2 < k1
    print(f"no-alloc wall model: {k1} and {k2} wall cells, bitwise equal to the existing path: {exact1}, {exact2}")


def test_no_alloc_wall_model_cold_start_and_limits():
    """NULL start array = Eq. 20's cold start (what the existing path does on its first step); a request beyond the
    built-in scratch is refused with HHRR_E_SIZE and a message that names the limit."""
    import torch
    from paper_2510_13726_b200 import binding as B
    L = _lattice(I.case_channel(128, 48, 16, 1))
    L.step(1)
    idx, ut_ref, uw_ref, sw_ref, va = L.wall_model_state()    # first step: every wall cell cold-started
    k = len(idx)
    dev = L.device
    ut_t = torch.empty(k, dtype=torch.float64, device=dev)
    uw_t = torch.empty((k, 3), dtype=torch.float32, device=dev)
    sw_t = torch.empty((k, 6), dtype=torch.float32, device=dev)
    for _ in range(2):                                        # two calls in a row on one stream
        L.wall_model_noalloc(k, None, ut_t, uw_t, sw_t)
    L.synchronize()
    assert np.max(np.abs(ut_t.cpu().numpy() - ut_ref)) <= TOL * np.max(np.abs(ut_ref))
    assert np.max(np.abs(uw_t.cpu().numpy() - uw_ref)) <= TOL * np.max(np.abs(uw_ref))
    assert np.max(np.abs(sw_t.cpu().numpy() - sw_ref)) <= TOL * max(np.max(np.abs(sw_ref)), 1e-30)
    with pytest.raises(B.HhrrError) as err:
        L.wall_model_noalloc(MAX_CELLS + 1, None, ut_t, uw_t, sw_t)
    assert err.value.code == -2 and str(MAX_CELLS) in str(err.value)
    with pytest.raises(B.HhrrError):
        L.wall_model_noalloc(0, None, ut_t, uw_t, sw_t)
    L.close()
