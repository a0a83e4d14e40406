"""Seeded random sequences of API calls on a small rotor lattice, the CUDA library and the oracle side by side (-m gpu).

The step schedule of the library keeps state between calls -- the geometry written ahead into the alternate set, the
wall-model state and its valid bits, the storage form of the populations, the force ring -- and every setter has to
leave that state consistent.  The parity tests walk the paths one at a time; here they are mixed: steps of varying
length, geometry evaluations between steps, the look-ahead switched off and on, the three kernel variants, other
z-chunk lengths and cluster sizes, the wall model switched off and on, a replaced rotor (other speed, sense and phase),
the bulk / FSI region split set and cleared, and a checkpoint restored into a fresh lattice.  After every block of
steps: cell types, tags, wall list and valid bits bit-exact, porosity, u_tau, flow and the forces of those steps at the
parity tolerance (the sequence is at most 40 steps long).
"""
import dataclasses

import numpy as np
import pytest

from paper_2510_13726_b200 import inputs as I
from test_parity_gpu import _gpu_lattice, _ora_lattice, compare_geometry, rel_linf

pytestmark = pytest.mark.gpu

TOL = 2e-5      # TOL10 = 1e-5 holds at 10 steps; these runs are up to 40 steps long


def _fresh_gpu(case, settings, q):
    """A new CUDA lattice in the state `settings` describes (what a restart would set up before loading a checkpoint)."""
    c = dataclasses.replace(case, rotor=settings["rotor"], wall_model=settings["wm"], fsi_boxes=settings["boxes"])
    G = _gpu_lattice(c, settings["variant"], q=q)
    G.set_lookahead(settings["lookahead"])
    G.set_launch_shape(*settings["shape"])
    return G


@pytest.mark.parametrize("q,seed", [(27, s) for s in range(11, 19)] + [(19, 21), (19, 22)])
def test_random_api_sequence_matches_the_oracle(oracle, q, seed):
    """q = 19: the D3Q19 library (libhhrr_q19.so) against the D3Q19 oracle."""
    if q == 19:
        oracle = oracle.view(19)
    rng = np.random.default_rng(seed)
    case = I.case_rotor(128, 48, 48, 12.0, 40, omega=0.02)
    split_boxes = I.with_region_split(case).fsi_boxes
    settings = dict(rotor=case.rotor, wm=True, boxes=None, variant=5, lookahead=True, shape=(0, 0))
    G, Oa = _gpu_lattice(case, 5, q=q), _ora_lattice(oracle, case)
    ops = ["step"] * 5 + ["update_geometry", "lookahead", "variant", "shape", "wm", "rotor", "region", "checkpoint"]
    done, log, worst = 0, [], 0.0
    while done < 40:
        op = ops[rng.integers(len(ops))]
        if op == "step":
            k = int(min(rng.choice([1, 1, 2, 3, 5]), 40 - done))
            G.step(k); Oa.step(k)
            done += k
            log.append(f"step({k})")
            try:
                compare_geometry(G, Oa, TOL)
            except AssertionError as e:
                raise AssertionError(f"{e} after: " + " ".join(log)) from None
            e_rho, e_v = rel_linf(*G.moments(), *Oa.moments())
            worst = max(worst, e_rho, e_v)
            assert e_rho <= TOL and e_v <= TOL, (e_rho, e_v, log)
            Fg, Fo = G.forces(done - k, k), Oa.forces(done - k, k)
            assert np.max(np.abs(Fg - Fo)) <= TOL * max(np.max(np.abs(Fo)), 1e-30), log
            Mg, Mo = G.torques(done - k, k), Oa.torques(done - k, k)
            assert np.max(np.abs(Mg - Mo)) <= TOL * max(np.max(np.abs(Mo)), 1e-30), log
        elif op == "update_geometry":
            G.update_geometry(); Oa.update_geometry()
            log.append(op)
            try:
                compare_geometry(G, Oa, TOL)
            except AssertionError as e:
                raise AssertionError(f"{e} after: " + " ".join(log)) from None
        elif op == "lookahead":
            settings["lookahead"] = bool(rng.integers(2))
            G.set_lookahead(settings["lookahead"])
            log.append(f"lookahead({settings['lookahead']})")
        elif op == "variant":
            settings["variant"] = int(rng.choice([0, 2, 5]))
            G.set_kernel_variant(settings["variant"])
            log.append(f"variant({settings['variant']})")
        elif op == "shape":
            settings["shape"] = (int(rng.choice([0, 5, 9, 16, 48])), int(rng.choice([0, 1, 2])))
            G.set_launch_shape(*settings["shape"])
            log.append(f"shape{settings['shape']}")
        elif op == "wm":
            settings["wm"] = bool(rng.integers(2))
            G.enable_wall_model(settings["wm"]); Oa.enable_wall_model(settings["wm"])
            log.append(f"wm({settings['wm']})")
        elif op == "rotor":
            settings["rotor"] = dict(case.rotor, omega=float(rng.uniform(-0.03, 0.03)), theta0=float(rng.uniform(0, 6.28)))
            G.set_rotor(**settings["rotor"]); Oa.set_rotor(**settings["rotor"])
            log.append("rotor(omega=%.3f)" % settings["rotor"]["omega"])
        elif op == "region":
            settings["boxes"] = None if settings["boxes"] else split_boxes
            G.set_fsi_region(settings["boxes"] or []); Oa.set_fsi_region(settings["boxes"] or [])
            log.append("region(%s)" % ("on" if settings["boxes"] else "off"))
        elif op == "checkpoint" and done > 0:
            # hhrr_set_wall_model_state evaluates the geometry of the step to come (include/hhrr.h): a checkpoint is
            # taken of an evaluated state, on both sides -- a setter since the last step may have left it pending
            G.update_geometry(); Oa.update_geometry()
            f, state, n = G.populations(), G.wall_model_state(), G.step_count()
            G.close()
            G = _fresh_gpu(case, settings, q)
            G.set_step_count(n); G.set_populations(f); G.set_wall_model_state(*state)
            log.append("checkpoint")
    G.check_finite()
    print(f"D3Q{q} seed {seed}: {len(log)} calls, worst rel-Linf {worst:.2e}: " + " ".join(log))
    G.close(); Oa.close()


@pytest.mark.parametrize("shape,seed", [((128, 24, 16), 31), ((128, 24, 16), 32), ((48, 20, 12), 33)])
def test_random_api_sequence_static_geometry(oracle, shape, seed):
    """The same on STATIC geometry: a wall with its wall-model layer (channel recipe, y MIRROR on top) and a ball whose
    position, velocity and tag change between steps; the wall function (Spalding / Musker) and the second readings of
    the wall model switched; the inflow fringe moved; wall model off and on.  128 x 24 x 16 runs the default kernel,
    48 x 20 x 12 cannot be tiled by it (variant 2 runs on post-stream storage)."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = shape
    base = I.case_channel(nx, ny, nz, 30)
    wall = np.asarray(base.phi, np.float64)

    def geometry(centre, r):
        ball = np.asarray(I.sphere_phi(nx, ny, nz, centre, r), np.float64)
        phi = np.minimum(wall, ball).astype(np.float32)
        tag = np.where(ball < wall, 2, 1).astype(np.uint8)
        return phi, tag

    G, Oa = _gpu_lattice(base, 5), _ora_lattice(oracle, base)
    ops = ["step"] * 5 + ["update_geometry", "variant", "lookahead", "ball", "body", "wall_function", "readings", "fringe", "wm"]
    done, log, worst = 0, [], 0.0
    while done < 30:
        op = ops[rng.integers(len(ops))]
        if op == "step":
            k = int(min(rng.choice([1, 1, 2, 3, 5]), 30 - done))
            G.step(k); Oa.step(k)
            done += k
            log.append(f"step({k})")
            try:
                compare_geometry(G, Oa, TOL)
            except AssertionError as e:
                raise AssertionError(f"{e} after: " + " ".join(log)) from None
            e_rho, e_v = rel_linf(*G.moments(), *Oa.moments())
            worst = max(worst, e_rho, e_v)
            assert e_rho <= TOL and e_v <= TOL, (e_rho, e_v, log)
            Fg, Fo = G.forces(done - k, k), Oa.forces(done - k, k)
            assert np.max(np.abs(Fg - Fo)) <= TOL * max(np.max(np.abs(Fo)), 1e-30), log
            Mg, Mo = G.torques(done - k, k), Oa.torques(done - k, k)
            assert np.max(np.abs(Mg - Mo)) <= TOL * max(np.max(np.abs(Mo)), 1e-30), log
        elif op == "update_geometry":
            G.update_geometry(); Oa.update_geometry()
            log.append(op)
            try:
                compare_geometry(G, Oa, TOL)
            except AssertionError as e:
                raise AssertionError(f"{e} after: " + " ".join(log)) from None
        elif op == "variant":
            v = int(rng.choice([0, 2, 5]))
            G.set_kernel_variant(v)
            log.append(f"variant({v})")
        elif op == "lookahead":
            b = bool(rng.integers(2))
            G.set_lookahead(b)
            log.append(f"lookahead({b})")
        elif op == "ball":
            c = (float(rng.uniform(0, nx)), float(rng.uniform(5, ny - 4)), float(rng.uniform(0, nz)))
            phi, tag = geometry(c, float(rng.uniform(2.0, 3.5)))
            for L in (G, Oa):
                L.set_static_geometry(phi, tag, None)
            log.append("ball(%.1f,%.1f,%.1f)" % c)
        elif op == "body":
            c = (float(rng.uniform(0, nx)), float(rng.uniform(0, ny)), float(rng.uniform(0, nz)))
            w = tuple(float(x) for x in rng.uniform(-0.004, 0.004, 3))
            v = tuple(float(x) for x in rng.uniform(-0.02, 0.02, 3))
            for L in (G, Oa):
                L.set_body(2, c, w, v)
            log.append("body")
        elif op == "wall_function":
            k = int(rng.integers(2))
            G.set_wall_function(k); Oa.set_wall_function(k)
            log.append(f"wall_function({k})")
        elif op == "readings":
            sl, sh = int(rng.integers(2)), int(rng.integers(2))
            G.set_wall_model_variant(sl, sh); Oa.set_wall_model_variant(sl, sh)
            log.append(f"readings({sl},{sh})")
        elif op == "fringe":
            x0 = int(rng.integers(0, nx - 4))
            u_in = (float(rng.uniform(0.02, 0.06)), 0.0, 0.0)
            G.set_fringe(x0, x0 + 3, u_in); Oa.set_fringe(x0, x0 + 3, u_in)
            log.append(f"fringe({x0})")
        elif op == "wm":
            b = bool(rng.integers(2))
            G.enable_wall_model(b); Oa.enable_wall_model(b)
            log.append(f"wm({b})")
    G.check_finite()
    print(f"static {shape} seed {seed}: {len(log)} calls, worst rel-Linf {worst:.2e}: " + " ".join(log))
    G.close(); Oa.close()
