"""Slab decomposition, host side (CPU): the halo plan of paper_2510_13726_b200/slabs.py drives TWO oracle lattices in
two gloo ranks; after every step the decomposed state must equal the undecomposed oracle lattice (the
decomposed run must equal the single-lattice oracle; nothing new on the oracle side)."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

NX, NY, NZ, STEPS = 8, 6, 20, 6


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _global_case(q):
    """Noisy flow with a body force, an inflow fringe crossing the slab faces and a small ball inside slab 0."""
    from paper_2510_13726_b200 import inputs as I
    rho, u = I.noisy_uniform(NX, NY, NZ, (0.03, -0.01, 0.02), 5e-3, 17)
    phi = I.sphere_phi(NX, NY, NZ, (4.0, 2.5, 4.5), 1.5)
    params = dict(tau0=0.56, sigma=0.6, smagorinsky_cs=0.1, body_force=(1e-5, 0.0, -2e-5))
    return rho.astype(np.float64), u.astype(np.float64), phi.astype(np.float64), params


def _make(O, nz, rho, u, phi, params):
    L = O.Lattice(O.make_params(NX, NY, nz, **params))
    L.set_static_geometry(phi, np.ones(phi.size, np.uint8))
    L.set_fringe(0, 2, (0.03, 0.0, 0.0))
    L.init_equilibrium(rho, u, False)
    return L


def _worker(rank, world, port, q, out):
    import torch
    import torch.distributed as dist
    from oracle import oracle as Om
    from paper_2510_13726_b200 import slabs as S
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    O = Om if q == 27 else Om.view(q)
    rho, u, phi, params = _global_case(q)
    z0, z1 = S.slab_range(NZ, rank, world)
    nz = z1 - z0 + 2
    L = _make(O, nz, S.slab_field(rho, NZ, NY, NX, rank, world), S.slab_field(u, NZ, NY, NX, rank, world),
              S.slab_field(phi, NZ, NY, NX, rank, world), params)
    lo, hi = (rank - 1) % world, (rank + 1) % world
    for _ in range(STEPS):
        L.step(1)
        f = L.populations().reshape(q, nz, NY, NX)
        send = [torch.from_numpy(S.pack_numpy(f, 0)), torch.from_numpy(S.pack_numpy(f, 1))]
        recv = [torch.empty_like(send[0]), torch.empty_like(send[1])]
        # messages between one pair of ranks are matched in order (see slabs.SlabLattice.transfer)
        ops = [dist.P2POp(dist.isend, send[0], lo), dist.P2POp(dist.isend, send[1], hi),
               dist.P2POp(dist.irecv, recv[1], hi), dist.P2POp(dist.irecv, recv[0], lo)]
        for w in dist.batch_isend_irecv(ops):
            w.wait()
        S.unpack_numpy(f, 0, recv[0].numpy())
        S.unpack_numpy(f, 1, recv[1].numpy())
        L.set_populations(f.reshape(q, -1))
    F = torch.from_numpy(L.forces().copy())
    dist.all_reduce(F)                                   # per-element forces: sum over the slabs
    out[rank] = (z0, z1, L.populations().reshape(q, nz, NY, NX)[:, 1:-1].copy(), F.numpy())
    dist.destroy_process_group()


@pytest.mark.parametrize("q", [27, 19])
def test_two_slabs_equal_the_single_lattice(oracle, q):
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, q, out), nprocs=world, join=True)
        res = dict(out)
    O = oracle if q == 27 else oracle.view(q)
    rho, u, phi, params = _global_case(q)
    G = _make(O, NZ, rho, u, phi, params)
    G.step(STEPS)
    fg = G.populations().reshape(q, NZ, NY, NX)
    for rank in range(world):
        z0, z1, f, F = res[rank]
        assert (z0, z1) == ((0, 10), (10, 20))[rank]
        assert np.max(np.abs(f - fg[:, z0:z1])) <= 1e-15
        assert np.allclose(F, G.forces(), rtol=1e-12, atol=1e-18)
    assert np.max(np.abs(G.forces()[-1, 1])) > 1e-4


def test_halo_plan_covers_every_population_once():
    """Per face the buffer carries Q planes: the outward movers of the halo plane, and from the last real plane every
    population the receiver's own collision has not already put into its halo plane (c_z = 0 and the outward ones)."""
    from paper_2510_13726_b200 import slabs as S
    for q in (27, 19):
        dirs = S.directions(q)
        for face in (0, 1):
            c = 1 if face else -1
            plan = S.halo_plan(q, face)
            assert len(plan) == q
            halo = sorted(p for p, k in plan if k == "halo")
            real = sorted(p for p, k in plan if k == "real")
            assert halo == [i for i, d in enumerate(dirs) if d[2] == c]
            assert real == sorted([i for i, d in enumerate(dirs) if d[2] == 0] + [i for i, d in enumerate(dirs) if d[2] == c])
    assert S.slab_range(364, 3, 8) == (138, 184) and sum(b - a for a, b in (S.slab_range(364, r, 8) for r in range(8))) == 364
