"""Slab decomposition on the GPU (run with -m gpu): hhrr_halo_pack / hhrr_halo_unpack and slabs.SlabLattice.

One process, one GPU: two slabs of a lattice are stepped in turn with the halo exchange after every step and must
reproduce the undecomposed lattice BIT FOR BIT (every cell runs the same arithmetic on the same inputs), forces and
torques summed over the slabs.  Two processes on two GPUs (NCCL send / recv): the same, skipped with fewer than two
devices."""
import os
import socket

import numpy as np
import pytest

from paper_2510_13726_b200 import inputs as I
from paper_2510_13726_b200 import slabs as S

pytestmark = pytest.mark.gpu

NX, NY, NZ = 128, 32, 40


def _global_case():
    rho, u = I.noisy_uniform(NX, NY, NZ, (0.03, -0.01, 0.02), 5e-3, 23)
    phi = I.sphere_phi(NX, NY, NZ, (40.0, 15.5, 9.5), 4.0)
    return dict(rho=rho, u=u, phi=phi, params=dict(I.DEFAULTS, tau0=0.5 + 3 * 3.156e-4))


def _lattice(q, nz, rho, u, phi, params, device="cuda:0"):
    from paper_2510_13726_b200 import binding as B
    L = B.Lattice(B.make_params(NX, NY, nz, **params), q=q, device=device)
    L.set_static_geometry(phi, np.ones(phi.size, np.uint8), None)
    L.set_fringe(0, 4, (0.03, 0.0, 0.0))
    L.enable_wall_model(True)
    L.init_equilibrium(rho, u, False)
    assert L.population_storage() == 1
    return L


def _slab(q, g, rank, world, device="cuda:0", group=None):
    f = lambda a: S.slab_field(np.asarray(a), NZ, NY, NX, rank, world)
    z0, z1 = S.slab_range(NZ, rank, world)
    L = _lattice(q, z1 - z0 + 2, f(g["rho"]), f(g["u"]), f(g["phi"]), g["params"], device)
    return S.SlabLattice(L, rank, world, group)


@pytest.mark.parametrize("q", [27, 19])
def test_two_slabs_on_one_gpu_equal_the_single_lattice(q):
    g = _global_case()
    G = _lattice(q, NZ, g["rho"], g["u"], g["phi"], g["params"])
    slabs = [_slab(q, g, r, 2) for r in range(2)]
    steps = 8
    G.step(steps)
    S.step_in_process(slabs, steps)
    fg = G.populations().reshape(q, NZ, NY, NX)
    for s in slabs:
        z0, z1 = S.slab_range(NZ, s.rank, 2)
        f = s.L.populations().reshape(q, z1 - z0 + 2, NY, NX)[:, 1:-1]
        assert np.array_equal(f, fg[:, z0:z1]), np.max(np.abs(f - fg[:, z0:z1]))
    F = sum(s.L.forces() for s in slabs)
    M = sum(s.L.torques() for s in slabs)
    assert np.max(np.abs(G.forces()[-1, 1])) > 1e-4
    assert np.allclose(F, G.forces(), rtol=1e-10, atol=1e-16)
    assert np.allclose(M[:, :, 2], G.torques()[:, :, 2], rtol=1e-9, atol=1e-13)   # body centre (0,0,0): z lever differs per slab
    assert len(slabs[0].L.wall_list()[0]) == len(G.wall_list()[0]) > 0 and len(slabs[1].L.wall_list()[0]) == 0
    for L in [G] + [s.L for s in slabs]:
        L.close()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q, steps, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device(f"cuda:{rank}"))
    s = _slab(q, _global_case(), rank, world, device=f"cuda:{rank}", group=dist.group.WORLD)
    s.step(steps)
    z0, z1 = S.slab_range(NZ, rank, world)
    out[rank] = (s.L.populations().reshape(q, z1 - z0 + 2, NY, NX)[:, 1:-1].copy(), s.total_forces())
    s.L.close()
    dist.destroy_process_group()


def test_two_slabs_on_two_gpus_equal_the_single_lattice():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    import torch.multiprocessing as mp
    q, steps, world = 27, 8, 2
    g = _global_case()
    G = _lattice(q, NZ, g["rho"], g["u"], g["phi"], g["params"])
    G.step(steps)
    fg = G.populations().reshape(q, NZ, NY, NX)
    Fg = G.forces()
    G.close()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), q, steps, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        z0, z1 = S.slab_range(NZ, rank, world)
        assert np.array_equal(res[rank][0], fg[:, z0:z1])
        assert np.allclose(res[rank][1], Fg, rtol=1e-10, atol=1e-16)
