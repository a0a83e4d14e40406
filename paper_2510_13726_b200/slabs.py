"""Slab decomposition along z with halo exchange.

The paper's multi-GPU runs give every GPU one block of the lattice (Fig. 13 :421-423: one turbine per
GPU, 384 GPUs).  Here a rank holds `nz_real` planes of the global lattice plus one HALO plane at either end on a
z-periodic local lattice; after every collide-stream step it exchanges, per face, Q planes of populations with its
neighbour (include/hhrr.h "Slab decomposition"):

    slot i of the buffer, c = c_z of the populations crossing the face:
      c_z(i) ==  c : population i of the sender's HALO plane      -> population i of the receiver's first REAL plane
      c_z(i) ==  0 : population i of the sender's last REAL plane -> population i of the receiver's HALO plane
      c_z(i) == -c : population j (= i with c_z reversed) of the sender's last REAL plane -> population j, HALO plane

`halo_plan` is that table as data; `pack_numpy` / `unpack_numpy` apply it to host arrays (the two-rank gloo test
drives two oracle lattices with it and compares with the undecomposed oracle lattice); `SlabLattice` applies it on the
GPU through hhrr_halo_pack / hhrr_halo_unpack and moves the buffers with torch.distributed (NCCL send / recv over
NVLink, one message per face and direction) or, inside one process, with device copies.  The per-element forces of all
ranks are combined with one all-reduce of n_steps x 16 x 3 doubles ("global reductions").

No arithmetic of the method lives here: only which plane of which population goes where.
"""
from __future__ import annotations

import numpy as np


def directions(q: int):
    """(cx, cy, cz) of the velocity set in the library's order (include/hhrr.h): D3Q27, or its |c|^2 <= 2 subset."""
    out = []
    for k in range(27):
        c = (k % 3 - 1, (k // 3) % 3 - 1, k // 9 - 1)
        if q == 19 and abs(c[0]) + abs(c[1]) + abs(c[2]) == 3:
            continue
        out.append(c)
    assert len(out) == q
    return out


def halo_plan(q: int, face: int):
    """For the SENDER's face (0 = low z, 1 = high z): list over buffer slots i of (population, 'halo' | 'real') to
    read; the receiver writes slot i to (population, 'real' | 'halo') -- the same population, the other kind of plane."""
    dirs = directions(q)
    c = 1 if face else -1
    plan = []
    for i, (cx, cy, cz) in enumerate(dirs):
        if cz == c:
            plan.append((i, "halo"))
        elif cz == 0:
            plan.append((i, "real"))
        else:
            plan.append((dirs.index((cx, cy, -cz)), "real"))
    return plan


def pack_numpy(f: np.ndarray, face: int) -> np.ndarray:
    """f: [q, nz, ny, nx] populations of a slab (planes 0 and nz-1 are halo planes).  Returns the buffer [q, ny, nx]."""
    q, nz = f.shape[0], f.shape[1]
    z = {"halo": nz - 1 if face else 0, "real": nz - 2 if face else 1}
    return np.stack([f[pop, z[kind]] for pop, kind in halo_plan(q, face)])


def unpack_numpy(f: np.ndarray, face: int, buf: np.ndarray) -> None:
    """Writes a buffer that arrived through `face` of this slab (packed by the neighbour with the opposite face)."""
    q, nz = f.shape[0], f.shape[1]
    z = {"halo": nz - 1 if face else 0, "real": nz - 2 if face else 1}
    other = {"halo": "real", "real": "halo"}
    for slot, (pop, kind) in enumerate(halo_plan(q, 1 - face)):
        f[pop, z[other[kind]]] = buf[slot]


def slab_range(nz_global: int, rank: int, world: int):
    """Real planes [z0, z1) of the global lattice owned by `rank` (contiguous, as even as possible)."""
    base, rem = divmod(nz_global, world)
    z0 = rank * base + min(rank, rem)
    return z0, z0 + base + (1 if rank < rem else 0)


def slab_field(a: np.ndarray, nz_global: int, ny: int, nx: int, rank: int, world: int) -> np.ndarray:
    """Slices a global per-cell array [..., nz*ny*nx] into the slab's [..., (nz_real+2)*ny*nx] with periodic halo planes."""
    z0, z1 = slab_range(nz_global, rank, world)
    g = a.reshape(a.shape[:-1] + (nz_global, ny, nx))
    idx = np.arange(z0 - 1, z1 + 1) % nz_global
    return np.ascontiguousarray(np.take(g, idx, axis=-3)).reshape(a.shape[:-1] + (-1,))


class SlabLattice:
    """One rank's slab on its GPU: a binding.Lattice of nz_real + 2 planes and the halo exchange after every step.

    group=None: single process; `neighbours` = (lower SlabLattice, upper SlabLattice) on the same or another device,
    the buffers are handed over with device copies (tests on one GPU; the caller steps the slabs in turn).
    group=a torch.distributed group: ranks lo / hi are the periodic neighbours along z."""

    def __init__(self, lattice, rank=0, world=1, group=None):
        import torch
        self.L, self.rank, self.world, self.group = lattice, rank, world, group
        n = lattice.halo_floats()
        dev = lattice.device
        self.send = [torch.empty(n, dtype=torch.float32, device=dev) for _ in range(2)]
        self.recv = [torch.empty(n, dtype=torch.float32, device=dev) for _ in range(2)]
        self.neighbours = None

    @property
    def lo(self):
        return (self.rank - 1) % self.world

    @property
    def hi(self):
        return (self.rank + 1) % self.world

    def pack(self):
        self.L.halo_pack(0, self.send[0])
        self.L.halo_pack(1, self.send[1])

    def transfer(self):
        """Moves send[face] to the neighbour's recv[1 - face]."""
        import torch
        if self.group is None:
            lower, upper = self.neighbours
            with torch.cuda.stream(self.L.stream):
                lower.recv[1].copy_(self.send[0], non_blocking=True)
                upper.recv[0].copy_(self.send[1], non_blocking=True)
            return
        import torch.distributed as dist
        if self.world == 1 or self.group == "self":   # periodic in z onto itself
            with torch.cuda.stream(self.L.stream):
                self.recv[1].copy_(self.send[0], non_blocking=True)
                self.recv[0].copy_(self.send[1], non_blocking=True)
            return
        with torch.cuda.stream(self.L.stream):
            # Messages between one pair of ranks are matched in order: with two ranks (both neighbours are the same
            # rank) the low-face message goes out first and is received first, into the peer's high-face buffer.
            ops = [dist.P2POp(dist.isend, self.send[0], self.lo, group=self.group),
                   dist.P2POp(dist.isend, self.send[1], self.hi, group=self.group),
                   dist.P2POp(dist.irecv, self.recv[1], self.hi, group=self.group),
                   dist.P2POp(dist.irecv, self.recv[0], self.lo, group=self.group)]
            for w in dist.batch_isend_irecv(ops):
                w.wait()

    def unpack(self):
        self.L.halo_unpack(0, self.recv[0])
        self.L.halo_unpack(1, self.recv[1])

    def step(self, n=1):
        """n time steps with the halo exchange after each (distributed use; in-process slabs are stepped by the caller
        in turn: pack all, transfer all, unpack all)."""
        for _ in range(n):
            self.L.step(1)
            self.pack()
            self.transfer()
            self.unpack()

    def total_forces(self, first=0, count=None):
        """Per-element forces summed over all ranks: one all-reduce of count x 16 x 3 doubles."""
        import torch
        F = self.L.forces(first, count)
        if self.group is None or self.group == "self" or self.world == 1:
            return F
        import torch.distributed as dist
        t = torch.from_numpy(F).to(self.L.device)
        dist.all_reduce(t, group=self.group)
        return t.cpu().numpy()


def step_in_process(slabs, n=1):
    """Steps slabs that live in ONE process (one after the other on the device) with the exchange after every step."""
    k = len(slabs)
    for i, s in enumerate(slabs):
        s.neighbours = (slabs[(i - 1) % k], slabs[(i + 1) % k])
    for _ in range(n):
        for s in slabs:
            s.L.step(1)
        for s in slabs:
            s.pack()
        for s in slabs:
            s.L.synchronize()
        for s in slabs:
            s.transfer()
        for s in slabs:
            s.L.synchronize()
        for s in slabs:
            s.unpack()
