"""Domain decomposition of a single-type mesh over ranks (section 3.6, Tables 6-7 :697-717): element
partition, ghost layers and the exchange tables of the per-stage halo update.  Host-side index bookkeeping only -- no
arithmetic of the method; the right-hand side of every rank runs in the library's kernels on the rank's sub-mesh.

Design: every rank owns a contiguous slab of elements and carries the elements within `hops` = 2
face-neighbour steps of its slab as ghosts.  The Navier-Stokes right-hand side of an element depends on its neighbours'
neighbours (compact LDG stencil with beta = +-1/2: common solution from one side, viscous flux from the other), so with the
ghost STATES up to date the right-hand side of every owned element on the sub-mesh equals the one on the whole mesh; the
faces where the ghost layer is cut get a dummy boundary condition whose influence stops inside the ghost layer.  One halo
exchange of state columns per right-hand side (point-to-point, no reduction) replaces the paper's two exchanges of
flux-point rows; the ghost elements are recomputed redundantly.

    plan = decompose(mesh, world_size)            # on every rank, deterministic
    sub  = plan.sub_mesh(rank)                     # mesh dictionary for fr_setup_mesh (cut faces: bc_id = plan.cut_bc)
    plan.send[rank][peer] / plan.recv[rank][peer]  # local element indices to pack for / unpack from `peer`
"""
import numpy as np


class Plan:
    def __init__(self, mesh, owner, hops, cut_bc):
        self.mesh, self.owner, self.hops, self.cut_bc = mesh, owner, hops, cut_bc
        self.world = int(owner.max()) + 1
        n_el = mesh["nodes"].shape[0]
        ifc = mesh["ifaces"]
        self.local = []   # global element ids of every rank's sub-mesh: owned first (ascending), then ghosts (ascending)
        self.n_owned = []
        for r in range(self.world):
            inside = owner == r
            owned = np.flatnonzero(inside)
            reach = inside.copy()
            for _ in range(hops):
                touch = reach[ifc[:, 0]] | reach[ifc[:, 2]]
                reach[ifc[touch, 0]] = True
                reach[ifc[touch, 2]] = True
            ghosts = np.flatnonzero(reach & ~inside)
            self.local.append(np.concatenate([owned, ghosts]))
            self.n_owned.append(owned.size)
        # exchange tables: rank r receives its ghost g from owner[g]; the owner sends its local index of g
        self.send = [dict() for _ in range(self.world)]
        self.recv = [dict() for _ in range(self.world)]
        pos = []
        for r in range(self.world):
            p = -np.ones(n_el, dtype=np.int64)
            p[self.local[r]] = np.arange(self.local[r].size)
            pos.append(p)
        for r in range(self.world):
            ghosts = self.local[r][self.n_owned[r]:]
            for peer in np.unique(owner[ghosts]):
                g = ghosts[owner[ghosts] == peer]          # ascending global ids: the same order on both sides
                self.recv[r][int(peer)] = pos[r][g]
                self.send[int(peer)][r] = pos[int(peer)][g]

    def sub_mesh(self, rank):
        """The rank's elements (owned + ghosts) as a mesh dictionary; interfaces with both sides present are kept, faces
        whose other side is absent become boundary faces with bc_id = cut_bc."""
        mesh, ids = self.mesh, self.local[rank]
        n_el = mesh["nodes"].shape[0]
        remap = -np.ones(n_el, dtype=np.int64)
        remap[ids] = np.arange(ids.size)
        ifc = mesh["ifaces"]
        inL, inR = remap[ifc[:, 0]] >= 0, remap[ifc[:, 2]] >= 0
        both = inL & inR
        sub_if = ifc[both].copy()
        sub_if[:, 0], sub_if[:, 2] = remap[sub_if[:, 0]], remap[sub_if[:, 2]]
        cutL, cutR = ifc[inL & ~inR], ifc[inR & ~inL]
        bf = [np.stack([remap[cutL[:, 0]], cutL[:, 1], np.full(len(cutL), self.cut_bc)], -1),
              np.stack([remap[cutR[:, 2]], cutR[:, 3], np.full(len(cutR), self.cut_bc)], -1)]
        old_b = mesh["bfaces"]
        if len(old_b):
            keep = remap[old_b[:, 0]] >= 0
            ob = old_b[keep].astype(np.int64).copy()
            ob[:, 0] = remap[ob[:, 0]]
            bf.append(ob)
        sub = dict(mesh)
        sub["nodes"] = np.ascontiguousarray(mesh["nodes"][ids])
        sub["ifaces"] = sub_if.astype(np.int32)
        sub["shifts"] = np.ascontiguousarray(mesh["shifts"][both])
        sub["bfaces"] = np.concatenate(bf).astype(np.int32).reshape(-1, 3)
        return sub

    def halo_bytes(self, rank, bytes_per_element):
        """bytes this rank sends per right-hand side"""
        return sum(v.size for v in self.send[rank].values()) * bytes_per_element


def decompose(mesh, world_size, hops=2, cut_bc=None):
    """Contiguous slabs of the element numbering (structured generators number x fastest, so slabs cut the slowest direction:
    minimal surface for box meshes).  cut_bc: bc_id given to cut faces (default: one past the largest bc_id in use)."""
    n_el = mesh["nodes"].shape[0]
    if world_size < 1 or world_size > n_el:
        raise ValueError("world_size out of range")
    owner = (np.arange(n_el) * world_size) // n_el
    if cut_bc is None:
        cut_bc = int(mesh["bfaces"][:, 2].max()) + 1 if len(mesh["bfaces"]) else 0
    return Plan(mesh, owner.astype(np.int64), hops, cut_bc)


def exchange_halo(plan, rank, state, dist, device_ops=None):
    """Updates the ghost columns of `state` ([N_u, N_V, >= n_local] array or tensor, element last) from their owners with
    point-to-point messages over `dist` (torch.distributed; NCCL on GPUs, gloo in the CPU tests).  Send buffers are packed by
    index_select on the state's device; all sends and receives are posted before any wait."""
    import torch

    t = state if isinstance(state, torch.Tensor) else torch.from_numpy(state)
    ops, bufs = [], []
    for peer, idx in sorted(plan.send[rank].items()):
        out = t.index_select(2, torch.as_tensor(idx, device=t.device)).contiguous()
        ops.append(dist.P2POp(dist.isend, out, peer))
    for peer, idx in sorted(plan.recv[rank].items()):
        buf = torch.empty((t.shape[0], t.shape[1], len(idx)), dtype=t.dtype, device=t.device)
        bufs.append((idx, buf))
        ops.append(dist.P2POp(dist.irecv, buf, peer))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    for idx, buf in bufs:
        t.index_copy_(2, torch.as_tensor(idx, device=t.device), buf)
    return state


class DistributedContext:
    """One rank of a domain-decomposed run: the library context of the rank's sub-mesh plus the halo exchange.  PyTorch is
    plumbing here (device buffers, torch.distributed point-to-point messages); the right-hand side and the register
    updates run in the library (fr_rhs, fr_state_lincomb)."""

    def __init__(self, mesh, disc, precision="f64", world=None, rank=None, bcs=None, cut_state=None):
        import torch
        import torch.distributed as dist

        from .binding import Context

        self.torch, self.dist = torch, dist
        self.world = dist.get_world_size() if world is None else world
        self.rank = dist.get_rank() if rank is None else rank
        self.plan = decompose(mesh, self.world)
        bcs = dict(bcs or {})
        # the state of the dummy boundary on cut faces never reaches an owned element; any admissible state will do
        bcs[self.plan.cut_bc] = ("sup-inflow", cut_state or dict(rho=1.0, v=(0.1,) * mesh["ndims"], p=1.0))
        self.ctx = Context(self.plan.sub_mesh(self.rank), bcs).setup_operators(precision=precision, **disc)
        self.n_owned, self.ids = self.plan.n_owned[self.rank], self.plan.local[self.rank]
        c = self.ctx
        tdt = torch.float64 if c.dtype == np.float64 else torch.float32
        self.shape = (c.Nu, c.NV, c.ld)
        self.k, self.tmp, self.acc = (torch.zeros(self.shape, dtype=tdt, device="cuda") for _ in range(3))
        self.work = torch.zeros(c.workspace_bytes, dtype=torch.uint8, device="cuda")
        self.stream = torch.cuda.current_stream().cuda_stream

    def rhs(self, u, out):
        """out = R(u) on the rank's elements (exact on the owned ones); the ghost columns of u are refreshed first"""
        if self.world > 1:
            exchange_halo(self.plan, self.rank, u, self.dist)
        self.ctx.rhs(u.data_ptr(), out.data_ptr(), self.work.data_ptr(), self.stream)

    def rk4_step(self, u, dt):
        """classical RK4 with a halo exchange in every stage"""
        lc, k, tmp, acc = self.ctx.state_lincomb, self.k, self.tmp, self.acc
        p = lambda t: t.data_ptr()
        self.rhs(u, k)
        lc([p(u), p(k)], [1, dt / 2], p(tmp), self.stream); lc([p(u), p(k)], [1, dt / 6], p(acc), self.stream)
        self.rhs(tmp, k)
        lc([p(u), p(k)], [1, dt / 2], p(tmp), self.stream); lc([p(acc), p(k)], [1, dt / 3], p(acc), self.stream)
        self.rhs(tmp, k)
        lc([p(u), p(k)], [1, dt], p(tmp), self.stream); lc([p(acc), p(k)], [1, dt / 3], p(acc), self.stream)
        self.rhs(tmp, k)
        lc([p(acc), p(k)], [1, dt / 6], p(u), self.stream)
