"""The N>1 path of bench.py is 'replicas only' (the north_star fixes one GPU, no sharding, no
collective on the data path): every rank runs the same workload and the only exchange is the
max-over-ranks reduction of the timed region.  This covers that host logic with world_size 2 on gloo."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_max_over_ranks_aggregation_gloo(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent("""
        import os, sys, json
        sys.path.insert(0, %r)
        import torch, torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")
        val = bench.aggregate_value(dof=1000, ms_step=ms, world=world)
        if rank == 0:
            print(json.dumps({"ms": ms, "val": val}))
        dist.destroy_process_group()
    """ % ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29517")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                          "--master-port", "29517", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json

    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["ms"] == 15.0  # the slower rank
    assert abs(d["val"] - 2 * 1000 / 15e-3 / 1e9) < 1e-12


def test_domain_decomposition_halo_exchange_gloo(tmp_path):
    """SURVEY 8(f) item 2, host side: the element partition with two ghost layers and one halo exchange of
    state columns per right-hand side (paper_1312_1638_b200/partition.py) reproduces the single-rank right-hand side and RK4
    state on the owned elements of every rank.  world_size 2 and 3 on gloo; the per-rank compute is the oracle (no GPU here),
    the exchange code is the one the GPU path uses."""
    script = tmp_path / "dd.py"
    script.write_text(textwrap.dedent("""
        import os, sys, json
        sys.path.insert(0, %r)
        import numpy as np, torch, torch.distributed as dist
        import workloads as W
        from oracle.fr_oracle import FROracle
        from paper_1312_1638_b200.partition import decompose, exchange_halo
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        mesh = W.box_mesh((5, 12), (1.0, 2.4), p_g=2, warp=lambda X: 0.02 * np.stack([np.sin(2 * np.pi * X[..., 0]) * np.sin(2 * np.pi * X[..., 1] / 2.4)] * 2, -1))
        disc = dict(p=3, system="navier-stokes", gamma=1.4, mu=0.02, Pr=0.71, beta=0.5, tau=0.1)
        full = FROracle(mesh, disc)
        X = np.asarray(full.xu_phys, float)
        U = np.ascontiguousarray(np.moveaxis(W.add_relative_noise(W.sinusoidal_2d(X / 2.4), 1e-2, 3), -1, 1))
        plan = decompose(mesh, world)
        ids, n_own = plan.local[rank], plan.n_owned[rank]
        assert n_own < ids.size < mesh["nodes"].shape[0]          # there are ghosts, and not the whole mesh
        sub = FROracle(plan.sub_mesh(rank), disc, {plan.cut_bc: ("sup-inflow", dict(rho=1.0, v=(0.3, 0.1), p=9.0))})
        def local_rhs(u_loc):
            u_loc[:, :, n_own:] = np.nan                            # ghost columns are stale until the exchange
            exchange_halo(plan, rank, u_loc, dist)
            return sub.rhs(u_loc)
        u = np.ascontiguousarray(U[:, :, ids])
        R = local_rhs(u.copy())
        R_ref = full.rhs(U)
        err_rhs = float(np.max(np.abs(R[:, :, :n_own] - R_ref[:, :, ids[:n_own]])) / np.max(np.abs(R_ref)))
        # two RK4 steps with a halo exchange in every stage
        dt, ref = 1e-4, U
        for _ in range(2):
            ref = full.rk4_step(ref, dt)
            k1 = local_rhs(u.copy()); k2 = local_rhs(u + dt / 2 * k1); k3 = local_rhs(u + dt / 2 * k2); k4 = local_rhs(u + dt * k3)
            u = u + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        err_rk = float(np.max(np.abs(u[:, :, :n_own] - ref[:, :, ids[:n_own]])))
        out = torch.tensor([err_rhs, err_rk, float(plan.halo_bytes(rank, U.shape[0] * U.shape[1] * 8))], dtype=torch.float64)
        dist.all_reduce(out, op=dist.ReduceOp.MAX)
        if rank == 0:
            print(json.dumps({"err_rhs": out[0].item(), "err_rk": out[1].item(), "halo_bytes": out[2].item(), "world": world}))
        dist.destroy_process_group()
    """ % ROOT))
    import json

    for world, port in ((2, 29531), (3, 29532)):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=%d" % world, "--master-addr", "127.0.0.1",
                              "--master-port", str(port), str(script)], capture_output=True, text=True, env=env, timeout=600)
        assert out.returncode == 0, out.stderr[-3000:]
        d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
        assert d["world"] == world and d["halo_bytes"] > 0
        assert d["err_rhs"] <= 1e-13 and d["err_rk"] <= 1e-13, d


def test_partition_plan_invariants():
    """Index bookkeeping of the domain decomposition (no communication): every element is owned once; ghosts are exactly the
    elements within two face-neighbour steps; send and receive tables of every pair of ranks list the same global elements in
    the same order; a sub-mesh covers each of its flux-point faces once (interfaces kept + cut faces + original boundaries)."""
    import numpy as np

    import workloads as W
    from paper_1312_1638_b200.partition import decompose

    for mesh, world in ((W.box_mesh((4, 4, 9), (1.0, 1.0, 2.0), periodic=(True, False, True)), 3), (W.tri_mesh(8, 1.0, 0.1, 3), 4)):
        n_el = mesh["nodes"].shape[0]
        plan = decompose(mesh, world)
        owned = np.concatenate([plan.local[r][: plan.n_owned[r]] for r in range(world)])
        assert np.array_equal(np.sort(owned), np.arange(n_el))
        nfaces = {"hex": 6, "tri": 3, "quad": 4}[mesh["etype"]]
        for r in range(world):
            ids = plan.local[r]
            for peer, idx in plan.recv[r].items():
                assert np.array_equal(ids[idx], plan.local[peer][plan.send[peer][r]])
                assert np.all(plan.owner[ids[idx]] == peer) and np.all(idx >= plan.n_owned[r])
            got = np.sort(np.concatenate([v for v in plan.recv[r].values()])) if plan.recv[r] else np.zeros(0, int)
            assert np.array_equal(got, np.arange(plan.n_owned[r], ids.size))  # every ghost is received exactly once
            sub = plan.sub_mesh(r)
            cover = np.zeros((ids.size, nfaces), dtype=int)
            np.add.at(cover, (sub["ifaces"][:, 0], sub["ifaces"][:, 1]), 1)
            np.add.at(cover, (sub["ifaces"][:, 2], sub["ifaces"][:, 3]), 1)
            np.add.at(cover, (sub["bfaces"][:, 0], sub["bfaces"][:, 1]), 1)
            assert np.all(cover == 1)
            # the owned elements and their neighbours' neighbours are all present: no cut face within one step of an owned element
            cut = sub["bfaces"][sub["bfaces"][:, 2] == plan.cut_bc][:, 0]
            near = np.zeros(ids.size, dtype=bool)
            near[: plan.n_owned[r]] = True
            touch = near[sub["ifaces"][:, 0]] | near[sub["ifaces"][:, 2]]
            near[sub["ifaces"][touch, 0]] = True
            near[sub["ifaces"][touch, 2]] = True
            assert not np.any(near[cut])
