"""Host logic of the sharded fine operator on CPU (-m "not gpu"): the rank grid, the split of a global field, and the
face exchange of paper_2111_05012_b200/sharded.py between world_size-2 gloo processes.

The exchange is checked end to end without any GPU arithmetic: each rank pads its sub-lattice with the faces it
RECEIVES (full spinors and the backward links, times the boundary phase of RankGrid.face_phase), applies the oracle's
D to the padded lattice, and the interior must equal its part of the oracle's D on the global lattice -- a face
routed to the wrong neighbour, slot or phase fails it."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DIMS, BC, RANKS = (4, 2, 2, 8), (1, -1, 1, -1), (1, 1, 1, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch
    import torch.distributed as dist
    import oracle
    from problems import custom_config, make_problem
    from paper_2111_05012_b200 import sharded as sh

    dist.init_process_group("gloo", rank=rank, world_size=world)
    grid = sh.RankGrid(RANKS, rank)
    prob = make_problem(custom_config(DIMS, (2, 2, 2, 2), 2, bc=BC, seed=3), coarse="none")
    cfg = prob.cfg
    ld = grid.local_dims(DIMS)
    want = sh.split_field(oracle.wilson_clover_mult(prob.psi[0], prob.U, prob.clover, cfg.kappa, DIMS, BC), DIMS, grid)

    lat = (ld[3], ld[2], ld[1], ld[0])
    psi = sh.split_field(prob.psi[0], DIMS, grid).reshape(lat + (4, 3))
    U = sh.split_field(prob.U, DIMS, grid, site_axis=1).reshape((4,) + lat + (3, 3))
    clover = sh.split_field(prob.clover, DIMS, grid).reshape(lat + (2, 6, 6))

    def faces(a):  # the t faces of a field whose first axis is t, as real tensors; slots 6 (t = 0) and 7 (t = L - 1)
        f = [None] * 8
        f[6] = torch.view_as_real(torch.from_numpy(np.ascontiguousarray(a[0])))
        f[7] = torch.view_as_real(torch.from_numpy(np.ascontiguousarray(a[-1])))
        return f

    def recv_like(f):
        return [None if b is None else torch.empty_like(b) for b in f]

    mask = grid.part_mask
    assert mask == 8
    s_psi, s_U = faces(psi), faces(U[3])
    g_psi = sh.exchange_faces(s_psi, recv_like(s_psi), grid, mask)
    g_U = sh.exchange_faces(s_U, recv_like(s_U), grid, mask)
    ph = grid.face_phase(BC)
    lo = torch.view_as_complex(g_psi[6]).numpy() * ph[6]     # from the -t neighbour: feeds the backward hop at t = 0
    hi = torch.view_as_complex(g_psi[7]).numpy() * ph[7]     # from the +t neighbour: feeds the forward hop at t = L - 1
    psi_pad = np.concatenate([lo[None], psi, hi[None]], axis=0)
    U_pad = np.zeros((4, ld[3] + 2) + lat[1:] + (3, 3), dtype=U.dtype)
    U_pad[:, 1:-1] = U
    U_pad[3, 0] = torch.view_as_complex(g_U[6]).numpy()      # U_t(x - t) of the first slice lives on the -t neighbour
    clover_pad = np.zeros((ld[3] + 2,) + lat[1:] + (2, 6, 6), dtype=clover.dtype)
    clover_pad[1:-1] = clover
    pdims = (ld[0], ld[1], ld[2], ld[3] + 2)
    Vp = int(np.prod(pdims))
    got = oracle.wilson_clover_mult(psi_pad.reshape(Vp, 4, 3), U_pad.reshape(4, Vp, 3, 3),
                                    clover_pad.reshape(Vp, 2, 6, 6), cfg.kappa, pdims, (BC[0], BC[1], BC[2], 1))
    got = got.reshape((ld[3] + 2,) + lat[1:] + (4, 3))[1:-1].reshape(-1, 4, 3)
    err = float(np.linalg.norm(got - want) / np.linalg.norm(want))
    # the cross-rank sum ShardedVcycle hands to the coarse solver's reduce hook
    t = torch.tensor([rank + 1.0, 2.0], dtype=torch.float64)
    sh.allreduce_sum()(t)
    assert t.tolist() == [3.0, 4.0], t
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, err, ph))


def test_world_size_2_gloo_face_exchange():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, err, ph in out:
        assert err <= 1e-13, (rank, err)
    assert out[0][2][6] == -1 and out[0][2][7] == 1          # rank 0 holds t = 0: only its backward hop wraps
    assert out[1][2][6] == 1 and out[1][2][7] == -1


def test_rank_grid_geometry():
    sys.path.insert(0, ROOT)
    from paper_2111_05012_b200 import sharded as sh
    g = sh.RankGrid((2, 1, 3, 2), 7)            # 7 = 1 + 2 * (0 + 1 * (0 + 3 * 1))
    assert g.world == 12 and g.coords == (1, 0, 0, 1) and g.rank_of(g.coords) == 7
    assert g.part_mask == 1 | 4 | 8
    assert g.neighbour(0, +1) == 6 and g.neighbour(0, -1) == 6        # two ranks: the same neighbour on both sides
    assert g.neighbour(1, +1) == 7                                    # one rank: its own neighbour
    assert g.neighbour(2, -1) == sh.RankGrid((2, 1, 3, 2), 0).rank_of((1, 0, 2, 1))
    assert g.neighbour(3, +1) == 1
    assert g.face_phase((-1, -1, -1, -1)) == [1, -1, 1, 1, -1, 1, 1, -1]
    assert g.local_dims((8, 4, 6, 4)) == (4, 4, 2, 2)
    with pytest.raises(ValueError):
        g.local_dims((8, 4, 7, 4))
    with pytest.raises(ValueError):
        sh.RankGrid((2, 2, 2, 2), 16)


def test_split_join_roundtrip_and_routing():
    sys.path.insert(0, ROOT)
    from paper_2111_05012_b200 import sharded as sh
    gd, ranks = (4, 2, 6, 4), (2, 1, 3, 2)
    V = int(np.prod(gd))
    a = np.arange(V * 3, dtype=np.float64).reshape(V, 3)
    parts = [sh.split_field(a, gd, sh.RankGrid(ranks, r)) for r in range(12)]
    assert np.array_equal(sh.join_field(parts, gd, ranks), a)
    b = np.arange(4 * V, dtype=np.float64).reshape(4, V)
    partsb = [sh.split_field(b, gd, sh.RankGrid(ranks, r), site_axis=1) for r in range(12)]
    assert np.array_equal(sh.join_field(partsb, gd, ranks, site_axis=1), b)
    # the local site (0,0,0,0) of rank r is the global site at r's corner
    g = sh.RankGrid(ranks, 7)
    ld = g.local_dims(gd)
    corner = [g.coords[mu] * ld[mu] for mu in range(4)]
    s = corner[0] + gd[0] * (corner[1] + gd[1] * (corner[2] + gd[2] * corner[3]))
    assert np.array_equal(parts[7][0], a[s])
    # routing: what rank r receives in slot 2 mu (from -mu) is the forward face its -mu neighbour sent
    sends = [[(r, f) for f in range(8)] for r in range(12)]
    recvs = sh.route_faces(sends, ranks, 15)
    for r in range(12):
        gr = sh.RankGrid(ranks, r)
        for mu in range(4):
            assert recvs[r][2 * mu] == (gr.neighbour(mu, -1), 2 * mu + 1)
            assert recvs[r][2 * mu + 1] == (gr.neighbour(mu, +1), 2 * mu)
