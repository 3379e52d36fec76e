"""The sharded fine operator against the oracle's D on the GLOBAL lattice
(-m gpu, through the C ABI).  One GPU plays the ranks one after the other: every rank's faces are packed, routed by
reference to the neighbour that needs them, and added after the interior pass -- the arithmetic and the indexing of a
multi-GPU run, without ranks that wait on one another.  Bars as for D itself: 1e-12 (fp64), 2e-6 (fp32) relative L2.
"""
import numpy as np
import pytest

import oracle
from problems import custom_config, make_problem, rel_l2
from test_gpu_parity import TOL, lq, rounded, to_dev  # noqa: F401  (lq is a fixture)

pytestmark = pytest.mark.gpu


def sharded_D(lq, prob, prec, ranks, part_mask=None, dagger=False, links12=False, psi=None):
    """D psi on the global lattice, computed rank by rank on sub-lattices with halo faces; returns (V, 4, 3)."""
    from paper_2111_05012_b200 import sharded as sh
    cfg = prob.cfg
    psi = prob.psi[0] if psi is None else psi
    world = int(np.prod(ranks))
    grids = [sh.RankGrid(ranks, r) for r in range(world)]
    mask = grids[0].part_mask if part_mask is None else part_mask
    ld = grids[0].local_dims(cfg.dims)
    loc = []
    for g in grids:
        U = lq.pack_gauge(to_dev(sh.split_field(prob.U, cfg.dims, g, site_axis=1), prec), ld, links12=links12)
        C = lq.pack_clover(to_dev(sh.split_field(prob.clover, cfg.dims, g), prec), ld)
        x = lq.pack_spinor(to_dev(sh.split_field(psi, cfg.dims, g), prec), ld)
        send = lq.halo_buffers(ld, mask, dtype=x.dtype)
        lq.wilson_clover_halo_pack(send, x, U, ld, mask, dagger=dagger, links12=links12)
        loc.append((U, C, x, send))
    recvs = sh.route_faces([l[3] for l in loc], ranks, mask)
    parts = []
    for g, (U, C, x, _), recv in zip(grids, loc, recvs):
        y = lq.empty_spinor(ld, dtype=x.dtype)
        y.fill_(7.0)
        lq.wilson_clover_mult_interior(y, x, U, C, cfg.kappa, ld, cfg.bc, mask, dagger=dagger, links12=links12)
        lq.wilson_clover_halo_add(y, recv, U, cfg.kappa, ld, g.face_phase(cfg.bc, mask), mask, dagger=dagger,
                                  links12=links12)
        parts.append(lq.unpack_spinor(y, ld).cpu().numpy())
    return sh.join_field(parts, cfg.dims, ranks)


def oracle_D(prob, prec, dagger=False, psi=None):
    cfg = prob.cfg
    psi = prob.psi[0] if psi is None else psi
    return oracle.wilson_clover_mult(rounded(psi, prec), rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa,
                                     cfg.dims, cfg.bc, dagger=dagger)


@pytest.fixture(scope="module")
def prob8():
    return make_problem(custom_config((8, 4, 6, 8), (2, 2, 2, 2), 2, bc=(1, 1, 1, -1)), coarse="none")


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("ranks", [(1, 1, 1, 2), (2, 1, 1, 1), (2, 2, 1, 2), (1, 1, 3, 4), (4, 2, 2, 2), (1, 1, 1, 1)])
def test_sharded_matches_global_oracle(lq, prob8, prec, ranks):
    want = oracle_D(prob8, prec)
    got = sharded_D(lq, prob8, prec, ranks)
    assert rel_l2(got, want) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dagger,links12", [(True, False), (False, True), (True, True)])
def test_sharded_dagger_and_12_real_links(lq, prob8, prec, dagger, links12):
    want = oracle_D(prob8, prec, dagger=dagger)
    got = sharded_D(lq, prob8, prec, (2, 1, 2, 2), dagger=dagger, links12=links12)
    assert rel_l2(got, want) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (-1, -1, -1, -1), (-1, 1, -1, 1)])
def test_boundary_phase_only_on_the_global_edge(lq, prec, bc):
    prob = make_problem(custom_config((4, 4, 4, 8), (2, 2, 2, 2), 2, bc=bc, seed=5), coarse="none")
    want = oracle_D(prob, prec)
    for ranks in [(2, 2, 2, 2), (1, 2, 1, 4), (4, 1, 1, 1)]:
        assert rel_l2(sharded_D(lq, prob, prec, ranks), want) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_self_neighbour_in_every_direction(lq, prob8, prec):
    """One rank, all four directions marked partitioned: the rank exchanges with itself -- the same operator."""
    want = oracle_D(prob8, prec)
    got = sharded_D(lq, prob8, prec, (1, 1, 1, 1), part_mask=15)
    assert rel_l2(got, want) <= TOL[prec]
    got = sharded_D(lq, prob8, prec, (1, 2, 1, 1), part_mask=2 | 8)
    assert rel_l2(got, want) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_odd_and_unit_local_extents(lq, prec):
    """Local extents 3, 5 and 1 (both faces of a direction are then the same site; sites sit on up to 8 faces)."""
    prob = make_problem(custom_config((3, 5, 2, 6), (1, 1, 1, 1), 1, bc=(1, -1, 1, -1), seed=9), coarse="none")
    want = oracle_D(prob, prec)
    for ranks, mask in [((1, 1, 2, 6), None), ((3, 5, 2, 1), None), ((1, 1, 1, 1), 15), ((3, 1, 2, 3), 15)]:
        assert rel_l2(sharded_D(lq, prob, prec, ranks, part_mask=mask), want) <= TOL[prec]


def test_sharded_operator_class_self_exchange(lq, prob8):
    """ShardedWilsonClover on one rank (pack || interior on two streams, then add) against the plain kernel."""
    import torch
    from paper_2111_05012_b200 import sharded as sh
    cfg = prob8.cfg
    U = lq.pack_gauge(to_dev(prob8.U, "f32"), cfg.dims)
    C = lq.pack_clover(to_dev(prob8.clover, "f32"), cfg.dims)
    x = lq.pack_spinor(to_dev(prob8.psi[0], "f32"), cfg.dims)
    op = sh.ShardedWilsonClover(U, C, cfg.kappa, cfg.dims, cfg.bc, sh.RankGrid((1, 1, 1, 1)), part_mask=15)
    y = lq.empty_spinor(cfg.dims)
    for dagger in (False, True):
        op.apply(y, x, dagger=dagger)
        torch.cuda.synchronize()
        got = lq.unpack_spinor(y, cfg.dims).cpu().numpy()
        assert rel_l2(got, oracle_D(prob8, "f32", dagger=dagger)) <= TOL["f32"]
    # bit-reproducible: fixed order of the face additions
    y2 = lq.empty_spinor(cfg.dims)
    op.apply(y2, x, dagger=True)
    torch.cuda.synchronize()
    assert torch.equal(y, y2)


def test_part_mask_zero_is_the_plain_operator(lq, prob8):
    import torch
    cfg = prob8.cfg
    U = lq.pack_gauge(to_dev(prob8.U, "f32"), cfg.dims)
    C = lq.pack_clover(to_dev(prob8.clover, "f32"), cfg.dims)
    x = lq.pack_spinor(to_dev(prob8.psi[0], "f32"), cfg.dims)
    y0, y1 = lq.empty_spinor(cfg.dims), lq.empty_spinor(cfg.dims)
    lq.wilson_clover_mult(y0, x, U, C, cfg.kappa, cfg.dims, cfg.bc)
    lq.wilson_clover_mult_interior(y1, x, U, C, cfg.kappa, cfg.dims, cfg.bc, 0)
    n0 = lq.launch_count()
    lq.wilson_clover_halo_pack([None] * 8, x, U, cfg.dims, 0)
    lq.wilson_clover_halo_add(y1, [None] * 8, U, cfg.kappa, cfg.dims, [1] * 8, 0)
    assert lq.launch_count() == n0
    assert float((y0 - y1).norm() / y0.norm()) <= 1e-7        # another instantiation of the same arithmetic


def test_halo_argument_errors(lq, prob8):
    cfg = prob8.cfg
    U = lq.pack_gauge(to_dev(prob8.U, "f32"), cfg.dims)
    x = lq.pack_spinor(to_dev(prob8.psi[0], "f32"), cfg.dims)
    y = lq.empty_spinor(cfg.dims)
    send = lq.halo_buffers(cfg.dims, 8)
    assert send[6].numel() == lq.halo_face_reals(cfg.dims, 3) == 12 * 8 * 4 * 6 and send[0] is None
    n0 = lq.launch_count()
    with pytest.raises(lq.LqcdError):
        lq.wilson_clover_halo_pack(send, x, U, cfg.dims, 16)             # part_mask out of range
    with pytest.raises(lq.LqcdError):
        lq.wilson_clover_halo_pack(send, x, U, cfg.dims, 1 | 8)          # direction 0 partitioned, no buffer
    with pytest.raises(lq.LqcdError):
        lq.wilson_clover_halo_add(y, send, U, cfg.kappa, cfg.dims, [1, 1, 1, 1, 1, 1, 0, 1], 8)   # phase 0
    with pytest.raises(lq.LqcdError):
        lq.wilson_clover_mult_interior(y, y, U, U, cfg.kappa, cfg.dims, cfg.bc, 8)               # out aliases in
    assert lq.launch_count() == n0                                       # nothing enqueued on error


# ---- the coarse operator and the block-local transfers on sub-lattices --------------------------------------------
def sharded_Dc(lq, A, xc, cdims, nvec, prec, ranks, part_mask=None, dagger=False):
    import torch
    from paper_2111_05012_b200 import sharded as sh
    world = int(np.prod(ranks))
    grids = [sh.RankGrid(ranks, r) for r in range(world)]
    mask = grids[0].part_mask if part_mask is None else part_mask
    lc = grids[0].local_dims(cdims)
    loc = []
    for g in grids:
        Al = to_dev(sh.split_field(A, cdims, g), prec)
        xl = to_dev(sh.split_field(xc, cdims, g), prec)
        send = lq.coarse_halo_buffers(lc, nvec, mask, dtype=torch.float32 if prec == "f32" else torch.float64)
        lq.coarse_halo_pack(send, xl, lc, nvec, mask)
        loc.append((Al, xl, send))
    recvs = sh.route_faces([l[2] for l in loc], ranks, mask)
    parts = []
    for (Al, xl, _), recv in zip(loc, recvs):
        y = torch.full_like(xl, 7.0)
        lq.coarse_mult_interior(y, xl, Al, lc, nvec, mask, dagger=dagger)
        lq.coarse_halo_add(y, recv, Al, lc, nvec, mask, dagger=dagger)
        parts.append(y.cpu().numpy())
    return sh.join_field(parts, cdims, ranks)


@pytest.fixture(scope="module")
def probc():
    # coarse lattice 4 x 2 x 6 x 4, N = 12 (a ragged row: 6 float4 / 12 double2 per row)
    return make_problem(custom_config((8, 4, 12, 8), (2, 2, 2, 2), 6, bc=(1, 1, 1, -1), seed=21))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dagger", [False, True])
def test_sharded_coarse_matches_global_oracle(lq, probc, prec, dagger):
    cfg = probc.cfg
    A, xc = rounded(probc.A, prec), rounded(probc.xc, prec)
    want = oracle.coarse_mult(xc, A, cfg.cdims, dagger=dagger)
    for ranks, mask in [((1, 1, 1, 2), None), ((2, 1, 3, 2), None), ((4, 2, 6, 4), None), ((1, 1, 1, 1), 15),
                        ((2, 2, 1, 1), 15), ((1, 1, 6, 1), 4 | 8)]:
        got = sharded_Dc(lq, A, xc, cfg.cdims, cfg.nvec, prec, ranks, part_mask=mask, dagger=dagger)
        assert rel_l2(got, want) <= TOL[prec], (ranks, mask)


def test_sharded_coarse_n64_and_class(lq):
    """N = 64 (the paper's size; the full-row fast path of k_coarse) and the ShardedCoarse class with self exchange."""
    import torch
    import lqcd_inputs as li
    from paper_2111_05012_b200 import sharded as sh
    cdims, nvec = (4, 4, 2, 6), 32
    rng = np.random.default_rng(5)
    Vc = int(np.prod(cdims))
    A = rounded(li.coarse_matrix_synthetic(rng, Vc, nvec), "f32")
    xc = rounded(li.coarse_vector(rng, Vc, nvec), "f32")
    want = oracle.coarse_mult(xc, A, cdims)
    assert rel_l2(sharded_Dc(lq, A, xc, cdims, nvec, "f32", (2, 1, 1, 3)), want) <= TOL["f32"]
    op = sh.ShardedCoarse(to_dev(A, "f32"), cdims, nvec, sh.RankGrid((1, 1, 1, 1)), part_mask=15)
    x = to_dev(xc, "f32")
    y = torch.empty_like(x)
    op.apply(y, x)
    torch.cuda.synchronize()
    assert rel_l2(y.cpu().numpy(), want) <= TOL["f32"]
    y1 = torch.empty_like(x)
    lq.coarse_mult(y1, x, to_dev(A, "f32"), cdims, nvec)
    y0 = torch.empty_like(x)
    lq.coarse_mult_interior(y0, x, to_dev(A, "f32"), cdims, nvec, 0)          # nothing partitioned: D_c itself
    assert torch.equal(y0, y1)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_transfers_are_block_local(lq, probc, prec):
    """A4/A5 need no exchange when the aggregates do not straddle ranks: restrict and prolong on the
    sub-lattices, with the null vectors of the local aggregates, reproduce the oracle on the global lattice."""
    import torch
    from paper_2111_05012_b200 import sharded as sh
    cfg = probc.cfg
    ranks = (2, 1, 3, 2)
    v, psi, xc = rounded(probc.v, prec), rounded(probc.psi[0], prec), rounded(probc.xc, prec)
    want_r = oracle.restrict(psi, v, cfg.dims, cfg.block)
    want_p = oracle.prolong(xc, v, cfg.dims, cfg.block)
    got_r, got_p = [], []
    for r in range(int(np.prod(ranks))):
        g = sh.RankGrid(ranks, r)
        ld, lc = g.local_dims(cfg.dims), g.local_dims(cfg.cdims)
        vl = lq.pack_nullvecs(to_dev(sh.split_field(v, cfg.dims, g, site_axis=1), prec), ld, cfg.block)
        x = lq.pack_spinor(to_dev(sh.split_field(psi, cfg.dims, g), prec), ld)
        yc = torch.empty((int(np.prod(lc)), 2, cfg.nvec), dtype=to_dev(np.zeros(1), prec).dtype, device="cuda")
        lq.restrict(yc, x, vl, ld, cfg.block, cfg.nvec)
        got_r.append(yc.cpu().numpy())
        yf = lq.empty_spinor(ld, dtype=x.dtype)
        lq.prolong(yf, to_dev(sh.split_field(xc, cfg.cdims, g), prec), vl, ld, cfg.block, cfg.nvec)
        got_p.append(lq.unpack_spinor(yf, ld).cpu().numpy())
    assert rel_l2(sh.join_field(got_r, cfg.cdims, ranks), want_r) <= TOL[prec]
    assert rel_l2(sh.join_field(got_p, cfg.dims, ranks), want_p) <= TOL[prec]


def test_coarse_halo_argument_errors(lq):
    import torch
    cdims, nvec = (2, 2, 2, 4), 4
    A = torch.zeros((32, 9, 8, 8), dtype=torch.complex64, device="cuda")
    x = torch.zeros((32, 2, 4), dtype=torch.complex64, device="cuda")
    y = torch.zeros_like(x)
    send = lq.coarse_halo_buffers(cdims, nvec, 8)
    assert send[7].numel() == lq.coarse_halo_face_reals(cdims, nvec, 3) == 8 * 16 and send[1] is None
    n0 = lq.launch_count()
    with pytest.raises(lq.LqcdError):
        lq.coarse_halo_pack(send, x, cdims, nvec, 1 | 8)                       # face 0 has no buffer
    with pytest.raises(lq.LqcdError):
        lq.coarse_halo_add(y, send, A, cdims, nvec, 4 | 8)                     # recv of direction 2 missing
    with pytest.raises(lq.LqcdError):
        lq.coarse_mult_interior(y, x, A, (2, 2, 1, 4), nvec, 8)                # extent 1 in an unpartitioned direction
    with pytest.raises(lq.LqcdError):
        lq.coarse_mult_interior(y, x, A, cdims, nvec, 16)
    assert lq.launch_count() == n0


# ---- peer-memory transport: the pack kernel stores straight into the neighbour's receive buffer -------------------
@pytest.fixture(scope="module")
def pg1():
    """A one-rank nccl process group (symmetric memory needs a group to rendezvous on)."""
    import socket
    import torch
    import torch.distributed as dist
    if dist.is_initialized():
        yield dist.group.WORLD
        return
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1,
                            device_id=torch.device("cuda", 0))
    yield dist.group.WORLD
    dist.destroy_process_group()


def test_peer_transport_fine_and_coarse(lq, prob8, probc, pg1):
    """transport="peer" on one rank: the faces live in symmetric memory and the pack kernels write them through the
    peer mapping (here the rank's own); three applications walk both halves of the double buffer."""
    import torch
    from paper_2111_05012_b200 import sharded as sh
    cfg = prob8.cfg
    U = lq.pack_gauge(to_dev(prob8.U, "f32"), cfg.dims)
    C = lq.pack_clover(to_dev(prob8.clover, "f32"), cfg.dims)
    try:
        op = sh.ShardedWilsonClover(U, C, cfg.kappa, cfg.dims, cfg.bc, sh.RankGrid((1, 1, 1, 1)), part_mask=15,
                                    transport="peer")
    except (RuntimeError, ImportError) as e:      # no symmetric-memory support on this box
        pytest.skip(f"symmetric memory unavailable: {e}")
    ref = sh.ShardedWilsonClover(U, C, cfg.kappa, cfg.dims, cfg.bc, sh.RankGrid((1, 1, 1, 1)), part_mask=15)
    rng = np.random.default_rng(77)
    for k in range(3):
        psi = rounded(rng.standard_normal((cfg.volume, 4, 3)) + 1j * rng.standard_normal((cfg.volume, 4, 3)), "f32")
        x = lq.pack_spinor(to_dev(psi, "f32"), cfg.dims)
        y, y0 = lq.empty_spinor(cfg.dims), lq.empty_spinor(cfg.dims)
        op.apply(y, x, dagger=bool(k & 1))
        ref.apply(y0, x, dagger=bool(k & 1))
        torch.cuda.synchronize()
        assert torch.equal(y, y0)                                        # same kernels, other buffers
        got = lq.unpack_spinor(y, cfg.dims).cpu().numpy()
        assert rel_l2(got, oracle_D(prob8, "f32", dagger=bool(k & 1), psi=psi)) <= TOL["f32"]
    cc = probc.cfg
    A, xc = rounded(probc.A, "f32"), rounded(probc.xc, "f32")
    opc = sh.ShardedCoarse(to_dev(A, "f32"), cc.cdims, cc.nvec, sh.RankGrid((1, 1, 1, 1)), part_mask=15,
                           transport="peer")
    xd = to_dev(xc, "f32")
    for k in range(3):
        yc = torch.empty_like(xd)
        opc.apply(yc, xd)
        torch.cuda.synchronize()
        assert rel_l2(yc.cpu().numpy(), oracle.coarse_mult(xc, A, cc.cdims)) <= TOL["f32"]


# ---- the residual and the SAP smoother on a sharded lattice ---------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("links12", [False, True])
def test_sharded_residual_matches_global_oracle(lq, prob8, prec, links12):
    """r = b - D x rank by rank: interior pass in residual form, faces added with -kappa."""
    from paper_2111_05012_b200 import sharded as sh
    cfg = prob8.cfg
    rng = np.random.default_rng(3)
    b = rounded(rng.standard_normal((cfg.volume, 4, 3)) + 1j * rng.standard_normal((cfg.volume, 4, 3)), prec)
    x = rounded(prob8.psi[0], prec)
    want = b - oracle.wilson_clover_mult(x, rounded(prob8.U, prec), rounded(prob8.clover, prec), cfg.kappa, cfg.dims,
                                         cfg.bc)
    for ranks, mask in [((2, 1, 3, 2), None), ((1, 1, 1, 1), 15)]:
        grids = [sh.RankGrid(ranks, r) for r in range(int(np.prod(ranks)))]
        mask = grids[0].part_mask if mask is None else mask
        ld = grids[0].local_dims(cfg.dims)
        loc = []
        for g in grids:
            U = lq.pack_gauge(to_dev(sh.split_field(prob8.U, cfg.dims, g, site_axis=1), prec), ld, links12=links12)
            C = lq.pack_clover(to_dev(sh.split_field(prob8.clover, cfg.dims, g), prec), ld)
            xl = lq.pack_spinor(to_dev(sh.split_field(x, cfg.dims, g), prec), ld)
            bl = lq.pack_spinor(to_dev(sh.split_field(b, cfg.dims, g), prec), ld)
            send = lq.halo_buffers(ld, mask, dtype=xl.dtype)
            lq.wilson_clover_halo_pack(send, xl, U, ld, mask, links12=links12)
            loc.append((U, C, xl, bl, send))
        recvs = sh.route_faces([l[4] for l in loc], ranks, mask)
        parts = []
        for g, (U, C, xl, bl, _), recv in zip(grids, loc, recvs):
            r = lq.empty_spinor(ld, dtype=xl.dtype)
            lq.wilson_clover_residual_interior(r, bl, xl, U, C, cfg.kappa, ld, cfg.bc, mask, links12=links12)
            lq.wilson_clover_halo_add(r, recv, U, -cfg.kappa, ld, g.face_phase(cfg.bc, mask), mask, links12=links12)
            parts.append(lq.unpack_spinor(r, ld).cpu().numpy())
        got = sh.join_field(parts, cfg.dims, ranks)
        assert np.linalg.norm(got - want) / np.linalg.norm(b) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sharded_sap_one_rank_self_exchange(lq, prec):
    """ShardedSAP with every direction partitioned on one rank is lqcd_sap: against the oracle's SAP."""
    import torch
    from paper_2111_05012_b200 import sharded as sh
    cfg = custom_config((8, 4, 4, 8), (2, 2, 2, 2), 1, bc=(1, 1, 1, -1), seed=31)
    prob = make_problem(cfg, n_rhs=2, coarse="none")
    U = lq.pack_gauge(to_dev(prob.U, prec), cfg.dims)
    C = lq.pack_clover(to_dev(prob.clover, prec), cfg.dims)
    b, x0 = rounded(prob.psi[0], prec), 0.1 * rounded(prob.psi[1], prec)
    op = sh.ShardedWilsonClover(U, C, cfg.kappa, cfg.dims, cfg.bc, sh.RankGrid((1, 1, 1, 1)), part_mask=15)
    sap = sh.ShardedSAP(op, cfg.block, n_sap=3, n_mr=4)
    bd = lq.pack_spinor(to_dev(b, prec), cfg.dims)
    x, r = lq.empty_spinor(cfg.dims, dtype=bd.dtype), lq.empty_spinor(cfg.dims, dtype=bd.dtype)
    sap.apply(x, r, bd)
    torch.cuda.synchronize()
    rx, rr = oracle.sap(b, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims, cfg.bc, cfg.block,
                        n_sap=3, n_mr=4)
    bar = 2 * 3 * 5 * TOL[prec]
    assert rel_l2(lq.unpack_spinor(x, cfg.dims).cpu().numpy(), rx) <= bar
    assert np.linalg.norm(lq.unpack_spinor(r, cfg.dims).cpu().numpy() - rr) / np.linalg.norm(b) <= bar
    # with an initial guess: x0 + SAP(b - D x0)
    r0 = b - oracle.wilson_clover_mult(x0, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims,
                                       cfg.bc)
    sx, _ = oracle.sap(r0, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims, cfg.bc, cfg.block,
                       n_sap=3, n_mr=4)
    x = lq.pack_spinor(to_dev(x0, prec), cfg.dims)
    sap.apply(x, r, bd, initial_guess=True, final_residual=False)
    torch.cuda.synchronize()
    assert rel_l2(lq.unpack_spinor(x, cfg.dims).cpu().numpy(), x0 + sx) <= bar


class ThreadCluster:
    """Virtual ranks as host threads of this process on one GPU: the exchange hook of the Sharded* classes meets at a
    host barrier (after a device synchronize: every rank's pack is complete) and hands each rank a COPY of the faces
    its neighbours packed.  Host threads wait, kernels never do."""

    def __init__(self, n):
        import threading
        self.n, self.barrier, self.board = n, threading.Barrier(n), [None] * n

    def exchange(self, send, recv, grid, mask, group=None):
        import torch
        from paper_2111_05012_b200 import sharded as sh
        torch.cuda.synchronize()
        self.board[grid.rank] = send
        self.barrier.wait()
        got = [None] * 8
        for mu in range(4):
            if (mask >> mu) & 1:
                got[2 * mu] = self.board[grid.neighbour(mu, -1)][2 * mu + 1].clone()
                got[2 * mu + 1] = self.board[grid.neighbour(mu, +1)][2 * mu].clone()
        torch.cuda.synchronize()
        self.barrier.wait()           # nobody repacks before everybody has its copies
        return got

    def run(self, fn):
        import threading
        err, out = [], [None] * self.n

        def body(r):
            try:
                out[r] = fn(r)
            except BaseException as e:   # noqa: BLE001  (release the others, then report)
                err.append(e)
                self.barrier.abort()

        ts = [threading.Thread(target=body, args=(r,)) for r in range(self.n)]
        for t in ts:
            t.start()
        for t in ts:
            t.join(timeout=300)
        if err:
            raise err[0]
        return out


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sharded_sap_four_ranks_lockstep(lq, prec):
    """SAP on a 4 x 4 x 12 x 8 lattice over a 1 x 1 x 2 x 2 grid of (thread) ranks against the oracle's SAP on the
    global lattice.  Three 2^4 domains per rank in z: the ranks with z coordinate 1 see the global colouring flipped."""
    import torch
    from paper_2111_05012_b200 import sharded as sh
    ranks, dom = (1, 1, 2, 2), (2, 2, 2, 2)
    cfg = custom_config((4, 4, 12, 8), dom, 1, bc=(1, 1, -1, -1), seed=41)
    prob = make_problem(cfg, coarse="none")
    b = rounded(prob.psi[0], prec)
    rx, rr = oracle.sap(b, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims, cfg.bc, dom,
                        n_sap=2, n_mr=3)
    cluster = ThreadCluster(4)
    assert [sh.domain_parity_flip(sh.RankGrid(ranks, r), (4, 4, 6, 4), dom) for r in range(4)] == [0, 1, 0, 1]

    def rank_main(rk):
        torch.cuda.set_device(0)
        g = sh.RankGrid(ranks, rk)
        ld = g.local_dims(cfg.dims)
        U = lq.pack_gauge(to_dev(sh.split_field(prob.U, cfg.dims, g, site_axis=1), prec), ld)
        C = lq.pack_clover(to_dev(sh.split_field(prob.clover, cfg.dims, g), prec), ld)
        bl = lq.pack_spinor(to_dev(sh.split_field(b, cfg.dims, g), prec), ld)
        op = sh.ShardedWilsonClover(U, C, cfg.kappa, ld, cfg.bc, g, exchange=cluster.exchange)
        x, r = lq.empty_spinor(ld, dtype=bl.dtype), lq.empty_spinor(ld, dtype=bl.dtype)
        sh.ShardedSAP(op, dom, n_sap=2, n_mr=3).apply(x, r, bl)
        torch.cuda.synchronize()
        return lq.unpack_spinor(x, ld).cpu().numpy(), lq.unpack_spinor(r, ld).cpu().numpy()

    out = cluster.run(rank_main)
    gx = sh.join_field([o[0] for o in out], cfg.dims, ranks)
    gr = sh.join_field([o[1] for o in out], cfg.dims, ranks)
    bar = 2 * 2 * 4 * TOL[prec]
    assert rel_l2(gx, rx) <= bar
    assert np.linalg.norm(gr - rr) / np.linalg.norm(b) <= bar


# ---- the coarse solver with hooks and the whole V-cycle on a sharded lattice ------------------------------------------
def vcycle_bar(prob, prec, n_coarse, n_sap, n_mr):
    from test_gpu_mg import cond_coarse
    return (2 * n_coarse * cond_coarse(prob, prec) + 2 + 2 * n_sap * (n_mr + 1)) * TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_bicgstab_hooks_equal_the_plain_solver(lq, probc, prec):
    """With apply = the library's own D_c and no reduce, the hooked solver IS lqcd_coarse_bicgstab, bit for bit."""
    import torch
    cc = probc.cfg
    A, b = to_dev(rounded(probc.A, prec), prec), to_dev(rounded(probc.xc, prec), prec)
    x0, x1 = torch.empty_like(b), torch.empty_like(b)
    lq.coarse_bicgstab(x0, b, A, cc.cdims, cc.nvec, 5)
    calls = []

    def apply(o, i):
        calls.append(1)
        lq.coarse_mult(o, i, A, cc.cdims, cc.nvec)

    lq.coarse_bicgstab_hooks(x1, b, cc.cdims, cc.nvec, 5, apply)
    torch.cuda.synchronize()
    assert len(calls) == 10 and torch.equal(x0, x1)
    with pytest.raises(ZeroDivisionError):          # an exception in a hook surfaces after the C call returns
        lq.coarse_bicgstab_hooks(x1, b, cc.cdims, cc.nvec, 2, lambda o, i: 1 / 0)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sharded_vcycle_one_rank_self_exchange(lq, prec):
    import torch
    from paper_2111_05012_b200 import sharded as sh
    cfg = custom_config((8, 4, 4, 8), (2, 2, 2, 2), 3, bc=(1, 1, 1, -1), seed=51)
    prob = make_problem(cfg)
    one = sh.RankGrid((1, 1, 1, 1))
    U = lq.pack_gauge(to_dev(prob.U, prec), cfg.dims)
    C = lq.pack_clover(to_dev(prob.clover, prec), cfg.dims)
    V = lq.pack_nullvecs(to_dev(prob.v, prec), cfg.dims, cfg.block)
    b = rounded(prob.psi[0], prec)
    fine = sh.ShardedWilsonClover(U, C, cfg.kappa, cfg.dims, cfg.bc, one, part_mask=15)
    coarse = sh.ShardedCoarse(to_dev(prob.A, prec), cfg.cdims, cfg.nvec, one, part_mask=15)
    bd = lq.pack_spinor(to_dev(b, prec), cfg.dims)
    for n_coarse, n_sap, n_mr in ((4, 2, 3), (3, 0, 3)):
        x = lq.empty_spinor(cfg.dims, dtype=bd.dtype)
        sh.ShardedVcycle(fine, coarse, V, cfg.block, cfg.nvec, n_coarse, n_sap, n_mr).apply(x, bd)
        torch.cuda.synchronize()
        ref = oracle.mg_vcycle(b, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims, cfg.bc,
                               cfg.block, rounded(prob.v, prec), rounded(prob.A, prec), n_coarse=n_coarse, n_sap=n_sap,
                               n_mr=n_mr)
        assert rel_l2(lq.unpack_spinor(x, cfg.dims).cpu().numpy(), ref) <= vcycle_bar(prob, prec, n_coarse, n_sap, n_mr)


def cluster_reduce(cluster, rank):
    """Sum of a tensor over the thread-ranks, in rank order, in place (the stand-in for the nccl all-reduce)."""
    import torch

    def reduce(t):
        torch.cuda.synchronize()
        cluster.board[rank] = t
        cluster.barrier.wait()
        total = cluster.board[0].clone()
        for r in range(1, cluster.n):
            total += cluster.board[r]
        torch.cuda.synchronize()
        cluster.barrier.wait()
        t.copy_(total)

    return reduce


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sharded_vcycle_four_ranks_lockstep(lq, prec):
    """The whole V-cycle on a 4 x 4 x 12 x 8 lattice over a 1 x 1 x 2 x 2 grid of thread-ranks (halo exchanges of D,
    D_c and the residual, dot products summed over the ranks) against the oracle's V-cycle on the global lattice."""
    import torch
    from paper_2111_05012_b200 import sharded as sh
    ranks, block = (1, 1, 2, 2), (2, 2, 2, 2)
    cfg = custom_config((4, 4, 12, 8), block, 2, bc=(1, 1, -1, -1), seed=61)
    prob = make_problem(cfg)
    b = rounded(prob.psi[0], prec)
    n_coarse, n_sap, n_mr = 4, 2, 3
    ref = oracle.mg_vcycle(b, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims, cfg.bc, block,
                           rounded(prob.v, prec), rounded(prob.A, prec), n_coarse=n_coarse, n_sap=n_sap, n_mr=n_mr)
    cluster = ThreadCluster(4)

    def rank_main(rk):
        torch.cuda.set_device(0)
        g = sh.RankGrid(ranks, rk)
        ld, lc = g.local_dims(cfg.dims), g.local_dims(cfg.cdims)
        U = lq.pack_gauge(to_dev(sh.split_field(prob.U, cfg.dims, g, site_axis=1), prec), ld)
        C = lq.pack_clover(to_dev(sh.split_field(prob.clover, cfg.dims, g), prec), ld)
        V = lq.pack_nullvecs(to_dev(sh.split_field(prob.v, cfg.dims, g, site_axis=1), prec), ld, block)
        A = to_dev(sh.split_field(prob.A, cfg.cdims, g), prec)
        bl = lq.pack_spinor(to_dev(sh.split_field(b, cfg.dims, g), prec), ld)
        fine = sh.ShardedWilsonClover(U, C, cfg.kappa, ld, cfg.bc, g, exchange=cluster.exchange)
        coarse = sh.ShardedCoarse(A, lc, cfg.nvec, g, exchange=cluster.exchange)
        x = lq.empty_spinor(ld, dtype=bl.dtype)
        sh.ShardedVcycle(fine, coarse, V, block, cfg.nvec, n_coarse, n_sap, n_mr,
                         reduce=cluster_reduce(cluster, rk)).apply(x, bl)
        torch.cuda.synchronize()
        return lq.unpack_spinor(x, ld).cpu().numpy()

    out = cluster.run(rank_main)
    got = sh.join_field(out, cfg.dims, ranks)
    assert rel_l2(got, ref) <= vcycle_bar(prob, prec, n_coarse, n_sap, n_mr)
