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
