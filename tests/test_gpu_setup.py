"""Parity of the device-side set-up kernels against the oracle's O3 / O4 / O6 (-m gpu)."""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle
from problems import config_problem, custom_config, make_problem, rel_l2

pytestmark = pytest.mark.gpu

CDT = {"f64": np.complex128, "f32": np.complex64}
# bars: fp64 1e-12 and fp32 2e-6 relative L2 (north_star), for F itself and for 1 + F as it enters Eq. 1
TOL = {"f64": 1e-12, "f32": 2e-6}


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available()
    import paper_2111_05012_b200 as lq
    return lq


def to_dev(a, prec):
    import torch
    return torch.from_numpy(np.ascontiguousarray(np.asarray(a).astype(CDT[prec]))).cuda()


def rounded(a, prec):
    return np.ascontiguousarray(np.asarray(a).astype(CDT[prec]))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name,dims", [("c1", None), ("c2", None), ("odd", (3, 5, 2, 6)), ("c3", None)])
def test_clover_from_links(lq, prec, name, dims):
    if dims is None:
        cfg = li.CONFIGS[name]
        U = li.make_host_fields(cfg, with_nullvecs=False).U
    else:
        cfg = custom_config(dims, (1, 1, 1, 1), 1)
        U = li.gauge_exp(np.random.default_rng(3), int(np.prod(dims)), 0.7)
    ref = oracle.clover_from_links(rounded(U, prec), cfg.kappa, cfg.csw, cfg.dims)
    Un = lq.pack_gauge(to_dev(U, prec), cfg.dims)
    got = lq.unpack_clover(lq.clover_from_links(Un, cfg.kappa, cfg.csw, cfg.dims), cfg.dims).cpu().numpy()
    assert np.array_equal(got, np.conj(np.swapaxes(got, -1, -2))), "exactly Hermitian by construction"
    eye = np.eye(6)
    err_op = rel_l2(got + eye, ref + eye)      # as it enters Eq. 1
    err_f = rel_l2(got, ref)
    print(f"clover {name} {prec}: rel L2 of F {err_f:.2e}, of 1+F {err_op:.2e}, max|F| {np.abs(ref).max():.3f}")
    assert err_f <= TOL[prec] and err_op <= TOL[prec]


@pytest.mark.parametrize("prec,name", [("f64", "c1"), ("f32", "c1"), ("f32", "c2"), ("f32", "c3")])
def test_orthonormalize_blocks(lq, prec, name):
    """Raw Gaussian null vectors -> device Gram-Schmidt vs the oracle's modified Gram-Schmidt (same unique result)."""
    cfg = li.CONFIGS[name]
    raw = li.make_host_fields(cfg).v
    ref = oracle.orthonormalize_blocks(rounded(raw, prec).astype(np.complex128), cfg.dims, cfg.block)
    vn = lq.pack_nullvecs(to_dev(raw, prec), cfg.dims, cfg.block)
    lq.orthonormalize_blocks(vn, cfg.dims, cfg.block, cfg.nvec)
    got = np.stack([lq.unpack_nullvec(vn, i, cfg.dims, cfg.block, cfg.nvec).cpu().numpy() for i in range(cfg.nvec)])
    assert rel_l2(got, ref) <= TOL[prec]
    worst = max(rel_l2(got[i], ref[i]) for i in range(cfg.nvec))   # the last vectors accumulate the most rounding
    assert worst <= 4 * TOL[prec], worst
    # valid on its own terms: R P = 1 on one aggregate (block-orthonormal columns)
    X, chi = 1, 1
    dom = np.all(li.site_coords(cfg.dims) // np.array(cfg.block) == np.array(li.site_coords(cfg.cdims)[X]), axis=1)
    cols = got[:, dom][:, :, 2 * chi:2 * chi + 2, :].reshape(cfg.nvec, -1).astype(np.complex128)
    gram = cols.conj() @ cols.T
    assert np.max(np.abs(gram - np.eye(cfg.nvec))) <= (1e-13 if prec == "f64" else 5e-6)


@pytest.mark.parametrize("prec,name", [("f64", "c1"), ("f32", "c1"), ("f32", "c2"), ("f32", "c3")])
def test_galerkin_coarse(lq, prec, name):
    """A = P^dag D P built on the device column by column vs the oracle's direct assembly (Eq. 7), same inputs."""
    prob = config_problem(name, 16 if name == "c2" else 1)
    cfg = prob.cfg
    Un = lq.pack_gauge(to_dev(prob.U, prec), cfg.dims)
    Cn = lq.pack_clover(to_dev(prob.clover, prec), cfg.dims)
    vn = lq.pack_nullvecs(to_dev(prob.v, prec), cfg.dims, cfg.block)
    n0 = lq.launch_count()
    got = lq.galerkin_coarse(Un, Cn, vn, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec).cpu().numpy()
    # per column: P e_J, D_SAP, 8 hops, the multi-restrict (one launch per 9 slices of 108 KB shared memory), 9 scatters
    assert lq.launch_count() - n0 == 2 * cfg.nvec * 20
    ref = oracle.galerkin_coarse(rounded(prob.U, prec), rounded(prob.clover, prec), rounded(prob.v, prec), cfg.kappa,
                                 cfg.dims, cfg.bc, cfg.block)
    assert rel_l2(got, ref) <= TOL[prec]
    for d in range(9):                                   # every one of the nine blocks on its own scale
        assert rel_l2(got[:, d], ref[:, d]) <= 2 * TOL[prec], d
    # and it drives the coarse operator like the oracle's matrix does
    import torch
    xc = to_dev(prob.xc, prec)
    yc = torch.empty_like(xc)
    lq.coarse_mult(yc, xc, to_dev(got, prec), cfg.cdims, cfg.nvec)
    ref_y = oracle.coarse_mult(rounded(prob.xc, prec), rounded(prob.A, prec), cfg.cdims)
    assert rel_l2(yc.cpu().numpy(), ref_y) <= 2 * TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_setup_edge_geometry(lq, prec):
    """odd block 3x2x2x4, nvec 3, mixed boundary conditions, coarse extents 2: orthonormalise + Galerkin"""
    cfg = custom_config((6, 4, 4, 8), (3, 2, 2, 4), 3, bc=(-1, 1, -1, 1))
    prob = make_problem(cfg)
    Un = lq.pack_gauge(to_dev(prob.U, prec), cfg.dims)
    Cn = lq.clover_from_links(Un, cfg.kappa, cfg.csw, cfg.dims)
    raw = li.make_host_fields(cfg).v
    vn = lq.pack_nullvecs(to_dev(raw, prec), cfg.dims, cfg.block)
    lq.orthonormalize_blocks(vn, cfg.dims, cfg.block, cfg.nvec)
    got = lq.galerkin_coarse(Un, Cn, vn, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec).cpu().numpy()
    # the whole device set-up chain (clover, orthonormalisation, Galerkin) against the whole oracle chain
    assert rel_l2(got, prob.A if prec == "f64" else oracle.galerkin_coarse(
        rounded(prob.U, prec).astype(np.complex128),
        oracle.clover_from_links(rounded(prob.U, prec).astype(np.complex128), cfg.kappa, cfg.csw, cfg.dims),
        oracle.orthonormalize_blocks(rounded(raw, prec).astype(np.complex128), cfg.dims, cfg.block),
        cfg.kappa, cfg.dims, cfg.bc, cfg.block)) <= (1e-12 if prec == "f64" else 3 * TOL[prec])


def test_clover_from_links_feeds_the_operator(lq):
    """D with the device-built clover term equals the oracle's D with the oracle's clover term (fp32, config 2)."""
    prec = "f32"
    prob = config_problem("c2", 16)
    cfg = prob.cfg
    Un = lq.pack_gauge(to_dev(prob.U, prec), cfg.dims)
    Cn = lq.clover_from_links(Un, cfg.kappa, cfg.csw, cfg.dims)
    x = lq.pack_spinor(to_dev(prob.psi[0], prec), cfg.dims)
    y = lq.empty_spinor(cfg.dims)
    lq.wilson_clover_mult(y, x, Un, Cn, cfg.kappa, cfg.dims, cfg.bc)
    got = lq.unpack_spinor(y, cfg.dims).cpu().numpy()
    U32 = rounded(prob.U, prec)
    # the oracle needs one precision for all inputs: promote the fp32-rounded fields to fp64
    U64, psi64 = U32.astype(np.complex128), rounded(prob.psi[0], prec).astype(np.complex128)
    ref = oracle.wilson_clover_mult(psi64, U64, oracle.clover_from_links(U64, cfg.kappa, cfg.csw, cfg.dims), cfg.kappa,
                                    cfg.dims, cfg.bc)
    assert rel_l2(got, ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,block,nvec,bc", [
    ((6, 4, 6, 4), (2, 2, 2, 2), 3, (1, 1, 1, -1)),     # odd coarse extents, coarse extent 2, odd N_nv
    ((4, 6, 4, 8), (2, 3, 2, 4), 5, (-1, 1, -1, 1)),    # non-cubic blocks, other boundary conditions
])
def test_setup_chain_edge_lattices(lq, prec, dims, block, nvec, bc):
    """clover term, block orthonormalisation and Galerkin assembly on odd lattices: each against the oracle"""
    from problems import custom_config
    import lqcd_inputs as li_
    cfg = custom_config(dims, block, nvec, bc=bc)
    hf = li_.make_host_fields(cfg, n_rhs=1, with_nullvecs=True)
    Un = lq.pack_gauge(to_dev(hf.U, prec), cfg.dims)
    Cn = lq.clover_from_links(Un, cfg.kappa, cfg.csw, cfg.dims)
    clov_ref = oracle.clover_from_links(rounded(hf.U, prec), cfg.kappa, cfg.csw, cfg.dims)
    assert rel_l2(lq.unpack_clover(Cn, cfg.dims).cpu().numpy(), clov_ref) <= 4 * TOL[prec]
    # from here on both sides consume the oracle's clover term and the oracle's orthonormal vectors
    v_ref = oracle.orthonormalize_blocks(rounded(hf.v, prec), cfg.dims, cfg.block)
    vn = lq.pack_nullvecs(to_dev(hf.v, prec), cfg.dims, cfg.block)
    lq.orthonormalize_blocks(vn, cfg.dims, cfg.block, cfg.nvec)
    got_v = np.stack([lq.unpack_nullvec(vn, i, cfg.dims, cfg.block, cfg.nvec).cpu().numpy() for i in range(cfg.nvec)])
    assert rel_l2(got_v, v_ref) <= 4 * TOL[prec]
    Cn2 = lq.pack_clover(to_dev(clov_ref, prec), cfg.dims)
    vn2 = lq.pack_nullvecs(to_dev(v_ref, prec), cfg.dims, cfg.block)
    got = lq.galerkin_coarse(Un, Cn2, vn2, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec).cpu().numpy()
    ref = oracle.galerkin_coarse(rounded(hf.U, prec), rounded(clov_ref, prec), rounded(v_ref, prec), cfg.kappa, cfg.dims,
                                 cfg.bc, cfg.block)
    assert rel_l2(got, ref) <= TOL[prec]
