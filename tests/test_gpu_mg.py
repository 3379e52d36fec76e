"""F3, second half, on the GPU against the oracle (-m gpu): the coarse BiCGStab with fixed iterations
and one V-cycle of the multigrid preconditioner, through the C ABI.

Bars.  One operator application keeps the north_star bars TOL1 (1e-12 fp64, 2e-6 fp32).
A k-iteration BiCGStab applies D_c 2k times; its iterate is a rational function of inner products, so the forward
error is bounded by (number of applications) x cond(D_c) x TOL1 -- cond(D_c) is computed in the test from the oracle's
dense coarse matrix where that is small enough, else the bound 30 (cond <= 17 measured on configs 1-2).  The V-cycle
adds the restriction, the prolongation and SAP's 2 n_sap (n_mr + 1) fine applications.
"""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle
from problems import check_bar, config_problem, rel_l2
from test_gpu_parity import Dev, rounded, to_dev

pytestmark = pytest.mark.gpu

TOL1 = {"f64": 1e-12, "f32": 2e-6}


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2111_05012_b200 as lq
    return lq


def cond_coarse(prob, prec):
    cfg = prob.cfg
    n = cfg.cvolume * 2 * cfg.nvec
    if n > 1024:
        return 30.0
    A = rounded(prob.A, prec).astype(np.complex128)
    M = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        M[:, k] = oracle.coarse_mult(e.reshape(-1, 2, cfg.nvec), A, cfg.cdims).ravel()
    return float(np.linalg.cond(M))


def gpu_bicgstab(lq, d, b, niter, want_r=True):
    import torch
    cfg = d.cfg
    bd = to_dev(b, d.prec)
    x = torch.full_like(bd, 9.0)
    r = torch.full_like(bd, 9.0) if want_r else None
    lq.coarse_bicgstab(x, bd, d.A, cfg.cdims, cfg.nvec, niter, r_out=r)
    return x.cpu().numpy(), (r.cpu().numpy() if want_r else None)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name", ["c1", "c2"])
def test_coarse_bicgstab(lq, prec, name):
    prob = config_problem(name)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    cond = cond_coarse(prob, prec)
    assert cond < 30
    b = prob.xc
    A = rounded(prob.A, prec)
    for niter in (0, 1, 3, 8):
        rx, rr = oracle.coarse_bicgstab(rounded(b, prec), A, cfg.cdims, cfg.nvec, niter)
        gx, gr = gpu_bicgstab(lq, d, b, niter)
        if niter == 0:
            assert not np.any(gx) and np.array_equal(gr, rounded(b, prec))
            continue
        bar = 2 * niter * cond * TOL1[prec]   # principled bound; check_bar also applies the tight bar
        check_bar(rel_l2(gx, rx), bar, prec, f"bicgstab {name} niter {niter}")
        check_bar(np.linalg.norm(gr - rr) / np.linalg.norm(b), bar, prec, f"bicgstab residual {name} {niter}")
    # without r_out: the same solution, bit for bit (fixed summation order)
    gx2, _ = gpu_bicgstab(lq, d, b, 8, want_r=False)
    assert np.array_equal(gx, gx2)
    # b = 0: every quotient has a vanishing denominator -> x = 0, no NaN
    gx0, gr0 = gpu_bicgstab(lq, d, np.zeros_like(b), 3)
    assert not np.any(gx0) and not np.any(gr0)


def gpu_vcycle(lq, d, b, n_coarse, n_sap, n_mr):
    cfg = d.cfg
    bn = lq.pack_spinor(to_dev(b, d.prec), cfg.dims)
    x = lq.empty_spinor(cfg.dims, dtype=bn.dtype)
    x.fill_(2.0)
    lq.mg_vcycle(x, bn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec, d.v, d.A, n_coarse=n_coarse,
                 n_sap=n_sap, n_mr=n_mr)
    return lq.unpack_spinor(x, cfg.dims).cpu().numpy()


def oracle_vcycle(prob, prec, b, n_coarse, n_sap, n_mr):
    cfg = prob.cfg
    return oracle.mg_vcycle(rounded(b, prec), rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa, cfg.dims,
                            cfg.bc, cfg.block, rounded(prob.v, prec), rounded(prob.A, prec), n_coarse=n_coarse,
                            n_sap=n_sap, n_mr=n_mr)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("path", [0, -1], ids=["resident", "generic"])
def test_c1_vcycle(lq, prec, path):
    prob = config_problem("c1")
    d = Dev(lq, prob, prec)
    cond = cond_coarse(prob, prec)
    b = prob.psi[0]
    lq.set_knob("sap_fused", path)
    try:
        for n_coarse, n_sap, n_mr in ((8, 4, 6), (3, 0, 6), (0, 2, 3), (0, 0, 0)):
            ref = oracle_vcycle(prob, prec, b, n_coarse, n_sap, n_mr)
            got = gpu_vcycle(lq, d, b, n_coarse, n_sap, n_mr)
            if not np.any(ref):
                assert not np.any(got)
                continue
            bar = (2 * n_coarse * cond + 2 + 2 * n_sap * (n_mr + 1)) * TOL1[prec]
            check_bar(rel_l2(got, ref), bar, prec, f"vcycle c1 {n_coarse},{n_sap},{n_mr} path {path}")
    finally:
        lq.set_knob("sap_fused", 0)
    # M ~ D^-1: the V-cycle with the paper's parameters reduces the residual of D x = b
    x = gpu_vcycle(lq, d, b, 8, 4, 6)
    cfg = prob.cfg
    res = rounded(b, prec) - oracle.wilson_clover_mult(x, rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa,
                                                       cfg.dims, cfg.bc)
    assert np.linalg.norm(res) < 0.1 * np.linalg.norm(b)


@pytest.mark.parametrize("name", ["c2", "c3"])
def test_vcycle_fp32_configs(lq, name):
    """config 2 (8^4, N_nv = 16) and config 3 (16^3 x 32, N_nv = 32, the V-cycle config): 4^4 domains, i.e. the
    shared-memory-resident smoother at its design size, the paper's parameters n_sap = 4, n_mr = 6."""
    prob = config_problem(name)
    d = Dev(lq, prob, "f32")
    b = prob.psi[0]
    n_coarse = 8 if name == "c2" else 4
    ref = oracle_vcycle(prob, "f32", b, n_coarse, 4, 6)
    got = gpu_vcycle(lq, d, b, n_coarse, 4, 6)
    bar = (2 * n_coarse * 30.0 + 2 + 2 * 4 * 7) * TOL1["f32"]
    check_bar(rel_l2(got, ref), bar, "f32", f"vcycle {name}")


def test_mg_error_codes(lq):
    import torch
    prob = config_problem("c1")
    cfg = prob.cfg
    d = Dev(lq, prob, "f32")
    x, b = lq.empty_spinor(cfg.dims), lq.empty_spinor(cfg.dims)
    xc = torch.zeros((cfg.cvolume, 2, cfg.nvec), dtype=torch.complex64, device="cuda")
    bc_ = torch.zeros_like(xc)

    def code(fn):
        try:
            fn()
        except lq.LqcdError as e:
            return e.code
        return 0

    n0 = lq.launch_count()
    vc = lambda **kw: lq.mg_vcycle(x, b, d.U, d.clover, cfg.kappa, cfg.dims, **{"bc": cfg.bc, "block": cfg.block,
                                                                                 "nvec": cfg.nvec, "nullvecs": d.v,
                                                                                 "A": d.A, **kw})
    assert code(lambda: vc(bc=(1, 1, 1, 2))) == lq.EINVAL
    assert code(lambda: vc(block=(4, 4, 4, 4))) == lq.EINVAL      # coarse extent 1
    assert code(lambda: vc(n_coarse=-1)) == lq.EINVAL
    assert code(lambda: lq.mg_vcycle(x, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec, d.v,
                                     d.A)) == lq.EINVAL
    assert "lqcd_mg_vcycle_f32" in lq.last_error()
    assert code(lambda: lq.coarse_bicgstab(xc, xc, d.A, cfg.cdims, cfg.nvec, 3)) == lq.EINVAL
    assert code(lambda: lq.coarse_bicgstab(xc, bc_, d.A, cfg.cdims, cfg.nvec, -1)) == lq.EINVAL
    assert code(lambda: lq.coarse_bicgstab(xc, bc_, d.A, (2, 2, 2, 1), cfg.nvec, 1)) == lq.EINVAL
    assert lq.launch_count() == n0, "nothing is enqueued on error"


@pytest.mark.parametrize("prec,name,nrhs", [("f64", "c1", 3), ("f32", "c1", 5), ("f32", "c2", 4), ("f32", "c3", 18)])
def test_coarse_bicgstab_mrhs(lq, prec, name, nrhs):
    """K independent BiCGStab recurrences that share the D_c applications (config 3: through the tensor-core kernel,
    two launches per application for 18 right-hand sides): every right-hand side against the oracle's single solve."""
    import torch
    prob = config_problem(name)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    cond = cond_coarse(prob, prec)
    rng = np.random.default_rng(123)
    bs = np.stack([li.coarse_vector(rng, cfg.cvolume, cfg.nvec) for _ in range(nrhs)])
    bs[-1] *= 1e-3                    # right-hand sides of different scale keep their own scalars
    niter = 5
    bd = to_dev(bs, prec)
    x, r = torch.full_like(bd, 7.0), torch.full_like(bd, 7.0)
    lq.coarse_bicgstab_mrhs(x, bd, d.A, cfg.cdims, cfg.nvec, niter, r_out=r)
    gx, gr = x.cpu().numpy(), r.cpu().numpy()
    A = rounded(prob.A, prec)
    bar = 2 * niter * cond * TOL1[prec]
    one = torch.empty_like(bd[0])
    for k in range(nrhs):
        rx, rr = oracle.coarse_bicgstab(rounded(bs[k], prec), A, cfg.cdims, cfg.nvec, niter)
        check_bar(rel_l2(gx[k], rx), bar, prec, f"bicgstab mrhs {name} k {k}")
        check_bar(np.linalg.norm(gr[k] - rr) / np.linalg.norm(bs[k]), bar, prec, f"bicgstab mrhs residual {name} k {k}")
    # and against the single-right-hand-side call on the GPU
    lq.coarse_bicgstab(one, bd[0].contiguous(), d.A, cfg.cdims, cfg.nvec, niter)
    assert rel_l2(gx[0], one.cpu().numpy()) <= bar


@pytest.mark.parametrize("prec,name,nrhs", [("f64", "c1", 3), ("f32", "c1", 4), ("f32", "c3", 3)])
def test_vcycle_mrhs(lq, prec, name, nrhs):
    """the V-cycle on several right-hand sides at once: every one against the oracle's single V-cycle"""
    import torch
    from problems import make_problem
    prob = make_problem(li.CONFIGS[name], n_rhs=nrhs)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    cond = cond_coarse(prob, prec)
    n_coarse, n_sap, n_mr = 4, 2, 6
    b = torch.stack([lq.pack_spinor(to_dev(p, prec), cfg.dims) for p in prob.psi])
    x = torch.full_like(b, 2.0)
    lq.mg_vcycle_mrhs(x, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec, d.v, d.A,
                      n_coarse=n_coarse, n_sap=n_sap, n_mr=n_mr)
    bar = (2 * n_coarse * cond + 2 + 2 * n_sap * (n_mr + 1)) * TOL1[prec]
    for k in range(nrhs):
        ref = oracle_vcycle(prob, prec, prob.psi[k], n_coarse, n_sap, n_mr)
        got = lq.unpack_spinor(x[k], cfg.dims).cpu().numpy()
        check_bar(rel_l2(got, ref), bar, prec, f"vcycle mrhs {name} k {k}")


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,block,nvec,bc", [
    ((6, 4, 6, 4), (2, 2, 2, 2), 3, (1, 1, 1, -1)),     # odd coarse extents (3, 2, 3, 2), odd N_nv, coarse extent 2
    ((4, 6, 4, 8), (2, 3, 2, 4), 5, (-1, 1, -1, 1)),    # non-cubic blocks, other boundary conditions
])
def test_vcycle_edge_lattices(lq, prec, dims, block, nvec, bc):
    """single and batched V-cycle on odd lattices against the oracle, including the degenerate iteration counts"""
    import torch
    from problems import custom_config, make_problem
    cfg = custom_config(dims, block, nvec, bc=bc)
    prob = make_problem(cfg, n_rhs=3)
    d = Dev(lq, prob, prec)
    cond = cond_coarse(prob, prec)
    assert cond < 200
    b = torch.stack([lq.pack_spinor(to_dev(p, prec), cfg.dims) for p in prob.psi])
    for n_coarse, n_sap, n_mr in ((4, 2, 4), (0, 1, 3), (2, 0, 3)):
        x = torch.full_like(b, 2.0)
        lq.mg_vcycle_mrhs(x, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec, d.v, d.A,
                          n_coarse=n_coarse, n_sap=n_sap, n_mr=n_mr)
        bar = (2 * n_coarse * cond + 2 + 2 * n_sap * (n_mr + 1)) * TOL1[prec]
        for k in range(3):
            ref = oracle_vcycle(prob, prec, prob.psi[k], n_coarse, n_sap, n_mr)
            got = lq.unpack_spinor(x[k], cfg.dims).cpu().numpy()
            check_bar(rel_l2(got, ref), bar, prec, f"vcycle mrhs edge {n_coarse},{n_sap},{n_mr} k {k}")
        # the single-right-hand-side call gives the same
        got1 = gpu_vcycle(lq, d, prob.psi[0], n_coarse, n_sap, n_mr)
        assert rel_l2(got1, lq.unpack_spinor(x[0], cfg.dims).cpu().numpy()) <= bar
