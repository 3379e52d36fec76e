"""F3 on the GPU against the oracle (-m gpu): Richardson residual, blocked BLAS-1, the inner-domain minimal-residual
solver M_SAP^(e/o) and the SAP listing, through the C ABI.

Bars.  A single operator application keeps the north_star bars (1e-12 fp64, 2e-6 fp32).  The iterations chain
applications with fixed counts; their rounding errors add at most linearly (the minimal-residual coefficient is a
ratio of two sums over the same data, so its relative perturbation is that of p = D_SAP rho), hence
  mr_domain_solve(n_mr):  n_mr x the single-application bar,
  sap(n_sap, n_mr):       2 n_sap (n_mr + 1) x the single-application bar
(DESIGN.md section 6.6).  Both code paths of the solver (shared-memory-resident and generic) are held to them.
"""
import numpy as np
import pytest

import oracle
from problems import check_bar, config_problem, custom_config, make_problem, rel_l2
from test_gpu_parity import CDT, Dev, rounded, to_dev

pytestmark = pytest.mark.gpu

TOL1 = {"f64": 1e-12, "f32": 2e-6}


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2111_05012_b200 as lq
    return lq


@pytest.fixture(params=[(0, 0), (0, -1), (-1, 0)], ids=["resident", "resident-smem", "generic"])
def path(lq, request):
    """the implementations of the inner-domain solver: resident (persistent, links and clover blocks parked in tensor
    memory, for fp32 4^4 domains on the tiled site order; elsewhere the same as the next), resident in shared memory
    only (one CTA per domain), generic"""
    lq.set_knob("sap_fused", request.param[0])
    lq.set_knob("sap_tmem", request.param[1])
    yield request.param[0]
    lq.set_knob("sap_fused", 0)
    lq.set_knob("sap_tmem", 0)


def fields(prob, prec):
    return rounded(prob.U, prec), rounded(prob.clover, prec)


def rdtype(lq, prec):
    import torch
    return torch.float32 if prec == "f32" else torch.float64


def gpu_mr(lq, d, r, domain, parity, niter, accumulate_into=None):
    import torch
    cfg = d.cfg
    rn = lq.pack_spinor(to_dev(r, d.prec), cfg.dims)
    ws = lq.mr_workspace(cfg.dims, domain, dtype=rdtype(lq, d.prec))
    if accumulate_into is None:
        z = lq.empty_spinor(cfg.dims, dtype=rn.dtype)
        z.fill_(5.0)  # must be overwritten everywhere
        lq.mr_domain_solve(z, rn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, domain, parity=parity, niter=niter, ws=ws)
    else:
        z = lq.pack_spinor(to_dev(accumulate_into, d.prec), cfg.dims)
        lq.mr_domain_solve(z, rn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, domain, parity=parity, niter=niter,
                           accumulate=True, ws=ws)
    torch.cuda.synchronize()
    return lq.unpack_spinor(z, cfg.dims).cpu().numpy()


def gpu_sap(lq, d, b, domain, n_sap, n_mr, x0=None, final_residual=True):
    cfg = d.cfg
    bn = lq.pack_spinor(to_dev(b, d.prec), cfg.dims)
    x = lq.empty_spinor(cfg.dims, dtype=bn.dtype) if x0 is None else lq.pack_spinor(to_dev(x0, d.prec), cfg.dims)
    if x0 is None:
        x.fill_(3.0)
    r = lq.empty_spinor(cfg.dims, dtype=bn.dtype)
    ws = lq.mr_workspace(cfg.dims, domain, dtype=rdtype(lq, d.prec))
    lq.sap(x, r, bn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, domain, n_sap=n_sap, n_mr=n_mr,
           initial_guess=x0 is not None, final_residual=final_residual, ws=ws)
    return lq.unpack_spinor(x, cfg.dims).cpu().numpy(), lq.unpack_spinor(r, cfg.dims).cpu().numpy()


# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("links12", [False, True])
def test_residual(lq, prec, links12):
    prob = config_problem("c1", 2)
    cfg = prob.cfg
    d = Dev(lq, prob, prec, links12=links12, coarse=False)
    b, x = prob.psi
    bn, xn = (lq.pack_spinor(to_dev(a, prec), cfg.dims) for a in (b, x))
    r = lq.empty_spinor(cfg.dims, dtype=bn.dtype)
    lq.wilson_clover_residual(r, bn, xn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, links12=links12)
    U, clov = fields(prob, prec)
    ref = rounded(b, prec) - oracle.wilson_clover_mult(rounded(x, prec), U, clov, cfg.kappa, cfg.dims, cfg.bc)
    assert rel_l2(lq.unpack_spinor(r, cfg.dims).cpu().numpy(), ref) <= TOL1[prec]
    # r must alias neither b (read through the read-only path) nor x: refused, nothing enqueued
    for bad in (bn, xn):
        with pytest.raises(lq.LqcdError) as e:
            lq.wilson_clover_residual(bad, bn, xn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, links12=links12)
        assert e.value.code == lq.EINVAL


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,domain", [
    ((4, 4, 4, 4), (2, 2, 2, 2)),
    ((8, 8, 8, 8), (4, 4, 4, 4)),
    ((6, 4, 2, 10), (3, 4, 1, 5)),
    ((3, 3, 3, 3), (3, 1, 3, 1)),     # V = 81: ragged chunk
    ((16, 8, 8, 8), (8, 4, 4, 4)),    # the paper's 8x4x4x4: 512 sites per domain
    ((4, 4, 4, 4), (4, 4, 4, 4)),     # one domain: the global dotc / axpy
])
def test_block_blas(lq, prec, dims, domain):
    import torch
    rng = np.random.default_rng(5)
    V = int(np.prod(dims))
    a, b = (rounded(rng.standard_normal((V, 4, 3)) + 1j * rng.standard_normal((V, 4, 3)), prec) for _ in range(2))
    an, bn = (lq.pack_spinor(to_dev(v, prec), dims) for v in (a, b))
    got = lq.block_dotc(an, bn, dims, domain).cpu().numpy()
    ref = oracle.block_dotc(a, b, dims, domain)
    # a dot product is compared on the scale of its terms: |<a|b>_X| <= |a|_X |b|_X
    scale = np.sqrt(oracle.block_dotc(a, a, dims, domain).real * oracle.block_dotc(b, b, dims, domain).real)
    assert np.max(np.abs(got - ref) / scale) <= TOL1[prec]
    nd = ref.size
    coef = rounded(rng.standard_normal(nd) + 1j * rng.standard_normal(nd), prec)
    lq.block_caxpy(bn, to_dev(coef, prec), an, dims, domain)
    assert rel_l2(lq.unpack_spinor(bn, dims).cpu().numpy(), oracle.block_caxpy(b, coef, a, dims, domain)) <= TOL1[prec]
    torch.cuda.synchronize()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_c1_mr_domain_solve(lq, prec, path):
    prob = config_problem("c1", 2)
    cfg = prob.cfg
    d = Dev(lq, prob, prec, coarse=False)
    U, clov = fields(prob, prec)
    r, y = prob.psi
    for parity in (0, 1, 2):
        for niter in (0, 1, 6):
            ref = oracle.mr_domain_solve(rounded(r, prec), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, parity,
                                         niter)
            got = gpu_mr(lq, d, r, cfg.block, parity, niter)
            if niter == 0:
                assert np.all(got == 0)
                continue
            check_bar(rel_l2(got, ref), niter * TOL1[prec], prec, f"mr parity {parity} niter {niter}")
            assert np.array_equal(got == 0, ref == 0), "exact zeros outside the selected group"
    # accumulate: y + M^(e) r, sites of odd domains untouched (bit for bit)
    ref = rounded(y, prec) + oracle.mr_domain_solve(rounded(r, prec), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block,
                                                    1, 6)
    got = gpu_mr(lq, d, r, cfg.block, 1, 6, accumulate_into=y)
    check_bar(rel_l2(got, ref), 6 * TOL1[prec], prec, "mr accumulate")
    untouched = oracle.mr_domain_solve(rounded(r, prec), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, 1, 1) == 0
    assert np.array_equal(got[untouched], rounded(y, prec)[untouched])


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,domain,bc", [
    ((8, 8, 8, 8), (4, 4, 4, 4), (1, 1, 1, -1)),       # config 2's lattice, the paper's typical 4^4 domain
    ((16, 8, 8, 8), (8, 4, 4, 4), (1, 1, 1, -1)),      # 8x4x4x4: generic path in both precisions
    ((6, 4, 2, 10), (3, 4, 1, 5), (-1, 1, -1, 1)),     # 60-site domains, single domain in y (wrap with bc), odd Lc[0]
    ((3, 3, 3, 3), (3, 1, 3, 1), (1, 1, 1, -1)),       # V = 81, 9-site domains, 9 domains (odd count)
    ((4, 4, 4, 8), (4, 4, 4, 8), (1, 1, 1, -1)),       # ONE domain: global minimal residual on D itself
])
def test_mr_edge_lattices(lq, prec, dims, domain, bc, path):
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc)
    prob = make_problem(cfg, coarse="none")
    if np.prod(domain) >= 512 and path == -1 and prec == "f64":
        pytest.skip("same path as the resident parametrisation")
    d = Dev(lq, prob, prec, coarse=False)
    U, clov = fields(prob, prec)
    r = prob.psi[0]
    for parity in (0, 1, 2):
        ref = oracle.mr_domain_solve(rounded(r, prec), U, clov, cfg.kappa, dims, bc, domain, parity, 6)
        got = gpu_mr(lq, d, r, domain, parity, 6)
        if not np.any(ref):  # e.g. odd group of a single-domain lattice
            assert not np.any(got)
            continue
        check_bar(rel_l2(got, ref), 6 * TOL1[prec], prec, f"mr edge parity {parity}")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_c1_sap(lq, prec, path):
    """config 1 with the paper's parameters n = 4, 6 inner iterations"""
    prob = config_problem("c1", 2)
    cfg = prob.cfg
    d = Dev(lq, prob, prec, coarse=False)
    U, clov = fields(prob, prec)
    b, x0 = prob.psi
    bar = 2 * 4 * 7 * TOL1[prec]
    rx, rr = oracle.sap(rounded(b, prec), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=4, n_mr=6)
    gx, gr = gpu_sap(lq, d, b, cfg.block, 4, 6)
    check_bar(rel_l2(gx, rx), bar, prec, "sap x")
    check_bar(np.linalg.norm(gr - rr) / np.linalg.norm(rounded(b, prec)), bar, prec, "sap r")  # on the scale of b
    assert np.linalg.norm(gr) < 0.05 * np.linalg.norm(b), "SAP(4) reduces the residual as in the oracle pin"
    # without the final residual the solution is the same, bit for bit
    gx2, _ = gpu_sap(lq, d, b, cfg.block, 4, 6, final_residual=False)
    assert np.array_equal(gx, gx2)
    # with an initial guess: x0 + SAP(b - D x0), i.e. the Richardson refinement with M_2 = SAP
    x0 = 0.1 * rounded(x0, prec)
    r0 = rounded(b, prec) - oracle.wilson_clover_mult(x0, U, clov, cfg.kappa, cfg.dims, cfg.bc)
    sx, sr = oracle.sap(r0, U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=3)
    gx, gr = gpu_sap(lq, d, b, cfg.block, 2, 3, x0=x0)
    check_bar(rel_l2(gx, x0 + sx), bar, prec, "sap initial guess x")
    check_bar(np.linalg.norm(gr - sr) / np.linalg.norm(rounded(b, prec)), bar, prec, "sap initial guess r")
    # n_sap = 0: x = 0, r = b
    gx, gr = gpu_sap(lq, d, b, cfg.block, 0, 6)
    assert not np.any(gx) and np.array_equal(gr, rounded(b, prec))


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_c2_lattice_sap(lq, prec):
    """8^4 with 4^4 domains: fp32 takes the shared-memory-resident kernel at its design size (256 sites, 168 KB),
    fp64 does not fit and takes the generic path."""
    cfg = custom_config((8, 8, 8, 8), (4, 4, 4, 4), 1, gauge="exp", eps=0.5, kappa=0.135, csw=1.0)
    prob = make_problem(cfg, coarse="none")
    d = Dev(lq, prob, prec, coarse=False)
    nbytes = lq.lib().lqcd_mr_workspace_bytes(lq._i4(cfg.dims), lq._i4(cfg.block), 4 if prec == "f32" else 8)
    assert (nbytes == 0) == (prec == "f32")
    U, clov = fields(prob, prec)
    b = prob.psi[0]
    rx, rr = oracle.sap(rounded(b, prec), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=4, n_mr=6)
    gx, gr = gpu_sap(lq, d, b, cfg.block, 4, 6)
    bar = 2 * 4 * 7 * TOL1[prec]
    check_bar(rel_l2(gx, rx), bar, prec, "sap x (edge)")
    check_bar(np.linalg.norm(gr - rr) / np.linalg.norm(b), bar, prec, "sap r (edge)")
    assert np.linalg.norm(gr) < np.linalg.norm(b)


def test_sap_error_codes(lq):
    prob = config_problem("c1")
    cfg = prob.cfg
    d = Dev(lq, prob, "f32", coarse=False)
    x, r, b = (lq.empty_spinor(cfg.dims) for _ in range(3))

    def code(fn):
        try:
            fn()
        except lq.LqcdError as e:
            return e.code
        return 0

    n0 = lq.launch_count()
    sap = lambda **kw: lq.sap(x, r, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, **{"domain": cfg.block, **kw})
    assert code(lambda: sap(domain=(3, 2, 2, 2))) == lq.EINVAL
    assert code(lambda: sap(n_sap=-1)) == lq.EINVAL
    assert code(lambda: lq.sap(x, x, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block)) == lq.EINVAL
    assert code(lambda: lq.sap(x, r, b, d.U, d.clover, cfg.kappa, cfg.dims, (1, 1, 1, 0), cfg.block)) == lq.EINVAL
    assert "lqcd_sap_f32" in lq.last_error()
    mr = lambda **kw: lq.mr_domain_solve(x, r, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, **kw)
    assert code(lambda: mr(niter=-2)) == lq.EINVAL
    assert code(lambda: lq.mr_domain_solve(x, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block)) == lq.EINVAL
    assert code(lambda: lq.wilson_clover_residual(x, b, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc)) == lq.EINVAL
    assert code(lambda: lq.block_dotc(x, b, cfg.dims, (3, 1, 1, 1))) == lq.EINVAL
    # the generic path without its workspace
    lq.set_knob("sap_fused", -1)
    try:
        assert code(lambda: sap()) == lq.EINVAL and "workspace" in lq.last_error()
    finally:
        lq.set_knob("sap_fused", 0)
    assert lq.launch_count() == n0, "nothing is enqueued on error"


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sap_mrhs_is_sap_per_rhs(lq, prec, path):
    """several right-hand sides on the resident operator: bit-identical with one call per right-hand side (both
    paths), hence covered by the oracle comparisons above; one right-hand side is checked against the oracle again"""
    import torch
    prob = make_problem(__import__("lqcd_inputs").CONFIGS["c1"], n_rhs=3, coarse="none")
    cfg = prob.cfg
    d = Dev(lq, prob, prec, coarse=False)
    b = torch.stack([lq.pack_spinor(to_dev(p, prec), cfg.dims) for p in prob.psi])
    ws = lq.mr_workspace(cfg.dims, cfg.block, dtype=rdtype(lq, prec))
    x, r = torch.full_like(b, 3.0), torch.full_like(b, 3.0)
    lq.sap_mrhs(x, r, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=4, ws=ws)
    x1, r1 = lq.empty_spinor(cfg.dims, dtype=b.dtype), lq.empty_spinor(cfg.dims, dtype=b.dtype)
    for k in range(3):
        lq.sap(x1, r1, b[k], d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=4, ws=ws)
        assert torch.equal(x[k], x1) and torch.equal(r[k], r1), k
    U, clov = fields(prob, prec)
    rx, rr = oracle.sap(rounded(prob.psi[2], prec), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=4)
    check_bar(rel_l2(lq.unpack_spinor(x[2], cfg.dims).cpu().numpy(), rx), 2 * 2 * 5 * TOL1[prec], prec, "sap mrhs")


def test_sap_mrhs_4x4_domains(lq):
    """8^4 with 4^4 domains in fp32: the compile-time 256-site resident kernel with its right-hand-side loop"""
    import torch
    cfg = custom_config((8, 8, 8, 8), (4, 4, 4, 4), 1, gauge="exp", eps=0.5, kappa=0.135, csw=1.0)
    prob = make_problem(cfg, n_rhs=4, coarse="none")
    d = Dev(lq, prob, "f32", coarse=False)
    b = torch.stack([lq.pack_spinor(to_dev(p, "f32"), cfg.dims) for p in prob.psi])
    x, r = torch.full_like(b, 3.0), torch.full_like(b, 3.0)
    lq.sap_mrhs(x, r, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=6)
    x1, r1 = lq.empty_spinor(cfg.dims), lq.empty_spinor(cfg.dims)
    for k in range(4):
        lq.sap(x1, r1, b[k], d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=6)
        assert torch.equal(x[k], x1) and torch.equal(r[k], r1), k


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 8, 4, 8), (16, 16, 16, 20)])
def test_mr_tensor_memory_is_bit_identical(lq, dims):
    """fp32, 4^4 domains, tiled site order: the persistent form of the resident solver (one CTA per SM walks the
    domains, the next domain staged by bulk copies under the current one's iterations) parks each thread's links and
    clover block in tensor memory after the first iteration (knob sap_tmem).  The parked bits
    are the staged fp32 values and the arithmetic is the same, so every result is bit-identical with the
    one-CTA-per-domain shared-memory kernel: all groups, with and without accumulation, 0 ... 7 iterations (fewer than
    2 iterations and the full grid of an odd Lc[0] take the other kernel by design), several right-hand sides on the
    resident operator, SAP.  (Against the oracle both run in test_mr_edge_lattices / test_c2_lattice_sap.)
    (12, 8, 4, 8): odd Lc[0], a direction spanned by one domain; (16, 16, 16, 20): more domains than SMs, so a CTA walks
    several domains (320, 160 per group, on 148 SMs: a ragged second round)."""
    import torch
    cfg = custom_config(dims, (4, 4, 4, 4), 1, gauge="exp", eps=0.5, kappa=0.135, csw=1.0, seed=21)
    prob = make_problem(cfg, n_rhs=3, coarse="none")
    d = Dev(lq, prob, "f32", coarse=False)
    b = torch.stack([lq.pack_spinor(to_dev(p, "f32"), cfg.dims) for p in prob.psi])
    out = {}
    for knob in (0, -1):
        lq.set_knob("sap_tmem", knob)
        try:
            res = []
            for parity in (0, 1, 2):
                for niter in (0, 1, 2, 7):
                    z = torch.full_like(b[0], 5.0)
                    lq.mr_domain_solve(z, b[0], d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, parity=parity,
                                       niter=niter)
                    y = b[1].clone()
                    lq.mr_domain_solve(y, b[0], d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, parity=parity,
                                       niter=niter, accumulate=True)
                    res += [z, y]
            x, r = torch.full_like(b, 3.0), torch.full_like(b, 3.0)
            lq.sap_mrhs(x, r, b, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=5)
            res += [x, r]
            torch.cuda.synchronize()
            out[knob] = res
        finally:
            lq.set_knob("sap_tmem", 0)
    assert len(out[0]) == len(out[-1])
    for k, (a, c) in enumerate(zip(out[0], out[-1])):
        assert torch.equal(a, c), k
    assert float(out[0][-2].abs().max()) > 0


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,domain,bc", [
    ((6, 4, 2, 10), (3, 4, 1, 5), (-1, 1, -1, 1)),     # odd domain counts (same-parity neighbours across the wrap),
                                                       # a direction spanned by one domain, one-site-thick domains
    ((3, 3, 3, 3), (3, 1, 3, 1), (1, 1, 1, -1)),       # V = 81, 9 domains
    ((16, 8, 8, 8), (8, 4, 4, 4), (1, 1, 1, -1)),      # the paper's 8x4x4x4 domains: generic path
])
def test_sap_edge_lattices(lq, prec, dims, domain, bc, path):
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc)
    prob = make_problem(cfg, coarse="none")
    if np.prod(domain) >= 512 and path == -1:
        pytest.skip("same path as the resident parametrisation")
    d = Dev(lq, prob, prec, coarse=False)
    U, clov = fields(prob, prec)
    b = prob.psi[0]
    rx, rr = oracle.sap(rounded(b, prec), U, clov, cfg.kappa, dims, bc, domain, n_sap=3, n_mr=4)
    gx, gr = gpu_sap(lq, d, b, domain, 3, 4)
    bar = 2 * 3 * 5 * TOL1[prec]
    check_bar(rel_l2(gx, rx), bar, prec, "sap x (edge)")
    check_bar(np.linalg.norm(gr - rr) / np.linalg.norm(b), bar, prec, "sap r (edge)")


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,domain,bc", [
    ((8, 8, 8, 8), (4, 4, 4, 4), (1, 1, 1, -1)),       # the resident kernel's design size (fp32)
    ((6, 4, 2, 10), (3, 4, 1, 5), (-1, 1, -1, 1)),     # odd domain counts, a direction spanned by one domain
    ((3, 3, 3, 3), (3, 1, 3, 1), (1, 1, 1, -1)),       # 9 domains, ragged chunk
    ((4, 4, 4, 8), (4, 4, 4, 8), (1, 1, 1, -1)),       # one domain: the odd group is empty
])
def test_sap_group_residual_is_the_full_residual(lq, prec, dims, domain, bc):
    """Between half sweeps SAP computes r = b - D x on the domains of the NEXT group only (knob sap_group_residual):
    the same numbers where they are read -- x and the final residual are bit-identical with the all-sites form."""
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc, seed=13)
    prob = make_problem(cfg, n_rhs=2, coarse="none")
    d = Dev(lq, prob, prec, coarse=False)
    b, x0 = prob.psi
    out = {}
    for knob in (0, -1):
        lq.set_knob("sap_group_residual", knob)
        try:
            out[knob] = (gpu_sap(lq, d, b, domain, 3, 4), gpu_sap(lq, d, b, domain, 2, 3, x0=0.1 * x0),
                         gpu_sap(lq, d, b, domain, 2, 3, final_residual=False)[0])
        finally:
            lq.set_knob("sap_group_residual", 0)
    (xa, ra), (xb, rb), xc = out[0]
    (xa1, ra1), (xb1, rb1), xc1 = out[-1]
    assert np.array_equal(xa, xa1) and np.array_equal(ra, ra1)
    assert np.array_equal(xb, xb1) and np.array_equal(rb, rb1)
    assert np.array_equal(xc, xc1)
    n0 = lq.launch_count()
    gpu_sap(lq, d, b, domain, 3, 4)
    # pack b, [zero-fill by memset], 6 half sweeps (one resident launch, or 1 + 2 n_mr generic ones) + 6 residuals
    assert lq.launch_count() - n0 >= 1 + 6 + 6
