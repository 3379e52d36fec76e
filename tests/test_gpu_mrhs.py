"""F4 on the GPU against the oracle (-m gpu): the coarse operator on K right-hand sides at once.  The definition is K
independent applications of Eq. 4/7, so the expected value is the oracle's coarse_mult per right-
hand side; the bar is the north_star's per-application bar (2e-6 fp32 -- also for the tensor-core path, whose 3xTF32
operand split is there to keep fp32 accuracy; 1e-12 fp64)."""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle
from problems import config_problem, rel_l2
from test_gpu_parity import Dev, rounded, to_dev

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-6}


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2111_05012_b200 as lq
    return lq


def rhs_set(cfg, nrhs, seed=77):
    rng = np.random.default_rng(seed)
    return np.stack([li.coarse_vector(rng, cfg.cvolume, cfg.nvec) for _ in range(nrhs)])


def gpu_mrhs(lq, d, xs, dagger=False):
    import torch
    x = to_dev(xs, d.prec)
    y = torch.full_like(x, 3.0)
    lq.coarse_mult_mrhs(y, x, d.A, d.cfg.cdims, d.cfg.nvec, dagger=dagger)
    torch.cuda.synchronize()
    return y.cpu().numpy()


@pytest.mark.parametrize("nrhs", [1, 3, 4, 16, 21, 64, 70])
def test_c3_tensor_core_path(lq, nrhs):
    """config 3 (coarse 4^3 x 8, N = 64, true Galerkin blocks): tcgen05 path, also ragged K and K > 16 (several launches)"""
    prob = config_problem("c3")
    cfg = prob.cfg
    d = Dev(lq, prob, "f32")
    xs = rhs_set(cfg, nrhs)
    n0 = lq.launch_count()
    got = gpu_mrhs(lq, d, xs)
    assert lq.launch_count() - n0 == (nrhs + 15) // 16, "one tensor-core launch per 16 right-hand sides"
    A = rounded(prob.A, "f32")
    worst = 0.0
    for k in range(nrhs):
        ref = oracle.coarse_mult(rounded(xs[k], "f32"), A, cfg.cdims)
        worst = max(worst, rel_l2(got[k], ref))
    assert worst <= TOL["f32"], worst
    # fixed summation order (per-stage accumulator chains added in stage order): bit-reproducible
    assert np.array_equal(got, gpu_mrhs(lq, d, xs))
    # the tensor-core path and the single-right-hand-side kernel agree to rounding
    lq.set_knob("mrhs_tensor", -1)
    try:
        alt = gpu_mrhs(lq, d, xs)
    finally:
        lq.set_knob("mrhs_tensor", 0)
    assert rel_l2(got, alt) <= TOL["f32"]


def test_c3_structured_inputs(lq):
    """unit vectors and a constant vector: a wrong neighbour, a transposed block or a swapped (re, im) row of the
    operand matrix cannot hide behind random data"""
    prob = config_problem("c3")
    cfg = prob.cfg
    d = Dev(lq, prob, "f32")
    xs = np.zeros((8, cfg.cvolume, 2, cfg.nvec), dtype=np.complex128)
    sites = [0, 1, cfg.cdims[0], cfg.cvolume - 1]
    for k, X in enumerate(sites):
        xs[k, X, k % 2, (5 * k) % cfg.nvec] = 1.0        # real unit vector at one site
        xs[4 + k, X, (k + 1) % 2, (7 * k + 3) % cfg.nvec] = 1j  # imaginary unit vector
    got = gpu_mrhs(lq, d, xs)
    A = rounded(prob.A, "f32")
    for k in range(8):
        ref = oracle.coarse_mult(xs[k], A.astype(np.complex128), cfg.cdims)
        assert rel_l2(got[k], ref) <= TOL["f32"], k
        assert np.array_equal(got[k] == 0, ref == 0), "exact zeros outside the stencil"


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name", ["c1", "c2"])
def test_generic_sizes(lq, prec, name):
    """N = 8 and N = 32 (and fp64): one single-right-hand-side application per vector; dagger form too"""
    prob = config_problem(name)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    xs = rhs_set(cfg, 5)
    A = rounded(prob.A, prec)
    for dagger in (False, True):
        got = gpu_mrhs(lq, d, xs, dagger=dagger)
        for k in range(5):
            ref = oracle.coarse_mult(rounded(xs[k], prec), A, cfg.cdims, dagger=dagger)
            assert rel_l2(got[k], ref) <= TOL[prec], (k, dagger)


def test_mrhs_error_codes(lq):
    import torch
    prob = config_problem("c1")
    cfg = prob.cfg
    d = Dev(lq, prob, "f32")
    x = torch.zeros((2, cfg.cvolume, 2, cfg.nvec), dtype=torch.complex64, device="cuda")
    y = torch.zeros_like(x)

    def code(fn):
        try:
            fn()
        except lq.LqcdError as e:
            return e.code
        return 0

    n0 = lq.launch_count()
    assert code(lambda: lq.coarse_mult_mrhs(x, x, d.A, cfg.cdims, cfg.nvec)) == lq.EINVAL
    with pytest.raises(ValueError, match="needs"):  # sizes are checked by the binding before the C call ...
        lq.coarse_mult_mrhs(y, x, d.A, (2, 2, 1, 2), cfg.nvec)
    st = torch.cuda.current_stream().cuda_stream   # ... and the C call refuses the geometry itself
    rc = lq.lib().lqcd_coarse_mult_mrhs_f32(y.data_ptr(), x.data_ptr(), d.A.data_ptr(), lq._i4((2, 2, 1, 2)), cfg.nvec,
                                            2, 0, st)
    assert rc == lq.EINVAL, "coarse extent 1"
    assert code(lambda: lq.coarse_mult_mrhs(y, x, d.A, cfg.cdims, 0)) == lq.EINVAL
    assert "lqcd_coarse_mult_mrhs_f32" in lq.last_error()
    assert lq.launch_count() == n0


# ---- the fine operator on several right-hand sides -----------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("links12", [False, True])
def test_c1_fine_mrhs(lq, prec, links12):
    import torch
    from problems import make_problem
    prob = make_problem(li.CONFIGS["c1"], n_rhs=5, coarse="none")
    cfg = prob.cfg
    d = Dev(lq, prob, prec, links12=links12, coarse=False)
    x = torch.stack([lq.pack_spinor(to_dev(p, prec), cfg.dims) for p in prob.psi])
    for dagger in (False, True):
        y = torch.full_like(x, 4.0)
        n0 = lq.launch_count()
        lq.wilson_clover_mult_mrhs(y, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, dagger=dagger, links12=links12)
        assert lq.launch_count() - n0 == 3, "two pairs and one odd right-hand side"
        for k in range(5):
            ref = oracle.wilson_clover_mult(rounded(prob.psi[k], prec), rounded(prob.U, prec), rounded(prob.clover, prec),
                                            cfg.kappa, cfg.dims, cfg.bc, dagger=dagger)
            assert rel_l2(lq.unpack_spinor(y[k], cfg.dims).cpu().numpy(), ref) <= TOL[prec], (k, dagger)
    # the pair kernel and the single-right-hand-side kernel do the same arithmetic in the same order: bit-identical
    y1 = torch.empty_like(x)
    lq.set_knob("fine_mrhs", -1)
    try:
        lq.wilson_clover_mult_mrhs(y1, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, dagger=True, links12=links12)
    finally:
        lq.set_knob("fine_mrhs", 0)
    assert torch.equal(y, y1)


@pytest.mark.parametrize("dims,bc", [((3, 3, 3, 3), (1, 1, 1, -1)), ((6, 4, 2, 10), (-1, 1, -1, 1)),
                                     ((16, 8, 8, 8), (1, 1, 1, -1))])
def test_fine_mrhs_edge_lattices(lq, dims, bc):
    import torch
    from problems import custom_config, make_problem
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc)
    prob = make_problem(cfg, n_rhs=2, coarse="none")
    d = Dev(lq, prob, "f32", coarse=False)
    x = torch.stack([lq.pack_spinor(to_dev(p, "f32"), dims) for p in prob.psi])
    y = torch.full_like(x, 4.0)
    lq.wilson_clover_mult_mrhs(y, x, d.U, d.clover, cfg.kappa, dims, bc)
    for k in range(2):
        ref = oracle.wilson_clover_mult(rounded(prob.psi[k], "f32"), rounded(prob.U, "f32"), rounded(prob.clover, "f32"),
                                        cfg.kappa, dims, bc)
        assert rel_l2(lq.unpack_spinor(y[k], dims).cpu().numpy(), ref) <= TOL["f32"], k


def test_tensor_core_path_coarse_extent_two(lq):
    """8^4 blocked 4^4 with N_nv = 32: coarse extent 2 in every direction (X + mu == X - mu: the forward and the
    backward block multiply the SAME neighbour vector), 16 coarse sites only -- fewer sites than SMs, one per CTA."""
    from problems import custom_config, make_problem
    cfg = custom_config((8, 8, 8, 8), (4, 4, 4, 4), 32, bc=(1, 1, 1, -1), kappa=0.135, csw=1.0)
    prob = make_problem(cfg)
    d = Dev(lq, prob, "f32")
    xs = rhs_set(cfg, 6)
    n0 = lq.launch_count()
    got = gpu_mrhs(lq, d, xs)
    assert lq.launch_count() - n0 == 1
    A = rounded(prob.A, "f32")
    for k in range(6):
        ref = oracle.coarse_mult(rounded(xs[k], "f32"), A, cfg.cdims)
        assert rel_l2(got[k], ref) <= TOL["f32"], k


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name,nrhs", [("c1", 11), ("c2", 5), ("c3", 9)])
def test_restrict_mrhs(lq, prec, name, nrhs):
    """several fine vectors restricted in one pass over the null vectors; groups of up to 9, ragged last group"""
    import torch
    if name == "c3" and prec == "f64":
        pytest.skip("config 3 is an fp32 config")
    prob = config_problem(name)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    rng = np.random.default_rng(9)
    psis = [rng.standard_normal((cfg.volume, 4, 3)) + 1j * rng.standard_normal((cfg.volume, 4, 3)) for _ in range(nrhs)]
    x = torch.stack([lq.pack_spinor(to_dev(p, prec), cfg.dims) for p in psis])
    out = torch.full((nrhs, cfg.cvolume, 2, cfg.nvec), 3.0, dtype=to_dev(np.zeros(1), prec).dtype, device="cuda")
    lq.restrict_mrhs(out, x, d.v, cfg.dims, cfg.block, cfg.nvec)
    got = out.cpu().numpy()
    one = torch.empty_like(out[0])
    for k in range(nrhs):
        ref = oracle.restrict(rounded(psis[k], prec), rounded(prob.v, prec), cfg.dims, cfg.block)
        assert rel_l2(got[k], ref) <= TOL[prec], k
        lq.restrict(one, x[k], d.v, cfg.dims, cfg.block, cfg.nvec)
        assert rel_l2(got[k], one.cpu().numpy()) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name,nrhs", [("c1", 11), ("c2", 5), ("c3", 9)])
def test_prolong_mrhs(lq, prec, name, nrhs):
    import torch
    if name == "c3" and prec == "f64":
        pytest.skip("config 3 is an fp32 config")
    prob = config_problem(name)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    xs = rhs_set(cfg, nrhs, seed=5)
    xd = to_dev(xs, prec)
    out = torch.full((nrhs, lq.native_spinor_reals(cfg.dims)), 3.0, dtype=d.U.dtype, device="cuda")
    lq.prolong_mrhs(out, xd, d.v, cfg.dims, cfg.block, cfg.nvec)
    for k in range(nrhs):
        ref = oracle.prolong(rounded(xs[k], prec), rounded(prob.v, prec), cfg.dims, cfg.block)
        assert rel_l2(lq.unpack_spinor(out[k], cfg.dims).cpu().numpy(), ref) <= TOL[prec], k


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_transfer_mrhs_large_and_odd_blocks(lq, prec):
    """8x4x4x4 blocks (24 / 48 KB per slice: fewer slices per group) and a 2x3x2x2 block with odd N_nv"""
    import torch
    from problems import custom_config, make_problem
    for dims, block, nvec, nrhs in (((16, 8, 8, 8), (8, 4, 4, 4), 4, 5), ((4, 6, 4, 4), (2, 3, 2, 2), 3, 10)):
        cfg = custom_config(dims, block, nvec)
        prob = make_problem(cfg, coarse="synthetic")
        d = Dev(lq, prob, prec)
        rng = np.random.default_rng(17)
        psis = [rng.standard_normal((cfg.volume, 4, 3)) + 1j * rng.standard_normal((cfg.volume, 4, 3))
                for _ in range(nrhs)]
        x = torch.stack([lq.pack_spinor(to_dev(p, prec), dims) for p in psis])
        out = torch.full((nrhs, cfg.cvolume, 2, nvec), 3.0, dtype=to_dev(np.zeros(1), prec).dtype, device="cuda")
        lq.restrict_mrhs(out, x, d.v, dims, block, nvec)
        xs = rhs_set(cfg, nrhs, seed=8)
        fine = torch.full_like(x, 3.0)
        lq.prolong_mrhs(fine, to_dev(xs, prec), d.v, dims, block, nvec)
        for k in range(nrhs):
            assert rel_l2(out[k].cpu().numpy(), oracle.restrict(rounded(psis[k], prec), rounded(prob.v, prec), dims,
                                                                block)) <= TOL[prec], (dims, k)
            assert rel_l2(lq.unpack_spinor(fine[k], dims).cpu().numpy(),
                          oracle.prolong(rounded(xs[k], prec), rounded(prob.v, prec), dims, block)) <= TOL[prec], (dims, k)


@pytest.mark.parametrize("cdims", [(3, 2, 3, 2), (2, 5, 3, 4), (7, 3, 2, 3)])
def test_tensor_core_path_odd_coarse_lattices(lq, cdims):
    """odd and mixed coarse extents (multiply-high division by 3, 5, 7; wraps in every direction), synthetic blocks"""
    import torch
    nv = 32
    Vc = int(np.prod(cdims))
    rng = np.random.default_rng(sum(cdims))
    A = li.coarse_matrix_synthetic(rng, Vc, nv)
    xs = np.stack([li.coarse_vector(rng, Vc, nv) for _ in range(7)])
    Ad, xd = to_dev(A, "f32"), to_dev(xs, "f32")
    y = torch.full_like(xd, 3.0)
    n0 = lq.launch_count()
    lq.coarse_mult_mrhs(y, xd, Ad, cdims, nv)
    assert lq.launch_count() - n0 == 1, "tensor-core path"
    got = y.cpu().numpy()
    for k in range(7):
        ref = oracle.coarse_mult(rounded(xs[k], "f32"), rounded(A, "f32"), cdims)
        assert rel_l2(got[k], ref) <= TOL["f32"], k
