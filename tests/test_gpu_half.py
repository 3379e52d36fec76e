"""GPU parity of the coarse operator on HALF storage (lqcd_coarse_mult_half): A_0 and the four
forward blocks only, the backward blocks being Gamma5c A_{+mu}(X - mu)^dag Gamma5c (Eqs. 2, 7).

The oracle knows nothing of half storage: its definition is the nine-block coarse_mult (Eq. 4 with the blocks of
Eq. 7).  Two kinds of input:
  * the true Galerkin matrix P^dag D P of configs 1-3 (oracle O6), which HAS the symmetry -- the half operator must
    reproduce the oracle's nine-block result at the single-application bars;
  * arbitrary forward blocks (edge sizes): the nine-block matrix the oracle gets is expanded from them on the host in
    numpy (conjugate transpose + signs, no arithmetic that could share a mistake with the kernel's index handling).
"""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle
from problems import config_problem, expand_half, rel_l2

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 2e-6}


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available()
    import paper_2111_05012_b200 as lq
    return lq


def rounded(a, prec):
    return a.astype(np.complex64) if prec == "f32" else a.astype(np.complex128)


def to_dev(a, prec):
    import torch
    return torch.from_numpy(np.ascontiguousarray(rounded(a, prec))).cuda()


def run_half(lq, Ah, xc, cdims, nvec, prec, dagger):
    import torch
    x, A = to_dev(xc, prec), to_dev(Ah, prec)
    y = torch.full_like(x, 7.0)   # the kernels must overwrite every entry
    lq.coarse_mult_half(y, x, A, cdims, nvec, dagger=dagger)
    return y.cpu().numpy()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name", ["c1", "c2", "c3"])
def test_half_storage_on_galerkin_matrix(lq, name, prec):
    """True P^dag D P (oracle O6): half storage, packed on the device, against the oracle's nine-block operator."""
    if name == "c3" and prec == "f64":
        pytest.skip("config 3 is fp32-only (BASELINE.json)")
    import torch
    prob = config_problem(name, 16 if name == "c2" else 1)
    cfg = prob.cfg
    A9 = to_dev(prob.A, prec)
    Ah = lq.pack_coarse_half(A9, cfg.cdims, cfg.nvec)
    assert Ah.shape == (cfg.cvolume, 5, 2 * cfg.nvec, 2 * cfg.nvec)
    assert torch.equal(Ah[:, 0], A9[:, 0]) and all(torch.equal(Ah[:, 1 + mu], A9[:, 1 + 2 * mu]) for mu in range(4))
    x = to_dev(prob.xc, prec)
    for dagger in (False, True):
        y = torch.full_like(x, 7.0)
        lq.coarse_mult_half(y, x, Ah, cfg.cdims, cfg.nvec, dagger=dagger)
        ref = oracle.coarse_mult(rounded(prob.xc, prec), rounded(prob.A, prec), cfg.cdims, dagger=dagger)
        assert rel_l2(y.cpu().numpy(), ref) <= TOL[prec], (name, prec, dagger)
        # and bit-reproducible: a second application gives the same bits (fixed summation order, no atomics)
        y2 = torch.empty_like(x)
        lq.coarse_mult_half(y2, x, Ah, cfg.cdims, cfg.nvec, dagger=dagger)
        assert torch.equal(y, y2)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("cdims,nvec", [
    ((2, 2, 2, 2), 4),     # coarse extent 2 everywhere: X + mu == X - mu
    ((3, 2, 5, 2), 1),     # N = 2: one vec16 (fp32) per row, odd extents
    ((4, 2, 2, 3), 3),     # odd nvec: a G5c sign change inside a vec16
    ((2, 4, 2, 2), 20),    # N = 40: ragged row (not a power of two)
    ((2, 2, 2, 2), 40),    # N = 80: several vec16 per lane per row
    ((6, 4, 4, 2), 32),    # the BASELINE block size N = 64
])
def test_half_storage_edge_sizes(lq, prec, cdims, nvec):
    rng = np.random.default_rng(1234 + nvec)
    Vc, n = int(np.prod(cdims)), 2 * nvec
    Ah = 0.1 * (rng.standard_normal((Vc, 5, n, n)) + 1j * rng.standard_normal((Vc, 5, n, n)))
    Ah[:, 0] += np.eye(n)
    xc = li.coarse_vector(rng, Vc, nvec)
    A9 = expand_half(rounded(Ah, prec), cdims, nvec)
    for dagger in (False, True):
        got = run_half(lq, Ah, xc, cdims, nvec, prec, dagger)
        ref = oracle.coarse_mult(rounded(xc, prec), A9, cdims, dagger=dagger)
        assert rel_l2(got, ref) <= TOL[prec], (cdims, nvec, prec, dagger)


def test_half_storage_equals_nine_block_kernel_on_device_built_operator(lq):
    """Config 3 with the operator bench.py times: clover, orthonormal null vectors and P^dag D P built by the device
    set-up (F2); the half-storage operator agrees with the nine-block kernel on the same matrix (both fp32)."""
    import torch
    cfg = li.CONFIGS["c3"]
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 9)
    U18 = lq.pack_gauge(li.t_gauge_field(cfg, gen, "cuda").to(torch.complex64), cfg.dims)
    clover = lq.clover_from_links(U18, cfg.kappa, cfg.csw, cfg.dims)
    v = torch.empty(lq.native_nullvecs_reals(cfg.dims, cfg.block, cfg.nvec), dtype=torch.float32, device="cuda")
    for i in range(cfg.nvec):
        lq.pack_nullvec(v, li.t_spinor(gen, cfg.volume, "cuda", torch.float32), i, cfg.dims, cfg.block, cfg.nvec)
    lq.orthonormalize_blocks(v, cfg.dims, cfg.block, cfg.nvec)
    assert lq.orthonormalize_degenerate_count() == 0
    A9 = lq.galerkin_coarse(U18, clover, v, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec)
    Ah = lq.pack_coarse_half(A9, cfg.cdims, cfg.nvec)
    x = li.t_coarse_vector(gen, cfg.cvolume, cfg.nvec, "cuda", torch.float32)
    y9, yh = torch.empty_like(x), torch.empty_like(x)
    for dagger in (False, True):
        lq.coarse_mult(y9, x, A9, cfg.cdims, cfg.nvec, dagger=dagger)
        lq.coarse_mult_half(yh, x, Ah, cfg.cdims, cfg.nvec, dagger=dagger)
        err = torch.linalg.vector_norm((yh - y9).to(torch.complex128)) / torch.linalg.vector_norm(y9.to(torch.complex128))
        # two fp32 evaluations of the same operator (the backward blocks of the device-built matrix carry their own
        # fp32 rounding): twice the single-application bar
        assert err.item() <= 2 * TOL["f32"], dagger


def test_half_storage_error_codes(lq):
    import torch
    prob = config_problem("c1")
    cfg = prob.cfg
    Ah = lq.pack_coarse_half(to_dev(prob.A, "f32"), cfg.cdims, cfg.nvec)
    x = to_dev(prob.xc, "f32")
    y = torch.empty_like(x)
    n0 = lq.launch_count()
    with pytest.raises(lq.LqcdError) as e:
        lq.coarse_mult_half(x, x, Ah, cfg.cdims, cfg.nvec)          # out aliases in
    assert e.value.code == lq.EINVAL
    with pytest.raises(ValueError, match="needs"):
        lq.coarse_mult_half(y, x, Ah[:-1], cfg.cdims, cfg.nvec)     # short matrix: refused by the binding
    with pytest.raises(ValueError, match="needs"):
        lq.coarse_mult_half(y, x, Ah, cfg.cdims, cfg.nvec, ws=torch.empty(64, dtype=torch.uint8, device="cuda"))
    ws = lq.coarse_half_workspace(cfg.cdims, cfg.nvec)
    st = torch.cuda.current_stream().cuda_stream
    rc = lq.lib().lqcd_coarse_mult_half_f32(y.data_ptr(), x.data_ptr(), Ah.data_ptr(), lq._i4((2, 2, 1, 2)), cfg.nvec, 0,
                                            ws.data_ptr(), st)
    assert rc == lq.EINVAL and "extent" in lq.lib().lqcd_last_error().decode()
    rc = lq.lib().lqcd_coarse_mult_half_f32(y.data_ptr(), x.data_ptr(), Ah.data_ptr(), lq._i4(cfg.cdims), cfg.nvec, 4,
                                            ws.data_ptr(), st)
    assert rc == lq.EINVAL, "unknown flag"
    assert lq.launch_count() == n0, "an erroring call must not enqueue anything"


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name", ["c1", "c2"])
def test_solvers_on_half_storage(lq, name, prec):
    """The coarse BiCGStab and the V-cycle with the coarse matrix in half storage against the oracle's solver on the
    nine-block Galerkin matrix (same recurrences; only the operator application differs)."""
    import torch
    from problems import check_bar
    from test_gpu_parity import Dev
    prob = config_problem(name, 16 if name == "c2" else 1)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    Ah = lq.pack_coarse_half(d.A, cfg.cdims, cfg.nvec)
    M = np.zeros((cfg.cvolume * 2 * cfg.nvec,) * 2, dtype=np.complex128) if cfg.cvolume * 2 * cfg.nvec <= 512 else None
    cond = 30.0
    if M is not None:  # dense D_c from the oracle's operator, for the principled bound
        n = M.shape[0]
        for j in range(n):
            e = np.zeros(n, dtype=np.complex128)
            e[j] = 1
            M[:, j] = oracle.coarse_mult(e.reshape(cfg.cvolume, 2, cfg.nvec), prob.A, cfg.cdims).ravel()
        cond = float(np.linalg.cond(M))
    b = to_dev(prob.xc, prec)
    for niter in (1, 5):
        x, r = torch.full_like(b, 3.0), torch.full_like(b, 3.0)
        lq.coarse_bicgstab(x, b, Ah, cfg.cdims, cfg.nvec, niter, r_out=r, half=True)
        rx, rr = oracle.coarse_bicgstab(rounded(prob.xc, prec), rounded(prob.A, prec), cfg.cdims, cfg.nvec, niter)
        check_bar(rel_l2(x.cpu().numpy(), rx), 2 * niter * cond * TOL[prec], prec, f"bicgstab half {name} {niter}")
        check_bar(np.linalg.norm(r.cpu().numpy() - rr) / np.linalg.norm(prob.xc), 2 * niter * cond * TOL[prec], prec,
                  f"bicgstab half residual {name} {niter}")
    n_coarse, n_sap, n_mr = 4, 2, 4
    bn = lq.pack_spinor(to_dev(prob.psi[0], prec), cfg.dims)
    xv = lq.empty_spinor(cfg.dims, dtype=bn.dtype)
    lq.mg_vcycle(xv, bn, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, cfg.nvec, d.v, Ah, n_coarse=n_coarse,
                 n_sap=n_sap, n_mr=n_mr, half=True)
    ref = oracle.mg_vcycle(rounded(prob.psi[0], prec), rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa,
                           cfg.dims, cfg.bc, cfg.block, rounded(prob.v, prec), rounded(prob.A, prec), n_coarse=n_coarse,
                           n_sap=n_sap, n_mr=n_mr)
    bar = (2 * n_coarse * cond + 2 + 2 * n_sap * (n_mr + 1)) * TOL[prec]
    check_bar(rel_l2(lq.unpack_spinor(xv, cfg.dims).cpu().numpy(), ref), bar, prec, f"vcycle half {name}")
