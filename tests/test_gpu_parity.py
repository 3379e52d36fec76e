"""Parity of the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element, on the same
seeded inputs (-m gpu).  Bars (BASELINE.json north_star): relative L2 per application <= 1e-12 in fp64 and
<= 2e-6 in fp32.  fp32 protocol (O9): every input is rounded to fp32 once, BOTH sides consume the
rounded values, the oracle promotes them and does all arithmetic in fp64.
"""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle
from problems import config_problem, custom_config, make_problem, rel_l2

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-6}
CDT = {"f64": np.complex128, "f32": np.complex64}


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2111_05012_b200 as lq  # raises if the CUDA library is missing: no fallback
    return lq


def to_dev(a, prec):
    import torch
    return torch.from_numpy(np.ascontiguousarray(np.asarray(a).astype(CDT[prec]))).cuda()


def rounded(a, prec):
    """the values both sides consume"""
    return np.ascontiguousarray(np.asarray(a).astype(CDT[prec]))


class Dev:
    """Device-resident native operator fields of a Problem in one precision."""

    def __init__(self, lq, prob, prec, links12=False, coarse=True):
        cfg = prob.cfg
        self.lq, self.prob, self.prec, self.cfg, self.links12 = lq, prob, prec, cfg, links12
        self.U = lq.pack_gauge(to_dev(prob.U, prec), cfg.dims, links12=links12)
        self.clover = lq.pack_clover(to_dev(prob.clover, prec), cfg.dims)
        self.v = self.A = None
        if coarse and prob.v is not None:
            self.v = lq.pack_nullvecs(to_dev(prob.v, prec), cfg.dims, cfg.block)
            self.A = to_dev(prob.A, prec)

    def D(self, psi, dagger=False):
        lq, cfg = self.lq, self.cfg
        x = lq.pack_spinor(to_dev(psi, self.prec), cfg.dims)
        y = lq.empty_spinor(cfg.dims, dtype=x.dtype)
        lq.wilson_clover_mult(y, x, self.U, self.clover, cfg.kappa, cfg.dims, cfg.bc, dagger=dagger,
                              links12=self.links12)
        return lq.unpack_spinor(y, cfg.dims).cpu().numpy()

    def Dsap(self, psi, domain, parity=0, dagger=False):
        lq, cfg = self.lq, self.cfg
        x = lq.pack_spinor(to_dev(psi, self.prec), cfg.dims)
        y = lq.empty_spinor(cfg.dims, dtype=x.dtype)
        y.fill_(7.0)  # the kernel must overwrite every site, also the zeroed ones of the other domain group
        lq.wilson_clover_dd_mult(y, x, self.U, self.clover, cfg.kappa, cfg.dims, cfg.bc, domain, parity=parity,
                                 dagger=dagger, links12=self.links12)
        return lq.unpack_spinor(y, cfg.dims).cpu().numpy()

    def Dc(self, xc, dagger=False):
        import torch
        x = to_dev(xc, self.prec)
        y = torch.empty_like(x)
        self.lq.coarse_mult(y, x, self.A, self.cfg.cdims, self.cfg.nvec, dagger=dagger)
        return y.cpu().numpy()

    def R(self, psi):
        import torch
        lq, cfg = self.lq, self.cfg
        x = lq.pack_spinor(to_dev(psi, self.prec), cfg.dims)
        y = torch.empty((cfg.cvolume, 2, cfg.nvec), dtype=to_dev(np.zeros(1), self.prec).dtype, device="cuda")
        lq.restrict(y, x, self.v, cfg.dims, cfg.block, cfg.nvec)
        return y.cpu().numpy()

    def P(self, xc):
        lq, cfg = self.lq, self.cfg
        x = to_dev(xc, self.prec)
        y = lq.empty_spinor(cfg.dims, dtype=self.U.dtype)
        lq.prolong(y, x, self.v, cfg.dims, cfg.block, cfg.nvec)
        return lq.unpack_spinor(y, cfg.dims).cpu().numpy()


def oracle_D(prob, psi, prec, dagger=False):
    cfg = prob.cfg
    return oracle.wilson_clover_mult(rounded(psi, prec), rounded(prob.U, prec), rounded(prob.clover, prec), cfg.kappa,
                                     cfg.dims, cfg.bc, dagger=dagger)


# ------------------------------------------------------------------------------------------------------
# layout helpers: bit-exact round trips
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 5, 2, 7), (6, 4, 2, 10)])
def test_pack_unpack_spinor_roundtrip(lq, prec, dims):
    rng = np.random.default_rng(5)
    psi = rounded(li.spinor(rng, int(np.prod(dims))), prec)
    back = lq.unpack_spinor(lq.pack_spinor(to_dev(psi, prec), dims), dims).cpu().numpy()
    assert np.array_equal(back, psi)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_pack_unpack_nullvec_roundtrip(lq, prec):
    dims, block, nvec = (8, 4, 4, 6), (4, 2, 2, 3), 3
    rng = np.random.default_rng(6)
    v = rounded(li.null_vectors(rng, nvec, int(np.prod(dims))), prec)
    nat = lq.pack_nullvecs(to_dev(v, prec), dims, block)
    for i in range(nvec):
        assert np.array_equal(lq.unpack_nullvec(nat, i, dims, block, nvec).cpu().numpy(), v[i])


# ------------------------------------------------------------------------------------------------------
# config 1: every row, fp64 and fp32
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("links12", [False, True])
@pytest.mark.parametrize("dagger", [False, True])
def test_c1_wilson_clover(lq, prec, links12, dagger):
    prob = config_problem("c1")
    d = Dev(lq, prob, prec, links12=links12, coarse=False)
    got = d.D(prob.psi[0], dagger=dagger)
    ref = oracle_D(prob, prob.psi[0], prec, dagger=dagger)
    assert rel_l2(got, ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dagger", [False, True])
def test_c1_coarse(lq, prec, dagger):
    prob = config_problem("c1")
    d = Dev(lq, prob, prec)
    got = d.Dc(prob.xc, dagger=dagger)
    ref = oracle.coarse_mult(rounded(prob.xc, prec), rounded(prob.A, prec), prob.cfg.cdims, dagger=dagger)
    assert rel_l2(got, ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_c1_restrict_prolong(lq, prec):
    prob = config_problem("c1")
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    got = d.R(prob.psi[0])
    ref = oracle.restrict(rounded(prob.psi[0], prec), rounded(prob.v, prec), cfg.dims, cfg.block)
    assert rel_l2(got, ref) <= TOL[prec]
    got = d.P(prob.xc)
    ref = oracle.prolong(rounded(prob.xc, prec), rounded(prob.v, prec), cfg.dims, cfg.block)
    assert rel_l2(got, ref) <= TOL[prec]


# ------------------------------------------------------------------------------------------------------
# F1: domain-decomposed operator D_SAP, all / even / odd domain groups
# ------------------------------------------------------------------------------------------------------
def oracle_Dsap(prob, psi, prec, domain, parity=0, dagger=False):
    cfg = prob.cfg
    return oracle.wilson_clover_dd_mult(rounded(psi, prec), rounded(prob.U, prec), rounded(prob.clover, prec),
                                        cfg.kappa, cfg.dims, cfg.bc, domain, parity=parity, dagger=dagger)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("links12", [False, True])
def test_c1_dsap(lq, prec, links12):
    prob = config_problem("c1")
    cfg = prob.cfg
    d = Dev(lq, prob, prec, links12=links12, coarse=False)
    psi = prob.psi[0]
    for parity in (0, 1, 2):
        for dagger in (False, True):
            got = d.Dsap(psi, cfg.block, parity=parity, dagger=dagger)
            ref = oracle_Dsap(prob, psi, prec, cfg.block, parity=parity, dagger=dagger)
            assert rel_l2(got, ref) <= TOL[prec], (parity, dagger)
            assert np.array_equal(got == 0, ref == 0), "exact zeros on the domains of the other group"
    # one domain spanning the lattice: D_SAP is D, bit for bit
    assert np.array_equal(d.Dsap(psi, cfg.dims), d.D(psi))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,domain,bc", [
    ((8, 8, 8, 8), (4, 4, 4, 4), (1, 1, 1, -1)),       # config 2's lattice and domains
    ((16, 8, 8, 8), (8, 4, 4, 4), (1, 1, 1, -1)),      # the paper's 8x4x4x4 domain
    ((6, 4, 2, 10), (3, 4, 1, 5), (-1, 1, -1, 1)),     # odd domains, single domain in y, one-site domains in z
    ((3, 3, 3, 3), (3, 1, 3, 1), (1, 1, 1, -1)),       # V = 81: ragged chunk
])
def test_dsap_edge_lattices(lq, prec, dims, domain, bc):
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc)
    prob = make_problem(cfg, coarse="none")
    d = Dev(lq, prob, prec, coarse=False)
    for parity, dagger in ((0, False), (1, True), (2, False)):
        got = d.Dsap(prob.psi[0], domain, parity=parity, dagger=dagger)
        ref = oracle_Dsap(prob, prob.psi[0], prec, domain, parity=parity, dagger=dagger)
        assert rel_l2(got, ref) <= TOL[prec], (parity, dagger)
        assert np.array_equal(got == 0, ref == 0)


# ------------------------------------------------------------------------------------------------------
# config 2: 8^4, block 4^4, nvec 16, fp32, 16 right-hand sides one at a time
# ------------------------------------------------------------------------------------------------------
def test_c2_sixteen_rhs(lq):
    prec = "f32"
    prob = config_problem("c2", 16)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    rng = np.random.default_rng(77)
    for k, psi in enumerate(prob.psi):
        assert rel_l2(d.D(psi), oracle_D(prob, psi, prec)) <= TOL[prec], f"D rhs {k}"
        xc = li.coarse_vector(rng, cfg.cvolume, cfg.nvec)
        ref = oracle.coarse_mult(rounded(xc, prec), rounded(prob.A, prec), cfg.cdims)
        assert rel_l2(d.Dc(xc), ref) <= TOL[prec], f"D_c rhs {k}"
    psi = prob.psi[3]
    assert rel_l2(d.D(psi, dagger=True), oracle_D(prob, psi, prec, dagger=True)) <= TOL[prec]
    assert rel_l2(d.R(psi), oracle.restrict(rounded(psi, prec), rounded(prob.v, prec), cfg.dims, cfg.block)) <= TOL[prec]
    assert rel_l2(d.P(prob.xc), oracle.prolong(rounded(prob.xc, prec), rounded(prob.v, prec), cfg.dims, cfg.block)) <= \
        TOL[prec]


# ------------------------------------------------------------------------------------------------------
# config 3: 16^3 x 32, Haar links, nvec 32, true Galerkin A; restrict -> coarse_mult -> prolong chained on the
# device as in a V-cycle (row A6), no host copies between the three kernels
# ------------------------------------------------------------------------------------------------------
def test_c3_vcycle_chain(lq):
    import torch
    prec = "f32"
    prob = config_problem("c3")
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    psi = prob.psi[0]
    # each step against the oracle on the same (rounded) input
    assert rel_l2(d.D(psi), oracle_D(prob, psi, prec)) <= TOL[prec]
    v32, A32 = rounded(prob.v, prec), rounded(prob.A, prec)
    r_ref = oracle.restrict(rounded(psi, prec), v32, cfg.dims, cfg.block)
    assert rel_l2(d.R(psi), r_ref) <= TOL[prec]
    c_ref = oracle.coarse_mult(rounded(prob.xc, prec), A32, cfg.cdims)
    assert rel_l2(d.Dc(prob.xc), c_ref) <= TOL[prec]
    p_ref = oracle.prolong(rounded(prob.xc, prec), v32, cfg.dims, cfg.block)
    assert rel_l2(d.P(prob.xc), p_ref) <= TOL[prec]
    # the chain, device-resident; the oracle chain runs in fp64 from the same fp32 input, so the bar is three
    # applications' worth of fp32 rounding
    x = lq.pack_spinor(to_dev(psi, prec), cfg.dims)
    xc = torch.empty((cfg.cvolume, 2, cfg.nvec), dtype=torch.complex64, device="cuda")
    yc = torch.empty_like(xc)
    y = lq.empty_spinor(cfg.dims)
    n0 = lq.launch_count()
    lq.restrict(xc, x, d.v, cfg.dims, cfg.block, cfg.nvec)
    lq.coarse_mult(yc, xc, d.A, cfg.cdims, cfg.nvec)
    lq.prolong(y, yc, d.v, cfg.dims, cfg.block, cfg.nvec)
    assert lq.launch_count() - n0 == 3
    got = lq.unpack_spinor(y, cfg.dims).cpu().numpy()
    ref = oracle.prolong(oracle.coarse_mult(r_ref, prob.A.astype(np.complex64).astype(np.complex128), cfg.cdims),
                         v32.astype(np.complex128), cfg.dims, cfg.block)
    assert rel_l2(got, ref) <= 3 * TOL[prec]


# ------------------------------------------------------------------------------------------------------
# edge cases: odd / ragged lattices (V not a multiple of 32), other boundary conditions, odd nvec, 8x4x4x4
# blocks (the paper's production block), coarse extent 2 with X+mu == X-mu
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,bc", [
    ((3, 3, 3, 3), (1, 1, 1, -1)),       # V = 81: ragged last chunk, no power-of-two tile
    ((6, 4, 2, 10), (-1, 1, -1, 1)),     # extent 2 (x+mu == x-mu), mixed boundary conditions
    ((2, 2, 2, 2), (-1, -1, -1, -1)),    # smallest lattice, all antiperiodic
    ((16, 4, 4, 4), (1, 1, 1, 1)),       # all periodic
])
def test_wilson_clover_edge_lattices(lq, prec, dims, bc):
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc)
    prob = make_problem(cfg, coarse="none")
    for links12 in (False, True):
        d = Dev(lq, prob, prec, links12=links12, coarse=False)
        for dagger in (False, True):
            got = d.D(prob.psi[0], dagger=dagger)
            assert rel_l2(got, oracle_D(prob, prob.psi[0], prec, dagger=dagger)) <= TOL[prec]


def _random_lattices(n, seed):
    """Seeded lattice shapes for the sweep below: extents 2..12, volume <= 6000 (the oracle stays fast); about half of
    them satisfy 4 | Lx, 4 | Ly, 2 | Lz (tiled native site order, a warp per layout tile), the others fall back to the
    canonical order with ragged chunks."""
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        if len(out) % 2 == 0:
            dims = (int(rng.choice([4, 8, 12])), int(rng.choice([4, 8])), int(rng.choice([2, 4, 6])),
                    int(rng.integers(2, 9)))
        else:
            dims = tuple(int(rng.integers(2, 8)) for _ in range(4))
        if int(np.prod(dims)) > 6000:
            continue
        bc = tuple(int(b) for b in rng.choice([1, -1], size=4))
        domain = tuple(int(rng.choice([d for d in range(1, L + 1) if L % d == 0])) for L in dims)
        tile = tuple(int(rng.choice([d for d in (1, 2, 4) if L % d == 0])) for L in dims)
        out.append((dims, bc, domain, tile, bool(rng.integers(2)), bool(rng.integers(2)), int(rng.integers(3))))
    return out


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("case", _random_lattices(10, 20211105), ids=lambda c: "x".join(map(str, c[0])))
def test_wilson_clover_random_lattices(lq, prec, case):
    """D, D^dag and D_SAP (all / even / odd domains) on seeded random lattice shapes, boundary conditions, domains,
    link storage and CTA tiles against the oracle: every index-decode path of the fine kernels (tiled and canonical
    site order, a warp per layout tile or not, automatic and user tiles)."""
    dims, bc, domain, tile, links12, dagger, parity = case
    cfg = custom_config(dims, (1, 1, 1, 1), 1, bc=bc)
    prob = make_problem(cfg, coarse="none")
    d = Dev(lq, prob, prec, links12=links12, coarse=False)
    psi = prob.psi[0]
    try:
        for user_tile in (None, tile):
            lq.set_fine_tile(user_tile)
            got = d.D(psi, dagger=dagger)
            assert rel_l2(got, oracle_D(prob, psi, prec, dagger=dagger)) <= TOL[prec], (case, user_tile)
            got = d.Dsap(psi, domain, parity=parity, dagger=dagger)
            ref = oracle_Dsap(prob, psi, prec, domain, parity=parity, dagger=dagger)
            assert rel_l2(got, ref) <= TOL[prec], (case, user_tile)
            assert np.array_equal(got == 0, ref == 0), (case, user_tile)
    finally:
        lq.set_fine_tile(None)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,block,nvec", [
    ((16, 8, 8, 8), (8, 4, 4, 4), 4),    # the paper's 8x4x4x4 block; coarse 2^4
    ((4, 6, 4, 6), (2, 3, 2, 2), 3),     # odd nvec, non-power-of-two block
    ((4, 4, 4, 8), (2, 2, 2, 2), 1),     # nvec = 1 (N = 2)
    ((8, 4, 4, 4), (2, 2, 2, 2), 20),    # N = 40: rows not a power of two
    ((4, 4, 4, 4), (2, 2, 2, 2), 40),    # N = 80 > 64: several vec16 per lane per row
    ((4, 4, 8, 4), (4, 4, 4, 4), 5),     # one aggregate thick in x, y, t (coarse 1x1x2x1): the transfers only
])
def test_coarse_and_transfer_edge_sizes(lq, prec, dims, block, nvec):
    cfg = custom_config(dims, block, nvec)
    thin = min(cfg.cdims) < 2    # aggregate-local operations accept it; the coarse stencil does not (Q8)
    prob = make_problem(cfg, coarse="galerkin" if nvec <= 4 else "synthetic")
    d = Dev(lq, prob, prec)
    psi = prob.psi[0]
    v, A = rounded(prob.v, prec), rounded(prob.A, prec)
    for dagger in (False, True):
        if thin:
            with pytest.raises(lq.LqcdError):
                d.Dc(prob.xc, dagger=dagger)
            continue
        ref = oracle.coarse_mult(rounded(prob.xc, prec), A, cfg.cdims, dagger=dagger)
        assert rel_l2(d.Dc(prob.xc, dagger=dagger), ref) <= TOL[prec]
    assert rel_l2(d.R(psi), oracle.restrict(rounded(psi, prec), v, cfg.dims, cfg.block)) <= TOL[prec]
    assert rel_l2(d.P(prob.xc), oracle.prolong(rounded(prob.xc, prec), v, cfg.dims, cfg.block)) <= TOL[prec]


def _random_coarse_sizes(n, seed):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        block = tuple(int(rng.choice([1, 2, 3, 4])) for _ in range(4))
        cdims = tuple(int(rng.integers(2, 5)) for _ in range(4))
        dims = tuple(b * c for b, c in zip(block, cdims))
        nvec = int(rng.choice([1, 2, 3, 5, 7, 8, 12, 16, 17, 24, 32, 33]))
        bvol, cvol = int(np.prod(block)), int(np.prod(cdims))
        if bvol < 2 or bvol * cvol > 6000 or cvol * nvec * nvec > 60000:
            continue
        out.append((dims, block, nvec))
    return out


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("dims,block,nvec", _random_coarse_sizes(8, 5012),
                         ids=lambda v: "x".join(map(str, v)) if isinstance(v, tuple) else str(v))
def test_coarse_and_transfer_random_sizes(lq, prec, dims, block, nvec):
    """coarse_mult (and its dagger), restrict and prolong on seeded random block shapes, coarse extents 2..4 and numbers
    of null vectors (rows spread over part of a warp, one warp, several vec16 per lane; ragged aggregates)."""
    cfg = custom_config(dims, block, nvec)
    prob = make_problem(cfg, coarse="synthetic")
    d = Dev(lq, prob, prec)
    v, A = rounded(prob.v, prec), rounded(prob.A, prec)
    for dagger in (False, True):
        ref = oracle.coarse_mult(rounded(prob.xc, prec), A, cfg.cdims, dagger=dagger)
        assert rel_l2(d.Dc(prob.xc, dagger=dagger), ref) <= TOL[prec], dagger
    psi = prob.psi[0]
    assert rel_l2(d.R(psi), oracle.restrict(rounded(psi, prec), v, cfg.dims, cfg.block)) <= TOL[prec]
    assert rel_l2(d.P(prob.xc), oracle.prolong(rounded(prob.xc, prec), v, cfg.dims, cfg.block)) <= TOL[prec]


def test_results_do_not_depend_on_tuning_knobs(lq):
    prob = config_problem("c2", 16)
    d = Dev(lq, prob, "f32")
    base = d.D(prob.psi[0])
    base_c = d.Dc(prob.xc)
    try:
        for tile in [(8, 4, 4, 1), (4, 4, 4, 4), (8, 8, 2, 2), (2, 2, 2, 2), (8, 1, 1, 1)]:
            lq.set_fine_tile(tile)
            assert np.array_equal(d.D(prob.psi[0]), base), tile
        lq.set_fine_tile(None)
        lq.set_knob("fine_tslab", 1)
        assert np.array_equal(d.D(prob.psi[0]), base)
        for rpw in (1, 2, 4):
            lq.set_knob("coarse_rows_per_warp", rpw)
            assert np.array_equal(d.Dc(prob.xc), base_c)
    finally:
        lq.set_fine_tile(None)
        lq.set_knob("fine_tslab", 0)
        lq.set_knob("coarse_rows_per_warp", 0)


# ------------------------------------------------------------------------------------------------------
# error behaviour of the C ABI (nothing is enqueued on error)
# ------------------------------------------------------------------------------------------------------
def test_error_codes(lq):
    import torch
    prob = config_problem("c1")
    cfg = prob.cfg
    d = Dev(lq, prob, "f32")
    x = lq.pack_spinor(to_dev(prob.psi[0], "f32"), cfg.dims)
    y = lq.empty_spinor(cfg.dims)
    n0 = lq.launch_count()

    def code(fn):
        with pytest.raises(lq.LqcdError) as e:
            fn()
        return e.value.code

    assert code(lambda: lq.wilson_clover_mult(x, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc)) == lq.EINVAL
    assert code(lambda: lq.wilson_clover_mult(y, x, d.U, d.clover, cfg.kappa, cfg.dims, (1, 1, 1, 0))) == lq.EINVAL
    assert code(lambda: lq.wilson_clover_mult(y, x, d.U, d.clover, cfg.kappa, (4, 4, 4, 0), cfg.bc)) == lq.EINVAL
    # a tensor of the wrong size never reaches the C call (the binding knows the sizes, tests/test_binding_checks.py) ...
    with pytest.raises(ValueError, match="needs"):
        lq.wilson_clover_mult(y[1:], x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc)
    # ... and the C call itself refuses a pointer that is not 16-byte aligned
    i4, st = lq._i4, torch.cuda.current_stream().cuda_stream
    rc = lq.lib().lqcd_wilson_clover_mult_f32(y.data_ptr() + 4, x.data_ptr(), d.U.data_ptr(), d.clover.data_ptr(),
                                              cfg.kappa, i4(cfg.dims), i4(cfg.bc), 0, st)
    assert rc == lq.EINVAL and "aligned" in lq.lib().lqcd_last_error().decode()
    xc = to_dev(prob.xc, "f32")
    yc = torch.empty_like(xc)
    with pytest.raises(ValueError, match="needs"):
        lq.coarse_mult(yc, xc, d.A, (2, 2, 2, 1), cfg.nvec)
    rc = lq.lib().lqcd_coarse_mult_f32(yc.data_ptr(), xc.data_ptr(), d.A.data_ptr(), i4((2, 2, 2, 1)), cfg.nvec, 0, st)
    assert rc == lq.EINVAL, "the 9-point coarse stencil needs coarse extents >= 2 (DESIGN.md Q8)"
    assert code(lambda: lq.coarse_mult(xc, xc, d.A, cfg.cdims, cfg.nvec)) == lq.EINVAL
    assert code(lambda: lq.restrict(yc, x, d.v, cfg.dims, (3, 2, 2, 2), cfg.nvec)) == lq.EINVAL
    assert code(lambda: lq.prolong(y, yc, d.v, cfg.dims, cfg.block, 0)) == lq.EINVAL
    assert "lqcd_prolong_f32" in lq.last_error()
    dd = lambda **kw: lq.wilson_clover_dd_mult(y, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, **kw)
    assert code(lambda: dd(domain=(3, 2, 2, 2))) == lq.EINVAL          # does not divide
    assert code(lambda: dd(domain=(2, 2, 2, 0))) == lq.EINVAL
    rc = lq.lib().lqcd_wilson_clover_dd_mult_f32(y.data_ptr(), x.data_ptr(), d.U.data_ptr(), d.clover.data_ptr(),
                                                 cfg.kappa, lq._i4(cfg.dims), lq._i4(cfg.bc), lq._i4(cfg.block),
                                                 lq.DOMAIN_EVEN | lq.DOMAIN_ODD, None)
    assert rc == lq.EINVAL, "even and odd at once"
    rc = lq.lib().lqcd_wilson_clover_mult_f32(y.data_ptr(), x.data_ptr(), d.U.data_ptr(), d.clover.data_ptr(),
                                              cfg.kappa, lq._i4(cfg.dims), lq._i4(cfg.bc), lq.DOMAIN_EVEN, None)
    assert rc == lq.EINVAL, "domain flags are not accepted by the plain operator"
    assert lq.launch_count() == n0, "an erroring call must not enqueue anything"
    with pytest.raises(ValueError):
        lq.wilson_clover_mult(y.cpu(), x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc)  # no CPU path


# ------------------------------------------------------------------------------------------------------
# host-vector entry points give the same numbers as the device-pointer ones
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_host_entry_points(lq, prec):
    import torch
    prob = config_problem("c2", 16)
    cfg = prob.cfg
    d = Dev(lq, prob, prec)
    rdt = torch.float32 if prec == "f32" else torch.float64
    ws = torch.empty(lq.host_workspace_bytes(cfg.dims, cfg.block, cfg.nvec, dtype=rdt), dtype=torch.uint8,
                     device="cuda")
    psi = torch.from_numpy(rounded(prob.psi[0], prec)).pin_memory()
    out = torch.empty_like(psi).pin_memory()
    lq.wilson_clover_mult_host(out, psi, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, ws)
    assert np.array_equal(out.numpy(), d.D(prob.psi[0]))
    lq.wilson_clover_mult_host(out, psi, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, ws, dagger=True)
    assert np.array_equal(out.numpy(), d.D(prob.psi[0], dagger=True))
    xc = torch.from_numpy(rounded(prob.xc, prec)).pin_memory()
    yc = torch.empty_like(xc).pin_memory()
    with pytest.raises(TypeError):  # host and device data of one call share one precision
        lq.coarse_mult_host(yc.to(torch.complex64 if prec == "f64" else torch.complex128), xc, d.A, cfg.cdims,
                            cfg.nvec, ws)
    lq.coarse_mult_host(yc, xc, d.A, cfg.cdims, cfg.nvec, ws)
    assert np.array_equal(yc.numpy(), d.Dc(prob.xc))
    lq.restrict_host(yc, psi, d.v, cfg.dims, cfg.block, cfg.nvec, ws)
    assert np.array_equal(yc.numpy(), d.R(prob.psi[0]))
    lq.prolong_host(out, xc, d.v, cfg.dims, cfg.block, cfg.nvec, ws)
    assert np.array_equal(out.numpy(), d.P(prob.xc))


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("dims,block", [((16, 16, 8, 24), (4, 4, 4, 4)), ((8, 8, 8, 36), (4, 4, 2, 3)),
                                        ((10, 10, 10, 36), (5, 5, 2, 3))])
def test_host_entry_points_slab_pipeline(lq, prec, dims, block):
    """A host vector travels in slabs of time slices: upload of slab k + 1 under pack / kernel / unpack of slab k under
    the download of slab k - 1 (host_api.cu; knob host_slab_mb sets the smallest slab, -1 the one-shot path).  The
    kernels are the same ones on a range of tiles / aggregates, so every result is bit-identical with the one-shot
    path and with the device-pointer calls; the launch counts show that the pipeline was taken.  Random native operator
    fields (the comparison is between paths, not against the oracle); (10, 10, 10, 36): canonical site order."""
    import torch
    nvec = 4
    rdt = torch.float32 if prec == "f32" else torch.float64
    cd = tuple(d // b for d, b in zip(dims, block))
    V, Vc = int(np.prod(dims)), int(np.prod(cd))
    g = torch.Generator(device="cuda")
    g.manual_seed(7)
    rnd = lambda n, s=1.0: torch.randn(n, generator=g, device="cuda", dtype=rdt) * s
    bc = (1, 1, 1, -1)
    U, U12 = rnd(lq.native_gauge_reals(dims)), rnd(lq.native_gauge_reals(dims, links12=True))
    clov, v = rnd(lq.native_clover_reals(dims), 0.1), rnd(lq.native_nullvecs_reals(dims, block, nvec))
    ws = torch.empty(lq.host_workspace_bytes(dims, block, nvec, dtype=rdt), dtype=torch.uint8, device="cuda")
    x_h = torch.randn((V, 4, 3, 2), dtype=rdt).pin_memory()
    xc_h = torch.randn((Vc, 2, nvec, 2), dtype=rdt).pin_memory()
    xn = lq.pack_spinor(x_h.cuda(), dims)
    # device-pointer results, canonical
    ref = {}
    for key, kw in (("D", {}), ("Ddag", {"dagger": True}), ("D12", {"links12": True})):
        y = lq.empty_spinor(dims, dtype=rdt)
        lq.wilson_clover_mult(y, xn, U12 if kw.get("links12") else U, clov, 0.13, dims, bc, **kw)
        ref[key] = torch.view_as_real(lq.unpack_spinor(y, dims)).cpu()
    yc = torch.zeros((Vc, 2, nvec, 2), dtype=rdt, device="cuda")
    lq.restrict(yc, xn, v, dims, block, nvec)
    ref["R"] = yc.cpu()
    y = lq.empty_spinor(dims, dtype=rdt)
    lq.prolong(y, xc_h.cuda(), v, dims, block, nvec)
    ref["P"] = torch.view_as_real(lq.unpack_spinor(y, dims)).cpu()
    launches = {}
    for knob in (1, -1):  # slabs of >= 1 MB / one-shot
        lq.set_knob("host_slab_mb", knob)
        try:
            out = torch.zeros_like(x_h).pin_memory()
            n0 = lq.launch_count()
            lq.wilson_clover_mult_host(out, x_h, U, clov, 0.13, dims, bc, ws)
            launches[knob] = lq.launch_count() - n0
            assert torch.equal(out, ref["D"]), knob
            lq.wilson_clover_mult_host(out, x_h, U, clov, 0.13, dims, bc, ws, dagger=True)
            assert torch.equal(out, ref["Ddag"]), knob
            lq.wilson_clover_mult_host(out, x_h, U12, clov, 0.13, dims, bc, ws, links12=True)
            assert torch.equal(out, ref["D12"]), knob
            oc = torch.zeros_like(xc_h).pin_memory()
            lq.restrict_host(oc, x_h, v, dims, block, nvec, ws)
            assert torch.equal(oc, ref["R"]), knob
            out.zero_()
            lq.prolong_host(out, xc_h, v, dims, block, nvec, ws)
            assert torch.equal(out, ref["P"]), knob
            # pageable host memory (the copies then block the host; the order of the pipeline still holds)
            xp, op = x_h.clone(), torch.zeros((V, 4, 3, 2), dtype=rdt)
            assert not xp.is_pinned() and not op.is_pinned()
            lq.wilson_clover_mult_host(op, xp, U, clov, 0.13, dims, bc, ws)
            assert torch.equal(op, ref["D"]), knob
        finally:
            lq.set_knob("host_slab_mb", 0)
    assert launches[-1] == 3
    slab_big_enough = V * 24 * x_h.element_size() >= 3 * (1 << 20)
    if slab_big_enough:
        assert launches[1] >= 9, "the slab pipeline was not taken"


# ------------------------------------------------------------------------------------------------------
# the native site order (tiled 4 x 4 x 2 chunks) is invisible through pack / unpack: the same
# canonical fields packed in canonical order (knob site_order = -1) give the same bits
# ------------------------------------------------------------------------------------------------------
def test_results_do_not_depend_on_the_site_order(lq):
    import torch
    prob = config_problem("c2", 16)
    cfg = prob.cfg
    assert cfg.dims[0] % 4 == 0 and cfg.dims[1] % 4 == 0 and cfg.dims[2] % 2 == 0, "config 2 takes the tiled order"
    outs = {}
    try:
        for order in (0, -1):
            lq.set_knob("site_order", order)
            d = Dev(lq, prob, "f32")                       # packs U, clover, null vectors in this order
            x = lq.pack_spinor(to_dev(prob.psi[0], "f32"), cfg.dims)
            r = lq.pack_spinor(to_dev(prob.psi[1], "f32"), cfg.dims)
            z = lq.empty_spinor(cfg.dims)
            lq.mr_domain_solve(z, r, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, parity=2, niter=3)
            xs, rs = lq.empty_spinor(cfg.dims), lq.empty_spinor(cfg.dims)
            lq.sap(xs, rs, x, d.U, d.clover, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=3)
            outs[order] = dict(
                D=d.D(prob.psi[0]), Ddag=d.D(prob.psi[0], dagger=True), Dsap=d.Dsap(prob.psi[0], cfg.block, parity=1),
                R=d.R(prob.psi[0]), P=d.P(prob.xc), mr=lq.unpack_spinor(z, cfg.dims).cpu().numpy(),
                sap=lq.unpack_spinor(xs, cfg.dims).cpu().numpy(), packed=x.cpu().numpy())
    finally:
        lq.set_knob("site_order", 0)
    assert not np.array_equal(outs[0]["packed"], outs[-1]["packed"]), "the two orders are different native layouts"
    for k in ("D", "Ddag", "Dsap", "R", "P", "mr", "sap"):
        assert np.array_equal(outs[0][k], outs[-1][k]), k
