"""Parity at BASELINE.json's full sizes (configs 4 and 5), in the launch configuration bench.py times (default
knobs), on SAMPLED outputs the oracle computes one by one, plus properties that hold at any size (-m gpu).

Inputs are generated on the device with the seeded generators of lqcd_inputs.py; the
oracle gets the very same fp32 values:
  * fine operator: time-slabs of the canonical fields are copied into lazily-committed full-size host arrays
    (only the touched pages exist), the oracle's *_sites entry point evaluates Eq. 1 at sampled sites whose
    neighbours all lie in those slabs (both t boundaries, the lattice corners and the bulk are covered);
  * coarse operator: the oracle's *_sites entry point takes only the nine blocks of the sampled coarse sites;
  * restrict / prolong are aggregate-local, so 16 sampled aggregates are gathered into a fake 8^4 lattice of
    4^4 blocks on which the oracle runs as it stands.
"""
import numpy as np
import pytest

import lqcd_inputs as li
import oracle

pytestmark = pytest.mark.gpu
TOL32 = 2e-6


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def site_index(dims, c):
    return c[..., 0] + dims[0] * (c[..., 1] + dims[1] * (c[..., 2] + dims[2] * c[..., 3]))


def sample_fine_sites(cfg, rng, n):
    """sites with t in {0, 1, Lt/2, Lt-1} (both sides of the antiperiodic boundary and the bulk) + the corners"""
    L = np.array(cfg.dims)
    ts = np.array([0, 1, L[3] // 2, L[3] - 1])
    c = np.stack([rng.integers(0, L[0], n), rng.integers(0, L[1], n), rng.integers(0, L[2], n),
                  ts[rng.integers(0, len(ts), n)]], axis=1)
    corners = np.array([[x, y, z, t] for x in (0, L[0] - 1) for y in (0, L[1] - 1) for z in (0, L[2] - 1)
                        for t in (0, L[3] - 1)])
    c = np.concatenate([corners, c])
    slabs = sorted({int(v) % int(L[3]) for t in ts for v in (t - 1, t, t + 1)})
    return site_index(cfg.dims, c).astype(np.int64), slabs


def lazily_filled(shape, dtype, dev_tensor, slabs, v3, site_axis):
    """full-size host array (uninitialised, pages committed on touch) holding only the given time-slabs"""
    host = np.empty(shape, dtype=dtype)
    for t in slabs:
        sl = [slice(None)] * len(shape)
        sl[site_axis] = slice(t * v3, (t + 1) * v3)
        host[tuple(sl)] = dev_tensor[tuple(sl)].cpu().numpy()
    return host


@pytest.fixture(scope="module")
def lq():
    import torch
    assert torch.cuda.is_available()
    import paper_2111_05012_b200 as lq
    return lq


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_wilson_clover_sampled(lq, name):
    import torch
    cfg = li.CONFIGS[name]
    V, L = cfg.volume, cfg.dims
    v3 = L[0] * L[1] * L[2]
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed)
    U = li.t_gauge_field(cfg, gen, "cuda").to(torch.complex64)
    cl = li.t_clover_synthetic(gen, V, "cuda")
    psi = li.t_spinor(gen, V, "cuda", torch.float32)
    chi = li.t_spinor(gen, V, "cuda", torch.float32)
    U18, U12 = lq.pack_gauge(U, L), lq.pack_gauge(U, L, links12=True)
    Cn = lq.pack_clover(cl, L)
    x, w = lq.pack_spinor(psi, L), lq.pack_spinor(chi, L)
    y = lq.empty_spinor(L)

    rng = np.random.default_rng(cfg.seed)
    sites, slabs = sample_fine_sites(cfg, rng, 3000)
    U_h = lazily_filled((4, V, 3, 3), np.complex64, U, slabs, v3, 1)
    cl_h = lazily_filled((V, 2, 6, 6), np.complex64, cl, slabs, v3, 0)
    psi_h = lazily_filled((V, 4, 3), np.complex64, psi, slabs, v3, 0)
    sites_d = torch.from_numpy(sites).cuda()

    results = {}
    for label, Un, dag, l12 in (("D", U18, False, False), ("Ddag", U18, True, False), ("D_links12", U12, False, True)):
        lq.wilson_clover_mult(y, x, Un, Cn, cfg.kappa, L, cfg.bc, dagger=dag, links12=l12)
        yc = lq.unpack_spinor(y, L)
        got = yc[sites_d].cpu().numpy()
        ref = oracle.wilson_clover_mult_sites(psi_h, U_h, cl_h, cfg.kappa, L, cfg.bc, sites, dagger=dag)
        assert np.isfinite(got).all()
        assert rel_l2(got, ref) <= TOL32, label
        # no sampled site is individually off either (catches a wrong neighbour at a single boundary site)
        per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(
            ref.reshape(len(sites), -1), axis=1)
        assert per_site.max() <= 5 * TOL32, (label, int(sites[per_site.argmax()]))
        results[label] = yc
    # F1: D_SAP with the aggregation block as domain, all domains and the even group
    for parity, dag in ((0, False), (1, True), (2, False)):
        lq.wilson_clover_dd_mult(y, x, U18, Cn, cfg.kappa, L, cfg.bc, cfg.block, parity=parity, dagger=dag)
        got = lq.unpack_spinor(y, L)[sites_d].cpu().numpy()
        ref = oracle.wilson_clover_dd_mult_sites(psi_h, U_h, cl_h, cfg.kappa, L, cfg.bc, cfg.block, sites,
                                                 parity=parity, dagger=dag)
        assert rel_l2(got, ref) <= TOL32, ("D_SAP", parity)
        assert np.array_equal(got == 0, ref == 0)
    # property at full size: gamma5-hermiticity <chi, D psi> = <D^dag chi, psi> (Eq. 2), fp64 sums
    lq.wilson_clover_mult(y, w, U18, Cn, cfg.kappa, L, cfg.bc, dagger=True)
    ddag_chi = lq.unpack_spinor(y, L)
    lhs = torch.sum(torch.conj(chi.to(torch.complex128)) * results["D"].to(torch.complex128))
    rhs = torch.sum(torch.conj(ddag_chi.to(torch.complex128)) * psi.to(torch.complex128))
    assert abs((lhs - rhs).item()) <= 1e-5 * abs(lhs.item())
    # 12-real links reproduce the 18-real result up to fp32 rounding of the rebuilt third row
    d = (results["D_links12"] - results["D"]).to(torch.complex128)
    assert (torch.linalg.vector_norm(d) / torch.linalg.vector_norm(results["D"].to(torch.complex128))).item() <= TOL32


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_coarse_sampled(lq, name):
    import torch
    cfg = li.CONFIGS[name]
    Lc, Vc, nv = cfg.cdims, cfg.cvolume, cfg.nvec
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 1)
    A = li.t_coarse_matrix_synthetic(gen, Vc, nv, "cuda")
    xc = li.t_coarse_vector(gen, Vc, nv, "cuda", torch.float32)
    yc = torch.empty_like(xc)
    rng = np.random.default_rng(cfg.seed + 1)
    Lca = np.array(Lc)
    corners = np.array([[x, y, z, t] for x in (0, Lca[0] - 1) for y in (0, Lca[1] - 1) for z in (0, Lca[2] - 1)
                        for t in (0, Lca[3] - 1)])
    rnd = np.stack([rng.integers(0, Lca[mu], 112) for mu in range(4)], axis=1)
    sites = site_index(Lc, np.concatenate([corners, rnd])).astype(np.int64)
    A_s = A[torch.from_numpy(sites).cuda()].cpu().numpy()
    xc_h = xc.cpu().numpy()
    for dag in (False, True):
        lq.coarse_mult(yc, xc, A, Lc, nv, dagger=dag)
        got = yc[torch.from_numpy(sites).cuda()].cpu().numpy()
        ref = oracle.coarse_mult_sites(xc_h, A_s, Lc, sites, dagger=dag)
        assert rel_l2(got, ref) <= TOL32, dag
        per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(
            ref.reshape(len(sites), -1), axis=1)
        assert per_site.max() <= 5 * TOL32
    # property at full size: linearity D_c(a x + z) = a D_c x + D_c z on the whole lattice
    z = li.t_coarse_vector(gen, Vc, nv, "cuda", torch.float32)
    a = 0.5 - 0.25j
    y1, y2, y3 = torch.empty_like(xc), torch.empty_like(xc), torch.empty_like(xc)
    lq.coarse_mult(y1, xc, A, Lc, nv)
    lq.coarse_mult(y2, z, A, Lc, nv)
    lq.coarse_mult(y3, (a * xc + z).contiguous(), A, Lc, nv)
    err = torch.linalg.vector_norm((y3 - (a * y1 + y2)).to(torch.complex128)) / torch.linalg.vector_norm(
        y3.to(torch.complex128))
    assert err.item() <= 4 * TOL32


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_coarse_half_storage_sampled(lq, name):
    """The coarse operator on half storage in bench.py's configuration: seeded forward blocks on
    the device; for the sampled sites the nine blocks the oracle needs are put together on the HOST from the half
    storage of the site and of its four backward neighbours (conjugate transpose and signs only)."""
    import torch
    cfg = li.CONFIGS[name]
    Lc, Vc, nv = cfg.cdims, cfg.cvolume, cfg.nvec
    n = 2 * nv
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 6)
    Ah = torch.view_as_complex(0.05 * torch.randn((Vc, 5, n, n, 2), generator=gen, device="cuda", dtype=torch.float32))
    Ah[:, 0] += torch.eye(n, device="cuda", dtype=torch.complex64)
    sg = torch.cat([torch.ones(nv), -torch.ones(nv)]).to("cuda")
    # (input preparation: the diagonal block of a Galerkin matrix obeys G5c A_0 G5c = A_0^dag -- needed by the
    # whole-lattice property below, not by the sampled comparison)
    Ah[:, 0] = 0.5 * (Ah[:, 0] + sg[None, :, None] * Ah[:, 0].conj().transpose(-1, -2) * sg[None, None, :])
    xc = li.t_coarse_vector(gen, Vc, nv, "cuda", torch.float32)
    yc = torch.empty_like(xc)
    ws = lq.coarse_half_workspace(Lc, nv)
    rng = np.random.default_rng(cfg.seed + 6)
    Lca = np.array(Lc)
    corners = np.array([[x, y, z, t] for x in (0, Lca[0] - 1) for y in (0, Lca[1] - 1) for z in (0, Lca[2] - 1)
                        for t in (0, Lca[3] - 1)])
    coords = np.concatenate([corners, np.stack([rng.integers(0, Lca[mu], 112) for mu in range(4)], axis=1)])
    sites = site_index(Lc, coords).astype(np.int64)
    sgn = np.concatenate([np.ones(nv), -np.ones(nv)])
    A_s = np.empty((len(sites), 9, n, n), dtype=np.complex64)
    own = Ah[torch.from_numpy(sites).cuda()].cpu().numpy()
    A_s[:, 0] = own[:, 0]
    for mu in range(4):
        A_s[:, 1 + 2 * mu] = own[:, 1 + mu]
        back = coords.copy()
        back[:, mu] = (back[:, mu] - 1) % Lca[mu]
        bsites = torch.from_numpy(site_index(Lc, back).astype(np.int64)).cuda()
        fb = Ah[bsites, 1 + mu].cpu().numpy()
        A_s[:, 2 + 2 * mu] = sgn[None, :, None] * np.conj(np.swapaxes(fb, 1, 2)) * sgn[None, None, :]
    xc_h = xc.cpu().numpy()
    for dag in (False, True):
        lq.coarse_mult_half(yc, xc, Ah, Lc, nv, dagger=dag, ws=ws)
        got = yc[torch.from_numpy(sites).cuda()].cpu().numpy()
        ref = oracle.coarse_mult_sites(xc_h, A_s, Lc, sites, dagger=dag)
        assert rel_l2(got, ref) <= TOL32, dag
        per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(
            ref.reshape(len(sites), -1), axis=1)
        assert per_site.max() <= 5 * TOL32
    # property on the whole lattice: <y, D_c x> = <D_c^dag y, x> (the half-storage operator and its dagger form)
    z = li.t_coarse_vector(gen, Vc, nv, "cuda", torch.float32)
    y1, y2 = torch.empty_like(xc), torch.empty_like(xc)
    lq.coarse_mult_half(y1, xc, Ah, Lc, nv, ws=ws)
    lq.coarse_mult_half(y2, z, Ah, Lc, nv, dagger=True, ws=ws)
    lhs = torch.sum(torch.conj(z).to(torch.complex128) * y1.to(torch.complex128))
    rhs = torch.sum(torch.conj(y2).to(torch.complex128) * xc.to(torch.complex128))
    scale = torch.linalg.vector_norm(z.to(torch.complex128)) * torch.linalg.vector_norm(y1.to(torch.complex128))
    assert (abs(lhs - rhs) / scale).item() <= TOL32


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_restrict_prolong_sampled(lq, name):
    import torch
    cfg = li.CONFIGS[name]
    L, b, nv, V, Vc, Lc = cfg.dims, cfg.block, cfg.nvec, cfg.volume, cfg.cvolume, cfg.cdims
    assert tuple(b) == (4, 4, 4, 4)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 2)
    rng = np.random.default_rng(cfg.seed + 2)
    # 16 sampled aggregates (the two opposite corners included) -> fake 8^4 lattice of 2^4 blocks
    Lca = np.array(Lc)
    Xs = np.stack([rng.integers(0, Lca[mu], 16) for mu in range(4)], axis=1)
    Xs[0] = 0
    Xs[1] = Lca - 1
    fdims = (8, 8, 8, 8)
    fc = li.site_coords(fdims)                       # fake fine coords
    k = site_index((2, 2, 2, 2), fc // 4)            # fake coarse site of each fake fine site
    real = site_index(L, Xs[k] * 4 + fc % 4)         # the real fine site it stands for
    real_d = torch.from_numpy(real.astype(np.int64)).cuda()
    Xreal = site_index(Lc, Xs).astype(np.int64)      # real coarse index of fake coarse site k
    Xreal_d = torch.from_numpy(Xreal).cuda()

    vn = torch.empty(lq.native_nullvecs_reals(L, b, nv), dtype=torch.float32, device="cuda")
    v_fake = np.empty((nv, 4096, 4, 3), dtype=np.complex64)
    scale = 1.0 / np.sqrt(2.0 * 6 * 256)
    for i in range(nv):
        vi = li.t_spinor(gen, V, "cuda", torch.float32) * scale
        lq.pack_nullvec(vn, vi, i, L, b, nv)
        v_fake[i] = vi[real_d].cpu().numpy()
        del vi
    psi = li.t_spinor(gen, V, "cuda", torch.float32)
    xc = li.t_coarse_vector(gen, Vc, nv, "cuda", torch.float32)
    x = lq.pack_spinor(psi, L)
    out_c = torch.empty((Vc, 2, nv), dtype=torch.complex64, device="cuda")
    out_f = lq.empty_spinor(L)
    lq.restrict(out_c, x, vn, L, b, nv)
    lq.prolong(out_f, xc, vn, L, b, nv)
    got_r = out_c[Xreal_d].cpu().numpy()
    ref_r = oracle.restrict(psi[real_d].cpu().numpy(), v_fake, fdims, b)
    assert rel_l2(got_r, ref_r) <= TOL32
    got_p = lq.unpack_spinor(out_f, L)[real_d].cpu().numpy()
    ref_p = oracle.prolong(xc[Xreal_d].cpu().numpy(), v_fake, fdims, b)
    assert rel_l2(got_p, ref_p) <= TOL32
    # property at full size: adjointness <restrict(psi), xc> = <psi, prolong(xc)> (Eqs. 5, 6), fp64 sums
    lhs = torch.sum(torch.conj(out_c.to(torch.complex128)) * xc.to(torch.complex128))
    rhs = torch.sum(torch.conj(psi.to(torch.complex128)) * lq.unpack_spinor(out_f, L).to(torch.complex128))
    assert abs((lhs - rhs).item()) <= 1e-5 * abs(lhs.item())


# ------------------------------------------------------------------------------------------------------------------
# F3 / F4 at full size
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_mr_domain_and_sap_sampled(lq, name):
    """The inner-domain solver is domain-local: 16 sampled 4^4 domains (both lattice corners included) are gathered
    into a fake 8^4 lattice of 2^4 domains on which the oracle runs as it stands (hops between domains are cut, so the
    fake neighbourhood is irrelevant).  Then SAP at full size: properties that hold at any size."""
    import torch
    cfg = li.CONFIGS[name]
    L, dom, V, Lc = cfg.dims, cfg.block, cfg.volume, cfg.cdims
    assert tuple(dom) == (4, 4, 4, 4)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 3)
    rng = np.random.default_rng(cfg.seed + 3)
    U = li.t_gauge_field(cfg, gen, "cuda").to(torch.complex64)
    cl = li.t_clover_synthetic(gen, V, "cuda")
    r = li.t_spinor(gen, V, "cuda", torch.float32)
    U18, Cn, rn = lq.pack_gauge(U, L), lq.pack_clover(cl, L), lq.pack_spinor(r, L)
    Lca = np.array(Lc)
    Xs = np.stack([rng.integers(0, Lca[mu], 16) for mu in range(4)], axis=1)
    Xs[0] = 0
    Xs[1] = Lca - 1
    fdims = (8, 8, 8, 8)
    fc = li.site_coords(fdims)
    k = site_index((2, 2, 2, 2), fc // 4)
    real = site_index(L, Xs[k] * 4 + fc % 4)
    real_d = torch.from_numpy(real.astype(np.int64)).cuda()
    U_f = U[:, real_d].cpu().numpy()
    cl_f = cl[real_d].cpu().numpy()
    r_f = r[real_d].cpu().numpy()
    ref = oracle.mr_domain_solve(r_f, U_f, cl_f, cfg.kappa, fdims, (1, 1, 1, 1), dom, 0, 6)
    z = lq.empty_spinor(L)
    z.fill_(1.0)
    lq.mr_domain_solve(z, rn, U18, Cn, cfg.kappa, L, cfg.bc, dom, parity=0, niter=6)   # resident kernel, all domains
    got = lq.unpack_spinor(z, L)[real_d].cpu().numpy()
    assert rel_l2(got, ref) <= 6 * TOL32
    # the half-grid accumulate form SAP uses: x += M^(e) r changes exactly the even domains, by the same z
    x = lq.pack_spinor(li.t_spinor(gen, V, "cuda", torch.float32), L)
    x0 = lq.unpack_spinor(x, L).clone()
    lq.mr_domain_solve(x, rn, U18, Cn, cfg.kappa, L, cfg.bc, dom, parity=1, niter=6, accumulate=True)
    dx = (lq.unpack_spinor(x, L) - x0)[real_d].cpu().numpy()
    even = (Xs.sum(axis=1) % 2 == 0)[k]
    assert not np.any(dx[~even]), "odd domains untouched, bit for bit"
    assert rel_l2(dx[even], ref[even]) <= 10 * TOL32   # (x0 + z) - x0: one more rounding on the scale of x0
    del x0, dx
    # SAP(2, 6) at full size: the residual it returns is b - D x of the x it returns (same kernel: bit-identical),
    # and every quantity is finite and smaller than the right-hand side
    xs, rs, chk = lq.empty_spinor(L), lq.empty_spinor(L), lq.empty_spinor(L)
    lq.sap(xs, rs, rn, U18, Cn, cfg.kappa, L, cfg.bc, dom, n_sap=2, n_mr=6)
    lq.wilson_clover_residual(chk, rn, xs, U18, Cn, cfg.kappa, L, cfg.bc)
    assert torch.equal(rs, chk)
    nb, nr = torch.linalg.vector_norm(rn.double()).item(), torch.linalg.vector_norm(rs.double()).item()
    assert np.isfinite(nr) and nr < 0.5 * nb, (nr, nb)


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_mrhs_sampled(lq, name):
    """F4 in bench.py's configuration: 16 coarse right-hand sides through the tensor-core kernel, sampled sites
    against the oracle; the pair kernel of the fine operator against the (sample-checked) single kernel."""
    import torch
    cfg = li.CONFIGS[name]
    Lc, Vc, nv = cfg.cdims, cfg.cvolume, cfg.nvec
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 4)
    A = li.t_coarse_matrix_synthetic(gen, Vc, nv, "cuda")
    K = 16
    xs = torch.view_as_complex(torch.randn((K, Vc, 2, nv, 2), generator=gen, device="cuda", dtype=torch.float32))
    ys = torch.empty_like(xs)
    lq.coarse_mult_mrhs(ys, xs, A, Lc, nv)
    rng = np.random.default_rng(cfg.seed + 4)
    Lca = np.array(Lc)
    corners = np.array([[x, y, z, t] for x in (0, Lca[0] - 1) for y in (0, Lca[1] - 1) for z in (0, Lca[2] - 1)
                        for t in (0, Lca[3] - 1)])
    rnd = np.stack([rng.integers(0, Lca[mu], 48) for mu in range(4)], axis=1)
    sites = site_index(Lc, np.concatenate([corners, rnd])).astype(np.int64)
    sites_d = torch.from_numpy(sites).cuda()
    A_s = A[sites_d].cpu().numpy()
    for k in (0, 7, 15):
        ref = oracle.coarse_mult_sites(xs[k].cpu().numpy(), A_s, Lc, sites)
        got = ys[k][sites_d].cpu().numpy()
        assert rel_l2(got, ref) <= TOL32, k
        per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(
            ref.reshape(len(sites), -1), axis=1)
        assert per_site.max() <= 5 * TOL32, k
    # every right-hand side, every site: agreement with the single-right-hand-side kernel to fp32 rounding
    y1 = torch.empty_like(xs[0])
    for k in range(K):
        lq.coarse_mult(y1, xs[k].contiguous(), A, Lc, nv)
        err = torch.linalg.vector_norm((ys[k] - y1).to(torch.complex128)) / torch.linalg.vector_norm(y1.to(torch.complex128))
        assert err.item() <= TOL32, k
    del A, xs, ys
    # fine operator on a pair of right-hand sides: bit-identical with two single applications
    L, V = cfg.dims, cfg.volume
    U = li.t_gauge_field(cfg, gen, "cuda").to(torch.complex64)
    U18 = lq.pack_gauge(U, L)
    del U
    Cn = lq.pack_clover(li.t_clover_synthetic(gen, V, "cuda"), L)
    x2 = torch.stack([lq.pack_spinor(li.t_spinor(gen, V, "cuda", torch.float32), L) for _ in range(2)])
    y2, ys1 = torch.empty_like(x2), lq.empty_spinor(L)
    for dag in (False, True):
        lq.wilson_clover_mult_mrhs(y2, x2, U18, Cn, cfg.kappa, L, cfg.bc, dagger=dag)
        for k in range(2):
            lq.wilson_clover_mult(ys1, x2[k], U18, Cn, cfg.kappa, L, cfg.bc, dagger=dag)
            assert torch.equal(y2[k], ys1), (dag, k)


# ------------------------------------------------------------------------------------------------------------------
# the fp64 kernel variants at full size (config 4; `bench.py --precision f64` times them), bar 1e-12 (north_star)
# ------------------------------------------------------------------------------------------------------------------
TOL64 = 1e-12


@pytest.mark.parametrize("name", ["c4", "c5"])
def test_fullsize_fp64_five_rows_sampled(lq, name):
    """Same sampling as the fp32 tests above, on complex128 inputs: the oracle's fp64-input entry points."""
    import torch
    cfg = li.CONFIGS[name]
    V, L, b, nv, Vc, Lc = cfg.volume, cfg.dims, cfg.block, cfg.nvec, cfg.cvolume, cfg.cdims
    v3 = L[0] * L[1] * L[2]
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 7)
    rng = np.random.default_rng(cfg.seed + 7)
    c128 = torch.complex128

    # ---- A1 / A2: D, D^dag, 12-real links ----
    U = li.t_gauge_field(cfg, gen, "cuda")
    assert U.dtype == c128
    cl = li.t_clover_synthetic(gen, V, "cuda").to(c128)
    psi = li.t_spinor(gen, V, "cuda", torch.float64)
    U18, U12 = lq.pack_gauge(U, L), lq.pack_gauge(U, L, links12=True)
    Cn = lq.pack_clover(cl, L)
    x = lq.pack_spinor(psi, L)
    y = lq.empty_spinor(L, dtype=torch.float64)
    assert U18.dtype == torch.float64 and x.dtype == torch.float64
    sites, slabs = sample_fine_sites(cfg, rng, 2000)
    U_h = lazily_filled((4, V, 3, 3), np.complex128, U, slabs, v3, 1)
    cl_h = lazily_filled((V, 2, 6, 6), np.complex128, cl, slabs, v3, 0)
    psi_h = lazily_filled((V, 4, 3), np.complex128, psi, slabs, v3, 0)
    sites_d = torch.from_numpy(sites).cuda()
    for label, Un, dag, l12 in (("D", U18, False, False), ("Ddag", U18, True, False), ("D_links12", U12, False, True)):
        lq.wilson_clover_mult(y, x, Un, Cn, cfg.kappa, L, cfg.bc, dagger=dag, links12=l12)
        got = lq.unpack_spinor(y, L)[sites_d].cpu().numpy()
        ref = oracle.wilson_clover_mult_sites(psi_h, U_h, cl_h, cfg.kappa, L, cfg.bc, sites, dagger=dag)
        assert got.dtype == np.complex128 and np.isfinite(got).all()
        assert rel_l2(got, ref) <= TOL64, label
        per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(
            ref.reshape(len(sites), -1), axis=1)
        assert per_site.max() <= 5 * TOL64, (label, int(sites[per_site.argmax()]))
    del U, cl, U18, U12, Cn, U_h, cl_h

    # ---- A3: coarse operator and its dagger ----
    A = li.t_coarse_matrix_synthetic(gen, Vc, nv, "cuda").to(c128)
    xc = li.t_coarse_vector(gen, Vc, nv, "cuda", torch.float64)
    yc = torch.empty_like(xc)
    Lca = np.array(Lc)
    corners = np.array([[x_, y_, z_, t_] for x_ in (0, Lca[0] - 1) for y_ in (0, Lca[1] - 1) for z_ in (0, Lca[2] - 1)
                        for t_ in (0, Lca[3] - 1)])
    rnd = np.stack([rng.integers(0, Lca[mu], 48) for mu in range(4)], axis=1)
    csites = site_index(Lc, np.concatenate([corners, rnd])).astype(np.int64)
    csites_d = torch.from_numpy(csites).cuda()
    A_s = A[csites_d].cpu().numpy()
    xc_h = xc.cpu().numpy()
    for dag in (False, True):
        lq.coarse_mult(yc, xc, A, Lc, nv, dagger=dag)
        got = yc[csites_d].cpu().numpy()
        ref = oracle.coarse_mult_sites(xc_h, A_s, Lc, csites, dagger=dag)
        assert rel_l2(got, ref) <= TOL64, dag
    del A, A_s
    torch.cuda.empty_cache()
    # (config 5: the fp64 null vectors are 65 GB on the device -- the size bench.py --precision f64 times; the oracle
    # only ever sees the 16 gathered aggregates)

    # ---- A4 / A5: 16 sampled aggregates gathered into a fake 8^4 lattice of 2^4 blocks (see the fp32 test) ----
    Xs = np.stack([rng.integers(0, Lca[mu], 16) for mu in range(4)], axis=1)
    Xs[0] = 0
    Xs[1] = Lca - 1
    fdims = (8, 8, 8, 8)
    fc = li.site_coords(fdims)
    k = site_index((2, 2, 2, 2), fc // 4)
    real = site_index(L, Xs[k] * 4 + fc % 4)
    real_d = torch.from_numpy(real.astype(np.int64)).cuda()
    Xreal_d = torch.from_numpy(site_index(Lc, Xs).astype(np.int64)).cuda()
    vn = torch.empty(lq.native_nullvecs_reals(L, b, nv), dtype=torch.float64, device="cuda")
    v_fake = np.empty((nv, 4096, 4, 3), dtype=np.complex128)
    scale = 1.0 / np.sqrt(2.0 * 6 * 256)
    for i in range(nv):
        vi = li.t_spinor(gen, V, "cuda", torch.float64) * scale
        lq.pack_nullvec(vn, vi, i, L, b, nv)
        v_fake[i] = vi[real_d].cpu().numpy()
        del vi
    out_c = torch.empty((Vc, 2, nv), dtype=c128, device="cuda")
    out_f = lq.empty_spinor(L, dtype=torch.float64)
    lq.restrict(out_c, x, vn, L, b, nv)
    lq.prolong(out_f, xc, vn, L, b, nv)
    ref_r = oracle.restrict(psi[real_d].cpu().numpy(), v_fake, fdims, b)
    assert rel_l2(out_c[Xreal_d].cpu().numpy(), ref_r) <= TOL64
    ref_p = oracle.prolong(xc[Xreal_d].cpu().numpy(), v_fake, fdims, b)
    assert rel_l2(lq.unpack_spinor(out_f, L)[real_d].cpu().numpy(), ref_p) <= TOL64


def test_fullsize_device_setup_sampled(lq):
    """The operators bench.py times are BUILT on the device (F2: clover term from the links, block-orthonormal null
    vectors, Galerkin P^dag D P).  At config 4 the oracle cannot build them on the whole lattice, but all three are
    local: the nine blocks A[X][.] of a coarse site, the orthonormal vectors on its aggregate and the clover term on
    its sites depend only on the links and raw vectors of the 3^4 aggregates around X.  For sampled X those are
    gathered into a 12^4 lattice (X in the middle; for the sample at the antiperiodic boundary X is placed last in t,
    so that its forward t hop wraps -- and takes its phase -- in the small lattice as it does in the real one) and the
    oracle runs its own set-up chain (O3, O4, O6) there from the RAW seeded inputs.  No oracle input is a CUDA output."""
    import torch
    cfg = li.CONFIGS["c4"]
    L, b, Lc, nv, V = cfg.dims, cfg.block, cfg.cdims, cfg.nvec, cfg.volume
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed + 21)
    U = li.t_gauge_field(cfg, gen, "cuda").to(torch.complex64)          # canonical (4, V, 3, 3), rounded once
    U18 = lq.pack_gauge(U, L)
    clover = lq.clover_from_links(U18, cfg.kappa, cfg.csw, L)
    vn = torch.empty(lq.native_nullvecs_reals(L, b, nv), dtype=torch.float32, device="cuda")
    # sampled coarse sites and the offset of X inside its 3^4 neighbourhood (mini coordinate of X)
    samples = [((3, 5, 2, 9), (1, 1, 1, 1)), ((0, Lc[1] - 1, 4, Lc[3] - 1), (1, 1, 1, 2))]
    mdims, mcd = (12, 12, 12, 12), (3, 3, 3, 3)
    mc = li.site_coords(mdims)                                           # (20736, 4) fine coordinates in the mini lattice
    gathers = []
    for X, off in samples:
        # mini aggregate m <-> real aggregate X + delta, delta = ((m - off + 1) mod 3) - 1 in {-1, 0, +1}: cyclic, so a
        # hop that wraps the mini lattice arrives at the aggregate the real hop arrives at
        real_c = np.stack([((X[mu] + (mc[:, mu] // b[mu] - off[mu] + 1) % 3 - 1) % Lc[mu]) * b[mu] + mc[:, mu] % b[mu]
                           for mu in range(4)], axis=1)
        gathers.append(torch.from_numpy(site_index(L, real_c).astype(np.int64)).cuda())
    raw = [np.empty((nv, len(mc), 4, 3), dtype=np.complex64) for _ in samples]
    for i in range(nv):
        vi = li.t_spinor(gen, V, "cuda", torch.float32)
        lq.pack_nullvec(vn, vi, i, L, b, nv)
        for k, g in enumerate(gathers):
            raw[k][i] = vi[g].cpu().numpy()
        del vi
    lq.orthonormalize_blocks(vn, L, b, nv)
    assert lq.orthonormalize_degenerate_count() == 0
    A = lq.galerkin_coarse(U18, clover, vn, cfg.kappa, L, cfg.bc, b, nv)
    clov_c = lq.unpack_clover(clover, L)                                 # canonical (V, 2, 6, 6)
    for k, ((X, off), g) in enumerate(zip(samples, gathers)):
        # the fp32-rounded inputs, promoted: the oracle's set-up chain runs in fp64 from here on
        Um = np.ascontiguousarray(U[:, g].cpu().numpy()).astype(np.complex128)
        clov_ref = oracle.clover_from_links(Um, cfg.kappa, cfg.csw, mdims)
        v_ref = oracle.orthonormalize_blocks(raw[k].astype(np.complex128), mdims, b)
        A_ref = oracle.galerkin_coarse(Um, clov_ref, v_ref, cfg.kappa, mdims, cfg.bc, b)
        mX = int(site_index(mcd, np.array(off)))                         # X inside the mini coarse lattice
        Xr = int(site_index(Lc, np.array(X)))
        in_X = np.nonzero(site_index(mcd, mc // 4) == mX)[0]             # its 256 fine sites (mini indices)
        # O3: the clover term on the aggregate's sites
        got_c = clov_c[g[torch.from_numpy(in_X).cuda()]].cpu().numpy()
        assert rel_l2(got_c, clov_ref[in_X]) <= 4 * TOL32, ("clover", X)
        # O4: the orthonormal vectors on the aggregate (the unique Q with positive diagonal, compared directly)
        for i in (0, 1, nv // 2, nv - 1):
            vi = lq.unpack_nullvec(vn, i, L, b, nv)
            assert rel_l2(vi[g[torch.from_numpy(in_X).cuda()]].cpu().numpy(), v_ref[i][in_X]) <= 8 * TOL32, ("v", X, i)
        # O6: all nine blocks of the coarse site
        got_A = A[Xr].cpu().numpy()
        assert rel_l2(got_A, A_ref[mX]) <= 2 * TOL32, ("A", X)
        for d in range(9):
            assert rel_l2(got_A[d], A_ref[mX][d]) <= 4 * TOL32, ("A block", X, d)
