"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

The paper prints no operator input/output values, so every pin is a closed form,
an invariant, a special case or a brute-force evaluation -- never the oracle's own formula retyped.
Each test names the mistake it is there to catch.
"""
import os

import numpy as np
import pytest

import lqcd_inputs as li
import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def zero_clover(V):
    return np.zeros((V, 2, 6, 6), dtype=np.complex128)


# ------------------------------------------------------------------------------------------------
# O1  gamma algebra (Eq. 2)
# ------------------------------------------------------------------------------------------------


def test_gamma_algebra():
    g = oracle.gamma()
    eye = np.eye(4)
    for mu in range(4):
        assert np.array_equal(g[mu], g[mu].conj().T), "gamma_mu Hermitian"
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.array_equal(anti, 2 * eye * (mu == nu)), "Clifford algebra"
        for sign in (+1, -1):
            proj = 0.5 * (eye + sign * g[mu])
            assert np.array_equal(proj @ proj, proj), "(1 +- gamma)/2 is a projector"
            assert np.linalg.matrix_rank(proj) == 2, "of rank 2"
    g5 = g[4]
    assert np.array_equal(g5, -g[0] @ g[1] @ g[2] @ g[3]), "gamma5 = -g1 g2 g3 g4 (Eq. 2)"
    assert np.array_equal(g5 @ g5, eye), "(gamma5)^2 = 1 (footnote 4, PAPER.md:90)"
    assert np.array_equal(g5, np.diag([-1, -1, 1, 1])), "chiral basis: gamma5 diagonal, chi=0 <-> spins 0,1"
    for mu in range(4):
        assert np.array_equal(g5 @ g[mu], -g[mu] @ g5), "gamma5 anticommutes with gamma_mu"


# ------------------------------------------------------------------------------------------------
# A1  free field: plane waves and the closed-form momentum-space operator
#     D psi = e^{ipx} M(p) chi,  M(p) = (1 - 2 kappa sum cos p) + 2 i kappa sum gamma_mu sin p_mu
#     (from Eq. 1 with U = 1, F = 0), eigenvalues 1 - 2k sum cos p +- 2 i k sqrt(sum sin^2 p), each x6.
#     Catches: wrong hop sign, wrong (1 -+ gamma) assignment, wrong neighbour, wrong bc phase, kappa.
# ------------------------------------------------------------------------------------------------


def plane_wave(dims, p):
    return np.exp(1j * (li.site_coords(dims) @ np.asarray(p)))


def momentum(dims, n, bc):
    return np.array([2 * np.pi * (n[mu] + (0.5 if bc[mu] == -1 else 0.0)) / dims[mu] for mu in range(4)])


def momentum_matrix(p, kappa, colour_phase=None):
    """12x12 M(p) in (spin, colour) order; colour_phase[mu][c] adds a constant abelian background."""
    g = oracle.gamma()
    M = np.zeros((4, 3, 4, 3), dtype=np.complex128)
    for c in range(3):
        q = p + (0 if colour_phase is None else colour_phase[:, c])
        m = (1 - 2 * kappa * np.sum(np.cos(q))) * np.eye(4) + 2j * kappa * sum(g[mu] * np.sin(q[mu]) for mu in range(4))
        M[:, c, :, c] = m
    return M.reshape(12, 12)


@pytest.mark.parametrize("dims,n,bc", [
    ((4, 4, 4, 4), (1, 2, 0, 1), (1, 1, 1, -1)),
    ((4, 6, 2, 8), (3, 1, 1, 5), (1, 1, 1, -1)),
    ((6, 4, 4, 2), (2, 3, 1, 0), (-1, 1, -1, 1)),
    ((3, 5, 2, 4), (1, 4, 1, 2), (1, -1, 1, -1)),
])
def test_free_field_plane_waves(dims, n, bc):
    kappa = 0.13
    V = int(np.prod(dims))
    U = li.gauge_unit(V)
    p = momentum(dims, n, bc)
    wave = plane_wave(dims, p)
    M = momentum_matrix(p, kappa)
    got = np.zeros((12, 12), dtype=np.complex128)
    for k in range(12):
        chi = np.zeros(12, dtype=np.complex128)
        chi[k] = 1.0
        psi = (wave[:, None] * chi[None, :]).reshape(V, 4, 3)
        out = oracle.wilson_clover_mult(psi, U, zero_clover(V), kappa, dims, bc)
        expect = (wave[:, None] * M[:, k][None, :]).reshape(V, 4, 3)
        assert rel(out, expect) < 1e-14
        got[:, k] = out.reshape(V, 12)[0] / wave[0]
    # representation-independent: spectrum of the extracted 12x12 equals the closed form
    lam = np.linalg.eigvals(got)
    a = 1 - 2 * kappa * np.sum(np.cos(p))
    b = 2 * kappa * np.sqrt(np.sum(np.sin(p) ** 2))
    assert np.allclose(lam.real, a, atol=1e-12)
    assert np.allclose(np.sort(lam.imag), np.array([-b] * 6 + [b] * 6), atol=1e-12)


def test_free_field_golden_eigenvalues():
    """tests/golden/free_field_eigenvalues.txt: closed-form values written by
    tests/golden/make_free_field_golden.py (pure math, no oracle, no CUDA)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "free_field_eigenvalues.txt")) if l.strip() and l[0] != "#"]
    for r in rows:
        dims = tuple(int(v) for v in r[0:4])
        n = tuple(int(v) for v in r[4:8])
        bc = tuple(int(v) for v in r[8:12])
        kappa, re, im = float(r[12]), float(r[13]), float(r[14])
        V = int(np.prod(dims))
        p = momentum(dims, n, bc)
        wave = plane_wave(dims, p)
        got = np.zeros((12, 12), dtype=np.complex128)
        for k in range(12):
            chi = np.zeros(12, dtype=np.complex128)
            chi[k] = 1.0
            psi = (wave[:, None] * chi[None, :]).reshape(V, 4, 3)
            out = oracle.wilson_clover_mult(psi, li.gauge_unit(V), zero_clover(V), kappa, dims, bc)
            got[:, k] = out.reshape(V, 12)[5] / wave[5]
        lam = np.linalg.eigvals(got)
        assert np.allclose(np.sort(lam.real), re, atol=2e-6)
        assert np.allclose(np.sort(np.abs(lam.imag)), im, atol=2e-6)


def test_kappa_mass_relation():
    """kappa = 1/(8 + 2 m0): at p = 0, periodic free field, D = (1 - 8 kappa) 1."""
    dims, bc = (4, 2, 3, 2), (1, 1, 1, 1)
    V = int(np.prod(dims))
    m0 = 0.37
    kappa = 1 / (8 + 2 * m0)
    psi = np.ones((V, 4, 3), dtype=np.complex128) * (0.3 - 0.8j)
    out = oracle.wilson_clover_mult(psi, li.gauge_unit(V), zero_clover(V), kappa, dims, bc)
    assert rel(out, (1 - 8 * kappa) * psi) < 1e-15
    assert abs((1 - 8 * kappa) - 2 * m0 * kappa) < 1e-15


def test_constant_abelian_background():
    """U_mu = diag(e^{i th_mu,c}) constant: colour c sees momentum p + theta_c.
    Catches U <-> U^dagger swapped between forward and backward hop, and colour-index mix-ups."""
    dims, bc, n = (4, 4, 2, 6), (1, 1, 1, -1), (1, 3, 1, 2)
    V = int(np.prod(dims))
    rng = np.random.default_rng(7)
    theta = rng.uniform(-1, 1, size=(4, 3))
    theta[:, 2] = -theta[:, 0] - theta[:, 1]  # det = 1
    U = np.zeros((4, V, 3, 3), dtype=np.complex128)
    for mu in range(4):
        for c in range(3):
            U[mu, :, c, c] = np.exp(1j * theta[mu, c])
    clov, off = oracle.clover_from_links(U, 0.13, 1.3, dims, return_offdiag=True)
    assert np.max(np.abs(clov)) < 1e-15 and off < 1e-15, "constant abelian field has zero field strength"
    kappa = 0.124
    p = momentum(dims, n, bc)
    wave = plane_wave(dims, p)
    M = momentum_matrix(p, kappa, colour_phase=theta)
    for k in (0, 4, 8, 11):
        chi = np.zeros(12, dtype=np.complex128)
        chi[k] = 1.0
        psi = (wave[:, None] * chi[None, :]).reshape(V, 4, 3)
        out = oracle.wilson_clover_mult(psi, U, clov, kappa, dims, bc)
        expect = (wave[:, None] * M[:, k][None, :]).reshape(V, 4, 3)
        assert rel(out, expect) < 1e-14


# ------------------------------------------------------------------------------------------------
# interacting field: config-1-like inputs
# ------------------------------------------------------------------------------------------------


@pytest.fixture(scope="module")
def c1():
    cfg = li.CONFIGS["c1"]
    f = li.make_host_fields(cfg, n_rhs=2)
    clov = oracle.clover_from_links(f.U, cfg.kappa, cfg.csw, cfg.dims)
    v = oracle.orthonormalize_blocks(f.v, cfg.dims, cfg.block)
    A = oracle.galerkin_coarse(f.U, clov, v, cfg.kappa, cfg.dims, cfg.bc, cfg.block)
    return dict(cfg=cfg, U=f.U, psi=f.psi, clov=clov, v=v, A=A, vraw=f.v)


def test_inputs_are_su3(c1):
    U = c1["U"]
    uu = U @ U.conj().swapaxes(-1, -2)
    assert np.max(np.abs(uu - np.eye(3))) < 1e-14
    assert np.max(np.abs(np.linalg.det(U) - 1)) < 1e-14
    # O8: third row = conj(row0 x row1) -- what the 12-real link compression relies on
    assert np.max(np.abs(np.conj(np.cross(U[..., 0, :], U[..., 1, :])) - U[..., 2, :])) < 1e-14
    Uh = li.gauge_haar(np.random.default_rng(3), 64)
    assert np.max(np.abs(Uh @ Uh.conj().swapaxes(-1, -2) - np.eye(3))) < 1e-13
    assert np.max(np.abs(np.linalg.det(Uh) - 1)) < 1e-13


def test_gamma5_hermiticity(c1):
    """Eq. 2: <x, D^dag y> = <D x, y>, D^dag via the DAGGER flag (gamma5 D gamma5)."""
    cfg = c1["cfg"]
    x, y = c1["psi"]
    Dx = oracle.wilson_clover_mult(x, c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc)
    Ddy = oracle.wilson_clover_mult(y, c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc, dagger=True)
    lhs = np.vdot(x, Ddy)
    rhs = np.vdot(Dx, y)
    assert abs(lhs - rhs) / abs(rhs) < 1e-13
    # and the flag really is gamma5 D gamma5
    g5 = np.array([-1, -1, 1, 1])[None, :, None]
    manual = g5 * oracle.wilson_clover_mult(g5 * y, c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc)
    assert rel(Ddy, manual) < 1e-15


def test_dagger_is_dense_adjoint():
    """On a 2x2x2x4 lattice (extent 2: x+mu == x-mu) build dense D and D^dag from unit vectors."""
    dims, bc = (2, 2, 2, 4), (1, 1, 1, -1)
    V = int(np.prod(dims))
    rng = np.random.default_rng(11)
    U = li.gauge_exp(rng, V, 0.6)
    clov = oracle.clover_from_links(U, 0.13, 1.2, dims)
    n = 12 * V
    D = np.zeros((n, n), dtype=np.complex128)
    Dd = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        D[:, k] = oracle.wilson_clover_mult(e.reshape(V, 4, 3), U, clov, 0.13, dims, bc).ravel()
        Dd[:, k] = oracle.wilson_clover_mult(e.reshape(V, 4, 3), U, clov, 0.13, dims, bc, dagger=True).ravel()
    assert np.max(np.abs(Dd - D.conj().T)) < 1e-14


def test_gauge_covariance(c1):
    """U'_mu(x) = g(x) U_mu(x) g^dag(x+mu), F' from U':  D[U'](g psi) = g D[U] psi.
    Catches a wrong link site/dagger in the hops and a mis-routed clover leaf."""
    cfg = c1["cfg"]
    V = cfg.volume
    rng = np.random.default_rng(5)
    g = li.random_gauge_transform(rng, V)
    Ug = np.empty_like(c1["U"])
    for mu in range(4):
        fwd = li.neighbour_index(cfg.dims, mu, +1)
        Ug[mu] = g @ c1["U"][mu] @ g[fwd].conj().swapaxes(-1, -2)
    clov_g = oracle.clover_from_links(Ug, cfg.kappa, cfg.csw, cfg.dims)
    psi = c1["psi"][0]
    gpsi = np.einsum("sab,sxb->sxa", g, psi)
    lhs = oracle.wilson_clover_mult(gpsi, Ug, clov_g, cfg.kappa, cfg.dims, cfg.bc)
    rhs = np.einsum("sab,sxb->sxa", g, oracle.wilson_clover_mult(psi, c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc))
    assert rel(lhs, rhs) < 1e-14


def test_clover_properties(c1):
    cfg = c1["cfg"]
    clov, off = oracle.clover_from_links(c1["U"], cfg.kappa, cfg.csw, cfg.dims, return_offdiag=True)
    assert off < 1e-16, "F commutes with gamma5: chirality-off-diagonal part vanishes"
    assert np.max(np.abs(clov - clov.conj().swapaxes(-1, -2))) < 1e-16, "F Hermitian (PAPER.md:50)"
    tr = np.trace(clov, axis1=-2, axis2=-1)
    assert np.max(np.abs(tr)) < 1e-15, "each chirality block traceless"
    assert 0.01 < np.max(np.abs(clov)) < 0.5
    free = oracle.clover_from_links(li.gauge_unit(cfg.volume), cfg.kappa, cfg.csw, cfg.dims)
    assert np.max(np.abs(free)) == 0.0, "F = 0 at U = 1"


def test_clover_constant_field_closed_form():
    """U_y(x) = exp(i B x_x T), T = diag(1,-1,0), B = 2 pi k / Lx, other links 1: all four xy leaves equal
    exp(i B T)  =>  F(x) = kappa c_sw sigma_xy (x) sin(B T), other planes 0.
    Catches a mis-oriented leaf, a wrong 1/8, a wrong mu<nu factor."""
    dims = (4, 4, 2, 2)
    V = int(np.prod(dims))
    kappa, csw, k = 0.13, 1.7, 1
    B = 2 * np.pi * k / dims[0]
    T = np.array([1.0, -1.0, 0.0])
    U = li.gauge_unit(V)
    xx = li.site_coords(dims)[:, 0]
    for c in range(3):
        U[1, :, c, c] = np.exp(1j * B * xx * T[c])
    clov = oracle.clover_from_links(U, kappa, csw, dims)
    g = oracle.gamma()
    sig_xy = (g[0] @ g[1] - g[1] @ g[0]) / 2j
    assert np.array_equal(sig_xy, np.diag([1, -1, 1, -1])), "sigma_xy = (tau3, tau3) in the chiral basis"
    F12 = np.kron(sig_xy, np.diag(np.sin(B * T))) * kappa * csw   # index = 3*alpha + c
    expect = np.stack([F12[0:6, 0:6], F12[6:12, 6:12]])
    assert np.max(np.abs(clov - expect[None])) < 1e-15


# ------------------------------------------------------------------------------------------------
# O4/O5  aggregates, restriction, prolongation (Eqs. 5, 6)
# ------------------------------------------------------------------------------------------------


def test_block_orthonormality_and_RP_identity(c1):
    cfg, v = c1["cfg"], c1["v"]
    rng = np.random.default_rng(9)
    xc = li.coarse_vector(rng, cfg.cvolume, cfg.nvec)
    back = oracle.restrict(oracle.prolong(xc, v, cfg.dims, cfg.block), v, cfg.dims, cfg.block)
    assert rel(back, xc) < 1e-14, "<I|J> = delta_IJ  =>  R P = 1 (PAPER.md:92)"
    psi = c1["psi"][0]
    pr = oracle.prolong(oracle.restrict(psi, v, cfg.dims, cfg.block), v, cfg.dims, cfg.block)
    pr2 = oracle.prolong(oracle.restrict(pr, v, cfg.dims, cfg.block), v, cfg.dims, cfg.block)
    assert rel(pr2, pr) < 1e-14, "P R idempotent"
    ratio = np.linalg.norm(pr) / np.linalg.norm(psi)
    assert 0.05 < ratio < 0.9, "x and x' are in general different (PAPER.md:101)"
    # explicit Gram matrix of one aggregate, straight from the definition
    X = 5
    Xc = np.array([X % 2, (X // 2) % 2, (X // 4) % 2, X // 8])
    co = li.site_coords(cfg.dims)
    mask = np.all(co // np.array(cfg.block) == Xc, axis=1)
    for chi in range(2):
        W = v[:, mask][:, :, 2 * chi:2 * chi + 2, :].reshape(cfg.nvec, -1)
        assert np.max(np.abs(W.conj() @ W.T - np.eye(cfg.nvec))) < 1e-14


def test_orthonormalisation_is_the_qr_factor_with_positive_diagonal(c1):
    """Gram-Schmidt in index order (reading Q6) computes, per aggregate (X, chi), the Q of the QR factorisation whose R
    has a positive diagonal -- and that Q is unique.  numpy.linalg.qr (Householder, LAPACK) is an independent route to
    it: its Q, with every column re-phased by the phase of R's diagonal entry, must equal the oracle's vectors column
    by column.  This pins the ORDER in which the vectors are orthogonalised (the Gram matrix and R P = 1 are blind to
    it), which the device set-up's parity test relies on."""
    cfg = c1["cfg"]
    raw = c1["vraw"]                                      # the Gaussian vectors the oracle orthonormalised
    v = c1["v"]
    L, b, nv = cfg.dims, cfg.block, cfg.nvec
    coords = li.site_coords(L)                           # (V, 4)
    cidx = sum((coords[:, mu] // b[mu]) * int(np.prod(cfg.cdims[:mu])) for mu in range(4))
    checked = 0
    for X in range(cfg.cvolume):
        sites = np.nonzero(cidx == X)[0]
        for chi in range(2):
            M = raw[:, sites][:, :, 2 * chi:2 * chi + 2, :].reshape(nv, -1).T      # columns = vectors
            Q, R = np.linalg.qr(M)
            d = np.diagonal(R)
            Qp = Q * (d / np.abs(d))[None, :]                                     # R's diagonal made positive
            got = v[:, sites][:, :, 2 * chi:2 * chi + 2, :].reshape(nv, -1).T
            assert np.max(np.abs(got - Qp)) < 1e-13, (X, chi)
            # triangularity: vector i lies in the span of the raw vectors 0..i
            T = np.conj(got.T) @ M
            assert np.max(np.abs(np.tril(T, -1))) < 1e-13
            checked += 1
    assert checked == 2 * cfg.cvolume


def test_restrict_prolong_adjoint_and_definition(c1):
    cfg, v = c1["cfg"], c1["v"]
    rng = np.random.default_rng(10)
    psi = c1["psi"][1]
    xc = li.coarse_vector(rng, cfg.cvolume, cfg.nvec)
    lhs = np.vdot(oracle.restrict(psi, v, cfg.dims, cfg.block), xc)
    rhs = np.vdot(psi, oracle.prolong(xc, v, cfg.dims, cfg.block))
    assert abs(lhs - rhs) / abs(rhs) < 1e-14, "<R psi, x_c> = <psi, P x_c>"
    # dense P (3072 x 128) assembled column by column from Eq. 6 and used for Eq. 5
    co = li.site_coords(cfg.dims)
    Xof = (co // np.array(cfg.block)) @ np.array([1, 2, 4, 8])
    P = np.zeros((cfg.volume, 4, 3, cfg.cvolume, 2, cfg.nvec), dtype=np.complex128)
    for i in range(cfg.nvec):
        for chi in range(2):
            P[np.arange(cfg.volume), 2 * chi:2 * chi + 2, :, Xof, chi, i] = v[i][:, 2 * chi:2 * chi + 2, :]
    P = P.reshape(cfg.volume * 12, cfg.cvolume * 2 * cfg.nvec)
    assert rel(oracle.prolong(xc, v, cfg.dims, cfg.block).ravel(), P @ xc.ravel()) < 1e-14
    assert rel(oracle.restrict(psi, v, cfg.dims, cfg.block).ravel(), P.conj().T @ psi.ravel()) < 1e-14


# ------------------------------------------------------------------------------------------------
# O6/O7  Galerkin coarse operator (Eq. 7) and its application
# ------------------------------------------------------------------------------------------------


def test_coarse_equals_dense_PdagDP(c1):
    """Brute force on config 1: dense D (3072^2) from unit vectors, dense P, y = P^dag D P x_c
    against the 9-point apply of the Galerkin blocks.  Coarse extent 2 in every direction
    (X+mu == X-mu), antiperiodic time."""
    cfg, v = c1["cfg"], c1["v"]
    n = cfg.volume * 12
    D = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        D[:, k] = oracle.wilson_clover_mult(e.reshape(-1, 4, 3), c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc).ravel()
    nc = cfg.cvolume * 2 * cfg.nvec
    P = np.zeros((n, nc), dtype=np.complex128)
    for k in range(nc):
        e = np.zeros(nc, dtype=np.complex128)
        e[k] = 1
        P[:, k] = oracle.prolong(e.reshape(cfg.cvolume, 2, cfg.nvec), v, cfg.dims, cfg.block).ravel()
    Dc = P.conj().T @ D @ P
    rng = np.random.default_rng(12)
    xc = li.coarse_vector(rng, cfg.cvolume, cfg.nvec)
    got = oracle.coarse_mult(xc, c1["A"], cfg.cdims)
    assert rel(got.ravel(), Dc @ xc.ravel()) < 1e-14
    gotd = oracle.coarse_mult(xc, c1["A"], cfg.cdims, dagger=True)
    assert rel(gotd.ravel(), Dc.conj().T @ xc.ravel()) < 1e-13, "Gamma5c D_c Gamma5c = D_c^dag"


def test_coarse_gamma5_block_relations(c1):
    """Gamma5c A0 Gamma5c = A0^dag and A_{-mu}(X+mu) = Gamma5c A_{+mu}(X)^dag Gamma5c."""
    cfg, A = c1["cfg"], c1["A"]
    nv = cfg.nvec
    g5c = np.diag(np.concatenate([-np.ones(nv), np.ones(nv)]))
    for X in range(cfg.cvolume):
        assert np.max(np.abs(g5c @ A[X, 0] @ g5c - A[X, 0].conj().T)) < 1e-15
    for mu in range(4):
        fwd = li.neighbour_index(cfg.cdims, mu, +1)
        for X in range(cfg.cvolume):
            lhs = A[fwd[X], 2 + 2 * mu]
            rhs = g5c @ A[X, 1 + 2 * mu].conj().T @ g5c
            assert np.max(np.abs(lhs - rhs)) < 1e-15


def test_half_storage_expansion_reproduces_the_galerkin_matrix(c1):
    """The test helper that turns half storage (A_0 and the forward blocks) back into nine blocks is
    what the half-storage GPU tests hand to the oracle: on the true P^dag D P of config 1 (coarse extent 2 in every
    direction: X + mu == X - mu) it must give back the oracle's own nine blocks, and the same on a lattice with
    distinct neighbours."""
    from problems import expand_half, make_problem, custom_config
    cfg, A = c1["cfg"], c1["A"]
    assert np.max(np.abs(expand_half(A[:, [0, 1, 3, 5, 7]], cfg.cdims, cfg.nvec) - A)) < 1e-15
    prob = make_problem(custom_config((6, 4, 8, 4), (2, 2, 2, 2), 2))
    A2 = prob.A
    assert np.max(np.abs(expand_half(A2[:, [0, 1, 3, 5, 7]], prob.cfg.cdims, 2) - A2)) < 1e-15


@pytest.mark.parametrize("dims,block,nvec,bc", [
    ((8, 4, 4, 8), (4, 2, 2, 2), 5, (1, 1, 1, -1)),
    ((4, 6, 4, 4), (2, 3, 1, 2), 3, (-1, 1, 1, -1)),
])
def test_galerkin_identity_as_operators(dims, block, nvec, bc):
    """coarse_mult(x_c) == restrict(D prolong(x_c)) without dense matrices."""
    V = int(np.prod(dims))
    rng = np.random.default_rng(21)
    U = li.gauge_haar(rng, V)
    kappa, csw = 0.135, 1.4
    clov = oracle.clover_from_links(U, kappa, csw, dims)
    v = oracle.orthonormalize_blocks(li.null_vectors(rng, nvec, V), dims, block)
    A = oracle.galerkin_coarse(U, clov, v, kappa, dims, bc, block)
    cdims = tuple(l // b for l, b in zip(dims, block))
    xc = li.coarse_vector(rng, int(np.prod(cdims)), nvec)
    lhs = oracle.coarse_mult(xc, A, cdims)
    rhs = oracle.restrict(oracle.wilson_clover_mult(oracle.prolong(xc, v, dims, block), U, clov, kappa, dims, bc), v, dims, block)
    assert rel(lhs, rhs) < 1e-13


# ------------------------------------------------------------------------------------------------
# entry-point variants agree with the pinned ones
# ------------------------------------------------------------------------------------------------


def test_f32in_and_sites_variants(c1):
    cfg = c1["cfg"]
    U32, psi32, clov32 = (li.round_to_f32(a) for a in (c1["U"], c1["psi"][0], c1["clov"]))
    v32, A32 = li.round_to_f32(c1["v"]), li.round_to_f32(c1["A"])
    up = lambda a: a.astype(np.complex128)
    for dag in (False, True):
        a = oracle.wilson_clover_mult(psi32, U32, clov32, cfg.kappa, cfg.dims, cfg.bc, dagger=dag)
        b = oracle.wilson_clover_mult(up(psi32), up(U32), up(clov32), cfg.kappa, cfg.dims, cfg.bc, dagger=dag)
        assert np.array_equal(a, b), "fp32-input entry point = fp64 arithmetic on the rounded values"
        sites = np.array([0, 17, 255, 64, 3])
        c = oracle.wilson_clover_mult_sites(psi32, U32, clov32, cfg.kappa, cfg.dims, cfg.bc, sites, dagger=dag)
        assert np.array_equal(c, a[sites])
    rng = np.random.default_rng(2)
    xc32 = li.round_to_f32(li.coarse_vector(rng, cfg.cvolume, cfg.nvec))
    for dag in (False, True):
        a = oracle.coarse_mult(xc32, A32, cfg.cdims, dagger=dag)
        assert np.array_equal(a, oracle.coarse_mult(up(xc32), up(A32), cfg.cdims, dagger=dag))
        sites = np.array([3, 0, 15])
        assert np.array_equal(oracle.coarse_mult_sites(xc32, A32[sites], cfg.cdims, sites, dagger=dag), a[sites])
    assert np.array_equal(oracle.restrict(psi32, v32, cfg.dims, cfg.block), oracle.restrict(up(psi32), up(v32), cfg.dims, cfg.block))
    assert np.array_equal(oracle.prolong(xc32, v32, cfg.dims, cfg.block), oracle.prolong(up(xc32), up(v32), cfg.dims, cfg.block))
    assert np.array_equal(oracle.galerkin_coarse(U32, clov32, v32, cfg.kappa, cfg.dims, cfg.bc, cfg.block),
                          oracle.galerkin_coarse(up(U32), up(clov32), up(v32), cfg.kappa, cfg.dims, cfg.bc, cfg.block))


def test_oracle_rejects_bad_arguments(c1):
    cfg = c1["cfg"]
    with pytest.raises(ValueError):
        oracle.wilson_clover_mult(c1["psi"][0], c1["U"], c1["clov"], cfg.kappa, cfg.dims, (1, 1, 1, 0))
    with pytest.raises(ValueError):
        oracle.restrict(c1["psi"][0], c1["v"], cfg.dims, (3, 2, 2, 2))
    with pytest.raises(ValueError):
        oracle.coarse_mult(np.zeros((4, 2, 2), dtype=np.complex128), np.zeros((4, 9, 4, 4), dtype=np.complex128), (1, 2, 2, 1))


# ------------------------------------------------------------------------------------------------
# F1  D_SAP: D with the interaction across domains switched off; even/odd domain groups.
#     Pinned to the (already pinned) D: dense D masked by "same domain", single-domain limit, block
#     structure, e + o = all, gamma5-hermiticity.
# ------------------------------------------------------------------------------------------------


def domain_index(dims, block):
    c = li.site_coords(dims) // np.array(block)
    lc = [d // b for d, b in zip(dims, block)]
    return c[:, 0] + lc[0] * (c[:, 1] + lc[1] * (c[:, 2] + lc[2] * c[:, 3])), c.sum(axis=1) % 2


@pytest.mark.parametrize("dims,block,bc", [
    ((4, 4, 2, 4), (2, 2, 1, 2), (1, 1, 1, -1)),   # extent-2 direction with two domains (x+mu == x-mu, both cross)
    ((4, 2, 2, 6), (2, 2, 2, 3), (-1, 1, 1, -1)),  # directions spanned by a single domain keep their wrapping hops
])
def test_dsap_is_dense_D_masked_by_domain(dims, block, bc):
    """Brute force: dense D from unit vectors (pinned above), entries between different domains zeroed."""
    V = int(np.prod(dims))
    rng = np.random.default_rng(21)
    U = li.gauge_exp(rng, V, 0.6)
    clov = oracle.clover_from_links(U, 0.13, 1.2, dims)
    n = 12 * V
    D = np.zeros((n, n), dtype=np.complex128)
    Ds = np.zeros((n, n), dtype=np.complex128)
    Dsd = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        e = e.reshape(V, 4, 3)
        D[:, k] = oracle.wilson_clover_mult(e, U, clov, 0.13, dims, bc).ravel()
        Ds[:, k] = oracle.wilson_clover_dd_mult(e, U, clov, 0.13, dims, bc, block).ravel()
        Dsd[:, k] = oracle.wilson_clover_dd_mult(e, U, clov, 0.13, dims, bc, block, dagger=True).ravel()
    dom, par = domain_index(dims, block)
    dom12, par12 = np.repeat(dom, 12), np.repeat(par, 12)
    same = dom12[:, None] == dom12[None, :]
    assert np.max(np.abs(Ds - np.where(same, D, 0))) < 1e-15
    assert np.max(np.abs(D - Ds)) > 1e-3, "the mask removes something"
    assert np.max(np.abs(Dsd - Ds.conj().T)) < 1e-14, "D_SAP^dag via gamma5 is the dense adjoint"
    # even / odd groups: P_e D_SAP P_e
    x = li.spinor(rng, V)
    for parity in (1, 2):
        keep = (par12 == parity - 1)
        ref = np.where(keep, Ds @ np.where(keep, x.ravel(), 0), 0)
        got = oracle.wilson_clover_dd_mult(x, U, clov, 0.13, dims, bc, block, parity=parity).ravel()
        assert np.max(np.abs(got - ref)) < 1e-14


def test_dsap_limits_and_structure(c1):
    cfg = c1["cfg"]
    U, clov, x, y = c1["U"], c1["clov"], c1["psi"][0], c1["psi"][1]
    args = (U, clov, cfg.kappa, cfg.dims, cfg.bc)
    # one domain = the whole lattice: nothing is switched off
    assert rel(oracle.wilson_clover_dd_mult(x, *args, cfg.dims), oracle.wilson_clover_mult(x, *args)) < 1e-15
    # domains of one site: only the site-diagonal part 1 + F survives
    site_diag = x + np.einsum("schkl,schl->schk", clov.reshape(-1, 2, 6, 6)[:, :, None].repeat(1, 2),
                              x.reshape(-1, 2, 1, 6)).reshape(x.shape)
    assert rel(oracle.wilson_clover_dd_mult(x, *args, (1, 1, 1, 1)), site_diag) < 1e-15
    # block structure: a source inside one domain stays inside it
    dom, par = domain_index(cfg.dims, cfg.block)
    src = np.where((dom == 5)[:, None, None], x, 0)
    out = oracle.wilson_clover_dd_mult(src, *args, cfg.block)
    assert np.max(np.abs(out[dom != 5])) == 0.0 and np.max(np.abs(out[dom == 5])) > 0.1
    # even + odd = all; gamma5-hermiticity <x, Dsap^dag y> = <Dsap x, y>
    full = oracle.wilson_clover_dd_mult(x, *args, cfg.block)
    e = oracle.wilson_clover_dd_mult(x, *args, cfg.block, parity=1)
    o = oracle.wilson_clover_dd_mult(x, *args, cfg.block, parity=2)
    assert np.array_equal(e + o, full)
    assert np.max(np.abs(e[par == 1])) == 0.0 and np.max(np.abs(o[par == 0])) == 0.0
    lhs = np.vdot(x, oracle.wilson_clover_dd_mult(y, *args, cfg.block, dagger=True))
    rhs = np.vdot(oracle.wilson_clover_dd_mult(x, *args, cfg.block), y)
    assert abs(lhs - rhs) < 1e-12 * abs(rhs)
    # f32-input and sampled-site variants agree with the full fp64-input call on fp32-representable data
    x32, U32, c32 = li.round_to_f32(x), li.round_to_f32(U), li.round_to_f32(clov)
    a = oracle.wilson_clover_dd_mult(x32, U32, c32, cfg.kappa, cfg.dims, cfg.bc, cfg.block, parity=2, dagger=True)
    b = oracle.wilson_clover_dd_mult(x32.astype(np.complex128), U32.astype(np.complex128), c32.astype(np.complex128),
                                     cfg.kappa, cfg.dims, cfg.bc, cfg.block, parity=2, dagger=True)
    assert np.array_equal(a, b)
    sites = np.array([0, 7, 100, 255])
    s = oracle.wilson_clover_dd_mult_sites(x32, U32, c32, cfg.kappa, cfg.dims, cfg.bc, cfg.block, sites, parity=2,
                                           dagger=True)
    assert np.array_equal(s, a[sites])


# ------------------------------------------------------------------------------------------------
# F3  blocked BLAS-1, the inner-domain minimal-residual solver and SAP
# ------------------------------------------------------------------------------------------------


def test_block_blas_against_numpy(c1):
    cfg = c1["cfg"]
    a, b = c1["psi"]
    dims, dom = cfg.dims, (2, 4, 1, 2)
    idx, _ = domain_index(dims, dom)
    nd = idx.max() + 1
    ref = np.array([np.vdot(a[idx == X], b[idx == X]) for X in range(nd)])
    assert np.max(np.abs(oracle.block_dotc(a, b, dims, dom) - ref)) < 1e-12
    coef = np.random.default_rng(4).standard_normal(nd) + 1j * np.random.default_rng(5).standard_normal(nd)
    assert np.max(np.abs(oracle.block_caxpy(b, coef, a, dims, dom) - (b + coef[idx][:, None, None] * a))) < 1e-13


def dense_of(apply, V):
    n = 12 * V
    M = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        M[:, k] = apply(e.reshape(V, 4, 3)).ravel()
    return M


def numpy_mr(A, r, niter):
    """textbook minimal-residual iteration on a dense matrix, z0 = 0"""
    z, rho = np.zeros_like(r), r.copy()
    for _ in range(niter):
        p = A @ rho
        alpha = np.vdot(p, rho) / np.vdot(p, p)
        z += alpha * rho
        rho -= alpha * p
    return z


def test_mr_domain_solve_is_mr_on_each_domain_block():
    """Brute force: dense D_SAP (pinned above) cut into its domain blocks, textbook MR on each block separately."""
    dims, dom, bc = (4, 2, 2, 4), (2, 2, 2, 2), (1, 1, 1, -1)
    V = int(np.prod(dims))
    rng = np.random.default_rng(31)
    U = li.gauge_exp(rng, V, 0.6)
    clov = oracle.clover_from_links(U, 0.13, 1.2, dims)
    r = li.spinor(rng, V)
    Ds = dense_of(lambda e: oracle.wilson_clover_dd_mult(e, U, clov, 0.13, dims, bc, dom), V)
    idx, par = domain_index(dims, dom)
    idx12, par12 = np.repeat(idx, 12), np.repeat(par, 12)
    for parity in (0, 1, 2):
        for niter in (1, 6):
            ref = np.zeros(12 * V, dtype=np.complex128)
            for X in range(idx.max() + 1):
                m = idx12 == X
                if parity and par12[m][0] != parity - 1:
                    continue
                ref[m] = numpy_mr(Ds[np.ix_(m, m)], r.ravel()[m], niter)
            got = oracle.mr_domain_solve(r, U, clov, 0.13, dims, bc, dom, parity, niter).ravel()
            assert np.max(np.abs(got - ref)) < 1e-13, (parity, niter)
    # enough iterations converge to the exact inverse on the selected group: D_SAP^(e) M^(e) r = P_e r
    z = oracle.mr_domain_solve(r, U, clov, 0.13, dims, bc, dom, 1, 200)
    keep = par12 == 0
    assert np.max(np.abs((Ds @ z.ravel())[keep] - r.ravel()[keep])) < 1e-10
    assert np.max(np.abs(z.ravel()[~keep])) == 0.0


def test_sap_listing(c1):
    """The listing of PAPER.md:127-131 retyped on top of dense matrices, and its invariants."""
    dims, dom, bc = (4, 2, 2, 4), (2, 2, 2, 2), (1, 1, 1, -1)
    V = int(np.prod(dims))
    rng = np.random.default_rng(32)
    U = li.gauge_exp(rng, V, 0.6)
    clov = oracle.clover_from_links(U, 0.13, 1.2, dims)
    b = li.spinor(rng, V)
    D = dense_of(lambda e: oracle.wilson_clover_mult(e, U, clov, 0.13, dims, bc), V)
    Ds = dense_of(lambda e: oracle.wilson_clover_dd_mult(e, U, clov, 0.13, dims, bc, dom), V)
    idx, par = domain_index(dims, dom)
    idx12, par12 = np.repeat(idx, 12), np.repeat(par, 12)

    def M(group, r, n_mr):  # block-wise textbook MR on the domains of one group
        z = np.zeros_like(r)
        for X in range(idx.max() + 1):
            m = idx12 == X
            if par12[m][0] == group:
                z[m] = numpy_mr(Ds[np.ix_(m, m)], r[m], n_mr)
        return z

    n_sap, n_mr = 3, 4
    x, r = np.zeros(12 * V, dtype=np.complex128), b.ravel().copy()
    norms = [np.linalg.norm(r)]
    for _ in range(n_sap):
        for group in (0, 1):
            x += M(group, r, n_mr)
            r = b.ravel() - D @ x
            norms.append(np.linalg.norm(r))
    gx, gr = oracle.sap(b, U, clov, 0.13, dims, bc, dom, n_sap=n_sap, n_mr=n_mr)
    assert np.max(np.abs(gx.ravel() - x)) < 1e-13 and np.max(np.abs(gr.ravel() - r)) < 1e-13
    assert all(b2 < b1 for b1, b2 in zip(norms, norms[1:])), "every half sweep reduces the residual here"
    assert norms[-1] < 0.05 * norms[0]
    # config 1 with the paper's parameters (n = 4, 6 MR iterations): the returned residual is the true residual
    cfg = c1["cfg"]
    x1, r1 = oracle.sap(c1["psi"][0], c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc, cfg.block)
    true_r = c1["psi"][0] - oracle.wilson_clover_mult(x1, c1["U"], c1["clov"], cfg.kappa, cfg.dims, cfg.bc)
    assert rel(r1, true_r) < 1e-13 and np.linalg.norm(r1) < 0.05 * np.linalg.norm(c1["psi"][0])


# ------------------------------------------------------------------------------------------------
# F3 (continued)  coarse BiCGStab with fixed iterations and the V-cycle
# ------------------------------------------------------------------------------------------------
def dense_coarse(A, cdims, nvec):
    n = int(np.prod(cdims)) * 2 * nvec
    M = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        M[:, k] = oracle.coarse_mult(e.reshape(-1, 2, nvec), A, cdims).ravel()
    return M


def test_coarse_bicgstab_against_scipy_and_dense_solve(c1):
    """An independent library routine (scipy.sparse.linalg.bicgstab, stopped after the same number of iterations) on
    the dense coarse matrix (itself pinned by brute force above), and the exact solution for many iterations."""
    import scipy.sparse.linalg as spla
    cfg = c1["cfg"]
    Dc = dense_coarse(c1["A"], cfg.cdims, cfg.nvec)
    rng = np.random.default_rng(41)
    b = li.coarse_vector(rng, cfg.cvolume, cfg.nvec)
    for niter in (1, 2, 5, 9):
        ref, info = spla.bicgstab(Dc, b.ravel(), x0=np.zeros(Dc.shape[0], dtype=np.complex128), rtol=1e-300, atol=0.0,
                                  maxiter=niter)
        assert info == niter  # stopped by the iteration count, not by convergence
        x, r = oracle.coarse_bicgstab(b, c1["A"], cfg.cdims, cfg.nvec, niter)
        assert rel(x.ravel(), ref) < 1e-11, niter
        assert np.linalg.norm(r.ravel() - (b.ravel() - Dc @ x.ravel())) < 1e-12 * np.linalg.norm(b), \
            "the recurrence residual is the true residual"
    x0, r0 = oracle.coarse_bicgstab(b, c1["A"], cfg.cdims, cfg.nvec, 0)
    assert not np.any(x0) and np.array_equal(r0, b)
    x, r = oracle.coarse_bicgstab(b, c1["A"], cfg.cdims, cfg.nvec, 60)
    assert rel(x.ravel(), np.linalg.solve(Dc, b.ravel())) < 1e-10
    # residual norms fall by orders of magnitude within the paper-like iteration counts ("not necessarily ... high
    # precision")
    assert np.linalg.norm(oracle.coarse_bicgstab(b, c1["A"], cfg.cdims, cfg.nvec, 8)[1]) < 1e-2 * np.linalg.norm(b)


def test_vcycle_structure_and_convergence(c1):
    cfg = c1["cfg"]
    U, clov, v, A = c1["U"], c1["clov"], c1["v"], c1["A"]
    b = c1["psi"][0]
    D = lambda y: oracle.wilson_clover_mult(y, U, clov, cfg.kappa, cfg.dims, cfg.bc)
    args = (U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, v, A)
    # (1) alone with an accurate coarse solve: Galerkin orthogonality R (b - D P D_c^-1 R b) = 0 because D_c = R D P
    x1 = oracle.mg_vcycle(b, *args, n_coarse=60, n_sap=0)
    assert np.linalg.norm(oracle.restrict(b - D(x1), v, cfg.dims, cfg.block)) < 1e-9 * np.linalg.norm(b)
    # ... and x1 lies in the range of P: P R x1 = x1
    assert rel(oracle.prolong(oracle.restrict(x1, v, cfg.dims, cfg.block), v, cfg.dims, cfg.block), x1) < 1e-13
    # (2) alone (no coarse iterations): the V-cycle is SAP
    assert rel(oracle.mg_vcycle(b, *args, n_coarse=0, n_sap=2, n_mr=3),
               oracle.sap(b, U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block, n_sap=2, n_mr=3)[0]) < 1e-14
    # both: the two Richardson refinements of PAPER.md:112 from the pinned parts
    xc, _ = oracle.coarse_bicgstab(oracle.restrict(b, v, cfg.dims, cfg.block), A, cfg.cdims, cfg.nvec, 8)
    y = oracle.prolong(xc, v, cfg.dims, cfg.block)
    y = y + oracle.sap(b - D(y), U, clov, cfg.kappa, cfg.dims, cfg.bc, cfg.block)[0]
    x = oracle.mg_vcycle(b, *args)
    assert rel(x, y) < 1e-13
    # M ~ D^-1: as a stationary iteration x += M (b - D x) the error against the DENSE solve contracts every cycle
    V = cfg.volume
    Dd = dense_of(D, V)
    exact = np.linalg.solve(Dd, b.ravel()).reshape(V, 4, 3)
    xk, errs = np.zeros_like(b), []
    for _ in range(4):
        xk = xk + oracle.mg_vcycle(b - D(xk), *args)
        errs.append(rel(xk, exact))
    assert errs[0] < 0.1 and all(e2 < 0.25 * e1 for e1, e2 in zip(errs, errs[1:])), errs
