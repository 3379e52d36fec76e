"""CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes marshalling around oracle/liblqcd_oracle.so (plain fp64 C, lqcd_oracle.c), which
restates the hot path of arXiv:2111.05012 from the paper's equations.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package; the product (paper_2111_05012_b200) never does, and this package never imports it.

All arrays are numpy, canonical layout (see lqcd_inputs.py).  complex128 inputs call the `_ref`
entry points, complex64 inputs the `_ref_f32in` ones (values promoted to fp64 on load, all
arithmetic fp64 -- parity protocol O9).  Outputs are complex128.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

DAGGER = 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
    return _lib


def threads() -> int:
    return int(lib().lqcd_oracle_threads_ref())


def set_threads(n: int) -> int:
    """OpenMP threads of the following oracle calls (1 ... all cores); returns the count in effect."""
    return int(lib().lqcd_oracle_set_threads_ref(C.c_int(int(n))))


def _i4(a):
    arr = (C.c_int * 4)(*[int(v) for v in a])
    return arr


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _kind(*arrs) -> str:
    """Entry-point suffix from the input dtype; all inputs must agree."""
    dts = {a.dtype for a in arrs}
    if dts == {np.dtype(np.complex128)}:
        return "_ref"
    if dts == {np.dtype(np.complex64)}:
        return "_ref_f32in"
    raise TypeError(f"oracle inputs must be all complex128 or all complex64, got {dts}")


def _c(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a)


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError(f"oracle {what} failed with code {rc}")


def gamma() -> np.ndarray:
    """(5, 4, 4): gamma_x, gamma_y, gamma_z, gamma_t, gamma5 = -g1 g2 g3 g4 (Eq. 2)."""
    g = np.zeros((5, 4, 4), dtype=np.complex128)
    lib().lqcd_gamma_ref(_ptr(g))
    return g


def wilson_clover_mult(psi, U, clover, kappa, dims, bc, dagger=False) -> np.ndarray:
    """Eq. 1; dagger: Eq. 2."""
    psi, U, clover = _c(psi), _c(U), _c(clover)
    V = int(np.prod(dims))
    assert psi.shape == (V, 4, 3) and U.shape == (4, V, 3, 3) and clover.shape == (V, 2, 6, 6)
    out = np.empty((V, 4, 3), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_wilson_clover_mult" + _kind(psi, U, clover))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(psi), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc),
            C.c_uint(DAGGER if dagger else 0))
    _check(rc, "wilson_clover_mult")
    return out


def wilson_clover_mult_sites(psi, U, clover, kappa, dims, bc, sites, dagger=False) -> np.ndarray:
    """The same operator at the listed canonical site indices only -> (len(sites), 4, 3)."""
    psi, U, clover = _c(psi), _c(U), _c(clover)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_wilson_clover_mult_sites" + _kind(psi, U, clover))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(psi), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc),
            C.c_uint(DAGGER if dagger else 0), _ptr(sites), C.c_long(len(sites)))
    _check(rc, "wilson_clover_mult_sites")
    return out


def clover_from_links(U, kappa, csw, dims, return_offdiag=False):
    """O3: F = kappa csw sum_{mu<nu} sigma_{mu nu} F_{mu nu} from plaquette leaves -> (V, 2, 6, 6)."""
    U = _c(U)
    V = int(np.prod(dims))
    assert U.shape == (4, V, 3, 3)
    out = np.empty((V, 2, 6, 6), dtype=np.complex128)
    off = C.c_double(0.0)
    fn = getattr(lib(), "lqcd_clover_from_links" + _kind(U))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(U), C.c_double(kappa), C.c_double(csw), _i4(dims), C.byref(off))
    _check(rc, "clover_from_links")
    return (out, off.value) if return_offdiag else out


def orthonormalize_blocks(v, dims, block) -> np.ndarray:
    """O4: block/chirality-wise modified Gram-Schmidt (twice) of the null vectors; returns a new array."""
    v = np.array(v, dtype=np.complex128, order="C", copy=True)
    nvec = v.shape[0]
    fn = lib().lqcd_orthonormalize_blocks_ref
    fn.restype = C.c_int
    rc = fn(_ptr(v), _i4(dims), _i4(block), C.c_int(nvec))
    _check(rc, "orthonormalize_blocks")
    return v


def restrict(psi, v, dims, block) -> np.ndarray:
    """Eq. 5 -> (Vc, 2, nvec)."""
    psi, v = _c(psi), _c(v)
    nvec = v.shape[0]
    Vc = int(np.prod([l // b for l, b in zip(dims, block)]))
    out = np.empty((Vc, 2, nvec), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_restrict" + _kind(psi, v))
    fn.restype = C.c_int
    _check(fn(_ptr(out), _ptr(psi), _ptr(v), _i4(dims), _i4(block), C.c_int(nvec)), "restrict")
    return out


def prolong(xc, v, dims, block) -> np.ndarray:
    """Eq. 6 -> (V, 4, 3)."""
    xc, v = _c(xc), _c(v)
    nvec = v.shape[0]
    V = int(np.prod(dims))
    out = np.empty((V, 4, 3), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_prolong" + _kind(xc, v))
    fn.restype = C.c_int
    _check(fn(_ptr(out), _ptr(xc), _ptr(v), _i4(dims), _i4(block), C.c_int(nvec)), "prolong")
    return out


def galerkin_coarse(U, clover, v, kappa, dims, bc, block) -> np.ndarray:
    """Eq. 7: nine N x N blocks per coarse site -> (Vc, 9, N, N)."""
    U, clover, v = _c(U), _c(clover), _c(v)
    nvec = v.shape[0]
    n = 2 * nvec
    Vc = int(np.prod([l // b for l, b in zip(dims, block)]))
    out = np.empty((Vc, 9, n, n), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_galerkin_coarse" + _kind(U, clover, v))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(U), _ptr(clover), _ptr(v), C.c_double(kappa), _i4(dims), _i4(bc), _i4(block),
            C.c_int(nvec))
    _check(rc, "galerkin_coarse")
    return out


def coarse_mult(xc, A, cdims, dagger=False) -> np.ndarray:
    """Eqs. 4, 7: 9-point block stencil -> (Vc, 2, nvec)."""
    xc, A = _c(xc), _c(A)
    Vc, _, nvec = xc.shape
    assert A.shape == (Vc, 9, 2 * nvec, 2 * nvec)
    out = np.empty((Vc, 2, nvec), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_coarse_mult" + _kind(xc, A))
    fn.restype = C.c_int
    _check(fn(_ptr(out), _ptr(xc), _ptr(A), _i4(cdims), C.c_int(nvec), C.c_uint(DAGGER if dagger else 0)),
           "coarse_mult")
    return out


def coarse_mult_sites(xc, A_sites, cdims, sites, dagger=False) -> np.ndarray:
    """coarse_mult at listed coarse sites; A_sites = A[sites] (len(sites), 9, N, N)."""
    xc, A_sites = _c(xc), _c(A_sites)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    _, _, nvec = xc.shape
    out = np.empty((len(sites), 2, nvec), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_coarse_mult_sites" + _kind(xc, A_sites))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(xc), _ptr(A_sites), _i4(cdims), C.c_int(nvec), C.c_uint(DAGGER if dagger else 0),
            _ptr(sites), C.c_long(len(sites)))
    _check(rc, "coarse_mult_sites")
    return out


def wilson_clover_dd_mult(psi, U, clover, kappa, dims, bc, domain, parity=0, dagger=False) -> np.ndarray:
    """F1, D_SAP: D with the hops across domain boundaries off; parity 0/1/2 = all/even/odd domains."""
    psi, U, clover = _c(psi), _c(U), _c(clover)
    V = int(np.prod(dims))
    assert psi.shape == (V, 4, 3) and U.shape == (4, V, 3, 3) and clover.shape == (V, 2, 6, 6)
    out = np.empty((V, 4, 3), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_wilson_clover_dd_mult" + _kind(psi, U, clover))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(psi), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc), _i4(domain),
            C.c_int(parity), C.c_uint(DAGGER if dagger else 0))
    _check(rc, "wilson_clover_dd_mult")
    return out


def wilson_clover_dd_mult_sites(psi, U, clover, kappa, dims, bc, domain, sites, parity=0, dagger=False) -> np.ndarray:
    """D_SAP at the listed canonical site indices only -> (len(sites), 4, 3)."""
    psi, U, clover = _c(psi), _c(U), _c(clover)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3), dtype=np.complex128)
    fn = getattr(lib(), "lqcd_wilson_clover_dd_mult_sites" + _kind(psi, U, clover))
    fn.restype = C.c_int
    rc = fn(_ptr(out), _ptr(psi), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc), _i4(domain),
            C.c_int(parity), C.c_uint(DAGGER if dagger else 0), _ptr(sites), C.c_long(len(sites)))
    _check(rc, "wilson_clover_dd_mult_sites")
    return out


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def block_dotc(a, b, dims, domain) -> np.ndarray:
    """F3, blocked BLAS-1: out[X] = <a|b> restricted to domain X (fp64 only)."""
    a, b = _c128(a), _c128(b)
    Vc = int(np.prod([l // d for l, d in zip(dims, domain)]))
    out = np.empty(Vc, dtype=np.complex128)
    fn = lib().lqcd_block_dotc_ref
    fn.restype = C.c_int
    _check(fn(_ptr(out), _ptr(a), _ptr(b), _i4(dims), _i4(domain)), "block_dotc")
    return out


def block_caxpy(y, coef, a, dims, domain) -> np.ndarray:
    """y + coef[X(x)] * a, one complex coefficient per domain; returns a new array."""
    y, coef, a = np.array(y, dtype=np.complex128, order="C", copy=True), _c128(coef), _c128(a)
    fn = lib().lqcd_block_caxpy_ref
    fn.restype = C.c_int
    _check(fn(_ptr(y), _ptr(coef), _ptr(a), _i4(dims), _i4(domain)), "block_caxpy")
    return y


def mr_domain_solve(r, U, clover, kappa, dims, bc, domain, parity, niter) -> np.ndarray:
    """z = M_SAP^(e/o) r: `niter` minimal-residual iterations per domain (Q17)."""
    r, U, clover = _c128(r), _c128(U), _c128(clover)
    z = np.empty_like(r)
    fn = lib().lqcd_mr_domain_solve_ref
    fn.restype = C.c_int
    _check(fn(_ptr(z), _ptr(r), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc), _i4(domain),
              C.c_int(parity), C.c_int(niter)), "mr_domain_solve")
    return z


def sap(b, U, clover, kappa, dims, bc, domain, n_sap=4, n_mr=6):
    """SAP with fixed iterations -> (x, final residual b - D x)."""
    b, U, clover = _c128(b), _c128(U), _c128(clover)
    x, r = np.empty_like(b), np.empty_like(b)
    fn = lib().lqcd_sap_ref
    fn.restype = C.c_int
    _check(fn(_ptr(x), _ptr(r), _ptr(b), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc), _i4(domain),
              C.c_int(n_sap), C.c_int(n_mr)), "sap")
    return x, r


def coarse_bicgstab(b, A, cdims, nvec, niter):
    """(1b) of PAPER.md:116: `niter` BiCGStab iterations (listing PAPER.md:71 with M = 1, x0 = 0; Q18)
    for D_c x = b -> (x, recurrence residual)."""
    b, A = _c128(b), _c128(A)
    x, r = np.empty_like(b), np.empty_like(b)
    fn = lib().lqcd_coarse_bicgstab_ref
    fn.restype = C.c_int
    _check(fn(_ptr(x), _ptr(r), _ptr(b), _ptr(A), _i4(cdims), C.c_int(nvec), C.c_int(niter)), "coarse_bicgstab")
    return x, r


def mg_vcycle(b, U, clover, kappa, dims, bc, block, v, A, n_coarse=8, n_sap=4, n_mr=6) -> np.ndarray:
    """x = M b: one V-cycle of the multigrid preconditioner."""
    b, U, clover, v, A = _c128(b), _c128(U), _c128(clover), _c128(v), _c128(A)
    x = np.empty_like(b)
    fn = lib().lqcd_mg_vcycle_ref
    fn.restype = C.c_int
    _check(fn(_ptr(x), _ptr(b), _ptr(U), _ptr(clover), C.c_double(kappa), _i4(dims), _i4(bc), _i4(block),
              C.c_int(v.shape[0]), _ptr(v), _ptr(A), C.c_int(n_coarse), C.c_int(n_sap), C.c_int(n_mr)), "mg_vcycle")
    return x
