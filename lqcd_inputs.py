"""Seeded synthetic input generators shared by the tests, the bench and the oracle pins.

This module holds NONE of the method's arithmetic (no Dirac operator, no clover term,
no orthonormalisation, no Galerkin product): it only draws random fields with the
shapes and distributions of the paper's workloads (BASELINE.json
`configs`).  It imports neither `oracle/` nor the CUDA package.

Canonical layouts; numpy complex = interleaved (re, im):
  gauge     U[mu][s][a][b]     complex, (U psi)_a = sum_b U_ab psi_b      shape (4, V, 3, 3)
  spinor    psi[s][alpha][c]   complex                                     shape (V, 4, 3)
  nullvecs  v[i][s][alpha][c]  complex                                     shape (nvec, V, 4, 3)
  clover    F[s][chi][6][6]    complex Hermitian blocks, k = 3*(alpha%2)+c shape (V, 2, 6, 6)
  coarse vec   x[X][chi][i]    complex                                     shape (Vc, 2, nvec)
  coarse mat   A[X][d][row][col], d=0 diag, 1+2mu forward, 2+2mu backward  shape (Vc, 9, N, N)
Site index s = x + Lx*(y + Ly*(z + Lz*t)); mu = 0..3 <-> x, y, z, t (paper's mu = 1..4,
PAPER.md:43).

The paper's gauge ensembles are not available; these seeded fields
stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

# --------------------------------------------------------------------------------------
# The five BASELINE.json configurations
# --------------------------------------------------------------------------------------


@dataclass(frozen=True)
class Config:
    name: str
    dims: tuple          # fine lattice (Lx, Ly, Lz, Lt)
    block: tuple         # aggregation block (bx, by, bz, bt)
    nvec: int            # N_nv, coarse dofs per site N = 2*nvec
    gauge: str           # "exp" (U = exp(i eps H)) or "haar"
    eps: float
    kappa: float
    csw: float
    seed: int = 1
    bc: tuple = (1, 1, 1, -1)   # periodic space, antiperiodic time

    @property
    def volume(self) -> int:
        return int(np.prod(self.dims))

    @property
    def cdims(self) -> tuple:
        return tuple(l // b for l, b in zip(self.dims, self.block))

    @property
    def cvolume(self) -> int:
        return int(np.prod(self.cdims))


CONFIGS = {
    "c1": Config("c1", (4, 4, 4, 4), (2, 2, 2, 2), 4, "exp", 0.3, 0.13, 1.0, seed=1),
    "c2": Config("c2", (8, 8, 8, 8), (4, 4, 4, 4), 16, "exp", 0.5, 0.135, 1.0, seed=2),
    "c3": Config("c3", (16, 16, 16, 32), (4, 4, 4, 4), 32, "haar", 0.0, 0.137, 1.6, seed=3),
    "c4": Config("c4", (32, 32, 32, 64), (4, 4, 4, 4), 32, "exp", 0.3, 0.1370, 1.7, seed=4),
    "c5": Config("c5", (48, 48, 48, 96), (4, 4, 4, 4), 32, "haar", 0.0, 0.1372, 1.7, seed=5),
}

# --------------------------------------------------------------------------------------
# host (numpy) generators -- configs c1..c3 and every CPU test
# --------------------------------------------------------------------------------------


def _cgauss(rng: np.random.Generator, shape) -> np.ndarray:
    """Complex Gaussian N(0,1) + i N(0,1)."""
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def reunitarize(u: np.ndarray) -> np.ndarray:
    """Project 3x3 matrices (..., 3, 3) to SU(3): Gram-Schmidt on rows 0, 1; row 2 = conj(row0 x row1)."""
    r0 = u[..., 0, :]
    r0 = r0 / np.linalg.norm(r0, axis=-1, keepdims=True)
    r1 = u[..., 1, :]
    r1 = r1 - np.sum(np.conj(r0) * r1, axis=-1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def gauge_exp(rng: np.random.Generator, volume: int, eps: float) -> np.ndarray:
    """U = exp(i eps H), H = (G + G^dag)/2 - tr/3, G complex Gaussian; then re-unitarised."""
    g = _cgauss(rng, (4, volume, 3, 3))
    h = 0.5 * (g + np.conj(np.swapaxes(g, -1, -2)))
    tr = np.trace(h, axis1=-2, axis2=-1) / 3.0
    h = h - tr[..., None, None] * np.eye(3)
    lam, vec = np.linalg.eigh(h)
    u = (vec * np.exp(1j * eps * lam)[..., None, :]) @ np.conj(np.swapaxes(vec, -1, -2))
    return reunitarize(u)


def gauge_haar(rng: np.random.Generator, volume: int) -> np.ndarray:
    """Haar-random SU(3): Q of QR of a complex Gaussian 3x3, columns re-phased by R_ii/|R_ii|, / det^(1/3)."""
    g = _cgauss(rng, (4, volume, 3, 3))
    q, r = np.linalg.qr(g)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    q = q * (d / np.abs(d))[..., None, :]
    det = np.linalg.det(q)
    q = q / np.exp(1j * np.angle(det) / 3.0)[..., None, None]
    return q


def gauge_unit(volume: int) -> np.ndarray:
    """Free field U = 1."""
    u = np.zeros((4, volume, 3, 3), dtype=np.complex128)
    u[..., 0, 0] = u[..., 1, 1] = u[..., 2, 2] = 1.0
    return u


def gauge_field(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    if cfg.gauge == "exp":
        return gauge_exp(rng, cfg.volume, cfg.eps)
    if cfg.gauge == "haar":
        return gauge_haar(rng, cfg.volume)
    raise ValueError(cfg.gauge)


def spinor(rng: np.random.Generator, volume: int) -> np.ndarray:
    return _cgauss(rng, (volume, 4, 3))


def null_vectors(rng: np.random.Generator, nvec: int, volume: int) -> np.ndarray:
    """Gaussian test vectors; NOT orthonormalised (that is oracle input-prep O4)."""
    return _cgauss(rng, (nvec, volume, 4, 3))


def coarse_vector(rng: np.random.Generator, cvolume: int, nvec: int) -> np.ndarray:
    return _cgauss(rng, (cvolume, 2, nvec))


def coarse_matrix_synthetic(rng: np.random.Generator, cvolume: int, nvec: int) -> np.ndarray:
    """Synthetic coarse blocks with Galerkin-like magnitudes: A0 = 1 + 0.1 G, hops 0.05 G."""
    n = 2 * nvec
    a = _cgauss(rng, (cvolume, 9, n, n))
    a[:, 0] *= 0.1
    a[:, 0] += np.eye(n)
    a[:, 1:] *= 0.05
    return a


def random_gauge_transform(rng: np.random.Generator, volume: int) -> np.ndarray:
    """g(x) in SU(3), shape (V, 3, 3) -- for the gauge-covariance pin."""
    return gauge_haar(rng, volume)[0]


@dataclass
class HostFields:
    cfg: Config
    U: np.ndarray
    psi: list = field(default_factory=list)
    v: np.ndarray | None = None


def make_host_fields(cfg: Config, n_rhs: int = 1, with_nullvecs: bool = True) -> HostFields:
    """Draw, in the fixed order gauge -> spinor(s) -> null vectors, the fp64 canonical fields of a config."""
    rng = np.random.default_rng(cfg.seed)
    u = gauge_field(cfg, rng)
    psis = [spinor(rng, cfg.volume) for _ in range(n_rhs)]
    v = null_vectors(rng, cfg.nvec, cfg.volume) if with_nullvecs else None
    return HostFields(cfg, u, psis, v)


def round_to_f32(a: np.ndarray) -> np.ndarray:
    """fp32 parity protocol: round every input once; both sides consume the rounded values."""
    if np.iscomplexobj(a):
        return a.astype(np.complex64)
    return a.astype(np.float32)


# --------------------------------------------------------------------------------------
# lattice index helpers (pure geometry, used by tests to build plane waves, gauge transforms)
# --------------------------------------------------------------------------------------


def site_coords(dims) -> np.ndarray:
    """(V, 4) integer coordinates of canonical site s = x + Lx (y + Ly (z + Lz t))."""
    lx, ly, lz, lt = dims
    s = np.arange(lx * ly * lz * lt)
    return np.stack([s % lx, (s // lx) % ly, (s // (lx * ly)) % lz, s // (lx * ly * lz)], axis=1)


def neighbour_index(dims, mu: int, sign: int) -> np.ndarray:
    """Canonical index of x + sign*mu_hat (periodic wrap) for every site."""
    c = site_coords(dims).copy()
    c[:, mu] = (c[:, mu] + sign) % dims[mu]
    lx, ly, lz, _ = dims
    return c[:, 0] + lx * (c[:, 1] + ly * (c[:, 2] + lz * c[:, 3]))


# --------------------------------------------------------------------------------------
# device (torch) generators -- configs c4/c5, where host generation is too slow.
# Same distributions; a different (torch) random stream.  Returned tensors are
# canonical-layout complex tensors on `device`.
# --------------------------------------------------------------------------------------


def _torch():
    import torch
    return torch


def t_cgauss(gen, shape, device, dtype=None):
    torch = _torch()
    rdt = torch.float64 if dtype is None else dtype
    re = torch.randn(shape, generator=gen, device=device, dtype=rdt)
    im = torch.randn(shape, generator=gen, device=device, dtype=rdt)
    return torch.complex(re, im)


def t_reunitarize(u):
    torch = _torch()
    r0 = u[..., 0, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
    r1 = u[..., 1, :]
    r1 = r1 - torch.sum(torch.conj(r0) * r1, dim=-1, keepdim=True) * r0
    r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
    r2 = torch.conj(torch.linalg.cross(r0, r1, dim=-1))
    return torch.stack([r0, r1, r2], dim=-2)


def t_gauge_haar(gen, volume: int, device, chunk: int = 1 << 21):
    """Haar SU(3): Gram-Schmidt of a complex Gaussian 3x3 (== QR with positive diagonal R), / det^(1/3)."""
    torch = _torch()
    out = torch.empty((4, volume, 3, 3), dtype=torch.complex128, device=device)
    flat = out.view(4 * volume, 3, 3)
    for lo in range(0, 4 * volume, chunk):
        hi = min(lo + chunk, 4 * volume)
        g = t_cgauss(gen, (hi - lo, 3, 3), device)
        r0 = g[:, 0, :]
        r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
        r1 = g[:, 1, :]
        r1 = r1 - torch.sum(torch.conj(r0) * r1, dim=-1, keepdim=True) * r0
        r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
        r2 = g[:, 2, :]
        r2 = r2 - torch.sum(torch.conj(r0) * r2, dim=-1, keepdim=True) * r0
        r2 = r2 - torch.sum(torch.conj(r1) * r2, dim=-1, keepdim=True) * r1
        r2 = r2 / torch.linalg.vector_norm(r2, dim=-1, keepdim=True)
        q = torch.stack([r0, r1, r2], dim=-2)
        det = torch.linalg.det(q)
        q = q / torch.exp(1j * torch.angle(det) / 3.0)[:, None, None]
        flat[lo:hi] = q
    return out


def t_gauge_exp(gen, volume: int, eps: float, device, chunk: int = 1 << 21):
    """U = exp(i eps H) by a 30-term Taylor series (|eps H| ~ 1), then re-unitarised."""
    torch = _torch()
    out = torch.empty((4, volume, 3, 3), dtype=torch.complex128, device=device)
    flat = out.view(4 * volume, 3, 3)
    eye = torch.eye(3, dtype=torch.complex128, device=device)
    for lo in range(0, 4 * volume, chunk):
        hi = min(lo + chunk, 4 * volume)
        g = t_cgauss(gen, (hi - lo, 3, 3), device)
        h = 0.5 * (g + torch.conj(g.transpose(-1, -2)))
        tr = torch.diagonal(h, dim1=-2, dim2=-1).sum(-1) / 3.0
        h = h - tr[:, None, None] * eye
        x = 1j * eps * h
        term = eye.expand_as(x).clone()
        u = term.clone()
        for k in range(1, 31):
            term = torch.bmm(term, x) / k
            u = u + term
        flat[lo:hi] = t_reunitarize(u)
    return out


def t_gauge_field(cfg: Config, gen, device):
    if cfg.gauge == "exp":
        return t_gauge_exp(gen, cfg.volume, cfg.eps, device)
    return t_gauge_haar(gen, cfg.volume, device)


def t_spinor(gen, volume: int, device, dtype=None):
    """Gaussian spinor (V, 4, 3); dtype = real dtype of the parts (float32 -> complex64)."""
    return t_cgauss(gen, (volume, 4, 3), device, dtype)


def t_coarse_vector(gen, cvolume: int, nvec: int, device, dtype=None):
    return t_cgauss(gen, (cvolume, 2, nvec), device, dtype)


def t_clover_synthetic(gen, volume: int, device, scale: float = 0.05, chunk: int = 1 << 20):
    """Synthetic clover term for the two largest configs: per site two Hermitian 6x6
    blocks F = scale * (G + G^dag) / 2, G complex Gaussian -- the magnitude of the true term at these kappa, c_sw
    (|F| ~ 0.05-0.15).  complex64, canonical (V, 2, 6, 6).  The operator takes F as an input, so parity and
    throughput do not depend on where F comes from."""
    torch = _torch()
    out = torch.empty((volume, 2, 6, 6), dtype=torch.complex64, device=device)
    for lo in range(0, volume, chunk):
        hi = min(lo + chunk, volume)
        g = t_cgauss(gen, (hi - lo, 2, 6, 6), device, torch.float32)
        out[lo:hi] = (0.5 * scale) * (g + torch.conj(g.transpose(-1, -2)))
    return out


def t_coarse_matrix_synthetic(gen, cvolume: int, nvec: int, device, chunk: int = 1 << 10):
    """Device version of coarse_matrix_synthetic: A0 = 1 + 0.1 G, hop blocks 0.05 G; complex64 (Vc, 9, N, N)."""
    torch = _torch()
    n = 2 * nvec
    out = torch.empty((cvolume, 9, n, n), dtype=torch.complex64, device=device)
    eye = torch.eye(n, dtype=torch.complex64, device=device)
    for lo in range(0, cvolume, chunk):
        hi = min(lo + chunk, cvolume)
        g = t_cgauss(gen, (hi - lo, 9, n, n), device, torch.float32)
        g[:, 0] *= 0.1
        g[:, 0] += eye
        g[:, 1:] *= 0.05
        out[lo:hi] = g
    return out
