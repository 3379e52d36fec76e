"""paper_2111_05012_b200 -- thin Python binding of the C ABI in include/lqcd_b200.h.

B200 (sm_100a) hot path of arXiv:2111.05012: fine Wilson-clover operator (Eq. 1) and its
gamma5-conjugate (Eq. 2), coarse 9-point block operator (Eqs. 4, 7),
restriction / prolongation (Eqs. 5, 6).  Functions have the names of the C entry points
without the `lqcd_` prefix and the precision suffix (picked from the tensor dtype).  This module marshals
arguments only: every step runs in the CUDA kernels of csrc/.  torch supplies device memory and streams.
There is no CPU fallback; nothing here imports oracle/.
"""
from __future__ import annotations

import ctypes as C

import torch

from . import _lib
from ._lib import c_int4

DAGGER = 1
LINKS_12 = 2
DOMAIN_EVEN = 4
DOMAIN_ODD = 8
ACCUMULATE = 16
SAP_INITIAL_GUESS = 32
SAP_NO_FINAL_RESIDUAL = 64

OK, EINVAL, EUNSUPPORTED, ECUDA = 0, -1, -2, -3


class LqcdError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        msg = _lib.load().lqcd_last_error().decode()
        super().__init__(f"{what} failed with code {code}: {msg}")


_binding_error = None  # message of the most recent refusal by the binding itself (cleared by the next C call)


class LqcdSizeError(LqcdError, ValueError):
    """A call refused by the binding BEFORE it reaches the library: a tensor (or workspace, or face buffer) whose size
    does not match the geometry.  Counts as LQCD_EINVAL (nothing is enqueued); also a ValueError."""

    def __init__(self, msg: str):
        global _binding_error
        self.code = EINVAL
        _binding_error = msg
        RuntimeError.__init__(self, msg)


def lib():
    return _lib.load()


def _i4(a):
    return c_int4(*[int(v) for v in a])


def _sfx(t: torch.Tensor) -> str:
    if t.dtype in (torch.float32, torch.complex64):
        return "f32"
    if t.dtype in (torch.float64, torch.complex128):
        return "f64"
    raise TypeError(f"unsupported dtype {t.dtype}")


def _real(t: torch.Tensor) -> torch.Tensor:
    """Real view of a contiguous real or complex tensor (no copy)."""
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return torch.view_as_real(t) if t.is_complex() else t


def _dev_ptr(t: torch.Tensor):
    if not t.is_cuda:
        raise ValueError("expected a CUDA tensor (there is no CPU path)")
    return C.c_void_p(_real(t).data_ptr())


def _host_ptr(t: torch.Tensor):
    if t.is_cuda:
        raise ValueError("expected a host tensor")
    return C.c_void_p(_real(t).data_ptr())


def _stream(stream=None, *likes):
    """The caller's stream, else the current stream of the device the call's tensors live on (which need not be the
    current device).  likes: tensors (or lists of tensors) of the call; the first CUDA tensor decides."""
    if stream is None:
        dev = None
        for t in likes:
            for u in (t if isinstance(t, (list, tuple)) else (t,)):
                if isinstance(u, torch.Tensor) and u.is_cuda:
                    dev = u.device
                    break
            if dev is not None:
                break
        stream = torch.cuda.current_stream(dev)
    return C.c_void_p(stream.cuda_stream)


def _check(rc: int, what: str):
    global _binding_error
    _binding_error = None
    if rc != 0:
        raise LqcdError(rc, what)


def _same_dtype(*ts):
    sf = {_sfx(t) for t in ts}
    if len(sf) != 1:
        raise TypeError("all tensors of one call must share one precision")
    return sf.pop()


def _rdtype(sfx: str):
    return torch.float32 if sfx == "f32" else torch.float64


# ---- argument checks: only the binding knows the tensors' sizes (the C side sees raw pointers) ---------------
import functools


def _t4(a):
    return tuple(int(v) for v in a)


@functools.lru_cache(maxsize=256)
def _sz(kind: str, a=None, b=None, n=0, flag=0) -> int:
    """Reals of one native field, asked of the library (lqcd_native_*_reals) and cached per geometry."""
    L = lib()
    if kind == "spinor":
        return int(L.lqcd_native_spinor_reals(c_int4(*a)))
    if kind == "gauge":
        return int(L.lqcd_native_gauge_reals(c_int4(*a), flag))
    if kind == "clover":
        return int(L.lqcd_native_clover_reals(c_int4(*a)))
    if kind == "nullvecs":
        return int(L.lqcd_native_nullvecs_reals(c_int4(*a), c_int4(*b), n))
    if kind == "cvec":
        return int(L.lqcd_native_coarse_vec_reals(c_int4(*a), n))
    if kind == "cmat":
        return int(L.lqcd_native_coarse_mat_reals(c_int4(*a), n))
    raise KeyError(kind)


def _cdims(dims, block):
    """Coarse dims; all zero (= 'invalid geometry', which the C call reports itself) if block does not divide dims."""
    if any(int(b) < 1 or int(l) % int(b) for l, b in zip(dims, block)):
        return (0, 0, 0, 0)
    return tuple(int(l) // int(b) for l, b in zip(dims, block))


def _reals(t) -> int:
    return int(t.numel()) * (2 if t.is_complex() else 1)


def _need(t, reals: int, name: str, exact: bool = True):
    """Raise ValueError before the ctypes call when tensor `t` does not hold `reals` reals (a size the library
    reported as 0 means invalid geometry: the C call then answers LQCD_EINVAL itself)."""
    if t is None or isinstance(t, DevPtr) or reals <= 0:
        return
    n = _reals(t)
    if (n != reals) if exact else (n < reals):
        raise LqcdSizeError(f"{name}: tensor of {n} reals, the call needs {'' if exact else 'at least '}{reals}")


def _need_bytes(t, nbytes: int, name: str):
    if t is None or isinstance(t, DevPtr):
        if nbytes > 0 and t is None:
            raise LqcdSizeError(f"{name}: the call needs a workspace of {nbytes} bytes")
        return
    have = int(t.numel()) * int(t.element_size())
    if have < nbytes:
        raise LqcdSizeError(f"{name}: workspace of {have} bytes, the call needs {nbytes}")


def _vol(dims) -> int:
    v = 1
    for d in dims:
        v *= int(d)
    return v


def _need_faces(bufs, reals8, part_mask: int, name: str):
    """bufs[8]: a face buffer of at least reals8[f] reals for every face f of a partitioned direction."""
    if len(bufs) != 8:
        raise LqcdSizeError(f"{name}: expected 8 face buffers (None for unpartitioned directions)")
    for f in range(8):
        if (int(part_mask) >> (f >> 1)) & 1:
            if bufs[f] is None:
                raise LqcdSizeError(f"{name}[{f}]: missing face buffer of a partitioned direction")
            _need(bufs[f], int(reals8[f]), f"{name}[{f}]", exact=False)


def _mr_ws_bytes(dims, domain, sfx: str) -> int:
    return int(lib().lqcd_mr_workspace_bytes(_i4(dims), _i4(domain), 4 if sfx == "f32" else 8))


def host_workspace_bytes_fine(dims, sfx: str = "f32") -> int:
    """Scratch the fine host call needs (no coarse slots)."""
    fn = lib().lqcd_host_workspace_bytes if sfx == "f32" else lib().lqcd_host_workspace_bytes_f64
    return int(fn(_i4(dims), None, 0))


def _need_fine(dims, links12=None, spinors=(), U=None, clover=None, k=1):
    d = _t4(dims)
    for name, t in spinors:
        _need(t, k * _sz("spinor", d), name)
    if U is not None:
        _need(U, _sz("gauge", d, flag=LINKS_12 if links12 else 0), "U")
    if clover is not None:
        _need(clover, _sz("clover", d), "clover")


def _need_transfer(dims, block, nvec, fine=(), coarse=(), nullvecs=None, k=1):
    d, b = _t4(dims), _t4(block)
    for name, t in fine:
        _need(t, k * _sz("spinor", d), name)
    for name, t in coarse:
        _need(t, k * _sz("cvec", _cdims(d, b), n=int(nvec)), name)
    if nullvecs is not None:
        _need(nullvecs, _sz("nullvecs", d, b, int(nvec)), "nullvecs")


def _need_coarse(cdims, nvec, vecs=(), A=None, k=1):
    c = _t4(cdims)
    for name, t in vecs:
        _need(t, k * _sz("cvec", c, n=int(nvec)), name)
    if A is not None:
        _need(A, _sz("cmat", c, n=int(nvec)), "A")



# ---- diagnostics / knobs ---------------------------------------------------------------------------
def version() -> int:
    return lib().lqcd_version()


def last_error() -> str:
    """Text of the most recent failure: the library's (thread-local) string, or the binding's own refusal."""
    return _binding_error if _binding_error is not None else lib().lqcd_last_error().decode()


def launch_count() -> int:
    return int(lib().lqcd_launch_count())


def set_fine_tile(tile=None):
    _check(lib().lqcd_set_fine_tile(_i4(tile) if tile is not None else None), "lqcd_set_fine_tile")


def set_knob(name: str, value: int):
    _check(lib().lqcd_set_knob(name.encode(), int(value)), "lqcd_set_knob")


# ---- native sizes ------------------------------------------------------------------------------------
def native_spinor_reals(dims) -> int:
    return int(lib().lqcd_native_spinor_reals(_i4(dims)))


def native_gauge_reals(dims, links12=False) -> int:
    return int(lib().lqcd_native_gauge_reals(_i4(dims), LINKS_12 if links12 else 0))


def native_clover_reals(dims) -> int:
    return int(lib().lqcd_native_clover_reals(_i4(dims)))


def native_nullvecs_reals(dims, block, nvec) -> int:
    return int(lib().lqcd_native_nullvecs_reals(_i4(dims), _i4(block), int(nvec)))


def native_coarse_vec_reals(cdims, nvec) -> int:
    return int(lib().lqcd_native_coarse_vec_reals(_i4(cdims), int(nvec)))


def native_coarse_mat_reals(cdims, nvec) -> int:
    return int(lib().lqcd_native_coarse_mat_reals(_i4(cdims), int(nvec)))


def host_workspace_bytes(dims, block, nvec, dtype=torch.float32) -> int:
    fn = lib().lqcd_host_workspace_bytes if dtype == torch.float32 else lib().lqcd_host_workspace_bytes_f64
    return int(fn(_i4(dims), _i4(block), int(nvec)))


def empty_spinor(dims, dtype=torch.float32, device="cuda") -> torch.Tensor:
    return torch.zeros(native_spinor_reals(dims), dtype=dtype, device=device)


# ---- layout helpers (allocate the destination, then one C call) ------------------------------------------
def pack_spinor(src: torch.Tensor, dims, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    sfx = _sfx(src)
    _need(src, 24 * _vol(dims), "src")
    _need(out, _sz("spinor", _t4(dims)), "out")
    dst = out if out is not None else torch.zeros(native_spinor_reals(dims), dtype=_rdtype(sfx), device=src.device)
    _check(getattr(lib(), f"lqcd_pack_spinor_{sfx}")(_dev_ptr(dst), _dev_ptr(src), _i4(dims), _stream(stream, src, out)),
           "lqcd_pack_spinor")
    return dst


def unpack_spinor(src: torch.Tensor, dims, stream=None) -> torch.Tensor:
    """native -> canonical complex tensor of shape (V, 4, 3)"""
    sfx = _sfx(src)
    _need(src, _sz("spinor", _t4(dims)), "src")
    v = 1
    for d in dims:
        v *= int(d)
    dst = torch.empty((v, 4, 3, 2), dtype=_rdtype(sfx), device=src.device)
    _check(getattr(lib(), f"lqcd_unpack_spinor_{sfx}")(_dev_ptr(dst), _dev_ptr(src), _i4(dims), _stream(stream, src)),
           "lqcd_unpack_spinor")
    return torch.view_as_complex(dst)


def pack_gauge(src: torch.Tensor, dims, links12=False, stream=None) -> torch.Tensor:
    sfx = _sfx(src)
    _need(src, 4 * 18 * _vol(dims), "src")
    dst = torch.zeros(native_gauge_reals(dims, links12), dtype=_rdtype(sfx), device=src.device)
    _check(getattr(lib(), f"lqcd_pack_gauge_{sfx}")(_dev_ptr(dst), _dev_ptr(src), _i4(dims),
                                                    LINKS_12 if links12 else 0, _stream(stream, src, links12)), "lqcd_pack_gauge")
    return dst


def pack_clover(src: torch.Tensor, dims, stream=None) -> torch.Tensor:
    sfx = _sfx(src)
    _need(src, 2 * 72 * _vol(dims), "src")
    dst = torch.zeros(native_clover_reals(dims), dtype=_rdtype(sfx), device=src.device)
    _check(getattr(lib(), f"lqcd_pack_clover_{sfx}")(_dev_ptr(dst), _dev_ptr(src), _i4(dims), _stream(stream, src)),
           "lqcd_pack_clover")
    return dst


def unpack_clover(src: torch.Tensor, dims, stream=None) -> torch.Tensor:
    """native -> canonical complex tensor of shape (V, 2, 6, 6) (full Hermitian blocks)"""
    sfx = _sfx(src)
    _need(src, _sz("clover", _t4(dims)), "src")
    v = 1
    for d in dims:
        v *= int(d)
    dst = torch.empty((v, 2, 6, 6, 2), dtype=_rdtype(sfx), device=src.device)
    _check(getattr(lib(), f"lqcd_unpack_clover_{sfx}")(_dev_ptr(dst), _dev_ptr(src), _i4(dims), _stream(stream, src)),
           "lqcd_unpack_clover")
    return torch.view_as_complex(dst)


def clover_from_links(U_native18: torch.Tensor, kappa, csw, dims, stream=None) -> torch.Tensor:
    """F2: the native clover field built on the device from the native 18-real links (Q1)."""
    sfx = _sfx(U_native18)
    _need_fine(dims, links12=False, U=U_native18)
    dst = torch.zeros(native_clover_reals(dims), dtype=_rdtype(sfx), device=U_native18.device)
    k = (C.c_float if sfx == "f32" else C.c_double)
    _check(getattr(lib(), f"lqcd_clover_from_links_{sfx}")(_dev_ptr(dst), _dev_ptr(U_native18), k(kappa), k(csw),
                                                           _i4(dims), _stream(stream, U_native18)), "lqcd_clover_from_links")
    return dst


def orthonormalize_blocks(nullvecs_native: torch.Tensor, dims, block, nvec, stream=None) -> torch.Tensor:
    """F2: in-place block/chirality-wise orthonormalisation of the native null vectors."""
    sfx = _sfx(nullvecs_native)
    _need_transfer(dims, block, nvec, nullvecs=nullvecs_native)
    _check(getattr(lib(), f"lqcd_orthonormalize_blocks_{sfx}")(_dev_ptr(nullvecs_native), _i4(dims), _i4(block),
                                                               int(nvec), _stream(stream, nullvecs_native)), "lqcd_orthonormalize_blocks")
    return nullvecs_native


def orthonormalize_degenerate_count(stream=None) -> int:
    """(aggregate, vector) pairs that orthonormalize_blocks wrote as zero since the last query (0 = full rank)."""
    n = int(lib().lqcd_orthonormalize_degenerate_count(_stream(stream)))
    if n < 0:
        raise LqcdError(n, "lqcd_orthonormalize_degenerate_count")
    return n


def galerkin_coarse(U_native18, clover, nullvecs, kappa, dims, bc, block, nvec, stream=None) -> torch.Tensor:
    """F2: the coarse matrix A[X][d][I][J] = <I|D_d|J> (Eq. 7) as a complex (Vc, 9, N, N) tensor."""
    sfx = _same_dtype(U_native18, clover, nullvecs)
    _need_fine(dims, links12=False, U=U_native18, clover=clover)
    _need_transfer(dims, block, nvec, nullvecs=nullvecs)
    rdt = _rdtype(sfx)
    cd = [int(l) // int(b) for l, b in zip(dims, block)]
    vc, n = cd[0] * cd[1] * cd[2] * cd[3], 2 * int(nvec)
    A = torch.zeros((vc, 9, n, n, 2), dtype=rdt, device=nullvecs.device)
    nbytes = int(lib().lqcd_galerkin_workspace_bytes(_i4(dims), _i4(block), int(nvec), 4 if sfx == "f32" else 8))
    ws = torch.empty(max(nbytes, 16), dtype=torch.uint8, device=nullvecs.device)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_galerkin_coarse_{sfx}")(_dev_ptr(A), _dev_ptr(U_native18), _dev_ptr(clover),
                                                         _dev_ptr(nullvecs), k, _i4(dims), _i4(bc), _i4(block),
                                                         int(nvec), _dev_ptr(ws), _stream(stream, U_native18, clover, nullvecs)),
           "lqcd_galerkin_coarse")
    return torch.view_as_complex(A)


def pack_nullvec(dst: torch.Tensor, src_vi: torch.Tensor, i: int, dims, block, nvec, stream=None):
    sfx = _same_dtype(dst, src_vi)
    _need_transfer(dims, block, nvec, nullvecs=dst)
    _need(src_vi, 24 * _vol(dims), "src_vi")
    _check(getattr(lib(), f"lqcd_pack_nullvec_{sfx}")(_dev_ptr(dst), _dev_ptr(src_vi), int(i), _i4(dims), _i4(block),
                                                      int(nvec), _stream(stream, dst, src_vi)), "lqcd_pack_nullvec")


def unpack_nullvec(src_native: torch.Tensor, i: int, dims, block, nvec, stream=None) -> torch.Tensor:
    sfx = _sfx(src_native)
    _need_transfer(dims, block, nvec, nullvecs=src_native)
    v = 1
    for d in dims:
        v *= int(d)
    dst = torch.empty((v, 4, 3, 2), dtype=_rdtype(sfx), device=src_native.device)
    _check(getattr(lib(), f"lqcd_unpack_nullvec_{sfx}")(_dev_ptr(dst), _dev_ptr(src_native), int(i), _i4(dims),
                                                        _i4(block), int(nvec), _stream(stream, src_native)), "lqcd_unpack_nullvec")
    return torch.view_as_complex(dst)


def pack_nullvecs(v: torch.Tensor, dims, block) -> torch.Tensor:
    """canonical (nvec, V, 4, 3) complex -> native; one lqcd_pack_nullvec call per vector."""
    sfx = _sfx(v)
    nvec = v.shape[0]
    dst = torch.zeros(native_nullvecs_reals(dims, block, nvec), dtype=_rdtype(sfx), device=v.device)
    for i in range(nvec):
        pack_nullvec(dst, v[i], i, dims, block, nvec)
    return dst


# ---- the hot path -------------------------------------------------------------------------------------
def wilson_clover_mult(out, inp, U, clover, kappa, dims, bc, dagger=False, links12=False, stream=None):
    """A1/A2: out = D in (or D^dag in), Eq. 1 / Eq. 2; all tensors native layout."""
    sfx = _same_dtype(out, inp, U, clover)
    _need_fine(dims, links12, (("out", out), ("in", inp)), U, clover)
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_wilson_clover_mult_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(U), _dev_ptr(clover),
                                                            k, _i4(dims), _i4(bc), flags, _stream(stream, out, inp, U, clover)),
           "lqcd_wilson_clover_mult")
    return out


def wilson_clover_dd_mult(out, inp, U, clover, kappa, dims, bc, domain, parity=0, dagger=False, links12=False,
                          stream=None):
    """F1: out = D_SAP in; parity 0 / 1 / 2 = all / even / odd domains (zero elsewhere)."""
    sfx = _same_dtype(out, inp, U, clover)
    _need_fine(dims, links12, (("out", out), ("in", inp)), U, clover)
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0) | {0: 0, 1: DOMAIN_EVEN, 2: DOMAIN_ODD}[parity]
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_wilson_clover_dd_mult_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(U),
                                                               _dev_ptr(clover), k, _i4(dims), _i4(bc), _i4(domain),
                                                               flags, _stream(stream, out, inp, U, clover)), "lqcd_wilson_clover_dd_mult")
    return out


def coarse_mult(out, inp, A, cdims, nvec, dagger=False, stream=None):
    """A3: out = D_c in, Eqs. 4, 7."""
    sfx = _same_dtype(out, inp, A)
    _need_coarse(cdims, nvec, (("out", out), ("in", inp)), A)
    _check(getattr(lib(), f"lqcd_coarse_mult_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(A), _i4(cdims), int(nvec),
                                                     DAGGER if dagger else 0, _stream(stream, out, inp, A, dagger)), "lqcd_coarse_mult")
    return out


def native_coarse_half_reals(cdims, nvec) -> int:
    return int(lib().lqcd_native_coarse_half_reals(_i4(cdims), int(nvec)))


def pack_coarse_half(A: torch.Tensor, cdims, nvec, stream=None) -> torch.Tensor:
    """Half storage of a coarse matrix: A_0 and the four forward blocks, complex (Vc, 5, N, N)."""
    sfx = _sfx(A)
    _need_coarse(cdims, nvec, A=A)
    n = 2 * int(nvec)
    Ah = torch.empty((_vol(cdims), 5, n, n, 2), dtype=_rdtype(sfx), device=A.device)
    _check(getattr(lib(), f"lqcd_pack_coarse_half_{sfx}")(_dev_ptr(Ah), _dev_ptr(A), _i4(cdims), int(nvec),
                                                          _stream(stream, A)), "lqcd_pack_coarse_half")
    return torch.view_as_complex(Ah)


def coarse_half_workspace(cdims, nvec, dtype=torch.float32, device="cuda") -> torch.Tensor:
    nb = int(lib().lqcd_coarse_half_workspace_bytes(_i4(cdims), int(nvec), 4 if dtype == torch.float32 else 8))
    return torch.empty(max(nb, 16), dtype=torch.uint8, device=device)


NOALLOC_SCRATCH_BYTES = 16 << 20  # LQCD_NOALLOC_SCRATCH_BYTES of include/lqcd_b200.h


def coarse_mult_half_noalloc(out, inp, Ah, cdims, nvec, dagger=False, stream=None):
    """lqcd_coarse_mult_half_noalloc_f32: coarse_mult_half (fp32) with its scratch in a static device array of the
    library (16 MiB) instead of a workspace -- the call allocates nothing.  Problems whose four scratch vectors exceed
    that are refused (LqcdError, EUNSUPPORTED); calls that overlap on the GPU race on the shared array."""
    sfx = _same_dtype(out, inp, Ah)
    if sfx != "f32":
        raise TypeError("coarse_mult_half_noalloc: fp32 only (the fp64 form takes a workspace: coarse_mult_half)")
    _need_coarse(cdims, nvec, (("out", out), ("in", inp)))
    _need(Ah, native_coarse_half_reals(cdims, nvec), "Ah")
    _check(lib().lqcd_coarse_mult_half_noalloc_f32(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(Ah), _i4(cdims), int(nvec),
                                                   DAGGER if dagger else 0, _stream(stream, out, inp, Ah)),
           "lqcd_coarse_mult_half_noalloc")
    return out


def coarse_mult_half(out, inp, Ah, cdims, nvec, dagger=False, ws=None, stream=None):
    """A3 on half storage: out = D_c in from A_0 and the forward blocks, the backward blocks being
    Gamma5c A_{+mu}(X - mu)^dag Gamma5c (Eqs. 2, 7)."""
    sfx = _same_dtype(out, inp, Ah)
    _need_coarse(cdims, nvec, (("out", out), ("in", inp)))
    _need(Ah, native_coarse_half_reals(cdims, nvec), "Ah")
    if ws is None:
        ws = coarse_half_workspace(cdims, nvec, _rdtype(sfx), out.device)
    _need_bytes(ws, int(lib().lqcd_coarse_half_workspace_bytes(_i4(cdims), int(nvec), 4 if sfx == "f32" else 8)), "ws")
    _check(getattr(lib(), f"lqcd_coarse_mult_half_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(Ah), _i4(cdims),
                                                          int(nvec), DAGGER if dagger else 0, _dev_ptr(ws),
                                                          _stream(stream, out, inp, Ah)), "lqcd_coarse_mult_half")
    return out


def restrict(out_c, in_f, nullvecs, dims, block, nvec, stream=None):
    """A4: Eq. 5.  (`restrict` is the paper's name; it shadows nothing in Python.)"""
    sfx = _same_dtype(out_c, in_f, nullvecs)
    _need_transfer(dims, block, nvec, (("in_f", in_f),), (("out_c", out_c),), nullvecs)
    _check(getattr(lib(), f"lqcd_restrict_{sfx}")(_dev_ptr(out_c), _dev_ptr(in_f), _dev_ptr(nullvecs), _i4(dims),
                                                  _i4(block), int(nvec), _stream(stream, out_c, in_f, nullvecs)), "lqcd_restrict")
    return out_c


def prolong(out_f, in_c, nullvecs, dims, block, nvec, stream=None):
    """A5: Eq. 6."""
    sfx = _same_dtype(out_f, in_c, nullvecs)
    _need_transfer(dims, block, nvec, (("out_f", out_f),), (("in_c", in_c),), nullvecs)
    _check(getattr(lib(), f"lqcd_prolong_{sfx}")(_dev_ptr(out_f), _dev_ptr(in_c), _dev_ptr(nullvecs), _i4(dims),
                                                 _i4(block), int(nvec), _stream(stream, out_f, in_c, nullvecs)), "lqcd_prolong")
    return out_f


# ---- F3: residual, blocked BLAS-1, inner-domain solver, SAP ------------------------------------------------------
def wilson_clover_residual(r, b, x, U, clover, kappa, dims, bc, links12=False, stream=None):
    """r = b - D x in one pass."""
    sfx = _same_dtype(r, b, x, U, clover)
    _need_fine(dims, links12, (("r", r), ("b", b), ("x", x)), U, clover)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_wilson_clover_residual_{sfx}")(_dev_ptr(r), _dev_ptr(b), _dev_ptr(x), _dev_ptr(U),
                                                                _dev_ptr(clover), k, _i4(dims), _i4(bc),
                                                                LINKS_12 if links12 else 0, _stream(stream, r, b, x, U)),
           "lqcd_wilson_clover_residual")
    return r


def _ndomains(dims, domain) -> int:
    n = 1
    for l, d in zip(dims, domain):
        n *= int(l) // int(d)
    return n


def block_dotc(a, b, dims, domain, stream=None) -> torch.Tensor:
    """out[X] = <a|b> restricted to domain X; complex tensor of one entry per domain."""
    sfx = _same_dtype(a, b)
    _need_fine(dims, spinors=(("a", a), ("b", b)))
    out = torch.zeros((_ndomains(dims, domain), 2), dtype=_rdtype(sfx), device=a.device)
    _check(getattr(lib(), f"lqcd_block_dotc_{sfx}")(_dev_ptr(out), _dev_ptr(a), _dev_ptr(b), _i4(dims), _i4(domain),
                                                    _stream(stream, a, b)), "lqcd_block_dotc")
    return torch.view_as_complex(out)


def block_caxpy(y, coef, a, dims, domain, stream=None):
    """y(x) += coef[X(x)] a(x)."""
    sfx = _same_dtype(y, coef, a)
    _need_fine(dims, spinors=(("y", y), ("a", a)))
    _need(coef, 2 * _ndomains(dims, domain), "coef")
    _check(getattr(lib(), f"lqcd_block_caxpy_{sfx}")(_dev_ptr(y), _dev_ptr(coef), _dev_ptr(a), _i4(dims), _i4(domain),
                                                     _stream(stream, y, coef, a)), "lqcd_block_caxpy")
    return y


def mr_workspace(dims, domain, dtype=torch.float32, device="cuda"):
    """Scratch for mr_domain_solve / sap (None when the shared-memory-resident kernel applies)."""
    n = int(lib().lqcd_mr_workspace_bytes(_i4(dims), _i4(domain), 4 if dtype == torch.float32 else 8))
    return torch.empty(n, dtype=torch.uint8, device=device) if n else None


def _ws_ptr(ws):
    return C.c_void_p(None) if ws is None else _dev_ptr(ws)


def mr_domain_solve(z, r, U, clover, kappa, dims, bc, domain, parity=0, niter=6, accumulate=False, ws=None,
                    stream=None):
    """z (+)= M_SAP^(g) r: niter minimal-residual iterations in every domain of group `parity`."""
    sfx = _same_dtype(z, r, U, clover)
    _need_fine(dims, False, (("z", z), ("r", r)), U, clover)
    _need_bytes(ws, _mr_ws_bytes(dims, domain, sfx), "ws")
    flags = {0: 0, 1: DOMAIN_EVEN, 2: DOMAIN_ODD}[parity] | (ACCUMULATE if accumulate else 0)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_mr_domain_solve_{sfx}")(_dev_ptr(z), _dev_ptr(r), _dev_ptr(U), _dev_ptr(clover), k,
                                                         _i4(dims), _i4(bc), _i4(domain), flags, int(niter),
                                                         _ws_ptr(ws), _stream(stream, z, r, U, clover)), "lqcd_mr_domain_solve")
    return z


def sap(x, r, b, U, clover, kappa, dims, bc, domain, n_sap=4, n_mr=6, initial_guess=False, final_residual=True,
        ws=None, stream=None):
    """SAP with fixed iterations: x = SAP_n(b) (or x0 + SAP_n(b - D x0)); r = b - D x."""
    sfx = _same_dtype(x, r, b, U, clover)
    _need_fine(dims, False, (("x", x), ("r", r), ("b", b)), U, clover)
    _need_bytes(ws, _mr_ws_bytes(dims, domain, sfx), "ws")
    flags = (SAP_INITIAL_GUESS if initial_guess else 0) | (0 if final_residual else SAP_NO_FINAL_RESIDUAL)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_sap_{sfx}")(_dev_ptr(x), _dev_ptr(r), _dev_ptr(b), _dev_ptr(U), _dev_ptr(clover), k,
                                             _i4(dims), _i4(bc), _i4(domain), int(n_sap), int(n_mr), flags,
                                             _ws_ptr(ws), _stream(stream, x, r, b, U)), "lqcd_sap")
    return x

def coarse_bicgstab(x, b, A, cdims, nvec, niter, r_out=None, ws=None, half=False, stream=None):
    """(1b) of PAPER.md:116: niter BiCGStab iterations (listing PAPER.md:71, M = 1, x0 = 0) for D_c x = b.
    half: A is the half storage of the coarse matrix (pack_coarse_half)."""
    sfx = _same_dtype(x, b, A)
    _need_coarse(cdims, nvec, (("x", x), ("b", b), ("r_out", r_out)), None if half else A)
    if half:
        _need(A, native_coarse_half_reals(cdims, nvec), "Ah")
    if ws is None:
        nb = int(lib().lqcd_coarse_bicgstab_workspace_bytes(_i4(cdims), int(nvec), 4 if sfx == "f32" else 8))
        ws = torch.empty(nb, dtype=torch.uint8, device=x.device)
    name = f"lqcd_coarse_bicgstab_{'half_' if half else ''}{sfx}"
    _check(getattr(lib(), name)(_dev_ptr(x), _ws_ptr(r_out), _dev_ptr(b), _dev_ptr(A), _i4(cdims), int(nvec), int(niter),
                                _dev_ptr(ws), _stream(stream, x, b, A, r_out)), name)
    return x


def mg_workspace(dims, block, nvec, dtype=torch.float32, device="cuda") -> torch.Tensor:
    nb = int(lib().lqcd_mg_workspace_bytes(_i4(dims), _i4(block), int(nvec), 4 if dtype == torch.float32 else 8))
    return torch.empty(nb, dtype=torch.uint8, device=device)


def mg_vcycle(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, A, n_coarse=8, n_sap=4, n_mr=6, ws=None,
              half=False, stream=None):
    """x = M b: one V-cycle of the multigrid preconditioner.  half: A is the half storage."""
    sfx = _same_dtype(x, b, U, clover, nullvecs, A)
    _need_fine(dims, False, (("x", x), ("b", b)), U, clover)
    _need_transfer(dims, block, nvec, nullvecs=nullvecs)
    if half:
        _need(A, native_coarse_half_reals(_cdims(dims, block), nvec), "Ah")
    else:
        _need_coarse(_cdims(dims, block), nvec, A=A)
    if ws is None:
        ws = mg_workspace(dims, block, nvec, dtype=_rdtype(sfx), device=x.device)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    name = f"lqcd_mg_vcycle_{'half_' if half else ''}{sfx}"
    _check(getattr(lib(), name)(_dev_ptr(x), _dev_ptr(b), _dev_ptr(U), _dev_ptr(clover), k, _i4(dims), _i4(bc),
                                _i4(block), int(nvec), _dev_ptr(nullvecs), _dev_ptr(A), int(n_coarse), int(n_sap),
                                int(n_mr), _dev_ptr(ws), _stream(stream, x, b, U, clover)), name)
    return x

def coarse_mult_mrhs(out, inp, A, cdims, nvec, dagger=False, stream=None):
    """F4: out[k] = D_c in[k] for all k at once; in, out of shape (K, Vc, 2, nvec) complex."""
    sfx = _same_dtype(out, inp, A)
    nrhs = int(inp.shape[0])
    _need_coarse(cdims, nvec, (("out", out), ("in", inp)), A, k=nrhs)
    _check(getattr(lib(), f"lqcd_coarse_mult_mrhs_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(A), _i4(cdims),
                                                          int(nvec), nrhs, DAGGER if dagger else 0, _stream(stream, out, inp, A, dagger)),
           "lqcd_coarse_mult_mrhs")
    return out

def wilson_clover_mult_mrhs(out, inp, U, clover, kappa, dims, bc, dagger=False, links12=False, stream=None):
    """F4: out[k] = D in[k] for all k at once; in, out of shape (K, native_spinor_reals(dims))."""
    sfx = _same_dtype(out, inp, U, clover)
    _need_fine(dims, links12, (("out", out), ("in", inp)), U, clover, k=int(inp.shape[0]))
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_wilson_clover_mult_mrhs_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(U),
                                                                 _dev_ptr(clover), k, _i4(dims), _i4(bc),
                                                                 int(inp.shape[0]), flags, _stream(stream, out, inp, U, clover)),
           "lqcd_wilson_clover_mult_mrhs")
    return out

def restrict_mrhs(out_c, in_f, nullvecs, dims, block, nvec, stream=None):
    """Eq. 5 for several fine vectors at once: in_f (K, native spinor), out_c (K, Vc, 2, nvec)."""
    sfx = _same_dtype(out_c, in_f, nullvecs)
    _need_transfer(dims, block, nvec, (("in_f", in_f),), (("out_c", out_c),), nullvecs, k=int(in_f.shape[0]))
    _check(getattr(lib(), f"lqcd_restrict_mrhs_{sfx}")(_dev_ptr(out_c), _dev_ptr(in_f), _dev_ptr(nullvecs), _i4(dims),
                                                       _i4(block), int(nvec), int(in_f.shape[0]), _stream(stream, out_c, in_f, nullvecs)),
           "lqcd_restrict_mrhs")
    return out_c

def coarse_bicgstab_mrhs(x, b, A, cdims, nvec, niter, r_out=None, ws=None, stream=None):
    """niter BiCGStab iterations for D_c x_k = b_k, all k at once; x, b of shape (K, Vc, 2, nvec)."""
    sfx = _same_dtype(x, b, A)
    nrhs = int(b.shape[0])
    _need_coarse(cdims, nvec, (("x", x), ("b", b), ("r_out", r_out)), A, k=nrhs)
    if ws is None:
        nb = int(lib().lqcd_coarse_bicgstab_mrhs_workspace_bytes(_i4(cdims), int(nvec), nrhs,
                                                                 4 if sfx == "f32" else 8))
        ws = torch.empty(nb, dtype=torch.uint8, device=x.device)
    _check(getattr(lib(), f"lqcd_coarse_bicgstab_mrhs_{sfx}")(_dev_ptr(x), _ws_ptr(r_out), _dev_ptr(b), _dev_ptr(A),
                                                              _i4(cdims), int(nvec), nrhs, int(niter), _dev_ptr(ws),
                                                              _stream(stream, x, b, A, r_out)), "lqcd_coarse_bicgstab_mrhs")
    return x

def prolong_mrhs(out_f, in_c, nullvecs, dims, block, nvec, stream=None):
    """Eq. 6 for several coarse vectors at once: in_c (K, Vc, 2, nvec), out_f (K, native spinor)."""
    sfx = _same_dtype(out_f, in_c, nullvecs)
    _need_transfer(dims, block, nvec, (("out_f", out_f),), (("in_c", in_c),), nullvecs, k=int(in_c.shape[0]))
    _check(getattr(lib(), f"lqcd_prolong_mrhs_{sfx}")(_dev_ptr(out_f), _dev_ptr(in_c), _dev_ptr(nullvecs), _i4(dims),
                                                      _i4(block), int(nvec), int(in_c.shape[0]), _stream(stream, out_f, in_c, nullvecs)),
           "lqcd_prolong_mrhs")
    return out_f


def mg_vcycle_mrhs(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, A, n_coarse=8, n_sap=4, n_mr=6, ws=None,
                   stream=None):
    """x[k] = M b[k] for all k: restrictions, coarse solves and prolongations shared, the smoother one by one."""
    sfx = _same_dtype(x, b, U, clover, nullvecs, A)
    nrhs = int(b.shape[0])
    _need_fine(dims, False, (("x", x), ("b", b)), U, clover, k=nrhs)
    _need_transfer(dims, block, nvec, nullvecs=nullvecs)
    _need_coarse(_cdims(dims, block), nvec, A=A)
    if ws is None:
        nb = int(lib().lqcd_mg_mrhs_workspace_bytes(_i4(dims), _i4(block), int(nvec), nrhs, 4 if sfx == "f32" else 8))
        ws = torch.empty(nb, dtype=torch.uint8, device=x.device)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_mg_vcycle_mrhs_{sfx}")(_dev_ptr(x), _dev_ptr(b), _dev_ptr(U), _dev_ptr(clover), k,
                                                        _i4(dims), _i4(bc), _i4(block), int(nvec), _dev_ptr(nullvecs),
                                                        _dev_ptr(A), nrhs, int(n_coarse), int(n_sap), int(n_mr),
                                                        _dev_ptr(ws), _stream(stream, x, b, U, clover)), "lqcd_mg_vcycle_mrhs")
    return x

def sap_mrhs(x, r, b, U, clover, kappa, dims, bc, domain, n_sap=4, n_mr=6, initial_guess=False, final_residual=True,
             ws=None, stream=None):
    """SAP for all right-hand sides b[k] at once; x, r, b of shape (K, native spinor)."""
    sfx = _same_dtype(x, r, b, U, clover)
    _need_fine(dims, False, (("x", x), ("r", r), ("b", b)), U, clover, k=int(b.shape[0]))
    flags = (SAP_INITIAL_GUESS if initial_guess else 0) | (0 if final_residual else SAP_NO_FINAL_RESIDUAL)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_sap_mrhs_{sfx}")(_dev_ptr(x), _dev_ptr(r), _dev_ptr(b), _dev_ptr(U), _dev_ptr(clover),
                                                  k, _i4(dims), _i4(bc), _i4(domain), int(b.shape[0]), int(n_sap),
                                                  int(n_mr), flags, _ws_ptr(ws), _stream(stream, x, r, b, U)), "lqcd_sap_mrhs")
    return x

# ---- end-to-end calls on host vectors (fp32) --------------------------------------------------------------
class DevPtr:
    """A raw device pointer standing in for a real tensor in this module's calls: what the library's callbacks hand
    back (lqcd_apply_fn).  dtype: torch.float32 / torch.float64."""

    is_cuda = True

    def __init__(self, ptr, dtype):
        self._ptr, self.dtype = int(ptr), dtype

    def data_ptr(self):
        return self._ptr

    def is_contiguous(self):
        return True

    def is_complex(self):
        return False


def coarse_bicgstab_hooks(x, b, cdims, nvec, niter, apply, reduce=None, r_out=None, ws=None, stream=None):
    """The coarse solver with the operator and the cross-rank sum supplied by the caller (sharded lattice):
    apply(out: DevPtr, inp: DevPtr) enqueues out = D_c inp on the current stream; reduce(t: Tensor) sums the real
    tensor t over the ranks in place (None: single rank).  The BiCGStab recurrences run in the library's kernels."""
    sfx = _same_dtype(x, b)
    _need_coarse(cdims, nvec, (("x", x), ("b", b), ("r_out", r_out)))
    rdt = _rdtype(sfx)
    if ws is None:
        nb = int(lib().lqcd_coarse_bicgstab_workspace_bytes(_i4(cdims), int(nvec), 4 if sfx == "f32" else 8))
        ws = torch.empty(nb, dtype=torch.uint8, device=x.device)
    st = _stream(stream, x, b, apply, reduce)
    failure = []

    def _apply(out_p, in_p, stream_p, _user):
        try:
            if (stream_p or 0) != (st.value or 0):
                raise RuntimeError("apply hook called on a foreign stream")
            apply(DevPtr(out_p, rdt), DevPtr(in_p, rdt))
            return 0
        except BaseException as e:  # noqa: BLE001 -- must not propagate through the C frame
            failure.append(e)
            return 1

    def _reduce(ptr, count, real_bytes, stream_p, _user):
        try:
            if (stream_p or 0) != (st.value or 0):
                raise RuntimeError("reduce hook called on a foreign stream")
            off = int(ptr) - ws.data_ptr()
            reduce(ws[off:off + int(count) * int(real_bytes)].view(rdt))
            return 0
        except BaseException as e:  # noqa: BLE001
            failure.append(e)
            return 1

    a_fn = _lib.APPLY_FN(_apply)
    r_fn = _lib.REDUCE_FN(_reduce) if reduce is not None else C.cast(None, _lib.REDUCE_FN)
    rc = getattr(lib(), f"lqcd_coarse_bicgstab_hooks_{sfx}")(_dev_ptr(x), _ws_ptr(r_out), _dev_ptr(b), _i4(cdims),
                                                            int(nvec), int(niter), a_fn, r_fn, None, _dev_ptr(ws), st)
    if failure:
        raise failure[0]
    _check(rc, "lqcd_coarse_bicgstab_hooks")
    return x


def halo_face_reals(dims, mu) -> int:
    return int(lib().lqcd_halo_face_reals(_i4(dims), int(mu)))


def halo_buffers(dims, part_mask, dtype=torch.float32, device="cuda"):
    """The 8 face buffers of one side of the exchange (None for unpartitioned directions)."""
    return [torch.empty(halo_face_reals(dims, f >> 1), dtype=dtype, device=device) if (part_mask >> (f >> 1)) & 1
            else None for f in range(8)]


def _p8(bufs):
    return (C.c_void_p * 8)(*[None if b is None else _real(b).data_ptr() for b in bufs])


def wilson_clover_halo_pack(send, inp, U, dims, part_mask, dagger=False, links12=False, stream=None):
    """Sharded D, step 1: the projected half spinors of the partitioned faces of `inp` into send[8]."""
    sfx = _same_dtype(inp, U, *[b for b in send if b is not None])
    _need_fine(dims, links12, (("in", inp),), U)
    _need_faces(send, [halo_face_reals(dims, f >> 1) for f in range(8)], part_mask, "send")
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0)
    _check(getattr(lib(), f"lqcd_wilson_clover_halo_pack_{sfx}")(_p8(send), _dev_ptr(inp), _dev_ptr(U), _i4(dims),
                                                                 int(part_mask), flags, _stream(stream, send, inp, U, dagger)),
           "lqcd_wilson_clover_halo_pack")
    return send


def wilson_clover_mult_interior(out, inp, U, clover, kappa, dims, bc, part_mask, dagger=False, links12=False,
                                stream=None):
    """Sharded D, step 2: D on the local lattice with the hops leaving it in partitioned directions switched off."""
    sfx = _same_dtype(out, inp, U, clover)
    _need_fine(dims, links12, (("out", out), ("in", inp)), U, clover)
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    _check(getattr(lib(), f"lqcd_wilson_clover_mult_interior_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(U),
                                                                     _dev_ptr(clover), k, _i4(dims), _i4(bc),
                                                                     int(part_mask), flags, _stream(stream, out, inp, U, clover)),
           "lqcd_wilson_clover_mult_interior")
    return out


def wilson_clover_residual_interior(r, b, x, U, clover, kappa, dims, bc, part_mask, links12=False, domain=None,
                                    parity=0, stream=None):
    """Sharded residual, interior pass: r = b - (D without the leaving hops) x; complete it with
    wilson_clover_halo_add(r, recv, U, -kappa, ...).  parity 1 / 2 with a domain: only the even / odd domains'
    sites are computed, the others left as they are."""
    sfx = _same_dtype(r, b, x, U, clover)
    _need_fine(dims, links12, (("r", r), ("b", b), ("x", x)), U, clover)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    flags = (LINKS_12 if links12 else 0) | {0: 0, 1: DOMAIN_EVEN, 2: DOMAIN_ODD}[parity]
    _check(getattr(lib(), f"lqcd_wilson_clover_residual_interior_{sfx}")(
        _dev_ptr(r), _dev_ptr(b), _dev_ptr(x), _dev_ptr(U), _dev_ptr(clover), k, _i4(dims), _i4(bc),
        None if domain is None else _i4(domain), int(part_mask), flags, _stream(stream, r, b, x, U)),
        "lqcd_wilson_clover_residual_interior")
    return r


def wilson_clover_halo_add(out, recv, U, kappa, dims, face_phase, part_mask, dagger=False, links12=False,
                           stream=None):
    """Sharded D, step 3: out -= kappa * (the hops served by the received faces recv[8])."""
    sfx = _same_dtype(out, U, *[b for b in recv if b is not None])
    _need_fine(dims, links12, (("out", out),), U)
    _need_faces(recv, [halo_face_reals(dims, f >> 1) for f in range(8)], part_mask, "recv")
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    ph = (C.c_int * 8)(*[int(v) for v in face_phase])
    _check(getattr(lib(), f"lqcd_wilson_clover_halo_add_{sfx}")(_dev_ptr(out), _p8(recv), _dev_ptr(U), k, _i4(dims),
                                                                ph, int(part_mask), flags, _stream(stream, out, recv, U, face_phase)),
           "lqcd_wilson_clover_halo_add")
    return out


def coarse_halo_face_reals(cdims, nvec, mu) -> int:
    return int(lib().lqcd_coarse_halo_face_reals(_i4(cdims), int(nvec), int(mu)))


def coarse_halo_buffers(cdims, nvec, part_mask, dtype=torch.float32, device="cuda"):
    return [torch.empty(coarse_halo_face_reals(cdims, nvec, f >> 1), dtype=dtype, device=device)
            if (part_mask >> (f >> 1)) & 1 else None for f in range(8)]


def coarse_halo_pack(send, inp, cdims, nvec, part_mask, stream=None):
    """Sharded D_c, step 1: the coarse vectors of the partitioned faces of `inp` into send[8]."""
    sfx = _same_dtype(inp, *[b for b in send if b is not None])
    _need_coarse(cdims, nvec, (("in", inp),))
    _need_faces(send, [coarse_halo_face_reals(cdims, nvec, f >> 1) for f in range(8)], part_mask, "send")
    _check(getattr(lib(), f"lqcd_coarse_halo_pack_{sfx}")(_p8(send), _dev_ptr(inp), _i4(cdims), int(nvec),
                                                          int(part_mask), _stream(stream, send, inp)), "lqcd_coarse_halo_pack")
    return send


def coarse_mult_interior(out, inp, A, cdims, nvec, part_mask, dagger=False, stream=None):
    """Sharded D_c, step 2: D_c on the local coarse lattice without the blocks of hops that leave it."""
    sfx = _same_dtype(out, inp, A)
    _need_coarse(cdims, nvec, (("out", out), ("in", inp)), A)
    _check(getattr(lib(), f"lqcd_coarse_mult_interior_{sfx}")(_dev_ptr(out), _dev_ptr(inp), _dev_ptr(A), _i4(cdims),
                                                              int(nvec), int(part_mask), DAGGER if dagger else 0,
                                                              _stream(stream, out, inp, A, dagger)), "lqcd_coarse_mult_interior")
    return out


def coarse_halo_add(out, recv, A, cdims, nvec, part_mask, dagger=False, stream=None):
    """Sharded D_c, step 3: out += the blocks of the leaving hops applied to the received faces recv[8]."""
    sfx = _same_dtype(out, A, *[b for b in recv if b is not None])
    _need_coarse(cdims, nvec, (("out", out),), A)
    _need_faces(recv, [coarse_halo_face_reals(cdims, nvec, f >> 1) for f in range(8)], part_mask, "recv")
    _check(getattr(lib(), f"lqcd_coarse_halo_add_{sfx}")(_dev_ptr(out), _p8(recv), _dev_ptr(A), _i4(cdims), int(nvec),
                                                         int(part_mask), DAGGER if dagger else 0, _stream(stream, out, recv, A, dagger)),
           "lqcd_coarse_halo_add")
    return out


def wilson_clover_mult_host(out_host, in_host, U, clover, kappa, dims, bc, ws, dagger=False, links12=False,
                            stream=None):
    sfx = _same_dtype(out_host, in_host, U, clover)
    _need_fine(dims, links12, U=U, clover=clover)
    _need(out_host, 24 * _vol(dims), "out_host")
    _need(in_host, 24 * _vol(dims), "in_host")
    _need_bytes(ws, host_workspace_bytes_fine(dims, sfx), "ws")
    flags = (DAGGER if dagger else 0) | (LINKS_12 if links12 else 0)
    k = C.c_float(kappa) if sfx == "f32" else C.c_double(kappa)
    what = f"lqcd_wilson_clover_mult_host_{sfx}"
    _check(getattr(lib(), what)(_host_ptr(out_host), _host_ptr(in_host), _dev_ptr(U), _dev_ptr(clover), k, _i4(dims),
                                _i4(bc), flags, _dev_ptr(ws), _stream(stream, out_host, in_host, U, clover)), what)
    return out_host


def coarse_mult_host(out_host, in_host, A, cdims, nvec, ws, dagger=False, stream=None):
    sfx = _same_dtype(out_host, in_host, A)
    what = f"lqcd_coarse_mult_host_{sfx}"
    _need_coarse(cdims, nvec, (("out_host", out_host), ("in_host", in_host)), A)
    _need_bytes(ws, 2 * ((_sz("cvec", _t4(cdims), n=int(nvec)) * (4 if sfx == "f32" else 8) + 255) // 256 * 256), "ws")
    _check(getattr(lib(), what)(_host_ptr(out_host), _host_ptr(in_host), _dev_ptr(A), _i4(cdims), int(nvec),
                                DAGGER if dagger else 0, _dev_ptr(ws), _stream(stream, out_host, in_host, A, ws)), what)
    return out_host


def restrict_host(out_c_host, in_f_host, nullvecs, dims, block, nvec, ws, stream=None):
    sfx = _same_dtype(out_c_host, in_f_host, nullvecs)
    what = f"lqcd_restrict_host_{sfx}"
    _need_transfer(dims, block, nvec, coarse=(("out_c_host", out_c_host),), nullvecs=nullvecs)
    _need(in_f_host, 24 * _vol(dims), "in_f_host")
    _need_bytes(ws, host_workspace_bytes(dims, block, nvec, _rdtype(sfx)), "ws")
    _check(getattr(lib(), what)(_host_ptr(out_c_host), _host_ptr(in_f_host), _dev_ptr(nullvecs), _i4(dims),
                                _i4(block), int(nvec), _dev_ptr(ws), _stream(stream, out_c_host, in_f_host, nullvecs, ws)), what)
    return out_c_host


def prolong_host(out_f_host, in_c_host, nullvecs, dims, block, nvec, ws, stream=None):
    sfx = _same_dtype(out_f_host, in_c_host, nullvecs)
    what = f"lqcd_prolong_host_{sfx}"
    _need_transfer(dims, block, nvec, coarse=(("in_c_host", in_c_host),), nullvecs=nullvecs)
    _need(out_f_host, 24 * _vol(dims), "out_f_host")
    _need_bytes(ws, host_workspace_bytes(dims, block, nvec, _rdtype(sfx)), "ws")
    _check(getattr(lib(), what)(_host_ptr(out_f_host), _host_ptr(in_c_host), _dev_ptr(nullvecs), _i4(dims),
                                _i4(block), int(nvec), _dev_ptr(ws), _stream(stream, out_f_host, in_c_host, nullvecs, ws)), what)
    return out_f_host
