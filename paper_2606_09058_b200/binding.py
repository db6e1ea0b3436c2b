"""Thin ctypes binding of libnao.so (include/nao.h).  Argument marshalling ONLY: every step of the path runs in
the library's CUDA kernels.  PyTorch supplies device memory and the stream, nothing else.

Storage convention (same as paper_2606_09058_b200.synth): a batch of matrices is a contiguous tensor of shape
(batch, n, n) holding COLUMN-MAJOR items, i.e. ``t[b, j, i] == M_b(i, j)``; ``t.mT`` is the mathematical matrix.
Real = torch.float64, complex = torch.complex128 (interleaved re, im).

There is no CPU fallback: if the CUDA library cannot be built/loaded, or a tensor is not on a CUDA device, the
call raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

NAO_REAL, NAO_COMPLEX = 0, 1
NAO_S_FACTORED, NAO_NC_BLOCK_S, NAO_TRD_ONE_STAGE, NAO_TRD_TWO_STAGE, NAO_LOWDIN = 1, 2, 4, 8, 16
NAO_STREAM_GROUPS_2, NAO_STREAM_GROUPS_4, NAO_STREAM_GROUPS_8 = 32, 64, 96
NAO_PRUNED_LEVEL = 1.0e4

_LIB = None
_vp, _i, _l, _d, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_long, ctypes.c_double, ctypes.c_size_t
_szp = ctypes.POINTER(ctypes.c_size_t)
_dp = ctypes.POINTER(ctypes.c_double)

_SIGNATURES = {
    "nao_geneig_workspace": ([_i, _i, _i, ctypes.c_uint, _szp], _i),
    "nao_geneig": ([_i, _i, _i, ctypes.c_uint, _vp, _l, _l, _vp, _l, _l, _vp, _vp, _l, _l, _vp, _sz, _vp, _vp], _i),
    "nao_geneig_partial": ([_i, _i, _i, ctypes.c_uint, _i, _vp, _l, _l, _vp, _l, _l, _vp, _vp, _l, _l, _vp, _sz, _vp, _vp], _i),
    "nao_occupied_count": ([_i, _i, _vp, _d, ctypes.POINTER(ctypes.c_int), _vp], _i),
    "nao_scf_step_workspace": ([_i, _i, _i, ctypes.c_uint, _szp], _i),
    "nao_scf_step": ([_i, _i, _i, ctypes.c_uint, _vp, _l, _l, _vp, _l, _l, _dp, _d, _d, _vp, _dp, _vp, _vp, _l, _l, _vp, _l, _l,
                     ctypes.POINTER(ctypes.c_int), _vp, _sz, _vp, _vp], _i),
    "nao_solve_host_workspace": ([_i, _i, _i, ctypes.c_uint, _i, _szp], _i),
    "nao_solve_host": ([_i, _i, _i, ctypes.c_uint, _vp, _vp, _i, _dp, _d, _d, _vp, _dp, _vp, _vp, _vp, _sz, _vp], _i),
    "nao_fermi_workspace": ([_i, _i, _szp], _i),
    "nao_fermi_mu": ([_i, _i, _vp, _dp, _d, _d, _dp, _vp, _vp, _vp], _i),
    "nao_fermi_mu_static": ([_i, _i, _vp, _dp, _d, _d, _dp, _vp, _vp], _i),
    "nao_density_workspace": ([_i, _i, _i, _szp], _i),
    "nao_density_matrix": ([_i, _i, _i, _vp, _l, _l, _vp, _vp, _l, _l, _vp, _sz, _vp], _i),
    "nao_energy_weights": ([_i, _i, _vp, _vp, _vp, _vp], _i),
    "nao_fold_workspace": ([_i, _i, _szp], _i),
    "nao_fold_density": ([_i, _i, _i, _i, _vp, _l, _l, _dp, _dp, _dp, _vp, _l, _l, _vp, _sz, _vp], _i),
    "nao_set_lowdin_threshold": ([_d], _i),
    "nao_status_string": ([_i], ctypes.c_char_p),
    "nao_version": ([], ctypes.c_char_p),
    "nao_launch_count": ([], _l),
    "nao_dmma_peak": ([_dp, _vp], _i),
    "nao_profile_enable": ([_i], _i),
    "nao_profile_read": ([_dp, _i], _i),
    "nao_profile_phase_name": ([_i], ctypes.c_char_p),
    "nao_profile_kernel": ([_i, _dp, _dp, ctypes.POINTER(ctypes.c_int)], _i),
    "nao_profile_kernel_name": ([_i], ctypes.c_char_p),
    "nao_profile_kernel_launches": ([_i, _dp, _i], _i),
    "nao_gemm": ([_i, _i, _i, _i, _i, _i, _d, _vp, _l, _l, _vp, _l, _l, _d, _vp, _l, _l, _i, _i, _vp], _i),
    "nao_potrf_trtri": ([_i, _i, _i, _vp, _l, _l, _vp, _vp, _vp, _vp], _i),
    "nao_heev_workspace": ([_i, _i, _i, ctypes.c_uint, _szp], _i),
    "nao_heev": ([_i, _i, _i, ctypes.c_uint, _vp, _l, _l, _vp, _vp, _l, _l, _vp, _sz, _vp, _vp], _i),
    "nao_stedc_workspace": ([_i, _i, _szp], _i),
    "nao_stedc": ([_i, _i, _vp, _vp, _vp, _vp, _l, _l, _vp, _sz, _vp, _vp], _i),
}
EXPORTS = tuple(_SIGNATURES)


class NaoError(RuntimeError):
    pass


class _Lib:
    """ctypes handle with typed signatures; a symbol the header declares but the library lacks raises on use."""

    def __init__(self, path):
        self._cdll = ctypes.CDLL(path)
        self.path = path

    def __getattr__(self, name):
        argtypes, restype = _SIGNATURES[name]
        fn = getattr(self._cdll, name)          # AttributeError if the library lacks a declared symbol
        fn.argtypes = argtypes
        fn.restype = restype
        setattr(self, name, fn)
        return fn


def lib():
    """Load (building if stale) libnao.so.  Raises if that is impossible -- there is no fallback path."""
    global _LIB
    if _LIB is None:
        _LIB = _Lib(_build.build())
    return _LIB


def _check(rc, what):
    if rc != 0:
        raise NaoError("%s failed: status %d (%s)" % (what, rc, lib().nao_status_string(rc).decode()))


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.float64:
        return NAO_REAL
    if t.dtype == torch.complex128:
        return NAO_COMPLEX
    raise TypeError("expected float64 or complex128, got %s" % t.dtype)


_DEVICE = None      # the library's per-process state is bound to the first device it is used on (include/nao.h)


def _dev(t: torch.Tensor, name: str):
    global _DEVICE
    if not t.is_cuda:
        raise NaoError("%s must be a CUDA tensor (no CPU path exists)" % name)
    if _DEVICE is None:
        _DEVICE = t.device.index
    if t.device.index != _DEVICE or t.device.index != torch.cuda.current_device():
        raise NaoError("%s is on cuda:%s; the library is bound to cuda:%s, which must be the current device "
                       "(one device per process)" % (name, t.device.index, _DEVICE))
    if not t.is_contiguous():
        raise NaoError("%s must be contiguous" % name)
    return t.data_ptr()


def _stream(t: torch.Tensor):
    return torch.cuda.current_stream(t.device).cuda_stream


def _workspace(nbytes: int, device) -> torch.Tensor:
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def launch_count() -> int:
    return int(lib().nao_launch_count())


def profile_enable(on: bool = True) -> None:
    lib().nao_profile_enable(int(on))


def profile_read() -> dict:
    """Phase durations (ms) of the last nao_geneig call made with profiling enabled."""
    buf = (ctypes.c_double * 16)()
    k = lib().nao_profile_read(buf, 16)
    return {lib().nao_profile_phase_name(i).decode(): buf[i] for i in range(k)}


def profile_kernel(slot: int) -> dict:
    """Summed per-launch timings of one kernel class since profile_enable(): ms, algorithmic work, launches."""
    ms, work, k = ctypes.c_double(0), ctypes.c_double(0), ctypes.c_int(0)
    _check(lib().nao_profile_kernel(slot, ctypes.byref(ms), ctypes.byref(work), ctypes.byref(k)), "nao_profile_kernel")
    return {"name": lib().nao_profile_kernel_name(slot).decode(), "ms": ms.value, "work": work.value, "launches": k.value}


def profile_kernel_launches(slot: int, max_launches: int = 2048) -> list:
    """Per-launch durations (ms) of one kernel class since profile_enable(), in launch order."""
    buf = (ctypes.c_double * max_launches)()
    k = lib().nao_profile_kernel_launches(slot, buf, max_launches)
    if k < 0:
        raise NaoError("nao_profile_kernel_launches failed: %d" % k)
    return [buf[i] for i in range(k)]


def dmma_peak() -> float:
    """Measured FP64 tensor-pipe peak (TFLOP/s) of the current device: register-resident DMMA loop."""
    out = ctypes.c_double(0.0)
    _check(lib().nao_dmma_peak(ctypes.byref(out), None), "nao_dmma_peak")
    return out.value


def version() -> str:
    return lib().nao_version().decode()


# ------------------------------------------------------------------------------------------------- entry points
def geneig_workspace(n: int, batch: int, dtype: int, flags: int = 0) -> int:
    out = ctypes.c_size_t(0)
    _check(lib().nao_geneig_workspace(n, batch, dtype, flags, ctypes.byref(out)), "nao_geneig_workspace")
    return out.value


def geneig(H: torch.Tensor, S: torch.Tensor, flags: int = 0, work: torch.Tensor | None = None, n_vec: int | None = None):
    """nao_geneig on (batch, n, n) column-major items.  S is overwritten by its factor (see nao.h).
    n_vec (optional): back-transform only the n_vec lowest eigenvectors (nao_geneig_partial); the other columns of C are zero.
    Returns (E (batch, n), C (batch, n, n) column-major items, info (batch,) int32 device tensor)."""
    batch, n, _ = H.shape
    dt = _dtype_code(H)
    if flags & NAO_NC_BLOCK_S:
        sb, sn = S.shape[0], S.shape[-1]
        strideS = 0 if sb == 1 else sn * sn
        lds = sn
    else:
        strideS, lds = (0 if (S.shape[0] == 1 and batch > 1) else n * n), n     # one S shared by all items
    E = torch.empty((batch, n), dtype=torch.float64, device=H.device)
    C = torch.empty_like(H)
    info = torch.zeros(batch, dtype=torch.int32, device=H.device)
    need = geneig_workspace(n, batch, dt, flags)
    if work is None or work.numel() < need:
        work = _workspace(need, H.device)
    if n_vec is None:
        rc = lib().nao_geneig(n, batch, dt, flags, _dev(H, "H"), n, n * n, _dev(S, "S"), lds, strideS, _dev(E, "E"),
                              _dev(C, "C"), n, n * n, _dev(work, "work"), work.numel(), _dev(info, "info"), _stream(H))
        _check(rc, "nao_geneig")
    else:
        rc = lib().nao_geneig_partial(n, batch, dt, flags, int(n_vec), _dev(H, "H"), n, n * n, _dev(S, "S"), lds, strideS,
                                      _dev(E, "E"), _dev(C, "C"), n, n * n, _dev(work, "work"), work.numel(),
                                      _dev(info, "info"), _stream(H))
        _check(rc, "nao_geneig_partial")
    return E, C, info


def scf_step(H: torch.Tensor, S: torch.Tensor, weights, n_electrons: float, kT: float, flags: int = 0,
             work: torch.Tensor | None = None, out_D: torch.Tensor | None = None):
    """nao_scf_step: eigenvalues, Fermi level, the occupied eigenvectors and the density matrix in one call.
    Returns dict(E, mu, F, C, D, n_vec, info)."""
    batch, n, _ = H.shape
    dt = _dtype_code(H)
    if flags & NAO_NC_BLOCK_S:
        sn = S.shape[-1]
        strideS, lds = (0 if S.shape[0] == 1 else sn * sn), sn
    else:
        strideS, lds = (0 if (S.shape[0] == 1 and batch > 1) else n * n), n
    need = ctypes.c_size_t(0)
    _check(lib().nao_scf_step_workspace(n, batch, dt, flags, ctypes.byref(need)), "nao_scf_step_workspace")
    if work is None or work.numel() < need.value:
        work = _workspace(need.value, H.device)
    E = torch.empty((batch, n), dtype=torch.float64, device=H.device)
    F = torch.empty_like(E)
    C = torch.empty_like(H)
    D = torch.empty_like(H) if out_D is None else out_D
    info = torch.zeros(batch, dtype=torch.int32, device=H.device)
    w = (ctypes.c_double * batch)(*[float(x) for x in weights])
    mu, nvec = ctypes.c_double(0.0), ctypes.c_int(0)
    rc = lib().nao_scf_step(n, batch, dt, flags, _dev(H, "H"), n, n * n, _dev(S, "S"), lds, strideS, w, float(n_electrons),
                            float(kT), _dev(E, "E"), ctypes.byref(mu), _dev(F, "F"), _dev(C, "C"), n, n * n, _dev(D, "D"), n, n * n,
                            ctypes.byref(nvec), _dev(work, "work"), work.numel(), _dev(info, "info"), _stream(H))
    _check(rc, "nao_scf_step")
    return dict(E=E, mu=mu.value, F=F, C=C, D=D, n_vec=nvec.value, info=info)


def occupied_count(F: torch.Tensor, threshold: float = 1e-17) -> int:
    """nao_occupied_count: number of leading eigenvectors the density matrix needs (1 + last level with f >= threshold)."""
    batch, n = F.shape
    out = ctypes.c_int(0)
    _check(lib().nao_occupied_count(n, batch, _dev(F, "F"), float(threshold), ctypes.byref(out), _stream(F)), "nao_occupied_count")
    return out.value


def fermi_mu(E: torch.Tensor, weights, n_electrons: float, kT: float):
    """nao_fermi_mu: E (batch, n) device tensor, weights = g*w_k per item (host sequence).  Returns (mu, F)."""
    batch, n = E.shape
    w = (ctypes.c_double * batch)(*[float(x) for x in weights])
    need = ctypes.c_size_t(0)
    _check(lib().nao_fermi_workspace(n, batch, ctypes.byref(need)), "nao_fermi_workspace")
    work = _workspace(need.value, E.device)
    F = torch.empty_like(E)
    mu = ctypes.c_double(0.0)
    rc = lib().nao_fermi_mu(n, batch, _dev(E, "E"), w, float(n_electrons), float(kT), ctypes.byref(mu), _dev(F, "F"),
                            _dev(work, "work"), _stream(E))
    _check(rc, "nao_fermi_mu")
    return mu.value, F


FERMI_STATIC_MAX_STATES = 65536


def fermi_mu_static(E: torch.Tensor, weights, n_electrons: float, kT: float, out: torch.Tensor | None = None):
    """nao_fermi_mu_static: the Fermi level and occupations without any workspace -- for callers that may not allocate
    device memory (the host program owns all of it, or cudaMalloc's device-wide synchronisation is not acceptable where
    the call is made).  The library's own fixed 1.5 MiB scratch array is used instead, so at most
    FERMI_STATIC_MAX_STATES = 65536 states (E.numel()) are accepted; more raises NaoError (status 5).  Pass `out`
    (same shape as E, float64, same device) to receive the occupations: then this wrapper allocates nothing on the
    device either; without it a result tensor is created here for convenience.  All calls share that scratch array: do
    not overlap two of them on different streams.  Returns (mu, F) exactly as fermi_mu does."""
    batch, n = E.shape
    w = (ctypes.c_double * batch)(*[float(x) for x in weights])
    F = torch.empty_like(E) if out is None else out
    if F.shape != E.shape or F.dtype != torch.float64:
        raise NaoError("out must be a float64 tensor of the shape of E")
    mu = ctypes.c_double(0.0)
    rc = lib().nao_fermi_mu_static(n, batch, _dev(E, "E"), w, float(n_electrons), float(kT), ctypes.byref(mu),
                                   _dev(F, "out"), _stream(E))
    _check(rc, "nao_fermi_mu_static")
    return mu.value, F


def density_matrix(C: torch.Tensor, F: torch.Tensor, out: torch.Tensor | None = None):
    """nao_density_matrix: D_b = C_b diag(F_b) C_b^H, (batch, n, n) column-major items."""
    batch, n, _ = C.shape
    dt = _dtype_code(C)
    D = torch.empty_like(C) if out is None else out
    need = ctypes.c_size_t(0)
    _check(lib().nao_density_workspace(n, batch, dt, ctypes.byref(need)), "nao_density_workspace")
    work = _workspace(need.value, C.device)
    rc = lib().nao_density_matrix(n, batch, dt, _dev(C, "C"), n, n * n, _dev(F, "F"), _dev(D, "D"), n, n * n,
                                  _dev(work, "work"), work.numel(), _stream(C))
    _check(rc, "nao_density_matrix")
    return D


def solve_host(Hh: torch.Tensor, Sh: torch.Tensor, weights, n_electrons: float, kT: float, flags: int = 0,
               device=None, work: torch.Tensor | None = None, Eh: torch.Tensor | None = None, Dh: torch.Tensor | None = None):
    """nao_solve_host: the whole step with HOST tensors (pinned for asynchronous copies): Hh (batch, n, n), Sh (batch or 1,
    nS, nS) column-major items.  Returns dict(E, mu, D, info) of host tensors; the current stream of `device` is
    synchronised before returning."""
    if Hh.is_cuda or Sh.is_cuda:
        raise NaoError("solve_host takes host tensors")
    batch, n, _ = Hh.shape
    dt = _dtype_code(Hh)
    dev = torch.device(device if device is not None else "cuda:0")
    shared = 1 if (Sh.shape[0] == 1 and (batch > 1 or bool(flags & NAO_NC_BLOCK_S))) else 0
    if Sh.shape[0] == 1 and batch == 1:
        shared = 0
    need = ctypes.c_size_t(0)
    _check(lib().nao_solve_host_workspace(n, batch, dt, flags, shared, ctypes.byref(need)), "nao_solve_host_workspace")
    if work is None or work.numel() < need.value:
        work = _workspace(need.value, dev)
    Eh = torch.empty((batch, n), dtype=torch.float64).pin_memory() if Eh is None else Eh
    Dh = torch.empty_like(Hh).pin_memory() if Dh is None else Dh
    info = torch.zeros(batch, dtype=torch.int32).pin_memory()
    w = (ctypes.c_double * batch)(*[float(x) for x in weights])
    mu = ctypes.c_double(0.0)
    stream = torch.cuda.current_stream(dev)
    rc = lib().nao_solve_host(n, batch, dt, flags, Hh.data_ptr(), Sh.data_ptr(), shared, w, float(n_electrons), float(kT),
                              Eh.data_ptr(), ctypes.byref(mu), Dh.data_ptr(), info.data_ptr(), _dev(work, "work"), work.numel(),
                              stream.cuda_stream)
    _check(rc, "nao_solve_host")
    stream.synchronize()
    return dict(E=Eh, mu=mu.value, D=Dh, info=info)


def set_lowdin_threshold(rel: float):
    """nao_set_lowdin_threshold: relative pruning threshold of the NAO_LOWDIN route (0 = no pruning)."""
    _check(lib().nao_set_lowdin_threshold(float(rel)), "nao_set_lowdin_threshold")


def energy_weights(E: torch.Tensor, F: torch.Tensor):
    """nao_energy_weights: f*e per state; density_matrix(C, energy_weights(E, F)) is the energy-weighted DM."""
    batch, n = E.shape
    FE = torch.empty_like(F)
    _check(lib().nao_energy_weights(n, batch, _dev(E, "E"), _dev(F, "F"), _dev(FE, "FE"), _stream(E)), "nao_energy_weights")
    return FE


def fold_density(Dk: torch.Tensor, kpts, weights, Rvecs, real_out: bool = True):
    """nao_fold_density: D(R) = sum_k w_k exp(-i k.R) D(k).  Dk: (nk, n, n) complex column-major items; kpts (nk, 3),
    weights (nk,), Rvecs (nR, 3) host sequences.  Returns (nR, n, n) float64 (real_out) or complex128."""
    nk, n, _ = Dk.shape
    if Dk.dtype != torch.complex128:
        raise TypeError("D(k) must be complex128")
    hk = (ctypes.c_double * (3 * nk))(*[float(x) for row in kpts for x in row])
    hw = (ctypes.c_double * nk)(*[float(x) for x in weights])
    nR = len(Rvecs)
    hR = (ctypes.c_double * (3 * nR))(*[float(x) for row in Rvecs for x in row])
    DR = torch.empty((nR, n, n), dtype=torch.float64 if real_out else torch.complex128, device=Dk.device)
    need = ctypes.c_size_t(0)
    _check(lib().nao_fold_workspace(nk, nR, ctypes.byref(need)), "nao_fold_workspace")
    work = _workspace(need.value, Dk.device)
    rc = lib().nao_fold_density(n, nk, nR, NAO_REAL if real_out else NAO_COMPLEX, _dev(Dk, "Dk"), n, n * n, hk, hw, hR,
                                _dev(DR, "DR"), n, n * n, _dev(work, "work"), work.numel(), _stream(Dk))
    _check(rc, "nao_fold_density")
    return DR


# ------------------------------------------------------------------------------------------ building blocks
def gemm(A: torch.Tensor, B: torch.Tensor, opA: int = 0, opB: int = 0, alpha: float = 1.0, beta: float = 0.0,
         C: torch.Tensor | None = None, lower_only: bool = False):
    """C <- alpha op(A) op(B) + beta C.  A, B, C are (batch, cols, rows) column-major items (see module doc)."""
    batch = A.shape[0]
    dt = _dtype_code(A)
    a_rows, a_cols = A.shape[2], A.shape[1]
    b_rows, b_cols = B.shape[2], B.shape[1]
    m, k = (a_rows, a_cols) if opA == 0 else (a_cols, a_rows)
    k2, n = (b_rows, b_cols) if opB == 0 else (b_cols, b_rows)
    assert k == k2, (k, k2)
    if C is None:
        C = torch.zeros((batch, n, m), dtype=A.dtype, device=A.device)
    rc = lib().nao_gemm(dt, opA, opB, m, n, k, alpha, _dev(A, "A"), a_rows, a_rows * a_cols, _dev(B, "B"), b_rows,
                        b_rows * b_cols, beta, _dev(C, "C"), m, m * n, batch, int(lower_only), _stream(A))
    _check(rc, "nao_gemm")
    return C


def potrf_trtri(S: torch.Tensor):
    """In place on S (batch, n, n): lower = L, strict upper = strict upper of L^{-H}.  Returns (Linv, info)."""
    batch, n, _ = S.shape
    dt = _dtype_code(S)
    W = torch.zeros_like(S)
    T = torch.empty_like(S)
    info = torch.zeros(batch, dtype=torch.int32, device=S.device)
    rc = lib().nao_potrf_trtri(n, batch, dt, _dev(S, "S"), n, n * n, _dev(W, "W"), _dev(T, "T"), _dev(info, "info"),
                               _stream(S))
    _check(rc, "nao_potrf_trtri")
    return W, info


def heev(A: torch.Tensor, flags: int = 0):
    """Standard Hermitian eigenproblem (lower triangle of A referenced, A destroyed).  Returns (E, Z, info)."""
    batch, n, _ = A.shape
    dt = _dtype_code(A)
    need = ctypes.c_size_t(0)
    _check(lib().nao_heev_workspace(n, batch, dt, flags, ctypes.byref(need)), "nao_heev_workspace")
    work = _workspace(need.value, A.device)
    E = torch.empty((batch, n), dtype=torch.float64, device=A.device)
    Z = torch.empty_like(A)
    info = torch.zeros(batch, dtype=torch.int32, device=A.device)
    rc = lib().nao_heev(n, batch, dt, flags, _dev(A, "A"), n, n * n, _dev(E, "E"), _dev(Z, "Z"), n, n * n,
                        _dev(work, "work"), work.numel(), _dev(info, "info"), _stream(A))
    _check(rc, "nao_heev")
    return E, Z, info


def stedc(d: torch.Tensor, e: torch.Tensor):
    """Symmetric tridiagonal eigenproblem by divide and conquer.  d (batch, n), e (batch, n) [last entry unused];
    both destroyed.  Returns (E (batch, n), Q (batch, n, n) column-major items, info)."""
    batch, n = d.shape
    need = ctypes.c_size_t(0)
    _check(lib().nao_stedc_workspace(n, batch, ctypes.byref(need)), "nao_stedc_workspace")
    work = _workspace(need.value, d.device)
    E = torch.empty_like(d)
    Q = torch.empty((batch, n, n), dtype=torch.float64, device=d.device)
    info = torch.zeros(batch, dtype=torch.int32, device=d.device)
    rc = lib().nao_stedc(n, batch, _dev(d, "d"), _dev(e, "e"), _dev(E, "E"), _dev(Q, "Q"), n, n * n,
                         _dev(work, "work"), work.numel(), _dev(info, "info"), _stream(d))
    _check(rc, "nao_stedc")
    return E, Q, info
