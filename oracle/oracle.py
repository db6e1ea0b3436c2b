"""ctypes front-end of the C oracle (nao_oracle.c).  TEST INFRASTRUCTURE ONLY.

All functions take and return *mathematical* matrices: numpy arrays with ``M[i, j]`` = element (i, j).
(The C code is column-major; the wrapper transposes on the way in and out.)
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build_oracle_lib(force: bool = False) -> str:
    src = [os.path.join(_HERE, "nao_oracle.c"), os.path.join(_HERE, "oracle_impl.h")]
    out = os.path.join(_HERE, "libnao_oracle.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < max(os.path.getmtime(s) for s in src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", out, src[0], "-lm"])
    return out


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build_oracle_lib())
    return _LIB


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _colmajor(M, dtype):
    """mathematical matrix -> freshly allocated column-major buffer (as a C-contiguous array of M^T)."""
    return np.array(np.asarray(M, dtype=dtype).T, order="C", copy=True)


def _is_complex(*arrs):
    return any(np.iscomplexobj(a) for a in arrs)


def geneig(H, S, lowdin: bool = False):
    """H C = S C diag(e) (Eq. 5/11/21).  Returns (e ascending, C with C^H S C = I, info dict)."""
    n = H.shape[0]
    cplx = _is_complex(H, S)
    dt = np.complex128 if cplx else np.float64
    h, s = _colmajor(H, dt), _colmajor(S, dt)
    e = np.empty(n, dtype=np.float64)
    c = np.empty((n, n), dtype=dt)
    sweeps = ctypes.c_int(0)
    lib = _lib()
    if lowdin:
        fn = lib.oracle_geneig_lowdin_z if cplx else lib.oracle_geneig_lowdin_d
        info = fn(ctypes.c_int(n), _p(h), _p(s), _p(e), _p(c))
    else:
        fn = lib.oracle_geneig_z if cplx else lib.oracle_geneig_d
        info = fn(ctypes.c_int(n), _p(h), _p(s), _p(e), _p(c), ctypes.byref(sweeps))
    if info != 0:
        raise np.linalg.LinAlgError(f"S not positive definite: leading minor {info}")
    return e, c.T.copy(), {"sweeps": sweeps.value}


def geneig_lowdin(H, S):
    """Same problem by the paper's Loewdin route."""
    return geneig(H, S, lowdin=True)


def geneig_lowdin_pruned(H, S, rel: float):
    """Loewdin route with pruning of near-dependent directions (PAPER.md:147, 159-163 for the route):
    S = U s U^H by Jacobi; keep the directions with s_i > rel * s_max; V = U_keep s_keep^{-1/2}; H' = V^H H V (long double
    products); H' C' = C' e by Jacobi; C = V C'.  Returns (e ascending, m values; C of shape (n, m), C^H S C = I_m)."""
    H = np.asarray(H)
    S = np.asarray(S)
    s, U = heev(S)
    keep = (s > 0) & (s > rel * s.max())
    ld = np.clongdouble if _is_complex(H, S) else np.longdouble
    V = U[:, keep].astype(ld) / np.sqrt(s[keep].astype(np.longdouble))
    Hp = V.conj().T @ (H.astype(ld) @ V)
    Hp = (Hp + Hp.conj().T) / 2
    e, Cp = heev(Hp.astype(np.complex128 if _is_complex(H, S) else np.float64))
    C = V @ Cp.astype(ld)
    return e, C.astype(np.complex128 if _is_complex(H, S) else np.float64)


def cholesky(S):
    """Lower Cholesky factor L of S (S = L L^H)."""
    n = S.shape[0]
    cplx = _is_complex(S)
    dt = np.complex128 if cplx else np.float64
    s = _colmajor(S, dt)
    fn = _lib().oracle_cholesky_z if cplx else _lib().oracle_cholesky_d
    info = fn(ctypes.c_int(n), _p(s))
    if info != 0:
        raise np.linalg.LinAlgError(f"S not positive definite: leading minor {info}")
    return s.T.copy()


def heev(A):
    """Hermitian eigen-decomposition by cyclic Jacobi: returns (e ascending, Z)."""
    n = A.shape[0]
    cplx = _is_complex(A)
    dt = np.complex128 if cplx else np.float64
    a = _colmajor(A, dt)
    e = np.empty(n)
    z = np.empty((n, n), dtype=dt)
    fn = _lib().oracle_heev_z if cplx else _lib().oracle_heev_d
    fn(ctypes.c_int(n), _p(a), _p(e), _p(z))
    return e, z.T.copy()


def fermi(e, weights, n_electrons: float, kT: float):
    """e: (batch, n) eigenvalues; weights: (batch,) g*w_k per item.  Returns (mu, f (batch, n))."""
    e = np.ascontiguousarray(np.atleast_2d(e), dtype=np.float64)
    w = np.repeat(np.asarray(weights, dtype=np.float64), e.shape[1]).copy()
    f = np.empty_like(e)
    mu = ctypes.c_double(0.0)
    info = _lib().oracle_fermi(ctypes.c_int(e.size), _p(e), _p(w), ctypes.c_double(n_electrons),
                               ctypes.c_double(kT), ctypes.byref(mu), _p(f))
    if info != 0:
        raise ValueError("n_electrons outside (0, sum of weights) or kT <= 0")
    return mu.value, f


def density(C, f):
    """D = C diag(f) C^H (north_star; Eq. 8/23)."""
    n = C.shape[0]
    cplx = _is_complex(C)
    dt = np.complex128 if cplx else np.float64
    c = _colmajor(C, dt)
    ff = np.ascontiguousarray(f, dtype=np.float64)
    d = np.empty((n, n), dtype=dt)
    fn = _lib().oracle_density_z if cplx else _lib().oracle_density_d
    fn(ctypes.c_int(n), _p(c), _p(ff), _p(d))
    return d.T.copy()


def energy_density(C, f, e):
    """Energy-weighted density matrix C diag(f e) C^H: the definition of `density` with the weights
    f_i e_i (one FP64 product per state)."""
    return density(C, np.asarray(f, dtype=np.float64) * np.asarray(e, dtype=np.float64))


def fold_density(Dk, kpts, weights, Rvecs):
    """Real-space density matrix D(R) = sum_k w_k exp(-i k.R) D(k): the inverse of the Bloch sum of Eq. 12 (PAPER.md:79-82,
    M(k) = sum_R exp(+i k.R) M(R), reading C8).  Dk: (nk, n, n) mathematical matrices; returns (nR, n, n)
    complex.  Long double throughout (phase, product and sum), written out term by term."""
    Dk = np.asarray(Dk)
    nk, n, _ = Dk.shape
    kp = np.asarray(kpts, dtype=np.longdouble).reshape(nk, 3)
    w = np.asarray(weights, dtype=np.longdouble).reshape(nk)
    Rv = np.asarray(Rvecs, dtype=np.longdouble).reshape(-1, 3)
    dre = Dk.real.astype(np.longdouble)
    dim = Dk.imag.astype(np.longdouble)
    out = np.empty((Rv.shape[0], n, n), dtype=np.complex128)
    for r in range(Rv.shape[0]):
        are = np.zeros((n, n), dtype=np.longdouble)
        aim = np.zeros((n, n), dtype=np.longdouble)
        for k in range(nk):
            phi = -(kp[k, 0] * Rv[r, 0] + kp[k, 1] * Rv[r, 1] + kp[k, 2] * Rv[r, 2])
            c, sn = w[k] * np.cos(phi), w[k] * np.sin(phi)
            are += c * dre[k] - sn * dim[k]
            aim += c * dim[k] + sn * dre[k]
        out[r] = are.astype(np.float64) + 1j * aim.astype(np.float64)
    return out


def solve_problem(prob, want_D: bool = True):
    """Whole hot path on a synth.Problem: eigenpairs per item, shared Fermi level, D per item."""
    es, Cs = [], []
    for b in range(prob.batch):
        e, C, _ = geneig(prob.H_full(b), prob.S_full(b))
        es.append(e)
        Cs.append(C)
    e = np.stack(es)
    mu, f = fermi(e, prob.weights, prob.n_electrons, prob.kT)
    out = {"e": e, "mu": mu, "f": f, "C": Cs}
    if want_D:
        out["D"] = [density(Cs[b], f[b]) for b in range(prob.batch)]
    return out
