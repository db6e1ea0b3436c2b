"""ctypes front-end of nao_synth.c: builds the five BASELINE.json configurations.

Storage convention used everywhere in this repo: a matrix is a numpy array of
shape (n, n) whose memory is COLUMN-MAJOR, i.e. ``arr[j, i] == M(i, j)``; use
``as_matrix(arr)`` (= ``arr.T``) to get the mathematical matrix.  Batches are
``(batch, n, n)`` arrays of such items.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

KT_DEFAULT = 9.5e-4  # Ha, 300 K smearing (BASELINE.json configs)

# (atoms, box side / bohr, periodic, kind, electrons)
CONFIGS = {
    0: dict(nat=8, L=5.4, periodic=False, kind="col_gamma_1spin", n_electrons=32.0),
    1: dict(nat=64, L=10.8, periodic=True, kind="col_k222_2spin", n_electrons=256.0),
    2: dict(nat=512, L=21.7, periodic=True, kind="col_gamma_2spin", n_electrons=2048.0),
    3: dict(nat=384, L=19.7, periodic=True, kind="nc_gamma", n_electrons=1536.0),
    4: dict(nat=1024, L=27.4, periodic=True, kind="nc_gamma", n_electrons=4096.0),
}


def build_synth_lib(force: bool = False) -> str:
    """Compile nao_synth.c with gcc (OpenMP) into libnao_synth.so next to it."""
    src = os.path.join(_HERE, "nao_synth.c")
    out = os.path.join(_HERE, "libnao_synth.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", out, src, "-lm"])
    return out


def _lib():
    global _LIB
    if _LIB is None:
        lib = ctypes.CDLL(build_synth_lib())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.nao_synth_hs.argtypes = [ctypes.c_uint64, ctypes.c_int, ctypes.c_double, ctypes.c_int, dp,
                                     ctypes.c_int, ctypes.c_double, dp, dp]
        lib.nao_synth_hs.restype = None
        lib.nao_synth_nc.argtypes = [ctypes.c_uint64, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                     ctypes.c_double, ctypes.c_double, dp, dp]
        lib.nao_synth_nc.restype = None
        lib.nao_synth_positions.argtypes = [ctypes.c_uint64, ctypes.c_int, ctypes.c_double, dp]
        lib.nao_synth_positions.restype = None
        _LIB = lib
    return _LIB


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def as_matrix(arr: np.ndarray) -> np.ndarray:
    """Column-major storage array (…, n, n) -> mathematical matrix view (…, n, n)."""
    return np.swapaxes(arr, -1, -2)


@dataclass
class Problem:
    """One SCF step's worth of inputs: a batch of (H, S) pencils sharing one Fermi level."""
    name: str
    n: int                      # order of H (2N for noncollinear)
    batch: int
    is_complex: bool
    nc_block_s: bool            # S is the N*N real overlap, H is 2N*2N complex (NAO_NC_BLOCK_S)
    H: np.ndarray               # (batch, n, n) column-major items, float64 or complex128
    S: np.ndarray               # (batch, n, n) like H, or (1, N, N) float64 when nc_block_s
    weights: np.ndarray         # (batch,) g * w_k per item
    n_electrons: float
    kT: float
    meta: dict = field(default_factory=dict)

    def S_full(self, b: int = 0) -> np.ndarray:
        """Mathematical S matrix of item b at the order of H (expands diag(S,S) for NC)."""
        if not self.nc_block_s:
            return as_matrix(self.S[b])
        s = as_matrix(self.S[0])
        N = s.shape[0]
        out = np.zeros((2 * N, 2 * N), dtype=np.complex128)
        out[:N, :N] = s
        out[N:, N:] = s
        return out

    def H_full(self, b: int = 0) -> np.ndarray:
        return as_matrix(self.H[b])


def _hs(seed, nat, L, periodic, kfrac, is_complex, d_shift):
    n = 13 * nat
    dt = np.complex128 if is_complex else np.float64
    H = np.empty((n, n), dtype=dt)
    S = np.empty((n, n), dtype=dt)
    k = np.ascontiguousarray(kfrac, dtype=np.float64)
    _lib().nao_synth_hs(seed, nat, float(L), int(periodic), _dp(k), int(is_complex), float(d_shift),
                        _dp(H.view(np.float64)), _dp(S.view(np.float64)))
    return H, S


def make_config(idx: int, nat: int | None = None, seed: int = 0, kT: float = KT_DEFAULT) -> Problem:
    """Build BASELINE.json config `idx`.  `nat` overrides the atom count to make a reduced-size
    replica from the same recipe (box side scaled to keep the atom density, 4 electrons/atom)."""
    cfg = dict(CONFIGS[idx])
    if nat is not None and nat != cfg["nat"]:
        cfg["L"] = cfg["L"] * (nat / cfg["nat"]) ** (1.0 / 3.0)
        if cfg["periodic"]:
            cfg["L"] = max(cfg["L"], 10.5)     # strictly above the 10 bohr cut-off: no orbital sees its own image
        cfg["n_electrons"] = 4.0 * nat
        cfg["nat"] = nat
    nat, L, periodic, kind = cfg["nat"], cfg["L"], cfg["periodic"], cfg["kind"]
    if periodic and L <= 10.0:
        raise ValueError("periodic replica too small: box side must exceed the 10 bohr cut-off")
    n = 13 * nat
    name = f"c{idx}" + ("" if nat == CONFIGS[idx]["nat"] else f"_nat{nat}")
    meta = dict(cfg, seed=seed, idx=idx)
    if kind == "col_gamma_1spin":
        H, S = _hs(seed, nat, L, periodic, (0, 0, 0), False, 0.0)
        return Problem(name, n, 1, False, False, H[None], S[None], np.array([2.0]), cfg["n_electrons"], kT, meta)
    if kind == "col_gamma_2spin":
        Hu, S = _hs(seed, nat, L, periodic, (0, 0, 0), False, -0.02)
        Hd, _ = _hs(seed, nat, L, periodic, (0, 0, 0), False, +0.02)
        return Problem(name, n, 2, False, False, np.stack([Hu, Hd]), np.stack([S, S]),
                       np.array([1.0, 1.0]), cfg["n_electrons"], kT, meta)
    if kind == "col_k222_2spin":
        ks = [(sx * 0.25, sy * 0.25, sz * 0.25) for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
        Hs, Ss = [], []
        for shift in (0.0, 0.02):
            for k in ks:
                H, S = _hs(seed, nat, L, periodic, k, True, shift)
                Hs.append(H)
                Ss.append(S)
        meta["kfrac"] = ks
        return Problem(name, n, 16, True, False, np.stack(Hs), np.stack(Ss),
                       np.full(16, 1.0 / 8.0), cfg["n_electrons"], kT, meta)
    if kind == "nc_gamma":
        H = np.empty((2 * n, 2 * n), dtype=np.complex128)
        S = np.empty((n, n), dtype=np.float64)
        _lib().nao_synth_nc(seed, nat, float(L), int(periodic), 0.05, 0.01, _dp(H.view(np.float64)), _dp(S))
        return Problem(name, 2 * n, 1, True, True, H[None], S[None], np.array([1.0]),
                       cfg["n_electrons"], kT, meta)
    raise ValueError(kind)
