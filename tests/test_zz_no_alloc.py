"""nao_fermi_mu_static: the Fermi-level entry point for callers that cannot allocate device memory.

Some users of this library run inside a host program that owns every byte of HBM itself (an SCF code with its own pool, a
plug-in that is handed only its input and output arrays) or call from a place where cudaMalloc's device-wide
synchronisation is not acceptable.  They have no workspace to pass, so nao_fermi_mu_static keeps its intermediates in a
fixed 1.5 MiB array built into the library (limit: 65536 states).  This file checks that it returns what the ordinary
nao_fermi_mu returns -- twice in a row, because all calls share that array and the second one starts from what the first
left in it -- and that sizes beyond the limit are refused.

The file name sorts after every other test file on purpose: pytest -x stops at the first failure, and a failure here must
not hide the parity tests.  The GPU test passes on its own in a fresh process (the first call then does the per-device
address look-up) and after the other tests.
"""
import ctypes

import numpy as np
import pytest

TOL_MU, TOL_F = 1e-10, 1e-9          # the bars of tests/test_gpu_parity.py (Fermi level, occupations)
DEV = "cuda:0"


def test_static_limit_is_checked_on_the_host():
    """More than NAO_FERMI_STATIC_MAX_STATES states: refused with status 5 before any CUDA call (runs without a GPU)."""
    from paper_2606_09058_b200 import binding
    lib = binding.lib()
    w = (ctypes.c_double * 2)(1.0, 1.0)
    mu = ctypes.c_double(0.0)
    n = binding.FERMI_STATIC_MAX_STATES // 2 + 1
    assert lib.nao_fermi_mu_static(n, 2, 1, w, 10.0, 1e-3, ctypes.byref(mu), 1, None) == 5
    assert b"65536" in lib.nao_status_string(5)
    assert lib.nao_fermi_mu_static(0, 2, 1, w, 10.0, 1e-3, ctypes.byref(mu), 1, None) == -1
    assert lib.nao_fermi_mu_static(8, 2, None, w, 10.0, 1e-3, ctypes.byref(mu), 1, None) == -3
    assert lib.nao_fermi_mu_static(8, 2, 1, w, 99.0, 1e-3, ctypes.byref(mu), 1, None) == 3     # NAO_ERR_ELECTRONS


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_path_twice():
    """Two calls in a row on different problems, the second SMALLER than the first so that the shared array still holds
    the first call's sorted states beyond the part the second call rewrites; each against nao_fermi_mu on the same
    input.  Outputs are caller-owned (`out=`), as they are for a caller that cannot allocate."""
    import torch
    import paper_2606_09058_b200 as nao
    nao.lib()
    rng = np.random.default_rng(11)
    cases = [
        # (batch, n, weights, electrons per unit weight and level, kT): a config-1-like batch, then a small gapped one
        (16, 832, [2.0 / 16] * 16, 0.31, 9.5e-4),
        (3, 50, [0.5, 0.25, 0.25], 0.27, 1.0e-2),
    ]
    for batch, n, w, filling, kT in cases:
        e = np.sort(rng.standard_normal((batch, n)), axis=1)
        ne = filling * sum(w) * n
        E = torch.from_numpy(e).to(DEV)
        mu_ref, F_ref = nao.fermi_mu(E, w, ne, kT)
        out = torch.full_like(E, -7.0)
        mu, F = nao.fermi_mu_static(E, w, ne, kT, out=out)
        torch.cuda.synchronize()
        assert F.data_ptr() == out.data_ptr()
        assert abs(mu - mu_ref) <= TOL_MU, (mu, mu_ref)
        assert float((F - F_ref).abs().max()) <= TOL_F
        assert abs(float((F.sum(dim=1) * torch.tensor(w, device=DEV, dtype=torch.float64)).sum()) - ne) <= 1e-9 * ne
    # the largest accepted size runs (64 items of 1024 levels = 65536 states), one state more is refused
    E = torch.from_numpy(np.sort(rng.standard_normal((64, 1024)), axis=1)).to(DEV)
    w = [1.0 / 64] * 64
    mu_ref, F_ref = nao.fermi_mu(E, w, 300.0, 2e-3)
    mu, F = nao.fermi_mu_static(E, w, 300.0, 2e-3)
    assert abs(mu - mu_ref) <= TOL_MU and float((F - F_ref).abs().max()) <= TOL_F
    with pytest.raises(nao.NaoError):
        nao.fermi_mu_static(torch.zeros((1, nao.FERMI_STATIC_MAX_STATES + 1), dtype=torch.float64, device=DEV), [2.0], 10.0, 1e-3)
