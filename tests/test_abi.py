"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/nao.h declares; argument validation happens on the host before any launch."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_09058_b200 import build as nao_build
    return nao_build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "nao.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nao_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(libpath):
    lib = ctypes.CDLL(libpath)
    names = _declared_symbols()
    assert len(names) >= 14
    for name in names:
        assert hasattr(lib, name), "libnao.so does not export %s" % name


def test_binding_covers_header():
    from paper_2606_09058_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()


def test_library_is_sm100a_with_fp64_tensor_instructions(libpath):
    """The GEMM core must contain DMMA (FP64 tensor) SASS for sm_100a."""
    import subprocess
    out = subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True).stdout
    assert "arch = sm_100a" in out
    assert "DMMA" in out and "gemm_kernel" in out


def test_host_side_argument_validation(libpath):
    """Bad arguments are rejected on the host with -(argument index): no CUDA call is made (works without a GPU)."""
    lib = ctypes.CDLL(libpath)
    sz = ctypes.c_size_t(0)
    assert lib.nao_geneig_workspace(0, 1, 0, 0, ctypes.byref(sz)) == -1
    assert lib.nao_geneig_workspace(8, 0, 0, 0, ctypes.byref(sz)) == -2
    assert lib.nao_geneig_workspace(8, 1, 7, 0, ctypes.byref(sz)) == -3
    assert lib.nao_geneig_workspace(7, 1, 1, 2, ctypes.byref(sz)) == -4      # NC needs even n
    assert lib.nao_geneig_workspace(104, 1, 0, 0, ctypes.byref(sz)) == 0 and sz.value > 104 * 104 * 8 * 2
    assert lib.nao_fermi_workspace(104, 1, ctypes.byref(sz)) == 0 and sz.value >= 2 * 104 * 8
    assert lib.nao_density_workspace(104, 3, 1, ctypes.byref(sz)) == 0 and sz.value > 0
    lib.nao_status_string.restype = ctypes.c_char_p
    assert lib.nao_status_string(0) == b"ok"
    assert b"workspace" in lib.nao_status_string(1)
    lib.nao_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.nao_version()
    # nao_fermi_mu: electron count outside (0, sum w n) is an error before anything is launched
    lib.nao_fermi_mu.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double),
                                 ctypes.c_double, ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.c_void_p,
                                 ctypes.c_void_p, ctypes.c_void_p]
    w = (ctypes.c_double * 1)(2.0)
    mu = ctypes.c_double(0)
    assert lib.nao_fermi_mu(4, 1, 1, w, 9.0, 1e-3, ctypes.byref(mu), 1, 1, None) == 3      # NAO_ERR_ELECTRONS
    assert lib.nao_fermi_mu(4, 1, 1, w, 2.0, 0.0, ctypes.byref(mu), 1, 1, None) == 3
    assert lib.nao_fermi_mu(4, 1, None, w, 2.0, 1e-3, ctypes.byref(mu), 1, 1, None) == -3
    # partial spectrum / fused step: the extra arguments are validated on the host as well
    vp, l, i = ctypes.c_void_p, ctypes.c_long, ctypes.c_int
    lib.nao_geneig_partial.argtypes = [i, i, i, ctypes.c_uint, i, vp, l, l, vp, l, l, vp, vp, l, l, vp, ctypes.c_size_t, vp, vp]
    assert lib.nao_geneig_partial(8, 1, 0, 0, 0, 1, 8, 64, 1, 8, 64, 1, 1, 8, 64, 1, 1 << 20, 1, None) == -5     # n_vec < 1
    assert lib.nao_geneig_partial(8, 1, 0, 0, 9, 1, 8, 64, 1, 8, 64, 1, 1, 8, 64, 1, 1 << 20, 1, None) == -5     # n_vec > n
    assert lib.nao_geneig_partial(8, 1, 0, 0, 4, None, 8, 64, 1, 8, 64, 1, 1, 8, 64, 1, 1 << 20, 1, None) == -6  # dH
    assert lib.nao_scf_step_workspace(104, 2, 0, 0, ctypes.byref(sz)) == 0 and sz.value > 2 * 104 * 104 * 8 * 2
    lib.nao_occupied_count.argtypes = [i, i, vp, ctypes.c_double, ctypes.POINTER(i), vp]
    cnt = i(0)
    assert lib.nao_occupied_count(0, 1, 1, 1e-17, ctypes.byref(cnt), None) == -1
    assert lib.nao_occupied_count(4, 1, None, 1e-17, ctypes.byref(cnt), None) == -3
    # the step after the path: energy weights and the k-fold
    dp = ctypes.POINTER(ctypes.c_double)
    lib.nao_energy_weights.argtypes = [i, i, vp, vp, vp, vp]
    assert lib.nao_energy_weights(0, 1, 1, 1, 1, None) == -1
    assert lib.nao_energy_weights(4, 1, 1, None, 1, None) == -4
    assert lib.nao_fold_workspace(8, 27, ctypes.byref(sz)) == 0 and sz.value >= 27 * 16 * 16
    assert lib.nao_fold_workspace(0, 27, ctypes.byref(sz)) == -1
    lib.nao_fold_density.argtypes = [i, i, i, i, vp, l, l, dp, dp, dp, vp, l, l, vp, ctypes.c_size_t, vp]
    k3 = (ctypes.c_double * 3)(0, 0, 0)
    assert lib.nao_fold_density(4, 1, 1, 5, 1, 4, 16, k3, k3, k3, 1, 4, 16, 1, 1 << 20, None) == -4      # out_dtype
    assert lib.nao_fold_density(4, 1, 1, 0, 1, 3, 16, k3, k3, k3, 1, 4, 16, 1, 1 << 20, None) == -6      # ldd < n
    assert lib.nao_fold_density(4, 1, 1, 0, 1, 4, 16, k3, None, k3, 1, 4, 16, 1, 1 << 20, None) == -9    # h_w
    assert lib.nao_fold_density(4, 1, 1, 0, 1, 4, 16, k3, k3, k3, 1, 4, 16, 1, 8, None) == 1             # workspace
    # host-buffer form of the step
    assert lib.nao_solve_host_workspace(104, 2, 0, 0, 1, ctypes.byref(sz)) == 0 and sz.value > 5 * 2 * 104 * 104 * 8
    lib.nao_solve_host.argtypes = [i, i, i, ctypes.c_uint, vp, vp, i, dp, ctypes.c_double, ctypes.c_double, vp, dp, vp, vp, vp,
                                   ctypes.c_size_t, vp]
    w1 = (ctypes.c_double * 1)(2.0)
    assert lib.nao_solve_host(8, 1, 0, 0, None, 1, 0, w1, 4.0, 1e-3, 1, ctypes.byref(mu), 1, 1, 1, 1 << 30, None) == -5
    assert lib.nao_solve_host(8, 1, 0, 1, 1, 1, 0, w1, 4.0, 1e-3, 1, ctypes.byref(mu), 1, 1, 1, 1 << 30, None) == -4      # S_FACTORED
    assert lib.nao_solve_host(8, 1, 0, 0, 1, 1, 0, w1, 4.0, 1e-3, 1, ctypes.byref(mu), 1, 1, 1, 64, None) == 1           # workspace
    # ... and its occupation arguments are checked before the eigensolve is paid for (same rules as nao_fermi_mu)
    assert lib.nao_solve_host(8, 1, 0, 0, 1, 1, 0, w1, 17.0, 1e-3, 1, ctypes.byref(mu), 1, 1, 1, 1 << 30, None) == 3     # N_e > sum w n
    assert lib.nao_solve_host(8, 1, 0, 0, 1, 1, 0, w1, 4.0, 0.0, 1, ctypes.byref(mu), 1, 1, 1, 1 << 30, None) == 3       # kT <= 0
    wneg = (ctypes.c_double * 1)(-1.0)
    assert lib.nao_solve_host(8, 1, 0, 0, 1, 1, 0, wneg, 4.0, 1e-3, 1, ctypes.byref(mu), 1, 1, 1, 1 << 30, None) == -8   # h_weight
    assert lib.nao_solve_host(8, 1, 0, 0, 1, 1, 0, None, 4.0, 1e-3, 1, ctypes.byref(mu), 1, 1, 1, 1 << 30, None) == -8
    # fused step: the same checks first, and the negative codes of the shared eigensolver count THIS signature's arguments
    lib.nao_scf_step.argtypes = [i, i, i, ctypes.c_uint, vp, l, l, vp, l, l, dp, ctypes.c_double, ctypes.c_double, vp, dp, vp,
                                 vp, l, l, vp, l, l, ctypes.POINTER(i), vp, ctypes.c_size_t, vp, vp]
    nv = i(0)

    def scf(n=8, batch=1, dH=1, ldh=8, dS=1, w=w1, ne=4.0, kT=1e-3, dE=1, dF=1, dC=1, ldc=8, dD=1, ldd=8, work=1, wb=1 << 30, info=1):
        return lib.nao_scf_step(n, batch, 0, 0, dH, ldh, 64, dS, 8, 64, w, ne, kT, dE, ctypes.byref(mu), dF, dC, ldc, 64, dD, ldd, 64,
                                ctypes.byref(nv), work, wb, info, None)
    assert scf(ne=17.0) == 3 and scf(ne=0.0) == 3 and scf(kT=-1.0) == 3
    assert scf(w=wneg) == -11 and scf(w=None) == -11
    assert scf(n=0) == -1 and scf(batch=0) == -2
    assert scf(dH=None) == -5 and scf(ldh=7) == -6 and scf(dS=None) == -8
    assert scf(dE=None) == -14 and scf(dF=None) == -16 and scf(dC=None) == -17 and scf(ldc=7) == -18
    assert scf(dD=None) == -20 and scf(ldd=7) == -21
    assert scf(work=None) == -24 and scf(info=None) == -26
    assert scf(wb=64) == 1
    # stream groups: the workspace query accounts for one slice per group; a batch smaller than the group count is one group
    plain, grouped = ctypes.c_size_t(0), ctypes.c_size_t(0)
    assert lib.nao_geneig_workspace(832, 16, 1, 0, ctypes.byref(plain)) == 0
    assert lib.nao_geneig_workspace(832, 16, 1, 64, ctypes.byref(grouped)) == 0 and grouped.value >= plain.value
    assert lib.nao_geneig_workspace(832, 1, 1, 96, ctypes.byref(grouped)) == 0
    assert lib.nao_geneig_workspace(832, 1, 1, 0, ctypes.byref(plain)) == 0 and grouped.value == plain.value
    lib.nao_set_lowdin_threshold.argtypes = [ctypes.c_double]
    assert lib.nao_set_lowdin_threshold(-1e-3) == -1 and lib.nao_set_lowdin_threshold(1.0) == -1
    assert lib.nao_set_lowdin_threshold(1e-8) == 0 and lib.nao_set_lowdin_threshold(0.0) == 0
    assert lib.nao_geneig_workspace(104, 1, 0, 16, ctypes.byref(sz)) == 0 and sz.value > 104 * 104 * 8 * 2      # NAO_LOWDIN


def test_no_product_import_of_oracle():
    """The product package must never import or call oracle/ (or a CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_09058_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "nao_oracle" not in text and "oracle_impl" not in text, f
