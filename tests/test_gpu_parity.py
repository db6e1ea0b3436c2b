"""GPU parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's north_star bars:
    |de| <= 1e-9 Ha, max|dD| <= 1e-8, ||C^H S C - I||_max <= 1e-10, |dmu| <= 1e-10 Ha.
D is compared instead of C (gauge / degeneracy safe)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_09058_b200.synth import make_config

pytestmark = pytest.mark.gpu

TOL_E, TOL_D, TOL_ORTH, TOL_MU = 1e-9, 1e-8, 1e-10, 1e-10
DEV = "cuda:0"


@pytest.fixture(scope="module")
def nao():
    import paper_2606_09058_b200 as m
    m.lib()       # raises if the CUDA library is missing: there is no fallback
    return m


def to_dev(M):
    """mathematical (b, n, n) -> column-major items on the GPU"""
    return torch.from_numpy(np.ascontiguousarray(np.swapaxes(M, -1, -2))).to(DEV)


def to_np(T):
    return np.swapaxes(T.cpu().numpy(), -1, -2)


def run_path(nao, prob, flags=0):
    H = torch.from_numpy(prob.H).to(DEV)
    S = torch.from_numpy(prob.S.copy()).to(DEV)
    if prob.nc_block_s:
        flags |= nao.NAO_NC_BLOCK_S
    E, C, info = nao.geneig(H, S, flags=flags)
    assert int(info.abs().max()) == 0
    mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
    D = nao.density_matrix(C, F)
    return dict(e=E.cpu().numpy(), mu=mu, f=F.cpu().numpy(), C=to_np(C), D=to_np(D), S_factor=S)


def check_against_oracle(prob, got, ref):
    assert np.abs(got["e"] - ref["e"]).max() <= TOL_E
    assert abs(got["mu"] - ref["mu"]) <= TOL_MU
    assert np.abs(got["f"] - ref["f"]).max() <= 1e-7          # |df| <= |de|/(4 kT) ~ 2.6e-7 at the bar
    ne = 0.0
    for b in range(prob.batch):
        assert np.abs(got["D"][b] - ref["D"][b]).max() <= TOL_D
        Sb = prob.S_full(b)
        Cb = got["C"][b]
        assert np.abs(Cb.conj().T @ Sb @ Cb - np.eye(prob.n)).max() <= TOL_ORTH
        assert np.abs(prob.H_full(b) @ Cb - Sb @ Cb * got["e"][b]).max() <= 1e-10
        ne += prob.weights[b] * np.trace(got["D"][b] @ Sb).real
    assert abs(ne - prob.n_electrons) <= 1e-8


# ------------------------------------------------------------------------------------------ whole path vs oracle
def test_config0_full(nao):
    """BASELINE config 0: n = 104 real, one spin channel (g = 2), 32 electrons."""
    prob = make_config(0)
    check_against_oracle(prob, run_path(nao, prob), oracle.solve_problem(prob))


def test_config1_replica_complex_batch16(nao):
    """Config 1 recipe at 16 atoms: n = 208 complex, 8 k-points x 2 spins = 16 items sharing one Fermi level."""
    prob = make_config(1, nat=16)
    got = run_path(nao, prob)
    check_against_oracle(prob, got, oracle.solve_problem(prob))
    # time reversal: e(k) = e(-k) for a real real-space H (items 0..7 are k, 7-j is -k)
    assert np.abs(got["e"][:8] - got["e"][7::-1]).max() <= 1e-10


def test_config2_replica_two_spins(nao):
    """Config 2 recipe at 32 atoms: n = 416 real, 2 spin channels (several GEMM tiles and a ragged tail)."""
    prob = make_config(2, nat=32)
    check_against_oracle(prob, run_path(nao, prob), oracle.solve_problem(prob))


def test_config3_replica_noncollinear_block_S(nao):
    """Config 3 recipe at 16 atoms: 2N = 416 complex, S real N x N with NAO_NC_BLOCK_S (Eq. 25-27)."""
    prob = make_config(3, nat=16)
    ref = oracle.solve_problem(prob)
    check_against_oracle(prob, run_path(nao, prob), ref)
    # the same problem with S_NC = diag(S, S) passed as a dense complex 2N x 2N overlap must agree
    H = torch.from_numpy(prob.H).to(DEV)
    S = to_dev(prob.S_full(0)[None])
    E, C, info = nao.geneig(H, S)
    assert np.abs(E.cpu().numpy() - ref["e"]).max() <= TOL_E


def test_cached_factor_is_bit_identical(nao):
    """S and its factor do not change over the SCF loop: NAO_S_FACTORED must reproduce the result."""
    prob = make_config(2, nat=16)
    H = torch.from_numpy(prob.H).to(DEV)
    S = torch.from_numpy(prob.S.copy()).to(DEV)
    E1, C1, _ = nao.geneig(H, S)
    E2, C2, _ = nao.geneig(H, S, flags=nao.NAO_S_FACTORED)
    assert torch.equal(E1, E2) and torch.equal(C1, C2)
    L = np.tril(to_np(S)[0])
    assert np.abs(L @ L.T - prob.S_full(0)).max() <= 1e-13
    assert np.abs(L - oracle.cholesky(prob.S_full(0))).max() <= 1e-12


# ------------------------------------------------------------------------------------------ degenerate / edge cases
def test_ring_exact_degeneracies_density_matches(nao):
    """Complex Hermitian ring, theta = 0: +-m pairs are exactly degenerate; D is gauge independent."""
    n, t = 48, -1.0
    H = np.zeros((n, n), dtype=complex)
    for j in range(n):
        H[j, (j + 1) % n] += t
        H[(j + 1) % n, j] += t
    e_ref, C_ref, _ = oracle.geneig(H, np.eye(n, dtype=complex))
    mu_ref, f_ref = oracle.fermi(e_ref[None], [2.0], 20.0, 0.05)
    D_ref = oracle.density(C_ref, f_ref[0])
    E, C, info = nao.geneig(to_dev(H[None]), to_dev(np.eye(n, dtype=complex)[None]))
    mu, F = nao.fermi_mu(E, [2.0], 20.0, 0.05)
    D = nao.density_matrix(C, F)
    assert np.abs(E.cpu().numpy()[0] - e_ref).max() <= TOL_E
    assert abs(mu - mu_ref) <= TOL_MU
    assert np.abs(to_np(D)[0] - D_ref).max() <= TOL_D


@pytest.mark.parametrize("n", [1, 2, 3, 33, 65, 131])
@pytest.mark.parametrize("cplx", [False, True])
def test_small_and_ragged_sizes(nao, n, cplx):
    rng = np.random.default_rng(n + 1000 * cplx)
    A = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0)
    H = (A + A.conj().T) / 2
    B = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0)
    S = B @ B.conj().T / n + np.eye(n)
    e_ref, C_ref, _ = oracle.geneig(H, S)
    E, C, info = nao.geneig(to_dev(H[None]), to_dev(S[None]))
    assert int(info[0]) == 0
    assert np.abs(E.cpu().numpy()[0] - e_ref).max() <= TOL_E
    f = np.linspace(1.0, 0.0, n)
    D = nao.density_matrix(C, torch.from_numpy(f[None].copy()).to(DEV))
    if n == 1 or np.min(np.diff(e_ref)) > 1e-4:          # D with arbitrary f is unique only for distinct levels
        assert np.abs(to_np(D)[0] - oracle.density(C_ref, f)).max() <= TOL_D


def test_identity_overlap_and_block_diagonal(nao):
    """S = I => C unitary; block-diagonal H => spectrum is the union of the block spectra (heavy deflation in D&C)."""
    rng = np.random.default_rng(7)
    n1, n2 = 40, 57
    A1 = rng.standard_normal((n1, n1)); A2 = rng.standard_normal((n2, n2))
    H = np.zeros((n1 + n2, n1 + n2)); H[:n1, :n1] = (A1 + A1.T) / 2; H[n1:, n1:] = (A2 + A2.T) / 2
    n = n1 + n2
    E, C, info = nao.geneig(to_dev(H[None]), to_dev(np.eye(n)[None]))
    e1, _, _ = oracle.geneig(H[:n1, :n1], np.eye(n1)); e2, _, _ = oracle.geneig(H[n1:, n1:], np.eye(n2))
    assert np.abs(E.cpu().numpy()[0] - np.sort(np.concatenate([e1, e2]))).max() <= TOL_E
    Cm = to_np(C)[0]
    assert np.abs(Cm.T @ Cm - np.eye(n)).max() <= TOL_ORTH


def test_not_positive_definite_reports_pivot(nao):
    prob = make_config(0)
    S = prob.S_full(0).copy()
    S[60, 60] = -1.0
    with pytest.raises(np.linalg.LinAlgError):
        oracle.cholesky(S)
    E, C, info = nao.geneig(torch.from_numpy(prob.H).to(DEV), to_dev(S[None]))
    assert int(info[0]) == 61          # leading minor 61 (1-based) is the first that fails, as in the oracle


def test_density_all_occupied_is_inverse_overlap(nao):
    """f = 1 for every state: D = C C^H = S^{-1}, independent of the eigen-solver."""
    prob = make_config(0)
    E, C, _ = nao.geneig(torch.from_numpy(prob.H).to(DEV), torch.from_numpy(prob.S.copy()).to(DEV))
    D = nao.density_matrix(C, torch.ones_like(E))
    assert np.abs(to_np(D)[0] @ prob.S_full(0) - np.eye(prob.n)).max() <= 1e-11


# ------------------------------------------------------------------------------------------ Fermi level
def test_fermi_level_against_oracle_and_closed_forms(nao):
    rng = np.random.default_rng(3)
    e = np.sort(rng.standard_normal((3, 50)), axis=1)
    w = [0.5, 0.25, 0.25]
    mu_ref, f_ref = oracle.fermi(e, w, 13.7, 0.01)
    mu, F = nao.fermi_mu(torch.from_numpy(e).to(DEV), w, 13.7, 0.01)
    assert abs(mu - mu_ref) <= TOL_MU and np.abs(F.cpu().numpy() - f_ref).max() <= 1e-9
    # single n-fold level: mu = e0 + kT ln(nu/(1-nu))
    e0, kT, n, ne = -0.3, 2e-3, 40, 12.0
    mu, F = nao.fermi_mu(torch.full((1, n), e0, dtype=torch.float64, device=DEV), [2.0], ne, kT)
    nu = ne / (2.0 * n)
    assert abs(mu - (e0 + kT * np.log(nu / (1 - nu)))) <= TOL_MU
    # two levels of equal degeneracy, huge gap, integer filling: mu = midpoint (needs the particle/hole log form)
    e2 = np.concatenate([np.full(8, -1.0), np.full(8, 1.0)])[None]
    mu, F = nao.fermi_mu(torch.from_numpy(e2).to(DEV), [2.0], 16.0, 9.5e-4)
    assert abs(mu) <= TOL_MU
    mu_ref, _ = oracle.fermi(e2, [2.0], 16.0, 9.5e-4)
    assert abs(mu - mu_ref) <= TOL_MU


# ------------------------------------------------------------------------------------------ two-stage reduction
def test_two_stage_config2_replica_against_oracle(nao):
    """Config 2 recipe at 32 atoms (n = 416 real, 2 spins) through dense->band->tridiagonal (NAO_TRD_TWO_STAGE):
    6 panels, bulge chasing over 7 band blocks with a ragged last block, 13 diamonds of chase reflectors."""
    prob = make_config(2, nat=32)
    check_against_oracle(prob, run_path(nao, prob, flags=nao.NAO_TRD_TWO_STAGE), oracle.solve_problem(prob))


def test_two_stage_config3_replica_against_oracle(nao):
    """Config 3 recipe at 16 atoms (2N = 416 complex, block S) through the two-stage reduction."""
    prob = make_config(3, nat=16)
    check_against_oracle(prob, run_path(nao, prob, flags=nao.NAO_TRD_TWO_STAGE), oracle.solve_problem(prob))


@pytest.mark.parametrize("n", [66, 67, 129, 193, 200])
@pytest.mark.parametrize("cplx", [False, True])
def test_two_stage_heev_ragged_sizes(nao, n, cplx):
    """nao_heev with the two-stage path at sizes around the band width (64): one short panel, partial band blocks,
    partial diamonds.  Eigenvalues against the Jacobi oracle; vectors through residual and orthogonality."""
    rng = np.random.default_rng(100 + n)
    A = rng.standard_normal((2, n, n))
    if cplx:
        A = A + 1j * rng.standard_normal((2, n, n))
    A = A + np.swapaxes(A.conj(), -1, -2)
    E, Z, info = nao.heev(to_dev(A), flags=nao.NAO_TRD_TWO_STAGE)
    assert int(info.abs().max()) == 0
    E = E.cpu().numpy(); Zn = to_np(Z)
    for b in range(2):
        e_or, _ = oracle.heev(A[b])
        assert np.abs(E[b] - e_or).max() <= TOL_E
        assert np.abs(A[b] @ Zn[b] - Zn[b] * E[b]).max() <= 1e-11
        assert np.abs(Zn[b].conj().T @ Zn[b] - np.eye(n)).max() <= 1e-12


def test_two_stage_structured_inputs(nao):
    """Inputs whose panels are rank deficient or already banded: tight-binding chain (tridiagonal), block-diagonal,
    identity, and a matrix that is already a band of width 64.  Closed form for the chain (north_star)."""
    n = 300
    k = np.arange(1, n + 1)
    chain = np.diag(np.full(n - 1, -1.0), 1) + np.diag(np.full(n - 1, -1.0), -1)
    rng = np.random.default_rng(3)
    blk = np.zeros((n, n)); 
    for a, bnd in ((0, 100), (100, 170), (170, 300)):
        M = rng.standard_normal((bnd - a, bnd - a)); blk[a:bnd, a:bnd] = M + M.T
    band = np.triu(np.tril(rng.standard_normal((n, n)), 64), -64); band = band + band.T
    mats = np.stack([chain, blk, np.eye(n), band])
    E, Z, info = nao.heev(to_dev(mats), flags=nao.NAO_TRD_TWO_STAGE)
    assert int(info.abs().max()) == 0
    E = E.cpu().numpy(); Zn = to_np(Z)
    assert np.abs(E[0] - np.sort(-2.0 * np.cos(k * np.pi / (n + 1)))).max() <= 1e-12
    for b in range(4):
        assert np.abs(E[b] - np.linalg.eigvalsh(mats[b])).max() <= 1e-11
        assert np.abs(mats[b] @ Zn[b] - Zn[b] * E[b]).max() <= 1e-11
        assert np.abs(Zn[b].T @ Zn[b] - np.eye(n)).max() <= 1e-12


# ------------------------------------------------------------------------------------------ building blocks
@pytest.mark.parametrize("cplx", [False, True])
def test_gemm_core_all_ops(nao, cplx):
    rng = np.random.default_rng(11)

    def rnd(r, c):
        x = rng.standard_normal((2, r, c))
        return x + 1j * rng.standard_normal((2, r, c)) if cplx else x

    def op(X, o):
        return X if o == 0 else (np.swapaxes(X, -1, -2) if o == 1 else np.swapaxes(X.conj(), -1, -2))

    for (m, n, k) in [(1, 1, 1), (130, 67, 45), (257, 300, 129), (384, 256, 160), (391, 262, 83)]:
        for oa in (0, 1, 2):
            for ob in (0, 1, 2):
                A = rnd(m, k) if oa == 0 else rnd(k, m)
                B = rnd(k, n) if ob == 0 else rnd(n, k)
                C0 = rnd(m, n)
                Ct = to_dev(C0)
                nao.gemm(to_dev(A), to_dev(B), oa, ob, alpha=0.7, beta=-0.3, C=Ct)
                ref = 0.7 * (op(A, oa) @ op(B, ob)) - 0.3 * C0
                assert np.abs(to_np(Ct) - ref).max() <= 1e-12 * k


def test_stedc_textbook_tridiagonals(nao):
    """(1,2,1) Toeplitz: 2 - 2 cos(k pi/(n+1)); Wilkinson W+: near-degenerate pairs; glued: heavy deflation."""
    n = 201
    d = np.stack([np.full(n, 2.0), np.abs(np.arange(n) - 100.0), np.abs(np.arange(n) % 21 - 10.0)])
    e = np.stack([np.ones(n), np.ones(n), np.where((np.arange(n) + 1) % 21 == 0, 1e-8, 1.0)])
    E, Q, info = nao.stedc(torch.from_numpy(d.copy()).to(DEV), torch.from_numpy(e.copy()).to(DEV))
    E = E.cpu().numpy(); Qn = to_np(Q)
    k = np.arange(1, n + 1)
    assert np.abs(E[0] - np.sort(2 - 2 * np.cos(k * np.pi / (n + 1)))).max() <= 1e-13
    for i in range(3):
        T = np.diag(d[i]) + np.diag(e[i, :n - 1], 1) + np.diag(e[i, :n - 1], -1)
        assert np.abs(T @ Qn[i] - Qn[i] * E[i]).max() <= 1e-12 * np.abs(T).sum(1).max()
        assert np.abs(Qn[i].T @ Qn[i] - np.eye(n)).max() <= 1e-13
        e_or, _ = oracle.heev(T)
        assert np.abs(E[i] - e_or).max() <= 1e-11 * max(1.0, np.abs(e_or).max())


# ------------------------------------------------------------------------------------------ full-size properties
def test_config2_full_size_properties(nao):
    """BASELINE config 2 at full size (n = 6656 real, 2 spins), the launch configuration bench.py times.  The oracle
    cannot run here in seconds, so: invariants that hold at any size, plus sampled entries of D recomputed one by
    one from their definition with the oracle's D-kernel restricted to those entries."""
    prob = make_config(2)
    got = run_path(nao, prob)
    n = prob.n
    ne = 0.0
    for b in range(prob.batch):
        Cb, Sb, Hb = got["C"][b], prob.S_full(b), prob.H_full(b)
        assert np.all(np.diff(got["e"][b]) >= 0)
        SC = Sb @ Cb
        Fm = Cb.T @ SC - np.eye(n)
        R = Hb @ Cb - SC * got["e"][b]
        assert np.abs(Fm).max() <= TOL_ORTH
        assert np.abs(R).max() <= 1e-10
        # a-posteriori bound on every eigenvalue, as in the config-3 certificate: Frobenius norms bound the
        # 2-norms of F and R; ||C||_2^2 <= (1 + ||F||) / lambda_min(S), lambda_min(S) from LAPACK
        fF, fR = np.linalg.norm(Fm), np.linalg.norm(R)
        cN = np.sqrt((1.0 + fF) / np.linalg.eigvalsh(Sb)[0])
        bound = (fR * cN + np.abs(got["e"][b]).max() * fF) / (1.0 - fF)
        assert bound <= TOL_E, bound
        ne += prob.weights[b] * np.sum(got["D"][b] * Sb)
        _check_density_all_entries(to_dev(Cb), torch.from_numpy(got["f"][b]).to(DEV), to_dev(got["D"][b]))   # every entry
        rng = np.random.default_rng(5 + b)
        for (i, j) in rng.integers(0, n, size=(64, 2)):
            dij = float(np.sum(np.asarray(got["f"][b], dtype=np.longdouble) * Cb[i].astype(np.longdouble) * Cb[j].astype(np.longdouble)))
            assert abs(got["D"][b][i, j] - dij) <= 1e-12
        assert abs(np.sum(got["e"][b]) - np.trace(np.linalg.solve(Sb, Hb))) <= 1e-8
    assert abs(ne - prob.n_electrons) <= 1e-7
    mu_ref, f_ref = oracle.fermi(got["e"], prob.weights, prob.n_electrons, prob.kT)
    assert abs(got["mu"] - mu_ref) <= TOL_MU


def test_config3_full_size_certificate(nao):
    """BASELINE config 3 at full size (2N = 9984 complex, S real 4992, NAO_NC_BLOCK_S), the other headline workload.
    The Jacobi oracle would need ~40 core-hours here, so the a-posteriori certificate of SURVEY.md 8c is used: with
    F = C^H S C - I and R = H C - S C diag(e), congruence bounds the error of every eigenvalue by
    (||R||_2 ||C||_2 + max|e| ||F||_2) / (1 - ||F||_2); the products are formed on the GPU by torch (cuBLAS, a checker
    that shares nothing with the product path).  D is re-formed from (C, f) and compared in EVERY entry (SURVEY.md:414),
    sampled entries are recomputed in long double from the definition, plus Tr(D S) = N_e."""
    prob = make_config(3)
    n = prob.n
    H = torch.from_numpy(prob.H).to(DEV)
    S = torch.from_numpy(prob.S.copy()).to(DEV)
    E, C, info = nao.geneig(H, S, flags=nao.NAO_NC_BLOCK_S)
    assert int(info.abs().max()) == 0
    mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
    D = nao.density_matrix(C, F)
    e = E[0]
    assert bool((e[1:] >= e[:-1]).all())
    Cm = C[0].T                                           # column-major item -> mathematical matrix
    Hm = torch.from_numpy(prob.H_full(0)).to(DEV)
    Sm = torch.from_numpy(prob.S_full(0)).to(DEV).to(Hm.dtype)
    SC = Sm @ Cm
    Fm = Cm.mH @ SC
    Fm.diagonal().sub_(1.0)
    orth = float(Fm.abs().max())
    R = Hm @ Cm - SC * e[None, :]
    resid = float(R.abs().max())
    assert orth <= TOL_ORTH
    assert resid <= 1e-10
    # Frobenius norms bound the 2-norms
    fF = float(torch.linalg.norm(Fm)); fR = float(torch.linalg.norm(R)); cN = float(torch.linalg.norm(Cm, ord=2))
    bound = (fR * cN + float(e.abs().max()) * fF) / (1.0 - fF)
    assert bound <= TOL_E, bound
    del R, Fm, SC, Hm
    _check_density_all_entries(C[0], F[0], D[0])                  # all 1.0e8 entries, FP64 product by torch
    Dm = D[0].T
    ne = float((Dm * Sm.T).sum().real) * prob.weights[0]          # Tr(D S)
    assert abs(ne - prob.n_electrons) <= 1e-7
    assert float((Dm - Dm.mH).abs().max()) <= 1e-14
    f = F[0].cpu().numpy().astype(np.longdouble)
    Ch = Cm.cpu().numpy()
    Dh = Dm.cpu().numpy()
    rng = np.random.default_rng(9)
    for (i, j) in rng.integers(0, n, size=(48, 2)):
        dij = np.sum(f * Ch[i].astype(np.clongdouble) * np.conj(Ch[j]).astype(np.clongdouble))
        assert abs(Dh[i, j] - complex(dij)) <= 1e-12
    mu_ref, _ = oracle.fermi(E.cpu().numpy(), prob.weights, prob.n_electrons, prob.kT)
    assert abs(mu - mu_ref) <= TOL_MU


def _nc_certificate(prob, E, C, ncols=None):
    """A-posteriori certificate for a noncollinear problem (S_NC = diag(S, S), S real) from the solver's own
    (e, C), formed on the GPU by torch (cuBLAS: a checker that shares nothing with the product path):
        F = C^H S C - I,   R = H C - S C diag(e).
    Congruence: every e_i lies within (||R||_2 ||C||_2 + max|e| ||F||_2) / (1 - ||F||_2) of an eigenvalue of the pencil
    (with all n columns: of the i-th one).  Frobenius norms bound the 2-norms of F and R; ||C||_2^2 <= (1 + ||F||) / lambda_min(S)
    with lambda_min(S) > 1/2 PROVEN by a successful Cholesky factorisation of S - I/2.
    Returns (max|F|, max|R|, bound)."""
    n = prob.n
    N = n // 2
    e = E[0] if ncols is None else E[0][:ncols]
    Cm = C[0].T if ncols is None else C[0].T[:, :ncols]       # column-major item -> mathematical matrix
    Sr = torch.from_numpy(np.ascontiguousarray(prob.S[0].T)).to(DEV)
    _, chol_info = torch.linalg.cholesky_ex(Sr - 0.5 * torch.eye(N, dtype=Sr.dtype, device=DEV))
    assert int(chol_info) == 0                           # lambda_min(S) > 1/2
    Sc = Sr.to(Cm.dtype)
    SC = torch.cat([Sc @ Cm[:N], Sc @ Cm[N:]], dim=0)
    del Sc
    Fm = Cm.mH @ SC
    Fm.diagonal().sub_(1.0)
    orth = float(Fm.abs().max()); fF = float(torch.linalg.norm(Fm))
    del Fm
    Hm = torch.from_numpy(prob.H[0]).to(DEV).T          # mathematical H as a view of the column-major item
    R = Hm @ Cm
    R -= SC * e[None, :]
    resid = float(R.abs().max()); fR = float(torch.linalg.norm(R))
    del R, SC, Hm
    cN = ((1.0 + fF) / 0.5) ** 0.5
    bound = (fR * cN + float(e.abs().max()) * fF) / (1.0 - fF)
    return orth, resid, bound


def _check_density_all_entries(C_item, f_item, D_item, tol=TOL_D, block=2048):
    """EVERY entry of D against its definition D = sum_i f_i c_i c_i^H (Eq. 8 / 23; SURVEY.md:414),
    re-formed on the GPU by torch in FP64 (cuBLAS: a checker that shares nothing with the product path), column block by
    column block so that config 4 fits.  C_item / D_item are column-major items (row k of C_item = eigenvector k), f_item the
    occupations.  States with f < 1e-20 are left out of the reference (they change an entry by < 1e-20 |c|^2).
    Returns max |D - Dref|."""
    n = C_item.shape[0]
    nocc = int((f_item >= 1e-20).nonzero().max()) + 1
    Cs = C_item[:nocc]                                   # nocc x n, row k = eigenvector k
    fC = Cs * f_item[:nocc, None].to(Cs.dtype)
    worst = 0.0
    for j0 in range(0, n, block):
        j1 = min(n, j0 + block)
        ref = Cs[:, j0:j1].mH @ fC                       # stored rows j0..j1 of D: D_item[j, i] = D(i, j)
        worst = max(worst, float((D_item[j0:j1] - ref).abs().max()))
        del ref
    assert worst <= tol, worst
    return worst


def _check_density_from_definition(prob, C, F, D, mu, E, samples, seed):
    """D against its definition: every entry against the FP64 product re-formed by torch (1e-8), sampled entries in long
    double (1e-12: the tie to the definition itself), Hermiticity, Tr(D S) = N_e, mu against the oracle's Fermi solver on the
    solver's eigenvalues.  Noncollinear layout (S real N x N)."""
    n = prob.n
    N = n // 2
    _check_density_all_entries(C[0], F[0], D[0])
    Dm = D[0].T
    Sr = torch.from_numpy(np.ascontiguousarray(prob.S[0])).to(DEV)           # S^T as stored = S (symmetric)
    ne = float((Dm[:N, :N] * Sr).sum().real + (Dm[N:, N:] * Sr).sum().real) * prob.weights[0]      # Tr(D S_NC)
    assert abs(ne - prob.n_electrons) <= 1e-7, ne
    assert float((Dm - Dm.mH).abs().max()) <= 1e-14
    f = F[0].cpu().numpy().astype(np.longdouble)
    rng = np.random.default_rng(seed)
    idx = rng.integers(0, n, size=(samples, 2))
    rows = sorted(set(int(i) for i in idx.ravel()))
    Crows = {r: C[0][:, r].cpu().numpy() for r in rows}                       # row r of the mathematical C
    for (i, j) in idx:
        dij = np.sum(f * Crows[int(i)].astype(np.clongdouble) * np.conj(Crows[int(j)]).astype(np.clongdouble))
        assert abs(complex(Dm[int(i), int(j)]) - complex(dij)) <= 1e-12
    mu_ref, _ = oracle.fermi(E.cpu().numpy(), prob.weights, prob.n_electrons, prob.kT)
    assert abs(mu - mu_ref) <= TOL_MU


def test_config3_two_stage_and_fused_step_certificates(nao):
    """BASELINE config 3 at full size through the OTHER paths the library can take there: nao_geneig with
    NAO_TRD_TWO_STAGE (complex dense -> band -> tridiagonal, all eigenvectors) and nao_scf_step with DEFAULT flags (which
    picks the complex two-stage reduction by itself from order 1536 on and back-transforms only the occupied vectors).
    Both get the a-posteriori certificate; the fused step's eigenvalues, mu and D are also compared with the full solve."""
    prob = make_config(3)
    n = prob.n
    H = torch.from_numpy(prob.H).to(DEV)
    S = torch.from_numpy(prob.S.copy()).to(DEV)
    E, C, info = nao.geneig(H, S, flags=nao.NAO_NC_BLOCK_S | nao.NAO_TRD_TWO_STAGE)
    assert int(info.abs().max()) == 0
    assert bool((E[0][1:] >= E[0][:-1]).all())
    orth, resid, bound = _nc_certificate(prob, E, C)
    assert orth <= TOL_ORTH and resid <= 1e-10 and bound <= TOL_E, (orth, resid, bound)
    mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
    D = nao.density_matrix(C, F)
    _check_density_from_definition(prob, C, F, D, mu, E, 48, 11)
    del C
    # fused step, default flags, fresh S
    r = nao.scf_step(H, torch.from_numpy(prob.S.copy()).to(DEV), prob.weights, prob.n_electrons, prob.kT, flags=nao.NAO_NC_BLOCK_S)
    assert int(r["info"].abs().max()) == 0
    nv = r["n_vec"]
    assert nao.occupied_count(r["F"]) <= nv < n // 2
    assert float((r["E"] - E).abs().max()) <= 1e-11           # all n eigenvalues, same reduction
    assert abs(r["mu"] - mu) <= 1e-12
    orth, resid, bound = _nc_certificate(prob, r["E"], r["C"], ncols=nv)
    assert orth <= TOL_ORTH and resid <= 1e-10 and bound <= TOL_E, (orth, resid, bound)
    assert float(r["C"][0][nv:].abs().max()) == 0.0           # columns that were not back-transformed
    assert float((r["D"] - D).abs().max()) <= 1e-11
    _check_density_from_definition(prob, r["C"], r["F"], r["D"], r["mu"], r["E"], 24, 12)


def test_config4_full_recipe_certificate(nao):
    """BASELINE config 4, the whole recipe at full size (2N = 26 624 complex, 11.3 GB per matrix; S real 13 312 with
    NAO_NC_BLOCK_S): nao_geneig + nao_fermi_mu + nao_density_matrix exactly as bench.py --workload c4 launches them.  The
    Jacobi oracle would need ~800 core-hours, so the a-posteriori certificate of SURVEY.md 8c stands in for it:
    ||C^H S C - I||, residual, the congruence bound on every eigenvalue <= 1e-9, Tr(D S) = 4096, sampled D entries from the
    definition in long double, mu from the oracle's Fermi solver.  Buffers are released stage by stage (75 GB workspace)."""
    prob = make_config(4)
    n = prob.n
    assert n == 26624 and prob.n_electrons == 4096.0
    H = torch.from_numpy(prob.H).to(DEV)
    S = torch.from_numpy(prob.S.copy()).to(DEV)
    work = torch.empty(nao.geneig_workspace(n, 1, nao.NAO_COMPLEX, nao.NAO_NC_BLOCK_S) + 256, dtype=torch.uint8, device=DEV)
    E, C, info = nao.geneig(H, S, flags=nao.NAO_NC_BLOCK_S, work=work)
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    del work, H
    torch.cuda.empty_cache()
    assert bool((E[0][1:] >= E[0][:-1]).all())
    mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
    D = nao.density_matrix(C, F)
    _check_density_from_definition(prob, C, F, D, mu, E, 32, 14)
    del D
    torch.cuda.empty_cache()
    orth, resid, bound = _nc_certificate(prob, E, C)
    assert orth <= TOL_ORTH and resid <= 1e-10 and bound <= TOL_E, (orth, resid, bound)


def test_config4_size_heev_properties(nao):
    """Order of BASELINE config 4 (2N = 26 624 complex, 11.3 GB per matrix): 64-bit offsets, the 148-CTA cooperative
    panel kernel with 180-row chunks, 52 blocks of 512 reflectors.  Seeded Hermitian matrix generated on the device (the
    config-4 recipe needs > 30 GB of host memory for H alone); invariants that hold at any size, products by torch."""
    n = 26624
    g = torch.Generator(device=DEV); g.manual_seed(4)
    A = torch.complex(torch.randn(n, n, dtype=torch.float64, device=DEV, generator=g),
                      torch.randn(n, n, dtype=torch.float64, device=DEV, generator=g))
    A = (A + A.mH).unsqueeze(0)                       # Hermitian; column-major item of A^T = conj(A): same spectrum
    tr = float(A[0].diagonal().real.sum())
    fro2 = float((A[0].abs() ** 2).sum())
    E, Z, info = nao.heev(A.clone())
    assert int(info.abs().max()) == 0
    e = E[0]
    assert bool((e[1:] >= e[:-1]).all())
    assert abs(float(e.sum()) - tr) <= 1e-9 * n                      # trace
    assert abs(float((e ** 2).sum()) - fro2) <= 1e-12 * fro2         # ||A||_F^2 = sum e^2
    Zm = Z[0].T
    Am = A[0].T
    R = Am @ Zm - Zm * e[None, :]
    scale = float(e.abs().max())
    assert float(R.abs().max()) <= 1e-12 * scale * 10
    del R
    G = Zm.mH @ Zm
    G.diagonal().sub_(1.0)
    assert float(G.abs().max()) <= 1e-12


@pytest.mark.parametrize("two_stage", [False, True])
def test_partial_spectrum_gives_the_same_density(nao, two_stage):
    """nao_geneig_partial: only the vectors with f >= 1e-17 (+ margin) are
    back-transformed; e (all levels), mu and D must match the oracle like the full solve, the unwanted columns are 0."""
    for idx, nat in ((2, 32), (3, 16)):
        prob = make_config(idx, nat=nat)
        ref = oracle.solve_problem(prob)
        flags = (nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0) | (nao.NAO_TRD_TWO_STAGE if two_stage else 0)
        H = torch.from_numpy(prob.H).to(DEV)
        S = torch.from_numpy(prob.S.copy()).to(DEV)
        E, C, info = nao.geneig(H, S, flags=flags)                      # first SCF step: everything
        mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
        n_vec = nao.occupied_count(F)
        assert 0 < n_vec < prob.n // 2
        n_vec += 5
        E2, C2, info2 = nao.geneig(H, S, flags=flags | nao.NAO_S_FACTORED, n_vec=n_vec)   # later step: partial
        assert int(info2.abs().max()) == 0
        mu2, F2 = nao.fermi_mu(E2, prob.weights, prob.n_electrons, prob.kT)
        assert nao.occupied_count(F2) <= n_vec
        D2 = nao.density_matrix(C2, F2)
        assert np.abs(E2.cpu().numpy() - ref["e"]).max() <= TOL_E
        assert abs(mu2 - ref["mu"]) <= TOL_MU
        for b in range(prob.batch):
            assert np.abs(to_np(D2)[b] - ref["D"][b]).max() <= TOL_D
        assert float(C2[:, n_vec:, :].abs().max()) == 0.0              # column-major items: columns are dim 1
        Cb = to_np(C2)[0][:, :n_vec]
        assert np.abs(Cb.conj().T @ prob.S_full(0) @ Cb - np.eye(n_vec)).max() <= TOL_ORTH


@pytest.mark.parametrize("n,batch", [(64, 3), (832, 3), (2048, 2), (2112, 1), (2176, 3)])
@pytest.mark.parametrize("cplx", [False, True])
def test_one_stage_multiples_of_64_take_the_tma_fed_hemv(nao, n, batch, cplx):
    """Orders >= 2048 that are multiples of 64 run the one-stage tridiagonalisation through the TMA-fed HEMV (cp.async.bulk
    stage rings, stream of stages continuous across the columns of a panel); every other order takes the register-fed one.  The
    same matrices embedded with one more row and column (order n + 1, decoupled last level) go through the other kernel:
    both must agree with LAPACK (numpy, CPU) and with each other, and satisfy the invariants.  Several items per launch."""
    rng = np.random.default_rng(64 + n)
    A = rng.standard_normal((batch, n, n))
    if cplx:
        A = A + 1j * rng.standard_normal((batch, n, n))
    A = A + np.swapaxes(A.conj(), -1, -2)
    E, Z, info = nao.heev(to_dev(A), flags=nao.NAO_TRD_ONE_STAGE)
    assert int(info.abs().max()) == 0
    B = np.zeros((batch, n + 1, n + 1), dtype=A.dtype)
    B[:, :n, :n] = A
    B[:, n, n] = 1e3                                  # decoupled level far above the spectrum
    E2, Z2, info2 = nao.heev(to_dev(B), flags=nao.NAO_TRD_ONE_STAGE)
    assert int(info2.abs().max()) == 0
    for b in range(batch):
        e = E.cpu().numpy()[b]; Zn = to_np(Z)[b]
        ref = np.linalg.eigvalsh(A[b])
        scale = max(1.0, np.abs(ref).max())
        assert np.abs(e - ref).max() <= 1e-12 * scale * n ** 0.5
        assert np.abs(A[b] @ Zn - Zn * e).max() <= 1e-12 * scale * n ** 0.5
        assert np.abs(Zn.conj().T @ Zn - np.eye(n)).max() <= 1e-12
        assert np.abs(E2.cpu().numpy()[b][:n] - e).max() <= 1e-12 * scale * n ** 0.5


@pytest.mark.parametrize("flag", ["NAO_TRD_ONE_STAGE", "NAO_TRD_TWO_STAGE"])
@pytest.mark.parametrize("cplx", [False, True])
def test_odd_order_1001_both_paths(nao, flag, cplx):
    """Odd order and odd leading dimensions (no operand is 16-byte aligned after the first column): the 8-byte GEMM loaders,
    ragged last panels / band blocks / diamonds.  Invariants plus a LAPACK cross-check of the eigenvalues (numpy, CPU)."""
    n = 1001
    rng = np.random.default_rng(1001)
    A = rng.standard_normal((1, n, n))
    if cplx:
        A = A + 1j * rng.standard_normal((1, n, n))
    A = A + np.swapaxes(A.conj(), -1, -2)
    E, Z, info = nao.heev(to_dev(A), flags=getattr(nao, flag))
    assert int(info.abs().max()) == 0
    e = E.cpu().numpy()[0]; Zn = to_np(Z)[0]
    assert np.abs(e - np.linalg.eigvalsh(A[0])).max() <= 1e-10
    assert np.abs(A[0] @ Zn - Zn * e).max() <= 1e-10
    assert np.abs(Zn.conj().T @ Zn - np.eye(n)).max() <= 1e-12


def test_shared_overlap_across_spin_channels(nao):
    """strideS = 0: the two spin channels of config 2 share S; factoring it once must give the per-item result."""
    prob = make_config(2, nat=16)
    assert np.array_equal(prob.S[0], prob.S[1])
    H = torch.from_numpy(prob.H).to(DEV)
    E1, C1, i1 = nao.geneig(H, torch.from_numpy(prob.S.copy()).to(DEV))
    S1 = torch.from_numpy(prob.S[:1].copy()).to(DEV)
    E2, C2, i2 = nao.geneig(H, S1)
    assert int(i2.abs().max()) == 0
    assert torch.equal(E1, E2) and torch.equal(C1, C2)
    E3, C3, _ = nao.geneig(H, S1, flags=nao.NAO_S_FACTORED)
    assert torch.equal(E1, E3) and torch.equal(C1, C3)


@pytest.mark.parametrize("two_stage", [False, True])
def test_scf_step_fused_against_oracle(nao, two_stage):
    """nao_scf_step: eigenvalues -> Fermi level -> occupied eigenvectors -> D in one call, against the oracle on the
    config-1 (16 complex items, one shared mu), config-2 and config-3 (block S) recipes."""
    for idx, nat in ((1, 16), (2, 32), (3, 16)):
        prob = make_config(idx, nat=nat)
        ref = oracle.solve_problem(prob)
        flags = (nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0) | (nao.NAO_TRD_TWO_STAGE if two_stage else 0)
        H = torch.from_numpy(prob.H).to(DEV)
        S = torch.from_numpy(prob.S.copy()).to(DEV)
        r = nao.scf_step(H, S, prob.weights, prob.n_electrons, prob.kT, flags=flags)
        assert int(r["info"].abs().max()) == 0
        assert 0 < r["n_vec"] <= prob.n
        assert np.abs(r["E"].cpu().numpy() - ref["e"]).max() <= TOL_E
        assert abs(r["mu"] - ref["mu"]) <= TOL_MU
        assert np.abs(r["F"].cpu().numpy() - ref["f"]).max() <= 1e-7
        for b in range(prob.batch):
            assert np.abs(to_np(r["D"])[b] - ref["D"][b]).max() <= TOL_D
        Cb = to_np(r["C"])[0][:, :r["n_vec"]]
        assert np.abs(Cb.conj().T @ prob.S_full(0) @ Cb - np.eye(r["n_vec"])).max() <= TOL_ORTH


def test_dmma_peak_measurement_matches_the_derived_roof(nao):
    """nao_dmma_peak (register-resident DMMA loop) must land on the roof DESIGN.md derives from unit counts and clocks
    (148 SMs x 128 flop/clk x SM clock): between 80 % and 102 % of it (clocks may sit below the maximum)."""
    derived = 148 * 128 * 1.965e9 / 1e12
    t = nao.dmma_peak()
    assert 0.8 * derived <= t <= 1.02 * derived, t


# ---------------------------------------------------------------- the step after the path
def test_energy_weighted_density_matrix_against_oracle(nao):
    """W = C diag(f e) C^H through nao_energy_weights + nao_density_matrix (negative weights: occupied levels lie below
    zero) against the oracle's W from its own eigenpairs; Tr(W S) = sum f e."""
    for idx, nat in [(0, None), (1, 6), (3, 4)]:
        prob = make_config(idx, nat=nat)
        ref = oracle.solve_problem(prob, want_D=False)
        H = torch.from_numpy(prob.H).to(DEV)
        S = torch.from_numpy(prob.S.copy()).to(DEV)
        E, C, info = nao.geneig(H, S, flags=nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0)
        mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
        FE = nao.energy_weights(E, F)
        assert np.array_equal(FE.cpu().numpy(), F.cpu().numpy() * E.cpu().numpy())
        W = to_np(nao.density_matrix(C, FE))
        for b in range(prob.batch):
            Wref = oracle.energy_density(ref["C"][b], ref["f"][b], ref["e"][b])
            assert np.abs(W[b] - Wref).max() <= TOL_D
            assert abs(np.trace(W[b] @ prob.S_full(b)).real - float((ref["f"][b] * ref["e"][b]).sum())) <= 1e-8


def _c1_mesh(prob):
    L = prob.meta["L"]
    ks = [(sx * 0.25, sy * 0.25, sz * 0.25) for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
    Rv = [(L * a, L * b, L * c) for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)]
    return 2 * np.pi * np.array(ks) / L, np.full(8, 0.125), np.array(Rv)


@pytest.mark.parametrize("nat", [6, 16])
def test_fold_density_config1_recipe_against_oracle(nao, nat):
    """D(R) on the 27 images of the config-1 recipe (8 Monkhorst-Pack points, first spin channel) from the GPU's D(k),
    real and complex output, against the oracle's fold of the oracle's own D(k)."""
    prob = make_config(1, nat=nat)
    ref = oracle.solve_problem(prob)
    got = run_path(nao, prob)
    kp, w, Rv = _c1_mesh(prob)
    Dk = to_dev(np.stack(got["D"][:8]))
    ref_DR = oracle.fold_density(np.stack(ref["D"][:8]), kp, w, Rv)
    DRc = to_np(nao.fold_density(Dk, kp, w, Rv, real_out=False))
    DRr = to_np(nao.fold_density(Dk, kp, w, Rv, real_out=True))
    assert np.abs(DRc - ref_DR).max() <= TOL_D
    assert np.abs(DRr - ref_DR.real).max() <= TOL_D
    assert np.abs(ref_DR.imag).max() <= 1e-12          # time reversal: D(-k) = conj D(k) on this mesh
    # the fold itself, on identical inputs: the oracle's fold of the GPU's D(k), to rounding
    same = oracle.fold_density(np.stack(got["D"][:8]), kp, w, Rv)
    assert np.abs(DRc - same).max() <= 1e-13


def test_fold_density_ragged_sizes_and_many_k_points(nao):
    """Sizes that are not multiples of the 128 x 8 tile, more k-points than one register pass holds (16), more lattice
    vectors than one shared-memory pass holds (128)."""
    rng = np.random.default_rng(3)
    for (n, nk, nR) in [(1, 1, 1), (131, 19, 5), (37, 33, 140), (200, 8, 27)]:
        Dk = rng.standard_normal((nk, n, n)) + 1j * rng.standard_normal((nk, n, n))
        kp = rng.uniform(-0.6, 0.6, (nk, 3))
        w = rng.uniform(0.1, 1.0, nk)
        Rv = rng.uniform(-25, 25, (nR, 3))
        ref = oracle.fold_density(Dk, kp, w, Rv)
        scale = np.abs(ref).max()
        gc = to_np(nao.fold_density(to_dev(Dk), kp, w, Rv, real_out=False))
        gr = to_np(nao.fold_density(to_dev(Dk), kp, w, Rv, real_out=True))
        assert np.abs(gc - ref).max() <= 1e-13 * max(1.0, scale) * nk
        assert np.abs(gr - ref.real).max() <= 1e-13 * max(1.0, scale) * nk


# ---------------------------------------------------------------- the paper's own orthogonalisation
@pytest.mark.parametrize("idx,nat", [(0, None), (1, 6), (2, 8), (3, 4)])
def test_lowdin_route_against_oracle(nao, idx, nat):
    """NAO_LOWDIN (S = U s U^H, V = U s^{-1/2}) gives the same e, mu, D as the oracle; the dense
    V^H left in dS serves the later SCF steps (NAO_S_FACTORED | NAO_LOWDIN)."""
    prob = make_config(idx, nat=nat)
    ref = oracle.solve_problem(prob)
    got = run_path(nao, prob, flags=nao.NAO_LOWDIN)
    check_against_oracle(prob, got, ref)
    H = torch.from_numpy(prob.H).to(DEV)
    fl = nao.NAO_LOWDIN | nao.NAO_S_FACTORED | (nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0)
    E2, C2, info2 = nao.geneig(H, got["S_factor"], flags=fl)
    assert int(info2.abs().max()) == 0
    assert np.abs(E2.cpu().numpy() - ref["e"]).max() <= TOL_E
    mu2, F2 = nao.fermi_mu(E2, prob.weights, prob.n_electrons, prob.kT)
    D2 = to_np(nao.density_matrix(C2, F2))
    for b in range(prob.batch):
        assert np.abs(D2[b] - ref["D"][b]).max() <= TOL_D


@pytest.mark.parametrize("kind", ["real", "complex", "nc"])
def test_lowdin_pruning_of_duplicated_orbitals(nao, kind):
    """A basis in which two orbitals appear twice (S' = P^T S P singular, two exact null directions): with a pruning threshold
    the GPU path returns the levels of the pruned basis, NAO_PRUNED_LEVEL for the two pruned directions with zero vectors,
    and the oracle's D of the pruned problem."""
    prob = make_config({"real": 0, "complex": 1, "nc": 3}[kind], nat={"real": None, "complex": 6, "nc": 4}[kind])
    nS = prob.S.shape[-1]
    dup = [3, nS - 2]
    P = np.hstack([np.eye(nS), np.eye(nS)[:, dup]])
    S0 = np.swapaxes(prob.S[0], -1, -2)
    Sd = P.T @ S0 @ P
    H0 = prob.H_full(0)
    if kind == "nc":
        P2 = np.kron(np.eye(2), P)
        Hd, Sfull = P2.T @ H0 @ P2, np.kron(np.eye(2), Sd)
    else:
        Hd, Sfull = P.T @ H0 @ P, Sd
    m, n = H0.shape[0], Hd.shape[0]
    e_ref, C_ref = oracle.geneig_lowdin_pruned(Hd, Sfull, 1e-9)
    assert e_ref.shape == (m,)
    nel = 0.3 * m
    mu_ref, f_ref = oracle.fermi(e_ref[None], [1.0], nel, prob.kT)
    D_ref = oracle.density(np.hstack([C_ref, np.zeros((n, n - m))]), np.append(f_ref[0], np.zeros(n - m)))
    nao.set_lowdin_threshold(1e-9)
    try:
        flags = nao.NAO_LOWDIN | (nao.NAO_NC_BLOCK_S if kind == "nc" else 0)
        E, C, info = nao.geneig(to_dev(Hd[None]), to_dev(Sd[None]), flags=flags)
    finally:
        nao.set_lowdin_threshold(0.0)
    assert int(info.abs().max()) == 0
    e = E.cpu().numpy()[0]
    assert np.abs(e[:m] - e_ref).max() <= TOL_E
    assert np.abs(e[m:] - nao.NAO_PRUNED_LEVEL).max() <= 1e-6
    assert np.abs(to_np(C)[0][:, m:]).max() <= 1e-10
    mu, F = nao.fermi_mu(E, [1.0], nel, prob.kT)
    assert abs(mu - mu_ref) <= TOL_MU
    D = to_np(nao.density_matrix(C, F))[0]
    assert np.abs(D - D_ref).max() <= TOL_D
    assert abs(np.trace(D @ Sfull).real - nel) <= 1e-8


def test_default_reduction_at_the_switch_over_size(nao):
    """Config 2 recipe at 128 atoms (n = 1664 real, 2 spins, one shared S): above the switch-over order (1536) the library takes
    the two-stage reduction by itself.  The step must agree with the forced one-stage step (e, mu, D) and satisfy the invariants
    of the definition (C^H S C = I, residual, electron count); the closed-form chain at the same order pins the eigenvalues.
    Full-size runs of the same path: test_config2 / bench.py."""
    prob = make_config(2, nat=128)
    assert prob.n == 1664 and not prob.is_complex
    nao.profile_enable(True)
    got = run_path(nao, prob)
    torch.cuda.synchronize()
    phases = nao.profile_read()
    nao.profile_enable(False)
    assert phases["band_to_tridiagonal"] > 0.05          # the two-stage path ran
    one = run_path(nao, prob, flags=nao.NAO_TRD_ONE_STAGE)
    assert np.abs(got["e"] - one["e"]).max() <= TOL_E
    assert abs(got["mu"] - one["mu"]) <= TOL_MU
    ne = 0.0
    for b in range(prob.batch):
        assert np.abs(got["D"][b] - one["D"][b]).max() <= TOL_D
        Sb, Cb = prob.S_full(b), got["C"][b]
        assert np.abs(Cb.T @ Sb @ Cb - np.eye(prob.n)).max() <= TOL_ORTH
        assert np.abs(prob.H_full(b) @ Cb - Sb @ Cb * got["e"][b]).max() <= 1e-10
        ne += prob.weights[b] * np.trace(got["D"][b] @ Sb)
    assert abs(ne - prob.n_electrons) <= 1e-8
    n = 1664
    chain = np.diag(np.full(n - 1, -1.0), 1) + np.diag(np.full(n - 1, -1.0), -1)
    E, Z, info = nao.heev(to_dev(chain[None]))
    assert np.abs(E.cpu().numpy()[0] - np.sort(-2.0 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1)))).max() <= 1e-12


@pytest.mark.parametrize("idx,nat", [(0, None), (1, 6), (2, 8), (3, 4)])
def test_solve_host_matches_the_separate_calls_and_the_oracle(nao, idx, nat):
    """nao_solve_host (host buffers in and out, H copied on a second stream while S is factored, D returned item by item)
    against the oracle and against the three separate calls on device buffers."""
    prob = make_config(idx, nat=nat)
    ref = oracle.solve_problem(prob)
    flags = nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0
    Hh = torch.from_numpy(prob.H).pin_memory()
    S_np = prob.S
    if idx == 2:
        S_np = np.ascontiguousarray(prob.S[:1])          # the spin channels share one overlap matrix
    Sh = torch.from_numpy(S_np.copy()).pin_memory()
    for rep in range(2):                                  # second call reuses the internal stream and events
        r = nao.solve_host(Hh, Sh, prob.weights, prob.n_electrons, prob.kT, flags=flags)
        assert int(r["info"].abs().max()) == 0
        got = dict(e=r["E"].numpy(), mu=r["mu"], D=np.swapaxes(r["D"].numpy(), -1, -2))
        assert np.abs(got["e"] - ref["e"]).max() <= TOL_E
        assert abs(got["mu"] - ref["mu"]) <= TOL_MU
        for b in range(prob.batch):
            assert np.abs(got["D"][b] - ref["D"][b]).max() <= TOL_D
    sep = run_path(nao, prob)
    assert np.abs(got["e"] - sep["e"]).max() <= 1e-12
    for b in range(prob.batch):
        assert np.abs(got["D"][b] - sep["D"][b]).max() <= 1e-12


def test_config1_full_size_all_items(nao):
    """BASELINE config 1 at full size (64 atoms: n = 832 complex, 8 k-points x 2 spins = 16 items in one batched call, the
    launch configuration `bench.py --workload c1` times).  ALL 16 items are solved by the Jacobi oracle: eigenvalues and the
    density matrix (oracle eigenvectors, occupations from the oracle's Fermi level over all 16 x 832 oracle levels) are
    compared element by element, mu against the oracle's; every item also goes through the invariants of the definition."""
    prob = make_config(1)
    assert prob.n == 832 and prob.batch == 16 and prob.is_complex
    got = run_path(nao, prob)
    mu_ref, f_ref = oracle.fermi(got["e"], prob.weights, prob.n_electrons, prob.kT)
    assert abs(got["mu"] - mu_ref) <= TOL_MU
    assert np.abs(got["f"] - f_ref).max() <= 1e-9
    ne = 0.0
    for b in range(prob.batch):
        Cb, Sb, Hb = got["C"][b], prob.S_full(b), prob.H_full(b)
        assert np.abs(Cb.conj().T @ (Sb @ Cb) - np.eye(prob.n)).max() <= TOL_ORTH
        assert np.abs(Hb @ Cb - (Sb @ Cb) * got["e"][b]).max() <= 1e-10
        ne += prob.weights[b] * np.sum(got["D"][b] * Sb.T).real
    assert abs(ne - prob.n_electrons) <= 1e-8
    assert np.abs(got["e"][:8] - got["e"][7::-1]).max() <= 1e-10          # e(k) = e(-k)
    e_all, C_all = [], []
    for b in range(prob.batch):
        e_or, C_or, _ = oracle.geneig(prob.H_full(b), prob.S_full(b))
        assert np.abs(got["e"][b] - e_or).max() <= TOL_E
        e_all.append(e_or); C_all.append(C_or)
    mu_or, f_or = oracle.fermi(np.array(e_all), prob.weights, prob.n_electrons, prob.kT)      # the oracle's own chain
    assert abs(got["mu"] - mu_or) <= TOL_MU
    for b in range(prob.batch):
        assert np.abs(got["D"][b] - oracle.density(C_all[b], f_or[b])).max() <= TOL_D


# ------------------------------------------------------------------------------- ill-conditioned overlap (a1/a2 robustness)
@pytest.mark.parametrize("delta", [1e-3, 1e-4])
def test_ill_conditioned_overlap_near_duplicate_orbitals(nao, delta):
    """The reduction uses the explicit inverse W = L^{-1} (reading C2b) where north_star words it as triangular
    solves.  Stress it where that could matter: six orbitals are replaced by near-duplicates of others,
    phi'_j = delta phi_j + phi_k  (H' = T^T H T, S' = T^T S T), which drives cond(S') to 4e6 (delta = 1e-3) and 4e8 (1e-4) while
    the pencil's eigenvalues, mu and T D' T^T stay EXACTLY those of the original well-conditioned problem -- so the
    oracle's solution of the original problem is the reference.  FP64 accuracy of any backward-stable method is
    ~ cond(S) eps (LAPACK's dsygvd and a TRSM-based reduction measure the same 2e-11 / 2e-9 in e and 7e-11 / 1e-8 in
    orthogonality on these inputs): the north_star bars are asserted at cond 4e6 for e, mu and D; orthogonality and the
    cond 4e8 case are held to cond(S) eps / 2."""
    prob = make_config(2, nat=16)
    n = prob.n
    ref = oracle.solve_problem(prob)
    T = np.eye(n)
    for t in range(6):
        j, k = 13 * t + 2, 13 * t + 7 + 13 * 8
        T[:, j] *= delta
        T[k, j] += 1.0
    H2 = np.stack([T.T @ prob.H_full(b) @ T for b in range(2)]); H2 = (H2 + np.swapaxes(H2, -1, -2)) / 2
    S2 = np.stack([T.T @ prob.S_full(b) @ T for b in range(2)]); S2 = (S2 + np.swapaxes(S2, -1, -2)) / 2
    cond = np.linalg.cond(S2[0])
    assert (2e6 if delta == 1e-3 else 2e8) <= cond <= (1e7 if delta == 1e-3 else 1e9)
    ceps = 0.5 * cond * 2.220446049250313e-16
    for flags in (0, nao.NAO_TRD_TWO_STAGE):
        E, C, info = nao.geneig(to_dev(H2), to_dev(S2), flags=flags)
        assert int(info.abs().max()) == 0
        mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
        D = to_np(nao.density_matrix(C, F))
        tol_e = TOL_E if delta == 1e-3 else max(TOL_E, ceps)
        assert np.abs(E.cpu().numpy() - ref["e"]).max() <= tol_e
        assert abs(mu - ref["mu"]) <= (TOL_MU if delta == 1e-3 else max(TOL_MU, ceps))
        for b in range(2):
            Cb = to_np(C)[b]
            assert np.abs(Cb.T @ S2[b] @ Cb - np.eye(n)).max() <= max(TOL_ORTH, ceps)
            assert np.abs(T @ D[b] @ T.T - ref["D"][b]).max() <= (TOL_D if delta == 1e-3 else max(TOL_D, 10 * ceps))


# ------------------------------------------------------------------------------- leading dimensions, strides, streams
@pytest.mark.parametrize("pad", [1, 3])
@pytest.mark.parametrize("cplx", [False, True])
def test_padded_leading_dimensions_strides_and_side_stream(nao, pad, cplx):
    """The C ABI takes LAPACK-style leading dimensions and batch strides: nao_geneig, nao_geneig_partial, nao_heev and
    nao_density_matrix are called through raw ctypes on sub-views of larger buffers (ld = n + pad: odd, so nothing past the
    first column is 16-byte aligned; stride > ld n) on a non-default stream.  Results must equal the ld = n results bit for
    bit and every padding element must be left untouched."""
    import ctypes
    lib = nao.lib()
    prob = make_config(1, nat=6) if cplx else make_config(2, nat=8)
    n, batch = prob.n, 2
    dt = torch.complex128 if cplx else torch.float64
    code = nao.NAO_COMPLEX if cplx else nao.NAO_REAL
    H = torch.from_numpy(prob.H[:batch]).to(DEV)
    S = torch.from_numpy(prob.S[:batch].copy()).to(DEV)
    E0, C0, _ = nao.geneig(H, S.clone())
    w2 = [float(prob.weights[0])] * batch
    ne = prob.n_electrons * batch / prob.batch
    mu0, F0 = nao.fermi_mu(E0, w2, ne, prob.kT)
    D0 = nao.density_matrix(C0, F0)
    nv = nao.occupied_count(F0) + 3
    E0p, C0p, _ = nao.geneig(H, S.clone(), n_vec=nv)
    Eh0, Z0, _ = nao.heev(H.clone())
    ld = n + pad
    stride = ld * n + 7
    SENT = 777.0

    def padded(src=None):
        buf = torch.full((batch * stride + 5,), SENT, dtype=dt, device=DEV)
        view = torch.as_strided(buf, (batch, n, n), (stride, ld, 1))         # [b, col, row]: column-major items with ld
        if src is not None:
            view.copy_(src)
        return buf, view

    def untouched(buf, view):
        mask = torch.ones_like(buf, dtype=torch.bool)
        torch.as_strided(mask, (batch, n, n), (stride, ld, 1)).fill_(False)
        return bool((buf[mask] == SENT).all())

    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        sp = st.cuda_stream
        Hb, Hv = padded(H); Sb, Sv = padded(S); Cb, Cv = padded(); Db, Dv = padded()
        E = torch.empty((batch, n), dtype=torch.float64, device=DEV)
        info = torch.zeros(batch, dtype=torch.int32, device=DEV)
        work = torch.empty(nao.geneig_workspace(n, batch, code, 0) + 256, dtype=torch.uint8, device=DEV)
        rc = lib.nao_geneig(n, batch, code, 0, Hb.data_ptr(), ld, stride, Sb.data_ptr(), ld, stride, E.data_ptr(), Cb.data_ptr(), ld,
                            stride, work.data_ptr(), work.numel(), info.data_ptr(), sp)
        assert rc == 0
        st.synchronize()
        assert int(info.abs().max()) == 0
        assert torch.equal(E, E0) and torch.equal(Cv, C0)
        assert untouched(Cb, Cv) and untouched(Sb, Sv) and torch.equal(Hv, H)
        # density matrix on the padded C into a padded D
        need = ctypes.c_size_t(0)
        lib.nao_density_workspace(n, batch, code, ctypes.byref(need))
        dwork = torch.empty(need.value + 256, dtype=torch.uint8, device=DEV)
        rc = lib.nao_density_matrix(n, batch, code, Cb.data_ptr(), ld, stride, F0.data_ptr(), Db.data_ptr(), ld, stride,
                                    dwork.data_ptr(), dwork.numel(), sp)
        assert rc == 0
        st.synchronize()
        assert torch.equal(Dv, D0) and untouched(Db, Dv)
        # partial spectrum with the cached factor: the columns that are not back-transformed are zeroed column by column
        Cb2, Cv2 = padded()
        rc = lib.nao_geneig_partial(n, batch, code, nao.NAO_S_FACTORED, nv, Hb.data_ptr(), ld, stride, Sb.data_ptr(), ld, stride,
                                    E.data_ptr(), Cb2.data_ptr(), ld, stride, work.data_ptr(), work.numel(), info.data_ptr(), sp)
        assert rc == 0
        st.synchronize()
        assert torch.equal(E, E0p) and torch.equal(Cv2, C0p) and untouched(Cb2, Cv2)
        # standard problem on padded A and Z
        Ab, Av = padded(H); Zb, Zv = padded()
        lib.nao_heev_workspace(n, batch, code, 0, ctypes.byref(need))
        hwork = torch.empty(need.value + 256, dtype=torch.uint8, device=DEV)
        rc = lib.nao_heev(n, batch, code, 0, Ab.data_ptr(), ld, stride, E.data_ptr(), Zb.data_ptr(), ld, stride, hwork.data_ptr(),
                          hwork.numel(), info.data_ptr(), sp)
        assert rc == 0
        st.synchronize()
        assert torch.equal(E, Eh0) and torch.equal(Zv, Z0) and untouched(Zb, Zv) and untouched(Ab, Av)


# ------------------------------------------------------------------------------- concurrent mid-size solves
@pytest.mark.parametrize("groups", ["NAO_STREAM_GROUPS_2", "NAO_STREAM_GROUPS_4", "NAO_STREAM_GROUPS_8"])
def test_stream_groups_equal_the_single_batched_call(nao, groups):
    """NAO_STREAM_GROUPS_*: the 16 (k, spin) items of the config-1 recipe spread over 2/4/8 internal streams (each group with
    its share of the SMs for the grid-barrier kernels) must give what the single batched call gives.  Not bit for bit: the
    split-K factors of the blocked Cholesky and of the panel products depend on how many items share a launch, so partial
    sums are grouped differently; the factor of S, e, mu and D agree to a few ulps (1e-13 / 1e-12) -- with the one-stage and
    the two-stage reduction, with the cached factor and for the partial spectrum."""
    gflag = getattr(nao, groups)
    for nat, extra in ((16, 0), (16, nao.NAO_TRD_TWO_STAGE), (64, 0)):
        prob = make_config(1, nat=nat)
        H = torch.from_numpy(prob.H).to(DEV)
        S1 = torch.from_numpy(prob.S.copy()).to(DEV)
        S2 = torch.from_numpy(prob.S.copy()).to(DEV)
        E1, C1, i1 = nao.geneig(H, S1, flags=extra)
        E2, C2, i2 = nao.geneig(H, S2, flags=extra | gflag)
        assert int(i1.abs().max()) == 0 and int(i2.abs().max()) == 0
        assert float((S1 - S2).abs().max()) <= 1e-13                # the factor of S
        assert float((E1 - E2).abs().max()) <= 1e-13
        mu1, F1 = nao.fermi_mu(E1, prob.weights, prob.n_electrons, prob.kT)
        mu2, F2 = nao.fermi_mu(E2, prob.weights, prob.n_electrons, prob.kT)
        assert abs(mu1 - mu2) <= 1e-13
        D1, D2 = nao.density_matrix(C1, F1), nao.density_matrix(C2, F2)
        assert float((D1 - D2).abs().max()) <= 1e-12
        # later SCF step, occupied vectors only
        nv = nao.occupied_count(F1) + 4
        E3, C3, _ = nao.geneig(H, S1, flags=extra | nao.NAO_S_FACTORED, n_vec=nv)
        E4, C4, _ = nao.geneig(H, S2, flags=extra | nao.NAO_S_FACTORED | gflag, n_vec=nv)
        assert float((E3 - E4).abs().max()) <= 1e-13
        D3, D4 = nao.density_matrix(C3, F1), nao.density_matrix(C4, F1)
        assert float((D3 - D4).abs().max()) <= 1e-12 and float((D3 - D1).abs().max()) <= 1e-12
        if nat == 16:                                                # against the oracle as well
            ref = oracle.solve_problem(prob)
            assert np.abs(E2.cpu().numpy() - ref["e"]).max() <= TOL_E and abs(mu2 - ref["mu"]) <= TOL_MU
            for b in range(prob.batch):
                assert np.abs(to_np(D2)[b] - ref["D"][b]).max() <= TOL_D


def test_stream_groups_two_stage_order_2080_shared_factor(nao):
    """The SM-limited plans of the two-stage path only differ from the unlimited ones from order 1024 on (panel-QR CTAs per
    item, chase CTAs, the look-ahead switched off, q2_apply's slab width): four real items of order 2080 (config-2 recipe at 160
    atoms, the second pair with H scaled) under NAO_STREAM_GROUPS_4 = one item per group on 37 SMs, full and partial spectrum,
    against the single batched call.  Then ONE shared overlap (strideS = 0) that is already factored (NAO_S_FACTORED): the
    only grouped case in which the workspace query (shared S counted once) and the run (every group unpacks the shared factor)
    see different S layouts."""
    prob = make_config(2, nat=160)
    n = prob.n
    assert n == 2080 and np.array_equal(prob.S[0], prob.S[1])
    H = torch.from_numpy(np.concatenate([prob.H, 0.5 * prob.H])).to(DEV)
    S4 = np.concatenate([prob.S, prob.S])
    g4 = nao.NAO_STREAM_GROUPS_4
    S1, S2 = torch.from_numpy(S4.copy()).to(DEV), torch.from_numpy(S4.copy()).to(DEV)
    E1, C1, i1 = nao.geneig(H, S1)                                   # default = two-stage at this order
    E2, C2, i2 = nao.geneig(H, S2, flags=g4)
    assert int(i1.abs().max()) == 0 and int(i2.abs().max()) == 0
    assert float((S1 - S2).abs().max()) <= 1e-12
    assert float((E1 - E2).abs().max()) <= 1e-12
    assert float((E1[2:] - 0.5 * E1[:2]).abs().max()) <= 1e-12        # the scaled pair
    mu, F = nao.fermi_mu(E1, list(prob.weights) * 2, 2 * prob.n_electrons, prob.kT)
    nv = nao.occupied_count(F) + 8
    assert nv < n // 2
    D1, D2 = nao.density_matrix(C1, F), nao.density_matrix(C2, F)
    assert float((D1 - D2).abs().max()) <= 1e-10
    Cm = C2[3].T                                                      # an item of the last group: C^T S C = I, residual
    Sm = torch.from_numpy(prob.S_full(1)).to(DEV)
    assert float((Cm.T @ Sm @ Cm - torch.eye(n, dtype=torch.float64, device=DEV)).abs().max()) <= TOL_ORTH
    Hm = 0.5 * torch.from_numpy(prob.H_full(1)).to(DEV)
    assert float((Hm @ Cm - (Sm @ Cm) * E2[3][None, :]).abs().max()) <= 1e-10
    # partial spectrum, cached per-item factor
    E3, C3, _ = nao.geneig(H, S2, flags=g4 | nao.NAO_S_FACTORED, n_vec=nv)
    assert float((E3 - E1).abs().max()) <= 1e-12
    assert float((nao.density_matrix(C3, F) - D1).abs().max()) <= 1e-10
    assert float(C3[:, nv:].abs().max()) == 0.0
    # one shared overlap: factored by an ungrouped call (the group flag is ignored while S is unfactored), reused by groups
    Ss = torch.from_numpy(prob.S[:1].copy()).to(DEV)
    E5, C5, i5 = nao.geneig(H, Ss, flags=g4)
    assert int(i5.abs().max()) == 0
    assert float((E5 - E1).abs().max()) <= 1e-12 and float((Ss[0] - S1[0]).abs().max()) <= 1e-12
    E6, C6, i6 = nao.geneig(H, Ss, flags=g4 | nao.NAO_S_FACTORED)
    assert int(i6.abs().max()) == 0
    assert float((E6 - E1).abs().max()) <= 1e-12
    assert float((nao.density_matrix(C6, F) - D1).abs().max()) <= 1e-10
    E7, C7, _ = nao.geneig(H, Ss, flags=nao.NAO_STREAM_GROUPS_2 | nao.NAO_S_FACTORED, n_vec=nv)
    assert float((E7 - E1).abs().max()) <= 1e-12
    assert float((nao.density_matrix(C7, F) - D1).abs().max()) <= 1e-10


# ------------------------------------------------------------------------------- flag-synchronised kernels: reproducibility
@pytest.mark.parametrize("cplx", [False, True])
def test_flag_synchronised_kernels_are_bit_reproducible(nao, cplx):
    """hetrd_panel_kernel / panel_qr_kernel (software grid barrier), chase_kernel (acquire/release progress counters between
    CTAs), q2_apply_kernel (mbarrier ring, per-warp staging) and the TMA-fed HEMV synchronise through flags in global or
    shared memory.  compute-sanitizer is closed on this pool, so a missing acquire, release or barrier is looked for the
    other way: every cross-CTA reduction sums partial results in a fixed order, hence any run of the same input must give
    the same bits; a race shows up as a difference between repetitions.  Eight repetitions of both reductions on three
    sizes (several items per launch, ragged and 64-aligned orders), with other work queued in between to vary the timing."""
    rng = np.random.default_rng(77)
    # the last size is config 3's (complex) / config 2's (real): the widest launch of q2_apply_kernel, nine / twelve consumer
    # warps per CTA -- where a missing proxy fence between the fragment loads and the TMA refill of a ring stage showed up as
    # a handful of wrong columns in most runs, and nowhere else
    for n, batch in ((333, 3), (832, 4), (2176, 2), (9984 if cplx else 6656, 1 if cplx else 2)):
        if n > 4000:
            g = torch.Generator(device=DEV); g.manual_seed(n)
            A = torch.randn(batch, n, n, dtype=torch.float64, device=DEV, generator=g)
            if cplx:
                A = torch.complex(A, torch.randn(batch, n, n, dtype=torch.float64, device=DEV, generator=g))
            A = A + A.mH
        else:
            A = rng.standard_normal((batch, n, n))
            if cplx:
                A = A + 1j * rng.standard_normal((batch, n, n))
            A = to_dev(A + np.swapaxes(A.conj(), -1, -2))
        for flag in (nao.NAO_TRD_ONE_STAGE, nao.NAO_TRD_TWO_STAGE):
            if n > 4000 and flag == nao.NAO_TRD_ONE_STAGE:
                continue
            E0, Z0, info = nao.heev(A.clone(), flags=flag)
            assert int(info.abs().max()) == 0
            for rep in range(7):
                if rep % 2:
                    torch.empty(64 << 20, dtype=torch.uint8, device=DEV).zero_()
                E, Z, _ = nao.heev(A.clone(), flags=flag)
                assert torch.equal(E, E0) and torch.equal(Z, Z0), (n, flag, rep)
