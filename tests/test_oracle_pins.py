"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the definition it pins: Eq. 5/11/21 for the eigenproblem, the
Fermi-Dirac occupation for mu/f, Eq. 8/23 for D, the Loewdin route
 as an independent second reduction, and SURVEY.md 8(c) "What pins each part".
"""
import numpy as np
import pytest
import scipy.linalg as sl

import oracle
from paper_2606_09058_b200.synth import make_config

KT = 9.5e-4


def chain(n, t=1.0):
    T = np.zeros((n, n))
    i = np.arange(n - 1)
    T[i, i + 1] = T[i + 1, i] = 1.0
    return t * T


def rand_herm(rng, n, cplx):
    A = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0)
    return (A + A.conj().T) / 2


def rand_spd(rng, n, cplx):
    A = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0)
    return A @ A.conj().T / n + np.eye(n)


# ---------------------------------------------------------------- closed forms
@pytest.mark.parametrize("n", [2, 3, 12, 51])
def test_tight_binding_chain_closed_form(n):
    """Open chain, S = I: e_k = 2 t cos(k pi/(n+1)), vectors sqrt(2/(n+1)) sin(j k pi/(n+1)) (north_star)."""
    t = -0.7
    e, C, _ = oracle.geneig(chain(n, t), np.eye(n))
    k = np.arange(1, n + 1)
    exact = np.sort(2 * t * np.cos(k * np.pi / (n + 1)))
    assert np.abs(e - exact).max() < 1e-13
    # eigenvectors are non-degenerate: compare up to sign
    order = np.argsort(2 * t * np.cos(k * np.pi / (n + 1)))
    j = np.arange(1, n + 1)[:, None]
    V = np.sqrt(2 / (n + 1)) * np.sin(j * k[order][None, :] * np.pi / (n + 1))
    assert np.abs(np.abs(C) - np.abs(V)).max() < 1e-12
    assert np.abs(C.T @ C - np.eye(n)).max() < 1e-13  # S = I  =>  C orthogonal


@pytest.mark.parametrize("n", [7, 40])
def test_chain_with_overlap_closed_form(n):
    """H = eps0 I + t T, S = I + s T commute: e_k = (eps0 + t tau_k)/(1 + s tau_k), tau_k = 2 cos(k pi/(n+1))."""
    eps0, t, s = -0.3, -0.8, 0.2
    T = chain(n)
    e, C, _ = oracle.geneig(eps0 * np.eye(n) + t * T, np.eye(n) + s * T)
    tau = 2 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1))
    assert np.abs(e - np.sort((eps0 + t * tau) / (1 + s * tau))).max() < 1e-13


@pytest.mark.parametrize("theta", [0.0, 0.37])
def test_ring_with_peierls_phase(theta):
    """Complex Hermitian ring, H_{j,j+1} = t e^{i theta}: e_m = 2 t cos(2 pi m/n + theta).  theta = 0 has exact
    +-m degeneracies; D is gauge independent and equals (1/n) sum_m f_m e^{i q_m (j-l)} (plane waves)."""
    n, t = 16, -1.0
    H = np.zeros((n, n), dtype=complex)
    for j in range(n):
        H[j, (j + 1) % n] += t * np.exp(1j * theta)
        H[(j + 1) % n, j] += t * np.exp(-1j * theta)
    e, C, _ = oracle.geneig(H, np.eye(n))
    q = 2 * np.pi * np.arange(n) / n
    em = 2 * t * np.cos(q + theta)            # plane wave c_j = e^{i q j}/sqrt(n):  (H c)_j = t(e^{i(q+theta)} + c.c.) c_j
    assert np.abs(e - np.sort(em)).max() < 1e-13
    kT = 0.05
    mu, f = oracle.fermi(e[None], [1.0], 5.0, kT)
    D = oracle.density(C, f[0])
    fm = 1 / (1 + np.exp((em - mu) / kT))
    j = np.arange(n)
    Dex = (np.exp(1j * q[None, None, :] * (j[:, None, None] - j[None, :, None])) * fm).sum(-1) / n
    assert np.abs(D - Dex).max() < 1e-12
    assert abs(np.trace(D).real - 5.0) < 1e-12


def _eig2x2_longdouble(H, S):
    """Roots of det(H - lam S) = 0 for a 2x2 Hermitian-definite pencil, in long double."""
    ld = np.longdouble
    h11, h22, s11, s22 = ld(H[0, 0].real), ld(H[1, 1].real), ld(S[0, 0].real), ld(S[1, 1].real)
    h12, s12 = complex(H[0, 1]), complex(S[0, 1])
    a = s11 * s22 - ld(abs(s12) ** 2)
    b = -(h11 * s22 + h22 * s11 - 2 * ld((h12 * np.conj(s12)).real))
    c = h11 * h22 - ld(abs(h12) ** 2)
    disc = np.sqrt(b * b - 4 * a * c)
    q = -(b + np.copysign(disc, b)) / 2
    r = sorted([q / a, c / q])
    return np.array(r, dtype=np.float64)


@pytest.mark.parametrize("cplx", [False, True])
def test_bruteforce_2x2_and_kron_4x4(cplx):
    rng = np.random.default_rng(5)
    for _ in range(20):
        H1, S1 = rand_herm(rng, 2, cplx), rand_spd(rng, 2, cplx)
        e, C, _ = oracle.geneig(H1, S1)
        ex1 = _eig2x2_longdouble(H1, S1)
        assert np.abs(e - ex1).max() < 1e-13 * max(1, np.abs(ex1).max())
        assert np.abs(H1 @ C - S1 @ C * e).max() < 1e-13
        # direct sum of two 2x2 pencils
        H2, S2 = rand_herm(rng, 2, cplx), rand_spd(rng, 2, cplx)
        ex2 = _eig2x2_longdouble(H2, S2)
        e4, _, _ = oracle.geneig(sl.block_diag(H1, H2), sl.block_diag(S1, S2))
        assert np.abs(e4 - np.sort(np.concatenate([ex1, ex2]))).max() < 1e-12
        # Kronecker: (H1 x S2 + S1 x H2, S1 x S2) has eigenvalues lam_i + mu_j
        ek, _, _ = oracle.geneig(np.kron(H1, S2) + np.kron(S1, H2), np.kron(S1, S2))
        assert np.abs(ek - np.sort((ex1[:, None] + ex2[None, :]).ravel())).max() < 1e-12


def test_noncollinear_common_axis_splitting():
    """H_NC = H0 (x) I2 + J S (x) (m.sigma) in the paper's spin-major block layout (Eq. 21, 25-27;
    PAPER.md:113-115, 175-179) with S_NC = diag(S, S): spectrum is {e_i(H0,S) +- J} exactly."""
    rng = np.random.default_rng(11)
    N, J = 9, 0.05
    H0, S = rand_herm(rng, N, False), rand_spd(rng, N, False)
    m = rng.standard_normal(3)
    m /= np.linalg.norm(m)
    Hnc = np.block([[H0 + J * m[2] * S, J * (m[0] - 1j * m[1]) * S], [J * (m[0] + 1j * m[1]) * S, H0 - J * m[2] * S]])
    Snc = np.block([[S, 0 * S], [0 * S, S]]).astype(complex)
    e0, _, _ = oracle.geneig(H0, S)
    e, C, _ = oracle.geneig(Hnc, Snc)
    assert np.abs(e - np.sort(np.concatenate([e0 - J, e0 + J]))).max() < 1e-13
    # spin-diagonal H_NC reproduces two collinear solves
    Hu, Hd = rand_herm(rng, N, False), rand_herm(rng, N, False)
    Hsd = np.block([[Hu, 0 * Hu], [0 * Hu, Hd]]).astype(complex)
    e2, _, _ = oracle.geneig(Hsd, Snc)
    eu, _, _ = oracle.geneig(Hu, S)
    ed, _, _ = oracle.geneig(Hd, S)
    assert np.abs(e2 - np.sort(np.concatenate([eu, ed]))).max() < 1e-13


# ---------------------------------------------------------------- invariants
@pytest.mark.parametrize("cplx,n", [(False, 31), (True, 24)])
def test_invariants_random_pencil(cplx, n):
    rng = np.random.default_rng(3)
    H, S = rand_herm(rng, n, cplx), rand_spd(rng, n, cplx)
    e, C, _ = oracle.geneig(H, S)
    assert np.all(np.diff(e) >= 0)
    assert np.abs(C.conj().T @ S @ C - np.eye(n)).max() < 1e-12          # C^H S C = I
    assert np.abs(H @ C - S @ C * e).max() < 1e-12                        # residual
    assert abs(e.sum() - np.trace(np.linalg.solve(S, H)).real) < 1e-11    # sum e = Tr(S^-1 H)
    # congruence invariance: (Q^H H Q, Q^H S Q) has the same spectrum
    Q = rand_herm(rng, n, cplx) + 3 * np.eye(n)
    e2, _, _ = oracle.geneig(Q.conj().T @ H @ Q, Q.conj().T @ S @ Q)
    assert np.abs(e - e2).max() < 1e-11
    # all f = 1:  D = C C^H = S^-1  (independent of the eigen-solver)
    D1 = oracle.density(C, np.ones(n))
    assert np.abs(D1 @ S - np.eye(n)).max() < 1e-12
    # Tr(D S) = electron count
    mu, f = oracle.fermi(e[None], [2.0], 2.0 * (n // 3) + 0.5, 0.01)
    D = oracle.density(C, f[0])
    assert abs(2.0 * np.trace(D @ S).real - (2.0 * (n // 3) + 0.5)) < 1e-11
    assert np.abs(D - D.conj().T).max() < 1e-15
    # LAPACK cross-check
    assert np.abs(e - sl.eigh(H, S, eigvals_only=True)).max() < 1e-12


@pytest.mark.parametrize("cplx", [False, True])
def test_lowdin_route_agrees_with_cholesky_route(cplx):
    """Paper's route S = U s U^H, V = U s^-1/2, H' = V^H H V, C = V C'."""
    rng = np.random.default_rng(8)
    n = 26
    H, S = rand_herm(rng, n, cplx), rand_spd(rng, n, cplx)
    e1, C1, _ = oracle.geneig(H, S)
    e2, C2, _ = oracle.geneig_lowdin(H, S)
    assert np.abs(e1 - e2).max() < 1e-12
    f = 1 / (1 + np.exp((e1 - np.median(e1)) / 0.1))
    assert np.abs(oracle.density(C1, f) - oracle.density(C2, f)).max() < 1e-12


def test_block_diagonal_union_and_unitary_C():
    rng = np.random.default_rng(2)
    A, B = rand_herm(rng, 5, True), rand_herm(rng, 8, True)
    e, C, _ = oracle.geneig(sl.block_diag(A, B), np.eye(13))
    ex = np.sort(np.concatenate([np.linalg.eigvalsh(A), np.linalg.eigvalsh(B)]))
    assert np.abs(e - ex).max() < 1e-13
    assert np.abs(C.conj().T @ C - np.eye(13)).max() < 1e-13


def test_cholesky_factor_and_failure_index():
    rng = np.random.default_rng(4)
    for cplx in (False, True):
        S = rand_spd(rng, 17, cplx)
        L = oracle.cholesky(S)
        assert np.abs(np.triu(L, 1)).max() == 0
        assert np.abs(L @ L.conj().T - S).max() < 1e-14
    S = np.eye(6)
    S[3, 3] = -1.0                     # leading minor 4 is not positive definite
    with pytest.raises(np.linalg.LinAlgError, match="leading minor 4"):
        oracle.cholesky(S)


def test_jacobi_on_textbook_tridiagonals():
    """Clement/Kac matrix (integer spectrum -(n-1), -(n-3), ..., n-1) and Wilkinson W21+ (near-degenerate pairs)."""
    n = 20
    k = np.arange(1, n)
    T = np.diag(np.sqrt(k * (n - k)), 1)
    T = T + T.T
    e, Z = oracle.heev(T)
    assert np.abs(e - np.arange(-(n - 1), n, 2)).max() < 1e-12
    W = np.diag(np.abs(np.arange(-10, 11)).astype(float)) + np.diag(np.ones(20), 1) + np.diag(np.ones(20), -1)
    e, Z = oracle.heev(W)
    assert abs(e[-1] - 10.746194182903393) < 1e-12      # largest eigenvalue of W21+ (Wilkinson 1965)
    assert e[-1] - e[-2] < 1e-12 + 1e-13 * 7 and e[-1] - e[-2] > 0   # pair agrees to ~7e-14
    assert np.abs(W @ Z - Z * e).max() < 1e-12
    assert np.abs(Z.T @ Z - np.eye(21)).max() < 1e-13


# ---------------------------------------------------------------- Fermi level
def test_fermi_single_degenerate_level():
    """n-fold level e0 with N_e electrons: mu = e0 + kT ln(nu/(1-nu)), nu = N_e/(g n)."""
    e0, n, g, Ne = -0.4, 10, 2.0, 7.0
    mu, f = oracle.fermi(np.full((1, n), e0), [g], Ne, KT)
    nu = Ne / (g * n)
    assert abs(mu - (e0 + KT * np.log(nu / (1 - nu)))) < 1e-15
    assert np.abs(f - nu).max() < 1e-13


def test_fermi_two_level_midpoint_even_in_a_huge_gap():
    for gap in (0.01, 1.0, 5.0):         # 5 Ha = 5263 kT: P and Q underflow in the plain form
        e = np.array([[-gap / 2] * 4 + [gap / 2] * 4]) + 0.123
        mu, f = oracle.fermi(e, [2.0], 8.0, KT)
        assert abs(mu - 0.123) < 1e-14


def test_fermi_particle_hole_symmetric_chain():
    """Bipartite chain at half filling: mu = 0 exactly, D_jj = 1/2."""
    n = 30
    e, C, _ = oracle.geneig(chain(n, -1.0), np.eye(n))
    mu, f = oracle.fermi(e[None], [2.0], float(n), 0.02)
    assert abs(mu) < 1e-14
    D = oracle.density(C, f[0])
    assert np.abs(np.diag(D) - 0.5).max() < 1e-13


def test_fermi_matches_bruteforce_root_and_shared_mu_over_batch():
    rng = np.random.default_rng(9)
    e = np.sort(rng.uniform(-1, 1, (4, 25)), axis=1)
    w = np.array([0.25, 0.25, 0.125, 0.375])
    Ne = 9.3
    mu, f = oracle.fermi(e, w, Ne, 0.01)
    assert abs((w[:, None] * f).sum() - Ne) < 1e-12
    import scipy.optimize as so
    g = lambda m: (w[:, None] / (1 + np.exp((e - m) / 0.01))).sum() - Ne
    assert abs(mu - so.brentq(g, -2, 2, xtol=1e-15, rtol=1e-15)) < 1e-12
    with pytest.raises(ValueError):
        oracle.fermi(e, w, 26.0, 0.01)


# ---------------------------------------------------------------- the paper-shaped workloads
def test_config0_against_lapack_and_invariants():
    p = make_config(0)
    r = oracle.solve_problem(p)
    H, S = p.H_full(0), p.S_full(0)
    assert np.abs(r["e"][0] - sl.eigh(H, S, eigvals_only=True)).max() < 1e-12
    C, D = r["C"][0], r["D"][0]
    assert np.abs(C.T @ S @ C - np.eye(p.n)).max() < 1e-12
    assert np.abs(H @ C - S @ C * r["e"][0]).max() < 1e-12
    assert abs(2.0 * np.trace(D @ S) - 32.0) < 1e-10                 # Tr(D S) = N_e (g = 2, reading C4)
    # gap of ~47 kT: mu must sit where particle and hole tails balance; check against the defining equation
    e, mu = r["e"][0], r["mu"]
    particles = (1 / (1 + np.exp((e[16:] - mu) / p.kT))).sum()
    holes = (1 / (1 + np.exp((mu - e[:16]) / p.kT))).sum()      # 1 - f without cancellation
    assert abs(particles - holes) < 1e-9 * particles
    fref = 1 / (1 + np.exp((e[16:24] - mu) / p.kT))
    assert np.abs(r["f"][0][16:24] / fref - 1).max() < 1e-11


def test_config1_replica_time_reversal_and_lapack():
    """e(k) = e(-k) for real real-space H (PAPER.md:224 uses it to halve the k-mesh); complex Hermitian items."""
    p = make_config(1, nat=6)
    assert p.is_complex and p.batch == 16 and p.n == 78
    e0, _, _ = oracle.geneig(p.H_full(0), p.S_full(0))     # k = (-,-,-)
    e7, _, _ = oracle.geneig(p.H_full(7), p.S_full(7))     # k = (+,+,+)
    assert np.abs(e0 - e7).max() < 1e-13
    assert np.abs(e0 - sl.eigh(p.H_full(0), p.S_full(0), eigvals_only=True)).max() < 1e-12
    assert np.abs(p.H_full(0) - p.H_full(7).conj()).max() < 1e-15


def test_config3_replica_noncollinear():
    p = make_config(3, nat=4)
    assert p.nc_block_s and p.n == 104
    r = oracle.solve_problem(p)
    H, S = p.H_full(0), p.S_full(0)
    assert np.abs(H - H.conj().T).max() < 1e-15
    assert np.abs(r["e"][0] - sl.eigh(H, S, eigvals_only=True)).max() < 1e-12
    assert abs(np.trace(r["D"][0] @ S).real - 16.0) < 1e-10


def test_generator_matrices_are_hermitian_and_spd():
    """The input generator must hand Hermitian H and Hermitian positive definite S to both sides (replicas included)."""
    for idx, nat in [(0, None), (1, 6), (1, 16), (2, 8), (3, 4)]:
        p = make_config(idx, nat=nat)
        for b in range(p.batch):
            H, S = p.H_full(b), p.S_full(b)
            assert np.abs(H - H.conj().T).max() < 1e-14
            assert np.abs(S - S.conj().T).max() < 1e-14
            assert np.linalg.eigvalsh(S).min() > 0.05


# ---------------------------------------------------------------- the step after the path
def test_energy_weighted_density_matrix_identities():
    """W = C diag(f e) C^H.  With every f = 1: S W S = H exactly (H C = S C e, C^{-1} = C^H S), whatever the solver;
    for Fermi occupations Tr(W S) = sum f_i e_i, the band energy (Eq. 7 PAPER.md:59 without the factor 2)."""
    rng = np.random.default_rng(11)
    for cplx in (False, True):
        n = 23
        H, S = rand_herm(rng, n, cplx), rand_spd(rng, n, cplx)
        e, C, _ = oracle.geneig(H, S)
        W1 = oracle.energy_density(C, np.ones(n), e)
        assert np.abs(S @ W1 @ S - H).max() < 1e-12
        mu, f = oracle.fermi(e[None], [2.0], 14.0, 0.05)
        W = oracle.energy_density(C, f[0], e)
        assert abs(np.trace(W @ S).real - float((f[0] * e).sum())) < 1e-12
        assert np.abs(W - W.conj().T).max() < 1e-15


def _mp_mesh(L):
    ks = [(sx * 0.25, sy * 0.25, sz * 0.25) for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
    return 2 * np.pi * np.array(ks) / L, np.full(8, 0.125)


def test_fold_density_inverts_the_bloch_sum_on_the_2x2x2_mesh():
    """Eq. 12: M(k) = sum_R exp(+i k.R) M(R).  On the 8 Monkhorst-Pack points k = (2 pi/L)(+-1/4)^3
    sum_k w_k exp(-i k.(R - R')) = prod_d cos(pi (R - R')_d / 2L), which is delta(R, R') for R, R' in {0, L}^3: the fold of
    the Bloch sum returns the real-space matrices.  Unsymmetric random M(R) catch a transposed operand, the R = (L,L,L)
    term catches a phase of the wrong sign."""
    rng = np.random.default_rng(5)
    L, n = 10.8, 7
    kp, w = _mp_mesh(L)
    Rv = L * np.array([(a, b, c) for a in (0, 1) for b in (0, 1) for c in (0, 1)], dtype=float)
    M = rng.standard_normal((8, n, n))
    Dk = np.array([sum(np.exp(1j * (k @ R)) * M[r] for r, R in enumerate(Rv)) for k in kp])
    DR = oracle.fold_density(Dk, kp, w, Rv)
    assert np.abs(DR - M).max() < 1e-14
    # the weighted average at R = 0, antiperiodicity under R -> R + 2L e_x and periodicity 4L of this mesh
    R0 = np.array([[0.0, 0.0, 0.0], [2 * L, 0.0, 0.0], [4 * L, 0.0, 0.0], [L, L, L], [3 * L, L, L]])
    D0 = oracle.fold_density(Dk, kp, w, R0)
    assert np.abs(D0[0] - np.tensordot(w, Dk, axes=1)).max() < 1e-15
    assert np.abs(D0[1] + D0[0]).max() < 1e-14 and np.abs(D0[2] - D0[0]).max() < 1e-14
    assert np.abs(D0[4] + D0[3]).max() < 1e-14


def test_fold_density_single_k_closed_form_and_reality():
    rng = np.random.default_rng(6)
    n = 5
    D = rng.standard_normal((1, n, n)) + 1j * rng.standard_normal((1, n, n))
    k = np.array([[0.31, -0.27, 0.11]])
    Rv = np.array([[3.0, 1.0, -2.0], [0.0, 0.0, 0.0], [-7.5, 2.25, 4.0]])
    DR = oracle.fold_density(D, k, [0.7], Rv)
    for r in range(3):
        ph = 0.7 * complex(np.cos(k[0] @ Rv[r]), -np.sin(k[0] @ Rv[r]))
        assert np.abs(DR[r] - ph * D[0]).max() < 1e-15
    # inversion-symmetric set with D(-k) = conj D(k): D(R) is real
    D2 = np.concatenate([D, D.conj()])
    DR2 = oracle.fold_density(D2, np.concatenate([k, -k]), [0.5, 0.5], Rv)
    assert np.abs(DR2.imag).max() < 1e-16
    assert np.abs(DR2[1].real - D[0].real).max() < 1e-16


# ---------------------------------------------------------------- Loewdin route with pruning
def test_pruned_lowdin_recovers_the_closed_form_spectrum_of_a_basis_with_a_duplicated_orbital():
    """Chain with overlap (closed form e_k = (eps0 + t tau_k)/(1 + s tau_k)) written in a basis in which orbital q appears
    twice: H' = P^T H P, S' = P^T S P with P = [I | e_q] is singular; pruning the null direction must give back exactly the
    n closed-form levels, and the density matrix maps back as P D' P^T = D.  With rel = 0 on a regular pencil the pruned
    route is the plain one."""
    n, eps0, t, sov, q = 12, -0.3, -1.0, 0.2, 4
    T = chain(n)
    H, S = eps0 * np.eye(n) + t * T, np.eye(n) + sov * T
    tau = 2 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1))
    closed = np.sort((eps0 + t * tau) / (1 + sov * tau))
    P = np.hstack([np.eye(n), np.eye(n)[:, [q]]])
    Hd, Sd = P.T @ H @ P, P.T @ S @ P
    assert abs(oracle.heev(Sd)[0][0]) < 1e-14       # singular overlap: one exact null direction
    e, C = oracle.geneig_lowdin_pruned(Hd, Sd, 1e-10)
    assert e.shape == (n,) and C.shape == (n + 1, n)
    assert np.abs(e - closed).max() < 1e-13
    assert np.abs(C.T @ Sd @ C - np.eye(n)).max() < 1e-13
    mu, f = oracle.fermi(e[None], [2.0], 10.0, 0.01)
    e0, C0, _ = oracle.geneig(H, S)
    D0 = oracle.density(C0, oracle.fermi(e0[None], [2.0], 10.0, 0.01)[1][0])
    assert np.abs(P @ oracle.density(np.hstack([C, np.zeros((n + 1, 1))]), np.append(f[0], 0.0)) @ P.T - D0).max() < 1e-13
    rng = np.random.default_rng(2)
    Hr, Sr = rand_herm(rng, 9, True), rand_spd(rng, 9, True)
    e1, C1 = oracle.geneig_lowdin_pruned(Hr, Sr, 0.0)
    e2, C2, _ = oracle.geneig(Hr, Sr)
    assert np.abs(e1 - e2).max() < 1e-13
    assert np.abs(oracle.density(C1, np.arange(9) / 9.0) - oracle.density(C2, np.arange(9) / 9.0)).max() < 1e-13
