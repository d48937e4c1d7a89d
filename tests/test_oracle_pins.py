"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

The paper prints no worked numerical example of D-slash, M or CG (SURVEY.md
section 4), so each part of oracle/lqcd_oracle.cpp is pinned by something that
is not the oracle itself:

  P1 free-field closed form in momentum space      (normalisation G1, phases G5, gamma table)
  P2 true adjointness and gamma5-hermiticity       (adjoint stencil, signs)
  P3 gauge covariance                              (link orientation, U vs U^dag, backward index)
  P4 dense 2^4 build from the Kronecker-delta form (everything, incl. N_mu = 2, G8)
  P5 M(mu)^dag M(mu) = M(0)^dag M(0) + 4 k^2 mu^2  (operator form of the det identity)
  P6 Schur identity against the dense matrix       (G3)
  P7 trivial limits
  P8 CG against a dense Hermitian solve, orthogonality of residuals
  P9 BiCGStab against a dense solve of Mhat and van der Vorst's recurrence on the dense matrix
  P10 fermion force = -dS/dU by central differences of the action built from dense matrices,
      force fields closing the even-odd system, gauge covariance (reading G16)
"""
import numpy as np
import pytest

import lattice_util as lu
import lqcd_inputs as gen

AP = gen.antiperiodic_t()
SEED = gen.BASE_SEED


def _rand_spinor(n, stream):
    return gen.spinor_gaussian(n, SEED, stream)


# --------------------------------------------------------------------------- gamma basis (G4)
def test_gamma_basis_clifford_and_matches_oracle(oracle_mod):
    g = [oracle_mod.gamma(m) for m in range(4)]
    g5 = oracle_mod.gamma(4)
    for m in range(4):
        assert np.array_equal(g[m], lu.GAMMA[m])
        assert np.allclose(g[m], g[m].conj().T)
        for n in range(4):
            anti = g[m] @ g[n] + g[n] @ g[m]
            assert np.allclose(anti, 2.0 * (m == n) * np.eye(4))  # {g_mu,g_nu} = 2 delta
        for s in (+1, -1):
            assert np.linalg.matrix_rank(np.eye(4) + s * g[m]) == 2
    assert np.allclose(g5, g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))


# --------------------------------------------------------------------------- P1 free field
@pytest.mark.parametrize("phases", [AP, np.array([1, 1, 1, 1], dtype=complex),
                                    np.exp(1j * np.pi * np.array([0.3, 0.0, 1.0, 0.5]))])
def test_p1_free_field_full_operator(oracle_mod, phases):
    dims = (4, 4, 6, 8)
    kappa, mu = 0.137, 0.21
    U = gen.gauge_unit(dims)
    rng = np.random.default_rng(7)
    for n in [(0, 0, 0, 0), (1, 0, 2, 3), (3, 2, 5, 1)]:
        p = lu.momentum(dims, phases, n)
        u = rng.normal(size=12) + 1j * rng.normal(size=12)
        psi = lu.plane_wave(dims, p, u)
        got = oracle_mod.m_full(dims, phases, U, psi, kappa, mu)
        A = np.eye(4) + 2j * kappa * mu * lu.GAMMA5
        want = lu.apply_spin(A + lu.free_h(p, kappa), psi)
        assert lu.rel_err(got, want) < 1e-14


def test_p1_free_field_hopping_blocks_and_mhat(oracle_mod):
    dims = (4, 4, 6, 8)
    kappa, mu = 0.137, 0.21
    U = gen.gauge_unit(dims)
    rng = np.random.default_rng(11)
    n = (1, 3, 2, 5)
    p = lu.momentum(dims, AP, n)
    u = rng.normal(size=12) + 1j * rng.normal(size=12)
    psi = lu.plane_wave(dims, p, u)
    h = lu.free_h(p, kappa)
    A = np.eye(4) + 2j * kappa * mu * lu.GAMMA5
    for parity in (0, 1):
        got = oracle_mod.dslash_eo(dims, AP, U, lu.to_half(dims, psi, 1 - parity), parity, kappa)
        want = lu.to_half(dims, lu.apply_spin(h, psi), parity)
        assert lu.rel_err(got, want) < 1e-14
    got = oracle_mod.mhat(dims, AP, U, lu.to_half(dims, psi, 0), kappa, mu)
    want = lu.to_half(dims, lu.apply_spin(A - h @ np.linalg.inv(A) @ h, psi), 0)
    assert lu.rel_err(got, want) < 1e-14


def test_p1_massless_zero_mode(oracle_mod):
    # kappa = (2(am+4))^-1: at m = 0, kappa = 1/8, the free Wilson operator
    # annihilates the constant mode.  This is what fixes -kappa (not -kappa/2) in eq. 6 (G1).
    dims = (4, 4, 4, 4)
    per = np.ones(4, dtype=complex)
    psi = np.ones((lu.volume(dims), 4, 3), dtype=complex)
    out = oracle_mod.m_full(dims, per, gen.gauge_unit(dims), psi, 0.125, 0.0)
    assert np.max(np.abs(out)) < 1e-15


# --------------------------------------------------------------------------- P2 adjoint / gamma5
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_p2_adjointness_and_gamma5_hermiticity_full(oracle_mod, dims):
    kappa, mu = 0.15, 0.1
    phases = np.exp(1j * np.pi * np.array([0.0, 0.25, 0.0, 1.0]))
    U = gen.gauge_haar(dims, SEED)
    V = lu.volume(dims)
    psi, phi = _rand_spinor(V, 6), _rand_spinor(V, 7)
    Mpsi = oracle_mod.m_full(dims, phases, U, psi, kappa, mu, 0)
    Mdphi = oracle_mod.m_full(dims, phases, U, phi, kappa, mu, 1)
    lhs, rhs = np.vdot(phi, Mpsi), np.vdot(Mdphi, psi)  # <phi, M psi> = <M^dag phi, psi>
    assert abs(lhs - rhs) / abs(lhs) < 1e-14
    # gamma5 M(mu) gamma5 = M(-mu)^dag
    g5Mg5 = lu.apply_spin(lu.GAMMA5, oracle_mod.m_full(dims, phases, U, lu.apply_spin(lu.GAMMA5, psi),
                                                       kappa, mu, 0))
    Mmdag = oracle_mod.m_full(dims, phases, U, psi, kappa, -mu, 1)
    assert lu.rel_err(g5Mg5, Mmdag) < 1e-14


def test_p2_adjointness_and_gamma5_hermiticity_eo(oracle_mod):
    dims = (4, 4, 4, 6)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    h = lu.volume(dims) // 2
    a, b = _rand_spinor(h, 6), _rand_spinor(h, 7)
    for parity in (0, 1):
        # <a_p, D_{p,1-p} b> = <(D_{p,1-p})^dag a, b>
        lhs = np.vdot(a, oracle_mod.dslash_eo(dims, AP, U, b, parity, kappa, 0))
        rhs = np.vdot(oracle_mod.dslash_eo(dims, AP, U, a, 1 - parity, kappa, 1), b)
        assert abs(lhs - rhs) / abs(lhs) < 1e-14
    lhs = np.vdot(a, oracle_mod.mhat(dims, AP, U, b, kappa, mu, 0))
    rhs = np.vdot(oracle_mod.mhat(dims, AP, U, a, kappa, mu, 1), b)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14
    g5 = lu.GAMMA5
    g5Mg5 = lu.apply_spin(g5, oracle_mod.mhat(dims, AP, U, lu.apply_spin(g5, a), kappa, mu, 0))
    assert lu.rel_err(g5Mg5, oracle_mod.mhat(dims, AP, U, a, kappa, -mu, 1)) < 1e-14


# --------------------------------------------------------------------------- P3 gauge covariance
def _gauge_transform(dims, U, g):
    X = lu.site_coords(dims)
    Up = np.empty_like(U)
    for m in range(4):
        Y = X.copy()
        Y[:, m] = (Y[:, m] + 1) % dims[m]
        gy = g[lu.lex_index(dims, Y)]
        Up[:, m] = np.einsum("sab,sbc,sdc->sad", g, U[:, m], gy.conj())  # g(x) U g(x+mu)^dag
    return Up


@pytest.mark.parametrize("dims", [(4, 2, 2, 4), (4, 4, 4, 4)])
def test_p3_gauge_covariance(oracle_mod, dims):
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    g = gen.su3_haar(V, SEED, gen.STREAM_GTRANS)
    Up = _gauge_transform(dims, U, g)
    psi = _rand_spinor(V, 6)
    lhs = oracle_mod.m_full(dims, AP, Up, lu.apply_colour(g, psi), kappa, mu)
    rhs = lu.apply_colour(g, oracle_mod.m_full(dims, AP, U, psi, kappa, mu))
    assert lu.rel_err(lhs, rhs) < 1e-14
    # even-odd operator: Mhat[U'] g_e psi_e = g_e Mhat[U] psi_e
    ge = lu.to_half(dims, g, 0)
    pe = lu.to_half(dims, psi, 0)
    for dagger in (0, 1):
        lhs = oracle_mod.mhat(dims, AP, Up, lu.apply_colour(ge, pe), kappa, mu, dagger)
        rhs = lu.apply_colour(ge, oracle_mod.mhat(dims, AP, U, pe, kappa, mu, dagger))
        assert lu.rel_err(lhs, rhs) < 1e-14


# --------------------------------------------------------------------------- P4 dense build
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 2)])
def test_p4_dense_build_entry_by_entry(oracle_mod, dims):
    kappa, mu = 0.15, 0.1
    phases = np.exp(1j * np.pi * np.array([0.0, 0.5, 0.0, 1.0]))
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    M = lu.dense_m(dims, phases, U, kappa, mu)
    n = 12 * V
    got = np.empty((n, n), dtype=complex)
    got_dag = np.empty((n, n), dtype=complex)
    for j in range(n):
        e = np.zeros(n, dtype=complex)
        e[j] = 1.0
        got[:, j] = oracle_mod.m_full(dims, phases, U, e.reshape(V, 4, 3), kappa, mu, 0).ravel()
        got_dag[:, j] = oracle_mod.m_full(dims, phases, U, e.reshape(V, 4, 3), kappa, mu, 1).ravel()
    assert np.max(np.abs(got - M)) < 1e-15
    assert np.max(np.abs(got_dag - M.conj().T)) < 1e-15
    # hopping blocks = off-diagonal parity blocks of the dense matrix
    ie, io = lu.dense_index(dims, 0), lu.dense_index(dims, 1)
    x = _rand_spinor(V // 2, 6)
    d_eo = oracle_mod.dslash_eo(dims, phases, U, x, 0, kappa)
    d_oe = oracle_mod.dslash_eo(dims, phases, U, x, 1, kappa)
    assert lu.rel_err(d_eo.ravel(), M[np.ix_(ie, io)] @ x.ravel()) < 1e-14
    assert lu.rel_err(d_oe.ravel(), M[np.ix_(io, ie)] @ x.ravel()) < 1e-14
    # the parity-diagonal blocks are site diagonal: 1 + 2 i kappa mu gamma5
    Mee = M[np.ix_(ie, ie)]
    assert np.allclose(Mee, np.kron(np.eye(V // 2), np.kron(np.eye(4) + 2j * kappa * mu * lu.GAMMA5, np.eye(3))))


# --------------------------------------------------------------------------- P5 paper's identity
def test_p5_twisted_mass_identity(oracle_mod):
    dims = (4, 4, 4, 4)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    psi = _rand_spinor(lu.volume(dims), 6)
    n_mu = np.linalg.norm(oracle_mod.m_full(dims, AP, U, psi, kappa, mu)) ** 2
    n_0 = np.linalg.norm(oracle_mod.m_full(dims, AP, U, psi, kappa, 0.0)) ** 2
    want = n_0 + 4 * kappa ** 2 * mu ** 2 * np.linalg.norm(psi) ** 2
    assert abs(n_mu - want) / want < 1e-14


# --------------------------------------------------------------------------- P6 Schur identity
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 4)])
def test_p6_schur_identity(oracle_mod, dims):
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    S = lu.dense_mhat(dims, AP, U, kappa, mu)
    x = _rand_spinor(lu.volume(dims) // 2, 6)
    assert lu.rel_err(oracle_mod.mhat(dims, AP, U, x, kappa, mu, 0).ravel(), S @ x.ravel()) < 1e-14
    assert lu.rel_err(oracle_mod.mhat(dims, AP, U, x, kappa, mu, 1).ravel(), S.conj().T @ x.ravel()) < 1e-14
    A = S.conj().T @ S
    assert lu.rel_err(oracle_mod.mdagm(dims, AP, U, x, kappa, mu).ravel(), A @ x.ravel()) < 1e-14
    # site-sampled evaluation agrees with the whole-field one
    sites = np.array([0, 3, len(x) - 1, len(x) // 2])
    for dagger in (0, 1):
        whole = oracle_mod.mhat(dims, AP, U, x, kappa, mu, dagger)
        assert lu.rel_err(oracle_mod.mhat_sites(dims, AP, U, x, sites, kappa, mu, dagger), whole[sites]) < 1e-15
    for parity in (0, 1):
        whole = oracle_mod.dslash_eo(dims, AP, U, x, parity, kappa)
        assert np.array_equal(oracle_mod.dslash_eo_sites(dims, AP, U, x, sites, parity, kappa), whole[sites])


def test_p6_full_solve_through_even_odd(oracle_mod):
    # M psi = eta solved via Mhat psi_e = eta_e - D_eo M_oo^-1 eta_o ; psi_o = M_oo^-1 (eta_o - D_oe psi_e)
    dims = (2, 2, 2, 4)
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    eta = _rand_spinor(V, 6)
    M = lu.dense_m(dims, AP, U, kappa, mu)
    psi = np.linalg.solve(M, eta.ravel()).reshape(V, 4, 3)
    pe, po = lu.to_half(dims, psi, 0), lu.to_half(dims, psi, 1)
    ee, eo_ = lu.to_half(dims, eta, 0), lu.to_half(dims, eta, 1)
    Ainv = np.linalg.inv(np.eye(4) + 2j * kappa * mu * lu.GAMMA5)
    rhs = ee - oracle_mod.dslash_eo(dims, AP, U, lu.apply_spin(Ainv, eo_), 0, kappa)
    assert lu.rel_err(oracle_mod.mhat(dims, AP, U, pe, kappa, mu), rhs) < 1e-13
    assert lu.rel_err(lu.apply_spin(Ainv, eo_ - oracle_mod.dslash_eo(dims, AP, U, pe, 1, kappa)), po) < 1e-13


# --------------------------------------------------------------------------- P7 trivial limits
def test_p7_trivial_limits(oracle_mod):
    dims = (4, 4, 4, 4)
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    psi = _rand_spinor(V, 6)
    assert np.array_equal(oracle_mod.m_full(dims, AP, U, psi, 0.0, 0.3), psi)  # kappa = 0 -> identity
    per = np.ones(4, dtype=complex)
    const = np.ones((V, 4, 3), dtype=complex)
    kappa, mu = 0.11, 0.4
    got = oracle_mod.m_full(dims, per, gen.gauge_unit(dims), const, kappa, mu)
    want = lu.apply_spin((1 - 8 * kappa) * np.eye(4) + 2j * kappa * mu * lu.GAMMA5, const)
    assert lu.rel_err(got, want) < 1e-15
    # full operator restricted to parity blocks = eo blocks + diagonal
    pe, po = lu.to_half(dims, psi, 0), lu.to_half(dims, psi, 1)
    full = oracle_mod.m_full(dims, AP, U, psi, kappa, mu)
    A = np.eye(4) + 2j * kappa * mu * lu.GAMMA5
    even = lu.apply_spin(A, pe) + oracle_mod.dslash_eo(dims, AP, U, po, 0, kappa)
    odd = lu.apply_spin(A, po) + oracle_mod.dslash_eo(dims, AP, U, pe, 1, kappa)
    assert lu.rel_err(lu.from_halves(dims, even, odd), full) < 1e-15


# --------------------------------------------------------------------------- P8 CG
def test_p8_cg_against_dense_solve(oracle_mod):
    dims = (2, 2, 2, 4)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    S = lu.dense_mhat(dims, AP, U, kappa, mu)
    A = S.conj().T @ S
    want = np.linalg.solve(A, b.ravel()).reshape(b.shape)
    st, x, iters, rr, rt = oracle_mod.cg_mdagm(dims, AP, U, b, kappa, mu, 1e-12, 500)
    assert st == 0 and 0 < iters < 200
    assert rr <= 1e-12 and rt < 2e-12
    assert lu.rel_err(x, want) < 1e-10
    # lambda_min(M^dag M) >= 4 kappa^2 mu^2 for the full operator (P5) -- and CG's A is positive
    assert np.linalg.eigvalsh(A).min() > 0


def test_p8_cg_iterates_follow_textbook_recurrence(oracle_mod):
    # k steps of the oracle == k steps of Hestenes-Stiefel on the dense matrix, written out in numpy
    dims = (2, 2, 2, 2)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    S = lu.dense_mhat(dims, AP, U, kappa, mu)
    A = S.conj().T @ S
    x = np.zeros(b.size, dtype=complex)
    r = b.ravel().copy()
    p = r.copy()
    rho = np.vdot(r, r).real
    resid = []
    for k in range(1, 6):
        q = A @ p
        alpha = rho / np.vdot(p, q).real
        x = x + alpha * p
        r_new = r - alpha * q
        rho1 = np.vdot(r_new, r_new).real
        resid.append(r_new)
        p = r_new + (rho1 / rho) * p
        r, rho = r_new, rho1
        st, xo, iters, rr, rt = oracle_mod.cg_mdagm(dims, AP, U, b, kappa, mu, 0.0, k)
        assert st == 1 and iters == k
        assert lu.rel_err(xo.ravel(), x) < 1e-12
        assert abs(rr - np.sqrt(rho / np.vdot(b, b).real)) < 1e-12
    # residuals mutually orthogonal
    for i in range(len(resid)):
        for j in range(i):
            assert abs(np.vdot(resid[i], resid[j])) < 1e-10 * np.linalg.norm(resid[i]) * np.linalg.norm(resid[j]) + 1e-12


def test_p8_cg_expected_iteration_counts(oracle_mod):
    # Haar links, kappa=.15, mu=.1 on 4^4 -> ~36 iterations to 1e-10
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    st, x, iters, rr, rt = oracle_mod.cg_mdagm(dims, AP, U, b, 0.15, 0.1, 1e-10, 2000)
    assert st == 0 and 20 <= iters <= 60
    assert rt < 1.05e-10 * 1.5
    assert lu.rel_err(oracle_mod.mdagm(dims, AP, U, x, 0.15, 0.1), b) < 2e-10


# --------------------------------------------------------------------------- P9 BiCGStab
def test_p9_bicgstab_against_dense_solve(oracle_mod):
    dims = (2, 2, 2, 4)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    S = lu.dense_mhat(dims, AP, U, kappa, mu)
    want = np.linalg.solve(S, b.ravel()).reshape(b.shape)
    st, x, iters, rr, rt = oracle_mod.bicgstab_mhat(dims, AP, U, b, kappa, mu, 1e-12, 500)
    assert st == 0 and 0 < iters < 200
    assert rr <= 1e-12 and rt < 5e-12
    assert lu.rel_err(x, want) < 1e-10
    # the true residual is the one of Mhat itself (not of the normal equations)
    assert abs(rt - np.linalg.norm(b.ravel() - S @ x.ravel()) / np.linalg.norm(b)) < 1e-13


def test_p9_bicgstab_iterates_follow_textbook_recurrence(oracle_mod):
    # k steps of the oracle == k steps of van der Vorst's algorithm in its original form
    # (rho_0 = alpha = omega_0 = 1, v_0 = p_0 = 0) written out in numpy on the dense matrix
    dims = (2, 2, 2, 2)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    S = lu.dense_mhat(dims, AP, U, kappa, mu)
    bv = b.ravel()
    x = np.zeros(bv.size, dtype=complex)
    r = bv.copy()
    rhat = bv.copy()
    rho = alpha = omega = 1.0 + 0j
    v = np.zeros_like(x)
    p = np.zeros_like(x)
    for k in range(1, 7):
        rho1 = np.vdot(rhat, r)
        beta = (rho1 / rho) * (alpha / omega)
        p = r + beta * (p - omega * v)
        v = S @ p
        alpha = rho1 / np.vdot(rhat, v)
        s = r - alpha * v
        t = S @ s
        omega = np.vdot(t, s) / np.vdot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho = rho1
        st, xo, iters, rr, rt = oracle_mod.bicgstab_mhat(dims, AP, U, b, kappa, mu, 0.0, k)
        assert st == 1 and iters == k
        assert lu.rel_err(xo.ravel(), x) < 1e-11
        assert abs(rr - np.linalg.norm(r) / np.linalg.norm(bv)) < 1e-11 * max(rr, 1e-3)
        # the recursive residual is the true one up to rounding at this size
        assert abs(rt - np.linalg.norm(bv - S @ x) / np.linalg.norm(bv)) < 1e-12


def test_p9_bicgstab_edge_cases_and_cost(oracle_mod):
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    n = lu.volume(dims) // 2
    b = gen.spinor_gaussian(n, SEED, gen.STREAM_SOURCE)
    st, x, iters, rr, rt = oracle_mod.bicgstab_mhat(dims, AP, U, np.zeros_like(b), 0.15, 0.1, 1e-10, 50)
    assert st == 0 and iters == 0 and np.all(x == 0)
    st, x, iters, rr, rt = oracle_mod.bicgstab_mhat(dims, AP, U, b, 0.15, 0.1, 1e-10, 3)
    assert st == 1 and iters == 3 and rr > 1e-10
    # kappa = 0: Mhat = 1 + 2 i kappa mu gamma5 = 1 -> one iteration
    st, x, iters, rr, rt = oracle_mod.bicgstab_mhat(dims, AP, U, b, 0.0, 0.1, 1e-12, 50)
    assert st == 0 and iters == 1 and lu.rel_err(x, b) < 1e-14
    # two Mhat applications per iteration vs CG's two on the normal equations: BiCGStab needs
    # fewer iterations than CG for the same reduction of its own residual (PAPER.md:94 names both)
    st, x, it_b, rr, rt = oracle_mod.bicgstab_mhat(dims, AP, U, b, 0.15, 0.1, 1e-10, 2000)
    st_c, xc, it_c, rr_c, rt_c = oracle_mod.cg_mdagm(dims, AP, U, b, 0.15, 0.1, 1e-10, 2000)
    assert st == 0 and st_c == 0 and it_b < it_c
    assert lu.rel_err(oracle_mod.mhat(dims, AP, U, x, 0.15, 0.1, 0), b) < 2e-10


# --------------------------------------------------------------------------- P10 fermion force
def _vary_link(U, s, m, a, w):
    U2 = U.copy()
    U2[s, m] = lu.exp_i_w_T(a, w) @ U[s, m]
    return U2


@pytest.mark.parametrize("dims,phases", [((2, 2, 2, 2), AP), ((4, 2, 2, 2), np.exp(1j * np.pi * np.array([0.3, 0.0, 1.0, 0.5])))])
def test_p10_outer_product_force_is_the_derivative_of_the_bilinear(oracle_mod, dims, phases):
    # F^a_mu(x) = d/dw 2 Re [Y^dag M(U_mu(x) -> exp(i w T^a) U_mu(x)) X] for ARBITRARY X, Y,
    # the matrix built densely in numpy (eq. 6); central differences, error O(h^2)
    kappa, h = 0.15, 1e-4
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    X, Y = _rand_spinor(V, 7), _rand_spinor(V, 8)
    F = oracle_mod.fermion_force(dims, phases, U, X, Y, kappa)
    assert F.shape == (V, 4, 8)
    rng = np.random.default_rng(5)
    links = [(0, 0), (V - 1, 3), (1, 1)] + [(int(rng.integers(V)), int(rng.integers(4))) for _ in range(5)]
    # every wrapping hop of the 2-extent directions is among them (x_mu = N_mu - 1 carries the phase)
    f = lambda Uv: 2.0 * np.real(np.vdot(Y.ravel(), lu.dense_m(dims, phases, Uv, kappa, 0.0) @ X.ravel()))
    for s, m in links:
        for a in range(8):
            fd = (f(_vary_link(U, s, m, a, h)) - f(_vary_link(U, s, m, a, -h))) / (2 * h)
            assert abs(F[s, m, a] - fd) < 1e-6 * max(1.0, abs(fd)), (s, m, a, F[s, m, a], fd)
    # the listed-links evaluator agrees with the whole-field one
    ss = np.array([l[0] for l in links]); mm = np.array([l[1] for l in links])
    assert np.array_equal(oracle_mod.fermion_force_links(dims, phases, U, X, Y, ss, mm, kappa), F[ss, mm])


def test_p10_force_is_minus_the_derivative_of_the_action(oracle_mod):
    # S[U] = phi^dag (Mhat^dag Mhat)^-1 phi from the dense Schur complement (numpy only);
    # F^a_mu(x) = -dS/dw (eq. 9) by central differences
    dims = (2, 2, 2, 2)
    kappa, mu, h = 0.15, 0.1, 1e-4
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    phi = gen.spinor_gaussian(V // 2, SEED, gen.STREAM_SOURCE)

    def action(Uv):
        S = lu.dense_mhat(dims, AP, Uv, kappa, mu)
        return np.real(np.vdot(phi.ravel(), np.linalg.solve(S.conj().T @ S, phi.ravel())))

    st, F, iters = oracle_mod.force_tm(dims, AP, U, phi, kappa, mu, 1e-13, 500)
    assert st == 0
    rng = np.random.default_rng(6)
    links = [(0, 3), (V - 1, 3), (5, 0)] + [(int(rng.integers(V)), int(rng.integers(4))) for _ in range(5)]
    for s, m in links:
        for a in range(8):
            fd = -(action(_vary_link(U, s, m, a, h)) - action(_vary_link(U, s, m, a, -h))) / (2 * h)
            assert abs(F[s, m, a] - fd) < 1e-6 * max(1.0, abs(fd)), (s, m, a, F[s, m, a], fd)
    assert np.max(np.abs(F)) > 1e-3      # not trivially zero


def test_p10_force_fields_close_the_even_odd_system(oracle_mod):
    # X_o, Y_o are defined so that (M X)_odd = 0, (M X)_even = Y_e = Mhat X_e, (M^dag Y)_odd = 0
    dims = (4, 2, 2, 4)
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    Xe = _rand_spinor(V // 2, 9)
    X, Y = oracle_mod.force_fields(dims, AP, U, Xe, kappa, mu)
    M = lu.dense_m(dims, AP, U, kappa, mu)
    MX = (M @ X.ravel()).reshape(V, 4, 3)
    MdY = (M.conj().T @ Y.ravel()).reshape(V, 4, 3)
    assert np.array_equal(lu.to_half(dims, X, 0), Xe)
    assert np.linalg.norm(lu.to_half(dims, MX, 1)) < 1e-14 * np.linalg.norm(X)
    assert lu.rel_err(lu.to_half(dims, MX, 0), lu.to_half(dims, Y, 0)) < 1e-14
    assert lu.rel_err(lu.to_half(dims, Y, 0).ravel(), lu.dense_mhat(dims, AP, U, kappa, mu) @ Xe.ravel()) < 1e-14
    assert np.linalg.norm(lu.to_half(dims, MdY, 1)) < 1e-14 * np.linalg.norm(Y)


def test_p10_force_gauge_covariance(oracle_mod):
    # U' = g U g^dag(x+mu), X' = g X, Y' = g Y  =>  F'^a T^a = g(x) (F^a T^a) g(x)^dag
    dims = (4, 2, 2, 4)
    kappa = 0.15
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    g = gen.su3_haar(V, SEED, gen.STREAM_GTRANS)
    X, Y = _rand_spinor(V, 7), _rand_spinor(V, 8)
    F = oracle_mod.fermion_force(dims, AP, U, X, Y, kappa)
    Up = _gauge_transform(dims, U, g)
    Fp = oracle_mod.fermion_force(dims, AP, Up, lu.apply_colour(g, X), lu.apply_colour(g, Y), kappa)
    want = np.einsum("sab,smbc,sdc->smad", g, lu.algebra_matrix(F), g.conj())
    assert lu.rel_err(lu.algebra_matrix(Fp), want) < 1e-14
