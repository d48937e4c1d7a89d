"""Pins of oracle/gauge_oracle.cpp (heatbath / overrelaxation, Fig. 2) against
what the paper and the mathematics fix (-m "not gpu").  Nothing here calls the CUDA path.

  P11 plaquette and staple: the average plaquette against an independent numpy build with
      np.roll (eq. 5 with c_1 = 0), unit and pure-gauge fields, gauge invariance; the staple
      through the exact identity S[U'] - S[U] = -(beta/3) Re tr((U' - U) A), S from the numpy build
  P12 overrelaxation: the action is unchanged, links stay in SU(3), the step is not the identity;
      on a field embedded in the (0,1) SU(2) subgroup the first subgroup step equals the textbook
      formula U' = V^dag U^dag V^dag, V = staple block / sqrt(det); one subgroup step twice = identity
  P13 heatbath: Kennedy-Pendleton samples against <g0> = I_2(lambda) / I_1(lambda) and
      <g0^2> (numerical integral), isotropy of the direction, counters of the generator against
      lqcd_inputs; strong-coupling plaquette <P> = beta/18 + beta^2/216 on a thermalised 4^4 field;
      beta -> infinity drives a cold start nowhere (links stay at 1 up to O(1/beta))
"""
import numpy as np
import pytest

import lattice_util as lu
import lqcd_inputs as gen

SEED = gen.BASE_SEED


# --------------------------------------------------------------------------- numpy reference
def _field(dims, U):
    """(V,4,3,3) lex-ordered -> (N3,N2,N1,N0,4,3,3)."""
    N = [int(n) for n in dims]
    return U.reshape(N[3], N[2], N[1], N[0], 4, 3, 3)


def _shift(F, mu):
    """F(x) -> F(x + mu): axis of direction mu is 3 - mu in the reshaped field."""
    return np.roll(F, -1, axis=3 - mu)


def np_plaquette(dims, U):
    F = _field(dims, U)
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Umu, Unu = F[..., mu, :, :], F[..., nu, :, :]
            P = Umu @ _shift(Unu, mu) @ np.conj(np.swapaxes(_shift(Umu, nu), -1, -2)) @ np.conj(np.swapaxes(Unu, -1, -2))
            tot += np.trace(P, axis1=-2, axis2=-1).real.sum() / 3.0
    return tot / (6 * lu.volume(dims))


def np_action(dims, U, beta):
    return beta * 6 * lu.volume(dims) * (1.0 - np_plaquette(dims, U))


def _is_su3(M, tol):
    M = M.reshape(-1, 3, 3)
    eye = np.eye(3)
    unit = np.abs(M @ np.conj(np.swapaxes(M, 1, 2)) - eye).max()
    det = np.abs(np.linalg.det(M) - 1.0).max()
    return unit < tol and det < tol


def _gauge_transform(dims, U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag."""
    F, G = _field(dims, U), g.reshape(tuple(int(n) for n in dims[::-1]) + (3, 3))
    out = np.empty_like(F)
    for mu in range(4):
        out[..., mu, :, :] = G @ F[..., mu, :, :] @ np.conj(np.swapaxes(_shift(G, mu), -1, -2))
    return out.reshape(U.shape)


# --------------------------------------------------------------------------- P11
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4), (2, 2, 2, 2)])
def test_p11_plaquette_matches_numpy_build(oracle_mod, dims):
    for U in (gen.gauge_haar(dims), gen.gauge_near_identity(dims, SEED, 0.3)):
        assert abs(oracle_mod.plaquette(dims, U) - np_plaquette(dims, U)) < 1e-14


def test_p11_plaquette_unit_and_pure_gauge(oracle_mod):
    dims = (4, 4, 2, 4)
    V = lu.volume(dims)
    U1 = gen.gauge_unit(dims)
    assert oracle_mod.plaquette(dims, U1) == 1.0
    g = gen.su3_haar(V, SEED, gen.STREAM_GTRANS)
    assert abs(oracle_mod.plaquette(dims, _gauge_transform(dims, U1, g)) - 1.0) < 1e-14
    U = gen.gauge_near_identity(dims, SEED, 0.4)
    assert abs(oracle_mod.plaquette(dims, _gauge_transform(dims, U, g)) - oracle_mod.plaquette(dims, U)) < 1e-14


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 2, 6), (2, 2, 2, 2)])
def test_p11_staple_is_the_derivative_of_the_action(oracle_mod, dims):
    """S is linear in each link: S[U'] - S[U] = -(beta/3) Re tr((U' - U) A) exactly, for ANY 3x3 U'.
    A transposed product, a missing dagger, a wrong neighbour or a missing staple breaks it."""
    beta = 5.7
    U = gen.gauge_haar(dims)
    V = lu.volume(dims)
    S0 = np_action(dims, U, beta)
    rng = np.random.default_rng(7)
    for site in rng.integers(0, V, 6):
        for mu in range(4):
            A = oracle_mod.staple(dims, U, site, mu)
            Un = U.copy()
            Un[site, mu] = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))   # not even unitary
            dS = np_action(dims, Un, beta) - S0
            want = -(beta / 3.0) * np.trace((Un[site, mu] - U[site, mu]) @ A).real
            assert abs(dS - want) < 1e-9 * max(1.0, abs(want)), (site, mu, dS, want)


def test_p11_staple_unit_field(oracle_mod):
    A = oracle_mod.staple((4, 4, 4, 4), gen.gauge_unit((4, 4, 4, 4)), 17, 2)
    assert np.array_equal(A, 6.0 * np.eye(3))


# --------------------------------------------------------------------------- P12
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 4, 2)])
def test_p12_overrelax_keeps_action_and_group(oracle_mod, dims):
    U = gen.gauge_near_identity(dims, SEED, 0.5)
    Un = oracle_mod.gauge_sweep(dims, U, 1, 0.0, SEED, 50)
    assert abs(np_plaquette(dims, Un) - np_plaquette(dims, U)) < 1e-13
    assert _is_su3(Un, 1e-13)
    assert np.abs(Un - U).reshape(-1, 9).max(axis=1).min() > 1e-3      # every link moved
    # and sub-sweep by sub-sweep, link by link: Re tr(U A) is unchanged for each updated link
    V = lu.volume(dims)
    sites = np.arange(V)
    for mu in (0, 3):
        new = oracle_mod.update_links(dims, U, sites, np.full(V, mu), 1, 0.0, SEED, 50)
        for s in (0, 5, V - 1):
            A = oracle_mod.staple(dims, U, s, mu)
            assert abs(np.trace(new[s] @ A).real - np.trace(U[s, mu] @ A).real) < 1e-12


def _embed01(M2):
    out = np.zeros(M2.shape[:-2] + (3, 3), dtype=np.complex128)
    out[..., :2, :2] = M2
    out[..., 2, 2] = 1.0
    return out


def test_p12_overrelax_reduces_to_textbook_su2(oracle_mod):
    """All links in the (0,1) subgroup: the first subgroup step must give U' = V^dag U^dag V^dag with
    V = (2x2 block of the staple sum) / sqrt(det) -- the SU(2) overrelaxation of [19]."""
    dims = (4, 4, 4, 4)
    V = lu.volume(dims)
    H = gen.su3_haar(4 * V, SEED, 9)[:, :2, :2]
    # SU(2) from the top-left block: m = a0 + i a.sigma built from the block's SU(2)-proportional part
    a0 = (H[:, 0, 0] + np.conj(H[:, 1, 1])) / 2
    b0 = (H[:, 0, 1] - np.conj(H[:, 1, 0])) / 2
    nrm = np.sqrt(np.abs(a0) ** 2 + np.abs(b0) ** 2)
    a0, b0 = a0 / nrm, b0 / nrm
    S2 = np.stack([np.stack([a0, b0], -1), np.stack([-np.conj(b0), np.conj(a0)], -1)], -2)
    U = _embed01(S2).reshape(V, 4, 3, 3)
    assert _is_su3(U, 1e-14)
    sites = np.array([0, 3, 77, V - 1])
    for mu in range(4):
        new = oracle_mod.update_links(dims, U, sites, np.full(len(sites), mu), 1, 0.0, SEED, 1, subgroups=1)
        for k, s in enumerate(sites):
            A2 = oracle_mod.staple(dims, U, s, mu)[:2, :2]          # a sum of SU(2) matrices: k * SU(2)
            Vm = A2 / np.sqrt(np.linalg.det(A2).real)
            u = U[s, mu][:2, :2]
            want = Vm.conj().T @ u.conj().T @ Vm.conj().T
            assert np.abs(new[k] - _embed01(want)).max() < 1e-13


def test_p12_single_subgroup_step_is_an_involution(oracle_mod):
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims)
    sites, mus = np.array([1, 100, 200]), np.array([0, 1, 3], dtype=np.int32)
    for sub in (1, 2, 4):
        once = oracle_mod.update_links(dims, U, sites, mus, 1, 0.0, SEED, 1, subgroups=sub)
        U2 = U.copy()
        U2[sites, mus] = once
        twice = oracle_mod.update_links(dims, U2, sites, mus, 1, 0.0, SEED, 1, subgroups=sub)
        assert np.abs(once - U[sites, mus]).max() > 1e-2
        assert np.abs(twice - U[sites, mus]).max() < 1e-13
        # G19: step i acts from the left in the subgroup (0,1), (1,2), (0,2): the third row is untouched
        spectator = {1: 2, 2: 0, 4: 1}[sub]
        assert np.array_equal(once[:, spectator, :], U[sites, mus][:, spectator, :])
        assert np.abs(once - U[sites, mus]).max(axis=(0, 2))[[r for r in range(3) if r != spectator]].min() > 1e-3


# --------------------------------------------------------------------------- P13
def test_p13_generator_counters_match_the_input_recipe(oracle_mod):
    """G21: the heatbath's uniforms are lqcd_inputs' counter-based stream with stream = tag.  With
    lambda huge every first attempt is accepted (delta ~ 0), so g = (1 - delta, direction from r5, r6)
    exposes r1..r3 (through delta) and r5, r6 directly."""
    lam, tag, n = 1e9, 77, 64
    g, att = oracle_mod.kp_samples(lam, SEED, tag, n)
    assert np.all(att == 1)
    base = np.arange(n, dtype=np.uint64) * np.uint64(4 * 33)
    r = [gen._uniform(SEED, tag, base + np.uint64(j)) for j in range(3)]
    delta = -(np.log(r[0]) + np.cos(2 * np.pi * r[1]) ** 2 * np.log(r[2])) / lam
    assert np.allclose(1.0 - g[:, 0], delta, rtol=1e-6, atol=0)
    r5 = gen._uniform(SEED, tag, base + np.uint64(4 * 32))
    r6 = gen._uniform(SEED, tag, base + np.uint64(4 * 32 + 1))
    rad = np.sqrt(1.0 - g[:, 0] ** 2)
    assert np.allclose(g[:, 3], rad * (2 * r5 - 1), rtol=1e-12, atol=1e-18)
    st = np.sqrt(1 - (2 * r5 - 1) ** 2)
    assert np.allclose(g[:, 1], rad * st * np.cos(2 * np.pi * r6), rtol=1e-9, atol=1e-18)
    assert np.allclose(g[:, 2], rad * st * np.sin(2 * np.pi * r6), rtol=1e-9, atol=1e-18)


@pytest.mark.parametrize("lam", [1.5, 6.0, 20.0])
def test_p13_kennedy_pendleton_distribution(oracle_mod, lam):
    """g0 has density sqrt(1 - g0^2) exp(lam g0) on [-1, 1]: <g0> = I_2(lam)/I_1(lam) (closed form),
    <g0^2> by quadrature; the direction is uniform on the sphere."""
    from scipy.special import ive
    n = 200000
    g, att = oracle_mod.kp_samples(lam, SEED, 5, n)
    ok = att > 0
    assert ok.mean() > (0.9 if lam >= 6 else 0.5)       # 32 attempts: failures are rare even at lam = 1.5
    g = g[ok]
    m = len(g)
    assert np.allclose(np.sum(g * g, axis=1), 1.0, atol=1e-14)
    mean_exact = ive(2, lam) / ive(1, lam)
    x = np.linspace(-1, 1, 400001)
    w = np.sqrt(1 - x * x) * np.exp(lam * (x - 1))
    m2_exact = np.sum(w * x * x) / np.sum(w)
    var = m2_exact - mean_exact ** 2
    assert abs(g[:, 0].mean() - mean_exact) < 5 * np.sqrt(var / m)
    assert abs((g[:, 0] ** 2).mean() - m2_exact) < 5 * np.sqrt(1.0 / m) * max(var, 0.05)
    # isotropy: components 1..3 have zero mean and equal second moments (1 - <g0^2>)/3
    s2 = (1 - m2_exact) / 3
    for c in (1, 2, 3):
        assert abs(g[:, c].mean()) < 5 * np.sqrt(s2 / m)
        assert abs((g[:, c] ** 2).mean() - s2) < 6 * s2 * np.sqrt(2.0 / m)
    # acceptance: mean number of attempts = 1 / P(accept) with P = E[sqrt(1 - delta/2)] under the
    # proposal density ~ sqrt(delta) exp(-lam delta): a loose closed-form-free bound
    assert att[ok].mean() < (1.1 if lam >= 20 else 1.5 if lam >= 6 else 4.0)


def test_p13_strong_coupling_plaquette(oracle_mod):
    """<P> = beta/18 + beta^2/216 + O(beta^4) for SU(3) with the Wilson action (strong-coupling
    expansion): pins lambda = 2 beta k / 3 and the heatbath as a whole.  4^4, hot start."""
    dims, beta = (4, 4, 4, 4), 1.2
    U = gen.gauge_haar(dims)
    vals = []
    for sweep in range(60):
        U = oracle_mod.gauge_sweep(dims, U, 0, beta, SEED, 1000 + sweep)
        if sweep >= 10:
            vals.append(np_plaquette(dims, U))
    assert _is_su3(U, 1e-12)
    want = beta / 18 + beta ** 2 / 216
    err = np.std(vals) / np.sqrt(len(vals)) * 2.0    # mild autocorrelation allowance
    assert abs(np.mean(vals) - want) < max(4 * err, 0.0025), (np.mean(vals), want, err)
    # and it is far from what a wrong lambda would give (beta_eff off by 3/2 or 2)
    assert abs(np.mean(vals) - 1.5 * beta / 18) > 0.01


def test_p13_weak_coupling_keeps_a_cold_start_cold(oracle_mod):
    """beta -> infinity: the Boltzmann weight pins every link to the minimum of the action; from a
    cold start 1 - <P> = O(1/beta) (lowest order: 1 - <P> ~ 2/beta for SU(3) in 4 dimensions)."""
    dims, beta = (4, 4, 4, 4), 600.0
    U = gen.gauge_unit(dims)
    for sweep in range(12):
        U = oracle_mod.gauge_sweep(dims, U, 0, beta, SEED, 2000 + sweep)
    p = np_plaquette(dims, U)
    assert 0.5 * 2 / beta < 1 - p < 1.5 * 2 / beta, (1 - p, 2 / beta)


def test_p13_heatbath_then_overrelax_compose(oracle_mod):
    """A heatbath sweep followed by overrelaxation sweeps keeps SU(3) and the action of the heatbath output."""
    dims = (4, 4, 4, 4)
    U = oracle_mod.gauge_sweep(dims, gen.gauge_haar(dims), 0, 5.7, SEED, 1)
    p = np_plaquette(dims, U)
    for k in range(4):
        U = oracle_mod.gauge_sweep(dims, U, 1, 5.7, SEED, 2 + k)
    assert abs(np_plaquette(dims, U) - p) < 1e-13
    assert _is_su3(U, 1e-13)


def test_subsweeps_compose_to_a_sweep(oracle_mod):
    dims = (4, 4, 2, 4)
    U = gen.gauge_near_identity(dims, SEED, 0.4)
    for mode in (0, 1):
        want = oracle_mod.gauge_sweep(dims, U, mode, 5.5, SEED, 9)
        got = U
        for mu in range(4):
            for par in (0, 1):
                got = oracle_mod.gauge_subsweep(dims, got, mu, par, mode, 5.5, SEED, 9)
        assert np.array_equal(got, want)
        # a sub-sweep touches only its own links, and equals the link-wise evaluator on them
        one = oracle_mod.gauge_subsweep(dims, U, 2, 1, mode, 5.5, SEED, 9)
        par = lu.site_parity(dims)
        mask = np.zeros((lu.volume(dims), 4), dtype=bool)
        mask[par == 1, 2] = True
        assert np.array_equal(one[~mask], U[~mask])
        sites = np.nonzero(par == 1)[0]
        assert np.array_equal(one[sites, 2], oracle_mod.update_links(dims, U, sites, np.full(len(sites), 2), mode, 5.5, SEED, 9))
