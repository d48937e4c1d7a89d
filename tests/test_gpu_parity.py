"""Parity of the CUDA path (through the C ABI) against the CPU oracle (-m gpu).

Bar (BASELINE.json north_star): relative L2 error <= 1e-13 in double, <= 1e-5 in
single (oracle fed the float-rounded inputs), on the same seeded inputs.  CG:
reading G14 of DESIGN.md (solution unique, iterates not bit-reproducible).
"""
import numpy as np
import pytest

import lattice_util as lu
import lqcd_inputs as gen

pytestmark = pytest.mark.gpu

TOL_D = 1e-13
TOL_S = 1e-5
AP = gen.antiperiodic_t()
SEED = gen.BASE_SEED


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1209_5942_b200.binding as b
    return b


class Lat:
    """One initialised lattice + uploaded gauge field under a given format."""

    def __init__(self, B, dims, phases, U, precision=0, recon=18):
        self.B, self.dims, self.phases, self.U = B, dims, np.asarray(phases, dtype=complex), U
        self.precision, self.recon = precision, recon
        B.lqcd_init(dims, self.phases)
        B.lqcd_set_format(precision, recon)
        B.lqcd_set_stream()
        self.g = B.upload_gauge(U)

    def dslash(self, x, parity, kappa):
        s = self.B.upload_spinor(x, 1 - parity)
        o = self.B.alloc_spinor()
        self.B.lqcd_dslash_eo(self.g, s, o, parity, kappa)
        return self.B.download_spinor(o, parity)

    def mtm(self, x, kappa, mu, dagger):
        s = self.B.upload_spinor(x, 0)
        o = self.B.alloc_spinor()
        self.B.lqcd_mtm(self.g, s, o, kappa, mu, dagger)
        return self.B.download_spinor(o, 0)

    def cg(self, b, kappa, mu, tol, maxit):
        s = self.B.upload_spinor(b, 0)
        x = self.B.alloc_spinor()
        st = self.B.lqcd_cg_mdagm(self.g, s, x, kappa, mu, tol, maxit)
        return st, self.B.download_spinor(x, 0), self.B.lqcd_cg_stats()

    def bicgstab(self, b, kappa, mu, tol, maxit):
        s = self.B.upload_spinor(b, 0)
        x = self.B.alloc_spinor()
        st = self.B.lqcd_bicgstab_mhat(self.g, s, x, kappa, mu, tol, maxit)
        return st, self.B.download_spinor(x, 0), self.B.lqcd_cg_stats()


def _round_inputs(U, x, precision):
    if precision == 0:
        return U, x
    return U.astype(np.complex64).astype(np.complex128), x.astype(np.complex64).astype(np.complex128)


GENERIC_PH = np.exp(1j * np.pi * np.array([0.3, 0.0, 1.0, 0.5]))


# --------------------------------------------------------------------------- config 1 and friends
@pytest.mark.parametrize("dims,phases", [
    ((4, 4, 4, 4), AP),            # BASELINE config 1
    ((2, 2, 2, 2), AP),            # N_mu = 2: both hops reach the same site (G8)
    ((2, 2, 2, 2), GENERIC_PH),
    ((4, 6, 2, 8), GENERIC_PH),    # unequal extents, complex phases on every wrap
    ((6, 4, 10, 4), AP),           # Vh = 480: ragged tail for 128-thread blocks
    ((8, 8, 8, 16), AP),           # BASELINE config 2 lattice: several blocks
])
def test_dslash_eo_matches_oracle(B, oracle_mod, dims, phases):
    kappa = 0.15
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    L = Lat(B, dims, phases, U)
    for parity in (0, 1):
        got = L.dslash(x, parity, kappa)
        want = oracle_mod.dslash_eo(dims, phases, U, x, parity, kappa)
        assert lu.rel_err(got, want) <= TOL_D
        # element by element too: no single site may be off
        assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))


@pytest.mark.parametrize("dims,phases", [((4, 4, 4, 4), AP), ((2, 2, 2, 2), GENERIC_PH),
                                         ((4, 6, 2, 8), GENERIC_PH), ((8, 8, 8, 16), AP)])
@pytest.mark.parametrize("dagger", [0, 1])
def test_mtm_matches_oracle(B, oracle_mod, dims, phases, dagger):
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    L = Lat(B, dims, phases, U)
    got = L.mtm(x, kappa, mu, dagger)
    want = oracle_mod.mhat(dims, phases, U, x, kappa, mu, dagger)
    assert lu.rel_err(got, want) <= TOL_D


@pytest.mark.parametrize("block", [32, 64, 96, 128])
def test_block_sizes(B, oracle_mod, block):
    dims = (6, 4, 10, 4)
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    L = Lat(B, dims, AP, U)
    B.lqcd_set_block_size(block)
    got = L.mtm(x, 0.15, 0.1, 0)
    assert lu.rel_err(got, oracle_mod.mhat(dims, AP, U, x, 0.15, 0.1, 0)) <= TOL_D


def test_pack_unpack_roundtrip_is_exact(B):
    dims = (4, 6, 2, 8)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    B.lqcd_init(dims, AP)
    for parity in (0, 1):
        s = B.upload_spinor(x, parity)
        assert np.array_equal(B.download_spinor(s, parity), x)
    B.lqcd_set_format(B.LQCD_SINGLE, 18)
    s = B.upload_spinor(x, 0)
    assert np.array_equal(B.download_spinor(s, 0), x.astype(np.complex64).astype(np.complex128))


# --------------------------------------------------------------------------- config 2: invariances on GPU output
def test_config2_gamma5_hermiticity_and_gauge_covariance_on_gpu(B, oracle_mod):
    dims = (8, 8, 8, 16)
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(V // 2, SEED)
    y = gen.spinor_gaussian(V // 2, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    Mx, Mdy = L.mtm(x, kappa, mu, 0), L.mtm(y, kappa, mu, 1)
    for dagger, got in ((0, Mx), (1, Mdy)):
        want = oracle_mod.mhat(dims, AP, U, x if dagger == 0 else y, kappa, mu, dagger)
        assert lu.rel_err(got, want) <= TOL_D
    # <y, M x> = <M^dag y, x>
    lhs, rhs = np.vdot(y, Mx), np.vdot(Mdy, x)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # gamma5 Mhat(mu) gamma5 = Mhat(-mu)^dag
    g5 = lu.GAMMA5
    lhs = lu.apply_spin(g5, L.mtm(lu.apply_spin(g5, x), kappa, mu, 0))
    assert lu.rel_err(lhs, L.mtm(x, kappa, -mu, 1)) < 1e-13
    # gauge covariance: Mhat[U'] g x = g Mhat[U] x
    g = gen.su3_haar(V, SEED, gen.STREAM_GTRANS)
    X = lu.site_coords(dims)
    Up = np.empty_like(U)
    for m in range(4):
        Y = X.copy()
        Y[:, m] = (Y[:, m] + 1) % dims[m]
        Up[:, m] = np.einsum("sab,sbc,sdc->sad", g, U[:, m], g[lu.lex_index(dims, Y)].conj())
    ge = lu.to_half(dims, g, 0)
    Lp = Lat(B, dims, AP, Up)
    assert lu.rel_err(Lp.mtm(lu.apply_colour(ge, x), kappa, mu, 0), lu.apply_colour(ge, Mx)) < 1e-13


def test_free_field_closed_form_on_gpu(B):
    dims = (4, 4, 6, 8)
    kappa, mu = 0.137, 0.21
    p = lu.momentum(dims, AP, (1, 3, 2, 5))
    rng = np.random.default_rng(3)
    u = rng.normal(size=12) + 1j * rng.normal(size=12)
    psi = lu.plane_wave(dims, p, u)
    h = lu.free_h(p, kappa)
    A = np.eye(4) + 2j * kappa * mu * lu.GAMMA5
    L = Lat(B, dims, AP, gen.gauge_unit(dims))
    got = L.mtm(lu.to_half(dims, psi, 0), kappa, mu, 0)
    want = lu.to_half(dims, lu.apply_spin(A - h @ np.linalg.inv(A) @ h, psi), 0)
    assert lu.rel_err(got, want) < 1e-13


# --------------------------------------------------------------------------- storage variants (config 5 formats)
@pytest.mark.parametrize("precision,recon,tol", [(0, 12, TOL_D), (1, 18, TOL_S), (1, 12, TOL_S)])
@pytest.mark.parametrize("dims,phases", [((4, 4, 4, 4), AP), ((4, 6, 2, 8), GENERIC_PH), ((8, 8, 8, 16), AP)])
def test_storage_variants(B, oracle_mod, precision, recon, tol, dims, phases):
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    Ur, xr = _round_inputs(U, x, precision)
    L = Lat(B, dims, phases, U, precision, recon)
    for parity in (0, 1):
        got = L.dslash(x, parity, kappa)
        assert lu.rel_err(got, oracle_mod.dslash_eo(dims, phases, Ur, xr, parity, kappa)) <= tol
    for dagger in (0, 1):
        got = L.mtm(x, kappa, mu, dagger)
        assert lu.rel_err(got, oracle_mod.mhat(dims, phases, Ur, xr, kappa, mu, dagger)) <= tol


def test_near_identity_links_config3_small(B, oracle_mod):
    dims = (8, 8, 8, 8)
    kappa, mu = 0.16, 0.05
    U = gen.gauge_near_identity(dims, SEED, 0.3)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    for recon in (18, 12):
        L = Lat(B, dims, AP, U, 0, recon)
        assert lu.rel_err(L.mtm(x, kappa, mu, 0), oracle_mod.mhat(dims, AP, U, x, kappa, mu, 0)) <= TOL_D


# --------------------------------------------------------------------------- CG
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 16)])
def test_cg_matches_oracle(B, oracle_mod, dims):
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    st, x, (iters, rr, rt) = L.cg(b, kappa, mu, tol, 2000)
    st_o, x_o, it_o, rr_o, rt_o = oracle_mod.cg_mdagm(dims, AP, U, b, kappa, mu, tol, 2000)
    assert st == 0 and st_o == 0
    assert abs(iters - it_o) <= 2
    assert rr <= tol
    # true residual of the GPU's x, evaluated by the ORACLE's operator
    r = b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)
    true_rel = np.linalg.norm(r) / np.linalg.norm(b)
    assert true_rel <= 1.05 * tol
    assert abs(rt - true_rel) <= 0.05 * tol          # the library's own true residual agrees
    assert lu.rel_err(x, x_o) <= 10 * 5.0 * tol       # 10 * sqrt(cond) * tol, cond ~ 10-25 (G14)


@pytest.mark.parametrize("k", [1, 3])
def test_cg_k_iterations_from_identical_state(B, oracle_mod, k):
    dims = (8, 8, 8, 16)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    st, x, (iters, rr, rt) = L.cg(b, kappa, mu, 0.0, k)
    st_o, x_o, it_o, rr_o, rt_o = oracle_mod.cg_mdagm(dims, AP, U, b, kappa, mu, 0.0, k)
    assert st == 1 and st_o == 1 and iters == k == it_o
    assert lu.rel_err(x, x_o) <= 1e-13 * (4 if k > 1 else 1)
    assert abs(rr - rr_o) <= 1e-12 * rr_o
    assert abs(rt - rt_o) <= 1e-10 * rt_o


def test_cg_edge_cases(B):
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    L = Lat(B, dims, AP, U)
    zero = np.zeros((lu.volume(dims) // 2, 4, 3), dtype=complex)
    st, x, (iters, rr, rt) = L.cg(zero, 0.15, 0.1, 1e-10, 50)     # b = 0 -> x = 0 at once
    assert st == 0 and iters == 0 and np.all(x == 0)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    st, x, (iters, rr, rt) = L.cg(b, 0.15, 0.1, 1e-10, 5)         # maxit too small
    assert st == B.LQCD_NOT_CONVERGED and iters == 5 and rr > 1e-10
    st, x, (iters, rr, rt) = L.cg(b, 0.0, 0.1, 1e-12, 50)         # kappa = 0: A = 1, one step
    assert st == 0 and iters == 1 and lu.rel_err(x, b) < 1e-14


def test_cg_single_precision_converges_loosely(B, oracle_mod):
    dims = (8, 8, 8, 16)
    kappa, mu, tol = 0.15, 0.1, 1e-5
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    for recon in (18, 12):
        L = Lat(B, dims, AP, U, 1, recon)
        st, x, (iters, rr, rt) = L.cg(b, kappa, mu, tol, 500)
        assert st == 0 and rr <= tol
        r = b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)
        assert np.linalg.norm(r) / np.linalg.norm(b) <= 20 * tol


# --------------------------------------------------------------------------- BiCGStab on Mhat
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 10, 4), (8, 8, 8, 16)])
def test_bicgstab_matches_oracle(B, oracle_mod, dims):
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    st, x, (iters, rr, rt) = L.bicgstab(b, kappa, mu, tol, 2000)
    st_o, x_o, it_o, rr_o, rt_o = oracle_mod.bicgstab_mhat(dims, AP, U, b, kappa, mu, tol, 2000)
    assert st == 0 and st_o == 0
    assert abs(iters - it_o) <= 2          # BiCGStab's iterates are sensitive to rounding (G14)
    assert rr <= tol
    # true residual of the GPU's x under the ORACLE's Mhat
    true_rel = np.linalg.norm(b - oracle_mod.mhat(dims, AP, U, x, kappa, mu, 0)) / np.linalg.norm(b)
    assert true_rel <= 1.05 * tol
    assert abs(rt - true_rel) <= 0.05 * tol
    assert lu.rel_err(x, x_o) <= 10 * 5.0 * tol


@pytest.mark.parametrize("k", [1, 3])
def test_bicgstab_k_iterations_from_identical_state(B, oracle_mod, k):
    dims = (8, 8, 8, 16)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    st, x, (iters, rr, rt) = L.bicgstab(b, kappa, mu, 0.0, k)
    st_o, x_o, it_o, rr_o, rt_o = oracle_mod.bicgstab_mhat(dims, AP, U, b, kappa, mu, 0.0, k)
    assert st == 1 and st_o == 1 and iters == k == it_o
    assert lu.rel_err(x, x_o) <= 1e-13 * (10 if k > 1 else 1)
    assert abs(rr - rr_o) <= 1e-11 * rr_o
    assert abs(rt - rt_o) <= 1e-10 * rt_o


def test_bicgstab_edge_cases_and_formats(B, oracle_mod):
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    L = Lat(B, dims, AP, U)
    n = lu.volume(dims) // 2
    zero = np.zeros((n, 4, 3), dtype=complex)
    st, x, (iters, rr, rt) = L.bicgstab(zero, 0.15, 0.1, 1e-10, 50)
    assert st == 0 and iters == 0 and np.all(x == 0)
    b = gen.spinor_gaussian(n, SEED, gen.STREAM_SOURCE)
    st, x, (iters, rr, rt) = L.bicgstab(b, 0.15, 0.1, 1e-10, 3)
    assert st == B.LQCD_NOT_CONVERGED and iters == 3 and rr > 1e-10
    st, x, (iters, rr, rt) = L.bicgstab(b, 0.0, 0.1, 1e-12, 50)      # kappa = 0: Mhat = 1
    assert st == 0 and iters == 1 and lu.rel_err(x, b) < 1e-14
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_bicgstab_mhat(L.g, 0, L.g, 0.1, 0.1, 1e-8, 10)
    assert e.value.status == B.LQCD_BAD_ARG
    # single precision and 12-real links converge to what single precision allows
    dims = (8, 8, 8, 16)
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    for precision, recon, tol in ((1, 18, 1e-5), (1, 12, 1e-5), (0, 12, 1e-10)):
        L = Lat(B, dims, AP, U, precision, recon)
        st, x, (iters, rr, rt) = L.bicgstab(b, 0.15, 0.1, tol, 500)
        assert st == 0 and rr <= tol
        true_rel = np.linalg.norm(b - oracle_mod.mhat(dims, AP, U, x, 0.15, 0.1, 0)) / np.linalg.norm(b)
        assert true_rel <= (20 if precision else 1.05) * tol


# --------------------------------------------------------------------------- ABI behaviour
def test_error_codes(B):
    import torch
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_init((4, 4, 5, 4), AP)
    assert e.value.status == B.LQCD_BAD_DIMS
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_init((4, 4, 4, 4), [1, 1, 1, 2.0])
    assert e.value.status == B.LQCD_BAD_DIMS
    B.lqcd_init((4, 4, 4, 4), AP)
    g, s, o = B.alloc_gauge(), B.alloc_spinor(), B.alloc_spinor()
    for call in (lambda: B.lqcd_dslash_eo(g, s, o, 2, 0.1),
                 lambda: B.lqcd_dslash_eo(g, s, s, 0, 0.1),
                 lambda: B.lqcd_dslash_eo(g, 0, o, 0, 0.1),
                 lambda: B.lqcd_dslash_eo(g, s, o, 0, float("nan")),
                 lambda: B.lqcd_mtm(g, s, o, 0.1, float("inf"), 0),
                 lambda: B.lqcd_cg_mdagm(g, s, o, 0.1, 0.1, 1e-8, 0),
                 lambda: B.lqcd_set_format(2, 18),
                 lambda: B.lqcd_set_format(0, 8)):
        with pytest.raises(B.LqcdError) as e:
            call()
        assert e.value.status == B.LQCD_BAD_ARG
    assert B.lqcd_gauge_bytes() == 256 * 576 and B.lqcd_spinor_bytes() == 128 * 192
    B.lqcd_set_format(B.LQCD_SINGLE, 12)
    assert B.lqcd_gauge_bytes() == 256 * 192 and B.lqcd_spinor_bytes() == 128 * 96
    torch.cuda.synchronize()


def test_host_entry_points(B, oracle_mod):
    dims = (8, 8, 8, 16)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
    B.lqcd_init(dims, AP)
    out = np.empty_like(x)
    n0 = B.lqcd_launch_count()
    B.lqcd_mtm_host(U, x, out, kappa, mu, 0)
    assert B.lqcd_launch_count() - n0 == 5      # 2 pack + 2 hopping + 1 unpack
    assert lu.rel_err(out, oracle_mod.mhat(dims, AP, U, x, kappa, mu, 0)) <= TOL_D
    sol = np.empty_like(x)
    st = B.lqcd_cg_mdagm_host(U, x, sol, kappa, mu, 1e-10, 1000)
    assert st == 0
    assert lu.rel_err(oracle_mod.mdagm(dims, AP, U, sol, kappa, mu), x) <= 1.05e-10


# --------------------------------------------------------------------------- full sizes, sampled
def _sample_sites(n, count, seed):
    rng = np.random.default_rng(seed)
    s = rng.integers(0, n, size=count)
    s[:4] = [0, 1, n - 1, n // 2]       # corners: wraps in every direction
    return np.unique(s)


@pytest.mark.parametrize("dims,near_id,kappa,mu", [
    ((16, 16, 16, 32), True, 0.16, 0.05),     # config 3
    ((24, 24, 24, 48), False, 0.15, 0.1),     # config 4 lattice
    ((32, 32, 32, 64), False, 0.15, 0.1),     # config 5 (bench workload), bench launch configuration
])
def test_full_size_sampled_sites(B, oracle_mod, dims, near_id, kappa, mu):
    h = lu.volume(dims) // 2
    if near_id:
        U, x = gen.gauge_near_identity(dims, SEED, 0.3), gen.spinor_gaussian(h, SEED)
    else:
        U, x, _ = _cached_fields(dims)
    sites = _sample_sites(h, 300, 17)
    L = Lat(B, dims, AP, U)
    for parity in (0, 1):
        got = L.dslash(x, parity, kappa)[sites]
        want = oracle_mod.dslash_eo_sites(dims, AP, U, x, sites, parity, kappa)
        assert lu.rel_err(got, want) <= TOL_D
    for dagger in (0, 1):
        got = L.mtm(x, kappa, mu, dagger)
        want = oracle_mod.mhat_sites(dims, AP, U, x, sites, kappa, mu, dagger)
        assert lu.rel_err(got[sites], want) <= TOL_D
        assert np.all(np.isfinite(got))
    # a property that holds at any size: <x, Mhat^dag Mhat x> = |Mhat x|^2 > 0
    Mx = L.mtm(x, kappa, mu, 0)
    MdMx = L.mtm(Mx, kappa, mu, 1)
    assert abs(np.vdot(x, MdMx) - np.vdot(Mx, Mx)) <= 1e-12 * np.vdot(Mx, Mx).real


_FIELD_CACHE = {}


def _cached_fields(dims):
    """Seeded Haar links, input spinor and source of a full-size lattice, generated once per test session
    (32^3 x 64 links take ~20 s to draw); read-only for every test that uses them."""
    if dims not in _FIELD_CACHE:
        h = lu.volume(dims) // 2
        _FIELD_CACHE[dims] = (gen.gauge_haar(dims, SEED), gen.spinor_gaussian(h, SEED),
                              gen.spinor_gaussian(h, SEED, gen.STREAM_SOURCE))
    return _FIELD_CACHE[dims]


# BASELINE.json configs[4]: "32^3 x 64 in both double and single precision (single also with 12-real gauge
# reconstruction)"; PAPER.md:267 (single precision), :205, :305 (REC12).  Same launch configuration as the
# timings of sweep.py / bench.py (default block size, whole-lattice launches).
@pytest.mark.parametrize("precision,recon,tol", [(0, 12, TOL_D), (1, 18, TOL_S), (1, 12, TOL_S)])
def test_config5_storage_variants_sampled_sites(B, oracle_mod, precision, recon, tol):
    dims = (32, 32, 32, 64)
    kappa, mu = 0.15, 0.1
    U, x, _ = _cached_fields(dims)
    h = lu.volume(dims) // 2
    sites = _sample_sites(h, 300, 29 + recon + precision)
    # the oracle is fed what the kernel is fed: inputs rounded to the storage precision
    Ur, xr = _round_inputs(U, x, precision)
    L = Lat(B, dims, AP, U, precision, recon)
    for parity in (0, 1):
        got = L.dslash(x, parity, kappa)
        want = oracle_mod.dslash_eo_sites(dims, AP, Ur, xr, sites, parity, kappa)
        assert lu.rel_err(got[sites], want) <= tol
        assert np.max(np.abs(got[sites] - want)) <= tol * np.max(np.abs(want))     # no single element off
        assert np.all(np.isfinite(got))
    for dagger in (0, 1):
        got = L.mtm(x, kappa, mu, dagger)
        want = oracle_mod.mhat_sites(dims, AP, Ur, xr, sites, kappa, mu, dagger)
        assert lu.rel_err(got[sites], want) <= tol
        assert np.max(np.abs(got[sites] - want)) <= tol * np.max(np.abs(want))
        assert np.all(np.isfinite(got))
    # holds at any size: <x, Mhat^dag Mhat x> = |Mhat x|^2 (to the storage precision)
    Mx = L.mtm(x, kappa, mu, 0)
    MdMx = L.mtm(Mx, kappa, mu, 1)
    assert abs(np.vdot(xr, MdMx) - np.vdot(Mx, Mx)) <= (1e-12 if precision == 0 else 1e-5) * np.vdot(Mx, Mx).real
    del L


@pytest.mark.parametrize("precision,recon,tol,slack", [(0, 12, 1e-10, 1.05), (1, 18, 1e-5, 20.0), (1, 12, 1e-5, 20.0)])
def test_config4_cg_24c48_storage_variants(B, oracle_mod, precision, recon, tol, slack):
    """CG on the config 4 lattice in the other three storage formats, the residual taken by the ORACLE's
    (double) operator: double/12 to the double bar; single to what the recursive residual in float delivers."""
    dims = (24, 24, 24, 48)
    kappa, mu = 0.15, 0.1
    U, _, b = _cached_fields(dims)
    L = Lat(B, dims, AP, U, precision, recon)
    st, x, (iters, rr, rt) = L.cg(b, kappa, mu, tol, 2000)
    assert st == 0 and 5 <= iters <= 80 and rr <= tol
    r = b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= slack * tol
    del L


def test_config5_mixed_and_bicgstab_solves_32c64(B, oracle_mod):
    """One mixed-precision solve (single/12 inner, double/18 outer) and one BiCGStab solve at the bench
    workload's size, each checked by ONE application of the oracle's operator to the GPU's solution."""
    dims = (32, 32, 32, 64)
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U, _, b = _cached_fields(dims)
    nb = np.linalg.norm(b)
    st, x, (iters, rr, rt), outer = _mixed_solve(B, dims, U, b, kappa, mu, tol, 2000)
    assert st == 0 and rr <= tol and outer >= 2 and 20 <= iters <= 120
    assert np.linalg.norm(b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)) / nb <= 1.05 * tol
    L = Lat(B, dims, AP, U)
    st, x, (iters, rr, rt) = L.bicgstab(b, kappa, mu, tol, 2000)
    assert st == 0 and rr <= tol and 5 <= iters <= 60
    true_rel = np.linalg.norm(b - oracle_mod.mhat(dims, AP, U, x, kappa, mu, 0)) / nb
    assert true_rel <= 1.05 * tol and abs(rt - true_rel) <= 0.05 * tol
    del L


def test_fields_beyond_4_gib_sampled_sites(B, oracle_mod):
    """Maximum sizes: at 48^3 x 96 the gauge field is 6.1 GB in both the canonical and the internal layout, so
    byte offsets pass 2^32 inside it (from the mu = 1 links of odd sites on).  Any arrangement of SU(3)
    matrices is a valid gauge field, so the big field is a fixed pseudo-random gather of the links of a
    seeded 16^3 x 32 Haar field (lattice_util.big_gauge; generating 42 M fresh links would take minutes); oracle and GPU get the same
    array.  Checked on sampled sites of both parities, in 18- and 12-real storage, plus the field-wide identity."""
    dims = (48, 48, 48, 96)
    V = lu.volume(dims)
    U = lu.big_gauge(dims, gen.gauge_haar((16, 16, 16, 32), SEED).reshape(-1, 3, 3))
    assert U.nbytes > 2 ** 32
    h = V // 2
    x = gen.spinor_gaussian(h, SEED)
    sites = _sample_sites(h, 300, 23)
    kappa, mu = 0.15, 0.1
    for recon in (18, 12):
        L = Lat(B, dims, AP, U, 0, recon)
        assert B.lqcd_gauge_bytes() > (2 ** 32 if recon == 18 else 2 ** 31)
        for parity in (0, 1):
            got = L.dslash(x, parity, kappa)[sites]
            want = oracle_mod.dslash_eo_sites(dims, AP, U, x, sites, parity, kappa)
            assert lu.rel_err(got, want) <= TOL_D
        for dagger in (0, 1):
            got = L.mtm(x, kappa, mu, dagger)
            want = oracle_mod.mhat_sites(dims, AP, U, x, sites, kappa, mu, dagger)
            assert lu.rel_err(got[sites], want) <= TOL_D
            assert np.all(np.isfinite(got))
        Mx = L.mtm(x, kappa, mu, 0)
        MdMx = L.mtm(Mx, kappa, mu, 1)
        assert abs(np.vdot(x, MdMx) - np.vdot(Mx, Mx)) <= 1e-12 * np.vdot(Mx, Mx).real
        del L


def test_config4_cg_24c48(B, oracle_mod):
    dims = (24, 24, 24, 48)
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U, _, b = _cached_fields(dims)
    L = Lat(B, dims, AP, U)
    st, x, (iters, rr, rt) = L.cg(b, kappa, mu, tol, 2000)
    assert st == 0 and 20 <= iters <= 80 and rr <= tol
    r = b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)     # one oracle application of A
    assert np.linalg.norm(r) / np.linalg.norm(b) <= 1.05 * tol


# --------------------------------------------------------------------------- mixed-precision CG
def _mixed_solve(B, dims, U, b, kappa, mu, tol, maxit, recon_d=18, recon_s=12, inner_tol=0.0):
    B.lqcd_init(dims, AP)
    B.lqcd_set_stream()
    B.lqcd_set_format(B.LQCD_SINGLE, recon_s)
    gs = B.upload_gauge(U)
    B.lqcd_set_format(B.LQCD_DOUBLE, recon_d)
    gd = B.upload_gauge(U)
    src = B.upload_spinor(b, 0)
    x = B.alloc_spinor()
    st = B.lqcd_cg_mdagm_mixed(gd, recon_d, gs, recon_s, src, x, kappa, mu, tol, maxit, inner_tol)
    return st, B.download_spinor(x, 0), B.lqcd_cg_stats(), B.lqcd_cg_outer_iterations()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 16)])
@pytest.mark.parametrize("recon_d,recon_s", [(18, 12), (18, 18), (12, 12)])
@pytest.mark.parametrize("tol,inner_tol", [(1e-10, 0.0), (1e-13, 0.0), (1e-10, 1e-4)])
def test_mixed_precision_cg_reaches_double_accuracy(B, oracle_mod, dims, recon_d, recon_s, tol, inner_tol):
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    st, x, (iters, rr, rt), outer = _mixed_solve(B, dims, U, b, kappa, mu, tol, 2000, recon_d, recon_s, inner_tol)
    assert st == 0 and outer >= 2 and iters > 0
    assert rr <= tol and rt == rr            # the outer residual is a true residual, evaluated in double
    # the same solution the double oracle finds: true residual under the ORACLE's operator, and x itself
    r = b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= 1.05 * tol + 2e-15
    st_o, x_o, it_o, rr_o, rt_o = oracle_mod.cg_mdagm(dims, AP, U, b, kappa, mu, min(tol, 1e-12), 2000)
    assert lu.rel_err(x, x_o) <= 10 * 5.0 * max(tol, 1e-12)
    # defect correction restarts the Krylov space: a bounded number of extra iterations
    assert iters <= 2.5 * it_o + 10


def test_mixed_precision_cg_edge_cases(B):
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    h = lu.volume(dims) // 2
    st, x, (iters, rr, rt), outer = _mixed_solve(B, dims, U, np.zeros((h, 4, 3), dtype=complex), 0.15, 0.1, 1e-10, 100)
    assert st == 0 and iters == 0 and outer == 0 and np.all(x == 0)
    b = gen.spinor_gaussian(h, SEED, gen.STREAM_SOURCE)
    st, x, (iters, rr, rt), outer = _mixed_solve(B, dims, U, b, 0.15, 0.1, 1e-10, 6)
    assert st == B.LQCD_NOT_CONVERGED and iters == 6 and rr > 1e-10
    gd, s = B.alloc_gauge(), B.alloc_spinor()
    for call in (lambda: B.lqcd_cg_mdagm_mixed(gd, 18, gd, 12, s, s, 0.1, 0.1, 1e-8, 10),
                 lambda: B.lqcd_cg_mdagm_mixed(gd, 17, gd, 12, s, B.alloc_spinor(), 0.1, 0.1, 1e-8, 10),
                 lambda: B.lqcd_cg_mdagm_mixed(gd, 18, gd, 12, s, B.alloc_spinor(), 0.1, 0.1, 1e-8, 10, 2.0)):
        with pytest.raises(B.LqcdError) as e:
            call()
        assert e.value.status == B.LQCD_BAD_ARG


def test_a_nan_source_is_a_breakdown_in_every_solver(B):
    """A NaN in b must never come back as 'converged': all three solvers return LQCD_BREAKDOWN (include/lqcd.h)."""
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    b[5, 2, 1] = np.nan
    L = Lat(B, dims, AP, U)
    for solve in (lambda: L.cg(b, 0.15, 0.1, 1e-10, 50), lambda: L.bicgstab(b, 0.15, 0.1, 1e-10, 50),
                  lambda: _mixed_solve(B, dims, U, b, 0.15, 0.1, 1e-10, 50)):
        with pytest.raises(B.LqcdError) as e:
            solve()
        assert e.value.status == B.LQCD_BREAKDOWN
    # ... and a NaN in the links
    Un = U.copy()
    Un[7, 1, 0, 0] = np.nan
    b = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    with pytest.raises(B.LqcdError) as e:
        _mixed_solve(B, dims, Un, b, 0.15, 0.1, 1e-10, 50)
    assert e.value.status == B.LQCD_BREAKDOWN


def test_mixed_precision_cg_24c48(B, oracle_mod):
    dims = (24, 24, 24, 48)
    kappa, mu, tol = 0.15, 0.1, 1e-10
    U, _, b = _cached_fields(dims)
    st, x, (iters, rr, rt), outer = _mixed_solve(B, dims, U, b, kappa, mu, tol, 2000)
    assert st == 0 and rr <= tol and 20 <= iters <= 120
    r = b - oracle_mod.mdagm(dims, AP, U, x, kappa, mu)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= 1.05 * tol


# --------------------------------------------------------------------------- full-lattice operator and solve
def _full_apply(B, L, dims, psi, kappa, mu):
    ie, io = B.upload_spinor(lu.to_half(dims, psi, 0), 0), B.upload_spinor(lu.to_half(dims, psi, 1), 1)
    oe, oo = B.alloc_spinor(), B.alloc_spinor()
    B.lqcd_mtm_full(L.g, ie, io, oe, oo, kappa, mu)
    return lu.from_halves(dims, B.download_spinor(oe, 0), B.download_spinor(oo, 1))


@pytest.mark.parametrize("dims,phases", [((4, 4, 4, 4), AP), ((2, 2, 2, 2), GENERIC_PH),
                                         ((4, 6, 2, 8), GENERIC_PH), ((8, 8, 8, 16), AP)])
@pytest.mark.parametrize("precision,recon,tol", [(0, 18, TOL_D), (1, 12, TOL_S)])
def test_mtm_full_matches_oracle_eq6(B, oracle_mod, dims, phases, precision, recon, tol):
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    psi = gen.spinor_gaussian(V, SEED)
    Ur, pr = _round_inputs(U, psi, precision)
    L = Lat(B, dims, phases, U, precision, recon)
    assert lu.rel_err(_full_apply(B, L, dims, psi, kappa, mu), oracle_mod.m_full(dims, phases, Ur, pr, kappa, mu)) <= tol
    assert lu.rel_err(_full_apply(B, L, dims, psi, 0.0, 0.3), oracle_mod.m_full(dims, phases, Ur, pr, 0.0, 0.3)) <= tol


def test_twisted_mass_identity_on_gpu(B):
    # PAPER.md:82 in operator form: |M(mu) psi|^2 = |M(0) psi|^2 + 4 kappa^2 mu^2 |psi|^2
    dims = (8, 8, 8, 16)
    kappa, mu = 0.15, 0.1
    U = gen.gauge_haar(dims, SEED)
    psi = gen.spinor_gaussian(lu.volume(dims), SEED)
    L = Lat(B, dims, AP, U)
    n_mu = np.linalg.norm(_full_apply(B, L, dims, psi, kappa, mu)) ** 2
    n_0 = np.linalg.norm(_full_apply(B, L, dims, psi, kappa, 0.0)) ** 2
    want = n_0 + 4 * kappa ** 2 * mu ** 2 * np.linalg.norm(psi) ** 2
    assert abs(n_mu - want) / want < 1e-13


def _full_solve(B, L, dims, eta, kappa, mu, tol, maxit):
    ee, eo_ = B.upload_spinor(lu.to_half(dims, eta, 0), 0), B.upload_spinor(lu.to_half(dims, eta, 1), 1)
    pe, po = B.alloc_spinor(), B.alloc_spinor()
    st = B.lqcd_solve_full(L.g, ee, eo_, pe, po, kappa, mu, tol, maxit)
    return st, lu.from_halves(dims, B.download_spinor(pe, 0), B.download_spinor(po, 1))


def test_solve_full_against_dense_solve(B):
    dims = (2, 2, 2, 4)
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    eta = gen.spinor_gaussian(V, SEED, gen.STREAM_SOURCE)
    want = np.linalg.solve(lu.dense_m(dims, AP, U, kappa, mu), eta.ravel()).reshape(V, 4, 3)
    L = Lat(B, dims, AP, U)
    st, psi = _full_solve(B, L, dims, eta, kappa, mu, 1e-13, 500)
    assert st == 0
    assert lu.rel_err(psi, want) < 1e-11


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 16)])
def test_solve_full_residual_under_oracle_operator(B, oracle_mod, dims):
    kappa, mu, tol = 0.15, 0.1, 1e-10
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    eta = gen.spinor_gaussian(V, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    st, psi = _full_solve(B, L, dims, eta, kappa, mu, tol, 2000)
    iters, rr, rt = B.lqcd_cg_stats()
    assert st == 0 and rr <= tol and iters > 0
    r = eta - oracle_mod.m_full(dims, AP, U, psi, kappa, mu)
    assert np.linalg.norm(r) / np.linalg.norm(eta) <= 10 * tol     # cond(Mhat) ~ 3-5 of slack
    # kappa = 0: M is site diagonal, no iteration needed
    st, psi = _full_solve(B, L, dims, eta, 0.0, 0.3, tol, 10)
    assert st == 0 and lu.rel_err(oracle_mod.m_full(dims, AP, U, psi, 0.0, 0.3), eta) < 1e-14


# --------------------------------------------------------------------------- fermion force
def _gpu_force(B, dims, phases, U, X, Y, kappa, precision=0, recon=18):
    L = Lat(B, dims, phases, U, precision, recon)
    xe, xo = B.upload_spinor(lu.to_half(dims, X, 0), 0), B.upload_spinor(lu.to_half(dims, X, 1), 1)
    ye, yo = B.upload_spinor(lu.to_half(dims, Y, 0), 0), B.upload_spinor(lu.to_half(dims, Y, 1), 1)
    f = B.alloc_force()
    B.lqcd_fermion_force(L.g, xe, xo, ye, yo, f, kappa)
    return B.download_force(f)


@pytest.mark.parametrize("dims,phases", [
    ((4, 4, 4, 4), AP),
    ((2, 2, 2, 2), GENERIC_PH),    # every forward hop in a 2-extent direction from x_mu = 1 wraps
    ((4, 6, 2, 8), GENERIC_PH),
    ((6, 4, 10, 4), AP),           # Vh = 480: a ragged last group of 32 sites
    ((8, 8, 8, 16), AP),
])
@pytest.mark.parametrize("precision,recon,tol", [(0, 18, TOL_D), (0, 12, TOL_D), (1, 18, TOL_S), (1, 12, TOL_S)])
def test_fermion_force_matches_oracle(B, oracle_mod, dims, phases, precision, recon, tol):
    kappa = 0.15
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    X = gen.spinor_gaussian(V, SEED, 7)
    Y = gen.spinor_gaussian(V, SEED, 8)
    Ur, Xr = _round_inputs(U, X, precision)
    _, Yr = _round_inputs(U, Y, precision)
    want = oracle_mod.fermion_force(dims, phases, Ur, Xr, Yr, kappa)
    got = _gpu_force(B, dims, phases, U, X, Y, kappa, precision, recon)
    assert got.shape == want.shape == (V, 4, 8)
    assert lu.rel_err(got, want) <= tol
    assert np.max(np.abs(got - want)) <= 10 * tol * np.max(np.abs(want))


def test_fermion_force_gauge_covariance_on_gpu(B):
    # F'^a T^a = g(x) (F^a T^a) g(x)^dag under U' = g U g^dag(x+mu), X' = g X, Y' = g Y -- no oracle involved
    dims = (8, 8, 8, 16)
    kappa = 0.15
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    g = gen.su3_haar(V, SEED, gen.STREAM_GTRANS)
    X, Y = gen.spinor_gaussian(V, SEED, 7), gen.spinor_gaussian(V, SEED, 8)
    F = _gpu_force(B, dims, AP, U, X, Y, kappa)
    Xc = lu.site_coords(dims)
    Up = np.empty_like(U)
    for m in range(4):
        Yc = Xc.copy()
        Yc[:, m] = (Yc[:, m] + 1) % dims[m]
        Up[:, m] = np.einsum("sab,sbc,sdc->sad", g, U[:, m], g[lu.lex_index(dims, Yc)].conj())
    Fp = _gpu_force(B, dims, AP, Up, lu.apply_colour(g, X), lu.apply_colour(g, Y), kappa)
    want = np.einsum("sab,smbc,sdc->smad", g, lu.algebra_matrix(F), g.conj())
    assert lu.rel_err(lu.algebra_matrix(Fp), want) < 1e-13


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 16)])
def test_force_tm_matches_oracle(B, oracle_mod, dims):
    # the whole force of S = phi^dag (Mhat^dag Mhat)^-1 phi: CG + odd-site fields + outer product
    kappa, mu, tol = 0.15, 0.1, 1e-12
    U = gen.gauge_haar(dims, SEED)
    phi = gen.spinor_gaussian(lu.volume(dims) // 2, SEED, gen.STREAM_SOURCE)
    st_o, want, it_o = oracle_mod.force_tm(dims, AP, U, phi, kappa, mu, tol, 2000)
    L = Lat(B, dims, AP, U)
    src = B.upload_spinor(phi, 0)
    f = B.alloc_force()
    st = B.lqcd_force_tm(L.g, src, f, kappa, mu, tol, 2000)
    iters, rr, rt = B.lqcd_cg_stats()
    got = B.download_force(f)
    assert st == 0 and st_o == 0 and abs(iters - it_o) <= 2
    # both solves stop at |r| <= tol |phi|; the force is bilinear in the solution: 2 sqrt(cond) tol of slack
    assert lu.rel_err(got, want) <= 100 * tol
    assert np.max(np.abs(want)) > 1e-3


def test_force_tm_is_minus_the_action_derivative_on_gpu(B):
    # independent of the oracle: central differences of S from the dense Schur complement (numpy)
    dims = (2, 2, 2, 2)
    kappa, mu, h = 0.15, 0.1, 1e-4
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    phi = gen.spinor_gaussian(V // 2, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    f = B.alloc_force()
    assert B.lqcd_force_tm(L.g, B.upload_spinor(phi, 0), f, kappa, mu, 1e-13, 500) == 0
    F = B.download_force(f)

    def action(Uv):
        S = lu.dense_mhat(dims, AP, Uv, kappa, mu)
        return np.real(np.vdot(phi.ravel(), np.linalg.solve(S.conj().T @ S, phi.ravel())))

    for s, m in [(0, 3), (V - 1, 3), (5, 0), (10, 1), (7, 2)]:
        for a in range(8):
            Up, Um = U.copy(), U.copy()
            Up[s, m] = lu.exp_i_w_T(a, h) @ U[s, m]
            Um[s, m] = lu.exp_i_w_T(a, -h) @ U[s, m]
            fd = -(action(Up) - action(Um)) / (2 * h)
            assert abs(F[s, m, a] - fd) < 1e-6 * max(1.0, abs(fd))


def test_force_edge_cases(B):
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, SEED)
    L = Lat(B, dims, AP, U)
    V = lu.volume(dims)
    assert B.lqcd_force_bytes() == V * 4 * 8 * 8         # 256 B per site
    zero = np.zeros((V // 2, 4, 3), dtype=complex)
    f = B.alloc_force()
    assert B.lqcd_force_tm(L.g, B.upload_spinor(zero, 0), f, 0.15, 0.1, 1e-10, 50) == 0
    assert np.all(B.download_force(f) == 0)                # phi = 0 -> X = Y = 0 -> F = 0
    phi = gen.spinor_gaussian(V // 2, SEED, gen.STREAM_SOURCE)
    assert B.lqcd_force_tm(L.g, B.upload_spinor(phi, 0), f, 0.0, 0.1, 1e-10, 50) == 0
    assert np.all(B.download_force(f) == 0)                # kappa = 0 -> no hopping term -> F = 0
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_fermion_force(L.g, 0, f, f, f, f, 0.1)
    assert e.value.status == B.LQCD_BAD_ARG


def test_fermion_force_full_size_sampled_links(B, oracle_mod):
    # BASELINE config 5 lattice: 300 sampled links through the oracle's link-wise evaluator
    dims = (32, 32, 32, 64)
    kappa = 0.15
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    X, Y = gen.spinor_gaussian(V, SEED, 7), gen.spinor_gaussian(V, SEED, 8)
    got = _gpu_force(B, dims, AP, U, X, Y, kappa)
    rng = np.random.default_rng(11)
    sites = np.concatenate([rng.integers(0, V, 290), [0, 1, V - 1, V - 2, V // 2, 31, 32, 1023, 32767, V - 32 * 32 * 32]])
    mus = np.concatenate([rng.integers(0, 4, 290), [0, 1, 2, 3, 0, 0, 1, 2, 3, 3]])
    want = oracle_mod.fermion_force_links(dims, AP, U, X, Y, sites, mus, kappa)
    assert lu.rel_err(got[sites, mus], want) <= TOL_D
    assert np.all(np.isfinite(got))


def test_fermion_force_beyond_4_gib_sampled_links(B, oracle_mod):
    """48^3 x 96: gauge field 6.1 GB, force field 2.7 GB; 300 sampled links against the oracle's link-wise evaluator."""
    dims = (48, 48, 48, 96)
    kappa = 0.15
    V = lu.volume(dims)
    U = lu.big_gauge(dims, gen.gauge_haar((16, 16, 16, 32), SEED).reshape(-1, 3, 3))
    X, Y = gen.spinor_gaussian(V, SEED, 7), gen.spinor_gaussian(V, SEED, 8)
    got = _gpu_force(B, dims, AP, U, X, Y, kappa)
    rng = np.random.default_rng(12)
    sites = np.concatenate([rng.integers(0, V, 294), [0, 1, V - 1, V - 2, V // 2, V - 48 * 48 * 48]])
    mus = np.concatenate([rng.integers(0, 4, 294), [0, 1, 2, 3, 0, 3]])
    want = oracle_mod.fermion_force_links(dims, AP, U, X, Y, sites, mus, kappa)
    assert lu.rel_err(got[sites, mus], want) <= TOL_D
    assert np.all(np.isfinite(got))


def test_cg_on_a_side_stream_graph_replay_matches_direct_launches(B, oracle_mod):
    """On a non-default stream the solver replays four iterations at a time as a cached CUDA graph (api.cu
    cg_graph_ready); the legacy default stream cannot be captured, so the tests above run direct launches.  Same
    kernels, same arguments, same order: x, the iteration count and the residuals must be bit-identical, a second
    solve (graph reused) and a solve with other parameters (graph rebuilt) included; and the oracle's operator
    confirms the residual."""
    import torch
    dims = (8, 8, 8, 16)
    U = gen.gauge_haar(dims, SEED)
    h = lu.volume(dims) // 2
    b = gen.spinor_gaussian(h, SEED, gen.STREAM_SOURCE)
    L = Lat(B, dims, AP, U)
    ref = {}
    for kappa, mu in ((0.15, 0.1), (0.14, 0.2)):
        st, x, stats = L.cg(b, kappa, mu, 1e-10, 500)
        assert st == 0
        ref[(kappa, mu)] = (x, stats)
    side = torch.cuda.Stream()
    B.lqcd_set_stream(side)
    with torch.cuda.stream(side):
        for kappa, mu in ((0.15, 0.1), (0.15, 0.1), (0.14, 0.2)):
            st, x, stats = L.cg(b, kappa, mu, 1e-10, 500)
            assert st == 0
            assert stats == ref[(kappa, mu)][1]
            assert np.array_equal(x, ref[(kappa, mu)][0])
        res = b - oracle_mod.mdagm(dims, AP, U, x, 0.14, 0.2)
        assert np.linalg.norm(res) <= 1.05e-10 * np.linalg.norm(b)
        # the three-step solver: lqcd_cg_iterate goes through the same graph
        s_ = B.upload_spinor(b, 0)
        xd = B.alloc_spinor()
        B.lqcd_cg_setup(L.g, s_, xd, 0.15, 0.1, 1e-10)
        B.lqcd_cg_iterate(200)
        assert B.lqcd_cg_finish() == 0
        assert B.lqcd_cg_stats() == ref[(0.15, 0.1)][1]
        assert np.array_equal(B.download_spinor(xd, 0), ref[(0.15, 0.1)][0])
    torch.cuda.synchronize()
    B.lqcd_set_stream()


def test_bicgstab_on_a_side_stream_graph_replay_matches_direct_launches(B, oracle_mod):
    """BiCGStab replays its four-iteration chunk (36 launches) through the same graph cache: bit-identical to direct
    launches, also when a CG solve (other graph kind, same cache slot) runs in between, in double and in single/12."""
    import torch
    dims = (8, 8, 8, 16)
    U = gen.gauge_haar(dims, SEED)
    h = lu.volume(dims) // 2
    b = gen.spinor_gaussian(h, SEED, gen.STREAM_SOURCE)
    for precision, recon, tol in ((0, 18, 1e-10), (1, 12, 1e-5)):
        L = Lat(B, dims, AP, U, precision, recon)
        B.lqcd_set_stream()
        st, x0, stats0 = L.bicgstab(b, 0.15, 0.1, tol, 500)
        assert st == 0
        side = torch.cuda.Stream()
        B.lqcd_set_stream(side)
        with torch.cuda.stream(side):
            for rep in range(3):
                st, x, stats = L.bicgstab(b, 0.15, 0.1, tol, 500)
                assert st == 0 and stats == stats0
                assert np.array_equal(x, x0)
                if rep == 0:
                    assert L.cg(b, 0.15, 0.1, tol, 500)[0] == 0
            if precision == 0:
                res = b - oracle_mod.mhat(dims, AP, U, x, 0.15, 0.1, 0)
                assert np.linalg.norm(res) <= 1.05 * tol * np.linalg.norm(b)
        torch.cuda.synchronize()
        B.lqcd_set_stream()


# --------------------------------------------------------------------------- staged variants of the hopping kernel
@pytest.mark.parametrize("variant", [1, 2, 3, 4, 5, 6, 7])
@pytest.mark.parametrize("precision,recon,tol", [(0, 18, TOL_D), (0, 12, TOL_D), (1, 18, TOL_S), (1, 12, TOL_S)])
def test_hopping_variants_match_oracle(B, oracle_mod, variant, precision, recon, tol):
    """lqcd_set_hop_variant: every staged variant of the hopping kernel (hopping_staged.cu) against the oracle, in every
    storage format, on a ragged lattice with complex phases on every wrap (Vh = 192: one and a half thread blocks) and on
    8^3 x 16; D_eo, D_oe, Mhat and Mhat^dag (plain and M_ee*aux epilogues).  The variant must also be bit-identical to
    the default kernel: same operations in the same order per site."""
    kappa, mu = 0.15, 0.1
    try:
        for dims, phases in (((4, 6, 2, 8), GENERIC_PH), ((8, 8, 8, 16), AP)):
            U = gen.gauge_haar(dims, SEED)
            x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
            Ur, xr = _round_inputs(U, x, precision)
            B.lqcd_set_hop_variant(0)
            L = Lat(B, dims, phases, U, precision, recon)
            ref = [L.dslash(x, 0, kappa), L.dslash(x, 1, kappa), L.mtm(x, kappa, mu, 0), L.mtm(x, kappa, mu, 1)]
            B.lqcd_set_hop_variant(variant)
            got = [L.dslash(x, 0, kappa), L.dslash(x, 1, kappa), L.mtm(x, kappa, mu, 0), L.mtm(x, kappa, mu, 1)]
            want = [oracle_mod.dslash_eo(dims, phases, Ur, xr, 0, kappa), oracle_mod.dslash_eo(dims, phases, Ur, xr, 1, kappa),
                    oracle_mod.mhat(dims, phases, Ur, xr, kappa, mu, 0), oracle_mod.mhat(dims, phases, Ur, xr, kappa, mu, 1)]
            for g_, w_, r_ in zip(got, want, ref):
                assert lu.rel_err(g_, w_) <= tol
                assert np.array_equal(g_, r_)
    finally:
        B.lqcd_set_hop_variant(0)
    with pytest.raises(B.LqcdError) as e:
        B.lqcd_set_hop_variant(99)
    assert e.value.status == B.LQCD_BAD_ARG


@pytest.mark.parametrize("precision,recon,tol", [(0, 18, TOL_D), (1, 12, TOL_S)])
def test_hopping_variants_at_the_bench_size(B, oracle_mod, precision, recon, tol):
    """The staged variants at 32^3 x 64, in the launch configuration sweep.py --hop-variant times (the tile order is only
    active where a z plane holds whole groups: 16 groups per plane here): D_eo and Mhat^dag bit-identical to the default
    kernel on the whole field, and against the oracle on 300 sampled sites; a CG solve with the tile order through the
    fused launches (modes 2, 3) bit-identical to the default."""
    dims = (32, 32, 32, 64)
    kappa, mu = 0.15, 0.1
    U, x, b = _cached_fields(dims)
    h = lu.volume(dims) // 2
    sites = _sample_sites(h, 300, 77 + recon)
    Ur, xr = _round_inputs(U, x, precision)
    try:
        B.lqcd_set_hop_variant(0)
        L = Lat(B, dims, AP, U, precision, recon)
        ref_d, ref_m = L.dslash(x, 0, kappa), L.mtm(x, kappa, mu, 1)
        assert lu.rel_err(ref_d[sites], oracle_mod.dslash_eo_sites(dims, AP, Ur, xr, sites, 0, kappa)) <= tol
        assert lu.rel_err(ref_m[sites], oracle_mod.mhat_sites(dims, AP, Ur, xr, sites, kappa, mu, 1)) <= tol
        st0, x0, stats0 = L.cg(b, kappa, mu, 0.0, 6)
        for variant in (2, 4, 5, 6, 7):
            B.lqcd_set_hop_variant(variant)
            assert np.array_equal(L.dslash(x, 0, kappa), ref_d), variant
            assert np.array_equal(L.mtm(x, kappa, mu, 1), ref_m), variant
        st6, x6, stats6 = L.cg(b, kappa, mu, 0.0, 6)      # variant 6 still selected
        assert (st6, stats6) == (st0, stats0) and np.array_equal(x6, x0)
    finally:
        B.lqcd_set_hop_variant(0)


def test_programmatic_dependent_launch_changes_nothing_but_the_time():
    """Launches on the legacy default stream chain the kernels of the CG and BiCGStab iterations by programmatic
    dependent launch (lqcd_internal.h: chain_prologue / launch_chained); LQCD_PDL=0 (read once per process) launches them
    the ordinary way.  Same kernels, same order: the solutions, iteration counts and residuals must be bit-identical."""
    import hashlib
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = (
        "import sys, hashlib, numpy as np; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
        "import lqcd_inputs as gen, lattice_util as lu, paper_1209_5942_b200.binding as B\n"
        "dims = (8, 8, 8, 16); U = gen.gauge_haar(dims); h = lu.volume(dims) // 2\n"
        "b = gen.spinor_gaussian(h, stream=gen.STREAM_SOURCE)\n"
        "B.lqcd_init(dims, gen.antiperiodic_t()); B.lqcd_set_stream(); g = B.upload_gauge(U); s = B.upload_spinor(b, 0)\n"
        "x = B.alloc_spinor(); out = []\n"
        "st = B.lqcd_cg_mdagm(g, s, x, 0.15, 0.1, 1e-10, 500); out += [st, B.lqcd_cg_stats(), hashlib.sha256(B.download_spinor(x, 0).tobytes()).hexdigest()]\n"
        "st = B.lqcd_bicgstab_mhat(g, s, x, 0.15, 0.1, 1e-10, 500); out += [st, B.lqcd_cg_stats(), hashlib.sha256(B.download_spinor(x, 0).tobytes()).hexdigest()]\n"
        "B.lqcd_mtm(g, s, x, 0.15, 0.1, 1); out += [hashlib.sha256(B.download_spinor(x, 0).tobytes()).hexdigest()]\n"
        "print('RESULT', out)\n" % (root, os.path.join(root, "tests")))
    res = []
    for pdl in ("1", "0"):
        r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600,
                           env=dict(os.environ, LQCD_PDL=pdl))
        assert r.returncode == 0, r.stderr[-2000:]
        res.append([l for l in r.stdout.splitlines() if l.startswith("RESULT")][0])
    assert res[0] == res[1]
    assert "RESULT [0, " in res[0]


def test_random_lattice_shapes_all_formats(B, oracle_mod):
    """Sixteen seeded random even extents between 2 and 12 (ragged warps, N_mu = 2 in some direction, extents that are
    not powers of two, z planes that do and do not hold whole 32-site groups), complex phases on every boundary, in all
    four storage formats: D_eo, D_oe and Mhat^dag against the oracle; the tile-order variant on the same shapes must
    reproduce the default bit for bit (it is active only where a z plane is a whole number of groups)."""
    rng = np.random.default_rng(1209_5942)
    shapes = {(2, 2, 2, 2), (12, 2, 2, 2), (2, 12, 2, 4)}
    while len(shapes) < 16:
        shapes.add(tuple(int(2 * rng.integers(1, 7)) for _ in range(4)))
    kappa, mu = 0.137, 0.21
    try:
        for dims in sorted(shapes):
            U = gen.gauge_haar(dims, SEED)
            x = gen.spinor_gaussian(lu.volume(dims) // 2, SEED)
            for precision, recon, tol in ((0, 18, TOL_D), (0, 12, TOL_D), (1, 18, TOL_S), (1, 12, TOL_S)):
                Ur, xr = _round_inputs(U, x, precision)
                B.lqcd_set_hop_variant(0)
                L = Lat(B, dims, GENERIC_PH, U, precision, recon)
                got = [L.dslash(x, 0, kappa), L.dslash(x, 1, kappa), L.mtm(x, kappa, mu, 1)]
                want = [oracle_mod.dslash_eo(dims, GENERIC_PH, Ur, xr, 0, kappa), oracle_mod.dslash_eo(dims, GENERIC_PH, Ur, xr, 1, kappa),
                        oracle_mod.mhat(dims, GENERIC_PH, Ur, xr, kappa, mu, 1)]
                for g_, w_ in zip(got, want):
                    assert lu.rel_err(g_, w_) <= tol, (dims, precision, recon)
                B.lqcd_set_hop_variant(6)
                for g_, t_ in zip(got, [L.dslash(x, 0, kappa), L.dslash(x, 1, kappa), L.mtm(x, kappa, mu, 1)]):
                    assert np.array_equal(g_, t_), (dims, precision, recon)
    finally:
        B.lqcd_set_hop_variant(0)
