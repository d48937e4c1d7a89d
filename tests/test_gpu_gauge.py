"""Parity of the pure-gauge kernels (gauge_update.cu: heatbath, overrelaxation, plaquette) against
oracle/gauge_oracle.cpp through the C ABI (-m gpu).  SURVEY.md section 8(f) row 4.

Bar: relative L2 error <= 1e-13 in double on the whole updated field and <= 1e-13 * max|U| element by
element.  The heatbath's accept/reject decisions are taken in double on both sides (DESIGN.md section
9); a flipped decision needs |r4^2 - (1 - delta/2)| ~ 1e-15, so in double no link may differ.  In
single precision (3x3 products in float, SU(2) step in double, oracle fed the float-rounded links) the
staples differ by float rounding, so a decision may flip on ~1e-7 of the links: those links are valid
heatbath samples but not comparable, the test bounds their number and checks that they are in SU(3).
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


def _setup(B, dims, U, precision=0, recon=18):
    B.lqcd_init(dims, AP)
    B.lqcd_set_format(precision, recon)
    B.lqcd_set_stream()
    return B.upload_gauge(U)


def _round(U, precision):
    return U if precision == 0 else U.astype(np.complex64).astype(np.complex128)


def _su3_defect(M):
    M = M.reshape(-1, 3, 3)
    return max(np.abs(M @ np.conj(np.swapaxes(M, 1, 2)) - np.eye(3)).max(), np.abs(np.linalg.det(M) - 1).max())


DIMS = [(4, 4, 4, 4),      # BASELINE config 1 lattice
        (2, 2, 2, 2),      # N_mu = 2: x+nu and x-nu are the same site
        (4, 6, 2, 8),      # unequal extents
        (6, 4, 10, 4),     # Vh = 480: ragged tail for 128-thread blocks
        (8, 8, 8, 16)]     # BASELINE config 2 lattice: several blocks


@pytest.mark.parametrize("dims", DIMS)
def test_unpack_gauge_roundtrip_and_plaquette(B, oracle_mod, dims):
    for U in (gen.gauge_haar(dims, SEED), gen.gauge_near_identity(dims, SEED, 0.3)):
        g = _setup(B, dims, U)
        assert np.array_equal(B.download_gauge(g), U)
        assert abs(B.lqcd_plaquette(g) - oracle_mod.plaquette(dims, U)) <= 1e-14
    g = _setup(B, dims, gen.gauge_unit(dims))
    assert B.lqcd_plaquette(g) == 1.0


@pytest.mark.parametrize("precision,recon,tol", [(0, 12, 1e-14), (1, 18, 1e-6), (1, 12, 1e-6)])
def test_plaquette_and_unpack_storage_variants(B, oracle_mod, precision, recon, tol):
    dims = (4, 6, 2, 8)
    U = gen.gauge_near_identity(dims, SEED, 0.3)
    g = _setup(B, dims, U, precision, recon)
    assert abs(B.lqcd_plaquette(g) - oracle_mod.plaquette(dims, _round(U, precision))) <= tol
    assert np.max(np.abs(B.download_gauge(g) - U)) <= (1e-14 if precision == 0 else 2e-7)


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("mode", [0, 1])
def test_subsweeps_match_oracle(B, oracle_mod, dims, mode):
    """Every (mu, parity) sub-sweep from the same input field; untouched links stay bit-identical."""
    beta, tag = 5.7, 11
    U = gen.gauge_near_identity(dims, SEED, 0.4)
    par = lu.site_parity(dims)
    for mu in range(4):
        for parity in (0, 1):
            g = _setup(B, dims, U)
            B.lqcd_gauge_update(g, mu, parity, mode, beta, SEED, tag)
            got = B.download_gauge(g)
            want = oracle_mod.gauge_subsweep(dims, U, mu, parity, mode, beta, SEED, tag)
            mask = np.zeros((lu.volume(dims), 4), dtype=bool)
            mask[par == parity, mu] = True
            assert np.array_equal(got[~mask], U[~mask])
            assert lu.rel_err(got[mask], want[mask]) <= TOL_D
            assert np.max(np.abs(got - want)) <= TOL_D
            assert np.min(np.abs(got[mask] - U[mask]).reshape(-1, 9).max(axis=1)) > 1e-6   # every link of the set moved


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 10, 4), (8, 8, 8, 16)])
def test_chained_sweeps_match_oracle(B, oracle_mod, dims):
    """Two heatbath and two overrelaxation sweeps chained on an ordered field (later sub-sweeps read
    earlier updates; rounding differences grow slowly here)."""
    beta = 5.7
    U = gen.gauge_near_identity(dims, SEED, 0.4)
    g = _setup(B, dims, U)
    want = U
    for k, mode in enumerate((0, 1, 0, 1)):
        B.lqcd_gauge_sweep(g, mode, beta, SEED, 20 + k)
        want = oracle_mod.gauge_sweep(dims, want, mode, beta, SEED, 20 + k)
        got = B.download_gauge(g)
        assert lu.rel_err(got, want) <= TOL_D * (k + 1), (k, mode)
        assert np.max(np.abs(got - want)) <= 2 * TOL_D * (k + 1)
    assert _su3_defect(got) < 1e-13
    assert abs(B.lqcd_plaquette(g) - oracle_mod.plaquette(dims, want)) < 1e-13


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 10, 4), (8, 8, 8, 16)])
def test_hot_start_sweeps_from_identical_state(B, oracle_mod, dims):
    """Disordered field at strong coupling (beta = 1.2: small lambda, many Kennedy-Pendleton
    rejections, staples that nearly cancel).  As a map of the field at fixed random numbers the update
    is chaotic here -- a rounding difference grows ~2.5x per SUB-sweep (measured)
    -- so, as for CG (reading G14), sweeps are compared one at a time from identical state."""
    beta = 1.2
    state = gen.gauge_haar(dims, SEED)
    for k, mode in enumerate((0, 1, 0)):
        g = _setup(B, dims, state)
        B.lqcd_gauge_sweep(g, mode, beta, SEED, 20 + k)
        want = oracle_mod.gauge_sweep(dims, state, mode, beta, SEED, 20 + k)
        got = B.download_gauge(g)
        assert lu.rel_err(got, want) <= 1e-11, (k, mode)          # 8 chained sub-sweeps: 1e-15 * 2.5^8 ~ 2e-12
        assert np.max(np.abs(got - want)) <= 1e-9
        assert _su3_defect(got) < 1e-13
        state = want
    # one sub-sweep from identical state meets the plain bar
    g = _setup(B, dims, state)
    B.lqcd_gauge_update(g, 1, 1, 0, beta, SEED, 99)
    want = oracle_mod.gauge_subsweep(dims, state, 1, 1, 0, beta, SEED, 99)
    assert lu.rel_err(B.download_gauge(g), want) <= TOL_D


def test_overrelax_keeps_the_action_on_gpu(B):
    dims = (8, 8, 8, 16)
    g = _setup(B, dims, gen.gauge_near_identity(dims, SEED, 0.5))
    p0 = B.lqcd_plaquette(g)
    for k in range(3):
        B.lqcd_gauge_sweep(g, B.LQCD_OVERRELAX, 0.0, 0, 0)
    assert abs(B.lqcd_plaquette(g) - p0) < 1e-13
    assert _su3_defect(B.download_gauge(g)) < 1e-13


def test_heatbath_strong_coupling_plaquette_on_gpu(B):
    """<P> = beta/18 + beta^2/216 (strong coupling), measured on the GPU's own chain: 8^4, hot start."""
    dims, beta = (8, 8, 8, 8), 1.2
    g = _setup(B, dims, gen.gauge_haar(dims, SEED))
    vals = []
    for sweep in range(40):
        B.lqcd_gauge_sweep(g, B.LQCD_HEATBATH, beta, SEED, 500 + sweep)
        if sweep >= 10:
            vals.append(B.lqcd_plaquette(g))
    want = beta / 18 + beta ** 2 / 216
    assert abs(np.mean(vals) - want) < 0.0015, (np.mean(vals), want)


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("mode", [0, 1])
def test_single_precision_sweep(B, oracle_mod, recon, mode):
    dims, beta = (8, 8, 8, 16), 5.7
    U = gen.gauge_near_identity(dims, SEED, 0.4)
    g = _setup(B, dims, U, 1, recon)
    B.lqcd_gauge_sweep(g, mode, beta, SEED, 31)
    got = B.download_gauge(g)
    want = oracle_mod.gauge_sweep(dims, _round(U, 1), mode, beta, SEED, 31)
    err = np.abs(got - want).reshape(-1, 9).max(axis=1)
    bad = err > 1e-4
    # a flipped accept/reject decision (heatbath only) changes a link completely and perturbs the
    # staples of its neighbours updated later in the sweep
    assert bad.sum() <= (0 if mode == 1 else 40), bad.sum()
    assert lu.rel_err(got.reshape(-1, 9)[~bad], want.reshape(-1, 9)[~bad]) <= TOL_S
    assert _su3_defect(got) < 5e-6


def test_double_recon12_sweep(B, oracle_mod):
    dims, beta = (4, 6, 2, 8), 5.7
    U = gen.gauge_near_identity(dims, SEED, 0.4)
    g = _setup(B, dims, U, 0, 12)
    want = U
    for k, mode in enumerate((0, 1)):
        B.lqcd_gauge_sweep(g, mode, beta, SEED, 40 + k)
        want = oracle_mod.gauge_sweep(dims, want, mode, beta, SEED, 40 + k)
    assert lu.rel_err(B.download_gauge(g), want) <= 1e-12     # third rows are rebuilt from rows 0, 1


def test_gauge_update_error_codes(B):
    dims = (4, 4, 4, 4)
    g = _setup(B, dims, gen.gauge_unit(dims))
    for args in [(4, 0, 0, 5.7, 1, 1), (0, 2, 0, 5.7, 1, 1), (0, 0, 2, 5.7, 1, 1), (0, 0, 0, float("nan"), 1, 1),
                 (0, 0, 0, 0.0, 1, 1), (0, 0, 0, -1.0, 1, 1), (0, 0, 0, 5.7, 1, 1 << 24)]:
        with pytest.raises(B.LqcdError) as ei:
            B.lqcd_gauge_update(g, *args)
        assert ei.value.status == B.LQCD_BAD_ARG
    with pytest.raises(B.LqcdError):
        B.lqcd_gauge_update(0, 0, 0, 0, 5.7, 1, 1)
    # cold start, beta huge: links stay at 1 up to O(1/beta); a unit field under overrelaxation is a fixed point
    B.lqcd_gauge_sweep(g, B.LQCD_OVERRELAX, 0.0, 0, 0)
    assert np.max(np.abs(B.download_gauge(g) - gen.gauge_unit(dims))) < 1e-15
    B.lqcd_finalize()
    with pytest.raises(B.LqcdError) as ei:
        B.lqcd_gauge_update(g, 0, 0, 0, 5.7, 1, 1)
    assert ei.value.status == B.LQCD_NOT_INITIALISED


def test_full_size_subsweep_sampled_links(B, oracle_mod):
    """BASELINE config 5 lattice (32^3 x 64), the launch configuration the sweep timing uses: one
    heatbath and one overrelaxation sub-sweep, 300 sampled updated links each against the oracle's
    link-wise evaluator, untouched links bit-identical on a sampled slab."""
    dims, beta = (32, 32, 32, 64), 5.7
    V = lu.volume(dims)
    U = gen.gauge_near_identity(dims, SEED, 0.3)
    rng = np.random.default_rng(3)
    coords_sum = lambda s: (s % 32) + (s // 32) % 32 + (s // 1024) % 32 + (s // 32768)
    for mode, mu, parity in ((0, 2, 1), (1, 0, 0), (0, 3, 0)):
        g = _setup(B, dims, U)
        B.lqcd_gauge_update(g, mu, parity, mode, beta, SEED, 77)
        got = B.download_gauge(g)
        cand = rng.integers(0, V, 2000)
        cand = np.concatenate([cand, [0, 1, V - 1, V - 2, 31, 32 * 32 * 32 - 1]])
        sites = cand[coords_sum(cand) % 2 == parity][:300]
        want = oracle_mod.update_links(dims, U, sites, np.full(len(sites), mu), mode, beta, SEED, 77)
        assert lu.rel_err(got[sites, mu], want) <= TOL_D
        assert np.max(np.abs(got[sites, mu] - want)) <= TOL_D
        other = cand[coords_sum(cand) % 2 != parity]
        assert np.array_equal(got[other], U[other])
        assert np.array_equal(got[sites][:, [m for m in range(4) if m != mu]], U[sites][:, [m for m in range(4) if m != mu]])
        del g, got


def test_subsweep_beyond_4_gib_sampled_links(B, oracle_mod):
    """48^3 x 96: the gauge field is 6.1 GB, byte offsets pass 2^32 inside it.  One overrelaxation sub-sweep on
    links stored beyond 4 GiB (odd sites, mu = 1) and one heatbath sub-sweep (even sites, mu = 3): 300 sampled
    updated links each against the oracle's link-wise evaluator, sampled untouched links bit-identical, and the
    average plaquette of the whole field against the oracle's."""
    dims, beta = (48, 48, 48, 96), 5.7
    V = lu.volume(dims)
    U = lu.big_gauge(dims, gen.gauge_near_identity((16, 16, 16, 32), SEED, 0.3).reshape(-1, 3, 3))
    assert U.nbytes > 2 ** 32
    rng = np.random.default_rng(5)
    coords_sum = lambda s: (s % 48) + (s // 48) % 48 + (s // 2304) % 48 + (s // 110592)
    g = _setup(B, dims, U)
    assert abs(B.lqcd_plaquette(g) - oracle_mod.plaquette(dims, U)) <= 1e-13
    del g
    for mode, mu, parity in ((1, 1, 1), (0, 3, 0)):
        g = _setup(B, dims, U)
        B.lqcd_gauge_update(g, mu, parity, mode, beta, SEED, 77)
        got = B.download_gauge(g)
        cand = np.concatenate([rng.integers(0, V, 2000), [0, 1, V - 1, V - 2, 47, 48 * 48 * 48 - 1]])
        sites = cand[coords_sum(cand) % 2 == parity][:300]
        want = oracle_mod.update_links(dims, U, sites, np.full(len(sites), mu), mode, beta, SEED, 77)
        assert lu.rel_err(got[sites, mu], want) <= TOL_D
        assert np.max(np.abs(got[sites, mu] - want)) <= TOL_D
        other = cand[coords_sum(cand) % 2 != parity]
        assert np.array_equal(got[other], U[other])
        del g, got


def test_recon12_rows_stay_orthonormal_over_many_sweeps(B):
    """12-real storage: without the re-orthonormalisation before the store the unitarity defect grows
    x1.35 per overrelaxation sweep in single precision (1e-5 -> 0.1 in 30 sweeps, measured)."""
    dims = (8, 8, 8, 16)
    g = _setup(B, dims, gen.gauge_near_identity(dims, SEED, 0.3), 1, 12)
    for k in range(6):
        B.lqcd_gauge_sweep(g, B.LQCD_HEATBATH, 5.7, SEED, 100 + k)
    p0 = B.lqcd_plaquette(g)
    for k in range(40):
        B.lqcd_gauge_sweep(g, B.LQCD_OVERRELAX, 0.0, 0, 0)
    assert _su3_defect(B.download_gauge(g)) < 5e-6
    assert abs(B.lqcd_plaquette(g) - p0) < 2e-6
