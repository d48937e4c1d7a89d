"""Out-of-bounds and uninitialised-read checks of every kernel through the C ABI (-m gpu).

compute-sanitizer is closed on this GPU pool, so the memory checks are our own: every device
buffer the tests hand to the library is the middle of a larger allocation whose two guard regions
(and the buffer itself) are pre-filled with 0xFF bytes -- a NaN in double and in single precision.

  * a store outside a buffer changes a guard byte            -> `check()` fails;
  * a load outside a buffer, or of an output element that was never written (pad sites of the
    ragged last group of 32, workspace the caller owns), that reaches a result makes it NaN
                                                              -> the parity / finiteness asserts fail.

Lattices are chosen for ragged tails: 6^4 has V/2 = 648 = 20 groups of 32 + 8 sites, 2^4 has 8 sites
(a quarter of one group), 6x4x10x4 fills 15 groups exactly (not a multiple of the 128-thread CTA).
"""
import numpy as np
import pytest

import lattice_util as lu
import lqcd_inputs as gen

pytestmark = pytest.mark.gpu

GUARD = 1 << 16          # bytes on each side; a multiple of 256 keeps the buffer's alignment
SEED = gen.BASE_SEED
PH = np.exp(1j * np.pi * np.array([0.3, 0.0, 1.0, 0.5]))
DIMS = [(6, 6, 6, 6), (2, 2, 2, 2), (6, 4, 10, 4)]
FORMATS = [(0, 18, 1e-13), (0, 12, 1e-13), (1, 18, 1e-5), (1, 12, 1e-5)]


@pytest.fixture()
def G():
    """The binding with alloc_gauge / alloc_spinor / alloc_force replaced by guarded allocations."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1209_5942_b200.binding as B

    class Guarded:
        def __init__(self):
            self.B = B
            self.bufs = []
            self.saved = (B.alloc_gauge, B.alloc_spinor, B.alloc_force)
            B.alloc_gauge = lambda device="cuda": self._alloc(B.lqcd_gauge_bytes(), device)
            B.alloc_spinor = lambda device="cuda": self._alloc(B.lqcd_spinor_bytes(), device)
            B.alloc_force = lambda device="cuda": self._alloc(B.lqcd_force_bytes(), device)

        def _alloc(self, nbytes, device):
            full = torch.full((nbytes + 2 * GUARD,), 0xFF, dtype=torch.uint8, device=device)
            self.bufs.append((full, nbytes))
            return full[GUARD:GUARD + nbytes]

        def check(self):
            torch.cuda.synchronize()
            for full, nbytes in self.bufs:
                assert bool((full[:GUARD] == 0xFF).all()), "store below a device buffer"
                assert bool((full[GUARD + nbytes:] == 0xFF).all()), "store above a device buffer"
            return len(self.bufs)

        def restore(self):
            B.alloc_gauge, B.alloc_spinor, B.alloc_force = self.saved

    g = Guarded()
    yield g
    g.restore()


def _round(a, precision):
    return a if precision == 0 else a.astype(np.complex64).astype(np.complex128)


def _finite(*arrays):
    for a in arrays:
        assert np.isfinite(a).all(), "NaN / inf in a result: out-of-bounds or uninitialised read"


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision,recon,tol", FORMATS)
def test_operator_calls_stay_inside_their_buffers(G, oracle_mod, dims, precision, recon, tol):
    B = G.B
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    Vh = V // 2
    U = gen.gauge_haar(dims, SEED)
    x = gen.spinor_gaussian(Vh, SEED)
    y = gen.spinor_gaussian(Vh, SEED, 9)
    Ur, xr, yr = _round(U, precision), _round(x, precision), _round(y, precision)
    B.lqcd_init(dims, PH)
    B.lqcd_set_format(precision, recon)
    B.lqcd_set_stream()
    g = B.upload_gauge(U)
    for parity in (0, 1):
        s, o = B.upload_spinor(x, 1 - parity), B.alloc_spinor()
        B.lqcd_dslash_eo(g, s, o, parity, kappa)
        got = B.download_spinor(o, parity)
        _finite(got)
        assert lu.rel_err(got, oracle_mod.dslash_eo(dims, PH, Ur, xr, parity, kappa)) <= tol
    s = B.upload_spinor(x, 0)
    for dagger in (0, 1):
        o = B.alloc_spinor()
        B.lqcd_mtm(g, s, o, kappa, mu, dagger)
        got = B.download_spinor(o, 0)
        _finite(got)
        assert lu.rel_err(got, oracle_mod.mhat(dims, PH, Ur, xr, kappa, mu, dagger)) <= tol
    so, oe, oo = B.upload_spinor(y, 1), B.alloc_spinor(), B.alloc_spinor()
    B.lqcd_mtm_full(g, s, so, oe, oo, kappa, mu)
    got = lu.from_halves(dims, B.download_spinor(oe, 0), B.download_spinor(oo, 1))
    _finite(got)
    assert lu.rel_err(got, oracle_mod.m_full(dims, PH, Ur, lu.from_halves(dims, xr, yr), kappa, mu)) <= tol
    _finite(B.download_gauge(g))
    assert G.check() >= 8


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision,recon", [(0, 18), (0, 12), (1, 12)])
def test_solver_calls_stay_inside_their_buffers(G, oracle_mod, dims, precision, recon):
    B = G.B
    kappa, mu = 0.15, 0.1
    tol = 1e-10 if precision == 0 else 1e-5
    Vh = lu.volume(dims) // 2
    U = gen.gauge_haar(dims, SEED)
    b = gen.spinor_gaussian(Vh, SEED, gen.STREAM_SOURCE)
    eta_o = gen.spinor_gaussian(Vh, SEED, 11)
    B.lqcd_init(dims, PH)
    B.lqcd_set_format(precision, recon)
    B.lqcd_set_stream()
    g = B.upload_gauge(U)
    s = B.upload_spinor(b, 0)
    x = B.alloc_spinor()
    assert B.lqcd_cg_mdagm(g, s, x, kappa, mu, tol, 500) == 0
    xs = B.download_spinor(x, 0)
    _finite(xs)
    assert lu.rel_err(oracle_mod.mdagm(dims, PH, U, xs, kappa, mu), b) <= (1.05 * tol if precision == 0 else 1e-3)
    x2 = B.alloc_spinor()
    assert B.lqcd_bicgstab_mhat(g, s, x2, kappa, mu, tol, 500) == 0
    xb = B.download_spinor(x2, 0)
    _finite(xb)
    assert lu.rel_err(oracle_mod.mhat(dims, PH, U, xb, kappa, mu, 0), b) <= (1.05 * tol if precision == 0 else 1e-3)
    so, pe, po = B.upload_spinor(eta_o, 1), B.alloc_spinor(), B.alloc_spinor()
    assert B.lqcd_solve_full(g, s, so, pe, po, kappa, mu, tol, 500) == 0
    _finite(B.download_spinor(pe, 0), B.download_spinor(po, 1))
    if precision == 0:
        B.lqcd_set_format(1, 12)
        gs = B.upload_gauge(U)
        B.lqcd_set_format(precision, recon)
        xm = B.alloc_spinor()
        assert B.lqcd_cg_mdagm_mixed(g, recon, gs, 12, s, xm, kappa, mu, 1e-10, 2000, 0.0) == 0
        got = B.download_spinor(xm, 0)
        _finite(got)
        assert lu.rel_err(oracle_mod.mdagm(dims, PH, U, got, kappa, mu), b) <= 1.05e-10
    assert G.check() >= 7


@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("precision,recon,tol", FORMATS)
def test_force_and_gauge_update_stay_inside_their_buffers(G, oracle_mod, dims, precision, recon, tol):
    B = G.B
    kappa, mu = 0.15, 0.1
    V = lu.volume(dims)
    U = gen.gauge_haar(dims, SEED)
    X, Y = gen.spinor_gaussian(V, SEED, 7), gen.spinor_gaussian(V, SEED, 8)
    Ur, Xr, Yr = _round(U, precision), _round(X, precision), _round(Y, precision)
    B.lqcd_init(dims, PH)
    B.lqcd_set_format(precision, recon)
    B.lqcd_set_stream()
    g = B.upload_gauge(U)
    xe, xo = B.upload_spinor(lu.to_half(dims, X, 0), 0), B.upload_spinor(lu.to_half(dims, X, 1), 1)
    ye, yo = B.upload_spinor(lu.to_half(dims, Y, 0), 0), B.upload_spinor(lu.to_half(dims, Y, 1), 1)
    f = B.alloc_force()
    B.lqcd_fermion_force(g, xe, xo, ye, yo, f, kappa)
    got = B.download_force(f)
    _finite(got)
    assert lu.rel_err(got, oracle_mod.fermion_force(dims, PH, Ur, Xr, Yr, kappa)) <= tol
    f2 = B.alloc_force()
    assert B.lqcd_force_tm(g, xe, f2, kappa, mu, 1e-10 if precision == 0 else 1e-5, 500) == 0
    _finite(B.download_force(f2))
    p0 = B.lqcd_plaquette(g)
    assert abs(p0 - oracle_mod.plaquette(dims, Ur)) <= (1e-13 if precision == 0 else 1e-6)
    B.lqcd_gauge_sweep(g, B.LQCD_OVERRELAX, 0.0, SEED, 1)
    assert abs(B.lqcd_plaquette(g) - p0) <= (1e-13 if precision == 0 else 1e-5)
    B.lqcd_gauge_sweep(g, B.LQCD_HEATBATH, 5.7, SEED, 2)
    Un = B.download_gauge(g)
    _finite(Un)
    if precision == 0 and recon == 18:
        want = oracle_mod.gauge_sweep(dims, oracle_mod.gauge_sweep(dims, U, 1, 0.0, SEED, 1), 0, 5.7, SEED, 2)
        assert lu.rel_err(Un, want) <= 1e-11
    assert G.check() >= 7
