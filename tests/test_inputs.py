"""Seeded input generators: structure of the synthetic workloads (DESIGN.md input recipe)."""
import numpy as np

import lqcd_inputs as gen


def _is_su3(U, tol=1e-13):
    n = U.reshape(-1, 3, 3)
    eye = np.eye(3)
    assert np.max(np.abs(np.einsum("nab,ncb->nac", n, n.conj()) - eye)) < tol
    assert np.max(np.abs(np.linalg.det(n) - 1.0)) < tol


def test_haar_links_are_su3_and_deterministic():
    dims = (4, 4, 4, 4)
    U = gen.gauge_haar(dims, 123)
    assert U.shape == (256, 4, 3, 3) and U.dtype == np.complex128
    _is_su3(U)
    assert np.array_equal(U, gen.gauge_haar(dims, 123))
    assert not np.array_equal(U, gen.gauge_haar(dims, 124))
    # counter based: a sub-range regenerates alone
    sub = gen.su3_haar(40, 123, gen.STREAM_GAUGE, first=100)
    assert np.array_equal(sub, U.reshape(-1, 3, 3)[100:140])


def test_haar_moments():
    U = gen.su3_haar(20000, 5, gen.STREAM_GTRANS)
    # Haar: E[U_ab] = 0, E[|U_ab|^2] = 1/3, E[|tr U|^2] = 1
    assert np.max(np.abs(U.mean(axis=0))) < 0.02
    assert np.max(np.abs((np.abs(U) ** 2).mean(axis=0) - 1.0 / 3.0)) < 0.01
    tr = np.trace(U, axis1=1, axis2=2)
    assert abs((np.abs(tr) ** 2).mean() - 1.0) < 0.05


def test_near_identity_links():
    dims = (4, 4, 4, 4)
    U = gen.gauge_near_identity(dims, 123, eps=0.3)
    _is_su3(U)
    tr = np.trace(U.reshape(-1, 3, 3), axis1=1, axis2=2).real / 3.0
    assert 0.85 < tr.mean() < 0.99   # close to, but not at, the identity
    U0 = gen.gauge_near_identity(dims, 123, eps=0.0)
    assert np.allclose(U0, gen.gauge_unit(dims), atol=1e-15)


def test_gaussian_spinors():
    s = gen.spinor_gaussian(50000, 9)
    assert s.shape == (50000, 4, 3)
    assert abs(s.real.mean()) < 0.01 and abs(s.imag.mean()) < 0.01
    assert abs(s.real.var() - 1.0) < 0.01 and abs(s.imag.var() - 1.0) < 0.01
    assert abs(np.mean(s.real * s.imag)) < 0.01
    assert np.array_equal(s[:10], gen.spinor_gaussian(10, 9))
    assert not np.array_equal(gen.spinor_gaussian(10, 9, gen.STREAM_SOURCE), s[:10])
