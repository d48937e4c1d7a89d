"""ctypes marshalling for oracle/lqcd_oracle.cpp -- TEST INFRASTRUCTURE ONLY.

No arithmetic of the method happens in this file: it checks shapes/dtypes,
passes pointers to the C++ oracle and returns numpy arrays in the canonical
layout (gauge (V,4,3,3), spinor (V,4,3) / (V/2,4,3), complex128).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lqcd_oracle.cpp")
_SRC_GAUGE = os.path.join(_HERE, "gauge_oracle.cpp")
_LIB = os.path.join(_HERE, "liblqcd_oracle.so")
_lib = None

_c_int_p = ctypes.POINTER(ctypes.c_int)
_c_dbl_p = ctypes.POINTER(ctypes.c_double)
_c_long_p = ctypes.POINTER(ctypes.c_long)


def build(force=False):
    """Compile the oracle with g++ (-O2, no FMA contraction, OpenMP over sites)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC),
                                                                            os.path.getmtime(_SRC_GAUGE)):
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-o", _LIB, _SRC, _SRC_GAUGE]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_cg_mdagm.restype = ctypes.c_int
        _lib.orc_bicgstab_mhat.restype = ctypes.c_int
        _lib.orc_num_threads.restype = ctypes.c_int
        _lib.orc_plaquette.restype = ctypes.c_double
    return _lib


def _dims(dims):
    d = np.ascontiguousarray(dims, dtype=np.int32)
    assert d.shape == (4,) and np.all(d >= 2) and np.all(d % 2 == 0), "extents must be even, >= 2"
    return d


def _phases(bc_phase):
    p = np.ascontiguousarray(np.asarray(bc_phase, dtype=np.complex128))
    assert p.shape == (4,)
    return p


def _c128(a, shape):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _ip(a):
    return a.ctypes.data_as(_c_int_p)


def _dp(a):
    return a.ctypes.data_as(_c_dbl_p)


def gamma(which):
    """gamma_mu for which in 0..3 (x,y,z,t), gamma5 for which == 4, as a 4x4 array."""
    out = np.zeros((4, 4), dtype=np.complex128)
    _load().orc_gamma(ctypes.c_int(which), _dp(out))
    return out


def m_full(dims, bc_phase, U, psi, kappa, mu, dagger=0):
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    psi = _c128(psi, (V, 4, 3))
    out = np.empty_like(psi)
    _load().orc_m_full(_ip(d), _dp(ph), _dp(U), _dp(psi), _dp(out), ctypes.c_double(kappa),
                       ctypes.c_double(mu), ctypes.c_int(dagger))
    return out


def dslash_eo(dims, bc_phase, U, half_in, parity, kappa, adjoint=0):
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    half_in = _c128(half_in, (V // 2, 4, 3))
    out = np.empty_like(half_in)
    _load().orc_dslash_eo(_ip(d), _dp(ph), _dp(U), _dp(half_in), _dp(out), ctypes.c_int(parity),
                          ctypes.c_double(kappa), ctypes.c_int(adjoint))
    return out


def dslash_eo_sites(dims, bc_phase, U, half_in, sites, parity, kappa, adjoint=0):
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    half_in = _c128(half_in, (V // 2, 4, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3), dtype=np.complex128)
    _load().orc_dslash_eo_sites(_ip(d), _dp(ph), _dp(U), _dp(half_in),
                                sites.ctypes.data_as(_c_long_p), ctypes.c_long(len(sites)),
                                _dp(out), ctypes.c_int(parity), ctypes.c_double(kappa),
                                ctypes.c_int(adjoint))
    return out


def mhat(dims, bc_phase, U, half_in, kappa, mu, dagger=0):
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    half_in = _c128(half_in, (V // 2, 4, 3))
    out = np.empty_like(half_in)
    _load().orc_mhat(_ip(d), _dp(ph), _dp(U), _dp(half_in), _dp(out), ctypes.c_double(kappa),
                     ctypes.c_double(mu), ctypes.c_int(dagger))
    return out


def mhat_sites(dims, bc_phase, U, half_in, sites, kappa, mu, dagger=0):
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    half_in = _c128(half_in, (V // 2, 4, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3), dtype=np.complex128)
    _load().orc_mhat_sites(_ip(d), _dp(ph), _dp(U), _dp(half_in),
                           sites.ctypes.data_as(_c_long_p), ctypes.c_long(len(sites)), _dp(out),
                           ctypes.c_double(kappa), ctypes.c_double(mu), ctypes.c_int(dagger))
    return out


def mdagm(dims, bc_phase, U, half_in, kappa, mu):
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    half_in = _c128(half_in, (V // 2, 4, 3))
    out = np.empty_like(half_in)
    _load().orc_mdagm(_ip(d), _dp(ph), _dp(U), _dp(half_in), _dp(out), ctypes.c_double(kappa),
                      ctypes.c_double(mu))
    return out


def cg_mdagm(dims, bc_phase, U, b, kappa, mu, tol, maxit):
    """Returns (status, x, iters, rel_resid_recursive, rel_resid_true)."""
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    b = _c128(b, (V // 2, 4, 3))
    x = np.empty_like(b)
    it = ctypes.c_int(0)
    rr = ctypes.c_double(0.0)
    rt = ctypes.c_double(0.0)
    st = _load().orc_cg_mdagm(_ip(d), _dp(ph), _dp(U), _dp(b), _dp(x), ctypes.c_double(kappa),
                              ctypes.c_double(mu), ctypes.c_double(tol), ctypes.c_int(maxit),
                              ctypes.byref(it), ctypes.byref(rr), ctypes.byref(rt))
    return st, x, it.value, rr.value, rt.value


def bicgstab_mhat(dims, bc_phase, U, b, kappa, mu, tol, maxit):
    """Returns (status, x, iters, rel_resid_recursive, rel_resid_true)."""
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    b = _c128(b, (V // 2, 4, 3))
    x = np.empty_like(b)
    it = ctypes.c_int(0)
    rr = ctypes.c_double(0.0)
    rt = ctypes.c_double(0.0)
    st = _load().orc_bicgstab_mhat(_ip(d), _dp(ph), _dp(U), _dp(b), _dp(x), ctypes.c_double(kappa),
                                   ctypes.c_double(mu), ctypes.c_double(tol), ctypes.c_int(maxit),
                                   ctypes.byref(it), ctypes.byref(rr), ctypes.byref(rt))
    return st, x, it.value, rr.value, rt.value


def fermion_force(dims, bc_phase, U, X, Y, kappa):
    """Outer-product force of two full-lattice spinor fields: F (V,4,8) float64."""
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    X = _c128(X, (V, 4, 3))
    Y = _c128(Y, (V, 4, 3))
    F = np.empty((V, 4, 8), dtype=np.float64)
    _load().orc_fermion_force(_ip(d), _dp(ph), _dp(U), _dp(X), _dp(Y), ctypes.c_double(kappa), _dp(F))
    return F


def fermion_force_links(dims, bc_phase, U, X, Y, sites, mus, kappa):
    """The same at the listed links (lex site, direction) only: (n,8) float64."""
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    X = _c128(X, (V, 4, 3))
    Y = _c128(Y, (V, 4, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    mus = np.ascontiguousarray(mus, dtype=np.int32)
    assert sites.shape == mus.shape
    F = np.empty((len(sites), 8), dtype=np.float64)
    _load().orc_fermion_force_links(_ip(d), _dp(ph), _dp(U), _dp(X), _dp(Y), sites.ctypes.data_as(_c_long_p),
                                    _ip(mus), ctypes.c_long(len(sites)), ctypes.c_double(kappa), _dp(F))
    return F


def force_fields(dims, bc_phase, U, X_even, kappa, mu):
    """Full-lattice (X, Y) of the even-odd force from X_e (see lqcd_oracle.cpp)."""
    d, ph = _dims(dims), _phases(bc_phase)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    X_even = _c128(X_even, (V // 2, 4, 3))
    X = np.empty((V, 4, 3), dtype=np.complex128)
    Y = np.empty_like(X)
    _load().orc_force_fields(_ip(d), _dp(ph), _dp(U), _dp(X_even), ctypes.c_double(kappa), ctypes.c_double(mu),
                             _dp(X), _dp(Y))
    return X, Y


def force_tm(dims, bc_phase, U, phi_even, kappa, mu, tol, maxit):
    """Force of S = phi^dag (Mhat^dag Mhat)^-1 phi: CG solve, force fields, outer product.
    Returns (status, F, iters)."""
    st, Xe, iters, rr, rt = cg_mdagm(dims, bc_phase, U, phi_even, kappa, mu, tol, maxit)
    X, Y = force_fields(dims, bc_phase, U, Xe, kappa, mu)
    return st, fermion_force(dims, bc_phase, U, X, Y, kappa), iters


# ----------------------------------------------------------------------------- gauge_oracle.cpp
def plaquette(dims, U):
    """Average plaquette (1/3) Re tr P over the 6 V plaquettes."""
    d = _dims(dims)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    return float(_load().orc_plaquette(_ip(d), _dp(U)))


def staple(dims, U, site, mu):
    """Staple sum A (3,3) of the link (lex site, mu): Re tr(U A) = sum over its 6 plaquettes."""
    d = _dims(dims)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    A = np.empty((3, 3), dtype=np.complex128)
    _load().orc_staple(_ip(d), _dp(U), ctypes.c_long(int(site)), ctypes.c_int(int(mu)), _dp(A))
    return A


def update_links(dims, U, sites, mus, mode, beta, seed, tag, subgroups=7):
    """Fig. 2 for the listed links, each computed from the same input field: (n,3,3)."""
    d = _dims(dims)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    mus = np.ascontiguousarray(mus, dtype=np.int32)
    assert sites.shape == mus.shape
    out = np.empty((len(sites), 3, 3), dtype=np.complex128)
    _load().orc_update_links(_ip(d), _dp(U), sites.ctypes.data_as(_c_long_p), _ip(mus), ctypes.c_long(len(sites)),
                             ctypes.c_int(mode), ctypes.c_int(subgroups), ctypes.c_double(beta),
                             ctypes.c_ulonglong(seed), ctypes.c_ulonglong(tag), _dp(out))
    return out


def gauge_subsweep(dims, U, mu, parity, mode, beta, seed, tag):
    """Update every link U_mu(x), parity(x) = parity; returns the new field (input untouched)."""
    d = _dims(dims)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3)).copy()
    _load().orc_gauge_subsweep(_ip(d), _dp(U), ctypes.c_int(mu), ctypes.c_int(parity), ctypes.c_int(mode),
                               ctypes.c_double(beta), ctypes.c_ulonglong(seed), ctypes.c_ulonglong(tag))
    return U


def gauge_sweep(dims, U, mode, beta, seed, tag):
    """One sweep (mu = 0..3, parity 0 then 1); mode 0 heatbath, 1 overrelax; returns the new field."""
    d = _dims(dims)
    V = int(np.prod(d))
    U = _c128(U, (V, 4, 3, 3)).copy()
    _load().orc_gauge_sweep(_ip(d), _dp(U), ctypes.c_int(mode), ctypes.c_double(beta), ctypes.c_ulonglong(seed),
                            ctypes.c_ulonglong(tag))
    return U


def kp_samples(lam, seed, tag, n):
    """n Kennedy-Pendleton samples: (g (n,4), attempts (n,)); attempts 0 = all rejected."""
    g = np.empty((n, 4), dtype=np.float64)
    att = np.empty(n, dtype=np.int32)
    _load().orc_kp_samples(ctypes.c_double(lam), ctypes.c_ulonglong(seed), ctypes.c_ulonglong(tag), ctypes.c_long(n),
                           _dp(g), _ip(att))
    return g, att


def num_threads():
    return int(_load().orc_num_threads())


def set_num_threads(n):
    """Threads of the oracle's OpenMP loops over independent sites (n <= 0: the default); returns the count in force."""
    lib = _load()
    lib.orc_set_num_threads.restype = ctypes.c_int
    return int(lib.orc_set_num_threads(ctypes.c_int(int(n))))
