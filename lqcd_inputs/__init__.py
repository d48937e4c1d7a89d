"""Seeded synthetic inputs shared by the oracle tests and the CUDA path's tests/bench.

This module holds NONE of the method's arithmetic (no gamma matrices, no
stencil, no lattice indexing): it only draws random fields in the canonical
interchange layout

    gauge   (V, 4, 3, 3) complex128   U[lex(x)][mu][a][b]
    spinor  (n, 4, 3)    complex128   psi[site][alpha][a]

Recipe (stands in for the paper's "prior generated"
beta = 3.9 configurations, which do not exist here):

* RNG: counter based.  u64 = splitmix64_mix(seed * 0x9E3779B97F4A7C15
  + stream * 2^40 + counter); uniform in (0, 1] from the top 53 bits; two
  uniforms -> Box-Muller -> one complex Gaussian (independent N(0,1) real and
  imaginary parts).  Every element's counter is a fixed function of its
  (site, mu, row, col) position, so any site subset can be regenerated alone.
* Haar SU(3) link: 3x3 complex Gaussian; rows 0, 1 by classical Gram-Schmidt;
  row 2 = conj(row0 x row1)  (Gram-Schmidt of the third row with the
  determinant phase removed).
* Near-identity link: G complex Gaussian, H = (G + G^dag)/2 - tr/3,
  U = exp(i eps H) by Taylor series, then re-unitarised as above.
* Spinors: 12 complex Gaussians per site.

Streams: 1 gauge, 2 input spinor, 3 CG source, 4 gauge transformation g(x),
5 near-identity H, 6+ free for tests.
"""
import numpy as np

BASE_SEED = 12095942
STREAM_GAUGE, STREAM_SPINOR, STREAM_SOURCE, STREAM_GTRANS, STREAM_NEARID = 1, 2, 3, 4, 5

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_CHUNK = 1 << 20  # complex numbers generated per chunk (bounds temporaries)


def _mix(z):
    """splitmix64 output function on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = z + _GOLD
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def _uniform(seed, stream, counter):
    """Uniform in (0, 1] for each uint64 counter."""
    with np.errstate(over="ignore"):
        base = np.uint64(seed) * _GOLD + (np.uint64(stream) << np.uint64(40))
        bits = _mix(base + counter)
    return ((bits >> np.uint64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)


def complex_gaussian(seed, stream, first, count):
    """`count` complex Gaussians with element indices first .. first+count-1."""
    out = np.empty(count, dtype=np.complex128)
    for lo in range(0, count, _CHUNK):
        hi = min(count, lo + _CHUNK)
        idx = np.arange(first + lo, first + hi, dtype=np.uint64)
        u1 = _uniform(seed, stream, idx * np.uint64(2))
        u2 = _uniform(seed, stream, idx * np.uint64(2) + np.uint64(1))
        r = np.sqrt(-2.0 * np.log(u1))
        th = (2.0 * np.pi) * u2
        out[lo:hi] = r * np.cos(th) + 1j * (r * np.sin(th))
    return out


def _unitarise(G):
    """(n,3,3) complex -> SU(3): Gram-Schmidt rows 0,1; row 2 = conj(row0 x row1)."""
    a = G[:, 0, :]
    a = a / np.linalg.norm(a, axis=1, keepdims=True)
    b = G[:, 1, :]
    b = b - a * np.sum(np.conj(a) * b, axis=1, keepdims=True)
    b = b / np.linalg.norm(b, axis=1, keepdims=True)
    c = np.conj(np.cross(a, b))
    return np.stack([a, b, c], axis=1)


def su3_haar(n, seed, stream, first=0):
    """n Haar-random SU(3) matrices, matrix k built from element indices 9(first+k) .. +8."""
    out = np.empty((n, 3, 3), dtype=np.complex128)
    step = _CHUNK // 9
    for lo in range(0, n, step):
        hi = min(n, lo + step)
        G = complex_gaussian(seed, stream, 9 * (first + lo), 9 * (hi - lo)).reshape(-1, 3, 3)
        out[lo:hi] = _unitarise(G)
    return out


def gauge_haar(dims, seed=BASE_SEED):
    V = int(np.prod(dims))
    return su3_haar(4 * V, seed, STREAM_GAUGE).reshape(V, 4, 3, 3)


def gauge_unit(dims):
    V = int(np.prod(dims))
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    U[:, :, 0, 0] = U[:, :, 1, 1] = U[:, :, 2, 2] = 1.0
    return U


def gauge_near_identity(dims, seed=BASE_SEED, eps=0.3):
    """U = exp(i eps H), H Gaussian traceless Hermitian; resembles a thermalised field."""
    V = int(np.prod(dims))
    n = 4 * V
    out = np.empty((n, 3, 3), dtype=np.complex128)
    step = _CHUNK // 9
    eye = np.eye(3, dtype=np.complex128)
    for lo in range(0, n, step):
        hi = min(n, lo + step)
        G = complex_gaussian(seed, STREAM_NEARID, 9 * lo, 9 * (hi - lo)).reshape(-1, 3, 3)
        H = 0.5 * (G + np.conj(np.swapaxes(G, 1, 2)))
        H = H - (np.trace(H, axis1=1, axis2=2) / 3.0)[:, None, None] * eye
        X = (1j * eps) * H
        term = np.broadcast_to(eye, X.shape).copy()
        acc = term.copy()
        for k in range(1, 40):
            term = np.matmul(term, X) / k
            acc += term
            if np.max(np.abs(term)) < 1e-18:
                break
        out[lo:hi] = _unitarise(acc)
    return out.reshape(V, 4, 3, 3)


def spinor_gaussian(n_sites, seed=BASE_SEED, stream=STREAM_SPINOR):
    return complex_gaussian(seed, stream, 0, 12 * n_sites).reshape(n_sites, 4, 3)


def antiperiodic_t():
    """Boundary phases e^{i pi theta_mu}: periodic in space, antiperiodic in time."""
    return np.array([1.0, 1.0, 1.0, -1.0], dtype=np.complex128)
