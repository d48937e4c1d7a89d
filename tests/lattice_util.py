"""Test-side helpers, written independently of both oracle/ and the CUDA path.

Lattice bookkeeping in numpy, the gamma basis retyped from DESIGN.md (reading
G4), a dense-matrix builder that follows the Kronecker-delta form of eq. 6
 literally, and plane waves for the free-field closed form.
"""
import numpy as np

# gamma basis, reading G4 (rows top to bottom)
_i = 1j
GAMMA = np.array([
    [[0, 0, 0, -_i], [0, 0, -_i, 0], [0, _i, 0, 0], [_i, 0, 0, 0]],      # gamma_x
    [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],          # gamma_y
    [[0, 0, -_i, 0], [0, 0, 0, _i], [_i, 0, 0, 0], [0, -_i, 0, 0]],      # gamma_z
    [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],            # gamma_t
], dtype=np.complex128)
GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)


def volume(dims):
    return int(np.prod(dims))


def site_coords(dims):
    """(V,4) integer coordinates of every site in lex order (x fastest)."""
    N = [int(n) for n in dims]
    s = np.arange(volume(dims))
    x0 = s % N[0]
    x1 = (s // N[0]) % N[1]
    x2 = (s // (N[0] * N[1])) % N[2]
    x3 = s // (N[0] * N[1] * N[2])
    return np.stack([x0, x1, x2, x3], axis=1)


def lex_index(dims, x):
    N = [int(n) for n in dims]
    x = np.asarray(x)
    return x[..., 0] + N[0] * (x[..., 1] + N[1] * (x[..., 2] + N[2] * x[..., 3]))


def site_parity(dims):
    return site_coords(dims).sum(axis=1) % 2


def eo_sites(dims, parity):
    """lex indices of the sites of the given parity, ordered by e = lex // 2."""
    par = site_parity(dims)
    lexs = np.nonzero(par == parity)[0]
    assert np.array_equal(lexs // 2, np.arange(len(lexs)))
    return lexs


def to_half(dims, full, parity):
    return np.ascontiguousarray(full[eo_sites(dims, parity)])


def from_halves(dims, even, odd):
    full = np.empty((volume(dims),) + even.shape[1:], dtype=even.dtype)
    full[eo_sites(dims, 0)] = even
    full[eo_sites(dims, 1)] = odd
    return full


def dense_m(dims, phases, U, kappa, mu):
    """Dense (12V x 12V) matrix of eq. 6 (reading G1: -kappa, 8 signed directions).

    Row/column index = 12*lex(x) + 3*alpha + a.  Blocks are added with +=, so
    that for N_mu = 2 the forward and backward hop to the same site both count
    (reading G8).
    """
    N = [int(n) for n in dims]
    V = volume(dims)
    X = site_coords(dims)
    M = np.zeros((12 * V, 12 * V), dtype=np.complex128)
    one4 = np.eye(4)
    diag = np.kron(one4 + 2j * kappa * mu * GAMMA5, np.eye(3))
    for s in range(V):
        x = X[s]
        M[12 * s:12 * s + 12, 12 * s:12 * s + 12] += diag
        for m in range(4):
            # forward: -kappa (1 - gamma_mu) U_mu(x) delta_{x+mu, y}
            y = x.copy()
            y[m] = (x[m] + 1) % N[m]
            sy = int(lex_index(dims, y))
            eta = phases[m] if x[m] == N[m] - 1 else 1.0
            M[12 * s:12 * s + 12, 12 * sy:12 * sy + 12] += -kappa * eta * np.kron(one4 - GAMMA[m], U[s, m])
            # backward: -kappa (1 + gamma_mu) U_mu(x-mu)^dag delta_{x-mu, y}
            y = x.copy()
            y[m] = (x[m] - 1) % N[m]
            sy = int(lex_index(dims, y))
            eta = np.conj(phases[m]) if x[m] == 0 else 1.0
            M[12 * s:12 * s + 12, 12 * sy:12 * sy + 12] += -kappa * eta * np.kron(
                one4 + GAMMA[m], U[sy, m].conj().T)
    return M


def dense_index(dims, parity):
    """Row indices of the dense matrix belonging to sites of one parity, eo ordered."""
    lexs = eo_sites(dims, parity)
    return (12 * lexs[:, None] + np.arange(12)[None, :]).reshape(-1)


def dense_mhat(dims, phases, U, kappa, mu):
    """Schur complement M_ee - M_eo M_oo^{-1} M_oe of the dense matrix (reading G3)."""
    M = dense_m(dims, phases, U, kappa, mu)
    ie, io = dense_index(dims, 0), dense_index(dims, 1)
    Mee, Meo = M[np.ix_(ie, ie)], M[np.ix_(ie, io)]
    Moe, Moo = M[np.ix_(io, ie)], M[np.ix_(io, io)]
    return Mee - Meo @ np.linalg.solve(Moo, Moe)


def momentum(dims, phases, n):
    """p_mu = (2 pi n_mu + pi theta_mu) / N_mu with phase_mu = exp(i pi theta_mu)."""
    theta = np.angle(np.asarray(phases, dtype=np.complex128)) / np.pi
    return (2.0 * np.pi * np.asarray(n, dtype=np.float64) + np.pi * theta) / np.asarray(dims, dtype=np.float64)


def plane_wave(dims, p, u):
    """psi(x) = exp(i p.x) u for a 12-vector u; returns (V,4,3)."""
    X = site_coords(dims).astype(np.float64)
    ph = np.exp(1j * (X @ p))
    return ph[:, None, None] * np.asarray(u).reshape(1, 4, 3)


def free_h(p, kappa):
    """h(p) = -2 kappa sum cos p_mu + 2 i kappa sum gamma_mu sin p_mu   (4x4, colour-diagonal)."""
    h = -2.0 * kappa * np.sum(np.cos(p)) * np.eye(4, dtype=np.complex128)
    for m in range(4):
        h = h + 2j * kappa * np.sin(p[m]) * GAMMA[m]
    return h


def apply_spin(mat4, psi):
    """(4x4 matrix acting on the Dirac index) psi[..., alpha, a]."""
    return np.einsum("ab,...bc->...ac", mat4, psi)


def apply_colour(g, psi):
    """g[site] (3x3) acting on the colour index of psi[site, alpha, a]."""
    return np.einsum("sab,sxb->sxa", g, psi)


def rel_err(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


# Gell-Mann matrices lambda^1..lambda^8 (standard order), retyped here independently of the
# oracle; the force components are taken along T^a = lambda^a / 2 (reading G16).
_s3 = 1.0 / np.sqrt(3.0)
GELL_MANN = np.array([
    [[0, 1, 0], [1, 0, 0], [0, 0, 0]],
    [[0, -_i, 0], [_i, 0, 0], [0, 0, 0]],
    [[1, 0, 0], [0, -1, 0], [0, 0, 0]],
    [[0, 0, 1], [0, 0, 0], [1, 0, 0]],
    [[0, 0, -_i], [0, 0, 0], [_i, 0, 0]],
    [[0, 0, 0], [0, 0, 1], [0, 1, 0]],
    [[0, 0, 0], [0, 0, -_i], [0, _i, 0]],
    [[_s3, 0, 0], [0, _s3, 0], [0, 0, -2 * _s3]],
], dtype=np.complex128)


def exp_i_w_T(a, w):
    """exp(i w T^a), T^a = lambda^a / 2, by eigendecomposition of the Hermitian generator."""
    ev, V = np.linalg.eigh(0.5 * GELL_MANN[a])
    return (V * np.exp(1j * w * ev)) @ V.conj().T


def algebra_matrix(F8):
    """sum_a F^a T^a for F8[..., 8] -> [..., 3, 3] (Hermitian, traceless)."""
    return 0.5 * np.einsum("...a,aij->...ij", F8, GELL_MANN)


def big_gauge(dims, small_links):
    """A gauge field for a lattice too large to generate link by link in a test: any arrangement of SU(3)
    matrices is a valid field, so link i of the big lattice is link (7919 i + 13) mod n of the seeded small
    field `small_links` (n, 3, 3).  Holds no method arithmetic; oracle and GPU are handed the same array."""
    V = volume(dims)
    idx = (np.arange(4 * V, dtype=np.int64) * 7919 + 13) % small_links.shape[0]
    return small_links[idx].reshape(V, 4, 3, 3)
