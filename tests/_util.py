"""Test-side helpers written independently of oracle/ and of the CUDA path.

Gamma matrices here are built from Pauli matrices (a second statement of the
DeGrand-Rossi convention of SURVEY.md 8(c)), not copied from the oracle.
"""
import numpy as np

S1 = np.array([[0, 1], [1, 0]], dtype=complex)
S2 = np.array([[0, -1j], [1j, 0]], dtype=complex)
S3 = np.array([[1, 0], [0, -1]], dtype=complex)
Z2 = np.zeros((2, 2), dtype=complex)
I2 = np.eye(2, dtype=complex)


def pauli_gammas():
    """DeGrand-Rossi: gamma_k = [[0, i e_k sigma_k], [-i e_k sigma_k, 0]], e = (+,-,+); gamma_t offdiag 1."""
    g = []
    for sig, e in ((S1, 1), (S2, -1), (S3, 1)):
        g.append(np.block([[Z2, 1j * e * sig], [-1j * e * sig, Z2]]))
    g.append(np.block([[Z2, I2], [I2, Z2]]))
    return g


GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(complex)


def cplx(a):
    """(..., 2) real array -> complex array."""
    return a[..., 0] + 1j * a[..., 1]


def reals(z, dtype=np.float64):
    """complex array -> (..., 2) real array."""
    return np.ascontiguousarray(np.stack([z.real, z.imag], axis=-1).astype(dtype))


def coords(dims):
    """(V4, 4) integer coordinates in lexicographic order, x0 fastest."""
    L0, L1, L2, L3 = dims
    x = np.arange(L0 * L1 * L2 * L3)
    return np.stack([x % L0, (x // L0) % L1, (x // (L0 * L1)) % L2, x // (L0 * L1 * L2)], axis=1)


def lex(dims, c):
    L0, L1, L2, L3 = dims
    return c[..., 0] + L0 * (c[..., 1] + L1 * (c[..., 2] + L2 * c[..., 3]))


def shift_index(dims, mu, step):
    """index array n with n[x] = lex(x + step*mu_hat) (periodic)."""
    c = coords(dims).copy()
    c[:, mu] = (c[:, mu] + step) % dims[mu]
    return lex(dims, c)


def rel_err(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def dense_dhop_matrix(dims, U, antiperiodic_t):
    """Brute-force D = sum_mu [(1-g_mu) (x) W_mu + (1+g_mu) (x) W_mu^dag], index (spin, site, colour).

    W_mu has the block sign*U_mu(x) at (x, x+mu_hat); the backward term appears only as the
    matrix adjoint, never coded by hand (pin P1 of SURVEY.md 8(c))."""
    V = int(np.prod(dims))
    Uc = cplx(U.astype(np.float64)).reshape(V, 4, 3, 3)
    g = pauli_gammas()
    c = coords(dims)
    D = np.zeros((4 * 3 * V, 4 * 3 * V), dtype=complex)
    one = np.eye(4, dtype=complex)
    for mu in range(4):
        W = np.zeros((3 * V, 3 * V), dtype=complex)
        nb = shift_index(dims, mu, +1)
        for x in range(V):
            wrap = mu == 3 and c[x, 3] == dims[3] - 1
            sign = (-1.0 if antiperiodic_t == 1 else 0.0 if antiperiodic_t == 2 else 1.0) if wrap else 1.0      # 2: open time boundary
            W[3 * x:3 * x + 3, 3 * nb[x]:3 * nb[x] + 3] += sign * Uc[x, mu]
        D += np.kron(one - g[mu], W) + np.kron(one + g[mu], W.conj().T)
    return D


def apply_dense(D, psi):
    """psi canonical (V, Ls, 4, 3, 2) -> D applied slice by slice, same layout, fp64."""
    z = cplx(psi.astype(np.float64))            # (V, Ls, 4, 3)
    V, Ls = z.shape[:2]
    out = np.empty_like(z)
    for s in range(Ls):
        v = z[:, s].transpose(1, 0, 2).reshape(-1)      # (spin, site, colour)
        out[:, s] = (D @ v).reshape(4, V, 3).transpose(1, 0, 2)
    return reals(out)
