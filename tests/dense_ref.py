"""Independent dense (numpy) statement of the operators, used ONLY to pin the oracle.

Shares nothing with oracle/tm_oracle.c: gamma matrices come from Kronecker products of
Pauli matrices, the operator is assembled as an explicit (12V x 12V) matrix from shift
(permutation) matrices, and inverses are numpy LU.  Index convention of the flattened
canonical arrays: row = ((site*4 + spin)*3 + colour), site = ((t*Lz+z)*Ly+y)*Lx+x.
"""
import numpy as np

_s0 = np.eye(2, dtype=complex)
_sx = np.array([[0, 1], [1, 0]], dtype=complex)
_sy = np.array([[0, -1j], [1j, 0]], dtype=complex)
_sz = np.array([[1, 0], [0, -1]], dtype=complex)

# reading 2: g_k = sigma_y (x) sigma_k, g_t = sigma_x (x) 1
GAMMA = [np.kron(_sy, _sx), np.kron(_sy, _sy), np.kron(_sy, _sz), np.kron(_sx, _s0)]
GAMMA5 = GAMMA[0] @ GAMMA[1] @ GAMMA[2] @ GAMMA[3]


def big_gamma(n):
    g = np.eye(4, dtype=complex)
    for m in range(4):
        if (n >> m) & 1:
            g = g @ GAMMA[m]
    return g


def _site(dims, c):
    lx, ly, lz, lt = dims
    return ((c[3] * lz + c[2]) * ly + c[1]) * lx + c[0]


def hop_blocks(U, dims, tb):
    """Return (F, B): lists over mu of (V*3 x V*3) colour-site matrices with
    F[mu][x,a; x+mu,b] = sign * U_mu(x)[a,b] and B[mu][x,a; x-mu,b] = sign * conj(U_mu(x-mu)[b,a]).
    Entries ADD when forward and backward neighbours coincide (L = 2)."""
    lx, ly, lz, lt = dims
    V = lx * ly * lz * lt
    Uf = np.asarray(U).reshape(V, 4, 3, 3)
    F = [np.zeros((V * 3, V * 3), dtype=complex) for _ in range(4)]
    B = [np.zeros((V * 3, V * 3), dtype=complex) for _ in range(4)]
    for t in range(lt):
        for z in range(lz):
            for y in range(ly):
                for x in range(lx):
                    c = [x, y, z, t]
                    s = _site(dims, c)
                    for m in range(4):
                        cp = list(c)
                        cp[m] += 1
                        sg = 1.0
                        if cp[m] == dims[m]:
                            cp[m] = 0
                            if m == 3:
                                sg = tb
                        sp = _site(dims, cp)
                        F[m][s * 3:s * 3 + 3, sp * 3:sp * 3 + 3] += sg * Uf[s, m]
                        B[m][sp * 3:sp * 3 + 3, s * 3:s * 3 + 3] += sg * Uf[s, m].conj().T
    return F, B


def _spin_colour(Asc, G, V):
    """(site,colour) matrix Asc and 4x4 spin matrix G -> (site,spin,colour) matrix."""
    A4 = Asc.reshape(V, 3, V, 3)
    out = np.einsum("xayb,st->xsaytb", A4, G)
    return out.reshape(V * 12, V * 12)


def dense_M(U, dims, kappa, mu, tb=-1):
    """M = 1 + 2 i kappa mu g5 - kappa sum_mu[(1-g_mu) F_mu + (1+g_mu) B_mu]  (BASELINE north_star)."""
    V = int(np.prod(dims))
    F, B = hop_blocks(U, dims, tb)
    one = np.eye(4)
    M = np.eye(V * 12, dtype=complex)
    M += 2j * kappa * mu * np.kron(np.eye(V), np.kron(GAMMA5, np.eye(3)))
    for m in range(4):
        M -= kappa * (_spin_colour(F[m], one - GAMMA[m], V) + _spin_colour(B[m], one + GAMMA[m], V))
    return M


def dense_cov_deriv(U, dims, m, tb=-1):
    """D_m = (F_m - B_m)/2 as a (site,spin,colour) matrix."""
    V = int(np.prod(dims))
    F, B = hop_blocks(U, dims, tb)
    return _spin_colour(0.5 * (F[m] - B[m]), np.eye(4), V)
