"""Independent numpy brute force used to PIN the oracle (tests only; shares no code with oracle/ or the
CUDA library).  Everything here is typed from the definitions in SURVEY.md §8(c) O1-O6:

  * gamma matrices typed entry by entry (chiral basis, O2), sigma_{mu nu} from the closed-form
    (upper, lower) Pauli blocks listed in O2 -- NOT from commutators as the oracle does;
  * clover leaves by np.roll shifts of whole link fields (O4) -- NOT by per-site index arithmetic;
  * the dense matrix M filled entry block by entry block with `+=` so coinciding neighbours on
    extent-2 lattices accumulate (O1, O3, O5).
"""
import numpy as np

I = 1j
GAMMA = np.array([
    [[0, 0, 0, -I], [0, 0, -I, 0], [0, I, 0, 0], [I, 0, 0, 0]],      # gamma_x
    [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],      # gamma_y
    [[0, 0, -I, 0], [0, 0, 0, I], [I, 0, 0, 0], [0, -I, 0, 0]],      # gamma_z
    [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],        # gamma_t
], dtype=np.complex128)
GAMMA5 = np.diag([1, 1, -1, -1]).astype(np.complex128)

S1 = np.array([[0, 1], [1, 0]], dtype=np.complex128)
S2 = np.array([[0, -I], [I, 0]], dtype=np.complex128)
S3 = np.array([[1, 0], [0, -1]], dtype=np.complex128)


def _bd(up, lo):
    z = np.zeros((4, 4), dtype=np.complex128)
    z[:2, :2] = up
    z[2:, 2:] = lo
    return z


# sigma_{mu nu} = (i/2)[gamma_mu, gamma_nu], (upper, lower) blocks as listed in SURVEY O2
SIGMA = {
    (0, 1): _bd(-S3, -S3),
    (0, 2): _bd(+S2, +S2),
    (0, 3): _bd(+S1, -S1),
    (1, 2): _bd(-S1, -S1),
    (1, 3): _bd(+S2, -S2),
    (2, 3): _bd(+S3, -S3),
}

_AXIS = {0: 3, 1: 2, 2: 1, 3: 0}  # mu -> axis of [t][z][y][x]


def shift(f, mu, d):
    """Field at x + d*mu^ (periodic)."""
    return np.roll(f, -d, axis=_AXIS[mu])


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def field_strength(U, mu, nu, trace_sub=True):
    """F_{mu nu}(x) on the whole lattice, [t][z][y][x][3][3] (O4)."""
    Um, Un = U[..., mu, :, :], U[..., nu, :, :]
    l1 = Um @ shift(Un, mu, 1) @ dag(shift(Um, nu, 1)) @ dag(Un)
    l2 = Un @ dag(shift(shift(Um, mu, -1), nu, 1)) @ dag(shift(Un, mu, -1)) @ shift(Um, mu, -1)
    l3 = dag(shift(Um, mu, -1)) @ dag(shift(shift(Un, mu, -1), nu, -1)) @ shift(shift(Um, mu, -1), nu, -1) @ shift(Un, nu, -1)
    l4 = dag(shift(Un, nu, -1)) @ shift(Um, nu, -1) @ shift(shift(Un, mu, 1), nu, -1) @ dag(Um)
    Q = l1 + l2 + l3 + l4
    G = (Q - dag(Q)) / 8.0
    if trace_sub:
        tr = np.einsum("...ii->...", G) / 3.0
        G = G - tr[..., None, None] * np.eye(3)
    return -I * G


def clover_blocks(U, kappa, csw, trace_sub=True):
    """A(x) = 1 - kappa*csw*sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x), [t][z][y][x][12][12]."""
    shape = U.shape[:4]
    A = np.zeros(shape + (12, 12), dtype=np.complex128)
    A[...] = np.eye(12)
    for (mu, nu), sig in SIGMA.items():
        F = field_strength(U, mu, nu, trace_sub)
        A -= kappa * csw * np.einsum("st,...ab->...satb", sig, F).reshape(shape + (12, 12))
    return A


def dense_M(dims, bc, U, kappa, csw, trace_sub=True):
    """Dense 12V x 12V matrix of M = A - kappa*D, filled block by block (O3, O5)."""
    lx, ly, lz, lt = dims
    L = (lx, ly, lz, lt)
    V = lx * ly * lz * lt
    A = clover_blocks(U, kappa, csw, trace_sub).reshape(V, 12, 12)
    Uf = U.reshape(V, 4, 3, 3)
    M = np.zeros((12 * V, 12 * V), dtype=np.complex128)
    one = np.eye(4)

    def idx(x):
        return x[0] + lx * (x[1] + ly * (x[2] + lz * x[3]))

    for t in range(lt):
        for z in range(lz):
            for y in range(ly):
                for x in range(lx):
                    c = [x, y, z, t]
                    i = idx(c)
                    M[12 * i:12 * i + 12, 12 * i:12 * i + 12] += A[i]
                    for mu in range(4):
                        f = list(c)
                        f[mu] = (c[mu] + 1) % L[mu]
                        j = idx(f)
                        eta = bc[mu] if c[mu] == L[mu] - 1 else 1
                        M[12 * i:12 * i + 12, 12 * j:12 * j + 12] += -kappa * eta * np.kron(one - GAMMA[mu], Uf[i, mu])
                        b = list(c)
                        b[mu] = (c[mu] - 1) % L[mu]
                        j = idx(b)
                        eta = bc[mu] if c[mu] == 0 else 1
                        M[12 * i:12 * i + 12, 12 * j:12 * j + 12] += -kappa * eta * np.kron(one + GAMMA[mu], Uf[j, mu].conj().T)
    return M


def parity_of_sites(dims):
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    return ((x + y + z + t) & 1).reshape(-1)


def dense_schur(dims, M):
    """S = M_ee - M_eo M_oo^{-1} M_oe from the dense M (O6); returns (S, even component indices)."""
    par = np.repeat(parity_of_sites(dims), 12)
    e = np.where(par == 0)[0]
    o = np.where(par == 1)[0]
    Mee, Meo, Moe, Moo = M[np.ix_(e, e)], M[np.ix_(e, o)], M[np.ix_(o, e)], M[np.ix_(o, o)]
    return Mee - Meo @ np.linalg.solve(Moo, Moe), e, o
