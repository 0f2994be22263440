"""Independent numpy restatements of textbook lattice quantities, used ONLY to pin the oracle.

Nothing here is shared with oracle/ or the CUDA path: whole-lattice array expressions with np.roll replace
the oracle's per-site index arithmetic, so an indexing, sign or transposition slip in the oracle shows up
as a disagreement.  Canonical layout: U[s, mu, r, c], s = x + Nx (y + Ny (z + Nz t)).
"""
import numpy as np

PAULI = np.array(
    [
        [[1, 0], [0, 1]],
        [[0, 1], [1, 0]],
        [[0, -1j], [1j, 0]],
        [[1, 0], [0, -1]],
    ],
    dtype=np.complex128,
)


def as_grid(U, dims):
    """(V,4,3,3) -> (Nt,Nz,Ny,Nx,4,3,3) view; direction mu lives on axis 3-mu."""
    Nx, Ny, Nz, Nt = dims
    return U.reshape(Nt, Nz, Ny, Nx, 4, 3, 3)


def shift(A, mu, step):
    """A(x) -> A(x + step*mu_hat) with periodic wrap (grid array, axis 3-mu)."""
    return np.roll(A, -step, axis=3 - mu)


def dag(A):
    return np.conj(np.swapaxes(A, -1, -2))


def plaquette(U, dims):
    G = as_grid(U, dims)
    acc = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Umu, Unu = G[..., mu, :, :], G[..., nu, :, :]
            P = Umu @ shift(Unu, mu, 1) @ dag(shift(Umu, nu, 1)) @ dag(Unu)
            acc += np.trace(P, axis1=-2, axis2=-1).real.sum()
    V = dims[0] * dims[1] * dims[2] * dims[3]
    return acc / (6 * 3 * V)


def functional(U, dims, nd=4):
    V = dims[0] * dims[1] * dims[2] * dims[3]
    return np.trace(U[:, :nd], axis1=-2, axis2=-1).real.sum() / (3 * nd * V)


def theta_from_A(U, dims, nd=4):
    """eq. 2.5 with the standard lattice definition: A_mu = [(U - U^dag)/(2i)]_traceless,
    Delta(x) = sum_mu [A_mu(x) - A_mu(x - mu)].  Returns per-site tr[Delta Delta^dag] as a grid."""
    G = as_grid(U, dims)
    eye = np.eye(3)
    Delta = 0
    for mu in range(nd):
        Umu = G[..., mu, :, :]
        A = (Umu - dag(Umu)) / 2j
        A = A - np.trace(A, axis1=-2, axis2=-1)[..., None, None] * eye / 3
        Delta = Delta + A - shift(A, mu, -1)
    return (np.abs(Delta) ** 2).sum(axis=(-1, -2))


def K_field(U, dims, nd=4):
    G = as_grid(U, dims)
    K = 0
    for mu in range(nd):
        Umu = G[..., mu, :, :]
        K = K + Umu + dag(shift(Umu, mu, -1))
    return K  # grid (Nt,Nz,Ny,Nx,3,3)


def quat_to_su2(q):
    """q0 + i (q1 s1 + q2 s2 + q3 s3) with explicit Pauli matrices (vectorised over leading axes)."""
    q = np.asarray(q, dtype=np.float64)
    return (
        q[..., 0, None, None] * PAULI[0]
        + 1j * (q[..., 1, None, None] * PAULI[1] + q[..., 2, None, None] * PAULI[2] + q[..., 3, None, None] * PAULI[3])
    )


def embed(q, i, j):
    m = quat_to_su2(q)
    G = np.eye(3, dtype=np.complex128)
    G[i, i], G[i, j], G[j, i], G[j, j] = m[0, 0], m[0, 1], m[1, 0], m[1, 1]
    return G


def gauge_transform(U, dims, g):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu)^dag, eq. 1.1; g is (V,3,3)."""
    Nx, Ny, Nz, Nt = dims
    G = as_grid(U, dims)
    gg = g.reshape(Nt, Nz, Ny, Nx, 3, 3)
    out = np.empty_like(G)
    for mu in range(4):
        out[..., mu, :, :] = gg @ G[..., mu, :, :] @ dag(shift(gg, mu, 1))
    return out.reshape(U.shape)


def site_coords(s, dims):
    Nx, Ny, Nz, Nt = dims
    x = s % Nx
    y = (s // Nx) % Ny
    z = (s // (Nx * Ny)) % Nz
    t = s // (Nx * Ny * Nz)
    return x, y, z, t
