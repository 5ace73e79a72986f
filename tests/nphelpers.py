"""Independent numpy restatements of the paper's definitions, used to pin the oracle.

Links are complex128 arrays [t][z][y][x][mu][row][col] (the canonical export layout). Nothing here
is shared with oracle/ or with the CUDA path: vectorised np.roll / einsum versions of eq 3, 4, 9.
"""
import numpy as np


def axis_of(mu):
    return 3 - mu  # x -> axis 3, y -> 2, z -> 1, t -> 0


def shifted(field, mu, d=1):
    """field(x + d*mu_hat) for a site field whose first four axes are t,z,y,x"""
    return np.roll(field, -d, axis=axis_of(mu))


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def random_sun(rng, N, shape=()):
    """Haar SU(N) via QR of a Ginibre matrix (Mezzadri's recipe), det fixed by a global phase."""
    z = (rng.standard_normal(shape + (N, N)) + 1j * rng.standard_normal(shape + (N, N))) / np.sqrt(2)
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=-2, axis2=-1)
    q = q * (d / np.abs(d))[..., None, :]
    det = np.linalg.det(q)
    return q / (det ** (1.0 / N))[..., None, None]


def random_links(rng, N, dims):
    Lx, Ly, Lz, Lt = dims
    return random_sun(rng, N, (Lt, Lz, Ly, Lx, 4))


def plaquette_field(links, mu, nu):
    """P_mu,nu(s) = U_mu(s) U_nu(s+mu) U_mu(s+nu)^dagger U_nu(s)^dagger   (eq 4)"""
    Um, Un = links[..., mu, :, :], links[..., nu, :, :]
    return Um @ shifted(Un, mu) @ dag(shifted(Um, nu)) @ dag(Un)


def mean_plaquette(links):
    N = links.shape[-1]
    V = int(np.prod(links.shape[:4]))
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            tot += np.trace(plaquette_field(links, mu, nu), axis1=-2, axis2=-1).real.sum()
    return tot / (6 * V * N)


def wilson_action(links, beta):
    """S_G = beta/Nc sum_s sum_{mu<nu} ReTr[1 - P]   (eq 3)"""
    N = links.shape[-1]
    V = int(np.prod(links.shape[:4]))
    return beta * 6 * V * (1.0 - mean_plaquette(links))


def polyakov(links):
    Lt = links.shape[0]
    N = links.shape[-1]
    P = links[0, ..., 3, :, :]
    for t in range(1, Lt):
        P = P @ links[t, ..., 3, :, :]
    return np.trace(P, axis1=-2, axis2=-1).mean() / N


def gauge_transform(links, G):
    """U_mu(x) -> G(x) U_mu(x) G(x+mu)^dagger"""
    out = np.empty_like(links)
    for mu in range(4):
        out[..., mu, :, :] = G @ links[..., mu, :, :] @ dag(shifted(G, mu))
    return out


def staple_field(links, mu):
    """eq 9 as printed, for every site at once."""
    Um = links[..., mu, :, :]
    S = np.zeros_like(Um)
    for nu in range(4):
        if nu == mu:
            continue
        Un = links[..., nu, :, :]
        S += Un @ shifted(Um, nu) @ dag(shifted(Un, mu))
        Un_d, Um_d = shifted(Un, nu, -1), shifted(Um, nu, -1)
        S += dag(Un_d) @ Um_d @ shifted(Un_d, mu)
    return S


def site_index(x, y, z, t, dims):
    Lx, Ly, Lz, Lt = dims
    return x + Lx * (y + Ly * (z + Lz * t))


def quat_to_su2(a):
    """eq 6: a0 + i a.sigma"""
    a0, a1, a2, a3 = a
    return np.array([[a0 + 1j * a3, a2 + 1j * a1], [-a2 + 1j * a1, a0 - 1j * a3]])


def unitarity_defect(links):
    N = links.shape[-1]
    return np.abs(links @ dag(links) - np.eye(N)).max()


def det_defect(links):
    return np.abs(np.linalg.det(links) - 1).max()
