"""numpy helpers for the oracle pins: 4-D views, np.roll shifts, gauge transforms.

Independent of oracle/qdp_oracle.c's index arithmetic: a field [V, ...] in
lexicographic order (x0 fastest) is viewed as [L3, L2, L1, L0, ...] and moved
with np.roll, so f(x + mu_hat) = roll(f, -1, axis=3-mu).
"""
import numpy as np


def view4(dims, f):
    L0, L1, L2, L3 = dims
    return f.reshape((L3, L2, L1, L0) + f.shape[1:])


def flat(dims, f4):
    V = dims[0] * dims[1] * dims[2] * dims[3]
    return np.ascontiguousarray(f4.reshape((V,) + f4.shape[4:]))


def sh(dims, f, mu, step=+1):
    """f(x + step*mu_hat), periodic."""
    return flat(dims, np.roll(view4(dims, f), -step, axis=3 - mu))


def coords(dims):
    L0, L1, L2, L3 = dims
    x3, x2, x1, x0 = np.indices((L3, L2, L1, L0))
    return np.stack([x0, x1, x2, x3], axis=-1).reshape(-1, 4)


def parity(dims):
    return coords(dims).sum(axis=1) & 1


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def gauge_transform(dims, u, g):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu)^dag."""
    out = np.empty_like(u)
    for mu in range(4):
        out[:, mu] = g @ u[:, mu] @ dag(sh(dims, g, mu))
    return out


def plaquette_np(dims, u, mu, nu):
    """Re tr P_{mu nu}(x) for every x, [V]."""
    P = u[:, mu] @ sh(dims, u[:, nu], mu) @ dag(sh(dims, u[:, mu], nu)) @ dag(u[:, nu])
    return np.trace(P, axis1=-2, axis2=-1).real


def staple_np(dims, u, mu, dirs):
    S = np.zeros_like(u[:, mu])
    for nu in dirs:
        if nu == mu:
            continue
        S += u[:, nu] @ sh(dims, u[:, mu], nu) @ dag(sh(dims, u[:, nu], mu))
        low = dag(u[:, nu]) @ u[:, mu] @ sh(dims, u[:, nu], mu)   # based at x - nu
        S += sh(dims, low, nu, -1)
    return S


def hop_np(dims, u, psi):
    chi = np.zeros_like(psi)
    for mu in range(4):
        chi += np.einsum("xab,xsb->xsa", u[:, mu], sh(dims, psi, mu))
        back = np.einsum("xba,xsb->xsa", np.conj(u[:, mu]), psi)   # U^dag(y) psi(y) at y
        chi += sh(dims, back, mu, -1)
    return chi
