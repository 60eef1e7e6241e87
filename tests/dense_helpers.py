"""Brute-force helpers for the oracle pins: dense matrices obtained by applying an
operator to every unit vector, site tables built with plain Python loops."""
import numpy as np


def volume(dims):
    return int(np.prod(dims))


def coords(dims):
    """[V][4] integer coordinates in lex order x + Lx*(y + Ly*(z + Lz*t)) (C1)."""
    Lx, Ly, Lz, Lt = dims
    out = np.zeros((volume(dims), 4), dtype=np.int64)
    for t in range(Lt):
        for z in range(Lz):
            for y in range(Ly):
                for x in range(Lx):
                    out[x + Lx * (y + Ly * (z + Lz * t))] = (x, y, z, t)
    return out


def parity(dims):
    return coords(dims).sum(axis=1) & 1


def dense_from_apply(apply, n_sites, site_mask=None):
    """Matrix of a linear map on [V][4][3] fields; optional restriction to masked sites."""
    n = n_sites * 12
    idx = np.arange(n).reshape(n_sites, 12)
    sel = idx.reshape(-1) if site_mask is None else idx[site_mask].reshape(-1)
    cols = []
    for j in sel:
        e = np.zeros(n, dtype=np.complex128)
        e[j] = 1.0
        cols.append(apply(e.reshape(n_sites, 4, 3)).reshape(-1)[sel])
    return np.stack(cols, axis=1)


def timeslice_projector_trace(dims, Gam, Minv):
    """sum_{x in t} tr[Gamma M^-1(x,x)] for every t; Minv is the dense [12V,12V] inverse."""
    V = volume(dims)
    Lt = dims[3]
    Vs = V // Lt
    out = np.zeros(Lt, dtype=np.complex128)
    G = np.kron(Gam, np.eye(3))
    for s in range(V):
        blk = Minv[12 * s:12 * s + 12, 12 * s:12 * s + 12]
        out[s // Vs] += np.trace(G @ blk)
    return out
