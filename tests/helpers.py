"""Small numpy helpers for the tests (no oracle/, no CUDA path)."""
from __future__ import annotations

import numpy as np


def site_grid(dims):
    """Integer array g[x3][x2][x1][x0] = site index s(x) (x0 fastest)."""
    L0, L1, L2, L3 = (int(d) for d in dims)
    return np.arange(L0 * L1 * L2 * L3, dtype=np.int64).reshape(L3, L2, L1, L0)


def neighbour_table(dims):
    """nbr[s][m]: m=0 -> s, 1+mu -> s(x+mu^), 5+mu -> s(x-mu^), built with np.roll."""
    g = site_grid(dims)
    V = g.size
    nbr = np.empty((V, 9), dtype=np.int64)
    nbr[:, 0] = g.reshape(-1)
    for mu in range(4):
        ax = 3 - mu
        nbr[:, 1 + mu] = np.roll(g, -1, axis=ax).reshape(-1)   # value at x is s(x+mu^)
        nbr[:, 5 + mu] = np.roll(g, +1, axis=ax).reshape(-1)   # value at x is s(x-mu^)
    return nbr


def assemble_dense(links, dims):
    """Dense (V Nc)^2 matrix of the stencil: block row s gets links[s][m] in block column
    nbr[s][m]; coinciding neighbours (extents 1 and 2) add up."""
    links = np.asarray(links)
    V, _, Nc, _ = links.shape
    nbr = neighbour_table(dims)
    A = np.zeros((V * Nc, V * Nc), dtype=np.complex128)
    for s in range(V):
        for m in range(9):
            t = nbr[s, m]
            A[s * Nc:(s + 1) * Nc, t * Nc:(t + 1) * Nc] += links[s, m]
    return A


def rel_l2(a, b):
    a = np.asarray(a).reshape(-1)
    b = np.asarray(b).reshape(-1)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def rel_l2_per_rhs(got, ref):
    """max over right-hand sides r of ||got[:,:,r]-ref[:,:,r]|| / ||ref[:,:,r]||."""
    got = np.asarray(got)
    ref = np.asarray(ref)
    nrhs = ref.shape[-1]
    return max(rel_l2(got[..., r], ref[..., r]) for r in range(nrhs))


def gamma_diag(Nc):
    g = np.ones(Nc)
    g[Nc // 2:] = -1.0
    return g
