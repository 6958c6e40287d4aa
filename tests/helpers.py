"""Small numpy helpers for the tests (no oracle/ import; only gpu_hat_links touches the CUDA path, lazily)."""
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


def gpu_hat_links(oracle_lib, dims, Nc, links_np):
    """Block-preconditioned links built by the PRODUCT (coarse_op_build_hat_links) from complex64 links on the
    host; returns the device tensor and its host copy (the same bits go to the oracle's apply), after
    checking them against the oracle's own fp64 solve at fp32 rounding level."""
    import torch
    import paper_2212_12559_b200 as cop
    links_d = torch.as_tensor(links_np, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links_d)
    hat_d = torch.empty_like(links_d)
    op.build_hat_links(hat_d)
    torch.cuda.synchronize()
    op.close()
    hat = hat_d.cpu().numpy()
    ref = oracle_lib.hat_links(links_np)
    d = np.linalg.norm((hat - ref).reshape(hat.shape[0], 9, -1), axis=2) / np.linalg.norm(ref.reshape(hat.shape[0], 9, -1), axis=2)
    assert d.max() <= 1e-6, f"device-built hat links differ from the oracle's: {d.max():.3e}"
    return hat_d, hat
