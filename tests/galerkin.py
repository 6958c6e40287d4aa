"""Brute-force Galerkin coarsening on a tiny lattice (numpy, dense) — oracle pin #1.

Follows PAPER.md:L41-43 (§2.1): near-null vectors -> chiral doubling with
(1 +- eps(x))/2, eps(x) = (-1)^{x0+x1+x2+x3} (§2.2) -> block
orthonormalisation over aggregates -> P, R = P^dagger -> A_hat = R A P.

Nothing here touches oracle/ or the CUDA path.  The fine operator is an explicit
nearest-neighbour staggered stencil with random n_f x n_f links,

    A_f = m + sum_mu 1/2 eta_mu(x) [ U_mu(x) delta_{x+mu^} - U_mu(x-mu^)^dagger delta_{x-mu^} ],
    eta_mu(x) = (-1)^{x0+...+x_{mu-1}},

held as a dense (V_f n_f)^2 matrix.  `coarse_dense` is the dense product P^dagger A_f P:
the coarse apply must equal coarse_dense @ v and the dagger apply coarse_dense^H @ v.
`links` holds the nine blocks per coarse site in the C-ABI order; forward and backward
hops that cross an aggregate face are kept apart, so coarse extents 2 and 1 (where
x+mu^ and x-mu^ coincide, or are x itself) stay well defined.
"""
from __future__ import annotations

import itertools

import numpy as np


def _sidx(x, dims):
    return x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))


def _coords(dims):
    # x0 fastest
    for x3, x2, x1, x0 in itertools.product(*(range(d) for d in reversed(dims))):
        yield (x0, x1, x2, x3)


def build(coarse_dims, block, n_f, n_vec, mass, seed):
    rng = np.random.default_rng(seed)
    cd = tuple(int(d) for d in coarse_dims)
    blk = tuple(int(b) for b in block)
    fd = tuple(c * b for c, b in zip(cd, blk))
    assert all(f % 2 == 0 for f in fd), "staggered phases need even fine extents"
    Vf, Vc = int(np.prod(fd)), int(np.prod(cd))
    Nc = 2 * n_vec
    nd = Vf * n_f

    U = (rng.standard_normal((4, Vf, n_f, n_f)) + 1j * rng.standard_normal((4, Vf, n_f, n_f))) / np.sqrt(2 * n_f)

    def blk_slice(s):
        return slice(s * n_f, (s + 1) * n_f)

    # parts of A_f: local (mass + hops inside an aggregate), forward / backward hops across a face
    A_local = np.zeros((nd, nd), dtype=np.complex128)
    A_fwd = [np.zeros((nd, nd), dtype=np.complex128) for _ in range(4)]
    A_bwd = [np.zeros((nd, nd), dtype=np.complex128) for _ in range(4)]
    for x in _coords(fd):
        s = _sidx(x, fd)
        A_local[blk_slice(s), blk_slice(s)] += mass * np.eye(n_f)
        for mu in range(4):
            eta = (-1) ** (sum(x[:mu]) % 2)
            xp = list(x); xp[mu] = (x[mu] + 1) % fd[mu]
            xm = list(x); xm[mu] = (x[mu] - 1) % fd[mu]
            sp, sm = _sidx(xp, fd), _sidx(xm, fd)
            fwd_crosses = (x[mu] % blk[mu]) == blk[mu] - 1
            bwd_crosses = (x[mu] % blk[mu]) == 0
            (A_fwd[mu] if fwd_crosses else A_local)[blk_slice(s), blk_slice(sp)] += 0.5 * eta * U[mu, s]
            (A_bwd[mu] if bwd_crosses else A_local)[blk_slice(s), blk_slice(sm)] += -0.5 * eta * U[mu, sm].conj().T
    A_f = A_local + sum(A_fwd) + sum(A_bwd)

    # prolongator: chirally doubled, block-orthonormalised random vectors
    phi = rng.standard_normal((nd, n_vec)) + 1j * rng.standard_normal((nd, n_vec))
    P = np.zeros((nd, Vc * Nc), dtype=np.complex128)
    agg_rows = {}
    for x in _coords(fd):
        c = _sidx(tuple(xi // b for xi, b in zip(x, blk)), cd)
        chi = sum(x) % 2                      # chi = 0 <-> eps(x) = +1 <-> projector (1+eps)/2
        agg_rows.setdefault((c, chi), []).extend(range(_sidx(x, fd) * n_f, (_sidx(x, fd) + 1) * n_f))
    for (c, chi), rows in agg_rows.items():
        rows = np.array(rows)
        assert len(rows) >= n_vec
        q, _ = np.linalg.qr(phi[rows, :])
        P[np.ix_(rows, c * Nc + chi * n_vec + np.arange(n_vec))] = q

    coarse_dense = P.conj().T @ A_f @ P

    def cblock(M, c, cp):
        return (P[:, c * Nc:(c + 1) * Nc].conj().T @ M @ P[:, cp * Nc:(cp + 1) * Nc])

    links = np.zeros((Vc, 9, Nc, Nc), dtype=np.complex128)
    for x in _coords(cd):
        c = _sidx(x, cd)
        links[c, 0] = cblock(A_local, c, c)
        for mu in range(4):
            xp = list(x); xp[mu] = (x[mu] + 1) % cd[mu]
            xm = list(x); xm[mu] = (x[mu] - 1) % cd[mu]
            links[c, 1 + mu] = cblock(A_fwd[mu], c, _sidx(xp, cd))
            links[c, 5 + mu] = cblock(A_bwd[mu], c, _sidx(xm, cd))
    return dict(coarse_dims=cd, Nc=Nc, links=links, coarse_dense=coarse_dense, P=P, A_f=A_f)
