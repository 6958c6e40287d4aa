"""Pins for the CA-GCR(s) oracle: it must produce the iterate
that minimises the residual over x0 + K_s(A, r0).  Pinned against scipy's GMRES (an independent library
routine that defines the same iterate), against the direct solve when s reaches the system size, and by
the orthogonality of the new residual to A K_s."""
import numpy as np
import pytest
import scipy.sparse.linalg as spla

import synth
from tests.helpers import assemble_dense, rel_l2


def _system(dims, Nc, seed, shift=12.0):
    links = synth.make_arbitrary_links(dims, Nc, seed).numpy()
    links[:, 0] += shift * np.eye(Nc, dtype=np.complex64)     # diagonally dominant: a smoother-friendly operator
    A = assemble_dense(links, dims)
    b = synth.make_vectors(dims, Nc, 1, seed + 1).numpy().reshape(-1)
    return links, A, b


def test_one_cycle_is_the_gmres_iterate(oracle_lib):
    dims, Nc, s = (2, 2, 2, 2), 4, 6
    links, A, b = _system(dims, Nc, 3)
    apply_fn = lambda v: A @ v.astype(np.complex128)
    x, norms = oracle_lib.cagcr(apply_fn, b, np.zeros_like(b), s, cycles=1)
    xg, info = spla.gmres(A, b.astype(np.complex128), x0=np.zeros(b.size, complex), restart=s, maxiter=1,
                          rtol=1e-30, atol=0.0)
    assert rel_l2(x, xg) < 1e-10
    assert abs(norms[1] - np.linalg.norm(b - A @ xg)) < 1e-10 * norms[0]
    assert norms[1] < norms[0]


def test_residual_is_orthogonal_to_A_times_krylov_space(oracle_lib):
    dims, Nc, s = (2, 2, 2, 4), 4, 8
    links, A, b = _system(dims, Nc, 5)
    apply_fn = lambda v: A @ v.astype(np.complex128)
    x0 = synth.make_vectors(dims, Nc, 1, 9).numpy().reshape(-1)
    x, norms = oracle_lib.cagcr(apply_fn, b, x0, s, cycles=1)
    r0 = b - A @ x0.astype(np.complex128)
    r = b - A @ x
    K = [r0]
    for _ in range(s - 1):
        K.append(A @ K[-1])
    AK = A @ np.stack(K, axis=1)
    AKn = AK / np.linalg.norm(AK, axis=0)
    assert np.abs(AKn.conj().T @ r).max() < 1e-5 * np.linalg.norm(r0)
    assert abs(np.linalg.norm(r) - norms[1]) < 1e-6 * norms[0]


def test_full_dimension_gives_the_direct_solution(oracle_lib):
    dims, Nc = (1, 1, 1, 2), 2          # 4 unknowns
    links, A, b = _system(dims, Nc, 7, shift=3.0)
    apply_fn = lambda v: A @ v.astype(np.complex128)
    x, norms = oracle_lib.cagcr(apply_fn, b, np.zeros_like(b), 4, cycles=1)
    assert rel_l2(x, np.linalg.solve(A, b.astype(np.complex128))) < 1e-10
    assert norms[1] < 1e-10 * norms[0]


def test_cycles_chain_and_match_restarted_gmres(oracle_lib):
    dims, Nc, s = (2, 2, 2, 2), 4, 4
    links, A, b = _system(dims, Nc, 11)
    apply_fn = lambda v: A @ v.astype(np.complex128)
    x, norms = oracle_lib.cagcr(apply_fn, b, np.zeros_like(b), s, cycles=3)
    assert len(norms) == 4 and all(norms[i + 1] < norms[i] for i in range(3))
    xg, _ = spla.gmres(A, b.astype(np.complex128), restart=s, maxiter=3, rtol=1e-30, atol=0.0)
    assert rel_l2(x, xg) < 1e-9


def test_with_the_oracle_apply_as_operator(oracle_lib):
    """The composition the GPU test uses: apply_fn = the pinned coarse apply."""
    dims, Nc, s = (2, 2, 2, 2), 8, 8
    links, A, b = _system(dims, Nc, 13)
    f = lambda v: oracle_lib.coarse_apply(dims, Nc, links, v.reshape(-1, Nc, 1)).reshape(-1)
    g = lambda v: A @ v.astype(np.complex128)
    xa, na = oracle_lib.cagcr(f, b, np.zeros_like(b), s)
    xb, nb = oracle_lib.cagcr(g, b, np.zeros_like(b), s)
    assert rel_l2(xa, xb) < 1e-9 and abs(na[1] - nb[1]) < 1e-9 * na[0]


def test_ill_conditioned_power_basis_still_reaches_the_gmres_optimum(oracle_lib):
    """s = 8 on a 256-unknown system: the power basis has cond ~1e9+, where a least-squares routine with a
    default singular-value cut-off silently returns a worse iterate (this pin exists because that happened).
    GMRES builds an orthonormal basis of the same space, so its residual is the true optimum."""
    dims, Nc, s = (2, 2, 2, 2), 16, 8
    links, A, b = _system(dims, Nc, 17)
    apply_fn = lambda v: A @ v.astype(np.complex128)
    x, norms = oracle_lib.cagcr(apply_fn, b, np.zeros_like(b), s, cycles=1)
    xg, _ = spla.gmres(A, b.astype(np.complex128), restart=s, maxiter=1, rtol=1e-30, atol=0.0)
    rg = np.linalg.norm(b - A @ xg)
    P = [b.astype(np.complex128)]
    for _ in range(s):
        P.append(A @ P[-1])
    assert np.linalg.cond(np.stack(P[1:], axis=1)) > 1e8
    assert abs(norms[1] - rg) < 1e-8 * rg
    assert abs(np.linalg.norm(b - A @ x) - rg) < 1e-8 * rg


def test_large_tall_basis_is_not_truncated(oracle_lib):
    """The exact scenario that exposed the cut-off: 12288 unknowns, s = 8, cond(Q) ~ 4e11 > 1/(eps * 12288).
    The returned residual must be orthogonal to every basis direction and no worse than the one the
    normal equations (a different route to the same minimiser) give."""
    dims, Nc, s = (4, 4, 4, 4), 48, 8
    links = synth.make_arbitrary_links(dims, Nc, 101).numpy()
    links[:, 0] += 12.0 * np.eye(Nc, dtype=np.complex64)
    b = synth.make_vectors(dims, Nc, 1, 102).numpy().reshape(-1)
    f = lambda v: oracle_lib.coarse_apply(dims, Nc, links, v.reshape(-1, Nc, 1)).reshape(-1)
    x, norms = oracle_lib.cagcr(f, b, np.zeros_like(b), s)
    P = [b]
    for _ in range(s):
        P.append(f(P[-1]).astype(np.complex64))
    Pm = np.stack([p.astype(np.complex128) for p in P], axis=1)
    Q = Pm[:, 1:]
    Qn = Q / np.linalg.norm(Q, axis=0)
    alpha_ne = np.linalg.solve(Qn.conj().T @ Qn, Qn.conj().T @ Pm[:, 0])
    r_ne = np.linalg.norm(Pm[:, 0] - Qn @ alpha_ne)
    assert norms[1] <= r_ne * (1 + 1e-3)
    r = b.astype(np.complex128) - f(x.astype(np.complex64))
    assert np.abs(Qn.conj().T @ r).max() < 1e-4 * norms[0]
    assert norms[1] < 1e-3 * norms[0]
