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
    assert rel_l2(x, xg) < 2e-6            # basis vectors rounded to complex64 in the oracle, not in scipy
    assert abs(norms[1] - np.linalg.norm(b - A @ xg)) < 2e-6 * norms[0]
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
    assert rel_l2(x, np.linalg.solve(A, b.astype(np.complex128))) < 1e-4
    assert norms[1] < 1e-4 * norms[0]


def test_cycles_chain_and_match_restarted_gmres(oracle_lib):
    dims, Nc, s = (2, 2, 2, 2), 4, 4
    links, A, b = _system(dims, Nc, 11)
    apply_fn = lambda v: A @ v.astype(np.complex128)
    x, norms = oracle_lib.cagcr(apply_fn, b, np.zeros_like(b), s, cycles=3)
    assert len(norms) == 4 and all(norms[i + 1] < norms[i] for i in range(3))
    xg, _ = spla.gmres(A, b.astype(np.complex128), restart=s, maxiter=3, rtol=1e-30, atol=0.0)
    assert rel_l2(x, xg) < 1e-5


def test_with_the_oracle_apply_as_operator(oracle_lib):
    """The composition the GPU test uses: apply_fn = the pinned coarse apply."""
    dims, Nc, s = (2, 2, 2, 2), 8, 8
    links, A, b = _system(dims, Nc, 13)
    f = lambda v: oracle_lib.coarse_apply(dims, Nc, links, v.reshape(-1, Nc, 1)).reshape(-1)
    g = lambda v: A @ v.astype(np.complex128)
    xa, na = oracle_lib.cagcr(f, b, np.zeros_like(b), s)
    xb, nb = oracle_lib.cagcr(g, b, np.zeros_like(b), s)
    assert rel_l2(xa, xb) < 1e-9 and abs(na[1] - nb[1]) < 1e-9 * na[0]
