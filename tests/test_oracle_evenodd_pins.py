"""Pins for the even/odd part of the oracle (parts apply O7, Schur complement,
block-preconditioned links).  None of these re-types the oracle's loops: they tie it to a dense
matrix assembled entry by entry from the operator's definition (tests/helpers.assemble_dense, built
with np.roll), to numpy's dense block algebra, and to the already pinned full apply."""
import numpy as np
import pytest

import synth
from tests.helpers import assemble_dense, rel_l2

TINY = [((2, 2, 2, 2), 6), ((4, 2, 2, 2), 4), ((2, 4, 2, 6), 2)]


def _setup(dims, Nc, seed, nrhs=1):
    links = synth.make_arbitrary_links(dims, Nc, seed).numpy()
    links[:, 0] += 2.0 * np.eye(Nc, dtype=np.complex64)          # keep X(x) well conditioned
    u = synth.make_vectors(dims, Nc, nrhs, seed + 1).numpy()
    w = synth.make_vectors(dims, Nc, nrhs, seed + 2).numpy()
    return links, u, w


def _site_mask(par, Nc, p):
    return np.repeat(par == p, Nc)


def test_site_parities_match_coordinates(oracle_lib):
    dims = (4, 2, 6, 2)
    par = oracle_lib.site_parities(dims)
    for s in (0, 1, 4, 5, 9, 47, 95):
        x0 = s % 4; x1 = (s // 4) % 2; x2 = (s // 8) % 6; x3 = s // 48
        assert par[s] == (x0 + x1 + x2 + x3) % 2
    assert par.sum() * 2 == par.size


@pytest.mark.parametrize("dims,Nc", TINY + [((3, 2, 1, 4), 4)])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("parity", [0, 1, 2])
@pytest.mark.parametrize("local", [0, 1, 2])
def test_parts_equals_dense_blocks(oracle_lib, dims, Nc, dagger, parity, local):
    """out = alpha*Loc + beta*Hop against the dense matrix split into its block-diagonal (X) and
    off-diagonal (hopping) parts; rows outside the parity set must come back as zero."""
    links, u, w = _setup(dims, Nc, 11, nrhs=2)
    V = links.shape[0]
    hop_only = links.copy(); hop_only[:, 0] = 0
    x_only = np.zeros_like(links); x_only[:, 0] = links[:, 0]
    H = assemble_dense(hop_only, dims)
    X = assemble_dense(x_only, dims)
    if dagger:
        H, X = H.conj().T, X.conj().T
    alpha, beta = 0.75, -1.25
    uu = u.reshape(V * Nc, 2).astype(np.complex128)
    ww = w.reshape(V * Nc, 2).astype(np.complex128)
    loc = {0: 0 * uu, 1: X @ uu, 2: uu}[local]
    ref = alpha * loc + beta * (H @ ww)
    par = oracle_lib.site_parities(dims)
    if parity != 2:
        ref[~_site_mask(par, Nc, parity)] = 0
    got = oracle_lib.coarse_apply_parts(dims, Nc, links, u if local else None, w, nrhs=2, dagger=dagger,
                                        parity=parity, local=local, alpha=alpha, beta=beta)
    assert rel_l2(got.reshape(V * Nc, 2), ref) < 1e-13
    if parity != 2:
        assert np.all(got.reshape(V * Nc, 2)[~_site_mask(par, Nc, parity)] == 0)


@pytest.mark.parametrize("dagger", [0, 1])
def test_parts_all_sites_is_the_full_apply(oracle_lib, dagger):
    dims, Nc = (3, 2, 4, 2), 8
    links, u, _ = _setup(dims, Nc, 5)
    a = oracle_lib.coarse_apply_parts(dims, Nc, links, u, u, dagger=dagger)
    b = oracle_lib.coarse_apply(dims, Nc, links, u, dagger=dagger)
    assert rel_l2(a, b) < 1e-14


def test_parts_int16_links_equal_dequantised(oracle_lib):
    dims, Nc = (2, 2, 2, 4), 8
    links, u, w = _setup(dims, Nc, 21)
    q, sc = oracle_lib.quantize_i16(links, Nc)
    deq = oracle_lib.dequantize_i16(q, sc, Nc).reshape(links.shape)
    hop = deq.copy(); hop[:, 0] = 0
    ref = assemble_dense(hop, dims) @ w.reshape(-1).astype(np.complex128)
    par = oracle_lib.site_parities(dims)
    ref[~_site_mask(par, Nc, 1)] = 0
    got = oracle_lib.coarse_apply_parts(dims, Nc, q.reshape(-1, 9, Nc, Nc, 2), None, w, parity=1, local=0,
                                        alpha=0.0, beta=1.0, link_precision=oracle_lib.LINK_I16, scales=sc)
    assert rel_l2(got.reshape(-1), ref) < 1e-13


@pytest.mark.parametrize("dims,Nc", TINY)
@pytest.mark.parametrize("parity", [0, 1])
def test_schur_apply_is_the_dense_schur_complement(oracle_lib, dims, Nc, parity):
    """S_p = A_pp - A_pq A_qq^{-1} A_qp computed by numpy on the assembled matrix."""
    links, u, _ = _setup(dims, Nc, 31)
    V = links.shape[0]
    A = assemble_dense(links, dims)
    par = oracle_lib.site_parities(dims)
    P, Q = _site_mask(par, Nc, parity), _site_mask(par, Nc, 1 - parity)
    S = A[np.ix_(P, P)] - A[np.ix_(P, Q)] @ np.linalg.solve(A[np.ix_(Q, Q)], A[np.ix_(Q, P)])
    v = u.reshape(-1).astype(np.complex128)
    ref = S @ v[P]
    got = oracle_lib.schur_apply(dims, Nc, links, u, parity).reshape(-1)
    # the oracle rounds the two intermediate vectors to complex64 (as the CUDA path stores them)
    assert rel_l2(got[P], ref) < 5e-7
    assert np.all(got[Q] == 0)


@pytest.mark.parametrize("dims,Nc", TINY)
def test_schur_solution_property(oracle_lib, dims, Nc):
    """If A x = b then S_e x_e = b_e - D_eo X_o^{-1} b_o: the reason the solver may iterate on one parity."""
    links, u, _ = _setup(dims, Nc, 41)
    A = assemble_dense(links, dims)
    par = oracle_lib.site_parities(dims)
    E, O = _site_mask(par, Nc, 0), _site_mask(par, Nc, 1)
    x = u.reshape(-1).astype(np.complex128)
    b = A @ x
    rhs = b[E] - A[np.ix_(E, O)] @ np.linalg.solve(A[np.ix_(O, O)], b[O])
    xe = np.where(E, x, 0).reshape(u.shape)
    got = oracle_lib.schur_apply(dims, Nc, links, xe, 0).reshape(-1)[E]
    assert rel_l2(got, rhs) < 5e-7


@pytest.mark.parametrize("dims,Nc", TINY)
@pytest.mark.parametrize("parity", [0, 1])
def test_hat_links_give_the_left_preconditioned_schur_operator(oracle_lib, dims, Nc, parity):
    """1 - Dhat_pq Dhat_qp (two hops on Yhat = X^{-1} Y) equals X_p^{-1} S_p built densely."""
    links, u, _ = _setup(dims, Nc, 51)
    A = assemble_dense(links, dims)
    par = oracle_lib.site_parities(dims)
    P, Q = _site_mask(par, Nc, parity), _site_mask(par, Nc, 1 - parity)
    S = A[np.ix_(P, P)] - A[np.ix_(P, Q)] @ np.linalg.solve(A[np.ix_(Q, Q)], A[np.ix_(Q, P)])
    ref = np.linalg.solve(A[np.ix_(P, P)], S @ u.reshape(-1).astype(np.complex128)[P])
    hat = oracle_lib.hat_links(links)
    assert np.allclose(hat[:, 0], np.eye(Nc))
    assert np.allclose(np.einsum("sij,smjk->smik", links[:, 0].astype(np.complex128), hat[:, 1:]), links[:, 1:],
                       atol=1e-6)
    got = oracle_lib.schur_hat_apply(dims, Nc, hat.astype(np.complex64), u, parity).reshape(-1)
    # hat links are rounded to complex64 before use: 6e-8 per entry, amplified by ||Dhat||^2
    assert rel_l2(got[P], ref) < 5e-6
    assert np.all(got[Q] == 0)


@pytest.mark.parametrize("parity", [0, 1])
def test_schur_hat_adjoint_identity(oracle_lib, parity):
    dims, Nc = (2, 4, 2, 2), 6
    links, u, w = _setup(dims, Nc, 61)
    hat = oracle_lib.hat_links(links).astype(np.complex64)
    par = oracle_lib.site_parities(dims)
    P = _site_mask(par, Nc, parity)
    a = np.where(P, u.reshape(-1), 0).reshape(u.shape)
    b = np.where(P, w.reshape(-1), 0).reshape(w.shape)
    Sb = oracle_lib.schur_hat_apply(dims, Nc, hat, b, parity).reshape(-1)
    Sda = oracle_lib.schur_hat_apply(dims, Nc, hat, a, parity, dagger=1).reshape(-1)
    lhs = np.vdot(a.reshape(-1).astype(np.complex128), Sb)
    rhs = np.vdot(Sda, b.reshape(-1).astype(np.complex128))
    assert abs(lhs - rhs) <= 1e-6 * abs(lhs)


def test_parts_rejects_bad_arguments(oracle_lib):
    dims, Nc = (2, 2, 2, 2), 4
    links, u, w = _setup(dims, Nc, 1)
    with pytest.raises(ValueError):
        oracle_lib.coarse_apply_parts(dims, Nc, links, u, w, parity=3)
    with pytest.raises(ValueError):
        oracle_lib.coarse_apply_parts(dims, Nc, links, None, w, local=1)
    with pytest.raises(ValueError):
        oracle_lib.schur_apply((3, 2, 2, 2), Nc, np.zeros((24, 9, Nc, Nc), np.complex64), np.zeros((24, Nc, 1), np.complex64), 0)


def test_hat_links_definition_by_multiplying_back(oracle_lib):
    """Pin of oracle.hat_links against its definition without re-calling the solver: X . Yhat_m = Y_m for
    m = 1..8, slot 0 = identity, or X . slot0 = identity with slot0_inverse (reading R21)."""
    dims, Nc = (2, 2, 2, 2), 12
    links = synth.make_gamma_hermitian_links(dims, Nc, 5).numpy().astype(np.complex128)
    hat = oracle_lib.hat_links(links)
    hat_inv = oracle_lib.hat_links(links, slot0_inverse=True)
    eye = np.eye(Nc)
    for s in range(links.shape[0]):
        X = links[s, 0]
        assert np.array_equal(hat[s, 0], eye)
        assert np.abs(X @ hat_inv[s, 0] - eye).max() < 1e-12
        for m in range(1, 9):
            assert np.abs(X @ hat[s, m] - links[s, m]).max() < 1e-12 * max(1.0, np.abs(links[s, m]).max() * np.linalg.cond(X))
            assert np.array_equal(hat[s, m], hat_inv[s, m])
