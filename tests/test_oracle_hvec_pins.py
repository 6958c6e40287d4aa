"""Pins for the half-precision vector part of the oracle (PAPER.md:L97:
16-bit fixed point with a per-site fp32 norm)."""
import numpy as np
import pytest

import synth
from tests.helpers import assemble_dense, rel_l2


def test_vector_quantiser_properties(oracle_lib):
    Nc, nrhs = 12, 3
    v = synth.make_vectors((2, 3, 2, 2), Nc, nrhs, 5).numpy()
    v[3] = 0                                   # an all-zero site
    v[5, :, 1] *= 1e-20                        # tiny but non-zero column
    q, norms = oracle_lib.quantize_vec_i16(v, Nc, nrhs)
    assert q.dtype == np.int16 and q.shape == (24, Nc, nrhs, 2) and norms.shape == (24, nrhs)
    vr = v.view(np.float32).reshape(24, Nc, nrhs, 2)
    amax = np.abs(vr).max(axis=(1, 3))
    assert np.array_equal(norms, np.where(amax == 0, 0, amax / np.float32(32767.0)).astype(np.float32))
    assert np.all(q[3] == 0) and np.all(norms[3] == 0)
    assert np.abs(q).max() <= 32767 and q.min() >= -32767
    deq = q.astype(np.float64) * norms[:, None, :, None].astype(np.float64)
    # 0.5 from rounding + the fp32 division's own rounding (32767 * 2^-24 = 0.002)
    assert np.all(np.abs(deq - vr) <= 0.503 * norms[:, None, :, None] + 1e-45)
    # the largest component of every (site, rhs) maps to +-32767
    assert np.all((np.abs(q).max(axis=(1, 3)) == 32767) | (amax == 0))
    # idempotent on dequantised data
    q2, n2 = oracle_lib.quantize_vec_i16(deq.astype(np.float32).view(np.complex64).reshape(24, Nc, nrhs), Nc, nrhs)
    assert np.array_equal(q2, q)


@pytest.mark.parametrize("dagger", [0, 1])
def test_hvec_apply_equals_apply_on_exactly_dequantised_vectors(oracle_lib, dagger):
    """With power-of-two norms q*norm is exact in fp32, so the pinned complex64 apply must agree."""
    dims, Nc, nrhs = (3, 2, 2, 4), 8, 2
    V = 48
    links = synth.make_arbitrary_links(dims, Nc, 3).numpy()
    rng = np.random.default_rng(7)
    q = rng.integers(-32767, 32768, size=(V, Nc, nrhs, 2)).astype(np.int16)
    norms = (2.0 ** rng.integers(-20, -10, size=(V, nrhs))).astype(np.float32)
    deq = (q.astype(np.float32) * norms[:, None, :, None]).view(np.complex64).reshape(V, Nc, nrhs)
    a = oracle_lib.coarse_apply_hvec(dims, Nc, links, q, norms, nrhs=nrhs, dagger=dagger)
    b = oracle_lib.coarse_apply(dims, Nc, links, deq, nrhs=nrhs, dagger=dagger)
    assert rel_l2(a, b) < 1e-15


def test_hvec_apply_against_dense_matrix_and_int16_links(oracle_lib):
    dims, Nc = (2, 2, 3, 2), 6
    V = 24
    links = synth.make_arbitrary_links(dims, Nc, 9).numpy()
    v = synth.make_vectors(dims, Nc, 1, 10).numpy()
    q, norms = oracle_lib.quantize_vec_i16(v, Nc, 1)
    deq = (q.astype(np.float64) * norms[:, None, :, None].astype(np.float64))
    x = (deq[..., 0] + 1j * deq[..., 1]).reshape(-1)
    ref = assemble_dense(links, dims) @ x
    got = oracle_lib.coarse_apply_hvec(dims, Nc, links, q, norms).reshape(-1)
    assert rel_l2(got, ref) < 1e-13
    lq, sc = oracle_lib.quantize_i16(links, Nc)
    ldeq = oracle_lib.dequantize_i16(lq, sc, Nc).reshape(V, 9, Nc, Nc)
    ref2 = assemble_dense(ldeq, dims).conj().T @ x
    got2 = oracle_lib.coarse_apply_hvec(dims, Nc, lq.reshape(V, 9, Nc, Nc, 2), q, norms, dagger=1,
                                        link_precision=oracle_lib.LINK_I16, scales=sc).reshape(-1)
    assert rel_l2(got2, ref2) < 1e-13


def test_half_vectors_cost_about_3e5_relative(oracle_lib):
    """Quantising the vector itself moves the result by ~1e-5..1e-4 (why parity is against the dequantised input)."""
    dims, Nc = (2, 2, 2, 2), 16
    links = synth.make_arbitrary_links(dims, Nc, 1).numpy()
    v = synth.make_vectors(dims, Nc, 1, 2).numpy()
    q, norms = oracle_lib.quantize_vec_i16(v, Nc, 1)
    a = oracle_lib.coarse_apply_hvec(dims, Nc, links, q, norms)
    b = oracle_lib.coarse_apply(dims, Nc, links, v)
    assert 1e-6 < rel_l2(a, b) < 2e-4


@pytest.mark.parametrize("dagger", [0, 1])
def test_hvec_sites_is_the_dense_operator_rows(oracle_lib, dagger):
    """coarse_apply_hvec_sites at a site list = those block rows of the dense operator (assembled with
    numpy from the dequantised links) times the exactly dequantised vector; int16 links, 2 RHS, extents 1-3."""
    dims, Nc, nrhs = (3, 2, 1, 2), 6, 2
    V = 12
    links = synth.make_arbitrary_links(dims, Nc, 21).numpy()
    lq, sc = oracle_lib.quantize_i16(links, Nc)
    ldeq = oracle_lib.dequantize_i16(lq, sc, Nc).reshape(V, 9, Nc, Nc)
    A = assemble_dense(ldeq, dims)
    if dagger:
        A = A.conj().T
    v = synth.make_vectors(dims, Nc, nrhs, 22).numpy()
    q, norms = oracle_lib.quantize_vec_i16(v, Nc, nrhs)
    deq = q.astype(np.float64) * norms[:, None, :, None].astype(np.float64)
    x = (deq[..., 0] + 1j * deq[..., 1]).reshape(V * Nc, nrhs)
    ref = (A @ x).reshape(V, Nc, nrhs)
    sites = np.array([11, 0, 5, 5, 7], dtype=np.int64)          # unordered, with a repeat
    got = oracle_lib.coarse_apply_hvec_sites(dims, Nc, lq.reshape(V, 9, Nc, Nc, 2), q, norms, sites, nrhs=nrhs,
                                             dagger=dagger, link_precision=oracle_lib.LINK_I16, scales=sc)
    assert got.shape == (5, Nc, nrhs)
    assert rel_l2(got, ref[sites]) < 1e-13
    full = oracle_lib.coarse_apply_hvec(dims, Nc, lq.reshape(V, 9, Nc, Nc, 2), q, norms, nrhs=nrhs, dagger=dagger,
                                        link_precision=oracle_lib.LINK_I16, scales=sc)
    assert np.array_equal(got, full[sites])
