"""Pins for the CPU oracle (oracle/coarse_oracle.cpp) — all CPU, `-m "not gpu"`.

The paper prints no worked numerical example for the coarse operator, so the oracle is
pinned to what the paper and the mathematics fix:

  1. brute-force Galerkin coarsening A_hat = P^dagger A P on tiny lattices
  2. unit-shift cases that are exact permutations of the input
  3. X-only case against a library einsum
  4. the adjoint identity <u, A v> = <A^dagger u, v> on arbitrary links (dagger)
  5. the Gamma-Hermiticity invariant on the generated links
  6. linearity; block apply = per-column single applies
  7. quantiser bounds ("16-bit fixed point"; BASELINE.json config 4)
  8. the storage count the paper prints, tests/golden/storage_count.txt

A dropped term, a swapped +-mu, a transposed operand, a wrong wrap or a wrong site order
each fail at least one of (1), (2), (4).
"""
import os

import numpy as np
import pytest

import synth
from tests import galerkin
from tests.helpers import (assemble_dense, gamma_diag, neighbour_table, rel_l2,
                           rel_l2_per_rhs, site_grid)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand_vec(rng, V, Nc, nrhs):
    return (rng.standard_normal((V, Nc, nrhs)) + 1j * rng.standard_normal((V, Nc, nrhs))).astype(np.complex64)


# ---------------------------------------------------------------- 1. Galerkin
GALERKIN_CASES = [
    # coarse dims, aggregate, n_f, n_vec
    ((3, 3, 3, 3), (2, 2, 2, 2), 1, 4),
    ((2, 2, 2, 2), (2, 2, 2, 2), 2, 3),
    ((3, 2, 1, 4), (2, 2, 2, 2), 2, 4),
    ((1, 1, 1, 1), (2, 2, 2, 2), 3, 24),      # complete basis: the Nc=48 KD supersite transform
    ((4, 3, 2, 3), (2, 2, 2, 2), 1, 2),
    ((2, 3, 2, 1), (4, 2, 2, 2), 1, 5),
]


@pytest.fixture(scope="module", params=range(len(GALERKIN_CASES)))
def galerkin_case(request):
    cd, blk, n_f, n_vec = GALERKIN_CASES[request.param]
    return galerkin.build(cd, blk, n_f, n_vec, mass=0.05, seed=100 + request.param)


def test_galerkin_blocks_reassemble_to_PAP(galerkin_case):
    """The nine-blocks-per-site layout, placed by the stencil definition, IS P^dagger A P."""
    g = galerkin_case
    A = assemble_dense(g["links"], g["coarse_dims"])
    assert rel_l2(A, g["coarse_dense"]) < 1e-13


@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("nrhs", [1, 3])
def test_oracle_equals_galerkin(oracle_lib, galerkin_case, dagger, nrhs):
    g = galerkin_case
    cd, Nc = g["coarse_dims"], g["Nc"]
    V = int(np.prod(cd))
    rng = np.random.default_rng(7)
    v = _rand_vec(rng, V, Nc, nrhs)
    links32 = g["links"].astype(np.complex64)
    got = oracle_lib.coarse_apply(cd, Nc, links32, v, nrhs=nrhs, dagger=dagger)
    M = g["coarse_dense"].conj().T if dagger else g["coarse_dense"]
    ref = (M @ v.astype(np.complex128).reshape(V * Nc, nrhs)).reshape(V, Nc, nrhs)
    # the only difference allowed is the fp32 rounding of the link entries handed to the oracle
    assert rel_l2_per_rhs(got, ref) < 5e-7
    # and with that rounding taken out (dense matrix rebuilt from the SAME fp32 links) it is exact
    A32 = assemble_dense(links32, cd)
    M32 = A32.conj().T if dagger else A32
    ref32 = (M32 @ v.astype(np.complex128).reshape(V * Nc, nrhs)).reshape(V, Nc, nrhs)
    assert rel_l2_per_rhs(got, ref32) < 1e-13


def test_galerkin_links_obey_generator_relation(galerkin_case):
    """Y_{-mu}(x+mu^) = Gamma Y_{+mu}(x)^dagger Gamma and X = Gamma X^dagger Gamma hold for links
    coarsened from a staggered stencil, i.e. the synthetic generator's relation is the physical one."""
    g = galerkin_case
    cd, Nc, links = g["coarse_dims"], g["Nc"], g["links"]
    gam = gamma_diag(Nc)
    gg = gam[:, None] * gam[None, :]
    nbr = neighbour_table(cd)
    scale = np.abs(links).max()
    for s in range(links.shape[0]):
        assert np.abs(links[s, 0] - gg * links[s, 0].conj().T).max() < 1e-13 * max(scale, 1)
        for mu in range(4):
            lhs = links[nbr[s, 1 + mu], 5 + mu]
            assert np.abs(lhs - gg * links[s, 1 + mu].conj().T).max() < 1e-13 * max(scale, 1)


# ---------------------------------------------------------------- 2. unit shifts
@pytest.mark.parametrize("dims", [(3, 2, 1, 4), (2, 2, 2, 2), (4, 3, 2, 5)])
def test_unit_shift_cases_are_exact(oracle_lib, dims):
    Nc, V = 4, int(np.prod(dims))
    g = site_grid(dims)
    # the input encodes its own coordinates: component a of site x holds (s(x) + 1) + i*(a+1)
    v = np.empty((V, Nc, 1), dtype=np.complex64)
    v[:, :, 0] = (np.arange(V)[:, None] + 1) + 1j * (np.arange(Nc)[None, :] + 1)
    for mu in range(4):
        for sign, m in ((+1, 1 + mu), (-1, 5 + mu)):
            links = np.zeros((V, 9, Nc, Nc), dtype=np.complex64)
            links[:, m] = np.eye(Nc)
            out = oracle_lib.coarse_apply(dims, Nc, links, v)
            src = np.roll(g, -sign, axis=3 - mu).reshape(-1)     # site x reads site x + sign*mu^
            assert np.array_equal(out[:, :, 0], v[src, :, 0].astype(np.complex128))
            # dagger of a pure forward shift is the backward shift (and vice versa)
            out_d = oracle_lib.coarse_apply(dims, Nc, links, v, dagger=1)
            src_d = np.roll(g, +sign, axis=3 - mu).reshape(-1)
            assert np.array_equal(out_d[:, :, 0], v[src_d, :, 0].astype(np.complex128))


# ---------------------------------------------------------------- 3. X only
def test_x_only_matches_einsum(oracle_lib):
    dims, Nc, nrhs = (3, 2, 2, 3), 6, 2
    V = int(np.prod(dims))
    rng = np.random.default_rng(3)
    links = np.zeros((V, 9, Nc, Nc), dtype=np.complex64)
    links[:, 0] = rng.standard_normal((V, Nc, Nc)) + 1j * rng.standard_normal((V, Nc, Nc))
    v = _rand_vec(rng, V, Nc, nrhs)
    X = links[:, 0].astype(np.complex128)
    v128 = v.astype(np.complex128)
    assert rel_l2(oracle_lib.coarse_apply(dims, Nc, links, v, nrhs=nrhs),
                  np.einsum("sij,sjr->sir", X, v128)) < 1e-14
    assert rel_l2(oracle_lib.coarse_apply(dims, Nc, links, v, nrhs=nrhs, dagger=1),
                  np.einsum("sji,sjr->sir", X.conj(), v128)) < 1e-14


# ---------------------------------------------------------------- 4. adjoint identity
@pytest.mark.parametrize("dims", [(1, 1, 1, 1), (2, 1, 3, 2), (4, 4, 4, 4), (3, 5, 2, 4)])
def test_adjoint_identity_arbitrary_links(oracle_lib, dims):
    Nc, V = 8, int(np.prod(dims))
    links = synth.make_arbitrary_links(dims, Nc, seed=11).numpy()
    rng = np.random.default_rng(5)
    u, v = _rand_vec(rng, V, Nc, 1), _rand_vec(rng, V, Nc, 1)
    Av = oracle_lib.coarse_apply(dims, Nc, links, v)
    Adu = oracle_lib.coarse_apply(dims, Nc, links, u, dagger=1)
    lhs = np.vdot(u.astype(np.complex128), Av)          # <u, A v>, conj on the left (reading R12)
    rhs = np.vdot(Adu, v.astype(np.complex128))         # <A^dagger u, v>
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)


# ---------------------------------------------------------------- 5. Gamma-Hermiticity
@pytest.mark.parametrize("dims,Nc", [((4, 4, 4, 4), 48), ((2, 3, 1, 4), 16)])
def test_gamma_hermiticity_of_generated_links(oracle_lib, dims, Nc):
    V = int(np.prod(dims))
    links = synth.make_gamma_hermitian_links(dims, Nc, seed=21).numpy()
    rng = np.random.default_rng(9)
    u, v = _rand_vec(rng, V, Nc, 1), _rand_vec(rng, V, Nc, 1)
    gam = gamma_diag(Nc)[None, :, None]
    GAv = gam * oracle_lib.coarse_apply(dims, Nc, links, v)
    GAu = gam * oracle_lib.coarse_apply(dims, Nc, links, u)
    lhs = np.vdot(u.astype(np.complex128), GAv)
    rhs = np.vdot(GAu, v.astype(np.complex128))
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)
    # equivalently A^dagger = Gamma A Gamma (a CHECK of the dagger path, not its implementation)
    Adv = oracle_lib.coarse_apply(dims, Nc, links, v, dagger=1)
    GAGv = gam * oracle_lib.coarse_apply(dims, Nc, links, (gam * v).astype(np.complex64))
    assert rel_l2(Adv, GAGv) < 1e-13


# ---------------------------------------------------------------- 6. linearity, block
def test_linearity(oracle_lib):
    dims, Nc = (3, 2, 2, 2), 8
    V = int(np.prod(dims))
    links = synth.make_arbitrary_links(dims, Nc, seed=31).numpy()
    # integer-valued inputs so that alpha*u + beta*v is exact in complex64
    rng = np.random.default_rng(13)
    u = (rng.integers(-8, 9, (V, Nc, 1)) + 1j * rng.integers(-8, 9, (V, Nc, 1))).astype(np.complex64)
    v = (rng.integers(-8, 9, (V, Nc, 1)) + 1j * rng.integers(-8, 9, (V, Nc, 1))).astype(np.complex64)
    alpha, beta = 2 - 3j, -1 + 4j
    w = (alpha * u + beta * v).astype(np.complex64)
    for dagger in (0, 1):
        Au = oracle_lib.coarse_apply(dims, Nc, links, u, dagger=dagger)
        Av = oracle_lib.coarse_apply(dims, Nc, links, v, dagger=dagger)
        Aw = oracle_lib.coarse_apply(dims, Nc, links, w, dagger=dagger)
        assert rel_l2(Aw, alpha * Au + beta * Av) < 1e-14


@pytest.mark.parametrize("dagger", [0, 1])
def test_block_apply_is_per_column(oracle_lib, dagger):
    dims, Nc, nrhs = (2, 3, 2, 2), 8, 5
    links = synth.make_arbitrary_links(dims, Nc, seed=41).numpy()
    v = synth.make_vectors(dims, Nc, nrhs, seed=42).numpy()
    blk = oracle_lib.coarse_apply(dims, Nc, links, v, nrhs=nrhs, dagger=dagger)
    for r in range(nrhs):
        col = oracle_lib.coarse_apply(dims, Nc, links, np.ascontiguousarray(v[:, :, r:r + 1]), dagger=dagger)
        assert np.array_equal(blk[:, :, r], col[:, :, 0])


def test_apply_sites_and_neighbours(oracle_lib):
    dims, Nc = (3, 4, 2, 3), 8
    V = int(np.prod(dims))
    links = synth.make_arbitrary_links(dims, Nc, seed=51).numpy()
    v = synth.make_vectors(dims, Nc, 2, seed=52).numpy()
    nbr = neighbour_table(dims)
    for s in (0, 5, V - 1):
        assert np.array_equal(oracle_lib.neighbours(dims, s), nbr[s])
    sites = np.array([0, 7, V - 1, 3, 3], dtype=np.int64)
    for dagger in (0, 1):
        full = oracle_lib.coarse_apply(dims, Nc, links, v, nrhs=2, dagger=dagger)
        part = oracle_lib.coarse_apply_sites(dims, Nc, links, v, sites, nrhs=2, dagger=dagger)
        assert np.array_equal(part, full[sites])


def test_bad_arguments_rejected(oracle_lib):
    links = np.zeros((1, 9, 2, 2), dtype=np.complex64)
    v = np.zeros((1, 2, 1), dtype=np.complex64)
    with pytest.raises(ValueError):
        oracle_lib.coarse_apply((1, 1, 1, 0), 2, links, v)
    with pytest.raises(ValueError):
        oracle_lib.coarse_apply((1, 1, 1, 1), 2, links, v, dagger=2)


# ---------------------------------------------------------------- 7. quantiser
def test_quantiser_properties(oracle_lib):
    Nc = 16
    links = synth.make_gamma_hermitian_links((2, 2, 2, 2), Nc, seed=61).numpy()
    links[3, 4] = 0                                   # an all-zero matrix
    links[5, 2] *= 1e-30                              # tiny but non-zero
    q, scales = oracle_lib.quantize_i16(links, Nc)
    flat = links.reshape(-1, Nc, Nc).view(np.float32).reshape(-1, Nc, Nc, 2)
    assert q.shape == flat.shape and scales.shape == (flat.shape[0],)
    assert q.min() >= -32767 and q.max() <= 32767
    amax = np.abs(flat).reshape(flat.shape[0], -1).max(axis=1)
    assert np.array_equal(scales, (amax / np.float32(32767.0)).astype(np.float32))
    deq = oracle_lib.dequantize_i16(q, scales, Nc)
    deq_f = np.stack([deq.real, deq.imag], axis=-1)
    err = np.abs(deq_f - flat.astype(np.float64)).reshape(flat.shape[0], -1).max(axis=1)
    # |deq - orig| <= scale/2, widened by the fp32 rounding of t = component/scale (|t| <= 32767,
    # so t is off by at most 32767 * 2^-24 before it is rounded to an integer)
    assert np.all(err <= (0.5 + 32767.0 * 2.0 ** -23) * scales.astype(np.float64))
    # the largest component maps to +-32767; the zero matrix round-trips to zeros with scale 0
    k = 3 * 9 + 4
    assert scales[k] == 0 and not q[k].any()
    nz = amax > 0
    assert np.all(np.abs(q).reshape(q.shape[0], -1).max(axis=1)[nz] == 32767)
    # idempotent: re-quantising the dequantised matrices gives the same integers
    q2, _ = oracle_lib.quantize_i16(deq.astype(np.complex64), Nc)
    # (deq cast to fp32 is q*scale rounded once; its max is 32767*scale so the scale is reproduced)
    assert np.abs(q2.astype(np.int32) - q.astype(np.int32)).max() <= 1
    assert (q2 != q).mean() < 1e-3


def test_quantiser_rounds_half_to_even_and_clamps(oracle_lib):
    Nc = 2
    m = np.zeros((1, Nc, Nc), dtype=np.complex64)
    # amax = 32767 -> scale exactly 1 -> q = rint(component)
    m[0, 0, 0] = 32767 + 2.5j
    m[0, 0, 1] = 3.5 - 2.5j
    m[0, 1, 0] = -32767 + 0.5j
    m[0, 1, 1] = -0.5 + 1.5j
    q, scales = oracle_lib.quantize_i16(m, Nc)
    assert scales[0] == 1.0
    assert q[0].tolist() == [[[32767, 2], [4, -2]], [[-32767, 0], [0, 2]]]


def test_i16_apply_equals_apply_on_dequantised_links(oracle_lib):
    """O3: the int16 path is the c64 definition evaluated on q*scale.  Checked against the dense
    assembly of the dequantised (double) links, which shares nothing with the oracle."""
    dims, Nc = (2, 3, 2, 2), 8
    V = int(np.prod(dims))
    links = synth.make_gamma_hermitian_links(dims, Nc, seed=71).numpy()
    q, scales = oracle_lib.quantize_i16(links, Nc)
    deq = oracle_lib.dequantize_i16(q, scales, Nc).reshape(V, 9, Nc, Nc)
    # dequantiser itself against plain numpy
    assert np.array_equal(deq.real, q[..., 0].astype(np.float64).reshape(V, 9, Nc, Nc)
                          * scales.astype(np.float64).reshape(V, 9, 1, 1))
    v = synth.make_vectors(dims, Nc, 2, seed=72).numpy()
    A = assemble_dense(deq, dims)
    for dagger in (0, 1):
        got = oracle_lib.coarse_apply(dims, Nc, q.reshape(V, 9, Nc, Nc, 2), v, nrhs=2, dagger=dagger,
                                      link_precision=oracle_lib.LINK_I16, scales=scales)
        M = A.conj().T if dagger else A
        ref = (M @ v.astype(np.complex128).reshape(V * Nc, 2)).reshape(V, Nc, 2)
        assert rel_l2_per_rhs(got, ref) < 1e-13


# ---------------------------------------------------------------- 8. the paper's storage count
def test_storage_count_golden():
    """nine 48^2 matrices per 2^4 super-site = 9*48^2/16 = 1296 complex per fine site."""
    vals = {}
    with open(os.path.join(GOLDEN, "storage_count.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                vals[k.strip()] = int(v)
    links = synth.make_gamma_hermitian_links((1, 1, 1, 1), vals["Nc"], seed=1)
    per_site = links.numel()                           # complex entries per coarse site
    assert links.shape[1] == vals["matrices_per_site"]
    assert per_site == vals["matrices_per_site"] * vals["Nc"] ** 2
    assert per_site // vals["fine_sites_per_supersite"] == vals["complex_per_fine_site"]
