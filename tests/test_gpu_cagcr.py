"""GPU parity for CA-GCR(s) against the oracle's definition
(least squares over the Krylov space, tests/test_oracle_cagcr_pins.py).

What is compared, and why: the minimised residual is what the method defines stably,
so ||b - A x_gpu|| (evaluated by the fp64 oracle apply) must match the oracle's optimum to 1e-4
relative, and the norms the solve kernel reports must match the true ones.  The iterate x itself is
compared too, at ONE bound for every s: 1e-5 relative, the tolerance of the apply (the Chebyshev basis on
the device-estimated interval keeps the basis well conditioned up to s = 16)."""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.helpers import gpu_hat_links, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible (there is no CPU fallback)")
    torch.cuda.set_device(0)


def _case(oracle_lib, dims, Nc, prec, s, cycles, x_is_zero, shift=12.0, seed=101):
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, seed, device="cuda")
    links[:, 0] += shift * torch.eye(Nc, dtype=torch.complex64, device="cuda")
    scales = scales_h = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links, scales_h = q, scales.cpu().numpy()
    links_h = links.cpu().numpy()
    b = synth.make_vectors(dims, Nc, 1, seed + 1, device="cuda")
    x = torch.zeros_like(b) if x_is_zero else 0.05 * synth.make_vectors(dims, Nc, 1, seed + 2, device="cuda")
    x0_h = x.cpu().numpy().reshape(-1)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    info = torch.zeros((cycles, 3), dtype=torch.float64, device="cuda")
    op.cagcr(b, x, s=s, cycles=cycles, x_is_zero=x_is_zero, info=info)
    torch.cuda.synchronize()
    assert op.last_launches == cycles * (2 * s + 2) + 2 + (0 if x_is_zero else 2)
    apply_fn = lambda v: oracle_lib.coarse_apply(dims, Nc, links_h, v.reshape(V, Nc, 1), link_precision=prec,
                                                 scales=scales_h).reshape(-1)
    b_h = b.cpu().numpy().reshape(-1)
    x_ref, norms = oracle_lib.cagcr(apply_fn, b_h, x0_h, s, cycles)
    x_gpu = x.cpu().numpy().reshape(-1)
    r_gpu = np.linalg.norm(b_h.astype(np.complex128) - apply_fn(x_gpu))
    info_h = info.cpu().numpy()
    # conditioning of the first cycle's basis (for the bound on x)
    P = [(b_h.astype(np.complex128) - (apply_fn(x0_h.astype(np.complex64)) if not x_is_zero else 0)).astype(np.complex64)]
    for _ in range(s):
        P.append(apply_fn(P[-1]).astype(np.complex64))
    condQ = np.linalg.cond(np.stack(P[1:], axis=1).astype(np.complex128))
    op.close()
    return dict(x_err=rel_l2(x_gpu, x_ref), r_gpu=r_gpu, norms=norms, info=info_h, condQ=condQ)


@pytest.mark.parametrize("dims,Nc", [((4, 4, 4, 4), 48), ((3, 2, 2, 4), 64), ((2, 2, 2, 2), 128)])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("s,cycles", [(8, 1), (4, 3), (1, 2), (16, 1)])
@pytest.mark.parametrize("x_is_zero", [True, False])
def test_cagcr_against_oracle(oracle_lib, dims, Nc, prec, s, cycles, x_is_zero):
    res = _case(oracle_lib, dims, Nc, prec, s, cycles, x_is_zero)
    norms, info = res["norms"], res["info"]
    # The oracle is the true minimiser (fp64 Arnoldi); the CUDA path reaches it on the Chebyshev basis of the
    # interval it estimates itself.  One bound for every s (the power basis this replaced needed 1e-4 at s = 8
    # and 1e-3 at s = 16, and dropped half its vectors there).
    floor = 2e-6 * norms[0]
    # the residual the GPU iterate really has is the oracle's optimum
    assert abs(res["r_gpu"] - norms[-1]) <= 1e-4 * norms[-1] + floor, (res["r_gpu"], norms)
    # what the solve kernel reports: ||r0||^2 per cycle and the predicted ||r||^2 after it
    for c in range(cycles):
        assert abs(np.sqrt(info[c, 0]) - norms[c]) <= 1e-4 * norms[c] + floor
        assert info[c, 2] == s                                          # the whole basis is kept, at every s
    assert abs(np.sqrt(max(info[-1, 1], 0.0)) - norms[-1]) <= 1e-3 * norms[-1] + 5 * floor
    # the iterate itself
    assert res["x_err"] <= 1e-5 * cycles, (res["x_err"], res["condQ"])


@pytest.mark.parametrize("s", [8, 16])
def test_cagcr_on_a_baseline_sized_lattice(oracle_lib, s):
    """BASELINE config C3's shape (8^3 x 12, Nc = 128; the paper's level-2 operator), one CA-GCR(s) cycle: the
    residual the device reports must be the residual the fp64 oracle apply measures for the device iterate,
    and a cycle must reduce it (the full minimiser is not recomputed at this size)."""
    cfg = synth.config("C3")
    dims, Nc = cfg["dims"], cfg["Nc"]
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device="cuda")
    links[:, 0] += 12.0 * torch.eye(Nc, dtype=torch.complex64, device="cuda")
    b = synth.make_vectors(dims, Nc, 1, cfg["seed"] + 1, device="cuda")
    x = torch.zeros_like(b)
    op = cop.CoarseOp(dims, Nc).set_links(links)
    info = torch.zeros((1, 3), dtype=torch.float64, device="cuda")
    op.cagcr(b, x, s=s, cycles=1, info=info)
    torch.cuda.synchronize()
    links_h = links.cpu().numpy()
    ax = oracle_lib.coarse_apply(dims, Nc, links_h, x.cpu().numpy())
    b_h = b.cpu().numpy().astype(np.complex128)
    r_true = np.linalg.norm(b_h - ax)
    r0 = np.linalg.norm(b_h)
    info_h = info.cpu().numpy()
    assert info_h[0, 2] == s
    assert abs(np.sqrt(info_h[0, 0]) - r0) <= 1e-6 * r0
    assert abs(np.sqrt(max(info_h[0, 1], 0.0)) - r_true) <= 1e-3 * r_true + 2e-6 * r0, (info_h, r_true)
    assert r_true < 1e-3 * r0
    op.close()


def test_cagcr_reduces_the_residual_on_a_baseline_shaped_operator(oracle_lib):
    """C1's generator (Gamma-Hermitian links) with a diagonal shift that makes it smoother-friendly."""
    res = _case(oracle_lib, (4, 4, 4, 4), 48, cop.LINK_C64, 8, 2, True, shift=10.0, seed=20221201)
    assert res["norms"][-1] < 0.05 * res["norms"][0]
    # two cycles take the fp64 oracle to 1e-6 of ||r0||; the complex64 iterate and residual recurrence of the
    # CUDA path stall at its single-precision floor (a few 1e-5): a smoother, not a solver
    assert res["r_gpu"] <= 1e-4 * res["norms"][0]


@pytest.mark.parametrize("dims,Nc", [((4, 4, 4, 4), 48), ((2, 4, 2, 4), 128)])
@pytest.mark.parametrize("parity", [0, 1])
@pytest.mark.parametrize("x_is_zero", [True, False])
def test_cagcr_on_the_schur_hat_operator(oracle_lib, dims, Nc, parity, x_is_zero):
    """The paper's level-2/3 combination (Table 1): CA-GCR(8) on the Schur-preconditioned operator."""
    V, s, cycles = synth.lattice_volume(dims), 8, 2
    links = synth.make_arbitrary_links(dims, Nc, 7).numpy()
    links[:, 0] += 6.0 * np.eye(Nc, dtype=np.complex64)
    hat_d, hat = gpu_hat_links(oracle_lib, dims, Nc, links)       # the block-preconditioned links come from the device
    par = oracle_lib.site_parities(dims)
    mask = torch.as_tensor(par == parity, device="cuda")
    b = synth.make_vectors(dims, Nc, 1, 8, device="cuda")
    b[~mask] = 0
    x = torch.zeros_like(b) if x_is_zero else 0.05 * synth.make_vectors(dims, Nc, 1, 9, device="cuda")
    x[~mask] = 0
    x0_h = x.cpu().numpy().reshape(-1)
    op = cop.CoarseOp(dims, Nc).set_links(hat_d)
    info = torch.zeros((cycles, 3), dtype=torch.float64, device="cuda")
    op.cagcr(b, x, s=s, cycles=cycles, x_is_zero=x_is_zero, info=info, schur_parity=parity)
    torch.cuda.synchronize()
    assert op.last_launches == cycles * (3 * s + 2) + 2 + (0 if x_is_zero else 3)
    f = lambda v: oracle_lib.schur_hat_apply(dims, Nc, hat, v.reshape(V, Nc, 1), parity).reshape(-1)
    b_h = b.cpu().numpy().reshape(-1)
    x_ref, norms = oracle_lib.cagcr(f, b_h, x0_h, s, cycles)
    x_gpu = x.cpu().numpy().reshape(-1)
    assert np.all(x_gpu.reshape(V, Nc)[par != parity] == 0)
    r_gpu = np.linalg.norm(b_h.astype(np.complex128) - f(x_gpu))
    assert abs(r_gpu - norms[-1]) <= 1e-4 * norms[-1] + 5e-5 * norms[0], (r_gpu, norms)
    assert norms[-1] < 0.1 * norms[0]
    info_h = info.cpu().numpy()
    assert abs(np.sqrt(info_h[0, 0]) - norms[0]) <= 1e-5 * norms[0]
    op.close()


def _cheb_case(oracle_lib, dims, Nc, prec, s, cycles, x_is_zero, lam=(7.5, 16.5), shift=12.0, seed=201):
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, seed, device="cuda")
    links[:, 0] += shift * torch.eye(Nc, dtype=torch.complex64, device="cuda")
    scales = scales_h = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links, scales_h = q, scales.cpu().numpy()
    links_h = links.cpu().numpy()
    b = synth.make_vectors(dims, Nc, 1, seed + 1, device="cuda")
    x = torch.zeros_like(b) if x_is_zero else 0.05 * synth.make_vectors(dims, Nc, 1, seed + 2, device="cuda")
    x0_h = x.cpu().numpy().reshape(-1)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    info = torch.zeros((cycles, 3), dtype=torch.float64, device="cuda")
    op.cagcr_cheb(b, x, lam[0], lam[1], s=s, cycles=cycles, x_is_zero=x_is_zero, info=info)
    torch.cuda.synchronize()
    assert op.last_launches == cycles * (2 * s + 2) + 1 + (0 if x_is_zero else 2)
    # the same start on the interval the library estimates itself, for comparison
    xp = torch.zeros_like(b) if x_is_zero else torch.as_tensor(x0_h.reshape(V, Nc, 1), device="cuda").clone()
    op.cagcr(b, xp, s=s, cycles=cycles, x_is_zero=x_is_zero)
    torch.cuda.synchronize()
    f = lambda v: oracle_lib.coarse_apply(dims, Nc, links_h, v.reshape(V, Nc, 1), link_precision=prec,
                                          scales=scales_h).reshape(-1)
    b_h = b.cpu().numpy().reshape(-1)
    x_ref, norms = oracle_lib.cagcr(f, b_h, x0_h, s, cycles)
    r_cheb = np.linalg.norm(b_h.astype(np.complex128) - f(x.cpu().numpy().reshape(-1)))
    r_pow = np.linalg.norm(b_h.astype(np.complex128) - f(xp.cpu().numpy().reshape(-1)))
    op.close()
    return r_cheb, r_pow, norms, info.cpu().numpy(), rel_l2(x.cpu().numpy().reshape(-1), x_ref)


@pytest.mark.parametrize("dims,Nc", [((4, 4, 4, 4), 48), ((2, 2, 2, 4), 128)])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("s,cycles", [(16, 1), (8, 2), (3, 2), (1, 1)])
@pytest.mark.parametrize("x_is_zero", [True, False])
def test_cagcr_chebyshev_basis(oracle_lib, dims, Nc, prec, s, cycles, x_is_zero):
    """Caller-supplied interval: the whole basis is kept at s = 16, the iterate matches the fp64 oracle to 1e-5
    (measured 2-3e-7) and the residual to the single-precision floor; the device-estimated interval
    (coarse_op_cagcr) reaches the same residual."""
    r_cheb, r_pow, norms, info, x_err = _cheb_case(oracle_lib, dims, Nc, prec, s, cycles, x_is_zero)
    assert np.all(info[:, 2] == s)                                    # no truncation, even at s = 16
    assert abs(r_cheb - norms[-1]) <= 1e-4 * norms[-1] + 2e-6 * norms[0], (r_cheb, r_pow, norms)
    assert abs(r_pow - r_cheb) <= 1e-4 * norms[-1] + 2e-6 * norms[0]  # estimated interval: the same minimum
    assert abs(np.sqrt(info[0, 0]) - norms[0]) <= 1e-5 * norms[0]
    assert x_err <= 1e-5, x_err                                       # the iterate itself, at every s


def test_cagcr_chebyshev_on_schur_operator_and_errors(oracle_lib):
    dims, Nc, parity, s = (4, 4, 4, 4), 48, 0, 12
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 7).numpy()
    links[:, 0] += 6.0 * np.eye(Nc, dtype=np.complex64)
    hat_d, hat = gpu_hat_links(oracle_lib, dims, Nc, links)
    par = oracle_lib.site_parities(dims)
    mask = torch.as_tensor(par == parity, device="cuda")
    b = synth.make_vectors(dims, Nc, 1, 8, device="cuda")
    b[~mask] = 0
    x = torch.zeros_like(b)
    op = cop.CoarseOp(dims, Nc).set_links(hat_d)
    info = torch.zeros((1, 3), dtype=torch.float64, device="cuda")
    op.cagcr_cheb(b, x, 0.3, 1.7, s=s, schur_parity=parity, info=info)       # Shat = 1 - Dhat Dhat: spectrum around 1
    torch.cuda.synchronize()
    f = lambda v: oracle_lib.schur_hat_apply(dims, Nc, hat, v.reshape(V, Nc, 1), parity).reshape(-1)
    b_h = b.cpu().numpy().reshape(-1)
    x_ref, norms = oracle_lib.cagcr(f, b_h, np.zeros_like(b_h), s, 1)
    r_gpu = np.linalg.norm(b_h.astype(np.complex128) - f(x.cpu().numpy().reshape(-1)))
    assert info[0, 2].item() == s
    assert abs(r_gpu - norms[-1]) <= 1e-4 * norms[-1] + 2e-6 * norms[0], (r_gpu, norms)
    assert rel_l2(x.cpu().numpy().reshape(-1), x_ref) <= 1e-5
    L = cop.lib()
    w = torch.zeros(cop.coarse_op_cagcr_cheb_work_bytes(op._h, s), dtype=torch.uint8, device="cuda")
    args = lambda lo, hi, sp: (op._h, b.data_ptr(), x.data_ptr(), s, 1, 1, lo, hi, sp, w.data_ptr(), None, None)
    assert L.coarse_op_cagcr_cheb(*args(2.0, 1.0, -1)) == cop.EINVAL
    assert L.coarse_op_cagcr_cheb(*args(1.0, 2.0, 2)) == cop.EINVAL
    assert L.coarse_op_cagcr_cheb(*args(1.0, 2.0, -1)) == cop.OK
    torch.cuda.synchronize()
    assert cop.coarse_op_cagcr_cheb_work_bytes(op._h, 17) == 0
    op.close()


def test_cagcr_is_bit_reproducible():
    dims, Nc = (4, 4, 2, 2), 48
    links = synth.make_arbitrary_links(dims, Nc, 1, device="cuda")
    links[:, 0] += 12.0 * torch.eye(Nc, dtype=torch.complex64, device="cuda")
    b = synth.make_vectors(dims, Nc, 1, 2, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links)
    outs = []
    for _ in range(2):
        x = torch.empty_like(b)
        op.cagcr(b, x, s=8, cycles=2)
        torch.cuda.synchronize()
        outs.append(x)
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[1]))
    op.close()


def test_cagcr_argument_errors():
    L = cop.lib()
    dims, Nc, V = (2, 2, 2, 2), 48, 16
    h = cop.coarse_op_create(dims, Nc, cop.LINK_C64)
    assert cop.coarse_op_cagcr_work_bytes(h, 8) >= 18 * V * Nc * 8
    assert cop.coarse_op_cagcr_work_bytes(h, 0) == 0 and cop.coarse_op_cagcr_work_bytes(h, 17) == 0
    b = torch.zeros((V, Nc, 1), dtype=torch.complex64, device="cuda")
    x = torch.zeros_like(b)
    w = torch.zeros(cop.coarse_op_cagcr_work_bytes(h, 8), dtype=torch.uint8, device="cuda")
    assert L.coarse_op_cagcr(h, b.data_ptr(), x.data_ptr(), 8, 1, 1, w.data_ptr(), None, None) == cop.ENOTREADY
    links = torch.zeros((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    assert L.coarse_op_set_links(h, links.data_ptr(), None) == cop.OK
    assert L.coarse_op_cagcr(h, b.data_ptr(), x.data_ptr(), 0, 1, 1, w.data_ptr(), None, None) == cop.EINVAL
    assert L.coarse_op_cagcr(h, b.data_ptr(), x.data_ptr(), 17, 1, 1, w.data_ptr(), None, None) == cop.EINVAL
    assert L.coarse_op_cagcr(h, b.data_ptr(), x.data_ptr(), 8, 0, 1, w.data_ptr(), None, None) == cop.EINVAL
    assert L.coarse_op_cagcr(h, None, x.data_ptr(), 8, 1, 1, w.data_ptr(), None, None) == cop.EINVAL
    # a zero operator: the Gram matrix is singular, the basis truncates to nothing and x stays 0
    info = torch.zeros(3, dtype=torch.float64, device="cuda")
    b.fill_(1.0)
    assert L.coarse_op_cagcr(h, b.data_ptr(), x.data_ptr(), 8, 1, 1, w.data_ptr(), info.data_ptr(), None) == cop.OK
    torch.cuda.synchronize()
    assert info[2].item() == 0 and torch.all(x == 0)
    cop.coarse_op_destroy(h)
