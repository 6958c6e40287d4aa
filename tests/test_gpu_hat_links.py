"""GPU parity for coarse_op_build_hat_links: the block-preconditioned
links Yhat_m = X^-1 Y_m and X^-1 itself, built on the device, against oracle.hat_links (numpy fp64 solve,
pinned in tests/test_oracle_evenodd_pins.py).  The kernel works in fp64 and rounds to complex64 once, so
the bound is fp32 rounding: relative L2 <= 1e-6 PER MATRIX (cond(X) of the generator's X is 5-30; the
fp64 factorisation error cond x 1e-16 is far below the final rounding).  Then the whole f1 chain runs
without the oracle's numpy in the product path: GPU hat links -> Schur-hat operator -> parity."""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.helpers import rel_l2_per_rhs

pytestmark = pytest.mark.gpu
TOL_MATRIX = 1e-6


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible (there is no CPU fallback)")
    torch.cuda.set_device(0)


def _per_matrix_err(got, ref):
    d = np.linalg.norm((got - ref).reshape(got.shape[0], 9, -1), axis=2)
    n = np.linalg.norm(ref.reshape(ref.shape[0], 9, -1), axis=2)
    return float((d / n).max())


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [6, 32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("slot0", [cop.HAT_SLOT0_IDENTITY, cop.HAT_SLOT0_XINV])
def test_hat_links_match_the_oracle(oracle_lib, dims, Nc, prec, slot0):
    if Nc >= 96 and dims == (4, 4, 4, 4):
        dims = (2, 2, 3, 2)                        # keep numpy's per-site solves in seconds
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, 31 + Nc, device="cuda")
    scales = None
    links_h = links.cpu().numpy().astype(np.complex128)
    links_d = links
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links_d = q
        links_h = oracle_lib.dequantize_i16(q.cpu().numpy(), scales.cpu().numpy(), Nc).reshape(V, 9, Nc, Nc)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links_d, scales)
    out = torch.full((V, 9, Nc, Nc), complex(float("nan"), float("nan")), dtype=torch.complex64, device="cuda")
    info = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    op.build_hat_links(out, slot0=slot0, info=info)
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    got = out.cpu().numpy()
    assert np.isfinite(got.view(np.float32)).all()
    ref = oracle_lib.hat_links(links_h, slot0_inverse=(slot0 == cop.HAT_SLOT0_XINV))
    err = _per_matrix_err(got.astype(np.complex128), ref)
    assert err <= TOL_MATRIX, f"per-matrix rel-L2 {err:.3e} dims={dims} Nc={Nc} prec={prec}"
    if slot0 == cop.HAT_SLOT0_IDENTITY:
        assert np.array_equal(got[:, 0], np.broadcast_to(np.eye(Nc, dtype=np.complex64), (V, Nc, Nc)))
    op.close()


def test_hat_links_need_pivoting_and_report_singular_sites(oracle_lib):
    """X with a zero leading entry (needs a row exchange) and one singular site."""
    dims, Nc = (2, 1, 1, 2), 8
    V = 4
    links = synth.make_arbitrary_links(dims, Nc, 3, device="cuda")
    links[0, 0, 0, 0] = 0                          # first pivot candidate is exactly zero
    links[1, 0] = torch.roll(torch.eye(Nc, dtype=torch.complex64, device="cuda"), 3, dims=0)   # a permutation matrix
    links[3, 0, :, 2] = 0                          # singular: a zero column
    op = cop.CoarseOp(dims, Nc).set_links(links)
    out = torch.empty((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    info = torch.zeros((1,), dtype=torch.int32, device="cuda")
    op.build_hat_links(out, slot0=cop.HAT_SLOT0_XINV, info=info)
    torch.cuda.synchronize()
    assert int(info.item()) == 1
    got = out.cpu().numpy()[:3].astype(np.complex128)
    ref = oracle_lib.hat_links(links.cpu().numpy()[:3], slot0_inverse=True)
    assert _per_matrix_err(got, ref) <= TOL_MATRIX
    op.close()


def test_hat_argument_errors():
    L = cop.lib()
    h = cop.coarse_op_create((2, 2, 2, 2), 8, cop.LINK_C64)
    links = torch.zeros((16, 9, 8, 8), dtype=torch.complex64, device="cuda")
    out = torch.zeros_like(links)
    work = torch.empty(cop.coarse_op_hat_work_bytes(h), dtype=torch.uint8, device="cuda")
    assert L.coarse_op_build_hat_links(h, out.data_ptr(), 0, work.data_ptr(), None, None) == cop.ENOTREADY
    assert L.coarse_op_set_links(h, links.data_ptr(), None) == cop.OK
    assert L.coarse_op_build_hat_links(h, links.data_ptr(), 0, work.data_ptr(), None, None) == cop.EINVAL   # in place
    assert L.coarse_op_build_hat_links(h, out.data_ptr(), 7, work.data_ptr(), None, None) == cop.EINVAL     # slot0 mode
    assert L.coarse_op_build_hat_links(h, out.data_ptr(), 0, None, None, None) == cop.EINVAL
    assert L.coarse_op_build_hat_links(h, out.data_ptr(), 0, out.data_ptr(), None, None) == cop.EINVAL      # work overlaps out
    cop.coarse_op_destroy(h)


@pytest.mark.parametrize("Nc,prec_hat", [(48, cop.LINK_C64), (64, cop.LINK_I16), (128, cop.LINK_C64)])
@pytest.mark.parametrize("parity", [0, 1])
@pytest.mark.parametrize("dagger", [0, 1])
def test_schur_hat_chain_entirely_on_the_gpu(oracle_lib, Nc, prec_hat, parity, dagger):
    """f1 end to end on the device: links -> coarse_op_build_hat_links (-> coarse_op_quantize_i16) -> two
    parity-restricted launches = Shat_p v = v - Dhat_pq Dhat_qp v.  The oracle gets the SAME hat links (the
    device-built bits, brought back) for the apply and, separately, checks them against its own solve."""
    dims = (4, 2, 2, 4) if Nc < 128 else (2, 2, 2, 2)
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, 77, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links)
    hat = torch.empty((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    op.build_hat_links(hat)
    torch.cuda.synchronize()
    ref_hat = oracle_lib.hat_links(links.cpu().numpy())
    assert _per_matrix_err(hat.cpu().numpy().astype(np.complex128), ref_hat) <= TOL_MATRIX
    hat_links_d, hat_scales, hat_h, hat_scales_h = hat, None, hat.cpu().numpy(), None
    if prec_hat == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        hat_scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(hat, Nc, q, hat_scales)
        torch.cuda.synchronize()
        hat_links_d, hat_h, hat_scales_h = q, q.cpu().numpy(), hat_scales.cpu().numpy()
    ophat = cop.CoarseOp(dims, Nc, prec_hat).set_links(hat_links_d, hat_scales)
    par = torch.as_tensor(oracle_lib.site_parities(dims), device="cuda")
    v = synth.make_vectors(dims, Nc, 1, 78, device="cuda")
    v[par != parity] = 0
    t = torch.zeros_like(v)
    out = torch.zeros_like(v)
    ophat.apply_parts(None, v, t, dagger=dagger, parity=1 - parity, local=cop.LOCAL_NONE, alpha=0.0, beta=1.0)
    ophat.apply_parts(v, t, out, dagger=dagger, parity=parity, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)
    torch.cuda.synchronize()
    q_par = 1 - parity
    tt = oracle_lib.coarse_apply_parts(dims, Nc, hat_h, None, v.cpu().numpy(), dagger=dagger, parity=q_par, local=0,
                                       alpha=0.0, beta=1.0, link_precision=prec_hat, scales=hat_scales_h)
    ref = oracle_lib.coarse_apply_parts(dims, Nc, hat_h, v.cpu().numpy(), tt.astype(np.complex64), dagger=dagger,
                                        parity=parity, local=2, alpha=1.0, beta=-1.0, link_precision=prec_hat,
                                        scales=hat_scales_h)
    mask = (par == parity).cpu().numpy()
    assert rel_l2_per_rhs(out.cpu().numpy()[mask], ref[mask]) <= 1e-5
    op.close(); ophat.close()
