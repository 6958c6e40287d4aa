"""GPU parity for the even/odd building block: coarse_op_apply_parts and the
Schur compositions built from it, against the oracle's O7 / schur_* (tests/test_oracle_evenodd_pins.py
pins those).  Tolerance as for the plain apply: relative L2 <= 1e-5 per output vector over the sites
of the parity set; sites of the other parity must be left untouched (checked with a NaN prefill)."""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.helpers import gpu_hat_links, rel_l2_per_rhs

pytestmark = pytest.mark.gpu
TOL = 1e-5


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible (there is no CPU fallback)")
    torch.cuda.set_device(0)


def _make(oracle_lib, dims, Nc, prec, seed, nrhs):
    links = synth.make_arbitrary_links(dims, Nc, seed, device="cuda")
    V = synth.lattice_volume(dims)
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        sc = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, sc)
        torch.cuda.synchronize()
        links_d, scales_d, links_h, scales_h = q, sc, q.cpu().numpy(), sc.cpu().numpy()
    else:
        links_d, scales_d, links_h, scales_h = links, None, links.cpu().numpy(), None
    u = synth.make_vectors(dims, Nc, nrhs, seed + 1, device="cuda")
    w = synth.make_vectors(dims, Nc, nrhs, seed + 2, device="cuda")
    return links_d, scales_d, links_h, scales_h, u, w


def _check_parts(oracle_lib, dims, Nc, prec, nrhs, dagger, parity, local, path, alpha=0.75, beta=-1.25, opts=None):
    V = synth.lattice_volume(dims)
    links_d, scales_d, links_h, scales_h, u, w = _make(oracle_lib, dims, Nc, prec, 4321, nrhs)
    out = torch.full((V, Nc, nrhs), complex(float("nan"), float("nan")), dtype=torch.complex64, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links_d, scales_d).set_option(cop.OPT_PATH, path)
    for k, v in (opts or {}).items():
        op.set_option(k, v)
    op.apply_parts(u if local else None, w, out, nrhs=nrhs, dagger=dagger, parity=parity, local=local,
                   alpha=alpha, beta=beta)
    torch.cuda.synchronize()
    if path != cop.PATH_TENSOR:
        want = 1
    elif prec == cop.LINK_I16:      # integer tensor-core kernel: + one scale pre-pass per operand and column group
        want = ((nrhs + 15) // 16) * (2 + (1 if local == 1 else 0))
    else:
        want = (nrhs + 15) // 16
    assert op.last_path == path and op.last_launches == want
    ref = oracle_lib.coarse_apply_parts(dims, Nc, links_h, u.cpu().numpy() if local else None, w.cpu().numpy(),
                                        nrhs=nrhs, dagger=dagger, parity=parity, local=local, alpha=alpha,
                                        beta=beta, link_precision=prec, scales=scales_h)
    got = out.cpu().numpy()
    par = oracle_lib.site_parities(dims)
    mask = np.ones(V, bool) if parity == 2 else (par == parity)
    assert np.isfinite(got[mask].view(np.float32)).all()
    assert np.isnan(got[~mask].view(np.float32)).all(), "sites of the other parity were written"
    err = rel_l2_per_rhs(got[mask], ref[mask])
    assert err <= TOL, f"rel-L2 {err:.3e} dims={dims} Nc={Nc} prec={prec} dagger={dagger} parity={parity} local={local}"
    op.close()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (6, 2, 4, 2)])
@pytest.mark.parametrize("Nc", [48, 64, 128])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("parity", [0, 1, 2])
@pytest.mark.parametrize("local", [0, 1, 2])
def test_parts_stream(oracle_lib, dims, Nc, prec, dagger, parity, local):
    if Nc == 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 4)
    _check_parts(oracle_lib, dims, Nc, prec, 1, dagger, parity, local, cop.PATH_STREAM)


@pytest.mark.parametrize("Nc", [32, 96, 192])
@pytest.mark.parametrize("dagger", [0, 1])
def test_parts_stream_other_nc_and_fine_geometry(oracle_lib, Nc, dagger):
    _check_parts(oracle_lib, (2, 2, 4, 2), Nc, cop.LINK_C64, 1, dagger, 1, 2, cop.PATH_STREAM)
    _check_parts(oracle_lib, (2, 2, 4, 2), Nc, cop.LINK_I16, 1, dagger, 0, 1, cop.PATH_STREAM,
                 opts={cop.OPT_FINE: 2, cop.OPT_STAGES: 3})


@pytest.mark.parametrize("nrhs", [1, 3])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("parity", [0, 1, 2])
@pytest.mark.parametrize("local", [0, 1, 2])
def test_parts_simple(oracle_lib, nrhs, dagger, parity, local):
    _check_parts(oracle_lib, (4, 2, 2, 4), 8, cop.LINK_C64, nrhs, dagger, parity, local, cop.PATH_SIMPLE)
    _check_parts(oracle_lib, (2, 2, 2, 2), 48, cop.LINK_I16, nrhs, dagger, parity, local, cop.PATH_SIMPLE)


@pytest.mark.parametrize("Nc", [48, 64, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [3, 8, 16, 18])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("parity", [0, 1, 2])
@pytest.mark.parametrize("local", [0, 1, 2])
def test_parts_tensor(oracle_lib, Nc, prec, nrhs, dagger, parity, local):
    """Multi-RHS parts apply on the TENSOR kernel: parity-restricted site list, X stage on / off, alpha and
    beta folded into the B operand, identity term added in the epilogue (L127/L135 + L200)."""
    dims = (2, 2, 4, 2) if Nc >= 128 else (4, 2, 2, 4)
    _check_parts(oracle_lib, dims, Nc, prec, nrhs, dagger, parity, local, cop.PATH_TENSOR)


@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [2, 3, 4])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("parity,local", [(0, 0), (1, 1), (2, 2), (0, 2), (1, 0), (2, 1)])
def test_parts_stream_few_rhs(oracle_lib, Nc, prec, nrhs, dagger, parity, local):
    """2-4 right-hand sides (3 = one propagator) of the parts apply on the STREAM-MR kernel: parity list,
    X stage on / off, alpha / beta folded into the vector operand, identity term added at the store."""
    dims = (2, 2, 4, 2) if Nc >= 128 else (4, 2, 2, 4)
    _check_parts(oracle_lib, dims, Nc, prec, nrhs, dagger, parity, local, cop.PATH_STREAM)


def test_parts_auto_routes_few_rhs():
    small, large = (2, 2, 2, 2), (4, 4, 4, 10)        # int16, 2-3 RHS: TENSOR needs two work items per SM, else STREAM-MR
    for dims, Nc, prec, nrhs, want in ((small, 48, cop.LINK_C64, 3, cop.PATH_STREAM), (small, 64, cop.LINK_I16, 4, cop.PATH_TENSOR),
                                       (large, 64, cop.LINK_I16, 2, cop.PATH_TENSOR), (small, 64, cop.LINK_I16, 2, cop.PATH_STREAM),
                                       (small, 48, cop.LINK_I16, 2, cop.PATH_STREAM), (large, 128, cop.LINK_I16, 3, cop.PATH_TENSOR),
                                       (small, 128, cop.LINK_I16, 3, cop.PATH_STREAM), (small, 128, cop.LINK_C64, 2, cop.PATH_STREAM)):
        V = synth.lattice_volume(dims)
        if prec == cop.LINK_C64:
            links, scales = torch.zeros((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda"), None
        else:
            links = torch.zeros((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
            scales = torch.ones((V, 9), dtype=torch.float32, device="cuda")
        u = torch.zeros((V, Nc, nrhs), dtype=torch.complex64, device="cuda")
        w, out = torch.zeros_like(u), torch.zeros_like(u)
        op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
        op.apply_parts(u, w, out, nrhs=nrhs, parity=cop.PARITY_ODD, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)
        torch.cuda.synchronize()
        assert op.last_path == want, (Nc, prec, nrhs, op.last_path)
        op.close()


def test_parts_auto_routes_multi_rhs_to_tensor():
    dims, Nc, nrhs = (2, 2, 2, 2), 48, 5
    links = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    u = synth.make_vectors(dims, Nc, nrhs, 6, device="cuda")
    w = synth.make_vectors(dims, Nc, nrhs, 7, device="cuda")
    out = torch.zeros_like(u)
    op = cop.CoarseOp(dims, Nc).set_links(links)
    op.apply_parts(u, w, out, nrhs=nrhs, parity=cop.PARITY_EVEN, local=cop.LOCAL_X, alpha=1.0, beta=-1.0)
    torch.cuda.synchronize()
    assert op.last_path == cop.PATH_TENSOR
    op.close()


def test_parts_all_sites_equals_plain_apply():
    dims, Nc = (4, 4, 2, 6), 64
    links = synth.make_gamma_hermitian_links(dims, Nc, 9, device="cuda")
    v = synth.make_vectors(dims, Nc, 1, 10, device="cuda")
    a, b = torch.empty_like(v), torch.empty_like(v)
    op = cop.CoarseOp(dims, Nc).set_links(links)
    for dagger in (0, 1):
        op.apply(v, a, dagger=dagger)
        op.apply_parts(v, v, b, dagger=dagger)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))   # same kernel schedule, scale 1.0
    op.close()


@pytest.mark.parametrize("dims,Nc", [((4, 4, 4, 4), 48), ((4, 2, 6, 2), 64), ((2, 4, 2, 4), 128)])
@pytest.mark.parametrize("parity", [0, 1])
@pytest.mark.parametrize("dagger", [0, 1])
def test_schur_hat_operator_two_launches(oracle_lib, dims, Nc, parity, dagger):
    """1 - Dhat_pq Dhat_qp on block-preconditioned links: two parts launches."""
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 77).numpy()
    links[:, 0] += 2.0 * np.eye(Nc, dtype=np.complex64)
    hat_d, hat = gpu_hat_links(oracle_lib, dims, Nc, links)       # built on the device; same bits for both sides
    v = synth.make_vectors(dims, Nc, 1, 78, device="cuda")
    par = torch.as_tensor(oracle_lib.site_parities(dims), device="cuda")
    v[par != parity] = 0
    op = cop.CoarseOp(dims, Nc).set_links(hat_d)
    t = torch.zeros_like(v)
    out = torch.full_like(v, float("nan"))
    op.apply_parts(None, v, t, dagger=dagger, parity=1 - parity, local=cop.LOCAL_NONE, alpha=0.0, beta=1.0)
    op.apply_parts(v, t, out, dagger=dagger, parity=parity, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)
    torch.cuda.synchronize()
    ref = oracle_lib.schur_hat_apply(dims, Nc, hat, v.cpu().numpy(), parity, dagger=dagger)
    mask = (par == parity).cpu().numpy()
    got = out.cpu().numpy()
    assert rel_l2_per_rhs(got[mask], ref[mask]) <= TOL
    op.close()


@pytest.mark.parametrize("parity", [0, 1])
def test_schur_complement_three_launches(oracle_lib, parity):
    """S_p v = X_p v - D_pq X_q^{-1} D_qp v with the inverse of X held as the local term of a second
    operator handle (links2[:,0] = X^{-1})."""
    dims, Nc = (4, 2, 2, 4), 48
    links = synth.make_arbitrary_links(dims, Nc, 91).numpy()
    links[:, 0] += 2.0 * np.eye(Nc, dtype=np.complex64)
    v = synth.make_vectors(dims, Nc, 1, 92, device="cuda")
    par = torch.as_tensor(oracle_lib.site_parities(dims), device="cuda")
    v[par != parity] = 0
    op = cop.CoarseOp(dims, Nc).set_links(torch.as_tensor(links, device="cuda"))
    xinv_d = torch.empty((synth.lattice_volume(dims), 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    op.build_hat_links(xinv_d, slot0=cop.HAT_SLOT0_XINV)          # X^-1 in slot 0, built on the device
    torch.cuda.synchronize()
    opi = cop.CoarseOp(dims, Nc).set_links(xinv_d)
    t, t2, out = torch.zeros_like(v), torch.zeros_like(v), torch.full_like(v, float("nan"))
    q = 1 - parity
    op.apply_parts(None, v, t, parity=q, local=cop.LOCAL_NONE, alpha=0.0, beta=1.0)
    opi.apply_parts(t, t, t2, parity=q, local=cop.LOCAL_X, alpha=1.0, beta=0.0)
    op.apply_parts(v, t2, out, parity=parity, local=cop.LOCAL_X, alpha=1.0, beta=-1.0)
    torch.cuda.synchronize()
    ref = oracle_lib.schur_apply(dims, Nc, links, v.cpu().numpy(), parity)
    mask = (par == parity).cpu().numpy()
    # X^{-1} rounded to complex64 vs the oracle's fp64 solve: one extra 6e-8 rounding, amplified by cond(X)
    assert rel_l2_per_rhs(out.cpu().numpy()[mask], ref[mask]) <= TOL
    op.close(); opi.close()


def test_parts_argument_errors():
    L = cop.lib()
    h = cop.coarse_op_create((3, 2, 2, 2), 48, cop.LINK_C64)
    V = 24
    links = torch.zeros((V, 9, 48, 48), dtype=torch.complex64, device="cuda")
    v = torch.zeros((V, 48, 1), dtype=torch.complex64, device="cuda")
    o = torch.zeros_like(v)
    args = lambda u, w, out, parity, local: (h, u, w, out, 1, 0, parity, local, 1.0, 1.0, None)
    assert L.coarse_op_apply_parts(*args(v.data_ptr(), v.data_ptr(), o.data_ptr(), 2, 1)) == cop.ENOTREADY
    assert L.coarse_op_set_links(h, links.data_ptr(), None) == cop.OK
    assert L.coarse_op_apply_parts(*args(v.data_ptr(), v.data_ptr(), o.data_ptr(), 0, 1)) == cop.EINVAL   # odd extent
    assert "even" in cop.coarse_op_last_error()
    assert L.coarse_op_apply_parts(*args(v.data_ptr(), v.data_ptr(), o.data_ptr(), 3, 1)) == cop.EINVAL
    assert L.coarse_op_apply_parts(*args(v.data_ptr(), v.data_ptr(), o.data_ptr(), 2, 5)) == cop.EINVAL
    assert L.coarse_op_apply_parts(*args(None, v.data_ptr(), o.data_ptr(), 2, 1)) == cop.EINVAL           # local term without u
    assert L.coarse_op_apply_parts(*args(v.data_ptr(), o.data_ptr(), o.data_ptr(), 2, 1)) == cop.EINVAL   # w overlaps out
    assert L.coarse_op_apply_parts(*args(o.data_ptr(), v.data_ptr(), o.data_ptr(), 2, 2)) == cop.OK       # identity: u == out is allowed
    assert L.coarse_op_apply_parts(*args(o.data_ptr(), v.data_ptr(), o.data_ptr(), 2, 1)) == cop.EINVAL   # X.u in place is a race
    assert "COARSE_LOCAL_X" in cop.coarse_op_last_error()
    big = torch.zeros((2 * V, 48, 1), dtype=torch.complex64, device="cuda")
    shifted = big.data_ptr() + 48 * 8                                                                       # overlaps big[:V] by all but one site
    assert L.coarse_op_apply_parts(*args(shifted, v.data_ptr(), big.data_ptr(), 2, 2)) == cop.EINVAL      # partial overlap
    assert "partially" in cop.coarse_op_last_error()
    assert L.coarse_op_apply_parts(*args(None, v.data_ptr(), o.data_ptr(), 2, 0)) == cop.OK
    torch.cuda.synchronize()
    cop.coarse_op_destroy(h)


@pytest.mark.parametrize("Nc,prec", [(96, cop.LINK_C64), (128, cop.LINK_I16), (48, cop.LINK_C64)])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("path", [cop.PATH_STREAM, cop.PATH_SIMPLE])
def test_parts_identity_in_place_values(oracle_lib, Nc, prec, dagger, path):
    """out = u - Hop(w) computed IN PLACE (u_dev == out_dev, COARSE_LOCAL_IDENTITY) on shapes whose sites
    are split over several (site, row-block) work items (Nc = 96 / 128, dagger = 0): every output element
    reads only its own u element, so the values must equal the out-of-place result of the oracle."""
    dims = (2, 4, 2, 2)
    V = synth.lattice_volume(dims)
    links_d, scales_d, links_h, scales_h, u, w = _make(oracle_lib, dims, Nc, prec, 977, 1)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links_d, scales_d).set_option(cop.OPT_PATH, path)
    buf = u.clone()
    op.apply_parts(buf, w, buf, dagger=dagger, parity=cop.PARITY_ALL, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)
    torch.cuda.synchronize()
    ref = oracle_lib.coarse_apply_parts(dims, Nc, links_h, u.cpu().numpy(), w.cpu().numpy(), dagger=dagger, parity=2,
                                        local=2, alpha=1.0, beta=-1.0, link_precision=prec, scales=scales_h)
    assert rel_l2_per_rhs(buf.cpu().numpy(), ref) <= TOL
    op.close()


@pytest.mark.parametrize("Nc,prec", [(96, cop.LINK_C64), (128, cop.LINK_I16), (192, cop.LINK_I16)])
@pytest.mark.parametrize("dagger", [0, 1])
def test_parts_identity_in_place_values_multi_rhs(oracle_lib, Nc, prec, dagger):
    """The same in-place update with several right-hand sides, on the tensor kernels (the identity term is read in
    the epilogue by the thread that then stores the element) and on STREAM-MR (read at the store)."""
    dims = (2, 4, 2, 2)
    for nrhs, want in ((5, cop.PATH_TENSOR), (3, cop.PATH_STREAM)):       # (32 sites: 2-3 RHS stay on STREAM-MR for int16 links too)
        links_d, scales_d, links_h, scales_h, u, w = _make(oracle_lib, dims, Nc, prec, 978, nrhs)
        op = cop.CoarseOp(dims, Nc, prec).set_links(links_d, scales_d)
        buf = u.clone()
        op.apply_parts(buf, w, buf, nrhs=nrhs, dagger=dagger, parity=cop.PARITY_ALL, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)
        torch.cuda.synchronize()
        assert op.last_path == want
        ref = oracle_lib.coarse_apply_parts(dims, Nc, links_h, u.cpu().numpy(), w.cpu().numpy(), nrhs=nrhs, dagger=dagger, parity=2,
                                            local=2, alpha=1.0, beta=-1.0, link_precision=prec, scales=scales_h)
        assert rel_l2_per_rhs(buf.cpu().numpy(), ref) <= TOL
        op.close()
