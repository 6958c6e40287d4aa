"""coarse_op_apply_static (include/coarse_op.h): the block apply on int16 links with the integer tensor-core kernel's
scratch in a file-scope __device__ array of the library, for callers that cannot call cudaMalloc.  Checked against the
existing path (coarse_op_apply on COARSE_PATH_TENSOR) within the tolerance of the other parity tests, on calls in a
row that share the array.  Named test_zz_* so that pytest collects it last: `pytest -x` then cannot hide other tests
behind a failure here.  Self-contained: passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest
import torch

import paper_2212_12559_b200 as cop
import synth

pytestmark = pytest.mark.gpu

TOL = 1e-5          # north_star tolerance, relative L2 per right-hand side (tests/test_gpu_parity.py)


def _rel_l2_per_rhs(got, ref):
    g = got.reshape(-1, got.shape[-1]).astype(np.complex128)
    r = ref.reshape(-1, ref.shape[-1]).astype(np.complex128)
    return float(np.max(np.linalg.norm(g - r, axis=0) / np.linalg.norm(r, axis=0)))


def _int16_op(dims, Nc, seed):
    V = synth.lattice_volume(dims)
    lc = synth.make_arbitrary_links(dims, Nc, seed, device="cuda")
    q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
    scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_i16(lc, Nc, q, scales)
    torch.cuda.synchronize()
    return cop.CoarseOp(dims, Nc, cop.LINK_I16).set_links(q, scales), q, scales


@pytest.mark.parametrize("Nc,dims", [(64, (3, 3, 3, 5)), (128, (2, 4, 2, 2))])
def test_apply_static_matches_existing_path_on_calls_in_a_row(Nc, dims):
    op, q, scales = _int16_op(dims, Nc, 31)
    ref_op = cop.CoarseOp(dims, Nc, cop.LINK_I16).set_links(q, scales).set_option(cop.OPT_PATH, cop.PATH_TENSOR)
    # calls in a row on one stream, sharing the static array: different vectors (other magnitudes -> other scales in
    # the scratch), column counts (16-, 8- and 4-wide tiles, several launches per call) and both modes
    calls = [(8, 0, 1.0), (8, 0, 37.5), (3, 1, 1e-3), (19, 0, 4.0), (8, 1, 1.0)]
    ins = [synth.make_vectors(dims, Nc, nrhs, 100 + i, device="cuda") * scale for i, (nrhs, _, scale) in enumerate(calls)]
    outs = [torch.full_like(v, float("nan")) for v in ins]
    refs = [torch.empty_like(v) for v in ins]
    for i, (nrhs, dagger, _) in enumerate(calls):
        if i == 1:
            # same kernels as call 0 (already loaded): the call must not change the free device memory.  (Up to three
            # tries: something else on the box allocating at that moment must not fail the test; an allocation of ours
            # would show every time.)
            unchanged = False
            for _ in range(3):
                torch.cuda.synchronize()
                free_before = torch.cuda.mem_get_info()[0]
                op.apply_static(ins[i], outs[i], nrhs=nrhs, dagger=dagger)
                torch.cuda.synchronize()
                unchanged = unchanged or torch.cuda.mem_get_info()[0] == free_before
                if unchanged:
                    break
            assert unchanged, "coarse_op_apply_static changed the free device memory"
        else:
            op.apply_static(ins[i], outs[i], nrhs=nrhs, dagger=dagger)
        assert op.last_path == cop.PATH_TENSOR and op.last_launches == 2 * ((nrhs + 15) // 16)
    torch.cuda.synchronize()
    for i, (nrhs, dagger, _) in enumerate(calls):
        ref_op.apply(ins[i], refs[i], nrhs=nrhs, dagger=dagger)
    torch.cuda.synchronize()
    for i, (nrhs, dagger, _) in enumerate(calls):
        got, ref = outs[i].cpu().numpy(), refs[i].cpu().numpy()
        assert np.isfinite(got.view(np.float32)).all()
        err = _rel_l2_per_rhs(got, ref)
        assert err <= TOL, f"call {i} (nrhs={nrhs}, dagger={dagger}): rel-L2 {err:.3e} > {TOL}"
    op.close()
    ref_op.close()


def test_apply_static_rejects_what_the_static_scratch_cannot_hold():
    # more sites than COARSE_STATIC_MAX_SITES
    dims, Nc = (4, 4, 8, 72), 32
    V = synth.lattice_volume(dims)
    assert V > cop.STATIC_MAX_SITES
    links = torch.zeros((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
    scales = torch.ones((V, 9), dtype=torch.float32, device="cuda")
    op = cop.CoarseOp(dims, Nc, cop.LINK_I16).set_links(links, scales)
    vin = torch.zeros((V, Nc, 2), dtype=torch.complex64, device="cuda")
    vout = torch.empty_like(vin)
    with pytest.raises(cop.CoarseOpError, match="COARSE_STATIC_MAX_SITES"):
        op.apply_static(vin, vout, nrhs=2)
    op.close()
    # complex64 links have no integer tensor-core kernel
    dims, Nc = (2, 2, 2, 2), 48
    links = torch.zeros((16, 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links)
    vin = torch.zeros((16, Nc, 2), dtype=torch.complex64, device="cuda")
    vout = torch.empty_like(vin)
    with pytest.raises(cop.CoarseOpError, match="int16"):
        op.apply_static(vin, vout, nrhs=2)
    op.close()
