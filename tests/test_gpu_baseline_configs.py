"""GPU parity at BASELINE.json's full sizes (configs C1..C5), in the launch configuration bench.py
times (AUTO path, default persistent grid).

Every config is compared with the oracle element by element over the WHOLE lattice, both modes
(tests/fullsize.py: the oracle evaluates its definition site by site over chunks of x3-slices, so
the 16 GB of C2 links never sit on the host at once).  The adjoint identity <u, A v> = <A^H u, v>
additionally ties the dagger kernel to the non-dagger kernel.
"""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.fullsize import whole_lattice_errors

pytestmark = pytest.mark.gpu

TOL = 1e-5                      # BASELINE.json north_star: relative L2 per output vector


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible (there is no CPU fallback)")
    torch.cuda.set_device(0)


def _build(name, oracle_lib):
    cfg = synth.config(name)
    dims, Nc, nrhs = cfg["dims"], cfg["Nc"], cfg["nrhs"]
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device="cuda")
    scales = None
    prec = cop.LINK_C64
    if cfg["links"] == "i16":
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        # quantiser parity on a slab of the real data (bit-exact)
        n = min(V, 512)
        q_ref, sc_ref = oracle_lib.quantize_i16(links[:n].cpu().numpy(), Nc)
        assert np.array_equal(scales[:n].cpu().numpy().reshape(-1), sc_ref)
        assert np.array_equal(q[:n].cpu().numpy().reshape(q_ref.shape), q_ref)
        del links
        links, prec = q, cop.LINK_I16
    vin = synth.make_vectors(dims, Nc, nrhs, cfg["seed"] + 1, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    return cfg, V, links, scales, prec, vin, op


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_baseline_config_parity(oracle_lib, name):
    cfg, V, links, scales, prec, vin, op = _build(name, oracle_lib)
    dims, Nc, nrhs = cfg["dims"], cfg["Nc"], cfg["nrhs"]
    outs = {}
    for dagger in (0, 1):
        vout = torch.full_like(vin, float("nan"))
        op.apply(vin, vout, nrhs=nrhs, dagger=dagger)
        torch.cuda.synchronize()
        assert op.last_launches >= 1
        assert torch.isfinite(torch.view_as_real(vout)).all()
        outs[dagger] = vout
    if nrhs == 1:
        assert op.last_path == cop.PATH_STREAM          # the configuration bench.py times
    else:
        assert op.last_path == cop.PATH_TENSOR          # C5: block apply on the tensor cores

    # EVERY output site against the oracle, element by element: the oracle's
    # per-site evaluation over chunks of x3-slices, links brought to the host chunk by chunk
    res = whole_lattice_errors(oracle_lib, dims, Nc, links, scales, prec, outs, nrhs, vin_h=vin.cpu().numpy())
    for dagger in (0, 1):
        err, worst_site, n_sites = res[dagger]
        assert n_sites == V
        assert err <= TOL, f"{name} dagger={dagger}: whole-lattice rel-L2 {err:.3e}"
        # per-site errors too: one wrong site must not hide in the norm
        assert worst_site <= 5 * TOL, f"{name} dagger={dagger}: worst site rel-L2 {worst_site:.3e}"
        print(f"{name} dagger={dagger}: {n_sites} sites compared, rel-L2 {err:.2e}, worst site {worst_site:.2e}")

    # whole-lattice property: <u, A v> = <A^H u, v>   (u = a second seeded vector)
    u = synth.make_vectors(dims, Nc, nrhs, cfg["seed"] + 2, device="cuda")
    Adu = torch.empty_like(u)
    op.apply(u, Adu, nrhs=nrhs, dagger=1)
    torch.cuda.synchronize()
    for r in range(nrhs):
        lhs = torch.vdot(u[:, :, r].reshape(-1).to(torch.complex128), outs[0][:, :, r].reshape(-1).to(torch.complex128))
        rhs = torch.vdot(Adu[:, :, r].reshape(-1).to(torch.complex128), vin[:, :, r].reshape(-1).to(torch.complex128))
        scale = torch.linalg.vector_norm(u[:, :, r].to(torch.complex128)) * \
            torch.linalg.vector_norm(outs[0][:, :, r].to(torch.complex128))
        assert abs(lhs - rhs).item() <= 1e-5 * scale.item()
    op.close()
