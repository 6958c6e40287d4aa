"""GPU parity at BASELINE.json's full sizes (configs C1..C5), in the launch configuration bench.py
times (AUTO path, default persistent grid).

Small configs are compared element by element over the whole lattice.  For the large ones the
oracle evaluates its definition one site at a time on SAMPLED output sites (lattice corners, the
first/last sites, and seeded random sites); only the link matrices and vectors those sites touch
are brought to the host.  At any size the adjoint identity <u, A v> = <A^H u, v> ties the dagger
kernel to the non-dagger kernel over the WHOLE lattice.
"""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.helpers import neighbour_table, rel_l2_per_rhs

pytestmark = pytest.mark.gpu

TOL = 1e-5                      # BASELINE.json north_star: relative L2 per output vector
FULL_COMPARE_MAX_CMAC = 1.2e9   # whole-lattice oracle apply stays within seconds below this


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


def _sample_sites(dims, V, n_random, seed):
    L0, L1, L2, L3 = dims
    corners = []
    for x3 in (0, L3 - 1):
        for x2 in (0, L2 - 1):
            for x1 in (0, L1 - 1):
                for x0 in (0, L0 - 1):
                    corners.append(x0 + L0 * (x1 + L1 * (x2 + L2 * x3)))
    rng = np.random.default_rng(seed)
    rnd = rng.integers(0, V, size=n_random)
    return np.unique(np.concatenate([np.array(corners + [0, 1, V - 2, V - 1]), rnd])).astype(np.int64)


def _host_sparse(t_dev, rows, shape_tail, dtype):
    """Host array of the full first dimension with only `rows` filled from the device tensor
    (untouched pages of np.empty are never committed)."""
    host = np.empty((t_dev.shape[0],) + shape_tail, dtype=dtype)
    idx = torch.as_tensor(rows, device=t_dev.device)
    host[rows] = t_dev[idx].cpu().numpy().reshape((len(rows),) + shape_tail)
    return host


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

    work = V * 9.0 * Nc * Nc * nrhs
    vin_h = vin.cpu().numpy()
    if work <= FULL_COMPARE_MAX_CMAC:
        links_h = links.cpu().numpy()
        scales_h = None if scales is None else scales.cpu().numpy()
        for dagger in (0, 1):
            ref = oracle_lib.coarse_apply(dims, Nc, links_h, vin_h, nrhs=nrhs, dagger=dagger,
                                          link_precision=prec, scales=scales_h)
            err = rel_l2_per_rhs(outs[dagger].cpu().numpy(), ref)
            assert err <= TOL, f"{name} dagger={dagger}: rel-L2 {err:.3e}"
    else:
        sites = _sample_sites(dims, V, 160 if nrhs == 1 else 48, cfg["seed"])
        nbr = neighbour_table(dims)
        need = np.unique(nbr[sites].reshape(-1))
        tail = (9, Nc, Nc, 2)
        links_h = _host_sparse(links if prec == cop.LINK_I16 else torch.view_as_real(links),
                               need, tail, np.int16 if prec == cop.LINK_I16 else np.float32)
        scales_h = None if scales is None else scales.cpu().numpy()
        for dagger in (0, 1):
            ref = oracle_lib.coarse_apply_sites(dims, Nc, links_h, vin_h, sites, nrhs=nrhs, dagger=dagger,
                                                link_precision=prec, scales=scales_h)
            got = outs[dagger][torch.as_tensor(sites, device="cuda")].cpu().numpy()
            err = rel_l2_per_rhs(got, ref)
            assert err <= TOL, f"{name} dagger={dagger}: sampled rel-L2 {err:.3e}"
            # per-site errors too: one wrong site must not hide in the norm
            per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / \
                np.linalg.norm(ref.reshape(len(sites), -1), axis=1)
            assert per_site.max() <= 5 * TOL

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
