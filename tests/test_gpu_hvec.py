"""GPU parity for half-precision input vectors: the vector
quantiser is integer work (bit-exact against the oracle's), the apply is compared with the oracle run
on the SAME int16 + norm arrays at the 1e-5 relative-L2 tolerance."""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.helpers import rel_l2_per_rhs

pytestmark = pytest.mark.gpu
TOL = 1e-5


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible (there is no CPU fallback)")
    torch.cuda.set_device(0)


def _quantise(oracle_lib, v, Nc, nrhs):
    V = v.shape[0]
    q = torch.empty((V, Nc, nrhs, 2), dtype=torch.int16, device="cuda")
    nm = torch.empty((V, nrhs), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_vec_i16(v, Nc, nrhs, q, nm)
    torch.cuda.synchronize()
    q_ref, nm_ref = oracle_lib.quantize_vec_i16(v.cpu().numpy(), Nc, nrhs)
    assert np.array_equal(nm.cpu().numpy(), nm_ref)
    assert np.array_equal(q.cpu().numpy(), q_ref)
    return q, nm, q_ref, nm_ref


def _run(oracle_lib, dims, Nc, prec, nrhs, dagger, path, opts=None, launches=1, pin_path=True):
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 55, device="cuda")
    scales = scales_h = None
    if prec == cop.LINK_I16:
        lq = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, lq, scales)
        torch.cuda.synchronize()
        links, scales_h = lq, scales.cpu().numpy()
    v = synth.make_vectors(dims, Nc, nrhs, 56, device="cuda")
    if V > 1:
        v[1] *= 1e-6                                # sites of very different magnitude: the norm must be per site
    if V > 2:
        v[2] = 0
    q, nm, q_h, nm_h = _quantise(oracle_lib, v, Nc, nrhs)
    out = torch.full((V, Nc, nrhs), complex(float("nan"), float("nan")), dtype=torch.complex64, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    if pin_path:
        op.set_option(cop.OPT_PATH, path)
    for k, val in (opts or {}).items():
        op.set_option(k, val)
    op.apply_hvec(q, nm, out, nrhs=nrhs, dagger=dagger)
    torch.cuda.synchronize()
    assert op.last_path == path and op.last_launches == launches
    ref = oracle_lib.coarse_apply_hvec(dims, Nc, links.cpu().numpy(), q_h, nm_h, nrhs=nrhs, dagger=dagger,
                                       link_precision=prec, scales=scales_h)
    got = out.cpu().numpy()
    assert np.isfinite(got.view(np.float32)).all()
    err = rel_l2_per_rhs(got, ref)
    assert err <= TOL, f"rel-L2 {err:.3e} dims={dims} Nc={Nc} prec={prec} nrhs={nrhs} dagger={dagger}"
    op.close()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_hvec_stream(oracle_lib, dims, Nc, prec, dagger):
    if Nc >= 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 3)
    _run(oracle_lib, dims, Nc, prec, 1, dagger, cop.PATH_STREAM)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (5, 3, 4, 7)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("team", [12, 14])
@pytest.mark.parametrize("dagger", [0, 1])
def test_hvec_stream_warp_teams(oracle_lib, dims, Nc, team, dagger):
    """int16 links AND int16 + norm vectors (the paper's storage for both, PAPER.md:L97 / L99) on the warp-team kernel
    (stream2_kernel.cuh, what AUTO runs on large lattices; forced here): 2 and 4 warps per team, ragged last round."""
    if Nc >= 128 and dims == (5, 3, 4, 7):
        dims = (5, 3, 2, 3)
    _run(oracle_lib, dims, Nc, cop.LINK_I16, 1, dagger, cop.PATH_STREAM, opts={cop.OPT_WARP_ITEMS: team})
    if dims == (3, 2, 1, 4):
        _run(oracle_lib, (5, 3, 2, 3), Nc, cop.LINK_I16, 1, dagger, cop.PATH_STREAM, opts={cop.OPT_WARP_ITEMS: team, cop.OPT_GRID: 3})


@pytest.mark.parametrize("grid,stages", [(1, 2), (7, 3), (1000, 12)])
def test_hvec_stream_any_grid(oracle_lib, grid, stages):
    for dagger in (0, 1):
        _run(oracle_lib, (5, 3, 4, 7), 48, cop.LINK_I16, 1, dagger, cop.PATH_STREAM,
             opts={cop.OPT_GRID: grid, cop.OPT_STAGES: stages})


@pytest.mark.parametrize("nrhs", [1, 3])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_hvec_simple(oracle_lib, nrhs, prec, dagger):
    _run(oracle_lib, (3, 2, 2, 2), 8, prec, nrhs, dagger, cop.PATH_SIMPLE)
    _run(oracle_lib, (2, 2, 1, 2), 48, prec, nrhs, dagger, cop.PATH_SIMPLE)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 3, 3, 5), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("nrhs", [2, 3, 8, 11, 16, 19])
@pytest.mark.parametrize("dagger", [0, 1])
def test_hvec_tensor_int16_links_int16_vectors(oracle_lib, dims, Nc, nrhs, dagger):
    """Several right-hand sides with the paper's storage for BOTH operands (16-bit links; 16-bit vectors
    with a per-site norm, L97) on the integer tensor cores: link bytes and vector bytes are the int8 operands, int32
    accumulation is exact.  Every compiled Nc (two sites per MMA tile at Nc <= 64: odd site count 135), 4-, 8- and
    16-wide column tiles, ragged widths, more than 16 columns (two launches); AUTO picks this path."""
    if Nc >= 96 and dims != (1, 1, 1, 1):
        dims = (2, 4, 2, 2) if dims == (4, 4, 4, 4) else (3, 1, 3, 2)
    _run(oracle_lib, dims, Nc, cop.LINK_I16, nrhs, dagger, cop.PATH_TENSOR, launches=(nrhs + 15) // 16, pin_path=False)


@pytest.mark.parametrize("grid", [1, 7])
def test_hvec_tensor_any_grid_and_single_rhs(oracle_lib, grid):
    """One CTA walking every item (rings wrap many times) and a ragged grid; 1 RHS on the tensor kernel when pinned."""
    for dagger in (0, 1):
        _run(oracle_lib, (3, 3, 3, 5), 64, cop.LINK_I16, 8, dagger, cop.PATH_TENSOR, opts={cop.OPT_GRID: grid})
        _run(oracle_lib, (5, 3, 2, 3), 128, cop.LINK_I16, 16, dagger, cop.PATH_TENSOR, opts={cop.OPT_GRID: grid})
        _run(oracle_lib, (3, 2, 1, 4), 48, cop.LINK_I16, 1, dagger, cop.PATH_TENSOR, opts={cop.OPT_GRID: grid})


@pytest.mark.parametrize("Nc,nrhs,applies", [(64, 8, 800), (128, 16, 400), (64, 1, 1200), (96, 1, 800)])
def test_hvec_tensor_bit_reproducible_under_stress(Nc, nrhs, applies):
    """Integer accumulation (1 RHS: fp32 in a fixed order) and a fixed schedule: every apply must equal the first one bit
    for bit (~55 work items per CTA; the link-slot release race of tests/test_gpu_parity.py's stress test would show up here the same way)."""
    dims = (8, 8, 8, 16)
    V = synth.lattice_volume(dims)
    lc = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    lq = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
    scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_i16(lc, Nc, lq, scales)
    del lc
    v = synth.make_vectors(dims, Nc, nrhs, 6, device="cuda")
    q = torch.empty((V, Nc, nrhs, 2), dtype=torch.int16, device="cuda")
    nm = torch.empty((V, nrhs), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_vec_i16(v, Nc, nrhs, q, nm)
    op = cop.CoarseOp(dims, Nc, cop.LINK_I16).set_links(lq, scales)
    refs = {}
    for dagger in (0, 1):
        refs[dagger] = torch.empty_like(v)
        op.apply_hvec(q, nm, refs[dagger], nrhs=nrhs, dagger=dagger)
    assert op.last_path == (cop.PATH_TENSOR if nrhs > 1 else cop.PATH_STREAM)      # 1 RHS: the warp-team kernel (8192 sites)
    out = torch.empty_like(v)
    bad = 0
    for it in range(applies):
        op.apply_hvec(q, nm, out, nrhs=nrhs, dagger=it % 2)
        bad += int(not torch.equal(torch.view_as_real(out), torch.view_as_real(refs[it % 2])))
    assert bad == 0, f"{bad} of {applies} applies differ from the first one"
    op.close()


@pytest.mark.parametrize("Nc,half_in", [(64, False), (64, True), (48, True), (128, False)])
def test_half_output_warp_teams_bit_reproducible_under_stress(Nc, half_in):
    """Half-precision output from the warp-team kernel on a lattice with many items per team: the 16-bit vectors, the norms
    and the complex64 result of every apply must equal the first one's (the team-wide maximum goes through a double-buffered
    shared-memory slot behind one named barrier per item)."""
    dims, applies = (8, 8, 8, 16), 600
    V = synth.lattice_volume(dims)
    lc = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    lq = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
    scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_i16(lc, Nc, lq, scales)
    del lc
    v = synth.make_vectors(dims, Nc, 1, 6, device="cuda")
    v[::7] *= 1e-3                                   # norms that differ from site to site
    q = nm = None
    if half_in:
        q = torch.empty((V, Nc, 1, 2), dtype=torch.int16, device="cuda")
        nm = torch.empty((V, 1), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_vec_i16(v, Nc, 1, q, nm)
    op = cop.CoarseOp(dims, Nc, cop.LINK_I16).set_links(lq, scales)
    src = q if half_in else v
    refs = {}
    for dagger in (0, 1):
        refs[dagger] = (torch.empty_like(v), torch.empty((V, Nc, 1, 2), dtype=torch.int16, device="cuda"),
                        torch.empty((V, 1), dtype=torch.float32, device="cuda"))
        op.apply_hout(src, nm, *refs[dagger], dagger=dagger)
    out, oq, on = torch.empty_like(v), torch.empty((V, Nc, 1, 2), dtype=torch.int16, device="cuda"), torch.empty((V, 1), dtype=torch.float32, device="cuda")
    bad = 0
    for it in range(applies):
        dg = it % 2
        op.apply_hout(src, nm, out, oq, on, dagger=dg)
        ok = torch.equal(torch.view_as_real(out), torch.view_as_real(refs[dg][0])) and torch.equal(oq, refs[dg][1]) and torch.equal(on, refs[dg][2])
        bad += int(not ok)
    assert bad == 0, f"{bad} of {applies} applies differ from the first one"
    # and the first one is right: the 16-bit result is the vector quantiser applied to the complex64 result
    q2 = torch.empty_like(oq)
    n2 = torch.empty_like(on)
    cop.coarse_op_quantize_vec_i16(refs[1][0], Nc, 1, q2, n2)
    torch.cuda.synchronize()
    assert torch.equal(q2, refs[1][1]) and torch.equal(n2, refs[1][2])
    op.close()


def test_hvec_multi_rhs_complex64_links_stay_on_simple(oracle_lib):
    _run(oracle_lib, (2, 2, 1, 2), 48, cop.LINK_C64, 3, 0, cop.PATH_SIMPLE, pin_path=False)


def test_hvec_full_size_c4_whole_lattice(oracle_lib):
    """BASELINE config C4 with half-precision input vectors, in the launch configuration of the bench:
    every output site against the oracle's O8 (`coarse_apply_hvec_sites`, the oracle's own apply_site)."""
    from tests.fullsize import whole_lattice_errors
    cfg = synth.config("C4")
    dims, Nc = cfg["dims"], cfg["Nc"]
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device="cuda")
    lq = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
    scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_i16(links, Nc, lq, scales)
    del links
    v = synth.make_vectors(dims, Nc, 1, cfg["seed"] + 1, device="cuda")
    q = torch.empty((V, Nc, 1, 2), dtype=torch.int16, device="cuda")
    nm = torch.empty((V, 1), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_vec_i16(v, Nc, 1, q, nm)
    op = cop.CoarseOp(dims, Nc, cop.LINK_I16).set_links(lq, scales)
    outs = {}
    for dagger in (0, 1):
        outs[dagger] = torch.full_like(v, float("nan"))
        op.apply_hvec(q, nm, outs[dagger], dagger=dagger)
        torch.cuda.synchronize()
        assert op.last_path == cop.PATH_STREAM
    res = whole_lattice_errors(oracle_lib, dims, Nc, lq, scales, cop.LINK_I16, outs, 1,
                               hvec=(q.cpu().numpy(), nm.cpu().numpy()))
    for dagger in (0, 1):
        err, worst_site, n_sites = res[dagger]
        assert n_sites == V and err <= TOL and worst_site <= 5 * TOL, (dagger, err, worst_site)
    op.close()


# ------------------------------------------------------------------ half-precision OUTPUT (coarse_op_apply_hout)
def _run_hout(oracle_lib, dims, Nc, prec, nrhs, dagger, half_in, opts=None, want_launches=None):
    """The complex64 result must match the oracle's apply (1e-5); the 16-bit result must be EXACTLY what the oracle's
    vector quantiser (pinned in tests/test_oracle_hvec_pins.py) makes of that complex64 result - the rounding decision is
    taken in fp32 on the same numbers on both sides - and must dequantise to the oracle's apply within half a step."""
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 65, device="cuda")
    scales = scales_h = None
    if prec == cop.LINK_I16:
        lq = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, lq, scales)
        torch.cuda.synchronize()
        links, scales_h = lq, scales.cpu().numpy()
    v = synth.make_vectors(dims, Nc, nrhs, 66, device="cuda")
    if V > 1:
        v[1] *= 1e-6
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    for k, val in (opts or {}).items():
        op.set_option(k, val)
    out = torch.full((V, Nc, nrhs), complex(float("nan"), float("nan")), dtype=torch.complex64, device="cuda")
    oq = torch.full((V, Nc, nrhs, 2), -7, dtype=torch.int16, device="cuda")
    on = torch.full((V, nrhs), float("nan"), dtype=torch.float32, device="cuda")
    if half_in:
        q, nm, q_h, nm_h = _quantise(oracle_lib, v, Nc, nrhs)
        ref = oracle_lib.coarse_apply_hvec(dims, Nc, links.cpu().numpy(), q_h, nm_h, nrhs=nrhs, dagger=dagger,
                                           link_precision=prec, scales=scales_h)
    else:
        q, nm = v, None
        ref = oracle_lib.coarse_apply(dims, Nc, links.cpu().numpy(), v.cpu().numpy(), nrhs=nrhs, dagger=dagger,
                                      link_precision=prec, scales=scales_h)
    for rep in range(2):                       # twice: the per-site counters must be back at zero
        oq.fill_(-7)
        op.apply_hout(q, nm, out, oq, on, nrhs=nrhs, dagger=dagger)
        torch.cuda.synchronize()
        if want_launches is not None:
            assert op.last_launches == want_launches
        got = out.cpu().numpy()
        assert rel_l2_per_rhs(got, ref) <= TOL
        q_ref, n_ref = oracle_lib.quantize_vec_i16(got, Nc, nrhs)
        assert np.array_equal(on.cpu().numpy(), n_ref)
        assert np.array_equal(oq.cpu().numpy(), q_ref)
        deq = on.cpu().numpy()[:, None, :] * (oq.cpu().numpy()[..., 0].astype(np.float64) + 1j * oq.cpu().numpy()[..., 1])
        step = on.cpu().numpy()[:, None, :]
        assert np.all(np.abs(deq - ref) <= 0.75 * step * np.sqrt(2) + 1e-5 * np.abs(ref).max())
    op.close()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("half_in", [False, True])
def test_half_precision_output_fused_epilogue(oracle_lib, dims, Nc, prec, dagger, half_in):
    """1 RHS: ONE launch; the CTA that finishes a site's last (site, row-block) item takes the norm and writes the int16
    vector (Nc >= 96 in dagger 0: several CTAs per site; dagger 1: one)."""
    if Nc >= 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 2)
    _run_hout(oracle_lib, dims, Nc, prec, 1, dagger, half_in, want_launches=1)


@pytest.mark.parametrize("grid,fine", [(1, 0), (5, 2), (1000, 0)])
def test_half_precision_output_any_grid(oracle_lib, grid, fine):
    for dagger in (0, 1):
        _run_hout(oracle_lib, (3, 2, 2, 4), 128, cop.LINK_I16, 1, dagger, False, opts={cop.OPT_GRID: grid, cop.OPT_FINE: fine})
        _run_hout(oracle_lib, (5, 3, 2, 3), 48, cop.LINK_C64, 1, dagger, True, opts={cop.OPT_GRID: grid})


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (5, 3, 2, 3)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("team", [12, 14])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("half_in", [False, True])
def test_half_precision_output_warp_teams(oracle_lib, dims, Nc, team, dagger, half_in):
    """Half-precision output on the warp-team kernel (int16 links; what AUTO runs on large lattices): dagger 1 and, where a
    work item is a whole site (Nc <= 64), dagger 0 - a team holds all rows of the site and takes the norm itself; the
    other shapes fall back to the cooperative kernel's site-owning CTAs.  PDL off so that both repetitions take this path."""
    if Nc >= 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 2)
    _run_hout(oracle_lib, dims, Nc, cop.LINK_I16, 1, dagger, half_in, opts={cop.OPT_WARP_ITEMS: team, cop.OPT_PDL: 2}, want_launches=1)


@pytest.mark.parametrize("nrhs", [3, 16])
def test_half_precision_output_multi_rhs_two_pass(oracle_lib, nrhs):
    """Several right-hand sides: the apply (STREAM-MR / tensor kernels), then the vector quantiser."""
    _run_hout(oracle_lib, (4, 2, 2, 2), 64, cop.LINK_C64, nrhs, 0, False, want_launches=2)
    _run_hout(oracle_lib, (2, 2, 2, 2), 128, cop.LINK_I16, nrhs, 1, False)


def test_half_precision_output_argument_errors():
    dims, Nc, V = (2, 2, 2, 2), 48, 16
    links = torch.zeros((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    v = torch.zeros((V, Nc, 1), dtype=torch.complex64, device="cuda")
    out, oq, on = torch.zeros_like(v), torch.zeros((V, Nc, 1, 2), dtype=torch.int16, device="cuda"), torch.zeros((V, 1), device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links)
    L = cop.lib()
    assert L.coarse_op_apply_hout(op._h, v.data_ptr(), None, out.data_ptr(), None, on.data_ptr(), 1, 0, None) == cop.EINVAL
    assert L.coarse_op_apply_hout(op._h, v.data_ptr(), None, v.data_ptr(), oq.data_ptr(), on.data_ptr(), 1, 0, None) == cop.EINVAL
    assert L.coarse_op_apply_hout(op._h, v.data_ptr(), None, out.data_ptr(), oq.data_ptr(), on.data_ptr(), 1, 0, None) == cop.OK
    torch.cuda.synchronize()
    assert torch.all(oq == 0) and torch.all(on == 0)          # a zero operator: norm 0, q 0
    op.close()
