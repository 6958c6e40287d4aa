"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerance (BASELINE.json north_star, written here as asked): relative L2 error per output vector
<= 1e-5 for complex64 links, and <= 1e-5 against the oracle run on the SAME int16 + scale arrays
(i.e. on the dequantised links) for int16 storage.  The quantiser is integer work: bit-exact.
"""
import numpy as np
import pytest
import torch

import synth
import paper_2212_12559_b200 as cop
from tests.helpers import rel_l2, rel_l2_per_rhs

pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests selected but no CUDA device is visible (there is no CPU fallback)")
    torch.cuda.set_device(0)


def _links_for(dims, Nc, prec, seed, hermitian, oracle_lib):
    """Returns (device link tensor, device scales or None, host links for the oracle, host scales)."""
    gen = synth.make_gamma_hermitian_links if hermitian else synth.make_arbitrary_links
    links = gen(dims, Nc, seed, device="cuda")
    if prec == cop.LINK_C64:
        return links, None, links.cpu().numpy(), None
    V = synth.lattice_volume(dims)
    q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
    sc = torch.empty((V, 9), dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_i16(links, Nc, q, sc)
    torch.cuda.synchronize()
    # the integers handed to BOTH sides come from the oracle's quantiser; the CUDA quantiser
    # must reproduce them bit for bit (checked here on every int16 case)
    q_ref, sc_ref = oracle_lib.quantize_i16(links.cpu().numpy(), Nc)
    assert np.array_equal(sc.cpu().numpy().reshape(-1), sc_ref)
    assert np.array_equal(q.cpu().numpy().reshape(q_ref.shape), q_ref)
    return q, sc, q_ref.reshape(V, 9, Nc, Nc, 2), sc_ref


def _run(oracle_lib, dims, Nc, prec, nrhs, dagger, path, seed=1234, hermitian=True, grid=0, opts=None):
    V = synth.lattice_volume(dims)
    links, scales, links_h, scales_h = _links_for(dims, Nc, prec, seed, hermitian, oracle_lib)
    vin = synth.make_vectors(dims, Nc, nrhs, seed + 1, device="cuda")
    vout = torch.full((V, Nc, nrhs), float("nan"), dtype=torch.complex64, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    op.set_option(cop.OPT_PATH, path)
    if grid:
        op.set_option(cop.OPT_GRID, grid)
    for k, v in (opts or {}).items():
        op.set_option(k, v)
    op.apply(vin, vout, nrhs=nrhs, dagger=dagger)
    torch.cuda.synchronize()
    assert op.last_launches >= 1
    if path != cop.PATH_AUTO:
        assert op.last_path == path
    got = vout.cpu().numpy()
    ref = oracle_lib.coarse_apply(dims, Nc, links_h, vin.cpu().numpy(), nrhs=nrhs, dagger=dagger,
                                  link_precision=prec, scales=scales_h)
    assert np.isfinite(got.view(np.float32)).all()
    err = rel_l2_per_rhs(got, ref)
    assert err <= TOL, f"rel-L2 {err:.3e} > {TOL} for dims={dims} Nc={Nc} prec={prec} nrhs={nrhs} dagger={dagger} path={path}"
    op.close()
    return err


SMALL_LATTICES = [(4, 4, 4, 4), (3, 2, 1, 4), (2, 2, 2, 2), (1, 1, 1, 1), (5, 3, 4, 7)]


@pytest.mark.parametrize("dims", SMALL_LATTICES)
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_stream_path_single_rhs(oracle_lib, dims, Nc, prec, dagger):
    if Nc >= 128 and dims == (5, 3, 4, 7):
        dims = (5, 3, 2, 3)               # keep the oracle's run time in seconds
    _run(oracle_lib, dims, Nc, prec, 1, dagger, cop.PATH_STREAM)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1), (5, 3, 4, 7)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("team", [12, 14])
def test_stream_warp_teams_single_rhs(oracle_lib, dims, Nc, prec, dagger, team):
    """The team-owned-stages STREAM variant (csrc/stream2_kernel.cuh), forced on every shape with 2 and 4
    warps per team: ragged item counts (fewer items than teams, ragged last round), extents 1 and 2,
    arbitrary links."""
    if Nc >= 128 and dims == (5, 3, 4, 7):
        dims = (5, 3, 2, 3)
    _run(oracle_lib, dims, Nc, prec, 1, dagger, cop.PATH_STREAM, opts={cop.OPT_WARP_ITEMS: team}, hermitian=False)


@pytest.mark.parametrize("grid,stages", [(1, 4), (3, 9), (2, 16), (1000, 0)])
def test_stream_warp_teams_any_grid(oracle_lib, grid, stages):
    """Many rounds per CTA (the multi-round ring bookkeeping), every ring depth the host may pick."""
    for dagger in (0, 1):
        for Nc, prec, team in ((64, cop.LINK_I16, 12), (48, cop.LINK_C64, 14), (192, cop.LINK_I16, 14), (128, cop.LINK_I16, 2)):
            opts = {cop.OPT_WARP_ITEMS: team}
            if stages:
                opts[cop.OPT_STAGES] = stages
            _run(oracle_lib, (5, 3, 2, 3), Nc, prec, 1, dagger, cop.PATH_STREAM, grid=grid, opts=opts)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [6, 8, 48, 64])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [1, 3, 16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_simple_path(oracle_lib, dims, Nc, prec, nrhs, dagger):
    _run(oracle_lib, dims, Nc, prec, nrhs, dagger, cop.PATH_SIMPLE)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (2, 2, 2, 2), (1, 1, 1, 1), (5, 3, 2, 3)])
@pytest.mark.parametrize("Nc", [48, 64, 128])
@pytest.mark.parametrize("nrhs", [8, 16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_tensor_path_block_apply(oracle_lib, dims, Nc, nrhs, dagger):
    """tcgen05 3xTF32 block apply: same 1e-5 bound as the CUDA-core paths (north_star (4))."""
    err = _run(oracle_lib, dims, Nc, cop.LINK_C64, nrhs, dagger, cop.PATH_TENSOR)
    assert err <= 3e-6, f"3xTF32 with per-matrix accumulator chains should sit near 1e-6, got {err:.2e}"


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [1, 3, 7, 8, 11, 16, 19, 40])
@pytest.mark.parametrize("dagger", [0, 1])
def test_tensor_path_every_shape(oracle_lib, dims, Nc, prec, nrhs, dagger):
    """The TENSOR kernel on every compiled Nc (Nc = 192: two output tiles per site), both link formats
    (int16: the paper's storage, decoded and split exactly), any nrhs: zero-padded 8- / 16-wide
    column tiles (3 = one propagator; odd row pitches), several launches beyond 16."""
    if Nc >= 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 2)               # keep the oracle's run time in seconds
    if nrhs == 40 and dims == (4, 4, 4, 4):
        dims = (2, 2, 2, 4)
    err = _run(oracle_lib, dims, Nc, prec, nrhs, dagger, cop.PATH_TENSOR, hermitian=(nrhs != 7))
    assert err <= 3e-6, f"3xTF32 with per-matrix accumulator chains should sit near 1e-6, got {err:.2e}"


@pytest.mark.parametrize("Nc", [32, 48, 64])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [3, 8, 16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_tensor_two_sites_per_tile_odd_site_count(oracle_lib, Nc, prec, nrhs, dagger):
    """Nc <= 64: a work item of the tensor kernels is a PAIR of sites sharing the 128-lane MMA tile.  135 sites: the
    last item has one site only (its second half must not store), with one CTA per item, several items per CTA and a
    single CTA walking all 68 items (rings wrap many times)."""
    for grid in (0, 7, 1):
        _run(oracle_lib, (3, 3, 3, 5), Nc, prec, nrhs, dagger, cop.PATH_TENSOR, seed=77 + grid, hermitian=False, grid=grid)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [2, 3, 8, 11, 16])
@pytest.mark.parametrize("dagger", [0, 1])
def test_block_path_cuda_cores(oracle_lib, dims, Nc, prec, nrhs, dagger):
    """CUDA-core block apply: every compiled Nc, both link formats, ragged nrhs (3 = one propagator,
    PAPER.md:L188; 11 leaves surplus lanes in the 16-wide mapping)."""
    if Nc >= 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 2)               # keep the oracle's run time in seconds
    _run(oracle_lib, dims, Nc, prec, nrhs, dagger, cop.PATH_BLOCK)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 2, 1, 4), (1, 1, 1, 1)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("nrhs", [2, 3, 4])
@pytest.mark.parametrize("dagger", [0, 1])
def test_stream_path_few_rhs(oracle_lib, dims, Nc, prec, nrhs, dagger):
    """STREAM-MR: 2-4 right-hand sides on the streaming kernel (3 RHS = one propagator)."""
    if Nc >= 128 and dims == (4, 4, 4, 4):
        dims = (2, 4, 2, 2)
    _run(oracle_lib, dims, Nc, prec, nrhs, dagger, cop.PATH_STREAM)


@pytest.mark.parametrize("grid,stages", [(1, 2), (7, 3), (1000, 12)])
def test_stream_few_rhs_any_grid(oracle_lib, grid, stages):
    for dagger in (0, 1):
        _run(oracle_lib, (5, 3, 4, 7), 48, cop.LINK_I16, 3, dagger, cop.PATH_STREAM, grid=grid,
             opts={cop.OPT_STAGES: stages}, hermitian=False)
        _run(oracle_lib, (3, 3, 2, 2), 128, cop.LINK_C64, 4, dagger, cop.PATH_STREAM, grid=grid,
             opts={cop.OPT_STAGES: stages})


@pytest.mark.parametrize("grid", [1, 7, 1000])
def test_block_path_any_grid(oracle_lib, grid):
    for dagger in (0, 1):
        _run(oracle_lib, (5, 3, 2, 3), 128, cop.LINK_C64, 16, dagger, cop.PATH_BLOCK, grid=grid)
        _run(oracle_lib, (5, 3, 4, 7), 48, cop.LINK_I16, 3, dagger, cop.PATH_BLOCK, grid=grid, hermitian=False,
             opts={cop.OPT_STAGES: 2})


def test_auto_path_selection():
    small, large = (2, 2, 2, 2), (4, 4, 4, 10)       # 16 sites; 640 sites: at least two tensor work items per SM
    cases = [(small, 48, cop.LINK_C64, 1, cop.PATH_STREAM), (small, 48, cop.LINK_C64, 16, cop.PATH_TENSOR),
             (small, 48, cop.LINK_C64, 3, cop.PATH_STREAM), (small, 64, cop.LINK_I16, 4, cop.PATH_TENSOR),
             # int16 links, 2-3 RHS: the integer tensor kernel on large lattices, STREAM-MR on tiny ones
             (large, 64, cop.LINK_I16, 2, cop.PATH_TENSOR), (small, 64, cop.LINK_I16, 2, cop.PATH_STREAM),
             (large, 128, cop.LINK_I16, 3, cop.PATH_TENSOR), (small, 128, cop.LINK_I16, 3, cop.PATH_STREAM),
             (large, 48, cop.LINK_I16, 3, cop.PATH_STREAM), (small, 48, cop.LINK_I16, 4, cop.PATH_TENSOR),
             (large, 32, cop.LINK_I16, 2, cop.PATH_TENSOR), (small, 64, cop.LINK_C64, 4, cop.PATH_TENSOR),
             (small, 32, cop.LINK_C64, 4, cop.PATH_STREAM),
             (small, 48, cop.LINK_C64, 5, cop.PATH_TENSOR), (small, 64, cop.LINK_I16, 16, cop.PATH_TENSOR),
             (small, 96, cop.LINK_C64, 8, cop.PATH_TENSOR), (small, 48, cop.LINK_C64, 17, cop.PATH_TENSOR),
             (small, 192, cop.LINK_I16, 12, cop.PATH_TENSOR), (small, 6, cop.LINK_C64, 2, cop.PATH_SIMPLE)]
    for dims, Nc, prec, nrhs, want in cases:
        V = synth.lattice_volume(dims)
        if prec == cop.LINK_C64:
            links, scales = torch.zeros((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda"), None
        else:
            links = torch.zeros((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
            scales = torch.ones((V, 9), dtype=torch.float32, device="cuda")
        vin = torch.zeros((V, Nc, nrhs), dtype=torch.complex64, device="cuda")
        vout = torch.empty_like(vin)
        op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
        op.apply(vin, vout, nrhs=nrhs)
        torch.cuda.synchronize()
        assert op.last_path == want, (Nc, prec, nrhs, op.last_path, want)
        if prec == cop.LINK_C64 and nrhs == 4:      # complex64, 4 RHS: only dagger = 0 leaves STREAM-MR (bank conflicts there)
            op.apply(vin, vout, nrhs=nrhs, dagger=1)
            torch.cuda.synchronize()
            assert op.last_path == cop.PATH_STREAM
        op.close()


@pytest.mark.parametrize("grid", [1, 7, 1000])
def test_tensor_path_any_grid(oracle_lib, grid):
    """Several sites per CTA (accumulator/operand rings wrap many times), ragged tail, idle CTAs."""
    for dagger in (0, 1):
        _run(oracle_lib, (5, 3, 2, 3), 128, cop.LINK_C64, 16, dagger, cop.PATH_TENSOR, grid=grid)
        _run(oracle_lib, (5, 3, 4, 7), 48, cop.LINK_C64, 8, dagger, cop.PATH_TENSOR, grid=grid, hermitian=False)


def test_tensor_path_matches_cuda_core_path_and_is_reproducible():
    dims, Nc, nrhs = (4, 3, 2, 5), 128, 16
    links = synth.make_arbitrary_links(dims, Nc, 21, device="cuda")
    vin = synth.make_vectors(dims, Nc, nrhs, 22, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links)
    outs = {}
    for path in (cop.PATH_SIMPLE, cop.PATH_TENSOR, cop.PATH_TENSOR):
        op.set_option(cop.OPT_PATH, path)
        vout = torch.empty_like(vin)
        op.apply(vin, vout, nrhs=nrhs, dagger=1)
        torch.cuda.synchronize()
        outs.setdefault(path, []).append(vout)
    a, b = outs[cop.PATH_TENSOR]
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))
    ref = outs[cop.PATH_SIMPLE][0].cpu().numpy()
    assert rel_l2_per_rhs(a.cpu().numpy(), ref) <= 3e-6
    op.close()


@pytest.mark.parametrize("Nc,prec,nrhs,applies", [(64, cop.LINK_C64, 16, 1200), (128, cop.LINK_I16, 16, 600),
                                                  (64, cop.LINK_I16, 8, 1200), (64, cop.LINK_I16, 3, 1200)])
def test_tensor_kernels_bit_reproducible_under_stress(Nc, prec, nrhs, applies):
    """Many applies on a lattice with ~55 work items per CTA: every result must equal the first one bit for bit.  (An
    earlier version released a link slot right after loading it, behind a fence only; the producer's next TMA write
    overtook the reads once in 600-2000 applies and a few rows of one site came out wrong.)"""
    dims = (8, 8, 8, 16)                  # (Nc = 64 int16: two sites per MMA tile, 8- and 4-wide column tiles)
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        links = q
    vin = synth.make_vectors(dims, Nc, nrhs, 6, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales).set_option(cop.OPT_PATH, cop.PATH_TENSOR)
    refs = {}
    for dagger in (0, 1):
        refs[dagger] = torch.empty_like(vin)
        op.apply(vin, refs[dagger], nrhs=nrhs, dagger=dagger)
    out = torch.empty_like(vin)
    bad = 0
    for it in range(applies):
        op.apply(vin, out, nrhs=nrhs, dagger=it % 2)
        bad += int(not torch.equal(torch.view_as_real(out), torch.view_as_real(refs[it % 2])))
    assert bad == 0, f"{bad} of {applies} applies differ from the first one"
    op.close()


@pytest.mark.parametrize("Nc,prec,nrhs,opts", [
    (48, cop.LINK_C64, 1, {}), (128, cop.LINK_C64, 1, {}), (64, cop.LINK_I16, 1, {}), (48, cop.LINK_I16, 1, {}),
    (64, cop.LINK_I16, 1, {cop.OPT_WARP_ITEMS: 1}), (64, cop.LINK_I16, 3, {}), (48, cop.LINK_C64, 4, {}),
    (64, cop.LINK_I16, 5, {cop.OPT_PATH: cop.PATH_BLOCK})])
def test_streaming_kernels_bit_reproducible_under_stress(Nc, prec, nrhs, opts):
    """The same watch on the TMA-ring kernels that run on the CUDA cores (cooperative and warp-team STREAM, STREAM-MR,
    BLOCK): 1000 applies on a lattice with ~55 work items per CTA, each equal to the first bit for bit."""
    dims = (8, 8, 8, 16)
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        links = q
    vin = synth.make_vectors(dims, Nc, nrhs, 6, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    for k, v in opts.items():
        op.set_option(k, v)
    refs = {}
    for dagger in (0, 1):
        refs[dagger] = torch.empty_like(vin)
        op.apply(vin, refs[dagger], nrhs=nrhs, dagger=dagger)
    out = torch.empty_like(vin)
    bad = 0
    for it in range(1000):
        op.apply(vin, out, nrhs=nrhs, dagger=it % 2)
        bad += int(not torch.equal(torch.view_as_real(out), torch.view_as_real(refs[it % 2])))
    assert bad == 0, f"{bad} of 1000 applies differ from the first one"
    op.close()


def test_tensor_path_unsupported_shapes():
    L = cop.lib()
    h = cop.coarse_op_create((2, 2, 2, 2), 80, cop.LINK_I16)          # Nc outside the compiled set
    assert L.coarse_op_set_option(h, cop.OPT_PATH, cop.PATH_TENSOR) == cop.EUNSUPPORTED
    cop.coarse_op_destroy(h)


@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
@pytest.mark.parametrize("bad", [float("nan"), float("inf")])
def test_tensor_paths_propagate_non_finite_inputs(prec, bad):
    """A NaN / Inf in one input vector entry must reach every output that reads it (a solver detects divergence that
    way), also on the integer tensor-core kernel whose fixed-point operand cannot represent it; other columns and
    sites that do not touch the entry stay finite."""
    dims, Nc, nrhs = (4, 4, 2, 2), 64, 8
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 31, device="cuda")
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        links = q
    vin = synth.make_vectors(dims, Nc, nrhs, 32, device="cuda")
    vin[5, 7, 2] = complex(bad, 0.0)
    vout = torch.empty_like(vin)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales).set_option(cop.OPT_PATH, cop.PATH_TENSOR)
    op.apply(vin, vout, nrhs=nrhs)
    torch.cuda.synchronize()
    fin = torch.isfinite(torch.view_as_real(vout)).all(dim=-1)          # [V][Nc][nrhs]
    assert not fin[5, :, 2].any()                                        # the site itself (X term), column 2
    assert fin[:, :, [0, 1, 3, 4, 5, 6, 7]].all()                        # other columns untouched
    assert fin[:, :, 2].any()                                            # sites that are no neighbours of site 5
    op.close()


def test_tensor_launch_count_beyond_16_rhs():
    dims, Nc = (2, 2, 2, 2), 64
    links = synth.make_arbitrary_links(dims, Nc, 3, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links).set_option(cop.OPT_PATH, cop.PATH_TENSOR)
    for nrhs, want in ((3, 1), (16, 1), (17, 2), (40, 3)):
        vin = synth.make_vectors(dims, Nc, nrhs, 4, device="cuda")
        vout = torch.empty_like(vin)
        op.apply(vin, vout, nrhs=nrhs)
        torch.cuda.synchronize()
        assert op.last_launches == want and op.last_path == cop.PATH_TENSOR
    op.close()


@pytest.mark.parametrize("dagger", [0, 1])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
def test_arbitrary_links_not_gamma_hermitian(oracle_lib, prec, dagger):
    """The dagger must be the true adjoint for ANY links (no Gamma shortcut in the library)."""
    _run(oracle_lib, (3, 4, 2, 5), 48, prec, 1, dagger, cop.PATH_STREAM, hermitian=False)
    _run(oracle_lib, (3, 4, 2, 5), 128, prec, 1, dagger, cop.PATH_STREAM, hermitian=False)


@pytest.mark.parametrize("grid", [1, 7, 148, 1000])
def test_stream_path_any_grid(oracle_lib, grid):
    """Several items per CTA, a ragged tail, and more CTAs than items."""
    for dagger in (0, 1):
        _run(oracle_lib, (5, 3, 4, 7), 48, cop.LINK_C64, 1, dagger, cop.PATH_STREAM, grid=grid)
        _run(oracle_lib, (3, 3, 2, 2), 128, cop.LINK_I16, 1, dagger, cop.PATH_STREAM, grid=grid)


@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
def test_stream_fine_geometry(oracle_lib, Nc, prec):
    """The small-lattice row-block split (PAPER.md:L99 'additional parallelism'), forced on, and the
    automatic choice on a lattice with fewer regular work items than SMs."""
    _run(oracle_lib, (3, 2, 1, 4), Nc, prec, 1, 0, cop.PATH_STREAM, opts={cop.OPT_FINE: 2})
    _run(oracle_lib, (2, 2, 1, 2), Nc, prec, 1, 0, cop.PATH_STREAM, opts={cop.OPT_FINE: 0}, hermitian=False)
    _run(oracle_lib, (3, 2, 1, 4), Nc, prec, 1, 0, cop.PATH_STREAM, opts={cop.OPT_FINE: 1})


@pytest.mark.parametrize("stages", [2, 3, 5, 12, 64])
@pytest.mark.parametrize("keep", [1, 2])
def test_stream_ring_depth_and_l2_policy(oracle_lib, stages, keep):
    for dagger in (0, 1):
        _run(oracle_lib, (5, 3, 4, 7), 48, cop.LINK_C64, 1, dagger, cop.PATH_STREAM,
             opts={cop.OPT_STAGES: stages, cop.OPT_KEEP_LINKS: keep})
        _run(oracle_lib, (3, 3, 2, 2), 192, cop.LINK_I16, 1, dagger, cop.PATH_STREAM,
             opts={cop.OPT_STAGES: stages, cop.OPT_KEEP_LINKS: keep})


def test_apply_is_graph_capturable(oracle_lib):
    """coarse_op_apply only enqueues: a chain of applies can be captured into one CUDA graph (how
    bench.py times L2-resident lattices and how a solver would drive it)."""
    dims, Nc = (4, 4, 4, 4), 48
    links = synth.make_gamma_hermitian_links(dims, Nc, 31, device="cuda")
    v0 = synth.make_vectors(dims, Nc, 1, 32, device="cuda")
    v1, v2 = torch.empty_like(v0), torch.empty_like(v0)
    op = cop.CoarseOp(dims, Nc).set_links(links)
    op.apply(v0, v1)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.graph(g, stream=side):
        op.apply(v0, v1, dagger=0)
        op.apply(v1, v2, dagger=1)          # A^H A v0: one CGNE normal-equation application
    torch.cuda.current_stream().wait_stream(side)
    v1.zero_(); v2.zero_()
    g.replay()
    torch.cuda.synchronize()
    links_h = links.cpu().numpy()
    ref1 = oracle_lib.coarse_apply(dims, Nc, links_h, v0.cpu().numpy(), dagger=0)
    ref2 = oracle_lib.coarse_apply(dims, Nc, links_h, ref1.astype(np.complex64), dagger=1)
    assert rel_l2_per_rhs(v1.cpu().numpy(), ref1) <= TOL
    assert rel_l2_per_rhs(v2.cpu().numpy(), ref2) <= 2 * TOL
    op.close()


@pytest.mark.parametrize("dims,Nc,prec", [((4, 4, 4, 4), 48, 0), ((2, 4, 2, 2), 192, 1), ((5, 3, 4, 7), 64, 1), ((1, 1, 1, 2), 32, 0)])
def test_programmatic_dependent_launch_chain(oracle_lib, dims, Nc, prec):
    """COARSE_OPT_PDL: a chain of applies where each kernel may start while its predecessor drains, including
    the ping-pong a -> b -> a whose second kernel WRITES the buffer the first one reads.  Results must be
    bit-identical to the same chain launched normally, and correct against the oracle."""
    V = synth.lattice_volume(dims)
    links, scales, links_h, scales_h = _links_for(dims, Nc, prec, 77, False, oracle_lib)
    if prec == cop.LINK_C64:
        links = links * 0.25                      # keep the 6-fold product's magnitude moderate
        links_h = links.cpu().numpy()
    else:
        scales = scales * 0.25
        scales_h = scales.cpu().numpy()
    v0 = synth.make_vectors(dims, Nc, 1, 78, device="cuda")
    outs = {}
    for pdl in (0, 1):
        op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales).set_option(cop.OPT_PDL, pdl)
        a, b = v0.clone(), torch.empty_like(v0)
        for k in range(6):
            op.apply(a, b, dagger=k & 1)
            a, b = b, a
        torch.cuda.synchronize()
        outs[pdl] = a.clone()
        op.close()
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[1]))
    ref = v0.cpu().numpy()
    for k in range(6):
        ref = oracle_lib.coarse_apply(dims, Nc, links_h, ref.astype(np.complex64), dagger=k & 1, link_precision=prec,
                                      scales=scales_h)
    assert rel_l2_per_rhs(outs[1].cpu().numpy(), ref) <= 6 * TOL


def test_pdl_with_parts_hvec_and_graph_capture(oracle_lib):
    dims, Nc = (4, 4, 2, 2), 48
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 5, device="cuda") * 0.25
    v = synth.make_vectors(dims, Nc, 1, 6, device="cuda")
    res = {}
    for pdl in (0, 1):
        op = cop.CoarseOp(dims, Nc).set_links(links).set_option(cop.OPT_PDL, pdl)
        t, out = torch.zeros_like(v), torch.zeros_like(v)
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.graph(g, stream=side):
            for _ in range(3):
                op.apply_parts(None, v, t, parity=cop.PARITY_ODD, local=cop.LOCAL_NONE, alpha=0.0, beta=1.0)
                op.apply_parts(v, t, out, parity=cop.PARITY_EVEN, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)
        torch.cuda.current_stream().wait_stream(side)
        g.replay()
        torch.cuda.synchronize()
        q = torch.empty((V, Nc, 1, 2), dtype=torch.int16, device="cuda")
        nm = torch.empty((V, 1), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_vec_i16(out, Nc, 1, q, nm)
        o2 = torch.empty_like(v)
        op.apply_hvec(q, nm, o2)
        torch.cuda.synchronize()
        res[pdl] = (out.clone(), o2.clone())
        op.close()
    assert torch.equal(torch.view_as_real(res[0][0]), torch.view_as_real(res[1][0]))
    assert torch.equal(torch.view_as_real(res[0][1]), torch.view_as_real(res[1][1]))


@pytest.mark.parametrize("dims", [(2, 4, 2, 2), (1, 1, 1, 1), (3, 2, 1, 4), (3, 3, 3, 5)])
@pytest.mark.parametrize("Nc", [32, 48, 64, 96, 128, 192])
@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
def test_split_dagger_on_tiny_lattices(oracle_lib, dims, Nc, prec):
    """dagger = 1 with fewer sites than SMs (the paper's level 3 has 32 sites per GPU): the contraction of
    a site is split over its row chunks - in thread-block clusters whose partial vectors meet in the first CTA's
    shared memory (auto, 2), or through a global workspace with a per-site counter (3).  Forcing it off (1) must give
    the same numbers up to summation order, all must match the oracle, and repeated launches must be bit-identical for
    any grid (one cluster walking every site: the inbox is double buffered; the chunk counters reset themselves).
    135 sites: several sites per cluster also in the default launch."""
    V = synth.lattice_volume(dims)
    links, scales, links_h, scales_h = _links_for(dims, Nc, prec, 61, False, oracle_lib)
    vin = synth.make_vectors(dims, Nc, 1, 62, device="cuda")
    ref = oracle_lib.coarse_apply(dims, Nc, links_h, vin.cpu().numpy(), dagger=1, link_precision=prec, scales=scales_h)
    for mode in (0, 1, 2, 3):
        op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales).set_option(cop.OPT_SPLIT_DAGGER, mode)
        out = torch.full_like(vin, float("nan"))
        op.apply(vin, out, dagger=1)
        torch.cuda.synchronize()
        assert op.last_path == cop.PATH_STREAM and op.last_launches == 1
        assert rel_l2_per_rhs(out.cpu().numpy(), ref) <= TOL
        for grid in (0, 1, 5, 9):                       # many launches, also with every chunk of a site on one CTA
            op.set_option(cop.OPT_GRID, grid)
            for _ in range(3):
                again = torch.full_like(vin, float("nan"))
                op.apply(vin, again, dagger=1)
                torch.cuda.synchronize()
                assert torch.equal(torch.view_as_real(again), torch.view_as_real(out))
        op.set_option(cop.OPT_GRID, 0)
        # dagger = 0 is untouched by the option
        op.apply(vin, out, dagger=0)
        torch.cuda.synchronize()
        assert op.last_launches == 1
        op.close()


@pytest.mark.parametrize("Nc,prec", [(192, cop.LINK_I16), (128, cop.LINK_C64), (48, cop.LINK_C64)])
def test_split_dagger_clusters_bit_reproducible_under_stress(Nc, prec):
    """The paper's level-3 volume (32 sites): 3000 alternating A / A^H applies in one stream (PDL chain, cluster launches for
    A^H), every result equal to the first one's bit for bit."""
    dims = (2, 4, 2, 2)
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        links = q
    vin = synth.make_vectors(dims, Nc, 1, 6, device="cuda")
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    refs = {}
    for dagger in (0, 1):
        refs[dagger] = torch.empty_like(vin)
        op.apply(vin, refs[dagger], dagger=dagger)
    outs = [torch.empty_like(vin) for _ in range(6)]
    bad = 0
    for rep in range(500):
        for k in range(6):
            op.apply(vin, outs[k], dagger=k % 2)
        torch.cuda.synchronize()
        for k in range(6):
            bad += int(not torch.equal(torch.view_as_real(outs[k]), torch.view_as_real(refs[k % 2])))
    assert bad == 0, f"{bad} of 3000 applies differ from the first one"
    op.close()


def test_read_probe_runs_and_validates_arguments():
    buf = torch.zeros(64 << 20, dtype=torch.uint8, device="cuda")
    assert cop.coarse_op_probe_read(buf, 16384, 6) == 64 << 20
    assert cop.coarse_op_probe_read(buf[: 100000], 16384, 2) == 6 * 16384
    torch.cuda.synchronize()
    L = cop.lib()
    assert L.coarse_op_probe_read(buf.data_ptr(), 1 << 20, 1000, 6, None) == cop.EINVAL
    assert L.coarse_op_probe_read(buf.data_ptr(), 1 << 20, 65536, 8, None) == cop.EINVAL     # does not fit smem
    assert L.coarse_op_probe_read(None, 1 << 20, 16384, 6, None) == cop.EINVAL
    assert L.coarse_op_probe_read(buf.data_ptr(), 100, 16384, 6, None) == cop.EINVAL


def test_bit_reproducible():
    dims, Nc = (4, 4, 4, 6), 64
    links = synth.make_gamma_hermitian_links(dims, Nc, 5, device="cuda")
    vin = synth.make_vectors(dims, Nc, 1, 6, device="cuda")
    op = cop.CoarseOp(dims, Nc).set_links(links)
    outs = []
    for _ in range(3):
        vout = torch.empty_like(vin)
        op.apply(vin, vout)
        torch.cuda.synchronize()
        outs.append(vout.clone())
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[1]))
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[2]))


def test_apply_host_matches_device_apply(oracle_lib):
    dims, Nc = (4, 3, 2, 5), 48
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, 8, device="cuda")
    vin = synth.make_vectors(dims, Nc, 1, 9, device="cpu").pin_memory()
    vout = torch.empty((V, Nc, 1), dtype=torch.complex64).pin_memory()
    op = cop.CoarseOp(dims, Nc).set_links(links)
    for dagger in (0, 1):
        op.apply_host(vin, vout, dagger=dagger)
        ref = oracle_lib.coarse_apply(dims, Nc, links.cpu().numpy(), vin.numpy(), dagger=dagger)
        assert rel_l2_per_rhs(vout.numpy(), ref) <= TOL


@pytest.mark.parametrize("prec", [cop.LINK_C64, cop.LINK_I16])
def test_apply_host_pipelined_path_is_bit_identical(oracle_lib, prec):
    """Large enough for coarse_op_apply_host's pipelined path (4 ranges of x3-slices, H2D / kernels / D2H on
    three streams): must equal the plain device apply bit for bit, for both modes, and repeatedly."""
    dims, Nc = (8, 8, 8, 24), 48
    V = synth.lattice_volume(dims)
    links, scales, _, _ = _links_for(dims, Nc, prec, 3, True, oracle_lib) if prec == cop.LINK_C64 else (None, None, None, None)
    if prec == cop.LINK_I16:
        lc = synth.make_gamma_hermitian_links(dims, Nc, 3, device="cuda")
        links = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(lc, Nc, links, scales)
        del lc
    vin_d = synth.make_vectors(dims, Nc, 1, 4, device="cuda")
    vin = vin_d.cpu().pin_memory()
    vout = torch.empty_like(vin).pin_memory()
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    for rep in range(2):
        for dagger in (0, 1):
            ref = torch.empty_like(vin_d)
            op.apply(vin_d, ref, dagger=dagger)
            torch.cuda.synchronize()
            vout.fill_(float("nan"))
            op.apply_host(vin, vout, dagger=dagger)
            assert op.last_launches == 4 and op.last_path == cop.PATH_STREAM
            assert torch.equal(torch.view_as_real(vout), torch.view_as_real(ref.cpu()))
    # and against the oracle on sampled sites
    sites = np.array([0, 1, 511, 512, V // 2, V - 513, V - 512, V - 1], dtype=np.int64)
    got = vout.numpy()[sites]
    refo = oracle_lib.coarse_apply_sites(dims, Nc, links.cpu().numpy(), vin.numpy(), sites, dagger=1,
                                         link_precision=prec, scales=None if scales is None else scales.cpu().numpy())
    assert rel_l2_per_rhs(got, refo) <= TOL
    op.close()


@pytest.mark.parametrize("Nc,prec,nrhs,want_path,launches", [
    (48, cop.LINK_I16, 3, cop.PATH_STREAM, 4), (64, cop.LINK_C64, 16, cop.PATH_TENSOR, 8),
    (48, cop.LINK_I16, 20, cop.PATH_TENSOR, 16), (64, cop.LINK_I16, 4, cop.PATH_TENSOR, 4)])
def test_apply_host_pipelined_multi_rhs_is_bit_identical(oracle_lib, Nc, prec, nrhs, want_path, launches):
    """The pipelined host path for several right-hand sides: STREAM-MR (3 = one propagator) and
    TENSOR launch ranges of x3-slices too; results must equal the device-resident apply bit for bit."""
    dims = (8, 8, 8, 16)                      # vectors of at least 4 MiB: the pipelined path
    V = synth.lattice_volume(dims)
    links = synth.make_arbitrary_links(dims, Nc, 5, device="cuda")
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device="cuda")
        scales = torch.empty((V, 9), dtype=torch.float32, device="cuda")
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links = q
    vin_d = synth.make_vectors(dims, Nc, nrhs, 6, device="cuda")
    vin = vin_d.cpu().pin_memory()
    vout = torch.empty_like(vin).pin_memory()
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    i8 = prec == cop.LINK_I16 and want_path == cop.PATH_TENSOR
    for dagger in (0, 1):
        ref_default = torch.empty_like(vin_d)
        op.apply(vin_d, ref_default, nrhs=nrhs, dagger=dagger)
        ref = ref_default
        if i8:
            # the device-resident apply runs int16 links on the integer tensor-core kernel; the site-range launches of
            # apply_host use the 3xTF32 kernel (include/coarse_op.h): bit-identical to THAT kernel, 1e-5 to the other
            # (the path is pinned for the comparison run: with the integer kernel switched off AUTO sends 2-4 RHS to STREAM)
            op.set_option(cop.OPT_TENSOR_I8, 1)
            op.set_option(cop.OPT_PATH, cop.PATH_TENSOR)
            ref = torch.empty_like(vin_d)
            op.apply(vin_d, ref, nrhs=nrhs, dagger=dagger)
            op.set_option(cop.OPT_TENSOR_I8, 0)
            op.set_option(cop.OPT_PATH, cop.PATH_AUTO)
        torch.cuda.synchronize()
        vout.fill_(float("nan"))
        op.apply_host(vin, vout, nrhs=nrhs, dagger=dagger)
        assert op.last_launches == launches and op.last_path == want_path
        assert torch.equal(torch.view_as_real(vout), torch.view_as_real(ref.cpu()))
        assert rel_l2_per_rhs(vout.numpy(), ref_default.cpu().numpy()) <= 3e-6
    op.close()


# ------------------------------------------------------------------ ABI behaviour
def test_error_codes():
    dims, Nc = (2, 2, 2, 2), 48
    V = 16
    with pytest.raises(cop.CoarseOpError):
        cop.coarse_op_create((2, 2, 0, 2), Nc, cop.LINK_C64)
    with pytest.raises(cop.CoarseOpError):
        cop.coarse_op_create(dims, 7, cop.LINK_C64)
    with pytest.raises(cop.CoarseOpError):
        cop.coarse_op_create(dims, Nc, 5)
    h = cop.coarse_op_create(dims, Nc, cop.LINK_C64)
    assert cop.coarse_op_link_bytes(h) == V * 9 * Nc * Nc * 8
    assert cop.coarse_op_scale_bytes(h) == 0
    assert cop.coarse_op_vector_bytes(h, 3) == V * Nc * 3 * 8
    vin = torch.zeros((V, Nc, 1), dtype=torch.complex64, device="cuda")
    vout = torch.zeros_like(vin)
    L = cop.lib()
    assert L.coarse_op_apply(h, vin.data_ptr(), vout.data_ptr(), 1, 0, None) == cop.ENOTREADY
    links = torch.zeros((V, 9, Nc, Nc), dtype=torch.complex64, device="cuda")
    assert L.coarse_op_set_links(h, links.data_ptr(), vin.data_ptr()) == cop.EINVAL      # scales with C64
    assert L.coarse_op_set_links(h, links.data_ptr() + 8, None) == cop.EINVAL            # misaligned
    assert L.coarse_op_set_links(h, links.data_ptr(), None) == cop.OK
    assert L.coarse_op_apply(h, vin.data_ptr(), vin.data_ptr(), 1, 0, None) == cop.EINVAL      # overlap
    assert L.coarse_op_apply(h, vin.data_ptr(), vout.data_ptr(), 0, 0, None) == cop.EINVAL     # nrhs
    assert L.coarse_op_apply(h, vin.data_ptr(), vout.data_ptr(), 1, 2, None) == cop.EINVAL     # dagger
    assert L.coarse_op_apply(h, None, vout.data_ptr(), 1, 0, None) == cop.EINVAL
    assert "dagger" in cop.coarse_op_last_error() or "NULL" in cop.coarse_op_last_error()
    assert L.coarse_op_set_option(h, cop.OPT_PATH, 99) == cop.EINVAL
    assert L.coarse_op_set_option(h, cop.OPT_STAGES, 1) == cop.EINVAL
    assert L.coarse_op_set_option(h, cop.OPT_FINE, 3) == cop.EINVAL
    assert L.coarse_op_set_option(h, cop.OPT_KEEP_LINKS, -1) == cop.EINVAL
    assert L.coarse_op_set_option(h, 77, 0) == cop.EINVAL
    assert L.coarse_op_apply(h, vin.data_ptr(), vout.data_ptr(), 1, 0, None) == cop.OK
    cop.coarse_op_destroy(h)
    cop.coarse_op_destroy(0)
    h16 = cop.coarse_op_create(dims, Nc, cop.LINK_I16)
    assert cop.coarse_op_link_bytes(h16) == V * 9 * Nc * Nc * 4
    assert cop.coarse_op_scale_bytes(h16) == V * 9 * 4
    assert L.coarse_op_set_links(h16, links.data_ptr(), None) == cop.EINVAL              # I16 needs scales
    cop.coarse_op_destroy(h16)
    h6 = cop.coarse_op_create(dims, 6, cop.LINK_C64)
    assert L.coarse_op_set_option(h6, cop.OPT_PATH, cop.PATH_STREAM) == cop.EUNSUPPORTED
    cop.coarse_op_destroy(h6)


def test_quantiser_edge_cases_bit_exact(oracle_lib):
    Nc = 16
    links = synth.make_gamma_hermitian_links((2, 2, 1, 2), Nc, 77, device="cuda")
    links[1, 3] = 0
    links[2, 5] *= 1e-30
    links[3, 0, 0, 0] = 1e30
    q = torch.empty(links.shape + (2,), dtype=torch.int16, device="cuda")
    sc = torch.empty(links.shape[:2], dtype=torch.float32, device="cuda")
    cop.coarse_op_quantize_i16(links, Nc, q, sc)
    torch.cuda.synchronize()
    q_ref, sc_ref = oracle_lib.quantize_i16(links.cpu().numpy(), Nc)
    assert np.array_equal(sc.cpu().numpy().reshape(-1), sc_ref)
    assert np.array_equal(q.cpu().numpy().reshape(q_ref.shape), q_ref)
