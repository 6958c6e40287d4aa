"""CPU check of tests/fullsize.py (the chunked whole-lattice comparison the GPU parity tests use):
chunking over x3-slices with wrap-around halos must reproduce the full oracle apply exactly, and one
wrong site must show up."""
import numpy as np
import pytest
import torch

import synth
from tests.fullsize import chunk_slices, whole_lattice_errors


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("slices", [1, 2, 5])
def test_chunked_comparison_equals_full_apply(oracle_lib, prec, slices):
    dims, Nc, nrhs = (2, 3, 2, 5), 6, 2
    V = 60
    links = synth.make_arbitrary_links(dims, Nc, 31)
    scales = None
    links_dev = links
    if prec == 1:
        q, sc = oracle_lib.quantize_i16(links.numpy(), Nc)
        links_dev = torch.from_numpy(q.reshape(V, 9, Nc, Nc, 2))
        scales = torch.from_numpy(sc.reshape(V, 9))
    vin = synth.make_vectors(dims, Nc, nrhs, 32)
    outs = {}
    for dg in (0, 1):
        ref = oracle_lib.coarse_apply(dims, Nc, links_dev.numpy(), vin.numpy(), nrhs=nrhs, dagger=dg,
                                      link_precision=prec, scales=None if scales is None else scales.numpy())
        outs[dg] = torch.from_numpy(ref.astype(np.complex64))
    res = whole_lattice_errors(oracle_lib, dims, Nc, links_dev, scales, prec, outs, nrhs, vin_h=vin.numpy(),
                               slices_per_chunk=slices)
    for dg in (0, 1):
        err, worst, n = res[dg]
        assert n == V and err < 2e-7 and worst < 2e-7          # complex64 rounding of the reference only
    # one wrong entry at one site must be seen
    outs[1][37, 2, 1] += 1e-3
    res = whole_lattice_errors(oracle_lib, dims, Nc, links_dev, scales, prec, outs, nrhs, vin_h=vin.numpy(),
                               slices_per_chunk=slices)
    assert res[1][1] > 5e-5 and res[0][1] < 2e-7


def test_chunks_cover_every_slice_once():
    for T, budget in ((24, 6 << 30), (12, 3 << 30), (5, 1), (1, 1 << 40)):
        ch = chunk_slices((16, 16, 16, T), 9 * 48 * 48 * 8, budget)
        assert [t for a, b in ch for t in range(a, b)] == list(range(T))
