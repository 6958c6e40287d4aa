"""Whole-lattice oracle comparison at BASELINE sizes without holding 16 GB of links on the host.

The oracle evaluates its definition one output site at a time (`coarse_apply_sites`, the same
`apply_site` as the full apply) and indexes the link array by GLOBAL site, so the host copy is a
full-size `np.empty` whose pages are committed only where a chunk's sites (and, for the dagger apply,
their x3-neighbours) live: chunks of x3-slices are brought over one after the other, every site of
the chunk is evaluated in both modes, and the chunk's pages are released before the next one.
EVERY output site of the lattice is compared ("per RHS r over the whole lattice").
No oracle/ import here: the caller passes the loaded oracle module in.
"""
from __future__ import annotations

import numpy as np
import torch


def host_mem_available_bytes() -> int:
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) * 1024
    except OSError:
        pass
    return 8 << 30


def chunk_slices(dims, bytes_per_site: int, budget_bytes: int):
    """Split the T = dims[3] x3-slices into chunks [t0, t1) such that a chunk plus one halo slice on
    either side stays under budget_bytes of host link storage."""
    T = int(dims[3])
    plane = int(dims[0]) * int(dims[1]) * int(dims[2])
    per_slice = plane * bytes_per_site
    k = max(1, int(budget_bytes // per_slice) - 2)
    return [(t0, min(T, t0 + k)) for t0 in range(0, T, k)]


def whole_lattice_errors(oracle_lib, dims, Nc, links_dev, scales_dev, link_precision, outs, nrhs,
                         vin_h=None, hvec=None, budget_bytes: int = 6 << 30, slices_per_chunk: int = 0):
    """Compare outs[dagger] (device tensors [V][Nc][nrhs] complex64) with the oracle at every site.

    links_dev: the device link tensor exactly as handed to the library (complex64 [V][9][Nc][Nc] or
    int16 [V][9][Nc][Nc][2]); vin_h: host complex64 input (plain apply) or hvec = (q_h, norms_h) for
    half-precision input vectors.  Returns {dagger: (max over r of rel-L2 over the WHOLE lattice,
    max per-site rel-L2, number of sites compared)}.
    """
    dims = tuple(int(d) for d in dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    T, plane = dims[3], V // dims[3]
    i16 = link_precision == 1
    flat = links_dev if i16 else torch.view_as_real(links_dev)
    tail = (9, Nc, Nc, 2)
    np_dtype = np.int16 if i16 else np.float32
    bytes_per_site = 9 * Nc * Nc * (4 if i16 else 8)
    budget = min(budget_bytes, max(1 << 30, host_mem_available_bytes() // 3))
    scales_h = None if scales_dev is None else scales_dev.cpu().numpy()
    num = {dg: np.zeros(nrhs) for dg in outs}
    den = {dg: np.zeros(nrhs) for dg in outs}
    worst_site = {dg: 0.0 for dg in outs}
    count = 0
    chunks = chunk_slices(dims, bytes_per_site, budget)
    if slices_per_chunk > 0:
        chunks = [(t0, min(T, t0 + slices_per_chunk)) for t0 in range(0, T, slices_per_chunk)]
    for t0, t1 in chunks:
        need = sorted({t % T for t in range(t0 - 1, t1 + 1)})
        links_h = np.empty((V,) + tail, dtype=np_dtype)          # virtual: only the needed slices are touched
        for t in need:
            links_h[t * plane:(t + 1) * plane] = flat[t * plane:(t + 1) * plane].cpu().numpy().reshape((plane,) + tail)
        sites = np.arange(t0 * plane, t1 * plane, dtype=np.int64)
        for dg, out_dev in outs.items():
            if hvec is None:
                ref = oracle_lib.coarse_apply_sites(dims, Nc, links_h, vin_h, sites, nrhs=nrhs, dagger=dg,
                                                    link_precision=link_precision, scales=scales_h)
            else:
                ref = oracle_lib.coarse_apply_hvec_sites(dims, Nc, links_h, hvec[0], hvec[1], sites, nrhs=nrhs,
                                                         dagger=dg, link_precision=link_precision, scales=scales_h)
            got = out_dev[t0 * plane:t1 * plane].cpu().numpy().astype(np.complex128)
            d = got - ref
            num[dg] += (np.abs(d) ** 2).sum(axis=(0, 1))
            den[dg] += (np.abs(ref) ** 2).sum(axis=(0, 1))
            per_site = np.sqrt((np.abs(d) ** 2).sum(axis=(1, 2)) / (np.abs(ref) ** 2).sum(axis=(1, 2)))
            worst_site[dg] = max(worst_site[dg], float(per_site.max()))
        count += len(sites)
        del links_h
    return {dg: (float(np.sqrt(num[dg] / den[dg]).max()), worst_site[dg], count) for dg in outs}
