"""Counter-based seeded generators for coarse-operator links and vectors.

Every value is a pure function of (seed, field id, flat index): a splitmix64
hash of the counter feeds a Box-Muller transform evaluated in float64, and the
result is cast to float32.  The same call therefore returns the same numbers no
matter how it is chunked.  The code is plain torch integer/float ops, so it runs
on the CPU (small test lattices) and on the GPU (BASELINE-size lattices, which
are far too large to ship or to draw on the host in reasonable time).  CPU and
CUDA `log`/`cos` may differ in the last bit; nothing relies on the two devices
agreeing: inputs are drawn once and the SAME bits are handed to the CUDA path
and to the oracle.

Structure of the inputs (BASELINE.json configs 1-5):
  * Y_{+mu}(x): every real component ~ N(0, 1/Nc)   ("Gaussian scaled by 1/sqrt(Nc)")
  * Y_{-mu}(x+mu^) = Gamma . Y_{+mu}(x)^dagger . Gamma,  Gamma = diag(I_{Nc/2}, -I_{Nc/2})
    (the "gamma5-Hermiticity on the coarse level" the chiral doubling preserves,
    PAPER.md:L41 §2.1)
  * X(x) = 0.1*I + 0.1*S(x),  S = (G + Gamma G^dagger Gamma)/2, G drawn like Y
  * vectors: every real component ~ N(0,1)

Layouts (the C-ABI's, include/coarse_op.h):
  links[s][m][i][j] complex64, m = 0:X, 1+mu:Y_{+mu}, 5+mu:Y_{-mu}; row-major
  vectors v[s][a][r] complex64, r (right-hand side) innermost
  site index s(x) = x0 + L0*(x1 + L1*(x2 + L2*x3))
"""
from __future__ import annotations

import math
from typing import Sequence

import torch

FIELD_YPLUS = 1
FIELD_G = 2
FIELD_IN = 3
FIELD_ANY = 4

_M64 = (1 << 64) - 1


def _signed(v: int) -> int:
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


_C0 = _signed(0x9E3779B97F4A7C15)
_C1 = _signed(0xBF58476D1CE4E5B9)
_C2 = _signed(0x94D049BB133111EB)


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """Logical right shift of an int64 tensor (torch's >> is arithmetic)."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 tensors (two's-complement wrap-around)."""
    z = z + _C0
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def _mix64_py(v: int) -> int:
    v = (v + 0x9E3779B97F4A7C15) & _M64
    v = ((v ^ (v >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    v = ((v ^ (v >> 27)) * 0x94D049BB133111EB) & _M64
    return v ^ (v >> 31)


def _key(seed: int, field: int) -> int:
    return _signed(_mix64_py(_mix64_py(seed & _M64) ^ (field * 0xD1B54A32D192ED03 & _M64)))


def normal(seed: int, field: int, start: int, count: int, device="cpu") -> torch.Tensor:
    """count standard normals (float64) for counters start..start+count-1."""
    c = torch.arange(start, start + count, dtype=torch.int64, device=device)
    key = _key(seed, field)
    h1 = _mix64(c * 2 + key)
    h2 = _mix64(c * 2 + 1 + key)
    inv53 = 1.0 / float(1 << 53)
    u1 = (_lsr(h1, 11).to(torch.float64) + 0.5) * inv53
    u2 = (_lsr(h2, 11).to(torch.float64) + 0.5) * inv53
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def lattice_volume(dims: Sequence[int]) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def site_index(x: Sequence[int], dims: Sequence[int]) -> int:
    return x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))


def _gamma_sign(Nc: int, device) -> torch.Tensor:
    g = torch.ones(Nc, dtype=torch.float64, device=device)
    g[Nc // 2:] = -1.0
    return g[:, None] * g[None, :]          # gamma_i * gamma_j


def make_gamma_hermitian_links(dims, Nc: int, seed: int, device="cpu",
                               chunk_sites: int = 2048) -> torch.Tensor:
    """links[V][9][Nc][Nc] complex64 with the Gamma-Hermitian structure above."""
    V = lattice_volume(dims)
    links = torch.empty((V, 9, Nc, Nc), dtype=torch.complex64, device=device)
    sigma = 1.0 / math.sqrt(Nc)
    gg = _gamma_sign(Nc, device)
    eye = torch.eye(Nc, dtype=torch.complex128, device=device)
    per_y = 4 * Nc * Nc * 2
    per_g = Nc * Nc * 2
    for s0 in range(0, V, chunk_sites):
        n = min(chunk_sites, V - s0)
        y = normal(seed, FIELD_YPLUS, s0 * per_y, n * per_y, device) * sigma
        y = torch.view_as_complex(y.view(n, 4, Nc, Nc, 2).to(torch.float32))
        links[s0:s0 + n, 1:5] = y
        g = normal(seed, FIELD_G, s0 * per_g, n * per_g, device) * sigma
        g = torch.view_as_complex(g.view(n, Nc, Nc, 2))
        s_mat = 0.5 * (g + gg * g.transpose(-1, -2).conj())
        links[s0:s0 + n, 0] = (0.1 * eye + 0.1 * s_mat).to(torch.complex64)
        del y, g, s_mat
    L0, L1, L2, L3 = (int(d) for d in dims)
    gg32 = gg.to(torch.float32)
    for mu in range(4):
        yp = links[:, 1 + mu].reshape(L3, L2, L1, L0, Nc, Nc)
        shifted = torch.roll(yp, shifts=1, dims=3 - mu)      # shifted[x] = Y_{+mu}(x - mu^)
        ym = gg32 * shifted.transpose(-1, -2).conj()
        links[:, 5 + mu] = ym.reshape(V, Nc, Nc)
        del shifted, ym
    return links


def make_arbitrary_links(dims, Nc: int, seed: int, device="cpu",
                         chunk_sites: int = 2048) -> torch.Tensor:
    """links[V][9][Nc][Nc] complex64, all nine matrices iid N(0, 1/Nc) per component
    (no Gamma structure: used for the adjoint identity, which must hold for any links)."""
    V = lattice_volume(dims)
    links = torch.empty((V, 9, Nc, Nc), dtype=torch.complex64, device=device)
    sigma = 1.0 / math.sqrt(Nc)
    per = 9 * Nc * Nc * 2
    for s0 in range(0, V, chunk_sites):
        n = min(chunk_sites, V - s0)
        y = normal(seed, FIELD_ANY, s0 * per, n * per, device) * sigma
        links[s0:s0 + n] = torch.view_as_complex(y.view(n, 9, Nc, Nc, 2).to(torch.float32))
    return links


def make_vectors(dims, Nc: int, nrhs: int, seed: int, device="cpu") -> torch.Tensor:
    """v[V][Nc][nrhs] complex64, iid complex Gaussian (each real component ~ N(0,1))."""
    V = lattice_volume(dims)
    n = V * Nc * nrhs * 2
    z = normal(seed, FIELD_IN, 0, n, device).to(torch.float32)
    return torch.view_as_complex(z.view(V, Nc, nrhs, 2))


# BASELINE.json configs (C1..C5).  "links": "c64" | "i16".
CONFIGS = {
    "C1": dict(dims=(4, 4, 4, 4), Nc=48, links="c64", nrhs=1, seed=20221201),
    "C2": dict(dims=(16, 16, 16, 24), Nc=48, links="c64", nrhs=1, seed=20221202),
    "C3": dict(dims=(8, 8, 8, 12), Nc=128, links="c64", nrhs=1, seed=20221203),
    "C4": dict(dims=(16, 16, 16, 24), Nc=64, links="i16", nrhs=1, seed=20221204),
    "C5": dict(dims=(8, 8, 8, 12), Nc=128, links="c64", nrhs=16, seed=20221205),
    # The paper's own per-GPU coarse volumes (not BASELINE configs, derived from
    # PAPER.md:L117/L125/L133 Table 1): local 24x48x24x36 / aggregate 4x6x6x6 = 6x8x4x6 sites at
    # level 2 (Nc = 64x2), / 3x2x2x3 = 2x4x2x2 sites at level 3 (Nc = 96x2); int16 links (L99).
    "P2": dict(dims=(6, 8, 4, 6), Nc=128, links="i16", nrhs=1, seed=20221206),
    "P3": dict(dims=(2, 4, 2, 2), Nc=192, links="i16", nrhs=1, seed=20221207),
}


def config(name: str) -> dict:
    return dict(CONFIGS[name])
