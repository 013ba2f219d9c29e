"""Seeded synthetic inputs for the COLA hot path (links, sources, gauge transforms).

This module holds NO arithmetic of the method (no Dirac operator, no clover term, no solver):
it only produces the arrays that both the CPU oracle (`oracle/`) and the CUDA library consume.
It imports neither of them.  Recipe: SURVEY.md §8(d) "Synthetic inputs" / BASELINE.json configs
(`BJ:cK`); the paper itself states no lattice sizes or couplings.

Counter-based generator, so a value depends only on (seed, stream, global index, k) and never on
layout, chunking or device:

    u64(seed, stream, idx, k) = splitmix64( seed XOR (stream << 56) XOR (idx*64 + k) )
    N(0,1) from two u64 by Box-Muller

`idx` = 4*i(x)+mu for links, i(x) for sites, with i(x) = x + Lx*(y + Ly*(z + Lz*t)).

Canonical array shapes (complex128, C order):
    links   U[t][z][y][x][mu][a][b]      (U psi)_a = sum_b U_ab psi_b
    spinor  psi[t][z][y][x][s][c]        s = spin 0..3, c = colour 0..2

Everything is implemented with torch ops so the same code runs on the CPU (small lattices, the
oracle's inputs) and on a CUDA device (the 48^3x96 / 64^3x128 fields); integer hashing is exact
on both, the floating-point part agrees to rounding.
"""
from __future__ import annotations

import math

import numpy as np
import torch

STREAM_LINKS = 1
STREAM_SOURCE = 2
STREAM_GAUGE_TRANSFORM = 3

_M64 = (1 << 64) - 1


def _i64(v: int) -> int:
    """Python int (mod 2^64) -> the same bit pattern as a signed 64-bit value."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 bit patterns."""
    return (x >> s) & _i64((1 << (64 - s)) - 1)


def splitmix64(x: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 bit patterns (wrapping arithmetic)."""
    z = x + _i64(0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _i64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _i64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def splitmix64_int(x: int) -> int:
    """Scalar pure-Python splitmix64 (used by tests to pin the tensor version)."""
    z = (x + 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def normals(seed: int, stream: int, idx: torch.Tensor, count: int) -> torch.Tensor:
    """`count` independent N(0,1) per entry of the int64 tensor `idx` -> float64 [..., count]."""
    if count > 32:
        raise ValueError("at most 32 normals per index (64 counters)")
    dev = idx.device
    k = torch.arange(count, dtype=torch.int64, device=dev)
    base = (idx.to(torch.int64) * 64).unsqueeze(-1)
    key = _i64(seed ^ (stream << 56))
    a = splitmix64((base + 2 * k) ^ key)
    b = splitmix64((base + 2 * k + 1) ^ key)
    u1 = (_lsr(a, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)
    u2 = (_lsr(b, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def volume(dims) -> int:
    lx, ly, lz, lt = dims
    return lx * ly * lz * lt


def _gell_mann(device) -> torch.Tensor:
    lam = np.zeros((8, 3, 3), dtype=np.complex128)
    lam[0][0, 1] = lam[0][1, 0] = 1
    lam[1][0, 1] = -1j
    lam[1][1, 0] = 1j
    lam[2][0, 0] = 1
    lam[2][1, 1] = -1
    lam[3][0, 2] = lam[3][2, 0] = 1
    lam[4][0, 2] = -1j
    lam[4][2, 0] = 1j
    lam[5][1, 2] = lam[5][2, 1] = 1
    lam[6][1, 2] = -1j
    lam[6][2, 1] = 1j
    lam[7] = np.diag([1, 1, -2]) / math.sqrt(3.0)
    return torch.from_numpy(lam).to(device)


def _expm_antihermitian(x: torch.Tensor) -> torch.Tensor:
    """exp(X) for a batch of small 3x3 matrices: scaling (2^-4) + 18-term Taylor + 4 squarings."""
    n_sq = 4
    y = x * (1.0 / (1 << n_sq))
    eye = torch.eye(3, dtype=x.dtype, device=x.device).expand_as(x)
    acc = eye.clone()
    term = eye.clone()
    for n in range(1, 19):
        term = torch.matmul(term, y) * (1.0 / n)
        acc = acc + term
    for _ in range(n_sq):
        acc = torch.matmul(acc, acc)
    return acc


def links_smooth(dims, eps: float, seed: int, device="cpu", chunk: int = 1 << 22) -> torch.Tensor:
    """U = exp(i*eps*H), H = sum_a w_a lambda_a/2, w_a ~ N(0,1)  (BJ:c1..c4)."""
    v = volume(dims)
    lam = _gell_mann(device)
    out = torch.empty((4 * v, 3, 3), dtype=torch.complex128, device=device)
    for lo in range(0, 4 * v, chunk):
        hi = min(4 * v, lo + chunk)
        idx = torch.arange(lo, hi, dtype=torch.int64, device=device)
        w = normals(seed, STREAM_LINKS, idx, 8).to(torch.complex128)
        h = torch.einsum("na,aij->nij", w, lam) * 0.5
        out[lo:hi] = _expm_antihermitian(1j * eps * h)
    lx, ly, lz, lt = dims
    return out.reshape(lt, lz, ly, lx, 4, 3, 3)


def links_haar(dims, seed: int, device="cpu") -> torch.Tensor:
    """Random SU(3) by Gram-Schmidt of two complex Gaussian rows, third row = conj(r1 x r2) (BJ:c0)."""
    v = volume(dims)
    idx = torch.arange(4 * v, dtype=torch.int64, device=device)
    g = normals(seed, STREAM_LINKS, idx, 12)
    g1 = torch.complex(g[:, 0:3], g[:, 3:6])
    g2 = torch.complex(g[:, 6:9], g[:, 9:12])
    r1 = g1 / torch.linalg.vector_norm(g1, dim=-1, keepdim=True)
    g2 = g2 - (r1.conj() * g2).sum(-1, keepdim=True) * r1
    r2 = g2 / torch.linalg.vector_norm(g2, dim=-1, keepdim=True)
    r3 = torch.linalg.cross(r1, r2).conj()
    lx, ly, lz, lt = dims
    return torch.stack([r1, r2, r3], dim=-2).reshape(lt, lz, ly, lx, 4, 3, 3).contiguous()


def links_unit(dims, device="cpu") -> torch.Tensor:
    lx, ly, lz, lt = dims
    u = torch.zeros((lt, lz, ly, lx, 4, 3, 3), dtype=torch.complex128, device=device)
    for a in range(3):
        u[..., a, a] = 1.0
    return u


def su3_site_field(dims, seed: int, device="cpu") -> torch.Tensor:
    """Random g(x) in SU(3) per site (stream 3) -> [t][z][y][x][3][3]."""
    v = volume(dims)
    idx = torch.arange(v, dtype=torch.int64, device=device)
    g = normals(seed, STREAM_GAUGE_TRANSFORM, idx, 12)
    g1 = torch.complex(g[:, 0:3], g[:, 3:6])
    g2 = torch.complex(g[:, 6:9], g[:, 9:12])
    r1 = g1 / torch.linalg.vector_norm(g1, dim=-1, keepdim=True)
    g2 = g2 - (r1.conj() * g2).sum(-1, keepdim=True) * r1
    r2 = g2 / torch.linalg.vector_norm(g2, dim=-1, keepdim=True)
    r3 = torch.linalg.cross(r1, r2).conj()
    lx, ly, lz, lt = dims
    return torch.stack([r1, r2, r3], dim=-2).reshape(lt, lz, ly, lx, 3, 3).contiguous()


def gauge_transform_links(u: torch.Tensor, g: torch.Tensor) -> torch.Tensor:
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger (periodic shift; index bookkeeping only)."""
    out = torch.empty_like(u)
    axis = {0: 3, 1: 2, 2: 1, 3: 0}  # mu -> tensor axis of [t][z][y][x]
    for mu in range(4):
        g_fwd = torch.roll(g, shifts=-1, dims=axis[mu])
        out[..., mu, :, :] = g @ u[..., mu, :, :] @ g_fwd.conj().transpose(-1, -2)
    return out


def gauge_transform_spinor(psi: torch.Tensor, g: torch.Tensor) -> torch.Tensor:
    return torch.einsum("tzyxab,tzyxsb->tzyxsa", g, psi)


def source_gaussian(dims, seed: int, device="cpu") -> torch.Tensor:
    """Complex Gaussian on all 24*V reals (BJ:c0, c2, c4)."""
    v = volume(dims)
    idx = torch.arange(v, dtype=torch.int64, device=device)
    g = normals(seed, STREAM_SOURCE, idx, 24)
    lx, ly, lz, lt = dims
    return torch.complex(g[:, 0:12], g[:, 12:24]).reshape(lt, lz, ly, lx, 4, 3).contiguous()


def source_point(dims, spin: int, colour: int, device="cpu") -> torch.Tensor:
    """Unit point source at the origin (BJ:c3: one per spin-colour component)."""
    lx, ly, lz, lt = dims
    psi = torch.zeros((lt, lz, ly, lx, 4, 3), dtype=torch.complex128, device=device)
    psi[0, 0, 0, 0, spin, colour] = 1.0
    return psi


def source_smeared(dims, u: torch.Tensor, alpha: float = 0.7, sweeps: int = 35,
                   spin: int = 0, colour: int = 0) -> torch.Tensor:
    """Gauge-covariant Gaussian smearing of a point source on time-slice 0 (BJ:c1).

    psi <- (1-alpha) psi + (alpha/6) sum_{j=x,y,z} [U_j(x) psi(x+j) + U_j(x-j)^dagger psi(x-j)],
    `sweeps` times, then unit L2 norm.  Only the right-hand side of a solve depends on this.
    """
    psi = source_point(dims, spin, colour, device=u.device)
    sl = psi[0]  # [z][y][x][s][c] on t = 0
    us = u[0]
    axis = {0: 2, 1: 1, 2: 0}
    for _ in range(sweeps):
        acc = torch.zeros_like(sl)
        for j in range(3):
            uj = us[..., j, :, :]
            fwd = torch.roll(sl, shifts=-1, dims=axis[j])
            acc = acc + torch.einsum("zyxab,zyxsb->zyxsa", uj, fwd)
            ub = torch.roll(uj, shifts=1, dims=axis[j])
            bwd = torch.roll(sl, shifts=1, dims=axis[j])
            acc = acc + torch.einsum("zyxba,zyxsb->zyxsa", ub.conj(), bwd)
        sl = (1.0 - alpha) * sl + (alpha / 6.0) * acc
    psi[0] = sl
    return psi / torch.linalg.vector_norm(psi)


def plaquette(u: torch.Tensor) -> float:
    """Average Re tr plaquette / 3 (a diagnostic of the generated field, quoted in DESIGN.md)."""
    axis = {0: 3, 1: 2, 2: 1, 3: 0}
    tot = 0.0
    n = 0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            umu = u[..., mu, :, :]
            unu = u[..., nu, :, :]
            unu_f = torch.roll(unu, shifts=-1, dims=axis[mu])
            umu_f = torch.roll(umu, shifts=-1, dims=axis[nu])
            p = umu @ unu_f @ umu_f.conj().transpose(-1, -2) @ unu.conj().transpose(-1, -2)
            tot += torch.einsum("...ii->...", p).real.mean().item() / 3.0
            n += 1
    return tot / n


# BASELINE.json configs[K]: (dims, link recipe, eps, kappa, csw, source recipe)
CONFIGS = {
    0: dict(dims=(4, 4, 4, 4), links="haar", eps=None, kappa=0.12, csw=1.0, source="gaussian"),
    1: dict(dims=(16, 16, 16, 32), links="smooth", eps=0.3, kappa=0.125, csw=1.0, source="smeared"),
    2: dict(dims=(32, 32, 32, 64), links="smooth", eps=0.3, kappa=0.1245, csw=1.0, source="gaussian"),
    3: dict(dims=(48, 48, 48, 96), links="smooth", eps=0.4, kappa=0.1248, csw=1.2, source="point"),
    4: dict(dims=(64, 64, 64, 128), links="smooth", eps=0.3, kappa=0.1247, csw=1.0, source="gaussian"),
}
BC = (1, 1, 1, -1)


def config_seed_links(k: int) -> int:
    return 20230200 + k


def config_seed_source(k: int) -> int:
    return 850 + k


def make_links(k: int, dims=None, device="cpu") -> torch.Tensor:
    """Links of config K, optionally on other extents (same distribution, same seed)."""
    c = CONFIGS[k]
    dims = tuple(dims or c["dims"])
    if c["links"] == "haar":
        return links_haar(dims, config_seed_links(k), device=device)
    return links_smooth(dims, c["eps"], config_seed_links(k), device=device)


def make_source(k: int, dims=None, u: torch.Tensor | None = None, device="cpu") -> torch.Tensor:
    c = CONFIGS[k]
    dims = tuple(dims or c["dims"])
    if c["source"] == "gaussian":
        return source_gaussian(dims, config_seed_source(k), device=device)
    if c["source"] == "smeared":
        if u is None:
            raise ValueError("smeared source needs the links")
        return source_smeared(dims, u)
    return source_point(dims, 0, 0, device=device)
