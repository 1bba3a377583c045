"""Seeded synthetic inputs for the generalized eigenproblem HC = eps SC (Eq. 2).

This module is shared by the CUDA path's tests/bench and by the oracle's tests.  It holds NONE of
the method's arithmetic (no Cholesky, inversion, products or eigensolves): it only materialises the
input matrices H, S and dense right-hand sides, from the recipe in BASELINE.json `configs` as read in
SURVEY.md section 8(d) / DESIGN.md "Input recipe".

The paper measures on unspecified FHI-aims matrices at N = 40960 (Table 1 caption); no
dataset is named.  These inputs stand in for them: an overlap matrix of unit-width s-type Gaussians
centred at random points (dense, SPD, cond ~ 1e4) and a Hamiltonian roughly proportional to -S with
a noisy scale and an on-site term.

Storage convention: matrices handed to the C ABI are COLUMN-MAJOR with
leading dimension = number of rows.  `colmajor_empty(rows, cols)` returns a torch tensor of logical
shape (rows, cols) and strides (1, rows), so `t.data_ptr()` is the column-major buffer and ordinary
torch indexing `t[i, j]` addresses A(i, j).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import torch

# mean number of neighbours within distance 2 targeted by the box scaling (BASELINE.json configs[1])
_NEIGHBOURS = 20.0
_RHO = _NEIGHBOURS / (4.0 * math.pi * 2.0 ** 3 / 3.0)  # points per unit volume = 0.5968
BASE_SEED = 20250204


@dataclass(frozen=True)
class Config:
    index: int
    N: int
    nev: int
    complex: bool
    box: float  # edge length L of the cube the points are drawn in

    @property
    def name(self) -> str:
        return f"cfg{self.index}_N{self.N}_{'c128' if self.complex else 'f64'}_nev{self.nev}"

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index


def scaled_box(N: int) -> float:
    """Cube edge that keeps ~20 neighbours within distance 2 (BASELINE.json configs[1])."""
    return (N / _RHO) ** (1.0 / 3.0)


# BASELINE.json `configs`, in order.  Config 3 ("built as in config 0" at N=8192) is read as: same
# recipe, box scaled like configs 1-4 (reading Q15: a 6x6x6 box with 8192 points would
# give cond(S) ~ 1e6, contradicting "cond <= 1e4").
CONFIGS = (
    Config(0, 256, 256, False, 6.0),
    Config(1, 4096, 1024, False, scaled_box(4096)),
    Config(2, 16384, 4096, False, scaled_box(16384)),
    Config(3, 8192, 2048, True, scaled_box(8192)),
    Config(4, 32768, 8192, False, scaled_box(32768)),
)

PHASE_K = 0.7  # config 3: exp(i k (x_i - x_j))


def colmajor_empty(rows: int, cols: int, dtype=torch.float64, device="cpu") -> torch.Tensor:
    """Logical (rows, cols) tensor whose storage is column-major, ld = rows."""
    return torch.empty((cols, rows), dtype=dtype, device=device).t()


def colmajor_zeros(rows: int, cols: int, dtype=torch.float64, device="cpu") -> torch.Tensor:
    return torch.zeros((cols, rows), dtype=dtype, device=device).t()


def to_colmajor(a: torch.Tensor) -> torch.Tensor:
    """Copy of a 2-D tensor with column-major storage (strides (1, rows))."""
    out = colmajor_empty(a.shape[0], a.shape[1], dtype=a.dtype, device=a.device)
    out.copy_(a)
    return out


def is_colmajor(a: torch.Tensor) -> bool:
    return a.dim() == 2 and (a.shape[0] <= 1 or a.stride(0) == 1) and \
        (a.shape[1] <= 1 or a.stride(1) == a.shape[0])


def _generator(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def points(N: int, box: float, gen: torch.Generator, device="cpu") -> torch.Tensor:
    """N points i.i.d. uniform in [0, box]^3."""
    return torch.rand((N, 3), dtype=torch.float64, device=device, generator=gen) * box


def mirror_upper_(A: torch.Tensor, chunk: int = 4096) -> torch.Tensor:
    """In place: the strictly-lower triangle becomes the (conjugate) transpose of the strictly-upper one;
    a complex diagonal is made exactly real.  Block by block, to bound temporaries."""
    N = A.shape[0]
    for i0 in range(0, N, chunk):
        i1 = min(N, i0 + chunk)
        blk = A[i0:i1, i0:i1]
        up = torch.triu(blk, 1)
        dg = torch.diag(torch.diagonal(blk).real.to(A.dtype))
        blk.copy_(up + up.conj().t() + dg)
        if i1 < N:
            A[i1:, i0:i1] = A[i0:i1, i1:].conj().t()
    return A


def overlap(r: torch.Tensor, jitter: float = 1e-3, chunk: int = 2048) -> torch.Tensor:
    """S_ij = exp(-0.5 |r_i - r_j|^2) + jitter * delta_ij, column-major, exactly symmetric.

    The squared distances are bitwise symmetric (explicit differences, not |a|^2+|b|^2-2ab), but a
    vectorised exp need not return the same bits for the same argument at two places of a tensor
    (seen on the GPU box's host CPU: S_ij and S_ji a few 1e-10 apart in the first call of a fresh
    process), so the lower triangle is mirrored from the upper one explicitly.
    """
    N = r.shape[0]
    S = colmajor_empty(N, N, device=r.device)
    for i0 in range(0, N, chunk):
        i1 = min(N, i0 + chunk)
        d2 = torch.zeros((i1 - i0, N), dtype=torch.float64, device=r.device)
        for c in range(3):
            diff = r[i0:i1, c].unsqueeze(1) - r[:, c].unsqueeze(0)
            d2 += diff * diff
        S[i0:i1, :] = torch.exp(-0.5 * d2)
    mirror_upper_(S)
    S.diagonal().add_(jitter)
    return S


def hamiltonian(S: torch.Tensor, gen: torch.Generator, chunk: int = 4096) -> torch.Tensor:
    """H_ij = -S_ij (1 + 0.1 g_ij) with g symmetric standard normal, plus diag uniform in [-2, 0]."""
    N = S.shape[0]
    dev = S.device
    H = colmajor_empty(N, N, device=dev)
    # g: draw a full matrix row-chunk by row-chunk, keep the upper triangle (incl. diagonal), mirror.
    for i0 in range(0, N, chunk):
        i1 = min(N, i0 + chunk)
        g = torch.randn((i1 - i0, N), dtype=torch.float64, device=dev, generator=gen)
        H[i0:i1, :] = g
    d = torch.rand((N,), dtype=torch.float64, device=dev, generator=gen) * 2.0 - 2.0
    # mirror upper -> lower, chunked to bound temporaries
    for i0 in range(0, N, chunk):
        i1 = min(N, i0 + chunk)
        blk = H[i0:i1, i0:i1]
        blk.copy_(torch.triu(blk) + torch.triu(blk, 1).t())
        if i1 < N:
            H[i1:, i0:i1] = H[i0:i1, i1:].t()
    H.mul_(0.1).add_(1.0).mul_(S).neg_()
    H.diagonal().add_(d)
    # step 3 reads one triangle of H, the oracle the whole matrix: the two must agree bit for bit
    return mirror_upper_(H)


def phase_factor(x: torch.Tensor, k: float = PHASE_K) -> torch.Tensor:
    """P_ij = exp(i k (x_i - x_j)), exactly Hermitian (lower triangle = conj of upper), column-major."""
    N = x.shape[0]
    ang = k * (x.unsqueeze(1) - x.unsqueeze(0))
    P = torch.complex(torch.cos(ang), torch.sin(ang))
    up = torch.triu(P, 1)
    P = up + up.conj().t() + torch.eye(N, dtype=torch.complex128, device=x.device)
    return to_colmajor(P)


@dataclass
class Pencil:
    N: int
    complex: bool
    H: torch.Tensor  # column-major N x N, symmetric / Hermitian, both triangles filled
    S: torch.Tensor  # column-major N x N, SPD / HPD
    r: torch.Tensor  # the points (N, 3)


def make_pencil(N: int, box: float, seed: int, complex: bool = False, device="cpu",
                jitter: float = 1e-3) -> Pencil:
    """The BASELINE.json recipe.  Draw order: r (N x 3), then g (row chunks), then d (N)."""
    gen = _generator(seed, device)
    r = points(N, box, gen, device)
    S = overlap(r, jitter)
    H = hamiltonian(S, gen)
    if complex:
        P = phase_factor(r[:, 0])
        S = to_colmajor(S.to(torch.complex128) * P)
        H = to_colmajor(H.to(torch.complex128) * P)
        # diagonals are exactly real by construction (P_ii = 1)
        mirror_upper_(S)
        mirror_upper_(H)
    if N <= 4096 and not (torch.equal(H, H.conj().t()) and torch.equal(S, S.conj().t())):
        raise RuntimeError("workloads.make_pencil: H or S is not exactly Hermitian")
    return Pencil(N, complex, H, S, r)


def make_config(cfg: Config | int, device="cpu") -> Pencil:
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    return make_pencil(cfg.N, cfg.box, cfg.seed, cfg.complex, device)


def small_pencil(N: int, seed: int = 1, complex: bool = False, device="cpu") -> Pencil:
    """Recipe at an arbitrary (small / ragged) N for parity tests; config-0 density (box 6 at N=256)."""
    box = 6.0 * (max(N, 1) / 256.0) ** (1.0 / 3.0)
    return make_pencil(N, box, BASE_SEED + 1000 + seed, complex, device)


def dense_rhs(N: int, nev: int, seed: int, complex: bool = False, device="cpu") -> torch.Tensor:
    """Seeded N x nev standard-normal block, column-major: a stand-in C~ for throughput runs and
    back-transform parity (any dense C~ is valid input to C = U^-1 C~)."""
    gen = _generator(BASE_SEED + 5000 + seed, device)
    out = colmajor_empty(N, nev, dtype=torch.complex128 if complex else torch.float64, device=device)
    re = torch.randn((nev, N), dtype=torch.float64, device=device, generator=gen)
    if complex:
        im = torch.randn((nev, N), dtype=torch.float64, device=device, generator=gen)
        out.copy_(torch.complex(re, im).t())
    else:
        out.copy_(re.t())
    return out


def nominal_flops(N: int, nev: int, complex: bool = False) -> dict:
    """Nominal flop counts the metric credits (BASELINE.json north_star): N^3/3 POTRF, N^3/3 TRTRI,
    N^3 transform, N^2 nev back-transform; complex = 4x real-equivalent."""
    f = 4.0 if complex else 1.0
    d = {
        "cholesky": f * N ** 3 / 3.0,
        "invert": f * N ** 3 / 3.0,
        "to_standard": f * float(N) ** 3,
        "backtransform": f * float(N) ** 2 * nev,
    }
    d["total"] = sum(d.values())
    return d
