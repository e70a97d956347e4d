"""Seeded synthetic inputs for MRCQR tests, smoke() and bench.py.

This module serves BOTH the CUDA path and the CPU oracle with the same A buffer and holds none of
the method's arithmetic (no draw of D/S, no transform, no factorization).  Recipe (DESIGN.md
"Input recipe", BASELINE.json `configs`):

    A = G * diag(sigma) * V^T,   G: m x n i.i.d. N(0,1) (seed_G),  V: Q-factor of an n x n
    Gaussian (seed_V),  sigma_i = 10^(-e * i / (n-1)), i = 0..n-1   (kappa(A) ~ 10^e).

The paper's own test matrices (eq. (3)) are A = U Sigma V^T with orthonormal
U, V from QR of uniform[-1,1] matrices and sigma_i = kappa^(1/2 - i/(n-1)); `make_paper_eq3`
builds those for the stability sweep.

Random numbers: uniform doubles u_k = (X(k) >> 11) * 2^-53 from the k-th output X(k) of a
splitmix64 stream (counter-based, so any slice can be generated on any device), Box-Muller
pairs, filled in column-major element order.  Implemented with torch int64 wrap-around
arithmetic so the same code runs on CPU and on the GPU; values are reproducible per device type
(libm vs CUDA log/cos differ in the last bits), which is all parity needs because both sides
always consume the very same buffer.

Returned matrices are torch float64 tensors of shape (n, m), C-contiguous: that IS the m x n
matrix in column-major order with lda = m (column j = row j of the tensor).
"""
import math

import torch

_GAMMA = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


def _s64(x):
    """python int (mod 2^64) -> signed 64-bit python int"""
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z, k):
    """logical shift right of an int64 tensor"""
    return (z >> k) & ((1 << (64 - k)) - 1)


def splitmix64_block(seed, start, count, device="cpu"):
    """int64 tensor holding the bit patterns of X(start) .. X(start+count-1)."""
    k = torch.arange(start + 1, start + count + 1, dtype=torch.int64, device=device)
    z = k * _s64(_GAMMA) + _s64(seed)
    z = (z ^ _lsr(z, 30)) * _s64(_M1)
    z = (z ^ _lsr(z, 27)) * _s64(_M2)
    return z ^ _lsr(z, 31)


def uniform_block(seed, start, count, device="cpu"):
    """float64 uniforms in [0,1): (X(k) >> 11) * 2^-53."""
    z = splitmix64_block(seed, start, count, device)
    return _lsr(z, 11).to(torch.float64) * (2.0 ** -53)


def normal_block(seed, start, count, device="cpu"):
    """`count` N(0,1) values for linear element indices start .. start+count-1 (start even).
    Element e uses the Box-Muller pair p = e // 2 built from u_{2p}, u_{2p+1}:
    even e -> r cos(2 pi u_{2p+1}), odd e -> r sin(2 pi u_{2p+1}), r = sqrt(-2 ln(1 - u_{2p}))."""
    assert start % 2 == 0
    npair = (count + 1) // 2
    u = uniform_block(seed, start, 2 * npair, device).view(npair, 2)
    r = torch.sqrt(-2.0 * torch.log1p(-u[:, 0]))
    ang = (2.0 * math.pi) * u[:, 1]
    z = torch.stack((r * torch.cos(ang), r * torch.sin(ang)), dim=1).reshape(-1)
    return z[:count]


def gaussian_colmajor(m, n, seed, device="cpu", chunk=1 << 24):
    """(n, m) tensor = column-major m x n matrix of N(0,1), element order column by column."""
    out = torch.empty((n, m), dtype=torch.float64, device=device)
    flat = out.view(-1)
    total = m * n
    for e0 in range(0, total, chunk):                            # chunk is even
        e1 = min(total, e0 + chunk)
        flat[e0:e1] = normal_block(seed, e0, e1 - e0, device)
    return out


def sigma_logspaced(n, exponent, device="cpu"):
    """sigma_i = 10^(-exponent * i/(n-1)), i = 0..n-1 (sigma = [1] for n = 1)."""
    if n == 1:
        return torch.ones(1, dtype=torch.float64, device=device)
    i = torch.arange(n, dtype=torch.float64, device=device)
    return torch.pow(torch.tensor(10.0, dtype=torch.float64, device=device), -exponent * i / (n - 1))


def orthogonal_factor(n, seed, device="cpu"):
    """V = Q-factor of an n x n Gaussian (always computed on the CPU for reproducibility)."""
    Gm = gaussian_colmajor(n, n, seed, "cpu").t().contiguous()
    V, _ = torch.linalg.qr(Gm)
    return V.to(device)


def make_A(m, n, exponent, seed_G, seed_V, device="cpu"):
    """BASELINE.json recipe: A = G diag(sigma) V^T.  Returns the (n, m) column-major tensor."""
    GT = gaussian_colmajor(m, n, seed_G, device)                 # (n, m): GT[j, r] = G[r, j]
    sig = sigma_logspaced(n, exponent, device)
    V = orthogonal_factor(n, seed_V, device)                     # (n, n)
    # A^T = V diag(sigma) G^T
    AT = (V * sig.unsqueeze(0)) @ GT
    return AT.contiguous()


def make_paper_eq3(m, n, kappa, seed_U, seed_V, device="cpu"):
    """Paper eq. (3): A = U Sigma V^T, U (m x n) and V (n x n) with orthonormal
    columns from QR of uniform[-1,1] matrices, sigma_i = kappa^(1/2 - i/(n-1)).  Returns (n, m)."""
    UT = (2.0 * uniform_block(seed_U, 0, m * n, device) - 1.0).view(n, m)
    U, _ = torch.linalg.qr(UT.t())                               # (m, n)
    Vm = (2.0 * uniform_block(seed_V, 0, n * n, "cpu") - 1.0).view(n, n).t().contiguous()
    V, _ = torch.linalg.qr(Vm)
    V = V.to(device)
    i = torch.arange(n, dtype=torch.float64, device=device)
    e = 0.5 - i / max(n - 1, 1)
    sig = torch.pow(torch.tensor(float(kappa), dtype=torch.float64, device=device), e)
    AT = (V * sig.unsqueeze(0)) @ U.t()
    return AT.contiguous()


# BASELINE.json `configs`.  exponent e: sigma from 1 to 10^-e.
CONFIGS = {
    "C0": dict(m=4096, n=16, s=32, prec=32, exponent=6, seed_G=0, seed_V=1, seed_draw=2),
    "C1": dict(m=1 << 20, n=64, s=128, prec=16, exponent=4, seed_G=10, seed_V=11, seed_draw=12),
    "C2": dict(m=1 << 20, n=128, s=256, prec=32, exponent=8, seed_G=20, seed_V=21, seed_draw=22),
    "C3": dict(m=1 << 21, n=256, s=512, prec=64, exponent=15, seed_G=30, seed_V=31, seed_draw=32),
}


def sweep_config(n, prec):
    """configs[4]: column sweep at m = 2^21, kappa ~ 1e4, s = 2n, seeds 40+n (G), +1 (V), +2 (draw)."""
    return dict(m=1 << 21, n=n, s=2 * n, prec=prec, exponent=4,
                seed_G=40 + n, seed_V=41 + n, seed_draw=42 + n)


def make_config(cfg, device="cpu"):
    return make_A(cfg["m"], cfg["n"], cfg["exponent"], cfg["seed_G"], cfg["seed_V"], device)
