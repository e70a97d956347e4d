"""Shared test helpers (no method arithmetic of the CUDA path, no oracle arithmetic)."""
import numpy as np
import torch

U = 1.1e-16          # north_star writes the Q tolerance as 10 * kappa * n * 1.1e-16


def to_np(T):
    """(n, m) C-contiguous tensor holding a column-major m x n matrix -> m x n numpy (Fortran order)."""
    return T.detach().cpu().numpy().T


def colmajor_to_dev(M, device="cuda"):
    """m x n numpy matrix -> (n, m) C-contiguous float64 tensor on `device` (column-major m x n)."""
    return torch.from_numpy(np.ascontiguousarray(np.asarray(M, dtype=np.float64).T)).to(device)


def draw_to_dev(signs, idx, device="cuda"):
    s = torch.from_numpy(np.ascontiguousarray(signs).view(np.int64).copy()).to(device)
    i = torch.from_numpy(np.ascontiguousarray(idx, dtype=np.int64).copy()).to(device)
    return s, i


def gpu_orth_error_fro(QT, block=1024):
    """||I - Q^T Q||_F on the device with block + pairwise-tree summation over rows (a plain long
    accumulation adds ~1e-14 of its own at m = 2^20).  Test infrastructure."""
    n, m = QT.shape
    nb = (m + block - 1) // block
    if nb * block != m:
        pad = torch.zeros((n, nb * block - m), dtype=QT.dtype, device=QT.device)
        QT = torch.cat([QT, pad], dim=1)
    G = None
    step = max(1, (1 << 28) // (n * n))                  # bound the temporary to ~2 GiB
    parts = []
    for b0 in range(0, nb, step):
        b1 = min(nb, b0 + step)
        Qb = QT[:, b0 * block:b1 * block].reshape(n, b1 - b0, block).permute(1, 0, 2)   # (nb, n, block)
        P = torch.bmm(Qb, Qb.transpose(1, 2))
        while P.shape[0] > 1:
            if P.shape[0] % 2:
                P = torch.cat([P, torch.zeros_like(P[:1])], dim=0)
            P = P[0::2] + P[1::2]
        parts.append(P[0])
    G = parts[0]
    for Pk in parts[1:]:
        G = G + Pk
    E = G - torch.eye(n, dtype=QT.dtype, device=QT.device)
    return float(torch.linalg.norm(E))


def gpu_residual_fro(AT, QT, Rt, chunk=1 << 18):
    """||A - Q R||_F / ||A||_F on the device; Rt is the (n,n) tensor holding column-major R."""
    n, m = AT.shape
    num = torch.zeros((), dtype=torch.float64, device=AT.device)
    den = torch.zeros((), dtype=torch.float64, device=AT.device)
    for c0 in range(0, m, chunk):
        c1 = min(m, c0 + chunk)
        D = AT[:, c0:c1] - Rt @ QT[:, c0:c1]                  # A^T - R^T Q^T
        num += (D * D).sum()
        den += (AT[:, c0:c1] ** 2).sum()
    return float(torch.sqrt(num / den))
