"""Closed forms used as pins.  Independent of oracle/ and of the CUDA path (test-only helpers)."""
import numpy as np


def wu_mesh_reff(M, N, r, s, x1, y1, x2, y2):
    """PAPER.md:49-52, Eq. (3) (Wu 2004, free-boundary M x N resistor mesh), reading G1:
    exactly as printed with 0-based x in [0, M-1], y in [0, N-1]; segments along x have resistance
    r, along y resistance s; theta_m = m*pi/M, phi_n = n*pi/N."""
    m = np.arange(1, M)[:, None]
    n = np.arange(1, N)[None, :]
    th = m * np.pi / M
    ph = n * np.pi / N
    num = (np.cos((x1 + 0.5) * th) * np.cos((y1 + 0.5) * ph)
           - np.cos((x2 + 0.5) * th) * np.cos((y2 + 0.5) * ph)) ** 2
    den = (1.0 - np.cos(th)) / r + (1.0 - np.cos(ph)) / s
    return (r / N) * abs(int(x1) - int(x2)) + (s / M) * abs(int(y1) - int(y2)) + 2.0 / (M * N) * float((num / den).sum())


def _dct_mode(L, k, j):
    return np.sqrt((1.0 if k == 0 else 2.0) / L) * np.cos((j + 0.5) * k * np.pi / L)


def product_graph_reff(nx, ny, nz, rx, ry, rz, u, v):
    """Two-point resistance on the path-graph product P_nx x P_ny x P_nz with uniform resistances
    rx, ry, rz per direction: R = sum_{(a,b,c) != 0} (phi_abc(u) - phi_abc(v))^2 / lambda_abc with
    orthonormal DCT-II modes, lambda = sum_dir (2 - 2 cos(k pi / L)) / r_dir.  u, v = (x, y, z)."""
    tot = 0.0
    for a in range(nx):
        for b in range(ny):
            for c in range(nz):
                if a == b == c == 0:
                    continue
                lam = ((2 - 2 * np.cos(a * np.pi / nx)) / rx + (2 - 2 * np.cos(b * np.pi / ny)) / ry
                       + (2 - 2 * np.cos(c * np.pi / nz)) / rz)
                pu = _dct_mode(nx, a, u[0]) * _dct_mode(ny, b, u[1]) * _dct_mode(nz, c, u[2])
                pv = _dct_mode(nx, a, v[0]) * _dct_mode(ny, b, v[1]) * _dct_mode(nz, c, v[2])
                tot += (pu - pv) ** 2 / lam
    return float(tot)
