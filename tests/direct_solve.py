"""Separable direct solver for LAYERED conductivity -- a pin for the oracle, not the oracle.

Textbook fast Poisson solve: with kappa depending on z only and adiabatic (Neumann) sides, the
lateral part of eq. (4) is kx(z) * L_x + ky(z) * L_y with L the 1-D Neumann
Laplacian, diagonalised by the DCT-II with eigenvalues 2 - 2 cos(pi m / n).  What is left is one
tridiagonal system of size nz per lateral mode (m_x, m_y), solved by the Thomas algorithm.
Shares no code with oracle/ or with the CUDA path; O(N log N), exact to round-off.
"""
import numpy as np
from scipy.fft import dctn, idctn


def solve_layered(nx, ny, nz, dx, dy, dz, kappa_layer, h_top, b, cvol=None, dt=0.0):
    dz = np.asarray(dz, dtype=np.float64)
    k = np.asarray(kappa_layer, dtype=np.float64)
    gx = k * dy * dz / dx                      # lateral conductance per layer (equal kappa both sides)
    gy = k * dx * dz / dy
    gz = dx * dy / (dz[:-1] / (2 * k[:-1]) + dz[1:] / (2 * k[1:]))   # between z and z+1
    lam_x = 2.0 - 2.0 * np.cos(np.pi * np.arange(nx) / nx)
    lam_y = 2.0 - 2.0 * np.cos(np.pi * np.arange(ny) / ny)
    bh = dctn(np.asarray(b, dtype=np.float64).reshape(nz, ny, nx), type=2, axes=(1, 2), norm="ortho")
    # tridiagonal in z for every (my, mx)
    diag = np.empty((nz, ny, nx))
    for z in range(nz):
        d = gx[z] * lam_x[None, :] + gy[z] * lam_y[:, None]
        if z > 0:
            d = d + gz[z - 1]
        if z + 1 < nz:
            d = d + gz[z]
        if z == nz - 1:
            d = d + h_top * dx * dy
        if cvol is not None and dt > 0:
            d = d + cvol[z] * dx * dy * dz[z] / dt
        diag[z] = d
    # Thomas: sub/super diagonal = -gz
    cp = np.empty((nz, ny, nx))
    dp = np.empty((nz, ny, nx))
    cp[0] = (-gz[0] / diag[0]) if nz > 1 else 0.0
    dp[0] = bh[0] / diag[0]
    for z in range(1, nz):
        den = diag[z] + gz[z - 1] * cp[z - 1]
        cp[z] = (-gz[z] / den) if z + 1 < nz else 0.0
        dp[z] = (bh[z] + gz[z - 1] * dp[z - 1]) / den
    xh = np.empty((nz, ny, nx))
    xh[nz - 1] = dp[nz - 1]
    for z in range(nz - 2, -1, -1):
        xh[z] = dp[z] - cp[z] * xh[z + 1]
    return idctn(xh, type=2, axes=(1, 2), norm="ortho").reshape(-1)
