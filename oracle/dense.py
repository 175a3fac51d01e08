"""Dense brute-force matrices from the closed forms, numpy fp64.  TEST INFRASTRUCTURE ONLY.

Independent of cp4d_ref.c (no call into it): the static Joseph matrix is typed from the closed form
A_k[b; iy,ix] = Lambda((x c + y s - s_b)/a_k)/a_k, Lambda(u) = max(0, 1-|u|)  (reading R3),
K1 = sum_j Phi[j,k] (x) A_k  (Eq. 9), K2 from Kronecker products of 1D forward
differences (reading R4).  Sizes: only for tiny grids (<= 32x32).
"""
import numpy as np


def joseph_matrix(n, nd, theta):
    c, s = np.cos(theta), np.sin(theta)
    a = max(abs(c), abs(s))
    x = np.arange(n) - (n - 1) / 2.0
    X, Y = np.meshgrid(x, x, indexing="xy")            # X[iy,ix] = x_ix, Y[iy,ix] = y_iy
    sb = np.arange(nd) - (nd - 1) / 2.0
    u = (X[None] * c + Y[None] * s - sb[:, None, None]) / a
    return (np.maximum(0.0, 1.0 - np.abs(u)) / a).reshape(nd, n * n)


def dense_K1(n, nz, nd, n_angles, n_half_rot, m, phi):
    """K1 as a (nz*n_angles*nd) x (nz*n*n*m) matrix for layouts g[z][k][b], f[z][iy][ix][j]."""
    n0 = n_angles // n_half_rot
    S1, V1 = n_angles * nd, n * n * m
    K = np.zeros((nz * S1, nz * V1))
    for k in range(n_angles):
        A = joseph_matrix(n, nd, k * np.pi / n0)        # (nd, n*n)
        blk = np.kron(A, phi[:, k][None, :])            # columns ordered (iy,ix) major, j minor
        for z in range(nz):
            K[z * S1 + k * nd: z * S1 + (k + 1) * nd, z * V1:(z + 1) * V1] = blk
    return K


def _fd(n):
    D = np.zeros((n, n))
    for i in range(n - 1):
        D[i, i], D[i, i + 1] = -1.0, 1.0
    return D


def dense_K2(n, nz, m, lambda2):
    """K2 = grad_{lambda2} as a (4V x V) matrix, component-major (x, y, z, t), f[z][iy][ix][j]."""
    Iz, Iy, Ix, Ij = np.eye(nz), np.eye(n), np.eye(n), np.eye(m)
    k4 = lambda a, b, c, d: np.kron(np.kron(np.kron(a, b), c), d)
    return np.vstack([k4(Iz, Iy, _fd(n), Ij), k4(Iz, _fd(n), Ix, Ij), k4(_fd(nz), Iy, Ix, Ij),
                      lambda2 * k4(Iz, Iy, Ix, _fd(m))])
