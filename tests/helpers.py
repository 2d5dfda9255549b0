"""Test-side helpers that are independent of both the oracle and the CUDA path."""
import itertools

import numpy as np


def dense_from_eq3(nx, ny, nz, h, eps_x, eps_y, eps_z, kbar2, periodic=False):
    """Dense A assembled row by row straight from PAPER.md Eq. 3 (lines 50-62), tiny grids only.

    Each of the six bracketed terms -h^-2 eps_f [phi(nbr) - phi(c)] contributes +eps_f/h^2 to the
    diagonal and, when the neighbour is an unknown (not a ghost node), -eps_f/h^2 to its column.
    """
    n = nx * ny * nz
    A = np.zeros((n, n))
    idx = lambda i, j, k: (k * ny + j) * nx + i
    for k, j, i in itertools.product(range(nz), range(ny), range(nx)):
        c = idx(i, j, k)
        faces = [
            (eps_x[k, j, i], (i - 1, j, k)), (eps_x[k, j, i + 1], (i + 1, j, k)),
            (eps_y[k, j, i], (i, j - 1, k)), (eps_y[k, j + 1, i], (i, j + 1, k)),
            (eps_z[k, j, i], (i, j, k - 1)), (eps_z[k + 1, j, i], (i, j, k + 1)),
        ]
        for e, (a, b_, c_) in faces:
            A[c, c] += e / h ** 2
            if 0 <= a < nx and 0 <= b_ < ny and 0 <= c_ < nz:
                A[c, idx(a, b_, c_)] -= e / h ** 2
            elif periodic:      # the neighbour across the box face is the node on the other side
                A[c, idx(a % nx, b_ % ny, c_ % nz)] -= e / h ** 2
        A[c, c] += kbar2[k, j, i]
    return A


def sine_mode(nx, ny, nz, p, q, r):
    """Discrete Dirichlet eigenvector sin(p pi (i+1)/(nx+1)) sin(q ..) sin(r ..), shape [nz][ny][nx]."""
    sx = np.sin(p * np.pi * (np.arange(nx) + 1) / (nx + 1))
    sy = np.sin(q * np.pi * (np.arange(ny) + 1) / (ny + 1))
    sz = np.sin(r * np.pi * (np.arange(nz) + 1) / (nz + 1))
    return sz[:, None, None] * sy[None, :, None] * sx[None, None, :]


def sine_eigenvalue(nx, ny, nz, h, eps, k2, p, q, r):
    """lambda_pqr = (4 eps/h^2)[sin^2(p pi/2(nx+1)) + sin^2(q pi/2(ny+1)) + sin^2(r pi/2(nz+1))] + k2."""
    s = (np.sin(p * np.pi / (2 * (nx + 1))) ** 2 + np.sin(q * np.pi / (2 * (ny + 1))) ** 2
         + np.sin(r * np.pi / (2 * (nz + 1))) ** 2)
    return 4.0 * eps / h ** 2 * s + k2


def uniform_eps(nx, ny, nz, eps):
    return (np.full((nz, ny, nx + 1), float(eps)), np.full((nz, ny + 1, nx), float(eps)),
            np.full((nz + 1, ny, nx), float(eps)))


def pack_bc(nx, ny, nz, h, fn):
    """Ghost values fn(x,y,z) in the bc packing order x-,x+,y-,y+,z-,z+ (node (i,j,k) at (ih,jh,kh))."""
    x, y, z = np.arange(nx) * h, np.arange(ny) * h, np.arange(nz) * h
    out = []
    for xg in (-h, nx * h):
        Z, Y = np.meshgrid(z, y, indexing="ij")
        out.append(fn(np.full_like(Z, xg), Y, Z).ravel())
    for yg in (-h, ny * h):
        Z, X = np.meshgrid(z, x, indexing="ij")
        out.append(fn(X, np.full_like(Z, yg), Z).ravel())
    for zg in (-h, nz * h):
        Y, X = np.meshgrid(y, x, indexing="ij")
        out.append(fn(X, Y, np.full_like(Y, zg)).ravel())
    return np.concatenate(out)
