"""ORACLE for the grid / stencil setup (NEXT row f1) -- test infrastructure, not product code.

The paper's stated next step is "integrated grid stencil setup on GPU".  What is set up is
the input of Eq. 3: the dielectric map "80 solvent / 1 solute" with "the weighted harmonic
average" on boundary-crossing grid edges, the Boltzmann coefficient in the solvent only (the
Stern mask lambda of Eq. 1-2), the grid charges q(i,j,k) of Eq. 3's right-hand side, and the
free-space boundary potentials.  The paper gives no formulas for these; the readings are
DESIGN.md Readings 8-11, 13, 18 (node is solute iff d^2 <= R^2 for some atom; face eps = 2 e1 e2/(e1+e2) of its
two nodes, ghost nodes are solvent; trilinear spreading to the 8 surrounding nodes; rhs = 4 pi q/h^3;
Debye-Hueckel ghost values sum_i q_i exp(-kappa r_i)/(eps_out r_i), kappa^2 = kbar2/eps_out).

Plain numpy / python loops in fp64, one atom or one term at a time, no blocking.  Shares no code with
paper_1704_02745_b200/ or workloads/.  Pins: tests/test_oracle_setup_pins.py.
"""
from __future__ import annotations

import math

import numpy as np


def solute_mask(nx, ny, nz, h, centres, radii):
    """mask[k][j][i] = True iff node (i h, j h, k h) lies within some atom sphere, d^2 <= R^2 (Reading 18)."""
    mask = np.zeros((nz, ny, nx), dtype=bool)
    for (cx, cy, cz), R in zip(np.asarray(centres, float), np.asarray(radii, float)):
        i_lo, i_hi = max(0, math.ceil((cx - R) / h)), min(nx - 1, math.floor((cx + R) / h))
        j_lo, j_hi = max(0, math.ceil((cy - R) / h)), min(ny - 1, math.floor((cy + R) / h))
        k_lo, k_hi = max(0, math.ceil((cz - R) / h)), min(nz - 1, math.floor((cz + R) / h))
        for k in range(k_lo, k_hi + 1):
            dz = k * h - cz
            for j in range(j_lo, j_hi + 1):
                dy = j * h - cy
                for i in range(i_lo, i_hi + 1):
                    dx = i * h - cx
                    if (dz * dz + dy * dy) + dx * dx <= R * R:
                        mask[k, j, i] = True
    return mask


def face_dielectrics(mask, eps_in, eps_out):
    """eps_x [nz][ny][nx+1], eps_y [nz][ny+1][nx], eps_z [nz+1][ny][nx]: harmonic mean of the two nodes a face
    joins; nodes outside the grid (the ghost layer) are solvent (Reading 11)."""
    nz, ny, nx = mask.shape

    def node_eps(k, j, i):
        if 0 <= k < nz and 0 <= j < ny and 0 <= i < nx and mask[k, j, i]:
            return float(eps_in)
        return float(eps_out)

    def hm(a, b):
        return 2.0 * a * b / (a + b)

    eps_x = np.empty((nz, ny, nx + 1))
    eps_y = np.empty((nz, ny + 1, nx))
    eps_z = np.empty((nz + 1, ny, nx))
    for k in range(nz):
        for j in range(ny):
            for f in range(nx + 1):
                eps_x[k, j, f] = hm(node_eps(k, j, f - 1), node_eps(k, j, f))
    for k in range(nz):
        for f in range(ny + 1):
            for i in range(nx):
                eps_y[k, f, i] = hm(node_eps(k, f - 1, i), node_eps(k, f, i))
    for f in range(nz + 1):
        for j in range(ny):
            for i in range(nx):
                eps_z[f, j, i] = hm(node_eps(f - 1, j, i), node_eps(f, j, i))
    return eps_x, eps_y, eps_z


def salt_map(mask, kbar2_solvent):
    """kbar2 on solvent nodes only, 0 inside the solute (Reading 10)."""
    return np.where(mask, 0.0, float(kbar2_solvent))


def grid_charges(nx, ny, nz, h, centres, charges):
    """q(i,j,k) of Eq. 3: every point charge spread trilinearly to its 8 surrounding nodes, atom by atom."""
    q = np.zeros((nz, ny, nx))
    for (cx, cy, cz), qa in zip(np.asarray(centres, float), np.asarray(charges, float)):
        g = (cx / h, cy / h, cz / h)
        base = [min(max(int(math.floor(g[d])), 0), n - 2) for d, n in enumerate((nx, ny, nz))]
        fr = [g[d] - base[d] for d in range(3)]
        for dz in (0, 1):
            wz = fr[2] if dz else 1.0 - fr[2]
            for dy in (0, 1):
                wy = fr[1] if dy else 1.0 - fr[1]
                for dx in (0, 1):
                    wx = fr[0] if dx else 1.0 - fr[0]
                    q[base[2] + dz, base[1] + dy, base[0] + dx] += qa * wz * wy * wx
    return q


def rhs_from_charges(q_node, h):
    """Right-hand side of Eq. 3 in the generator's units (Reading 8): 4 pi q / h^3."""
    return 4.0 * math.pi * q_node / h ** 3


def ghost_positions(nx, ny, nz, h):
    """Ghost-node coordinates in the bc packing order x-, x+ ([nz][ny]), y-, y+ ([nz][nx]), z-, z+ ([ny][nx])."""
    out = []
    for xg in (-h, nx * h):
        out += [(xg, j * h, k * h) for k in range(nz) for j in range(ny)]
    for yg in (-h, ny * h):
        out += [(i * h, yg, k * h) for k in range(nz) for i in range(nx)]
    for zg in (-h, nz * h):
        out += [(i * h, j * h, zg) for j in range(ny) for i in range(nx)]
    return np.array(out, dtype=np.float64)


def debye_huckel_boundary(nx, ny, nz, h, centres, charges, eps_out, kappa):
    """Free-space Dirichlet values (Reading 13): sum_i q_i exp(-kappa r_i) / (eps_out r_i) at every
    ghost node, atoms added in index order."""
    g = ghost_positions(nx, ny, nz, h)
    c = np.asarray(centres, float)
    q = np.asarray(charges, float)
    out = np.zeros(g.shape[0])
    for a in range(c.shape[0]):                       # one atom at a time, all ghost nodes vectorised
        dx, dy, dz = g[:, 0] - c[a, 0], g[:, 1] - c[a, 1], g[:, 2] - c[a, 2]
        r = np.sqrt((dx * dx + dy * dy) + dz * dz)
        out += q[a] * (np.exp(-kappa * r) / r)
    return out / eps_out


def setup(nx, ny, nz, h, centres, radii, charges, eps_in, eps_out, kbar2_solvent):
    """All fields pb_create takes, from atoms: dict(mask, eps_x, eps_y, eps_z, kbar2, rhs, bc)."""
    mask = solute_mask(nx, ny, nz, h, centres, radii)
    eps_x, eps_y, eps_z = face_dielectrics(mask, eps_in, eps_out)
    kappa = math.sqrt(kbar2_solvent / eps_out)
    return dict(mask=mask, eps_x=eps_x, eps_y=eps_y, eps_z=eps_z, kbar2=salt_map(mask, kbar2_solvent),
                rhs=rhs_from_charges(grid_charges(nx, ny, nz, h, centres, charges), h),
                bc=debye_huckel_boundary(nx, ny, nz, h, centres, charges, eps_out, kappa))
