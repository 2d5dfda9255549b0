"""Seeded synthetic Poisson-Boltzmann problems: the five `configs` of BASELINE.json.

What this module produces is *input data only* -- the four coefficient fields of
PAPER.md Eq. 3 (face dielectrics eps_i, eps_j, eps_k and the nodal Boltzmann
coefficient kappa^2), the charge right-hand side and the
free-space Dirichlet values on a ghost layer around the grid.
The recipe (restated in DESIGN.md) stands in for the Amber
benchmark structures the paper measured on, which are not available here.

Conventions (shared by the oracle and the CUDA library):
  * node (i,j,k) sits at (i*h, j*h, k*h); arrays are C-ordered [k][j][i], x fastest;
  * eps_x has shape [nz][ny][nx+1]; face f lies between node i=f-1 and node i=f, so
    f=0 and f=nx touch the ghost layer.  eps_y [nz][ny+1][nx], eps_z [nz+1][ny][nx];
  * lengths in Angstrom, charges in e, potential in e/Angstrom (Gaussian-style units):
    -div(eps grad phi) + kbar2*phi = rhs with rhs = 4*pi*q_node/h^3;
  * bc packs the ghost Dirichlet values as x-, x+ ([nz][ny] each), y-, y+ ([nz][nx]),
    z-, z+ ([ny][nx]).

Nothing here solves or applies the operator.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED0 = 170402745

# kbar2 = eps_out * kappa_D^2 = 2 N_A e^2 I / (eps0 kB T) for a 1:1 salt of ionic strength I
# (SI, CODATA-2018), I = 0.15 mol/L = 150 mol/m^3, T = 300 K, converted m^-2 -> Angstrom^-2.
_NA = 6.02214076e23
_E = 1.602176634e-19
_EPS0 = 8.8541878128e-12
_KB = 1.380649e-23
KBAR2_150MM_300K = 2.0 * _NA * _E * _E * 150.0 / (_EPS0 * _KB * 300.0) * 1e-20  # = 1.26456 A^-2


@dataclass
class PBInputs:
    nx: int
    ny: int
    nz: int
    h: float
    eps_x: np.ndarray
    eps_y: np.ndarray
    eps_z: np.ndarray
    kbar2: np.ndarray
    rhs: np.ndarray
    bc: np.ndarray
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return self.nx * self.ny * self.nz

    def args(self):
        """Positional arrays in the order both pb_create and the oracle take them."""
        return (self.nx, self.ny, self.nz, self.h, self.eps_x, self.eps_y, self.eps_z,
                self.kbar2, self.rhs, self.bc)


def bc_size(nx: int, ny: int, nz: int) -> int:
    return 2 * (nz * ny + nz * nx + ny * nx)


# --------------------------------------------------------------------------------------
# atoms
# --------------------------------------------------------------------------------------
def _fix_total_charge(q: np.ndarray) -> np.ndarray:
    """'total rounded to an integer': shift every charge by the same amount."""
    tot = q.sum()
    return q - (tot - round(tot)) / q.size


def atoms_uniform(n_atoms: int, lo, hi, rng: np.random.Generator) -> np.ndarray:
    lo = np.asarray(lo, float)
    hi = np.asarray(hi, float)
    return lo + (hi - lo) * rng.random((n_atoms, 3))


class _CellList:
    """Uniform cell list over points kept as python tuples (the walk is a scalar loop)."""

    def __init__(self, cell: float):
        self.cell = cell
        self.cells: dict[tuple, list] = {}
        self.pos: list = []

    def _key(self, p):
        c = self.cell
        return (math.floor(p[0] / c), math.floor(p[1] / c), math.floor(p[2] / c))

    def add(self, p) -> int:
        idx = len(self.pos)
        self.pos.append(p)
        self.cells.setdefault(self._key(p), []).append(idx)
        return idx

    def pop(self):
        idx = len(self.pos) - 1
        p = self.pos.pop()
        self.cells[self._key(p)].remove(idx)

    def clash(self, p, dmin2: float, skip_from: int) -> bool:
        """True if any stored point with index < skip_from is closer than sqrt(dmin2)."""
        kx, ky, kz = self._key(p)
        cells = self.cells
        pos = self.pos
        px, py, pz = p
        for ax in (kx - 1, kx, kx + 1):
            for ay in (ky - 1, ky, ky + 1):
                for az in (kz - 1, kz, kz + 1):
                    lst = cells.get((ax, ay, az))
                    if not lst:
                        continue
                    for idx in lst:
                        if idx >= skip_from:
                            continue
                        q = pos[idx]
                        dx = q[0] - px
                        dy = q[1] - py
                        dz = q[2] - pz
                        if dx * dx + dy * dy + dz * dz < dmin2:
                            return True
        return False


def _walk_once(n_atoms, lo, hi, rng, cl: _CellList, bond, dmin, max_reject):
    """Grow one self-avoiding chain inside the box [lo,hi]; returns False if it stalls."""
    dmin2 = dmin * dmin
    base = len(cl.pos)
    # start: uniform in the confinement, clear of earlier chains
    for _ in range(10000):
        p = tuple(lo[d] + (hi[d] - lo[d]) * rng.random() for d in range(3))
        if not cl.clash(p, dmin2, base):
            break
    else:
        return False
    cl.add(p)
    total_reject = 0
    rejects = 0
    while len(cl.pos) - base < n_atoms:
        last = cl.pos[-1]
        v = rng.standard_normal(3)
        s = bond / math.sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2])
        c = (last[0] + s * v[0], last[1] + s * v[1], last[2] + s * v[2])
        ok = (lo[0] <= c[0] <= hi[0]) and (lo[1] <= c[1] <= hi[1]) and (lo[2] <= c[2] <= hi[2])
        # atoms 1 and 2 bonds back are exempt; everything else (incl. other chains) >= dmin
        if ok and cl.clash(c, dmin2, len(cl.pos) - 2):
            ok = False
        if ok:
            cl.add(c)
            rejects = 0
            continue
        rejects += 1
        total_reject += 1
        if total_reject > max_reject:
            return False
        if rejects >= 50:
            npop = min(10, len(cl.pos) - base - 1)
            for _ in range(npop):
                cl.pop()
            rejects = 0
    return True


def atoms_random_walk(n_chains: int, n_per_chain: int, confinements, seed: int,
                      bond: float = 1.5, dmin: float = 3.0, max_reject: int = 1_000_000):
    """Self-avoiding random-walk chains (bond 1.5 A, >= 3 A from atoms >= 3 bonds away).

    `confinements` is a list of (lo, hi) boxes, one per chain, sharing one exclusion list.
    If a walk stalls, all confinements are scaled by 5 % about their common centre and the
    whole construction restarts from the same seed.  Returns (rng, centres, scale_used).
    """
    scale = 1.0
    los = np.array([c[0] for c in confinements], float)
    his = np.array([c[1] for c in confinements], float)
    centre = 0.5 * (los.min(axis=0) + his.max(axis=0))
    while True:
        rng = np.random.Generator(np.random.PCG64(seed))
        cl = _CellList(dmin)
        good = True
        for ch in range(n_chains):
            lo = centre + scale * (los[ch] - centre)
            hi = centre + scale * (his[ch] - centre)
            if not _walk_once(n_per_chain, lo, hi, rng, cl, bond, dmin, max_reject):
                good = False
                break
        if good:
            return rng, np.array(cl.pos, float), scale
        scale *= 1.05


# --------------------------------------------------------------------------------------
# grid fields
# --------------------------------------------------------------------------------------
def solute_mask(nx, ny, nz, h, centres, radii) -> np.ndarray:
    """Node is solute iff it lies within any atom sphere (d^2 <= R^2); bool [nz][ny][nx]."""
    mask = np.zeros((nz, ny, nx), bool)
    for (cx, cy, cz), R in zip(centres, radii):
        i0, i1 = max(0, math.ceil((cx - R) / h)), min(nx - 1, math.floor((cx + R) / h))
        j0, j1 = max(0, math.ceil((cy - R) / h)), min(ny - 1, math.floor((cy + R) / h))
        k0, k1 = max(0, math.ceil((cz - R) / h)), min(nz - 1, math.floor((cz + R) / h))
        if i0 > i1 or j0 > j1 or k0 > k1:
            continue
        dx = np.arange(i0, i1 + 1) * h - cx
        dy = np.arange(j0, j1 + 1) * h - cy
        dz = np.arange(k0, k1 + 1) * h - cz
        d2 = dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2
        mask[k0:k1 + 1, j0:j1 + 1, i0:i1 + 1] |= d2 <= R * R
    return mask


def face_eps_from_mask(mask: np.ndarray, eps_in: float, eps_out: float):
    """Harmonic mean 2 e1 e2/(e1+e2) of the two nodes a face joins; ghost nodes are solvent."""
    nz, ny, nx = mask.shape
    node = np.where(mask, eps_in, eps_out).astype(np.float64)
    pad = np.full((nz + 2, ny + 2, nx + 2), float(eps_out))
    pad[1:-1, 1:-1, 1:-1] = node

    def hm(a, b):
        return 2.0 * a * b / (a + b)

    c = pad[1:-1, 1:-1, :]
    eps_x = hm(c[:, :, :-1], c[:, :, 1:])
    c = pad[1:-1, :, 1:-1]
    eps_y = hm(c[:, :-1, :], c[:, 1:, :])
    c = pad[:, 1:-1, 1:-1]
    eps_z = hm(c[:-1, :, :], c[1:, :, :])
    return (np.ascontiguousarray(eps_x), np.ascontiguousarray(eps_y), np.ascontiguousarray(eps_z))


def spread_trilinear(nx, ny, nz, h, centres, charges) -> np.ndarray:
    """Trilinear spreading of point charges to the 8 surrounding nodes; returns q_node."""
    q = np.zeros((nz, ny, nx))
    c = np.asarray(centres, float) / h
    i0 = np.clip(np.floor(c).astype(np.int64), 0, [nx - 2, ny - 2, nz - 2])
    f = c - i0
    for dz in (0, 1):
        wz = f[:, 2] if dz else 1.0 - f[:, 2]
        for dy in (0, 1):
            wy = f[:, 1] if dy else 1.0 - f[:, 1]
            for dx in (0, 1):
                wx = f[:, 0] if dx else 1.0 - f[:, 0]
                np.add.at(q, (i0[:, 2] + dz, i0[:, 1] + dy, i0[:, 0] + dx), charges * wz * wy * wx)
    return q


def ghost_coords(nx, ny, nz, h) -> np.ndarray:
    """Coordinates of the ghost nodes in `bc` packing order; [bc_size, 3]."""
    x = np.arange(nx) * h
    y = np.arange(ny) * h
    z = np.arange(nz) * h
    out = []
    for xg in (-h, nx * h):                       # x-, x+ : [nz][ny]
        Z, Y = np.meshgrid(z, y, indexing="ij")
        out.append(np.stack([np.full_like(Z, xg), Y, Z], -1).reshape(-1, 3))
    for yg in (-h, ny * h):                       # y-, y+ : [nz][nx]
        Z, X = np.meshgrid(z, x, indexing="ij")
        out.append(np.stack([X, np.full_like(Z, yg), Z], -1).reshape(-1, 3))
    for zg in (-h, nz * h):                       # z-, z+ : [ny][nx]
        Y, X = np.meshgrid(y, x, indexing="ij")
        out.append(np.stack([X, Y, np.full_like(Y, zg)], -1).reshape(-1, 3))
    return np.concatenate(out, 0)


def debye_huckel_ghost(nx, ny, nz, h, centres, charges, eps_out, kappa, device=None) -> np.ndarray:
    """Free-space boundary values sum_i q_i exp(-kappa r_i)/(eps_out r_i) on the ghost layer.

    Exact sum over all atoms, chunked; torch is used only as a vectorised array library
    (on the GPU when one is present, which is what makes config 5's 5e10 terms practical).
    """
    import torch

    if device is None:
        device = "cuda" if torch.cuda.is_available() else "cpu"
    g = torch.from_numpy(ghost_coords(nx, ny, nz, h)).to(device)
    c = torch.from_numpy(np.ascontiguousarray(centres, dtype=np.float64)).to(device)
    q = torch.from_numpy(np.ascontiguousarray(charges, dtype=np.float64)).to(device)
    out = torch.empty(g.shape[0], dtype=torch.float64, device=device)
    chunk = max(1, int(3e7) // max(1, c.shape[0]))
    for s in range(0, g.shape[0], chunk):
        gg = g[s:s + chunk]
        # |g-c|^2 by explicit differences (no cancellation-prone expansion)
        d2 = ((gg[:, None, 0] - c[None, :, 0]) ** 2 + (gg[:, None, 1] - c[None, :, 1]) ** 2
              + (gg[:, None, 2] - c[None, :, 2]) ** 2)
        r = torch.sqrt(d2)
        out[s:s + chunk] = (torch.exp(-kappa * r) / r) @ q
    return (out / eps_out).cpu().numpy()


def assemble(nx, ny, nz, h, centres, radii, charges, eps_in, eps_out, kbar2_solvent,
             name="", device=None, extra=None) -> PBInputs:
    mask = solute_mask(nx, ny, nz, h, centres, radii)
    eps_x, eps_y, eps_z = face_eps_from_mask(mask, eps_in, eps_out)
    kbar2 = np.where(mask, 0.0, float(kbar2_solvent))
    qn = spread_trilinear(nx, ny, nz, h, centres, charges)
    rhs = 4.0 * math.pi * qn / h ** 3
    kappa = math.sqrt(kbar2_solvent / eps_out)
    bc = debye_huckel_ghost(nx, ny, nz, h, centres, charges, eps_out, kappa, device=device)
    meta = dict(name=name, centres=np.asarray(centres, float), radii=np.asarray(radii, float),
                charges=np.asarray(charges, float), eps_in=eps_in, eps_out=eps_out,
                kbar2_solvent=kbar2_solvent, kappa=kappa,
                solute_fraction=float(mask.mean()))
    if extra:
        meta.update(extra)
    return PBInputs(nx, ny, nz, h, eps_x, eps_y, eps_z, np.ascontiguousarray(kbar2),
                    np.ascontiguousarray(rhs), bc, meta)


# --------------------------------------------------------------------------------------
# the configs
# --------------------------------------------------------------------------------------
def born_ion(n: int = 33, h: float = 0.5, radius: float = 2.0, q: float = 1.0,
             eps_in: float = 1.0, eps_out: float = 80.0, centre=None) -> PBInputs:
    """Config 1: one charged sphere, no salt, ghost values q/(eps_out r)."""
    L = (n - 1) * h
    c = np.array([[L / 2, L / 2, L / 2]] if centre is None else [centre], float)
    return assemble(n, n, n, h, c, np.array([radius]), np.array([q]), eps_in, eps_out, 0.0,
                    name=f"born_{n}")


def _chain_config(cfg, n, n_chains, n_per_chain, eps_in, device, n_side=None):
    h = 0.5
    L = (n - 1) * h
    side = L / 1.5                       # the paper's fill ratio 1.5
    lo0 = (L - side) / 2
    if n_chains == 1:
        conf = [((lo0,) * 3, (lo0 + side,) * 3)]
    else:                                # z-slabs separated by 3 A gaps
        gap = 3.0
        t = (side - (n_chains - 1) * gap) / n_chains
        conf = [((lo0, lo0, lo0 + s * (t + gap)), (lo0 + side, lo0 + side, lo0 + s * (t + gap) + t))
                for s in range(n_chains)]
    rng, centres, scale = atoms_random_walk(n_chains, n_per_chain, conf, SEED0 + cfg)
    centres = centres - centres.mean(0) + L / 2          # re-centre
    na = centres.shape[0]
    radii = rng.uniform(1.2, 2.0, na)
    charges = _fix_total_charge(rng.normal(0.0, 0.4, na))
    return assemble(n, n, n, h, centres, radii, charges, eps_in, 80.0, KBAR2_150MM_300K,
                    name=f"cfg{cfg}_{n}", device=device,
                    extra=dict(confinement_scale=scale, n_chains=n_chains))


def make_config(cfg: int, device=None, n_atoms=None) -> PBInputs:
    """BASELINE.json configs 1..5 (index = position in `configs`, 1-based).

    RNG: numpy PCG64(170402745 + cfg); draw order centres -> radii -> charges.
    `n_atoms` overrides the atom count (used only by tests that want a cheaper generator run).
    """
    if cfg == 1:
        return born_ion()
    if cfg == 2:
        n, h = 65, 0.5
        L = (n - 1) * h
        rng = np.random.Generator(np.random.PCG64(SEED0 + cfg))
        na = n_atoms or 200
        centres = atoms_uniform(na, (0.2 * L,) * 3, (0.8 * L,) * 3, rng)
        radii = rng.uniform(1.2, 2.0, na)
        charges = _fix_total_charge(rng.normal(0.0, 0.4, na))
        return assemble(n, n, n, h, centres, radii, charges, 1.0, 80.0, KBAR2_150MM_300K,
                        name="cfg2_65", device=device)
    if cfg == 3:
        return _chain_config(3, 129, 1, n_atoms or 2000, 1.0, device)
    if cfg == 4:
        return _chain_config(4, 257, 1, n_atoms or 20000, 4.0, device)
    if cfg == 5:
        return _chain_config(5, 385, 3, n_atoms or 20000, 1.0, device)
    raise ValueError(f"unknown config {cfg}")


def perturbed_charge_values(inp: PBInputs, s: int) -> np.ndarray:
    """Charges of batch member s (q_i += N(0,0.05), total re-fixed); RNG PCG64(170402745 + 1000 + s)."""
    m = inp.meta
    rng = np.random.Generator(np.random.PCG64(SEED0 + 1000 + s))
    return _fix_total_charge(m["charges"] + rng.normal(0.0, 0.05, m["charges"].size))


def perturbed_charges(inp: PBInputs, s: int, device=None):
    """Batch member s of config 5's 50-solve batch: q_i += N(0,0.05), total re-fixed.

    Same operator; returns (rhs, bc) for pb_set_rhs.  RNG PCG64(170402745 + 1000 + s).
    """
    m = inp.meta
    q = perturbed_charge_values(inp, s)
    qn = spread_trilinear(inp.nx, inp.ny, inp.nz, inp.h, m["centres"], q)
    rhs = 4.0 * math.pi * qn / inp.h ** 3
    bc = debye_huckel_ghost(inp.nx, inp.ny, inp.nz, inp.h, m["centres"], q, m["eps_out"],
                            m["kappa"], device=device)
    return np.ascontiguousarray(rhs), bc


def random_operator(nx, ny, nz, seed, h=0.5, salted=True, two_valued=True) -> PBInputs:
    """Structure-free random SPD operator for SpMV / small-solve parity (anisotropic, odd sizes).

    Face dielectrics are drawn per face (two-valued 1/80 with ~40 % low, or U[1,80]); kbar2 is
    U[0,2] on ~60 % of the nodes; rhs ~ N(0,1); ghost values ~ U(-1,1).
    """
    rng = np.random.Generator(np.random.PCG64(SEED0 + 7919 * seed + 13))

    def eps(shape):
        if two_valued:
            return np.where(rng.random(shape) < 0.4, 1.0, 80.0)
        return rng.uniform(1.0, 80.0, shape)

    eps_x = eps((nz, ny, nx + 1))
    eps_y = eps((nz, ny + 1, nx))
    eps_z = eps((nz + 1, ny, nx))
    if salted:
        kbar2 = np.where(rng.random((nz, ny, nx)) < 0.6, rng.uniform(0.0, 2.0, (nz, ny, nx)), 0.0)
    else:
        kbar2 = np.zeros((nz, ny, nx))
    rhs = rng.standard_normal((nz, ny, nx))
    bc = rng.uniform(-1.0, 1.0, bc_size(nx, ny, nz))
    return PBInputs(nx, ny, nz, h, eps_x, eps_y, eps_z, kbar2, rhs, bc,
                    dict(name=f"rand_{nx}x{ny}x{nz}_s{seed}"))
