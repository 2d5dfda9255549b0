"""-m "not gpu": pins of the grid-setup oracle (oracle/pbsetup_ref.py) against things fixed outside of it:
brute-force lattice counts, the three face values a two-valued dielectric map can take, exact moment
conservation of trilinear spreading, closed-form single-charge potentials, and the analytic fixtures of
tests/golden/born_analytic.txt."""
import itertools
import math

import numpy as np

from oracle import pbsetup_ref as S


def test_mask_is_the_lattice_ball_brute_force():
    # sphere R = 2 A centred on node (16,16,16), h = 0.5: nodes with i^2+j^2+k^2 <= 16 (integer arithmetic)
    n, h = 33, 0.5
    m = S.solute_mask(n, n, n, h, [[8.0, 8.0, 8.0]], [2.0])
    count = sum(1 for i, j, k in itertools.product(range(-5, 6), repeat=3) if i * i + j * j + k * k <= 16)
    assert m.sum() == count == 257
    assert m[16, 16, 20] and m[16, 20, 16] and m[20, 16, 16] and not m[16, 16, 21]      # d^2 <= R^2 inclusive
    # off-centre atom near a corner: clipped bounding box, brute force over every node
    c, R = [0.3, 15.9, 7.77], 1.7
    m2 = S.solute_mask(n, n, n, h, [c], [R])
    brute = np.zeros_like(m2)
    for k, j, i in itertools.product(range(n), repeat=3):
        brute[k, j, i] = (i * h - c[0]) ** 2 + (j * h - c[1]) ** 2 + (k * h - c[2]) ** 2 <= R * R + 1e-12
    assert np.array_equal(m2, brute)
    # union of two atoms
    m3 = S.solute_mask(n, n, n, h, [[8.0, 8.0, 8.0], c], [2.0, R])
    assert np.array_equal(m3, m | m2)


def test_face_values_and_shapes():
    n, h = 9, 0.5
    mask = S.solute_mask(n, n + 1, n + 2, h, [[2.0, 2.2, 2.4]], [1.1])
    ex, ey, ez = S.face_dielectrics(mask, 1.0, 80.0)
    nz, ny, nx = mask.shape
    assert ex.shape == (nz, ny, nx + 1) and ey.shape == (nz, ny + 1, nx) and ez.shape == (nz + 1, ny, nx)
    vals = {1.0, 80.0, 2.0 * 80.0 / 81.0}
    for a in (ex, ey, ez):
        assert set(np.unique(a)) <= vals
    # a face is low-dielectric iff both its nodes are solute, mixed iff exactly one is; ghost nodes are solvent
    node = np.pad(mask, 1)
    assert np.array_equal(ex == 1.0, node[1:-1, 1:-1, :-1] & node[1:-1, 1:-1, 1:])
    assert np.array_equal(ey == 80.0, ~node[1:-1, :-1, 1:-1] & ~node[1:-1, 1:, 1:-1])
    assert np.array_equal(ez == 2.0 * 80.0 / 81.0, node[:-1, 1:-1, 1:-1] ^ node[1:, 1:-1, 1:-1])
    assert np.all(ex[:, :, 0] == 80.0) and np.all(ez[-1] == 80.0)
    k2 = S.salt_map(mask, 1.26456)
    assert np.all(k2[mask] == 0.0) and np.all(k2[~mask] == 1.26456)


def test_trilinear_conserves_charge_and_dipole():
    rng = np.random.default_rng(3)
    nx, ny, nz, h = 11, 9, 7, 0.5
    c = rng.uniform([0.2, 0.2, 0.2], [(nx - 1) * h - 0.2, (ny - 1) * h - 0.2, (nz - 1) * h - 0.2], (40, 3))
    q = rng.normal(0, 0.4, 40)
    g = S.grid_charges(nx, ny, nz, h, c, q)
    z, y, x = np.meshgrid(np.arange(nz) * h, np.arange(ny) * h, np.arange(nx) * h, indexing="ij")
    assert abs(g.sum() - q.sum()) < 1e-13
    for coord, col in ((x, 0), (y, 1), (z, 2)):          # first moments are reproduced exactly by trilinear weights
        assert abs((g * coord).sum() - (q * c[:, col]).sum()) < 1e-12
    # a charge on a node stays on that node; at most 8 nodes per charge
    g1 = S.grid_charges(nx, ny, nz, h, [[2.0, 1.5, 1.0]], [0.7])
    assert g1[2, 3, 4] == 0.7 and np.count_nonzero(g1) == 1
    assert np.count_nonzero(S.grid_charges(nx, ny, nz, h, [[2.1, 1.6, 1.2]], [1.0])) == 8
    assert np.allclose(S.rhs_from_charges(g1, h)[2, 3, 4], 4 * math.pi * 0.7 / 0.125)


def test_debye_huckel_closed_forms():
    nx, ny, nz, h = 5, 4, 3, 0.5
    c = np.array([[1.0, 0.75, 0.5]])
    gp = S.ghost_positions(nx, ny, nz, h)
    assert gp.shape == (2 * (nz * ny + nz * nx + ny * nx), 3)
    assert np.allclose(gp[0], [-h, 0, 0]) and np.allclose(gp[nz * ny], [nx * h, 0, 0])
    assert np.allclose(gp[2 * nz * ny + 1], [h, -h, 0]) and np.allclose(gp[-1], [(nx - 1) * h, (ny - 1) * h, nz * h])
    r = np.linalg.norm(gp - c[0], axis=1)
    kap = 0.1257
    bc = S.debye_huckel_boundary(nx, ny, nz, h, c, [1.3], 80.0, kap)
    assert np.allclose(bc, 1.3 * np.exp(-kap * r) / (80.0 * r), rtol=1e-14)
    assert np.allclose(S.debye_huckel_boundary(nx, ny, nz, h, c, [1.0], 80.0, 0.0), 1.0 / (80.0 * r), rtol=1e-14)
    # superposition
    c2 = np.array([[1.0, 0.75, 0.5], [0.3, 1.2, 0.9]])
    b2 = S.debye_huckel_boundary(nx, ny, nz, h, c2, [0.4, -0.9], 80.0, kap)
    b2s = (S.debye_huckel_boundary(nx, ny, nz, h, c2[:1], [0.4], 80.0, kap)
           + S.debye_huckel_boundary(nx, ny, nz, h, c2[1:], [-0.9], 80.0, kap))
    assert np.allclose(b2, b2s, rtol=1e-13)
    # golden: exterior Born potential at r = 6 A (tests/golden/born_analytic.txt: phi_exterior_r6)
    assert abs(1.0 / (80.0 * 6.0) - 0.0020833333333333333) < 1e-18


def test_setup_feeds_the_solver_oracle_born_ion():
    """End to end through both oracles: atoms -> fields -> Jacobi-PCG reproduces the Born reaction field (5 %)."""
    from oracle import pbref

    n, h = 33, 0.5
    f = S.setup(n, n, n, h, [[8.0, 8.0, 8.0]], [2.0], [1.0], 1.0, 80.0, 0.0)
    sol = pbref.PBRef(n, n, n, h, f["eps_x"], f["eps_y"], f["eps_z"], f["kbar2"], f["rhs"], f["bc"]).solve(1e-10, 2000)
    one = np.ones_like(f["eps_x"]), np.ones_like(f["eps_y"]), np.ones_like(f["eps_z"])
    bc_vac = S.debye_huckel_boundary(n, n, n, h, [[8.0, 8.0, 8.0]], [1.0], 1.0, 0.0)
    vac = pbref.PBRef(n, n, n, h, *one, None, f["rhs"], bc_vac).solve(1e-10, 2000)
    rf = sol["phi"][16, 16, 16] - vac["phi"][16, 16, 16]
    assert abs(rf - (-0.49375)) < 0.05 * 0.49375
