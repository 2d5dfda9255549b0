"""-m "not gpu": pins of the grid-setup oracle (oracle/pbsetup_ref.py) against things fixed outside of it:
brute-force lattice counts, the three face values a two-valued dielectric map can take, exact moment
conservation of trilinear spreading, closed-form single-charge potentials, and the analytic fixtures of
tests/golden/born_analytic.txt."""
import itertools
import os
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


# ---------------------------------------------------------------------------------------------
# Reading 9: kbar2 = eps_out * kappa_D^2, "+ kappa^2 phi" of Eq. 3 with "all the related
# coefficients in Boltzmann term ... absorbed into kappa^2".  Pins with salt != 0 (catch kappa = sqrt(kbar2),
# kappa = kbar2/eps_out, a dropped Boltzmann term, a wrong unit conversion of the ionic strength).
# ---------------------------------------------------------------------------------------------
def _kbar2_from_codata(ionic_mol_per_l, temp_k):
    """2 N_A e^2 I / (eps0 kB T) in 1/Angstrom^2 -- CODATA-2018 constants written out here, not imported."""
    n_a, e, eps0, k_b = 6.02214076e23, 1.602176634e-19, 8.8541878128e-12, 1.380649e-23
    per_m2 = 2.0 * n_a * e * e * (ionic_mol_per_l * 1000.0) / (eps0 * k_b * temp_k)
    return per_m2 * 1e-20


def test_debye_length_of_the_configs_salt():
    """0.15 M 1:1 salt, 300 K, eps_out = 80: Debye length 7.954 A (tests/golden/debye_length.txt), i.e.
    kbar2 = eps_out / lambda_D^2 = 1.26456 A^-2 -- the constant workloads/ hands to both sides."""
    from workloads import KBAR2_150MM_300K

    golden = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "debye_length.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]
                golden[k] = float(v)
    kb = _kbar2_from_codata(0.15, 300.0)
    assert abs(kb - golden["kbar2_150mM_300K_per_A2"]) < 5e-6
    assert abs(math.sqrt(80.0 / kb) - golden["debye_length_A_eps80"]) < 5e-4
    assert abs(KBAR2_150MM_300K - kb) < 1e-12
    # textbook cross-check (water, 25 C, eps = 78.5): lambda_D = 3.04 A / sqrt(I[mol/l]) to three digits
    assert abs(math.sqrt(78.5 / _kbar2_from_codata(1.0, 298.15)) - 3.04) < 0.01


def test_setup_kappa_with_salt_closed_form_boundary():
    """setup() must put kappa = sqrt(kbar2_solvent / eps_out) into the Debye-Hueckel ghost values: one charge,
    salt on, against q exp(-r/lambda_D)/(eps_out r) with lambda_D from the CODATA formula above."""
    nx, ny, nz, h = 7, 6, 5, 0.5
    kb = _kbar2_from_codata(0.15, 300.0)
    lam = math.sqrt(80.0 / kb)
    c = np.array([[1.3, 1.1, 0.9]])
    f = S.setup(nx, ny, nz, h, c, [1.0], [0.8], 1.0, 80.0, kb)
    r = np.linalg.norm(S.ghost_positions(nx, ny, nz, h) - c[0], axis=1)
    assert np.allclose(f["bc"], 0.8 * np.exp(-r / lam) / (80.0 * r), rtol=1e-13)
    assert np.all(f["kbar2"][~f["mask"]] == kb) and np.all(f["kbar2"][f["mask"]] == 0.0)
    # the two plausible misreadings are far outside that tolerance
    for wrong in (math.sqrt(kb), kb / 80.0):
        assert not np.allclose(f["bc"], 0.8 * np.exp(-wrong * r) / (80.0 * r), rtol=1e-3)


def test_yukawa_potential_pins_the_boltzmann_term():
    """One point charge in uniform salted solvent (eps = 80 everywhere, kbar2 = eps kappa^2 on every node): the
    solution of Eq. 3 is the screened Coulomb potential q exp(-kappa r)/(eps r).  setup() -> Jacobi-PCG oracle must
    reproduce it to discretisation accuracy (measured 0.8 % for r >= 3 A at h = 0.5 A; a missing '+kappa^2 phi'
    gives 35 %, kappa = sqrt(kbar2) or kbar2/eps in the boundary values 100 % and more)."""
    from oracle import pbref

    n, h = 41, 0.5
    kb = _kbar2_from_codata(0.15, 300.0)
    kappa = math.sqrt(kb / 80.0)
    c = [[10.25, 10.25, 10.25]]                        # cell centre: the general 8-node spreading, no solute node
    f = S.setup(n, n, n, h, c, [1e-3], [1.0], 80.0, 80.0, kb)
    assert not f["mask"].any() and np.all(f["kbar2"] == kb)
    sol = pbref.PBRef(n, n, n, h, f["eps_x"], f["eps_y"], f["eps_z"], f["kbar2"], f["rhs"], f["bc"]).solve(1e-11, 5000)
    z, y, x = np.meshgrid(*(np.arange(n) * h,) * 3, indexing="ij")
    r = np.sqrt((x - c[0][0]) ** 2 + (y - c[0][1]) ** 2 + (z - c[0][2]) ** 2)
    ana = np.exp(-kappa * r) / (80.0 * r)
    far = r >= 3.0
    assert sol["status"] == 0
    assert np.max(np.abs(sol["phi"] - ana)[far] / ana[far]) < 0.015
    # without the Boltzmann term the same boundary values give a visibly different interior
    nosalt = pbref.PBRef(n, n, n, h, f["eps_x"], f["eps_y"], f["eps_z"], None, f["rhs"], f["bc"]).solve(1e-11, 5000)
    assert np.max(np.abs(nosalt["phi"] - ana)[far] / ana[far]) > 0.2
