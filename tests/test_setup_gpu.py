"""-m gpu: NEXT row f1 -- pb_create_from_atoms (grid / stencil setup on the GPU) against oracle/pbsetup_ref.py.

Bar: integer-like decisions (solute mask, which of the three face values, salt on/off) bit-exact; face values
bit-exact (same IEEE operations); trilinear charges 1e-13 (atomic accumulation order); Debye-Hueckel ghost values
1e-12 relative to the sum of |terms| (exp differs by an ulp between libm and CUDA); then the solve through the
atom-built handle against the solver oracle fed by the setup oracle."""
import math

import numpy as np
import pytest

from workloads import pb_inputs as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg(cuda_device):
    from paper_1704_02745_b200 import build as pb_build

    pb_build.build()
    import paper_1704_02745_b200 as p

    p.load_library()
    return p


def atoms(n_atoms, nx, ny, nz, h, seed):
    rng = np.random.Generator(np.random.PCG64(W.SEED0 + 500 + seed))
    L = np.array([(nx - 1) * h, (ny - 1) * h, (nz - 1) * h])
    c = W.atoms_uniform(n_atoms, 0.15 * L, 0.85 * L, rng)
    c[0] = [0.2, 0.3, L[2] - 0.1]                       # one atom hugging a corner: clipped bounding box
    r = rng.uniform(1.2, 2.0, n_atoms)
    q = rng.normal(0.0, 0.4, n_atoms)
    return c, r, q


@pytest.mark.parametrize("shape,na", [((21, 17, 13), 12), ((33, 33, 33), 1), ((40, 23, 31), 60)])
def test_fields_match_setup_oracle(pkg, shape, na):
    from oracle import pbsetup_ref as S

    nx, ny, nz = shape
    h, eps_in, eps_out, kb = 0.5, 1.0, 80.0, W.KBAR2_150MM_300K
    if na == 1:
        c, r, q = np.array([[8.0, 8.0, 8.0]]), np.array([2.0]), np.array([1.0])      # config 1 (Born ion)
    else:
        c, r, q = atoms(na, nx, ny, nz, h, na)
    ref = S.setup(nx, ny, nz, h, c, r, q, eps_in, eps_out, kb)
    with pkg.PBSolver.from_atoms(nx, ny, nz, h, c, r, q, eps_in, eps_out, kb) as s:
        for name in ("eps_x", "eps_y", "eps_z", "kbar2"):
            assert np.array_equal(s.field(name), ref[name]), name           # bit-exact
        rhs = s.field("rhs")
        assert np.max(np.abs(rhs - ref["rhs"])) <= 1e-13 * np.max(np.abs(ref["rhs"]))
        assert np.array_equal(rhs != 0, ref["rhs"] != 0)
        bc = s.field("bc")
        kappa = math.sqrt(kb / eps_out)
        g = S.ghost_positions(nx, ny, nz, h)
        rr = np.linalg.norm(g[:, None, :] - c[None, :, :], axis=2)
        scale = (np.abs(q)[None, :] * np.exp(-kappa * rr) / rr).sum(1) / eps_out
        assert np.all(np.abs(bc - ref["bc"]) <= 1e-12 * scale)
        # new charges on the same atoms (pb_set_charges): rhs and bc follow, operator untouched
        q2 = q + 0.05
        s.set_charges(q2)
        ref2 = S.setup(nx, ny, nz, h, c, r, q2, eps_in, eps_out, kb)
        assert np.max(np.abs(s.field("rhs") - ref2["rhs"])) <= 1e-13 * np.max(np.abs(ref2["rhs"]))
        assert np.all(np.abs(s.field("bc") - ref2["bc"]) <= 1e-12 * (scale + 0.05 * (np.exp(-kappa * rr) / rr).sum(1) / eps_out))
        assert np.array_equal(s.field("eps_x"), ref["eps_x"])


@pytest.mark.parametrize("kb", [0.0, 2.0e5])
def test_boundary_sum_salt_extremes(pkg, kb):
    """The fp64 boundary sum outside its everyday range: no salt (kappa = 0, every exponential is exactly 1) and a
    screening so strong (kappa r up to ~800) that the kernel's fitted exp routine does not apply and the library one is
    used (dh_fast_range) -- ghost values against the setup oracle, 1e-12 of the sum of |terms|."""
    from oracle import pbsetup_ref as S

    nx, ny, nz, h, eps_in, eps_out = 21, 17, 13, 0.5, 1.0, 80.0
    c, r, q = atoms(12, nx, ny, nz, h, 12)
    ref = S.setup(nx, ny, nz, h, c, r, q, eps_in, eps_out, kb)
    kappa = math.sqrt(kb / eps_out)
    g = S.ghost_positions(nx, ny, nz, h)
    rr = np.linalg.norm(g[:, None, :] - c[None, :, :], axis=2)
    scale = (np.abs(q)[None, :] * np.exp(-kappa * rr) / rr).sum(1) / eps_out
    with pkg.PBSolver.from_atoms(nx, ny, nz, h, c, r, q, eps_in, eps_out, kb) as s:
        bc = s.field("bc")
    assert np.all(np.isfinite(bc)) and np.all(np.abs(bc - ref["bc"]) <= 1e-12 * scale + 1e-300)
    if kb == 0.0:
        assert np.max(np.abs(bc)) > 0.0


def test_fp32_boundary_sum(pkg):
    """pb_set_setup_precision(PB_F32): the Debye-Hueckel ghost values with every term in fp32 (hardware rsqrt / exp2,
    Kahan partial sums) stay within 2e-6 of the sum of |terms| of the fp64 setup oracle (an fp32 term carries a few
    1e-7; the bound is on the term scale because charges of both signs cancel), the charge grid stays fp64-exact, and
    an fp32 solve on that boundary is still within the fp32 bar of the oracle's solve on the exact boundary."""
    from oracle import pbref, pbsetup_ref as S

    nx, ny, nz, h = 40, 23, 31, 0.5
    eps_in, eps_out, kb = 1.0, 80.0, W.KBAR2_150MM_300K
    c, r, q = atoms(300, nx, ny, nz, h, 61)              # more than one 256-atom tile, odd tail
    c = c[:299]; r = r[:299]; q = q[:299]
    q2 = q + 0.05
    ref = S.setup(nx, ny, nz, h, c, r, q2, eps_in, eps_out, kb)
    kappa = math.sqrt(kb / eps_out)
    g = S.ghost_positions(nx, ny, nz, h)
    rr = np.linalg.norm(g[:, None, :] - c[None, :, :], axis=2)
    scale = (np.abs(q2)[None, :] * np.exp(-kappa * rr) / rr).sum(1) / eps_out
    o = pbref.PBRef(nx, ny, nz, h, ref["eps_x"], ref["eps_y"], ref["eps_z"], ref["kbar2"], ref["rhs"],
                    ref["bc"]).solve(1e-10, 5000)
    with pkg.PBSolver.from_atoms(nx, ny, nz, h, c, r, q, eps_in, eps_out, kb) as s:
        s.set_setup_precision("f32")
        s.set_charges(q2)
        bc32 = s.field("bc")
        err = np.abs(bc32 - ref["bc"])
        assert np.all(err <= 2e-6 * scale)
        assert np.max(err / scale) > 1e-12               # it really is the fp32 kernel
        assert np.max(np.abs(s.field("rhs") - ref["rhs"])) <= 1e-13 * np.max(np.abs(ref["rhs"]))
        g32 = s.solve(1e-5, 5000, "f32")
        s.set_setup_precision("f64")
        s.set_charges(q2)
        assert np.all(np.abs(s.field("bc") - ref["bc"]) <= 1e-12 * scale)
    assert np.max(np.abs(g32["phi"] - o["phi"])) <= 1e-4 * np.max(np.abs(o["phi"]))


def test_solve_through_atom_built_handle(pkg):
    from oracle import pbref, pbsetup_ref as S

    nx, ny, nz, h = 40, 23, 31, 0.5
    c, r, q = atoms(60, nx, ny, nz, h, 60)
    f = S.setup(nx, ny, nz, h, c, r, q, 1.0, 80.0, W.KBAR2_150MM_300K)
    o = pbref.PBRef(nx, ny, nz, h, f["eps_x"], f["eps_y"], f["eps_z"], f["kbar2"], f["rhs"], f["bc"]).solve(1e-10, 5000)
    with pkg.PBSolver.from_atoms(nx, ny, nz, h, c, r, q, 1.0, 80.0, W.KBAR2_150MM_300K) as s:
        g = s.solve(1e-10, 5000, "f64")
        g32 = s.solve(1e-5, 5000, "f32")
    scale = np.max(np.abs(o["phi"]))
    assert g["status"] == 0 and abs(g["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"]))
    assert np.max(np.abs(g["phi"] - o["phi"])) <= 1e-8 * scale
    assert np.max(np.abs(g32["phi"] - o["phi"])) <= 1e-4 * scale


def test_from_atoms_edge_cases(pkg):
    # no atoms: pure solvent, zero rhs and ghost values -> phi = 0 in 0 iterations
    with pkg.PBSolver.from_atoms(9, 8, 7, 0.5, np.zeros((0, 3)), np.zeros(0), np.zeros(0), 1.0, 80.0, 1.0) as s:
        assert np.all(s.field("eps_y") == 80.0) and np.all(s.field("kbar2") == 1.0) and not s.field("rhs").any()
        g = s.solve(1e-8, 50, "f64")
        assert g["iters"] == 0 and not g["phi"].any()
    with pytest.raises(pkg.PBError):
        pkg.PBSolver.from_atoms(1, 8, 7, 0.5, np.zeros((1, 3)), np.ones(1), np.ones(1), 1.0, 80.0, 1.0)
    with pytest.raises(pkg.PBError):
        pkg.PBSolver.from_atoms(9, 8, 7, 0.5, np.ones((1, 3)), np.ones(1), np.ones(1), -1.0, 80.0, 1.0)


def test_atoms_outside_the_box_are_rejected_and_charges_are_reproducible(pkg):
    """An atom outside [0, (n-1)h]^3 would get extrapolated trilinear weights (and, on a ghost node, 1/0 in the
    boundary sum): PB_ERR_INVALID_ARG.  The charge grid accumulates in 64-bit fixed point, so repeated spreading of
    the same charges is bit-identical even where many atoms share nodes."""
    nx, ny, nz, h = 21, 17, 13, 0.5
    c, r, q = atoms(40, nx, ny, nz, h, 9)
    for bad in ([-0.1, 2.0, 2.0], [2.0, (ny - 1) * h + 0.01, 2.0], [2.0, 2.0, float("nan")]):
        cb = c.copy()
        cb[5] = bad
        with pytest.raises(pkg.PBError) as e:
            pkg.PBSolver.from_atoms(nx, ny, nz, h, cb, r, q, 1.0, 80.0, 1.0)
        assert e.value.status == pkg.binding.PB_ERR_INVALID_ARG
    c[:20] = c[20:] + 0.01                                # pairs of atoms in the same cell: shared nodes
    with pkg.PBSolver.from_atoms(nx, ny, nz, h, c, r, q, 1.0, 80.0, 1.0) as s:
        first = s.field("rhs")
        for _ in range(3):
            s.set_charges(q)
            assert np.array_equal(s.field("rhs"), first)
        with pytest.raises(pkg.PBError):
            s.set_charges(np.where(np.arange(40) == 3, np.inf, q))
