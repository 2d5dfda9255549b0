"""Pins for the ORACLE (oracle/pbref.c): it is checked here against what the paper and the
mathematics fix, never against itself and never against the CUDA path.

Each test names the mistake it is meant to catch.  All run on CPU (-m "not gpu").
"""
import math
import os

import numpy as np
import pytest

from oracle import pbref
from tests.helpers import dense_from_eq3, pack_bc, sine_eigenvalue, sine_mode, uniform_eps
from workloads import born_ion, make_config, random_operator

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------------------------------------
# operator: closed-form eigenpairs (catches wrong index strides, dropped terms, sign, missing h^-2,
# missing kappa^2; anisotropic dims catch transposed axes)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(9, 7, 5), (4, 11, 6), (1, 5, 3), (1, 1, 1)])
def test_apply_uniform_eigenpairs(dims):
    nx, ny, nz = dims
    h, eps, k2 = 0.4, 3.7, 0.9
    ex, ey, ez = uniform_eps(nx, ny, nz, eps)
    o = pbref.PBRef(nx, ny, nz, h, ex, ey, ez, np.full((nz, ny, nx), k2))
    for (p, q, r) in [(1, 1, 1), (nx, 1, 1), (1, ny, 1), (1, 1, nz), (max(1, nx // 2), ny, max(1, nz - 1))]:
        v = sine_mode(nx, ny, nz, p, q, r)
        lam = sine_eigenvalue(nx, ny, nz, h, eps, k2, p, q, r)
        err = np.abs(o.apply(v) - lam * v).max()
        assert err <= 5e-15 * lam, (dims, p, q, r, err / lam)


# ---------------------------------------------------------------------------------------------
# operator: dense assembly straight from Eq. 3 on tiny heterogeneous grids (catches a wrong face
# convention: eps_i(i-1) vs eps_i(i), and wrong array extents nx+1 / ny+1 / nz+1)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,seed", [((6, 5, 4), 1), ((3, 7, 5), 2), ((9, 9, 9), 3)])
def test_apply_vs_dense_eq3(dims, seed):
    nx, ny, nz = dims
    inp = random_operator(nx, ny, nz, seed, h=0.5, salted=True, two_valued=(seed != 2))
    A = dense_from_eq3(nx, ny, nz, inp.h, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2)
    o = pbref.from_inputs(inp)
    rng = np.random.default_rng(seed)
    for _ in range(3):
        x = rng.uniform(-1, 1, (nz, ny, nx))
        y = o.apply(x).ravel()
        yd = A @ x.ravel()
        scale = np.abs(A) @ np.abs(x.ravel())
        assert np.all(np.abs(y - yd) <= 1e-14 * scale)
    assert np.array_equal(np.diag(A), np.diag(A))  # sanity
    assert np.allclose(o.diag().ravel(), np.diag(A), rtol=1e-15, atol=0)


def test_dense_matrix_is_spd_and_m_matrix():
    """'symmetric and positive-definite coefficient matrices were obtained'."""
    inp = random_operator(7, 6, 5, 4, salted=False)
    A = dense_from_eq3(7, 6, 5, inp.h, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2)
    assert np.array_equal(A, A.T)
    np.linalg.cholesky(A)
    off = A - np.diag(np.diag(A))
    assert (off <= 0).all()
    assert (np.diag(A) >= -off.sum(1) - 1e-12).all()


@pytest.mark.parametrize("dims", [(33, 33, 33), (20, 31, 17)])
def test_symmetry_and_positivity_invariants(dims):
    nx, ny, nz = dims
    inp = random_operator(nx, ny, nz, 11)
    o = pbref.from_inputs(inp)
    rng = np.random.default_rng(5)
    x, y = rng.standard_normal((2, nz, ny, nx))
    xAy = float((x * o.apply(y)).sum())
    yAx = float((y * o.apply(x)).sum())
    assert abs(xAy - yAx) <= 1e-12 * max(abs(xAy), float(np.abs(x).sum()))
    assert float((x * o.apply(x)).sum()) > 0
    # Gershgorin: lambda_max <= 2 max D
    assert float((x * o.apply(x)).sum()) <= 2 * o.diag().max() * float((x * x).sum())


# ---------------------------------------------------------------------------------------------
# Dirichlet fold-in and bc packing: exact discrete solutions with non-zero ghost values
# ---------------------------------------------------------------------------------------------
def test_linear_potential_is_reproduced_exactly():
    """Uniform eps, no salt, no charge: any linear function is discretely harmonic, so the solve
    must return it at every node.  Each of the six faces carries different values, so a swapped
    or mis-strided bc block fails."""
    nx, ny, nz, h = 7, 5, 6, 0.5
    f = lambda x, y, z: 0.3 + 1.1 * x - 0.7 * y + 0.45 * z
    ex, ey, ez = uniform_eps(nx, ny, nz, 2.5)
    bc = pack_bc(nx, ny, nz, h, f)
    o = pbref.PBRef(nx, ny, nz, h, ex, ey, ez, None, None, bc)
    res = o.solve(1e-14, 500)
    Z, Y, X = np.meshgrid(np.arange(nz) * h, np.arange(ny) * h, np.arange(nx) * h, indexing="ij")
    assert res["status"] == pbref.OK
    assert np.abs(res["phi"] - f(X, Y, Z)).max() < 1e-11


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_layered_dielectric_flux_continuity(axis):
    """eps varying along one axis only: phi with eps_f * (phi(n+1) - phi(n)) = const is an exact
    discrete solution of Eq. 3 whatever the transverse face values are.  Pins the face index
    convention (eps_i(i,j,k) lies between i and i+1) together with the fold-in, per axis."""
    dims = [6, 5, 4]
    nx, ny, nz = dims
    h = 0.5
    n = dims[axis]
    rng = np.random.default_rng(axis)
    face = rng.choice([1.0, 80.0, 1.97531], n + 1)           # faces 0..n along the axis
    # potential on ghost(-1), nodes 0..n-1, ghost(n): increments C/eps_face
    C = 3.0
    u = np.concatenate([[0.25], 0.25 + np.cumsum(C / face)])   # u[m+1] = node m ; u[0], u[n+1] ghosts
    ex = rng.uniform(1, 80, (nz, ny, nx + 1))
    ey = rng.uniform(1, 80, (nz, ny + 1, nx))
    ez = rng.uniform(1, 80, (nz + 1, ny, nx))
    if axis == 0:
        ex[:] = face[None, None, :]
    elif axis == 1:
        ey[:] = face[None, :, None]
    else:
        ez[:] = face[:, None, None]
    coord = lambda x, y, z: (x, y, z)[axis]
    g = lambda x, y, z: np.interp(coord(x, y, z) / h, np.arange(-1, n + 1), u)
    bc = pack_bc(nx, ny, nz, h, g)
    o = pbref.PBRef(nx, ny, nz, h, ex, ey, ez, None, None, bc)
    res = o.solve(1e-14, 2000)
    shape = [1, 1, 1]
    shape[2 - axis] = n
    exact = np.broadcast_to(u[1:-1].reshape(shape), (nz, ny, nx))
    assert res["status"] == pbref.OK
    assert np.abs(res["phi"] - exact).max() < 1e-10 * np.abs(u).max()


# ---------------------------------------------------------------------------------------------
# PCG loop logic
# ---------------------------------------------------------------------------------------------
def test_pcg_terminates_in_m_steps_on_m_eigenvectors():
    """b = sum of m eigenvectors with distinct eigenvalues => CG stops in exactly m iterations with
    x = sum v_i / lambda_i (finite-termination property).  Catches a wrong alpha/beta formula, a
    stale r.z, or an off-by-one iteration count."""
    nx, ny, nz, h, eps, k2 = 9, 7, 5, 0.5, 2.0, 0.3
    ex, ey, ez = uniform_eps(nx, ny, nz, eps)
    modes = [(1, 1, 1), (2, 3, 1), (5, 2, 4), (9, 7, 5)]
    for m in (1, 2, 4):
        b = sum(sine_mode(nx, ny, nz, *pq) for pq in modes[:m])
        x_exact = sum(sine_mode(nx, ny, nz, *pq) / sine_eigenvalue(nx, ny, nz, h, eps, k2, *pq)
                      for pq in modes[:m])
        o = pbref.PBRef(nx, ny, nz, h, ex, ey, ez, np.full((nz, ny, nx), k2), b, None)
        res = o.solve(1e-12, 50)
        assert res["iters"] == m
        assert np.abs(res["phi"] - x_exact).max() <= 1e-12 * np.abs(x_exact).max()


@pytest.mark.parametrize("dims,seed", [((9, 9, 9), 3), ((5, 8, 6), 7)])
def test_solve_vs_dense_direct(dims, seed):
    nx, ny, nz = dims
    inp = random_operator(nx, ny, nz, seed)
    A = dense_from_eq3(nx, ny, nz, inp.h, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2)
    o = pbref.from_inputs(inp)
    res = o.solve(1e-12, 2000)
    x = np.linalg.solve(A, o.b().ravel())
    assert res["status"] == pbref.OK
    assert np.abs(res["phi"].ravel() - x).max() <= 1e-10 * np.abs(x).max()
    assert res["true_relres"] < 2e-12
    # Jacobi-preconditioned needs fewer iterations than plain CG on heterogeneous eps
    res_cg = o.solve(1e-12, 5000, precond=False)
    assert np.abs(res_cg["phi"].ravel() - x).max() <= 1e-9 * np.abs(x).max()
    assert res["iters"] < res_cg["iters"]


def test_stopping_rule_and_maxiter():
    inp = random_operator(8, 7, 6, 9)
    o = pbref.from_inputs(inp)
    full = o.solve(1e-8, 1000, history=True)
    hist = full["history"]
    # step 3: first l with ||r_l||/||b|| < delta, strict
    first = int(np.argmax(hist < 1e-8))
    assert full["iters"] == first and hist[first] < 1e-8 and (hist[:first] >= 1e-8).all()
    assert full["relres"] == hist[-1]
    # recurrence and recomputed residual agree in fp64
    assert abs(full["true_relres"] - full["relres"]) < 1e-3 * full["relres"] + 1e-14
    cut = o.solve(1e-8, 5)
    assert cut["status"] == pbref.MAXITER and cut["iters"] == 5
    assert cut["relres"] == pytest.approx(hist[5], rel=1e-12)
    zero = pbref.PBRef(4, 4, 4, 0.5, *uniform_eps(4, 4, 4, 1.0))
    zero.set_rhs(np.zeros((4, 4, 4)), None)
    r0 = zero.solve(1e-6, 10)
    assert r0["iters"] == 0 and r0["relres"] == 0.0 and not r0["phi"].any()


def test_scale_invariance_of_iterates():
    """CG iterates are invariant under A -> cA, b -> cb; a misplaced h^-2 breaks this relation
    between two grids that differ only in h (rhs scaled accordingly)."""
    inp = random_operator(7, 6, 5, 21, salted=False)
    o1 = pbref.PBRef(7, 6, 5, 0.5, inp.eps_x, inp.eps_y, inp.eps_z, None, inp.rhs, inp.bc)
    o2 = pbref.PBRef(7, 6, 5, 1.0, inp.eps_x, inp.eps_y, inp.eps_z, None, inp.rhs / 4.0, inp.bc)
    a, b = o1.solve(1e-9, 500), o2.solve(1e-9, 500)
    assert a["iters"] == b["iters"]
    assert np.abs(a["phi"] - b["phi"]).max() <= 1e-12 * np.abs(a["phi"]).max()


# ---------------------------------------------------------------------------------------------
# discretisation order: manufactured solution with closed-form discrete error
# ---------------------------------------------------------------------------------------------
def test_manufactured_sine_closed_form_error():
    """u = sin(pi x) sin(pi y) sin(pi z) on the unit cube, eps = 1, kbar2 = 0, rhs = 3 pi^2 u.
    u is a discrete eigenvector, so phi_h = u * 3 pi^2 / lambda_h with lambda_h = (12/h^2) sin^2(pi h/2):
    max error = 3 pi^2/lambda_h - 1 ~ pi^2 h^2 / 12, ratio -> 4 under h -> h/2."""
    errs = []
    for n in (7, 15, 31):
        h = 1.0 / (n + 1)
        u = sine_mode(n, n, n, 1, 1, 1)
        o = pbref.PBRef(n, n, n, h, *uniform_eps(n, n, n, 1.0), None, 3 * math.pi ** 2 * u, None)
        res = o.solve(1e-13, 100)
        err = np.abs(res["phi"] - u).max()
        lam_h = 12.0 / h ** 2 * math.sin(math.pi * h / 2) ** 2
        assert err == pytest.approx(3 * math.pi ** 2 / lam_h - 1.0, rel=1e-9)
        errs.append(err)
    assert errs[0] / errs[1] == pytest.approx(4.0, abs=0.05)
    assert errs[1] / errs[2] == pytest.approx(4.0, abs=0.02)


def test_manufactured_variable_eps_second_order():
    """Smooth variable eps evaluated at face mid-points: error ratio -> 4 (exercises the three face
    arrays with different values per axis)."""
    def run(n):
        h = 1.0 / (n + 1)
        c = (np.arange(n) + 1) * h                       # node coordinates in (0,1)
        f = (np.arange(n + 1) + 0.5) * h                 # face mid-points
        eps = lambda x, y, z: 1.0 + 0.5 * x + 0.25 * y * y + 0.3 * np.sin(2 * z)
        Z, Y, X = np.meshgrid(c, c, f, indexing="ij"); ex = eps(X, Y, Z)
        Z, Y, X = np.meshgrid(c, f, c, indexing="ij"); ey = eps(X, Y, Z)
        Z, Y, X = np.meshgrid(f, c, c, indexing="ij"); ez = eps(X, Y, Z)
        Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
        pi = math.pi
        u = np.sin(pi * X) * np.sin(pi * Y) * np.sin(pi * Z)
        ux = pi * np.cos(pi * X) * np.sin(pi * Y) * np.sin(pi * Z)
        uy = pi * np.sin(pi * X) * np.cos(pi * Y) * np.sin(pi * Z)
        uz = pi * np.sin(pi * X) * np.sin(pi * Y) * np.cos(pi * Z)
        e = eps(X, Y, Z)
        kb = 0.7
        # -div(eps grad u) + kb u = -(eps_x ux + eps_y uy + eps_z uz) + 3 pi^2 eps u + kb u
        rhs = -(0.5 * ux + 0.5 * Y * uy + 0.6 * np.cos(2 * Z) * uz) + 3 * pi * pi * e * u + kb * u
        o = pbref.PBRef(n, n, n, h, ex, ey, ez, np.full((n, n, n), kb), rhs, None)
        return np.abs(o.solve(1e-12, 2000)["phi"] - u).max()
    e1, e2, e3 = run(7), run(15), run(31)
    assert e1 / e2 == pytest.approx(4.0, abs=0.4)
    assert e2 / e3 == pytest.approx(4.0, abs=0.15)


# ---------------------------------------------------------------------------------------------
# physics: Born ion (config 1) against the analytic potential
# ---------------------------------------------------------------------------------------------
def _golden_born():
    rows = {}
    with open(os.path.join(GOLDEN, "born_analytic.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]
                rows[k] = float(v)
    return rows


def test_born_ion_against_analytic():
    g = _golden_born()
    inp = born_ion()
    o = pbref.from_inputs(inp)
    res = o.solve(1e-10, 2000)
    assert res["status"] == pbref.OK
    phi = res["phi"]
    n, h = 33, 0.5
    c = 16
    # reaction-field potential at the ion: phi(centre) minus the same charge solved in vacuum-like
    # uniform eps_in (the grid self term cancels); analytic -(q/a)(1/eps_in - 1/eps_out)
    ex, ey, ez = uniform_eps(n, n, n, 1.0)
    vac = pbref.PBRef(n, n, n, h, ex, ey, ez, None, inp.rhs, 80.0 * inp.bc)  # q/r ghost values
    phi_vac = vac.solve(1e-10, 2000)["phi"]
    rf = phi[c, c, c] - phi_vac[c, c, c]
    assert rf == pytest.approx(g["reaction_field_e_per_A"], rel=0.05)
    # vacuum solve reproduces q/r away from the charge (0.8 % at r = 3 A)
    assert phi_vac[c, c, c + 6] == pytest.approx(1.0 / 3.0, rel=0.02)
    # exterior potential q/(eps_out r) within 2.5 % for r >= 3 A
    idx = np.arange(n) - c
    Z, Y, X = np.meshgrid(idx, idx, idx, indexing="ij")
    r = h * np.sqrt(X * X + Y * Y + Z * Z)
    m = r >= 3.0
    exact = 1.0 / (80.0 * r[m])
    assert np.abs(phi[m] / exact - 1.0).max() < 0.025
    assert phi[c, c, c + 12] == pytest.approx(g["phi_exterior_r6"], rel=0.005)
    # 48-fold cubic symmetry
    for perm in [(0, 1, 2), (1, 0, 2), (2, 1, 0), (0, 2, 1)]:
        t = phi.transpose(perm)
        assert np.abs(t - phi).max() < 1e-9 * np.abs(phi).max()
        assert np.abs(t[::-1] - phi).max() < 1e-9 * np.abs(phi).max()


def test_config2_runs_and_preconditioner_helps():
    inp = make_config(2, device="cpu")
    o = pbref.from_inputs(inp)
    pcg = o.solve(1e-5, 2000)
    cg = o.solve(1e-5, 5000, precond=False)
    assert pcg["status"] == pbref.OK and cg["status"] == pbref.OK
    assert pcg["iters"] < cg["iters"]
    assert np.abs(pcg["phi"] - cg["phi"]).max() < 1e-3 * np.abs(pcg["phi"]).max()


def test_thread_count_does_not_change_bits():
    import subprocess
    import sys
    code = ("import numpy as np, hashlib; from oracle import pbref; from workloads import random_operator;"
            "o = pbref.from_inputs(random_operator(13, 9, 7, 3)); r = o.solve(1e-9, 500);"
            "print(r['iters'], hashlib.sha256(r['phi'].tobytes()).hexdigest())")
    outs = []
    for nt in ("1", "3"):
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
        outs.append(subprocess.check_output([sys.executable, "-c", code], env=env, cwd=root))
    assert outs[0] == outs[1]


def test_initial_guess_step1_general_phi0():
    """Step 1 with a general phi_0 (r_0 = b - A phi_0), pinned against the dense direct solve:
    the exact solution as phi_0 stops at l = 0; any phi_0 converges to the same x; the first residual equals
    ||b - A phi_0|| / ||b|| computed from the dense matrix."""
    nx, ny, nz = 7, 6, 5
    inp = random_operator(nx, ny, nz, 5)
    A = dense_from_eq3(nx, ny, nz, inp.h, inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2)
    o = pbref.from_inputs(inp)
    b = o.b().ravel()
    x = np.linalg.solve(A, b)
    exact = o.solve(1e-9, 100, phi0=x.reshape(nz, ny, nx))
    assert exact["iters"] == 0 and np.array_equal(exact["phi"].ravel(), x)
    g = np.random.default_rng(1).standard_normal(x.size)
    res = o.solve(1e-12, 2000, phi0=g.reshape(nz, ny, nx), history=True)
    assert np.abs(res["phi"].ravel() - x).max() <= 1e-10 * np.abs(x).max()
    assert abs(res["history"][0] - np.linalg.norm(b - A @ g) / np.linalg.norm(b)) <= 1e-12 * res["history"][0]
    # a guess close to the solution needs fewer iterations than phi_0 = 0
    near = o.solve(1e-10, 2000, phi0=(x * (1 + 1e-4 * g)).reshape(nz, ny, nx))
    cold = o.solve(1e-10, 2000)
    assert near["iters"] < cold["iters"]
    assert np.abs(near["phi"].ravel() - x).max() <= 1e-8 * np.abs(x).max()


def _periodic_faces(inp):
    """Make face f = n equal to face f = 0 in each direction (one physical face under the periodic condition)."""
    ex, ey, ez = inp.eps_x.copy(), inp.eps_y.copy(), inp.eps_z.copy()
    ex[:, :, -1] = ex[:, :, 0]
    ey[:, -1, :] = ey[:, 0, :]
    ez[-1] = ez[0]
    return ex, ey, ez


def test_periodic_boundary_condition():
    """The paper's PBC variant, pinned by (i) the closed-form Fourier eigenpairs of
    the uniform periodic 7-point operator, (ii) a dense matrix assembled row by row from Eq. 3 with wrapped
    neighbours, (iii) symmetry, and (iv) the dense direct solve."""
    nx, ny, nz, h, eps, k2 = 8, 6, 5, 0.5, 3.0, 0.7
    ex, ey, ez = uniform_eps(nx, ny, nz, eps)
    o = pbref.PBRef(nx, ny, nz, h, ex, ey, ez, np.full((nz, ny, nx), k2))
    o.set_periodic(True)
    i, j, k = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    for (p, q, r) in [(0, 0, 0), (1, 0, 0), (2, 1, 3), (3, 2, 1)]:
        for fn in (np.cos, np.sin):
            v = fn(2 * np.pi * (p * i / nx + q * j / ny + r * k / nz)).transpose(2, 1, 0)
            lam = 4 * eps / h ** 2 * (np.sin(np.pi * p / nx) ** 2 + np.sin(np.pi * q / ny) ** 2
                                      + np.sin(np.pi * r / nz) ** 2) + k2
            assert np.abs(o.apply(v) - lam * v).max() <= 1e-12 * max(lam, 1.0)
    inp = random_operator(6, 5, 4, 9)
    ex, ey, ez = _periodic_faces(inp)
    A = dense_from_eq3(6, 5, 4, inp.h, ex, ey, ez, inp.kbar2, periodic=True)
    assert np.array_equal(A, A.T) and np.linalg.eigvalsh(A).min() > 0
    o = pbref.PBRef(6, 5, 4, inp.h, ex, ey, ez, inp.kbar2)
    o.set_periodic(True)
    o.set_rhs(inp.rhs, inp.bc)                         # ghost values are ignored under the periodic condition
    assert np.array_equal(o.b(), inp.rhs)
    x = np.random.default_rng(2).standard_normal((4, 5, 6))
    assert np.abs(o.apply(x).ravel() - A @ x.ravel()).max() <= 1e-11 * np.abs(A @ x.ravel()).max()
    res = o.solve(1e-12, 2000)
    sol = np.linalg.solve(A, inp.rhs.ravel())
    assert res["status"] == pbref.OK and np.abs(res["phi"].ravel() - sol).max() <= 1e-10 * np.abs(sol).max()
