"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances are BASELINE.json's north_star: fp64 SpMV 1e-12 (componentwise backward measure, DESIGN.md
Reading 20), fp64 solve to 1e-10 within 1e-8 max|phi|, fp32 solve to 1e-5 within 1e-4 max|phi|,
iteration counts within 5 % (at least +-1).
"""
import numpy as np
import pytest

from tests.helpers import sine_eigenvalue, sine_mode, uniform_eps
from workloads import born_ion, make_config, random_operator

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg(cuda_device):
    from paper_1704_02745_b200 import build as pb_build

    pb_build.build()
    import paper_1704_02745_b200 as p

    p.load_library()          # fail loudly if the extension is missing
    return p


@pytest.fixture(scope="module")
def pbref():
    from oracle import pbref as m

    return m


def backward_bound(inp, x, periodic=False):
    """(D|x| + sum_f eps_f |x_nbr|)/h^2 per node: the scale of the terms of one row of Eq. 3 (DESIGN.md Reading 20).
    Periodic: the neighbour across a box face is the node on the opposite side, so its
    |x| counts too (wrap padding instead of the zero ghost layer)."""
    ax = np.abs(x)
    p = np.pad(ax, 1, mode="wrap") if periodic else np.pad(ax, 1)
    ex, ey, ez = inp.eps_x, inp.eps_y, inp.eps_z
    s = (ex[:, :, :-1] * (p[1:-1, 1:-1, :-2] + ax) + ex[:, :, 1:] * (p[1:-1, 1:-1, 2:] + ax)
         + ey[:, :-1, :] * (p[1:-1, :-2, 1:-1] + ax) + ey[:, 1:, :] * (p[1:-1, 2:, 1:-1] + ax)
         + ez[:-1, :, :] * (p[:-2, 1:-1, 1:-1] + ax) + ez[1:, :, :] * (p[2:, 1:-1, 1:-1] + ax))
    return s / inp.h ** 2 + inp.kbar2 * ax


SPMV_SHAPES = [(1, 1, 1), (2, 1, 3), (13, 9, 7), (33, 31, 29), (77, 97, 99), (130, 21, 37), (263, 19, 18),
               (524, 6, 5)]


@pytest.mark.parametrize("shape", SPMV_SHAPES)
def test_spmv_fp64_matches_oracle(pkg, pbref, shape):
    nx, ny, nz = shape
    inp = random_operator(nx, ny, nz, seed=nx + ny + nz, two_valued=(nx % 2 == 1))
    x = np.random.default_rng(5 + nx).uniform(-1, 1, (nz, ny, nx))
    ref = pbref.from_inputs(inp)
    with pkg.PBSolver(*inp.args()) as s:
        y = s.apply(x, "f64")
        yr = ref.apply(x)
        bound = backward_bound(inp, x)
        assert np.all(np.abs(y - yr) <= 1e-12 * bound + 1e-300), np.max(np.abs(y - yr) / (bound + 1e-300))
        assert np.max(np.abs(y - yr)) <= 1e-13 * np.max(np.abs(yr))
        # derived setup quantities (row a0): diagonal and folded right-hand side
        np.testing.assert_allclose(s.diag(), ref.diag(), rtol=1e-14, atol=0)
        np.testing.assert_allclose(s.b(), ref.b(), rtol=1e-13, atol=1e-13 * np.max(np.abs(ref.b())))
    ref.close()


@pytest.mark.parametrize("shape", [(13, 9, 7), (77, 97, 99), (130, 21, 37)])
def test_spmv_fp32_matches_oracle(pkg, pbref, shape):
    nx, ny, nz = shape
    inp = random_operator(nx, ny, nz, seed=3)
    x = np.random.default_rng(9).uniform(-1, 1, (nz, ny, nx)).astype(np.float32)
    ref = pbref.from_inputs(inp)
    with pkg.PBSolver(*inp.args()) as s:
        y = s.apply(x, "f32")
        assert y.dtype == np.float32
        yr = ref.apply(x.astype(np.float64))
        bound = backward_bound(inp, x.astype(np.float64))
        assert np.all(np.abs(y - yr) <= 8 * 6e-8 * bound)
    ref.close()


def test_spmv_eigenvector_closed_form(pkg):
    """Independent of the oracle: uniform eps, kbar2 = k -> A v_pqr = lambda_pqr v_pqr (closed form)."""
    nx, ny, nz, h, eps, k2 = 21, 14, 9, 0.5, 3.0, 0.7
    ex, ey, ez = uniform_eps(nx, ny, nz, eps)
    with pkg.PBSolver(nx, ny, nz, h, ex, ey, ez, np.full((nz, ny, nx), k2)) as s:
        for (p, q, r) in [(1, 1, 1), (3, 2, 5), (nx, ny, nz)]:
            v = sine_mode(nx, ny, nz, p, q, r)
            lam = sine_eigenvalue(nx, ny, nz, h, eps, k2, p, q, r)
            assert np.max(np.abs(s.apply(v) - lam * v)) <= 5e-14 * lam


def test_spmv_device_pointers(pkg, pbref, cuda_device):
    import torch

    inp = random_operator(45, 23, 11, seed=8)
    ref = pbref.from_inputs(inp)
    dev = [torch.from_numpy(np.ascontiguousarray(a)).to(cuda_device) for a in
           (inp.eps_x, inp.eps_y, inp.eps_z, inp.kbar2, inp.rhs, inp.bc)]
    x = np.random.default_rng(1).uniform(-1, 1, (inp.nz, inp.ny, inp.nx))
    with pkg.PBSolver(inp.nx, inp.ny, inp.nz, inp.h, *dev) as s:
        y = s.apply(torch.from_numpy(x).to(cuda_device))
        assert y.is_cuda
        yr = ref.apply(x)
        assert np.max(np.abs(y.cpu().numpy() - yr)) <= 1e-13 * np.max(np.abs(yr))
        out = torch.empty((inp.nz, inp.ny, inp.nx), dtype=torch.float64, device=cuda_device)
        g = s.solve(1e-10, 5000, "f64", out=out)
        o = ref.solve(1e-10, 5000)
        assert g["status"] == 0
        assert np.max(np.abs(out.cpu().numpy() - o["phi"])) <= 1e-8 * np.max(np.abs(o["phi"]))
    ref.close()


# the three ways pb_solve can run an iteration: the default choice (cooperative kernel on L2-resident grids, else
# k_pcg_fused), one fused kernel per iteration forced (persist = 0), K_spmv + K_vec forced (persist = 0, fused = 0)
PATHS = {"default": None, "fused": dict(persist=0), "two-kernel": dict(persist=0, fused=0)}


def check_solve(pkg, pbref, inp, prec, tol, maxiter=20000, check_every=16, options=None):
    ref = pbref.from_inputs(inp)
    o = ref.solve(tol, maxiter)
    o_tight = ref.solve(1e-10, maxiter) if tol > 1e-10 else o
    with pkg.PBSolver(*inp.args(), options=options) as s:
        g = s.solve(tol, maxiter, prec, check_every=check_every)
        if options is not None:
            pl = s.plan(prec)
            assert pl["persist"] == 0 and pl["fused"] == options.get("fused", 1), pl
    ref.close()
    scale = np.max(np.abs(o_tight["phi"]))
    lim = 1e-8 if prec == "f64" and tol <= 1e-10 else 1e-4
    assert g["status"] == 0 and o["status"] == 0
    assert g["relres"] < tol
    assert abs(g["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (g["iters"], o["iters"])
    err = np.max(np.abs(g["phi"] - o["phi"])) / scale
    err_t = np.max(np.abs(g["phi"] - o_tight["phi"])) / scale
    assert err <= lim and err_t <= lim, (err, err_t)
    return g, o


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("shape", [(5, 4, 3), (13, 9, 7), (33, 31, 29), (130, 21, 37)])
def test_solve_fp64_random(pkg, pbref, shape, path):
    check_solve(pkg, pbref, random_operator(*shape, seed=11, two_valued=(shape[0] != 130)), "f64", 1e-10, options=PATHS[path])


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("shape", [(13, 9, 7), (33, 31, 29), (130, 21, 37)])
def test_solve_fp32_random(pkg, pbref, shape, path):
    check_solve(pkg, pbref, random_operator(*shape, seed=12, two_valued=(shape[0] != 130)), "f32", 1e-5, options=PATHS[path])


def test_solve_born_config1(pkg, pbref):
    g, o = check_solve(pkg, pbref, born_ion(), "f64", 1e-10)
    # physics pin repeated on the GPU result: reaction field at the ion within 5 % of -0.49375 e/A
    inp = born_ion()
    c = 16
    ex, ey, ez = uniform_eps(33, 33, 33, 1.0)
    from workloads.pb_inputs import debye_huckel_ghost

    bc = debye_huckel_ghost(33, 33, 33, 0.5, inp.meta["centres"], inp.meta["charges"], 1.0, 0.0, device="cpu")
    with pkg.PBSolver(33, 33, 33, 0.5, ex, ey, ez, None, inp.rhs, bc) as s:
        vac = s.solve(1e-10, 5000, "f64")
    rf = g["phi"][c, c, c] - vac["phi"][c, c, c]
    assert abs(rf - (-0.49375)) <= 0.05 * 0.49375


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_solve_config2_65(pkg, pbref, prec, tol, path):
    check_solve(pkg, pbref, make_config(2), prec, tol, options=PATHS[path])


@pytest.mark.slow
def test_solve_config3_129_fp32(pkg, pbref):
    check_solve(pkg, pbref, make_config(3), "f32", 1e-5, check_every=32)


def test_edge_zero_rhs_maxiter_and_latch(pkg, pbref):
    inp = random_operator(19, 11, 6, seed=4)
    ref = pbref.from_inputs(inp)
    with pkg.PBSolver(*inp.args()) as s:
        # maxiter hit: same iterate as the oracle stopped at the same l
        g = s.solve(1e-12, 7, "f64", check_every=3)
        o = ref.solve(1e-12, 7)
        assert g["status"] == pkg.binding.PB_ERR_MAXITER and o["status"] == pbref.MAXITER
        assert g["iters"] == 7 == o["iters"]
        assert np.max(np.abs(g["phi"] - o["phi"])) <= 1e-10 * np.max(np.abs(o["phi"]))
        assert abs(g["relres"] - o["relres"]) <= 1e-8 * o["relres"]
        g0 = s.solve(1e-6, 0, "f64")
        assert g0["status"] == pkg.binding.PB_ERR_MAXITER and g0["iters"] == 0 and not g0["phi"].any()
        # the returned iterate does not depend on how often the host polls; bitwise run-to-run determinism
        runs = [s.solve(1e-9, 5000, "f64", check_every=ce) for ce in (1, 5, 64, 5)]
        for r in runs[1:]:
            assert r["iters"] == runs[0]["iters"] and r["relres"] == runs[0]["relres"]
            assert np.array_equal(r["phi"], runs[0]["phi"])
        # b = 0 -> phi = 0, iters = 0, relres = 0
        s.set_rhs(None, None)
        z = s.solve(1e-6, 100, "f32")
        assert z["status"] == 0 and z["iters"] == 0 and z["relres"] == 0.0 and not z["phi"].any()
        # same operator, new right-hand side (pb_set_rhs)
        inp2 = random_operator(19, 11, 6, seed=5)
        s.set_rhs(inp2.rhs, inp2.bc)
        ref.set_rhs(inp2.rhs, inp2.bc)
        g2, o2 = s.solve(1e-10, 5000, "f64"), ref.solve(1e-10, 5000)
        assert np.max(np.abs(g2["phi"] - o2["phi"])) <= 1e-8 * np.max(np.abs(o2["phi"]))
    ref.close()


def test_edge_not_spd_and_bad_args(pkg):
    inp = random_operator(6, 5, 4, seed=2, salted=False)
    ex = inp.eps_x.copy()
    ex[:] = 0.0
    ey, ez = np.zeros_like(inp.eps_y), np.zeros_like(inp.eps_z)
    with pytest.raises(pkg.PBError) as e:
        pkg.PBSolver(6, 5, 4, 0.5, ex, ey, ez)
    assert e.value.status == pkg.binding.PB_ERR_NOT_SPD
    with pkg.PBSolver(*inp.args()) as s:
        with pytest.raises(pkg.PBError):
            s.solve(-1.0, 10)
        with pytest.raises(pkg.PBError):
            s.solve(1e-5, 10, check_every=0)


def test_fp32_true_residual_reported(pkg, pbref):
    """fp32 storage: the recurrence residual passes 1e-5 and the true residual b - A phi (computed by the
    oracle in fp64 from the GPU's phi) stays of the same order (SURVEY hard part 4)."""
    inp = make_config(2)
    ref = pbref.from_inputs(inp)
    with pkg.PBSolver(*inp.args()) as s:
        g = s.solve(1e-5, 5000, "f32")
    b = ref.b()
    true = np.linalg.norm(b - ref.apply(g["phi"].astype(np.float64))) / np.linalg.norm(b)
    ref.close()
    assert true < 5e-5, true


@pytest.mark.slow
def test_fullsize_385_spmv_and_solve_properties(pkg, pbref):
    """BASELINE.json's full size (385^3) in the launch configuration bench.py times: SpMV compared
    element by element with the oracle (one pass is cheap), the fp32 solve checked by properties
    that hold at any size: recurrence residual < tol, true residual (oracle arithmetic) small."""
    n = 385
    inp = random_operator(n, n, n, seed=385, two_valued=True)
    ref = pbref.from_inputs(inp)
    x = np.random.default_rng(385).uniform(-1, 1, (n, n, n))
    with pkg.PBSolver(*inp.args()) as s:
        y = s.apply(x, "f64")
        yr = ref.apply(x)
        assert np.max(np.abs(y - yr)) <= 1e-13 * np.max(np.abs(yr))
        bound = backward_bound(inp, x)
        assert np.all(np.abs(y - yr) <= 1e-12 * bound)
        del y, yr, bound, x
        g = s.solve(1e-5, 5000, "f32", check_every=32)
        assert g["status"] == 0 and g["relres"] < 1e-5
        b = ref.b()
        true = np.linalg.norm(b - ref.apply(g["phi"].astype(np.float64))) / np.linalg.norm(b)
        assert true < 1e-4, true
    ref.close()


# per-handle options (pb_set_option): forced tiles / rings / grids of k_spmv_tma, the static plan, the autotuned plan
TILE_CONFIGS = [dict(autotune=0), dict(tile_txv=7, tile_ty=3, ring_slots=3, blocks_per_sm=2, tile_tz=5),
                dict(tile_txv=20, tile_ty=8, ring_slots=6, blocks_per_sm=1, tile_tz=99),
                dict(tile_txv=5, tile_ty=2, ring_slots=4, blocks_per_sm=4, tile_tz=1),
                dict(tile_txv=13, tile_ty=5, ring_slots=5, blocks_per_sm=3, tile_tz=33), dict()]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_tiling_independence(pkg, pbref, prec):
    """Every tile / ring / grid configuration of k_spmv_tma (halo boxes, TMA zero fill, ring hand-off, ragged
    tiles) must give the SAME SpMV bit for bit -- a node's arithmetic does not depend on the tiling -- and
    solves that agree with the oracle.  (compute-sanitizer is closed on this pool; this is the race/halo check.)"""
    inp = random_operator(77, 45, 38, seed=21)
    dt = np.float64 if prec == "f64" else np.float32
    x = np.random.default_rng(2).uniform(-1, 1, (inp.nz, inp.ny, inp.nx)).astype(dt)
    ref = pbref.from_inputs(inp)
    tol = 1e-10 if prec == "f64" else 1e-5
    o = ref.solve(tol, 5000)
    scale = np.max(np.abs(o["phi"]))
    y0 = None
    for cfg in TILE_CONFIGS:
        # small grid: persist=0 forces the two-kernel TMA path under test
        with pkg.PBSolver(*inp.args(), options=dict(cfg, persist=0, fused=0)) as s:
            y = s.apply(x, prec)
            runs = [s.solve(tol, 5000, prec, check_every=9) for _ in range(2)]
            plan = s.plan(prec)
        if "tile_txv" in cfg:
            assert (plan["txv"], plan["ty"], plan["ring_slots"], plan["blocks_per_sm"]) == (
                cfg["tile_txv"], cfg["tile_ty"], cfg["ring_slots"], cfg["blocks_per_sm"]), (cfg, plan)
            assert plan["tz"] == min(cfg["tile_tz"], inp.nz) and not plan["autotuned"] and not plan["persist"]
        if y0 is None:
            y0 = y
        assert np.array_equal(y, y0), cfg
        assert np.array_equal(runs[0]["phi"], runs[1]["phi"]) and runs[0]["iters"] == runs[1]["iters"], cfg
        assert abs(runs[0]["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), cfg
        assert np.max(np.abs(runs[0]["phi"] - o["phi"])) <= (1e-8 if prec == "f64" else 1e-4) * scale, cfg
    ref.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_tiling_independence_with_both_palettes(pkg, prec):
    """k_spmv_tma with the face palette AND Dinv read through the diagonal palette (haloed byte box, every lead-in
    0/4/8/12 of the 16-byte aligned box start under the forced tilings): the SpMV and one PCG step's vectors must be
    bit-identical across tilings and identical to the word formats (PB_PALETTE_DS=0, PB_PALETTE=0)."""
    inp = random_operator(77, 45, 38, seed=33, salted=False, two_valued=True)      # kbar2 = 0: few distinct diagonals
    dt = np.float64 if prec == "f64" else np.float32
    x = np.random.default_rng(5).uniform(-1, 1, (inp.nz, inp.ny, inp.nx)).astype(dt)
    ref_y = ref_p = ref_ap = None
    for fmt in (dict(), dict(palette_diag_spmv=0), dict(palette=0)):
        for cfg in TILE_CONFIGS:
            with pkg.PBSolver(*inp.args(), options={**cfg, **fmt, "persist": 0, "fused": 0}) as s:
                y = s.apply(x, prec)
                if not fmt:
                    assert s.palette_size() > 0 and s.diag_palette_size() > 0
                    assert s.bytes_per_node(prec, 0) == 6 * x.itemsize + 4
                s.solve_begin(prec)
                s.iterate(prec, 2)
                p2, ap2 = s.vector("p"), s.vector("Ap")
            if ref_y is None:
                ref_y, ref_p, ref_ap = y, p2, ap2
            assert np.array_equal(y, ref_y), (fmt, cfg)
            # p and Ap after two iterations: alpha/beta come from tiling-dependent summation orders, so compare
            # to rounding, not bitwise
            eps = 1e-5 if prec == "f32" else 1e-13
            assert np.max(np.abs(p2 - ref_p)) <= eps * np.max(np.abs(ref_p)), (fmt, cfg)
            assert np.max(np.abs(ap2 - ref_ap)) <= eps * np.max(np.abs(ref_ap)), (fmt, cfg)


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_unpreconditioned_cg_variant(pkg, pbref, prec, tol):
    """NEXT row f3: the paper's GPU/CG = the same recurrence with M = I.  Same parity bar;
    and Jacobi needs fewer iterations than CG on heterogeneous eps."""
    inp = born_ion()
    ref = pbref.from_inputs(inp)
    o_cg = ref.solve(tol, 5000, precond=False)
    o_pcg = ref.solve(tol, 5000, precond=True)
    with pkg.PBSolver(*inp.args()) as s:
        s.set_preconditioner(False)
        g_cg = s.solve(tol, 5000, prec)
        s.set_preconditioner(True)
        g_pcg = s.solve(tol, 5000, prec)
    ref.close()
    scale = np.max(np.abs(o_pcg["phi"]))
    lim = 1e-8 if prec == "f64" else 1e-4
    for g, o in ((g_cg, o_cg), (g_pcg, o_pcg)):
        assert g["status"] == 0
        assert abs(g["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (g["iters"], o["iters"])
        assert np.max(np.abs(g["phi"] - o["phi"])) <= lim * scale
    assert g_pcg["iters"] < g_cg["iters"]


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_palette_and_full_precision_coefficients_agree(pkg, pbref, prec, tol):
    """The coefficient palette (<= 256 distinct face values stored as bytes + table) is an exact storage format:
    the SpMV must be bit-identical with the full-precision face arrays (PB_PALETTE=0), and operators with more
    than 256 distinct values must fall back to them."""
    inp = make_config(2)                       # molecular map: eps in {1, 80, 160/81}
    x = np.random.default_rng(4).uniform(-1, 1, (inp.nz, inp.ny, inp.nx)).astype(np.float64 if prec == "f64" else np.float32)
    with pkg.PBSolver(*inp.args()) as s:
        y_pal = s.apply(x, prec)
        assert s.palette_size() == 4       # the three face values and the pad value 0
        g_pal = s.solve(tol, 5000, prec)
        # the same handle with the palette switched off: work arrays and plan are rebuilt (options are handle state)
        s.set_option("palette", 0)
        y_full = s.apply(x, prec)
        assert s.palette_size() == 0 and s.get_option("palette") == 0
        g_full = s.solve(tol, 5000, prec)
    assert np.array_equal(y_pal, y_full)
    assert abs(g_pal["iters"] - g_full["iters"]) <= 1
    assert np.max(np.abs(g_pal["phi"] - g_full["phi"])) <= (1e-9 if prec == "f64" else 1e-4) * np.max(np.abs(g_full["phi"]))
    many = random_operator(21, 9, 8, seed=6, two_valued=False)      # ~5000 distinct face values
    with pkg.PBSolver(*many.args()) as s:
        s.prepare(prec)
        assert s.palette_size() == 0


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_warm_start_matches_oracle(pkg, pbref, prec, tol, path):
    """NEXT row f2 (part): pb_solve_from = step 1 with a given phi_0.  Snapshot-style use: solve,
    perturb the charges (new rhs and ghost values), restart from the previous potential.  Iteration counts and
    potentials must match the oracle run from the same phi_0; the restart must need fewer iterations.  On each of the
    three solve paths (the fused one takes its warm start through the same k_warm step as the two-kernel one)."""
    inp = make_config(2)
    from workloads import perturbed_charges

    rhs2, bc2 = perturbed_charges(inp, 0, device="cpu")
    ref = pbref.from_inputs(inp)
    dt = np.float64 if prec == "f64" else np.float32
    with pkg.PBSolver(*inp.args(), options=PATHS[path]) as s:
        if path == "fused":
            assert s.plan(prec)["fused"] == 1
        first = s.solve(tol, 5000, prec)
        s.set_rhs(rhs2, bc2)
        ref.set_rhs(rhs2, bc2)
        cold = s.solve(tol, 5000, prec)
        warm = s.solve(tol, 5000, prec, phi0=first["phi"].copy())
        again = s.solve(tol, 5000, prec, phi0=warm["phi"].astype(dt))       # already converged -> 0 or 1 iterations
    o_warm = ref.solve(tol, 5000, phi0=first["phi"].astype(np.float64))
    o_cold = ref.solve(tol, 5000)
    ref.close()
    scale = np.max(np.abs(o_cold["phi"]))
    lim = 1e-8 if prec == "f64" else 1e-4
    assert warm["status"] == 0 and warm["relres"] < tol
    assert abs(warm["iters"] - o_warm["iters"]) <= max(1, round(0.05 * o_warm["iters"])), (warm["iters"], o_warm["iters"])
    assert np.max(np.abs(warm["phi"] - o_warm["phi"])) <= lim * scale
    assert np.max(np.abs(warm["phi"] - cold["phi"])) <= 10 * lim * scale
    assert warm["iters"] < cold["iters"]
    assert again["iters"] <= 1


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_persistent_and_two_kernel_paths_agree(pkg, pbref, prec, tol):
    """NEXT row f2 (part): L2-resident grids run steps 3-8 in one cooperative kernel (k_pcg_persistent); larger ones
    (or PB_PERSIST=0) through k_spmv_tma + k_vec.  Both must meet the oracle bar, agree with each other, stop on
    maxiter identically, honour the M = I variant and a warm start, and be bitwise repeatable."""
    inp = make_config(2)
    ref = pbref.from_inputs(inp)
    o = ref.solve(tol, 5000)
    o_cg = ref.solve(tol, 5000, precond=False)
    o7 = ref.solve(tol, 7)
    ref.close()
    scale = np.max(np.abs(o["phi"]))
    lim = 1e-8 if prec == "f64" else 1e-4
    res = {}
    for mode in ("1", "0"):
        with pkg.PBSolver(*inp.args(), options=dict(persist=int(mode))) as s:
            a, b = s.solve(tol, 5000, prec), s.solve(tol, 5000, prec)
            assert s.plan(prec)["persist"] == int(mode)
            assert np.array_equal(a["phi"], b["phi"]) and a["iters"] == b["iters"]
            m7 = s.solve(tol, 7, prec)
            w = s.solve(tol, 5000, prec, phi0=a["phi"].copy())
            s.set_preconditioner(False)
            cg = s.solve(tol, 5000, prec)
        res[mode] = (a, m7, cg, w)
    for a, m7, cg, w in res.values():
        assert a["status"] == 0 and abs(a["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"]))
        assert np.max(np.abs(a["phi"] - o["phi"])) <= lim * scale
        assert m7["status"] == pkg.binding.PB_ERR_MAXITER and m7["iters"] == 7
        assert np.max(np.abs(m7["phi"] - o7["phi"])) <= lim * scale
        assert abs(cg["iters"] - o_cg["iters"]) <= max(1, round(0.05 * o_cg["iters"]))
        assert w["iters"] <= 1
    assert np.max(np.abs(res["1"][0]["phi"] - res["0"][0]["phi"])) <= lim * scale


@pytest.mark.slow
def test_config5_headline_parity_full_size(pkg, pbref):
    """BASELINE.json configs[4] (385^3, 60 000 atoms) exactly as bench.py runs it (autotuned plan, palette,
    check_every 32): the fp32 solve to 1e-5 and the fp64 solve to 1e-10 against the full oracle solves -- every node,
    the north-star tolerances.  (The oracle needs about a minute on the GPU box's host cores.)"""
    inp = make_config(5, device="cuda")
    ref = pbref.from_inputs(inp)
    o32 = ref.solve(1e-5, 5000)
    o64 = ref.solve(1e-10, 5000)
    ref.close()
    scale = np.max(np.abs(o64["phi"]))
    with pkg.PBSolver(*inp.args()) as s:
        g32 = s.solve(1e-5, 20000, "f32", check_every=32)
        g64 = s.solve(1e-10, 20000, "f64", check_every=32)
        assert s.palette_size() == 4
    assert g32["status"] == 0 and g64["status"] == 0
    assert abs(g32["iters"] - o32["iters"]) <= round(0.05 * o32["iters"]), (g32["iters"], o32["iters"])
    assert abs(g64["iters"] - o64["iters"]) <= round(0.05 * o64["iters"]), (g64["iters"], o64["iters"])
    e32 = np.max(np.abs(g32["phi"] - o32["phi"])) / scale
    e32t = np.max(np.abs(g32["phi"] - o64["phi"])) / scale
    e64 = np.max(np.abs(g64["phi"] - o64["phi"])) / scale
    print(f"config5: fp32 iters {g32['iters']} (oracle {o32['iters']}) err {e32:.2e} / {e32t:.2e}; "
          f"fp64 iters {g64['iters']} (oracle {o64['iters']}) err {e64:.2e}")
    assert e32 <= 1e-4 and e32t <= 1e-4 and e64 <= 1e-8


def _periodic_inputs(shape, seed):
    inp = random_operator(*shape, seed=seed)
    inp.eps_x[:, :, -1] = inp.eps_x[:, :, 0]        # face f = n is face f = 0 under the periodic condition
    inp.eps_y[:, -1, :] = inp.eps_y[:, 0, :]
    inp.eps_z[-1] = inp.eps_z[0]
    return inp


@pytest.mark.parametrize("shape", [(1, 1, 1), (2, 3, 1), (13, 9, 7), (77, 45, 38), (130, 21, 37)])
def test_periodic_boundary_spmv(pkg, pbref, shape):
    """NEXT row f3: the paper's PBC variant -- index wraps instead of ghost zeros."""
    nx, ny, nz = shape
    inp = _periodic_inputs(shape, 31)
    ref = pbref.from_inputs(inp)
    ref.set_periodic(True)
    x = np.random.default_rng(3).uniform(-1, 1, (nz, ny, nx))
    with pkg.PBSolver(*inp.args()) as s:
        y_dir = s.apply(x, "f64")
        s.set_periodic(True)
        y = s.apply(x, "f64")
        y32 = s.apply(x.astype(np.float32), "f32")
        s.set_periodic(False)
        assert np.array_equal(s.apply(x, "f64"), y_dir)
    yr = ref.apply(x)
    bound = backward_bound(inp, x, periodic=True) + 1e-300
    assert np.all(np.abs(y - yr) <= 1e-12 * bound)
    assert np.all(np.abs(y32 - yr) <= 2e-6 * bound)
    ref.close()


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
@pytest.mark.parametrize("persist", ["1", "0"])
def test_periodic_boundary_solve(pkg, pbref, prec, tol, persist):
    inp = _periodic_inputs((45, 23, 19), 32)
    ref = pbref.from_inputs(inp)
    ref.set_periodic(True)
    ref.set_rhs(inp.rhs, inp.bc)
    o = ref.solve(tol, 5000)
    ref.close()
    with pkg.PBSolver(*inp.args(), options=dict(persist=int(persist))) as s:
        s.set_periodic(True)
        assert np.allclose(s.b(), inp.rhs, rtol=1e-14)       # no ghost fold-in
        g = s.solve(tol, 5000, prec, check_every=8)
        g2 = s.solve(tol, 5000, prec, check_every=8)
    scale = np.max(np.abs(o["phi"]))
    assert g["status"] == 0 and abs(g["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (g["iters"], o["iters"])
    assert np.max(np.abs(g["phi"] - o["phi"])) <= (1e-8 if prec == "f64" else 1e-4) * scale
    assert np.array_equal(g["phi"], g2["phi"])


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_diagonal_palette_is_exact(pkg, prec, tol):
    """k_vec reading Dinv through the diagonal palette (index byte + table of (T)(1/d)) must reproduce the Dinv-array
    run bit for bit; an operator whose salt map varies from node to node must fall back to the array."""
    inp = make_config(2)
    # persist=0: the two-kernel path is the one that uses k_vec; autotune=0: the same static plan in both runs,
    # hence the same reduction order
    with pkg.PBSolver(*inp.args(), options=dict(persist=0, autotune=0, fused=0)) as s:
        a = s.solve(tol, 5000, prec)
        assert 0 < s.diag_palette_size() <= 56 and s.plan(prec)["diag_palette_vec"] == 1
        s.set_option("palette_diag", 0)
        b = s.solve(tol, 5000, prec)
        assert s.diag_palette_size() == 0 and s.plan(prec)["diag_palette_vec"] == 0
    many = random_operator(21, 9, 8, seed=6, two_valued=True, salted=True)    # kbar2 ~ U[0,2] per node
    with pkg.PBSolver(*many.args()) as s:
        s.prepare(prec)
        assert s.palette_size() > 0 and s.diag_palette_size() == 0
    assert a["iters"] == b["iters"] and np.array_equal(a["phi"], b["phi"])


def test_randomised_shapes_and_options(pkg, pbref):
    """Seeded sweep over odd shapes and every switch (periodic / Dirichlet, Jacobi / M = I, palette or not, persistent
    or two-kernel path, fp32 / fp64, warm start): SpMV within the componentwise bound, solves within the north-star
    tolerances of the oracle run with the same options."""
    rng = np.random.default_rng(20260704)
    for case in range(24):
        nx, ny, nz = (int(v) for v in rng.integers(1, 41, 3))
        periodic, jacobi, two_valued = bool(rng.integers(2)), bool(rng.integers(2)), bool(rng.integers(2))
        persist, prec = int(rng.integers(2)), ("f64", "f32")[int(rng.integers(2))]
        inp = _periodic_inputs((nx, ny, nz), 100 + case) if periodic else random_operator(nx, ny, nz, seed=100 + case)
        if not two_valued:
            inp.eps_x[...] = rng.uniform(1, 80, inp.eps_x.shape)
            if periodic:
                inp.eps_x[:, :, -1] = inp.eps_x[:, :, 0]
        tol = 1e-10 if prec == "f64" else 1e-5
        ref = pbref.from_inputs(inp)
        ref.set_periodic(periodic)
        ref.set_rhs(inp.rhs, inp.bc)
        o = ref.solve(tol, 4000, precond=jacobi)
        x = rng.uniform(-1, 1, (nz, ny, nx))
        yr = ref.apply(x)
        with pkg.PBSolver(*inp.args(), options=dict(persist=persist)) as s:
            s.set_periodic(periodic)
            s.set_preconditioner(jacobi)
            y = s.apply(x.astype(np.float64 if prec == "f64" else np.float32), prec)
            g = s.solve(tol, 4000, prec, check_every=int(rng.integers(1, 40)))
            w = s.solve(tol, 4000, prec, phi0=g["phi"].copy())
        ref.close()
        tag = (case, nx, ny, nz, periodic, jacobi, two_valued, persist, prec)
        bound = backward_bound(inp, x, periodic=periodic) + 1e-300
        assert np.all(np.abs(y - yr) <= (1e-12 if prec == "f64" else 2e-6) * bound), tag
        assert g["status"] == o["status"] == 0, tag
        assert abs(g["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), tag + (g["iters"], o["iters"])
        scale = np.max(np.abs(o["phi"])) + 1e-300
        assert np.max(np.abs(g["phi"] - o["phi"])) <= (1e-8 if prec == "f64" else 1e-4) * scale, tag
        assert w["iters"] <= 1, tag


def test_true_residual_matches_oracle(pkg, pbref):
    """pb_residual = ||b - A phi|| / ||b|| against the oracle's recomputed residual (Reading 5), and the fp32 story of
    SURVEY hard part 4: the recurrence residual passes 1e-7 while the true residual of the fp32 iterate stagnates."""
    inp = make_config(2)
    ref = pbref.from_inputs(inp)
    o = ref.solve(1e-6, 5000)
    b = ref.b()
    with pkg.PBSolver(*inp.args()) as s:
        assert abs(s.residual(o["phi"], "f64") - o["true_relres"]) <= 1e-6 * o["true_relres"]
        assert s.residual(np.zeros_like(o["phi"]), "f64") == 1.0
        g = s.solve(1e-7, 5000, "f32")
        t32 = s.residual(g["phi"], "f32")
        t64 = s.residual(g["phi"].astype(np.float64), "f64")
    true = np.linalg.norm(b - ref.apply(g["phi"].astype(np.float64))) / np.linalg.norm(b)
    ref.close()
    assert g["relres"] < 1e-7 < true                      # fp32 storage: recurrence below, truth above
    assert abs(t64 - true) <= 1e-6 * true and abs(t32 - true) <= 0.2 * true


@pytest.mark.parametrize("path", ["default", "fused"])
@pytest.mark.parametrize("cfg", [2, "born", "random"])
def test_mixed_precision_refinement_matches_fp64_oracle(pkg, pbref, cfg, path):
    """NEXT row f3 (fp32-inner / fp64-outer iterative refinement): the result is the solution of A phi = b to 1e-10 on
    the TRUE residual -- same bar as the fp64 solve (within 1e-8 max|phi| of the oracle run to 1e-10) -- although every
    PCG iteration ran in fp32; a plain fp32 solve cannot get there (its true residual stagnates near 1e-6)."""
    inp = make_config(2) if cfg == 2 else born_ion() if cfg == "born" else random_operator(45, 31, 38, seed=8)
    ref = pbref.from_inputs(inp)
    o = ref.solve(1e-10, 5000)
    b = ref.b()
    with pkg.PBSolver(*inp.args(), options=PATHS[path]) as s:      # "fused": the corrections run through k_pcg_fused
        g = s.solve_refined(1e-10, 5000)
        assert g["status"] == 0 and g["relres"] <= 1e-10 and 2 <= g["outer"] <= 6
        assert abs(s.residual(g["phi"], "f64") - g["relres"]) <= 1e-3 * g["relres"] + 1e-16
        f = s.solve(1e-10, 5000, "f32")                      # wf.b must have been rebuilt after the refinement
        d = s.solve(1e-10, 5000, "f64")
    true = np.linalg.norm(b - ref.apply(g["phi"])) / np.linalg.norm(b)
    ref.close()
    scale = np.max(np.abs(o["phi"]))
    assert true <= 2e-10
    assert np.max(np.abs(g["phi"] - o["phi"])) <= 1e-8 * scale
    assert np.max(np.abs(d["phi"] - o["phi"])) <= 1e-8 * scale
    assert np.max(np.abs(f["phi"] - o["phi"])) <= 1e-4 * scale
    assert g["iters"] <= 4 * o["iters"]


@pytest.mark.parametrize("persist", ["0", "1"])
def test_refinement_periodic_and_two_kernel_path(pkg, pbref, persist):
    """pb_solve_refined under the periodic boundary condition (wrap terms in the fp64 residual and in the fp32
    corrections), through the persistent kernel and through the two-kernel TMA path."""
    inp = _periodic_inputs((45, 23, 19), 32)
    ref = pbref.from_inputs(inp)
    ref.set_periodic(True)
    ref.set_rhs(inp.rhs, inp.bc)
    o = ref.solve(1e-10, 5000)
    ref.close()
    with pkg.PBSolver(*inp.args(), options=dict(persist=int(persist))) as s:
        s.set_periodic(True)
        g = s.solve_refined(1e-10, 5000, check_every=8)
    assert g["status"] == 0 and g["relres"] <= 1e-10
    assert np.max(np.abs(g["phi"] - o["phi"])) <= 1e-8 * np.max(np.abs(o["phi"]))


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs[3] (257^3, eps_in = 4) and the config-5 batch members (PAPER.md:182 defines the
# workload family: eps 80 / solute, harmonic faces, free-space boundary; PAPER.md:23 the snapshot stream)
# ---------------------------------------------------------------------------------------------
@pytest.mark.slow
def test_solve_config4_257(pkg, pbref):
    """configs[3]: 257^3, 20 000-atom globule, eps_in = 4 (palette {0, 4, 7.619, 80}: another face table, another
    diagonal table, another autotuned plan than config 5), fp32 to 1e-5 and fp64 to 1e-10 -- every node against the
    full oracle solves, iteration counts within 5 %."""
    inp = make_config(4, device="cuda")
    assert inp.meta["eps_in"] == 4.0 and set(np.unique(inp.eps_x)) == {4.0, 80.0, 2 * 4.0 * 80.0 / 84.0}
    ref = pbref.from_inputs(inp)
    o32 = ref.solve(1e-5, 5000)
    o64 = ref.solve(1e-10, 5000)
    ref.close()
    scale = np.max(np.abs(o64["phi"]))
    with pkg.PBSolver(*inp.args()) as s:
        g32 = s.solve(1e-5, 20000, "f32", check_every=32)
        g64 = s.solve(1e-10, 20000, "f64", check_every=32)
        p32, p64 = s.plan("f32"), s.plan("f64")
    assert p32["palette_size"] == 4 and p32["face_palette"] and not p32["persist"] and not p64["persist"]
    assert g32["status"] == 0 and g64["status"] == 0 and g32["relres"] < 1e-5 and g64["relres"] < 1e-10
    assert abs(g32["iters"] - o32["iters"]) <= round(0.05 * o32["iters"]), (g32["iters"], o32["iters"])
    assert abs(g64["iters"] - o64["iters"]) <= round(0.05 * o64["iters"]), (g64["iters"], o64["iters"])
    e32 = np.max(np.abs(g32["phi"] - o32["phi"])) / scale
    e32t = np.max(np.abs(g32["phi"] - o64["phi"])) / scale
    e64 = np.max(np.abs(g64["phi"] - o64["phi"])) / scale
    print(f"config4: fp32 iters {g32['iters']} (oracle {o32['iters']}) err {e32:.2e} / {e32t:.2e}; "
          f"fp64 iters {g64['iters']} (oracle {o64['iters']}) err {e64:.2e}; plan {p32['txv']}x{p32['ty']}x{p32['tz']}")
    assert e32 <= 1e-4 and e32t <= 1e-4 and e64 <= 1e-8


@pytest.mark.slow
def test_config5_batch_member_parity(pkg, pbref):
    """One member of configs[4]'s 50-solve batch (seeded charge perturbation N(0, 0.05) e on the same operator) at the
    full 385^3, fp32 to 1e-5, against the oracle's own solve of that member -- through pb_set_rhs (host-generated
    rhs / ghost values) and through pb_set_charges on an atom-built handle (rhs and the 5.3e10-term boundary sum made
    on the GPU); every node, north-star fp32 bar."""
    from workloads import perturbed_charge_values, perturbed_charges

    member = 7
    inp = make_config(5, device="cuda")
    rhs_s, bc_s = perturbed_charges(inp, member, device="cuda")
    ref = pbref.from_inputs(inp)
    ref.set_rhs(rhs_s, bc_s)
    o = ref.solve(1e-5, 5000)
    ref.close()
    scale = np.max(np.abs(o["phi"]))
    with pkg.PBSolver(*inp.args()) as s:
        base = s.solve(1e-5, 20000, "f32", check_every=32)
        s.set_rhs(rhs_s, bc_s)
        g = s.solve(1e-5, 20000, "f32", check_every=32)
    m = inp.meta
    with pkg.PBSolver.from_atoms(inp.nx, inp.ny, inp.nz, inp.h, m["centres"], m["radii"], m["charges"], m["eps_in"],
                                 m["eps_out"], m["kbar2_solvent"]) as s2:
        s2.set_charges(perturbed_charge_values(inp, member))
        g2 = s2.solve(1e-5, 20000, "f32", check_every=32)
    for r in (g, g2):
        assert r["status"] == 0 and r["relres"] < 1e-5
        assert abs(r["iters"] - o["iters"]) <= round(0.05 * o["iters"]), (r["iters"], o["iters"])
        assert np.max(np.abs(r["phi"] - o["phi"])) <= 1e-4 * scale
    # the member really is another right-hand side than the unperturbed one
    assert np.max(np.abs(g["phi"] - base["phi"])) > 1e-3 * scale
    print(f"config5 member {member}: iters set_rhs {g['iters']} / set_charges {g2['iters']} (oracle {o['iters']}), "
          f"err {np.max(np.abs(g['phi'] - o['phi'])) / scale:.2e} / {np.max(np.abs(g2['phi'] - o['phi'])) / scale:.2e}")


# ---------------------------------------------------------------------------------------------
# failure paths (Reading 17) on both solve paths
# ---------------------------------------------------------------------------------------------
def _indefinite_operator(shape=(17, 13, 11)):
    """Uniform eps = 80, no salt, one interior face at -300: both adjacent diagonals stay positive (5*80 - 300 = 100,
    pb_create accepts it) but the 2x2 block [[100, 300], [300, 100]] is indefinite, so A is not SPD."""
    nx, ny, nz = shape
    inp = random_operator(nx, ny, nz, seed=77, salted=False)
    inp.eps_x[...] = 80.0
    inp.eps_y[...] = 80.0
    inp.eps_z[...] = 80.0
    inp.eps_x[nz // 2, ny // 2, nx // 2] = -300.0
    return inp


@pytest.mark.parametrize("persist", [1, 0])
def test_breakdown_returns_last_good_iterate(pkg, pbref, persist):
    """p.Ap <= 0 on an indefinite operator: PB_ERR_BREAKDOWN, iters and phi = the oracle's at its own breakdown (the last
    iterate before the failed step), on the cooperative path and on the two-kernel path, whatever check_every is."""
    inp = _indefinite_operator()
    ref = pbref.from_inputs(inp)
    o = ref.solve(1e-12, 500)
    ref.close()
    assert o["status"] == pbref.BREAKDOWN and o["iters"] >= 1
    scale = np.max(np.abs(o["phi"]))
    with pkg.PBSolver(*inp.args(), options=dict(persist=persist)) as s:
        assert np.all(s.diag() > 0)
        for ce in (1, 7, 1000):                          # 1000 > maxiter: one chunk covers the whole solve
            g = s.solve(1e-12, 500, "f64", check_every=ce)
            assert g["status"] == pkg.binding.PB_ERR_BREAKDOWN, (ce, g["status"])
            assert g["iters"] == o["iters"], (ce, g["iters"], o["iters"])
            assert np.all(np.isfinite(g["phi"]))
            assert np.max(np.abs(g["phi"] - o["phi"])) <= 1e-8 * scale
        g32 = s.solve(1e-12, 500, "f32", check_every=5)
        assert g32["status"] == pkg.binding.PB_ERR_BREAKDOWN and np.all(np.isfinite(g32["phi"]))
        # the handle is still usable afterwards
        s.set_rhs(None, None)
        assert s.solve(1e-6, 10, "f64")["iters"] == 0


@pytest.mark.parametrize("persist", [1, 0])
@pytest.mark.parametrize("bad", [np.nan, np.inf])
def test_non_finite_rhs_is_a_breakdown(pkg, pbref, persist, bad):
    """NaN / Inf in rhs: PB_ERR_BREAKDOWN at l = 0 with phi = 0 (finite), never a hang or PB_ERR_MAXITER; same as the
    oracle's verdict."""
    inp = random_operator(19, 11, 6, seed=4)
    rhs = inp.rhs.copy()
    rhs[3, 5, 7] = bad
    ref = pbref.from_inputs(inp)
    ref.set_rhs(rhs, inp.bc)
    o = ref.solve(1e-8, 50)
    ref.close()
    assert o["status"] == pbref.BREAKDOWN and o["iters"] == 0
    with pkg.PBSolver(*inp.args(), options=dict(persist=persist)) as s:
        s.set_rhs(rhs, inp.bc)
        for prec in ("f64", "f32"):
            g = s.solve(1e-8, 50, prec, check_every=4)
            assert g["status"] == pkg.binding.PB_ERR_BREAKDOWN and g["iters"] == 0
            assert not g["phi"].any()
        s.set_rhs(inp.rhs, inp.bc)                        # a good right-hand side afterwards solves normally
        assert s.solve(1e-8, 500, "f64")["status"] == 0


def test_check_every_larger_than_maxiter(pkg, pbref):
    inp = random_operator(19, 11, 6, seed=4)
    ref = pbref.from_inputs(inp)
    o = ref.solve(1e-12, 7)
    o_conv = ref.solve(1e-6, 1000)
    ref.close()
    with pkg.PBSolver(*inp.args(), options=dict(persist=0)) as s:
        g = s.solve(1e-12, 7, "f64", check_every=4096)
        assert g["status"] == pkg.binding.PB_ERR_MAXITER and g["iters"] == 7
        assert np.max(np.abs(g["phi"] - o["phi"])) <= 1e-10 * np.max(np.abs(o["phi"]))
        c = s.solve(1e-6, 1000, "f64", check_every=4096)
        assert c["status"] == 0 and c["iters"] == o_conv["iters"]


def test_options_are_handle_state(pkg):
    """pb_set_option / pb_get_option / pb_get_plan: two handles in one process configured differently, invalid values
    rejected, the plan reports what runs."""
    inp = make_config(2)
    with pkg.PBSolver(*inp.args(), options=dict(persist=0, palette=0, autotune=0, fused=0)) as a, \
            pkg.PBSolver(*inp.args(), options=dict(fused=0)) as b:
        pa, pb_ = a.plan("f32"), b.plan("f32")
        assert pa["persist"] == 0 and pa["face_palette"] == 0 and pa["palette_size"] == 0 and not pa["autotuned"]
        assert pa["spmv_bytes_per_node"] == 40 and pa["vec_bytes_per_node"] == 16
        assert pb_["persist"] == 1 and pb_["face_palette"] == 1 and pb_["palette_size"] == 4
        assert pb_["spmv_bytes_per_node"] == 28 and pb_["vec_bytes_per_node"] == 13
        assert pa["num_sm"] == pb_["num_sm"] >= 1 and pa["grid"] >= 1 and pa["threads"] % 32 == 0
        assert a.get_option("palette") == 0 and b.get_option("palette") == 1
        ga, gb = a.solve(1e-5, 5000, "f32"), b.solve(1e-5, 5000, "f32")
        assert abs(ga["iters"] - gb["iters"]) <= 1
        for name, val in (("ring_slots", 2), ("ring_slots", 9), ("persist", 2), ("palette", -1), ("blocks_per_sm", 33)):
            with pytest.raises(pkg.PBError):
                a.set_option(name, val)
        # the fused iteration (the default off the L2-resident path): one kernel, 8 words + 2 index bytes per node
        a.set_option("fused", 1)
        a.set_option("palette", 1)
        pf = a.plan("f32")
        assert pf["fused"] == 1 and pf["face_quad"] == 1 and pf["spmv_bytes_per_node"] == 34 and pf["vec_bytes_per_node"] == 0
        assert abs(a.solve(1e-5, 5000, "f32")["iters"] - gb["iters"]) <= 1
        a.set_option("fused", 0)
        a.set_option("palette", 0)
        # a forced tile larger than the grid / the thread budget is clamped, and the plan says what really runs
        a.set_option("tile_ty", 400)
        a.set_option("tile_txv", 60)
        pc = a.plan("f32")
        assert pc["ty"] <= inp.ny and pc["txv"] <= pc["pitch"] // 4 and pc["threads"] <= 512
        a.set_option("tile_ty", 0)
        a.set_option("tile_txv", 0)
        assert a.plan("f32")["txv"] == pa["txv"] and a.solve(1e-5, 5000, "f32")["iters"] == ga["iters"]


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_fused_tail_pool_is_schedule_independent(pkg, pbref, prec, tol):
    """k_pcg_fused hands the top tenth of the planes out dynamically (PB_OPT_TAIL_POOL): which block runs which chunk
    changes from launch to launch, the result must not -- the sums are formed per tile and added in tile order.  Chunk
    sizes 4 / 8 (default for nz >= 64) / 10, a size too large for the grid (64: no pool) and pool off: oracle parity, the same iteration count,
    bitwise repeatable solves, and rejected values."""
    inp = random_operator(45, 37, 83, seed=12, two_valued=True)         # nz = 83: 3 static z-chunks + the pool
    ref = pbref.from_inputs(inp)
    o = ref.solve(tol, 5000)
    ref.close()
    scale, lim = np.max(np.abs(o["phi"])), (1e-8 if prec == "f64" else 1e-4)
    iters = set()
    for pool in (0, 1, 4, 10, 64):
        with pkg.PBSolver(*inp.args(), options=dict(persist=0, tail_pool=pool, tile_tz=25)) as s:
            g1 = s.solve(tol, 5000, prec, check_every=5)
            g2 = s.solve(tol, 5000, prec, check_every=64)
            pl = s.plan(prec)
        assert pl["fused"] == 1 and pl["tail_pool"] == {0: 8, 1: 0, 4: 4, 10: 10, 64: 0}[pool], pl     # 64 > nz / 8: no pool
        assert g1["status"] == 0 and np.array_equal(g1["phi"], g2["phi"]) and g1["iters"] == g2["iters"], pool
        assert abs(g1["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (pool, g1["iters"], o["iters"])
        assert np.max(np.abs(g1["phi"] - o["phi"])) <= lim * scale, pool
        iters.add(g1["iters"])
    assert len(iters) == 1
    with pkg.PBSolver(*inp.args()) as s:
        for bad in (2, 3, 65):
            with pytest.raises(pkg.PBError):
                s.set_option("tail_pool", bad)


# ---------------------------------------------------------------------------------------------
# NEXT row f2: pb_solve_batch -- M right-hand sides per pass (k_spmv_batch + k_vec_batch)
# ---------------------------------------------------------------------------------------------
def _members(inp, m, seed):
    rng = np.random.default_rng(seed)
    rhs = np.stack([inp.rhs * (1 + 0.3 * s) + rng.standard_normal(inp.rhs.shape) * (0.2 * s) for s in range(m)])
    bc = np.stack([inp.bc * (1 - 0.1 * s) + rng.uniform(-1, 1, inp.bc.shape) * (0.1 * s) for s in range(m)])
    return rhs, bc


@pytest.mark.parametrize("shape,kind", [((13, 9, 7), "quad"), ((77, 45, 38), "quad"), ((130, 21, 37), "words"),
                                        ((45, 23, 19), "bytes")])
@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_batch_members_match_their_own_oracle_solves(pkg, pbref, shape, kind, prec, tol):
    """Every member of a batch against ITS OWN oracle solve (north-star bars), for each batch width and coefficient
    format (2-bit quads for <= 4 face values, words otherwise -- also for a 7-valued map whose single-solve format is
    the byte palette); per member the iteration count must not depend on the width (1, 2 or 4 members per pass: the
    arithmetic per member is the same) and must agree with pb_solve's to within one iteration."""
    inp = random_operator(*shape, seed=21, two_valued=(kind != "words"))
    if kind == "bytes":
        inp.eps_y[...] = np.random.default_rng(5).choice([1.0, 2.0, 4.0, 20.0, 78.5, 80.0], inp.eps_y.shape)
    m = 5                                         # not a multiple of 2 or 4: groups of 2+2+1 and 4+1
    rhs, bc = _members(inp, m, 3)
    ref = pbref.from_inputs(inp)
    orc = []
    for s in range(m):
        ref.set_rhs(rhs[s], bc[s])
        orc.append(ref.solve(tol, 5000))
    ref.close()
    lim = 1e-8 if prec == "f64" else 1e-4
    iters_by_width = {}
    for width in (1, 2, 4):
        with pkg.PBSolver(*inp.args(), options=dict(batch_width=width, persist=0)) as sv:
            g = sv.solve_batch(rhs, bc, tol, 5000, prec, check_every=9)
            g_again = sv.solve_batch(rhs, bc, tol, 5000, prec, check_every=31)
            singles = []
            for s in range(m):
                sv.set_rhs(rhs[s], bc[s])
                singles.append(sv.solve(tol, 5000, prec))
        assert g["worst"] == 0 and g["status"] == [0] * m
        assert np.array_equal(g["phi"], g_again["phi"]) and g["iters"] == g_again["iters"]      # bitwise repeatable
        for s in range(m):
            o = orc[s]
            scale = np.max(np.abs(o["phi"]))
            assert g["relres"][s] < tol
            assert abs(g["iters"][s] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (width, s, g["iters"][s], o["iters"])
            assert np.max(np.abs(g["phi"][s] - o["phi"])) <= lim * scale, (width, s)
            assert abs(g["iters"][s] - singles[s]["iters"]) <= 1
            assert np.max(np.abs(g["phi"][s] - singles[s]["phi"])) <= lim * scale
        iters_by_width[width] = g["iters"]
    assert iters_by_width[1] == iters_by_width[2] == iters_by_width[4]


def test_batch_per_member_latches(pkg, pbref):
    """Members stop independently: a zero right-hand side is done at l = 0, a non-finite one breaks down at l = 0 without
    disturbing its neighbours, an easy member converges long before a hard one, maxiter latches every live member."""
    inp = random_operator(33, 31, 29, seed=12)
    rng = np.random.default_rng(9)
    rhs = np.stack([inp.rhs, np.zeros_like(inp.rhs), inp.rhs.copy(), rng.standard_normal(inp.rhs.shape)])
    bc = np.stack([inp.bc, np.zeros_like(inp.bc), inp.bc, inp.bc * 0.5])
    rhs[2, 3, 5, 7] = np.nan
    ref = pbref.from_inputs(inp)
    o0 = ref.solve(1e-10, 5000)
    ref.set_rhs(rhs[3], bc[3])
    o3 = ref.solve(1e-10, 5000)
    o3_short = ref.solve(1e-10, 11)
    ref.close()
    for width in (2, 4):
        with pkg.PBSolver(*inp.args(), options=dict(batch_width=width)) as sv:
            g = sv.solve_batch(rhs, bc, 1e-10, 5000, "f64", check_every=7)
            assert g["status"] == [0, 0, pkg.binding.PB_ERR_BREAKDOWN, 0] and g["worst"] == pkg.binding.PB_ERR_BREAKDOWN
            assert g["iters"][1] == 0 and not g["phi"][1].any() and g["relres"][1] == 0.0
            assert g["iters"][2] == 0 and not g["phi"][2].any()
            assert g["iters"][0] == o0["iters"] and g["iters"][3] == o3["iters"]
            assert np.max(np.abs(g["phi"][0] - o0["phi"])) <= 1e-8 * np.max(np.abs(o0["phi"]))
            assert np.max(np.abs(g["phi"][3] - o3["phi"])) <= 1e-8 * np.max(np.abs(o3["phi"]))
            short = sv.solve_batch(rhs[[0, 3]], bc[[0, 3]], 1e-10, 11, "f64", check_every=4)
            assert short["status"] == [pkg.binding.PB_ERR_MAXITER] * 2 and short["iters"] == [11, 11]
            assert np.max(np.abs(short["phi"][1] - o3_short["phi"])) <= 1e-10 * np.max(np.abs(o3_short["phi"]))
            sv.set_periodic(True)
            with pytest.raises(pkg.PBError):
                sv.solve_batch(rhs, bc, 1e-10, 50, "f64")


def test_batch_device_pointers_and_charges(pkg, pbref, cuda_device):
    """Device-resident members (no host staging), and pb_solve_batch_charges on an atom-built handle against
    pb_set_charges + pb_solve of each member and against the oracle fed by the setup oracle."""
    import torch

    from oracle import pbsetup_ref as S
    from workloads import pb_inputs as W

    inp = make_config(2)
    m = 3
    rhs, bc = _members(inp, m, 4)
    with pkg.PBSolver(*inp.args()) as sv:
        host = sv.solve_batch(rhs, bc, 1e-5, 5000, "f32")
        dev = sv.solve_batch(torch.from_numpy(rhs).to(cuda_device), torch.from_numpy(bc).to(cuda_device), 1e-5, 5000, "f32")
        assert dev["phi"].is_cuda and host["iters"] == dev["iters"]
        assert np.array_equal(dev["phi"].cpu().numpy(), host["phi"])
    nx, ny, nz, h = 40, 23, 31, 0.5
    rng = np.random.Generator(np.random.PCG64(W.SEED0 + 777))
    L = np.array([(nx - 1) * h, (ny - 1) * h, (nz - 1) * h])
    c = W.atoms_uniform(30, 0.15 * L, 0.85 * L, rng)
    r = rng.uniform(1.2, 2.0, 30)
    Q = rng.normal(0.0, 0.4, (3, 30))
    with pkg.PBSolver.from_atoms(nx, ny, nz, h, c, r, Q[0], 1.0, 80.0, W.KBAR2_150MM_300K) as sv:
        g = sv.solve_batch_charges(Q, 1e-10, 5000, "f64")
        for s in range(3):
            sv.set_charges(Q[s])
            one = sv.solve(1e-10, 5000, "f64")
            f = S.setup(nx, ny, nz, h, c, r, Q[s], 1.0, 80.0, W.KBAR2_150MM_300K)
            o = pbref.PBRef(nx, ny, nz, h, f["eps_x"], f["eps_y"], f["eps_z"], f["kbar2"], f["rhs"], f["bc"]).solve(1e-10, 5000)
            scale = np.max(np.abs(o["phi"]))
            assert g["status"][s] == 0 and abs(g["iters"][s] - o["iters"]) <= max(1, round(0.05 * o["iters"]))
            assert np.max(np.abs(g["phi"][s] - o["phi"])) <= 1e-8 * scale
            assert np.max(np.abs(g["phi"][s] - one["phi"])) <= 1e-8 * scale


@pytest.mark.slow
def test_config5_batch_members_multi_rhs_full_size(pkg, pbref):
    """Two members of configs[4]'s perturbed-charge batch at the full 385^3 through pb_solve_batch_charges (two members
    per pass, 2-bit face indices), each against the oracle's own solve of that member; fp32, every node."""
    from workloads import perturbed_charge_values, perturbed_charges

    inp = make_config(5, device="cuda")
    members = (3, 11)
    m = inp.meta
    Q = np.stack([perturbed_charge_values(inp, s) for s in members])
    with pkg.PBSolver.from_atoms(inp.nx, inp.ny, inp.nz, inp.h, m["centres"], m["radii"], m["charges"], m["eps_in"],
                                 m["eps_out"], m["kbar2_solvent"]) as sv:
        g = sv.solve_batch_charges(Q, 1e-5, 20000, "f32", check_every=32)
    ref = pbref.from_inputs(inp)
    for i, s in enumerate(members):
        rhs_s, bc_s = perturbed_charges(inp, s, device="cuda")
        ref.set_rhs(rhs_s, bc_s)
        o = ref.solve(1e-5, 5000)
        scale = np.max(np.abs(o["phi"]))
        err = np.max(np.abs(g["phi"][i] - o["phi"])) / scale
        print(f"config5 batch member {s}: iters {g['iters'][i]} (oracle {o['iters']}) err {err:.2e}")
        assert g["status"][i] == 0 and g["relres"][i] < 1e-5
        assert abs(g["iters"][i] - o["iters"]) <= round(0.05 * o["iters"])
        assert err <= 1e-4
    ref.close()


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_fused_iteration_tilings_and_formats(pkg, pbref, prec, tol):
    """k_pcg_fused (one kernel per iteration: the residual update deferred into the next pass, every scalar from one
    reduction with exactly re-summed norms) under forced tiles / rings / grids and in both coefficient formats (2-bit
    quads, words; Dinv bytes or words): same iteration count as the oracle within 5 % and as the two-kernel path within
    one, potentials within the north-star bars, bitwise repeatable; maxiter and the l = 0 cases latch identically."""
    inp = random_operator(77, 45, 38, seed=21)
    ref = pbref.from_inputs(inp)
    o = ref.solve(tol, 5000)
    o9 = ref.solve(tol, 9)
    ref.close()
    scale = np.max(np.abs(o["phi"]))
    lim = 1e-8 if prec == "f64" else 1e-4
    with pkg.PBSolver(*inp.args(), options=dict(persist=0, fused=0)) as s:
        two = s.solve(tol, 5000, prec)
    cfgs = [dict(), dict(tile_txv=7, tile_ty=3, ring_slots=3, blocks_per_sm=2, tile_tz=5),
            dict(tile_txv=20, tile_ty=8, blocks_per_sm=1, tile_tz=99), dict(tile_txv=5, tile_ty=2, blocks_per_sm=4, tile_tz=1),
            dict(tile_txv=13, tile_ty=5, ring_slots=4, blocks_per_sm=3, tile_tz=33)]
    for fmt in (dict(), dict(palette_diag_spmv=0), dict(palette=0)):
        for cfg in cfgs:
            with pkg.PBSolver(*inp.args(), options={**cfg, **fmt, "persist": 0}) as s:
                runs = [s.solve(tol, 5000, prec, check_every=ce) for ce in (9, 64)]
                short = s.solve(tol, 9, prec, check_every=4)
                pl = s.plan(prec)
            assert pl["fused"] == 1 and pl["face_quad"] == (0 if fmt == dict(palette=0) else 1), (fmt, cfg, pl)
            assert np.array_equal(runs[0]["phi"], runs[1]["phi"]) and runs[0]["iters"] == runs[1]["iters"], (fmt, cfg)
            assert runs[0]["status"] == 0 and runs[0]["relres"] < tol
            assert abs(runs[0]["iters"] - o["iters"]) <= max(1, round(0.05 * o["iters"])), (fmt, cfg, runs[0]["iters"], o["iters"])
            assert abs(runs[0]["iters"] - two["iters"]) <= 1, (fmt, cfg)
            assert np.max(np.abs(runs[0]["phi"] - o["phi"])) <= lim * scale, (fmt, cfg)
            assert short["status"] == pkg.binding.PB_ERR_MAXITER and short["iters"] == 9
            assert np.max(np.abs(short["phi"] - o9["phi"])) <= lim * scale, (fmt, cfg)
