"""-m "not gpu": the algebra behind k_pcg_fused (DESIGN.md Reading 23), checked on the CPU against the oracle.

The fused pass defers the residual update of iteration l into the pass of iteration l+1 and takes every scalar from ONE
reduction.  This file restates that recurrence in plain numpy fp64 -- with the ORACLE's operator (pbref.apply) and
diagonal, nothing from the CUDA path -- and checks that it is the PCG of PAPER.md:104-126: the same iterates, the same
residual history, the same stopping iteration as the oracle's solve, and the identities the kernel's finaliser relies
on (S1 = z_l . A p_{l+1} = p.Ap - beta_l W by the symmetry of A;  r_{l+1}.z_{l+1} = U1 - 2 alpha S1 + alpha^2 S2).
A wrong sign, a wrong index (beta_l for beta_{l+1}, W on the wrong pair of vectors) or an off-by-one in the lagged
stopping test fails it."""
import numpy as np
import pytest

from oracle import pbref
from workloads import born_ion, random_operator


def fused_passes(ref, tol, maxiter):
    """The sequence of passes of k_pcg_fused, in the kernel's notation.  Pass number l + 1 (l = 0, 1, ...) reads the
    buffer set {r_{l-1}, A p_l, p_l, x_{l-1}} and the scalars alpha_l, beta_l; it forms r_l, x_l, p_{l+1}, A p_{l+1} and
    the five sums, from which its finaliser takes alpha_{l+1}, beta_{l+1} -- or stops, on ||r_l||."""
    A = ref.apply
    b, dinv = ref.b(), 1.0 / ref.diag()
    bb = float(np.sum(b * b))
    # k_init: x = 0, r = b, p = 0, "A p_0" = 0, alpha = beta = 0
    r, q, p, x = b.copy(), np.zeros_like(b), np.zeros_like(b), np.zeros_like(b)
    alpha = beta = 0.0
    hist, checks = [], []
    for l in range(maxiter + 2):
        r = r - alpha * q                          # r_l (the deferred step 5; r_0 = b)
        x = x + alpha * p                          # phi_l
        z = dinv * r
        p_new = z + beta * p                       # p_{l+1} (steps 6-7; p_1 = z_0)
        v = A(p_new)                               # A p_{l+1}
        pAp, S2, W = np.sum(p_new * v), np.sum(dinv * v * v), np.sum(q * p_new)
        U1, U2 = np.sum(dinv * r * r), np.sum(r * r)
        hist.append(np.sqrt(U2 / bb))
        if U2 < tol * tol * bb or l >= maxiter:    # step 3 on the exact ||r_l||, one pass late; x = phi_l is final
            return dict(phi=x, iters=l, history=np.array(hist), checks=checks)
        S1 = pAp - beta * W                        # z_l . A p_{l+1}
        alpha_new = U1 / pAp                       # step 5
        rz_new = U1 - 2.0 * alpha_new * S1 + alpha_new * alpha_new * S2
        checks.append((S1, float(np.sum(z * v)), rz_new, float(np.sum(dinv * (r - alpha_new * v) ** 2)), U1))
        alpha, beta = alpha_new, rz_new / U1       # step 7
        q, p = v, p_new
    raise AssertionError("unreachable")


@pytest.mark.parametrize("case", ["born", "random", "random_salted"])
def test_fused_recurrence_is_the_pcg_of_the_paper(case):
    inp = born_ion() if case == "born" else random_operator(13, 9, 7, seed=4, salted=(case == "random_salted"))
    ref = pbref.from_inputs(inp)
    tol = 1e-9
    o = ref.solve(tol, 2000, history=True)
    f = fused_passes(ref, tol, 2000)
    ref.close()
    # the same stopping iteration and the same residual history as the listing (tested before step 4)
    assert f["iters"] == o["iters"]
    assert np.allclose(f["history"], o["history"], rtol=1e-6, atol=0.0)
    assert np.max(np.abs(f["phi"] - o["phi"])) <= 1e-9 * np.max(np.abs(o["phi"]))
    # the identities of the single reduction hold to rounding in every pass (relative to the size of their terms)
    for S1, zv, rz_new, rz_direct, U1 in f["checks"]:
        assert abs(S1 - zv) <= 1e-9 * (abs(zv) + U1)
        assert abs(rz_new - rz_direct) <= 1e-9 * U1


def test_fused_recurrence_edge_cases():
    """b = 0 stops in pass 1 with l = 0 and phi = 0; maxiter stops with l = maxiter and the iterate phi_maxiter of the
    oracle (PB_ERR_MAXITER semantics, Reading 17)."""
    inp = random_operator(9, 7, 5, seed=2)
    ref = pbref.from_inputs(inp)
    o5 = ref.solve(1e-12, 5)
    f5 = fused_passes(ref, 1e-12, 5)
    assert f5["iters"] == 5 == o5["iters"]
    assert np.max(np.abs(f5["phi"] - o5["phi"])) <= 1e-12 * np.max(np.abs(o5["phi"]))
    ref.set_rhs(np.zeros_like(inp.rhs), np.zeros_like(inp.bc))
    f0 = fused_passes(ref, 1e-5, 100) if float(np.sum(ref.b() ** 2)) > 0 else dict(iters=0, phi=np.zeros_like(inp.rhs))
    ref.close()
    assert f0["iters"] == 0 and not np.any(f0["phi"])
