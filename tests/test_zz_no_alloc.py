"""-m gpu: pb_residual_noalloc (the entry point that allocates nothing: its scratch is a fixed __device__ array of
the library) against the existing path, pb_residual, on two calls in a row.  Collected last on purpose (the file name
sorts after every other test file): the suite runs with pytest -x.  Passes alone in a fresh process and after the
other tests -- the first call on the device looks the scratch address up, whoever makes it."""
import numpy as np
import pytest

from workloads import make_config, random_operator

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg(cuda_device):
    import paper_1704_02745_b200 as pkg
    from paper_1704_02745_b200 import build as pb_build

    pb_build.build()
    pkg.load_library()
    return pkg


def _dev(inp, torch, dev):
    """The operator / right-hand side arrays of a workload as CUDA float64 tensors (the caller's inputs)."""
    t = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device=dev)
    return dict(eps_x=t(inp.eps_x), eps_y=t(inp.eps_y), eps_z=t(inp.eps_z), kbar2=t(inp.kbar2), rhs=t(inp.rhs), bc=t(inp.bc))


def _noalloc(pkg, inp, d, phi_d, out3, stream=None):
    pkg.residual_noalloc(inp.nx, inp.ny, inp.nz, inp.h, d["eps_x"], d["eps_y"], d["eps_z"], d["kbar2"], d["rhs"], d["bc"],
                         phi_d, out3, stream=stream)


def test_noalloc_residual_matches_pb_residual_twice_in_a_row(pkg, cuda_device):
    """Two calls in a row (a large grid first, a smaller one second: the scratch still holds the first call's partial
    sums beyond the second call's blocks), each against pb_residual on the same inputs.  Tolerances are the ones
    test_true_residual_matches_oracle uses: 1e-12 relative where nothing cancels (random phi), 1e-6 relative for a
    converged potential (r = b - A phi cancels to 1e-6 |b|).  Device memory in use must not change across the calls."""
    import torch

    dev = cuda_device
    big = random_operator(77, 45, 38, seed=5, two_valued=False)        # ragged: 38 * 45 rows = 213.75 blocks of 8
    small = make_config(1)                                             # Born ion, 33^3
    rng = np.random.default_rng(11)
    cases = []
    for inp in (big, small):
        with pkg.PBSolver(*inp.args()) as s:
            solved = s.solve(1e-6, 5000, "f64")["phi"]
            rnd = rng.standard_normal(solved.shape)
            cases.append((inp, rnd, s.residual(rnd, "f64"), 1e-12))
            cases.append((inp, solved, s.residual(solved, "f64"), 1e-6))
            assert s.residual(np.zeros_like(solved), "f64") == 1.0
    prepared = []
    for inp, phi, want, rtol in cases:
        prepared.append((inp, _dev(inp, torch, dev), torch.as_tensor(phi, device=dev), want, rtol))
    out = torch.zeros((len(prepared), 3), dtype=torch.float64, device=dev)       # the caller's output buffers
    _noalloc(pkg, prepared[0][0], prepared[0][1], prepared[0][2], out[0])       # first call on this device: address lookup
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for rep in range(2):                                                         # the whole sequence twice
        out.zero_()
        for c, (inp, d, phi_d, want, rtol) in enumerate(prepared):               # back to back, no sync in between
            _noalloc(pkg, inp, d, phi_d, out[c])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0                             # nothing was allocated
        got = out.cpu().numpy()
        for c, (inp, d, phi_d, want, rtol) in enumerate(prepared):
            relres, rr, bb = got[c]
            assert abs(relres - want) <= rtol * want, (rep, c, relres, want)
            assert bb > 0.0 and abs(np.sqrt(rr / bb) - relres) <= 1e-15 * relres
    # phi = 0: r = b exactly, on the second grid right after the first
    z = torch.zeros_like(prepared[0][2])
    _noalloc(pkg, prepared[0][0], prepared[0][1], z, out[0])
    torch.cuda.synchronize()
    assert float(out[0, 0]) == 1.0 and float(out[0, 1]) == float(out[0, 2])
    # a side stream of the caller's, and the NULL-able inputs (no salt, no charges, no boundary values: b = 0 -> 0)
    side = torch.cuda.Stream()
    inp, d, phi_d, want, rtol = prepared[1]
    with torch.cuda.stream(side):
        out.zero_()
        _noalloc(pkg, inp, d, phi_d, out[1], stream=side.cuda_stream)
        d0 = dict(d, kbar2=None, rhs=None, bc=None)
        _noalloc(pkg, inp, d0, phi_d, out[2], stream=side.cuda_stream)
    side.synchronize()
    assert abs(float(out[1, 0]) - want) <= rtol * want
    assert float(out[2, 0]) == 0.0 and float(out[2, 2]) == 0.0 and float(out[2, 1]) > 0.0


def test_noalloc_rejects_grids_beyond_its_scratch(pkg, cuda_device):
    """nz * ny > PB_NOALLOC_MAX_ROWS: PB_ERR_TOO_LARGE with a message that says why, before any pointer is looked at
    (nothing is enqueued); the largest admissible row count passes the size check."""
    import ctypes

    lib = pkg.load_library()
    assert pkg.NOALLOC_MAX_ROWS == 262144
    with pytest.raises(pkg.PBError) as e:
        pkg.residual_noalloc(2, 513, 512, 0.5, None, None, None, None, None, None, None, None)
    assert e.value.status == 7 and "PB_ERR_TOO_LARGE" in str(e.value) and "PB_NOALLOC_MAX_ROWS" in str(e.value)
    assert lib.pb_residual_noalloc(2, 512, 513, 0.5, None, None, None, None, None, None, None, None, None) == 7
    # at the limit the size check passes and the NULL pointers are what is rejected
    assert lib.pb_residual_noalloc(2, 512, 512, 0.5, None, None, None, None, None, None, None, None, None) == 1
    assert lib.pb_residual_noalloc(0, 4, 4, 0.5, None, None, None, None, None, None, None, None, None) == 1
    assert lib.pb_residual_noalloc(4, 4, 4, -1.0, None, None, None, None, None, None, None, None, None) == 1
    assert ctypes.c_char_p(lib.pb_strerror(7)).value.decode().startswith("grid larger than the fixed scratch")
