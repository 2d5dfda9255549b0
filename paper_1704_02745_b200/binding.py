"""ctypes binding of include/pb.h -- same names, argument marshalling only.

Arrays may be numpy arrays / CPU torch tensors (passed as PB_HOST pointers) or CUDA torch
tensors (passed as PB_DEVICE pointers).  PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

PB_F32, PB_F64 = 0, 1
PB_HOST, PB_DEVICE = 0, 1
PB_OK, PB_ERR_INVALID_ARG, PB_ERR_ALLOC, PB_ERR_CUDA, PB_ERR_NOT_SPD, PB_ERR_BREAKDOWN, PB_ERR_MAXITER = range(7)
STATUS_NAMES = {0: "PB_OK", 1: "PB_ERR_INVALID_ARG", 2: "PB_ERR_ALLOC", 3: "PB_ERR_CUDA",
                4: "PB_ERR_NOT_SPD", 5: "PB_ERR_BREAKDOWN", 6: "PB_ERR_MAXITER", 7: "PB_ERR_TOO_LARGE"}

# every symbol include/pb.h declares
EXPORTS = ("pb_create", "pb_set_rhs", "pb_apply", "pb_solve", "pb_solve_begin", "pb_iterate",
           "pb_destroy", "pb_strerror", "pb_query", "pb_version", "pb_profile", "pb_launch_count", "pb_set_preconditioner", "pb_create_from_atoms",
           "pb_set_charges", "pb_get_field", "pb_palette_size", "pb_solve_from", "pb_set_boundary",
           "pb_diag_palette_size", "pb_residual", "pb_bytes_per_node", "pb_solve_refined", "pb_set_setup_precision", "pb_set_option", "pb_get_option",
           "pb_prepare", "pb_get_plan", "pb_solve_batch", "pb_solve_batch_charges", "pb_create_slab", "pb_slab_begin",
           "pb_slab_step", "pb_slab_pointers", "pb_slab_latch", "pb_slab_result", "pb_residual_noalloc")

# pb_option (include/pb.h), by name
OPTIONS = {"persist": 0, "persist_max_mb": 1, "persist_fused_max_knodes": 2, "persist_blocks_per_sm": 3,
           "palette": 4, "palette_diag": 5, "palette_diag_spmv": 6, "autotune": 7, "tile_txv": 8, "tile_ty": 9,
           "tile_tz": 10, "ring_slots": 11, "blocks_per_sm": 12, "vec_blocks_per_sm": 13, "graph": 14, "l2_hints": 15,
           "batch_width": 16, "fused": 17, "tail_pool": 18}


class PBPlan(ctypes.Structure):
    """pb_plan of include/pb.h."""
    _fields_ = [(n, ctypes.c_int) for n in (
        "precision", "num_sm", "persist", "persist_fused", "persist_grid", "palette_size", "diag_palette_size",
        "face_palette", "diag_palette_vec", "diag_palette_spmv", "txv", "ty", "tz", "ring_slots", "blocks_per_sm",
        "tiles", "grid", "threads", "smem_bytes", "autotuned", "vec_grid", "vec_threads", "spmv_bytes_per_node",
        "vec_bytes_per_node", "pitch", "fused", "face_quad", "coef_slots", "tail_pool")] + [("reserved", ctypes.c_int * 4)]


_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


class PBError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        super().__init__(f"{where}: {STATUS_NAMES.get(status, status)} ({pb_strerror(status)})")


def lib_path() -> str:
    return os.path.join(_HERE, "libpb.so")


def load_library():
    """Load libpb.so (built in-tree by paper_1704_02745_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} not found: build it with `python -m paper_1704_02745_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    lib.pb_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, cd, vp, vp, vp, vp, vp, vp, ci, vp]
    lib.pb_set_rhs.argtypes = [vp, vp, vp, ci]
    lib.pb_apply.argtypes = [vp, ci, vp, vp, ci]
    lib.pb_solve.argtypes = [vp, cd, ci, ci, ci, vp, ci, ctypes.POINTER(ci), ctypes.POINTER(cd)]
    lib.pb_solve_begin.argtypes = [vp, ci]
    lib.pb_solve_from.argtypes = [vp, cd, ci, ci, ci, vp, vp, ci, ctypes.POINTER(ci), ctypes.POINTER(cd)]
    lib.pb_iterate.argtypes = [vp, ci, ci]
    lib.pb_destroy.argtypes = [vp]
    lib.pb_query.argtypes = [vp, ci, vp]
    lib.pb_strerror.argtypes = [ci]
    lib.pb_strerror.restype = ctypes.c_char_p
    lib.pb_version.restype = ci
    lib.pb_profile.argtypes = [vp, ci, ci, ctypes.POINTER(cd), ctypes.POINTER(cd)]
    lib.pb_launch_count.argtypes = [vp]
    lib.pb_set_preconditioner.argtypes = [vp, ci]
    lib.pb_set_boundary.argtypes = [vp, ci]
    lib.pb_bytes_per_node.argtypes = [vp, ci, ci]
    lib.pb_bytes_per_node.restype = ci
    lib.pb_solve_refined.argtypes = [vp, cd, ci, cd, ci, vp, ci, ctypes.POINTER(ci), ctypes.POINTER(ci),
                                     ctypes.POINTER(cd)]
    lib.pb_set_setup_precision.argtypes = [vp, ci]
    lib.pb_residual.argtypes = [vp, ci, vp, ci, ctypes.POINTER(cd)]
    lib.pb_create_from_atoms.argtypes = [ctypes.POINTER(vp), ci, ci, ci, cd, ci, vp, vp, vp, cd, cd, cd, ci, vp]
    lib.pb_set_charges.argtypes = [vp, vp, ci]
    lib.pb_get_field.argtypes = [vp, ci, vp]
    lib.pb_palette_size.argtypes = [vp]
    lib.pb_diag_palette_size.argtypes = [vp]
    lib.pb_launch_count.restype = ctypes.c_longlong
    lib.pb_solve_batch.argtypes = [vp, ci, vp, vp, cd, ci, ci, ci, vp, ci, ctypes.POINTER(ci), ctypes.POINTER(cd),
                                   ctypes.POINTER(ci)]
    lib.pb_solve_batch_charges.argtypes = [vp, ci, vp, cd, ci, ci, ci, vp, ci, ctypes.POINTER(ci), ctypes.POINTER(cd),
                                           ctypes.POINTER(ci)]
    lib.pb_create_slab.argtypes = [ctypes.POINTER(vp), ci, ci, ci, cd, vp, vp, vp, vp, vp, vp, ci, vp, ci, ci]
    lib.pb_slab_begin.argtypes = [vp, ci, cd, ci]
    lib.pb_slab_step.argtypes = [vp, ci]
    lib.pb_slab_pointers.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_size_t)]
    lib.pb_slab_latch.argtypes = [vp, ctypes.POINTER(ci), ctypes.POINTER(ci), ctypes.POINTER(ci), ctypes.POINTER(cd)]
    lib.pb_slab_result.argtypes = [vp, vp, ci]
    lib.pb_set_option.argtypes = [vp, ci, ci]
    lib.pb_get_option.argtypes = [vp, ci, ctypes.POINTER(ci)]
    lib.pb_prepare.argtypes = [vp, ci]
    lib.pb_get_plan.argtypes = [vp, ci, ctypes.POINTER(PBPlan)]
    lib.pb_residual_noalloc.argtypes = [ci, ci, ci, cd, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    for name in EXPORTS:
        getattr(lib, name)
    _lib = lib
    return lib


def pb_strerror(status: int) -> str:
    try:
        return load_library().pb_strerror(int(status)).decode()
    except Exception:
        return "?"


NOALLOC_MAX_ROWS = 262144      # PB_NOALLOC_MAX_ROWS of include/pb.h


def residual_noalloc(nx, ny, nz, h, eps_x, eps_y, eps_z, kbar2, rhs, bc, phi, out3, stream=None):
    """pb_residual_noalloc: ||b - A phi|| / ||b|| without any allocation, for callers that cannot call cudaMalloc.

    Every array is a CUDA float64 tensor (contiguous, on the current device; kbar2 / rhs / bc may be None); `out3` is
    the caller's 3-element CUDA float64 tensor {relres, ||r||^2, ||b||^2}, written asynchronously on `stream` (a raw
    cudaStream_t value; None = the legacy default stream).  Argument marshalling only; nothing is copied or allocated.
    Grids with nz * ny > NOALLOC_MAX_ROWS raise PBError(PB_ERR_TOO_LARGE).  Calls share one fixed scratch array per
    GPU: do not let two of them overlap on the device."""
    def dptr(t, name, count):
        if t is None:
            return None
        if not (_is_torch(t) and t.is_cuda and str(t.dtype) == "torch.float64" and t.is_contiguous() and t.numel() == count):
            raise ValueError(f"{name}: expected a contiguous CUDA float64 tensor of {count} elements")
        return ctypes.c_void_p(t.data_ptr())

    nx, ny, nz = int(nx), int(ny), int(nz)
    n = nx * ny * nz
    nbc = 2 * (nz * ny + nz * nx + ny * nx)
    big = nz * ny > NOALLOC_MAX_ROWS          # let the library reject it (before it looks at any pointer)
    args = [(eps_x, "eps_x", nz * ny * (nx + 1)), (eps_y, "eps_y", nz * (ny + 1) * nx), (eps_z, "eps_z", (nz + 1) * ny * nx),
            (kbar2, "kbar2", n), (rhs, "rhs", n), (bc, "bc", nbc), (phi, "phi", n), (out3, "out3", 3)]
    ptrs = [None if big else dptr(t, nm, c) for t, nm, c in args]
    st = load_library().pb_residual_noalloc(nx, ny, nz, float(h), *ptrs, ctypes.c_void_p(stream) if stream else None)
    if st != PB_OK:
        raise PBError(st, "pb_residual_noalloc")
    return out3


def _is_torch(a) -> bool:
    return type(a).__module__.startswith("torch")


def _marshal(a, dtype, count=None, name="array"):
    """-> (pointer, memspace, keepalive).  None -> (NULL, None, None)."""
    if a is None:
        return None, None, None
    if _is_torch(a):
        import torch

        want = {np.float64: torch.float64, np.float32: torch.float32}[dtype]
        if a.dtype != want:
            raise TypeError(f"{name}: expected {want}, got {a.dtype}")
        a = a.contiguous()
        if count is not None and a.numel() != count:
            raise ValueError(f"{name}: expected {count} elements, got {a.numel()}")
        return ctypes.c_void_p(a.data_ptr()), (PB_DEVICE if a.is_cuda else PB_HOST), a
    arr = np.ascontiguousarray(a, dtype=dtype)
    if count is not None and arr.size != count:
        raise ValueError(f"{name}: expected {count} elements, got {arr.size}")
    return ctypes.c_void_p(arr.ctypes.data), PB_HOST, arr


def _one_space(spaces, default=PB_HOST):
    s = {x for x in spaces if x is not None}
    if len(s) > 1:
        raise ValueError("all arrays of one call must live in the same memory space (host or device)")
    return s.pop() if s else default


def _prec(precision):
    if precision in (PB_F32, "f32", "fp32", "float32", np.float32):
        return PB_F32, np.float32
    if precision in (PB_F64, "f64", "fp64", "float64", np.float64):
        return PB_F64, np.float64
    raise ValueError(f"unknown precision {precision!r}")


class PBSolver:
    """One operator (Eq. 3) on one device/stream: pb_create ... pb_destroy."""

    def __init__(self, nx, ny, nz, h, eps_x, eps_y, eps_z, kbar2=None, rhs=None, bc=None, stream=None, options=None):
        lib = load_library()
        self.nx, self.ny, self.nz, self.h = int(nx), int(ny), int(nz), float(h)
        n = self.nx * self.ny * self.nz
        nbc = 2 * (self.nz * self.ny + self.nz * self.nx + self.ny * self.nx)
        f8 = np.float64
        ex, s1, k1 = _marshal(eps_x, f8, self.nz * self.ny * (self.nx + 1), "eps_x")
        ey, s2, k2 = _marshal(eps_y, f8, self.nz * (self.ny + 1) * self.nx, "eps_y")
        ez, s3, k3 = _marshal(eps_z, f8, (self.nz + 1) * self.ny * self.nx, "eps_z")
        kb, s4, k4 = _marshal(kbar2, f8, n, "kbar2")
        rh, s5, k5 = _marshal(rhs, f8, n, "rhs")
        bv, s6, k6 = _marshal(bc, f8, nbc, "bc")
        where = _one_space([s1, s2, s3, s4, s5, s6])
        self._h = ctypes.c_void_p()
        st = lib.pb_create(ctypes.byref(self._h), self.nx, self.ny, self.nz, self.h, ex, ey, ez, kb, rh, bv,
                           where, ctypes.c_void_p(int(stream) if stream else None))
        del k1, k2, k3, k4, k5, k6
        if st != PB_OK:
            self._h = None
            raise PBError(st, "pb_create")
        self.set_options(options)

    @classmethod
    def from_atoms(cls, nx, ny, nz, h, centres, radii, charges, eps_in, eps_out, kbar2_solvent, stream=None,
                   options=None):
        """pb_create_from_atoms: grid / stencil setup on the GPU (mask, face eps, salt map, charges, DH ghosts)."""
        lib = load_library()
        self = cls.__new__(cls)
        self.nx, self.ny, self.nz, self.h = int(nx), int(ny), int(nz), float(h)
        na = int(np.asarray(radii).shape[0]) if not _is_torch(radii) else int(radii.numel())
        c, s1, k1 = _marshal(centres, np.float64, 3 * na, "centres")
        r, s2, k2 = _marshal(radii, np.float64, na, "radii")
        q, s3, k3 = _marshal(charges, np.float64, na, "charges")
        self._h = ctypes.c_void_p()
        st = lib.pb_create_from_atoms(ctypes.byref(self._h), self.nx, self.ny, self.nz, self.h, na, c, r, q,
                                      float(eps_in), float(eps_out), float(kbar2_solvent), _one_space([s1, s2, s3]),
                                      ctypes.c_void_p(int(stream) if stream else None))
        del k1, k2, k3
        if st != PB_OK:
            self._h = None
            raise PBError(st, "pb_create_from_atoms")
        self.n_atoms = na
        self.set_options(options)
        return self

    def set_option(self, name, value):
        """pb_set_option: per-handle tunable (names in OPTIONS); drops the work arrays / plan if the value changes."""
        st = load_library().pb_set_option(self._h, OPTIONS[name], int(value))
        if st != PB_OK:
            raise PBError(st, f"pb_set_option({name}, {value})")

    def set_options(self, options):
        for k, v in (options or {}).items():
            self.set_option(k, v)

    def get_option(self, name) -> int:
        out = ctypes.c_int(0)
        st = load_library().pb_get_option(self._h, OPTIONS[name], ctypes.byref(out))
        if st != PB_OK:
            raise PBError(st, "pb_get_option")
        return out.value

    def prepare(self, precision):
        """pb_prepare: build the work arrays of a precision and pick its launch plan now."""
        st = load_library().pb_prepare(self._h, _prec(precision)[0])
        if st != PB_OK:
            raise PBError(st, "pb_prepare")

    def plan(self, precision) -> dict:
        """pb_get_plan as a dict (tile, ring, grids, palettes, bytes per node)."""
        pl = PBPlan()
        st = load_library().pb_get_plan(self._h, _prec(precision)[0], ctypes.byref(pl))
        if st != PB_OK:
            raise PBError(st, "pb_get_plan")
        return {n: getattr(pl, n) for n, _ in PBPlan._fields_ if n != "reserved"}

    def set_charges(self, charges):
        q, sp, keep = _marshal(charges, np.float64, self.n_atoms, "charges")
        st = load_library().pb_set_charges(self._h, q, sp)
        del keep
        if st != PB_OK:
            raise PBError(st, "pb_set_charges")

    def field(self, name):
        """Dense fp64 input field held by the handle: eps_x, eps_y, eps_z, kbar2, rhs or bc (numpy)."""
        nx, ny, nz = self.nx, self.ny, self.nz
        shapes = {"eps_x": (nz, ny, nx + 1), "eps_y": (nz, ny + 1, nx), "eps_z": (nz + 1, ny, nx),
                  "kbar2": (nz, ny, nx), "rhs": (nz, ny, nx), "bc": (2 * (nz * ny + nz * nx + ny * nx),)}
        which = list(shapes).index(name)
        out = np.empty(shapes[name], dtype=np.float64)
        st = load_library().pb_get_field(self._h, which, ctypes.c_void_p(out.ctypes.data))
        if st != PB_OK:
            raise PBError(st, "pb_get_field")
        return out

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    def set_rhs(self, rhs, bc):
        n = self.nx * self.ny * self.nz
        nbc = 2 * (self.nz * self.ny + self.nz * self.nx + self.ny * self.nx)
        rh, s1, k1 = _marshal(rhs, np.float64, n, "rhs")
        bv, s2, k2 = _marshal(bc, np.float64, nbc, "bc")
        st = load_library().pb_set_rhs(self._h, rh, bv, _one_space([s1, s2]))
        del k1, k2
        if st != PB_OK:
            raise PBError(st, "pb_set_rhs")

    def apply(self, x, precision=None):
        """y = A x (Eq. 3 left-hand side, ghost x = 0).  numpy in -> numpy out; CUDA tensor in -> CUDA tensor out."""
        if precision is None:
            is32 = (str(x.dtype).endswith("float32"))
            precision = PB_F32 if is32 else PB_F64
        pc, dt = _prec(precision)
        n = self.nx * self.ny * self.nz
        xp, sx, keep = _marshal(x, dt, n, "x")
        if _is_torch(x):
            import torch

            y = torch.empty(self.shape, dtype=keep.dtype, device=keep.device)
            yp = ctypes.c_void_p(y.data_ptr())
        else:
            y = np.empty(self.shape, dtype=dt)
            yp = ctypes.c_void_p(y.ctypes.data)
        st = load_library().pb_apply(self._h, pc, xp, yp, sx)
        if st != PB_OK:
            raise PBError(st, "pb_apply")
        return y

    def solve(self, tol, maxiter, precision="f64", check_every=32, out=None, phi0=None):
        """Jacobi-PCG.  Returns dict(phi, iters, relres, status).

        `out`: optional numpy array / torch tensor (host or CUDA) receiving phi; default a new numpy array.
        PB_ERR_MAXITER and PB_ERR_BREAKDOWN are reported in `status`, other errors raise.
        """
        pc, dt = _prec(precision)
        n = self.nx * self.ny * self.nz
        if out is None:
            out = np.empty(self.shape, dtype=dt)
        if not _is_torch(out) and (out.dtype != dt or not out.flags.c_contiguous):
            raise TypeError("out must be a C-contiguous array of the requested precision")
        op, so, keep = _marshal(out, dt, n, "out")
        if _is_torch(out) and keep.data_ptr() != out.data_ptr():
            raise TypeError("out must be contiguous")
        it = ctypes.c_int(0)
        rel = ctypes.c_double(0.0)
        if phi0 is None:
            st = load_library().pb_solve(self._h, float(tol), int(maxiter), pc, int(check_every), op, so,
                                         ctypes.byref(it), ctypes.byref(rel))
        else:   # initial guess (pb_solve_from): same precision and memory space as the output
            gp, sg, keep0 = _marshal(phi0, dt, n, "phi0")
            if sg != so:
                raise ValueError("phi0 and out must live in the same memory space")
            st = load_library().pb_solve_from(self._h, float(tol), int(maxiter), pc, int(check_every), gp, op, so,
                                              ctypes.byref(it), ctypes.byref(rel))
            del keep0
        if st not in (PB_OK, PB_ERR_MAXITER, PB_ERR_BREAKDOWN):
            raise PBError(st, "pb_solve")
        return dict(phi=out, iters=it.value, relres=rel.value, status=st)

    def _batch_out(self, m, dt, out, like):
        n = self.nx * self.ny * self.nz
        if out is None:
            if like is not None and _is_torch(like) and like.is_cuda:
                import torch

                out = torch.empty((m,) + self.shape, dtype={np.float32: torch.float32, np.float64: torch.float64}[dt],
                                  device=like.device)
            else:
                out = np.empty((m,) + self.shape, dtype=dt)
        if not _is_torch(out) and (out.dtype != dt or not out.flags.c_contiguous):
            raise TypeError("out must be a C-contiguous array of the requested precision")
        op, so, keep = _marshal(out, dt, m * n, "out")
        if _is_torch(out) and keep.data_ptr() != out.data_ptr():
            raise TypeError("out must be contiguous")
        return out, op, so

    def solve_batch(self, rhs, bc, tol, maxiter, precision="f32", check_every=32, out=None):
        """pb_solve_batch: m right-hand sides on this operator, PB_OPT_BATCH_WIDTH members per kernel pass.
        rhs [m][nz][ny][nx], bc [m][nbc] (numpy / CUDA tensors, same memory space; either may be None = 0).
        Returns dict(phi [m][nz][ny][nx], iters [m], relres [m], status [m], worst)."""
        pc, dt = _prec(precision)
        n = self.nx * self.ny * self.nz
        nbc = 2 * (self.nz * self.ny + self.nz * self.nx + self.ny * self.nx)
        src = rhs if rhs is not None else bc
        if src is None:
            raise ValueError("rhs and bc cannot both be None")
        m = int(src.shape[0])
        rh, s1, k1 = _marshal(rhs, np.float64, m * n, "rhs")
        bv, s2, k2 = _marshal(bc, np.float64, m * nbc, "bc")
        out, op, so = self._batch_out(m, dt, out, src)
        where = _one_space([s1, s2, so])
        it, rel, stt = (ctypes.c_int * m)(), (ctypes.c_double * m)(), (ctypes.c_int * m)()
        st = load_library().pb_solve_batch(self._h, m, rh, bv, float(tol), int(maxiter), pc, int(check_every), op, where,
                                           it, rel, stt)
        del k1, k2
        if st not in (PB_OK, PB_ERR_MAXITER, PB_ERR_BREAKDOWN):
            raise PBError(st, "pb_solve_batch")
        return dict(phi=out, iters=list(it), relres=list(rel), status=list(stt), worst=st)

    def solve_batch_charges(self, charges, tol, maxiter, precision="f32", check_every=32, out=None):
        """pb_solve_batch_charges: member s = charge set charges[s] on the atoms of a from_atoms handle."""
        pc, dt = _prec(precision)
        m = int(charges.shape[0])
        q, sq, kq = _marshal(charges, np.float64, m * self.n_atoms, "charges")
        out, op, so = self._batch_out(m, dt, out, charges)
        where = _one_space([sq, so])
        it, rel, stt = (ctypes.c_int * m)(), (ctypes.c_double * m)(), (ctypes.c_int * m)()
        st = load_library().pb_solve_batch_charges(self._h, m, q, float(tol), int(maxiter), pc, int(check_every), op,
                                                   where, it, rel, stt)
        del kq
        if st not in (PB_OK, PB_ERR_MAXITER, PB_ERR_BREAKDOWN):
            raise PBError(st, "pb_solve_batch_charges")
        return dict(phi=out, iters=list(it), relres=list(rel), status=list(stt), worst=st)

    def solve_refined(self, tol, maxiter, inner_tol=1e-5, check_every=32, out=None):
        """Mixed-precision iterative refinement (pb_solve_refined): fp64 potential and true residual, fp32 Jacobi-PCG
        corrections.  Returns dict(phi [fp64], outer, iters [inner PCG iterations in total], relres [TRUE], status)."""
        n = self.nx * self.ny * self.nz
        if out is None:
            out = np.empty(self.shape, dtype=np.float64)
        if not _is_torch(out) and (out.dtype != np.float64 or not out.flags.c_contiguous):
            raise TypeError("out must be a C-contiguous float64 array")
        op, so, keep = _marshal(out, np.float64, n, "out")
        if _is_torch(out) and keep.data_ptr() != out.data_ptr():
            raise TypeError("out must be contiguous")
        outer, it, rel = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_double(0.0)
        st = load_library().pb_solve_refined(self._h, float(tol), int(maxiter), float(inner_tol), int(check_every),
                                             op, so, ctypes.byref(outer), ctypes.byref(it), ctypes.byref(rel))
        if st not in (PB_OK, PB_ERR_MAXITER, PB_ERR_BREAKDOWN):
            raise PBError(st, "pb_solve_refined")
        return dict(phi=out, outer=outer.value, iters=it.value, relres=rel.value, status=st)

    def set_setup_precision(self, precision):
        """'f64' (default) or 'f32': arithmetic of the Debye-Hueckel boundary sum in set_charges."""
        pc, _ = _prec(precision)
        st = load_library().pb_set_setup_precision(self._h, pc)
        if st != PB_OK:
            raise PBError(st, "pb_set_setup_precision")

    def set_preconditioner(self, jacobi: bool):
        """True (default): Jacobi-PCG; False: unpreconditioned CG (M = I)."""
        st = load_library().pb_set_preconditioner(self._h, 1 if jacobi else 0)
        if st != PB_OK:
            raise PBError(st, "pb_set_preconditioner")

    def set_periodic(self, periodic: bool):
        """False (default): Dirichlet ghost layer; True: periodic boundary condition."""
        st = load_library().pb_set_boundary(self._h, 1 if periodic else 0)
        if st != PB_OK:
            raise PBError(st, "pb_set_boundary")

    def residual(self, phi, precision=None):
        """True relative residual ||b - A phi|| / ||b|| of `phi` (numpy or CUDA tensor), pb_residual."""
        if precision is None:
            precision = PB_F32 if str(phi.dtype).endswith("float32") else PB_F64
        pc, dt = _prec(precision)
        pp, sp, keep = _marshal(phi, dt, self.nx * self.ny * self.nz, "phi")
        out = ctypes.c_double(0.0)
        st = load_library().pb_residual(self._h, pc, pp, sp, ctypes.byref(out))
        del keep
        if st != PB_OK:
            raise PBError(st, "pb_residual")
        return out.value

    def bytes_per_node(self, precision, kernel):
        """Bytes per node and launch of kernel 0 (k_spmv_tma) / 1 (k_vec) in this handle's storage format."""
        pc, _ = _prec(precision)
        n = load_library().pb_bytes_per_node(self._h, pc, int(kernel))
        if n < 0:
            raise PBError(PB_ERR_CUDA, "pb_bytes_per_node")
        return n

    def solve_begin(self, precision):
        st = load_library().pb_solve_begin(self._h, _prec(precision)[0])
        if st != PB_OK:
            raise PBError(st, "pb_solve_begin")

    def iterate(self, precision, n_iter):
        st = load_library().pb_iterate(self._h, _prec(precision)[0], int(n_iter))
        if st != PB_OK:
            raise PBError(st, "pb_iterate")

    def profile(self, precision, n_iter):
        """Mean device ms of (K_spmv, K_vec) over n_iter iterations continuing the current state."""
        a, b = ctypes.c_double(0.0), ctypes.c_double(0.0)
        st = load_library().pb_profile(self._h, _prec(precision)[0], int(n_iter), ctypes.byref(a), ctypes.byref(b))
        if st != PB_OK:
            raise PBError(st, "pb_profile")
        return a.value, b.value

    def palette_size(self) -> int:
        return int(load_library().pb_palette_size(self._h))

    def diag_palette_size(self) -> int:
        return int(load_library().pb_diag_palette_size(self._h))

    def launch_count(self) -> int:
        return int(load_library().pb_launch_count(self._h))

    def _query(self, what):
        out = np.empty(self.shape, dtype=np.float64)
        st = load_library().pb_query(self._h, what, ctypes.c_void_p(out.ctypes.data))
        if st != PB_OK:
            raise PBError(st, "pb_query")
        return out

    def state(self):
        """Device-resident PCG scalars (pb_query what=2) as a dict; diagnostics only."""
        out = np.zeros(10)
        st = load_library().pb_query(self._h, 2, ctypes.c_void_p(out.ctypes.data))
        if st != PB_OK:
            raise PBError(st, "pb_query")
        keys = ("rz", "pAp", "rr", "bb", "alpha", "beta", "l", "done", "status", "iters")
        return dict(zip(keys, out.tolist()))

    def vector(self, name):
        """Work vector 'r', 'Dinv', 'p', 'Ap' or 'x' of the last solve (h^2-scaled system), as fp64 numpy.
        'x' is the stored phi: the update alpha*p of the latest iteration is still pending (see k_finish)."""
        return self._query({"r": 3, "Dinv": 4, "p": 5, "Ap": 6, "x": 7}[name])

    def diag(self):
        return self._query(0)

    def b(self):
        return self._query(1)

    def close(self):
        if getattr(self, "_h", None):
            load_library().pb_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
