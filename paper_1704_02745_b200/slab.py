"""One Jacobi-PCG solve over several GPUs: z-slab decomposition (the paper's node had
two GPUs).

Every step of the method runs in the CUDA library (pb_slab_* of include/pb.h: K_spmv and K_vec on the rank's slab with
one ghost plane of r, p and Dinv on either side, the scalar steps after each all-reduce).  This module is plumbing
only: it cuts the inputs into slabs, moves the boundary planes between neighbouring ranks and all-reduces the three
dot products -- over NCCL (torch.distributed) between processes, by plain device copies between slabs that live in
the same process (which is how the path is exercised on a single GPU: all slabs in one process, one stream).

Per iteration and rank: 2 x 2 planes of ny*pitch elements to each neighbour (r and p boundary planes) and two
all-reduces (1 and 2 doubles).  At 385^3 fp32 a plane is 0.6 MB: the exchange is latency-, not bandwidth-bound
(SURVEY.md section 5), so strong scaling of one solve is limited by the two all-reduce latencies per iteration.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import binding as B


def partition(nz: int, nslabs: int):
    """Contiguous z ranges [(z0, nz_local)] -- as even as possible, the first nz % nslabs slabs one plane thicker."""
    if nslabs < 1 or nslabs > nz:
        raise ValueError("need 1 <= nslabs <= nz")
    base, extra = divmod(nz, nslabs)
    out, z0 = [], 0
    for s in range(nslabs):
        n = base + (1 if s < extra else 0)
        out.append((z0, n))
        z0 += n
    return out


def slab_inputs(nx, ny, nz, eps_x, eps_y, eps_z, kbar2, rhs, bc, z0, nzl):
    """The part of the global inputs (layouts of pb_create) that slab [z0, z0 + nzl) owns.  eps_z keeps the nzl + 1
    faces of its planes (an interface face goes to both neighbours); the z- / z+ entries of bc are the global ones at
    the bottom / top slab and zeros across an interface (the library ignores them there)."""
    ex = np.ascontiguousarray(eps_x[z0:z0 + nzl])
    ey = np.ascontiguousarray(eps_y[z0:z0 + nzl])
    ez = np.ascontiguousarray(eps_z[z0:z0 + nzl + 1])
    kb = None if kbar2 is None else np.ascontiguousarray(kbar2[z0:z0 + nzl])
    rh = None if rhs is None else np.ascontiguousarray(rhs[z0:z0 + nzl])
    bcl = None
    if bc is not None:
        bc = np.asarray(bc)
        n_zy, n_zx, n_xy = nz * ny, nz * nx, ny * nx
        xm, xp = bc[:n_zy].reshape(nz, ny), bc[n_zy:2 * n_zy].reshape(nz, ny)
        o = 2 * n_zy
        ym, yp = bc[o:o + n_zx].reshape(nz, nx), bc[o + n_zx:o + 2 * n_zx].reshape(nz, nx)
        o += 2 * n_zx
        zm, zp = bc[o:o + n_xy], bc[o + n_xy:o + 2 * n_xy]
        zero = np.zeros(n_xy)
        bcl = np.concatenate([xm[z0:z0 + nzl].ravel(), xp[z0:z0 + nzl].ravel(), ym[z0:z0 + nzl].ravel(),
                              yp[z0:z0 + nzl].ravel(), zm if z0 == 0 else zero, zp if z0 + nzl == nz else zero])
    return ex, ey, ez, kb, rh, bcl


class _DevMem:
    """Raw device memory as a __cuda_array_interface__ object (wrapped by torch.as_tensor, no copy)."""

    def __init__(self, ptr, count, typestr):
        self.__cuda_array_interface__ = {"shape": (int(count),), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2}


class SlabRank:
    """One slab = one pb handle made by pb_create_slab, plus torch views of its exchange buffers and scalars."""

    def __init__(self, index, nslabs, nx, ny, nzl, h, eps_x, eps_y, eps_z, kbar2, rhs, bc, stream, options=None):
        import torch

        lib = B.load_library()
        self.index, self.nslabs, self.nx, self.ny, self.nz, self.h = index, nslabs, int(nx), int(ny), int(nzl), float(h)
        f8 = np.float64
        n = self.nx * self.ny * self.nz
        ex, s1, k1 = B._marshal(eps_x, f8, self.nz * self.ny * (self.nx + 1), "eps_x")
        ey, s2, k2 = B._marshal(eps_y, f8, self.nz * (self.ny + 1) * self.nx, "eps_y")
        ez, s3, k3 = B._marshal(eps_z, f8, (self.nz + 1) * self.ny * self.nx, "eps_z")
        kb, s4, k4 = B._marshal(kbar2, f8, n, "kbar2")
        rh, s5, k5 = B._marshal(rhs, f8, n, "rhs")
        bv, s6, k6 = B._marshal(bc, f8, 2 * (self.nz * self.ny + self.nz * self.nx + self.ny * self.nx), "bc")
        self._h = ctypes.c_void_p()
        st = lib.pb_create_slab(ctypes.byref(self._h), self.nx, self.ny, self.nz, self.h, ex, ey, ez, kb, rh, bv,
                                B._one_space([s1, s2, s3, s4, s5, s6]), ctypes.c_void_p(int(stream)),
                                1 if index > 0 else 0, 1 if index < nslabs - 1 else 0)
        if st != B.PB_OK:
            self._h = None
            raise B.PBError(st, "pb_create_slab")
        for k, v in (options or {}).items():
            st = lib.pb_set_option(self._h, B.OPTIONS[k], int(v))
            if st != B.PB_OK:
                raise B.PBError(st, f"pb_set_option({k})")
        self._torch = torch
        self.views = None

    def begin(self, precision, tol, maxiter):
        pc, dt = B._prec(precision)
        st = B.load_library().pb_slab_begin(self._h, pc, float(tol), int(maxiter))
        if st != B.PB_OK:
            raise B.PBError(st, "pb_slab_begin")
        ptrs = (ctypes.c_void_p * 8)()
        pbytes = ctypes.c_size_t(0)
        st = B.load_library().pb_slab_pointers(self._h, ptrs, ctypes.byref(pbytes))
        if st != B.PB_OK:
            raise B.PBError(st, "pb_slab_pointers")
        torch = self._torch
        esz = 4 if pc == B.PB_F32 else 8
        ts = "<f4" if pc == B.PB_F32 else "<f8"
        pe = pbytes.value // esz                                  # elements per plane

        def view(i, count, typestr=ts):
            return torch.as_tensor(_DevMem(ptrs[i], count, typestr), device="cuda")

        self.dtype = dt
        self.views = dict(send=view(0, 4 * pe), recv=view(1, 4 * pe), pAp=view(2, 1, "<f8"), rzrr=view(3, 2, "<f8"),
                          dinv_lo=view(4, pe), dinv_hi=view(5, pe), dinv_below=view(6, pe), dinv_above=view(7, pe))
        self.plane = pe

    def step(self, which):
        st = B.load_library().pb_slab_step(self._h, int(which))
        if st != B.PB_OK:
            raise B.PBError(st, f"pb_slab_step({which})")

    def latch(self):
        d, it, stt, rel = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int(0), ctypes.c_double(0.0)
        st = B.load_library().pb_slab_latch(self._h, ctypes.byref(d), ctypes.byref(it), ctypes.byref(stt), ctypes.byref(rel))
        if st != B.PB_OK:
            raise B.PBError(st, "pb_slab_latch")
        return dict(done=bool(d.value), iters=it.value, status=stt.value, relres=rel.value)

    def result(self, device=False):
        """This rank's planes of phi: a numpy array, or (device=True) a CUDA tensor -- no copy to the host."""
        if device:
            torch = self._torch
            out = torch.empty((self.nz, self.ny, self.nx), device="cuda",
                              dtype=torch.float32 if self.dtype == np.float32 else torch.float64)
            st = B.load_library().pb_slab_result(self._h, ctypes.c_void_p(out.data_ptr()), B.PB_DEVICE)
        else:
            out = np.empty((self.nz, self.ny, self.nx), dtype=self.dtype)
            st = B.load_library().pb_slab_result(self._h, ctypes.c_void_p(out.ctypes.data), B.PB_HOST)
        if st != B.PB_OK:
            raise B.PBError(st, "pb_slab_result")
        return out

    def close(self):
        if getattr(self, "_h", None):
            self.views = None
            B.load_library().pb_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class SlabComm:
    """The ranks' exchange.  `owner[s]` = process (torch.distributed rank) that holds slab s; slabs of the calling
    process exchange by device copies, slabs of different processes through torch.distributed (NCCL on GPUs; gloo in
    the CPU tests, where the 'device buffers' are plain CPU tensors)."""

    def __init__(self, owner, my_process=0, dist=None):
        self.owner, self.me, self.dist = list(owner), int(my_process), dist
        self.nslabs = len(self.owner)
        self.graphs = {}          # CUDA graphs of an iteration chunk, per set of ranks (solve_slabs)
        if dist is None and any(o != self.me for o in self.owner):
            raise ValueError("slabs on other processes need torch.distributed")

    def local(self):
        return [s for s, o in enumerate(self.owner) if o == self.me]

    def all_reduce(self, tensors):
        """tensors: {slab index: tensor} of this process's slabs; afterwards every one holds the sum over ALL slabs."""
        loc = self.local()
        total = tensors[loc[0]].clone()
        for s in loc[1:]:
            total += tensors[s]
        if self.dist is not None and any(o != self.me for o in self.owner):
            self.dist.all_reduce(total)
        for s in loc:
            tensors[s].copy_(total)

    def exchange(self, send, recv, halves):
        """send / recv: {slab index: tensor}; every tensor is two halves of `halves` elements -- [to / from the slab
        below | to / from the slab above].  Slab s's lower half goes to the upper half of slab s-1's receive buffer, its
        upper half to the lower half of slab s+1's."""
        ops = []
        for s in self.local():
            for nbr, mine, theirs in ((s - 1, 0, 1), (s + 1, 1, 0)):
                if nbr < 0 or nbr >= self.nslabs:
                    continue
                src = send[s][mine * halves:(mine + 1) * halves]
                if self.owner[nbr] == self.me:
                    recv[nbr][theirs * halves:(theirs + 1) * halves].copy_(src)
                else:
                    dst = recv[s][mine * halves:(mine + 1) * halves]       # what the neighbour sends back to me
                    ops.append(self.dist.P2POp(self.dist.isend, src, self.owner[nbr]))
                    ops.append(self.dist.P2POp(self.dist.irecv, dst, self.owner[nbr]))
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()


def solve_slabs(ranks, comm, tol, maxiter, precision="f32", check_every=32, use_graph=True, device_result=False):
    """Jacobi-PCG on the slabs of this process (`ranks`: {slab index: SlabRank}), in step with the
    other processes through `comm`.  Returns {slab index: dict(phi [nz_local][ny][nx], iters, relres, status)}."""
    ids = sorted(ranks)
    for s in ids:
        ranks[s].begin(precision, tol, maxiter)                    # steps 1-2 on the slab: local r.z, r.r
    comm.all_reduce({s: ranks[s].views["rzrr"] for s in ids})
    for s in ids:
        ranks[s].step(3)                                           # ||b||^2, r_0.z_0, beta = 0, the l = 0 test
    # Dinv ghost planes, once: plane 0 -> the slab below, plane nz-1 -> the slab above
    pe = ranks[ids[0]].plane
    torch = ranks[ids[0]]._torch
    dsend = {s: torch.cat([ranks[s].views["dinv_lo"], ranks[s].views["dinv_hi"]]) for s in ids}
    drecv = {s: torch.zeros_like(dsend[s]) for s in ids}
    comm.exchange(dsend, drecv, pe)
    for s in ids:
        if s > 0:
            ranks[s].views["dinv_below"].copy_(drecv[s][:pe])
        if s < comm.nslabs - 1:
            ranks[s].views["dinv_above"].copy_(drecv[s][pe:])

    def halo():
        for s in ids:
            ranks[s].step(4)
        comm.exchange({s: ranks[s].views["send"] for s in ids}, {s: ranks[s].views["recv"] for s in ids}, 2 * pe)
        for s in ids:
            ranks[s].step(5)

    def chunk():
        for _ in range(check_every):
            for s in ids:
                ranks[s].step(0)                                   # K_spmv; local p.Ap
            comm.all_reduce({s: ranks[s].views["pAp"] for s in ids})
            for s in ids:
                ranks[s].step(1)                                   # alpha; K_vec; local r.z, r.r
            comm.all_reduce({s: ranks[s].views["rzrr"] for s in ids})
            for s in ids:
                ranks[s].step(2)                                   # beta, stopping rule (same decision everywhere)
            halo()

    halo()
    # check_every iterations -- kernels, copies and NCCL calls alike -- captured once into a CUDA graph on the ranks'
    # stream and replayed until the latch is set (kernels after the latch do nothing); eager launches if capture fails
    # (the graph is kept on the communicator and reused by later solves of the same ranks: the captured kernels and
    # copies address the handles' own buffers, which stay put until an option or the precision changes)
    graph = None
    if use_graph:
        key = (tuple(id(ranks[s]) for s in ids), tuple(int(ranks[s].views["send"].data_ptr()) for s in ids),
               str(precision), int(check_every))
        graph = comm.graphs.get(key)
        if graph is None:
            try:
                torch.cuda.synchronize()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=torch.cuda.current_stream()):
                    chunk()
                comm.graphs[key] = graph
            except Exception:
                graph = None
                torch.cuda.synchronize()
    done, l = False, 0                                             # (the capture itself executed nothing)
    while not done:
        if graph is not None:
            graph.replay()
        else:
            chunk()
        l += check_every
        done = ranks[ids[0]].latch()["done"] or l > maxiter + 2 * check_every
    out = {}
    for s in ids:
        st = ranks[s].latch()
        out[s] = dict(phi=ranks[s].result(device=device_result), iters=st["iters"], relres=st["relres"], status=st["status"])
    return out
