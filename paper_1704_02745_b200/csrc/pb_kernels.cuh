// pb_kernels.cuh -- the hot-path kernels of the matrix-free Jacobi-PCG iteration.
//
//   k_spmv_tma (pb_spmv_tma.cuh): z = Dinv r (step 6), p <- z + beta*p (step 7), the deferred
//            phi += alpha p of step 5, Ap = A'p rebuilt on the fly from the face dielectrics of
//            Eq. 3, and the p.Ap dot of step 5 in the epilogue.
//   k_vec  : alpha = rz/pAp (read from the device state); r -= alpha Ap (step 5); r.z = sum r^2 Dinv
//            (Jacobi) and r.r; then beta (step 7) and the stopping rule of step 3.
//   k_init : steps 1-2 with phi_0 = 0;  k_warm: step 1 with a given phi_0.
//   k_finish : the last pending phi += alpha p and the un-padding of phi (row a6).
//
// The solver works on the h^2-scaled system A' = h^2 A, b' = h^2 b (CG iterates and the
// relative residual are invariant under this scaling); see DESIGN.md.
//
// Internal (padded) layout, element type T in {float,double}, row pitch P elements
// (P >= nx+1, P*sizeof(T) a multiple of 32 B), x fastest:
//   node arrays  [nz][ny][P]      p (two ping-pong buffers), Ap, x, r, b, D, Dinv, tmp (pb_apply input)
//   exm          [nz][ny][P]      exm[k][j][i]  = eps_x face between i-1 and i (i = 0..nx), else 0
//   eym          [nz][ny+1][P]    eym[k][f][i]  = eps_y face between j=f-1 and j=f
//   ezm          [nz+1][ny][P]    ezm[f][j][i]  = eps_z face between k=f-1 and k=f
// Pad columns (i >= nx) hold 0 in every vector and coefficient except D = Dinv = 1 and
// exm[nx] (the right-hand face of node nx-1); k_spmv writes A'p = 0 there explicitly, so the
// pads stay exactly 0 through the iteration and never contribute to a dot product.
#pragma once
#include "pb_internal.cuh"
#include "pb_tma.cuh"

namespace pb {

// ---------------------------------------------------------------------------------------
// finaliser shared by k_vec and k_init: beta (step 7) and the stopping rule (step 3)
// ---------------------------------------------------------------------------------------
// init: 0 = an iteration, 1 = steps 1-2 with phi_0 = 0 (r_0 = b), 2 = steps 1-2 with a given phi_0 (||b||^2 kept)
__device__ __forceinline__ void finish_iteration(State *st, double rz_new, double rr, int init)
{
    if (init) {
        if (init == 1) st->bb = rr;  // r_0 = b (phi_0 = 0)
        st->beta = 0.0;              // first k_spmv gives p_0 = z_0 (step 2)
        st->iter_cur = 0;
    } else {
        st->beta = rz_new / st->rz;  // step 7
        st->iter_cur += 1;           // step 4 (counted once the update of step 5 is done)
    }
    st->rz = rz_new;
    st->rr = rr;
    if (!st->latch) return;
    if (init == 2) { st->done = 0; st->status = 0; }   // re-decide what the phi_0 = 0 pass latched
    const double bb = st->bb;
    const int l = st->iter_cur;
    if (!isfinite(rr) || !isfinite(rz_new)) { st->done = 1; st->iters = l; st->status = 5; }
    else if (bb == 0.0 || rr < st->tol2 * bb) { st->done = 1; st->iters = l; st->status = 0; }  // step 3
    else if (l >= st->maxiter) { st->done = 1; st->iters = l; st->status = 6; }
}

template <typename T>
struct VecArgs {
    T *r;
    const T *Ap, *Dinv;
    const T *b;               // k_init only
    T *x, *pzero;             // k_init only: phi_0 = 0 and the p buffer to clear
    size_t nvec;              // number of 16-byte vectors in a padded node array
    int precond;              // 1: Jacobi (z = Dinv r), 0: M = I (z = r)
    int l2hints;              // 1: keep r and Dinv in L2 for the next k_spmv_tma, stream Ap
    const unsigned char *dvi; // PALD: one index byte per node into dlut instead of the Dinv word (k_vec only)
    const T *dlut;            // PALD: 256 values of Dinv
    State *st;
    double *partials;         // 2 per block
};

// stage 1 + stage 2 of the two dots of k_vec / k_init, then the finaliser
__device__ __forceinline__ void reduce_and_finish(State *st, double *partials, double s_rz, double s_rr,
                                                  double *red, int *s_last, int init)
{
    const double t_rz = block_sum(s_rz, red);
    const double t_rr = block_sum(s_rr, red);
    const int nblk = gridDim.x;
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = t_rz;
        partials[nblk + blockIdx.x] = t_rr;
        __threadfence();
        const unsigned int t = atomicAdd(&st->ticket_vec, 1u);
        *s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (*s_last) {
        __threadfence();
        const double rz = final_sum(partials, nblk, red);
        const double rr = final_sum(partials + nblk, nblk, red);
        if (threadIdx.x == 0) {
            st->ticket_vec = 0u;
            if (st->slab) { st->loc_rz = rz; st->loc_rr = rr; }      // local sums: k_slab_finish after the all-reduce
            else finish_iteration(st, rz, rr, init);
        }
    }
}

// 4 words per node: reads r, Ap, Dinv; writes r.  The sweep runs from the END of the arrays
// towards the start: k_spmv_tma finishes at high z, so its last-written Ap lines are still in L2.
template <typename T, bool PALD>
__global__ void __launch_bounds__(256) k_vec(const VecArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    __shared__ double red[32];
    __shared__ int s_last;
    __shared__ T dlut[PALD ? 256 : 1];
    if (a.st->done) return;
    if (PALD) {
        for (int i = threadIdx.x; i < 256; i += blockDim.x) dlut[i] = a.dlut[i];
        __syncthreads();
    }
    const T alpha = (T)a.st->alpha;
    const uint64_t pol_keep = l2_policy((a.l2hints & 1) ? 2 : 0), pol_stream = l2_policy((a.l2hints & 2) ? 1 : 0);
    double s_rz = 0.0, s_rr = 0.0;
    // two vectors per thread and pass (both fully coalesced across the warp): all loads are issued before the first
    // use, which is what keeps enough bytes in flight when a vector is only two fp64 nodes
    const size_t chunk = 2 * (size_t)blockDim.x, stride = (size_t)gridDim.x * chunk;
    for (size_t v0 = (size_t)blockIdx.x * chunk + threadIdx.x; v0 < a.nvec; v0 += stride) {
        const size_t v1 = v0 + blockDim.x;
        const bool two = v1 < a.nvec;
        const size_t idx0 = (a.nvec - 1 - v0) * VEC, idx1 = two ? (a.nvec - 1 - v1) * VEC : idx0;
        Vec<T> r0, q0, d0, r1, q1, d1;
        ld16_hint(r0.a, a.r + idx0, pol_keep);
        ld16_hint(q0.a, a.Ap + idx0, pol_stream);
        ld16_hint(r1.a, a.r + idx1, pol_keep);
        ld16_hint(q1.a, a.Ap + idx1, pol_stream);
        if (PALD) {
            const uint32_t w0 = (VEC == 4) ? *reinterpret_cast<const uint32_t *>(a.dvi + idx0)
                                           : (uint32_t)*reinterpret_cast<const unsigned short *>(a.dvi + idx0);
            const uint32_t w1 = (VEC == 4) ? *reinterpret_cast<const uint32_t *>(a.dvi + idx1)
                                           : (uint32_t)*reinterpret_cast<const unsigned short *>(a.dvi + idx1);
#pragma unroll
            for (int e = 0; e < VEC; e++) { d0.a[e] = dlut[(w0 >> (8 * e)) & 255u]; d1.a[e] = dlut[(w1 >> (8 * e)) & 255u]; }
        } else {
            ld16_hint(d0.a, a.Dinv + idx0, pol_keep);
            ld16_hint(d1.a, a.Dinv + idx1, pol_keep);
        }
#pragma unroll
        for (int e = 0; e < VEC; e++) {
            r0.a[e] = fma(-alpha, q0.a[e], r0.a[e]);      // r_l = r_{l-1} - alpha A p     (step 5)
            const T zv = a.precond ? d0.a[e] * r0.a[e] : r0.a[e];   // M z_l = r_l, M = D or I   (step 6)
            s_rz = fma((double)r0.a[e], (double)zv, s_rz);
            s_rr = fma((double)r0.a[e], (double)r0.a[e], s_rr);
        }
        st16_hint(a.r + idx0, r0.a, pol_keep);
        if (two) {
#pragma unroll
            for (int e = 0; e < VEC; e++) {
                r1.a[e] = fma(-alpha, q1.a[e], r1.a[e]);
                const T zv = a.precond ? d1.a[e] * r1.a[e] : r1.a[e];
                s_rz = fma((double)r1.a[e], (double)zv, s_rz);
                s_rr = fma((double)r1.a[e], (double)r1.a[e], s_rr);
            }
            st16_hint(a.r + idx1, r1.a, pol_keep);
        }
    }
    reduce_and_finish(a.st, a.partials, s_rz, s_rr, red, &s_last, 0);
}

// k_vec for M right-hand sides on one operator: member s lives at r + s*stride, Ap + s*stride,
// its scalars in st[s], its partials at partials + s*2*gridDim.x.  Dinv (word or palette byte) is read once per node
// for all members; a member whose latch is set is skipped.  Per member the arithmetic and the order of the
// reduction are those of k_vec run with one vector per thread and pass.
template <typename T, bool PALD, int M>
__global__ void __launch_bounds__(256) k_vec_batch(const VecArgs<T> a, size_t stride)
{
    constexpr int VEC = VecN<T>::value;
    __shared__ double red[32];
    __shared__ int s_last;
    __shared__ T dlut[PALD ? 256 : 1];
    bool live[M];
    T alpha[M];
    bool any = false;
#pragma unroll
    for (int s = 0; s < M; s++) { live[s] = !a.st[s].done; any |= live[s]; alpha[s] = (T)a.st[s].alpha; }
    if (!any) return;
    if (PALD) {
        for (int i = threadIdx.x; i < 256; i += blockDim.x) dlut[i] = a.dlut[i];
        __syncthreads();
    }
    double s_rz[M], s_rr[M];
#pragma unroll
    for (int s = 0; s < M; s++) { s_rz[s] = 0.0; s_rr[s] = 0.0; }
    const size_t step = (size_t)gridDim.x * blockDim.x;
    for (size_t v0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v0 < a.nvec; v0 += step) {
        const size_t idx = (a.nvec - 1 - v0) * VEC;
        Vec<T> r[M], q[M], d;
#pragma unroll
        for (int s = 0; s < M; s++)
            if (live[s]) { r[s] = ldv(a.r + s * stride + idx); q[s] = ldv(a.Ap + s * stride + idx); }
        if (PALD) {
            const uint32_t w = (VEC == 4) ? *reinterpret_cast<const uint32_t *>(a.dvi + idx)
                                          : (uint32_t)*reinterpret_cast<const unsigned short *>(a.dvi + idx);
#pragma unroll
            for (int e = 0; e < VEC; e++) d.a[e] = dlut[(w >> (8 * e)) & 255u];
        } else {
            d = ldv(a.Dinv + idx);
        }
#pragma unroll
        for (int s = 0; s < M; s++) {
            if (!live[s]) continue;
#pragma unroll
            for (int e = 0; e < VEC; e++) {
                r[s].a[e] = fma(-alpha[s], q[s].a[e], r[s].a[e]);              // r_l = r_{l-1} - alpha A p   (step 5)
                const T zv = a.precond ? d.a[e] * r[s].a[e] : r[s].a[e];       // M z_l = r_l                (step 6)
                s_rz[s] = fma((double)r[s].a[e], (double)zv, s_rz[s]);
                s_rr[s] = fma((double)r[s].a[e], (double)r[s].a[e], s_rr[s]);
            }
            stv(a.r + s * stride + idx, r[s]);
        }
    }
    const int nblk = gridDim.x;
    double t_rz[M], t_rr[M];
#pragma unroll
    for (int s = 0; s < M; s++) { t_rz[s] = block_sum(s_rz[s], red); t_rr[s] = block_sum(s_rr[s], red); }
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < M; s++) {
            a.partials[(size_t)s * 2 * nblk + blockIdx.x] = t_rz[s];
            a.partials[(size_t)s * 2 * nblk + nblk + blockIdx.x] = t_rr[s];
        }
        __threadfence();
        const unsigned int t = atomicAdd(&a.st->ticket_vec, 1u);
        s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
#pragma unroll
        for (int s = 0; s < M; s++) {
            const double rz = final_sum(a.partials + (size_t)s * 2 * nblk, nblk, red);
            const double rr = final_sum(a.partials + (size_t)s * 2 * nblk + nblk, nblk, red);
            if (threadIdx.x == 0 && live[s]) finish_iteration(a.st + s, rz, rr, 0);
        }
        if (threadIdx.x == 0) a.st->ticket_vec = 0u;
    }
}

// steps 1-2 with phi_0 = 0: x = 0, r = b, p buffer cleared, r.z and r.r
template <typename T>
__global__ void __launch_bounds__(256) k_init(const VecArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    __shared__ double red[32];
    __shared__ int s_last;
    double s_rz = 0.0, s_rr = 0.0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < a.nvec; v += stride) {
        const size_t idx = v * VEC;
        const Vec<T> rv = ldv(a.b + idx);
        const Vec<T> dv = ldv(a.Dinv + idx);
#pragma unroll
        for (int e = 0; e < VEC; e++) {
            const T zv = a.precond ? dv.a[e] * rv.a[e] : rv.a[e];
            s_rz = fma((double)rv.a[e], (double)zv, s_rz);
            s_rr = fma((double)rv.a[e], (double)rv.a[e], s_rr);
        }
        stv(a.x + idx, zerov<T>());
        stv(a.pzero + idx, zerov<T>());
        stv(a.r + idx, rv);
    }
    reduce_and_finish(a.st, a.partials, s_rz, s_rr, red, &s_last, 1);
}

// step 1 with a given initial guess (r_0 = b - A phi_0), run after k_init and after k_spmv_tma<MODE 1>
// has put A'phi_0 into Ap:  x = phi_0 (padded, in `x0`),  r = b - A'phi_0,  r.z and r.r;  ||b||^2 stays from k_init.
template <typename T>
__global__ void __launch_bounds__(256) k_warm(const VecArgs<T> a, const T *__restrict__ x0)
{
    constexpr int VEC = VecN<T>::value;
    __shared__ double red[32];
    __shared__ int s_last;
    double s_rz = 0.0, s_rr = 0.0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < a.nvec; v += stride) {
        const size_t idx = v * VEC;
        Vec<T> rv = ldv(a.b + idx);
        const Vec<T> qv = ldv(a.Ap + idx);
        const Vec<T> dv = ldv(a.Dinv + idx);
#pragma unroll
        for (int e = 0; e < VEC; e++) {
            rv.a[e] = rv.a[e] - qv.a[e];
            const T zv = a.precond ? dv.a[e] * rv.a[e] : rv.a[e];
            s_rz = fma((double)rv.a[e], (double)zv, s_rz);
            s_rr = fma((double)rv.a[e], (double)rv.a[e], s_rr);
        }
        stv(a.x + idx, ldv(x0 + idx));
        stv(a.r + idx, rv);
    }
    reduce_and_finish(a.st, a.partials, s_rz, s_rr, red, &s_last, 2);
}

// row a6: phi_out (dense [nz][ny][nx], type S) = x + alpha*p -- the phi update of the last
// iteration, which k_spmv_tma would have applied one kernel later (alpha = 0 after a breakdown
// or when no iteration ran).
template <typename T, typename S>
__global__ void k_finish(const T *__restrict__ x, const T *__restrict__ pbuf0, const T *__restrict__ pbuf1,
                         const State *st, S *dst, int nx, int P, size_t rows, const T *__restrict__ x_alt = nullptr)
{
    if (x_alt && st->xbuf) x = x_alt;          // k_pcg_fused double-buffers x: st->xbuf names the current one
    const T alpha = (T)st->alpha;
    const T *p = (st->iter_cur & 1) ? pbuf1 : pbuf0;
    const size_t total = rows * nx;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % nx);
        const size_t row = t / nx;
        // alpha = 0: nothing pending (no iteration ran, or a breakdown: p may hold non-finite values, 0*NaN = NaN)
        dst[t] = (alpha == T(0)) ? (S)x[row * P + i] : (S)fma(alpha, p[row * P + i], x[row * P + i]);
    }
}

}  // namespace pb

// ---------------------------------------------------------------------------------------
// Periodic boundary condition.  k_spmv_tma computes A'p with p = 0 outside the
// grid; under the periodic condition the neighbour across a box face is the node on the opposite side, so the
// nodes of the boundary shell lack the terms  -eps_face * p(opposite node).  k_wrap adds them (one thread per
// shell node, so every A'p entry has one writer), corrects p.Ap and recomputes alpha with the stopping checks of
// the k_spmv_tma finaliser.  In a matrix-free kernel the paper's "6 extra bands" are just these index wraps.
// ---------------------------------------------------------------------------------------
namespace pb {

template <typename T>
struct WrapArgs {
    const T *pbuf0, *pbuf1;   // MODE 0: p = buf[(l+1)&1] (what k_spmv_tma just wrote);  MODE 1: pbuf0 = the input vector
    T *Ap;
    const double *eps_x, *eps_y, *eps_z;   // dense fp64 inputs: only the outer faces f = 0 and f = n are read
    int nx, ny, nz, P;
    double out_scale;         // MODE 1
    State *st;
    double *partials;
};

template <typename T, int MODE>
__global__ void __launch_bounds__(256) k_wrap(const WrapArgs<T> a)
{
    __shared__ double red[32];
    __shared__ int s_last;
    const T *p = a.pbuf0;
    if (MODE == 0) {
        if (a.st->done) return;
        p = (a.st->iter_cur & 1) ? a.pbuf0 : a.pbuf1;
    }
    const int nx = a.nx, ny = a.ny, nz = a.nz, P = a.P;
    // shell nodes, each owned once: the two z faces (full planes), then the y faces of the inner planes, then the x faces
    const size_t n_z = (size_t)(nz > 1 ? 2 : 1) * ny * nx;
    const int kin = nz > 2 ? nz - 2 : 0;                       // inner planes 1..nz-2
    const size_t n_y = (size_t)kin * (ny > 1 ? 2 : 1) * nx;
    const int jin = ny > 2 ? ny - 2 : 0;
    const size_t n_x = (size_t)kin * jin * (nx > 1 ? 2 : 1);
    const size_t total = n_z + n_y + n_x;
    double acc = 0.0;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
        int i, j, k;
        if (t < n_z) {
            const size_t u = t % ((size_t)ny * nx);
            k = (t < (size_t)ny * nx) ? 0 : nz - 1; j = (int)(u / nx); i = (int)(u % nx);
        } else if (t < n_z + n_y) {
            const size_t v = t - n_z, per_k = (size_t)(ny > 1 ? 2 : 1) * nx, u = v % per_k;
            k = 1 + (int)(v / per_k); j = (u < (size_t)nx) ? 0 : ny - 1; i = (int)(u % nx);
        } else {
            const size_t v = t - n_z - n_y, per_j = (nx > 1 ? 2 : 1), per_k = (size_t)jin * per_j, u = v % per_k;
            k = 1 + (int)(v / per_k); j = 1 + (int)(u / per_j); i = (u % per_j) ? nx - 1 : 0;
        }
        const size_t row = (size_t)k * ny + j, idx = row * P + i;
        T d = T(0);                                            // the missing terms -eps_f * p(opposite)
        if (i == 0)      d = fma(-(T)a.eps_x[row * (nx + 1)], p[row * P + nx - 1], d);
        if (i == nx - 1) d = fma(-(T)a.eps_x[row * (nx + 1) + nx], p[row * P], d);
        if (j == 0)      d = fma(-(T)a.eps_y[((size_t)k * (ny + 1)) * nx + i], p[((size_t)k * ny + ny - 1) * P + i], d);
        if (j == ny - 1) d = fma(-(T)a.eps_y[((size_t)k * (ny + 1) + ny) * nx + i], p[((size_t)k * ny) * P + i], d);
        if (k == 0)      d = fma(-(T)a.eps_z[(size_t)j * nx + i], p[((size_t)(nz - 1) * ny + j) * P + i], d);
        if (k == nz - 1) d = fma(-(T)a.eps_z[((size_t)nz * ny + j) * nx + i], p[((size_t)j) * P + i], d);
        if (MODE == 1) d = (T)((double)d * a.out_scale);
        a.Ap[idx] += d;
        if (MODE == 0) acc = fma((double)p[idx], (double)d, acc);
    }
    if (MODE == 0) {
        const double tot = block_sum(acc, red);
        const int nblk = gridDim.x;
        if (threadIdx.x == 0) {
            a.partials[blockIdx.x] = tot;
            __threadfence();
            const unsigned int t = atomicAdd(&a.st->ticket_spmv, 1u);
            s_last = (t == (unsigned int)(nblk - 1));
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            const double dp = final_sum(a.partials, nblk, red);
            if (threadIdx.x == 0) {
                State *st = a.st;
                st->ticket_spmv = 0u;
                const double pAp = st->pAp + dp;
                st->pAp = pAp;
                if (!(pAp > 0.0) || !isfinite(pAp)) {
                    if (st->latch) { st->done = 1; st->iters = st->iter_cur; st->status = 5; }
                    st->alpha = 0.0;
                } else {
                    st->alpha = st->rz / pAp;
                }
            }
        }
    }
}

// ||b - A'phi||^2 and ||b||^2 (A'phi in Ap): the TRUE residual of a given potential, as opposed to the recurrence
// residual the iteration tests (DESIGN.md Reading 5).  Same two-stage deterministic reduction; result in st->rr, st->bb.
template <typename T>
__global__ void __launch_bounds__(256) k_true_residual(const T *__restrict__ b, const T *__restrict__ Ap, size_t nvec,
                                                       State *st, double *partials, T *rout = nullptr)
{
    constexpr int VEC = VecN<T>::value;
    __shared__ double red[32];
    __shared__ int s_last;
    double s_rr = 0.0, s_bb = 0.0;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < nvec; v += (size_t)gridDim.x * blockDim.x) {
        Vec<T> bv = ldv(b + v * VEC);
        const Vec<T> qv = ldv(Ap + v * VEC);
#pragma unroll
        for (int e = 0; e < VEC; e++) {
            const double d = (double)bv.a[e] - (double)qv.a[e];
            s_rr = fma(d, d, s_rr);
            s_bb = fma((double)bv.a[e], (double)bv.a[e], s_bb);
            bv.a[e] = (T)d;
        }
        if (rout) stv(rout + v * VEC, bv);          // r = b - A'phi kept (iterative refinement)
    }
    const double t_rr = block_sum(s_rr, red), t_bb = block_sum(s_bb, red);
    const int nblk = gridDim.x;
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = t_rr;
        partials[nblk + blockIdx.x] = t_bb;
        __threadfence();
        s_last = (atomicAdd(&st->ticket_vec, 1u) == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        const double rr = final_sum(partials, nblk, red), bb = final_sum(partials + nblk, nblk, red);
        if (threadIdx.x == 0) { st->ticket_vec = 0u; st->rr = rr; st->bb = bb; }
    }
}

// Mixed-precision iterative refinement: the fp64 residual becomes the fp32 right-hand side, and
// the fp32 correction x + alpha p (its last update still pending, as in k_finish) is added to the fp64 potential.
template <typename S, typename T>
__global__ void k_repad(const S *__restrict__ src, int Ps, T *dst, int Pd, int nx, size_t rows)
{
    const size_t total = rows * Pd;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % Pd);
        const size_t row = t / Pd;
        dst[t] = (i < nx) ? (T)src[row * Ps + i] : T(0);
    }
}

template <typename T, typename S>
__global__ void k_finish_add(const T *__restrict__ x, const T *__restrict__ pbuf0, const T *__restrict__ pbuf1,
                             const State *st, S *acc, int nx, int P, int Pacc, size_t rows,
                             const T *__restrict__ x_alt = nullptr)
{
    if (x_alt && st->xbuf) x = x_alt;          // k_pcg_fused double-buffers x (as in k_finish)
    const T alpha = (T)st->alpha;
    const T *p = (st->iter_cur & 1) ? pbuf1 : pbuf0;
    const size_t total = rows * nx;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % nx);
        const size_t row = t / nx;
        acc[row * Pacc + i] += (alpha == T(0)) ? (S)x[row * P + i] : (S)fma(alpha, p[row * P + i], x[row * P + i]);
    }
}

}  // namespace pb

// ---------------------------------------------------------------------------------------
// z-slab decomposition of one solve over several GPUs (the paper's node had two GPUs,
// PAPER.md:184).  Each rank owns nz_local planes plus one ghost plane of r, p and Dinv on either side; per iteration
// the ranks exchange the boundary planes of r and p and all-reduce p.Ap and {r.z, r.r} (the caller does both, with
// NCCL through torch.distributed; the sums live in the State).  These kernels are the scalar steps that follow an
// all-reduce -- the same decisions as the single-GPU finalisers, taken identically on every rank.
// ---------------------------------------------------------------------------------------
namespace pb {

__global__ void k_slab_alpha(State *st)        // after the all-reduce of st->pAp: step 5
{
    if (st->done) return;
    const double pAp = st->pAp;
    if (!(pAp > 0.0) || !isfinite(pAp)) {
        if (st->latch) { st->done = 1; st->iters = st->iter_cur; st->status = 5; }
        st->alpha = 0.0;
    } else {
        st->alpha = st->rz / pAp;
    }
}

__global__ void k_slab_finish(State *st, int init)   // after the all-reduce of {loc_rz, loc_rr}: steps 3 and 7
{
    if (!init && st->done) return;
    finish_iteration(st, st->loc_rz, st->loc_rr, init);
}

// boundary planes -> send buffer [r_lo | p_lo | r_hi | p_hi] (p = the buffer the NEXT k_spmv_tma reads), and
// receive buffer [r_below | p_below | r_above | p_above] -> ghost planes.  `plane` = ny*P elements.
template <typename T>
__global__ void k_slab_pack(const T *__restrict__ r, const T *__restrict__ p0, const T *__restrict__ p1,
                            const State *st, T *send, size_t plane, int nz)
{
    const T *p = (st->iter_cur & 1) ? p1 : p0;
    const size_t top = (size_t)(nz - 1) * plane;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < plane; t += (size_t)gridDim.x * blockDim.x) {
        send[t] = r[t];
        send[plane + t] = p[t];
        send[2 * plane + t] = r[top + t];
        send[3 * plane + t] = p[top + t];
    }
}

template <typename T>
__global__ void k_slab_unpack(T *r, T *p0, T *p1, const State *st, const T *__restrict__ recv, size_t plane, int nz,
                              int iface_lo, int iface_hi)
{
    T *p = (st->iter_cur & 1) ? p1 : p0;
    const size_t above = (size_t)nz * plane;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < plane; t += (size_t)gridDim.x * blockDim.x) {
        if (iface_lo) { (r - plane)[t] = recv[t]; (p - plane)[t] = recv[plane + t]; }
        if (iface_hi) { r[above + t] = recv[2 * plane + t]; p[above + t] = recv[3 * plane + t]; }
    }
}

}  // namespace pb
