// pb_kernels.cuh -- the hot-path kernels of the matrix-free Jacobi-PCG iteration.
//
//   k_spmv : step 7b + step 5a of PAPER.md:118-124:  p <- z + beta*p  (folded in from the
//            previous iteration), Ap = A'p rebuilt on the fly from the face dielectrics of
//            Eq. 3, and the p.Ap dot of step 5 in the epilogue.
//   k_vec  : steps 5b-7a: alpha = rz/pAp; x += alpha p; r -= alpha Ap; z = Dinv r (Jacobi,
//            PAPER.md:138-140); r.z and r.r; then beta and the stopping rule of step 3.
//   k_init : steps 1-2 with phi_0 = 0.
//
// The solver works on the h^2-scaled system A' = h^2 A, b' = h^2 b (CG iterates and the
// relative residual are invariant under this scaling); see DESIGN.md.
//
// Internal (padded) layout, element type T in {float,double}, row pitch P elements
// (P >= nx+1, P*sizeof(T) a multiple of 32 B), x fastest:
//   node arrays  [nz][ny][P]      z, p (two ping-pong buffers), Ap, x, r, b, D, Dinv
//   exm          [nz][ny][P]      exm[k][j][i]  = eps_x face between i-1 and i (i = 0..nx), else 0
//   eym          [nz][ny+1][P]    eym[k][f][i]  = eps_y face between j=f-1 and j=f
//   ezm          [nz+1][ny][P]    ezm[f][j][i]  = eps_z face between k=f-1 and k=f
// Pad columns (i >= nx) hold 0 in every vector and coefficient except D = Dinv = 1 and
// exm[nx] (the right-hand face of node nx-1); k_spmv writes A'p = 0 there explicitly, so the
// pads stay exactly 0 through the iteration and never contribute to a dot product.
#pragma once
#include "pb_internal.cuh"

namespace pb {

template <typename T>
struct SpmvArgs {
    const T *z;              // MODE 0: z_l ; MODE 1: the input vector x
    T *pbuf0, *pbuf1;        // ping-pong p; iteration l reads buf[l&1], writes buf[(l+1)&1]
    T *Ap;                   // output A'p (MODE 1: A x, scaled by out_scale)
    const T *exm, *eym, *ezm, *D;
    int nx, ny, nz, P;
    int TXV, TY, TZ;         // tile: TXV 16-byte vectors wide, TY rows, TZ planes marched per block
    int ntx, nty, ntz;
    State *st;
    double *partials;        // one per block
    double out_scale;        // MODE 1 only
};

// MODE 0: PCG step (p update + A'p + p.Ap);  MODE 1: plain y = scale * A' x
template <typename T, int MODE>
__global__ void __launch_bounds__(512) k_spmv(const SpmvArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    __shared__ int s_last;
    T *sm = reinterpret_cast<T *>(smem_raw);

    const int tid = threadIdx.x, nthr = blockDim.x;
    const T *pin = nullptr;
    T *pout = nullptr;
    T beta = T(0);
    if (MODE == 0) {
        if (a.st->done) return;
        const int it = a.st->iter_cur;
        beta = (T)a.st->beta;
        pin = (it & 1) ? a.pbuf1 : a.pbuf0;
        pout = (it & 1) ? a.pbuf0 : a.pbuf1;
    }
    const int nx = a.nx, ny = a.ny, nz = a.nz, P = a.P;
    const int TXV = a.TXV, TY = a.TY;
    int b = blockIdx.x;
    const int bx = b % a.ntx; b /= a.ntx;
    const int by = b % a.nty;
    const int bz = b / a.nty;
    const int tx = tid % TXV, ty = tid / TXV;
    const int x0 = bx * TXV * VEC, j0 = by * TY;
    const int i0 = x0 + tx * VEC, j = j0 + ty;
    const bool intile = ty < TY;                 // blockDim is rounded up to whole warps
    const bool active = intile && (i0 < P) && (j < ny);
    const int k0 = bz * a.TZ, k1 = min(k0 + a.TZ, nz);
    const int SW = TXV * VEC + 2 * VEC;          // smem row: VEC pad | TXV*VEC data | VEC pad
    const int planeSz = (TY + 2) * SW;
    const int nvalid = nx - i0;                  // elements e < nvalid of this thread's vector are grid nodes

    // p_new = z + beta*p_old at an arbitrary position (0 outside the grid: ghost p = 0)
    auto pnew_vec = [&](int k, int jj, int ii) -> Vec<T> {
        if (k < 0 || k >= nz || jj < 0 || jj >= ny || ii >= P) return zerov<T>();
        const size_t idx = ((size_t)k * ny + jj) * P + ii;
        Vec<T> zv = ldv(a.z + idx);
        if (MODE == 0) {
            const Vec<T> pv = ldv(pin + idx);
#pragma unroll
            for (int e = 0; e < VEC; e++) zv.a[e] = fma(beta, pv.a[e], zv.a[e]);
        }
        return zv;
    };
    auto pnew_scalar = [&](int k, int jj, int ii) -> T {
        if (k < 0 || k >= nz || jj < 0 || jj >= ny || ii < 0 || ii >= P) return T(0);
        const size_t idx = ((size_t)k * ny + jj) * P + ii;
        T zv = a.z[idx];
        if (MODE == 0) zv = fma(beta, pin[idx], zv);
        return zv;
    };
    // stage plane k of p_new into shared buffer s: own vector + the tile's halo rows/columns
    auto stage = [&](int s, int k, const Vec<T> &own) {
        T *pl = sm + s * planeSz;
        if (intile) stv(pl + (ty + 1) * SW + VEC + tx * VEC, own);
        for (int h = tid; h < 2 * TXV; h += nthr) {           // halo rows j0-1 and j0+TY
            const int side = h / TXV, hx = h - side * TXV;
            const int jj = side ? j0 + TY : j0 - 1;
            stv(pl + (side ? TY + 1 : 0) * SW + VEC + hx * VEC, pnew_vec(k, jj, x0 + hx * VEC));
        }
        for (int c = tid; c < 2 * TY; c += nthr) {            // halo columns x0-1 and x0+TXV*VEC
            const int side = c / TY, r = c - side * TY;
            const int ii = side ? x0 + TXV * VEC : x0 - 1;
            pl[(r + 1) * SW + (side ? VEC + TXV * VEC : VEC - 1)] = pnew_scalar(k, j0 + r, ii);
        }
    };

    int sb = 0;
    Vec<T> pm = active ? pnew_vec(k0 - 1, j, i0) : zerov<T>();
    Vec<T> pc = active ? pnew_vec(k0, j, i0) : zerov<T>();
    stage(sb, k0, pc);
    Vec<T> ezc = active ? ldv(a.ezm + ((size_t)k0 * ny + j) * P + i0) : zerov<T>();
    __syncthreads();

    double acc = 0.0;
    for (int k = k0; k < k1; k++) {
        const int sn = (sb == 2) ? 0 : sb + 1;
        const Vec<T> pn = active ? pnew_vec(k + 1, j, i0) : zerov<T>();
        if (k + 1 < k1) stage(sn, k + 1, pn);
        const Vec<T> ezn = active ? ldv(a.ezm + ((size_t)(k + 1) * ny + j) * P + i0) : zerov<T>();
        if (active) {
            const size_t idx = ((size_t)k * ny + j) * P + i0;
            const Vec<T> d = ldv(a.D + idx);
            const Vec<T> ex = ldv(a.exm + idx);
            const T exr = (i0 + VEC < P) ? a.exm[idx + VEC] : T(0);
            const size_t yidx = ((size_t)k * (ny + 1) + j) * P + i0;
            const Vec<T> eyl = ldv(a.eym + yidx);
            const Vec<T> eyh = ldv(a.eym + yidx + P);
            const T *srow = sm + sb * planeSz + (ty + 1) * SW + VEC + tx * VEC;
            const Vec<T> up = ldv(srow - SW);
            const Vec<T> dn = ldv(srow + SW);
            const T left = srow[-1], right = srow[VEC];
            Vec<T> ap;
#pragma unroll
            for (int e = 0; e < VEC; e++) {
                const T pl = (e == 0) ? left : pc.a[e == 0 ? 0 : e - 1];
                const T pr = (e == VEC - 1) ? right : pc.a[e == VEC - 1 ? e : e + 1];
                const T exh = (e == VEC - 1) ? exr : ex.a[e == VEC - 1 ? e : e + 1];
                T v = d.a[e] * pc.a[e];
                v = fma(-ex.a[e], pl, v);
                v = fma(-exh, pr, v);
                v = fma(-eyl.a[e], up.a[e], v);
                v = fma(-eyh.a[e], dn.a[e], v);
                v = fma(-ezc.a[e], pm.a[e], v);
                v = fma(-ezn.a[e], pn.a[e], v);
                if (e >= nvalid) v = T(0);     // pad column: exm[nx] is node nx-1's face, not a row of A
                if (MODE == 0) acc = fma((double)pc.a[e], (double)v, acc);
                ap.a[e] = (MODE == 1) ? (T)((double)v * a.out_scale) : v;
            }
            stv(a.Ap + idx, ap);
            if (MODE == 0) stv(pout + idx, pc);
        }
        __syncthreads();
        pm = pc; pc = pn; ezc = ezn; sb = sn;
    }

    if (MODE == 0) {
        // stage 1 -> per-block partial; stage 2 by the last block to take a ticket
        const double tot = block_sum(acc, red);
        const int nblk = gridDim.x;
        if (tid == 0) {
            a.partials[blockIdx.x] = tot;
            __threadfence();
            const unsigned int t = atomicAdd(&a.st->ticket_spmv, 1u);
            s_last = (t == (unsigned int)(nblk - 1));
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            const double pAp = final_sum(a.partials, nblk, red);
            if (tid == 0) {
                State *st = a.st;
                st->ticket_spmv = 0u;
                st->pAp = pAp;
                if (!(pAp > 0.0) || !isfinite(pAp)) {          // breakdown: not SPD / NaN
                    if (st->latch) { st->done = 1; st->iters = st->iter_cur; st->status = 5; }
                    st->alpha = 0.0;
                } else {
                    st->alpha = st->rz / pAp;                   // step 5
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// finaliser shared by k_vec and k_init: beta (step 7) and the stopping rule (step 3)
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void finish_iteration(State *st, double rz_new, double rr, bool init)
{
    if (init) {
        st->bb = rr;                 // r_0 = b (phi_0 = 0)
        st->beta = 0.0;              // first k_spmv gives p_0 = z_0 (step 2)
        st->iter_cur = 0;
    } else {
        st->beta = rz_new / st->rz;  // step 7
        st->iter_cur += 1;           // step 4 (counted once the update of step 5 is done)
    }
    st->rz = rz_new;
    st->rr = rr;
    if (!st->latch) return;
    const double bb = st->bb;
    const int l = st->iter_cur;
    if (!isfinite(rr) || !isfinite(rz_new)) { st->done = 1; st->iters = l; st->status = 5; }
    else if (bb == 0.0 || rr < st->tol2 * bb) { st->done = 1; st->iters = l; st->status = 0; }  // step 3
    else if (l >= st->maxiter) { st->done = 1; st->iters = l; st->status = 6; }
}

template <typename T>
struct VecArgs {
    const T *pbuf0, *pbuf1;   // k_vec reads the buffer k_spmv just wrote: buf[(l+1)&1]
    T *x, *r, *z;
    const T *Ap, *Dinv;
    const T *b;               // k_init only
    T *pzero;                 // k_init only: p buffer to clear
    size_t nvec;              // number of 16-byte vectors in a padded node array
    State *st;
    double *partials;         // 2 per block
};

template <typename T>
__global__ void __launch_bounds__(256) k_vec(const VecArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    __shared__ double red[32];
    __shared__ int s_last;
    if (a.st->done) return;
    const int it = a.st->iter_cur;
    const T *p = (it & 1) ? a.pbuf0 : a.pbuf1;
    const T alpha = (T)a.st->alpha;
    double s_rz = 0.0, s_rr = 0.0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < a.nvec; v += stride) {
        const size_t idx = v * VEC;
        Vec<T> xv = ldv(a.x + idx);
        const Vec<T> pv = ldv(p + idx);
        Vec<T> rv = ldv(a.r + idx);
        const Vec<T> qv = ldv(a.Ap + idx);
        const Vec<T> dv = ldv(a.Dinv + idx);
        Vec<T> zv;
#pragma unroll
        for (int e = 0; e < VEC; e++) {
            xv.a[e] = fma(alpha, pv.a[e], xv.a[e]);       // phi_l = phi_{l-1} + alpha p   (step 5)
            rv.a[e] = fma(-alpha, qv.a[e], rv.a[e]);      // r_l = r_{l-1} - alpha A p     (step 5)
            zv.a[e] = dv.a[e] * rv.a[e];                  // M z_l = r_l, M = D            (step 6)
            s_rz = fma((double)rv.a[e], (double)zv.a[e], s_rz);
            s_rr = fma((double)rv.a[e], (double)rv.a[e], s_rr);
        }
        stv(a.x + idx, xv);
        stv(a.r + idx, rv);
        stv(a.z + idx, zv);
    }
    const double t_rz = block_sum(s_rz, red);
    const double t_rr = block_sum(s_rr, red);
    const int nblk = gridDim.x;
    if (threadIdx.x == 0) {
        a.partials[blockIdx.x] = t_rz;
        a.partials[nblk + blockIdx.x] = t_rr;
        __threadfence();
        const unsigned int t = atomicAdd(&a.st->ticket_vec, 1u);
        s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        const double rz = final_sum(a.partials, nblk, red);
        const double rr = final_sum(a.partials + nblk, nblk, red);
        if (threadIdx.x == 0) {
            a.st->ticket_vec = 0u;
            finish_iteration(a.st, rz, rr, false);
        }
    }
}

// steps 1-2 with phi_0 = 0: x = 0, r = b, z = Dinv r, p buffer cleared
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
        Vec<T> zv;
#pragma unroll
        for (int e = 0; e < VEC; e++) {
            zv.a[e] = dv.a[e] * rv.a[e];
            s_rz = fma((double)rv.a[e], (double)zv.a[e], s_rz);
            s_rr = fma((double)rv.a[e], (double)rv.a[e], s_rr);
        }
        stv(a.x + idx, zerov<T>());
        stv(a.pzero + idx, zerov<T>());
        stv(a.r + idx, rv);
        stv(a.z + idx, zv);
    }
    const double t_rz = block_sum(s_rz, red);
    const double t_rr = block_sum(s_rr, red);
    const int nblk = gridDim.x;
    if (threadIdx.x == 0) {
        a.partials[blockIdx.x] = t_rz;
        a.partials[nblk + blockIdx.x] = t_rr;
        __threadfence();
        const unsigned int t = atomicAdd(&a.st->ticket_vec, 1u);
        s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        const double rz = final_sum(a.partials, nblk, red);
        const double rr = final_sum(a.partials + nblk, nblk, red);
        if (threadIdx.x == 0) {
            a.st->ticket_vec = 0u;
            finish_iteration(a.st, rz, rr, true);
        }
    }
}

}  // namespace pb
