// pb_persist.cuh -- the whole PCG loop (steps 3-8) as ONE persistent cooperative kernel, for grids
// whose working set lives in the 126 MB L2: there two launches per iteration cost more than the data movement
// (SURVEY.md 8(f) f2).  Same arithmetic as k_spmv_tma / k_vec (z = Dinv r, p = z + beta p, Ap rebuilt from the
// face dielectrics of Eq. 3 with D = 1/Dinv, alpha, x, r, beta), three grid-wide barriers per iteration instead
// of two kernel launches, every scalar kept in registers by every block (each block sums the per-block partials
// in the same fixed order, so all blocks take the same decisions and the loop exit is uniform).  No host
// involvement at all until the latch is read after the kernel.
#pragma once
#include <cooperative_groups.h>
#include "pb_internal.cuh"

namespace pb {

template <typename T>
struct PersistArgs {
    T *x, *r, *p0, *p1, *Ap;
    const T *Dinv, *exm, *eym, *ezm;
    int nx, ny, nz, P;
    int precond;
    int periodic;            // 1: neighbours wrap, 0: ghost p = 0
    State *st;
    double *partials;        // 3 regions of gridDim.x doubles: p.Ap | r.z | r.r
};

// sum of n per-block partials in fixed order, result broadcast to every thread of the block
__device__ __forceinline__ double all_sum(const double *partials, int n, double *red, double *bcast)
{
    const double t = final_sum(partials, n, red);
    if (threadIdx.x == 0) *bcast = t;
    __syncthreads();
    const double v = *bcast;
    __syncthreads();
    return v;
}

// FUSED: p = z + beta p is recomputed at the centre and its six neighbours inside the stencil pass (21 instead of 7
// L1/L2-resident loads) instead of in a pass of its own: two grid barriers per iteration instead of three, which is
// what counts on grids so small that the barriers dominate.
template <typename T, bool FUSED>
__global__ void __launch_bounds__(256, FUSED ? 2 : 3) k_pcg_persistent(const PersistArgs<T> a)
{
    namespace cg = cooperative_groups;
    constexpr int VEC = VecN<T>::value;
    cg::grid_group grid = cg::this_grid();
    __shared__ double red[32];
    __shared__ double bcast;
    State *st = a.st;
    const int nx = a.nx, ny = a.ny, nz = a.nz, P = a.P;
    const int rowvecs = P / VEC;
    const size_t nvec = (size_t)nz * ny * rowvecs;
    const size_t stride = (size_t)gridDim.x * blockDim.x, first = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int G = gridDim.x;
    const bool precond = a.precond != 0, per = a.periodic != 0;

    // every block carries the scalars of PAPER.md:106-126 in registers
    double rz = st->rz, rr = st->rr;
    const double bb = st->bb, tol2 = st->tol2;
    const int maxiter = st->maxiter;
    int done = st->done, status = st->status, l = 0;
    T beta = T(0);
    T *pin = a.p0, *pout = a.p1;              // k_init cleared p0

    // p_new = z + beta p_old at an arbitrary vector / scalar position (steps 6-7)
    auto pnew_v = [&](const T *pin_, size_t idx) -> Vec<T> {
        const Vec<T> rv = ldv(a.r + idx), dv = ldv(a.Dinv + idx), po = ldv(pin_ + idx);
        Vec<T> pn;
#pragma unroll
        for (int e = 0; e < VEC; e++) pn.a[e] = fma(beta, po.a[e], precond ? dv.a[e] * rv.a[e] : rv.a[e]);
        return pn;
    };
    auto pnew_s = [&](const T *pin_, size_t idx) -> T {
        return fma(beta, pin_[idx], precond ? a.Dinv[idx] * a.r[idx] : a.r[idx]);
    };

    while (!done) {
        if (!FUSED) {
            // step 6-7: z = Dinv r (or r), p = z + beta p
            for (size_t v = first; v < nvec; v += stride) stv(pout + v * VEC, pnew_v(pin, v * VEC));
            grid.sync();
        }
        // step 5a: Ap = A'p from the face dielectrics (ghost p = 0), partial p.Ap
        double acc = 0.0;
        for (size_t v = first; v < nvec; v += stride) {
            const int iv = (int)(v % rowvecs);
            const size_t row = v / rowvecs;
            const int j = (int)(row % ny), k = (int)(row / ny), i0 = iv * VEC;
            const size_t idx = v * VEC;
            // neighbour values of p: read back (three-barrier form) or recomputed from r, Dinv, p_old (FUSED)
            auto PV = [&](size_t at) -> Vec<T> { return FUSED ? pnew_v(pin, at) : ldv(pout + at); };
            auto PS = [&](size_t at) -> T { return FUSED ? pnew_s(pin, at) : pout[at]; };
            const Vec<T> pc = PV(idx);
            if (FUSED) stv(pout + idx, pc);
            const size_t rowbase = idx - i0, planebase = (size_t)k * ny * P, colbase = (size_t)j * P + i0;
            const Vec<T> up = (j > 0) ? PV(idx - P) : (per ? PV(planebase + (size_t)(ny - 1) * P + i0) : zerov<T>());
            const Vec<T> dn = (j < ny - 1) ? PV(idx + P) : (per ? PV(planebase + i0) : zerov<T>());
            const Vec<T> pm = (k > 0) ? PV(idx - (size_t)ny * P) : (per ? PV((size_t)(nz - 1) * ny * P + colbase) : zerov<T>());
            const Vec<T> pp = (k < nz - 1) ? PV(idx + (size_t)ny * P) : (per ? PV(colbase) : zerov<T>());
            const T left = (i0 > 0) ? PS(idx - 1) : (per ? PS(rowbase + nx - 1) : T(0));
            const T right = (i0 + VEC < P) ? PS(idx + VEC) : T(0);
            const T wrap0 = per ? PS(rowbase) : T(0);         // right neighbour of node nx-1
            const Vec<T> dinv = ldv(a.Dinv + idx), ex = ldv(a.exm + idx);
            const T exr = (i0 + VEC < P) ? a.exm[idx + VEC] : T(0);
            const size_t yidx = ((size_t)k * (ny + 1) + j) * P + i0;
            const Vec<T> eyl = ldv(a.eym + yidx), eyh = ldv(a.eym + yidx + P);
            const Vec<T> ezl = ldv(a.ezm + idx), ezh = ldv(a.ezm + idx + (size_t)ny * P);
            Vec<T> ap;
#pragma unroll
            for (int e = 0; e < VEC; e++) {
                const T pl = (e == 0) ? left : pc.a[e == 0 ? 0 : e - 1];
                T pr = (e == VEC - 1) ? right : pc.a[e == VEC - 1 ? e : e + 1];
                if (i0 + e == nx - 1) pr = wrap0;             // pad column (0) or, periodic, node 0 of the row
                const T exh = (e == VEC - 1) ? exr : ex.a[e == VEC - 1 ? e : e + 1];
                T s = rcp_rn(dinv.a[e]) * pc.a[e];            // D = 1/Dinv, as in k_spmv_tma
                s = fma(-ex.a[e], pl, s);
                s = fma(-exh, pr, s);
                s = fma(-eyl.a[e], up.a[e], s);
                T w = -eyh.a[e] * dn.a[e];
                w = fma(-ezl.a[e], pm.a[e], w);
                w = fma(-ezh.a[e], pp.a[e], w);
                s += w;
                if (i0 + e >= nx) s = T(0);
                acc = fma((double)pc.a[e], (double)s, acc);
                ap.a[e] = s;
            }
            stv(a.Ap + idx, ap);
        }
        const double t_b = block_sum(acc, red);
        if (threadIdx.x == 0) a.partials[blockIdx.x] = t_b;
        grid.sync();
        const double pAp = all_sum(a.partials, G, red, &bcast);
        if (!(pAp > 0.0) || !isfinite(pAp)) { done = 1; status = 5; break; }     // breakdown; x = last good iterate
        const T alpha = (T)(rz / pAp);                                           // step 5
        // step 5b: x += alpha p, r -= alpha Ap;  r.z and r.r
        double s_rz = 0.0, s_rr = 0.0;
        for (size_t v = first; v < nvec; v += stride) {
            const size_t idx = v * VEC;
            Vec<T> xv = ldv(a.x + idx), rv = ldv(a.r + idx);
            const Vec<T> pc = ldv(pout + idx), qv = ldv(a.Ap + idx), dv = ldv(a.Dinv + idx);
#pragma unroll
            for (int e = 0; e < VEC; e++) {
                xv.a[e] = fma(alpha, pc.a[e], xv.a[e]);
                rv.a[e] = fma(-alpha, qv.a[e], rv.a[e]);
                const T zv = precond ? dv.a[e] * rv.a[e] : rv.a[e];
                s_rz = fma((double)rv.a[e], (double)zv, s_rz);
                s_rr = fma((double)rv.a[e], (double)rv.a[e], s_rr);
            }
            stv(a.x + idx, xv);
            stv(a.r + idx, rv);
        }
        const double t_rz = block_sum(s_rz, red), t_rr = block_sum(s_rr, red);
        if (threadIdx.x == 0) { a.partials[G + blockIdx.x] = t_rz; a.partials[2 * G + blockIdx.x] = t_rr; }
        grid.sync();
        const double rz_new = all_sum(a.partials + G, G, red, &bcast);
        rr = all_sum(a.partials + 2 * G, G, red, &bcast);
        beta = (T)(rz_new / rz);                                                 // step 7
        rz = rz_new;
        l++;                                                                     // step 4
        if (!isfinite(rr) || !isfinite(rz_new)) { done = 1; status = 5; }
        else if (rr < tol2 * bb) { done = 1; status = 0; }                       // step 3
        else if (l >= maxiter) { done = 1; status = 6; }
        T *t = pin; pin = pout; pout = t;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st->rz = rz; st->rr = rr; st->beta = (double)beta;
        st->alpha = 0.0;                         // x is fully updated: nothing pending for k_finish
        st->iter_cur = l; st->iters = l; st->done = 1; st->status = status;
    }
}

}  // namespace pb
