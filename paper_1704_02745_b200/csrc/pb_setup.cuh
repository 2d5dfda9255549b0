// pb_setup.cuh -- one-time setup kernels (row a0 of the hot-path table): build the padded
// coefficient arrays, the Jacobi diagonal D = diag(A') and its inverse,
// and the right-hand side of Eq. 4 with the ghost Dirichlet values folded in
// (PAPER.md:50-68, 182).  Inputs are the caller's dense fp64 arrays (device copies).
#pragma once
#include "pb_internal.cuh"

namespace pb {

// exm/eym/ezm/D/Dinv in precision T from the fp64 inputs; h^2-scaled system:
//   D'(c) = sum of the six face eps touching c + h^2 kbar2(c)     (coefficient of phi(i,j,k) in Eq. 3, times h^2)
template <typename T>
__global__ void k_setup_coeff(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                              const double *__restrict__ eps_z, const double *__restrict__ kbar2,
                              double h2, int nx, int ny, int nz, int P,
                              T *exm, T *eym, T *ezm, T *D, T *Dinv, int *bad)
{
    const size_t total = (size_t)(nz + 1) * (ny + 1) * P;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % P);
        const size_t q = t / P;
        const int j = (int)(q % (ny + 1));
        const int k = (int)(q / (ny + 1));
        if (k < nz && j < ny) {
            const size_t row = (size_t)k * ny + j;
            exm[row * P + i] = (i <= nx) ? (T)eps_x[row * (nx + 1) + i] : T(0);
            double d = 1.0;
            if (i < nx) {
                d = eps_x[row * (nx + 1) + i] + eps_x[row * (nx + 1) + i + 1]
                  + eps_y[((size_t)k * (ny + 1) + j) * nx + i] + eps_y[((size_t)k * (ny + 1) + j + 1) * nx + i]
                  + eps_z[row * nx + i] + eps_z[((size_t)(k + 1) * ny + j) * nx + i];
                if (kbar2) d += h2 * kbar2[row * nx + i];
                if (!(d > 0.0) || !isfinite(d)) *bad = 1;
            }
            D[row * P + i] = (T)d;
            Dinv[row * P + i] = (T)(1.0 / d);
        }
        if (k < nz)
            eym[((size_t)k * (ny + 1) + j) * P + i] = (i < nx) ? (T)eps_y[((size_t)k * (ny + 1) + j) * nx + i] : T(0);
        if (j < ny)
            ezm[((size_t)k * ny + j) * P + i] = (i < nx) ? (T)eps_z[((size_t)k * ny + j) * nx + i] : T(0);
    }
}

// b'(c) = h^2 rhs(c) + sum over ghost neighbours g of c of eps_face(c,g) * bc(g)
// bc packing: x-, x+ ([nz][ny]), y-, y+ ([nz][nx]), z-, z+ ([ny][nx]).
template <typename T>
__global__ void k_setup_b(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                          const double *__restrict__ eps_z, const double *__restrict__ rhs,
                          const double *__restrict__ bc, double h2, int nx, int ny, int nz, int P, T *b)
{
    const size_t total = (size_t)nz * ny * P;
    const size_t o_xp = (size_t)nz * ny, o_ym = 2 * o_xp, o_yp = o_ym + (size_t)nz * nx,
                 o_zm = o_yp + (size_t)nz * nx, o_zp = o_zm + (size_t)ny * nx;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % P);
        const size_t row = t / P;
        const int j = (int)(row % ny);
        const int k = (int)(row / ny);
        double v = 0.0;
        if (i < nx) {
            if (rhs) v = h2 * rhs[row * nx + i];
            if (bc) {
                if (i == 0)      v += eps_x[row * (nx + 1)] * bc[(size_t)k * ny + j];
                if (i == nx - 1) v += eps_x[row * (nx + 1) + nx] * bc[o_xp + (size_t)k * ny + j];
                if (j == 0)      v += eps_y[((size_t)k * (ny + 1)) * nx + i] * bc[o_ym + (size_t)k * nx + i];
                if (j == ny - 1) v += eps_y[((size_t)k * (ny + 1) + ny) * nx + i] * bc[o_yp + (size_t)k * nx + i];
                if (k == 0)      v += eps_z[(size_t)j * nx + i] * bc[o_zm + (size_t)j * nx + i];
                if (k == nz - 1) v += eps_z[((size_t)nz * ny + j) * nx + i] * bc[o_zp + (size_t)j * nx + i];
            }
        }
        b[t] = (T)v;
    }
}

// dense [nz][ny][nx] (type S) -> padded [nz][ny][P] (type T), pad = 0
template <typename T, typename S>
__global__ void k_pad(const S *__restrict__ src, T *dst, int nx, int P, size_t rows)
{
    const size_t total = rows * P;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % P);
        const size_t row = t / P;
        dst[t] = (i < nx) ? (T)src[row * nx + i] : T(0);
    }
}

// padded [nz][ny][P] (type T) -> dense [nz][ny][nx] (type S), times scale
template <typename T, typename S>
__global__ void k_unpad(const T *__restrict__ src, S *dst, int nx, int P, size_t rows, double scale)
{
    const size_t total = rows * nx;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % nx);
        const size_t row = t / nx;
        dst[t] = (S)((double)src[row * P + i] * scale);
    }
}

__global__ void k_set_state(State *st, double tol2, int maxiter, int latch)
{
    st->tol2 = tol2;
    st->maxiter = maxiter;
    st->latch = latch;
    st->done = 0;
    st->iters = 0;
    st->status = 0;
    st->iter_cur = 0;
    st->ticket_spmv = 0u;
    st->ticket_vec = 0u;
    st->alpha = 0.0;
    st->beta = 0.0;
}

}  // namespace pb
