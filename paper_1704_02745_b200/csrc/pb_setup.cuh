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
            if (exm) exm[row * P + i] = (i <= nx) ? (T)eps_x[row * (nx + 1) + i] : T(0);
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
        if (k < nz && eym)
            eym[((size_t)k * (ny + 1) + j) * P + i] = (i < nx) ? (T)eps_y[((size_t)k * (ny + 1) + j) * nx + i] : T(0);
        if (j < ny && ezm)
            ezm[((size_t)k * ny + j) * P + i] = (i < nx) ? (T)eps_z[((size_t)k * ny + j) * nx + i] : T(0);
    }
}

// b'(c) = h^2 rhs(c) + sum over ghost neighbours g of c of eps_face(c,g) * bc(g)
// bc packing: x-, x+ ([nz][ny]), y-, y+ ([nz][nx]), z-, z+ ([ny][nx]).
template <typename T>
__global__ void k_setup_b(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                          const double *__restrict__ eps_z, const double *__restrict__ rhs,
                          const double *__restrict__ bc, double h2, int nx, int ny, int nz, int P, T *b,
                          int iface_lo = 0, int iface_hi = 0)   // z-slab: the plane below / above belongs to a neighbour rank
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
                if (k == 0 && !iface_lo)      v += eps_z[(size_t)j * nx + i] * bc[o_zm + (size_t)j * nx + i];
                if (k == nz - 1 && !iface_hi) v += eps_z[((size_t)nz * ny + j) * nx + i] * bc[o_zp + (size_t)j * nx + i];
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

__global__ void k_set_state(State *st, double tol2, int maxiter, int latch, int slab = 0)
{
    st->slab = slab;
    st->xbuf = 0;
    st->pool_ctr = 0u;
    st->loc_rz = 0.0;
    st->loc_rr = 0.0;
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

// ---------------------------------------------------------------------------------------
// Coefficient palette.  A molecular dielectric map takes very few distinct face values (eps_in,
// eps_out and their harmonic mean), so the three face arrays can be stored exactly
// as one byte per face indexing a table of <= 256 values -- a storage format in the sense of
// PAPER.md:251-261 (fewer bytes per row than DIA's seven bands), decoded on the fly in k_spmv_tma.
// Operators with more than 256 distinct face values keep the full-precision arrays.
// ---------------------------------------------------------------------------------------
namespace pb {

constexpr int kPalMax = 256;
constexpr int kPalHash = 1024;
constexpr unsigned long long kPalEmpty = 0xFFFFFFFFFFFFFFFFull;

struct PalTable {
    unsigned long long keys[kPalHash];   // open-addressing set of the distinct bit patterns
    int count;
    int overflow;
    int n;                               // final size (k_pal_finish)
    double vals[kPalMax];                // sorted ascending
};

__global__ void k_pal_reset(PalTable *t)
{
    for (int i = threadIdx.x; i < kPalHash; i += blockDim.x) t->keys[i] = kPalEmpty;
    if (threadIdx.x == 0) { t->count = 0; t->overflow = 0; t->n = 0; }
}

__device__ __forceinline__ void pal_insert(PalTable *t, double v)
{
    const unsigned long long bits = (unsigned long long)__double_as_longlong(v);
    unsigned int slot = (unsigned int)((bits * 0x9E3779B97F4A7C15ull) >> 54);      // 10 bits
    for (int probe = 0; probe < kPalHash; probe++, slot = (slot + 1) & (kPalHash - 1)) {
        const unsigned long long cur = t->keys[slot];
        if (cur == bits) return;
        if (cur == kPalEmpty) {
            const unsigned long long old = atomicCAS(&t->keys[slot], kPalEmpty, bits);
            if (old == kPalEmpty) { if (atomicAdd(&t->count, 1) >= kPalMax) t->overflow = 1; return; }
            if (old == bits) return;
        }
    }
    t->overflow = 1;
}

// collect the distinct values of one dense fp64 array (consecutive equal values are skipped cheaply)
__global__ void k_pal_collect(const double *__restrict__ a, size_t n, PalTable *t)
{
    volatile int *ovf = &t->overflow;
    if (*ovf) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) pal_insert(t, 0.0);                   // the pad value
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double v = a[i];
        if (i > 0 && a[i - 1] == v && (i % 4096)) continue;                         // run of equal values
        pal_insert(t, v);
        if (*ovf) return;
    }
}

// one block: gather the keys and sort them ascending by value (rank sort, <= 256 entries)
__global__ void k_pal_finish(PalTable *t)
{
    __shared__ double v[kPalMax];
    __shared__ int cnt;
    if (threadIdx.x == 0) {
        cnt = 0;
        if (!t->overflow)
            for (int i = 0; i < kPalHash && cnt < kPalMax; i++)
                if (t->keys[i] != kPalEmpty) v[cnt++] = __longlong_as_double((long long)t->keys[i]);
    }
    __syncthreads();
    const int n = t->overflow ? 0 : cnt;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        int rank = 0;
        for (int j = 0; j < n; j++) rank += (v[j] < v[i]) || (v[j] == v[i] && j < i);
        t->vals[rank] = v[i];
    }
    if (threadIdx.x == 0) t->n = n;
}

__device__ __forceinline__ unsigned char pal_index(const PalTable *t, double v)
{
    int lo = 0, hi = t->n - 1;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (t->vals[mid] < v) lo = mid + 1; else hi = mid; }
    return (unsigned char)lo;
}

// byte index arrays in the padded layouts of exm / eym / ezm (row pitch Pb bytes, Pb >= P), pad = index of 0.0.
// Every byte is the table index times `scale` (the element size of the decoding table, n * scale <= 256): the
// kernel then adds the byte to the table's address with no shift.
__global__ void k_setup_pal_idx(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                                const double *__restrict__ eps_z, int nx, int ny, int nz, int Pb, int scale,
                                const PalTable *t, unsigned char *exi, unsigned char *eyi, unsigned char *ezi)
{
    const unsigned char zero = (unsigned char)(pal_index(t, 0.0) * scale);
    const size_t total = (size_t)(nz + 1) * (ny + 1) * Pb;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(q % Pb);
        const size_t u = q / Pb;
        const int j = (int)(u % (ny + 1)), k = (int)(u / (ny + 1));
        if (k < nz && j < ny)
            exi[((size_t)k * ny + j) * Pb + i] = (i <= nx) ? (unsigned char)(pal_index(t, eps_x[((size_t)k * ny + j) * (nx + 1) + i]) * scale) : zero;
        if (k < nz)
            eyi[((size_t)k * (ny + 1) + j) * Pb + i] = (i < nx) ? (unsigned char)(pal_index(t, eps_y[((size_t)k * (ny + 1) + j) * nx + i]) * scale) : zero;
        if (j < ny)
            ezi[((size_t)k * ny + j) * Pb + i] = (i < nx) ? (unsigned char)(pal_index(t, eps_z[((size_t)k * ny + j) * nx + i]) * scale) : zero;
    }
}

// Quad index arrays for palettes of at most four values (k_spmv_quad): 2 bits per face, four consecutive nodes of a
// row per byte (node i -> bits 2(i&3) of byte i>>2), rows of Pq bytes.  exq holds the MINUS x-face of every node
// (face i), exqp its PLUS x-face (face i+1), eyq / ezq the minus y- / z-faces with one extra row / plane (the plus
// face of a node is the minus face of its neighbour).  Pad nodes (i >= nx) get the index of 0.0.
__global__ void k_setup_quad_idx(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                                 const double *__restrict__ eps_z, int nx, int ny, int nz, int Pq,
                                 const PalTable *t, unsigned char *exq, unsigned char *exqp, unsigned char *eyq,
                                 unsigned char *ezq)
{
    const unsigned int zero = pal_index(t, 0.0);
    const size_t total = (size_t)(nz + 1) * (ny + 1) * Pq;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const int bq = (int)(q % Pq);
        const size_t u = q / Pq;
        const int j = (int)(u % (ny + 1)), k = (int)(u / (ny + 1));
        unsigned int bm = 0, bp = 0, by = 0, bz = 0;
        for (int f = 0; f < 4; f++) {
            const int i = 4 * bq + f;
            unsigned int im = zero, ip = zero, iy = zero, iz = zero;
            if (i < nx) {
                if (k < nz && j < ny) {
                    im = pal_index(t, eps_x[((size_t)k * ny + j) * (nx + 1) + i]);
                    ip = pal_index(t, eps_x[((size_t)k * ny + j) * (nx + 1) + i + 1]);
                }
                if (k < nz) iy = pal_index(t, eps_y[((size_t)k * (ny + 1) + j) * nx + i]);
                if (j < ny) iz = pal_index(t, eps_z[((size_t)k * ny + j) * nx + i]);
            }
            bm |= im << (2 * f); bp |= ip << (2 * f); by |= iy << (2 * f); bz |= iz << (2 * f);
        }
        if (k < nz && j < ny) {
            exq[((size_t)k * ny + j) * Pq + bq] = (unsigned char)bm;
            exqp[((size_t)k * ny + j) * Pq + bq] = (unsigned char)bp;
        }
        if (k < nz) eyq[((size_t)k * (ny + 1) + j) * Pq + bq] = (unsigned char)by;
        if (j < ny) ezq[((size_t)k * ny + j) * Pq + bq] = (unsigned char)bz;
    }
}

// The same indices in ONE array [4][nz+1][ny+1][Pq] = {ez, ex-, ex+, ey} (k_pcg_fused fetches the four boxes of a
// plane with one TMA instruction); entries outside an array's own range hold the index of 0.0 and are never used.
__global__ void k_setup_quad4(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                              const double *__restrict__ eps_z, int nx, int ny, int nz, int Pq, const PalTable *t,
                              unsigned char *q4)
{
    const unsigned int zero = pal_index(t, 0.0);
    const size_t total = (size_t)(nz + 1) * (ny + 1) * Pq;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const int bq = (int)(q % Pq);
        const size_t u = q / Pq;
        const int j = (int)(u % (ny + 1)), k = (int)(u / (ny + 1));
        unsigned int bm = 0, bp = 0, by = 0, bz = 0;
        for (int f = 0; f < 4; f++) {
            const int i = 4 * bq + f;
            unsigned int im = zero, ip = zero, iy = zero, iz = zero;
            if (i < nx) {
                if (k < nz && j < ny) {
                    im = pal_index(t, eps_x[((size_t)k * ny + j) * (nx + 1) + i]);
                    ip = pal_index(t, eps_x[((size_t)k * ny + j) * (nx + 1) + i + 1]);
                }
                if (k < nz) iy = pal_index(t, eps_y[((size_t)k * (ny + 1) + j) * nx + i]);
                if (j < ny) iz = pal_index(t, eps_z[((size_t)k * ny + j) * nx + i]);
            }
            bm |= im << (2 * f); bp |= ip << (2 * f); by |= iy << (2 * f); bz |= iz << (2 * f);
        }
        q4[q] = (unsigned char)bz;
        q4[total + q] = (unsigned char)bm;
        q4[2 * total + q] = (unsigned char)bp;
        q4[3 * total + q] = (unsigned char)by;
    }
}

template <typename T>
__global__ void k_pal_lut(const PalTable *t, T *lut)
{
    for (int i = threadIdx.x; i < kPalMax; i += blockDim.x) lut[i] = (i < t->n) ? (T)t->vals[i] : T(0);
}

}  // namespace pb

// ---------------------------------------------------------------------------------------
// Diagonal palette.  With palette-able face dielectrics and a two-valued salt map the Jacobi diagonal
// D' = sum of six face eps + h^2 kbar2 also takes few distinct values (56 at most for three face values), so k_vec
// can read one index byte per node instead of a Dinv word.  The table holds the fp64 diagonals; the lookup table
// in precision T is (T)(1/d), bit-identical to the Dinv array k_setup_coeff writes.
// ---------------------------------------------------------------------------------------
namespace pb {

__device__ __forceinline__ double diag_of(const double *eps_x, const double *eps_y, const double *eps_z,
                                          const double *kbar2, double h2, int nx, int ny, int i, int j, int k)
{
    const size_t row = (size_t)k * ny + j;
    double d = eps_x[row * (nx + 1) + i] + eps_x[row * (nx + 1) + i + 1]
             + eps_y[((size_t)k * (ny + 1) + j) * nx + i] + eps_y[((size_t)k * (ny + 1) + j + 1) * nx + i]
             + eps_z[row * nx + i] + eps_z[((size_t)(k + 1) * ny + j) * nx + i];
    if (kbar2) d += h2 * kbar2[row * nx + i];
    return d;
}

// SPD check of pb_create: every diagonal entry of Eq. 3 must be positive and finite (M = D must be invertible,
// PAPER.md:138-140; "symmetric and positive-definite coefficient matrices")
__global__ void k_check_diag(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                             const double *__restrict__ eps_z, const double *__restrict__ kbar2, double h2,
                             int nx, int ny, int nz, int *bad)
{
    const size_t n = (size_t)nx * ny * nz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(q % nx), j = (int)((q / nx) % ny), k = (int)(q / ((size_t)nx * ny));
        const double d = diag_of(eps_x, eps_y, eps_z, kbar2, h2, nx, ny, i, j, k);
        if (!(d > 0.0) || !isfinite(d)) *bad = 1;
    }
}

__global__ void k_pal_collect_diag(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                                   const double *__restrict__ eps_z, const double *__restrict__ kbar2, double h2,
                                   int nx, int ny, int nz, PalTable *t)
{
    volatile int *ovf = &t->overflow;
    if (*ovf) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) pal_insert(t, 1.0);                   // the pad value
    const size_t n = (size_t)nx * ny * nz;
    double prev = -1.0;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(q % nx), j = (int)((q / nx) % ny), k = (int)(q / ((size_t)nx * ny));
        const double d = diag_of(eps_x, eps_y, eps_z, kbar2, h2, nx, ny, i, j, k);
        if (d == prev) continue;
        prev = d;
        pal_insert(t, d);
        if (*ovf) return;
    }
}

// byte index of D per padded node ([nz][ny][P], pad = index of 1.0)
__global__ void k_setup_diag_idx(const double *__restrict__ eps_x, const double *__restrict__ eps_y,
                                 const double *__restrict__ eps_z, const double *__restrict__ kbar2, double h2,
                                 int nx, int ny, int nz, int P, int scale, const PalTable *t, unsigned char *dvi)
{
    const unsigned char one = (unsigned char)(pal_index(t, 1.0) * scale);
    const size_t total = (size_t)nz * ny * P;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(q % P);
        const size_t row = q / P;
        const int j = (int)(row % ny), k = (int)(row / ny);
        dvi[q] = (i < nx) ? (unsigned char)(pal_index(t, diag_of(eps_x, eps_y, eps_z, kbar2, h2, nx, ny, i, j, k)) * scale) : one;
    }
}

template <typename T>
__global__ void k_pal_lut_dinv(const PalTable *t, T *lut)
{
    for (int i = threadIdx.x; i < kPalMax; i += blockDim.x) lut[i] = (i < t->n) ? (T)(1.0 / t->vals[i]) : T(1);
}

}  // namespace pb
