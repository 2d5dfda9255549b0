// pb_grid.cuh -- grid / stencil setup on the GPU (NEXT row f1; the paper's own stated next step,
// "integrated grid stencil setup on GPU"): from atoms (centres, radii, charges) to the
// inputs of Eq. 3: solute mask, harmonic-mean face dielectrics, salt map
// (Stern mask of Eq. 1-2), trilinearly spread grid charges, and the free-space Debye-Hueckel ghost values
// (PAPER.md:182).  Readings: DESIGN.md 8-11, 13, 18.  fp64 throughout; decisions that produce integers
// (inside / outside a sphere, the base node of a charge) use explicitly rounded operations (__dmul_rn ...)
// so that no FMA contraction can flip them relative to a plain IEEE evaluation.
#pragma once
#include <cuda_runtime.h>
#include "pb_internal.cuh"

namespace pb {

// one block per atom (grid-stride): mark every node of the atom's bounding box with d^2 <= R^2
__global__ void k_grid_mask(const double *__restrict__ c, const double *__restrict__ rad, int n_atoms,
                            int nx, int ny, int nz, double h, unsigned char *mask)
{
    for (int a = blockIdx.x; a < n_atoms; a += gridDim.x) {
        const double cx = c[3 * a], cy = c[3 * a + 1], cz = c[3 * a + 2], R = rad[a];
        const int i_lo = max(0, (int)ceil((cx - R) / h)), i_hi = min(nx - 1, (int)floor((cx + R) / h));
        const int j_lo = max(0, (int)ceil((cy - R) / h)), j_hi = min(ny - 1, (int)floor((cy + R) / h));
        const int k_lo = max(0, (int)ceil((cz - R) / h)), k_hi = min(nz - 1, (int)floor((cz + R) / h));
        if (i_lo > i_hi || j_lo > j_hi || k_lo > k_hi) continue;
        const int bx = i_hi - i_lo + 1, by = j_hi - j_lo + 1, bz = k_hi - k_lo + 1;
        const double R2 = __dmul_rn(R, R);
        for (int t = threadIdx.x; t < bx * by * bz; t += blockDim.x) {
            const int i = i_lo + t % bx, j = j_lo + (t / bx) % by, k = k_lo + t / (bx * by);
            const double dx = __dsub_rn(__dmul_rn((double)i, h), cx);
            const double dy = __dsub_rn(__dmul_rn((double)j, h), cy);
            const double dz = __dsub_rn(__dmul_rn((double)k, h), cz);
            const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dz, dz), __dmul_rn(dy, dy)), __dmul_rn(dx, dx));
            if (d2 <= R2) mask[((size_t)k * ny + j) * nx + i] = 1;   // every writer stores the same value
        }
    }
}

__device__ __forceinline__ double node_eps(const unsigned char *mask, int nx, int ny, int nz, int k, int j, int i,
                                           double eps_in, double eps_out)
{
    if (k < 0 || k >= nz || j < 0 || j >= ny || i < 0 || i >= nx) return eps_out;   // ghost layer = solvent
    return mask[((size_t)k * ny + j) * nx + i] ? eps_in : eps_out;
}
__device__ __forceinline__ double harmonic(double a, double b)
{
    return __ddiv_rn(__dmul_rn(__dmul_rn(2.0, a), b), __dadd_rn(a, b));
}

// face dielectrics (harmonic mean of the two nodes a face joins) and the salt map, one pass over (nz+1)(ny+1)(nx+1)
__global__ void k_grid_faces(const unsigned char *__restrict__ mask, int nx, int ny, int nz, double eps_in,
                             double eps_out, double kbar2_solvent, double *eps_x, double *eps_y, double *eps_z,
                             double *kbar2)
{
    const size_t total = (size_t)(nz + 1) * (ny + 1) * (nx + 1);
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(t % (nx + 1));
        const size_t q = t / (nx + 1);
        const int j = (int)(q % (ny + 1)), k = (int)(q / (ny + 1));
        const double e = node_eps(mask, nx, ny, nz, k, j, i, eps_in, eps_out);
        if (k < nz && j < ny)
            eps_x[((size_t)k * ny + j) * (nx + 1) + i] = harmonic(node_eps(mask, nx, ny, nz, k, j, i - 1, eps_in, eps_out), e);
        if (k < nz && i < nx)
            eps_y[((size_t)k * (ny + 1) + j) * nx + i] = harmonic(node_eps(mask, nx, ny, nz, k, j - 1, i, eps_in, eps_out), e);
        if (j < ny && i < nx)
            eps_z[((size_t)k * ny + j) * nx + i] = harmonic(node_eps(mask, nx, ny, nz, k - 1, j, i, eps_in, eps_out), e);
        if (k < nz && j < ny && i < nx)
            kbar2[((size_t)k * ny + j) * nx + i] = mask[((size_t)k * ny + j) * nx + i] ? 0.0 : kbar2_solvent;
    }
}

// Atom check + charge scale, one block, fixed order: every centre must lie inside the box [0,(n-1)h]^3 (an atom
// outside would get extrapolated -- negative -- trilinear weights, and one sitting on a ghost node a 1/0 in the
// boundary sum), and sum |q_a| bounds every node's accumulated charge, which fixes the fixed-point scale below.
__global__ void k_grid_check(const double *__restrict__ c, const double *__restrict__ charge, int n_atoms,
                             int nx, int ny, int nz, double h, double *sum_abs, int *bad)
{
    __shared__ double red[32];
    double s = 0.0;
    const double hi[3] = {(nx - 1) * h, (ny - 1) * h, (nz - 1) * h};
    for (int a = threadIdx.x; a < n_atoms; a += blockDim.x) {
        s += fabs(charge[a]);
        for (int d = 0; d < 3; d++) {
            const double v = c[3 * a + d];
            if (!(v >= 0.0 && v <= hi[d])) *bad = 1;          // also catches NaN
        }
        if (!isfinite(charge[a])) *bad = 1;
    }
    const double tot = block_sum(s, red);
    if (threadIdx.x == 0) *sum_abs = tot;
}

// fixed-point scale 2^(62 - e) with sum|q| < 2^e: every partial sum fits a signed 64-bit integer
__device__ __forceinline__ int spread_shift(double sum_abs)
{
    int e = 0;
    if (sum_abs > 0.0) frexp(sum_abs, &e);
    return 62 - e;
}

// Trilinear spreading of the point charges to their 8 surrounding nodes (q(i,j,k) of Eq. 3).  Nodes
// shared by several atoms are accumulated with integer atomics in 64-bit fixed point (resolution sum|q| * 2^-62,
// far below an fp64 ulp of any node charge that matters): integer addition is associative, so the result does not
// depend on the order in which the atoms arrive -- bitwise reproducible, unlike a floating-point atomicAdd.
// `acc` is the rhs buffer viewed as int64 and zeroed before; k_grid_rhs converts it in place.
__global__ void k_grid_spread(const double *__restrict__ c, const double *__restrict__ charge, int n_atoms,
                              int nx, int ny, int nz, double h, const double *sum_abs, long long *acc)
{
    const double scale = ldexp(1.0, spread_shift(*sum_abs));
    for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < n_atoms; a += gridDim.x * blockDim.x) {
        const double g[3] = {c[3 * a] / h, c[3 * a + 1] / h, c[3 * a + 2] / h};
        const int n[3] = {nx, ny, nz};
        int base[3];
        double fr[3];
        for (int d = 0; d < 3; d++) {
            base[d] = min(max((int)floor(g[d]), 0), n[d] - 2);
            fr[d] = __dsub_rn(g[d], (double)base[d]);
        }
        const double qa = charge[a];
        for (int dz = 0; dz < 2; dz++) {
            const double wz = dz ? fr[2] : __dsub_rn(1.0, fr[2]);
            for (int dy = 0; dy < 2; dy++) {
                const double wy = dy ? fr[1] : __dsub_rn(1.0, fr[1]);
                for (int dx = 0; dx < 2; dx++) {
                    const double wx = dx ? fr[0] : __dsub_rn(1.0, fr[0]);
                    const double v = __dmul_rn(__dmul_rn(__dmul_rn(qa, wz), wy), wx);
                    const long long fx = __double2ll_rn(__dmul_rn(v, scale));
                    if (fx != 0)
                        atomicAdd((unsigned long long *)&acc[((size_t)(base[2] + dz) * ny + base[1] + dy) * nx + base[0] + dx],
                                  (unsigned long long)fx);
                }
            }
        }
    }
}

// rhs = (4 pi) q / h^3 in place, q = fixed-point accumulator * 2^-shift
__global__ void k_grid_rhs(double *q, size_t n, double four_pi, double h3, const double *sum_abs)
{
    const double inv = ldexp(1.0, -spread_shift(*sum_abs));
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const double qn = __dmul_rn((double)reinterpret_cast<const long long *>(q)[t], inv);
        q[t] = __ddiv_rn(__dmul_rn(four_pi, qn), h3);
    }
}

// fp64 1/sqrt(d2) for the boundary sum: MUFU.RSQ seed on the value rounded to fp32 (2^-22) and ONE third-order Newton
// step (error (5/16) e^3 ~ 3e-21 relative, i.e. correctly rounded up to the last DFMA).  d2 in [2^-126, 2^127].
__device__ __forceinline__ double dh_rsqrt(double d2)
{
    float s;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(__double2float_rn(d2)));
    const double y = (double)s;
    const double e = fma(-(d2 * y), y, 1.0);                   // 1 - d2 y^2
    return fma(y, fma(0.375, e, 0.5) * e, y);                  // y (1 + e/2 + 3 e^2/8)
}

// fp64 exp(x) for -700 < x <= 0: x = (64 n + k) ln2/64 + f, |f| <= ln2/128; exp(x) = 2^n * 2^(k/64) * exp(f) with a
// 64-entry table (shared memory) and a degree-5 Taylor polynomial (remainder f^6/6! < 4e-17); no special cases --
// the argument range is fixed by the geometry (kappa r <= a few hundred).
constexpr int DH_EXP_TAB = 64;
__device__ __forceinline__ double dh_exp_neg(double x, const double *tab)
{
    const double MAGIC = 6755399441055744.0;                   // 1.5 * 2^52: the integer lands in the low word
    const double t = fma(x, 92.332482616893657, MAGIC);        // 64 / ln 2
    const int m = __double2loint(t);
    const double mf = t - MAGIC;
    double f = fma(mf, -1.08304246932675596326e-02, x);        // ln2_hi / 64 (32 significant bits: mf * it is exact)
    f = fma(mf, -2.98158582698529328128e-12, f);               // ln2_lo / 64
    double p = fma(f, 1.0 / 120.0, 1.0 / 24.0);
    p = fma(p, f, 1.0 / 6.0);
    p = fma(p, f, 0.5);
    p = fma(p, f, 1.0);
    p = fma(p, f, 1.0);
    p *= tab[m & (DH_EXP_TAB - 1)];
    return __hiloint2double(__double2hiint(p) + ((m >> 6) << 20), __double2loint(p));   // * 2^n (stays normal)
}

// Debye-Hueckel ghost values: bc[g] = (1/eps_out) sum_a q_a exp(-kappa r_ga)/r_ga, atoms in index order.
// One thread per ghost node, atoms staged through shared memory in tiles of DH_TILE.  Plain-ALU-bound (fp64 pipe /
// issue): 1/r and exp come from the two routines above instead of the general-purpose library ones.
// FAST = false: the library rsqrt / exp (any argument), for geometries outside the range the fitted routines assume
// (dh_fast_range below; no molecular grid gets there).
constexpr int DH_TILE = 256;
inline bool dh_fast_range(int nx, int ny, int nz, double h, double kappa)
{
    const double rmax2 = h * h * ((double)(nx + 1) * (nx + 1) + (double)(ny + 1) * (ny + 1) + (double)(nz + 1) * (nz + 1));
    return h * h >= 1e-30 && rmax2 <= 1e30 && kappa * sqrt(rmax2) <= 700.0;      // d2 within fp32 range, exp normal
}
template <bool FAST>
__global__ void __launch_bounds__(DH_TILE) k_grid_dh(const double *__restrict__ c, const double *__restrict__ charge,
                                                     int n_atoms, int nx, int ny, int nz, double h, double eps_out,
                                                     double kappa, double *bc)
{
    __shared__ double sc[DH_TILE][4];
    __shared__ double tab[DH_EXP_TAB];
    if (threadIdx.x < DH_EXP_TAB) tab[threadIdx.x] = exp2((double)threadIdx.x / DH_EXP_TAB);   // 2^(k/64), library exp2 (< 1 ulp)
    const size_t n_xy = (size_t)ny * nx, n_zy = (size_t)nz * ny, n_zx = (size_t)nz * nx;
    const size_t nbc = 2 * (n_zy + n_zx + n_xy);
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    double gx = 0.0, gy = 0.0, gz = 0.0;
    if (t < 2 * n_zy) {                                   // x-, x+ : [nz][ny]
        const size_t u = t % n_zy;
        gx = (t < n_zy) ? -h : nx * h; gy = (double)(u % ny) * h; gz = (double)(u / ny) * h;
    } else if (t < 2 * n_zy + 2 * n_zx) {                 // y-, y+ : [nz][nx]
        const size_t v = t - 2 * n_zy, u = v % n_zx;
        gy = (v < n_zx) ? -h : ny * h; gx = (double)(u % nx) * h; gz = (double)(u / nx) * h;
    } else if (t < nbc) {                                 // z-, z+ : [ny][nx]
        const size_t v = t - 2 * n_zy - 2 * n_zx, u = v % n_xy;
        gz = (v < n_xy) ? -h : nz * h; gx = (double)(u % nx) * h; gy = (double)(u / nx) * h;
    }
    const double nkappa = -kappa;
    double acc = 0.0;
    for (int a0 = 0; a0 < n_atoms; a0 += DH_TILE) {
        const int a = a0 + threadIdx.x;
        if (a < n_atoms) { sc[threadIdx.x][0] = c[3 * a]; sc[threadIdx.x][1] = c[3 * a + 1]; sc[threadIdx.x][2] = c[3 * a + 2]; sc[threadIdx.x][3] = charge[a]; }
        __syncthreads();
        const int m = min(DH_TILE, n_atoms - a0);
#pragma unroll 4
        for (int s = 0; s < m; s++) {
            const double dx = gx - sc[s][0], dy = gy - sc[s][1], dz = gz - sc[s][2];
            const double d2 = (dx * dx + dy * dy) + dz * dz;
            const double ir = FAST ? dh_rsqrt(d2) : rsqrt(d2);          // 1/r, and r = d2/r: no division
            const double x = nkappa * (d2 * ir);
            acc = fma(sc[s][3], (FAST ? dh_exp_neg(x, tab) : exp(x)) * ir, acc);
        }
        __syncthreads();
    }
    if (t < nbc) bc[t] = acc / eps_out;
}

// The same boundary sum with every term evaluated in fp32 (coordinates relative to the box centre, MUFU rsqrt / ex2,
// Kahan-compensated fp32 partial sums per atom tile, tiles added in fp64): ~2 special-function operations per term
// instead of an fp64 rsqrt and exp, for callers who solve in fp32 anyway (pb_set_setup_precision).  Values agree with
// the fp64 kernel to a few 1e-7 of the largest term.
__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__global__ void __launch_bounds__(DH_TILE) k_grid_dh_f32(const double *__restrict__ c, const double *__restrict__ charge,
                                                         int n_atoms, int nx, int ny, int nz, double h, double eps_out,
                                                         double kappa, double *bc)
{
    __shared__ float4 sc[DH_TILE];
    const size_t n_xy = (size_t)ny * nx, n_zy = (size_t)nz * ny, n_zx = (size_t)nz * nx;
    const size_t nbc = 2 * (n_zy + n_zx + n_xy);
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const double cx = 0.5 * (nx - 1) * h, cy = 0.5 * (ny - 1) * h, cz = 0.5 * (nz - 1) * h;   // box centre
    double gx = 0.0, gy = 0.0, gz = 0.0;
    if (t < 2 * n_zy) {                                   // x-, x+ : [nz][ny]
        const size_t u = t % n_zy;
        gx = (t < n_zy) ? -h : nx * h; gy = (double)(u % ny) * h; gz = (double)(u / ny) * h;
    } else if (t < 2 * n_zy + 2 * n_zx) {                 // y-, y+ : [nz][nx]
        const size_t v = t - 2 * n_zy, u = v % n_zx;
        gy = (v < n_zx) ? -h : ny * h; gx = (double)(u % nx) * h; gz = (double)(u / nx) * h;
    } else if (t < nbc) {                                 // z-, z+ : [ny][nx]
        const size_t v = t - 2 * n_zy - 2 * n_zx, u = v % n_xy;
        gz = (v < n_xy) ? -h : nz * h; gx = (double)(u % nx) * h; gy = (double)(u / nx) * h;
    }
    const float fx = (float)(gx - cx), fy = (float)(gy - cy), fz = (float)(gz - cz);
    const float nk = (float)(-kappa * 1.4426950408889634);          // exp(-kappa r) = 2^(nk r)
    double acc = 0.0;
    for (int a0 = 0; a0 < n_atoms; a0 += DH_TILE) {
        const int a = a0 + threadIdx.x;
        if (a < n_atoms)
            sc[threadIdx.x] = make_float4((float)(c[3 * a] - cx), (float)(c[3 * a + 1] - cy), (float)(c[3 * a + 2] - cz),
                                          (float)charge[a]);
        __syncthreads();
        const int m = min(DH_TILE, n_atoms - a0);
        float s0 = 0.f, k0 = 0.f, s1 = 0.f, k1 = 0.f;     // two Kahan sums (even / odd atoms)
        int s = 0;
        for (; s + 1 < m; s += 2) {
            const float4 A = sc[s], B = sc[s + 1];
            const float ax = fx - A.x, ay = fy - A.y, az = fz - A.z, bx = fx - B.x, by = fy - B.y, bz = fz - B.z;
            const float da = fmaf(az, az, fmaf(ay, ay, ax * ax)), db = fmaf(bz, bz, fmaf(by, by, bx * bx));
            const float ia = mufu_rsq(da), ib = mufu_rsq(db);
            const float ta = A.w * (mufu_ex2(nk * (da * ia)) * ia), tb = B.w * (mufu_ex2(nk * (db * ib)) * ib);
            const float ya = ta - k0, yb = tb - k1;
            const float ua = s0 + ya, ub = s1 + yb;
            k0 = (ua - s0) - ya; k1 = (ub - s1) - yb;
            s0 = ua; s1 = ub;
        }
        if (s < m) {
            const float4 A = sc[s];
            const float ax = fx - A.x, ay = fy - A.y, az = fz - A.z;
            const float da = fmaf(az, az, fmaf(ay, ay, ax * ax));
            const float ia = mufu_rsq(da);
            const float ya = A.w * (mufu_ex2(nk * (da * ia)) * ia) - k0;
            const float ua = s0 + ya;
            k0 = (ua - s0) - ya; s0 = ua;
        }
        acc += (double)s0 + (double)s1;
        __syncthreads();
    }
    if (t < nbc) bc[t] = acc / eps_out;
}

}  // namespace pb
