// pb_noalloc.cu -- pb_residual_noalloc: the true relative residual ||b - A phi|| / ||b|| of Eq. 3 / Eq. 4
// (the quantity pb_residual reports, DESIGN.md Reading 5) for callers that cannot allocate: code
// under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The entry point calls no
// cudaMalloc / cudaFree / allocating library routine and does not synchronise: it enqueues one 256-byte memset and
// one kernel on the caller's stream.
//
// The kernel is a variant of k_true_residual (pb_kernels.cuh): the same two-stage deterministic reduction (per-block
// partial sums, the last block to take a ticket adds them in block order), but its scratch -- the partial sums and
// the ticket -- lives in a file-scope __device__ array of FIXED size instead of the handle's cudaMalloc'ed
// `partials`, and A phi and b are formed on the fly from the caller's dense fp64 arrays (no padded work arrays).
//
// Limits and sharing (stated in include/pb.h too):
//   * kNoAllocMaxRows = 262 144 grid rows (nz * ny, e.g. 512 x 512): one block per 8 rows, 32 768 blocks at most,
//     two partial sums each -> 512 KiB + 256 B of device memory held by every GPU that loads the library, until exit.
//   * every call on a device shares the array: calls that overlap on the GPU (two streams, two host threads) race.
//     The array keeps the last call's partial sums; the only word that must start at zero, the ticket, is cleared
//     on the stream before every launch.
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <mutex>

#include "../../include/pb.h"

namespace {

constexpr int kRowsPerBlock = 8;                          // one warp per grid row (k, j)
constexpr int kNoAllocMaxRows = PB_NOALLOC_MAX_ROWS;      // 262 144
constexpr int kNoAllocMaxBlocks = kNoAllocMaxRows / kRowsPerBlock;
constexpr int kTicketOffset = 2 * kNoAllocMaxBlocks;      // doubles; the ticket sits in its own 256-byte tail
constexpr int kMaxDevices = 64;

// [0, B): per-block ||r||^2;  [B, 2B): per-block ||b||^2 (B = kNoAllocMaxBlocks);  then 256 bytes holding the ticket
static __device__ __align__(256) double g_noalloc_scratch[2 * kNoAllocMaxBlocks + 32];

// Device address of the array, per device.  In host code `g_noalloc_scratch` is only a host-side stand-in for the
// symbol; the address a kernel may use comes from cudaGetSymbolAddress with that device current.
std::mutex g_mu;
double *g_scratch_ptr[kMaxDevices] = {nullptr};

pb_status scratch_for_current_device(double **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return PB_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) { cudaGetLastError(); return PB_ERR_CUDA; }
        g_scratch_ptr[dev] = static_cast<double *>(p);
    }
    *out = g_scratch_ptr[dev];
    return PB_OK;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// sum of n doubles by one block, in a fixed order (thread t adds elements t, t + 256, ...; then a fixed tree)
__device__ double ordered_sum(const double *v, int n, double *red)
{
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s += __ldcg(v + i);   // written by other SMs: read through L2
    s = warp_sum(s);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) t += red[w];
    return t;                                   // valid in thread 0
}

// h^2-scaled system (the relative residual does not depend on the scaling): with eps_f the six face values of node c,
//   (A' phi)(c) = (sum_f eps_f + h^2 kbar2(c)) phi(c) - sum_f eps_f phi(neighbour_f),  phi = 0 on the ghost layer
//   b'(c)       = h^2 rhs(c) + sum over ghost neighbours g of c of eps_face(c, g) bc(g)                 (Eq. 4)
// Layouts as pb_create: eps_x [nz][ny][nx+1], eps_y [nz][ny+1][nx], eps_z [nz+1][ny][nx], kbar2 / rhs / phi
// [nz][ny][nx], bc = the six ghost faces x-, x+ ([nz][ny]), y-, y+ ([nz][nx]), z-, z+ ([ny][nx]).
__global__ void __launch_bounds__(kRowsPerBlock * 32)
k_residual_noalloc(const double *__restrict__ eps_x, const double *__restrict__ eps_y, const double *__restrict__ eps_z,
                   const double *__restrict__ kbar2, const double *__restrict__ rhs, const double *__restrict__ bc,
                   const double *__restrict__ phi, double h2, int nx, int ny, int nz, double *scratch, double *out)
{
    __shared__ double red[2 * kRowsPerBlock];
    __shared__ int s_last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long rows = (long long)nz * ny;
    const long long row = (long long)blockIdx.x * kRowsPerBlock + warp;
    double s_rr = 0.0, s_bb = 0.0;
    if (row < rows) {
        const int j = (int)(row % ny), k = (int)(row / ny);
        const size_t o_xp = (size_t)nz * ny, o_ym = 2 * o_xp, o_yp = o_ym + (size_t)nz * nx,
                     o_zm = o_yp + (size_t)nz * nx, o_zp = o_zm + (size_t)ny * nx;
        const double *ex = eps_x + (size_t)row * (nx + 1);
        const double *eym = eps_y + ((size_t)k * (ny + 1) + j) * nx, *eyp = eym + nx;
        const double *ezm = eps_z + (size_t)row * nx, *ezp = ezm + (size_t)ny * nx;
        const double *pc = phi + (size_t)row * nx;
        const ptrdiff_t pl = (ptrdiff_t)ny * nx;              // elements per plane
        for (int i = lane; i < nx; i += 32) {
            const double exm_ = ex[i], exp_ = ex[i + 1], eym_ = eym[i], eyp_ = eyp[i], ezm_ = ezm[i], ezp_ = ezp[i];
            double d = exm_ + exp_ + eym_ + eyp_ + ezm_ + ezp_;
            if (kbar2) d += h2 * kbar2[(size_t)row * nx + i];
            double b = rhs ? h2 * rhs[(size_t)row * nx + i] : 0.0;
            double ap = d * pc[i];
            if (i > 0) ap -= exm_ * pc[i - 1];               else if (bc) b += exm_ * bc[(size_t)k * ny + j];
            if (i < nx - 1) ap -= exp_ * pc[i + 1];          else if (bc) b += exp_ * bc[o_xp + (size_t)k * ny + j];
            if (j > 0) ap -= eym_ * pc[i - nx];              else if (bc) b += eym_ * bc[o_ym + (size_t)k * nx + i];
            if (j < ny - 1) ap -= eyp_ * pc[i + nx];         else if (bc) b += eyp_ * bc[o_yp + (size_t)k * nx + i];
            if (k > 0) ap -= ezm_ * pc[i - pl];              else if (bc) b += ezm_ * bc[o_zm + (size_t)j * nx + i];
            if (k < nz - 1) ap -= ezp_ * pc[i + pl];         else if (bc) b += ezp_ * bc[o_zp + (size_t)j * nx + i];
            const double r = b - ap;
            s_rr = fma(r, r, s_rr);
            s_bb = fma(b, b, s_bb);
        }
    }
    s_rr = warp_sum(s_rr);
    s_bb = warp_sum(s_bb);
    if (lane == 0) { red[warp] = s_rr; red[kRowsPerBlock + warp] = s_bb; }
    __syncthreads();
    const int nblk = gridDim.x;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + kTicketOffset);
    if (threadIdx.x == 0) {
        double t_rr = 0.0, t_bb = 0.0;
        for (int w = 0; w < kRowsPerBlock; w++) { t_rr += red[w]; t_bb += red[kRowsPerBlock + w]; }
        scratch[blockIdx.x] = t_rr;
        scratch[kNoAllocMaxBlocks + blockIdx.x] = t_bb;
        __threadfence();
        s_last = (atomicAdd(ticket, 1u) == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        const double rr = ordered_sum(scratch, nblk, red);
        __syncthreads();
        const double bb = ordered_sum(scratch + kNoAllocMaxBlocks, nblk, red);
        if (threadIdx.x == 0) {
            *ticket = 0u;
            out[0] = bb > 0.0 ? sqrt(rr / bb) : 0.0;
            out[1] = rr;
            out[2] = bb;
        }
    }
}

}  // namespace

extern "C" pb_status pb_residual_noalloc(int nx, int ny, int nz, double h, const double *eps_x, const double *eps_y,
                                         const double *eps_z, const double *kbar2, const double *rhs, const double *bc,
                                         const double *phi, double *out3, void *cuda_stream)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(h > 0.0) || h != h || h > 1e300) return PB_ERR_INVALID_ARG;
    if ((long long)nz * ny > (long long)kNoAllocMaxRows) return PB_ERR_TOO_LARGE;     // before any pointer is touched
    if ((double)nx * ny * nz > 2.0e9) return PB_ERR_TOO_LARGE;
    if (!eps_x || !eps_y || !eps_z || !phi || !out3) return PB_ERR_INVALID_ARG;
    double *scratch = nullptr;
    const pb_status s = scratch_for_current_device(&scratch);
    if (s != PB_OK) return s;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long rows = (long long)nz * ny;
    const int grid = (int)((rows + kRowsPerBlock - 1) / kRowsPerBlock);
    // the ticket must start at zero (a call whose kernel never ran to its end could have left it elsewhere)
    if (cudaMemsetAsync(scratch + kTicketOffset, 0, 256, st) != cudaSuccess) { cudaGetLastError(); return PB_ERR_CUDA; }
    k_residual_noalloc<<<grid, kRowsPerBlock * 32, 0, st>>>(eps_x, eps_y, eps_z, kbar2, rhs, bc, phi, h * h, nx, ny, nz,
                                                           scratch, out3);
    if (cudaGetLastError() != cudaSuccess) return PB_ERR_CUDA;
    return PB_OK;
}
