// pb_internal.cuh -- device-side state, vector types and the deterministic two-stage
// reduction shared by the kernels of the Jacobi-PCG hot path.
// Product code: nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pb {

// ---------------------------------------------------------------------------------------
// Device-resident solver state: every scalar of PAPER.md:106-126 lives here, so the host
// never reads a dot product.  One instance per handle.
// ---------------------------------------------------------------------------------------
struct State {
    double rz;        // r_{l-1}^T z_{l-1}                     (step 5 numerator, step 7 denominator)
    double pAp;       // p^T A p                               (step 5 denominator)
    double rr;        // ||r_l||^2                             (step 3)
    double bb;        // ||b||^2                               (step 3)
    double alpha;     // alpha_l, written by the K_spmv finaliser
    double beta;      // beta_l,  written by the K_vec finaliser (0 before the first product)
    double tol2;      // delta^2
    int done;         // latch: 1 once the stopping rule, maxiter or a breakdown fired
    int iters;        // l at the moment `done` was latched
    int status;       // pb_status latched with `done`
    int iter_cur;     // l: number of completed iterations (also selects the p ping-pong buffer)
    int maxiter;
    int latch;        // 0: never latch (pb_iterate / benchmarking), 1: normal
    unsigned int ticket_spmv;
    unsigned int ticket_vec;
    // z-slab decomposition of ONE solve over several GPUs (pb_slab_*): the finalisers leave the
    // LOCAL sums here (pAp above, r.z / r.r below); the caller all-reduces them over the ranks in place, and the
    // k_slab_alpha / k_slab_finish kernels then take the same decisions on every rank
    double loc_rz, loc_rr;
    int slab;
    int xbuf;         // k_pcg_fused: which of its two x buffers holds the current iterate (0 after k_init)
    unsigned int pool_ctr;   // k_pcg_fused: next chunk of the dynamically scheduled tail (0 between launches)
    int pad2_;
};

// 16-byte vector of T: 4 floats or 2 doubles -> one 128-bit load/store per thread
template <typename T> struct Vec;
template <> struct alignas(16) Vec<float>  { float a[4]; };
template <> struct alignas(16) Vec<double> { double a[2]; };
template <typename T> struct VecN { static constexpr int value = 16 / sizeof(T); };

template <typename T> __device__ __forceinline__ Vec<T> ldv(const T *p) {
    return *reinterpret_cast<const Vec<T> *>(p);
}
template <typename T> __device__ __forceinline__ void stv(T *p, const Vec<T> &v) {
    *reinterpret_cast<Vec<T> *>(p) = v;
}
template <typename T> __device__ __forceinline__ Vec<T> zerov() {
    Vec<T> v;
#pragma unroll
    for (int e = 0; e < VecN<T>::value; e++) v.a[e] = T(0);
    return v;
}

// ---------------------------------------------------------------------------------------
// Deterministic reduction, stage 1: fixed-shape warp-shuffle tree, then a fixed-order sum
// of the warp partials by thread 0.  All threads of the block must call it.
// `scratch` holds >= 32 doubles per value.  Result valid in thread 0.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double block_sum(double v, double *scratch) {
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    if (lane == 0) scratch[w] = v;
    __syncthreads();
    double tot = 0.0;
    if (tid == 0)
        for (int i = 0; i < nw; i++) tot += scratch[i];
    __syncthreads();
    return tot;
}

// Stage 2 helper: the calling block (the last one to take a ticket) sums `n` per-block
// partials in a fixed order: thread t adds partials t, t+B, t+2B, ... then block_sum.
__device__ __forceinline__ double final_sum(const double *partials, int n, double *scratch) {
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v += __ldcg(partials + i);
    return block_sum(v, scratch);
}

}  // namespace pb
