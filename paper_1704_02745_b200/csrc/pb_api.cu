// pb_api.cu -- the C ABI of include/pb.h on top of the sm_100a kernels.
// Host logic only: argument checks, device memory, tile selection, the launch sequence of
// the PCG loop with its poll-every-k convergence latch, CUDA graphs.
// No step of the method runs on the host.  Product code: shares nothing with oracle/.
#include "../../include/pb.h"
#include "pb_kernels.cuh"
#include "pb_spmv_tma.cuh"
#include "pb_spmv_batch.cuh"
#include "pb_fused.cuh"
#include "pb_persist.cuh"
#include "pb_setup.cuh"
#include "pb_grid.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

using namespace pb;

namespace {

// Work set of pb_solve_batch: M members' vectors side by side ([M][npad], 4-D tensor maps), the
// coefficient arrays in the format k_spmv_batch reads (2-bit quads or words; unscaled Dinv index bytes), its plan.
template <typename T>
struct BatchWork {
    int cap = 0;                                   // members the vector arrays hold
    T *r = nullptr, *x = nullptr, *p0 = nullptr, *p1 = nullptr, *Ap = nullptr, *b = nullptr;
    T *r2 = nullptr, *Ap2 = nullptr;               // fused iteration (k_pcg_fused): second buffers of r and A p
    T *vblock = nullptr;                           // the one allocation behind r, Ap, p0, x, r2, Ap2, p1, x2 (in this order)
    T *x2 = nullptr;                               // fused iteration: second buffer of x (State::xbuf names the current one)
    unsigned char *cq4 = nullptr;                  // k_pcg_fused: {ez, ex-, ex+, ey} quad indices as one array
    CUtensorMap tm_q4;
    bool fused = false;                            // the plan / maps / graph below are the fused kernel's
    FusedMaps vm;
    bool coef_ready = false, quad = false, pald = false, own_words = false;
    unsigned char *exq = nullptr, *exqp = nullptr, *eyq = nullptr, *ezq = nullptr, *dviu = nullptr;
    T *exm = nullptr, *eym = nullptr, *ezm = nullptr;   // word format (aliases of Work's arrays unless own_words)
    int Pq = 0;
    int M = 0;                                     // members the plan / tensor maps / graph were built for
    int TXV = 0, TY = 0, TZ = 0, ntx = 0, nty = 0, ntz = 0, nsv = 0, nsc = 0, bps = 0, grid = 0, threads = 0;
    size_t smem = 0;
    int vec_grid = 0;
    int tuned = 0;                                 // the fused plan was chosen by timing candidates
    int zs = 0, pc = 0, npool = 0;                 // k_pcg_fused: static tiles over [0, zs), pool chunks of pc planes above
    CUtensorMap tm_r, tm_p0, tm_p1, tm_x, tm_dinv, tm_exm, tm_exp, tm_ey, tm_ez;
    cudaGraphExec_t graph = nullptr;
    int graph_iters = 0;
};

template <typename T>
struct Work {
    BatchWork<T> bw;
    T *exm = nullptr, *eym = nullptr, *ezm = nullptr, *D = nullptr, *Dinv = nullptr, *b = nullptr;
    T *x = nullptr, *r = nullptr, *tmp = nullptr, *p0 = nullptr, *p1 = nullptr, *Ap = nullptr;   // tmp: pb_apply input
    int P = 0;
    size_t npad = 0;                 // nz*ny*P
    size_t goff = 0;                 // z-slab mode: r, p0, p1, Dinv start one ghost plane (ny*P elements) into their allocation
    bool ready = false, b_ready = false;
    int vec_grid = 0;
    cudaGraphExec_t graph = nullptr;
    int graph_iters = 0;
    // TMA pipeline configuration of k_spmv_tma (tile, ring depth, persistent grid, tensor maps)
    int qTXV = 0, qTY = 0, qTZ = 0, qntx = 0, qnty = 0, qntz = 0, qns = 0, qgrid = 0, qthreads = 0, qbps = 0;
    bool qtuned = false;
    size_t qsmem = 0;
    CUtensorMap tm_r, tm_tmp, tm_dinv, tm_p0, tm_p1, tm_x, tm_ex, tm_ey, tm_ez;
    // L2-resident grids: the whole loop as one cooperative kernel (pb_persist.cuh)
    bool persist = false, pfused = false;
    int pgrid = 0;
    // coefficient palette (pb_setup.cuh): byte face indices + table, instead of exm/eym/ezm
    bool pal = false;
    unsigned char *exi = nullptr, *eyi = nullptr, *ezi = nullptr;
    T *lut = nullptr;
    // diagonal palette for k_vec: index byte per node + Dinv table
    bool pald = false;
    unsigned char *dvi = nullptr;
    size_t qmaxdyn = 224 * 1024;     // dynamic shared memory the chosen k_spmv_tma variant may use
    unsigned char *dvib = nullptr;   // the same indices in rows of Pb bytes (TMA strides are multiples of 16)
    bool pald_s = false;             // k_spmv_tma reads Dinv through the index tensor too
    T *dlut = nullptr;
    int Pb = 0;
};

}  // namespace

struct pb_handle {
    int nx, ny, nz;
    double h;
    int device;
    cudaStream_t stream;
    bool own_stream;
    double *eps_x, *eps_y, *eps_z, *kbar2, *rhs, *bc;   // dense fp64 device copies of the inputs
    State *st;
    double *partials;
    size_t partials_cap;
    int *bad;
    int *pinned;                 // 2 x 4 ints, page-locked
    State *pinned_state;
    cudaEvent_t ev[2];
    void *stage;                 // dense staging buffer for host <-> device vectors
    size_t stage_bytes;
    Work<float> wf;
    Work<double> wd;
    int opt[PB_OPT_COUNT_];     // per-handle options (pb_set_option); no environment variables except PB_VERBOSE
    int nsm;                     // multiprocessors of the device (cudaDevAttrMultiProcessorCount)
    long long launches;          // kernels enqueued so far (graph-contained ones included)
    int precond;                 // 1 Jacobi (default), 0 none
    int periodic;                // 0 Dirichlet ghost layer (free-space condition, default), 1 periodic
    bool slab = false;           // z-slab rank of a multi-GPU solve (pb_create_slab): ghost planes, local sums only
    int iface_lo = 0, iface_hi = 0;   // the plane below / above belongs to a neighbour rank (not the Dirichlet ghost layer)
    void *slab_send = nullptr, *slab_recv = nullptr;   // 4 planes each: [r_lo | p_lo | r_hi | p_hi]
    size_t slab_plane_bytes = 0;
    int slab_prec = -1;
    PalTable *pal_table;         // device; distinct face values of the operator
    PalTable *pald_table;        // device; distinct diagonal values
    int pald_n;                  // -1 unknown, 0 none, else table size
    int pal_n;                   // -1: not examined yet, 0: more than 256 distinct values, else the table size
    // pb_create_from_atoms keeps the atom geometry for pb_set_charges
    double *atoms_c;             // [n_atoms][3], device
    double *atoms_q = nullptr;   // [n_atoms] charges + 2 doubles of scratch, device (pb_set_charges; allocated once)
    int n_atoms;
    double atoms_eps_out, atoms_kappa;
    bool dh_f32 = false;         // pb_set_charges evaluates the Debye-Hueckel boundary terms in fp32
    int last_prec;               // precision of the last pb_solve/pb_solve_begin (for pb_query 3..7)
    bool last_fused = false;     // the last pb_solve / pb_solve_begin ran k_pcg_fused on the batch work set
};

namespace {

#define PB_CUDA(call)                                                          \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) {                                              \
            if (verbose())                                                     \
                fprintf(stderr, "pb: %s failed: %s (%s:%d)\n", #call,          \
                        cudaGetErrorString(e__), __FILE__, __LINE__);          \
            cudaGetLastError();                                                \
            return (e__ == cudaErrorMemoryAllocation) ? PB_ERR_ALLOC : PB_ERR_CUDA; \
        }                                                                      \
    } while (0)

// cudaMalloc / cudaFree can return cudaSuccess and still leave a non-sticky "invalid argument" in the runtime's
// last-error slot (observed on driver 580.159 / CUDA 12.9); clear it so later launch checks see only their own errors.
#define PB_ALLOC(call)            \
    do {                          \
        PB_CUDA(call);            \
        (void)cudaGetLastError(); \
    } while (0)

#define PB_TRY(expr)                       \
    do {                                   \
        pb_status s__ = (expr);            \
        if (s__ != PB_OK) return s__;      \
    } while (0)

template <typename T> Work<T> &work(pb_handle *h);
template <> Work<float> &work<float>(pb_handle *h) { return h->wf; }
template <> Work<double> &work<double>(pb_handle *h) { return h->wd; }

bool verbose() { static const bool v = getenv("PB_VERBOSE") != nullptr; return v; }

void default_options(int *opt)
{
    opt[PB_OPT_PERSIST] = 1; opt[PB_OPT_PERSIST_MAX_MB] = 100; opt[PB_OPT_PERSIST_FUSED_MAX_KNODES] = 600;
    opt[PB_OPT_PERSIST_BLOCKS_PER_SM] = 4; opt[PB_OPT_PALETTE] = 1; opt[PB_OPT_PALETTE_DIAG] = 1;
    opt[PB_OPT_PALETTE_DIAG_SPMV] = 1; opt[PB_OPT_AUTOTUNE] = 1; opt[PB_OPT_TILE_TXV] = 0; opt[PB_OPT_TILE_TY] = 0;
    opt[PB_OPT_TILE_TZ] = 0; opt[PB_OPT_RING_SLOTS] = 0; opt[PB_OPT_BLOCKS_PER_SM] = 0; opt[PB_OPT_VEC_BLOCKS_PER_SM] = 0;
    opt[PB_OPT_GRAPH] = 1; opt[PB_OPT_L2_HINTS] = 0; opt[PB_OPT_BATCH_WIDTH] = 1; opt[PB_OPT_FUSED] = 1;
}

inline int grid_for(size_t n, int block, int cap)
{
    size_t g = (n + block - 1) / block;
    if (g > (size_t)cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}


template <typename T>
pb_status alloc_arr(T **p, size_t n)
{
    PB_ALLOC(cudaMalloc((void **)p, (n + 64) * sizeof(T)));   // slack: vector tails never fault
    return PB_OK;
}

template <typename T>
void free_batch(BatchWork<T> &b)
{
    if (b.vblock) cudaFree(b.vblock);
    if (b.b) cudaFree(b.b);
    b.vblock = b.b = b.r = b.x = b.p0 = b.p1 = b.Ap = b.r2 = b.Ap2 = b.x2 = nullptr;
    unsigned char **idx[] = {&b.exq, &b.exqp, &b.eyq, &b.ezq, &b.dviu, &b.cq4};
    for (unsigned char **a : idx) { if (*a) cudaFree(*a); *a = nullptr; }
    if (b.own_words) { T **wa[] = {&b.exm, &b.eym, &b.ezm}; for (T **a : wa) { if (*a) cudaFree(*a); } }
    b.exm = b.eym = b.ezm = nullptr;
    if (b.graph) { cudaGraphExecDestroy(b.graph); b.graph = nullptr; }
    b.cap = 0; b.M = 0; b.coef_ready = false; b.own_words = false;
}

template <typename T>
void free_work(Work<T> &w)
{
    free_batch(w.bw);
    T **ghosted[] = {&w.Dinv, &w.r, &w.p0, &w.p1};
    for (T **a : ghosted) { if (*a) cudaFree(*a - w.goff); *a = nullptr; }
    w.goff = 0;
    T **arrs[] = {&w.exm, &w.eym, &w.ezm, &w.D, &w.b, &w.x, &w.tmp, &w.Ap};
    for (T **a : arrs) { if (*a) cudaFree(*a); *a = nullptr; }
    if (w.graph) { cudaGraphExecDestroy(w.graph); w.graph = nullptr; }
    unsigned char **idx[] = {&w.exi, &w.eyi, &w.ezi};
    for (unsigned char **a : idx) { if (*a) cudaFree(*a); *a = nullptr; }
    if (w.lut) { cudaFree(w.lut); w.lut = nullptr; }
    if (w.dvi) { cudaFree(w.dvi); w.dvi = nullptr; }
    if (w.dvib) { cudaFree(w.dvib); w.dvib = nullptr; }
    if (w.dlut) { cudaFree(w.dlut); w.dlut = nullptr; }
    w.ready = w.b_ready = false;
}

template <typename T>
pb_status build_b(pb_handle *h, Work<T> &w)
{
    const double h2 = h->h * h->h;
    k_setup_b<T><<<grid_for(w.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(
        h->eps_x, h->eps_y, h->eps_z, h->rhs, h->periodic ? nullptr : h->bc, h2, h->nx, h->ny, h->nz, w.P, w.b,
        h->iface_lo, h->iface_hi);
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    w.b_ready = true;
    return PB_OK;
}

template <typename T> pb_status setup_tma(pb_handle *h, Work<T> &w);
template <typename T> pb_status tune_vec(pb_handle *h, Work<T> &w);
pb_status ensure_stage(pb_handle *h, size_t bytes);

template <typename T> pb_status build_work(pb_handle *h, Work<T> &w);

// Lazily build the arrays of precision T (setup row a0).  Any failure frees what was allocated so far.
template <typename T>
pb_status ensure(pb_handle *h)
{
    Work<T> &w = work<T>(h);
    if (w.ready) {
        if (!w.b_ready) PB_TRY(build_b<T>(h, w));
        return PB_OK;
    }
    const pb_status s = build_work<T>(h, w);
    if (s != PB_OK) { cudaStreamSynchronize(h->stream); cudaGetLastError(); free_work(w); }
    return s;
}

template <typename T>
pb_status build_work(pb_handle *h, Work<T> &w)
{
    const int align = 32 / (int)sizeof(T);
    w.P = ((h->nx + 1 + align - 1) / align) * align;
    {
        // Row pitch such that the x tiling of the TMA kernels is EXACT (rows of ntx tiles of txv vectors, same rule as the
        // plans below): with a ragged last tile -- its boxes hang over the tensor's edge by more than the one halo vector
        // -- k_pcg_fused's 4-D boxes lose the L2 reuse of the y-halo rows (measured: DRAM reads 1.26x-1.5x the stored
        // bytes, 8.4-9.2 instead of 6.2-7.0 ps per node at 465^3 ... 513^3 fp32).  Costs at most a few pad vectors per row.
        constexpr int VEC = VecN<T>::value;
        const int maxv = 240 / VEC - 2;
        const int rowvecs = w.P / VEC;
        int ntx = (rowvecs + 32) / 64;
        if (ntx < 1) ntx = 1;
        while ((rowvecs + ntx - 1) / ntx > maxv) ntx++;
        int txv = (rowvecs + ntx - 1) / ntx;
        if (((ntx * txv) & 1) && txv + 1 <= maxv) txv++;           // rows stay a multiple of 32 bytes (two vectors)
        if (!((ntx * txv) & 1) && sizeof(T) == 4) w.P = ntx * txv * VEC;     // fp64: measured no gain (385^3: -3 %)
    }
    w.npad = (size_t)h->nz * h->ny * w.P;
    const size_t n_ey = (size_t)h->nz * (h->ny + 1) * w.P, n_ez = (size_t)(h->nz + 1) * h->ny * w.P;
    // distinct face values of the operator -> palette or full-precision face arrays (decided once per handle)
    if (h->pal_n < 0) {
        h->pal_n = 0;
        if (h->opt[PB_OPT_PALETTE]) {
            if (!h->pal_table) PB_ALLOC(cudaMalloc((void **)&h->pal_table, sizeof(PalTable)));
            k_pal_reset<<<1, 256, 0, h->stream>>>(h->pal_table);
            const size_t ns[3] = {(size_t)h->nz * h->ny * (h->nx + 1), (size_t)h->nz * (h->ny + 1) * h->nx,
                                  (size_t)(h->nz + 1) * h->ny * h->nx};
            const double *arrs[3] = {h->eps_x, h->eps_y, h->eps_z};
            for (int a = 0; a < 3; a++)
                k_pal_collect<<<grid_for(ns[a], 256, h->nsm * 8), 256, 0, h->stream>>>(arrs[a], ns[a], h->pal_table);
            k_pal_finish<<<1, 256, 0, h->stream>>>(h->pal_table);
            PB_CUDA(cudaGetLastError());
            int n = 0;
            PB_CUDA(cudaMemcpyAsync(&n, &h->pal_table->n, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            PB_CUDA(cudaStreamSynchronize(h->stream));
            h->pal_n = n;
            h->launches += 5;
        }
    }
    if (h->pald_n < 0) {
        h->pald_n = 0;
        if (h->pal_n > 0 && h->opt[PB_OPT_PALETTE_DIAG]) {     // few face values -> few diagonals (unless kbar2 varies)
            if (!h->pald_table) PB_ALLOC(cudaMalloc((void **)&h->pald_table, sizeof(PalTable)));
            k_pal_reset<<<1, 256, 0, h->stream>>>(h->pald_table);
            k_pal_collect_diag<<<grid_for((size_t)h->nx * h->ny * h->nz, 256, h->nsm * 8), 256, 0, h->stream>>>(
                h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->h * h->h, h->nx, h->ny, h->nz, h->pald_table);
            k_pal_finish<<<1, 256, 0, h->stream>>>(h->pald_table);
            PB_CUDA(cudaGetLastError());
            int n = 0;
            PB_CUDA(cudaMemcpyAsync(&n, &h->pald_table->n, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
            PB_CUDA(cudaStreamSynchronize(h->stream));
            h->pald_n = n;
            h->launches += 3;
        }
    }
    // k_spmv_tma decodes through tables addressed by pre-scaled index bytes: n * sizeof(T) <= 256 entries-bytes
    w.pal = h->pal_n > 0 && (size_t)h->pal_n * sizeof(T) <= 256;
    w.pald = w.pal && h->pald_n > 0;
    // (z-slab mode: Dinv words in the SpMV -- its ghost planes come from the neighbour rank, whose palette differs)
    w.pald_s = w.pald && (size_t)h->pald_n * sizeof(T) <= 256 && h->opt[PB_OPT_PALETTE_DIAG_SPMV] != 0 && !h->slab;
    w.Pb = (w.P + 15) / 16 * 16;
    // working set (11 node-sized arrays) small enough to live in L2 -> persistent cooperative kernel for pb_solve
    {
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device);
        const double mb = 11.0 * (double)w.npad * sizeof(T) / 1.0e6;
        w.persist = coop && h->opt[PB_OPT_PERSIST] != 0 && mb <= (double)h->opt[PB_OPT_PERSIST_MAX_MB] && !h->slab;
    }
    pb_status s = PB_OK;
    if (w.pal && w.persist &&
        ((s = alloc_arr(&w.exm, w.npad)) || (s = alloc_arr(&w.eym, n_ey)) || (s = alloc_arr(&w.ezm, n_ez)))) {
        free_work(w);
        return s;
    }
    if (w.pald && ((s = alloc_arr(&w.dvi, w.npad)) || (s = alloc_arr(&w.dlut, (size_t)kPalMax)))) {
        free_work(w);
        return s;
    }
    if (w.pald_s && (s = alloc_arr(&w.dvib, (size_t)h->nz * h->ny * w.Pb))) { free_work(w); return s; }
    if (w.pal) {
        const size_t b_ex = (size_t)h->nz * h->ny * w.Pb, b_ey = (size_t)h->nz * (h->ny + 1) * w.Pb,
                     b_ez = (size_t)(h->nz + 1) * h->ny * w.Pb;
        if ((s = alloc_arr(&w.exi, b_ex)) || (s = alloc_arr(&w.eyi, b_ey)) || (s = alloc_arr(&w.ezi, b_ez)) ||
            (s = alloc_arr(&w.lut, (size_t)kPalMax))) { free_work(w); return s; }
    } else if ((s = alloc_arr(&w.exm, w.npad)) || (s = alloc_arr(&w.eym, n_ey)) || (s = alloc_arr(&w.ezm, n_ez))) {
        free_work(w);
        return s;
    }
    if ((s = alloc_arr(&w.D, w.npad)) || (s = alloc_arr(&w.b, w.npad)) || (s = alloc_arr(&w.x, w.npad)) ||
        (s = alloc_arr(&w.tmp, w.npad)) || (s = alloc_arr(&w.Ap, w.npad))) {
        free_work(w);
        return s;
    }
    {   // the haloed arrays; in z-slab mode with one ghost plane below plane 0 and one above plane nz-1 (zeroed: the
        // Dirichlet ghost layer where there is no neighbour rank; Dinv = 1 there so that p_new(ghost) = 0 exactly)
        const size_t gp = h->slab ? (size_t)h->ny * w.P : 0;
        T **ghosted[] = {&w.Dinv, &w.r, &w.p0, &w.p1};
        for (T **a : ghosted) {
            if ((s = alloc_arr(a, w.npad + 2 * gp))) { w.goff = 0; free_work(w); return s; }
            if (gp) PB_CUDA(cudaMemsetAsync(*a, 0, (w.npad + 2 * gp) * sizeof(T), h->stream));
        }
        for (T **a : ghosted) *a += gp;
        w.goff = gp;
    }
    w.vec_grid = grid_for(w.npad / VecN<T>::value, 512, h->nsm * (h->opt[PB_OPT_VEC_BLOCKS_PER_SM] > 0 ? h->opt[PB_OPT_VEC_BLOCKS_PER_SM] : 4));   // 2 vectors per thread and pass
    if (w.persist) {
        // tiny grids: barriers dominate -> the two-barrier form that recomputes p at the neighbours
        w.pfused = (double)w.npad <= (double)h->opt[PB_OPT_PERSIST_FUSED_MAX_KNODES] * 1.0e3;
        int bps = 0;
        const cudaError_t eo = w.pfused ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_pcg_persistent<T, true>, 256, 0)
                                        : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_pcg_persistent<T, false>, 256, 0);
        if (eo != cudaSuccess) { cudaGetLastError(); bps = 0; }
        if (bps < 1) { w.persist = false; bps = 1; }      // no co-residency on this device/partition: two-kernel path
        bps = bps > h->opt[PB_OPT_PERSIST_BLOCKS_PER_SM] ? h->opt[PB_OPT_PERSIST_BLOCKS_PER_SM] : bps;
        w.pgrid = grid_for(w.npad / VecN<T>::value, 256, h->nsm * bps);
    }
    size_t need = (size_t)h->nsm * 16 > (size_t)2 * w.vec_grid ? (size_t)h->nsm * 16 : (size_t)2 * w.vec_grid;
    if ((size_t)3 * w.pgrid > need) need = (size_t)3 * w.pgrid;
    if (need > h->partials_cap) {
        if (h->partials) cudaFree(h->partials);
        h->partials = nullptr;
        h->partials_cap = 0;
        PB_ALLOC(cudaMalloc((void **)&h->partials, need * sizeof(double)));
        h->partials_cap = need;
    }
    PB_CUDA(cudaMemsetAsync(h->bad, 0, sizeof(int), h->stream));
    const size_t total = (size_t)(h->nz + 1) * (h->ny + 1) * w.P;
    k_setup_coeff<T><<<grid_for(total, 256, h->nsm * 16), 256, 0, h->stream>>>(
        h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->h * h->h, h->nx, h->ny, h->nz, w.P,
        w.exm, w.eym, w.ezm, w.D, w.Dinv, h->bad);
    if (w.pal) {
        k_setup_pal_idx<<<grid_for((size_t)(h->nz + 1) * (h->ny + 1) * w.Pb, 256, h->nsm * 16), 256, 0, h->stream>>>(
            h->eps_x, h->eps_y, h->eps_z, h->nx, h->ny, h->nz, w.Pb, (int)sizeof(T), h->pal_table, w.exi, w.eyi, w.ezi);
        k_pal_lut<T><<<1, 256, 0, h->stream>>>(h->pal_table, w.lut);
        h->launches += 2;
    }
    if (w.pald) {
        k_setup_diag_idx<<<grid_for(w.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(
            h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->h * h->h, h->nx, h->ny, h->nz, w.P, 1, h->pald_table, w.dvi);
        k_pal_lut_dinv<T><<<1, 256, 0, h->stream>>>(h->pald_table, w.dlut);
        h->launches += 2;
        if (w.pald_s) {
            k_setup_diag_idx<<<grid_for((size_t)h->nz * h->ny * w.Pb, 256, h->nsm * 16), 256, 0, h->stream>>>(
                h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->h * h->h, h->nx, h->ny, h->nz, w.Pb, (int)sizeof(T), h->pald_table, w.dvib);
            h->launches += 1;
        }
    }
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    PB_TRY(build_b<T>(h, w));
    PB_TRY(setup_tma<T>(h, w));
    PB_TRY(tune_vec<T>(h, w));
    w.ready = true;
    return PB_OK;
}

template <typename T>
VecArgs<T> vec_args(pb_handle *h, Work<T> &w)
{
    VecArgs<T> a;
    a.r = w.r; a.Ap = w.Ap; a.Dinv = w.Dinv; a.b = w.b; a.x = w.x; a.pzero = w.p0; a.l2hints = h->opt[PB_OPT_L2_HINTS]; a.precond = h->precond; a.dvi = w.dvi; a.dlut = w.dlut; a.nvec = w.npad / VecN<T>::value; a.st = h->st; a.partials = h->partials;
    return a;
}


// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    }
    return fn;
}

// 3-D tensor [planes][rows][P] of T, box = bx elements x by rows x 1 plane, zero fill outside
template <typename T>
pb_status make_map(CUtensorMap *tm, const T *ptr, int P, int rows, int planes, int bx, int by)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return PB_ERR_CUDA;
    const cuuint64_t dims[3] = {(cuuint64_t)P, (cuuint64_t)rows, (cuuint64_t)planes};
    const cuuint64_t strides[2] = {(cuuint64_t)P * sizeof(T), (cuuint64_t)P * rows * sizeof(T)};
    const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = fn(tm, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3,
                          (void *)ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        if (verbose()) fprintf(stderr, "pb: cuTensorMapEncodeTiled failed (%d)\n", (int)r);
        return PB_ERR_CUDA;
    }
    return PB_OK;
}

// byte tensor [planes][rows][Pb] of face indices, box = bw bytes x by rows x 1 plane, zero fill outside
pb_status make_map_u8(CUtensorMap *tm, const unsigned char *ptr, int Pb, int rows, int planes, int bw, int by)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return PB_ERR_CUDA;
    const cuuint64_t dims[3] = {(cuuint64_t)Pb, (cuuint64_t)rows, (cuuint64_t)planes};
    const cuuint64_t strides[2] = {(cuuint64_t)Pb, (cuuint64_t)Pb * rows};
    const cuuint32_t box[3] = {(cuuint32_t)bw, (cuuint32_t)by, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void *)ptr, dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? PB_OK : PB_ERR_CUDA;
}

struct TileCfg { int TXV, TY, NS, bps, TZ; };   // TZ = 0: derive from the tile count

// z split of a tile column: blocks stride over the tile list, so the launch lasts ceil(tiles / slots) tiles.  Take
// the split whose tile count fills those waves best (a count just above a multiple of the grid wastes up to a whole
// wave), charging each tile its two halo planes (about one plane's worth of traffic); fewest tiles on ties.
inline int choose_tz(int nz, int xy, int slots)
{
    double best = -1.0;
    int best_ntz = 1;
    const int max_ntz = nz / 8 > 1 ? nz / 8 : 1;
    for (int ntz = 1; ntz <= max_ntz && (long)xy * ntz <= 8L * slots + xy; ntz++) {
        const int tz = (nz + ntz - 1) / ntz;
        const long tiles = (long)xy * ((nz + tz - 1) / tz);
        const long waves = (tiles + slots - 1) / slots;
        const double fill = (double)tiles / (double)(waves * slots);
        const double score = fill * tz / (tz + 1.0);
        if (score > best + 1e-9) { best = score; best_ntz = ntz; }
    }
    return (nz + best_ntz - 1) / best_ntz;
}

// apply one tile / ring / grid configuration: sizes, persistent grid, tensor maps
template <typename T>
pb_status configure_tma(pb_handle *h, Work<T> &w, const TileCfg &c)
{
    constexpr int VEC = VecN<T>::value;
    const int rowvecs = w.P / VEC;
    const int TXV = c.TXV, TY = c.TY, NS = c.NS;
    w.qTXV = TXV; w.qTY = TY; w.qns = NS; w.qbps = c.bps;
    w.qntx = (rowvecs + TXV - 1) / TXV;
    w.qnty = (h->ny + TY - 1) / TY;
    w.qthreads = (spmv_row_threads(TXV) * TY + 31) / 32 * 32 + 32;
    const SlotLayout L = slot_layout(TXV, TY, w.pal ? VEC : 0, w.pald_s);
    w.qsmem = (size_t)NS * L.slot + 128;
    if (w.qsmem > w.qmaxdyn || w.qthreads > 512 || NS < 3 || NS > kMaxStages) return PB_ERR_INVALID_ARG;
    const int slots = h->nsm * c.bps;
    const int xy = w.qntx * w.qnty;
    int TZ = c.TZ;
    if (TZ <= 0) TZ = choose_tz(h->nz, xy, slots);
    if (TZ > h->nz) TZ = h->nz;
    w.qTZ = TZ;
    w.qntz = (h->nz + TZ - 1) / TZ;
    const long ntiles = (long)xy * w.qntz;
    w.qgrid = (int)(ntiles < slots ? ntiles : slots);
    const int gpl = w.goff ? 2 : 0;      // z-slab mode: ghost planes in the haloed tensors (the kernel adds zoff = 1)
    PB_TRY(make_map<T>(&w.tm_r, w.r - w.goff, w.P, h->ny, h->nz + gpl, (TXV + 2) * VEC, TY + 2));
    PB_TRY(make_map<T>(&w.tm_tmp, w.tmp, w.P, h->ny, h->nz, (TXV + 2) * VEC, TY + 2));
    if (w.pald_s) PB_TRY(make_map_u8(&w.tm_dinv, w.dvib, w.Pb, h->ny, h->nz, L.bwd, TY + 2));
    else PB_TRY(make_map<T>(&w.tm_dinv, w.Dinv - w.goff, w.P, h->ny, h->nz + gpl, (TXV + 2) * VEC, TY + 2));
    PB_TRY(make_map<T>(&w.tm_p0, w.p0 - w.goff, w.P, h->ny, h->nz + gpl, (TXV + 2) * VEC, TY + 2));
    PB_TRY(make_map<T>(&w.tm_p1, w.p1 - w.goff, w.P, h->ny, h->nz + gpl, (TXV + 2) * VEC, TY + 2));
    PB_TRY(make_map<T>(&w.tm_x, w.x, w.P, h->ny, h->nz, TXV * VEC, TY));
    if (w.pal) {
        PB_TRY(make_map_u8(&w.tm_ex, w.exi, w.Pb, h->ny, h->nz, L.bw, TY));
        PB_TRY(make_map_u8(&w.tm_ey, w.eyi, w.Pb, h->ny + 1, h->nz, L.bw, TY + 1));
        PB_TRY(make_map_u8(&w.tm_ez, w.ezi, w.Pb, h->ny, h->nz + 1, L.bw, TY));
    } else {
        PB_TRY(make_map<T>(&w.tm_ex, w.exm, w.P, h->ny, h->nz, (TXV + 1) * VEC, TY));
        PB_TRY(make_map<T>(&w.tm_ey, w.eym, w.P, h->ny + 1, h->nz, TXV * VEC, TY + 1));
        PB_TRY(make_map<T>(&w.tm_ez, w.ezm, w.P, h->ny, h->nz + 1, TXV * VEC, TY));
    }
    return PB_OK;
}

template <typename T, int MODE> void launch_spmv(pb_handle *h, Work<T> &w, double out_scale);

// deepest ring (<= 6 slots) that lets `bps` blocks of this tile share one SM's shared memory
inline int ring_depth(int TXV, int TY, int bps, int pal_vec, bool pald)
{
    // 227 KB per SM, 1 KB reserved per block, statics (barriers, reduction scratch, up to three 256-entry tables)
    const size_t per_block = (size_t)232448 / bps - 1024 - 3200 - (pald ? 2 * 256 * (16 / pal_vec) : 0);
    int NS = (int)(per_block / slot_layout(TXV, TY, pal_vec, pald).slot);
    return NS > 6 ? 6 : NS;
}

// Tile / ring / grid selection for k_spmv_tma.  Explicit PB_TXV/PB_TY/PB_NS/PB_BPS/PB_TZ win; otherwise a
// short list of candidates (x splits of about 0.5-1 KB rows, 2-8 rows, 1-4 blocks per SM, the deepest ring
// that fits) is timed on the handle's own arrays -- three launches each -- and the fastest is kept, like an
// FFT plan.  PB_AUTOTUNE=0 takes the first feasible candidate instead (fully static choice).
template <typename T>
pb_status setup_tma(pb_handle *h, Work<T> &w)
{
    constexpr int VEC = VecN<T>::value;
    const int rowvecs = w.P / VEC;
    // box inner dimension <= 256 elements (byte-index boxes: the haloed row plus 16 bytes of lead-in)
    const int maxv = (w.pal ? 240 : 256) / VEC - 2;
    // dynamic + static shared memory <= 227 KB per block; the static part depends on the variant (its tables)
    auto allow = [&](auto kernel, size_t *max_dyn) -> pb_status {
        cudaFuncAttributes fa;
        PB_CUDA(cudaFuncGetAttributes(&fa, kernel));
        const size_t lim = (size_t)232448 - fa.sharedSizeBytes;
        PB_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lim));
        if (max_dyn) *max_dyn = lim;
        return PB_OK;
    };
    size_t lim0 = 0, lim1 = 0;
    if (w.pald_s) { PB_TRY(allow(k_spmv_tma<T, 0, true, true>, &lim0)); PB_TRY(allow(k_spmv_tma<T, 1, true, true>, &lim1)); }
    else if (w.pal) { PB_TRY(allow(k_spmv_tma<T, 0, true, false>, &lim0)); PB_TRY(allow(k_spmv_tma<T, 1, true, false>, &lim1)); }
    else { PB_TRY(allow(k_spmv_tma<T, 0, false, false>, &lim0)); PB_TRY(allow(k_spmv_tma<T, 1, false, false>, &lim1)); }
    w.qmaxdyn = lim0 < lim1 ? lim0 : lim1;
    int ntx0 = (rowvecs + 32) / 64;                                  // rows of about 64 vectors (1 KB)
    if (ntx0 < 1) ntx0 = 1;
    while ((rowvecs + ntx0 - 1) / ntx0 > maxv) ntx0++;
    TileCfg cand[64];
    int nc = 0;
    const int *o = h->opt;
    auto opt_or = [&](pb_option k, int dflt) { return o[k] > 0 ? o[k] : dflt; };
    const bool forced = o[PB_OPT_TILE_TXV] > 0 || o[PB_OPT_TILE_TY] > 0 || o[PB_OPT_RING_SLOTS] > 0 ||
                        o[PB_OPT_BLOCKS_PER_SM] > 0 || o[PB_OPT_TILE_TZ] > 0;
    if (forced) {
        TileCfg c;
        c.TXV = opt_or(PB_OPT_TILE_TXV, (rowvecs + ntx0 - 1) / ntx0);
        if (c.TXV < 1) c.TXV = 1;
        if (c.TXV > maxv) c.TXV = maxv;
        if (c.TXV > rowvecs) c.TXV = rowvecs;
        c.TY = opt_or(PB_OPT_TILE_TY, 4);
        if (c.TY < 1) c.TY = 1;
        if (c.TY > h->ny) c.TY = h->ny;
        while (spmv_row_threads(c.TXV) * c.TY > 448 && c.TY > 1) c.TY--;
        c.bps = opt_or(PB_OPT_BLOCKS_PER_SM, ring_depth(c.TXV, c.TY, 2, w.pal ? VEC : 0, w.pald_s) >= 4 ? 2 : 1);
        if (c.bps < 1) c.bps = 1;
        c.NS = opt_or(PB_OPT_RING_SLOTS, ring_depth(c.TXV, c.TY, c.bps, w.pal ? VEC : 0, w.pald_s));
        c.TZ = o[PB_OPT_TILE_TZ];
        cand[nc++] = c;
    } else {
        static const int tys[] = {8, 4, 6, 3, 2};
        for (int dx = 0; dx < 2; dx++) {
            const int ntx = ntx0 + dx;
            const int TXV = (rowvecs + ntx - 1) / ntx;
            if (dx && TXV * VEC < 64) break;
            for (int ty : tys) {
                int TY = ty > h->ny ? h->ny : ty;
                if (spmv_row_threads(TXV) * TY > 448) continue;
                for (int bps = 1; bps <= 4; bps++) {
                    const int NS = ring_depth(TXV, TY, bps, w.pal ? VEC : 0, w.pald_s);
                    if (NS < 4 && !(NS == 3 && bps >= 2)) continue;
                    const int cthreads = ((spmv_row_threads(TXV) * TY + 31) / 32 * 32) * bps;
                    if (cthreads < 256 || cthreads > 1024) continue;     // consumer threads per SM
                    if (nc < 64) cand[nc++] = TileCfg{TXV, TY, NS, bps, 0};
                }
            }
        }
        if (nc == 0) cand[nc++] = TileCfg{(rowvecs + ntx0 - 1) / ntx0, h->ny < 4 ? h->ny : 4, 4, 1, 0};
    }
    int best = 0;
    const bool tune = nc > 1 && h->opt[PB_OPT_AUTOTUNE] != 0 && (double)h->nx * h->ny * h->nz >= 2.0e5;
    if (tune) {
        cudaEvent_t e0, e1;
        PB_CUDA(cudaEventCreate(&e0));
        PB_CUDA(cudaEventCreate(&e1));
        PB_CUDA(cudaMemsetAsync(w.r, 0, w.npad * sizeof(T), h->stream));
        PB_CUDA(cudaMemsetAsync(w.p0, 0, w.npad * sizeof(T), h->stream));
        PB_CUDA(cudaMemsetAsync(w.p1, 0, w.npad * sizeof(T), h->stream));
        PB_CUDA(cudaMemsetAsync(w.x, 0, w.npad * sizeof(T), h->stream));
        k_set_state<<<1, 1, 0, h->stream>>>(h->st, 1.0, 0, 0);
        float tbest = 1e30f;
        float tms[64];
        for (int i = 0; i < nc; i++) {
            tms[i] = 1e30f;
            if (configure_tma<T>(h, w, cand[i]) != PB_OK) continue;
            if ((size_t)w.qgrid > h->partials_cap) continue;
            launch_spmv<T, 0>(h, w, 1.0);
            cudaEventRecord(e0, h->stream);
            for (int rep = 0; rep < 3; rep++) launch_spmv<T, 0>(h, w, 1.0);
            cudaEventRecord(e1, h->stream);
            if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
                cudaEventDestroy(e0); cudaEventDestroy(e1);
                return PB_ERR_CUDA;
            }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (verbose())
                fprintf(stderr, "pb: tune TXV=%d TY=%d NS=%d bps=%d TZ=%d grid=%d: %.4f ms\n", cand[i].TXV, cand[i].TY,
                        cand[i].NS, cand[i].bps, w.qTZ, w.qgrid, ms / 3);
            tms[i] = ms;
            if (ms < tbest) { tbest = ms; best = i; }
        }
        // second pass: the three fastest plans are within the noise of three launches of each other; time them
        // again the way the solver runs them -- alternating with k_vec, twelve iterations each
        int fin[3] = {-1, -1, -1};
        for (int f = 0; f < 3; f++) {
            float tb = 1e30f;
            for (int i = 0; i < nc; i++)
                if (tms[i] < tb && i != fin[0] && i != fin[1]) { tb = tms[i]; fin[f] = i; }
        }
        if (fin[1] >= 0 && (size_t)2 * w.vec_grid <= h->partials_cap) {
            const VecArgs<T> va = vec_args<T>(h, w);
            tbest = 1e30f;
            for (int f = 0; f < 3 && fin[f] >= 0; f++) {
                if (configure_tma<T>(h, w, cand[fin[f]]) != PB_OK) continue;
                cudaEventRecord(e0, h->stream);
                for (int rep = 0; rep < 12; rep++) {
                    launch_spmv<T, 0>(h, w, 1.0);
                    if (w.pald) k_vec<T, true><<<w.vec_grid, 256, 0, h->stream>>>(va);
                    else k_vec<T, false><<<w.vec_grid, 256, 0, h->stream>>>(va);
                }
                cudaEventRecord(e1, h->stream);
                if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
                    cudaEventDestroy(e0); cudaEventDestroy(e1);
                    return PB_ERR_CUDA;
                }
                float ms = 0.f;
                cudaEventElapsedTime(&ms, e0, e1);
                if (verbose())
                    fprintf(stderr, "pb: tune (pass 2) TXV=%d TY=%d NS=%d bps=%d: %.4f ms per iteration\n", cand[fin[f]].TXV,
                            cand[fin[f]].TY, cand[fin[f]].NS, cand[fin[f]].bps, ms / 12);
                if (ms < tbest) { tbest = ms; best = fin[f]; }
            }
        }
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
    }
    PB_TRY(configure_tma<T>(h, w, cand[best]));
    w.qtuned = tune;
    if (verbose())
        fprintf(stderr, "pb: palette %d (diagonal %d); k_spmv_tma<%s> TXV=%d TY=%d TZ=%d NS=%d bps=%d tiles=%d grid=%d threads=%d smem=%zu%s\n",
                h->pal_n, w.pald_s ? h->pald_n : 0, sizeof(T) == 4 ? "f32" : "f64", w.qTXV, w.qTY, w.qTZ, w.qns, cand[best].bps,
                w.qntx * w.qnty * w.qntz, w.qgrid, w.qthreads, w.qsmem, tune ? " (autotuned)" : "");
    return PB_OK;
}

// one launch of the SpMV kernel (MODE 0: PCG step, MODE 1: y = scale*A'x)
template <typename T, int MODE>
void launch_spmv(pb_handle *h, Work<T> &w, double out_scale)
{
    TmaArgs<T> a;
    a.pbuf0 = w.p0; a.pbuf1 = w.p1; a.Ap = w.Ap; a.x = w.x;
    a.nx = h->nx; a.ny = h->ny; a.nz = h->nz; a.P = w.P;
    a.TXV = w.qTXV; a.TY = w.qTY; a.TZ = w.qTZ; a.ntx = w.qntx; a.nty = w.qnty; a.ntz = w.qntz;
    a.ntiles = w.qntx * w.qnty * w.qntz; a.nstage = w.qns; a.l2hints = h->opt[PB_OPT_L2_HINTS]; a.precond = h->precond;
    a.zoff = (MODE == 0 && w.goff) ? 1 : 0;
    a.st = h->st; a.partials = h->partials; a.out_scale = out_scale;
    a.lut = w.lut; a.dlut = w.dlut;
    if (w.pald_s)
        k_spmv_tma<T, MODE, true, true><<<w.qgrid, w.qthreads, w.qsmem, h->stream>>>(
            MODE == 0 ? w.tm_r : w.tm_tmp, w.tm_dinv, w.tm_p0, w.tm_p1, w.tm_x, w.tm_ex, w.tm_ey, w.tm_ez, a);
    else if (w.pal)
        k_spmv_tma<T, MODE, true, false><<<w.qgrid, w.qthreads, w.qsmem, h->stream>>>(
            MODE == 0 ? w.tm_r : w.tm_tmp, w.tm_dinv, w.tm_p0, w.tm_p1, w.tm_x, w.tm_ex, w.tm_ey, w.tm_ez, a);
    else
        k_spmv_tma<T, MODE, false, false><<<w.qgrid, w.qthreads, w.qsmem, h->stream>>>(
            MODE == 0 ? w.tm_r : w.tm_tmp, w.tm_dinv, w.tm_p0, w.tm_p1, w.tm_x, w.tm_ex, w.tm_ey, w.tm_ez, a);
}

// k_vec is a plain stream, but its rate depends measurably on how many blocks share an SM (DRAM page / bank
// interleaving of the concurrent streams): time 3-8 blocks per SM once per handle, like the SpMV plan.
template <typename T>
pb_status tune_vec(pb_handle *h, Work<T> &w)
{
    if (h->opt[PB_OPT_VEC_BLOCKS_PER_SM] > 0 || h->opt[PB_OPT_AUTOTUNE] == 0 || (double)h->nx * h->ny * h->nz < 2.0e6) return PB_OK;
    cudaEvent_t e0, e1;
    PB_CUDA(cudaEventCreate(&e0));
    PB_CUDA(cudaEventCreate(&e1));
    PB_CUDA(cudaMemsetAsync(w.r, 0, w.npad * sizeof(T), h->stream));
    PB_CUDA(cudaMemsetAsync(w.Ap, 0, w.npad * sizeof(T), h->stream));
    k_set_state<<<1, 1, 0, h->stream>>>(h->st, 1.0, 0, 0);
    static const int cand[] = {3, 4, 5, 6, 8};
    float tbest = 1e30f;
    int best = w.vec_grid;
    for (int c : cand) {
        w.vec_grid = grid_for(w.npad / VecN<T>::value, 512, h->nsm * c);
        if ((size_t)2 * w.vec_grid > h->partials_cap) continue;
        const VecArgs<T> va = vec_args<T>(h, w);
        auto launch = [&]() {
            if (w.pald) k_vec<T, true><<<w.vec_grid, 256, 0, h->stream>>>(va);
            else k_vec<T, false><<<w.vec_grid, 256, 0, h->stream>>>(va);
        };
        launch();
        cudaEventRecord(e0, h->stream);
        for (int rep = 0; rep < 3; rep++) launch();
        cudaEventRecord(e1, h->stream);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
            cudaEventDestroy(e0); cudaEventDestroy(e1);
            return PB_ERR_CUDA;
        }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (verbose()) fprintf(stderr, "pb: tune k_vec %d blocks/SM (grid %d): %.4f ms\n", c, w.vec_grid, ms / 3);
        if (ms < tbest) { tbest = ms; best = w.vec_grid; }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    w.vec_grid = best;
    return PB_OK;
}

// periodic boundary condition: the wrap terms k_spmv_tma cannot see (k_wrap), right after it
template <typename T, int MODE>
void launch_wrap(pb_handle *h, Work<T> &w, double out_scale)
{
    if (!h->periodic) return;
    WrapArgs<T> a;
    a.pbuf0 = MODE == 0 ? w.p0 : w.tmp; a.pbuf1 = w.p1; a.Ap = w.Ap;
    a.eps_x = h->eps_x; a.eps_y = h->eps_y; a.eps_z = h->eps_z;
    a.nx = h->nx; a.ny = h->ny; a.nz = h->nz; a.P = w.P; a.out_scale = out_scale;
    a.st = h->st; a.partials = h->partials;
    const size_t shell = 2 * ((size_t)h->ny * h->nx + (size_t)h->nz * h->nx + (size_t)h->nz * h->ny);
    k_wrap<T, MODE><<<grid_for(shell, 256, h->nsm * 8), 256, 0, h->stream>>>(a);
    h->launches += 1;
}

// enqueue n PCG iterations: (k_spmv, k_vec) pairs, nothing else
template <typename T>
pb_status enqueue_iterations(pb_handle *h, Work<T> &w, int n)
{
    const VecArgs<T> va = vec_args<T>(h, w);
    for (int it = 0; it < n; it++) {
        launch_spmv<T, 0>(h, w, 1.0);
        launch_wrap<T, 0>(h, w, 1.0);
        if (w.pald) k_vec<T, true><<<w.vec_grid, 256, 0, h->stream>>>(va);
        else k_vec<T, false><<<w.vec_grid, 256, 0, h->stream>>>(va);
    }
    PB_CUDA(cudaGetLastError());
    h->launches += 2LL * n;
    return PB_OK;
}

template <typename T>
pb_status begin_solve(pb_handle *h, double tol, int maxiter, int latch, const void *phi0 = nullptr,
                      pb_memspace where = PB_DEVICE)
{
    PB_TRY(ensure<T>(h));
    Work<T> &w = work<T>(h);
    h->last_prec = sizeof(T) == 4 ? PB_F32 : PB_F64;
    k_set_state<<<1, 1, 0, h->stream>>>(h->st, tol * tol, maxiter, latch);
    k_init<T><<<w.vec_grid, 256, 0, h->stream>>>(vec_args<T>(h, w));
    PB_CUDA(cudaGetLastError());
    h->launches += 2;
    if (phi0) {   // step 1 with a given phi_0: x = phi_0, r = b - A phi_0
        const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
        const T *src = (const T *)phi0;
        if (where == PB_HOST) {
            PB_TRY(ensure_stage(h, n * sizeof(T)));
            PB_CUDA(cudaMemcpyAsync(h->stage, phi0, n * sizeof(T), cudaMemcpyHostToDevice, h->stream));
            src = (const T *)h->stage;
        }
        k_pad<T, T><<<grid_for(w.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(src, w.tmp, h->nx, w.P, rows);
        launch_spmv<T, 1>(h, w, 1.0);                      // Ap = A' phi_0
        launch_wrap<T, 1>(h, w, 1.0);
        k_warm<T><<<w.vec_grid, 256, 0, h->stream>>>(vec_args<T>(h, w), w.tmp);
        PB_CUDA(cudaGetLastError());
        h->launches += 3;
    }
    return PB_OK;
}

template <typename T>
pb_status get_graph(pb_handle *h, Work<T> &w, int m)
{
    if (w.graph && w.graph_iters == m) return PB_OK;
    if (w.graph) { cudaGraphExecDestroy(w.graph); w.graph = nullptr; }
    cudaGraph_t g = nullptr;
    PB_CUDA(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
    pb_status s = enqueue_iterations<T>(h, w, m);
    h->launches -= (2LL + (h->periodic ? 1 : 0)) * m;          // captured, not executed
    cudaError_t e = cudaStreamEndCapture(h->stream, &g);
    if (s != PB_OK || e != cudaSuccess || !g) { cudaGetLastError(); return PB_ERR_CUDA; }
    e = cudaGraphInstantiate(&w.graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { w.graph = nullptr; cudaGetLastError(); return PB_ERR_CUDA; }
    w.graph_iters = m;
    return PB_OK;
}

pb_status ensure_stage(pb_handle *h, size_t bytes)
{
    if (bytes <= h->stage_bytes) return PB_OK;
    if (h->stage) PB_ALLOC(cudaFree(h->stage));
    h->stage = nullptr;
    h->stage_bytes = 0;
    PB_ALLOC(cudaMalloc(&h->stage, bytes));
    h->stage_bytes = bytes;
    return PB_OK;
}

// pb_solve takes the one-kernel-per-iteration path unless the problem needs a special one
template <typename T>
bool fused_eligible(pb_handle *h)
{
    if (!h->opt[PB_OPT_FUSED] || h->periodic || h->slab) return false;
    if (ensure<T>(h) != PB_OK) return false;
    return !work<T>(h).persist && work<T>(h).npad < ((size_t)1 << 32);   // k_pcg_fused indexes elements with 32 bits
}

struct DevTmp {                      // frees its device allocations on scope exit
    void *p[12]; int n = 0;
    ~DevTmp() { for (int i = 0; i < n; i++) if (p[i]) cudaFree(p[i]); }
    pb_status get(void **out, size_t bytes) {
        *out = nullptr;
        PB_ALLOC(cudaMalloc(out, bytes ? bytes : 8));
        p[n++] = *out;
        return PB_OK;
    }
    void release(void *q) { for (int i = 0; i < n; i++) if (p[i] == q) p[i] = nullptr; }
};

pb_status charges_to_rhs_bc(const double *d_c, const double *d_q, int n_atoms, int nx, int ny, int nz, double hh,
                            double eps_out, double kappa, double *d_rhs, double *d_bc, double *scratch, int nsm,
                            cudaStream_t st, bool dh_f32 = false);
pb_status take_copy(pb_handle *h, double **dst, const double *src, size_t n, pb_memspace where);

#include "pb_api_batch.cuh"

// pb_solve_begin: steps 1-2 without a latch, on the path pb_solve would take
template <typename T>
pb_status begin_any(pb_handle *h)
{
    h->last_fused = false;
    if (fused_eligible<T>(h)) {
        PB_TRY(ensure_batch<T>(h, 1, true));
        PB_TRY(init_batch<T>(h, 1, 1.0, 0, 0, work<T>(h).b));
        h->last_fused = true;
        return PB_OK;
    }
    return begin_solve<T>(h, 1.0, 0, 0);
}

// steps 1-8 until the device latch is set (converged, maxiter or breakdown); the iterate stays on the device
template <typename T>
pb_status run_solve(pb_handle *h, double tol, int maxiter, int check_every, const void *phi0, pb_memspace where,
                    bool allow_fused = true)
{
    h->last_fused = false;
    if (allow_fused && fused_eligible<T>(h)) {
        // one kernel per iteration (k_pcg_fused) on the batch work set, right-hand side = this handle's b
        Work<T> &wq = work<T>(h);
        PB_TRY(ensure_batch<T>(h, 1, true));
        PB_TRY(run_batch<T>(h, 1, tol, maxiter, check_every, wq.b, phi0, where));
        h->last_fused = true;
        return PB_OK;
    }
    PB_TRY(begin_solve<T>(h, tol, maxiter, 1, phi0, where));
    Work<T> &w = work<T>(h);
    const int m = check_every;
    if (w.persist) {
        // L2-resident grid: steps 3-8 in one cooperative kernel, exit decided on the device
        PersistArgs<T> pa;
        pa.x = w.x; pa.r = w.r; pa.p0 = w.p0; pa.p1 = w.p1; pa.Ap = w.Ap;
        pa.Dinv = w.Dinv; pa.exm = w.exm; pa.eym = w.eym; pa.ezm = w.ezm;
        pa.nx = h->nx; pa.ny = h->ny; pa.nz = h->nz; pa.P = w.P; pa.precond = h->precond; pa.periodic = h->periodic;
        pa.st = h->st; pa.partials = h->partials;
        void *kargs[] = {(void *)&pa};
        const void *fn = w.pfused ? (const void *)k_pcg_persistent<T, true> : (const void *)k_pcg_persistent<T, false>;
        if (cudaLaunchCooperativeKernel(fn, dim3(w.pgrid), dim3(256), kargs, 0, h->stream) == cudaSuccess) {
            h->launches += 1;
        } else {
            // e.g. fewer SMs available than the occupancy query promised (MPS / MIG): fall back for good
            cudaGetLastError();
            if (verbose()) fprintf(stderr, "pb: cooperative launch refused, using the two-kernel path\n");
            w.persist = false;
        }
    }
    bool graph_ok = !w.persist && h->opt[PB_OPT_GRAPH] && get_graph<T>(h, w, m) == PB_OK;
    // chunk c is enqueued before the latch of chunk c-1 is waited for, so the device never idles
    const long max_chunks = (long)maxiter / m + 2;
    int seen_done = w.persist ? 1 : 0;
    for (long c = 0; c < max_chunks + 1 && !seen_done; c++) {
        if (graph_ok) { PB_CUDA(cudaGraphLaunch(w.graph, h->stream)); h->launches += (2LL + (h->periodic ? 1 : 0)) * m; }
        else PB_TRY(enqueue_iterations<T>(h, w, m));
        int *slot = h->pinned + 4 * (c & 1);
        PB_CUDA(cudaMemcpyAsync(slot, &h->st->done, 4 * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaEventRecord(h->ev[c & 1], h->stream));
        if (c >= 1) {
            PB_CUDA(cudaEventSynchronize(h->ev[(c - 1) & 1]));
            seen_done = h->pinned[4 * ((c - 1) & 1)];
        }
    }
    return PB_OK;
}

template <typename T>
pb_status solve_impl(pb_handle *h, double tol, int maxiter, int check_every, void *phi_out,
                     pb_memspace where, int *iters_out, double *relres_out, const void *phi0 = nullptr)
{
    PB_TRY(run_solve<T>(h, tol, maxiter, check_every, phi0, where));
    Work<T> &w = work<T>(h);
    // a6: un-pad x -> phi_out, read the final scalars
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    T *dst = (T *)phi_out;
    if (where == PB_HOST) { PB_TRY(ensure_stage(h, n * sizeof(T))); dst = (T *)h->stage; }
    if (h->last_fused)
        k_finish<T, T><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(w.bw.x, w.bw.p0, w.bw.p1, h->st, dst, h->nx, w.P, rows,
                                                                             w.bw.x2);
    else
        k_finish<T, T><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(w.x, w.p0, w.p1, h->st, dst, h->nx, w.P, rows);
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    if (where == PB_HOST)
        PB_CUDA(cudaMemcpyAsync(phi_out, dst, n * sizeof(T), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    const State &st = *h->pinned_state;
    if (!st.done) return PB_ERR_CUDA;   // cannot happen: maxiter latches
    if (iters_out) *iters_out = st.iters;
    if (relres_out) *relres_out = (st.bb > 0.0) ? sqrt(st.rr / st.bb) : 0.0;
    return (pb_status)st.status;
}

// Mixed-precision iterative refinement: the potential and the true residual r = b - A phi live in
// fp64 (k_spmv_tma<double, MODE 1> + k_true_residual); each correction A d = r is a Jacobi-PCG solve in fp32 (the
// same kernels as pb_solve) to `inner_tol` relative to ||r||; phi += d in fp64.  The result meets
// the fp64 tolerance on the TRUE residual at close to the fp32 iteration rate.
pb_status refined_impl(pb_handle *h, double tol, int maxiter, double inner_tol, int check_every, double *phi_out,
                       pb_memspace where, int *outer_out, int *iters_out, double *relres_out)
{
    PB_TRY(ensure<double>(h));
    PB_TRY(ensure<float>(h));
    Work<double> &wd = h->wd;
    Work<float> &wf = h->wf;
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    const size_t nvec_d = wd.npad / VecN<double>::value;
    // phi (padded fp64) is kept in wd.tmp, the input tensor of the MODE 1 SpMV
    PB_CUDA(cudaMemsetAsync(wd.tmp, 0, wd.npad * sizeof(double), h->stream));
    int total = 0, outer = 0;
    double relres = 1.0;
    pb_status status = PB_ERR_MAXITER;
    for (;; outer++) {
        launch_spmv<double, 1>(h, wd, 1.0);
        launch_wrap<double, 1>(h, wd, 1.0);
        k_set_state<<<1, 1, 0, h->stream>>>(h->st, 1.0, 0, 0);
        k_true_residual<double><<<grid_for(nvec_d, 256, h->nsm * 4), 256, 0, h->stream>>>(wd.b, wd.Ap, nvec_d, h->st,
                                                                                          h->partials, wd.r);
        PB_CUDA(cudaGetLastError());
        h->launches += 3;
        PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaStreamSynchronize(h->stream));
        const double rr = h->pinned_state->rr, bb = h->pinned_state->bb;
        relres = bb > 0.0 ? sqrt(rr / bb) : 0.0;
        if (!(relres == relres)) { status = PB_ERR_BREAKDOWN; break; }
        if (relres <= tol) { status = PB_OK; break; }
        if (total >= maxiter || outer >= 40) break;
        // correction solve in fp32 on the right-hand side r; the last one only has to close the remaining gap
        double tin = 0.3 * tol / relres;
        if (tin < inner_tol) tin = inner_tol;
        if (tin > 0.1) tin = 0.1;
        k_repad<double, float><<<grid_for(wf.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(wd.r, wd.P, wf.b, wf.P,
                                                                                           h->nx, rows);
        h->launches += 1;
        wf.b_ready = true;
        const pb_status rs = run_solve<float>(h, tin, maxiter - total, check_every, nullptr, PB_DEVICE);
        wf.b_ready = false;                      // wf.b holds a residual, not b: rebuilt before the next plain solve
        if (rs != PB_OK) return rs;
        if (h->last_fused)                       // the correction went through k_pcg_fused (its own vectors)
            k_finish_add<float, double><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(
                wf.bw.x, wf.bw.p0, wf.bw.p1, h->st, wd.tmp, h->nx, wf.P, wd.P, rows, wf.bw.x2);
        else
            k_finish_add<float, double><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(
                wf.x, wf.p0, wf.p1, h->st, wd.tmp, h->nx, wf.P, wd.P, rows);
        PB_CUDA(cudaGetLastError());
        h->launches += 1;
        PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaStreamSynchronize(h->stream));
        total += h->pinned_state->iters;
        if (h->pinned_state->status == (int)PB_ERR_BREAKDOWN) { status = PB_ERR_BREAKDOWN; break; }
    }
    h->last_prec = PB_F64;
    double *dst = phi_out;
    if (where == PB_HOST) { PB_TRY(ensure_stage(h, n * sizeof(double))); dst = (double *)h->stage; }
    k_unpad<double, double><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(wd.tmp, dst, h->nx, wd.P, rows, 1.0);
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    if (where == PB_HOST)
        PB_CUDA(cudaMemcpyAsync(phi_out, dst, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    if (outer_out) *outer_out = outer;
    if (iters_out) *iters_out = total;
    if (relres_out) *relres_out = relres;
    return status;
}


// ---- NEXT row f4: one solve over several GPUs, z-slab decomposition -------------------------
// The library provides the per-rank pieces; the ranks' exchange (halo planes, scalar all-reduces) is the caller's --
// torch.distributed / NCCL in paper_1704_02745_b200/slab.py.
template <typename T>
pb_status slab_begin(pb_handle *h, double tol, int maxiter)
{
    PB_TRY(ensure<T>(h));
    Work<T> &w = work<T>(h);
    const size_t plane = (size_t)h->ny * w.P;
    if (h->slab_prec != (int)(sizeof(T) == 4 ? PB_F32 : PB_F64) || !h->slab_send) {
        if (h->slab_send) { cudaFree(h->slab_send); h->slab_send = nullptr; }
        if (h->slab_recv) { cudaFree(h->slab_recv); h->slab_recv = nullptr; }
        PB_ALLOC(cudaMalloc(&h->slab_send, 4 * plane * sizeof(T)));
        PB_ALLOC(cudaMalloc(&h->slab_recv, 4 * plane * sizeof(T)));
        PB_CUDA(cudaMemsetAsync(h->slab_recv, 0, 4 * plane * sizeof(T), h->stream));
        h->slab_plane_bytes = plane * sizeof(T);
        h->slab_prec = sizeof(T) == 4 ? PB_F32 : PB_F64;
    }
    h->last_prec = sizeof(T) == 4 ? PB_F32 : PB_F64;
    // ghost planes of both p buffers start at 0 (p_0 = z_0: beta = 0 multiplies them, they must be finite)
    PB_CUDA(cudaMemsetAsync(w.p0 - w.goff, 0, (w.npad + 2 * w.goff) * sizeof(T), h->stream));
    PB_CUDA(cudaMemsetAsync(w.p1 - w.goff, 0, (w.npad + 2 * w.goff) * sizeof(T), h->stream));
    k_set_state<<<1, 1, 0, h->stream>>>(h->st, tol * tol, maxiter, 1, 1);
    k_init<T><<<w.vec_grid, 256, 0, h->stream>>>(vec_args<T>(h, w));       // local r.z, r.r -> State::loc_*
    PB_CUDA(cudaGetLastError());
    h->launches += 2;
    return PB_OK;
}

template <typename T>
pb_status slab_pack(pb_handle *h, bool unpack)
{
    Work<T> &w = work<T>(h);
    if (!w.ready || !h->slab_send) return PB_ERR_INVALID_ARG;
    const size_t plane = (size_t)h->ny * w.P;
    const int g = grid_for(plane, 256, h->nsm * 4);
    if (unpack) k_slab_unpack<T><<<g, 256, 0, h->stream>>>(w.r, w.p0, w.p1, h->st, (const T *)h->slab_recv, plane, h->nz,
                                                          h->iface_lo, h->iface_hi);
    else k_slab_pack<T><<<g, 256, 0, h->stream>>>(w.r, w.p0, w.p1, h->st, (T *)h->slab_send, plane, h->nz);
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    return PB_OK;
}

template <typename T>
pb_status slab_step(pb_handle *h, int which)
{
    Work<T> &w = work<T>(h);
    if (!w.ready) return PB_ERR_INVALID_ARG;
    if (which == 0) {
        launch_spmv<T, 0>(h, w, 1.0);                                        // local p.Ap -> State::pAp
    } else {
        k_slab_alpha<<<1, 1, 0, h->stream>>>(h->st);                        // pAp is global now
        const VecArgs<T> va = vec_args<T>(h, w);
        if (w.pald) k_vec<T, true><<<w.vec_grid, 256, 0, h->stream>>>(va);  // local r.z, r.r -> State::loc_*
        else k_vec<T, false><<<w.vec_grid, 256, 0, h->stream>>>(va);
        h->launches += 1;
    }
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    return PB_OK;
}

template <typename T>
pb_status apply_impl(pb_handle *h, const void *x, void *y, pb_memspace where)
{
    PB_TRY(ensure<T>(h));
    Work<T> &w = work<T>(h);
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    const T *src = (const T *)x;
    T *dst = (T *)y;
    if (where == PB_HOST) {
        PB_TRY(ensure_stage(h, n * sizeof(T)));
        PB_CUDA(cudaMemcpyAsync(h->stage, x, n * sizeof(T), cudaMemcpyHostToDevice, h->stream));
        src = (const T *)h->stage;
        dst = (T *)h->stage;
    }
    const int g = grid_for(w.npad, 256, h->nsm * 16);
    k_pad<T, T><<<g, 256, 0, h->stream>>>(src, w.tmp, h->nx, w.P, rows);
    launch_spmv<T, 1>(h, w, 1.0 / (h->h * h->h));
    launch_wrap<T, 1>(h, w, 1.0 / (h->h * h->h));
    k_unpad<T, T><<<g, 256, 0, h->stream>>>(w.Ap, dst, h->nx, w.P, rows, 1.0);
    PB_CUDA(cudaGetLastError());
    h->launches += 3;
    if (where == PB_HOST)
        PB_CUDA(cudaMemcpyAsync(y, dst, n * sizeof(T), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    return PB_OK;
}

template <typename T>
int bytes_per_node_impl(pb_handle *h, int kernel)
{
    if (ensure<T>(h) != PB_OK) return -1;
    Work<T> &w = work<T>(h);
    const int e = (int)sizeof(T);
    if (fused_eligible<T>(h)) {
        // k_pcg_fused: r, A p, p, x in; r, p, x, A p out (8 words); Dinv; the three faces (quad: ex twice, 4 x 2 bits)
        if (kernel == 1) return 0;
        if (ensure_batch<T>(h, 1, true) != PB_OK) return -1;
        const BatchWork<T> &b = w.bw;
        return 8 * e + (b.pald ? 1 : e) + (b.quad ? 1 : 3 * e);
    }
    if (kernel == 0)      // r, p_old, x in; p, x, Ap out; Dinv; three face coefficients
        return 6 * e + (w.pald_s ? 1 : e) + (w.pal ? 3 : 3 * e);
    return 3 * e + (w.pald ? 1 : e);      // r, Ap in; r out; Dinv
}

// true residual ||b - A phi|| / ||b|| of a caller-supplied potential, in the arithmetic of precision T
template <typename T>
pb_status residual_impl(pb_handle *h, const void *phi, pb_memspace where, double *relres_out)
{
    PB_TRY(ensure<T>(h));
    Work<T> &w = work<T>(h);
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    const T *src = (const T *)phi;
    if (where == PB_HOST) {
        PB_TRY(ensure_stage(h, n * sizeof(T)));
        PB_CUDA(cudaMemcpyAsync(h->stage, phi, n * sizeof(T), cudaMemcpyHostToDevice, h->stream));
        src = (const T *)h->stage;
    }
    k_pad<T, T><<<grid_for(w.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(src, w.tmp, h->nx, w.P, rows);
    launch_spmv<T, 1>(h, w, 1.0);
    launch_wrap<T, 1>(h, w, 1.0);
    k_set_state<<<1, 1, 0, h->stream>>>(h->st, 1.0, 0, 0);
    k_true_residual<T><<<grid_for(w.npad / VecN<T>::value, 256, h->nsm * 4), 256, 0, h->stream>>>(
        w.b, w.Ap, w.npad / VecN<T>::value, h->st, h->partials);
    PB_CUDA(cudaGetLastError());
    h->launches += 4;
    PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    const State &st = *h->pinned_state;
    *relres_out = (st.bb > 0.0) ? sqrt(st.rr / st.bb) : 0.0;
    return PB_OK;
}

// copy a caller array (host or device) into a fresh/existing device array of n doubles
pb_status take_copy(pb_handle *h, double **dst, const double *src, size_t n, pb_memspace where)
{
    if (!src) {
        if (*dst) cudaFree(*dst);
        *dst = nullptr;
        return PB_OK;
    }
    if (!*dst) PB_ALLOC(cudaMalloc((void **)dst, (n + 8) * sizeof(double)));
    PB_CUDA(cudaMemcpyAsync(*dst, src, n * sizeof(double),
                            where == PB_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, h->stream));
    return PB_OK;
}

bool valid_space(pb_memspace w) { return w == PB_HOST || w == PB_DEVICE; }
bool valid_prec(pb_precision p) { return p == PB_F32 || p == PB_F64; }

}  // namespace

namespace {
template <typename T>
pb_status profile_impl(pb_handle *h, int n_iter, double *ms_spmv, double *ms_vec)
{
    Work<T> &w = work<T>(h);
    if (!w.ready) return PB_ERR_INVALID_ARG;
    const int ne = 2 * n_iter + 1;
    cudaEvent_t *ev = (cudaEvent_t *)calloc(ne, sizeof(cudaEvent_t));
    if (!ev) return PB_ERR_ALLOC;
    pb_status s = PB_OK;
    auto body = [&]() -> pb_status {
        for (int i = 0; i < ne; i++) PB_CUDA(cudaEventCreate(&ev[i]));
        const VecArgs<T> va = vec_args<T>(h, w);
        PB_CUDA(cudaEventRecord(ev[0], h->stream));
        if (h->last_fused) {
            // one kernel per iteration: its time is reported as "spmv", "vec" is 0
            for (int it = 0; it < n_iter; it++) {
                PB_TRY(enqueue_batch_iterations<T>(h, w, 1));
                PB_CUDA(cudaEventRecord(ev[it + 1], h->stream));
            }
            PB_CUDA(cudaStreamSynchronize(h->stream));
            double a = 0.0;
            for (int it = 0; it < n_iter; it++) {
                float t1 = 0.f;
                PB_CUDA(cudaEventElapsedTime(&t1, ev[it], ev[it + 1]));
                a += t1;
            }
            if (ms_spmv) *ms_spmv = a / n_iter;
            if (ms_vec) *ms_vec = 0.0;
            return PB_OK;
        }
        for (int it = 0; it < n_iter; it++) {
            launch_spmv<T, 0>(h, w, 1.0);
            launch_wrap<T, 0>(h, w, 1.0);
            PB_CUDA(cudaEventRecord(ev[2 * it + 1], h->stream));
            if (w.pald) k_vec<T, true><<<w.vec_grid, 256, 0, h->stream>>>(va);
            else k_vec<T, false><<<w.vec_grid, 256, 0, h->stream>>>(va);
            PB_CUDA(cudaEventRecord(ev[2 * it + 2], h->stream));
        }
        PB_CUDA(cudaGetLastError());
        h->launches += 2LL * n_iter;
        PB_CUDA(cudaStreamSynchronize(h->stream));
        double a = 0.0, b = 0.0;
        for (int it = 0; it < n_iter; it++) {
            float t1 = 0.f, t2 = 0.f;
            PB_CUDA(cudaEventElapsedTime(&t1, ev[2 * it], ev[2 * it + 1]));
            PB_CUDA(cudaEventElapsedTime(&t2, ev[2 * it + 1], ev[2 * it + 2]));
            a += t1; b += t2;
        }
        if (ms_spmv) *ms_spmv = a / n_iter;
        if (ms_vec) *ms_vec = b / n_iter;
        return PB_OK;
    };
    s = body();
    for (int i = 0; i < ne; i++) if (ev[i]) cudaEventDestroy(ev[i]);
    free(ev);
    return s;
}
}  // namespace

extern "C" {

pb_status pb_destroy(pb_handle *h)
{
    if (!h) return PB_OK;
    cudaSetDevice(h->device);
    if (h->stream) cudaStreamSynchronize(h->stream);
    free_work(h->wf);
    free_work(h->wd);
    double **ins[] = {&h->eps_x, &h->eps_y, &h->eps_z, &h->kbar2, &h->rhs, &h->bc};
    for (double **a : ins) if (*a) cudaFree(*a);
    if (h->st) cudaFree(h->st);
    if (h->partials) cudaFree(h->partials);
    if (h->bad) cudaFree(h->bad);
    if (h->stage) cudaFree(h->stage);
    if (h->slab_send) cudaFree(h->slab_send);
    if (h->slab_recv) cudaFree(h->slab_recv);
    if (h->atoms_c) cudaFree(h->atoms_c);
    if (h->atoms_q) cudaFree(h->atoms_q);
    if (h->pal_table) cudaFree(h->pal_table);
    if (h->pald_table) cudaFree(h->pald_table);
    if (h->pinned) cudaFreeHost(h->pinned);
    if (h->pinned_state) cudaFreeHost(h->pinned_state);
    for (int i = 0; i < 2; i++) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
    cudaGetLastError();
    delete h;
    return PB_OK;
}

pb_status pb_create(pb_handle **out, int nx, int ny, int nz, double hh,
                    const double *eps_x, const double *eps_y, const double *eps_z,
                    const double *kbar2, const double *rhs, const double *bc,
                    pb_memspace where, void *cuda_stream)
{
    if (!out) return PB_ERR_INVALID_ARG;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1 || !(hh > 0.0) || !std::isfinite(hh) || !eps_x || !eps_y || !eps_z ||
        !valid_space(where))
        return PB_ERR_INVALID_ARG;
    if ((double)nx * ny * nz > 2.0e9) return PB_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return PB_ERR_CUDA; }
    pb_handle *h = new (std::nothrow) pb_handle();
    if (!h) return PB_ERR_ALLOC;
    h->nx = nx; h->ny = ny; h->nz = nz; h->h = hh;
    default_options(h->opt);
    h->precond = 1;
    h->pal_n = -1;
    h->pald_n = -1;
    pb_status s = PB_OK;
    auto body = [&]() -> pb_status {
        PB_CUDA(cudaGetDevice(&h->device));
        PB_CUDA(cudaDeviceGetAttribute(&h->nsm, cudaDevAttrMultiProcessorCount, h->device));
        if (h->nsm < 1) return PB_ERR_CUDA;
        if (cuda_stream) { h->stream = (cudaStream_t)cuda_stream; h->own_stream = false; }
        else { PB_CUDA(cudaStreamCreate(&h->stream)); h->own_stream = true; }   // blocking: orders with stream 0
        PB_ALLOC(cudaMalloc((void **)&h->st, kMaxBatch * sizeof(State)));      // st[0]: pb_solve; st[0..M): pb_solve_batch
        PB_CUDA(cudaMemsetAsync(h->st, 0, kMaxBatch * sizeof(State), h->stream));
        PB_ALLOC(cudaMalloc((void **)&h->bad, sizeof(int)));
        PB_ALLOC(cudaHostAlloc((void **)&h->pinned, 8 * sizeof(int), cudaHostAllocDefault));
        PB_ALLOC(cudaHostAlloc((void **)&h->pinned_state, 2 * kMaxBatch * sizeof(State), cudaHostAllocDefault));
        PB_CUDA(cudaEventCreateWithFlags(&h->ev[0], cudaEventDisableTiming));
        PB_CUDA(cudaEventCreateWithFlags(&h->ev[1], cudaEventDisableTiming));
        const size_t n = (size_t)nx * ny * nz;
        PB_TRY(take_copy(h, &h->eps_x, eps_x, (size_t)nz * ny * (nx + 1), where));
        PB_TRY(take_copy(h, &h->eps_y, eps_y, (size_t)nz * (ny + 1) * nx, where));
        PB_TRY(take_copy(h, &h->eps_z, eps_z, (size_t)(nz + 1) * ny * nx, where));
        PB_TRY(take_copy(h, &h->kbar2, kbar2, n, where));
        PB_TRY(take_copy(h, &h->rhs, rhs, n, where));
        PB_TRY(take_copy(h, &h->bc, bc, 2 * ((size_t)nz * ny + (size_t)nz * nx + (size_t)ny * nx), where));
        // SPD check on the diagonal alone; the padded work arrays of a precision and its launch
        // plan are built on first use (or by pb_prepare), so an fp32-only caller never pays for the fp64 set
        PB_CUDA(cudaMemsetAsync(h->bad, 0, sizeof(int), h->stream));
        k_check_diag<<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(h->eps_x, h->eps_y, h->eps_z, h->kbar2,
                                                                        hh * hh, nx, ny, nz, h->bad);
        PB_CUDA(cudaGetLastError());
        h->launches += 1;
        int bad = 0;
        PB_CUDA(cudaMemcpyAsync(&bad, h->bad, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaStreamSynchronize(h->stream));
        if (bad) return PB_ERR_NOT_SPD;
        return PB_OK;
    };
    s = body();
    if (s != PB_OK) { pb_destroy(h); return s; }
    *out = h;
    return PB_OK;
}

pb_status pb_set_rhs(pb_handle *h, const double *rhs, const double *bc, pb_memspace where)
{
    if (!h || !valid_space(where)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    const size_t n = (size_t)h->nx * h->ny * h->nz;
    PB_TRY(take_copy(h, &h->rhs, rhs, n, where));
    PB_TRY(take_copy(h, &h->bc, bc, 2 * ((size_t)h->nz * h->ny + (size_t)h->nz * h->nx + (size_t)h->ny * h->nx), where));
    h->wf.b_ready = false;
    h->wd.b_ready = false;
    if (h->wf.ready) PB_TRY(build_b<float>(h, h->wf));
    if (h->wd.ready) PB_TRY(build_b<double>(h, h->wd));
    PB_CUDA(cudaStreamSynchronize(h->stream));   // the inputs are copied: the caller may free or overwrite them on return
    return PB_OK;
}

pb_status pb_create_slab(pb_handle **out, int nx, int ny, int nz, double hh,
                         const double *eps_x, const double *eps_y, const double *eps_z,
                         const double *kbar2, const double *rhs, const double *bc,
                         pb_memspace where, void *cuda_stream, int neighbour_below, int neighbour_above)
{
    PB_TRY(pb_create(out, nx, ny, nz, hh, eps_x, eps_y, eps_z, kbar2, rhs, bc, where, cuda_stream));
    (*out)->slab = true;
    (*out)->iface_lo = neighbour_below ? 1 : 0;
    (*out)->iface_hi = neighbour_above ? 1 : 0;
    return PB_OK;
}

pb_status pb_slab_begin(pb_handle *h, pb_precision prec, double tol, int maxiter)
{
    if (!h || !h->slab || !valid_prec(prec) || !(tol > 0.0) || maxiter < 0 || h->periodic) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? slab_begin<float>(h, tol, maxiter) : slab_begin<double>(h, tol, maxiter);
}

pb_status pb_slab_step(pb_handle *h, int which)
{
    if (!h || !h->slab || h->slab_prec < 0 || which < 0 || which > 5) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    const bool f32 = h->slab_prec == PB_F32;
    switch (which) {
    case 0: case 1: return f32 ? slab_step<float>(h, which) : slab_step<double>(h, which);
    case 2: case 3:
        k_slab_finish<<<1, 1, 0, h->stream>>>(h->st, which == 3 ? 1 : 0);
        PB_CUDA(cudaGetLastError());
        h->launches += 1;
        return PB_OK;
    case 4: return f32 ? slab_pack<float>(h, false) : slab_pack<double>(h, false);
    default: return f32 ? slab_pack<float>(h, true) : slab_pack<double>(h, true);
    }
}

pb_status pb_slab_pointers(pb_handle *h, void **ptrs, size_t *plane_bytes)
{
    if (!h || !h->slab || h->slab_prec < 0 || !ptrs || !plane_bytes) return PB_ERR_INVALID_ARG;
    const size_t pb_ = h->slab_plane_bytes;
    char *dinv = h->slab_prec == PB_F32 ? (char *)h->wf.Dinv : (char *)h->wd.Dinv;
    ptrs[0] = h->slab_send;                                  // [r_lo | p_lo | r_hi | p_hi], 4 planes
    ptrs[1] = h->slab_recv;                                  // [r_below | p_below | r_above | p_above]
    ptrs[2] = &h->st->pAp;                                   // 1 double: local p.Ap, all-reduced in place
    ptrs[3] = &h->st->loc_rz;                                // 2 doubles: local r.z, r.r, all-reduced in place
    ptrs[4] = dinv;                                          // Dinv plane 0        (to the rank below, once)
    ptrs[5] = dinv + (size_t)(h->nz - 1) * pb_;              // Dinv plane nz-1     (to the rank above, once)
    ptrs[6] = dinv - pb_;                                    // Dinv ghost plane -1 (from the rank below)
    ptrs[7] = dinv + (size_t)h->nz * pb_;                    // Dinv ghost plane nz (from the rank above)
    *plane_bytes = pb_;
    return PB_OK;
}

pb_status pb_slab_latch(pb_handle *h, int *done, int *iters, int *status, double *relres)
{
    if (!h || !h->slab) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    const State &st = *h->pinned_state;
    if (done) *done = st.done;
    if (iters) *iters = st.done ? st.iters : st.iter_cur;
    if (status) *status = st.status;
    if (relres) *relres = (st.bb > 0.0) ? sqrt(st.rr / st.bb) : 0.0;
    return PB_OK;
}

pb_status pb_slab_result(pb_handle *h, void *phi_out, pb_memspace where)
{
    if (!h || !h->slab || h->slab_prec < 0 || !phi_out || !valid_space(where)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    const size_t esz = h->slab_prec == PB_F32 ? 4 : 8;
    void *dst = phi_out;
    if (where == PB_HOST) { PB_TRY(ensure_stage(h, n * esz)); dst = h->stage; }
    const int g = grid_for(n, 256, h->nsm * 16);
    if (h->slab_prec == PB_F32)
        k_finish<float, float><<<g, 256, 0, h->stream>>>(h->wf.x, h->wf.p0, h->wf.p1, h->st, (float *)dst, h->nx, h->wf.P, rows);
    else
        k_finish<double, double><<<g, 256, 0, h->stream>>>(h->wd.x, h->wd.p0, h->wd.p1, h->st, (double *)dst, h->nx, h->wd.P, rows);
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    if (where == PB_HOST) PB_CUDA(cudaMemcpyAsync(phi_out, dst, n * esz, cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    return PB_OK;
}

pb_status pb_set_option(pb_handle *h, pb_option opt, int value)
{
    if (!h || (int)opt < 0 || (int)opt >= (int)PB_OPT_COUNT_ || value < 0) return PB_ERR_INVALID_ARG;
    switch (opt) {
    case PB_OPT_PERSIST: case PB_OPT_PALETTE: case PB_OPT_PALETTE_DIAG: case PB_OPT_PALETTE_DIAG_SPMV:
    case PB_OPT_AUTOTUNE: case PB_OPT_GRAPH: case PB_OPT_FUSED:
        if (value > 1) return PB_ERR_INVALID_ARG;
        break;
    case PB_OPT_PERSIST_BLOCKS_PER_SM:
        if (value < 1 || value > 32) return PB_ERR_INVALID_ARG;
        break;
    case PB_OPT_RING_SLOTS:
        if (value != 0 && (value < 3 || value > kMaxStages)) return PB_ERR_INVALID_ARG;
        break;
    case PB_OPT_BATCH_WIDTH:
        if (value != 1 && value != 2 && value != 4) return PB_ERR_INVALID_ARG;
        break;
    case PB_OPT_TAIL_POOL:
        if (value != 0 && value != 1 && (value < 4 || value > 64)) return PB_ERR_INVALID_ARG;
        break;
    case PB_OPT_BLOCKS_PER_SM: case PB_OPT_VEC_BLOCKS_PER_SM:
        if (value > 32) return PB_ERR_INVALID_ARG;
        break;
    default: break;
    }
    if (h->opt[opt] == value) return PB_OK;
    PB_CUDA(cudaSetDevice(h->device));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    h->opt[opt] = value;
    // work arrays, palettes and plans depend on the options: drop them, the next use rebuilds
    free_work(h->wf);
    free_work(h->wd);
    h->pal_n = -1;
    h->pald_n = -1;
    return PB_OK;
}

pb_status pb_get_option(pb_handle *h, pb_option opt, int *value_out)
{
    if (!h || !value_out || (int)opt < 0 || (int)opt >= (int)PB_OPT_COUNT_) return PB_ERR_INVALID_ARG;
    *value_out = h->opt[opt];
    return PB_OK;
}

pb_status pb_prepare(pb_handle *h, pb_precision prec)
{
    if (!h || !valid_prec(prec)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    PB_TRY(prec == PB_F32 ? ensure<float>(h) : ensure<double>(h));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    return PB_OK;
}

pb_status pb_get_plan(pb_handle *h, pb_precision prec, pb_plan *out)
{
    if (!h || !out || !valid_prec(prec)) return PB_ERR_INVALID_ARG;
    PB_TRY(pb_prepare(h, prec));
    memset(out, 0, sizeof(*out));
    out->precision = (int)prec;
    out->num_sm = h->nsm;
    out->palette_size = h->pal_n > 0 ? h->pal_n : 0;
    out->diag_palette_size = h->pald_n > 0 ? h->pald_n : 0;
    auto fill = [&](const auto &w) {
        out->persist = w.persist; out->persist_fused = w.persist && w.pfused; out->persist_grid = w.persist ? w.pgrid : 0;
        out->face_palette = w.pal; out->diag_palette_vec = w.pald; out->diag_palette_spmv = w.pald_s;
        out->txv = w.qTXV; out->ty = w.qTY; out->tz = w.qTZ; out->ring_slots = w.qns; out->blocks_per_sm = w.qbps;
        out->tiles = w.qntx * w.qnty * w.qntz; out->grid = w.qgrid; out->threads = w.qthreads;
        out->smem_bytes = (int)w.qsmem; out->autotuned = w.qtuned;
        out->vec_grid = w.vec_grid; out->vec_threads = 256; out->pitch = w.P;
    };
    if (prec == PB_F32) fill(h->wf); else fill(h->wd);
    out->spmv_bytes_per_node = pb_bytes_per_node(h, prec, 0);      // (builds the fused plan when pb_solve takes that path)
    auto fill_fused = [&](const auto &w) {
        const auto &b = w.bw;
        if (!(b.fused && b.M == 1)) return;
        out->fused = 1;
        out->txv = b.TXV; out->ty = b.TY; out->tz = b.TZ; out->ring_slots = b.nsv; out->blocks_per_sm = b.bps;
        out->tiles = b.ntx * b.nty * b.ntz; out->grid = b.grid; out->threads = b.threads; out->smem_bytes = (int)b.smem;
        out->autotuned = b.tuned; out->vec_grid = 0; out->vec_threads = 0;
        out->face_quad = b.quad; out->coef_slots = b.nsc; out->tail_pool = b.pc;
    };
    const bool fz = prec == PB_F32 ? fused_eligible<float>(h) : fused_eligible<double>(h);
    if (fz) { if (prec == PB_F32) fill_fused(h->wf); else fill_fused(h->wd); }
    out->vec_bytes_per_node = pb_bytes_per_node(h, prec, 1);
    return PB_OK;
}

pb_status pb_apply(pb_handle *h, pb_precision prec, const void *x, void *y, pb_memspace where)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !x || !y || x == y || !valid_prec(prec) || !valid_space(where)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? apply_impl<float>(h, x, y, where) : apply_impl<double>(h, x, y, where);
}

pb_status pb_solve(pb_handle *h, double tol, int maxiter, pb_precision prec, int check_every,
                   void *phi_out, pb_memspace where, int *iters_out, double *relres_out)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !phi_out || !(tol > 0.0) || !std::isfinite(tol) || maxiter < 0 || check_every < 1 ||
        !valid_prec(prec) || !valid_space(where))
        return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? solve_impl<float>(h, tol, maxiter, check_every, phi_out, where, iters_out, relres_out)
                          : solve_impl<double>(h, tol, maxiter, check_every, phi_out, where, iters_out, relres_out);
}

pb_status pb_solve_batch(pb_handle *h, int m, const double *rhs, const double *bc, double tol, int maxiter,
                         pb_precision prec, int check_every, void *phi_out, pb_memspace where, int *iters_out,
                         double *relres_out, int *status_out)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || m < 1 || !phi_out || !(tol > 0.0) || !std::isfinite(tol) || maxiter < 0 || check_every < 1 ||
        !valid_prec(prec) || !valid_space(where))
        return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? solve_batch_impl<float>(h, m, rhs, bc, nullptr, where, tol, maxiter, check_every, phi_out,
                                                    iters_out, relres_out, status_out)
                          : solve_batch_impl<double>(h, m, rhs, bc, nullptr, where, tol, maxiter, check_every, phi_out,
                                                     iters_out, relres_out, status_out);
}

pb_status pb_solve_batch_charges(pb_handle *h, int m, const double *charges, double tol, int maxiter,
                                 pb_precision prec, int check_every, void *phi_out, pb_memspace where, int *iters_out,
                                 double *relres_out, int *status_out)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || m < 1 || !h->atoms_c || (h->n_atoms && !charges) || !phi_out || !(tol > 0.0) || !std::isfinite(tol) ||
        maxiter < 0 || check_every < 1 || !valid_prec(prec) || !valid_space(where))
        return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? solve_batch_impl<float>(h, m, nullptr, nullptr, charges, where, tol, maxiter, check_every,
                                                    phi_out, iters_out, relres_out, status_out)
                          : solve_batch_impl<double>(h, m, nullptr, nullptr, charges, where, tol, maxiter, check_every,
                                                     phi_out, iters_out, relres_out, status_out);
}

pb_status pb_solve_from(pb_handle *h, double tol, int maxiter, pb_precision prec, int check_every,
                        const void *phi0, void *phi_out, pb_memspace where, int *iters_out, double *relres_out)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !phi_out || !(tol > 0.0) || !std::isfinite(tol) || maxiter < 0 || check_every < 1 ||
        !valid_prec(prec) || !valid_space(where))
        return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32
               ? solve_impl<float>(h, tol, maxiter, check_every, phi_out, where, iters_out, relres_out, phi0)
               : solve_impl<double>(h, tol, maxiter, check_every, phi_out, where, iters_out, relres_out, phi0);
}

pb_status pb_solve_refined(pb_handle *h, double tol, int maxiter, double inner_tol, int check_every, double *phi_out,
                           pb_memspace where, int *outer_out, int *iters_out, double *relres_out)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !phi_out || !(tol > 0.0) || !(inner_tol > 0.0) || maxiter < 0 || check_every < 1 || !valid_space(where))
        return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return refined_impl(h, tol, maxiter, inner_tol, check_every, phi_out, where, outer_out, iters_out, relres_out);
}

pb_status pb_residual(pb_handle *h, pb_precision prec, const void *phi, pb_memspace where, double *relres_out)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !phi || !relres_out || !valid_prec(prec) || !valid_space(where)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? residual_impl<float>(h, phi, where, relres_out)
                          : residual_impl<double>(h, phi, where, relres_out);
}

pb_status pb_set_preconditioner(pb_handle *h, int kind)
{
    if (!h || (kind != 0 && kind != 1)) return PB_ERR_INVALID_ARG;
    if (h->precond != kind) {
        h->precond = kind;
        // captured graphs hold the kernel arguments by value
        if (h->wf.graph) { cudaGraphExecDestroy(h->wf.graph); h->wf.graph = nullptr; }
        if (h->wd.graph) { cudaGraphExecDestroy(h->wd.graph); h->wd.graph = nullptr; }
        if (h->wf.bw.graph) { cudaGraphExecDestroy(h->wf.bw.graph); h->wf.bw.graph = nullptr; }
        if (h->wd.bw.graph) { cudaGraphExecDestroy(h->wd.bw.graph); h->wd.bw.graph = nullptr; }
    }
    return PB_OK;
}

pb_status pb_set_boundary(pb_handle *h, int kind)
{
    if (!h || (kind != 0 && kind != 1)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    if (h->periodic != kind) {
        h->periodic = kind;
        if (h->wf.graph) { cudaGraphExecDestroy(h->wf.graph); h->wf.graph = nullptr; }
        if (h->wd.graph) { cudaGraphExecDestroy(h->wd.graph); h->wd.graph = nullptr; }
        if (h->wf.bw.graph) { cudaGraphExecDestroy(h->wf.bw.graph); h->wf.bw.graph = nullptr; }
        if (h->wd.bw.graph) { cudaGraphExecDestroy(h->wd.bw.graph); h->wd.bw.graph = nullptr; }
        h->wf.b_ready = false;           // b loses / regains the ghost fold-in
        h->wd.b_ready = false;
        if (h->wf.ready) PB_TRY(build_b<float>(h, h->wf));
        if (h->wd.ready) PB_TRY(build_b<double>(h, h->wd));
    }
    return PB_OK;
}

pb_status pb_solve_begin(pb_handle *h, pb_precision prec)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !valid_prec(prec)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? begin_any<float>(h) : begin_any<double>(h);
}

pb_status pb_iterate(pb_handle *h, pb_precision prec, int n_iter)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !valid_prec(prec) || n_iter < 0) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    if (prec == PB_F32) {
        if (!h->wf.ready) return PB_ERR_INVALID_ARG;
        return h->last_fused ? enqueue_batch_iterations<float>(h, h->wf, n_iter) : enqueue_iterations<float>(h, h->wf, n_iter);
    }
    if (!h->wd.ready) return PB_ERR_INVALID_ARG;
    return h->last_fused ? enqueue_batch_iterations<double>(h, h->wd, n_iter) : enqueue_iterations<double>(h, h->wd, n_iter);
}

pb_status pb_profile(pb_handle *h, pb_precision prec, int n_iter, double *ms_spmv, double *ms_vec)
{
    if (h && h->slab) return PB_ERR_INVALID_ARG;      // a z-slab rank is driven through pb_slab_* only
    if (!h || !valid_prec(prec) || n_iter < 1) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    return prec == PB_F32 ? profile_impl<float>(h, n_iter, ms_spmv, ms_vec)
                          : profile_impl<double>(h, n_iter, ms_spmv, ms_vec);
}

long long pb_launch_count(pb_handle *h) { return h ? h->launches : 0; }

int pb_palette_size(pb_handle *h) { return (h && h->pal_n > 0) ? h->pal_n : 0; }

int pb_bytes_per_node(pb_handle *h, pb_precision prec, int kernel)
{
    if (!h || !valid_prec(prec) || kernel < 0 || kernel > 1) return -1;
    if (cudaSetDevice(h->device) != cudaSuccess) return -1;
    return prec == PB_F32 ? bytes_per_node_impl<float>(h, kernel) : bytes_per_node_impl<double>(h, kernel);
}

int pb_diag_palette_size(pb_handle *h) { return (h && h->pald_n > 0) ? h->pald_n : 0; }

pb_status pb_query(pb_handle *h, int what, double *out_host)
{
    if (!h || !out_host || what < 0 || what > 7) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    if (what == 2) {
        PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaStreamSynchronize(h->stream));
        const State &st = *h->pinned_state;
        const double v[10] = {st.rz, st.pAp, st.rr, st.bb, st.alpha, st.beta, (double)st.iter_cur,
                              (double)st.done, (double)st.status, (double)st.iters};
        memcpy(out_host, v, sizeof(v));
        return PB_OK;
    }
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    PB_TRY(ensure_stage(h, n * sizeof(double)));
    if (what >= 3) {   // work vectors of the last solve, h^2-scaled system, converted to fp64
        const int g = grid_for(n, 256, h->nsm * 16);
        if (h->last_prec == PB_F32) {
            Work<float> &w = h->wf;
            if (!w.ready) return PB_ERR_INVALID_ARG;
            const float *src[] = {w.r, w.Dinv, nullptr, w.Ap, w.x};
            const float *sp = src[what - 3];
            if (h->last_fused && what != 4) {      // k_pcg_fused: the buffers the NEXT pass reads (r is one update behind)
                PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
                PB_CUDA(cudaStreamSynchronize(h->stream));
                const int par = h->pinned_state->iter_cur & 1;
                const float *fs[] = {par ? w.bw.r2 : w.bw.r, nullptr, par ? w.bw.p1 : w.bw.p0, par ? w.bw.Ap2 : w.bw.Ap,
                                     h->pinned_state->xbuf ? w.bw.x2 : w.bw.x};
                sp = fs[what - 3];
            }
            if (!sp) { PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
                       PB_CUDA(cudaStreamSynchronize(h->stream)); sp = (h->pinned_state->iter_cur & 1) ? w.p1 : w.p0; }
            k_unpad<float, double><<<g, 256, 0, h->stream>>>(sp, (double *)h->stage, h->nx, w.P, rows, 1.0);
        } else {
            Work<double> &w = h->wd;
            if (!w.ready) return PB_ERR_INVALID_ARG;
            const double *src[] = {w.r, w.Dinv, nullptr, w.Ap, w.x};
            const double *sp = src[what - 3];
            if (h->last_fused && what != 4) {
                PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
                PB_CUDA(cudaStreamSynchronize(h->stream));
                const int par = h->pinned_state->iter_cur & 1;
                const double *fs[] = {par ? w.bw.r2 : w.bw.r, nullptr, par ? w.bw.p1 : w.bw.p0, par ? w.bw.Ap2 : w.bw.Ap,
                                     h->pinned_state->xbuf ? w.bw.x2 : w.bw.x};
                sp = fs[what - 3];
            }
            if (!sp) { PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, sizeof(State), cudaMemcpyDeviceToHost, h->stream));
                       PB_CUDA(cudaStreamSynchronize(h->stream)); sp = (h->pinned_state->iter_cur & 1) ? w.p1 : w.p0; }
            k_unpad<double, double><<<g, 256, 0, h->stream>>>(sp, (double *)h->stage, h->nx, w.P, rows, 1.0);
        }
        PB_CUDA(cudaGetLastError());
        PB_CUDA(cudaMemcpyAsync(out_host, h->stage, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaStreamSynchronize(h->stream));
        return PB_OK;
    }
    PB_TRY(ensure<double>(h));
    Work<double> &w = h->wd;
    k_unpad<double, double><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(
        what == 0 ? w.D : w.b, (double *)h->stage, h->nx, w.P, rows, 1.0 / (h->h * h->h));
    PB_CUDA(cudaGetLastError());
    PB_CUDA(cudaMemcpyAsync(out_host, h->stage, n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    return PB_OK;
}

const char *pb_strerror(pb_status s)
{
    switch (s) {
    case PB_OK: return "ok";
    case PB_ERR_INVALID_ARG: return "invalid argument";
    case PB_ERR_ALLOC: return "out of memory";
    case PB_ERR_CUDA: return "CUDA error or no CUDA device (this library has no CPU fallback)";
    case PB_ERR_NOT_SPD: return "operator not symmetric positive definite (non-positive or non-finite diagonal)";
    case PB_ERR_BREAKDOWN: return "PCG breakdown (p.Ap <= 0 or non-finite value)";
    case PB_ERR_MAXITER: return "maximum number of iterations reached before convergence";
    case PB_ERR_TOO_LARGE: return "grid larger than the fixed scratch of pb_residual_noalloc (nz * ny > PB_NOALLOC_MAX_ROWS)";
    }
    return "unknown status";
}

int pb_version(void) { return 100; }

}  // extern "C"

// ---- NEXT row f1: grid / stencil setup on the GPU ---------------------------------------------------------
namespace {

// rhs (dense [nz][ny][nx]) and bc from charges on the stored / given atom geometry.  `scratch` = one double
// (sum |q|) followed by one int (the bad-atom flag), device.
pb_status charges_to_rhs_bc(const double *d_c, const double *d_q, int n_atoms, int nx, int ny, int nz, double hh,
                            double eps_out, double kappa, double *d_rhs, double *d_bc, double *scratch, int nsm,
                            cudaStream_t st, bool dh_f32)
{
    const size_t n = (size_t)nx * ny * nz;
    const size_t nbc = 2 * ((size_t)nz * ny + (size_t)nz * nx + (size_t)ny * nx);
    int *d_bad = reinterpret_cast<int *>(scratch + 1);
    PB_CUDA(cudaMemsetAsync(scratch, 0, 2 * sizeof(double), st));
    PB_CUDA(cudaMemsetAsync(d_rhs, 0, n * sizeof(double), st));
    k_grid_check<<<1, 1024, 0, st>>>(d_c, d_q, n_atoms, nx, ny, nz, hh, scratch, d_bad);
    k_grid_spread<<<grid_for((size_t)n_atoms, 128, nsm * 8), 128, 0, st>>>(d_c, d_q, n_atoms, nx, ny, nz, hh, scratch,
                                                                         reinterpret_cast<long long *>(d_rhs));
    k_grid_rhs<<<grid_for(n, 256, nsm * 16), 256, 0, st>>>(d_rhs, n, 4.0 * 3.141592653589793, pow(hh, 3.0), scratch);
    if (dh_f32)
        k_grid_dh_f32<<<(unsigned)((nbc + DH_TILE - 1) / DH_TILE), DH_TILE, 0, st>>>(d_c, d_q, n_atoms, nx, ny, nz, hh,
                                                                                    eps_out, kappa, d_bc);
    else if (dh_fast_range(nx, ny, nz, hh, kappa))
        k_grid_dh<true><<<(unsigned)((nbc + DH_TILE - 1) / DH_TILE), DH_TILE, 0, st>>>(d_c, d_q, n_atoms, nx, ny, nz, hh,
                                                                                      eps_out, kappa, d_bc);
    else
        k_grid_dh<false><<<(unsigned)((nbc + DH_TILE - 1) / DH_TILE), DH_TILE, 0, st>>>(d_c, d_q, n_atoms, nx, ny, nz, hh,
                                                                                       eps_out, kappa, d_bc);
    PB_CUDA(cudaGetLastError());
    int bad = 0;
    PB_CUDA(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    return bad ? PB_ERR_INVALID_ARG : PB_OK;      // an atom outside the box [0,(n-1)h]^3 or a non-finite charge
}
}  // namespace

extern "C" pb_status pb_create_from_atoms(pb_handle **out, int nx, int ny, int nz, double hh, int n_atoms,
                                          const double *centres, const double *radii, const double *charges,
                                          double eps_in, double eps_out, double kbar2_solvent,
                                          pb_memspace where, void *cuda_stream)
{
    if (!out) return PB_ERR_INVALID_ARG;
    *out = nullptr;
    if (nx < 2 || ny < 2 || nz < 2 || !(hh > 0.0) || !std::isfinite(hh) || n_atoms < 0 || (n_atoms && (!centres || !radii || !charges)) ||
        !(eps_in > 0.0) || !(eps_out > 0.0) || !(kbar2_solvent >= 0.0) || !valid_space(where))
        return PB_ERR_INVALID_ARG;
    if ((double)nx * ny * nz > 2.0e9) return PB_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return PB_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;     // NULL: legacy default stream, ordered before the handle's own
    const size_t n = (size_t)nx * ny * nz;
    const size_t nbc = 2 * ((size_t)nz * ny + (size_t)nz * nx + (size_t)ny * nx);
    const cudaMemcpyKind kind = where == PB_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    int dev = 0, nsm = 0;
    PB_CUDA(cudaGetDevice(&dev));
    PB_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    DevTmp tmp;
    double *d_c, *d_R, *d_q, *ex, *ey, *ez, *kb, *rhs, *bc, *scratch;
    unsigned char *mask;
    PB_TRY(tmp.get((void **)&scratch, 2 * sizeof(double)));
    PB_TRY(tmp.get((void **)&d_c, (size_t)n_atoms * 3 * sizeof(double)));
    PB_TRY(tmp.get((void **)&d_R, (size_t)n_atoms * sizeof(double)));
    PB_TRY(tmp.get((void **)&d_q, (size_t)n_atoms * sizeof(double)));
    PB_TRY(tmp.get((void **)&mask, n));
    PB_TRY(tmp.get((void **)&ex, (size_t)nz * ny * (nx + 1) * sizeof(double)));
    PB_TRY(tmp.get((void **)&ey, (size_t)nz * (ny + 1) * nx * sizeof(double)));
    PB_TRY(tmp.get((void **)&ez, (size_t)(nz + 1) * ny * nx * sizeof(double)));
    PB_TRY(tmp.get((void **)&kb, n * sizeof(double)));
    PB_TRY(tmp.get((void **)&rhs, n * sizeof(double)));
    PB_TRY(tmp.get((void **)&bc, nbc * sizeof(double)));
    if (n_atoms) {
        PB_CUDA(cudaMemcpyAsync(d_c, centres, (size_t)n_atoms * 3 * sizeof(double), kind, st));
        PB_CUDA(cudaMemcpyAsync(d_R, radii, (size_t)n_atoms * sizeof(double), kind, st));
        PB_CUDA(cudaMemcpyAsync(d_q, charges, (size_t)n_atoms * sizeof(double), kind, st));
    }
    PB_CUDA(cudaMemsetAsync(mask, 0, n, st));
    if (n_atoms) k_grid_mask<<<n_atoms < 65535 ? n_atoms : 65535, 128, 0, st>>>(d_c, d_R, n_atoms, nx, ny, nz, hh, mask);
    const size_t nf = (size_t)(nz + 1) * (ny + 1) * (nx + 1);
    k_grid_faces<<<grid_for(nf, 256, nsm * 16), 256, 0, st>>>(mask, nx, ny, nz, eps_in, eps_out, kbar2_solvent,
                                                                 ex, ey, ez, kb);
    PB_CUDA(cudaGetLastError());
    const double kappa = sqrt(kbar2_solvent / eps_out);
    PB_TRY(charges_to_rhs_bc(d_c, d_q, n_atoms, nx, ny, nz, hh, eps_out, kappa, rhs, bc, scratch, nsm, st));
    pb_handle *h = nullptr;
    PB_TRY(pb_create(&h, nx, ny, nz, hh, ex, ey, ez, kb, rhs, bc, PB_DEVICE, cuda_stream));
    h->atoms_c = d_c; tmp.release(d_c);
    h->n_atoms = n_atoms; h->atoms_eps_out = eps_out; h->atoms_kappa = kappa;
    h->launches += 6;
    *out = h;
    return PB_OK;
}

extern "C" pb_status pb_set_charges(pb_handle *h, const double *charges, pb_memspace where)
{
    if (!h || !h->atoms_c || (h->n_atoms && !charges) || !valid_space(where)) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    const size_t n = (size_t)h->nx * h->ny * h->nz;
    const size_t nbc = 2 * ((size_t)h->nz * h->ny + (size_t)h->nz * h->nx + (size_t)h->ny * h->nx);
    if (!h->atoms_q) PB_ALLOC(cudaMalloc((void **)&h->atoms_q, ((size_t)h->n_atoms + 2) * sizeof(double)));
    double *d_q = h->atoms_q, *scratch = h->atoms_q + h->n_atoms;
    PB_CUDA(cudaMemcpyAsync(d_q, charges, (size_t)h->n_atoms * sizeof(double),
                            where == PB_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, h->stream));
    if (!h->rhs) PB_ALLOC(cudaMalloc((void **)&h->rhs, (n + 8) * sizeof(double)));
    if (!h->bc) PB_ALLOC(cudaMalloc((void **)&h->bc, (nbc + 8) * sizeof(double)));
    PB_TRY(charges_to_rhs_bc(h->atoms_c, d_q, h->n_atoms, h->nx, h->ny, h->nz, h->h, h->atoms_eps_out,
                             h->atoms_kappa, h->rhs, h->bc, scratch, h->nsm, h->stream, h->dh_f32));
    h->launches += 4;
    h->wf.b_ready = false;
    h->wd.b_ready = false;
    if (h->wf.ready) PB_TRY(build_b<float>(h, h->wf));
    if (h->wd.ready) PB_TRY(build_b<double>(h, h->wd));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    return PB_OK;
}

extern "C" pb_status pb_set_setup_precision(pb_handle *h, pb_precision prec)
{
    if (!h || !valid_prec(prec)) return PB_ERR_INVALID_ARG;
    h->dh_f32 = (prec == PB_F32);
    return PB_OK;
}

extern "C" pb_status pb_get_field(pb_handle *h, int which, double *out_host)
{
    if (!h || !out_host || which < 0 || which > 5) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(h->device));
    const size_t n = (size_t)h->nx * h->ny * h->nz;
    const size_t sizes[6] = {(size_t)h->nz * h->ny * (h->nx + 1), (size_t)h->nz * (h->ny + 1) * h->nx,
                             (size_t)(h->nz + 1) * h->ny * h->nx, n, n,
                             2 * ((size_t)h->nz * h->ny + (size_t)h->nz * h->nx + (size_t)h->ny * h->nx)};
    const double *src[6] = {h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->rhs, h->bc};
    if (!src[which]) { memset(out_host, 0, sizes[which] * sizeof(double)); return PB_OK; }   // NULL input = zeros
    PB_CUDA(cudaMemcpyAsync(out_host, src[which], sizes[which] * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    PB_CUDA(cudaStreamSynchronize(h->stream));
    return PB_OK;
}
