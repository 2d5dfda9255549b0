// pb_api_batch.cuh -- host logic of pb_solve_batch / pb_solve_batch_charges (NEXT row f2 of SURVEY.md 8(f): M
// right-hand sides per pass through k_spmv_batch + k_vec_batch).  Included by pb_api.cu inside its anonymous
// namespace, after the single-solve helpers it builds on (ensure, make_map, vec_args, k_init, k_finish ...).
#pragma once

// 4-D tensor [M][planes][rows][P] of T (member = coordinate 3), box = bx elements x by rows x 1 plane x 1 member
template <typename T>
pb_status make_map4(CUtensorMap *tm, const T *ptr, int P, int rows, int planes, int members, int bx, int by, int bm = 1,
                    size_t member_stride = 0)       // elements between two members (0: dense, P * rows * planes)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return PB_ERR_CUDA;
    const cuuint64_t dims[4] = {(cuuint64_t)P, (cuuint64_t)rows, (cuuint64_t)planes, (cuuint64_t)members};
    const cuuint64_t strides[3] = {(cuuint64_t)P * sizeof(T), (cuuint64_t)P * rows * sizeof(T),
                                   (cuuint64_t)(member_stride ? member_stride : (size_t)P * rows * planes) * sizeof(T)};
    const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1u, (cuuint32_t)bm};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = fn(tm, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4,
                          (void *)ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? PB_OK : PB_ERR_CUDA;
}

// 4-D byte tensor [members][planes][rows][Pb], box = bw bytes x by rows x 1 plane x bm members
inline pb_status make_map4_u8(CUtensorMap *tm, const unsigned char *ptr, int Pb, int rows, int planes, int members, int bw,
                              int by, int bm)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return PB_ERR_CUDA;
    const cuuint64_t dims[4] = {(cuuint64_t)Pb, (cuuint64_t)rows, (cuuint64_t)planes, (cuuint64_t)members};
    const cuuint64_t strides[3] = {(cuuint64_t)Pb, (cuuint64_t)Pb * rows, (cuuint64_t)Pb * rows * planes};
    const cuuint32_t box[4] = {(cuuint32_t)bw, (cuuint32_t)by, 1u, (cuuint32_t)bm};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, (void *)ptr, dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                          CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? PB_OK : PB_ERR_CUDA;
}

template <typename T, bool QUAD, bool PALD, int M>
pb_status batch_kernel_attr(size_t *max_dyn)
{
    cudaFuncAttributes fa;
    PB_CUDA(cudaFuncGetAttributes(&fa, k_spmv_batch<T, QUAD, PALD, M>));
    const size_t lim = (size_t)232448 - fa.sharedSizeBytes;
    PB_CUDA(cudaFuncSetAttribute(k_spmv_batch<T, QUAD, PALD, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lim));
    *max_dyn = lim;
    return PB_OK;
}
template <typename T, int M>
pb_status batch_kernel_attr_fmt(bool quad, bool pald, size_t *max_dyn)
{
    if (quad) return pald ? batch_kernel_attr<T, true, true, M>(max_dyn) : batch_kernel_attr<T, true, false, M>(max_dyn);
    return pald ? batch_kernel_attr<T, false, true, M>(max_dyn) : batch_kernel_attr<T, false, false, M>(max_dyn);
}

template <typename T, bool QUAD, bool PALD>
pb_status fused_kernel_attr(size_t *max_dyn)
{
    cudaFuncAttributes fa;
    PB_CUDA(cudaFuncGetAttributes(&fa, k_pcg_fused<T, QUAD, PALD>));
    const size_t lim = (size_t)232448 - fa.sharedSizeBytes;
    PB_CUDA(cudaFuncSetAttribute(k_pcg_fused<T, QUAD, PALD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lim));
    *max_dyn = lim;
    return PB_OK;
}
template <typename T>
pb_status fused_kernel_attr_fmt(bool quad, bool pald, size_t *max_dyn)
{
    if (quad) return pald ? fused_kernel_attr<T, true, true>(max_dyn) : fused_kernel_attr<T, true, false>(max_dyn);
    return pald ? fused_kernel_attr<T, false, true>(max_dyn) : fused_kernel_attr<T, false, false>(max_dyn);
}

template <typename T> pb_status enqueue_batch_iterations(pb_handle *h, Work<T> &w, int n_iter);

// coefficient arrays, vectors, plan and tensor maps of the batch path for M members; `fused`: of k_pcg_fused (one
// kernel per iteration, one member) instead of k_spmv_batch + k_vec_batch
template <typename T>
pb_status ensure_batch(pb_handle *h, int M, bool fused = false)
{
    constexpr int VEC = VecN<T>::value;
    PB_TRY(ensure<T>(h));
    Work<T> &w = work<T>(h);
    BatchWork<T> &b = w.bw;
    pb_status s = PB_OK;
    const size_t rows = (size_t)h->nz * h->ny;
    if (!b.coef_ready) {
        b.quad = h->pal_n > 0 && h->pal_n <= 4 && h->opt[PB_OPT_PALETTE] != 0;
        b.pald = w.pald && h->opt[PB_OPT_PALETTE_DIAG_SPMV] != 0;
        b.Pq = ((w.P + 3) / 4 + 15) / 16 * 16;
        if (b.quad) {
            const size_t b_ex = rows * b.Pq, b_ey = (size_t)h->nz * (h->ny + 1) * b.Pq, b_ez = (size_t)(h->nz + 1) * h->ny * b.Pq;
            if ((s = alloc_arr(&b.exq, b_ex)) || (s = alloc_arr(&b.exqp, b_ex)) || (s = alloc_arr(&b.eyq, b_ey)) ||
                (s = alloc_arr(&b.ezq, b_ez))) { free_batch(b); return s; }
            if (!w.lut) {
                if ((s = alloc_arr(&w.lut, (size_t)kPalMax))) { free_batch(b); return s; }
                k_pal_lut<T><<<1, 256, 0, h->stream>>>(h->pal_table, w.lut);
            }
            k_setup_quad_idx<<<grid_for((size_t)(h->nz + 1) * (h->ny + 1) * b.Pq, 256, h->nsm * 16), 256, 0, h->stream>>>(
                h->eps_x, h->eps_y, h->eps_z, h->nx, h->ny, h->nz, b.Pq, h->pal_table, b.exq, b.exqp, b.eyq, b.ezq);
            h->launches += 1;
        } else if (w.exm) {
            b.exm = w.exm; b.eym = w.eym; b.ezm = w.ezm;
        } else {
            // a byte-palette operator (5..64 face values): the batch kernel reads full words, built here once
            const size_t n_ey = (size_t)h->nz * (h->ny + 1) * w.P, n_ez = (size_t)(h->nz + 1) * h->ny * w.P;
            b.own_words = true;
            if ((s = alloc_arr(&b.exm, w.npad)) || (s = alloc_arr(&b.eym, n_ey)) || (s = alloc_arr(&b.ezm, n_ez))) {
                free_batch(b);
                return s;
            }
            k_setup_coeff<T><<<grid_for((size_t)(h->nz + 1) * (h->ny + 1) * w.P, 256, h->nsm * 16), 256, 0, h->stream>>>(
                h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->h * h->h, h->nx, h->ny, h->nz, w.P,
                b.exm, b.eym, b.ezm, w.D, w.Dinv, h->bad);
            h->launches += 1;
        }
        if (b.pald) {
            if ((s = alloc_arr(&b.dviu, rows * w.Pb))) { free_batch(b); return s; }
            k_setup_diag_idx<<<grid_for(rows * w.Pb, 256, h->nsm * 16), 256, 0, h->stream>>>(
                h->eps_x, h->eps_y, h->eps_z, h->kbar2, h->h * h->h, h->nx, h->ny, h->nz, w.Pb, 1, h->pald_table, b.dviu);
            h->launches += 1;
        }
        PB_CUDA(cudaGetLastError());
        b.coef_ready = true;
    }
    if (b.cap < M) {
        if (b.vblock) cudaFree(b.vblock);
        if (b.b) cudaFree(b.b);
        b.vblock = b.b = nullptr;
        b.cap = 0; b.M = 0;
        // one allocation, buffer set 0 then buffer set 1: the four arrays of a set are consecutive (k_pcg_fused fetches
        // their boxes with one TMA instruction, pb_fused.cuh)
        const size_t each = (size_t)M * w.npad;
        if ((s = alloc_arr(&b.vblock, 8 * each)) || (s = alloc_arr(&b.b, each))) { free_batch(b); return s; }
        b.r = b.vblock; b.Ap = b.r + each; b.p0 = b.Ap + each; b.x = b.p0 + each;
        b.r2 = b.x + each; b.Ap2 = b.r2 + each; b.p1 = b.Ap2 + each; b.x2 = b.p1 + each;
        b.cap = M;
    }
    if (fused && b.quad && !b.cq4) {
        const size_t one = (size_t)(h->nz + 1) * (h->ny + 1) * b.Pq;
        if ((s = alloc_arr(&b.cq4, 4 * one))) { free_batch(b); return s; }
        k_setup_quad4<<<grid_for(one, 256, h->nsm * 16), 256, 0, h->stream>>>(h->eps_x, h->eps_y, h->eps_z, h->nx, h->ny, h->nz,
                                                                               b.Pq, h->pal_table, b.cq4);
        PB_CUDA(cudaGetLastError());
        h->launches += 1;
    }
    if (b.M == M && b.fused == fused) return PB_OK;
    if (b.graph) { cudaGraphExecDestroy(b.graph); b.graph = nullptr; }
    // plan: rows of about 1 KB like k_spmv_tma, four rows, two blocks per SM (one for M = 4: its registers), rings as
    // deep as the shared memory allows
    size_t max_dyn = 0;
    if (fused) {
        if (M != 1) return PB_ERR_INVALID_ARG;
        PB_TRY((fused_kernel_attr_fmt<T>(b.quad, b.pald, &max_dyn)));
    } else if (M == 1) PB_TRY((batch_kernel_attr_fmt<T, 1>(b.quad, b.pald, &max_dyn)));
    else if (M == 2) PB_TRY((batch_kernel_attr_fmt<T, 2>(b.quad, b.pald, &max_dyn)));
    else PB_TRY((batch_kernel_attr_fmt<T, 4>(b.quad, b.pald, &max_dyn)));
    const int max_threads = (!fused && M >= 4) ? 256 : 512;      // the kernels' launch bounds
    const int rowvecs = w.P / VEC;
    const int maxv = ((b.pald || b.quad) ? 240 : 256) / VEC - 2;
    int ntx0 = (rowvecs + 32) / 64;
    if (ntx0 < 1) ntx0 = 1;
    while ((rowvecs + ntx0 - 1) / ntx0 > maxv) ntx0++;
    const int *o = h->opt;
    // the plan for tile rows of `txv_c` vectors (0: the option, else rows of about 1 KB), and its tensor maps
    auto plan_with = [&](int txv_c, int pool_c = 0) -> pb_status {
    b.TXV = o[PB_OPT_TILE_TXV] > 0 ? o[PB_OPT_TILE_TXV] : txv_c > 0 ? txv_c : (rowvecs + ntx0 - 1) / ntx0;
    if (b.TXV > maxv) b.TXV = maxv;
    if (b.TXV > rowvecs) b.TXV = rowvecs;
    b.TY = o[PB_OPT_TILE_TY] > 0 ? o[PB_OPT_TILE_TY] : 4;
    if (b.TY > h->ny) b.TY = h->ny;
    const int max_ct = max_threads - 64;
    while (spmv_row_threads(b.TXV) * b.TY > max_ct && b.TY > 1) b.TY--;
    // k_pcg_fused takes 128 registers per thread: two blocks share an SM only up to 256 threads each (measured at 385^3
    // fp64: 65 x 3 tiles, two blocks per SM, 0.654 ms per pass against 0.742 ms for 65 x 4 with one block)
    if (fused && o[PB_OPT_TILE_TY] <= 0 && o[PB_OPT_BLOCKS_PER_SM] != 1)
        while ((spmv_row_threads(b.TXV) * b.TY + 31) / 32 * 32 + 32 > 256 && b.TY > 2) b.TY--;
    b.threads = (spmv_row_threads(b.TXV) * b.TY + 31) / 32 * 32 + 32;
    if (fused) {       // k_pcg_fused: one halo cell per consumer thread at most
        const int halo = (2 * b.TXV + 2 * b.TY + 31) / 32 * 32 + 32;
        if (halo > b.threads) b.threads = halo;
        if (b.threads > max_threads) return PB_ERR_INVALID_ARG;
    }
    const FusedLayout FL = fused_layout(b.TXV, b.TY, VEC, b.quad, b.pald);
    const BatchLayout &L = FL.B;
    const long vslot = fused ? (long)FL.vslot : (long)L.vslot;
    const long cslot = fused ? (long)FL.cslot : (long)L.cslot, pnb = fused ? (long)FL.pn : (long)L.pn;
    // blocks per SM / coefficient ring depth: the first combination that leaves the vector ring M + 2 slots (the
    // consumers work on one member's plane while M more are in flight), else the one with the deepest vector ring
    const int forced_bps = o[PB_OPT_BLOCKS_PER_SM];
    const int try_bps[3] = {max_threads == 256 ? 1 : 2, 1, 1}, try_nsc[3] = {4, 4, 3};
    b.nsv = 0;
    for (int t = 0; t < 3; t++) {
        const int bps = forced_bps > 0 ? forced_bps : try_bps[t], nsc = try_nsc[t];
        const long fixed = (long)nsc * cslot + (fused ? (long)kFusedPlanes : 2L * M) * pnb + 128 +
                           (fused ? (long)fused_fixed_smem((int)sizeof(T), b.quad, b.pald) : 0L);
        long budget = (long)((size_t)232448 / bps) - 1024 - (long)((size_t)232448 - max_dyn) - fixed;   // per-SM share
        if ((long)max_dyn - fixed < budget) budget = (long)max_dyn - fixed;                              // per-block cap
        int nsv = budget > 0 ? (int)(budget / vslot) : 0;
        if (nsv > kMaxStages) nsv = kMaxStages;
        if (nsv > b.nsv) { b.nsv = nsv; b.nsc = nsc; b.bps = bps; }
        if (b.nsv >= M + 2) break;
    }
    if (o[PB_OPT_RING_SLOTS] > 0 && o[PB_OPT_RING_SLOTS] < b.nsv) b.nsv = o[PB_OPT_RING_SLOTS];
    if (b.nsv < 2) return PB_ERR_INVALID_ARG;
    b.smem = fused ? fused_smem(FL, b.nsv, b.nsc, (int)sizeof(T), b.quad, b.pald) : batch_smem(L, b.nsv, b.nsc, M);
    b.ntx = (rowvecs + b.TXV - 1) / b.TXV;
    b.nty = (h->ny + b.TY - 1) / b.TY;
    const int slots = h->nsm * b.bps, xy = b.ntx * b.nty;
    // k_pcg_fused: the planes [zs, nz) form the dynamically scheduled pool (pool_c planes per chunk, about a twentieth of
    // nz: at full clock 5-15 % are equally good, under the power cap of a long run the smaller pool's extra halo planes
    // cost less -- 385^3 fp32 sustained: 10 % pool -1 %, 5 % pool +0.7 % against none)
    b.zs = h->nz; b.pc = 0; b.npool = 0;
    if (fused && pool_c >= 4 && h->nz >= 8 * pool_c) {
        int nch = (h->nz + 10 * pool_c) / (20 * pool_c);
        if (nch < 1) nch = 1;
        b.pc = pool_c; b.zs = h->nz - nch * pool_c; b.npool = nch * xy;
    }
    b.TZ = o[PB_OPT_TILE_TZ] > 0 ? o[PB_OPT_TILE_TZ] : choose_tz(b.zs, xy, slots);
    if (b.TZ > b.zs) b.TZ = b.zs;
    b.ntz = (b.zs + b.TZ - 1) / b.TZ;
    const long ntiles = (long)xy * b.ntz;
    b.grid = (int)(ntiles < slots ? ntiles : slots);
    b.vec_grid = grid_for(w.npad / VEC, 256, h->nsm * 8);
    size_t need = (size_t)M * b.grid > (size_t)2 * M * b.vec_grid ? (size_t)M * b.grid : (size_t)2 * M * b.vec_grid;
    if (fused && (size_t)kFusedSums * ((size_t)ntiles + b.npool) > need) need = (size_t)kFusedSums * ((size_t)ntiles + b.npool);
    if (need > h->partials_cap) {
        PB_CUDA(cudaStreamSynchronize(h->stream));
        if (h->partials) cudaFree(h->partials);
        h->partials = nullptr;
        h->partials_cap = 0;
        PB_ALLOC(cudaMalloc((void **)&h->partials, need * sizeof(double)));
        h->partials_cap = need;
        // graphs captured earlier hold the old pointer
        if (h->wf.graph) { cudaGraphExecDestroy(h->wf.graph); h->wf.graph = nullptr; }
        if (h->wd.graph) { cudaGraphExecDestroy(h->wd.graph); h->wd.graph = nullptr; }
        if (h->wf.bw.graph) { cudaGraphExecDestroy(h->wf.bw.graph); h->wf.bw.graph = nullptr; }
        if (h->wd.bw.graph) { cudaGraphExecDestroy(h->wd.bw.graph); h->wd.bw.graph = nullptr; }
    }
    const int hx = (b.TXV + 2) * VEC, hy = b.TY + 2;
    PB_TRY(make_map4<T>(&b.tm_r, b.r, w.P, h->ny, h->nz, M, hx, hy));
    PB_TRY(make_map4<T>(&b.tm_p0, b.p0, w.P, h->ny, h->nz, M, hx, hy));
    PB_TRY(make_map4<T>(&b.tm_p1, b.p1, w.P, h->ny, h->nz, M, hx, hy));
    PB_TRY(make_map4<T>(&b.tm_x, b.x, w.P, h->ny, h->nz, M, b.TXV * VEC, b.TY));
    if (fused) {       // M = 1: (r, Ap, p0, x) and (r2, Ap2, p1, x2) as four members each
        const size_t each = (size_t)b.cap * w.npad;                  // the arrays were sized for b.cap members
        PB_TRY(make_map4<T>(&b.vm.set0, b.r, w.P, h->ny, h->nz, 4, hx, hy, 4, each));
        PB_TRY(make_map4<T>(&b.vm.set1, b.r2, w.P, h->ny, h->nz, 4, hx, hy, 4, each));
        if (b.quad) PB_TRY(make_map4_u8(&b.tm_q4, b.cq4, b.Pq, h->ny + 1, h->nz + 1, 4, L.bwq, b.TY + 1, 4));
    }
    if (b.pald) PB_TRY(make_map_u8(&b.tm_dinv, b.dviu, w.Pb, h->ny, h->nz, L.bwd, hy));
    else PB_TRY(make_map<T>(&b.tm_dinv, w.Dinv, w.P, h->ny, h->nz, hx, hy));
    if (b.quad) {
        PB_TRY(make_map_u8(&b.tm_exm, b.exq, b.Pq, h->ny, h->nz, L.bwq, b.TY));
        PB_TRY(make_map_u8(&b.tm_exp, b.exqp, b.Pq, h->ny, h->nz, L.bwq, b.TY));
        PB_TRY(make_map_u8(&b.tm_ey, b.eyq, b.Pq, h->ny + 1, h->nz, L.bwq, b.TY + 1));
        PB_TRY(make_map_u8(&b.tm_ez, b.ezq, b.Pq, h->ny, h->nz + 1, L.bwq, b.TY));
    } else {
        PB_TRY(make_map<T>(&b.tm_exm, b.exm, w.P, h->ny, h->nz, (b.TXV + 1) * VEC, b.TY));
        b.tm_exp = b.tm_exm;
        PB_TRY(make_map<T>(&b.tm_ey, b.eym, w.P, h->ny + 1, h->nz, b.TXV * VEC, b.TY + 1));
        PB_TRY(make_map<T>(&b.tm_ez, b.ezm, w.P, h->ny, h->nz + 1, b.TXV * VEC, b.TY));
    }
    if (fused && !b.quad) b.tm_q4 = b.tm_dinv;       // word format: the merged quad box does not exist (never fetched)
    b.M = M;
    b.fused = fused;
    return PB_OK;
    };
    // measured at 385^3 at full clock: 5-15 % of the planes in chunks of 6-13 take 5-7 % (fp32) / 10 % (fp64) off a pass
    const int pool_forced = o[PB_OPT_TAIL_POOL] >= 4 ? o[PB_OPT_TAIL_POOL] : (o[PB_OPT_TAIL_POOL] == 0 && h->nz >= 64) ? 8 : 0;
    PB_TRY(plan_with(0, pool_forced));
    b.tuned = 0;
    const bool forced = o[PB_OPT_TILE_TXV] > 0 || o[PB_OPT_TILE_TY] > 0 || o[PB_OPT_TILE_TZ] > 0 || o[PB_OPT_RING_SLOTS] > 0 ||
                        o[PB_OPT_BLOCKS_PER_SM] > 0;
    if (fused && o[PB_OPT_AUTOTUNE] && !forced && (size_t)h->nx * h->ny * h->nz >= ((size_t)1 << 21)) {
        // Like an FFT plan: time the pass for rows cut into ntx0 - 1 ... ntx0 + 2 tiles on the handle's own arrays (their
        // contents do not matter: no latch, every solve re-initialises them) and keep the fastest.  Which width wins
        // depends on how well neighbouring tiles stay in step (L2 reuse of the halo rows), not only on the tile shape:
        // e.g. 481 x 481 x 257 fp64 0.917 ms with 61 x 3 tiles, 0.739 ms with 82 x 2.
        int cand[4], nc = 0;
        for (int ntx = ntx0 > 1 ? ntx0 - 1 : 1; ntx <= ntx0 + 2 && nc < 4; ntx++) {
            const int txv = (rowvecs + ntx - 1) / ntx;
            if (txv > maxv || txv < 8) continue;
            if (nc && cand[nc - 1] == txv) continue;
            cand[nc++] = txv;
        }
        if (nc > 1) {
            cudaEvent_t e0 = nullptr, e1 = nullptr;
            if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess) {
                float best = 1e30f;
                int best_txv = 0;
                const int txv_std = (rowvecs + ntx0 - 1) / ntx0;
                for (int c = 0; c < nc; c++) {
                    const int txv_c = cand[c];
                    if (plan_with(txv_c, pool_forced) != PB_OK) continue;
                    k_set_state<<<1, 1, 0, h->stream>>>(h->st, 1.0, 0, 0);
                    if (enqueue_batch_iterations<T>(h, w, 2) != PB_OK) continue;          // warm-up (both buffer sets)
                    cudaEventRecord(e0, h->stream);
                    if (enqueue_batch_iterations<T>(h, w, 6) != PB_OK) continue;
                    cudaEventRecord(e1, h->stream);
                    float ms = 0.f;
                    if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) {
                        cudaGetLastError();
                        continue;
                    }
                    if (verbose()) fprintf(stderr, "pb: fused plan candidate TXV=%d TY=%d TZ=%d pool=%d: %.4f ms per pass\n", b.TXV, b.TY, b.TZ, b.pc, ms / 6);
                    // six passes are a noisy sample: another width has to beat the standard one (rows of about 1 KB) by 3 %
                    if (txv_c == txv_std) { if (ms * 0.97f < best) { best = ms * 0.97f; best_txv = txv_c; } }
                    else if (ms < best) { best = ms; best_txv = txv_c; }
                }
                PB_TRY(plan_with(best_txv, pool_forced));
                b.tuned = best_txv > 0;
            }
            if (e0) cudaEventDestroy(e0);
            if (e1) cudaEventDestroy(e1);
            PB_CUDA(cudaGetLastError());
        }
    }
    if (verbose())
        fprintf(stderr, "pb: %s plan<%s> M=%d %s%s TXV=%d TY=%d TZ=%d vector slots=%d coefficient slots=%d bps=%d tiles=%d (+%d pool chunks of %d planes) grid=%d threads=%d smem=%zu%s\n",
                fused ? "fused" : "batch", sizeof(T) == 4 ? "f32" : "f64", M, b.quad ? "quad" : "words", b.pald ? "+diag palette" : "", b.TXV, b.TY, b.TZ,
                b.nsv, b.nsc, b.bps, b.ntx * b.nty * b.ntz, b.npool, b.pc, b.grid, b.threads, b.smem, b.tuned ? " (autotuned)" : "");
    return PB_OK;
}

template <typename T, bool QUAD, bool PALD, int M>
void launch_batch_kernels(pb_handle *h, Work<T> &w, int n_iter)
{
    BatchWork<T> &b = w.bw;
    BatchArgs<T> a;
    a.pbuf0 = b.p0; a.pbuf1 = b.p1; a.Ap = b.Ap; a.x = b.x; a.npad = w.npad;
    a.nx = h->nx; a.ny = h->ny; a.nz = h->nz; a.P = w.P;
    a.TXV = b.TXV; a.TY = b.TY; a.TZ = b.TZ; a.ntx = b.ntx; a.nty = b.nty; a.ntz = b.ntz;
    a.ntiles = b.ntx * b.nty * b.ntz; a.nsv = b.nsv; a.nsc = b.nsc; a.precond = h->precond;
    a.st = h->st; a.partials = h->partials; a.lut = w.lut; a.dlut = w.dlut;
    VecArgs<T> v = vec_args<T>(h, w);
    v.r = b.r; v.Ap = b.Ap;
    for (int it = 0; it < n_iter; it++) {
        k_spmv_batch<T, QUAD, PALD, M><<<b.grid, b.threads, b.smem, h->stream>>>(
            b.tm_r, b.tm_dinv, b.tm_p0, b.tm_p1, b.tm_x, b.tm_exm, b.tm_exp, b.tm_ey, b.tm_ez, a);
        if (w.pald) k_vec_batch<T, true, M><<<b.vec_grid, 256, 0, h->stream>>>(v, w.npad);
        else k_vec_batch<T, false, M><<<b.vec_grid, 256, 0, h->stream>>>(v, w.npad);
    }
}

template <typename T, bool QUAD, bool PALD>
void launch_fused_kernels(pb_handle *h, Work<T> &w, int n_iter)
{
    BatchWork<T> &b = w.bw;
    FusedArgs<T> a;
    a.r0 = b.r; a.r1 = b.r2; a.Ap0 = b.Ap; a.Ap1 = b.Ap2; a.p0 = b.p0; a.p1 = b.p1; a.x0 = b.x; a.x1 = b.x2;
    a.nx = h->nx; a.ny = h->ny; a.nz = h->nz; a.P = w.P;
    a.TXV = b.TXV; a.TY = b.TY; a.TZ = b.TZ; a.ntx = b.ntx; a.nty = b.nty; a.ntz = b.ntz;
    a.ntiles = b.ntx * b.nty * b.ntz; a.nsv = b.nsv; a.nsc = b.nsc; a.precond = h->precond;
    a.st = h->st; a.partials = h->partials; a.lut = w.lut; a.dlut = w.dlut;
    a.nct = b.threads - 32;
    a.zs = b.zs; a.pc = b.pc; a.npool = b.npool; a.ncol = b.ntx * b.nty;
    a.sQ = (size_t)(b.Ap - b.r) * sizeof(T); a.sP = (size_t)(b.p0 - b.r) * sizeof(T); a.sX = (size_t)(b.x - b.r) * sizeof(T);
    fused_args_layout(a, fused_layout(b.TXV, b.TY, VecN<T>::value, QUAD, PALD));
    for (int it = 0; it < n_iter; it++)
        k_pcg_fused<T, QUAD, PALD><<<b.grid, b.threads, b.smem, h->stream>>>(b.vm, b.tm_dinv, b.tm_q4, b.tm_exm, b.tm_ey,
                                                                           b.tm_ez, a);
}

template <typename T>
pb_status enqueue_batch_iterations(pb_handle *h, Work<T> &w, int n_iter)
{
    const BatchWork<T> &b = w.bw;
    if (b.fused) {
        if (b.quad) { if (b.pald) launch_fused_kernels<T, true, true>(h, w, n_iter); else launch_fused_kernels<T, true, false>(h, w, n_iter); }
        else { if (b.pald) launch_fused_kernels<T, false, true>(h, w, n_iter); else launch_fused_kernels<T, false, false>(h, w, n_iter); }
        PB_CUDA(cudaGetLastError());
        h->launches += (long long)n_iter;
        return PB_OK;
    }
#define PB_BATCH_CASE(Q, D, MM) launch_batch_kernels<T, Q, D, MM>(h, w, n_iter)
#define PB_BATCH_M(Q, D) do { if (b.M == 1) PB_BATCH_CASE(Q, D, 1); else if (b.M == 2) PB_BATCH_CASE(Q, D, 2); else PB_BATCH_CASE(Q, D, 4); } while (0)
    if (b.quad) { if (b.pald) PB_BATCH_M(true, true); else PB_BATCH_M(true, false); }
    else { if (b.pald) PB_BATCH_M(false, true); else PB_BATCH_M(false, false); }
#undef PB_BATCH_M
#undef PB_BATCH_CASE
    PB_CUDA(cudaGetLastError());
    h->launches += 2LL * n_iter;
    return PB_OK;
}

// M members: steps 1-8 until every member's latch is set; member s's right-hand side b is in w.bw.b + s*npad
// steps 1-2 of every member (x = 0, r = b, p cleared, ||b||^2, the l = 0 test); `single_b`: the one right-hand side
// of pb_solve (w.b) instead of the members' own (w.bw.b)
template <typename T>
pb_status init_batch(pb_handle *h, int M, double tol, int maxiter, int latch, const T *single_b)
{
    Work<T> &w = work<T>(h);
    BatchWork<T> &b = w.bw;
    h->last_prec = sizeof(T) == 4 ? PB_F32 : PB_F64;
    if (b.fused) PB_CUDA(cudaMemsetAsync(b.Ap, 0, (size_t)M * w.npad * sizeof(T), h->stream));   // "A p_0" = 0: r_0 = b
    for (int s = 0; s < M; s++) {
        k_set_state<<<1, 1, 0, h->stream>>>(h->st + s, tol * tol, maxiter, latch);
        VecArgs<T> va = vec_args<T>(h, w);
        va.r = b.r + s * w.npad; va.b = single_b ? single_b : b.b + s * w.npad; va.x = b.x + s * w.npad;
        va.pzero = b.p0 + s * w.npad;
        va.st = h->st + s;
        k_init<T><<<w.vec_grid, 256, 0, h->stream>>>(va);
    }
    PB_CUDA(cudaGetLastError());
    h->launches += 2LL * M;
    return PB_OK;
}

// step 1 with a given phi_0 on the batch work set, member 0, after init_batch: x = phi_0,
// r = b - A'phi_0 (A'phi_0 through k_spmv_tma<MODE 1> on the handle's own arrays), r.z, r.r, the l = 0 test again;
// k_pcg_fused's first pass then finds exactly what it finds after a cold start (alpha = beta = 0, "A p_0" = 0, p = 0)
template <typename T>
pb_status warm_batch(pb_handle *h, const T *b_rhs, const void *phi0, pb_memspace where)
{
    Work<T> &w = work<T>(h);
    BatchWork<T> &b = w.bw;
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    const T *src = (const T *)phi0;
    if (where == PB_HOST) {
        PB_TRY(ensure_stage(h, n * sizeof(T)));
        PB_CUDA(cudaMemcpyAsync(h->stage, phi0, n * sizeof(T), cudaMemcpyHostToDevice, h->stream));
        src = (const T *)h->stage;
    }
    k_pad<T, T><<<grid_for(w.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(src, w.tmp, h->nx, w.P, rows);
    launch_spmv<T, 1>(h, w, 1.0);                      // w.Ap = A' phi_0
    VecArgs<T> va = vec_args<T>(h, w);
    va.r = b.r; va.x = b.x; va.b = b_rhs;
    k_warm<T><<<w.vec_grid, 256, 0, h->stream>>>(va, w.tmp);
    PB_CUDA(cudaGetLastError());
    h->launches += 3;
    return PB_OK;
}

template <typename T>
pb_status run_batch(pb_handle *h, int M, double tol, int maxiter, int check_every, const T *single_b = nullptr,
                    const void *phi0 = nullptr, pb_memspace phi0_where = PB_DEVICE)
{
    Work<T> &w = work<T>(h);
    BatchWork<T> &b = w.bw;
    PB_TRY(init_batch<T>(h, M, tol, maxiter, 1, single_b));
    if (phi0) {
        if (M != 1 || !single_b) return PB_ERR_INVALID_ARG;
        PB_TRY(warm_batch<T>(h, single_b, phi0, phi0_where));
    }
    const int m = check_every;
    const long long per_iter = b.fused ? 1 : 2;
    bool graph_ok = false;
    if (h->opt[PB_OPT_GRAPH]) {
        if (!(b.graph && b.graph_iters == m)) {
            if (b.graph) { cudaGraphExecDestroy(b.graph); b.graph = nullptr; }
            cudaGraph_t g = nullptr;
            PB_CUDA(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
            const pb_status cs = enqueue_batch_iterations<T>(h, w, m);
            h->launches -= per_iter * m;
            const cudaError_t e = cudaStreamEndCapture(h->stream, &g);
            if (cs == PB_OK && e == cudaSuccess && g && cudaGraphInstantiate(&b.graph, g, 0) == cudaSuccess) b.graph_iters = m;
            else { b.graph = nullptr; cudaGetLastError(); }
            if (g) cudaGraphDestroy(g);
        }
        graph_ok = b.graph != nullptr;
    }
    const long max_chunks = (long)maxiter / m + 2;
    bool all_done = false;
    for (long c = 0; c < max_chunks + 1 && !all_done; c++) {
        if (graph_ok) { PB_CUDA(cudaGraphLaunch(b.graph, h->stream)); h->launches += per_iter * m; }
        else PB_TRY(enqueue_batch_iterations<T>(h, w, m));
        State *slot = h->pinned_state + kMaxBatch * (c & 1);
        PB_CUDA(cudaMemcpyAsync(slot, h->st, M * sizeof(State), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaEventRecord(h->ev[c & 1], h->stream));
        if (c >= 1) {
            PB_CUDA(cudaEventSynchronize(h->ev[(c - 1) & 1]));
            const State *prev = h->pinned_state + kMaxBatch * ((c - 1) & 1);
            all_done = true;
            for (int s = 0; s < M; s++) all_done = all_done && prev[s].done;
        }
    }
    return PB_OK;
}

// fold member s's right-hand side (dense rhs / bc on the device) into w.bw.b + s*npad
template <typename T>
pb_status batch_fold(pb_handle *h, Work<T> &w, int s, const double *d_rhs, const double *d_bc)
{
    const double h2 = h->h * h->h;
    k_setup_b<T><<<grid_for(w.npad, 256, h->nsm * 16), 256, 0, h->stream>>>(
        h->eps_x, h->eps_y, h->eps_z, d_rhs, h->periodic ? nullptr : d_bc, h2, h->nx, h->ny, h->nz, w.P, w.bw.b + s * w.npad);
    PB_CUDA(cudaGetLastError());
    h->launches += 1;
    return PB_OK;
}

// pb_solve_batch / pb_solve_batch_charges: members in groups of the batch width; each group = fold the members'
// right-hand sides, run_batch, un-pad the potentials
template <typename T>
pb_status solve_batch_impl(pb_handle *h, int m, const double *rhs, const double *bc, const double *charges,
                           pb_memspace where, double tol, int maxiter, int check_every, void *phi_out,
                           int *iters_out, double *relres_out, int *status_out)
{
    PB_TRY(ensure<T>(h));
    Work<T> &w = work<T>(h);
    const size_t rows = (size_t)h->nz * h->ny, n = rows * h->nx;
    const size_t nbc = 2 * ((size_t)h->nz * h->ny + (size_t)h->nz * h->nx + (size_t)h->ny * h->nx);
    const int width = h->opt[PB_OPT_BATCH_WIDTH];
    if (h->periodic) return PB_ERR_INVALID_ARG;         // the batch kernels implement the free-space (ghost-layer) condition
    if (where == PB_HOST) PB_TRY(ensure_stage(h, n * sizeof(T)));
    DevTmp tmp;
    double *d_q = nullptr, *scratch = nullptr;
    if (charges) {
        PB_TRY(tmp.get((void **)&d_q, (size_t)(h->n_atoms ? h->n_atoms : 1) * sizeof(double)));
        PB_TRY(tmp.get((void **)&scratch, 2 * sizeof(double)));
    }
    pb_status worst = PB_OK;
    for (int g0 = 0; g0 < m;) {
        int M = width;
        while (M > m - g0) M >>= 1;
        PB_TRY(ensure_batch<T>(h, M, h->opt[PB_OPT_FUSED] != 0 && M == 1));
        for (int s = 0; s < M; s++) {
            const int mem = g0 + s;
            if (charges) {
                PB_CUDA(cudaMemcpyAsync(d_q, charges + (size_t)mem * h->n_atoms, (size_t)h->n_atoms * sizeof(double),
                                        where == PB_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, h->stream));
                if (!h->rhs) PB_ALLOC(cudaMalloc((void **)&h->rhs, (n + 8) * sizeof(double)));
                if (!h->bc) PB_ALLOC(cudaMalloc((void **)&h->bc, (nbc + 8) * sizeof(double)));
                PB_TRY(charges_to_rhs_bc(h->atoms_c, d_q, h->n_atoms, h->nx, h->ny, h->nz, h->h, h->atoms_eps_out,
                                         h->atoms_kappa, h->rhs, h->bc, scratch, h->nsm, h->stream, h->dh_f32));
                h->launches += 4;
                PB_TRY(batch_fold<T>(h, w, s, h->rhs, h->bc));
                h->wf.b_ready = false; h->wd.b_ready = false;      // the handle's own rhs now is the last member's
            } else if (where == PB_DEVICE) {
                PB_TRY(batch_fold<T>(h, w, s, rhs ? rhs + (size_t)mem * n : nullptr, bc ? bc + (size_t)mem * nbc : nullptr));
            } else {
                PB_TRY(take_copy(h, &h->rhs, rhs ? rhs + (size_t)mem * n : nullptr, n, PB_HOST));
                PB_TRY(take_copy(h, &h->bc, bc ? bc + (size_t)mem * nbc : nullptr, nbc, PB_HOST));
                PB_TRY(batch_fold<T>(h, w, s, h->rhs, h->bc));
                PB_CUDA(cudaStreamSynchronize(h->stream));          // h->rhs / h->bc are reused by the next member
                h->wf.b_ready = false; h->wd.b_ready = false;
            }
        }
        PB_TRY(run_batch<T>(h, M, tol, maxiter, check_every));
        for (int s = 0; s < M; s++) {
            const int mem = g0 + s;
            T *dst = (T *)phi_out + (size_t)mem * n;
            T *dev_dst = where == PB_HOST ? (T *)h->stage : dst;
            k_finish<T, T><<<grid_for(n, 256, h->nsm * 16), 256, 0, h->stream>>>(
                w.bw.x + s * w.npad, w.bw.p0 + s * w.npad, w.bw.p1 + s * w.npad, h->st + s, dev_dst, h->nx, w.P, rows,
                w.bw.fused ? w.bw.x2 : nullptr);
            PB_CUDA(cudaGetLastError());
            h->launches += 1;
            if (where == PB_HOST) {
                PB_CUDA(cudaMemcpyAsync(dst, dev_dst, n * sizeof(T), cudaMemcpyDeviceToHost, h->stream));
                PB_CUDA(cudaStreamSynchronize(h->stream));          // the staging buffer is reused by the next member
            }
        }
        PB_CUDA(cudaMemcpyAsync(h->pinned_state, h->st, M * sizeof(State), cudaMemcpyDeviceToHost, h->stream));
        PB_CUDA(cudaStreamSynchronize(h->stream));
        for (int s = 0; s < M; s++) {
            const State &st = h->pinned_state[s];
            if (!st.done) return PB_ERR_CUDA;
            if (iters_out) iters_out[g0 + s] = st.iters;
            if (relres_out) relres_out[g0 + s] = (st.bb > 0.0) ? sqrt(st.rr / st.bb) : 0.0;
            if (status_out) status_out[g0 + s] = st.status;
            if (st.status == (int)PB_ERR_BREAKDOWN) worst = PB_ERR_BREAKDOWN;
            else if (st.status == (int)PB_ERR_MAXITER && worst == PB_OK) worst = PB_ERR_MAXITER;
        }
        g0 += M;
    }
    return worst;
}
