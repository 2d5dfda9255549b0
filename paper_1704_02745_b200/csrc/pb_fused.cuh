// pb_fused.cuh -- ONE kernel per PCG iteration: k_spmv_batch (pb_spmv_batch.cuh) with K_vec folded in.
//
// The two-kernel iteration (K_spmv, K_vec) needs two passes because step 5's alpha needs
// p.Ap (a reduction over the whole grid) before r can be updated, and step 7's beta needs r_new.z_new (a second one)
// before p can.  Here the residual update of iteration l is DEFERRED into the pass of iteration
// l+1 -- r_l = r_{l-1} - alpha_l A p_l is formed where r and A p_l are staged anyway, halo cells included -- and the
// scalars of iteration l+1 all come out of ONE reduction at the end of that pass:
//     p.Ap = sum p v,  v = A p_{l+1}                                                  (step 5)
//     r_l.z_l = U1 = sum Dinv r_l^2,   r_l.r_l = U2 = sum r_l^2                          (exact, of the stored r_l)
//     alpha = U1 / p.Ap
//     r_{l+1}.z_{l+1} = U1 - 2 alpha S1 + alpha^2 S2,   S1 = sum Dinv r_l v,  S2 = sum Dinv v^2    (r_{l+1} = r_l - alpha v)
//     r_{l+1}.r_{l+1} = U2 - 2 alpha T1 + alpha^2 T2,   T1 = sum r_l v,       T2 = sum v^2
//     beta = r_{l+1}.z_{l+1} / U1                                                        (step 7)
// These are the algebraic expansions of the very dot products K_vec computes; because U1 and U2 are re-summed from
// the stored r_l in every pass, the expansion is only ever one step deep (no drift: the classical single-reduction
// recurrences carry the norms along and lose them after ~1/eps of reduction).  In exact arithmetic the iterates are
// those of PAPER.md:104-126; in floating point alpha and beta agree with the two-kernel path to rounding.
// The stopping rule (step 3) is applied to the predicted ||r_{l+1}||, so the solve stops at the same l.
//
// Bytes per node and iteration: reads r, A p_l, p (haloed), x, Dinv, three faces; writes r, p, x, A p_{l+1}:
// 8 words + 2 index bytes in the quad format with the diagonal palette (34 B fp32, 66 B fp64) instead of 41 / 77 B
// in two kernels; r, p and A p are double-buffered (a neighbouring tile reads the old plane while this one writes).
// Everything else -- rings, p_new planes, coefficient formats, per-member latches -- is k_spmv_batch's.
#pragma once
#include "pb_internal.cuh"
#include "pb_tma.cuh"
#include "pb_spmv_tma.cuh"
#include "pb_spmv_batch.cuh"
#include "pb_kernels.cuh"

namespace pb {

constexpr int kFusedSums = 7;        // p.Ap, S1, S2, T1, T2, U1, U2

// vector slot of the fused kernel: r, A p (old) and p (old) haloed, x un-haloed
struct FusedLayout {
    BatchLayout B;
    size_t oAq, vslot;
};
__host__ __device__ inline FusedLayout fused_layout(int TXV, int TY, int vec, bool quad, bool pald)
{
    FusedLayout F;
    F.B = batch_layout(TXV, TY, vec, quad, pald);
    F.oAq = F.B.vslot;
    F.vslot = F.oAq + align128(F.B.bZ);
    return F;
}
__host__ __device__ inline size_t fused_smem(const FusedLayout &F, int nsv, int nsc, int M)
{
    return (size_t)nsv * F.vslot + (size_t)nsc * F.B.cslot + (size_t)2 * M * F.B.pn + 128;
}

template <typename T>
struct FusedArgs {
    T *r0, *r1, *Ap0, *Ap1, *p0, *p1;   // [M][npad] each: iteration with iter_cur = l reads buffer l & 1, writes the other
    T *x;
    size_t npad;
    int nx, ny, nz, P;
    int TXV, TY, TZ;
    int ntx, nty, ntz, ntiles;
    int nsv, nsc;
    int precond;
    State *st;               // [M]
    double *partials;        // [M][kFusedSums][gridDim.x]
    const T *lut;
    const T *dlut;
};

// the six ping-pong vector tensors (4-D [M][nz][ny][P], member = coordinate 3), in one kernel parameter
struct FusedMaps { CUtensorMap r0, r1, q0, q1, p0, p1; };

template <typename T, bool QUAD, bool PALD, int M>
__global__ void __launch_bounds__(M >= 2 ? 256 : 512)
k_pcg_fused(const __grid_constant__ FusedMaps vm, const __grid_constant__ CUtensorMap tm_dinv,
            const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_exm,
            const __grid_constant__ CUtensorMap tm_exp, const __grid_constant__ CUtensorMap tm_ey,
            const __grid_constant__ CUtensorMap tm_ez, const FusedArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t vfull[kMaxStages], vempty[kMaxStages];
    __shared__ __align__(8) uint64_t cfull[kMaxCoefStages], cempty[kMaxCoefStages];
    __shared__ double red[32];
    __shared__ int s_last;
    __shared__ __align__(16) T qtab[QUAD ? 256 * 4 : 4];   // qtab[b][f] = lut[(b >> 2f) & 3]: four face values per byte
    __shared__ __align__(16) T ddtab[PALD ? 512 : 2];      // {Dinv, D} pairs

    const int tid = threadIdx.x;
    const int nthr = blockDim.x;
    const int NCT = nthr - 32;                 // consumer threads (whole warps); the last warp produces
    const int NCW = NCT >> 5;
    const int warp = tid >> 5, lane = tid & 31;
    const bool is_producer = (warp == NCW);

    // per-member scalars; a member whose latch is set is skipped by producer and consumers alike
    T beta[M], alpha_prev[M];                  // beta_l and alpha_l: r_l = r_{l-1} - alpha_l A p_l, x += alpha_l p_l, p_{l+1} = z_l + beta_l p_l
    bool live[M];
    int parity[M];
    bool any = false;
#pragma unroll
    for (int s = 0; s < M; s++) {
        const State *st = a.st + s;
        live[s] = !st->done;
        any |= live[s];
        beta[s] = (T)st->beta;
        alpha_prev[s] = (T)st->alpha;          // alpha of the previous iteration (0 before the first)
        parity[s] = st->iter_cur & 1;
    }
    if (!any) return;

    const int nx = a.nx, ny = a.ny, nz = a.nz, P = a.P;
    const int TXV = a.TXV, TY = a.TY, TZ = a.TZ, NSV = a.nsv, NSC = a.nsc;
    const FusedLayout F = fused_layout(TXV, TY, VEC, QUAD, PALD);
    const BatchLayout &L = F.B;
    unsigned char *vbase = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *cbase = vbase + (size_t)NSV * F.vslot;
    unsigned char *pnbase = cbase + (size_t)NSC * L.cslot;   // PN[s][parity] at pnbase + (2 s + parity) * L.pn

    if (tid == 0) {
        for (int i = 0; i < NSV; i++) { mbar_init(&vfull[i], 1); mbar_init(&vempty[i], NCW); }
        for (int i = 0; i < NSC; i++) { mbar_init(&cfull[i], 1); mbar_init(&cempty[i], 1); }
        mbar_fence_init();
    }
    if (QUAD)
        for (int b = tid; b < 256; b += nthr) {
#pragma unroll
            for (int f = 0; f < 4; f++) qtab[b * 4 + f] = a.lut[(b >> (2 * f)) & 3];
        }
    if (PALD)
        for (int i = tid; i < 256; i += nthr) { const T d = a.dlut[i]; ddtab[2 * i] = d; ddtab[2 * i + 1] = rcp_rn(d); }
    __syncthreads();

    double acc[M][kFusedSums];                 // per thread: p.Ap, S1, S2, T1, T2, U1, U2 (see the header)
#pragma unroll
    for (int s = 0; s < M; s++)
#pragma unroll
        for (int q = 0; q < kFusedSums; q++) acc[s][q] = 0.0;

    if (is_producer) {
        if (lane == 0) {
            int vs = 0, cs = 0;
            uint32_t vph = 0, cph = 0;
            for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
                int b = tile;
                const int bx = b % a.ntx; b /= a.ntx;
                const int by = b % a.nty;
                const int bz = b / a.nty;
                const int x0 = bx * TXV * VEC, j0 = by * TY;
                const int k0 = bz * TZ, k1 = min(k0 + TZ, nz);
                const int xd = PALD ? ((x0 - VEC) & ~15) : x0 - VEC;   // byte-index box: 16-byte aligned start
                const int xq = QUAD ? ((x0 >> 2) & ~15) : x0;          // quad-index boxes likewise
                for (int q = k0 - 1; q <= k1; q++) {
                    const bool centre = (q >= k0) && (q < k1);
                    const bool ez = (q >= k0);
                    {   // coefficient item q
                        mbar_wait(&cempty[cs], cph ^ 1);
                        unsigned char *slot = cbase + cs * (uint32_t)L.cslot;
                        uint32_t bytes = L.bDv;
                        if (ez) bytes += L.bEZ;
                        if (centre) bytes += L.bEXM + L.bEXP + L.bEY;
                        mbar_expect_tx(&cfull[cs], bytes);
                        tma_load_3d(slot + L.oDv, &tm_dinv, xd, j0 - 1, q, &cfull[cs]);
                        if (ez) tma_load_3d(slot + L.oEZ, &tm_ez, xq, j0, q, &cfull[cs]);
                        if (centre) {
                            tma_load_3d(slot + L.oEXM, &tm_exm, xq, j0, q, &cfull[cs]);
                            if (QUAD) tma_load_3d(slot + L.oEXP, &tm_exp, xq, j0, q, &cfull[cs]);
                            tma_load_3d(slot + L.oEY, &tm_ey, xq, j0, q, &cfull[cs]);
                        }
                        cs = (cs + 1 == NSC) ? 0 : cs + 1; cph ^= (cs == 0);
                    }
#pragma unroll
                    for (int s = 0; s < M; s++) {
                        if (!live[s]) continue;
                        mbar_wait(&vempty[vs], vph ^ 1);
                        unsigned char *slot = vbase + vs * (uint32_t)F.vslot;
                        mbar_expect_tx(&vfull[vs], 3 * L.bZ + (centre ? L.bX : 0u));
                        tma_load_4d(slot + L.oR, parity[s] ? &vm.r1 : &vm.r0, x0 - VEC, j0 - 1, q, s, &vfull[vs]);
                        tma_load_4d(slot + F.oAq, parity[s] ? &vm.q1 : &vm.q0, x0 - VEC, j0 - 1, q, s, &vfull[vs]);
                        tma_load_4d(slot + L.oPp, parity[s] ? &vm.p1 : &vm.p0, x0 - VEC, j0 - 1, q, s, &vfull[vs]);
                        if (centre) tma_load_4d(slot + L.oX, &tm_x, x0, j0, q, s, &vfull[vs]);
                        vs = (vs + 1 == NSV) ? 0 : vs + 1; vph ^= (vs == 0);
                    }
                }
            }
        }
        __syncwarp();
    } else {
        const int BWc = TXV + 2;                       // vectors per row of the haloed boxes
        const int TXP = spmv_row_threads(TXV);
        const int tx = tid % TXP, ty = tid / TXP;
        const bool intile = ty < TY && tx < TXV;
        const int own = (ty + 1) * BWc + tx + 1;       // own cell in the haloed boxes
        const int own_d = (ty + 1) * L.bwd + (tx + 1) * VEC;   // PALD: its byte offset in the Dinv-index box
        const int cown = ty * TXV + tx;                // own cell in the un-haloed boxes
        const int nextra = 2 * TXV + 2 * TY;           // halo cells: two rows, two columns
        const bool precond = a.precond != 0;
        auto halo_cell = [&](int h) -> int {
            if (h < TXV) return h + 1;
            if (h < 2 * TXV) return (TY + 1) * BWc + (h - TXV) + 1;
            const int cc = h - 2 * TXV, side = cc / TY, r = cc - side * TY;
            return (r + 1) * BWc + (side ? TXV + 1 : 0);
        };
        auto cell_d = [&](int c) -> int { const int row = c / BWc; return row * L.bwd + (c - row * BWc) * VEC; };
        const int extra0 = (NCT - 1 - tid < nextra) ? halo_cell(NCT - 1 - tid) : -1;   // this thread's halo cell
        const int extra0_d = (PALD && extra0 >= 0) ? cell_d(extra0) : 0;
        int lead_d = 0;                                // PALD: bytes between the Dinv-index box's aligned start and x0 - VEC
        int qoff = 0, qfield = 0;                      // QUAD: byte (in a box row) and field offset of this thread's nodes

        // Dinv (and D = 1/Dinv when `D` is given) of haloed-box cell c of a coefficient slot
        auto load_dinv = [&](const unsigned char *cslot, int c, int cd, Vec<T> &dinv, Vec<T> *D) {
            if (PALD) {
                const unsigned char *p = cslot + L.oDv + lead_d + cd;
                const uint32_t w = (VEC == 4) ? *reinterpret_cast<const uint32_t *>(p)
                                              : (uint32_t)*reinterpret_cast<const unsigned short *>(p);
#pragma unroll
                for (int e = 0; e < VEC; e++) {
                    const uint32_t i = (w >> (8 * e)) & 255u;
                    const T *pr = reinterpret_cast<const T *>(reinterpret_cast<const unsigned char *>(ddtab) + i * (2 * sizeof(T)));
                    if (sizeof(T) == 4) {
                        const float2 v = *reinterpret_cast<const float2 *>(pr);
                        dinv.a[e] = (T)v.x; if (D) D->a[e] = (T)v.y;
                    } else {
                        const double2 v = *reinterpret_cast<const double2 *>(pr);
                        dinv.a[e] = (T)v.x; if (D) D->a[e] = (T)v.y;
                    }
                }
            } else {
                dinv = reinterpret_cast<const Vec<T> *>(cslot + L.oDv)[c];
                if (D) {
#pragma unroll
                    for (int e = 0; e < VEC; e++) D->a[e] = rcp_rn(dinv.a[e]);
                }
            }
        };
        // VEC face coefficients of this thread's nodes, row `row` of a coefficient box
        auto coef = [&](const unsigned char *box, int row, int row_vecs) -> Vec<T> {
            if (QUAD) {
                const uint32_t b = box[row * L.bwq + qoff];
                return *reinterpret_cast<const Vec<T> *>(reinterpret_cast<const unsigned char *>(qtab) + b * (4 * sizeof(T)) + qfield);
            }
            return reinterpret_cast<const Vec<T> *>(box)[row * row_vecs + tx];
        };
        auto release_vslot = [&](int s_) { __syncwarp(); if (lane == 0) mbar_arrive(&vempty[s_]); };

        int vs = 0, cs = 0;                            // ring slots of the next items and their phase parities
        uint32_t vph = 0, cph = 0;
        auto vadvance = [&]() { vs = (vs + 1 == NSV) ? 0 : vs + 1; vph ^= (vs == 0); };
        auto cadvance = [&]() { cs = (cs + 1 == NSC) ? 0 : cs + 1; cph ^= (cs == 0); };
        const size_t plane = (size_t)ny * P;

        for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
            int b = tile;
            const int bx = b % a.ntx; b /= a.ntx;
            const int by = b % a.nty;
            const int bz = b / a.nty;
            const int x0 = bx * TXV * VEC, j0 = by * TY;
            const int i0 = x0 + tx * VEC, j = j0 + ty;
            const bool active = intile && (i0 < P) && (j < ny);
            const int nvalid = nx - i0;
            const int k0 = bz * TZ, k1 = min(k0 + TZ, nz);
            lead_d = (x0 - VEC) & 15;
            if (QUAD) { qoff = (i0 >> 2) - ((x0 >> 2) & ~15); qfield = (i0 & 3) * (int)sizeof(T); }
            size_t idx = ((size_t)k0 * ny + j) * P + i0;

            Vec<T> pm[M], pc[M], pn[M], rc[M], rn[M];     // p_new of planes k-1, k, k+1 and r_l of planes k, k+1 (own column)
#pragma unroll
            for (int s = 0; s < M; s++) {
                pm[s] = zerov<T>(); pc[s] = zerov<T>(); pn[s] = zerov<T>(); rc[s] = zerov<T>(); rn[s] = zerov<T>();
            }
            Vec<T> Dc = zerov<T>(), Dn = zerov<T>(), ezc = zerov<T>(), ezn = zerov<T>();
            Vec<T> dvc = zerov<T>(), dvn = zerov<T>();    // Dinv of planes k, k+1 (own column): z_l = Dinv r_l in the sums

            // "update" of plane kk (the items at the ring heads): p_new of every live member -- own cell into out[s],
            // and for a plane this tile writes (centre) the haloed box into PN[s][kk & 1], the deferred phi update
            // and D; the vector slots are handed back, the coefficient slot stays (returned in cslot_out)
            auto update = [&](int kk, bool centre, Vec<T> *out, Vec<T> *rout, Vec<T> &Dout, Vec<T> &dvout, Vec<T> &ezout,
                              bool want_ez, size_t xidx) -> const unsigned char * {
                mbar_wait(&cfull[cs], cph);
                const unsigned char *cslot = cbase + cs * (uint32_t)L.cslot;
                Vec<T> dv = zerov<T>(), dvh = zerov<T>();
                if (intile) load_dinv(cslot, own, own_d, dv, centre ? &Dout : nullptr);
                dvout = dv;
                if (centre && extra0 >= 0) load_dinv(cslot, extra0, extra0_d, dvh, nullptr);
                if (want_ez) ezout = intile ? coef(cslot + L.oEZ, ty, TXV) : zerov<T>();
#pragma unroll
                for (int s = 0; s < M; s++) {
                    if (!live[s]) continue;
                    mbar_wait(&vfull[vs], vph);
                    const unsigned char *sl = vbase + vs * (uint32_t)F.vslot;
                    const Vec<T> *R = reinterpret_cast<const Vec<T> *>(sl + L.oR);
                    const Vec<T> *AQ = reinterpret_cast<const Vec<T> *>(sl + F.oAq);
                    const Vec<T> *Pp = reinterpret_cast<const Vec<T> *>(sl + L.oPp);
                    Vec<T> *PN = reinterpret_cast<Vec<T> *>(pnbase + (size_t)(2 * s + (kk & 1)) * L.pn);
                    // r_l = r_{l-1} - alpha_l A p_l (the deferred step 5), then p_{l+1} = Dinv r_l + beta_l p_l (steps 6-7)
                    auto pnew = [&](int c, const Vec<T> &d, Vec<T> *pold, Vec<T> *rnew) -> Vec<T> {
                        Vec<T> v = R[c];
                        const Vec<T> qv = AQ[c];
                        const Vec<T> pv = Pp[c];
#pragma unroll
                        for (int e = 0; e < VEC; e++) v.a[e] = fma(-alpha_prev[s], qv.a[e], v.a[e]);
                        if (pold) *pold = pv;
                        if (rnew) *rnew = v;
                        if (precond) {
#pragma unroll
                            for (int e = 0; e < VEC; e++) v.a[e] = fma(beta[s], pv.a[e], d.a[e] * v.a[e]);
                        } else {
#pragma unroll
                            for (int e = 0; e < VEC; e++) v.a[e] = fma(beta[s], pv.a[e], v.a[e]);
                        }
                        return v;
                    };
                    Vec<T> v = zerov<T>(), rl = zerov<T>();
                    if (intile) {
                        Vec<T> po;
                        v = pnew(own, dv, &po, &rl);
                        if (centre) {
                            PN[own] = v;
                            if (active) {
                                stv((parity[s] ? a.r0 : a.r1) + (size_t)s * a.npad + xidx, rl);     // r_l
                                // phi_{l-1} = phi_{l-2} + alpha_{l-1} p_{l-2}  (step 5 of the previous iteration)
                                Vec<T> xv = reinterpret_cast<const Vec<T> *>(sl + L.oX)[cown];
#pragma unroll
                                for (int e = 0; e < VEC; e++) xv.a[e] = fma(alpha_prev[s], po.a[e], xv.a[e]);
                                stv(a.x + (size_t)s * a.npad + xidx, xv);
                            }
                        }
                    }
                    if (centre) {
                        if (extra0 >= 0) PN[extra0] = pnew(extra0, dvh, nullptr, nullptr);
                        for (int h = NCT - 1 - tid + NCT; h < nextra; h += NCT) {   // only when the halo outnumbers the threads
                            const int c = halo_cell(h);
                            Vec<T> d2;
                            load_dinv(cslot, c, PALD ? cell_d(c) : 0, d2, nullptr);
                            PN[c] = pnew(c, d2, nullptr, nullptr);
                        }
                    }
                    out[s] = v;
                    rout[s] = rl;
                    consume(v.a[0]);            // R, AQ and Pp of the own cell have been read (x: the store above)
                    release_vslot(vs);
                    vadvance();
                }
                return cslot;
            };

            // item k0-1: only the own column's values are needed; its coefficient slot goes back after a barrier
            {
                const int c0 = cs;
                update(k0 - 1, false, pm, rn, Dn, dvn, ezn, false, idx);
                cadvance();
                named_bar_sync(1, NCT);
                if (tid == 0) mbar_arrive(&cempty[c0]);
            }
            // item k0
            int ck = cs;
            const unsigned char *cslotk = update(k0, true, pc, rc, Dc, dvc, ezc, true, idx);
            cadvance();
            named_bar_sync(1, NCT);

            for (int k = k0; k < k1; k++, idx += plane) {
                const int c1 = cs;
                const unsigned char *cslot1 = update(k + 1, k + 1 < k1, pn, rn, Dn, dvn, ezn, true, idx + plane);
                cadvance();
                if (active) {
                    // the six face coefficients and D of this thread's nodes: decoded once, used by every member
                    Vec<T> exl, exh;
                    if (QUAD) {
                        exl = coef(cslotk + L.oEXM, ty, 0);
                        exh = coef(cslotk + L.oEXP, ty, 0);
                    } else {
                        exl = coef(cslotk + L.oEXM, ty, TXV + 1);
                        const T exr = reinterpret_cast<const Vec<T> *>(cslotk + L.oEXM)[ty * (TXV + 1) + tx + 1].a[0];
#pragma unroll
                        for (int e = 0; e < VEC; e++) exh.a[e] = (e == VEC - 1) ? exr : exl.a[e == VEC - 1 ? e : e + 1];
                    }
                    const Vec<T> eyl = coef(cslotk + L.oEY, ty, TXV), eyh = coef(cslotk + L.oEY, ty + 1, TXV);
#pragma unroll
                    for (int s = 0; s < M; s++) {
                        if (!live[s]) continue;
                        const Vec<T> *Zk = reinterpret_cast<const Vec<T> *>(pnbase + (size_t)(2 * s + (k & 1)) * L.pn);
                        const Vec<T> up = Zk[own - BWc], dn = Zk[own + BWc];
                        const T left = Zk[own - 1].a[VEC - 1], right = Zk[own + 1].a[0];
                        Vec<T> ap;
                        // per-plane partial sums in T over this thread's VEC nodes, then one fp64 add per sum
                        T s_pv = T(0), s_zv = T(0), s_dvv = T(0), s_rv = T(0), s_vv = T(0), s_zr = T(0), s_rr = T(0);
#pragma unroll
                        for (int e = 0; e < VEC; e++) {
                            const T pl = (e == 0) ? left : pc[s].a[e == 0 ? 0 : e - 1];
                            const T pr = (e == VEC - 1) ? right : pc[s].a[e == VEC - 1 ? e : e + 1];
                            // same order of operations as k_spmv_tma
                            T v = Dc.a[e] * pc[s].a[e];
                            v = fma(-exl.a[e], pl, v);
                            v = fma(-exh.a[e], pr, v);
                            v = fma(-eyl.a[e], up.a[e], v);
                            T w = -eyh.a[e] * dn.a[e];
                            w = fma(-ezc.a[e], pm[s].a[e], w);
                            w = fma(-ezn.a[e], pn[s].a[e], w);
                            v += w;
                            if (e >= nvalid) v = T(0);     // pad column
                            const T rl = rc[s].a[e];
                            const T zl = precond ? dvc.a[e] * rl : rl;          // z_l = M^-1 r_l
                            const T dv_v = precond ? dvc.a[e] * v : v;
                            s_pv = fma(pc[s].a[e], v, s_pv);
                            s_zv = fma(zl, v, s_zv);
                            s_dvv = fma(dv_v, v, s_dvv);
                            s_rv = fma(rl, v, s_rv);
                            s_vv = fma(v, v, s_vv);
                            s_zr = fma(zl, rl, s_zr);
                            s_rr = fma(rl, rl, s_rr);
                            ap.a[e] = v;
                        }
                        acc[s][0] += (double)s_pv; acc[s][1] += (double)s_zv; acc[s][2] += (double)s_dvv;
                        acc[s][3] += (double)s_rv; acc[s][4] += (double)s_vv; acc[s][5] += (double)s_zr;
                        acc[s][6] += (double)s_rr;
                        stv((parity[s] ? a.Ap0 : a.Ap1) + (size_t)s * a.npad + idx, ap);
                        stv((parity[s] ? a.p0 : a.p1) + (size_t)s * a.npad + idx, pc[s]);
                    }
                }
                named_bar_sync(1, NCT);   // p_new(k+1) boxes complete; everyone is done with coefficient slot ck and p_new(k)
                if (tid == 0) mbar_arrive(&cempty[ck]);
#pragma unroll
                for (int s = 0; s < M; s++) { pm[s] = pc[s]; pc[s] = pn[s]; rc[s] = rn[s]; }
                ezc = ezn; Dc = Dn; dvc = dvn; ck = c1; cslotk = cslot1;
            }
            // coefficient item k1: only Dinv and ez of the own column were used, before the last barrier
            if (tid == 0) mbar_arrive(&cempty[ck]);
        }
    }

    // stage 1 -> per-block partials; stage 2 by the last block to take a ticket (fixed order: deterministic); then every
    // scalar of the iteration (header) and the stopping rule of step 3 (finish_iteration, pb_kernels.cuh)
    const int nblk = gridDim.x;
#pragma unroll
    for (int s = 0; s < M; s++)
#pragma unroll
        for (int q = 0; q < kFusedSums; q++) {
            const double t = block_sum(acc[s][q], red);
            if (tid == 0) a.partials[((size_t)s * kFusedSums + q) * nblk + blockIdx.x] = t;
        }
    if (tid == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(&a.st->ticket_spmv, 1u);
        s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
#pragma unroll
        for (int s = 0; s < M; s++) {
            double sum[kFusedSums];
#pragma unroll
            for (int q = 0; q < kFusedSums; q++) sum[q] = final_sum(a.partials + ((size_t)s * kFusedSums + q) * nblk, nblk, red);
            if (tid == 0 && live[s]) {
                State *st = a.st + s;
                const double pAp = sum[0], S1 = sum[1], S2 = sum[2], T1 = sum[3], T2 = sum[4], U1 = sum[5], U2 = sum[6];
                st->pAp = pAp;
                st->rz = U1;                                    // r_l.z_l and ||r_l||^2 of the stored r_l, exactly
                st->rr = U2;
                if (!(pAp > 0.0) || !isfinite(pAp) || !isfinite(U1) || !isfinite(U2)) {   // breakdown: not SPD / NaN
                    if (st->latch) { st->done = 1; st->iters = st->iter_cur; st->status = 5; }
                    st->alpha = 0.0;                            // x already holds the last good iterate
                } else {
                    const double alpha = U1 / pAp;              // step 5
                    st->alpha = alpha;
                    double rz_new = fma(alpha, fma(alpha, S2, -2.0 * S1), U1);     // r_{l+1}.z_{l+1}
                    double rr_new = fma(alpha, fma(alpha, T2, -2.0 * T1), U2);     // ||r_{l+1}||^2
                    if (rz_new < 0.0) rz_new = 0.0;             // cancellation at the rounding floor
                    if (rr_new < 0.0) rr_new = 0.0;
                    finish_iteration(st, rz_new, rr_new, 0);    // beta (step 7), l + 1 (step 4), stopping rule (step 3)
                }
            }
        }
        if (tid == 0) a.st->ticket_spmv = 0u;
    }
}

}  // namespace pb
