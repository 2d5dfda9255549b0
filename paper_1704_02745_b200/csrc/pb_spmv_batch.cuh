// pb_spmv_batch.cuh -- K_spmv for M right-hand sides on ONE operator in one pass ("multi-RHS
// kernels that read the coefficient arrays once for m right-hand sides"; the paper's motivation is "thousands to
// millions of snapshots" of one molecule).
//
// Per right-hand side s the computation is exactly k_spmv_tma's (pb_spmv_tma.cuh): z = Dinv r (step 6, Jacobi,
// PAPER.md:138-140), p <- z + beta_s p (step 7), the deferred x += alpha_s p_old (step 5), Ap = A'p with the rows of
// Eq. 3 rebuilt from the face dielectrics, partial p.Ap (step 5) -- same operations in the same
// order per node, so member s of a batch takes bit for bit the iterates of a single solve with the same tile plan.
// What is shared by the M members: the coefficient boxes of a plane (staged once by the TMA producer), their decode
// into registers (D, Dinv, the six face values), the ring hand-off and the plane barrier.
//
// Structure (one persistent block per tile column, one producer lane, NCW consumer warps):
//   coefficient ring  item q = { Dinv(q) (haloed), ez(q), ex-(q), ex+(q), ey(q) }                 one per plane
//   vector ring       item (q, s) = { r_s(q), p_old_s(q) (haloed), x_s(q) }                       M per plane
//   p_new planes      PN[s][q & 1]: the haloed p_new box of member s, double-buffered, plain shared memory
// A vector slot goes back to the producer as soon as its plane has been turned into p_new (every warp arrives once
// it has read its cells; the slots are only ever READ by the generic proxy, so no proxy fence is needed); a
// coefficient slot after the plane barrier that follows the stencil of its plane (one elected thread arrives).
// Coefficient formats: QUAD -- face palettes of at most four values (every molecular map: 0, eps_in, eps_out and their
// harmonic mean) as 2-bit indices, four nodes per byte, decoded four at a time through a 256-entry
// table of quadruples (eps_x stored twice, as the minus and the plus face of each node); otherwise full words.
// PALD -- Dinv as one index byte per node into a table of {Dinv, D = 1/Dinv} pairs; otherwise Dinv words.
#pragma once
#include "pb_internal.cuh"
#include "pb_tma.cuh"
#include "pb_spmv_tma.cuh"

namespace pb {

constexpr int kMaxBatch = 4;          // right-hand sides per pass (compile-time M in {1, 2, 4})
constexpr int kMaxCoefStages = 4;

// bytes per row of a quad-index box: the tile row's TXV*VEC nodes span at most TXV*VEC/4 + 1 bytes, the box starts
// at a 16-byte aligned byte (up to 15 bytes of lead-in), rows are multiples of 16 bytes (TMA)
__host__ __device__ inline int quad_row_bytes(int TXV, int vec) { return ((TXV * vec + 3) / 4 + 1 + 15 + 15) / 16 * 16; }

struct BatchLayout {
    uint32_t bZ, bX, bDv, bEZ, bEXM, bEXP, bEY;   // exact box bytes (what the TMA delivers)
    int bwq;                                      // QUAD: bytes per row of a quad-index box
    int bwd;                                      // PALD: bytes per row of the haloed Dinv-index box
    size_t oR, oPp, oX, vslot;                    // vector slot
    size_t oDv, oEZ, oEXM, oEXP, oEY, cslot;      // coefficient slot
    size_t pn;                                    // bytes of ONE p_new plane buffer (haloed box)
};
__host__ __device__ inline BatchLayout batch_layout(int TXV, int TY, int vec, bool quad, bool pald)
{
    BatchLayout L;
    L.bZ = (uint32_t)(TY + 2) * (TXV + 2) * 16;
    L.bX = (uint32_t)TY * TXV * 16;
    L.bwd = pald ? ((TXV + 2) * vec + 16 + 15) / 16 * 16 : 0;
    L.bDv = pald ? (uint32_t)(TY + 2) * L.bwd : L.bZ;
    if (quad) {
        L.bwq = quad_row_bytes(TXV, vec);
        L.bEZ = L.bEXM = L.bEXP = (uint32_t)TY * L.bwq;
        L.bEY = (uint32_t)(TY + 1) * L.bwq;
    } else {
        L.bwq = 0;
        L.bEZ = L.bX;
        L.bEXM = (uint32_t)TY * (TXV + 1) * 16;   // one extra vector: the plus face of the row's last node
        L.bEXP = 0;
        L.bEY = (uint32_t)(TY + 1) * TXV * 16;
    }
    L.oR = 0;
    L.oPp = L.oR + align128(L.bZ);
    L.oX = L.oPp + align128(L.bZ);
    L.vslot = L.oX + align128(L.bX);
    L.oDv = 0;
    L.oEZ = L.oDv + align128(L.bDv);
    L.oEXM = L.oEZ + align128(L.bEZ);
    L.oEXP = L.oEXM + align128(L.bEXM);
    L.oEY = L.oEXP + align128(L.bEXP);
    L.cslot = L.oEY + align128(L.bEY);
    L.pn = align128(L.bZ);
    return L;
}
// dynamic shared memory of one block
__host__ __device__ inline size_t batch_smem(const BatchLayout &L, int nsv, int nsc, int M)
{
    return (size_t)nsv * L.vslot + (size_t)nsc * L.cslot + (size_t)2 * M * L.pn + 128;
}

template <typename T>
struct BatchArgs {
    T *pbuf0, *pbuf1;        // [M][npad]: iteration l of member s reads buf[l_s & 1], writes buf[(l_s + 1) & 1]
    T *Ap, *x;               // [M][npad]
    size_t npad;             // elements between two members
    int nx, ny, nz, P;
    int TXV, TY, TZ;
    int ntx, nty, ntz, ntiles;
    int nsv, nsc;            // ring depths: vector slots, coefficient slots
    int precond;
    State *st;               // [M]
    double *partials;        // [M][gridDim.x]
    const T *lut;            // QUAD: the (<= 4) face values, ascending
    const T *dlut;           // PALD: the distinct values of Dinv (index = byte of the Dinv-index tensor, unscaled)
};

// vector tensors are 4-D [M][nz][ny][P] (member = coordinate 3), coefficient tensors 3-D
template <typename T, bool QUAD, bool PALD, int M>
__global__ void __launch_bounds__(M >= 4 ? 256 : 512)
k_spmv_batch(const __grid_constant__ CUtensorMap tm_r, const __grid_constant__ CUtensorMap tm_dinv,
             const __grid_constant__ CUtensorMap tm_p0, const __grid_constant__ CUtensorMap tm_p1,
             const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_exm,
             const __grid_constant__ CUtensorMap tm_exp, const __grid_constant__ CUtensorMap tm_ey,
             const __grid_constant__ CUtensorMap tm_ez, const BatchArgs<T> a)
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
    T beta[M], alpha_prev[M];
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
    const BatchLayout L = batch_layout(TXV, TY, VEC, QUAD, PALD);
    unsigned char *vbase = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *cbase = vbase + (size_t)NSV * L.vslot;
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

    double acc[M];
#pragma unroll
    for (int s = 0; s < M; s++) acc[s] = 0.0;

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
                        unsigned char *slot = vbase + vs * (uint32_t)L.vslot;
                        mbar_expect_tx(&vfull[vs], 2 * L.bZ + (centre ? L.bX : 0u));
                        tma_load_4d(slot + L.oR, &tm_r, x0 - VEC, j0 - 1, q, s, &vfull[vs]);
                        tma_load_4d(slot + L.oPp, parity[s] ? &tm_p1 : &tm_p0, x0 - VEC, j0 - 1, q, s, &vfull[vs]);
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

            Vec<T> pm[M], pc[M], pn[M];
#pragma unroll
            for (int s = 0; s < M; s++) { pm[s] = zerov<T>(); pc[s] = zerov<T>(); pn[s] = zerov<T>(); }
            Vec<T> Dc = zerov<T>(), Dn = zerov<T>(), ezc = zerov<T>(), ezn = zerov<T>();

            // "update" of plane kk (the items at the ring heads): p_new of every live member -- own cell into out[s],
            // and for a plane this tile writes (centre) the haloed box into PN[s][kk & 1], the deferred phi update
            // and D; the vector slots are handed back, the coefficient slot stays (returned in cslot_out)
            auto update = [&](int kk, bool centre, Vec<T> *out, Vec<T> &Dout, Vec<T> &ezout, bool want_ez, size_t xidx)
                -> const unsigned char * {
                mbar_wait(&cfull[cs], cph);
                const unsigned char *cslot = cbase + cs * (uint32_t)L.cslot;
                Vec<T> dv = zerov<T>(), dvh = zerov<T>();
                if (intile) load_dinv(cslot, own, own_d, dv, centre ? &Dout : nullptr);
                if (centre && extra0 >= 0) load_dinv(cslot, extra0, extra0_d, dvh, nullptr);
                if (want_ez) ezout = intile ? coef(cslot + L.oEZ, ty, TXV) : zerov<T>();
#pragma unroll
                for (int s = 0; s < M; s++) {
                    if (!live[s]) continue;
                    mbar_wait(&vfull[vs], vph);
                    const unsigned char *sl = vbase + vs * (uint32_t)L.vslot;
                    const Vec<T> *R = reinterpret_cast<const Vec<T> *>(sl + L.oR);
                    const Vec<T> *Pp = reinterpret_cast<const Vec<T> *>(sl + L.oPp);
                    Vec<T> *PN = reinterpret_cast<Vec<T> *>(pnbase + (size_t)(2 * s + (kk & 1)) * L.pn);
                    auto pnew = [&](int c, const Vec<T> &d, Vec<T> *pold) -> Vec<T> {
                        Vec<T> v = R[c];
                        const Vec<T> pv = Pp[c];
                        if (pold) *pold = pv;
                        if (precond) {
#pragma unroll
                            for (int e = 0; e < VEC; e++) v.a[e] = fma(beta[s], pv.a[e], d.a[e] * v.a[e]);
                        } else {
#pragma unroll
                            for (int e = 0; e < VEC; e++) v.a[e] = fma(beta[s], pv.a[e], v.a[e]);
                        }
                        return v;
                    };
                    Vec<T> v = zerov<T>();
                    if (intile) {
                        Vec<T> po;
                        v = pnew(own, dv, &po);
                        if (centre) {
                            PN[own] = v;
                            if (active) {
                                // phi_{l-1} = phi_{l-2} + alpha_{l-1} p_{l-2}  (step 5 of the previous iteration)
                                Vec<T> xv = reinterpret_cast<const Vec<T> *>(sl + L.oX)[cown];
#pragma unroll
                                for (int e = 0; e < VEC; e++) xv.a[e] = fma(alpha_prev[s], po.a[e], xv.a[e]);
                                stv(a.x + (size_t)s * a.npad + xidx, xv);
                            }
                        }
                    }
                    if (centre) {
                        if (extra0 >= 0) PN[extra0] = pnew(extra0, dvh, nullptr);
                        for (int h = NCT - 1 - tid + NCT; h < nextra; h += NCT) {   // only when the halo outnumbers the threads
                            const int c = halo_cell(h);
                            Vec<T> d2;
                            load_dinv(cslot, c, PALD ? cell_d(c) : 0, d2, nullptr);
                            PN[c] = pnew(c, d2, nullptr);
                        }
                    }
                    out[s] = v;
                    consume(v.a[0]);            // R and Pp of the own cell have been read (x: the store above)
                    release_vslot(vs);
                    vadvance();
                }
                return cslot;
            };

            // item k0-1: only the own column's values are needed; its coefficient slot goes back after a barrier
            {
                const int c0 = cs;
                update(k0 - 1, false, pm, Dn, ezn, false, idx);
                cadvance();
                named_bar_sync(1, NCT);
                if (tid == 0) mbar_arrive(&cempty[c0]);
            }
            // item k0
            int ck = cs;
            const unsigned char *cslotk = update(k0, true, pc, Dc, ezc, true, idx);
            cadvance();
            named_bar_sync(1, NCT);

            for (int k = k0; k < k1; k++, idx += plane) {
                const int c1 = cs;
                const unsigned char *cslot1 = update(k + 1, k + 1 < k1, pn, Dn, ezn, true, idx + plane);
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
                            acc[s] = fma((double)pc[s].a[e], (double)v, acc[s]);
                            ap.a[e] = v;
                        }
                        stv(a.Ap + (size_t)s * a.npad + idx, ap);
                        stv((parity[s] ? a.pbuf0 : a.pbuf1) + (size_t)s * a.npad + idx, pc[s]);
                    }
                }
                named_bar_sync(1, NCT);   // p_new(k+1) boxes complete; everyone is done with coefficient slot ck and p_new(k)
                if (tid == 0) mbar_arrive(&cempty[ck]);
#pragma unroll
                for (int s = 0; s < M; s++) { pm[s] = pc[s]; pc[s] = pn[s]; }
                ezc = ezn; Dc = Dn; ck = c1; cslotk = cslot1;
            }
            // coefficient item k1: only Dinv and ez of the own column were used, before the last barrier
            if (tid == 0) mbar_arrive(&cempty[ck]);
        }
    }

    // stage 1 -> per-block partials; stage 2 by the last block to take a ticket (fixed order: deterministic)
    const int nblk = gridDim.x;
    double tot[M];
#pragma unroll
    for (int s = 0; s < M; s++) tot[s] = block_sum(acc[s], red);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < M; s++) a.partials[(size_t)s * nblk + blockIdx.x] = tot[s];
        __threadfence();
        const unsigned int t = atomicAdd(&a.st->ticket_spmv, 1u);
        s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
#pragma unroll
        for (int s = 0; s < M; s++) {
            const double pAp = final_sum(a.partials + (size_t)s * nblk, nblk, red);
            if (tid == 0 && live[s]) {
                State *st = a.st + s;
                st->pAp = pAp;
                if (!(pAp > 0.0) || !isfinite(pAp)) {          // breakdown: not SPD / NaN
                    if (st->latch) { st->done = 1; st->iters = st->iter_cur; st->status = 5; }
                    st->alpha = 0.0;                            // x already holds the last good iterate
                } else {
                    st->alpha = st->rz / pAp;                   // step 5
                }
            }
        }
        if (tid == 0) a.st->ticket_spmv = 0u;
    }
}

}  // namespace pb
