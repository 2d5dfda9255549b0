// pb_spmv_quad.cuh -- K_spmv for operators whose face dielectrics take at most FOUR distinct values (pad value 0
// included): every molecular map built from eps_in, eps_out and their harmonic mean is one.
//
// Same computation as k_spmv_tma (pb_spmv_tma.cuh; PAPER.md:118-124 steps 5-7 with the Jacobi M of PAPER.md:138-140
// and the rows of Eq. 3, rebuilt on the fly), same persistent warp-specialised TMA ring, same
// arithmetic per node bit for bit.  What differs is the storage format of the coefficients and how the consumer
// warps spend their instructions (the byte-palette kernel had become issue-bound: ~300 warp instructions per plane,
// a fifth of them table look-ups):
//   * face coefficients as 2-bit palette indices, FOUR NODES PER BYTE (exq/exqp/eyq/ezq): one LDS.U8 + one LDS.128
//     from a 256-entry table of decoded quadruples yields four coefficients (was LDS + 4 PRMT + 4 LDS), and the
//     three face arrays cost 1 byte per node instead of 3 (eps_x is stored twice, as the minus and the plus face of
//     each node, so the plus faces need no shifted access);
//   * Dinv and D = 1/Dinv come from ONE 64/128-bit look-up in a table of pairs; D is carried in registers to the
//     plane's stencil one step later instead of being looked up again;
//   * p_new planes live in their own double-buffered shared array instead of being written back into the TMA slot:
//     the slots are only ever read by the generic proxy, so handing them back needs no fence.proxy.async, and one
//     elected thread arrives for the whole block after the plane barrier;
//   * the deferred phi update (x += alpha_prev p_old) happens where p_old is in registers anyway.
#pragma once
#include "pb_internal.cuh"
#include "pb_tma.cuh"
#include "pb_spmv_tma.cuh"

namespace pb {

// bytes per row of a quad-index box: the tile row's TXV*VEC nodes span at most TXV*VEC/4 + 1 bytes, the box starts
// at a 16-byte aligned byte (up to 15 bytes of lead-in), rows are multiples of 16 bytes (TMA)
__host__ __device__ inline int quad_row_bytes(int TXV, int vec) { return ((TXV * vec + 3) / 4 + 1 + 15 + 15) / 16 * 16; }

struct QuadLayout {
    uint32_t bZ, bX, bDv, bQ, bQy;           // exact box bytes (what the TMA delivers)
    int bwq;                                 // bytes per row of a quad-index box
    int bwd;                                 // PALD: bytes per row of the haloed Dinv-index box
    size_t oR, oPp, oX, oDv, oEZ, oEXM, oEXP, oEY, slot;
    size_t pn;                               // bytes of ONE p_new plane buffer (haloed box)
};
__host__ __device__ inline QuadLayout quad_layout(int TXV, int TY, int vec, bool pald)
{
    QuadLayout L;
    L.bZ = (uint32_t)(TY + 2) * (TXV + 2) * 16;
    L.bX = (uint32_t)TY * TXV * 16;
    L.bwd = pald ? ((TXV + 2) * vec + 16 + 15) / 16 * 16 : 0;
    L.bDv = pald ? (uint32_t)(TY + 2) * L.bwd : L.bZ;
    L.bwq = quad_row_bytes(TXV, vec);
    L.bQ = (uint32_t)TY * L.bwq;
    L.bQy = (uint32_t)(TY + 1) * L.bwq;
    L.oR = 0;
    L.oPp = L.oR + align128(L.bZ);
    L.oX = L.oPp + align128(L.bZ);
    L.oDv = L.oX + align128(L.bX);
    L.oEZ = L.oDv + align128(L.bDv);
    L.oEXM = L.oEZ + align128(L.bQ);
    L.oEXP = L.oEXM + align128(L.bQ);
    L.oEY = L.oEXP + align128(L.bQ);
    L.slot = L.oEY + align128(L.bQy);
    L.pn = align128(L.bZ);
    return L;
}

template <typename T>
struct QuadArgs {
    T *pbuf0, *pbuf1;        // iteration l reads buf[l&1] (through its tensor map), writes buf[(l+1)&1]
    T *Ap;
    T *x;
    int nx, ny, nz, P;
    int TXV, TY, TZ;
    int ntx, nty, ntz, ntiles;
    int nstage;
    int precond;
    State *st;
    double *partials;
    double out_scale;        // MODE 1 only
    const T *lut;            // the (<= 4) face values, ascending
    const T *dlut;           // PALD: the distinct values of Dinv (index = byte of the Dinv-index tensor, unscaled)
};

// MODE 0: PCG step;  MODE 1: y = out_scale * A' v  (v behind tm_r)
// PALD: Dinv is a byte-index tensor (haloed box) decoded through a table of {Dinv, D} pairs; else a word tensor
template <typename T, int MODE, bool PALD>
__global__ void __launch_bounds__(512)
k_spmv_quad(const __grid_constant__ CUtensorMap tm_r, const __grid_constant__ CUtensorMap tm_dinv,
            const __grid_constant__ CUtensorMap tm_p0, const __grid_constant__ CUtensorMap tm_p1,
            const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_exm,
            const __grid_constant__ CUtensorMap tm_exp, const __grid_constant__ CUtensorMap tm_ey,
            const __grid_constant__ CUtensorMap tm_ez, const QuadArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[kMaxStages];
    __shared__ __align__(8) uint64_t empty_bar[kMaxStages];
    __shared__ double red[32];
    __shared__ int s_last;
    __shared__ __align__(16) T qtab[256 * 4];              // qtab[b][f] = lut[(b >> 2f) & 3]: four face values per byte
    __shared__ __align__(16) T ddtab[PALD ? 512 : 2];      // {Dinv, D} pairs

    const int tid = threadIdx.x;
    const int nthr = blockDim.x;
    const int NCT = nthr - 32;                 // consumer threads (whole warps); the last warp produces
    const int NCW = NCT >> 5;
    const int warp = tid >> 5, lane = tid & 31;
    const bool is_producer = (warp == NCW);

    T beta = T(0), alpha_prev = T(0);
    const CUtensorMap *tm_pin = &tm_p0;
    T *pout = nullptr;
    if (MODE == 0) {
        if (a.st->done) return;
        const int it = a.st->iter_cur;
        beta = (T)a.st->beta;
        alpha_prev = (T)a.st->alpha;           // alpha of the previous iteration (0 before the first)
        tm_pin = (it & 1) ? &tm_p1 : &tm_p0;
        pout = (it & 1) ? a.pbuf0 : a.pbuf1;
    }
    const int nx = a.nx, ny = a.ny, nz = a.nz, P = a.P;
    const int TXV = a.TXV, TY = a.TY, TZ = a.TZ, NS = a.nstage;
    const QuadLayout L = quad_layout(TXV, TY, VEC, PALD);
    unsigned char *base = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *pnbase = base + (size_t)NS * L.slot;    // two p_new plane buffers behind the ring

    if (tid == 0) {
        for (int s = 0; s < NS; s++) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        mbar_fence_init();
    }
    for (int b = tid; b < 256; b += nthr) {
#pragma unroll
        for (int f = 0; f < 4; f++) qtab[b * 4 + f] = a.lut[(b >> (2 * f)) & 3];
    }
    if (PALD)
        for (int i = tid; i < 256; i += nthr) { const T d = a.dlut[i]; ddtab[2 * i] = d; ddtab[2 * i + 1] = rcp_rn(d); }
    __syncthreads();

    double acc = 0.0;
    if (is_producer) {
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
                int b = tile;
                const int bx = b % a.ntx; b /= a.ntx;
                const int by = b % a.nty;
                const int bz = b / a.nty;
                const int x0 = bx * TXV * VEC, j0 = by * TY;
                const int k0 = bz * TZ, k1 = min(k0 + TZ, nz);
                const int xd = PALD ? ((x0 - VEC) & ~15) : x0 - VEC;   // byte-index box: 16-byte aligned start
                const int xq = (x0 >> 2) & ~15;                        // quad-index boxes likewise
                for (int q = k0 - 1; q <= k1; q++, s = (s + 1 == NS) ? 0 : s + 1, ph ^= (s == 0)) {
                    mbar_wait(&empty_bar[s], ph ^ 1);
                    unsigned char *slot = base + s * (uint32_t)L.slot;
                    const bool centre = (q >= k0) && (q < k1);
                    const bool ez = (q >= k0);
                    uint32_t bytes = (MODE == 0) ? 2 * L.bZ + L.bDv : L.bZ;
                    if (ez) bytes += L.bQ;
                    if (centre) bytes += 2 * L.bQ + L.bQy + (MODE == 0 ? L.bX : L.bDv);
                    mbar_expect_tx(&full_bar[s], bytes);
                    tma_load_3d(slot + L.oR, &tm_r, x0 - VEC, j0 - 1, q, &full_bar[s]);
                    if (MODE == 0) {
                        tma_load_3d(slot + L.oDv, &tm_dinv, xd, j0 - 1, q, &full_bar[s]);
                        tma_load_3d(slot + L.oPp, tm_pin, x0 - VEC, j0 - 1, q, &full_bar[s]);
                    } else if (centre) {
                        tma_load_3d(slot + L.oDv, &tm_dinv, xd, j0 - 1, q, &full_bar[s]);
                    }
                    if (ez) tma_load_3d(slot + L.oEZ, &tm_ez, xq, j0, q, &full_bar[s]);
                    if (centre) {
                        if (MODE == 0) tma_load_3d(slot + L.oX, &tm_x, x0, j0, q, &full_bar[s]);
                        tma_load_3d(slot + L.oEXM, &tm_exm, xq, j0, q, &full_bar[s]);
                        tma_load_3d(slot + L.oEXP, &tm_exp, xq, j0, q, &full_bar[s]);
                        tma_load_3d(slot + L.oEY, &tm_ey, xq, j0, q, &full_bar[s]);
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
        const int cown = ty * TXV + tx;                // own cell in the x box
        const int nextra = 2 * TXV + 2 * TY;           // halo cells: two rows, two columns
        const bool precond = a.precond != 0;
        auto halo_cell = [&](int h) -> int {
            if (h < TXV) return h + 1;
            if (h < 2 * TXV) return (TY + 1) * BWc + (h - TXV) + 1;
            const int cc = h - 2 * TXV, side = cc / TY, r = cc - side * TY;
            return (r + 1) * BWc + (side ? TXV + 1 : 0);
        };
        const int extra0 = (NCT - 1 - tid < nextra) ? halo_cell(NCT - 1 - tid) : -1;   // this thread's halo cell
        auto cell_d = [&](int c) -> int { const int row = c / BWc; return row * L.bwd + (c - row * BWc) * VEC; };
        const int extra0_d = (PALD && extra0 >= 0) ? cell_d(extra0) : 0;
        int lead_d = 0;                                // PALD: bytes between the Dinv-index box's aligned start and x0 - VEC
        int qoff = 0;                                  // byte (in a quad box row) and field offset of this thread's nodes
        int qfield = 0;

        // {Dinv, D} of the VEC nodes whose index bytes start at p
        auto decode_dd = [&](const unsigned char *p, Vec<T> &dinv, Vec<T> &D) {
            const uint32_t w = (VEC == 4) ? *reinterpret_cast<const uint32_t *>(p)
                                          : (uint32_t)*reinterpret_cast<const unsigned short *>(p);
#pragma unroll
            for (int e = 0; e < VEC; e++) {
                const uint32_t i = (w >> (8 * e)) & 255u;
                if (sizeof(T) == 4) {
                    const float2 v = *reinterpret_cast<const float2 *>(reinterpret_cast<const unsigned char *>(ddtab) + i * 8);
                    dinv.a[e] = (T)v.x; D.a[e] = (T)v.y;
                } else {
                    const double2 v = *reinterpret_cast<const double2 *>(reinterpret_cast<const unsigned char *>(ddtab) + i * 16);
                    dinv.a[e] = (T)v.x; D.a[e] = (T)v.y;
                }
            }
        };
        // VEC face coefficients of this thread's nodes, row `row` of a quad box
        auto coefq = [&](const unsigned char *box, int row) -> Vec<T> {
            const uint32_t b = box[row * L.bwq + qoff];
            return *reinterpret_cast<const Vec<T> *>(reinterpret_cast<const unsigned char *>(qtab) + b * (4 * sizeof(T)) + qfield);
        };
        // p_new = Dinv*r + beta*p_old (steps 6-7) of haloed-box cell c; also Dinv's partner D when asked for
        auto pnew_cell = [&](const unsigned char *slot, int c, int cd, Vec<T> *Dout, Vec<T> *pold_out) -> Vec<T> {
            Vec<T> v = reinterpret_cast<const Vec<T> *>(slot + L.oR)[c];
            if (MODE == 0) {
                const Vec<T> pv = reinterpret_cast<const Vec<T> *>(slot + L.oPp)[c];
                if (pold_out) *pold_out = pv;
                Vec<T> dv, D;
                if (PALD) {
                    decode_dd(slot + L.oDv + lead_d + cd, dv, D);
                } else {
                    dv = reinterpret_cast<const Vec<T> *>(slot + L.oDv)[c];
                    if (Dout) {
#pragma unroll
                        for (int e = 0; e < VEC; e++) D.a[e] = rcp_rn(dv.a[e]);
                    }
                }
                if (Dout) *Dout = D;
                if (precond) {
#pragma unroll
                    for (int e = 0; e < VEC; e++) v.a[e] = fma(beta, pv.a[e], dv.a[e] * v.a[e]);
                } else {
#pragma unroll
                    for (int e = 0; e < VEC; e++) v.a[e] = fma(beta, pv.a[e], v.a[e]);
                }
            }
            return v;
        };

        int rs = 0;                                    // ring slot of the next item and its phase parity
        uint32_t rp = 0;
        auto advance = [&]() { rs = (rs + 1 == NS) ? 0 : rs + 1; rp ^= (rs == 0); };
        const uint32_t slot_bytes = (uint32_t)L.slot;
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
            qoff = (i0 >> 2) - ((x0 >> 2) & ~15);
            qfield = (i0 & 3) * (int)sizeof(T);
            size_t idx = ((size_t)k0 * ny + j) * P + i0;

            // update of the plane in slot `sl` that becomes plane kk of the march: own p_new (returned), and -- for a
            // plane this tile writes -- the haloed p_new box into PN[kk & 1], the deferred phi update, and D
            auto update = [&](const unsigned char *sl, int kk, bool centre, Vec<T> &Dout, size_t xidx) -> Vec<T> {
                Vec<T> v = zerov<T>();
                Vec<T> *PN = reinterpret_cast<Vec<T> *>(pnbase + (size_t)(kk & 1) * L.pn);
                if (intile) {
                    Vec<T> po;
                    v = pnew_cell(sl, own, own_d, centre ? &Dout : nullptr, &po);
                    if (centre) {
                        PN[own] = v;
                        if (MODE == 0 && active) {
                            // phi_{l-1} = phi_{l-2} + alpha_{l-1} p_{l-2}  (step 5 of the previous iteration)
                            Vec<T> xv = reinterpret_cast<const Vec<T> *>(sl + L.oX)[cown];
#pragma unroll
                            for (int e = 0; e < VEC; e++) xv.a[e] = fma(alpha_prev, po.a[e], xv.a[e]);
                            stv(a.x + xidx, xv);
                        }
                        if (MODE == 1) {
                            if (PALD) { Vec<T> dv; decode_dd(sl + L.oDv + lead_d + own_d, dv, Dout); }
                            else {
                                const Vec<T> dv = reinterpret_cast<const Vec<T> *>(sl + L.oDv)[own];
#pragma unroll
                                for (int e = 0; e < VEC; e++) Dout.a[e] = rcp_rn(dv.a[e]);
                            }
                        }
                    }
                }
                if (centre) {
                    if (extra0 >= 0) PN[extra0] = pnew_cell(sl, extra0, extra0_d, nullptr, nullptr);
                    for (int h = NCT - 1 - tid + NCT; h < nextra; h += NCT) {      // only when the halo outnumbers the threads
                        const int c = halo_cell(h);
                        PN[c] = pnew_cell(sl, c, PALD ? cell_d(c) : 0, nullptr, nullptr);
                    }
                }
                return v;
            };

            // item k0-1: only the own column's value is needed
            Vec<T> Dc = zerov<T>(), Dn = zerov<T>();
            mbar_wait(&full_bar[rs], rp);
            Vec<T> pm = update(base + rs * slot_bytes, k0 - 1, false, Dn, idx);
            __syncwarp();
            named_bar_sync(1, NCT);                   // every consumer has read the slot (and is done with the previous tile)
            if (tid == 0) mbar_arrive(&empty_bar[rs]);
            advance();
            // item k0
            int sk = rs;
            mbar_wait(&full_bar[sk], rp);
            const unsigned char *slotk = base + sk * slot_bytes;
            Vec<T> pc = update(slotk, k0, true, Dc, idx);
            Vec<T> ezc = intile ? coefq(slotk + L.oEZ, ty) : zerov<T>();
            advance();
            named_bar_sync(1, NCT);

            for (int k = k0; k < k1; k++, idx += plane) {
                const int s1 = rs;
                mbar_wait(&full_bar[s1], rp);
                const unsigned char *slot1 = base + s1 * slot_bytes;
                const Vec<T> pn = update(slot1, k + 1, k + 1 < k1, Dn, idx + plane);
                const Vec<T> ezn = intile ? coefq(slot1 + L.oEZ, ty) : zerov<T>();
                if (active) {
                    const Vec<T> *Zk = reinterpret_cast<const Vec<T> *>(pnbase + (size_t)(k & 1) * L.pn);   // p_new(k) box
                    const Vec<T> up = Zk[own - BWc], dn = Zk[own + BWc];
                    const T left = Zk[own - 1].a[VEC - 1], right = Zk[own + 1].a[0];
                    const Vec<T> exl = coefq(slotk + L.oEXM, ty), exh = coefq(slotk + L.oEXP, ty);
                    const Vec<T> eyl = coefq(slotk + L.oEY, ty), eyh = coefq(slotk + L.oEY, ty + 1);
                    Vec<T> ap;
#pragma unroll
                    for (int e = 0; e < VEC; e++) {
                        const T pl = (e == 0) ? left : pc.a[e == 0 ? 0 : e - 1];
                        const T pr = (e == VEC - 1) ? right : pc.a[e == VEC - 1 ? e : e + 1];
                        // two short FMA chains instead of one of seven (latency), summed at the end; same order of
                        // operations as k_spmv_tma
                        T v = Dc.a[e] * pc.a[e];
                        v = fma(-exl.a[e], pl, v);
                        v = fma(-exh.a[e], pr, v);
                        v = fma(-eyl.a[e], up.a[e], v);
                        T w = -eyh.a[e] * dn.a[e];
                        w = fma(-ezc.a[e], pm.a[e], w);
                        w = fma(-ezn.a[e], pn.a[e], w);
                        v += w;
                        if (e >= nvalid) v = T(0);     // pad column
                        if (MODE == 0) acc = fma((double)pc.a[e], (double)v, acc);
                        ap.a[e] = (MODE == 1) ? (T)((double)v * a.out_scale) : v;
                    }
                    stv(a.Ap + idx, ap);
                    if (MODE == 0) stv(pout + idx, pc);
                }
                named_bar_sync(1, NCT);   // p_new(k+1) box complete; everyone is done with slot sk and with p_new(k)
                if (tid == 0) mbar_arrive(&empty_bar[sk]);
                pm = pc; pc = pn; ezc = ezn; Dc = Dn; sk = s1; slotk = slot1;
                advance();
            }
            // item k1: only its own-column values were used, by the update of the last step -- every consumer read
            // them before that step's barrier, so the slot goes back right away
            if (tid == 0) mbar_arrive(&empty_bar[sk]);
        }
    }

    if (MODE == 0) {
        const double tot = block_sum(acc, red);
        const int nblk = gridDim.x;
        if (tid == 0) {
            a.partials[blockIdx.x] = tot;
            __threadfence();
            const unsigned int t = atomicAdd(&a.st->ticket_spmv, 1u);
            s_last = (t == (unsigned int)(nblk - 1));
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            const double pAp = final_sum(a.partials, nblk, red);
            if (tid == 0) {
                State *st = a.st;
                st->ticket_spmv = 0u;
                st->pAp = pAp;
                if (!(pAp > 0.0) || !isfinite(pAp)) {          // breakdown: not SPD / NaN
                    if (st->latch) { st->done = 1; st->iters = st->iter_cur; st->status = 5; }
                    st->alpha = 0.0;                            // x already holds the last good iterate
                } else {
                    st->alpha = st->rz / pAp;                   // step 5
                }
            }
        }
    }
}

}  // namespace pb
