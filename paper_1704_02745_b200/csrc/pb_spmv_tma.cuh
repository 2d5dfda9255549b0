// pb_spmv_tma.cuh -- K_spmv, the dominant kernel of the PCG iteration, as a persistent,
// warp-specialised TMA pipeline for sm_100a.
//
// Computes:  z = Dinv*r (step 6, Jacobi) ; p <- z + beta*p (step 7) ;
// x += alpha_prev * p_old (the phi update of step 5, deferred by one kernel) ; Ap = A'p ; partial p.Ap
// (step 5), with A' rebuilt on the fly from the face dielectrics of Eq. 3 and
// D = 1/Dinv.  z is never stored: 10 words per node (reads r, Dinv, p, x, eps_x, eps_y, eps_z;
// writes p, x, Ap) against k_vec's 4 -- the 14-word split of SURVEY.md section 8(d).
//
// Structure.  A tile is TXV 16-byte vectors x TY rows x TZ planes.  Blocks are persistent and
// stride over the tile list.  One producer lane streams "items" (one z-plane of the tile each)
// through an NS-deep shared-memory ring with cp.async.bulk.tensor (TMA) and mbarriers:
//     item q = { r(q), Dinv(q), p_old(q) boxes with a 1-row / 1-vector halo,  ezm(q),  x(q), exm(q), eym(q) }
// Out-of-range box elements are zero-filled by the TMA unit: that is the ghost layer p = 0.
// The consumer warps turn the r box into p_new = Dinv*r + beta*p_old in place (halo included:
// the neighbours' p_new is recomputed, never re-read), keep the k-1/k/k+1 values of their own
// column in registers, take the in-plane neighbours from the ring, and write Ap and p_new with
// 128-bit stores.  One named barrier per plane among the consumers; no __syncthreads in the loop.
#pragma once
#include "pb_internal.cuh"
#include "pb_tma.cuh"

namespace pb {

constexpr int kMaxStages = 8;

__device__ __forceinline__ float rcp_rn(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double rcp_rn(double x) { return __drcp_rn(x); }

template <typename T>
struct TmaArgs {
    T *pbuf0, *pbuf1;        // iteration l reads buf[l&1] (through its tensor map), writes buf[(l+1)&1]
    T *Ap;
    T *x;                    // phi, updated with the previous iteration's alpha (MODE 0)
    int nx, ny, nz, P;
    int TXV, TY, TZ;
    int ntx, nty, ntz, ntiles;
    int nstage;
    int precond;             // 1: M = diag(A) (Jacobi); 0: M = I (plain CG)
    int zoff;                // z-slab mode: the haloed tensors (r, Dinv, p) start one GHOST plane below plane 0
    int l2hints;             // 1: evict_last on r/Dinv/Ap (re-read by k_vec), evict_first on the streamed arrays
    State *st;
    double *partials;        // one per block
    double out_scale;        // MODE 1 only
    const T *lut;            // PAL only: palette values (256 entries)
    const T *dlut;           // PALD only: the distinct values of Dinv (256 entries)
};

__host__ __device__ inline int spmv_row_threads(int TXV) { return (TXV + 7) & ~7; }   // consumer threads per tile row
__host__ __device__ inline size_t align128(size_t v) { return (v + 127) & ~(size_t)127; }

// byte sizes of the boxes of one item (also the smem carve-up of a ring slot).  With a coefficient
// palette the three face boxes hold one byte per face, rows of `bw` bytes (a multiple of 16 for the TMA).
struct SlotLayout {
    size_t szZ, szD, szEX, szEY, szEZ, szDv, slot;
    size_t oR, oDv, oPp, oEZ, oX, oEX, oEY;   // offsets of the boxes inside a slot
    uint32_t bZ, bD, bEX, bEY, bEZ, bDv;      // exact box bytes (what the TMA delivers)
    int bw;                                   // palette only: bytes per row of a face-index box
    int bwd;                                  // diagonal palette only: bytes per row of the haloed Dinv-index box
};
__host__ __device__ inline SlotLayout slot_layout(int TXV, int TY, int pal_vec /* 0: no palette, else VEC */,
                                                  bool pald = false) {
    SlotLayout L;
    L.bZ = (uint32_t)(TY + 2) * (TXV + 2) * 16;
    L.bD = (uint32_t)TY * TXV * 16;
    L.bwd = pald ? ((TXV + 2) * pal_vec + 16 + 15) / 16 * 16 : 0;
    L.bDv = pald ? (uint32_t)(TY + 2) * L.bwd : L.bZ;
    if (pal_vec) {
        L.bw = (TXV * pal_vec + 16 + 15) / 16 * 16;   // box starts at x0 rounded down to 16 B: up to 16-VEC bytes of lead-in
        L.bEX = (uint32_t)TY * L.bw; L.bEY = (uint32_t)(TY + 1) * L.bw; L.bEZ = (uint32_t)TY * L.bw;
    } else {
        L.bw = 0;
        L.bEX = (uint32_t)TY * (TXV + 1) * 16; L.bEY = (uint32_t)(TY + 1) * TXV * 16; L.bEZ = L.bD;
    }
    L.szZ = align128(L.bZ); L.szD = align128(L.bD); L.szEX = align128(L.bEX);
    L.szEY = align128(L.bEY); L.szEZ = align128(L.bEZ); L.szDv = align128(L.bDv);
    L.oR = 0; L.oDv = L.szZ; L.oPp = L.oDv + L.szDv;
    L.oEZ = L.oPp + L.szZ; L.oX = L.oEZ + L.szEZ; L.oEX = L.oX + L.szD; L.oEY = L.oEX + L.szEX;
    L.slot = L.oEY + L.szEY;
    return L;
}

// MODE 0: PCG step;  MODE 1: y = out_scale * A' v  (v behind tm_r; no Dinv scaling, no p_old, no x, no dot)
// PAL: the eps_x/eps_y/eps_z maps are byte-index tensors decoded through the 256-entry table a.lut
// PALD (with PAL): Dinv too is a byte-index tensor (haloed box), decoded through a.dlut; D = 1/Dinv from a second
// table built at kernel start with the same correctly rounded reciprocal
template <typename T, int MODE, bool PAL, bool PALD>
__global__ void __launch_bounds__(512)
k_spmv_tma(const __grid_constant__ CUtensorMap tm_r, const __grid_constant__ CUtensorMap tm_dinv,
           const __grid_constant__ CUtensorMap tm_p0, const __grid_constant__ CUtensorMap tm_p1,
           const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_ex,
           const __grid_constant__ CUtensorMap tm_ey, const __grid_constant__ CUtensorMap tm_ez,
           const TmaArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[kMaxStages];
    __shared__ __align__(8) uint64_t empty_bar[kMaxStages];
    __shared__ double red[32];
    __shared__ int s_last;
    __shared__ T lut[PAL ? 256 : 1];
    __shared__ T lutDinv[PALD ? 256 : 1];
    __shared__ T lutD[PALD ? 256 : 1];

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
    const SlotLayout L = slot_layout(TXV, TY, PAL ? VEC : 0, PALD);
    // 128-byte aligned ring base; plain pointer arithmetic on the __shared__ symbol keeps the address space known
    // to the compiler (LDS/STS instead of generic LD/ST)
    unsigned char *base = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);

    if (tid == 0) {
        for (int s = 0; s < NS; s++) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], NCW); }
        mbar_fence_init();
    }
    if (PAL)
        for (int i = tid; i < 256; i += nthr) lut[i] = a.lut[i];
    if (PALD)
        for (int i = tid; i < 256; i += nthr) { const T d = a.dlut[i]; lutDinv[i] = d; lutD[i] = rcp_rn(d); }
    __syncthreads();

    double acc = 0.0;
    if (is_producer) {
        if (lane == 0) {
            const uint64_t pol_keep = l2_policy((a.l2hints & 1) ? 2 : 0), pol_stream = l2_policy((a.l2hints & 2) ? 1 : 0),
                           pol_pold = l2_policy((a.l2hints & 4) ? 1 : 0);
            int s = 0;                                  // ring slot of the next item and its phase parity
            uint32_t ph = 0;
            for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
                int b = tile;
                const int bx = b % a.ntx; b /= a.ntx;
                const int by = b % a.nty;
                const int bz = b / a.nty;
                const int x0 = bx * TXV * VEC, j0 = by * TY;
                const int k0 = bz * TZ, k1 = min(k0 + TZ, nz);
                for (int q = k0 - 1; q <= k1; q++, s = (s + 1 == NS) ? 0 : s + 1, ph ^= (s == 0)) {
                    mbar_wait(&empty_bar[s], ph ^ 1);
                    unsigned char *slot = base + s * (uint32_t)L.slot;
                    const bool centre = (q >= k0) && (q < k1);   // q is a plane this tile writes
                    const bool ez = (q >= k0);
                    uint32_t bytes = (MODE == 0) ? 2 * L.bZ + L.bDv : L.bZ;
                    if (ez) bytes += L.bEZ;
                    if (centre) bytes += L.bEX + L.bEY + (MODE == 0 ? L.bD : L.bDv);
                    const int xd = PALD ? ((x0 - VEC) & ~15) : x0 - VEC;   // byte-index box: 16-byte aligned start
                    mbar_expect_tx(&full_bar[s], bytes);
                    const int qh = q + a.zoff;                  // plane of the haloed tensors (ghost plane = plane 0 in slab mode)
                    tma_load_3d_hint(slot + L.oR, &tm_r, x0 - VEC, j0 - 1, qh, &full_bar[s], pol_keep);
                    if (MODE == 0) {
                        tma_load_3d_hint(slot + L.oDv, &tm_dinv, xd, j0 - 1, qh, &full_bar[s], pol_keep);
                        tma_load_3d_hint(slot + L.oPp, tm_pin, x0 - VEC, j0 - 1, qh, &full_bar[s], pol_pold);
                    } else if (centre) {
                        tma_load_3d_hint(slot + L.oDv, &tm_dinv, xd, j0 - 1, qh, &full_bar[s], pol_keep);
                    }
                    const int xc = PAL ? (x0 & ~15) : x0;      // byte-index boxes start 16-byte aligned
                    if (ez) tma_load_3d_hint(slot + L.oEZ, &tm_ez, xc, j0, q, &full_bar[s], pol_stream);
                    if (centre) {
                        if (MODE == 0) tma_load_3d_hint(slot + L.oX, &tm_x, x0, j0, q, &full_bar[s], pol_stream);
                        tma_load_3d_hint(slot + L.oEX, &tm_ex, xc, j0, q, &full_bar[s], pol_stream);
                        tma_load_3d_hint(slot + L.oEY, &tm_ey, xc, j0, q, &full_bar[s], pol_stream);
                    }
                }
            }
        }
        __syncwarp();
    } else {
        const int BWc = TXV + 2;                       // vectors per row of the haloed boxes
        // a tile row takes a multiple of 8 threads: a quarter-warp (one 128-byte shared-memory wavefront of a 16-byte
        // access) then never straddles two rows of the haloed boxes, whose 2-vector gap would make it a bank conflict
        const int TXP = spmv_row_threads(TXV);
        const int tx = tid % TXP, ty = tid / TXP;
        const bool intile = ty < TY && tx < TXV;
        const int own = (ty + 1) * BWc + tx + 1;       // own cell in the haloed boxes
        const int own_d = (ty + 1) * L.bwd + (tx + 1) * VEC;   // PALD: its byte offset in the Dinv-index box
        int lead_d = 0;                                // PALD: bytes between that box's aligned start and x0 - VEC
        const int cown = ty * TXV + tx;                // own cell in the x / ezm / eym boxes
        const int nextra = 2 * TXV + 2 * TY;           // halo cells: two rows, two columns
        const bool precond = a.precond != 0;
        const uint64_t pol_keep = l2_policy((a.l2hints & 1) ? 2 : 0), pol_stream = l2_policy((a.l2hints & 2) ? 1 : 0);

        // halo cell h of the haloed boxes: two rows (above / below the tile), then two columns (left / right)
        auto halo_cell = [&](int h) -> int {
            if (h < TXV) return h + 1;
            if (h < 2 * TXV) return (TY + 1) * BWc + (h - TXV) + 1;
            const int cc = h - 2 * TXV, side = cc / TY, r = cc - side * TY;
            return (r + 1) * BWc + (side ? TXV + 1 : 0);
        };
        const int extra0 = (NCT - 1 - tid < nextra) ? halo_cell(NCT - 1 - tid) : -1;   // this thread's halo cell
        auto cell_d = [&](int c) -> int { const int row = c / BWc; return row * L.bwd + (c - row * BWc) * VEC; };
        const int extra0_d = (PALD && extra0 >= 0) ? cell_d(extra0) : 0;
        // VEC values of a table selected by the VEC index bytes at p.  The bytes are pre-scaled byte offsets into
        // the table (k_setup_pal_idx): one PRMT and one LDS per value.
        auto entry = [&](const T *table, uint32_t off) -> T {
            return *reinterpret_cast<const T *>(reinterpret_cast<const unsigned char *>(table) + off);
        };
        auto decode = [&](const T *table, const unsigned char *p) -> Vec<T> {
            const uint32_t w = (VEC == 4) ? *reinterpret_cast<const uint32_t *>(p)
                                          : (uint32_t)*reinterpret_cast<const unsigned short *>(p);
            Vec<T> v;
#pragma unroll
            for (int e = 0; e < VEC; e++) v.a[e] = entry(table, __byte_perm(w, 0u, 0x4440u + e));
            return v;
        };
        // p_new = Dinv*r + beta*p_old (steps 6-7) in place in the r box; returns the own cell's p_new
        auto pnew_cell = [&](Vec<T> *R, const Vec<T> *Dv, const Vec<T> *Pp, int c, int cd) -> Vec<T> {
            Vec<T> v = R[c];
            if (MODE == 0) {
                const Vec<T> pv = Pp[c];
                if (precond) {
                    const Vec<T> dv = PALD ? decode(lutDinv, reinterpret_cast<const unsigned char *>(Dv) + lead_d + cd)
                                           : Dv[c];
#pragma unroll
                    for (int e = 0; e < VEC; e++) v.a[e] = fma(beta, pv.a[e], dv.a[e] * v.a[e]);
                } else {
#pragma unroll
                    for (int e = 0; e < VEC; e++) v.a[e] = fma(beta, pv.a[e], v.a[e]);
                }
            }
            return v;
        };
        auto update = [&](unsigned char *slot, bool with_halo) -> Vec<T> {
            Vec<T> *R = reinterpret_cast<Vec<T> *>(slot + L.oR);
            const Vec<T> *Dv = reinterpret_cast<const Vec<T> *>(slot + L.oDv);
            const Vec<T> *Pp = reinterpret_cast<const Vec<T> *>(slot + L.oPp);
            Vec<T> v = zerov<T>();
            if (intile) {
                v = pnew_cell(R, Dv, Pp, own, own_d);
                if (MODE == 0 && with_halo) R[own] = v;
            }
            if (MODE == 0 && with_halo) {
                if (extra0 >= 0) R[extra0] = pnew_cell(R, Dv, Pp, extra0, extra0_d);
                for (int h = NCT - 1 - tid + NCT; h < nextra; h += NCT) {      // only when the halo outnumbers the threads
                    const int c = halo_cell(h);
                    R[c] = pnew_cell(R, Dv, Pp, c, PALD ? cell_d(c) : 0);
                }
            }
            return v;
        };
        // VEC face coefficients starting at this thread's first node, row `row` of a face box
        int lead = 0;                                  // PAL: bytes between the aligned box start and x0
        auto coef = [&](const unsigned char *box, int row, int row_vecs) -> Vec<T> {
            if (!PAL) return reinterpret_cast<const Vec<T> *>(box)[row * row_vecs + tx];
            return decode(lut, box + row * L.bw + lead + tx * VEC);
        };
        auto release = [&](int s) {                    // this warp is done with ring slot s
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[s]);
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
            lead = x0 & 15;
            lead_d = (x0 - VEC) & 15;

            // item k0-1: only the own column's value is needed
            mbar_wait(&full_bar[rs], rp);
            Vec<T> pm = update(base + rs * slot_bytes, false);
            release(rs);
            advance();
            // item k0
            int sk = rs;
            mbar_wait(&full_bar[sk], rp);
            unsigned char *slotk = base + sk * slot_bytes;
            Vec<T> pc = update(slotk, true);
            Vec<T> ezc = intile ? coef(slotk + L.oEZ, ty, TXV) : zerov<T>();
            advance();
            named_bar_sync(1, NCT);

            size_t idx = ((size_t)k0 * ny + j) * P + i0;
            for (int k = k0; k < k1; k++, idx += plane) {
                const int s1 = rs;
                mbar_wait(&full_bar[s1], rp);
                unsigned char *slot1 = base + s1 * slot_bytes;
                const Vec<T> pn = update(slot1, k + 1 < k1);
                const Vec<T> ezn = intile ? coef(slot1 + L.oEZ, ty, TXV) : zerov<T>();
                if (active) {
                    const Vec<T> *Zk = reinterpret_cast<const Vec<T> *>(slotk + L.oR);     // p_new(k) box
                    const Vec<T> up = Zk[own - BWc], dn = Zk[own + BWc];
                    const T left = Zk[own - 1].a[VEC - 1], right = Zk[own + 1].a[0];
                    // D = 1/Dinv (correctly rounded): the diagonal of Eq. 3
                    Vec<T> D;
                    if (PALD) {
                        D = decode(lutD, slotk + L.oDv + lead_d + own_d);
                    } else {
                        const Vec<T> dinv = reinterpret_cast<const Vec<T> *>(slotk + L.oDv)[own];
#pragma unroll
                        for (int e = 0; e < VEC; e++) D.a[e] = rcp_rn(dinv.a[e]);
                    }
                    const Vec<T> ex = coef(slotk + L.oEX, ty, TXV + 1);
                    const T exr = PAL ? entry(lut, slotk[L.oEX + ty * L.bw + lead + tx * VEC + VEC])
                                      : reinterpret_cast<const Vec<T> *>(slotk + L.oEX)[ty * (TXV + 1) + tx + 1].a[0];
                    const Vec<T> eyl = coef(slotk + L.oEY, ty, TXV), eyh = coef(slotk + L.oEY, ty + 1, TXV);
                    Vec<T> ap;
#pragma unroll
                    for (int e = 0; e < VEC; e++) {
                        const T pl = (e == 0) ? left : pc.a[e == 0 ? 0 : e - 1];
                        const T pr = (e == VEC - 1) ? right : pc.a[e == VEC - 1 ? e : e + 1];
                        const T exh = (e == VEC - 1) ? exr : ex.a[e == VEC - 1 ? e : e + 1];
                        // two short FMA chains instead of one of seven (latency), summed at the end
                        T v = D.a[e] * pc.a[e];
                        v = fma(-ex.a[e], pl, v);
                        v = fma(-exh, pr, v);
                        v = fma(-eyl.a[e], up.a[e], v);
                        T w = -eyh.a[e] * dn.a[e];
                        w = fma(-ezc.a[e], pm.a[e], w);
                        w = fma(-ezn.a[e], pn.a[e], w);
                        v += w;
                        if (e >= nvalid) v = T(0);     // pad column: exm[nx] is node nx-1's face, not a row of A
                        if (MODE == 0) acc = fma((double)pc.a[e], (double)v, acc);
                        ap.a[e] = (MODE == 1) ? (T)((double)v * a.out_scale) : v;
                    }
                    st16_hint(a.Ap + idx, ap.a, pol_keep);
                    if (MODE == 0) {
                        st16_hint(pout + idx, pc.a, pol_stream);
                        // phi_{l-1} = phi_{l-2} + alpha_{l-1} p_{l-2}  (step 5 of the previous iteration)
                        Vec<T> xv = reinterpret_cast<const Vec<T> *>(slotk + L.oX)[cown];
                        const Vec<T> po = reinterpret_cast<const Vec<T> *>(slotk + L.oPp)[own];
#pragma unroll
                        for (int e = 0; e < VEC; e++) xv.a[e] = fma(alpha_prev, po.a[e], xv.a[e]);
                        st16_hint(a.x + idx, xv.a, pol_stream);
                    }
                }
                named_bar_sync(1, NCT);   // p_new(k+1) box complete; everyone is done with slot sk
                release(sk);
                pm = pc; pc = pn; ezc = ezn; sk = s1; slotk = slot1;
                advance();
            }
            release(sk);                  // item k1 (only its own-column values were used)
        }
    }

    if (MODE == 0) {
        // stage 1 -> per-block partial; stage 2 by the last block to take a ticket (fixed order: deterministic)
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
                if (st->slab) {
                    // z-slab mode: this is the LOCAL sum; alpha follows in k_slab_alpha after the all-reduce
                } else if (!(pAp > 0.0) || !isfinite(pAp)) {          // breakdown: not SPD / NaN
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
