// pb_fused.cuh -- ONE kernel per PCG iteration: K_spmv with K_vec folded in ("single-reduction PCG").
//
// The two-kernel iteration (K_spmv, K_vec) needs two passes over the grid because step 5's
// alpha needs p.Ap (a reduction over the whole grid) before r can be updated, and step 7's beta needs r_new.z_new (a
// second one) before p can.  Here the residual update of iteration l is DEFERRED into the pass of
// iteration l+1 -- r_l = r_{l-1} - alpha_l A p_l is formed where r and A p_l are staged anyway, halo cells included --
// and every scalar of iteration l+1 comes out of ONE reduction at the end of that pass.  With v = A p_{l+1}:
//     p.Ap = sum p_{l+1} v                                                               (step 5)
//     U1 = sum Dinv r_l^2 = r_l.z_l,   U2 = sum r_l^2                (re-summed EXACTLY from the stored r_l, every pass)
//     alpha_{l+1} = U1 / p.Ap
//     r_{l+1}.z_{l+1} = U1 - 2 alpha S1 + alpha^2 S2,   S2 = sum Dinv v^2,   S1 = z_l.v = p.Ap - beta_l W,
//                                                       W = sum (A p_l) p_{l+1}  (= p_l . A p_{l+1}: A is symmetric)
//     beta_{l+1} = r_{l+1}.z_{l+1} / U1                                                 (step 7)
// These are algebraic expansions of the very dot products K_vec computes, one step deep: U1 is re-summed in every pass,
// so nothing drifts (the classical single-reduction recurrences carry the norms along and lose them after ~1/eps of
// reduction).  W is summed where A p_l and p_{l+1} meet (the update stage), S2 and p.Ap where v is made (the stencil).
// The stopping rule (step 3) is applied to U2, the exact ||r_l||^2 of the stored residual, at the end of
// pass l+1: the solve stops at the same l as the two-kernel path and the oracle, and pays one extra pass per solve
// (x already holds phi_l then: the deferred update x += alpha_l p_l is part of this pass; alpha is zeroed so that
// k_finish adds nothing).  In exact arithmetic the iterates are those of PAPER.md:104-126.
//
// Bytes per node and iteration: reads r, A p_l, p (haloed), x, Dinv, the three faces; writes r, p, x, A p_{l+1}:
// 8 words + 2 index bytes in the quad format with the diagonal palette (34 B fp32, 66 B fp64) instead of 41 / 77 B
// in two kernels; r, p and A p are double-buffered (a neighbouring tile reads the old plane while this one writes).
//
// Structure: k_spmv_batch's (pb_spmv_batch.cuh) -- a vector ring {r, A p_l, p_l haloed, x} released right after the
// update stage, a coefficient ring held one step longer -- with the per-thread state cut to the bone (128 registers,
// two blocks per SM): p_new lives in THREE shared planes (k-1, k, k+1) and is re-read from there instead of being
// rotated through registers (measured: holding the own-cell values in registers costs spills and 8 % of the time); the step is unrolled twice so that D, Dinv and the z-face of
// planes k / k+1 alternate between two register sets without moves; every shared address is a 32-bit slot base plus
// a per-thread offset computed once, the slot-internal offsets come ready-made from the host (FusedArgs, constant
// bank) and the tables / barriers sit at compile-time offsets of the same window (FusedSm), so that nothing of the
// layout is re-derived inside the loop; inactive lanes run the same instructions on in-range cells and are masked
// out of the stores and the sums; the five sums are carried in fp32 over two planes (8 nodes) and then added to the
// thread's fp64 accumulators.
// Measured at 385^3 fp32 (profiles/r2_ncu_full_fused.txt): 651 K SM cycles per launch whatever the instruction count
// (192 M warp instructions before this layout, 145 M with it): the pass runs at 5.8 TB/s of DRAM traffic at 1.93 GHz
// (90 % of the measured copy rate) and follows the SM clock under the power cap (0.364 ms at 1.75 GHz).
#pragma once
#include "pb_internal.cuh"
#include "pb_tma.cuh"
#include "pb_spmv_tma.cuh"
#include "pb_spmv_batch.cuh"
#include "pb_kernels.cuh"

namespace pb {

constexpr int kFusedSums = 5;        // p.Ap, S2, W, U1, U2
constexpr int kFusedPlanes = 3;      // p_new planes k-1, k, k+1

// Slot layout.  The producer warp's TMA issue rate bounds this kernel (measured: leaving out three of nine small boxes
// per plane, 2 % of the bytes, took 7.5 % off the pass), so the boxes of one plane are fetched with as few TMA
// instructions as the tensors allow:
//   vector slot       ONE 4-D box {r, A p, p, x} (all haloed, hy rows): the vectors live in one allocation, buffer
//                     set 0 = (r0, Ap0, p0, x0) followed by set 1, each set four consecutive "members" of a tensor
//                     [4][nz][ny][P]; x is double-buffered like the others (same bytes: one read, one write), so
//                     that the slot looks the same in both parities (State::xbuf names the current x)
//   coefficient slot  the Dinv box (index bytes or words), then -- quad format -- ONE 4-D box {ez, ex-, ex+, ey} of a
//                     tensor [4][nz+1][ny+1][Pq] (TY + 1 rows each), or -- word format -- the three face boxes
struct FusedLayout {
    BatchLayout B;                       // box sizes
    uint32_t bZ, vslot;                  // one haloed vector box; the vector slot (four of them)
    uint32_t bDv, bQ4, oEZ, oEXM, oEXP, oEY, cslot;
    uint32_t pn;
};
__host__ __device__ inline FusedLayout fused_layout(int TXV, int TY, int vec, bool quad, bool pald)
{
    FusedLayout F;
    F.B = batch_layout(TXV, TY, vec, quad, pald);
    F.bZ = F.B.bZ;
    F.vslot = (uint32_t)align128(4 * (size_t)F.bZ);
    F.bDv = F.B.bDv;
    F.oEZ = (uint32_t)align128(F.bDv);
    if (quad) {
        const uint32_t S = (uint32_t)(TY + 1) * (uint32_t)F.B.bwq;   // one array of the merged quad box
        F.bQ4 = 4 * S;
        F.oEXM = F.oEZ + S; F.oEXP = F.oEZ + 2 * S; F.oEY = F.oEZ + 3 * S;
        F.cslot = F.oEZ + (uint32_t)align128(F.bQ4);
    } else {
        F.bQ4 = 0;
        F.oEXM = F.oEZ + (uint32_t)align128(F.B.bEZ);
        F.oEXP = F.oEXM;
        F.oEY = F.oEXM + (uint32_t)align128(F.B.bEXM);
        F.cslot = F.oEY + (uint32_t)align128(F.B.bEY);
    }
    F.pn = (uint32_t)align128(F.bZ);
    return F;
}

// fixed part of the block's shared memory (byte offsets from the 128-byte aligned start of the dynamic window): the
// mbarriers, the reduction scratch, the two lookup tables; the rings and the p_new planes follow at `ring`
template <typename T, bool QUAD, bool PALD>
struct FusedSm {
    static constexpr uint32_t vfull = 0, vempty = 64, cfull = 128, cempty = 160;     // 8 + 8 + 4 + 4 mbarriers
    static constexpr uint32_t red = 256, last = 896;                                 // red: [kFusedSums][16 warps] doubles
    static constexpr uint32_t tq = 904;                                              // 16 tile ids (producer -> consumers)
    static constexpr uint32_t qtab = 1024;                                           // [256][4] face values
    static constexpr uint32_t ddtab = qtab + (QUAD ? 1024u * (uint32_t)sizeof(T) : 0u);   // [256] {Dinv, D}
    static constexpr uint32_t ring = ddtab + (PALD ? 512u * (uint32_t)sizeof(T) : 0u);
};
static_assert(kMaxStages <= 8 && kMaxCoefStages <= 4, "FusedSm reserves 8 + 8 + 4 + 4 mbarriers");
inline size_t fused_fixed_smem(int elt, bool quad, bool pald)
{
    return 1024 + (quad ? (size_t)1024 * elt : 0) + (pald ? (size_t)512 * elt : 0);
}
inline size_t fused_smem(const FusedLayout &F, int nsv, int nsc, int elt, bool quad, bool pald)
{
    return fused_fixed_smem(elt, quad, pald) + (size_t)nsv * F.vslot + (size_t)nsc * F.cslot +
           (size_t)kFusedPlanes * F.pn + 128;
}

template <typename T>
struct FusedArgs {
    T *r0, *r1, *Ap0, *Ap1, *p0, *p1, *x0, *x1;   // iteration with iter_cur = l reads buffer set l & 1, writes the other
    int nx, ny, nz, P;
    int TXV, TY, TZ;
    int ntx, nty, ntz, ntiles;
    int nsv, nsc;
    int precond;
    int nct;                 // consumer threads (whole warps); one more warp produces
    // tiles: `ntiles` static ones over the planes [0, zs), handed out blockIdx.x, + gridDim.x, ...; then `npool` chunks of
    // `pc` planes over [zs, nz), every column again, fetched from a device-wide counter by whichever block runs out of
    // static tiles first (the blocks' speeds differ by several per cent from launch to launch)
    int zs, pc, npool, ncol;
    // the slot layout (fused_layout), bytes: coefficient slot {Dinv @0, ez @oEZ, ex- @oEXM, ex+ @oEXP, ey @oEY}, one
    // p_new plane; box sizes for expect_tx (bQ4: the merged quad box; bEZ, bC: the word-format face boxes)
    uint32_t vslot, cslot, pn, bZ, oEZ, oEXM, oEXP, oEY, bwq, bwd;
    uint32_t bDv, bQ4, bEZ, bC;
    size_t sQ, sP, sX;       // bytes from a cell of r to the same cell of A p, p, x in the written buffer set
    State *st;
    double *partials;        // [kFusedSums][ntiles + npool]: the sums of every tile
    const T *lut;
    const T *dlut;
};
template <typename T>
inline void fused_args_layout(FusedArgs<T> &a, const FusedLayout &F)
{
    const BatchLayout &L = F.B;
    a.vslot = F.vslot; a.cslot = F.cslot; a.pn = F.pn; a.bZ = F.bZ;
    a.oEZ = F.oEZ; a.oEXM = F.oEXM; a.oEXP = F.oEXP; a.oEY = F.oEY;
    a.bwq = (uint32_t)L.bwq; a.bwd = (uint32_t)L.bwd;
    a.bDv = F.bDv; a.bQ4 = F.bQ4; a.bEZ = L.bEZ; a.bC = L.bEXM + L.bEY;
}

// tile id -> column (bx, by) and plane range [k0, k1)
template <typename T>
__device__ __forceinline__ void fused_tile(const FusedArgs<T> &a, int t, int &bx, int &by, int &k0, int &k1)
{
    if (t < a.ntiles) {
        bx = t % a.ntx; t /= a.ntx;
        by = t % a.nty;
        k0 = (t / a.nty) * a.TZ;
        k1 = min(k0 + a.TZ, a.zs);
    } else {
        t -= a.ntiles;
        const int col = t % a.ncol;
        bx = col % a.ntx; by = col / a.ntx;
        k0 = a.zs + (t / a.ncol) * a.pc;
        k1 = min(k0 + a.pc, a.nz);
    }
}

// the two vector tensors ([4][nz][ny][P]: buffer set 0, buffer set 1) in one kernel parameter
struct FusedMaps { CUtensorMap set0, set1; };

template <typename T, bool QUAD, bool PALD>
__global__ void __launch_bounds__(512)
k_pcg_fused(const __grid_constant__ FusedMaps vm, const __grid_constant__ CUtensorMap tm_dinv,
            const __grid_constant__ CUtensorMap tm_q4, const __grid_constant__ CUtensorMap tm_exm,
            const __grid_constant__ CUtensorMap tm_ey, const __grid_constant__ CUtensorMap tm_ez, const FusedArgs<T> a)
{
    constexpr int VEC = VecN<T>::value;
    constexpr uint32_t ES = (uint32_t)sizeof(T);
    using SM = FusedSm<T, QUAD, PALD>;
    extern __shared__ __align__(128) unsigned char smem_raw[];

    const int tid = threadIdx.x;
    const int NCT = a.nct;
    const int warp = tid >> 5, lane = tid & 31;
    const bool is_producer = (warp == (NCT >> 5));

    if (a.st->done) return;
    const T beta = (T)a.st->beta;              // beta_l:  p_{l+1} = z_l + beta_l p_l
    const T alpha = (T)a.st->alpha;            // alpha_l: r_l = r_{l-1} - alpha_l A p_l,  phi_l = phi_{l-1} + alpha_l p_l
    const int parity = a.st->iter_cur & 1;

    // sb: shared-window address of the block's 128-byte aligned area; gb: the same place as a generic pointer
    const uint32_t sb = (smem_u32(smem_raw) + 127u) & ~127u;
    unsigned char *const gb = smem_raw + (sb - smem_u32(smem_raw));
    double *const red = reinterpret_cast<double *>(gb + SM::red);
    int *const s_last = reinterpret_cast<int *>(gb + SM::last);
    const uint32_t sm_v = sb + SM::ring;                           // vector ring
    const uint32_t sm_c = sm_v + (uint32_t)a.nsv * a.vslot;        // coefficient ring
    const uint32_t sm_pn = sm_c + (uint32_t)a.nsc * a.cslot;       // the three p_new planes

    if (tid == 0) {
        for (int i = 0; i < a.nsv; i++) { mbar_init_a(sb + SM::vfull + 8u * i, 1); mbar_init_a(sb + SM::vempty + 8u * i, NCT >> 5); }
        for (int i = 0; i < a.nsc; i++) { mbar_init_a(sb + SM::cfull + 8u * i, 1); mbar_init_a(sb + SM::cempty + 8u * i, 1); }
        mbar_fence_init();
    }
    if (QUAD) {
        T *qtab = reinterpret_cast<T *>(gb + SM::qtab);            // qtab[b][f] = lut[(b >> 2f) & 3]: four face values per byte
        for (int b = tid; b < 256; b += blockDim.x) {
#pragma unroll
            for (int f = 0; f < 4; f++) qtab[b * 4 + f] = a.lut[(b >> (2 * f)) & 3];
        }
    }
    if (PALD) {
        T *ddtab = reinterpret_cast<T *>(gb + SM::ddtab);          // {Dinv, D} pairs
        for (int i = tid; i < 256; i += blockDim.x) { const T d = a.dlut[i]; ddtab[2 * i] = d; ddtab[2 * i + 1] = rcp_rn(d); }
    }
    __syncthreads();

    double a_pAp = 0.0, a_S2 = 0.0, a_W = 0.0, a_U1 = 0.0, a_U2 = 0.0;
    const int nx = a.nx, ny = a.ny, nz = a.nz, P = a.P;
    const int TXV = a.TXV, TY = a.TY, TZ = a.TZ;

    if (is_producer) {
        // the whole warp runs the loop (uniform control flow: coordinates, addresses and byte counts stay in uniform
        // registers, no per-thread waterfall around the TMA instructions); lane 0 issues
        {
            const bool leader = lane == 0;
            int vs = 0, cs = 0;
            uint32_t vph = 0, cph = 0;
            const CUtensorMap *tv = parity ? &vm.set1 : &vm.set0;
            int next_static = blockIdx.x;
            for (uint32_t seq = 0;; seq++) {
                int tile = -1;
                if (next_static < a.ntiles) { tile = next_static; next_static += gridDim.x; }
                else if (a.npool > 0) {
                    unsigned int c = 0;
                    if (leader) c = atomicAdd(&a.st->pool_ctr, 1u);
                    c = __shfl_sync(0xffffffffu, c, 0);
                    if (c < (unsigned int)a.npool) tile = a.ntiles + (int)c;
                }
                // the tile id reaches the consumers with the first item of the tile (the arrive below releases it)
                if (leader) asm volatile("st.shared.s32 [%0], %1;" ::"r"(sb + SM::tq + 4u * (seq & 15u)), "r"(tile) : "memory");
                if (tile < 0) {                                        // end marker: an item without data
                    const uint32_t full = sb + SM::cfull + 8u * cs;
                    mbar_wait_a(full + (SM::cempty - SM::cfull), cph ^ 1);
                    if (leader) mbar_arrive_a(full);
                    break;
                }
                int bx, by, k0, k1;
                fused_tile(a, tile, bx, by, k0, k1);
                const int x0 = bx * TXV * VEC, j0 = by * TY;
                const int xd = PALD ? ((x0 - VEC) & ~15) : x0 - VEC;   // byte-index box: 16-byte aligned start
                const int xq = QUAD ? ((x0 >> 2) & ~15) : x0;          // quad-index boxes likewise
                for (int q = k0 - 1; q <= k1; q++) {
                    const bool centre = (q >= k0) && (q < k1);
                    const bool ez = (q >= k0);
                    {   // coefficient item q: Dinv, and from plane k0 on the faces (ex, ey go unused at q = k1)
                        const uint32_t full = sb + SM::cfull + 8u * cs, slot = sm_c + (uint32_t)cs * a.cslot;
                        mbar_wait_a(full + (SM::cempty - SM::cfull), cph ^ 1);
                        if (leader) {
                            if (QUAD) {
                                mbar_expect_tx_a(full, a.bDv + (ez ? a.bQ4 : 0u));
                                tma_load_3d_a(slot, &tm_dinv, xd, j0 - 1, q, full);
                                if (ez) tma_load_4d_a(slot + a.oEZ, &tm_q4, xq, j0, q, 0, full);
                            } else {
                                mbar_expect_tx_a(full, a.bDv + (ez ? a.bEZ : 0u) + (centre ? a.bC : 0u));
                                tma_load_3d_a(slot, &tm_dinv, xd, j0 - 1, q, full);
                                if (ez) tma_load_3d_a(slot + a.oEZ, &tm_ez, xq, j0, q, full);
                                if (centre) {
                                    tma_load_3d_a(slot + a.oEXM, &tm_exm, xq, j0, q, full);
                                    tma_load_3d_a(slot + a.oEY, &tm_ey, xq, j0, q, full);
                                }
                            }
                        }
                        cs = (cs + 1 == a.nsc) ? 0 : cs + 1; cph ^= (cs == 0);
                    }
                    {   // vector item q: one box {r, A p, p, x} of the buffer set this pass reads
                        const uint32_t full = sb + SM::vfull + 8u * vs, slot = sm_v + (uint32_t)vs * a.vslot;
                        mbar_wait_a(full + (SM::vempty - SM::vfull), vph ^ 1);
                        if (leader) {
                            mbar_expect_tx_a(full, 4u * a.bZ);
                            tma_load_4d_a(slot, tv, x0 - VEC, j0 - 1, q, 0, full);
                        }
                        vs = (vs + 1 == a.nsv) ? 0 : vs + 1; vph ^= (vs == 0);
                    }
                }
            }
        }
        __syncwarp();
    } else {
        // ---- consumer warps ---------------------------------------------------------------------------------
        const uint32_t BWc = (uint32_t)TXV + 2u;       // vectors per row of the haloed boxes
        const int TXP = spmv_row_threads(TXV);
        const int tx0 = tid % TXP, ty0 = tid / TXP;
        const bool intile = ty0 < TY && tx0 < TXV;
        // lanes outside the tile run the same instructions on cell (0, 0) of the tile and are masked out below
        const int tx = intile ? tx0 : 0, ty = intile ? ty0 : 0;
        const uint32_t t_own = ((uint32_t)(ty + 1) * BWc + (uint32_t)tx + 1u) * 16u;   // own cell in a haloed box / p_new plane
        const uint32_t t_c = (uint32_t)(ty * TXV + tx) * 16u;                          // own cell in an un-haloed box
        const uint32_t oQ = a.bZ, oP = 2u * a.bZ, oX = 3u * a.bZ;                      // the vector slot holds (r, A p, p, x)
        // halo cells (two rows, two columns): one per thread, from the last thread down (the host sizes the block so
        // that the consumer threads cover them: nct >= 2 TXV + 2 TY)
        const int nextra = 2 * TXV + 2 * TY;
        auto halo_cell = [&](int h) -> int {
            if (h < TXV) return h + 1;
            if (h < 2 * TXV) return (TY + 1) * (int)BWc + (h - TXV) + 1;
            const int cc = h - 2 * TXV, side = cc / TY, r = cc - side * TY;
            return (r + 1) * (int)BWc + (side ? TXV + 1 : 0);
        };
        auto cell_d = [&](int c) -> uint32_t { const int row = c / (int)BWc; return (uint32_t)row * a.bwd + (uint32_t)(c - row * (int)BWc) * VEC; };
        const int extra0 = (NCT - 1 - tid < nextra) ? halo_cell(NCT - 1 - tid) : -1;
        const bool has_x0 = extra0 >= 0;
        const uint32_t t_dx = has_x0 ? (uint32_t)extra0 * 16u - t_own : 0u;            // the halo cell, relative to the own cell
        const bool precond = a.precond != 0;
        // the buffer set this pass writes: r at out0, then A p, p, x at the constant strides of the allocation
        char *const out0 = reinterpret_cast<char *>(parity ? a.r0 : a.r1);
        // per tile (the aligned starts of the byte boxes depend on x0): offsets within a coefficient slot
        uint32_t t_dv = 0, t_dvx = 0, t_ez = 0, t_exm = 0, sbq = sb;

        // Dinv and D = 1/Dinv of VEC nodes: index bytes at `addr` -> pair table, or Dinv words at `addr`
        auto load_dinv = [&](uint32_t addr, Vec<T> &dinv, Vec<T> &D) {
            if (PALD) {
                const uint32_t w = (VEC == 4) ? lds_u32(addr) : lds_u16(addr);
#pragma unroll
                for (int e = 0; e < VEC; e++)
                    lds_pair_o<SM::ddtab>(dinv.a[e], D.a[e], sb + __byte_perm(w, 0u, 0x4440u | (uint32_t)e) * (2u * ES));
            } else {
                lds_vec(dinv.a, addr);
#pragma unroll
                for (int e = 0; e < VEC; e++) D.a[e] = rcp_rn(dinv.a[e]);
            }
            if (!precond) {                                            // M = I: z = r (1 * r is exact)
#pragma unroll
                for (int e = 0; e < VEC; e++) dinv.a[e] = T(1);
            }
        };
        // VEC face coefficients: quad byte at `addr` -> table of quadruples, or words at `addr`
        auto coef = [&](uint32_t addr) -> Vec<T> {
            Vec<T> v;
            if (QUAD) lds_vec_o<SM::qtab>(v.a, sbq + lds_u8(addr) * (4u * ES));
            else lds_vec(v.a, addr);
            return v;
        };

        // ring heads: slot index, phase parity and the slot's shared address, advanced together
        int vs = 0, cs = 0;
        uint32_t vph = 0, cph = 0;
        const size_t plane_b = (size_t)ny * (size_t)P * sizeof(T);     // bytes per plane
        // fp32: the sums over (at most) two planes, then added to the fp64 accumulators (flush); fp64: the thread's sums
        // themselves (inactive lanes are masked where they are formed)
        constexpr bool F32 = sizeof(T) == 4;
        T s_pv = T(0), s_dvv = T(0), s_w = T(0), s_u1 = T(0), s_u2 = T(0);

        for (uint32_t seq = 0;; seq++) {
            // the producer's tile sequence: its id comes with the first item of the tile
            mbar_wait_a(sb + SM::cfull + 8u * cs, cph);
            int tile;
            asm volatile("ld.shared.s32 %0, [%1];" : "=r"(tile) : "r"(sb + SM::tq + 4u * (seq & 15u)));
            if (tile < 0) break;
            int bx, by, k0, k1;
            fused_tile(a, tile, bx, by, k0, k1);
            const int x0 = bx * TXV * VEC, j0 = by * TY;
            const int i0 = x0 + tx * VEC, j = j0 + ty;
            const bool active = intile && (i0 < P) && (j < ny);
            const int nvalid = active ? nx - i0 : 0;   // inactive lanes: A p = 0 (their Dinv may be a zero-filled 0, D = inf)
            if (PALD) {
                const uint32_t lead_d = (uint32_t)(x0 - VEC) & 15u;
                t_dv = lead_d + (uint32_t)(ty + 1) * a.bwd + (uint32_t)(tx + 1) * VEC;
                t_dvx = has_x0 ? lead_d + cell_d(extra0) : 0u;
            } else {
                t_dv = t_own;
                t_dvx = t_own + t_dx;
            }
            if (QUAD) {
                const uint32_t t_q = (uint32_t)ty * a.bwq + (uint32_t)((i0 >> 2) - ((x0 >> 2) & ~15));
                sbq = sb + (uint32_t)(i0 & 3) * ES;                    // fp64: which half of the quadruple
                t_ez = t_q;                                            // + a.oEZ / oEXM / oEXP / oEY where it is used
            } else {
                t_ez = t_c;
                t_exm = a.oEXM + t_c + (uint32_t)ty * 16u;             // rows of TXV + 1 vectors
            }
            const uint32_t ey_row = QUAD ? a.bwq : (uint32_t)TXV * 16u;
            // this thread's cell of plane k in the written r array (inactive lanes never use it)
            char *po = out0 + (size_t)(uint32_t)((k0 * ny + j) * P + i0) * sizeof(T);
            // own-cell addresses in the three p_new planes: plane q lives in buffer q mod 3, rotated as the march advances
            uint32_t pn_m = sm_pn + t_own, pn_c = pn_m + a.pn, pn_n = pn_c + a.pn;

            // "update" of the plane at the ring heads -> p_new plane whose own-cell address is `pnw`:
            // r_l = r_{l-1} - alpha_l A p_l, p_{l+1} = Dinv r_l + beta_l p_l on the own cell (returned; always stored into the plane)
            // and, for a plane this tile writes (centre), on the halo cells; r_l stored; the deferred phi update; the sums
            // U1, U2, W.  The vector slot is handed back; the coefficient slot stays (its address is returned).
            auto update = [&](uint32_t pnw, bool centre, bool want_ez, char *pout, Vec<T> &pnew, Vec<T> &Dout, Vec<T> &dvout,
                              Vec<T> &ezout) -> uint32_t {
                mbar_wait_a(sb + SM::cfull + 8u * cs, cph);
                const uint32_t cslot = sm_c + (uint32_t)cs * a.cslot;
                Vec<T> dvh, dummy;
                load_dinv(cslot + t_dv, dvout, Dout);
                if (centre && has_x0) load_dinv(cslot + t_dvx, dvh, dummy);
                if (want_ez) ezout = coef(cslot + t_ez + a.oEZ);
                mbar_wait_a(sb + SM::vfull + 8u * vs, vph);
                const uint32_t sl = sm_v + (uint32_t)vs * a.vslot + t_own;
                Vec<T> rl, qv, pv;
                lds_vec(rl.a, sl);
                lds_vec(qv.a, sl + oQ);
                lds_vec(pv.a, sl + oP);
#pragma unroll
                for (int e = 0; e < VEC; e++) {
                    rl.a[e] = fma(-alpha, qv.a[e], rl.a[e]);                   // r_l (the deferred step 5)
                    pnew.a[e] = fma(beta, pv.a[e], dvout.a[e] * rl.a[e]);      // p_{l+1} (steps 6-7)
                }
                sts_vec(pnw, pnew.a);
                if (centre) {
                    Vec<T> xv;
                    lds_vec(xv.a, sl + oX);
#pragma unroll
                    for (int e = 0; e < VEC; e++) xv.a[e] = fma(alpha, pv.a[e], xv.a[e]);   // phi_l = phi_{l-1} + alpha_l p_l
                    if (F32 || active) {
#pragma unroll
                        for (int e = 0; e < VEC; e++) {
                            s_u1 = fma(dvout.a[e] * rl.a[e], rl.a[e], s_u1);    // r_l.z_l
                            s_u2 = fma(rl.a[e], rl.a[e], s_u2);                 // ||r_l||^2
                            s_w = fma(qv.a[e], pnew.a[e], s_w);                 // (A p_l).p_{l+1}
                        }
                    }
                    if (active) {
                        stv(reinterpret_cast<T *>(pout), rl);
                        stv(reinterpret_cast<T *>(pout + a.sX), xv);
                    }
                    if (has_x0) {
                        const uint32_t h0 = sl + t_dx;
                        Vec<T> r2, q2, p2;
                        lds_vec(r2.a, h0);
                        lds_vec(q2.a, h0 + oQ);
                        lds_vec(p2.a, h0 + oP);
#pragma unroll
                        for (int e = 0; e < VEC; e++) {
                            r2.a[e] = fma(-alpha, q2.a[e], r2.a[e]);
                            r2.a[e] = fma(beta, p2.a[e], dvh.a[e] * r2.a[e]);
                        }
                        sts_vec(pnw + t_dx, r2.a);
                    }
                }
                consume(pnew.a[0]);         // r, A p and p of the own cell have been read (x, halo: the stores above)
                __syncwarp();
                if (lane == 0) mbar_arrive_o<SM::vempty>(sb + 8u * vs);
                vs++;
                if (vs == a.nsv) { vs = 0; vph ^= 1u; }
                return cslot;
            };
            auto cnext = [&]() { cs++; if (cs == a.nsc) { cs = 0; cph ^= 1u; } };

            // the stencil of plane k: p_new(k) from plane buffer pc_a (own cell, in-plane neighbours), p_new(k-1) from pm_a,
            // p_new(k+1) = pn (fresh from the update); coefficient slot cslotk; D, Dinv, ez of plane k and ez of plane k+1
            auto stencil = [&](uint32_t cslotk, uint32_t pm_a, uint32_t pc_a, const Vec<T> &pn, const Vec<T> &D, const Vec<T> &dv,
                               const Vec<T> &ezc, const Vec<T> &ezn, char *pout) {
                Vec<T> pc, pm, up, dn, exh;
                T left, right;
                lds_vec(pc.a, pc_a);
                lds_vec(pm.a, pm_a);
                lds_vec(up.a, pc_a - BWc * 16u);
                lds_vec(dn.a, pc_a + BWc * 16u);
                lds_one_o<-(int)sizeof(T)>(left, pc_a);
                lds_one_o<16>(right, pc_a);
                const Vec<T> exl = coef(QUAD ? cslotk + t_ez + a.oEXM : cslotk + t_exm);
                if (QUAD) {
                    exh = coef(cslotk + t_ez + a.oEXP);
                } else {
                    T exr;
                    lds_one_o<16>(exr, cslotk + t_exm);                // the plus face of this vector's last node
#pragma unroll
                    for (int e = 0; e < VEC; e++) exh.a[e] = (e == VEC - 1) ? exr : exl.a[e == VEC - 1 ? e : e + 1];
                }
                const Vec<T> eyl = coef(cslotk + t_ez + a.oEY), eyh = coef(cslotk + t_ez + a.oEY + ey_row);
                Vec<T> ap;
#pragma unroll
                for (int e = 0; e < VEC; e++) {
                    const T pl = (e == 0) ? left : pc.a[e == 0 ? 0 : e - 1];
                    const T pr = (e == VEC - 1) ? right : pc.a[e == VEC - 1 ? e : e + 1];
                    // same order of operations as k_spmv_tma
                    T v = D.a[e] * pc.a[e];
                    v = fma(-exl.a[e], pl, v);
                    v = fma(-exh.a[e], pr, v);
                    v = fma(-eyl.a[e], up.a[e], v);
                    T w = -eyh.a[e] * dn.a[e];
                    w = fma(-ezc.a[e], pm.a[e], w);
                    w = fma(-ezn.a[e], pn.a[e], w);
                    ap.a[e] = v + w;
                }
                if (nvalid < VEC) {                    // pad columns (and inactive lanes): A p = 0
#pragma unroll
                    for (int e = 0; e < VEC; e++) if (e >= nvalid) ap.a[e] = T(0);
                }
                if (F32 || active) {
#pragma unroll
                    for (int e = 0; e < VEC; e++) {
                        s_pv = fma(pc.a[e], ap.a[e], s_pv);
                        s_dvv = fma(dv.a[e] * ap.a[e], ap.a[e], s_dvv);
                    }
                }
                if (active) {
                    stv(reinterpret_cast<T *>(pout + a.sQ), ap);
                    stv(reinterpret_cast<T *>(pout + a.sP), pc);
                }
            };
            // the two-plane sums -> the thread's fp64 accumulators
            auto flush = [&]() {
                if (F32) {
                    if (active) {
                        a_pAp += (double)s_pv; a_S2 += (double)s_dvv; a_W += (double)s_w; a_U1 += (double)s_u1; a_U2 += (double)s_u2;
                    }
                    s_pv = T(0); s_dvv = T(0); s_w = T(0); s_u1 = T(0); s_u2 = T(0);
                }
            };

            Vec<T> Da, Db, dva, dvb, eza, ezb, pnv;
            // item k0-1: the own column's p_new(k0-1) into plane buffer m; its coefficient slot goes back after a barrier
            {
                const uint32_t c0 = sb + SM::cempty + 8u * cs;
                update(pn_m, false, false, po, pnv, Da, dva, eza);
                cnext();
                named_bar_sync(1, NCT);
                if (tid == 0) mbar_arrive_a(c0);
            }
            // item k0 -> plane buffer c;  D, Dinv, ez of plane k0 in set a
            int csk = cs;                                       // the coefficient slot of plane k
            update(pn_c, true, true, po, pnv, Da, dva, eza);
            cnext();
            named_bar_sync(1, NCT);

            // one step: update plane k+1 (set `n`), stencil of plane k (set `c`), barrier, hand the coefficient slot back
            auto step = [&](int k, Vec<T> &Dc, Vec<T> &dvc, Vec<T> &ezc, Vec<T> &Dn, Vec<T> &dvn, Vec<T> &ezn) {
                const int cs1 = cs;
                update(pn_n, k + 1 < k1, true, po + plane_b, pnv, Dn, dvn, ezn);
                cnext();
                stencil(sm_c + (uint32_t)csk * a.cslot, pn_m, pn_c, pnv, Dc, dvc, ezc, ezn, po);
                named_bar_sync(1, NCT);   // p_new(k+1) complete; everyone is done with coefficient slot csk and plane buffer m
                if (tid == 0) mbar_arrive_o<SM::cempty>(sb + 8u * (uint32_t)csk);
                csk = cs1;
                const uint32_t t = pn_m; pn_m = pn_c; pn_c = pn_n; pn_n = t;
                po += plane_b;
            };
            int k = k0;
            for (; k + 1 < k1; k += 2) {
                step(k, Da, dva, eza, Db, dvb, ezb);
                step(k + 1, Db, dvb, ezb, Da, dva, eza);
                flush();
            }
            if (k < k1) step(k, Da, dva, eza, Db, dvb, ezb);
            flush();
            // coefficient item k1: only Dinv and ez of the own column were used, before the last barrier
            if (tid == 0) mbar_arrive_o<SM::cempty>(sb + 8u * (uint32_t)csk);
            // the five sums of THIS TILE -> partials[q][tile] (consumer warps in warp order): the value does not depend on
            // which block ran the tile, so the result of the pass is the same whatever the dynamic schedule was
            {
                if (!F32) {
                    a_pAp = (double)s_pv; a_S2 = (double)s_dvv; a_W = (double)s_w; a_U1 = (double)s_u1; a_U2 = (double)s_u2;
                    s_pv = T(0); s_dvv = T(0); s_w = T(0); s_u1 = T(0); s_u2 = T(0);
                }
                const double sums[kFusedSums] = {a_pAp, a_S2, a_W, a_U1, a_U2};
#pragma unroll
                for (int q = 0; q < kFusedSums; q++) {
                    const double t = warp_sum(sums[q]);
                    if (lane == 0) red[q * 16 + warp] = t;
                }
                named_bar_sync(1, NCT);
                if (tid < kFusedSums) {
                    double t = 0.0;
                    for (int w = 0; w < (NCT >> 5); w++) t += red[tid * 16 + w];
                    a.partials[(size_t)tid * (size_t)(a.ntiles + a.npool) + tile] = t;
                    __threadfence();
                }
                a_pAp = 0.0; a_S2 = 0.0; a_W = 0.0; a_U1 = 0.0; a_U2 = 0.0;
            }
        }
    }

    // stage 2 by the last block to take a ticket: warp q adds the tiles' partials of sum q in tile order (deterministic,
    // and independent of the grid size and of the dynamic schedule); then every scalar of the iteration (header) and
    // the stopping rule of step 3
    const int nblk = gridDim.x;
    const int nwarp = (int)(blockDim.x >> 5);
    __syncthreads();
    if (tid == 0) {
        const unsigned int t = atomicAdd(&a.st->ticket_spmv, 1u);
        *s_last = (t == (unsigned int)(nblk - 1));
    }
    __syncthreads();
    if (*s_last) {
        __threadfence();
        const int ntot = a.ntiles + a.npool;
        for (int q = warp; q < kFusedSums; q += nwarp) {
            const double *pq = a.partials + (size_t)q * ntot;
            double v = 0.0;
            for (int i = lane; i < ntot; i += 32) v += __ldcg(pq + i);
            v = warp_sum(v);
            if (lane == 0) red[q] = v;
        }
        __syncthreads();
        double sum[kFusedSums];
#pragma unroll
        for (int q = 0; q < kFusedSums; q++) sum[q] = red[q];
        if (tid == 0) {
            State *st = a.st;
            st->ticket_spmv = 0u;
            st->pool_ctr = 0u;
            const double pAp = sum[0], S2 = sum[1], W = sum[2], U1 = sum[3], U2 = sum[4];
            const int l = st->iter_cur;                         // this pass formed r_l and phi_l
            st->pAp = pAp;
            st->rz = U1;                                        // r_l.z_l and ||r_l||^2 of the stored r_l, exactly
            st->rr = U2;
            st->alpha = 0.0;                                    // unless another iteration follows: x = phi_l is final
            st->xbuf = parity ^ 1;                              // ... and sits in the buffer set this pass wrote
            if (st->latch && (!isfinite(U1) || !isfinite(U2))) { st->done = 1; st->iters = l; st->status = 5; }
            else if (st->latch && (st->bb == 0.0 || U2 < st->tol2 * st->bb)) { st->done = 1; st->iters = l; st->status = 0; }  // step 3
            else if (st->latch && l >= st->maxiter) { st->done = 1; st->iters = l; st->status = 6; }
            else if (!(pAp > 0.0) || !isfinite(pAp)) {          // breakdown: not SPD / NaN; x holds the last good iterate
                if (st->latch) { st->done = 1; st->iters = l; st->status = 5; }
            } else {
                const double al = U1 / pAp;                     // step 5
                const double S1 = pAp - st->beta * W;           // z_l.A p_{l+1}
                double rz_new = fma(al, fma(al, S2, -2.0 * S1), U1);   // r_{l+1}.z_{l+1}
                if (rz_new < 0.0) rz_new = 0.0;                 // cancellation at the rounding floor
                st->alpha = al;
                st->beta = rz_new / U1;                         // step 7
                st->iter_cur = l + 1;                           // step 4
            }
        }
    }
}

}  // namespace pb
