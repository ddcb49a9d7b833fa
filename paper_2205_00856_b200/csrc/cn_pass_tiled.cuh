// Tiled pass kernel for sm_100a: the hot path.
//
// One CTA owns a tile of TPB*8 consecutive points = a whole number of blocks.  The tile of psi, of the
// stored inverse pivots q and of gamma is brought in by three TMA tensor loads (cp.async.bulk.tensor,
// SASS UTMALDG) from 2-D views [N/8][8 points] with the 128-byte (64-byte for gamma) shared-memory
// swizzle, so that HBM sees only full-line coalesced traffic while thread t can read "its" row of
// 8 consecutive points conflict-free: that is the transposition from the paper's "conventional layout"
// to one contiguous chunk per thread.  The new psi leaves through the same swizzled
// buffer with one TMA tensor store (UTMASTG).
//
// Inside a block the RD / RU sweeps are first-order linear recurrences.  A thread
// sweeps its 8 points serially; the chunks of one block are chained by the affine-map scan of
// cn_common.cuh (warp shuffles carry the interface values).  A joint line resets the recurrence
// (A = 0), so blocks stay independent exactly as in the paper.
//
//   P1 (finish step k):  E = scaled T^dagger psi (Eq. 3) -> RD with the new support value of the joint
//                        above as inflow -> RU + SS with the support value of the own joint -> new psi.
//   P2 (start step k+1): E of the new psi -> RD, RU with zero support values -> JD / JU contributions
//                        slotD[w], slotU[w-1] (two slots per joint line instead of atomics).
//
// gamma is NOT read: mu_i = p_i + q_{i-1} with p_i = 1 / q_i (the block-local pivot recurrence, cn_factor.cuh), so
// gamma_i = -Re(1 / q_i + q_{i-1}) costs one real reciprocal per point (at a block's first row mu_f = 1 / q_f; on a
// joint line, where q := 1 is stored, gamma comes from the O(P) array gamJ).  HBM bytes moved per point of a fused pass:
// psi in 16 + q 16 + psi out 16 = 48, against the 56 of the formulation that also stores gamma (SURVEY 8d's minimum).
#pragma once
#include <cuda.h>
#include "cn_common.cuh"

struct cn_true { static constexpr bool value = true; };
struct cn_false { static constexpr bool value = false; };

struct cn_tiled_params {
    int64_t nchunks; // chunks (8 points) in the array the tensor maps describe: N / 8, or one streamed part of it
    int64_t chunk0;  // global index of its first chunk (0 unless psi is streamed part by part, ooc_* in cn_api.cu)
    int64_t P;
    int64_t cutMask; // ~0: one system.  k - 1 (k a power of two): the array holds independent systems of k blocks each
                     // (cn_plan_set_systems): a block whose index is a multiple of k has the virtual joint line "psi = 0"
                     // above it, exactly like block 0 of a single system (reading R8)
    double rho;
    const cplx *psi_raw; // prologue only: old psi for the tile's left halo (same array as tmPsi)
    const cplx *supOld;  // psi^k   at the joint lines (RS output of the previous step)
    const cplx *supNew;  // psi^k+1 at the joint lines (RS output of this step)
    cplx *slotD, *slotU;
    cplx *supInit; // prologue only: receives psi^0 at the joint lines
    const double *gamJ; // gamma on the joint lines (gamma of every other row is recovered from the stored pivots)
};

CN_DEVINL uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

CN_DEVINL void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
CN_DEVINL void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
CN_DEVINL void mbar_wait(uint64_t *bar, uint32_t phase)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(phase)
            : "memory");
    } while (!done);
}
CN_DEVINL void tma_load_2d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
CN_DEVINL void tma_store_2d(const CUtensorMap *map, const void *src, int c0, int c1)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(map),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1)
                 : "memory");
}
CN_DEVINL void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// shared-memory bytes of one CTA: one in-flight input tile (psi, q, gamma), one output staging tile, scan scratch
template <int TPB>
constexpr size_t tiled_smem_bytes()
{
    return (size_t)TPB * (128 + 128 + 128) + (size_t)(TPB / 32) * (2 * 2 + 2) * sizeof(cplx) + 16;
}

// TPB threads, 8 points per thread, 2^LOGC chunks (threads) per block.  PERSISTENT: CTA b handles tiles
// b, b + gridDim.x, ...; the TMA loads of the next tile are issued as soon as the current tile has been
// copied to registers, so they overlap the whole computation of the current tile.
template <int TPB, int LOGC, bool P1, bool P2, int MINB>
__global__ void __launch_bounds__(TPB, MINB)
k_pass_tiled(const __grid_constant__ CUtensorMap tmPsi, const __grid_constant__ CUtensorMap tmQ,
             const __grid_constant__ CUtensorMap tmGam, const cn_tiled_params prm)
{
    constexpr int CPB = 1 << LOGC;          // chunks per block
    constexpr bool XWARP = (LOGC > 5);      // a block spans several warps
    constexpr int WSTEPS = XWARP ? 5 : LOGC; // shuffle-scan steps inside a warp
    constexpr int NW = TPB / 32;
    constexpr int WPB = XWARP ? (CPB / 32) : 1; // warps per block
    static_assert(CPB <= TPB, "a block must fit in one tile");

    extern __shared__ __align__(1024) uint8_t smem[];
    cplx *const s_psi = (cplx *)smem;
    cplx *const s_q = (cplx *)(smem + (size_t)TPB * 128);
    cplx *const s_out = (cplx *)(smem + (size_t)TPB * 256);
    cplx *const s_scan = (cplx *)(smem + (size_t)TPB * 384); // [2 buffers][A,B][NW]
    cplx *const s_edge = s_scan + 2 * 2 * NW;                // [2][NW] edge exchange between warps
    uint64_t *const bar = (uint64_t *)(s_edge + 2 * NW);

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const double rho = prm.rho;
    const cplx zero = cmake(0.0, 0.0);
    const int64_t ntiles = (prm.nchunks + TPB - 1) / TPB;

    auto issue_loads = [&](int64_t tile) {
        const int64_t r0 = tile * TPB;
        mbar_expect_tx(bar, (uint32_t)(TPB * 256));
#pragma unroll
        for (int r = 0; r < TPB; r += 256) {
            tma_load_2d((uint8_t *)s_psi + (size_t)r * 128, &tmPsi, bar, 0, (int)(r0 + r));
            tma_load_2d((uint8_t *)s_q + (size_t)r * 128, &tmQ, bar, 0, (int)(r0 + r));
        }
    };

    if (t == 0) {
        if ((smem_u32(smem) & 1023u) != 0) __trap(); // the swizzle patterns below assume a 1 KiB aligned base
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if ((int64_t)blockIdx.x < ntiles) issue_loads(blockIdx.x); // psi: written two kernels ago, complete
    }
    pdl_wait();              // the RS kernel before this one has delivered supNew
    pdl_launch_dependents(); // the next RS kernel may become resident as soon as CTAs retire
    __syncthreads();

    uint32_t phase = 0;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t row0 = tile * TPB;
        const int64_t c = row0 + t;         // chunk index inside the array
        const int64_t cg = prm.chunk0 + c;  // global chunk index (chunk0 is a multiple of CPB)
        const bool active = c < prm.nchunks;
        const bool isFirst = (c & (CPB - 1)) == 0;
        const bool isLast = (c & (CPB - 1)) == CPB - 1;
        const int64_t w = cg >> LOGC;
        const bool top = (w & prm.cutMask) == 0;                 // first block of a system
        const bool bottom = ((w + 1) & prm.cutMask) == 0 || w == prm.P - 1; // last block of a system

        // the few values that live on the joint lines (issued before waiting for the tile)
        cplx supN = zero;       // new value of the own joint line (last chunk of a block)
        cplx jointAbove = zero; // new value of the joint line above the block of this thread
        if (P1 && active) {
            if (isLast) supN = prm.supNew[w];
            if (!top) jointAbove = prm.supNew[w - 1];
        }
        double gJ = 2.0; // gamma of the own joint line (last chunk of a block)
        if (active && isLast) gJ = prm.gamJ[w];
        cplx oldAbove = zero; // OLD psi just above the tile (needed by thread 0 only)
        // (prologue of a streamed part: the row above it is a joint line whose psi^0 the previous part recorded)
        if (t == 0 && !top) oldAbove = P1 ? prm.supOld[w - 1] : (c > 0 ? prm.psi_raw[8 * c - 1] : prm.supInit[w - 1]);

        mbar_wait(bar, phase);
        phase ^= 1;

        // ---- registers <- swizzled shared memory ------------------------------------------------------
        cplx v[8], qv[8];
        double g[8];
        const int sw = t & 7;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            v[j] = s_psi[t * 8 + (j ^ sw)];
            qv[j] = s_q[t * 8 + (j ^ sw)];
        }
        cplx vlo = oldAbove, vhi = zero, qm1 = cmake(1.0, 0.0); // the row above a tile is a joint line
        if (t > 0) {
            vlo = s_psi[(t - 1) * 8 + (7 ^ ((t - 1) & 7))];
            qm1 = s_q[(t - 1) * 8 + (7 ^ ((t - 1) & 7))];
        }
        // gamma_j = -Re(mu_j), mu_j = 1 / q_j + q_{j-1}; nothing is subtracted at a block's first row (its pivot is mu_f)
        // (the lanes beyond the end of the array hold q = 0: `pad` keeps their reciprocal finite, the unpredicated scans
        // multiply what those lanes hold by A = 0)
        const double pad = active ? 0.0 : 1.0;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const double qpx = (j == 0) ? (isFirst ? 0.0 : qm1.x) : qv[j - 1].x;
            const double r = rcp_pos(fma(qv[j].x, qv[j].x, fma(qv[j].y, qv[j].y, pad)));
            g[j] = -fma(qv[j].x, r, qpx);
        }
        if (isLast) g[7] = gJ;
        if (t < TPB - 1) vhi = s_psi[(t + 1) * 8 + ((t + 1) & 7)];
        if (isFirst && top) vlo = zero;       // nothing above the first row of a system
        if (!P1 && isFirst) jointAbove = vlo; // prologue: psi^0 of the joint above

        // everybody has its copy: refill the input buffers with the next tile while this one is computed.
        // The refill is a write of the ASYNC proxy (TMA); a CTA barrier alone orders only generic-proxy accesses, and
        // shared-memory loads still queued in the LSU when the barrier opens were overtaken by a fast (L2-resident)
        // TMA write: wrong halo values in the first chunks of a tile, about once in 20 calls at N = 2^21, m = 8.
        // fence.proxy.async orders this thread's earlier generic reads before the later async-proxy writes.
        fence_proxy_async();
        __syncthreads();
        if (t == 0 && tile + gridDim.x < ntiles) issue_loads(tile + gridDim.x);

        // chunk multipliers: Qp = prod_{j<7} (-q_j);  RD map A = (-q_{-1}) Qp,  RU map A = Qp (-q_7)
        cplx Qp = cneg(qv[0]);
#pragma unroll
        for (int j = 1; j < 7; ++j) Qp = cmul(Qp, cneg(qv[j]));
        const cplx fwdA = isLast ? zero : cmul(cneg(qm1), Qp);
        const cplx bwdA = isLast ? zero : cmul(Qp, cneg(qv[7]));

        // exclusive inflow of a forward (RD) chain; tin = value on the joint line above the block.
        // Across the warps of one block the per-warp maps are composed by a second shuffle scan that every
        // warp of the block runs redundantly on the WPB aggregates (no serial chain, one barrier).
        auto scan_fwd = [&](cplx A, cplx B, cplx tin, int buf, auto zin) -> cplx {
            constexpr bool ZEROIN = decltype(zin)::value;
            warp_scan_affine<+1, WSTEPS>(A, B, lane);
            cplx carry = tin;
            if (XWARP) {
                cplx *sA = s_scan + buf * 2 * NW, *sB = sA + NW;
                if (lane == 31) {
                    sA[warp] = A;
                    sB[warp] = B;
                }
                __syncthreads();
                const int vb = warp & ~(WPB - 1); // first warp of this block
                cplx wA = cmake(1.0, 0.0), wB = zero;
                if (lane < WPB) {
                    wA = sA[vb + lane];
                    wB = sB[vb + lane];
                }
                warp_scan_affine<+1, (LOGC > 5 ? LOGC - 5 : 0)>(wA, wB, lane);
                const int src = warp - vb - 1; // composite of warps vb .. warp-1
                cplx cA = shfl_c(wA, src < 0 ? 0 : src), cB = shfl_c(wB, src < 0 ? 0 : src);
                if (src >= 0) carry = cfma(cA, tin, cB);
            }
            cplx Be = shfl_up_c(B, 1);
            cplx r = Be;
            if (XWARP || !ZEROIN) { // with nothing entering the block the composed A is never needed (dead code)
                cplx Ae = shfl_up_c(A, 1);
                r = cfma(Ae, carry, Be);
            }
            return (lane == 0) ? carry : r;
        };
        // exclusive inflow of a backward (RU) chain; nothing enters a block from below (joint resets)
        auto scan_bwd = [&](cplx A, cplx B, int buf) -> cplx {
            warp_scan_affine<-1, WSTEPS>(A, B, lane);
            cplx carry = zero;
            if (XWARP) {
                cplx *sA = s_scan + buf * 2 * NW, *sB = sA + NW;
                if (lane == 0) {
                    sA[warp] = A;
                    sB[warp] = B;
                }
                __syncthreads();
                const int vb = warp & ~(WPB - 1);
                cplx wA = cmake(1.0, 0.0), wB = zero;
                if (lane < WPB) {
                    wA = sA[vb + lane];
                    wB = sB[vb + lane];
                }
                warp_scan_affine<-1, (LOGC > 5 ? LOGC - 5 : 0)>(wA, wB, lane);
                const int src = warp - vb + 1; // composite of warps warp+1 .. last, applied to 0
                cplx cB = shfl_c(wB, src > 31 ? 31 : src);
                if (src < WPB) carry = cB;
            }
            cplx Be = shfl_down_c(B, 1);
            cplx r = Be;
            if (XWARP) {
                cplx Ae = shfl_down_c(A, 1);
                r = cfma(Ae, carry, Be);
            }
            return (lane == 31) ? carry : r;
        };

        if (P1) {
            // ---- Eq. 3 fused into RD -------------------------------------------------
            cplx E[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                cplx lo = (j == 0) ? vlo : v[j - 1];
                cplx hi = (j == 7) ? vhi : v[j + 1];
                E[j] = rhs_E(g[j], rho, v[j], lo, hi);
            }
            // a block inside one warp: the support value of the joint above enters the block's first chunk directly,
            // so that A = 0 at every chain start and the scan needs no lane predicate (warp_scan_affine_uncond)
            cplx D = (!XWARP && isFirst) ? jointAbove : zero;
#pragma unroll
            for (int j = 0; j < 8; ++j) D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
            if (isLast) D = supN; // the joint line carries its new support value
            cplx in;
            if (XWARP) {
                in = scan_fwd(fwdA, D, jointAbove, 0, cn_false());
            } else {
                cplx A = isFirst ? zero : fwdA;
                warp_scan_affine_uncond<+1, WSTEPS>(A, D);
                in = shfl_up_c(D, 1);
                if (isFirst) in = jointAbove;
            }
            D = in;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
                E[j] = D; // E now holds d after RD
            }
            // ---- RU + SS: x_j = q_j (d_j - x_{j+1}) -----------------------------------------------------
            cplx X = cmul(qv[7], E[7]);
            if (isLast) X = supN;
#pragma unroll
            for (int j = 6; j >= 0; --j) X = cmul(qv[j], csub(E[j], X));
            cplx xin;
            if (XWARP) {
                xin = scan_bwd(bwdA, X, 1);
            } else { // bwdA = 0 on a block's last chunk: every chain of this direction starts with A = 0
                cplx A = bwdA, Bx = X;
                warp_scan_affine_uncond<-1, WSTEPS>(A, Bx);
                xin = shfl_down_c(Bx, 1); // ignored by a block's last chunk
            }
            X = cmul(qv[7], csub(E[7], xin));
            if (isLast) X = supN;
            v[7] = X;
#pragma unroll
            for (int j = 6; j >= 0; --j) {
                X = cmul(qv[j], csub(E[j], X));
                v[j] = X;
            }
            // ---- new psi -> swizzled staging tile -> one TMA tensor store ---------------------------------
            if (t == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); // previous store drained
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 8; ++j) s_out[t * 8 + (j ^ sw)] = v[j];
            fence_proxy_async();
            __syncthreads();
            if (t == 0) {
#pragma unroll
                for (int r = 0; r < TPB; r += 256)
                    tma_store_2d(&tmPsi, (uint8_t *)s_out + (size_t)r * 128, 0, (int)(row0 + r));
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        }

        if (P2) {
            // ---- neighbours of the NEW psi ------------------------------------------------------------
            cplx xlo = shfl_up_c(v[7], 1), xhi = shfl_down_c(v[0], 1);
            if (XWARP) {
                cplx *eLo = s_edge, *eHi = s_edge + NW;
                if (lane == 31) eLo[warp] = v[7];
                if (lane == 0) eHi[warp] = v[0];
                __syncthreads();
                if (lane == 0 && warp > 0) xlo = eLo[warp - 1];
                if (lane == 31 && warp < NW - 1) xhi = eHi[warp + 1];
            }
            if (isFirst) xlo = jointAbove; // also covers lane 0 when blocks do not span warps
            if (isLast) xhi = zero;
            cplx E[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                cplx lo = (j == 0) ? xlo : v[j - 1];
                cplx hi = (j == 7) ? xhi : v[j + 1];
                E[j] = rhs_E(g[j], rho, v[j], lo, hi);
            }
            const cplx EJ = E[7]; // for a last chunk: E of the joint line without its psi_{J+1} term (JD part)
            cplx D = zero;
#pragma unroll
            for (int j = 0; j < 8; ++j) D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
            if (isLast) D = zero;
            cplx in;
            if (XWARP) {
                in = scan_fwd(fwdA, D, zero, 1, cn_true());
            } else {
                cplx A = isFirst ? zero : fwdA;
                warp_scan_affine_uncond<+1, WSTEPS>(A, D);
                in = shfl_up_c(D, 1);
                if (isFirst) in = zero;
            }
            D = in;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
                E[j] = D;
            }
            cplx Y = cmul(qv[7], E[7]);
            if (isLast) Y = zero;
            Y = cmul(qv[6], csub(E[6], Y));
            const cplx yn = Y; // local solution next to the own joint (meaningful for a last chunk)
#pragma unroll
            for (int j = 5; j >= 0; --j) Y = cmul(qv[j], csub(E[j], Y));
            cplx yin;
            if (XWARP) {
                yin = scan_bwd(bwdA, Y, 0);
            } else {
                cplx A = bwdA, By = Y;
                warp_scan_affine_uncond<-1, WSTEPS>(A, By);
                yin = shfl_down_c(By, 1);
                if (isLast) yin = zero;
            }
            if (active) {
                if (isLast) {
                    prm.slotD[w] = csub(EJ, yn);
                    if (bottom) prm.slotU[w] = zero;
                    if (!P1) prm.supInit[w] = v[7];
                }
                if (isFirst && !top) {
                    cplx y0 = cfma(bwdA, yin, Y); // isLast && isFirst: bwdA = 0 and Y is already exact
                    prm.slotU[w - 1] = cneg(cadd(v[0], y0));
                }
            }
        }
    }
    if (P1 && t == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}
