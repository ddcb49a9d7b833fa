// Many-systems sweep (config C4; operator splitting reduces N-D to series of 1-D problems, PAPER.md:74,
// 209-211): nsys independent tridiagonal systems that SHARE the plan's matrix, advanced by one CN step.
//
// Every system is solved entirely on chip, so psi crosses HBM once in and once out (32 B per point).  The
// partition of a system is mapped onto the machine's own levels, the paper's nested scheme
// (Eq. 6) applied downwards:
//     level 0   one thread  = one block of 8 (x-sweep) or 16 (y-sweep) consecutive rows, in registers
//     level 1   one warp    = the blocks of its lanes, interface values carried by warp shuffles
//     level 2   one CTA     = its warps, interface values through shared memory
//     level 3   one cluster = up to 8 CTAs, interface values through distributed shared memory
// At every level the d-side of a sweep restricted to a part is the affine map "value entering the part ->
// value leaving it" (cn_common.cuh); composing the maps of the parts before a part gives its inflow, which is
// the RS + SS of that level.  Because the matrix is shared, the stored factors are the inverse pivots of
// the downward elimination of the WHOLE system (one block per system), kept in registers
// (x) or shared memory (y) for the lifetime of the persistent CTA: they never touch HBM again.
//
//   k_batched_x  rows of a system are contiguous (elem_stride == 1).  psi tiles move by TMA tensor loads /
//                stores with the 128-byte swizzle (the transposition to one chunk per thread, as in
//                cn_pass_tiled.cuh).
//   k_batched_y  systems are interleaved (sys_stride == 1, rows elem_stride apart): a strip of 8 adjacent
//                systems is 128 B wide; thread (g, c) owns 16 rows of column c, so global accesses are
//                whole lines without any transposition.  The strip arrives by TMA (prefetched one strip
//                ahead), the new psi leaves by 128-bit stores straight from registers.
//   k_batched_v_sweep  any N, any strides: one thread per system, in-place serial sweeps (correctness path; also the
//                sweep of systems with a matrix of their own each, cn_plan_set_systems).
#pragma once
#include <cuda.h>
#include "cn_common.cuh"
#include "cn_pass_tiled.cuh"

// ---- cluster helpers ---------------------------------------------------------------------------------
CN_DEVINL uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
CN_DEVINL void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
CN_DEVINL void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// store a complex value into the shared memory of CTA `rank` of this cluster at the address `p` has here
CN_DEVINL void dsmem_store(cplx *p, uint32_t rank, cplx v)
{
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(p)), "r"(rank));
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(remote), "d"(v.x), "d"(v.y) : "memory");
}

// The same store, asynchronous, completing 16 bytes of the transaction count of mbarrier `bar` IN THE DESTINATION
// CTA: the receiver waits on its own mbarrier and needs neither a cluster barrier nor a memory fence.
CN_DEVINL void dsmem_store_signal(cplx *p, uint64_t *bar, uint32_t rank, cplx v)
{
    uint32_t remote, rbar;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(p)), "r"(rank));
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rbar) : "r"(smem_u32(bar)), "r"(rank));
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(remote),
                 "d"(v.x), "d"(v.y), "r"(rbar)
                 : "memory");
}

// plain (non-tensor) bulk copy global -> shared memory, completing `bytes` of the transaction count of `bar`
CN_DEVINL void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
CN_DEVINL void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
CN_DEVINL void tma_store_3d(const CUtensorMap *map, const void *src, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}

struct cn_bx_params {
    int64_t nsys;
    int64_t sys_stride; // complex elements between systems
    double rho;
    const cplx *psi_raw; // halo rows at CTA edges inside a cluster
    const cplx *qB;      // inverse pivots of the whole-system downward elimination
    const double *gam;
};

#define CN_BX_TPB 256
#define CN_BATCHED_NMAX (1 << 20) // largest N for which cn_factorize also keeps whole-system pivots

// shared memory of k_batched_x: two psi tiles, the per-tile B aggregates and mailboxes, and the CONSTANT multipliers of
// every scan step (the matrix is the same for every system and every tile, so the A side of all scans is computed once)
constexpr size_t batched_x_smem_bytes()
{
    return (size_t)CN_BX_TPB * 256                               // s_psi, s_out
           + (size_t)2 * (CN_BX_TPB / 32) * sizeof(cplx)          // s_wB   [2 dirs][NW]
           + (size_t)4 * 8 * sizeof(cplx) + 32                    // s_mailB, s_mailA [2 dirs][8 ranks] each; 4 mbarriers
           + (size_t)10 * CN_BX_TPB * sizeof(cplx)                // s_M [2][4][TPB], s_Ae [2][TPB]
           + (size_t)8 * (CN_BX_TPB / 32) * sizeof(cplx)          // s_wM [2][3][NW], s_cA [2][NW]
           + (size_t)2 * sizeof(cplx);                            // s_halo [2]
}

// 256 threads x 8 points.  LOGC = log2(chunks per system) when a system fits one CTA (CL == 1, several
// systems per tile); CL > 1: one system = CL CTAs of a cluster (LOGC == 8, every CTA chains all its chunks).
//
// Scans: a sweep restricted to a chunk is the affine map x -> A x + B (cn_common.cuh); A depends on the matrix alone.
// All A products of the Kogge-Stone steps -- warp level, warps of a CTA, CTAs of a cluster -- are therefore computed
// ONCE before the tile loop and kept as multipliers (0 where a lane has no partner); per tile a scan step is one
// shuffle of B and one complex fused multiply-add.
template <int LOGC, int CL>
__global__ void __launch_bounds__(CN_BX_TPB, 2)
k_batched_x(const __grid_constant__ CUtensorMap tmPsi, const cn_bx_params prm)
{
    constexpr int TPB = CN_BX_TPB;
    constexpr int CPS = (1 << LOGC) * CL;     // chunks per system
    constexpr int CPB = 1 << LOGC;            // chunks chained inside this CTA
    constexpr int SPT = TPB / CPB;            // systems per tile (CL == 1)
    constexpr bool XWARP = (LOGC > 5);
    constexpr int WSTEPS = XWARP ? 5 : LOGC;
    constexpr int XSTEPS = XWARP ? LOGC - 5 : 0;
    constexpr int NW = TPB / 32;
    constexpr int WPB = XWARP ? (CPB / 32) : 1;
    static_assert(CL == 1 || LOGC == 8, "a cluster chains whole CTAs");

    extern __shared__ __align__(1024) uint8_t smem[];
    cplx *const s_psi = (cplx *)smem;
    cplx *const s_out = (cplx *)(smem + (size_t)TPB * 128);
    cplx *const s_wB = (cplx *)(smem + (size_t)TPB * 256); // [2 dirs][NW]        per-tile B aggregate of every warp
    cplx *const s_mailB = s_wB + 2 * NW;                   // [2 dirs][8 ranks]   per-tile B aggregate of every CTA
    cplx *const s_mailA = s_mailB + 16;                    // [2 dirs][8 ranks]   constant A aggregate of every CTA
    uint64_t *const bar = (uint64_t *)(s_mailA + 16);      // [0] TMA loads, [1] downward mailbox, [2] upward mailbox
    cplx *const s_M = (cplx *)(bar + 4);                   // [2][4][TPB]  multiplier of warp-scan steps 1..4
    cplx *const s_Ae = s_M + 8 * TPB;                      // [2][TPB]     inclusive A of the neighbouring lane
    cplx *const s_wM = s_Ae + 2 * TPB;                     // [2][3][NW]   multipliers of the scan over the warp aggregates
    cplx *const s_cA = s_wM + 6 * NW;                      // [2][NW]      A of the warps of this block before this warp
    cplx *const s_halo = s_cA + 2 * NW;                    // [2]          old psi just above / below this CTA's rows (CL > 1)

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const uint32_t rank = (CL > 1) ? cluster_ctarank() : 0u;
    const int64_t cid = blockIdx.x / CL, ncl = gridDim.x / CL;
    const int64_t ntiles = (CL > 1) ? prm.nsys : (prm.nsys + SPT - 1) / SPT;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    const double rho = prm.rho;
    const int pos = (CL > 1) ? (int)rank * TPB + t : (t & (CPB - 1)); // chunk position inside its system
    const bool sysFirst = pos == 0, sysLast = pos == CPS - 1;
    const int vb = warp & ~(WPB - 1), wl = vb + (lane & (WPB - 1)); // first warp of this block; this lane's warp slot

    // A tile and, inside a cluster, the two halo rows at the CTA edges (old psi: the neighbour CTA stores its new rows
    // only after it has received this CTA's aggregates of that tile, which are sent after the loads have landed); the
    // halos travel with the tile, one tile ahead, so no global load sits on the critical path of a tile.
    auto issue_load = [&](int64_t tile) {
        if (CL > 1) {
            mbar_expect_tx(bar, (uint32_t)(TPB * 128) + (rank > 0 ? 16u : 0u) + (rank < CL - 1 ? 16u : 0u));
            tma_load_3d(s_psi, &tmPsi, bar, 0, (int)rank * TPB, (int)tile);
            const cplx *row = prm.psi_raw + tile * prm.sys_stride + (int64_t)rank * (TPB * 8);
            if (rank > 0) bulk_load(s_halo, row - 1, 16u, bar);
            if (rank < CL - 1) bulk_load(s_halo + 1, row + TPB * 8, 16u, bar);
        } else {
            mbar_expect_tx(bar, (uint32_t)(TPB * 128));
            tma_load_3d(s_psi, &tmPsi, bar, 0, 0, (int)(tile * SPT));
        }
    };

    // ---- per-thread constants of the shared matrix: live in registers for the whole kernel -----------
    cplx qv[8];
    double g[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        qv[j] = prm.qB[8 * pos + j];
        g[j] = prm.gam[8 * pos + j];
    }
    const cplx qm1 = sysFirst ? zero : prm.qB[8 * pos - 1];

    if (t == 0) {
        if ((smem_u32(smem) & 1023u) != 0) __trap();
        mbar_init(bar, 1);
        mbar_init(bar + 1, 1);
        mbar_init(bar + 2, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (CL > 1) { // every CTA of the cluster is resident before anything is stored into its shared memory
        cluster_arrive();
        cluster_wait();
    }

    // ---- the A side of every scan, once (the matrix side) --------------------------------------
    cplx M0[2]; // multiplier of warp-scan step 0, in registers; steps 1..4 in s_M
    {
        cplx Qp = cneg(qv[0]);
#pragma unroll
        for (int j = 1; j < 7; ++j) Qp = cmul(Qp, cneg(qv[j]));
        const cplx chunkA[2] = {sysFirst ? zero : cmul(cneg(qm1), Qp),  // nothing enters a system from above
                                sysLast ? zero : cmul(Qp, cneg(qv[7]))}; // ... nor from below (Dirichlet)
#pragma unroll
        for (int di = 0; di < 2; ++di) { // 0: information flows to higher chunks (downward sweep), 1: to lower chunks
            cplx A = chunkA[di];
            M0[di] = zero;
#pragma unroll
            for (int k = 0; k < WSTEPS; ++k) {
                const int d = 1 << k;
                const bool ok = (di == 0) ? (lane >= d) : (lane + d < 32);
                const cplx Mk = ok ? A : zero;
                if (k == 0) M0[di] = Mk;
                else s_M[(di * 4 + k - 1) * TPB + t] = Mk;
                const cplx As = (di == 0) ? shfl_up_c(A, d) : shfl_down_c(A, d);
                if (ok) A = cmul(A, As);
            }
            s_Ae[di * TPB + t] = (di == 0) ? shfl_up_c(A, 1) : shfl_down_c(A, 1);
            cplx aggA = A;
            if (XWARP) {
                if (lane == (di == 0 ? 31 : 0)) s_cA[di * NW + warp] = A; // for now: the aggregate of this warp
                __syncthreads();
                cplx wA = s_cA[di * NW + wl];
#pragma unroll
                for (int k = 0; k < XSTEPS; ++k) {
                    const int d = 1 << k, l = lane & (WPB - 1);
                    const bool ok = (di == 0) ? (l >= d) : (l + d < WPB);
                    if (lane < WPB && warp == vb) s_wM[(di * 3 + k) * NW + wl] = ok ? wA : zero;
                    const cplx As = (di == 0) ? shfl_up_c(wA, d) : shfl_down_c(wA, d);
                    if (ok) wA = cmul(wA, As);
                }
                aggA = shfl_c(wA, di == 0 ? WPB - 1 : 0);
                const int src = (di == 0) ? warp - vb - 1 : warp - vb + 1;
                const bool has = (di == 0) ? (src >= 0) : (src < WPB);
                const cplx xA = shfl_c(wA, has ? src : 0);
                __syncthreads(); // every warp has read the aggregates
                if (lane == 0) s_cA[di * NW + warp] = has ? xA : one;
            }
            if (CL > 1 && warp == 0 && lane < CL) { // the aggregate of this CTA to the CTAs that chain after it
                const bool wants = (di == 0) ? ((uint32_t)lane > rank) : ((uint32_t)lane < rank);
                if (wants) dsmem_store(s_mailA + di * 8 + rank, (uint32_t)lane, aggA);
            }
        }
    }
    pdl_wait(); // psi is the output of the preceding sweep
    pdl_launch_dependents();
    if (t == 0 && cid < ntiles) issue_load(cid);
    if (CL > 1) { // the A aggregates have arrived everywhere
        cluster_arrive();
        cluster_wait();
    } else {
        __syncthreads();
    }

    // value entering this thread's chunk from the chunks before it in direction DIR (B: what leaves the chunk when
    // nothing enters it); per step one shuffle and one complex fused multiply-add against the stored multipliers
    uint32_t xphase = 0;
    auto inflow = [&](auto dirtag, cplx B) -> cplx {
        constexpr int DIR = decltype(dirtag)::value;
        constexpr int di = DIR > 0 ? 0 : 1;
        {
            const cplx Bs = (DIR > 0) ? shfl_up_c(B, 1) : shfl_down_c(B, 1);
            B = cfma(M0[di], Bs, B);
        }
#pragma unroll
        for (int k = 1; k < WSTEPS; ++k) {
            const cplx Bs = (DIR > 0) ? shfl_up_c(B, 1 << k) : shfl_down_c(B, 1 << k);
            B = cfma(s_M[(di * 4 + k - 1) * TPB + t], Bs, B);
        }
        cplx cB = zero; // what enters this warp
        if (XWARP) {
            if (lane == (DIR > 0 ? 31 : 0)) s_wB[di * NW + warp] = B;
            __syncthreads();
            cplx wB = s_wB[di * NW + wl];
#pragma unroll
            for (int k = 0; k < XSTEPS; ++k) {
                const cplx Bs = (DIR > 0) ? shfl_up_c(wB, 1 << k) : shfl_down_c(wB, 1 << k);
                wB = cfma(s_wM[(di * 3 + k) * NW + wl], Bs, wB);
            }
            const int src = (DIR > 0) ? warp - vb - 1 : warp - vb + 1;
            const bool has = (DIR > 0) ? (src >= 0) : (src < WPB);
            const cplx xB = shfl_c(wB, has ? src : 0);
            if (has) cB = xB;
            if (CL > 1) {
                // level 3: the aggregates travel by asynchronous DSMEM stores that signal the receiver's mbarrier: a
                // CTA waits only for the CTAs it depends on, never for the whole cluster.  A sender can never be a
                // whole tile ahead of a receiver: it needs that receiver's aggregate of the opposite direction to
                // finish its own tile.
                const cplx aggB = shfl_c(wB, DIR > 0 ? WPB - 1 : 0);
                cplx *mA = s_mailA + di * 8, *mB = s_mailB + di * 8;
                uint64_t *mb = bar + 1 + di;
                if (warp == 0 && lane < CL) {
                    const bool wants = (DIR > 0) ? ((uint32_t)lane > rank) : ((uint32_t)lane < rank);
                    if (wants) dsmem_store_signal(mB + rank, mb, (uint32_t)lane, aggB);
                }
                const int nsend = (DIR > 0) ? (int)rank : CL - 1 - (int)rank;
                if (nsend > 0) mbar_wait(mb, xphase);
                cplx cin = zero;
                if (DIR > 0) {
                    for (int u = 0; u < (int)rank; ++u) cin = cfma(mA[u], cin, mB[u]);
                } else {
                    for (int u = CL - 1; u > (int)rank; --u) cin = cfma(mA[u], cin, mB[u]);
                }
                cB = cfma(s_cA[di * NW + warp], cin, cB);
            }
        }
        const cplx Be = (DIR > 0) ? shfl_up_c(B, 1) : shfl_down_c(B, 1);
        const bool first = (DIR > 0) ? (lane == 0) : (lane == 31);
        return first ? cB : cfma(s_Ae[di * TPB + t], cB, Be);
    };

    uint32_t phase = 0;
    for (int64_t tile = cid; tile < ntiles; tile += ncl) {
        cplx vlo = zero, vhi = zero;
        if (CL > 1 && t == 0) { // arm this tile's mailboxes: 16 bytes (B) from every CTA this one depends on
            if (rank > 0) mbar_expect_tx(bar + 1, rank * 16u);
            if (rank < CL - 1) mbar_expect_tx(bar + 2, (CL - 1 - rank) * 16u);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        if (CL > 1) { // halo rows at the CTA edges inside a cluster
            if (t == 0 && rank > 0) vlo = s_halo[0];
            if (t == TPB - 1 && rank < CL - 1) vhi = s_halo[1];
        }

        cplx v[8];
        const int sw = t & 7;
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = s_psi[t * 8 + (j ^ sw)];
        if (t > 0 && !sysFirst) vlo = s_psi[(t - 1) * 8 + (7 ^ ((t - 1) & 7))];
        if (t < TPB - 1 && !sysLast) vhi = s_psi[(t + 1) * 8 + ((t + 1) & 7)];
        fence_proxy_async(); // generic reads above before the async-proxy refill below (see cn_pass_tiled.cuh)
        __syncthreads();
        if (t == 0 && tile + ncl < ntiles) issue_load(tile + ncl);

        // ---- Eq. 3 fused into the downward sweep -------------------------------------
        cplx E[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            cplx lo = (j == 0) ? vlo : v[j - 1];
            cplx hi = (j == 7) ? vhi : v[j + 1];
            E[j] = rhs_E(g[j], rho, v[j], lo, hi);
        }
        cplx D = zero;
#pragma unroll
        for (int j = 0; j < 8; ++j) D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
        D = inflow(std::integral_constant<int, +1>{}, D);
        if (sysFirst) D = zero;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
            E[j] = D;
        }
        // ---- upward sweep + substitution: x_j = q_j (d_j - x_{j+1}) ------------------------------------
        cplx X = zero;
#pragma unroll
        for (int j = 7; j >= 0; --j) X = cmul(qv[j], csub(E[j], X));
        X = inflow(std::integral_constant<int, -1>{}, X);
        if (sysLast) X = zero;
#pragma unroll
        for (int j = 7; j >= 0; --j) {
            X = cmul(qv[j], csub(E[j], X));
            v[j] = X;
        }
        // ---- new psi -> swizzled staging tile -> one TMA tensor store -------------------------------------
        if (t == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();
#pragma unroll
        for (int j = 0; j < 8; ++j) s_out[t * 8 + (j ^ sw)] = v[j];
        fence_proxy_async();
        __syncthreads();
        if (t == 0) {
            if (CL > 1) tma_store_3d(&tmPsi, s_out, 0, (int)rank * TPB, (int)tile);
            else tma_store_3d(&tmPsi, s_out, 0, 0, (int)(tile * SPT));
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        xphase ^= 1;
    }
    if (t == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    if (CL > 1) { // nobody leaves while a neighbour may still address its shared memory
        cluster_arrive();
        cluster_wait();
    }
}

// =========================================== y-sweep ===================================================
struct cn_by_params {
    int64_t nsys;  // number of systems (columns)
    int64_t pitch; // complex elements between consecutive rows of a system (elem_stride)
    double rho;
    cplx *psi;
    const cplx *qB;
    const double *gam;
};

// padded index of the per-row constants in shared memory: one pad slot per 16 rows, so that the row
// groups of a warp (16 rows apart) broadcast from different banks
CN_DEVINL int by_pad(int l) { return l + (l >> 4); }

// NC = columns (systems) of a strip: 8 (128 B per row) or 4 (64 B per row: twice the rows per CTA at the same tile size,
// so half the CTAs per cluster for a long system).  GPW = 32 / NC row groups per warp.
template <int LOGG, int NC>
struct by_layout {
    static constexpr int G = 1 << LOGG, RC = 16 * G, GPW = 32 / NC, NW = (G / GPW > 0) ? G / GPW : 1;
    static constexpr int L1 = (NC == 8) ? 2 : 3;                               // log2(GPW)
    static constexpr size_t off_q = (size_t)RC * NC * 16;                      // after psi [RC rows][NC columns]
    static constexpr size_t n_q = RC + RC / 16 + 2;                            // logical index row + 1, padded
    static constexpr size_t off_g = off_q + n_q * 16;
    static constexpr size_t n_g = (RC + RC / 16 + 2) & ~(size_t)1;
    static constexpr size_t off_M1 = off_g + n_g * 8;                          // [2 dirs][L1][G]   level-1 multipliers
    static constexpr size_t off_Ae = off_M1 + (size_t)2 * L1 * G * 16;         // [2][G]     inclusive A of the group before
    static constexpr size_t off_aggA = off_Ae + (size_t)2 * G * 16;            // [2][NW]    A aggregate of every warp
    static constexpr size_t off_cA = off_aggA + (size_t)2 * NW * 16;           // [2][NW]    A of the warps before a warp
    static constexpr size_t off_rM = off_cA + (size_t)2 * NW * 16;             // [2][L1][GPW] multipliers over the roles
    static constexpr size_t off_aggB = off_rM + (size_t)2 * L1 * GPW * 16;     // [2][NW][NC] per-strip B aggregates
    static constexpr size_t off_mailA = off_aggB + (size_t)2 * NW * NC * 16;   // [2][8 ranks]
    static constexpr size_t off_mailB = off_mailA + (size_t)2 * 8 * 16;        // [2][8 ranks][NC]
    static constexpr size_t off_bar = off_mailB + (size_t)2 * 8 * NC * 16;
    static constexpr size_t bytes = off_bar + 32; // [0] TMA loads, [1] downward mailbox, [2] upward mailbox
};
template <int LOGG, int NC>
constexpr size_t batched_y_smem_bytes()
{
    return by_layout<LOGG, NC>::bytes;
}

// Thread (g, c): rows 16 g .. 16 g + 15 of this CTA's part of column c of the strip.  lane = c + NC gl,
// g = GPW warp + gl.  G = 2^LOGG row groups per CTA, TPB = NC G threads, CL CTAs per system (CL > 1 needs TPB = 512).
// As in k_batched_x the A side of every scan is computed once per kernel (the matrix is shared by all systems); the
// multipliers of a thread depend on its row group alone, so they are stored per group and broadcast to its NC lanes.
template <int LOGG, int CL, int NC>
__global__ void __launch_bounds__(NC << LOGG, 1) // (two CTAs of 256 threads at 128 registers: slower, measured)
k_batched_y(const __grid_constant__ CUtensorMap tmPsi, const cn_by_params prm)
{
    typedef by_layout<LOGG, NC> LY;
    constexpr int G = LY::G, TPB = NC * G, RC = LY::RC, GPW = LY::GPW, NW = LY::NW, L1 = LY::L1;
    constexpr int KW = (NW + GPW - 1) / GPW; // warps covered by one lane role in the cross-warp scan
    constexpr int BOXR = RC < 256 ? RC : 256;
    static_assert(NC == 8 || NC == 4, "columns per strip");
    static_assert(G >= GPW && TPB <= 512, "32..512 threads");
    static_assert(CL == 1 || TPB == 512, "a cluster chains whole CTAs");

    extern __shared__ __align__(1024) uint8_t smem[];
    cplx *const s_psi = (cplx *)smem;
    cplx *const s_q = (cplx *)(smem + LY::off_q);
    double *const s_g = (double *)(smem + LY::off_g);
    cplx *const s_M1 = (cplx *)(smem + LY::off_M1);
    cplx *const s_Ae = (cplx *)(smem + LY::off_Ae);
    cplx *const s_aggA = (cplx *)(smem + LY::off_aggA);
    cplx *const s_cA = (cplx *)(smem + LY::off_cA);
    cplx *const s_rM = (cplx *)(smem + LY::off_rM);
    cplx *const s_aggB = (cplx *)(smem + LY::off_aggB);
    cplx *const s_mailA = (cplx *)(smem + LY::off_mailA);
    cplx *const s_mailB = (cplx *)(smem + LY::off_mailB);
    uint64_t *const bar = (uint64_t *)(smem + LY::off_bar);

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int c = lane & (NC - 1), gl = lane / NC, g = GPW * warp + gl;
    const uint32_t rank = (CL > 1) ? cluster_ctarank() : 0u;
    // loop control out of special registers and the constant bank alone (unsigned: shifts, no division), so that it can be
    // rematerialised instead of being kept in local memory (see the end of the strip loop)
    const uint32_t cid = blockIdx.x / CL, ncl = gridDim.x / CL;
    const uint32_t nstrips = (uint32_t)((prm.nsys + NC - 1) / NC);
    const int grow0 = (int)rank * RC + 16 * g; // first row of this thread inside its system
    cplx *const gthread = prm.psi + c + (int64_t)grow0 * prm.pitch; // row grow0 of column c of strip 0
    const bool sysFirst = (rank == 0 && g == 0), sysLast = (rank == CL - 1 && g == G - 1);
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    const double rho = prm.rho;

    auto issue_load = [&](uint32_t strip) {
        mbar_expect_tx(bar, (uint32_t)(RC * NC * 16));
#pragma unroll
        for (int r = 0; r < RC; r += BOXR)
            tma_load_2d((uint8_t *)s_psi + (size_t)r * NC * 16, &tmPsi, bar, (int)(strip * 2 * NC), (int)(rank * RC + r));
    };

    // ---- constants of the shared matrix for this CTA's rows: shared memory, loaded once ---------------
    for (int l = t; l <= RC; l += TPB) { // logical index l = local row + 1
        const int64_t row = (int64_t)rank * RC + l - 1;
        s_q[by_pad(l)] = (row >= 0) ? prm.qB[row] : zero;
        if (l < RC) s_g[by_pad(l)] = prm.gam[row + 1];
    }
    if (t == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 1, 1);
        mbar_init(bar + 2, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (CL > 1) { // every CTA of the cluster is resident before anything is stored into its shared memory
        cluster_arrive();
        cluster_wait();
    } else {
        __syncthreads();
    }

    // chain positions: roles of the cross-warp scan (role r composes chain positions [r KW, r KW + KW))
    const int posF = warp, posB = NW - 1 - warp; // chain position of this warp, downward / upward
    // ---- the A side of every scan, once ---------------------------------------------------------
    {
        cplx pm = one; // prod_{j=0..14} (-q_{row0+j})
#pragma unroll
        for (int j = 0; j < 15; ++j) pm = cmul(pm, cneg(s_q[by_pad(16 * g + j + 1)]));
        const cplx chunkA[2] = {sysFirst ? zero : cmul(cneg(s_q[by_pad(16 * g)]), pm),
                                sysLast ? zero : cmul(pm, cneg(s_q[by_pad(16 * g + 16)]))};
#pragma unroll
        for (int di = 0; di < 2; ++di) { // 0: downward (to higher rows), 1: upward
            cplx A = chunkA[di];
#pragma unroll
            for (int k = 0; k < L1; ++k) { // level 1: the row groups of a warp (lanes NC apart)
                const int d = NC << k;
                const bool ok = (di == 0) ? (lane >= d) : (lane + d < 32);
                if (c == 0) s_M1[(di * L1 + k) * G + g] = ok ? A : zero;
                const cplx As = (di == 0) ? shfl_up_c(A, d) : shfl_down_c(A, d);
                if (ok) A = cmul(A, As);
            }
            {
                const cplx Ae = (di == 0) ? shfl_up_c(A, NC) : shfl_down_c(A, NC);
                if (c == 0) s_Ae[di * G + g] = Ae;
            }
            const int lastRoleLane = c + NC * ((di == 0) ? GPW - 1 : 0);
            cplx aggA = shfl_c(A, lastRoleLane), cA = one;
            if (NW > 1) { // level 2: warps.  chain position of warp w: w (downward) or NW-1-w (upward)
                if (lane == lastRoleLane && c == 0) s_aggA[di * NW + warp] = A;
                __syncthreads();
                const int role = (di == 0) ? gl : GPW - 1 - gl;
                cplx a = one;
#pragma unroll
                for (int i = 0; i < KW; ++i) {
                    const int p = role * KW + i;
                    if (p < NW) a = cmul(s_aggA[di * NW + ((di == 0) ? p : NW - 1 - p)], a);
                }
#pragma unroll
                for (int k = 0; k < L1; ++k) { // inclusive over roles
                    const int d = NC << k;
                    const bool ok = (di == 0) ? (lane >= d) : (lane + d < 32);
                    if (warp == 0 && c == 0) s_rM[(di * L1 + k) * GPW + gl] = ok ? a : zero;
                    const cplx as = (di == 0) ? shfl_up_c(a, d) : shfl_down_c(a, d);
                    if (ok) a = cmul(a, as);
                }
                aggA = shfl_c(a, lastRoleLane);
                // exclusive over roles, then the warps of the own role before the own warp
                const int mypos = (di == 0) ? posF : posB, grole = mypos / KW, irole = mypos % KW;
                cplx ea = (di == 0) ? shfl_up_c(a, NC) : shfl_down_c(a, NC);
                if (role == 0) ea = one;
                cA = shfl_c(ea, c + NC * ((di == 0) ? grole : GPW - 1 - grole));
#pragma unroll
                for (int i = 0; i < KW - 1; ++i) {
                    if (i < irole) {
                        const int p = grole * KW + i;
                        cA = cmul(s_aggA[di * NW + ((di == 0) ? p : NW - 1 - p)], cA);
                    }
                }
                if (lane == 0) s_cA[di * NW + warp] = cA;
            }
            if (CL > 1 && warp == 0 && c == 0) { // the aggregate of this CTA to the CTAs that chain after it
#pragma unroll
                for (int k = 0; k < (8 + GPW - 1) / GPW; ++k) {
                    const uint32_t dst = (uint32_t)gl + GPW * k;
                    const bool wants = dst < (uint32_t)CL && ((di == 0) ? (dst > rank) : (dst < rank));
                    if (wants) dsmem_store(s_mailA + di * 8 + rank, dst, aggA);
                }
            }
        }
    }
    pdl_wait();
    pdl_launch_dependents();
    if (t == 0 && cid < nstrips) issue_load(cid);
    if (CL > 1) { // the A aggregates have arrived everywhere
        cluster_arrive();
        cluster_wait();
    } else {
        __syncthreads();
    }

    // value entering this thread's 16 rows from the rows before them in direction DIR, for its column (B: what leaves
    // the 16 rows when nothing enters them); level 3 as in k_batched_x: asynchronous DSMEM stores that signal the
    // receiver's mbarrier (16 NC bytes per sender: the per-column B)
    uint32_t par = 0; // parity of the number of strips this CTA has finished: the phase of all three mbarriers
    auto inflow = [&](auto dirtag, cplx B) -> cplx {
        constexpr int DIR = decltype(dirtag)::value;
        constexpr int di = DIR > 0 ? 0 : 1;
#pragma unroll
        for (int k = 0; k < L1; ++k) {
            const cplx Bs = (DIR > 0) ? shfl_up_c(B, NC << k) : shfl_down_c(B, NC << k);
            B = cfma(s_M1[(di * L1 + k) * G + g], Bs, B);
        }
        const int lastRoleLane = c + NC * ((DIR > 0) ? GPW - 1 : 0);
        cplx cB = zero, aggB;
        if (NW > 1) {
            cplx *const sB = s_aggB + di * NW * NC;
            const cplx *const sA = s_aggA + di * NW;
            if (gl == (DIR > 0 ? GPW - 1 : 0)) sB[warp * NC + c] = B;
            __syncthreads();
            const int role = (DIR > 0) ? gl : GPW - 1 - gl;
            cplx b = zero;
#pragma unroll
            for (int i = 0; i < KW; ++i) {
                const int p = role * KW + i;
                if (p < NW) {
                    const int w = (DIR > 0) ? p : NW - 1 - p;
                    b = cfma(sA[w], b, sB[w * NC + c]);
                }
            }
#pragma unroll
            for (int k = 0; k < L1; ++k) { // inclusive over roles
                const cplx bs = (DIR > 0) ? shfl_up_c(b, NC << k) : shfl_down_c(b, NC << k);
                b = cfma(s_rM[(di * L1 + k) * GPW + gl], bs, b);
            }
            aggB = shfl_c(b, lastRoleLane);
            const int mypos = (DIR > 0) ? posF : posB, grole = mypos / KW, irole = mypos % KW;
            cplx eb = (DIR > 0) ? shfl_up_c(b, NC) : shfl_down_c(b, NC);
            if (role == 0) eb = zero;
            cB = shfl_c(eb, c + NC * ((DIR > 0) ? grole : GPW - 1 - grole));
#pragma unroll
            for (int i = 0; i < KW - 1; ++i) {
                if (i < irole) {
                    const int p = grole * KW + i;
                    const int w = (DIR > 0) ? p : NW - 1 - p;
                    cB = cfma(sA[w], cB, sB[w * NC + c]);
                }
            }
        } else {
            aggB = shfl_c(B, lastRoleLane);
        }
        if (CL > 1) {
            const cplx *mA = s_mailA + di * 8;
            cplx *mB = s_mailB + di * 8 * NC;
            uint64_t *mb = bar + 1 + di;
            if (warp == 0) { // lane (c, gl): destination ranks gl, gl + GPW
#pragma unroll
                for (int k = 0; k < (8 + GPW - 1) / GPW; ++k) {
                    const uint32_t dst = (uint32_t)gl + GPW * k;
                    const bool wants = dst < (uint32_t)CL && ((DIR > 0) ? (dst > rank) : (dst < rank));
                    if (wants) dsmem_store_signal(mB + rank * NC + c, mb, dst, aggB);
                }
            }
            const int nsend = (DIR > 0) ? (int)rank : CL - 1 - (int)rank;
            if (nsend > 0) mbar_wait(mb, par);
            cplx cin = zero;
            if (DIR > 0) {
                for (int u = 0; u < (int)rank; ++u) cin = cfma(mA[u], cin, mB[u * NC + c]);
            } else {
                for (int u = CL - 1; u > (int)rank; --u) cin = cfma(mA[u], cin, mB[u * NC + c]);
            }
            cB = (NW > 1) ? cfma(s_cA[di * NW + warp], cin, cB) : cin;
        }
        const cplx Be = (DIR > 0) ? shfl_up_c(B, NC) : shfl_down_c(B, NC);
        const bool first = (DIR > 0) ? (gl == 0) : (gl == GPW - 1);
        return first ? cB : cfma(s_Ae[di * G + g], cB, Be);
    };

    for (uint32_t it = 0; cid + it * ncl < nstrips;) { // one loop-carried counter: strip and phase follow from it
        const uint32_t strip = cid + it * ncl;
        par = it & 1u;
        const bool hasNext = strip + ncl < nstrips;
        const bool colOK = (int64_t)strip * NC + c < prm.nsys;
        cplx *const gcol = gthread + (int64_t)strip * NC; // this thread's first row of its column of this strip
        // halo rows at the CTA edges inside a cluster: old psi from global memory (the neighbour CTA stores its
        // new rows only after it has received this CTA's aggregates of this strip).  Bringing them in with the strip
        // by bulk copies, as k_batched_x does, measured slower here (0.629 against 0.616 ms at C4).
        cplx vlo = zero, vhi = zero;
        if (CL > 1 && t == 0) { // arm this strip's mailboxes
            if (rank > 0) mbar_expect_tx(bar + 1, rank * (uint32_t)(16 * NC));
            if (rank < CL - 1) mbar_expect_tx(bar + 2, (CL - 1 - rank) * (uint32_t)(16 * NC));
        }
        if (CL > 1 && colOK) {
            if (g == 0 && rank > 0) vlo = gcol[-prm.pitch];
            if (g == G - 1 && rank < CL - 1) vhi = gcol[16 * prm.pitch];
        }
        mbar_wait(bar, par);
        cplx v[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = s_psi[(16 * g + j) * NC + c];
        if (g > 0) vlo = s_psi[(16 * g - 1) * NC + c];
        if (g < G - 1) vhi = s_psi[(16 * g + 16) * NC + c];
        fence_proxy_async(); // generic reads above before the async-proxy refill below (see cn_pass_tiled.cuh)
        __syncthreads();
        if (t == 0 && hasNext) issue_load(strip + ncl);

        // ---- Eq. 3 in place: v_j <- E_j ------------------------------------------------------------------
        {
            cplx prev = vlo;
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const cplx cur = v[j];
                const cplx hi = (j == 15) ? vhi : v[j + 1];
                v[j] = rhs_E(s_g[by_pad(16 * g + j)], rho, cur, prev, hi);
                prev = cur;
            }
        }
        // ---- downward sweep ----------------------------------------------------------------------------
        cplx D = zero;
#pragma unroll
        for (int j = 0; j < 16; ++j) D = cfnma(s_q[by_pad(16 * g + j)], D, v[j]);
        D = inflow(std::integral_constant<int, +1>{}, D);
        if (sysFirst) D = zero;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            D = cfnma(s_q[by_pad(16 * g + j)], D, v[j]);
            v[j] = D;
        }
        // ---- upward sweep + substitution -----------------------------------------------------------------
        cplx X = zero;
#pragma unroll
        for (int j = 15; j >= 0; --j) X = cmul(s_q[by_pad(16 * g + j + 1)], csub(v[j], X));
        X = inflow(std::integral_constant<int, -1>{}, X);
        if (sysLast) X = zero;
#pragma unroll
        for (int j = 15; j >= 0; --j) {
            X = cmul(s_q[by_pad(16 * g + j + 1)], csub(v[j], X));
            v[j] = X;
        }
        // The loop control is decided BEFORE the stores, and nothing of it lives in local memory: with 128 registers for
        // 16 points per thread the register allocator spills, and a reload issued after the 16 stores of a strip waits
        // behind them in the load/store queue (the trip count reloaded there held 6 % of the stall samples of this
        // kernel: 0.614 -> 0.566 ms at C4 for this alone).
        int more = hasNext;
        ++it;
        asm volatile("" : "+r"(more));
        if (colOK) {
#pragma unroll
            for (int j = 0; j < 16; ++j) gcol[j * prm.pitch] = v[j];
        }
        if (!more) break;
    }
    if (CL > 1) {
        cluster_arrive();
        cluster_wait();
    }
}

// ---- systems with a potential of their own each (cn_plan_set_systems), any dense layout: one thread per system ------
// Row i of system k lives at [k ss + i es] in V, q, gamma and psi alike.  Factor side: gamma and the
// inverse pivots of the downward elimination of every system (one block per system); d side: Eq. 3
// fused into the downward sweep, then the upward sweep + substitution, in place.  With interleaved systems (ss == 1)
// the threads of a warp touch consecutive addresses in every row.  The correctness path of the general layouts;
// contiguous systems of 8 * 2^k rows run on the tiled kernels instead (cn_pass_tiled.cuh, cutMask).
__global__ void k_batched_v_factor(int64_t N, int64_t nsys, int64_t es, int64_t ss, double two_dx2, double rho,
                                   const double *__restrict__ V, cplx *__restrict__ q, double *__restrict__ gam,
                                   int *__restrict__ err)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nsys) return;
    const int64_t o = k * ss;
    cplx qprev = cmake(0.0, 0.0);
    bool bad = false;
    for (int64_t i = 0; i < N; ++i) {
        const double g = fma(two_dx2, V[o + i * es], 2.0);
        gam[o + i * es] = g;
        const cplx p = cmake(-g - qprev.x, rho - qprev.y);
        if (!cfinite_nonzero(p)) bad = true;
        qprev = crecip(p);
        q[o + i * es] = qprev;
    }
    if (bad) atomicExch(err, 1);
}

// Rows are handled in batches of CN_BV_U: all loads of a batch are issued before its serial arithmetic and its stores (the
// in-place update keeps the compiler from hoisting loads over stores by itself), so a thread has CN_BV_U rows of three
// arrays in flight instead of one -- the difference between a latency-bound and a bandwidth-bound sweep when there are
// only a few thousand systems.
#define CN_BV_U 16
// qes / qss: strides of q and gamma (es / ss for systems with a matrix of their own; 1 / 0 for a shared matrix).
__global__ void __launch_bounds__(32)
k_batched_v_sweep(int64_t N, int64_t nsys, int64_t es, int64_t ss, double rho, cplx *__restrict__ psi,
                  const cplx *__restrict__ q, const double *__restrict__ gam, int64_t qes, int64_t qss)
{
    constexpr int U = CN_BV_U;
    pdl_wait();
    pdl_launch_dependents();
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nsys) return;
    cplx *p = psi + k * ss;
    const cplx *qk = q + k * qss;
    const double *gk = gam + k * qss;
    const cplx zero = cmake(0.0, 0.0);
    // Eq. 3 fused into the downward sweep: D_i = E_i - q_{i-1} D_{i-1}, D overwrites psi
    cplx lo = zero, cur = p[0], D = zero, qprev = zero;
    for (int64_t i0 = 0; i0 < N; i0 += U) {
        cplx hv[U], qv[U];
        double gv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t r = i0 + u;
            hv[u] = (r + 1 < N) ? p[(r + 1) * es] : zero;
            qv[u] = (r < N) ? qk[r * qes] : zero;
            gv[u] = (r < N) ? gk[r * qes] : 0.0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t r = i0 + u;
            if (r < N) {
                const cplx E = rhs_E(gv[u], rho, cur, lo, hv[u]);
                D = cfnma(qprev, D, E);
                p[r * es] = D;
                qprev = qv[u];
                lo = cur;
                cur = hv[u];
            }
        }
    }
    // upward sweep + substitution: x_i = q_i (D_i - x_{i+1})
    cplx x = zero;
    for (int64_t i1 = N; i1 > 0; i1 -= U) {
        cplx dv[U], qv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t r = i1 - 1 - u;
            dv[u] = (r >= 0) ? p[r * es] : zero;
            qv[u] = (r >= 0) ? qk[r * qes] : zero;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t r = i1 - 1 - u;
            if (r >= 0) {
                x = cmul(qv[u], csub(dv[u], x));
                p[r * es] = x;
            }
        }
    }
}

// whole-system inverse pivots (one block per system): p_0 = mu_0, p_i = mu_i - q_{i-1}, q_i = 1 / p_i
__global__ void k_factor_whole(int64_t N, double rho, const double *__restrict__ gam, cplx *__restrict__ qB,
                               int *__restrict__ err)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    cplx qprev = cmake(0.0, 0.0);
    bool bad = false;
    for (int64_t i = 0; i < N; ++i) {
        cplx p = cmake(-gam[i] - qprev.x, rho - qprev.y);
        if (!cfinite_nonzero(p)) bad = true;
        qprev = crecip(p);
        qB[i] = qprev;
    }
    if (bad) atomicExch(err, 1);
}
