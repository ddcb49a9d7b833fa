// RS stage: solve the reduced tridiagonal system on the joint lines.
//
// The paper solves it serially ("implemented serially", beta * n_bl in its model) and
// notes that the reduced system can itself be solved by the same partition method, level after level
// (Eq. 6:  N[M_0] = sum (RD+RU+JU+JD)[M_i] + RS[M_last] + sum SS[M_i]).
// Here:
//   * k_rs_top<K>     -- RS[M_last]: the pre-factored system of the last level is solved by ONE CTA;
//                        every thread owns K consecutive rows held in registers, the threads are chained
//                        by the affine-map scan of cn_common.cuh (serial depth K instead of n).
//   * k_rs_reduce     -- (RD+RU+JD+JU)[M_i], i >= 1, d-side only: one WARP per group of G joint lines of
//                        level i, 8 rows per lane in registers; emits two slots per joint line of level i+1.
//   * k_rs_subst      -- SS[M_i], i >= 1: one warp per group, given the two support values of level i+1.
//   * k_rs_serial     -- the paper-literal variant (one thread, plain Thomas on the joint lines), kept
//                        for the P sweep (CN_OPT_RS_LEVELS = -1).
// All matrix-side quantities (local pivots, fill-in, the next level's matrix) are produced once by the
// factor kernels at the end of this file.
//
// A level is a general complex tridiagonal system (sub_i, diag_i, sup_i), i = 0..n-1.  Group g owns rows
// [g G, min((g+1) G, n)); its LAST row is the joint line of the next level, the rows before it are its
// interior.  Stored per interior row:  l_i = sub_i * rp_{i-1}  (rp := 1 above the first interior row, so
// that "D above the group := support value of the joint above" works as in the pass kernels),
// rp_i = 1 / pivot_i,  u_i = sup_i * rp_i.
#pragma once
#include "cn_common.cuh"
#include "cn_factor.cuh" // cn_mob

CN_DEVINL cplx shard_rhs(const cplx *gathered, int64_t S, int64_t nt, int64_t w); // cn_shard.cuh (sharded last level)

#define CN_RS_G 256          // joint lines per group
#define CN_RS_TOP_THREADS 1024

// Exclusive scan of affine maps over all threads of a CTA (blockDim.x a multiple of 32, <= 1024).
// (A, B) is this thread's map in direction DIR; returns the value ENTERING this thread when `tin` enters
// the first thread of the direction.  sA, sB: 32 cplx each, free again after the next barrier of the caller.
template <int DIR>
CN_DEVINL cplx cta_scan_excl(cplx A, cplx B, cplx tin, cplx *sA, cplx *sB)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    warp_scan_affine<DIR, 5>(A, B, lane);
    if (lane == (DIR > 0 ? 31 : 0)) {
        sA[warp] = A;
        sB[warp] = B;
    }
    __syncthreads();
    cplx wA = cmake(1.0, 0.0), wB = cmake(0.0, 0.0);
    if (lane < nwarps) {
        wA = sA[lane];
        wB = sB[lane];
    }
    warp_scan_affine<DIR, 5>(wA, wB, lane);
    const int src = (DIR > 0) ? warp - 1 : warp + 1; // inclusive composite of all warps before this one
    const bool has = (DIR > 0) ? (src >= 0) : (src < nwarps);
    const int srcc = has ? src : lane;
    cplx cA = shfl_c(wA, srcc), cB = shfl_c(wB, srcc);
    cplx carry = has ? cfma(cA, tin, cB) : tin;
    cplx Ae = (DIR > 0) ? shfl_up_c(A, 1) : shfl_down_c(A, 1);
    cplx Be = (DIR > 0) ? shfl_up_c(B, 1) : shfl_down_c(B, 1);
    const bool first = (DIR > 0) ? (lane == 0) : (lane == 31);
    cplx r = cfma(Ae, carry, Be);
    return first ? carry : r;
}

// ---- RS[M_last]: one CTA, K rows per thread in registers ---------------------------------------------
// R_w = rD[w] + rU[w]  (the two extra elements per joint line of PAPER.md:102, summed here)
// forward   R'_w = R_w - lw_w R'_{w-1},   back substitution  X_w = rq_w R'_w - uw_w X_{w+1}
template <int K>
__global__ void __launch_bounds__(CN_RS_TOP_THREADS, 1)
k_rs_top(int64_t n, const cplx *__restrict__ rD, const cplx *__restrict__ rU, const cplx *__restrict__ lw,
         const cplx *__restrict__ rq, const cplx *__restrict__ uw, cplx *__restrict__ X)
{
    __shared__ cplx sA[2][32], sB[2][32];
    const int t = threadIdx.x;
    const int64_t w0 = (int64_t)t * K;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    cplx l[K], r[K], u[K], R[K];
    // the factors do not depend on the preceding kernel: fetch them before waiting for it
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const bool in = w0 + k < n;
        l[k] = in ? lw[w0 + k] : zero;
        r[k] = in ? rq[w0 + k] : zero;
        u[k] = in ? uw[w0 + k] : zero;
    }
    pdl_wait();
#pragma unroll
    for (int k = 0; k < K; ++k) R[k] = (w0 + k < n) ? cadd(ld_dep(rD + w0 + k), ld_dep(rU + w0 + k)) : zero;
    pdl_launch_dependents();

    cplx A = one, B = zero;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        B = cfnma(l[k], B, R[k]);
        A = cmul(cneg(l[k]), A);
    }
    cplx in = cta_scan_excl<+1>(A, B, zero, sA[0], sB[0]);
#pragma unroll
    for (int k = 0; k < K; ++k) {
        in = cfnma(l[k], in, R[k]);
        R[k] = cmul(r[k], in); // rq_w R'_w
    }
    A = one;
    B = zero;
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        B = cfnma(u[k], B, R[k]);
        A = cmul(cneg(u[k]), A);
    }
    in = cta_scan_excl<-1>(A, B, zero, sA[1], sB[1]);
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        in = cfnma(u[k], in, R[k]);
        if (w0 + k < n) X[w0 + k] = in;
    }
}

// ---- paper-literal serial RS: plain Thomas back/forward substitution by one thread ----------------------
__global__ void k_rs_serial(int64_t n, const cplx *__restrict__ rD, const cplx *__restrict__ rU,
                            const cplx *__restrict__ lw, const cplx *__restrict__ rq, const cplx *__restrict__ uw,
                            cplx *__restrict__ X)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    pdl_wait();
    pdl_launch_dependents();
    cplx prev = cmake(0.0, 0.0);
    for (int64_t w = 0; w < n; ++w) {
        prev = cfnma(lw[w], prev, cadd(ld_dep(rD + w), ld_dep(rU + w)));
        X[w] = prev;
    }
    prev = cmake(0.0, 0.0);
    for (int64_t w = n - 1; w >= 0; --w) {
        prev = cfnma(uw[w], prev, cmul(rq[w], X[w]));
        X[w] = prev;
    }
}

// ---- (RD+RU+JD+JU)[M_i], d-side: group g of level i -> slots of joint line g of level i+1 ----------------
// One WARP per group of CN_RS_G = 256 joint lines: lane t owns the CN_RS_K = 8 consecutive rows g0 + 8 t ...
// in registers and the lanes are chained by the warp scan of cn_common.cuh (no shared memory, no barrier).
// Nothing enters a group during the reduction (zero support values), so the composed A of the scan is dead.
#define CN_RS_K (CN_RS_G / 32)
#define CN_RS_WARPS 4 // groups per CTA of the group kernels

// Coalesced transfer of one group's rows between global memory and the lanes' registers (lane t owns rows 8 t .. 8 t + 7)
// through a swizzled 4 KB shared-memory buffer of the warp: a warp-level load touches 4 lines instead of 32.
CN_DEVINL int rs_swz(int r) { return (r & ~7) | ((r ^ (r >> 3)) & 7); }
template <bool DEP>
CN_DEVINL void rs_load_rows(const cplx *__restrict__ src, int ng, cplx *sbuf, int lane, cplx (&out)[CN_RS_G / 32])
{
#pragma unroll
    for (int k = 0; k < CN_RS_G / 32; ++k) {
        const int r = k * 32 + lane;
        cplx v = cmake(0.0, 0.0);
        if (r < ng) v = DEP ? ld_dep(src + r) : src[r];
        sbuf[rs_swz(r)] = v;
    }
    __syncwarp();
#pragma unroll
    for (int j = 0; j < CN_RS_G / 32; ++j) out[j] = sbuf[rs_swz(lane * 8 + j)];
    __syncwarp();
}
CN_DEVINL void rs_store_rows(cplx *__restrict__ dst, int ng, cplx *sbuf, int lane, const cplx (&in)[CN_RS_G / 32])
{
#pragma unroll
    for (int j = 0; j < CN_RS_G / 32; ++j) sbuf[rs_swz(lane * 8 + j)] = in[j];
    __syncwarp();
#pragma unroll
    for (int k = 0; k < CN_RS_G / 32; ++k) {
        const int r = k * 32 + lane;
        if (r < ng) dst[r] = sbuf[rs_swz(r)];
    }
    __syncwarp();
}

// The same for up to three arrays at once: all global loads are issued before the first shared-memory round trip, so a
// warp pays one memory latency for the lot (sbuf: 3 buffers of CN_RS_G elements).
template <bool DEP, int NA>
CN_DEVINL void rs_load_rows_n(const cplx *const (&src)[NA], const int (&lim)[NA], cplx *sbuf, int lane,
                              cplx (&out)[NA][CN_RS_G / 32])
{
    cplx tmp[NA][CN_RS_G / 32];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int k = 0; k < CN_RS_G / 32; ++k) {
            const int r = k * 32 + lane;
            tmp[a][k] = cmake(0.0, 0.0);
            if (r < lim[a]) tmp[a][k] = DEP ? ld_dep(src[a] + r) : src[a][r];
        }
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int k = 0; k < CN_RS_G / 32; ++k) sbuf[a * CN_RS_G + rs_swz(k * 32 + lane)] = tmp[a][k];
    __syncwarp();
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int j = 0; j < CN_RS_G / 32; ++j) out[a][j] = sbuf[a * CN_RS_G + rs_swz(lane * 8 + j)];
    __syncwarp();
}

__global__ void __launch_bounds__(32 * CN_RS_WARPS)
k_rs_reduce(int64_t n, const cplx *__restrict__ rD, const cplx *__restrict__ rU, const cplx *__restrict__ l,
            const cplx *__restrict__ rp, const cplx *__restrict__ u, const cplx *__restrict__ sub,
            const cplx *__restrict__ sup, cplx *__restrict__ outD, cplx *__restrict__ outU, int above = 0,
            const int64_t *__restrict__ off = nullptr, int64_t noff = 0)
{   // above: the rows of a shard that another shard precedes (cn_shard.cuh): group 0 has a real joint line above it,
    // whose coupling sup[-1] and slot outU[-1] are the guard elements of the arrays
    // off != NULL: caller-placed joint lines ("blocks may differ in size"), blocks of at most CN_RS_G rows:
    // group g = rows [off[g], off[g+1])
    constexpr int K = CN_RS_K;
    const int lane = threadIdx.x & 31;
    const int64_t ngroups = off ? noff : (n + CN_RS_G - 1) / CN_RS_G;
    const int64_t g = (int64_t)blockIdx.x * CN_RS_WARPS + (threadIdx.x >> 5);
    const bool live = g < ngroups; // whole warps only: the shuffles below stay convergent
    const int64_t g0 = !live ? 0 : (off ? off[g] : g * CN_RS_G);
    const int ng = live ? (off ? (int)(off[g + 1] - g0) : (int)((n - g0 < CN_RS_G) ? (n - g0) : CN_RS_G)) : 0;
    const int r0 = lane * K; // first row of this lane inside the group
    const cplx zero = cmake(0.0, 0.0);
    __shared__ cplx sbuf_all[CN_RS_WARPS][3 * CN_RS_G];
    cplx *const sbuf = sbuf_all[threadIdx.x >> 5];
    cplx F[3][K], R[K];
    {   // rows >= ng - 1 (the joint line and beyond) read as 0
        const cplx *const src[3] = {l + g0, rp + g0, u + g0};
        const int lim[3] = {ng - 1, ng - 1, ng - 1};
        rs_load_rows_n<false, 3>(src, lim, sbuf, lane, F);
    }
    cplx (&lk)[K] = F[0], (&rpk)[K] = F[1], (&uk)[K] = F[2];
    cplx subJ = zero, supAbove = zero;
    if (live && lane == 0) {
        subJ = sub[g0 + ng - 1];
        if (g > 0 || above) supAbove = sup[g0 - 1];
    }
    pdl_wait();
    {
        cplx RR[2][K];
        const cplx *const src[2] = {rD + g0, rU + g0};
        const int lim[2] = {ng, ng};
        rs_load_rows_n<true, 2>(src, lim, sbuf, lane, RR);
#pragma unroll
        for (int k = 0; k < K; ++k) R[k] = cadd(RR[0][k], RR[1][k]);
    }
    pdl_launch_dependents();
    // the joint line's own right-hand side (lane 0 needs it)
    cplx Rj = zero;
#pragma unroll
    for (int k = 0; k < K; ++k)
        if (r0 + k == ng - 1) Rj = R[k];
    Rj = shfl_c(Rj, ng > 0 ? (ng - 1) / K : 0);
    // RD: D_i = R_i - l_i D_{i-1} on the interior rows, D := 0 on the joint line and beyond
    cplx A = cmake(1.0, 0.0), B = zero;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        B = (r0 + k < ng - 1) ? cfnma(lk[k], B, R[k]) : zero;
        A = cmul(cneg(lk[k]), A);
    }
    if (lane == 0) A = zero; // nothing enters the group through the scan: no lane predicate needed
    warp_scan_affine_uncond<+1, 5>(A, B);
    cplx in = shfl_up_c(B, 1);
    if (lane == 0) in = zero;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        in = (r0 + k < ng - 1) ? cfnma(lk[k], in, R[k]) : zero;
        R[k] = cmul(rpk[k], in); // rp_i D_i
    }
    // RU + local solution: y_i = rp_i D_i - u_i y_{i+1}, y := 0 on the joint line
    A = cmake(1.0, 0.0);
    B = zero;
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        B = cfnma(uk[k], B, R[k]);
        A = cmul(cneg(uk[k]), A);
    }
    warp_scan_affine_uncond<-1, 5>(A, B); // u = 0 on the joint line and beyond: A = 0 at the chain start
    in = shfl_down_c(B, 1);
    if (lane == 31) in = zero;
    cplx yN = zero, y0 = zero; // y next to the own joint (row ng-2) and y of the first row
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        in = cfnma(uk[k], in, R[k]);
        if (r0 + k == ng - 2) yN = in;
        if (k == 0) y0 = in;
    }
    yN = shfl_c(yN, ng > 1 ? (ng - 2) / K : 0);
    if (live && lane == 0) {
        outD[g] = (ng >= 2) ? cfnma(subJ, yN, Rj) : Rj;                        // JD
        if (g > 0 || above) {
            cplx ju = (ng >= 2) ? cneg(cmul(supAbove, y0)) : zero; // JU
            if (g == 0) ju = cadd(ju, ld_dep(rU - 1)); // (a shard's first group) the guard of this level rides along
            outU[g - 1] = ju;
        }
    }
}

// ---- SS[M_i]: group g of level i from the support values of level i+1 (one warp per group, as above) -------
// KT > 0: the LAST level (ntop <= 128 KT rows) is solved inside this kernel, redundantly by every CTA, from the slots
// topD / topU the reduction kernel just wrote -- one launch less on the per-step chain (reduce -> substitute instead
// of reduce -> last level -> substitute); Xup is then not read.  KT == 0: Xup comes from k_rs_top.
template <int KT>
__global__ void __launch_bounds__(32 * CN_RS_WARPS)
k_rs_subst(int64_t n, const cplx *__restrict__ rD, const cplx *__restrict__ rU, const cplx *__restrict__ l,
           const cplx *__restrict__ rp, const cplx *__restrict__ u, const cplx *__restrict__ Xup,
           cplx *__restrict__ X, int64_t ntop, const cplx *topD, const cplx *topU, const cplx *__restrict__ lw,
           const cplx *__restrict__ rq, const cplx *__restrict__ uw, const cplx *Xabove = nullptr,
           const int64_t *__restrict__ off = nullptr, int64_t noff = 0, cplx *guardOut = nullptr,
           const cplx *gathered = nullptr, int64_t nshards = 1, int64_t toff = 0, cplx *xaboveOut = nullptr)
{   // Xabove (KT == 0 only): support value of the joint line above group 0 when a shard precedes this one (cn_shard.cuh)
    // off: caller-placed joint lines (see k_rs_reduce)
    // guardOut: a shard's level-0 substitution also leaves the support value of the row above the shard in the guard
    //           element of the level-0 array, where the pass kernel expects it
    // gathered (KT > 0): the last level is the WHOLE system's (nshards records, shard_rhs), this shard's rows start at
    //           toff; xaboveOut receives the support value of the row above the shard for the levels below
    constexpr int K = CN_RS_K;
    const int lane = threadIdx.x & 31;
    const int64_t ngroups = off ? noff : (n + CN_RS_G - 1) / CN_RS_G;
    const int64_t g = (int64_t)blockIdx.x * CN_RS_WARPS + (threadIdx.x >> 5);
    const bool live = g < ngroups;
    const int64_t g0 = !live ? 0 : (off ? off[g] : g * CN_RS_G);
    const int ng = live ? (off ? (int)(off[g + 1] - g0) : (int)((n - g0 < CN_RS_G) ? (n - g0) : CN_RS_G)) : 0;
    const int r0 = lane * K;
    const cplx zero = cmake(0.0, 0.0);
    __shared__ cplx sbuf_all[CN_RS_WARPS][3 * CN_RS_G];
    cplx *const sbuf = sbuf_all[threadIdx.x >> 5];
    cplx F[3][K], R[K];
    {
        const cplx *const src[3] = {l + g0, rp + g0, u + g0};
        const int lim[3] = {ng - 1, ng - 1, ng - 1};
        rs_load_rows_n<false, 3>(src, lim, sbuf, lane, F);
    }
    cplx (&lk)[K] = F[0], (&rpk)[K] = F[1], (&uk)[K] = F[2];
    {   // the right-hand sides were written two kernels ago: complete (interior rows only)
        cplx RR[2][K];
        const cplx *const src[2] = {rD + g0, rU + g0};
        const int lim[2] = {ng - 1, ng - 1};
        rs_load_rows_n<false, 2>(src, lim, sbuf, lane, RR);
#pragma unroll
        for (int k = 0; k < K; ++k) R[k] = cadd(RR[0][k], RR[1][k]);
    }
    cplx XL = zero, XJ = zero;
    if (KT > 0) {
        // ---- RS[M_last] by the whole CTA (as k_rs_top), result in shared memory ------------------------------
        constexpr int KK = KT > 0 ? KT : 1;
        const int t = threadIdx.x;
        const int64_t w0 = (int64_t)t * KK;
        const cplx one = cmake(1.0, 0.0);
        cplx tl[KK], tr[KK], tu[KK], tR[KK];
#pragma unroll
        for (int k = 0; k < KK; ++k) {
            const bool in = w0 + k < ntop;
            tl[k] = in ? lw[w0 + k] : zero;
            tr[k] = in ? rq[w0 + k] : zero;
            tu[k] = in ? uw[w0 + k] : zero;
        }
        pdl_wait();
#pragma unroll
        for (int k = 0; k < KK; ++k) {
            tR[k] = zero;
            if (w0 + k < ntop)
                tR[k] = gathered ? shard_rhs(gathered, nshards, ntop / nshards, w0 + k)
                                 : cadd(ld_dep(topD + w0 + k), ld_dep(topU + w0 + k));
        }
        pdl_launch_dependents();
        __syncthreads(); // every warp is done with its transfer buffer: the buffers become the scratch of the solve
        cplx *const sX = &sbuf_all[0][0];                    // [32 * CN_RS_WARPS * 8] <= 1024 values
        cplx *const sA = sX + 32 * CN_RS_WARPS * 8, *const sB = sA + 64; // [2][32] each
        cplx A = one, B = zero;
#pragma unroll
        for (int k = 0; k < KK; ++k) {
            B = cfnma(tl[k], B, tR[k]);
            A = cmul(cneg(tl[k]), A);
        }
        cplx in = cta_scan_excl<+1>(A, B, zero, sA, sB);
#pragma unroll
        for (int k = 0; k < KK; ++k) {
            in = cfnma(tl[k], in, tR[k]);
            tR[k] = cmul(tr[k], in);
        }
        A = one;
        B = zero;
#pragma unroll
        for (int k = KK - 1; k >= 0; --k) {
            B = cfnma(tu[k], B, tR[k]);
            A = cmul(cneg(tu[k]), A);
        }
        in = cta_scan_excl<-1>(A, B, zero, sA + 32, sB + 32);
#pragma unroll
        for (int k = KK - 1; k >= 0; --k) {
            in = cfnma(tu[k], in, tR[k]);
            if (w0 + k < ntop) sX[w0 + k] = in;
        }
        __syncthreads();
        if (live) {
            if (toff + g > 0) XL = sX[toff + g - 1];
            XJ = sX[toff + g];
            if (g == 0 && lane == 0 && toff > 0) {
                if (xaboveOut) *xaboveOut = XL;
                if (guardOut) *guardOut = XL;
            }
        }
        __syncthreads(); // sX is read: the warps may use their transfer buffers again (rs_store_rows below)
    } else {
        pdl_wait();
        if (live) {
            if (g > 0) XL = ld_dep(Xup + g - 1);
            else if (Xabove) {
                XL = ld_dep(Xabove);
                if (lane == 0 && guardOut) *guardOut = XL;
            }
            XJ = ld_dep(Xup + g);
        }
        pdl_launch_dependents();
    }
    // RD with the support value of the joint above entering the first row (rp := 1 there, see the header)
    cplx A = cmake(1.0, 0.0), B = (lane == 0) ? XL : zero;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        B = cfnma(lk[k], B, R[k]);
        A = cmul(cneg(lk[k]), A);
    }
    if (lane == 0) A = zero; // nothing enters the group through the scan: no lane predicate needed
    warp_scan_affine_uncond<+1, 5>(A, B);
    cplx in = shfl_up_c(B, 1);
    if (lane == 0) in = XL;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        in = cfnma(lk[k], in, R[k]);
        R[k] = cmul(rpk[k], in);
    }
    // SS: x_i = rp_i D_i - u_i x_{i+1}, x := X_g on the joint line
    A = cmake(1.0, 0.0);
    B = zero;
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        B = (r0 + k == ng - 1) ? XJ : cfnma(uk[k], B, R[k]);
        A = cmul(cneg(uk[k]), A);
    }
    warp_scan_affine_uncond<-1, 5>(A, B); // u = 0 on the joint line and beyond: A = 0 at the chain start
    in = shfl_down_c(B, 1);
    if (lane == 31) in = zero;
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        in = (r0 + k == ng - 1) ? XJ : cfnma(uk[k], in, R[k]);
        R[k] = in;
    }
    rs_store_rows(X + g0, ng, sbuf, lane, R);
}

// ---- paper-shaped group kernels: ONE THREAD serves one group of G joint lines (any G) ------------------------
// The multi-iteration GPU program of PAPER.md:276 ("interleaving" the block kernels for the nested method): the same
// stages as k_rs_reduce / k_rs_subst by serial sweeps straight in global memory.  X of the level is the scratch for
// rp_i D_i between the two sweeps.  Used when CN_OPT_RS_GROUP is not 256 (the nested-level study).
__global__ void k_rs_reduce_thread(int64_t n, int64_t G, const cplx *__restrict__ rD, const cplx *__restrict__ rU,
                                   const cplx *__restrict__ l, const cplx *__restrict__ rp, const cplx *__restrict__ u,
                                   const cplx *__restrict__ sub, const cplx *__restrict__ sup, cplx *scratch,
                                   cplx *__restrict__ outD, cplx *__restrict__ outU)
{
    pdl_wait();
    pdl_launch_dependents();
    const int64_t ngroups = (n + G - 1) / G;
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    const int64_t g0 = g * G, J = ((g0 + G < n) ? (g0 + G) : n) - 1;
    const cplx zero = cmake(0.0, 0.0);
    cplx D = zero;
    for (int64_t i = g0; i < J; ++i) {
        D = cfnma(l[i], D, cadd(ld_dep(rD + i), ld_dep(rU + i)));
        scratch[i] = cmul(rp[i], D);
    }
    cplx y = zero, yN = zero;
    for (int64_t i = J - 1; i >= g0; --i) {
        y = cfnma(u[i], y, scratch[i]);
        if (i == J - 1) yN = y;
    }
    const cplx RJ = cadd(ld_dep(rD + J), ld_dep(rU + J));
    outD[g] = (J > g0) ? cfnma(sub[J], yN, RJ) : RJ;
    if (g > 0) outU[g - 1] = (J > g0) ? cneg(cmul(sup[g0 - 1], y)) : zero;
}

__global__ void k_rs_subst_thread(int64_t n, int64_t G, const cplx *__restrict__ rD, const cplx *__restrict__ rU,
                                  const cplx *__restrict__ l, const cplx *__restrict__ rp, const cplx *__restrict__ u,
                                  const cplx *__restrict__ Xup, cplx *X)
{
    pdl_wait();
    pdl_launch_dependents();
    const int64_t ngroups = (n + G - 1) / G;
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    const int64_t g0 = g * G, J = ((g0 + G < n) ? (g0 + G) : n) - 1;
    cplx D = (g > 0) ? ld_dep(Xup + g - 1) : cmake(0.0, 0.0);
    for (int64_t i = g0; i < J; ++i) {
        D = cfnma(l[i], D, cadd(ld_dep(rD + i), ld_dep(rU + i)));
        X[i] = cmul(rp[i], D);
    }
    cplx x = ld_dep(Xup + g);
    X[J] = x;
    for (int64_t i = J - 1; i >= g0; --i) {
        x = cfnma(u[i], x, X[i]);
        X[i] = x;
    }
}

// ======================================= factor side (once per plan) =======================================

// level-0 reduced matrix from the block corner entries produced by k_factor_blocks (cn_factor.cuh)
// (gamJ != NULL: gamma of joint line w is gamJ[w] instead of gam[J_w] -- out-of-core mode, gamma not resident)
__global__ void k_rs_assemble0(int64_t P, int64_t N, double rho, const double *__restrict__ gam,
                               const double *__restrict__ gamJ,
                               const cplx *__restrict__ redSubD, const cplx *__restrict__ redDiagD,
                               const cplx *__restrict__ redSupU, const cplx *__restrict__ redDiagU,
                               cplx *__restrict__ sub, cplx *__restrict__ diag, cplx *__restrict__ sup,
                               int above = 0, cplx *__restrict__ diagAboveAcc = nullptr, int64_t cutMask = ~(int64_t)0)
{   // above (cn_shard.cuh): row 0 keeps its coupling to the last row of the preceding shard; that row's coupling to row 0
    // goes to the guard sup[-1] and the diagonal term this shard's first block adds to it opens the sum *diagAboveAcc
    int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= P) return;
    if (above && w == 0) {
        sup[-1] = redSupU[-1];
        *diagAboveAcc = redDiagU[-1];
    }
    const int64_t J = ((N % P == 0) ? (w + 1) * (N / P) : (int64_t)(((__int128)(w + 1) * N) / P)) - 1;
    const double gJ = gamJ ? gamJ[w] : gam[J];
    cplx d = cmake(-gJ + redDiagD[w].x, rho + redDiagD[w].y);
    cplx s = cmake(0.0, 0.0);
    if (w < P - 1) {
        d = cadd(d, redDiagU[w]);
        s = redSupU[w];
    }
    sub[w] = ((w & cutMask) != 0 || above) ? redSubD[w] : cmake(0.0, 0.0); // (cutMask: independent systems, cn_pass_tiled.cuh)
    diag[w] = d;
    sup[w] = s;
}

// one thread per group of a non-last level: local LU of the interior rows, responses to unit support
// values, and from them the rows of the next level's matrix (the JD / JU matrix side)
__global__ void k_rs_factor_level(int64_t n, int64_t G, const cplx *__restrict__ sub, const cplx *__restrict__ diag,
                                  const cplx *__restrict__ sup, cplx *__restrict__ l, cplx *__restrict__ rp,
                                  cplx *__restrict__ u, cplx *__restrict__ tmp, cplx *__restrict__ sub2,
                                  cplx *__restrict__ diag2, cplx *__restrict__ diag2U, cplx *__restrict__ sup2,
                                  int *__restrict__ err)
{
    const int64_t ngroups = (n + G - 1) / G;
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    const int64_t g0 = g * G;
    const int64_t J = ((g0 + G < n) ? (g0 + G) : n) - 1;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    bool bad = false;
    cplx prp = one, psup = zero, Dal = one; // Dal: forward sweep of the response to X_{g-1} = 1
    for (int64_t i = g0; i < J; ++i) {
        cplx li = cmul(sub[i], prp);
        cplx piv = cfnma(li, psup, diag[i]);
        if (!cfinite_nonzero(piv)) bad = true;
        cplx r = crecip(piv);
        l[i] = li;
        rp[i] = r;
        u[i] = cmul(sup[i], r);
        Dal = cneg(cmul(li, Dal));
        tmp[i] = Dal;
        prp = r;
        psup = sup[i];
    }
    l[J] = zero;
    rp[J] = zero;
    u[J] = zero;
    const bool has = J > g0;
    // alpha_i: response to (X_{g-1}, X_g) = (1, 0);  beta_i: response to (0, 1)
    cplx al = zero, be = one, alLast = zero, beLast = zero;
    for (int64_t i = J - 1; i >= g0; --i) {
        al = cfnma(u[i], al, cmul(rp[i], tmp[i]));
        be = cneg(cmul(u[i], be));
        if (i == J - 1) {
            alLast = al;
            beLast = be;
        }
    }
    // row J of this level:  sub_J x_{J-1} + diag_J x_J + sup_J x_{J+1} = R_J
    sub2[g] = (g == 0) ? zero : (has ? cmul(sub[J], alLast) : sub[J]);
    diag2[g] = has ? cfma(sub[J], beLast, diag[J]) : diag[J];
    if (g > 0) {
        const cplx sa = sup[g0 - 1];
        diag2U[g - 1] = has ? cmul(sa, al) : zero;
        sup2[g - 1] = has ? cmul(sa, be) : sa;
    }
    if (g == ngroups - 1) {
        diag2U[g] = zero;
        sup2[g] = zero;
    }
    if (bad) atomicExch(err, 1);
}

// The same for groups of CN_RS_G = 256 rows by ONE WARP per group, 8 rows per lane in registers (rows moved coalesced
// through the swizzled buffer of rs_load_rows_n).  Every serial recurrence of the thread-per-group kernel above becomes
// a warp scan over the lanes:
//   * pivots: rp_i = 1 / (diag_i - sub_i sup_{i-1} rp_{i-1}) is a Moebius map of rp_{i-1} (cn_factor.cuh); the lanes'
//     2x2 matrices are composed by a Kogge-Stone scan, then every lane recomputes its 8 rows from its true inflow;
//   * Dal_i = prod_{k <= i} (-l_k) (forward response to a unit support value above the group): multiplicative scan;
//   * al_i = rp_i Dal_i - u_i al_{i+1} and be_i = prod_{k >= i} (-u_k): ONE backward affine scan gives both (be is its A).
// The thread-per-group kernel pays a global-memory latency per row (268 us for 512 groups at C2), its shared-memory
// variant with one serial lane took 45 us, this one takes a few us -- it runs once per step under cn_step_td.
#define CN_RS_FL_WARPS 4
__global__ void __launch_bounds__(32 * CN_RS_FL_WARPS)
k_rs_factor_level_smem(int64_t n, const cplx *__restrict__ sub, const cplx *__restrict__ diag,
                       const cplx *__restrict__ sup, cplx *__restrict__ l, cplx *__restrict__ rp, cplx *__restrict__ u,
                       cplx *__restrict__ sub2, cplx *__restrict__ diag2, cplx *__restrict__ diag2U,
                       cplx *__restrict__ sup2, int *__restrict__ err, int above = 0,
                       const int64_t *__restrict__ off = nullptr, int64_t noff = 0)
{   // above (cn_shard.cuh): group 0 is treated like any later group; its JU matrix side goes to the guards [-1]
    // off: caller-placed joint lines with blocks of at most CN_RS_G rows (see k_rs_reduce)
    constexpr int K = CN_RS_K;
    __shared__ cplx sbuf_all[CN_RS_FL_WARPS][3 * CN_RS_G];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    cplx *const sbuf = sbuf_all[wp];
    const int64_t ngroups = off ? noff : (n + CN_RS_G - 1) / CN_RS_G;
    const int64_t g = (int64_t)blockIdx.x * CN_RS_FL_WARPS + wp;
    if (g >= ngroups) return; // whole warps
    const int64_t g0 = off ? off[g] : g * CN_RS_G;
    const int ng = off ? (int)(off[g + 1] - g0) : (int)((n - g0 < CN_RS_G) ? (n - g0) : CN_RS_G);
    const int nj = ng - 1; // interior rows; row nj is the joint line
    const int r0 = lane * K;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    cplx F[3][K];
    {
        const cplx *const src[3] = {sub + g0, diag + g0, sup + g0};
        const int lim[3] = {ng, ng, ng};
        rs_load_rows_n<false, 3>(src, lim, sbuf, lane, F);
    }
    cplx (&sb)[K] = F[0], (&dg)[K] = F[1], (&sp)[K] = F[2];
    // the joint line's own entries, for lane 0
    cplx subJ = zero, diagJ = zero;
#pragma unroll
    for (int k = 0; k < K; ++k)
        if (r0 + k == nj) {
            subJ = sb[k];
            diagJ = dg[k];
        }
    subJ = shfl_c(subJ, nj / K);
    diagJ = shfl_c(diagJ, nj / K);
    // sup of the row before each own row (0 before the group's first row: nothing is eliminated against the joint above)
    cplx spPrev0 = shfl_up_c(sp[K - 1], 1);
    if (lane == 0) spPrev0 = zero;
    // ---- pivots: Moebius maps of the own rows, scan, recompute ----------------------------------------------------
    cn_mob M{one, zero, zero, one};
#pragma unroll
    for (int k = 0; k < K; ++k) {
        if (r0 + k < nj) {
            const cplx ci = cmul(sb[k], (k == 0) ? spPrev0 : sp[k - 1]); // (row 0 of the group: spPrev0 = 0, a constant map)
            cn_mob Rm; // [[0, 1], [-c_i, d_i]] * M
            Rm.a = M.c;
            Rm.b = M.d;
            Rm.c = csub(cmul(dg[k], M.c), cmul(ci, M.a));
            Rm.d = csub(cmul(dg[k], M.d), cmul(ci, M.b));
            M = mob_scale(Rm);
        }
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int dd = 1 << k;
        cn_mob S = mob_shfl(M, lane - dd < 0 ? 0 : lane - dd);
        if (lane >= dd) M = mob_scale(mob_mul(M, S));
    }
    cn_mob Pm = mob_shfl(M, lane == 0 ? 0 : lane - 1);
    cplx rprev = (lane == 0) ? one : cmul(Pm.b, crecip_fast(Pm.d)); // rp := 1 above the first interior row
    bool bad = false;
    cplx lk[K], rpk[K], uk[K];
    cplx pl = one; // product of (-l) over the own interior rows
#pragma unroll
    for (int k = 0; k < K; ++k) {
        lk[k] = rpk[k] = uk[k] = zero;
        if (r0 + k < nj) {
            const cplx li = cmul(sb[k], rprev);
            const cplx piv = cfnma(li, (k == 0) ? spPrev0 : sp[k - 1], dg[k]);
            if (!cfinite_nonzero(piv)) bad = true;
            const cplx r = crecip_fast(piv);
            lk[k] = li;
            rpk[k] = r;
            uk[k] = cmul(sp[k], r);
            pl = cmul(pl, cneg(li));
            rprev = r;
        }
    }
    // ---- Dal_i = prod_{k <= i} (-l_k): multiplicative scan over the lanes, then the own rows -----------------------
    cplx pin = pl;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int dd = 1 << k;
        const cplx s = shfl_up_c(pin, dd);
        if (lane >= dd) pin = cmul(pin, s);
    }
    cplx Dal = shfl_up_c(pin, 1);
    if (lane == 0) Dal = one;
    // ---- backward affine scan: al_i = rp_i Dal_i - u_i al_{i+1}, be_i = -u_i be_{i+1} ---------------------------------
    cplx Rk[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        Rk[k] = zero;
        if (r0 + k < nj) {
            Dal = cneg(cmul(lk[k], Dal));
            Rk[k] = cmul(rpk[k], Dal);
        }
    }
    cplx A = one, B = zero;
    cplx alLast = zero, beLast = zero;
#pragma unroll
    for (int k = K - 1; k >= 0; --k) {
        if (r0 + k < nj) {
            B = cfnma(uk[k], B, Rk[k]);
            A = cmul(cneg(uk[k]), A);
            if (r0 + k == nj - 1) {
                alLast = Rk[k];
                beLast = cneg(uk[k]);
            }
        }
    }
    warp_scan_affine<-1, 5>(A, B, lane); // lane 0: the composite of all interior rows, applied to (al, be) = (0, 1) below
    const int lastLane = nj > 0 ? (nj - 1) / K : 0;
    alLast = shfl_c(alLast, lastLane);
    beLast = shfl_c(beLast, lastLane);
    if (lane == 0) {
        const bool has = nj > 0;
        const cplx al = B, be = A;
        sub2[g] = (g == 0 && !above) ? zero : (has ? cmul(subJ, alLast) : subJ);
        diag2[g] = has ? cfma(subJ, beLast, diagJ) : diagJ;
        if (g > 0 || above) {
            const cplx sa = sup[g0 - 1];
            diag2U[g - 1] = has ? cmul(sa, al) : zero;
            sup2[g - 1] = has ? cmul(sa, be) : sa;
        }
        if (g == ngroups - 1) {
            diag2U[g] = zero;
            sup2[g] = zero;
        }
    }
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicExch(err, 1);
    rs_store_rows(l + g0, ng, sbuf, lane, lk);
    rs_store_rows(rp + g0, ng, sbuf, lane, rpk);
    rs_store_rows(u + g0, ng, sbuf, lane, uk);
}

// LU of the last level's matrix by ONE WARP: rq_i = 1 / (diag_i - sub_i sup_{i-1} rq_{i-1}) is a Moebius map of
// rq_{i-1} (row matrix [[0, 1], [-sub_i sup_{i-1}, diag_i]], cn_factor.cuh); every lane composes the maps of its
// ceil(n/32) consecutive rows, a Kogge-Stone scan over the lanes gives each lane its inflow (row 0 has sub = 0, so
// everything is a constant map), and the lane recomputes its rows serially.  lw_w = sub_w rq_{w-1}, uw_w = sup_w rq_w.
__global__ void __launch_bounds__(32)
k_rs_factor_top_scan(int64_t n, const cplx *__restrict__ sub, const cplx *__restrict__ diag,
                     const cplx *__restrict__ sup, cplx *__restrict__ lw, cplx *__restrict__ rq, cplx *__restrict__ uw,
                     int *__restrict__ err)
{
    const int lane = threadIdx.x;
    const int64_t R = (n + 31) / 32, i0 = lane * R, i1 = (i0 + R < n) ? (i0 + R) : n;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    cn_mob M{one, zero, zero, one};
    cplx supprev = (i0 > 0 && i0 < n) ? sup[i0 - 1] : zero;
    const cplx sup0 = supprev;
    for (int64_t i = i0; i < i1; ++i) {
        const cplx ci = (i > 0) ? cmul(sub[i], supprev) : zero, di = diag[i];
        cn_mob Rm; // [[0, 1], [-c_i, d_i]] * M
        Rm.a = M.c;
        Rm.b = M.d;
        Rm.c = csub(cmul(di, M.c), cmul(ci, M.a));
        Rm.d = csub(cmul(di, M.d), cmul(ci, M.b));
        M = mob_scale(Rm);
        supprev = sup[i];
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int dd = 1 << k;
        cn_mob S = mob_shfl(M, lane - dd < 0 ? 0 : lane - dd);
        if (lane >= dd) M = mob_scale(mob_mul(M, S));
    }
    cn_mob Pm = mob_shfl(M, lane == 0 ? 0 : lane - 1);
    cplx rqprev = (lane == 0) ? zero : cmul(Pm.b, crecip_fast(Pm.d));
    bool bad = false;
    supprev = sup0;
    for (int64_t i = i0; i < i1; ++i) {
        const cplx si = sup[i];
        cplx lq = (i > 0) ? cmul(sub[i], rqprev) : zero;
        cplx piv = cfnma(lq, supprev, diag[i]);
        if (!cfinite_nonzero(piv)) bad = true;
        cplx r = crecip_fast(piv);
        lw[i] = lq;
        rq[i] = r;
        uw[i] = cmul(si, r);
        rqprev = r;
        supprev = si;
    }
    if (bad) atomicMax(err, 1); // (max: keeps the 2 of k_shard_assemble_top)
}

// diag += diagU (the two-writer accumulation of the next level's diagonal)
// (diagAboveAcc: a shard with a predecessor also sums what its first groups add to the diagonal of the row above it)
__global__ void k_rs_add(int64_t n, cplx *__restrict__ diag, const cplx *__restrict__ diagU,
                         cplx *__restrict__ diagAboveAcc = nullptr)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) diag[i] = cadd(diag[i], diagU[i]);
    if (i == 0 && diagAboveAcc) *diagAboveAcc = cadd(*diagAboveAcc, diagU[-1]);
}

