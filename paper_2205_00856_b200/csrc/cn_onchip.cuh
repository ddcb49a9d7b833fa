// Whole-system on-chip stepper for small N (config C1: N = 4096 is 64 KB of psi -- the entire problem lives in the
// registers of ONE CTA, and a cn_step(nsteps) call is ONE launch that loops over the steps on chip).
//
// The method is the same nest as everywhere else (PAPER.md:128-149 applied downwards): a thread's 8 consecutive
// rows are a block of the finest level (RD / RU / SS by serial sweeps in registers), the blocks of
// a warp are chained by the affine-map warp scan (the reduced system of that level), the warps through shared
// memory (the next level).  Stored factors: the inverse pivots qB of the downward elimination of the whole system
// and gamma, read ONCE per call; psi is read once and written once per call, so the per-step
// cost is pure latency and FP64 issue on one SM: 3 CTA barriers and two scans.  Eq. 3 is fused into the downward
// sweep.
#pragma once
#include "cn_common.cuh"

#define CN_ONCHIP_NMAX 4096 // 512 threads x 8 rows at 128 registers per thread

// Dynamic shared memory of k_onchip_steps<TPB>: the A-side of both CTA scans.  The matrix never changes inside the
// kernel, so every A product of the Kogge-Stone steps is a per-thread constant: it is computed ONCE before the step
// loop and the per-step scans move only B (one complex fused multiply-add per step instead of two products).
template <int TPB>
constexpr size_t onchip_smem_bytes()
{
    return (size_t)(2 * 5 * TPB + 2 * TPB + 2 * 5 * 32 + 2 * 32 + 64) * sizeof(cplx);
}

template <int TPB>
__global__ void __launch_bounds__(TPB, 1)
k_onchip_steps(int64_t N, int64_t nsteps, double rho, cplx *psi, const cplx *__restrict__ qB,
               const double *__restrict__ gam)
{
    extern __shared__ __align__(16) uint8_t onchip_smem[];
    cplx *const sM = (cplx *)onchip_smem;    // [2 dirs][5 steps][TPB]  multiplier of the warp-level step (0 = no partner)
    cplx *const sAe = sM + 2 * 5 * TPB;      // [2][TPB]               inclusive A of the neighbouring lane
    cplx *const sWm = sAe + 2 * TPB;         // [2][5][32]             multipliers of the scan over the warp aggregates
    cplx *const sWB = sWm + 2 * 5 * 32;      // [2][32]                per-warp aggregates B of the current step
    cplx *const eLo = sWB + 2 * 32, *const eHi = eLo + 32;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    constexpr int NW = TPB / 32;
    const int64_t r0 = 8 * (int64_t)t;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);

    // ---- the matrix side: constants of this thread's 8 rows (rows >= N behave as psi = 0, q = 0) ----------
    cplx qv[8];
    double g[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const bool in = r0 + j < N;
        qv[j] = in ? qB[r0 + j] : zero;
        g[j] = in ? gam[r0 + j] : 0.0;
    }
    const cplx qm1 = (t > 0 && r0 - 1 < N) ? qB[r0 - 1] : zero;
    {
        cplx Qp = cneg(qv[0]);
#pragma unroll
        for (int j = 1; j < 7; ++j) Qp = cmul(Qp, cneg(qv[j]));
        const cplx chunkA[2] = {cmul(cneg(qm1), Qp),   // downward: 0 for the first chunk
                                cmul(Qp, cneg(qv[7]))}; // upward
#pragma unroll
        for (int dir = 0; dir < 2; ++dir) { // 0: information flows to higher threads, 1: to lower threads
            cplx A = chunkA[dir];
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const int d = 1 << k;
                const bool ok = dir == 0 ? (lane >= d) : (lane + d < 32);
                sM[(dir * 5 + k) * TPB + t] = ok ? A : zero;
                const cplx As = dir == 0 ? shfl_up_c(A, d) : shfl_down_c(A, d);
                if (ok) A = cmul(A, As);
            }
            sAe[dir * TPB + t] = dir == 0 ? shfl_up_c(A, 1) : shfl_down_c(A, 1);
            if (lane == (dir == 0 ? 31 : 0)) sWB[dir * 32 + warp] = A; // borrowed for the aggregates A
            __syncthreads();
            cplx wA = (lane < NW) ? sWB[dir * 32 + lane] : one;
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const int d = 1 << k;
                const bool ok = dir == 0 ? (lane >= d) : (lane + d < 32);
                if (warp == 0) sWm[(dir * 5 + k) * 32 + lane] = ok ? wA : zero;
                const cplx wAs = dir == 0 ? shfl_up_c(wA, d) : shfl_down_c(wA, d);
                if (ok) wA = cmul(wA, wAs);
            }
        }
        __syncthreads();
    }
    // value entering this thread in direction dir when nothing enters the system (B-only scan, see above)
    auto scan_in = [&](int dir, cplx B) -> cplx {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const int d = 1 << k;
            const cplx Bs = dir == 0 ? shfl_up_c(B, d) : shfl_down_c(B, d);
            B = cfma(sM[(dir * 5 + k) * TPB + t], Bs, B);
        }
        if (lane == (dir == 0 ? 31 : 0)) sWB[dir * 32 + warp] = B;
        __syncthreads();
        cplx wB = (lane < NW) ? sWB[dir * 32 + lane] : zero;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const int d = 1 << k;
            const cplx wBs = dir == 0 ? shfl_up_c(wB, d) : shfl_down_c(wB, d);
            wB = cfma(sWm[(dir * 5 + k) * 32 + lane], wBs, wB);
        }
        const int src = dir == 0 ? warp - 1 : warp + 1; // inclusive composite of all warps before this one
        const bool has = dir == 0 ? (src >= 0) : (src < NW);
        const cplx cB = shfl_c(wB, has ? src : lane);
        const cplx carry = has ? cB : zero;
        const cplx Be = dir == 0 ? shfl_up_c(B, 1) : shfl_down_c(B, 1);
        const bool first = dir == 0 ? (lane == 0) : (lane == 31);
        return first ? carry : cfma(sAe[dir * TPB + t], carry, Be);
    };

    pdl_wait(); // psi may be the output of the preceding kernel on the stream
    pdl_launch_dependents();
    cplx v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = (r0 + j < N) ? psi[r0 + j] : zero;

    for (int64_t s = 0; s < nsteps; ++s) {
        // ---- neighbours of this chunk ------------------------------------------------------------------
        cplx vlo = shfl_up_c(v[7], 1), vhi = shfl_down_c(v[0], 1);
        if (NW > 1) {
            if (lane == 31) eLo[warp] = v[7];
            if (lane == 0) eHi[warp] = v[0];
            __syncthreads();
            if (lane == 0 && warp > 0) vlo = eLo[warp - 1];
            if (lane == 31 && warp < NW - 1) vhi = eHi[warp + 1];
        }
        if (t == 0) vlo = zero;
        if (t == TPB - 1) vhi = zero;
        // ---- Eq. 3 fused into RD ------------------------------------------------------
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
        D = scan_in(0, D);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
            E[j] = D;
        }
        // ---- RU + SS: x_j = q_j (d_j - x_{j+1}) -----------------------------------------
        cplx X = zero;
#pragma unroll
        for (int j = 7; j >= 0; --j) X = cmul(qv[j], csub(E[j], X));
        X = scan_in(1, X);
#pragma unroll
        for (int j = 7; j >= 0; --j) {
            X = cmul(qv[j], csub(E[j], X));
            v[j] = X;
        }
    }
#pragma unroll
    for (int j = 0; j < 8; ++j)
        if (r0 + j < N) psi[r0 + j] = v[j];
}
