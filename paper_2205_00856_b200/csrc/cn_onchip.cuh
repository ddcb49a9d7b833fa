// Whole-system on-chip stepper for small N (config C1: N = 4096 is 64 KB of psi -- the entire problem lives in the
// registers of ONE CTA, and a cn_step(nsteps) call is ONE launch that loops over the steps on chip).
//
// The method is the same nest as everywhere else (PAPER.md:128-149 applied downwards): a thread's 8 consecutive
// rows are a block of the finest level (RD / RU / SS by serial sweeps in registers), the blocks of
// a warp are chained by the affine-map warp scan (the reduced system of that level), the warps through shared
// memory (the next level).  Stored factors: the inverse pivots qB of the downward elimination of the whole system
// and gamma, read ONCE per call; psi is read once and written once per call, so the per-step
// cost is pure latency: 3 CTA barriers and two scans.  Eq. 3 is fused into the downward sweep.
#pragma once
#include "cn_common.cuh"
#include "cn_reduced.cuh" // cta_scan_excl

#define CN_ONCHIP_NMAX 4096 // 512 threads x 8 rows at 128 registers per thread

template <int TPB>
__global__ void __launch_bounds__(TPB, 1)
k_onchip_steps(int64_t N, int64_t nsteps, double rho, cplx *psi, const cplx *__restrict__ qB,
               const double *__restrict__ gam)
{
    __shared__ cplx sA[2][32], sB[2][32], eLo[32], eHi[32];
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    constexpr int NW = TPB / 32;
    const int64_t r0 = 8 * (int64_t)t;
    const cplx zero = cmake(0.0, 0.0);

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
    cplx Qp = cneg(qv[0]);
#pragma unroll
    for (int j = 1; j < 7; ++j) Qp = cmul(Qp, cneg(qv[j]));
    const cplx fwdA = cmul(cneg(qm1), Qp); // 0 for the first chunk: nothing enters the system
    const cplx bwdA = cmul(Qp, cneg(qv[7]));

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
        D = cta_scan_excl<+1>(fwdA, D, zero, sA[0], sB[0]);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            D = cfnma((j == 0) ? qm1 : qv[j - 1], D, E[j]);
            E[j] = D;
        }
        // ---- RU + SS: x_j = q_j (d_j - x_{j+1}) -----------------------------------------
        cplx X = zero;
#pragma unroll
        for (int j = 7; j >= 0; --j) X = cmul(qv[j], csub(E[j], X));
        X = cta_scan_excl<-1>(bwdA, X, zero, sA[1], sB[1]);
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
