// RS stage: solve the reduced tridiagonal system on the joint lines.
//
// The paper solves it serially ("implemented serially", beta * n_bl in its model) and
// notes that it can itself be parallelised.  Here the pre-factored system is
// solved by ONE CTA: every thread owns a contiguous chunk of joint lines, sweeps it serially, and the
// chunks are chained by the affine-map scan of cn_common.cuh, so the serial depth is P / threads.
#pragma once
#include "cn_common.cuh"

// Exclusive scan over the threads of a CTA.  (A, B) is this thread's chunk map; returns the value
// entering this thread's chunk, given `tin` entering the first chunk in direction DIR.
// sA, sB: shared arrays of >= 32 cplx, not in use by anyone else until the trailing barrier.
template <int DIR>
CN_DEVINL cplx block_scan_affine_excl(cplx A, cplx B, cplx tin, cplx *sA, cplx *sB)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    warp_scan_affine<DIR, 5>(A, B, lane);
    if (lane == (DIR > 0 ? 31 : 0)) {
        sA[warp] = A;
        sB[warp] = B;
    }
    __syncthreads();
    cplx carry = tin;
    if (DIR > 0) {
        for (int v = 0; v < warp; ++v) carry = cfma(sA[v], carry, sB[v]);
    } else {
        for (int v = nwarps - 1; v > warp; --v) carry = cfma(sA[v], carry, sB[v]);
    }
    cplx Ae = (DIR > 0) ? shfl_up_c(A, 1) : shfl_down_c(A, 1);
    cplx Be = (DIR > 0) ? shfl_up_c(B, 1) : shfl_down_c(B, 1);
    const bool first = (DIR > 0) ? (lane == 0) : (lane == 31);
    cplx in = first ? carry : cfma(Ae, carry, Be);
    __syncthreads();
    return in;
}

// R_w = slotD[w] + slotU[w]  (the two extra elements per joint line of PAPER.md:102, summed here)
__global__ void __launch_bounds__(1024, 1)
k_rs_single(int64_t P, const cplx *__restrict__ slotD, const cplx *__restrict__ slotU,
            const cplx *__restrict__ lw, const cplx *__restrict__ rq, const cplx *__restrict__ uw,
            cplx *__restrict__ sup)
{
    __shared__ cplx sA[32], sB[32];
    const int T = blockDim.x, t = threadIdx.x;
    const int64_t K = (P + T - 1) / T;
    const int64_t w0 = (int64_t)t * K, w1 = (w0 + K < P) ? (w0 + K) : P;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);

    // forward elimination  R'_w = R_w - lw_w R'_{w-1}   (e_d / f_d on the joint lines)
    cplx A = one, B = zero;
    for (int64_t w = w0; w < w1; ++w) {
        cplx l = lw[w];
        B = cfnma(l, B, cadd(slotD[w], slotU[w]));
        A = cmul(cneg(l), A);
    }
    cplx in = block_scan_affine_excl<+1>(A, B, zero, sA, sB);
    for (int64_t w = w0; w < w1; ++w) {
        in = cfnma(lw[w], in, cadd(slotD[w], slotU[w]));
        sup[w] = in; // R'_w, same thread reads it back below
    }
    // back substitution  Psi_w = rq_w R'_w - uw_w Psi_{w+1}
    A = one;
    B = zero;
    for (int64_t w = w1 - 1; w >= w0; --w) {
        cplx u = uw[w];
        B = cfnma(u, B, cmul(rq[w], sup[w]));
        A = cmul(cneg(u), A);
    }
    in = block_scan_affine_excl<-1>(A, B, zero, sA, sB);
    for (int64_t w = w1 - 1; w >= w0; --w) {
        in = cfnma(uw[w], in, cmul(rq[w], sup[w]));
        sup[w] = in;
    }
}
