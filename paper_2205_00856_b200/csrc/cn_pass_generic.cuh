// Generic pass kernels: one thread serves one block, conventional layout, global memory accessed
// directly -- the shape of the paper's own CUDA kernels, kept as the path that
// accepts ANY (N, P) including unequal blocks, blocks with one interior row and blocks that are a
// joint line only.  It is the correctness fallback, not the fast path (cn_pass_tiled.cuh).
//
// One pass = [P1] finish step k:   RHS (Eq. 3) fused into the downward sweep RD,
//                                  upward sweep + SS with the two support values,
//                                  psi written in place;
//            [P2] start step k+1:  RHS of the new psi, RD and RU with zero support values, and the
//                                  JD / JU contributions to the two neighbouring joint lines, written
//                                  to two slots per joint line instead of atomics.
// P1 and P2 of successive steps are fused in one kernel ("integration between the substitution and
// reduction stages of the successive implicit steps").
#pragma once
#include "cn_factor.cuh"

template <bool P1, bool P2>
__global__ void k_pass_generic(cn_geom g, double rho, cplx *__restrict__ psi, const cplx *__restrict__ q,
                               const double *__restrict__ gam, cplx *__restrict__ work,
                               const cplx *__restrict__ supOld, const cplx *__restrict__ supNew,
                               cplx *__restrict__ slotD, cplx *__restrict__ slotU, cplx *__restrict__ supInit)
{
    pdl_wait();
    pdl_launch_dependents();
    int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= g.P) return;
    const int64_t f = g.off(w), J = g.off(w + 1) - 1;
    const cplx zero = cmake(0.0, 0.0);

    if (P1) {
        // old psi at the joint above comes from the previous RS output: the neighbour may already have
        // overwritten psi[f-1] with the new value (in-place update hazard, SURVEY 7 "hard parts")
        cplx lo = (w > 0) ? supOld[w - 1] : zero;
        cplx Dprev = (w > 0) ? supNew[w - 1] : zero; // D at a joint line := its new support value
        cplx qprev = cmake(1.0, 0.0);
        cplx cur = psi[f];
        for (int64_t i = f; i < J; ++i) {
            cplx hi = psi[i + 1];
            cplx E = rhs_E(gam[i], rho, cur, lo, hi);
            cplx D = cfnma(qprev, Dprev, E); // RD on d:  d_i += r_i d_{i-1}   (Eq. 11)
            work[i] = D;
            qprev = q[i];
            Dprev = D;
            lo = cur;
            cur = hi;
        }
        cplx x = supNew[w];
        psi[J] = x;
        for (int64_t i = J - 1; i >= f; --i) { // RU + SS:  x_i = q_i (D_i - x_{i+1})
            x = cmul(q[i], csub(work[i], x));
            psi[i] = x;
        }
    }
    if (P2) {
        cplx lo;
        if (P1) lo = (w > 0) ? supNew[w - 1] : zero;
        else lo = (w > 0) ? psi[f - 1] : zero; // prologue: nobody writes psi
        cplx Dprev = zero, qprev = cmake(1.0, 0.0);
        cplx cur = psi[f];
        for (int64_t i = f; i < J; ++i) {
            cplx hi = psi[i + 1];
            cplx E = rhs_E(gam[i], rho, cur, lo, hi);
            cplx D = cfnma(qprev, Dprev, E);
            work[i] = D;
            qprev = q[i];
            Dprev = D;
            lo = cur;
            cur = hi;
        }
        // here cur = psi_J (new), lo = psi_{J-1} (new; the joint above if the block has no interior row)
        cplx y = zero, yn = zero;
        for (int64_t i = J - 1; i >= f; --i) {
            y = cmul(q[i], csub(work[i], y));
            if (i == J - 1) yn = y;
        }
        // JD: E_J without its psi_{J+1} term, minus the local solution next to the joint
        cplx EJ = rhs_E(gam[J], rho, cur, lo, zero);
        slotD[w] = csub(EJ, yn);
        // JU: the psi_{J+1} term of the joint above and the local solution next to it
        if (w > 0) slotU[w - 1] = cneg(cadd(psi[f], y)); // J == f: psi[f] is the joint itself and y = 0
        if (w == g.P - 1) slotU[w] = zero;
        if (!P1) supInit[w] = cur;
    }
}
