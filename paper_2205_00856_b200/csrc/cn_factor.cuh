// cn_factorize kernels: everything of RD / RU / JD / JU / RS that does not touch d
// ("storage of a column of r_i factors ... most of the operations for these two
// stages can be carried without the knowledge of the solution vector d").
//
// Stored per point i (scaled system, cn_common.cuh):
//   q_i   = 1 / p_i, the inverse pivot of the block-local downward elimination (RD)
//           p_f = mu_f,  p_i = mu_i - q_{i-1}   for the interior rows f..J-1 of a block,
//           q_J = 1 at a joint line (the coupling of the next block's first row to the joint).
//           Because both off-diagonals of the scaled matrix are 1, q_{i-1} IS the RD multiplier
//           r_i of PAPER.md:306-316 (up to sign) and q_i is the 1/a_i of the SS stage.
//   gam_i = gamma_i = 2 + 2 dx^2 V_i  (real), diagonal of the scaled T^dagger / -T.
// Stored per joint line w: the LU factors (lw, rq, uw) of the reduced matrix of the RS stage
// (PAPER.md:112-114), whose rows are
//   -Z^w_{n,1} Psi_{w-1} + (mu_J - Z^w_{n,n} - Z^{w+1}_{1,1}) Psi_w - Z^{w+1}_{1,n} Psi_{w+1} = R_w
// with Z^w the inverse of block w's interior matrix (these are the fill-in columns b_i, c_i of
// PAPER.md:98 evaluated at the rows next to the joints, i.e. exactly what JD / JU add to a_J).
#pragma once
#include "cn_common.cuh"

struct cn_geom {
    int64_t N, P;
    // block w owns rows [off(w), off(w+1)), joint line J_w = off(w+1) - 1
    __host__ __device__ __forceinline__ int64_t off(int64_t w) const
    {
        return (N % P == 0) ? w * (N / P) : (int64_t)(((__int128)w * N) / P);
    }
};

// one thread per block: pivots, gamma, corner entries of Z^w
__global__ void k_factor_blocks(cn_geom g, double two_dx2, double rho, const double *__restrict__ V,
                                cplx *__restrict__ q, double *__restrict__ gam,
                                cplx *__restrict__ redSubD, cplx *__restrict__ redDiagD,
                                cplx *__restrict__ redSupU, cplx *__restrict__ redDiagU, int *__restrict__ err)
{
    int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= g.P) return;
    const int64_t f = g.off(w), J = g.off(w + 1) - 1;
    const int64_t n = J - f; // interior rows
    cplx qprev = cmake(0.0, 0.0);
    cplx prod = cmake(1.0, 0.0); // prod_{i=f}^{J-2} (-q_i)
    bool bad = false;
    for (int64_t i = f; i < J; ++i) {
        double gi = fma(two_dx2, V[i], 2.0);
        gam[i] = gi;
        cplx p = cmake(-gi - qprev.x, rho - qprev.y);
        if (!cfinite_nonzero(p)) bad = true;
        cplx qi = crecip(p);
        q[i] = qi;
        if (i < J - 1) prod = cmul(prod, cneg(qi));
        qprev = qi;
    }
    gam[J] = fma(two_dx2, V[J], 2.0);
    q[J] = cmake(1.0, 0.0);
    if (n >= 1) {
        cplx Znn = qprev;
        cplx Zn1 = cmul(qprev, prod);
        // upward pivots (the RU direction) only to get Z_{1,1} = 1 / pu_f; nothing of it is stored
        cplx qu = cmake(0.0, 0.0);
        for (int64_t i = J - 1; i >= f; --i) {
            cplx p = cmake(-gam[i] - qu.x, rho - qu.y);
            if (!cfinite_nonzero(p)) bad = true;
            qu = crecip(p);
        }
        redSubD[w] = cneg(Zn1);
        redDiagD[w] = cneg(Znn);
        if (w > 0) {
            redSupU[w - 1] = cneg(Zn1); // Z is complex symmetric: Z_{1,n} = Z_{n,1}
            redDiagU[w - 1] = cneg(qu);
        }
    } else { // no interior row: the two joint lines are coupled directly by the off-diagonal 1
        redSubD[w] = cmake(1.0, 0.0);
        redDiagD[w] = cmake(0.0, 0.0);
        if (w > 0) {
            redSupU[w - 1] = cmake(1.0, 0.0);
            redDiagU[w - 1] = cmake(0.0, 0.0);
        }
    }
    if (bad) atomicExch(err, 1);
}

// The same for one streamed part of the system (out-of-core mode, cn_ooc.cuh): nb equal blocks of m rows whose
// V / q / gamma live in part-local arrays; block wl of the part is block w0 + wl of the system.  red* may be
// NULL (per-step recomputation of the factors: "neither the matrix nor the wavefunction ever need to be placed
// entirely on a single process").
// V and gam may be the SAME array (gamma replaces V in place).
__global__ void k_factor_part(int64_t nb, int64_t m, int64_t w0, double two_dx2, double rho, const double *V,
                              cplx *__restrict__ q, double *gam, cplx *__restrict__ redSubD,
                              cplx *__restrict__ redDiagD, cplx *__restrict__ redSupU, cplx *__restrict__ redDiagU,
                              int *__restrict__ err)
{
    int64_t wl = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (wl >= nb) return;
    const int64_t f = wl * m, J = f + m - 1, w = w0 + wl;
    cplx qprev = cmake(0.0, 0.0), prod = cmake(1.0, 0.0);
    bool bad = false;
    for (int64_t i = f; i < J; ++i) {
        double gi = fma(two_dx2, V[i], 2.0);
        gam[i] = gi;
        cplx p = cmake(-gi - qprev.x, rho - qprev.y);
        if (!cfinite_nonzero(p)) bad = true;
        cplx qi = crecip(p);
        q[i] = qi;
        if (i < J - 1) prod = cmul(prod, cneg(qi));
        qprev = qi;
    }
    gam[J] = fma(two_dx2, V[J], 2.0);
    q[J] = cmake(1.0, 0.0);
    if (redSubD) {
        if (m >= 2) {
            cplx Znn = qprev, Zn1 = cmul(qprev, prod), qu = cmake(0.0, 0.0);
            for (int64_t i = J - 1; i >= f; --i) {
                cplx p = cmake(-gam[i] - qu.x, rho - qu.y);
                if (!cfinite_nonzero(p)) bad = true;
                qu = crecip(p);
            }
            redSubD[w] = cneg(Zn1);
            redDiagD[w] = cneg(Znn);
            if (w > 0) {
                redSupU[w - 1] = cneg(Zn1);
                redDiagU[w - 1] = cneg(qu);
            }
        } else {
            redSubD[w] = cmake(1.0, 0.0);
            redDiagD[w] = cmake(0.0, 0.0);
            if (w > 0) {
                redSupU[w - 1] = cmake(1.0, 0.0);
                redDiagU[w - 1] = cmake(0.0, 0.0);
            }
        }
    }
    if (bad) atomicExch(err, 1);
}

// diagonal of the joint lines for the level-0 reduced matrix when gamma is not resident: gJ[w] = gamma_{J_w}
__global__ void k_joint_gamma(int64_t nb, int64_t m, int64_t w0, const double *__restrict__ gam, double *__restrict__ gJ)
{
    int64_t wl = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (wl < nb) gJ[w0 + wl] = gam[wl * m + m - 1];
}

// serial LU of the reduced matrix (once per plan): lw_w = sub_w * rq_{w-1}, rq_w = 1/pivot, uw_w = sup_w * rq_w
__global__ void k_factor_reduced(cn_geom g, double rho, const double *__restrict__ gam,
                                 const cplx *__restrict__ redSubD, const cplx *__restrict__ redDiagD,
                                 const cplx *__restrict__ redSupU, const cplx *__restrict__ redDiagU,
                                 cplx *__restrict__ lw, cplx *__restrict__ rq, cplx *__restrict__ uw,
                                 int *__restrict__ err)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    cplx rqprev = cmake(0.0, 0.0), supprev = cmake(0.0, 0.0);
    bool bad = false;
    for (int64_t w = 0; w < g.P; ++w) {
        const int64_t J = g.off(w + 1) - 1;
        cplx diag = cmake(-gam[J] + redDiagD[w].x, rho + redDiagD[w].y);
        cplx sup = cmake(0.0, 0.0);
        if (w < g.P - 1) {
            diag = cadd(diag, redDiagU[w]);
            sup = redSupU[w];
        }
        cplx l = (w > 0) ? cmul(redSubD[w], rqprev) : cmake(0.0, 0.0);
        cplx piv = cfnma(l, supprev, diag);
        if (!cfinite_nonzero(piv)) bad = true;
        cplx r = crecip(piv);
        lw[w] = l;
        rq[w] = r;
        uw[w] = cmul(sup, r);
        rqprev = r;
        supprev = sup;
    }
    if (bad) atomicExch(err, 1);
}
