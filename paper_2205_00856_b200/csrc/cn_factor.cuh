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
                                cplx *__restrict__ redSupU, cplx *__restrict__ redDiagU, int *__restrict__ err,
                                double *__restrict__ gamJ = nullptr) // gamJ: also gamma of the joint lines, per block
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
    if (gamJ) gamJ[w] = gam[J];
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

// ---- the same, chunk-parallel: one THREAD per chunk of 8 rows, a block = 2^LOGC consecutive lanes of a warp --------
// The pivot recurrence q_i = 1 / (mu_i - q_{i-1}) is a Moebius map of q_{i-1}; maps compose as 2x2 matrices
// [[a, b], [c, d]] : q -> (a q + b) / (c q + d), row i contributing [[0, 1], [-1, mu_i]].  Every thread multiplies the
// matrices of its 8 rows, a segmented Kogge-Stone scan over the lanes of the block composes them (a block's first
// chunk is entered by q = 0, so its map is the CONSTANT b / d and everything downstream of it is constant too), and
// each thread then recomputes its own 8 pivots serially from its true inflow.  Of the upward elimination only
// Z_{1,1} = (block matrix)^-1_{1,1} is needed; solving A x = e_1 with the downward factors (y_i = prod_{k<i} (-q_k),
// x_i = q_i (y_i - x_{i+1})) gives the closed form  Z_{1,1} = sum_i q_i prod_{k<i} q_k^2  over the block's interior rows:
// a running product in the same serial loop and one segmented SUM over the lanes of the block -- no second Moebius
// scan (it cost a third of this kernel's FP64 work).  The matrix of a chunk is rescaled by a power of two (a Moebius
// map does not change when its matrix is scaled), so |mu|^8 never overflows; the scan then multiplies at most 2^LOGC
// matrices with components below 2, which needs no further rescaling.
// Memory: a thread reads 64 contiguous bytes of V and writes 128 of q and 64 of gamma -- whole sectors, against one
// 8-byte access per row and per thread in k_factor_blocks (619 us at C2, P = 2^17; this kernel: see DESIGN.md 8c).
struct cn_mob {
    cplx a, b, c, d;
};
CN_DEVINL cn_mob mob_row(cn_mob M, cplx mu) // [[0, 1], [-1, mu]] * M
{
    cn_mob R;
    R.a = M.c;
    R.b = M.d;
    R.c = cmsub(mu, M.c, M.a);
    R.d = cmsub(mu, M.d, M.b);
    return R;
}
CN_DEVINL cn_mob mob_mul(cn_mob H, cn_mob L) // H * L : first L, then H
{
    cn_mob R;
    R.a = cfma(H.a, L.a, cmul(H.b, L.c));
    R.b = cfma(H.a, L.b, cmul(H.b, L.d));
    R.c = cfma(H.c, L.a, cmul(H.d, L.c));
    R.d = cfma(H.c, L.b, cmul(H.d, L.d));
    return R;
}
CN_DEVINL cn_mob mob_scale(cn_mob M)
{
    // scale by the power of two that brings the largest component into [1, 2): exact, and no division
    const double s = fmax(fmax(fmax(fabs(M.a.x), fabs(M.a.y)), fmax(fabs(M.b.x), fabs(M.b.y))),
                          fmax(fmax(fabs(M.c.x), fabs(M.c.y)), fmax(fabs(M.d.x), fabs(M.d.y))));
    const int e = (int)((__double_as_longlong(s) >> 52) & 0x7ff); // biased exponent
    double r = 1.0;
    if (e > 0 && e < 0x7ff && e < 2046 - 1) r = __longlong_as_double((long long)(2046 - e) << 52); // 2^(1023 - e)
    M.a = cmake(M.a.x * r, M.a.y * r);
    M.b = cmake(M.b.x * r, M.b.y * r);
    M.c = cmake(M.c.x * r, M.c.y * r);
    M.d = cmake(M.d.x * r, M.d.y * r);
    return M;
}
CN_DEVINL cn_mob mob_shfl(cn_mob M, int src)
{
    cn_mob R;
    R.a = shfl_c(M.a, src);
    R.b = shfl_c(M.b, src);
    R.c = shfl_c(M.c, src);
    R.d = shfl_c(M.d, src);
    return R;
}

template <int LOGC>
__global__ void __launch_bounds__(128)
k_factor_blocks_chunked(int64_t nchunks, double two_dx2, double rho, const double *__restrict__ V,
                        const double *__restrict__ tdG, double tdF, // potential = V + tdF * tdG when tdG != NULL (cn_step_td)
                        cplx *__restrict__ q, double *__restrict__ gam, cplx *__restrict__ redSubD,
                        cplx *__restrict__ redDiagD, cplx *__restrict__ redSupU, cplx *__restrict__ redDiagU,
                        int *__restrict__ err, int above = 0, // above: a shard precedes this one (cn_shard.cuh): the first
                                                              // block's JU matrix side goes to the guard element [-1]
                        int64_t cutMask = ~(int64_t)0,        // independent systems of cutMask + 1 blocks (cn_pass_tiled.cuh)
                        double *__restrict__ gamJ = nullptr)  // also gamma of the joint lines, per block
{
    constexpr int CPB = 1 << LOGC;
    const int lane = threadIdx.x & 31;
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; // nchunks is a multiple of 32: whole warps
    if (c >= nchunks) return;
    const int pos = lane & (CPB - 1); // chunk position inside its block
    const bool isFirst = pos == 0, isLast = pos == CPB - 1;
    const int64_t w = c >> LOGC;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    double g[8];
    {
        const double2 *v2 = reinterpret_cast<const double2 *>(V + 8 * c);
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            double2 vv = v2[jj];
            if (tdG) {
                const double2 gg = reinterpret_cast<const double2 *>(tdG + 8 * c)[jj];
                vv.x = fma(tdF, gg.x, vv.x);
                vv.y = fma(tdF, gg.y, vv.y);
            }
            g[2 * jj] = fma(two_dx2, vv.x, 2.0);
            g[2 * jj + 1] = fma(two_dx2, vv.y, 2.0);
        }
        if (gam) { // (NULL under cn_step_td: the tiled pass recovers gamma from q, only gamJ is needed)
            double2 *g2 = reinterpret_cast<double2 *>(gam + 8 * c);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) g2[jj] = make_double2(g[2 * jj], g[2 * jj + 1]);
        }
    }
    const int nrow = isLast ? 7 : 8; // the joint line (row 7 of a block's last chunk) is not part of the recurrence
    // ---- downward: inflow of every chunk -----------------------------------------------------------------
    cn_mob M{one, zero, zero, one};
#pragma unroll
    for (int j = 0; j < 8; ++j)
        if (j < nrow) M = mob_row(M, cmake(-g[j], rho));
    if (isFirst) { M.a = zero; M.c = zero; } // entered by q = 0: the constant map b / d
    M = mob_scale(M);
#pragma unroll
    for (int k = 0; k < LOGC; ++k) {
        const int dd = 1 << k;
        cn_mob S = mob_shfl(M, lane - dd < 0 ? 0 : lane - dd);
        if (pos >= dd) M = mob_mul(M, S); // scaled chunk maps: <= 2 * 16^LOGC after the scan, no rescaling needed
    }
    cn_mob Pm = mob_shfl(M, lane == 0 ? 0 : lane - 1); // inclusive map of the chunk above: a constant inside a block
    cplx qin = isFirst ? zero : cmul(Pm.b, crecip_fast(Pm.d));
    bool bad = false;
    cplx pp = one, qlast = zero; // product of (-q) over this chunk's rows except the block's last interior row
    cplx tq = zero, zacc = zero;  // q_j prod_{k<j} q_k^2 over the rows of this chunk (k from the chunk's first row), its sum
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        if (j < nrow) {
            cplx p = cmake(-g[j] - qin.x, rho - qin.y);
            if (!cfinite_nonzero(p)) bad = true;
            const cplx qnew = crecip_fast(p);
            q[8 * c + j] = qnew;
            if (!(isLast && j == 6)) pp = cmul(pp, cneg(qnew));
            tq = (j == 0) ? qnew : cmul(cmul(tq, qlast), qnew);
            zacc = cadd(zacc, tq);
            qlast = qnew;
            qin = qnew;
        }
    }
    if (isLast) {
        q[8 * c + 7] = one;
        if (gamJ) gamJ[w] = g[7];
    }
#pragma unroll
    for (int k = 0; k < LOGC; ++k) { // product over the block, wanted at its last chunk
        const int dd = 1 << k;
        cplx sp = shfl_c(pp, lane - dd < 0 ? 0 : lane - dd);
        if (pos >= dd) pp = cmul(pp, sp);
    }
    // ---- Z_{1,1} = sum over the block of (prod of (-q) over the chunks before)^2 * (this chunk's sum) ----------------
    cplx yin = shfl_up_c(pp, 1); // inclusive product of the chunks before this one (all of them whole chunks)
    if (isFirst) yin = one;
    cplx zs = cmul(cmul(yin, yin), zacc);
#pragma unroll
    for (int k = 0; k < LOGC; ++k) {
        const int dd = 1 << k;
        const cplx s = shfl_down_c(zs, dd);
        if (pos + dd < CPB) zs = cadd(zs, s);
    }
    if (isLast) {
        const cplx Zn1 = cmul(qlast, pp);
        redSubD[w] = cneg(Zn1);
        redDiagD[w] = cneg(qlast);
        if ((w & cutMask) != 0 || above) redSupU[w - 1] = cneg(Zn1);
    }
    if (isFirst && ((w & cutMask) != 0 || above)) redDiagU[w - 1] = cneg(zs);
    if (bad) atomicExch(err, 1);
}

// potential of one driven step, V + f g (cn_step_td with the thread-per-block factor kernel)
__global__ void k_td_potential(int64_t N, const double *__restrict__ V0, const double *__restrict__ g, double f,
                               double *__restrict__ V)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) V[i] = fma(f, g[i], V0[i]);
}

// The same for one streamed part of the system (out-of-core mode, ooc_* in cn_api.cu): nb equal blocks of m rows whose
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
