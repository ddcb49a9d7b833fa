// Sharded mode: ONE system spread over several processes / GPUs, the wave function never gathered
// (PAPER.md:94, 161-165), one small exchange around the RS stage per step (section 5.2.1; the
// process layout of PAPER.md:282-288, section 6.2).
//
// A shard owns a contiguous range of rows = a whole number of blocks, with its own q, gamma, slots and its own nested
// RS levels (cn_reduced.cuh) built over ITS joint lines only.  The last row of a shard is a joint line at every level
// (the last row of the last group always is), so the shard is one block of the partition method applied once more at
// the top (Eq. 6): the reduced system of the last level is the concatenation of the shards' last
// levels, nt rows each, and is the only thing solved from exchanged data.
//   * matrix side, once per (H, dt): a shard's first block / first groups produce, level by level,
//     what they add to the diagonal of the row ABOVE the shard and that row's coupling to the shard's first row; both
//     land in the guard elements [-1] of the level arrays.  Record sent: [sum of the diagonal terms, coupling at the
//     last level, then sub / diag / sup of the shard's nt last-level rows].  Every shard assembles and factors the whole
//     last-level matrix (S nt rows) from the gathered records: RS replicated, no root process.
//   * per step: the JU contribution of the first block / first groups to the row above the shard is one value per level
//     (guard [-1] of every rU array); they all add into that row's last-level right-hand side, so every reduction
//     carries the guard of its level into the guard of the next.  Record sent: the two right-hand-side slots of the nt
//     last-level rows with that guard = 2 nt values (shard_rhs below) -- with nt = 1 exactly the two values per process
//     of PAPER.md:175 for a pre-factored matrix.  The replicated last level is solved from the gathered records
//     (k_shard_top, or inside the substitution kernel of the level below when it is small) and hands every shard the
//     support values of its own rows and of the row above it.
#pragma once
#include "cn_reduced.cuh"

// Per-step record of a shard, 2 nt values: [rD[0..nt), guard, rU[0..nt-1)] -- the two right-hand-side slots of its nt
// last-level rows exactly as its kernels write them (the record IS the storage of those arrays: nothing is packed),
// with the guard element of rU -- the JU contributions of all levels to the row above the shard, carried up level by
// level by k_rs_reduce -- in the middle, where rU[-1] lives.  rU of a shard's last row comes from the next shard (its
// guard) and has no slot.  Right-hand side of last-level row w of the whole system:
CN_DEVINL cplx shard_rhs(const cplx *gathered, int64_t S, int64_t nt, int64_t w)
{
    const int64_t rr = w / nt, j = w - rr * nt;
    const cplx *rec = gathered + rr * (2 * nt);
    cplx R = ld_dep(rec + j);
    if (j < nt - 1) R = cadd(R, ld_dep(rec + nt + 1 + j));
    else if (rr + 1 < S) R = cadd(R, ld_dep(gathered + (rr + 1) * (2 * nt) + nt)); // JU of the next shard
    return R;
}

// RS[M_last] of the sharded system, replicated on every shard: right-hand side of row
// w = r nt + j from the gathered records (shard_rhs), pre-factored matrix (lw, rq, uw), ONE CTA,
// K rows per thread (the structure of k_rs_top).  X: all S nt support values; guard0 (may be NULL): receives the
// support value of the row above this shard, X[toff - 1], where the level-0 array of the pass kernels expects it.
template <int K>
__global__ void __launch_bounds__(CN_RS_TOP_THREADS, 1)
k_shard_top(int64_t S, int64_t nt, const cplx *__restrict__ gathered, const cplx *__restrict__ lw,
            const cplx *__restrict__ rq, const cplx *__restrict__ uw, cplx *__restrict__ X, int64_t toff,
            cplx *__restrict__ guard0)
{
    __shared__ cplx sA[2][32], sB[2][32];
    const int t = threadIdx.x;
    const int64_t n = S * nt, w0 = (int64_t)t * K;
    const cplx zero = cmake(0.0, 0.0), one = cmake(1.0, 0.0);
    cplx l[K], r[K], u[K], R[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const bool in = w0 + k < n;
        l[k] = in ? lw[w0 + k] : zero;
        r[k] = in ? rq[w0 + k] : zero;
        u[k] = in ? uw[w0 + k] : zero;
    }
    pdl_wait();
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int64_t w = w0 + k;
        R[k] = (w < n) ? shard_rhs(gathered, S, nt, w) : zero;
    }
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
        R[k] = cmul(r[k], in);
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
        if (w0 + k < n) {
            X[w0 + k] = in;
            if (guard0 && w0 + k == toff - 1) *guard0 = in;
        }
    }
}

// matrix record of this shard (3 nt + 3 values): [diagonal terms for the row above, its coupling at the last level,
// sub, diag, sup, stamp = (nt, shard index)]; the stamp lets the receiver reject records of unequal shards
#define CN_SHARD_MREC(nt) (3 * (nt) + 3)
__global__ void k_shard_pack_matrix(int64_t nt, const cplx *__restrict__ sub, const cplx *__restrict__ diag,
                                    const cplx *__restrict__ sup, const cplx *__restrict__ diagAboveAcc, int above,
                                    int shard, cplx *__restrict__ rec)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < nt) {
        rec[2 + j] = sub[j];
        rec[2 + nt + j] = diag[j];
        rec[2 + 2 * nt + j] = sup[j];
    }
    if (j == 0) {
        rec[0] = above ? *diagAboveAcc : cmake(0.0, 0.0);
        rec[1] = above ? sup[-1] : cmake(0.0, 0.0);
        rec[2 + 3 * nt] = cmake((double)nt, (double)shard);
    }
}

// the whole last-level matrix (S nt rows) from the gathered matrix records
// (err := 2 when a record does not carry the stamp (nt, r): shards of unequal shape, or records out of rank order)
__global__ void k_shard_assemble_top(int64_t S, int64_t nt, const cplx *__restrict__ gathered, cplx *__restrict__ sub,
                                     cplx *__restrict__ diag, cplx *__restrict__ sup, int *__restrict__ err)
{
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= S * nt) return;
    const int64_t len = CN_SHARD_MREC(nt), r = w / nt, j = w - r * nt;
    const cplx *rec = gathered + r * len;
    if (j == 0 && !(rec[2 + 3 * nt].x == (double)nt && rec[2 + 3 * nt].y == (double)r)) atomicMax(err, 2);
    cplx d = rec[2 + nt + j], s = rec[2 + 2 * nt + j];
    if (j == nt - 1) { // the shard's last row: the next shard's first block / first groups complete it
        s = cmake(0.0, 0.0);
        if (r + 1 < S) {
            const cplx *nx = gathered + (r + 1) * len;
            d = cadd(d, nx[0]);
            s = nx[1];
        }
    }
    sub[w] = (w == 0) ? cmake(0.0, 0.0) : rec[2 + j];
    diag[w] = d;
    sup[w] = s;
}
