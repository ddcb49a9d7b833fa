// C-ABI of the library (include/cn_nshape.h): plan management, factorization and the step drivers.
// Host logic only; every arithmetic step of the path runs in the kernels of cn_*.cuh.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cn_nshape.h"
#include "cn_common.cuh"
#include "cn_factor.cuh"
#include "cn_pass_generic.cuh"
#include "cn_pass_tiled.cuh"
#include "cn_reduced.cuh"
#include "cn_batched.cuh"
#include "cn_onchip.cuh"
#include "cn_shard.cuh"

typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct cn_plan {
    int64_t N = 0, P = 0; // P: blocks the kernels work with (= Pu unless cn_factorize sub-partitions, see there)
    int64_t Pu = 0;       // the caller's partition count
    double dx = 0, dt = 0, rho = 0, two_dx2 = 0;
    // device state
    double *dV = nullptr;
    cplx *q = nullptr;
    double *gam = nullptr;
    cplx *lw = nullptr, *rq = nullptr, *uw = nullptr; // LU factors of the LAST RS level
    cplx *slotD = nullptr, *slotU = nullptr, *sup[2] = {nullptr, nullptr};
    cplx *work = nullptr;
    cplx *qB = nullptr; // whole-system inverse pivots for cn_batched_sweep (N <= CN_BATCHED_NMAX)
    int *derr = nullptr;
    // out-of-core mode (cn_ooc: psi in pinned host memory, streamed part by part)
    double *hV = nullptr;      // pinned host copy of V when it may not stay on the device
    bool ooc = false;
    int64_t partPts = 0;       // points per streamed part (a multiple of the tile and of the block size)
    int64_t nparts = 0;
    static const int NB = 3;   // parts in flight: copy in | compute | copy out
    cplx *bPsi[NB] = {nullptr, nullptr, nullptr}, *bQ[NB] = {nullptr, nullptr, nullptr};
    double *bV[NB] = {nullptr, nullptr, nullptr}; // V on arrival, gamma after k_factor_part (in place)
    CUtensorMap tmPsiB[NB], tmQB[NB], tmGamB[NB];
    double *gamJ = nullptr;    // gamma on the joint lines (the only per-point factor data kept, O(P))
    cudaStream_t sIn = nullptr, sCmp = nullptr, sOut = nullptr;
    cudaEvent_t evIn[NB] = {}, evCmp[NB] = {}, evFree[NB] = {}, evFork = nullptr, evJoin[3] = {};
    std::vector<cudaEvent_t> evHost; // per part: its new psi has landed in host memory
    size_t device_bytes = 0;
    std::vector<void *> owned; // every device allocation of the factorization (freed by free_factors)
    // RS levels: lv[0] is the reduced system on the P joint lines, lv[i+1] the reduced
    // system of lv[i] partitioned into groups of CN_RS_G rows; the last level is solved by one CTA
    struct rs_level {
        int64_t n = 0;
        cplx *sub = nullptr, *diag = nullptr, *sup = nullptr; // matrix of this level
        cplx *l = nullptr, *rp = nullptr, *u = nullptr;       // group-local factors (all but the last level)
        cplx *rD = nullptr, *rU = nullptr, *X = nullptr;      // two rhs slots per row, solution (levels >= 1)
    };
    std::vector<rs_level> lv;
    int64_t *off0 = nullptr; // caller-placed joint lines of level 0 (cn_tridiag_create_blocks): group g = rows [off0[g], off0[g+1])
    int64_t noff0 = 0;       // number of such groups
    // configuration
    int opt_path = 0, opt_tile_threads = 0, opt_rs_topmax = 4096, opt_rs_levels = 0, opt_profile = 0, opt_onchip = 1;
    int opt_pdl = 1, opt_rs_group = CN_RS_G, opt_rs_serial_top = 0, opt_rs_top_in_subst = 1, opt_keep_p = 0, opt_by_cols = 0;
    int64_t opt_rs_top_in_subst_max = 256; // measured at C2: faster up to 256 rows (160.8 vs 163.0 us), slower from 512 on
    // time-dependent H (cn_step_td): spatial shape g of the driving term, the potential of the current step and the
    // temporaries of the factorization kept alive so that cn_step_td never allocates
    double *tdG = nullptr, *tdV = nullptr;
    cplx *tdRed = nullptr;
    int64_t tdRedP = 0;
    // many systems with a potential of their own each (cn_plan_set_systems): the plan's N rows are nsys systems
    int sysMode = 0;        // 0 one system; 1 contiguous systems on the tiled kernels (cuts, cn_pass_tiled.cuh); 2 generic
    int sysWant = 0;        // what cn_plan_set_systems asked for (cn_factorize settles sysMode)
    int64_t sysN = 0, sysCount = 0, sysEs = 0, sysSs = 0; // rows per system, systems, strides (complex elements)
    // sharded mode (cn_shard_*; cn_shard.cuh): this plan holds rows of ONE system that nshards processes share
    int shard = 0, nshards = 1;
    bool above = false, below = false; // a shard precedes / follows this one
    int64_t nt = 0;                    // rows of this shard's last RS level (equal on all shards)
    cplx *topX[2] = {nullptr, nullptr}; // support values of the whole last level (nshards * nt), ping-pong like sup[]
    cplx *gsub = nullptr, *gdiag = nullptr, *gsup = nullptr; // the whole last-level matrix, assembled from the records
    cplx *diagAcc = nullptr;           // what this shard adds to the diagonal of the row above it, summed over the levels
    int sh_out = 1;                    // sup[] / topX[] buffer the pending RS writes
    bool sh_local_done = false;        // cn_shard_factorize_local has run, cn_shard_factorize_finish is due
    cplx *xbuf = nullptr;              // send / receive records of cn_shard_factorize / cn_shard_run
    // profiling (CN_OPT_PROFILE): event pairs around fused-pass (kind 0) and RS (kind 1) launches
    struct ev_pair { cudaEvent_t a, b; int kind; };
    std::vector<ev_pair> ev_pool;
    size_t ev_used = 0;
    size_t budget = 0;
    // derived at factorize
    bool factorized = false;
    int path = 0; // 1 generic, 2 tiled
    int tpb = 0, logc = 0;
    int grid_tiled = 0; // persistent grid of the tiled pass kernel
    // tensor maps
    encode_tiled_fn encode = nullptr;
    CUtensorMap tmQ, tmGam, tmPsi;
    const void *tmPsiFor = nullptr;
    // batched sweep: tensor map of the last (psi, nsys, strides) and the persistent grid of its kernel
    CUtensorMap tmBatch;
    const void *tmBatchFor = nullptr;
    int64_t tmBatchKey[3] = {0, 0, 0};
    int batchGrid = 0;
    int sms = 0;
    // bookkeeping
    int last_cuda = 0;
    int64_t launches = 0;
};

static cn_status cuda_fail(cn_plan *p, cudaError_t e)
{
    if (p) p->last_cuda = (int)e;
    return CN_ECUDA;
}
#define CN_CUDA(p, call)                                   \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return cuda_fail((p), e__); \
    } while (0)

template <typename T>
static cn_status dev_alloc(cn_plan *p, T **ptr, size_t count)
{
    size_t bytes = count * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    cudaError_t e = cudaMalloc((void **)ptr, bytes);
    if (e != cudaSuccess) {
        p->last_cuda = (int)e;
        (void)cudaGetLastError();
        return (e == cudaErrorMemoryAllocation) ? CN_ENOMEM : CN_ECUDA;
    }
    p->device_bytes += bytes;
    p->owned.push_back((void *)*ptr);
    return CN_OK;
}

// the same with one guard element in front (index -1), zeroed: sharded plans keep there what belongs to the row above
// the shard (cn_shard.cuh); `guard` = false is plain dev_alloc
template <typename T>
static cn_status dev_alloc_g(cn_plan *p, T **ptr, size_t count, bool guard)
{
    if (!guard) return dev_alloc(p, ptr, count);
    T *raw = nullptr;
    cn_status st = dev_alloc(p, &raw, count + 1);
    if (st != CN_OK) return st;
    if (cudaMemset(raw, 0, sizeof(T)) != cudaSuccess) return CN_ECUDA;
    *ptr = raw + 1;
    return CN_OK;
}

static void free_factors(cn_plan *p)
{
    for (void *x : p->owned) cudaFree(x);
    p->owned.clear();
    p->lv.clear();
    p->device_bytes = p->dV ? sizeof(double) * (size_t)p->N : 0;
    p->ooc = false;
    p->q = nullptr; p->gam = nullptr; p->lw = p->rq = p->uw = nullptr;
    p->slotD = p->slotU = nullptr; p->sup[0] = p->sup[1] = nullptr; p->work = nullptr; p->derr = nullptr;
    p->qB = nullptr;
    p->gamJ = nullptr;
    p->off0 = nullptr;
    p->topX[0] = p->topX[1] = nullptr; p->gsub = p->gdiag = p->gsup = nullptr; p->diagAcc = nullptr;
    p->sh_local_done = false;
    for (int b = 0; b < cn_plan::NB; ++b) { p->bPsi[b] = nullptr; p->bQ[b] = nullptr; p->bV[b] = nullptr; }
    p->factorized = false;
    p->tmPsiFor = nullptr;
    p->tmBatchFor = nullptr;
}

extern "C" const char *cn_version(void) { return "cn_nshape 0.2 (sm_100a)"; }

extern "C" const char *cn_status_string(cn_status s)
{
    switch (s) {
    case CN_OK: return "CN_OK";
    case CN_EINVAL: return "CN_EINVAL: invalid argument";
    case CN_ENOMEM: return "CN_ENOMEM: out of memory or device budget too small";
    case CN_ECUDA: return "CN_ECUDA: CUDA error (see cn_last_cuda_error)";
    case CN_ENOTFACTORIZED: return "CN_ENOTFACTORIZED: call cn_factorize first";
    case CN_EBREAKDOWN: return "CN_EBREAKDOWN: zero or non-finite pivot";
    case CN_ETOOLARGE: return "CN_ETOOLARGE: N exceeds CN_STATIC_NMAX (4096), the static device scratch of cn_step_static";
    }
    return "unknown cn_status";
}

extern "C" cn_status cn_last_cuda_error(const cn_plan *plan, int *cuda_err)
{
    if (!plan || !cuda_err) return CN_EINVAL;
    *cuda_err = plan->last_cuda;
    return CN_OK;
}

extern "C" cn_status cn_plan_create(cn_plan **out, int64_t N, int64_t P, double dx, double dt, const double *V)
{
    if (!out) return CN_EINVAL;
    *out = nullptr;
    if (!V || N < 2 || P < 1 || P > N) return CN_EINVAL;
    if (!std::isfinite(dx) || !std::isfinite(dt) || dx <= 0.0 || dt == 0.0) return CN_EINVAL;
    cn_plan *p = new (std::nothrow) cn_plan();
    if (!p) return CN_ENOMEM;
    p->N = N; p->P = P; p->Pu = P; p->dx = dx; p->dt = dt;
    p->rho = 4.0 * dx * dx / dt; // 1 / s
    p->two_dx2 = 2.0 * dx * dx;
    cn_status st = dev_alloc(p, &p->dV, (size_t)N);
    if (st != CN_OK) { delete p; return st; }
    p->owned.clear(); // V lives as long as the plan; `owned` lists what cn_factorize allocates
    // V may be a host or a device pointer; cudaMemcpyDefault resolves it (UVA)
    cudaError_t e = cudaMemcpy(p->dV, V, sizeof(double) * (size_t)N, cudaMemcpyDefault);
    if (e != cudaSuccess) { cudaFree(p->dV); delete p; return CN_ECUDA; }
    *out = p;
    return CN_OK;
}

extern "C" cn_status cn_destroy(cn_plan *plan)
{
    if (!plan) return CN_EINVAL;
    free_factors(plan);
    if (plan->dV) cudaFree(plan->dV);
    if (plan->tdG) cudaFree(plan->tdG);
    if (plan->tdV) cudaFree(plan->tdV);
    if (plan->tdRed) cudaFree(plan->tdRed);
    if (plan->xbuf) cudaFree(plan->xbuf);
    if (plan->hV) cudaFreeHost(plan->hV);
    if (plan->sIn) cudaStreamDestroy(plan->sIn);
    if (plan->sCmp) cudaStreamDestroy(plan->sCmp);
    if (plan->sOut) cudaStreamDestroy(plan->sOut);
    for (int b = 0; b < cn_plan::NB; ++b) {
        if (plan->evIn[b]) cudaEventDestroy(plan->evIn[b]);
        if (plan->evCmp[b]) cudaEventDestroy(plan->evCmp[b]);
        if (plan->evFree[b]) cudaEventDestroy(plan->evFree[b]);
        if (plan->evJoin[b]) cudaEventDestroy(plan->evJoin[b]);
    }
    if (plan->evFork) cudaEventDestroy(plan->evFork);
    for (auto &e : plan->evHost) cudaEventDestroy(e);
    for (auto &e : plan->ev_pool) {
        cudaEventDestroy(e.a);
        cudaEventDestroy(e.b);
    }
    delete plan;
    return CN_OK;
}

// device bytes the in-core path needs: V, q, gamma (psi is the caller's) + the O(P) reduced-system arrays
static size_t incore_bytes(const cn_plan *p)
{
    const int64_t P = p->P > p->Pu ? p->P : p->Pu;
    return (size_t)p->N * (8 + 16 + 8) + (size_t)P * 16 * 14;
}

extern "C" cn_status cn_plan_set_device_budget(cn_plan *plan, size_t bytes)
{
    if (!plan) return CN_EINVAL;
    free_factors(plan);
    plan->budget = bytes;
    const bool want_host = bytes != 0 && incore_bytes(plan) > bytes;
    const size_t vb = sizeof(double) * (size_t)plan->N;
    if (want_host && !plan->hV) { // V leaves the device: keep a pinned host copy to stream from
        CN_CUDA(plan, cudaMallocHost((void **)&plan->hV, vb));
        CN_CUDA(plan, cudaMemcpy(plan->hV, plan->dV, vb, cudaMemcpyDeviceToHost));
        cudaFree(plan->dV);
        plan->dV = nullptr;
    } else if (!want_host && plan->hV) {
        CN_CUDA(plan, cudaMalloc((void **)&plan->dV, vb));
        CN_CUDA(plan, cudaMemcpy(plan->dV, plan->hV, vb, cudaMemcpyHostToDevice));
        cudaFreeHost(plan->hV);
        plan->hV = nullptr;
    }
    plan->device_bytes = plan->dV ? vb : 0;
    return CN_OK;
}

extern "C" cn_status cn_plan_set_option(cn_plan *plan, cn_option key, int64_t value)
{
    if (!plan) return CN_EINVAL;
    switch (key) {
    case CN_OPT_PATH:
        if (value < 0 || value > 2) return CN_EINVAL;
        plan->opt_path = (int)value;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_TILE_THREADS:
        if (value != 0 && value != 32 && value != 64 && value != 128 && value != 256 && value != 512) return CN_EINVAL;
        plan->opt_tile_threads = (int)value;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_RS_TOPMAX:
        if (value < 1 || value > 8 * CN_RS_TOP_THREADS) return CN_EINVAL;
        plan->opt_rs_topmax = (int)value;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_PDL:
        plan->opt_pdl = value ? 1 : 0;
        return CN_OK;
    case CN_OPT_ONCHIP:
        plan->opt_onchip = value ? 1 : 0;
        return CN_OK;
    case CN_OPT_RS_GROUP:
        if (value < 2 || value > (1 << 20)) return CN_EINVAL;
        plan->opt_rs_group = (int)value;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_RS_SERIAL_TOP:
        plan->opt_rs_serial_top = value ? 1 : 0;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_RS_TOP_IN_SUBST:
        plan->opt_rs_top_in_subst = value ? 1 : 0;
        plan->opt_rs_top_in_subst_max = value > 1 ? (value > 1024 ? 1024 : value) : 256; // value > 1: the row limit
        return CN_OK;
    case CN_OPT_KEEP_P:
        plan->opt_keep_p = value ? 1 : 0;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_BY_COLS:
        if (value != 0 && value != 4 && value != 8) return CN_EINVAL;
        plan->opt_by_cols = (int)value;
        plan->tmBatchFor = nullptr;
        return CN_OK;
    case CN_OPT_RS_LEVELS:
        if (value < -1 || value > 8) return CN_EINVAL;
        plan->opt_rs_levels = (int)value;
        plan->factorized = false;
        return CN_OK;
    case CN_OPT_PROFILE:
        plan->opt_profile = value ? 1 : 0;
        return CN_OK;
    }
    return CN_EINVAL;
}

// the whole system is stepped on chip by one CTA (cn_onchip.cuh) when nothing asks for a particular kernel family
static bool onchip_active(const cn_plan *p)
{
    return p->opt_onchip && p->opt_path == 0 && p->opt_rs_levels == 0 && !p->opt_profile && !p->ooc && p->qB && !p->sysMode &&
           p->N <= CN_ONCHIP_NMAX;
}

extern "C" cn_status cn_plan_get_info(const cn_plan *plan, cn_plan_info *info)
{
    if (!plan || !info) return CN_EINVAL;
    memset(info, 0, sizeof *info);
    info->N = plan->N; info->P = plan->Pu;
    info->P_effective = plan->P;
    info->path = onchip_active(plan) ? 3 : plan->path;
    info->tile_threads = plan->tpb;
    info->tile_points = plan->ooc ? plan->partPts : (int64_t)plan->tpb * 8;
    info->rs_levels = (plan->opt_rs_levels < 0) ? -1 : (int32_t)plan->lv.size();
    info->out_of_core = plan->ooc ? 1 : 0;
    info->device_bytes = plan->device_bytes;
    info->launches = plan->launches;
    info->bytes_per_point_step = (plan->path == 2) ? 48.0 : 56.0; // the tiled pass recovers gamma from q: psi 16 + q 16 in, psi 16 out
    return CN_OK;
}

// ---- tensor maps ---------------------------------------------------------------------------------------
static cn_status get_encoder(cn_plan *p)
{
    if (p->encode) return CN_OK;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CN_CUDA(p, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return CN_ECUDA;
    p->encode = (encode_tiled_fn)fn;
    return CN_OK;
}

// 2-D view [rows = N/8][inner doubles] of a contiguous array; inner = 16 (complex) or 8 (real)
static cn_status make_map(cn_plan *p, CUtensorMap *map, const void *base, int inner, int box_rows, int64_t rows = 0)
{
    cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)(rows ? rows : p->N / 8)};
    cuuint64_t strides[1] = {(cuuint64_t)inner * 8};
    cuuint32_t box[2] = {(cuuint32_t)inner, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = p->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE,
                           inner == 16 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        p->last_cuda = (int)cudaErrorInvalidValue;
        return CN_ECUDA;
    }
    return CN_OK;
}

// ---- kernel dispatch of the tiled path ---------------------------------------------------------------
typedef void (*tiled_kernel_t)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const cn_tiled_params);

template <int TPB, int LOGC, int MODE>
static tiled_kernel_t tiled_kernel_inst()
{
    constexpr int MINB = (TPB == 32) ? 16 : (TPB == 64) ? 8 : ((TPB == 128) ? 4 : (TPB == 256 ? 2 : 1));
    if (MODE == 0) return k_pass_tiled<TPB, LOGC, false, true, MINB>;
    if (MODE == 1) return k_pass_tiled<TPB, LOGC, true, true, MINB>;
    return k_pass_tiled<TPB, LOGC, true, false, MINB>;
}

template <int TPB, int MODE>
static tiled_kernel_t tiled_kernel_for_logc(int logc)
{
    switch (logc) {
    case 0: return tiled_kernel_inst<TPB, 0, MODE>();
    case 1: return tiled_kernel_inst<TPB, 1, MODE>();
    case 2: return tiled_kernel_inst<TPB, 2, MODE>();
    case 3: return tiled_kernel_inst<TPB, 3, MODE>();
    case 4: return tiled_kernel_inst<TPB, 4, MODE>();
    case 5: return tiled_kernel_inst<TPB, 5, MODE>();
    case 6: if (TPB >= 64) return tiled_kernel_inst<(TPB >= 64 ? TPB : 64), 6, MODE>(); break;
    case 7: if (TPB >= 128) return tiled_kernel_inst<(TPB >= 128 ? TPB : 128), 7, MODE>(); break;
    case 8: if (TPB >= 256) return tiled_kernel_inst<(TPB >= 256 ? TPB : 256), 8, MODE>(); break;
    case 9: if (TPB >= 512) return tiled_kernel_inst<(TPB >= 512 ? TPB : 512), 9, MODE>(); break;
    }
    return nullptr;
}

static tiled_kernel_t tiled_kernel(int tpb, int logc, int mode)
{
#define CN_PICK(T)                                               \
    if (tpb == T) {                                              \
        if (mode == 0) return tiled_kernel_for_logc<T, 0>(logc); \
        if (mode == 1) return tiled_kernel_for_logc<T, 1>(logc); \
        return tiled_kernel_for_logc<T, 2>(logc);                \
    }
    CN_PICK(32)
    CN_PICK(64)
    CN_PICK(128)
    CN_PICK(256)
    CN_PICK(512)
#undef CN_PICK
    return nullptr;
}

static size_t tiled_smem(int tpb)
{
    return tpb == 32 ? tiled_smem_bytes<32>() : tpb == 64 ? tiled_smem_bytes<64>()
                     : (tpb == 128 ? tiled_smem_bytes<128>() : (tpb == 256 ? tiled_smem_bytes<256>() : tiled_smem_bytes<512>()));
}


// ---- out-of-core mode (config C5) -----------------------------------------------------
// psi stays in the caller's PINNED HOST memory and V in the plan's pinned copy.  The system is streamed in parts
// of partPts points (whole blocks, whole tiles): copy in (psi 16 B + V 8 B per point) | k_factor_part + fused pass
// | copy out (16 B per point) on three streams over NB rotating device buffers.  Only the joint-line arrays (slots,
// support values, reduced-system factors: O(P)) persist on the device between passes.
static cn_status ooc_setup(cn_plan *p, int64_t m)
{
    const int64_t N = p->N, P = p->P;
    cn_status st;
    // what is already owned (joint-line arrays) + the transient of the factorization; the rest: NB parts of 40 B per point
    const size_t fixed = p->device_bytes + (size_t)P * 16 * 6;
    const int64_t unit = ((int64_t)p->tpb * 8 > m) ? (int64_t)p->tpb * 8 : m; // both are powers of two times 8
    if (p->budget <= fixed) return CN_ENOMEM;
    int64_t pts = (int64_t)((p->budget - fixed) / (cn_plan::NB * 40));
    if (pts > (1LL << 23)) pts = 1LL << 23; // 128 MB of psi per copy is plenty to reach the link rate
    pts = pts / unit * unit;
    if (pts < unit) return CN_ENOMEM;
    if (pts > N) pts = (N + unit - 1) / unit * unit;
    p->partPts = pts;
    p->nparts = (N + pts - 1) / pts;
    if ((st = get_encoder(p)) != CN_OK) return st;
    const int box_rows = p->tpb < 256 ? p->tpb : 256;
    for (int b = 0; b < cn_plan::NB; ++b) {
        if ((st = dev_alloc(p, &p->bPsi[b], (size_t)pts)) != CN_OK) return st;
        if ((st = dev_alloc(p, &p->bQ[b], (size_t)pts)) != CN_OK) return st;
        if ((st = dev_alloc(p, &p->bV[b], (size_t)pts)) != CN_OK) return st;
        // a last part shorter than the buffers leaves the tail of its last tile untouched: the inactive lanes of that
        // tile must read finite values (0 * garbage in the unpredicated scans would be NaN for Inf / NaN garbage)
        CN_CUDA(p, cudaMemset(p->bPsi[b], 0, sizeof(cplx) * (size_t)pts));
        CN_CUDA(p, cudaMemset(p->bQ[b], 0, sizeof(cplx) * (size_t)pts));
        CN_CUDA(p, cudaMemset(p->bV[b], 0, sizeof(double) * (size_t)pts));
        if ((st = make_map(p, &p->tmPsiB[b], p->bPsi[b], 16, box_rows, pts / 8)) != CN_OK) return st;
        if ((st = make_map(p, &p->tmQB[b], p->bQ[b], 16, box_rows, pts / 8)) != CN_OK) return st;
        if ((st = make_map(p, &p->tmGamB[b], p->bV[b], 8, box_rows, pts / 8)) != CN_OK) return st;
        if (!p->evIn[b]) {
            CN_CUDA(p, cudaEventCreateWithFlags(&p->evIn[b], cudaEventDisableTiming));
            CN_CUDA(p, cudaEventCreateWithFlags(&p->evCmp[b], cudaEventDisableTiming));
            CN_CUDA(p, cudaEventCreateWithFlags(&p->evFree[b], cudaEventDisableTiming));
            CN_CUDA(p, cudaEventCreateWithFlags(&p->evJoin[b], cudaEventDisableTiming));
        }
    }
    if (!p->sIn) {
        CN_CUDA(p, cudaStreamCreateWithFlags(&p->sIn, cudaStreamNonBlocking));
        CN_CUDA(p, cudaStreamCreateWithFlags(&p->sCmp, cudaStreamNonBlocking));
        CN_CUDA(p, cudaStreamCreateWithFlags(&p->sOut, cudaStreamNonBlocking));
        CN_CUDA(p, cudaEventCreateWithFlags(&p->evFork, cudaEventDisableTiming));
    }
    while ((int64_t)p->evHost.size() < p->nparts) {
        cudaEvent_t e;
        CN_CUDA(p, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        p->evHost.push_back(e);
    }
    for (int mode = 0; mode < 3; ++mode) {
        tiled_kernel_t k = tiled_kernel(p->tpb, p->logc, mode);
        if (!k) return CN_EINVAL;
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tiled_smem(p->tpb)));
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    }
    int dev = 0, sms = 0, per_sm = 0;
    CN_CUDA(p, cudaGetDevice(&dev));
    CN_CUDA(p, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CN_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)tiled_kernel(p->tpb, p->logc, 1), p->tpb,
                                                             tiled_smem(p->tpb)));
    if (per_sm < 1) return CN_ECUDA;
    const int64_t tiles = (pts / 8 + p->tpb - 1) / p->tpb, slots = (int64_t)sms * per_sm;
    p->grid_tiled = (int)(tiles < slots ? tiles : slots);
    return CN_OK;
}

// The arithmetic of the factorization: every matrix-side quantity of RD/RU/JD/JU from the potential
// `Vsrc`, the reduced matrices of all RS levels and their factors.  Launches only (no allocation, no synchronisation):
// cn_factorize calls it once, cn_step_td once per step with the potential of that step.  `red`: CN_RED_COUNT(P) complex
// scratch = six arrays of P values, each with a guard element in front (used by sharded plans only).
#define CN_RED_COUNT(P) (6 * ((size_t)(P) + 1))
static cn_status factor_compute(cn_plan *p, const double *Vsrc, cplx *red, int64_t m, cudaStream_t stream, bool whole = true,
                                const double *tdG = nullptr, double tdF = 0.0)
{
    const int64_t N = p->N, P = p->P;
    const int nlv = (int)p->lv.size();
    cn_status st;
    const int64_t Pg = P + 1;
    cplx *redSubD = red + 1, *redDiagD = red + Pg + 1, *redSupU = red + 2 * Pg + 1, *redDiagU = red + 3 * Pg + 1;
    cplx *tmpA = red + 4 * Pg + 1, *tmpB = red + 5 * Pg + 1;
    const int above = p->above ? 1 : 0;
    const bool sharded = p->nshards > 1;
    const int64_t cutMask = (p->sysMode == 1) ? p->sysN / m - 1 : ~(int64_t)0; // blocks per system - 1 (a power of two)
    CN_CUDA(p, cudaMemsetAsync(red, 0, sizeof(cplx) * CN_RED_COUNT(P), stream));
    CN_CUDA(p, cudaMemsetAsync(p->derr, 0, sizeof(int), stream));
    CN_CUDA(p, cudaMemsetAsync(p->slotU, 0, sizeof(cplx) * (size_t)P, stream));

    cn_geom g{N, P};
    const int T = 128;
    if (!p->ooc) {
        // blocks of 8 * 2^k <= 256 rows (the shapes of the tiled path): chunk-parallel pivots by the Moebius-map scan
        int logc = -1;
        if (m >= 8 && m <= 256 && (m & (m - 1)) == 0 && (N / 8) % 32 == 0) {
            logc = 0;
            while ((8LL << logc) < m) ++logc;
        }
        const int64_t nch = N / 8;
        const unsigned gridc = (unsigned)((nch + 127) / 128);
        // (a driven step does not store gamma: the tiled pass recovers it from q and reads only gamJ; the factorization of
        // the static H at the end of cn_step_td and cn_factorize write it for the kernels that want it)
        double *const gamOut = (tdG && p->path == 2) ? nullptr : p->gam;
#define CN_FB(L) k_factor_blocks_chunked<L><<<gridc, 128, 0, stream>>>(nch, p->two_dx2, p->rho, Vsrc, tdG, tdF, p->q, gamOut, redSubD, redDiagD, redSupU, redDiagU, p->derr, above, cutMask, p->gamJ)
        switch (logc) {
        case 0: CN_FB(0); break;
        case 1: CN_FB(1); break;
        case 2: CN_FB(2); break;
        case 3: CN_FB(3); break;
        case 4: CN_FB(4); break;
        case 5: CN_FB(5); break;
        default:
            if (sharded || p->sysMode) return CN_EINVAL; // these need blocks of 8 * 2^k <= 256 rows, whole warps of chunks
            if (tdG) { // the thread-per-block kernel takes the potential of the step ready-made
                k_td_potential<<<(unsigned)((N + 255) / 256), 256, 0, stream>>>(N, Vsrc, tdG, tdF, p->tdV);
                Vsrc = p->tdV;
                p->launches += 1;
            }
            k_factor_blocks<<<(unsigned)((P + T - 1) / T), T, 0, stream>>>(g, p->two_dx2, p->rho, Vsrc, p->q, p->gam, redSubD,
                                                                          redDiagD, redSupU, redDiagU, p->derr, p->gamJ);
        }
#undef CN_FB
    } else {
        // stream V through the device once, part by part: only the corner entries of every block's inverse and
        // gamma on the joint lines stay (O(P)); q and gamma are recomputed per part in every pass of cn_step
        if ((st = ooc_setup(p, m)) != CN_OK) return st;
        for (int64_t i = 0; i < p->nparts; ++i) {
            const int b = (int)(i % cn_plan::NB);
            const int64_t r0 = i * p->partPts, n = (N - r0 < p->partPts) ? (N - r0) : p->partPts;
            CN_CUDA(p, cudaMemcpyAsync(p->bV[b], p->hV + r0, sizeof(double) * (size_t)n, cudaMemcpyHostToDevice, stream));
            const int64_t nb = n / m;
            k_factor_part<<<(unsigned)((nb + T - 1) / T), T, 0, stream>>>(nb, m, r0 / m, p->two_dx2, p->rho, p->bV[b], p->bQ[b],
                                                                         p->bV[b], redSubD, redDiagD, redSupU, redDiagU,
                                                                         p->derr);
            k_joint_gamma<<<(unsigned)((nb + T - 1) / T), T, 0, stream>>>(nb, m, r0 / m, p->bV[b], p->gamJ);
            p->launches += 2;
        }
    }
    k_rs_assemble0<<<(unsigned)((P + T - 1) / T), T, 0, stream>>>(P, N, p->rho, p->gam, p->gamJ, redSubD, redDiagD, redSupU,
                                                                 redDiagU, p->lv[0].sub, p->lv[0].diag, p->lv[0].sup, above,
                                                                 p->diagAcc, cutMask);
    p->launches += 2;
    if (p->qB && whole) { // one block per system: the factors of cn_batched_sweep and of the on-chip stepper
        k_factor_whole<<<1, 32, 0, stream>>>(N, p->rho, p->gam, p->qB, p->derr);
        p->launches += 1;
    }
    for (int i = 0; i + 1 < nlv; ++i) {
        cn_plan::rs_level &L = p->lv[i], &U = p->lv[i + 1];
        if (p->opt_rs_group == CN_RS_G)
            k_rs_factor_level_smem<<<(unsigned)((U.n + CN_RS_FL_WARPS - 1) / CN_RS_FL_WARPS), 32 * CN_RS_FL_WARPS, 0, stream>>>(
                L.n, L.sub, L.diag, L.sup, L.l, L.rp, L.u, U.sub, U.diag, tmpB, U.sup, p->derr, above);
        else
        k_rs_factor_level<<<(unsigned)((U.n + T - 1) / T), T, 0, stream>>>(L.n, (int64_t)p->opt_rs_group, L.sub, L.diag, L.sup, L.l, L.rp, L.u, tmpA,
                                                                         U.sub, U.diag, tmpB, U.sup, p->derr);
        k_rs_add<<<(unsigned)((U.n + T - 1) / T), T, 0, stream>>>(U.n, U.diag, tmpB, above ? p->diagAcc : nullptr);
        p->launches += 2;
    }
    if (!sharded) { // (a sharded plan's last level is factored from the gathered records, cn_shard_factorize_finish)
        cn_plan::rs_level &L = p->lv.back();
        k_rs_factor_top_scan<<<1, 32, 0, stream>>>(L.n, L.sub, L.diag, L.sup, p->lw, p->rq, p->uw, p->derr);
        p->launches += 1;
    }
    return CN_OK;
}

static cn_status td_scratch(cn_plan *p);

// ---- factorize ----------------------------------------------------------------------------------------
// the partition the kernels work with (see cn_factorize) and, for a sharded plan, the rows nt of its last RS level
static void choose_partition(const cn_plan *p, int64_t *Peff, int64_t *nt)
{
    const int64_t N = p->N;
    int64_t P = p->Pu;
    if (p->sysMode == 1) { // blocks of the largest 8 * 2^k <= 256 rows that divides a SYSTEM
        int64_t me = 8;
        while (me < 256 && p->sysN % (2 * me) == 0) me *= 2;
        P = N / me;
    } else if (p->opt_path != 1 && !p->opt_keep_p && N % 8 == 0) {
        const int64_t mu = (N % p->Pu == 0) ? N / p->Pu : 0;
        const bool fits = mu >= 8 && mu <= 256 && (mu & (mu - 1)) == 0;
        if (!fits) {
            int64_t me = 8;
            while (me < 256 && N % (2 * me) == 0) me *= 2;
            P = N / me;
        }
    }
    *Peff = P;
    if (nt) { // levels are added while the shard's system exceeds its share of what one CTA solves (8192 rows in all)
        int64_t topmax = 8 * CN_RS_TOP_THREADS / p->nshards;
        if (topmax > p->opt_rs_topmax) topmax = p->opt_rs_topmax;
        int64_t n = P;
        while (n > topmax && n > 1) n = (n + CN_RS_G - 1) / CN_RS_G;
        *nt = n;
    }
}

static cn_status factorize_impl(cn_plan *p, cudaStream_t stream, cplx *msend);

extern "C" cn_status cn_factorize(cn_plan *p, void *stream_)
{
    if (!p) return CN_EINVAL;
    if (p->nshards > 1) return CN_EINVAL; // a sharded plan is factored by cn_shard_factorize_local / _finish
    return factorize_impl(p, (cudaStream_t)stream_, nullptr);
}

// msend != NULL: sharded plan; everything but the last RS level, whose rows go to the matrix record msend (DEVICE)
static cn_status factorize_impl(cn_plan *p, cudaStream_t stream, cplx *msend)
{
    free_factors(p);
    const int64_t N = p->N;
    const bool sharded = p->nshards > 1;
    p->sysMode = 0;
    if (p->sysWant) {
        if (sharded || p->hV) return CN_EINVAL;
        // contiguous systems of 8 * 2^k rows made of a power-of-two number of blocks: the tiled kernels with cuts
        int64_t me = 8;
        while (me < 256 && p->sysN % (2 * me) == 0) me *= 2;
        const int64_t k = (p->sysN % me == 0) ? p->sysN / me : 0;
        const bool fast = p->sysWant == 1 && p->opt_path != 1 && k >= 1 && (k & (k - 1)) == 0 && (N / 8) % 32 == 0;
        if (p->opt_path == 2 && !fast) return CN_EINVAL;
        p->sysMode = fast ? 1 : 2;
    }
    if (p->sysMode == 2) { // any dense layout: per-system pivots by one thread per system (cn_batched.cuh)
        cn_status st;
        if ((st = dev_alloc(p, &p->q, (size_t)N)) != CN_OK) return st;
        if ((st = dev_alloc(p, &p->gam, (size_t)N)) != CN_OK) return st;
        if ((st = dev_alloc(p, &p->derr, 1)) != CN_OK) return st;
        CN_CUDA(p, cudaMemsetAsync(p->derr, 0, sizeof(int), stream));
        const int T = 64;
        k_batched_v_factor<<<(unsigned)((p->sysCount + T - 1) / T), T, 0, stream>>>(p->sysN, p->sysCount, p->sysEs, p->sysSs,
                                                                                   p->two_dx2, p->rho, p->dV, p->q, p->gam,
                                                                                   p->derr);
        p->launches += 1;
        int herr = 0;
        CN_CUDA(p, cudaMemcpyAsync(&herr, p->derr, sizeof(int), cudaMemcpyDeviceToHost, stream));
        CN_CUDA(p, cudaStreamSynchronize(stream));
        if (herr) return CN_EBREAKDOWN;
        p->P = p->sysCount;
        p->path = 1;
        p->factorized = true;
        return CN_OK;
    }
    // The partition the kernels work with.  psi does not depend on it (direct solver), and the tiled kernels want equal
    // blocks of 8 * 2^k rows: up to 256 rows a block lives inside one warp (shuffle scans only), 512..4096 rows span
    // several warps (shared-memory scans and CTA barriers: 189-235 us per C2 step against 158), more does not fit a
    // CTA tile, and any other shape (N % P != 0, m = 300, m = 768 ...) would fall to the generic thread-per-block
    // kernels (10-500 times slower at C2).  So unless the caller's blocks already have 8 * 2^k <= 256 rows, the auto
    // and the forced-tiled paths partition the system themselves into blocks of the largest 8 * 2^k <= 256 rows that
    // divides N -- the same method one level down.  CN_OPT_KEEP_P = 1 and the generic path
    // (CN_OPT_PATH = 1) take the caller's P literally.
    choose_partition(p, &p->P, sharded ? &p->nt : nullptr);
    const int64_t P = p->P;

    // choose the path
    const bool uniform = (N % P == 0);
    const int64_t m = uniform ? N / P : 0;
    bool tiled_ok = uniform && m >= 8 && (m % 8 == 0) && (((m / 8) & (m / 8 - 1)) == 0) && (m / 8 <= 512);
    int logc = 0;
    if (tiled_ok)
        while ((8LL << logc) < m) ++logc;
    int tpb = 0;
    if (tiled_ok) {
        const int cpb = 1 << logc;
        // small tiles since the pass stopped staging gamma (25 KB of shared memory per 64 threads): eight CTAs of two
        // warps per SM interleave their load and compute phases more finely than two of eight -- 144 against 153 us per
        // C2 step in a 100-step call (32 threads: the same; the two-pass step of cn_step_td prefers 128: 391 / 394 / 400 us)
        tpb = p->opt_tile_threads ? p->opt_tile_threads : 64;
        if (tpb < cpb) tpb = (cpb <= 64) ? 64 : ((cpb <= 128) ? 128 : (cpb <= 256 ? 256 : 512));
        if (p->opt_tile_threads && p->opt_tile_threads < cpb) tiled_ok = false;
    }
    if (p->opt_path == 2 && !tiled_ok) return CN_EINVAL;
    // sharded: the tiled kernels on blocks inside one warp, resident, warp-per-group RS levels chosen by the library
    if (p->sysMode == 1 && (!tiled_ok || logc > 5)) return CN_EINVAL; // cannot happen: choose_partition picked the blocks
    if (sharded && (!tiled_ok || p->opt_path == 1 || logc > 5 || (N / 8) % 32 != 0 || p->hV || p->opt_rs_levels != 0 ||
                    p->opt_rs_group != CN_RS_G || p->opt_rs_serial_top))
        return CN_EINVAL;
    p->path = (p->opt_path == 1 || !tiled_ok) ? 1 : 2;
    p->tpb = (p->path == 2) ? tpb : 0;
    p->logc = logc;

    cn_status st;
    p->ooc = (p->hV != nullptr); // V was moved to the host by cn_plan_set_device_budget: stream everything
    if (p->ooc && p->path != 2) return CN_EINVAL; // the streamed mode exists for the tiled kernels only
    if (!p->ooc) {
        if ((st = dev_alloc(p, &p->q, (size_t)N)) != CN_OK) return st;
        if ((st = dev_alloc(p, &p->gam, (size_t)N)) != CN_OK) return st;
    }
    // gamma on the joint lines: all the tiled pass reads of gamma (the rest it recovers from q); all there is out of core
    if (p->ooc || p->path == 2)
        if ((st = dev_alloc_g(p, &p->gamJ, (size_t)P, sharded)) != CN_OK) return st;
    if ((st = dev_alloc_g(p, &p->slotD, (size_t)P, sharded)) != CN_OK) return st;
    if ((st = dev_alloc_g(p, &p->slotU, (size_t)P, sharded)) != CN_OK) return st;
    if ((st = dev_alloc(p, &p->derr, 1)) != CN_OK) return st;
    if (p->path == 1)
        if ((st = dev_alloc(p, &p->work, (size_t)N)) != CN_OK) return st;
    if (N <= CN_BATCHED_NMAX && !p->ooc && !sharded && !p->sysMode)
        if ((st = dev_alloc(p, &p->qB, (size_t)N)) != CN_OK) return st;

    // RS levels: lv[0] has P rows; add levels of ceil(n / G) rows until the last one fits the single CTA
    {
        int64_t topmax = (p->opt_rs_levels < 0) ? INT64_MAX : p->opt_rs_topmax;
        if (sharded && topmax > 8 * CN_RS_TOP_THREADS / p->nshards) topmax = 8 * CN_RS_TOP_THREADS / p->nshards;
        int64_t n = P;
        for (;;) {
            cn_plan::rs_level L;
            L.n = n;
            p->lv.push_back(L);
            const int nl = (int)p->lv.size();
            const bool want_more = (p->opt_rs_levels > 0) ? (nl < p->opt_rs_levels) : (n > topmax);
            if (!want_more || n <= (sharded ? 1 : 2)) break;
            n = (n + p->opt_rs_group - 1) / p->opt_rs_group;
        }
        if (p->opt_rs_levels >= 0 && !p->opt_rs_serial_top && p->lv.back().n > 8 * CN_RS_TOP_THREADS) return CN_EINVAL;
    }
    const int nlv = (int)p->lv.size();
    for (int i = 0; i < nlv; ++i) {
        cn_plan::rs_level &L = p->lv[i];
        const size_t n = (size_t)L.n;
        if ((st = dev_alloc(p, &L.sub, n)) != CN_OK) return st;
        if ((st = dev_alloc(p, &L.diag, n)) != CN_OK) return st;
        if ((st = dev_alloc_g(p, &L.sup, n, sharded)) != CN_OK) return st;
        if (i < nlv - 1) {
            if ((st = dev_alloc(p, &L.l, n)) != CN_OK) return st;
            if ((st = dev_alloc(p, &L.rp, n)) != CN_OK) return st;
            if ((st = dev_alloc(p, &L.u, n)) != CN_OK) return st;
        }
        if (i == 0) {
            L.rD = p->slotD;
            L.rU = p->slotU;
        } else {
            if ((st = dev_alloc(p, &L.rD, n)) != CN_OK) return st;
            if ((st = dev_alloc_g(p, &L.rU, n, sharded)) != CN_OK) return st;
            if (!(sharded && i == nlv - 1)) // (a sharded plan's last level lives in topX[], see below)
                if ((st = dev_alloc(p, &L.X, n)) != CN_OK) return st;
            CN_CUDA(p, cudaMemsetAsync(L.rU, 0, sizeof(cplx) * n, stream)); // rU[last] stays 0
        }
    }
    // last level: its factors; for a sharded plan the whole last level of all shards (nshards * nt rows, replicated)
    const size_t ntop = sharded ? (size_t)p->nshards * (size_t)p->nt : (size_t)p->lv.back().n;
    if (sharded && p->lv.back().n != p->nt) return CN_EINVAL; // choose_partition and the loop above must agree
    if ((st = dev_alloc(p, &p->lw, ntop)) != CN_OK) return st;
    if ((st = dev_alloc(p, &p->rq, ntop)) != CN_OK) return st;
    if ((st = dev_alloc(p, &p->uw, ntop)) != CN_OK) return st;
    if (sharded) {
        for (int b = 0; b < 2; ++b) {
            if ((st = dev_alloc(p, &p->topX[b], ntop)) != CN_OK) return st;
            CN_CUDA(p, cudaMemsetAsync(p->topX[b], 0, sizeof(cplx) * ntop, stream));
        }
        if ((st = dev_alloc(p, &p->gsub, ntop)) != CN_OK || (st = dev_alloc(p, &p->gdiag, ntop)) != CN_OK ||
            (st = dev_alloc(p, &p->gsup, ntop)) != CN_OK || (st = dev_alloc(p, &p->diagAcc, 1)) != CN_OK)
            return st;
        CN_CUDA(p, cudaMemsetAsync(p->diagAcc, 0, sizeof(cplx), stream));
    }
    // support values on the joint lines, old and new (ping-pong).  Sharded: with one guard element in front (the row
    // above the shard); when level 0 is the last level they are this shard's window of topX[]
    const int64_t toff = (int64_t)p->shard * p->nt;
    for (int b = 0; b < 2; ++b) {
        if (sharded && nlv == 1) p->sup[b] = p->topX[b] + toff;
        else if ((st = dev_alloc_g(p, &p->sup[b], (size_t)P, sharded)) != CN_OK) return st;
    }

    // temporaries of the factorization (freed below)
    cplx *red = nullptr;
    CN_CUDA(p, cudaMalloc((void **)&red, sizeof(cplx) * CN_RED_COUNT(P)));
    if ((st = factor_compute(p, p->dV, red, m, stream)) != CN_OK) { cudaFree(red); return st; }
    if (sharded) {
        const cn_plan::rs_level &L = p->lv.back();
        k_shard_pack_matrix<<<(unsigned)((p->nt + 127) / 128), 128, 0, stream>>>(p->nt, L.sub, L.diag, L.sup, p->diagAcc,
                                                                             p->above ? 1 : 0, p->shard, msend);
        p->launches += 1;
    }
    int herr = 0;
    cudaError_t e = cudaMemcpyAsync(&herr, p->derr, sizeof(int), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    cudaFree(red);
    if (e != cudaSuccess) return cuda_fail(p, e);
    if (herr) return CN_EBREAKDOWN;

    if (p->path == 2 && !p->ooc) {
        if ((st = get_encoder(p)) != CN_OK) return st;
        const int box_rows = p->tpb < 256 ? p->tpb : 256;
        if ((st = make_map(p, &p->tmQ, p->q, 16, box_rows)) != CN_OK) return st;
        if ((st = make_map(p, &p->tmGam, p->gam, 8, box_rows)) != CN_OK) return st;
        for (int mode = 0; mode < 3; ++mode) {
            tiled_kernel_t k = tiled_kernel(p->tpb, p->logc, mode);
            if (!k) return CN_EINVAL;
            CN_CUDA(p, cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)tiled_smem(p->tpb)));
            CN_CUDA(p, cudaFuncSetAttribute((const void *)k, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        }
        // persistent grid: one CTA per resident slot (148 SMs x resident CTAs per SM), never more than tiles
        int dev = 0, sms = 0, per_sm = 0;
        CN_CUDA(p, cudaGetDevice(&dev));
        CN_CUDA(p, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CN_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)tiled_kernel(p->tpb, p->logc, 1),
                                                                 p->tpb, tiled_smem(p->tpb)));
        if (per_sm < 1) return CN_ECUDA;
        const int64_t tiles = (N / 8 + p->tpb - 1) / p->tpb;
        const int64_t slots = (int64_t)sms * per_sm;
        p->grid_tiled = (int)(tiles < slots ? tiles : slots);
    }
    {
        int dev = 0;
        CN_CUDA(p, cudaGetDevice(&dev));
        CN_CUDA(p, cudaDeviceGetAttribute(&p->sms, cudaDevAttrMultiProcessorCount, dev));
    }
    if (p->qB && N <= CN_ONCHIP_NMAX) { // the on-chip stepper's dynamic shared memory, once per plan (not per cn_step)
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k_onchip_steps<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)onchip_smem_bytes<32>()));
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k_onchip_steps<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)onchip_smem_bytes<64>()));
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k_onchip_steps<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)onchip_smem_bytes<128>()));
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k_onchip_steps<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)onchip_smem_bytes<256>()));
        CN_CUDA(p, cudaFuncSetAttribute((const void *)k_onchip_steps<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)onchip_smem_bytes<512>()));
    }
    if (sharded) { // the last level is still to come (cn_shard_factorize_finish)
        p->sh_local_done = true;
        return CN_OK;
    }
    p->factorized = true;
    return td_scratch(p);
}

// ---- profiling aid ---------------------------------------------------------------------------------------
static int prof_begin(cn_plan *p, int kind, cudaStream_t stream)
{
    if (!p->opt_profile) return -1;
    if (p->ev_used == p->ev_pool.size()) {
        if (p->ev_pool.size() >= 8192) return -1; // enough samples; later launches go unbracketed
        cn_plan::ev_pair e;
        if (cudaEventCreate(&e.a) != cudaSuccess || cudaEventCreate(&e.b) != cudaSuccess) return -1;
        p->ev_pool.push_back(e);
    }
    int i = (int)p->ev_used++;
    p->ev_pool[i].kind = kind;
    cudaEventRecord(p->ev_pool[i].a, stream);
    return i;
}
static void prof_end(cn_plan *p, int i, cudaStream_t stream)
{
    if (i >= 0) cudaEventRecord(p->ev_pool[i].b, stream);
}

extern "C" cn_status cn_plan_get_profile(cn_plan *p, double *out)
{
    if (!p || !out) return CN_EINVAL;
    out[0] = out[1] = out[2] = out[3] = 0.0;
    for (size_t i = 0; i < p->ev_used; ++i) {
        float ms = 0.f;
        CN_CUDA(p, cudaEventSynchronize(p->ev_pool[i].b));
        CN_CUDA(p, cudaEventElapsedTime(&ms, p->ev_pool[i].a, p->ev_pool[i].b));
        out[2 * p->ev_pool[i].kind] += ms;
        out[2 * p->ev_pool[i].kind + 1] += 1.0;
    }
    p->ev_used = 0;
    return CN_OK;
}

// ---- one pass + RS ------------------------------------------------------------------------------------
// every kernel of the per-step chain goes through here; pdl = programmatic stream serialization (cn_common.cuh)
template <typename... KArgs, typename... Args>
static cudaError_t launch_k(void (*k)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t stream,
                            bool pdl, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, k, args...);
}

// mode 0: prologue (P2 only), 1: fused (P1 + P2), 2: epilogue (P1 only)
static cn_status launch_pass(cn_plan *p, cplx *psi, int mode, int cur, cudaStream_t stream)
{
    const cplx *supOld = p->sup[cur ^ 1], *supNew = p->sup[cur];
    const int pi = (mode == 1) ? prof_begin(p, 0, stream) : -1;
    const bool pdl = p->opt_pdl && mode != 0 && !p->opt_profile;
    cudaError_t e;
    if (p->path == 2) {
        cn_tiled_params prm;
        prm.nchunks = p->N / 8;
        prm.chunk0 = 0;
        prm.P = p->P;
        prm.cutMask = (p->sysMode == 1) ? p->sysN / (p->N / p->P) - 1 : ~(int64_t)0;
        prm.rho = p->rho;
        prm.psi_raw = psi;
        prm.supOld = supOld;
        prm.supNew = supNew;
        prm.slotD = p->slotD;
        prm.slotU = p->slotU;
        prm.supInit = p->sup[0];
        prm.gamJ = p->gamJ;
        if (p->above) {
            // a shard with a predecessor: its blocks are numbered from 1, so that "the joint line above block w" is
            // index w - 1 >= 0 for every block -- for the first one the guard element in front of the arrays, which
            // holds what belongs to the last row of the preceding shard (the same mechanism as a streamed part)
            prm.chunk0 = (int64_t)1 << p->logc;
            prm.supOld -= 1; prm.supNew -= 1; prm.slotD -= 1; prm.slotU -= 1; prm.supInit -= 1; prm.gamJ -= 1;
            prm.P += 1;
        }
        if (p->nshards > 1) prm.P = 0; // no block of a shard clears slotU of "the last joint line": that slot belongs to the
                                       // next shard (or, on the last shard, stays at the 0 of the factorization)
        tiled_kernel_t k = tiled_kernel(p->tpb, p->logc, mode);
        e = launch_k(k, (unsigned)p->grid_tiled, (unsigned)p->tpb, tiled_smem(p->tpb), stream, pdl, p->tmPsi, p->tmQ,
                     p->tmGam, prm);
    } else {
        cn_geom g{p->N, p->P};
        const int T = 64;
        const unsigned grid = (unsigned)((p->P + T - 1) / T);
        auto k = (mode == 0) ? k_pass_generic<false, true> : (mode == 1 ? k_pass_generic<true, true> : k_pass_generic<true, false>);
        e = launch_k(k, grid, T, 0, stream, pdl, g, p->rho, psi, (const cplx *)p->q, (const double *)p->gam, p->work,
                     supOld, supNew, p->slotD, p->slotU, p->sup[0]);
    }
    prof_end(p, pi, stream);
    p->launches += 1;
    if (e != cudaSuccess) return cuda_fail(p, e);
    return CN_OK;
}

template <int K>
static cudaError_t launch_top_k(cn_plan *p, const cn_plan::rs_level &L, cplx *X, cudaStream_t stream, bool pdl)
{
    int T = CN_RS_TOP_THREADS;
    while (T > 32 && (int64_t)(T / 2) * K >= L.n) T /= 2;
    return launch_k(k_rs_top<K>, 1u, (unsigned)T, 0, stream, pdl, L.n, (const cplx *)L.rD, (const cplx *)L.rU,
                    (const cplx *)p->lw, (const cplx *)p->rq, (const cplx *)p->uw, X);
}

// RS of one step: (RD+RU+JD+JU) level by level, RS of the last level, SS level by level (Eq. 6)
// Sharded plans (cn_shard.cuh) run it in two halves around the exchange: phase 1 = the reductions and the record `rec`
// to send, phase 2 = the replicated last level from the gathered records `rec`, then the substitutions.
static cn_status launch_rs(cn_plan *p, int out, cudaStream_t stream, int phase = 0, cplx *rec = nullptr)
{
    const bool pdl = p->opt_pdl && !p->opt_profile;
    const int nlv = (int)p->lv.size();
    const int pi = prof_begin(p, 1, stream);
    cudaError_t e = cudaSuccess;
    const bool sharded = p->nshards > 1;
    const int above = p->above ? 1 : 0;
    const int64_t toff = (int64_t)p->shard * p->nt;
    p->lv[0].X = p->sup[out];
    if (sharded) p->lv.back().X = p->topX[out] + toff; // (nlv == 1: sup[out] is that window already)
    const cplx *Xabove = (sharded && above) ? p->topX[out] + toff - 1 : nullptr;
    const int nsep = nlv - 1; // group levels: one reduce and one substitute kernel each
    const bool tg = p->opt_rs_group != CN_RS_G; // one thread per group of any size (paper-shaped, cn_reduced.cuh)
    // the last level is solved inside the substitution kernel of the level below it (one launch less per step)
    const bool tis = !tg && !sharded && p->opt_rs_top_in_subst && p->opt_rs_levels >= 0 && !p->opt_rs_serial_top &&
                     nlv >= 2 && p->lv.back().n <= p->opt_rs_top_in_subst_max;
    const int64_t G = p->opt_rs_group;
    for (int i = 0; i < nsep && e == cudaSuccess && phase != 2; ++i) {
        const cn_plan::rs_level &L = p->lv[i], &U = p->lv[i + 1];
        const int64_t *off = (i == 0) ? p->off0 : nullptr; // caller-placed joint lines: ragged blocks of at most 256 rows
        if (tg)
            e = launch_k(k_rs_reduce_thread, (unsigned)((U.n + 63) / 64), 64u, 0, stream, pdl, L.n, G, (const cplx *)L.rD,
                         (const cplx *)L.rU, (const cplx *)L.l, (const cplx *)L.rp, (const cplx *)L.u, (const cplx *)L.sub,
                         (const cplx *)L.sup, L.X, U.rD, U.rU);
        else
        e = launch_k(k_rs_reduce, (unsigned)((U.n + CN_RS_WARPS - 1) / CN_RS_WARPS), 32u * CN_RS_WARPS, 0, stream, pdl, L.n, (const cplx *)L.rD,
                     (const cplx *)L.rU, (const cplx *)L.l, (const cplx *)L.rp, (const cplx *)L.u, (const cplx *)L.sub,
                     (const cplx *)L.sup, U.rD, U.rU, above, off, p->noff0);
        p->launches += 1;
    }
    // (sharded, phase 1: the last level's right-hand-side slots ARE the record to send, shard_bind_record; nothing to pack)
    if (phase == 1) {
        prof_end(p, pi, stream);
        return e == cudaSuccess ? CN_OK : cuda_fail(p, e);
    }
    // sharded: RS of the whole last level (nshards * nt rows), replicated, from the gathered records `rec`; inside the
    // substitution kernel of the level below when it is small enough, else by k_shard_top.  Whichever kernel comes first
    // is launched WITHOUT programmatic serialization: the work before it on the stream is the caller's exchange.
    const int64_t ntopS = (int64_t)p->nshards * p->nt;
    const bool stis = sharded && nlv >= 2 && p->opt_rs_top_in_subst && ntopS <= 1024;
    if (sharded && !stis && e == cudaSuccess) {
        const int64_t n = ntopS;
        cplx *guard0 = (above && nlv >= 2) ? p->sup[out] - 1 : nullptr;
        int T = CN_RS_TOP_THREADS;
#define CN_STOP(K)                                                                                                     \
    {                                                                                                                  \
        while (T > 32 && (int64_t)(T / 2) * K >= n) T /= 2;                                                            \
        e = launch_k(k_shard_top<K>, 1u, (unsigned)T, 0, stream, false, (int64_t)p->nshards, p->nt, (const cplx *)rec, \
                     (const cplx *)p->lw, (const cplx *)p->rq, (const cplx *)p->uw, p->topX[out], toff, guard0);       \
    }
        if (n <= CN_RS_TOP_THREADS) CN_STOP(1)
        else if (n <= 2 * CN_RS_TOP_THREADS) CN_STOP(2)
        else if (n <= 4 * CN_RS_TOP_THREADS) CN_STOP(4)
        else CN_STOP(8)
#undef CN_STOP
        p->launches += 1;
    }
    if (e == cudaSuccess && !tis && !sharded) {
        const cn_plan::rs_level &L = p->lv.back();
        if (p->opt_rs_levels < 0 || p->opt_rs_serial_top)
            e = launch_k(k_rs_serial, 1u, 32u, 0, stream, pdl, L.n, (const cplx *)L.rD, (const cplx *)L.rU,
                         (const cplx *)p->lw, (const cplx *)p->rq, (const cplx *)p->uw, L.X);
        else if (L.n <= CN_RS_TOP_THREADS) e = launch_top_k<1>(p, L, L.X, stream, pdl);
        else if (L.n <= 2 * CN_RS_TOP_THREADS) e = launch_top_k<2>(p, L, L.X, stream, pdl);
        else if (L.n <= 4 * CN_RS_TOP_THREADS) e = launch_top_k<4>(p, L, L.X, stream, pdl);
        else e = launch_top_k<8>(p, L, L.X, stream, pdl);
        p->launches += 1;
    }
    for (int i = nsep - 1; i >= 0 && e == cudaSuccess; --i) {
        const cn_plan::rs_level &L = p->lv[i], &U = p->lv[i + 1];
        const int64_t *off = (i == 0) ? p->off0 : nullptr;
        if (tg)
            e = launch_k(k_rs_subst_thread, (unsigned)((U.n + 63) / 64), 64u, 0, stream, pdl, L.n, G, (const cplx *)L.rD,
                         (const cplx *)L.rU, (const cplx *)L.l, (const cplx *)L.rp, (const cplx *)L.u, (const cplx *)U.X, L.X);
        else {
            const unsigned gr = (unsigned)((U.n + CN_RS_WARPS - 1) / CN_RS_WARPS);
            const int64_t T = 32 * CN_RS_WARPS;
            const bool top_here = (tis || stis) && i == nlv - 2;        // the last level is solved inside this launch
            const int64_t ntop = stis ? ntopS : U.n;
            const int kt = top_here ? (ntop <= T ? 1 : (ntop <= 2 * T ? 2 : (ntop <= 4 * T ? 4 : 8))) : 0;
            cplx *guardOut = (sharded && above && i == 0) ? p->sup[out] - 1 : nullptr; // level 0 leaves X of the row above
            const cplx *gath = (stis && top_here) ? (const cplx *)rec : nullptr;
            cplx *xaboveOut = (stis && top_here && above) ? p->topX[out] + toff - 1 : nullptr;
            const bool pdl_here = pdl && !(stis && top_here);         // (first kernel after the caller's exchange)
#define CN_SUBST(KT) launch_k(k_rs_subst<KT>, gr, 32u * CN_RS_WARPS, 0, stream, pdl_here, L.n, (const cplx *)L.rD, (const cplx *)L.rU, \
                              (const cplx *)L.l, (const cplx *)L.rp, (const cplx *)L.u, (const cplx *)U.X, L.X, ntop,                \
                              (const cplx *)U.rD, (const cplx *)U.rU, (const cplx *)p->lw, (const cplx *)p->rq, (const cplx *)p->uw, \
                              Xabove, off, p->noff0, guardOut, gath, (int64_t)p->nshards,          \
                              stis ? toff : (int64_t)0, xaboveOut)
            e = kt == 0 ? CN_SUBST(0) : (kt == 1 ? CN_SUBST(1) : (kt == 2 ? CN_SUBST(2) : (kt == 4 ? CN_SUBST(4) : CN_SUBST(8))));
#undef CN_SUBST
        }
        p->launches += 1;
    }
    prof_end(p, pi, stream);
    if (e != cudaSuccess) return cuda_fail(p, e);
    return CN_OK;
}

// one pass over all parts: mode 0 prologue (no copy out), 1 fused, 2 epilogue; `first` = psi on the host is the caller's
static cn_status ooc_pass(cn_plan *p, cplx *hpsi, int mode, int cur, bool first)
{
    const int64_t N = p->N, m = N / p->P;
    const int T = 128;
    tiled_kernel_t k = tiled_kernel(p->tpb, p->logc, mode);
    for (int64_t i = 0; i < p->nparts; ++i) {
        const int b = (int)(i % cn_plan::NB);
        const int64_t r0 = i * p->partPts, n = (N - r0 < p->partPts) ? (N - r0) : p->partPts;
        // copy in: the buffer must be free, and the part's new psi of the previous pass must have landed
        CN_CUDA(p, cudaStreamWaitEvent(p->sIn, p->evFree[b], 0));
        if (!first) CN_CUDA(p, cudaStreamWaitEvent(p->sIn, p->evHost[i], 0));
        CN_CUDA(p, cudaMemcpyAsync(p->bPsi[b], hpsi + r0, sizeof(cplx) * (size_t)n, cudaMemcpyHostToDevice, p->sIn));
        CN_CUDA(p, cudaMemcpyAsync(p->bV[b], p->hV + r0, sizeof(double) * (size_t)n, cudaMemcpyHostToDevice, p->sIn));
        CN_CUDA(p, cudaEventRecord(p->evIn[b], p->sIn));
        // compute: factors of the part (recomputed instead of stored), then the pass
        CN_CUDA(p, cudaStreamWaitEvent(p->sCmp, p->evIn[b], 0));
        const int64_t nb = n / m;
        k_factor_part<<<(unsigned)((nb + T - 1) / T), T, 0, p->sCmp>>>(nb, m, r0 / m, p->two_dx2, p->rho, p->bV[b], p->bQ[b],
                                                                      p->bV[b], nullptr, nullptr, nullptr, nullptr, p->derr);
        cn_tiled_params prm;
        prm.nchunks = n / 8;
        prm.chunk0 = r0 / 8;
        prm.P = p->P;
        prm.cutMask = ~(int64_t)0;
        prm.rho = p->rho;
        prm.psi_raw = p->bPsi[b];
        prm.supOld = p->sup[cur ^ 1];
        prm.supNew = p->sup[cur];
        prm.slotD = p->slotD;
        prm.slotU = p->slotU;
        prm.supInit = p->sup[0];
        prm.gamJ = p->gamJ;
        const int64_t tiles = (n / 8 + p->tpb - 1) / p->tpb;
        const unsigned grid = (unsigned)(tiles < p->grid_tiled ? tiles : p->grid_tiled);
        cudaError_t e = launch_k(k, grid, (unsigned)p->tpb, tiled_smem(p->tpb), p->sCmp, false, p->tmPsiB[b], p->tmQB[b],
                                 p->tmGamB[b], prm);
        p->launches += 2;
        if (e != cudaSuccess) return cuda_fail(p, e);
        CN_CUDA(p, cudaEventRecord(p->evCmp[b], p->sCmp));
        if (mode != 0) {
            CN_CUDA(p, cudaStreamWaitEvent(p->sOut, p->evCmp[b], 0));
            CN_CUDA(p, cudaMemcpyAsync(hpsi + r0, p->bPsi[b], sizeof(cplx) * (size_t)n, cudaMemcpyDeviceToHost, p->sOut));
            CN_CUDA(p, cudaEventRecord(p->evFree[b], p->sOut));
            CN_CUDA(p, cudaEventRecord(p->evHost[i], p->sOut));
        } else {
            CN_CUDA(p, cudaEventRecord(p->evFree[b], p->sCmp));
        }
    }
    return CN_OK;
}

static cn_status ooc_step(cn_plan *p, cplx *hpsi, int64_t nsteps, cudaStream_t stream)
{
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, hpsi) != cudaSuccess || pa.type != cudaMemoryTypeHost) {
        (void)cudaGetLastError();
        return CN_EINVAL; // out-of-core mode streams psi from PINNED host memory
    }
    cn_status st;
    CN_CUDA(p, cudaEventRecord(p->evFork, stream));
    CN_CUDA(p, cudaStreamWaitEvent(p->sIn, p->evFork, 0));
    CN_CUDA(p, cudaStreamWaitEvent(p->sCmp, p->evFork, 0));
    CN_CUDA(p, cudaStreamWaitEvent(p->sOut, p->evFork, 0));
    if ((st = ooc_pass(p, hpsi, 0, /*cur=*/1, true)) != CN_OK) return st;
    if ((st = launch_rs(p, 1, p->sCmp)) != CN_OK) return st;
    int cur = 1;
    for (int64_t k = 1; k < nsteps; ++k) {
        if ((st = ooc_pass(p, hpsi, 1, cur, k == 1)) != CN_OK) return st;
        if ((st = launch_rs(p, cur ^ 1, p->sCmp)) != CN_OK) return st;
        cur ^= 1;
    }
    if ((st = ooc_pass(p, hpsi, 2, cur, nsteps == 1)) != CN_OK) return st;
    cudaStream_t ss[3] = {p->sIn, p->sCmp, p->sOut};
    for (int i = 0; i < 3; ++i) {
        CN_CUDA(p, cudaEventRecord(p->evJoin[i], ss[i]));
        CN_CUDA(p, cudaStreamWaitEvent(stream, p->evJoin[i], 0));
    }
    return CN_OK;
}

extern "C" cn_status cn_step(cn_plan *p, void *psi_, int64_t nsteps, void *stream_)
{
    if (!p || !psi_ || nsteps < 0) return CN_EINVAL;
    if (((uintptr_t)psi_ & 15) != 0) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    if (nsteps == 0) return CN_OK;
    cudaStream_t stream = (cudaStream_t)stream_;
    cplx *psi = (cplx *)psi_;
    cn_status st;
    if (p->nshards > 1) return CN_EINVAL; // a sharded plan is stepped by cn_shard_prologue / _advance / _epilogue
    if (p->ooc) return ooc_step(p, psi, nsteps, stream);
    if (p->sysMode == 2) {
        const int T = 32; // few systems: small CTAs spread the warps over the SMs
        for (int64_t k = 0; k < nsteps; ++k) {
            cudaError_t e = launch_k(k_batched_v_sweep, (unsigned)((p->sysCount + T - 1) / T), (unsigned)T, 0, stream, false,
                                     p->sysN, p->sysCount, p->sysEs, p->sysSs, p->rho, psi, (const cplx *)p->q,
                                     (const double *)p->gam, p->sysEs, p->sysSs);
            p->launches += 1;
            if (e != cudaSuccess) return cuda_fail(p, e);
        }
        return CN_OK;
    }
    if (onchip_active(p)) {
        // one launch for the whole call: psi, q and gamma are read once, the steps loop on chip
        const int64_t chunks = (p->N + 7) / 8;
        const bool pdl = p->opt_pdl != 0;
        cudaError_t e;
#define CN_ONCHIP(T)                                                                                              \
    launch_k(k_onchip_steps<T>, 1u, (unsigned)T, onchip_smem_bytes<T>(), stream, pdl, p->N, nsteps, p->rho, psi, \
             (const cplx *)p->qB, (const double *)p->gam)
        if (chunks <= 32) e = CN_ONCHIP(32);
        else if (chunks <= 64) e = CN_ONCHIP(64);
        else if (chunks <= 128) e = CN_ONCHIP(128);
        else if (chunks <= 256) e = CN_ONCHIP(256);
        else e = CN_ONCHIP(512);
#undef CN_ONCHIP
        p->launches += 1;
        if (e != cudaSuccess) return cuda_fail(p, e);
        return CN_OK;
    }
    if (p->path == 2 && p->tmPsiFor != psi_) {
        const int box_rows = p->tpb < 256 ? p->tpb : 256;
        if ((st = make_map(p, &p->tmPsi, psi_, 16, box_rows)) != CN_OK) return st;
        p->tmPsiFor = psi_;
    }
    // prologue: RHS + RD/RU/JD/JU of step 1; also records psi^0 on the joint lines in sup[0]
    if ((st = launch_pass(p, psi, 0, /*cur=*/1, stream)) != CN_OK) return st;
    if ((st = launch_rs(p, 1, stream)) != CN_OK) return st;
    int cur = 1; // sup[cur] = new support values, sup[cur^1] = old psi on the joint lines
    for (int64_t k = 1; k < nsteps; ++k) {
        if ((st = launch_pass(p, psi, 1, cur, stream)) != CN_OK) return st;
        if ((st = launch_rs(p, cur ^ 1, stream)) != CN_OK) return st;
        cur ^= 1;
    }
    return launch_pass(p, psi, 2, cur, stream);
}

// ---- time-dependent Hamiltonian (the propagator uses H(t + dt/2)) ---------------------
// H(t) = H0 + f(t) g(x): V_j(t_k + dt/2) = V_j + f_k g_j, e.g. g = x and f = the laser field.  Every step
// has its own T, so the factorization is redone on the device inside the step loop -- launches only,
// no allocation, no synchronisation -- and a step is prologue (RHS + RD/RU/JD/JU) -> RS -> epilogue (SS) with the
// factors of that step.  SS(k) cannot be fused with RD/RU(k+1) here: the two use different matrices.

// scratch of the per-step factorization of cn_step_td, sized for the partition in use; called by whichever of
// cn_plan_set_td_shape / cn_factorize comes second, so that cn_step_td itself never allocates
static cn_status td_scratch(cn_plan *p)
{
    if (!p->tdG || !p->factorized || (p->tdRed && p->tdRedP == p->P)) return CN_OK;
    if (p->tdRed) cudaFree(p->tdRed);
    p->tdRed = nullptr;
    p->tdRedP = 0;
    CN_CUDA(p, cudaMalloc((void **)&p->tdRed, sizeof(cplx) * CN_RED_COUNT(p->P)));
    p->tdRedP = p->P;
    return CN_OK;
}

extern "C" cn_status cn_plan_set_td_shape(cn_plan *p, const double *g)
{
    if (!p || !g) return CN_EINVAL;
    if (!p->dV) return CN_EINVAL; // not for streamed (out-of-core) plans
    const size_t vb = sizeof(double) * (size_t)p->N;
    if (!p->tdG) {
        CN_CUDA(p, cudaMalloc((void **)&p->tdG, vb));
        CN_CUDA(p, cudaMalloc((void **)&p->tdV, vb));
    }
    CN_CUDA(p, cudaMemcpy(p->tdG, g, vb, cudaMemcpyDefault));
    return td_scratch(p);
}

extern "C" cn_status cn_step_td(cn_plan *p, void *psi_, int64_t nsteps, const double *field, void *stream_)
{
    if (!p || !psi_ || nsteps < 0 || (nsteps > 0 && !field)) return CN_EINVAL;
    if (((uintptr_t)psi_ & 15) != 0) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    if (p->ooc || !p->tdG || p->sysMode || p->nshards > 1) return CN_EINVAL;
    if (nsteps == 0) return CN_OK;
    for (int64_t k = 0; k < nsteps; ++k)
        if (!std::isfinite(field[k])) return CN_EINVAL; // nothing has been enqueued yet
    cudaStream_t stream = (cudaStream_t)stream_;
    cplx *psi = (cplx *)psi_;
    cn_status st;
    if (!p->tdRed || p->tdRedP != p->P) return CN_EINVAL; // td_scratch() ran at set_td_shape / factorize: cannot happen
    if (p->path == 2 && p->tmPsiFor != psi_) {
        const int box_rows = p->tpb < 256 ? p->tpb : 256;
        if ((st = make_map(p, &p->tmPsi, psi_, 16, box_rows)) != CN_OK) return st;
        p->tmPsiFor = psi_;
    }
    const int64_t m = (p->N % p->P == 0) ? p->N / p->P : 0;
    // a launch that fails mid-loop leaves the plan with the factors of that step: the plan is then marked
    // unfactorized, so that a later cn_step cannot silently use the wrong matrix
    auto run = [&]() -> cn_status {
        cn_status s;
        for (int64_t k = 0; k < nsteps; ++k) {
            if ((s = factor_compute(p, p->dV, p->tdRed, m, stream, false, p->tdG, field[k])) != CN_OK) return s;
            if ((s = launch_pass(p, psi, 0, /*cur=*/1, stream)) != CN_OK) return s;
            if ((s = launch_rs(p, 1, stream)) != CN_OK) return s;
            if ((s = launch_pass(p, psi, 2, /*cur=*/1, stream)) != CN_OK) return s;
        }
        // leave the plan with the factors of the static H again, so that cn_step keeps its meaning
        if ((s = factor_compute(p, p->dV, p->tdRed, m, stream, false)) != CN_OK) return s;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(p, e);
        return CN_OK;
    };
    st = run();
    if (st != CN_OK) p->factorized = false;
    return st;
}

// ---- general complex tridiagonal front end (Eq. 5) ---------------------------------------
// b_i x_{i-1} + a_i x_i + c_i x_{i+1} = d_i for ARBITRARY complex b, a, c (non-constant off-diagonals, any N), solved
// by the same N-shaped partition scheme: the system is handed to the nested-level machinery of cn_reduced.cuh as its
// level 0 (groups of 256 rows = the blocks of PAPER.md:90-94, the last row of a group = its joint line; reduce =
// RD+RU+JD+JU on the d-side, Eq. 6), so every kernel on this path is one the CN stepper already uses.
struct cn_tridiag {
    cn_plan *p = nullptr;
    cplx *zero = nullptr; // the second right-hand-side slot of level 0, always 0 here
};

extern "C" cn_status cn_tridiag_destroy(cn_tridiag *t)
{
    if (!t) return CN_EINVAL;
    if (t->p) {
        free_factors(t->p);
        delete t->p;
    }
    delete t;
    return CN_OK;
}

static cn_status tridiag_create_impl(cn_tridiag **out, int64_t N, const void *b, const void *a, const void *c,
                                     int64_t P, const int64_t *joints, void *stream_);

extern "C" cn_status cn_tridiag_create(cn_tridiag **out, int64_t N, const void *b, const void *a, const void *c,
                                       void *stream_)
{
    return tridiag_create_impl(out, N, b, a, c, 0, nullptr, stream_);
}

// caller-placed joint lines ("the blocks may differ in size"): block w = rows (joints[w-1], joints[w]],
// its last row joints[w] is its joint line; joints = P strictly increasing HOST values, joints[P-1] = N - 1
extern "C" cn_status cn_tridiag_create_blocks(cn_tridiag **out, int64_t N, const void *b, const void *a, const void *c,
                                              int64_t P, const int64_t *joints, void *stream_)
{
    if (!out) return CN_EINVAL;
    *out = nullptr;
    if (P < 1 || P > N || !joints) return CN_EINVAL;
    for (int64_t w = 0; w < P; ++w)
        if (joints[w] < 0 || joints[w] >= N || (w > 0 && joints[w] <= joints[w - 1])) return CN_EINVAL;
    if (joints[P - 1] != N - 1) return CN_EINVAL;
    return tridiag_create_impl(out, N, b, a, c, P, joints, stream_);
}

static cn_status tridiag_create_impl(cn_tridiag **out, int64_t N, const void *b, const void *a, const void *c,
                                     int64_t P, const int64_t *joints, void *stream_)
{
    if (!out) return CN_EINVAL;
    *out = nullptr;
    if (N < 1 || !b || !a || !c) return CN_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_;
    cn_tridiag *t = new (std::nothrow) cn_tridiag;
    cn_plan *p = new (std::nothrow) cn_plan;
    if (!t || !p) { delete t; delete p; return CN_ENOMEM; }
    t->p = p;
    p->N = N; p->P = N; p->Pu = N;
    p->path = 1;
    cn_status st = CN_OK;
    auto fail = [&](cn_status e) { cn_tridiag_destroy(t); return e; };
    {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&p->sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
            return fail(CN_ECUDA);
    }
    // Caller-placed joint lines: every one of them is a joint line of the first level.  A block of more than 256 rows is
    // partitioned again by the library (more joint lines inside it, every 256 rows from its first row: the same method
    // one level down; x does not depend on the partition), so that every block of the first level fits
    // the warp-per-group kernels.
    std::vector<int64_t> off;
    if (joints) {
        off.push_back(0);
        for (int64_t w = 0; w < P; ++w) {
            const int64_t end = joints[w] + 1;
            while (end - off.back() > CN_RS_G) off.push_back(off.back() + CN_RS_G);
            off.push_back(end);
        }
    }
    const int64_t P1 = joints ? (int64_t)off.size() - 1 : 0; // blocks of the first level
    // levels: n_0 = N, n_{i+1} = ceil(n_i / 256) while n_i > 4096; with caller-placed joint lines n_1 = P1
    for (int64_t n = N;;) {
        cn_plan::rs_level L;
        L.n = n;
        p->lv.push_back(L);
        const bool ragged0 = joints && p->lv.size() == 1;
        if (!ragged0 && (n <= p->opt_rs_topmax || n <= 2)) break;
        n = ragged0 ? P1 : (n + CN_RS_G - 1) / CN_RS_G;
    }
    if (joints) {
        if ((st = dev_alloc(p, &p->off0, (size_t)P1 + 1)) != CN_OK) { cn_tridiag_destroy(t); return st; }
        if (cudaMemcpy(p->off0, off.data(), sizeof(int64_t) * ((size_t)P1 + 1), cudaMemcpyHostToDevice) != cudaSuccess) {
            cn_tridiag_destroy(t);
            return CN_ECUDA;
        }
        p->noff0 = P1;
    }
    const int nlv = (int)p->lv.size();
    for (int i = 0; i < nlv; ++i) {
        cn_plan::rs_level &L = p->lv[i];
        const size_t n = (size_t)L.n;
        if ((st = dev_alloc(p, &L.sub, n)) != CN_OK || (st = dev_alloc(p, &L.diag, n)) != CN_OK ||
            (st = dev_alloc(p, &L.sup, n)) != CN_OK)
            return fail(st);
        if (i < nlv - 1)
            if ((st = dev_alloc(p, &L.l, n)) != CN_OK || (st = dev_alloc(p, &L.rp, n)) != CN_OK ||
                (st = dev_alloc(p, &L.u, n)) != CN_OK)
                return fail(st);
        if (i > 0) {
            if ((st = dev_alloc(p, &L.rD, n)) != CN_OK || (st = dev_alloc(p, &L.rU, n)) != CN_OK ||
                (st = dev_alloc(p, &L.X, n)) != CN_OK)
                return fail(st);
            if (cudaMemsetAsync(L.rU, 0, sizeof(cplx) * n, stream) != cudaSuccess) return fail(CN_ECUDA);
        }
    }
    const size_t ntop = (size_t)p->lv.back().n;
    cplx *tmpB = nullptr;
    const size_t n1 = joints ? (size_t)P1 : (size_t)((N + CN_RS_G - 1) / CN_RS_G);
    if ((st = dev_alloc(p, &p->lw, ntop)) != CN_OK || (st = dev_alloc(p, &p->rq, ntop)) != CN_OK ||
        (st = dev_alloc(p, &p->uw, ntop)) != CN_OK || (st = dev_alloc(p, &p->derr, 1)) != CN_OK ||
        (st = dev_alloc(p, &t->zero, (size_t)N)) != CN_OK || (st = dev_alloc(p, &tmpB, n1)) != CN_OK)
        return fail(st);
    cn_plan::rs_level &L0 = p->lv[0];
    const size_t nb = sizeof(cplx) * (size_t)N;
    if (cudaMemsetAsync(t->zero, 0, nb, stream) != cudaSuccess || cudaMemsetAsync(p->derr, 0, sizeof(int), stream) != cudaSuccess ||
        cudaMemcpyAsync(L0.sub, b, nb, cudaMemcpyDefault, stream) != cudaSuccess ||
        cudaMemcpyAsync(L0.diag, a, nb, cudaMemcpyDefault, stream) != cudaSuccess ||
        cudaMemcpyAsync(L0.sup, c, nb, cudaMemcpyDefault, stream) != cudaSuccess ||
        cudaMemsetAsync(L0.sub, 0, sizeof(cplx), stream) != cudaSuccess ||               // b_1 = 0
        cudaMemsetAsync(L0.sup + (N - 1), 0, sizeof(cplx), stream) != cudaSuccess)       // c_N = 0
        return fail(CN_ECUDA);
    const int T = 128;
    for (int i = 0; i + 1 < nlv; ++i) {
        cn_plan::rs_level &L = p->lv[i], &U = p->lv[i + 1];
        k_rs_factor_level_smem<<<(unsigned)((U.n + CN_RS_FL_WARPS - 1) / CN_RS_FL_WARPS), 32 * CN_RS_FL_WARPS, 0, stream>>>(
            L.n, L.sub, L.diag, L.sup, L.l, L.rp, L.u, U.sub, U.diag, tmpB, U.sup, p->derr, 0, (i == 0) ? p->off0 : nullptr,
            (i == 0) ? p->noff0 : 0);
        k_rs_add<<<(unsigned)((U.n + T - 1) / T), T, 0, stream>>>(U.n, U.diag, tmpB, nullptr);
    }
    k_rs_factor_top_scan<<<1, 32, 0, stream>>>(p->lv.back().n, p->lv.back().sub, p->lv.back().diag, p->lv.back().sup, p->lw,
                                               p->rq, p->uw, p->derr);
    int herr = 0;
    if (cudaMemcpyAsync(&herr, p->derr, sizeof(int), cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
        cudaStreamSynchronize(stream) != cudaSuccess)
        return fail(CN_ECUDA);
    if (herr) return fail(CN_EBREAKDOWN);
    p->factorized = true;
    *out = t;
    return CN_OK;
}

extern "C" cn_status cn_tridiag_solve(cn_tridiag *t, const void *d, void *x, void *stream_)
{
    if (!t || !t->p || !d || !x) return CN_EINVAL;
    if ((((uintptr_t)d) & 15) != 0 || (((uintptr_t)x) & 15) != 0) return CN_EINVAL;
    cn_plan *p = t->p;
    cn_plan::rs_level &L0 = p->lv[0];
    L0.rD = (cplx *)d; // read only
    L0.rU = t->zero;
    p->sup[0] = (cplx *)x;
    return launch_rs(p, 0, (cudaStream_t)stream_);
}

// ---- batched sweep (config C4) --------------------------------------------------------------------------
typedef void (*bx_kernel_t)(const CUtensorMap, const cn_bx_params);
typedef void (*by_kernel_t)(const CUtensorMap, const cn_by_params);
#define CN_BY_COLS4_FROM_LOG2N 99 // auto: strips of 4 columns for systems of at least 2^this rows

static bx_kernel_t bx_kernel(int logc, int cl)
{
    if (cl == 1) {
        switch (logc) {
        case 3: return k_batched_x<3, 1>;
        case 4: return k_batched_x<4, 1>;
        case 5: return k_batched_x<5, 1>;
        case 6: return k_batched_x<6, 1>;
        case 7: return k_batched_x<7, 1>;
        case 8: return k_batched_x<8, 1>;
        }
        return nullptr;
    }
    if (logc != 8) return nullptr;
    if (cl == 2) return k_batched_x<8, 2>;
    if (cl == 4) return k_batched_x<8, 4>;
    if (cl == 8) return k_batched_x<8, 8>;
    return nullptr;
}

static by_kernel_t by_kernel(int logg, int cl, int nc, size_t *smem)
{
#define CN_BY(L, C, NC)                          \
    {                                            \
        *smem = batched_y_smem_bytes<L, NC>();   \
        return k_batched_y<L, C, NC>;            \
    }
    if (nc == 4) { // strips of 4 columns: up to 2048 rows per CTA
        if (cl == 1) {
            switch (logg) {
            case 3: CN_BY(3, 1, 4)
            case 4: CN_BY(4, 1, 4)
            case 5: CN_BY(5, 1, 4)
            case 6: CN_BY(6, 1, 4)
            case 7: CN_BY(7, 1, 4)
            }
            return nullptr;
        }
        if (logg != 7) return nullptr;
        if (cl == 2) CN_BY(7, 2, 4)
        if (cl == 4) CN_BY(7, 4, 4)
        return nullptr;
    }
    if (cl == 1) {
        switch (logg) {
        case 2: CN_BY(2, 1, 8)
        case 3: CN_BY(3, 1, 8)
        case 4: CN_BY(4, 1, 8)
        case 5: CN_BY(5, 1, 8)
        case 6: CN_BY(6, 1, 8)
        }
        return nullptr;
    }
    if (logg != 6) return nullptr;
    if (cl == 2) CN_BY(6, 2, 8)
    if (cl == 4) CN_BY(6, 4, 8)
    if (cl == 8) CN_BY(6, 8, 8)
#undef CN_BY
    return nullptr;
}

// launch with a cluster dimension (and programmatic stream serialization) on a persistent grid
template <typename K, typename... Args>
static cudaError_t launch_cluster(K k, unsigned grid, unsigned block, size_t smem, unsigned cl, cudaStream_t stream,
                                  bool pdl, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[2];
    int na = 0;
    if (cl > 1) {
        at[na].id = cudaLaunchAttributeClusterDimension;
        at[na].val.clusterDim.x = cl;
        at[na].val.clusterDim.y = 1;
        at[na].val.clusterDim.z = 1;
        ++na;
    }
    if (pdl) {
        at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, k, args...);
}

// persistent grid (in CTAs) of a kernel launched in clusters of `cl`
template <typename K>
static cn_status persistent_grid(cn_plan *p, K k, unsigned block, size_t smem, unsigned cl, int64_t work, int *grid)
{
    CN_CUDA(p, cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int64_t slots = 0;
    if (cl > 1) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(cl * 1024, 1, 1);
        cfg.blockDim = dim3(block, 1, 1);
        cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = cl;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        int ncl = 0;
        CN_CUDA(p, cudaOccupancyMaxActiveClusters(&ncl, (const void *)k, &cfg));
        slots = ncl;
    } else {
        int per_sm = 0;
        CN_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)k, (int)block, smem));
        slots = (int64_t)per_sm * p->sms;
    }
    if (slots < 1) return CN_ECUDA;
    const int64_t n = work < slots ? work : slots;
    *grid = (int)(n * cl);
    return CN_OK;
}

extern "C" cn_status cn_batched_sweep(cn_plan *p, void *psi_, int64_t nsys, int64_t es, int64_t ss, int64_t nsteps,
                                      void *stream_)
{
    if (!p || !psi_ || nsys < 1 || nsteps < 0 || es < 1 || ss < 1) return CN_EINVAL;
    if (((uintptr_t)psi_ & 15) != 0) return CN_EINVAL;
    const int64_t N = p->N;
    const bool xs = (es == 1 && (ss >= N || nsys == 1)), ys = (ss == 1 && es >= nsys && !xs);
    if (!xs && !ys) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    if (!p->qB) return CN_EINVAL; // N > CN_BATCHED_NMAX, or a streamed (out-of-core) plan
    if (nsteps == 0) return CN_OK;
    cudaStream_t stream = (cudaStream_t)stream_;
    cplx *psi = (cplx *)psi_;
    // no programmatic dependent launch here: CTAs of the next sweep that become resident early fragment the
    // cluster placement of a persistent grid (measured: x/y alternation 1.93 ms with, 1.44 ms without)
    const bool pdl = false;
    cn_status st;

    // shape of the fast kernels: N = 8 * 2^k (x) / 16 * 2^k (y), at most 8 CTAs of a cluster per system
    int lg = -1;
    if ((N & (N - 1)) == 0)
        for (lg = 0; (1LL << lg) < N; ++lg) {}
    int path = 0, logp = 0, cl = 1; // 0 generic, 1 x, 2 y
    // columns per strip of the y kernel: 4 from 2048 rows on (half the CTAs per cluster), else 8
    const int nc = (lg >= 7 && (p->opt_by_cols == 4 || (p->opt_by_cols == 0 && lg >= CN_BY_COLS4_FROM_LOG2N))) ? 4 : 8;
    if (p->opt_path != 1 && lg >= 6 && lg <= 14 && nsys < (1LL << 31) && ss < (1LL << 36) && es < (1LL << 36)) {
        if (xs && lg <= 14) {
            path = 1;
            logp = lg - 3;
            if (logp > 8) {
                cl = 1 << (logp - 8);
                logp = 8;
            }
        } else if (ys && lg <= 13 && nsys >= 8) {
            const int cap = (nc == 4) ? 7 : 6; // row groups of 16 rows per CTA: 512 threads
            path = 2;
            logp = lg - 4;
            if (logp > cap) {
                cl = 1 << (logp - cap);
                logp = cap;
            }
        }
    }
    const bool fresh = !(p->tmBatchFor == psi_ && p->tmBatchKey[0] == nsys && p->tmBatchKey[1] == es &&
                         p->tmBatchKey[2] == ss);
    cudaError_t e = cudaSuccess;
    if (path == 1) {
        bx_kernel_t k = bx_kernel(logp, cl);
        if (!k) return CN_EINVAL;
        const int cpb = 1 << logp, spt = CN_BX_TPB / cpb;
        if (fresh) {
            if ((st = get_encoder(p)) != CN_OK) return st;
            cuuint64_t dims[3] = {16, (cuuint64_t)(N / 8), (cuuint64_t)nsys};
            cuuint64_t strides[2] = {128, (cuuint64_t)ss * 16};
            cuuint32_t box[3] = {16, (cuuint32_t)cpb, (cuuint32_t)(cl > 1 ? 1 : spt)};
            cuuint32_t estr[3] = {1, 1, 1};
            if (nsys == 1) strides[1] = (cuuint64_t)N * 16;
            CUresult r = p->encode(&p->tmBatch, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, psi_, dims, strides, box, estr,
                                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return cuda_fail(p, cudaErrorInvalidValue);
            const int64_t ntiles = cl > 1 ? nsys : (nsys + spt - 1) / spt;
            if ((st = persistent_grid(p, k, CN_BX_TPB, batched_x_smem_bytes(), cl, ntiles, &p->batchGrid)) != CN_OK)
                return st;
        }
        cn_bx_params prm{nsys, ss, p->rho, psi, p->qB, p->gam};
        for (int64_t s = 0; s < nsteps && e == cudaSuccess; ++s) {
            e = launch_cluster(k, (unsigned)p->batchGrid, CN_BX_TPB, batched_x_smem_bytes(), (unsigned)cl, stream, pdl,
                               p->tmBatch, prm);
            p->launches += 1;
        }
    } else if (path == 2) {
        size_t smem = 0;
        by_kernel_t k = by_kernel(logp, cl, nc, &smem);
        if (!k) return CN_EINVAL;
        const int tpb = nc << logp, rc = 16 << logp;
        if (fresh) {
            if ((st = get_encoder(p)) != CN_OK) return st;
            cuuint64_t dims[2] = {(cuuint64_t)(2 * nsys), (cuuint64_t)N};
            cuuint64_t strides[1] = {(cuuint64_t)es * 16};
            cuuint32_t box[2] = {(cuuint32_t)(2 * nc), (cuuint32_t)(rc < 256 ? rc : 256)};
            cuuint32_t estr[2] = {1, 1};
            CUresult r = p->encode(&p->tmBatch, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, psi_, dims, strides, box, estr,
                                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return cuda_fail(p, cudaErrorInvalidValue);
            if ((st = persistent_grid(p, k, tpb, smem, cl, (nsys + nc - 1) / nc, &p->batchGrid)) != CN_OK) return st;
        }
        cn_by_params prm{nsys, es, p->rho, psi, p->qB, p->gam};
        for (int64_t s = 0; s < nsteps && e == cudaSuccess; ++s) {
            e = launch_cluster(k, (unsigned)p->batchGrid, (unsigned)tpb, smem, (unsigned)cl, stream, pdl, p->tmBatch, prm);
            p->launches += 1;
        }
    } else {
        const int T = 32;
        for (int64_t s = 0; s < nsteps && e == cudaSuccess; ++s) {
            e = launch_k(k_batched_v_sweep, (unsigned)((nsys + T - 1) / T), (unsigned)T, 0, stream, pdl, N, nsys, es, ss, p->rho,
                         psi, (const cplx *)p->qB, (const double *)p->gam, (int64_t)1, (int64_t)0);
            p->launches += 1;
        }
    }
    if (path != 0 && fresh) {
        p->tmBatchFor = psi_;
        p->tmBatchKey[0] = nsys;
        p->tmBatchKey[1] = es;
        p->tmBatchKey[2] = ss;
    }
    if (e != cudaSuccess) return cuda_fail(p, e);
    return CN_OK;
}

// ---- many systems with a potential of their own each ---------------------------------
extern "C" cn_status cn_plan_set_systems(cn_plan *p, int64_t nsys, int64_t elem_stride, int64_t sys_stride)
{
    if (!p || nsys < 1 || p->N % nsys != 0 || p->nshards > 1) return CN_EINVAL;
    const int64_t n = p->N / nsys;
    if (n < 2) return CN_EINVAL;
    const bool contiguous = elem_stride == 1 && (sys_stride == n || nsys == 1);
    const bool interleaved = sys_stride == 1 && elem_stride == nsys && !contiguous;
    if (!contiguous && !interleaved) return CN_EINVAL; // dense layouts only: V, psi and the factors share one indexing
    p->sysWant = contiguous ? 1 : 2;
    p->sysN = n;
    p->sysCount = nsys;
    p->sysEs = elem_stride;
    p->sysSs = contiguous ? n : 1;
    p->factorized = false;
    return CN_OK;
}

extern "C" cn_status cn_batched_sweep_v(cn_plan *p, void *psi, int64_t nsteps, void *stream)
{
    if (!p || !p->sysWant) return CN_EINVAL;
    return cn_step(p, psi, nsteps, stream);
}

// ---- sharded mode (kernels and record layout in cn_shard.cuh) ------
extern "C" cn_status cn_shard_plan_create(cn_plan **out, int64_t N_local, int64_t P_local, double dx, double dt,
                                          const double *V_local, int32_t shard, int32_t nshards)
{
    if (!out) return CN_EINVAL;
    *out = nullptr;
    if (nshards < 1 || nshards > 1024 || shard < 0 || shard >= nshards) return CN_EINVAL;
    if (N_local % 256 != 0 || N_local < 256) return CN_EINVAL; // whole warps of 8-row chunks (tiled kernels only)
    cn_status st = cn_plan_create(out, N_local, P_local, dx, dt, V_local);
    if (st != CN_OK) return st;
    cn_plan *p = *out;
    p->shard = shard;
    p->nshards = nshards;
    p->above = shard > 0;
    p->below = shard < nshards - 1;
    return CN_OK;
}

extern "C" cn_status cn_shard_counts(const cn_plan *p, int64_t *matrix_count, int64_t *step_count)
{
    if (!p || !matrix_count || !step_count) return CN_EINVAL;
    int64_t Peff = 0, nt = 0;
    choose_partition(p, &Peff, &nt);
    *matrix_count = CN_SHARD_MREC(nt);
    *step_count = 2 * nt;
    return CN_OK;
}

extern "C" cn_status cn_shard_factorize_local(cn_plan *p, void *matrix_send, void *stream_)
{
    if (!p || !matrix_send || (((uintptr_t)matrix_send) & 15) != 0) return CN_EINVAL;
    if (p->nshards == 1) { // one shard is the whole system: nothing to exchange, the record stays unused
        cn_status st = factorize_impl(p, (cudaStream_t)stream_, nullptr);
        if (st == CN_OK) p->sh_local_done = true;
        return st;
    }
    return factorize_impl(p, (cudaStream_t)stream_, (cplx *)matrix_send);
}

extern "C" cn_status cn_shard_factorize_finish(cn_plan *p, const void *matrix_all, void *stream_)
{
    if (!p || !p->sh_local_done) return CN_EINVAL;
    if (p->nshards == 1) return CN_OK;
    if (!matrix_all || (((uintptr_t)matrix_all) & 15) != 0) return CN_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_;
    const int64_t n = (int64_t)p->nshards * p->nt;
    CN_CUDA(p, cudaMemsetAsync(p->derr, 0, sizeof(int), stream));
    k_shard_assemble_top<<<(unsigned)((n + 127) / 128), 128, 0, stream>>>((int64_t)p->nshards, p->nt, (const cplx *)matrix_all,
                                                                         p->gsub, p->gdiag, p->gsup, p->derr);
    k_rs_factor_top_scan<<<1, 32, 0, stream>>>(n, p->gsub, p->gdiag, p->gsup, p->lw, p->rq, p->uw, p->derr);
    p->launches += 2;
    int herr = 0;
    CN_CUDA(p, cudaMemcpyAsync(&herr, p->derr, sizeof(int), cudaMemcpyDeviceToHost, stream));
    CN_CUDA(p, cudaStreamSynchronize(stream));
    if (herr >= 2) return CN_EINVAL; // records of shards with another shape, or not in rank order
    if (herr) return CN_EBREAKDOWN;
    p->factorized = true;
    return CN_OK;
}

extern "C" cn_status cn_shard_edge(cn_plan *p, const void *psi, void *edge_send, void *stream_)
{
    if (!p || !psi || !edge_send) return CN_EINVAL;
    CN_CUDA(p, cudaMemcpyAsync(edge_send, (const cplx *)psi + (p->N - 1), sizeof(cplx), cudaMemcpyDeviceToDevice,
                               (cudaStream_t)stream_));
    return CN_OK;
}

static cn_status shard_map_psi(cn_plan *p, void *psi_)
{
    if (p->tmPsiFor == psi_) return CN_OK;
    const int box_rows = p->tpb < 256 ? p->tpb : 256;
    cn_status st = make_map(p, &p->tmPsi, psi_, 16, box_rows);
    if (st == CN_OK) p->tmPsiFor = psi_;
    return st;
}

// The right-hand-side slots of the shard's last RS level live in the record to send (layout: shard_rhs, cn_shard.cuh)
static void shard_bind_record(cn_plan *p, cplx *rec)
{
    cn_plan::rs_level &T = p->lv.back();
    T.rD = rec;
    T.rU = rec + p->nt + 1; // rU[-1] = rec[nt]: the guard
    if (p->lv.size() == 1) { // level 0 is the last level: the pass kernel writes the record
        p->slotD = T.rD;
        p->slotU = T.rU;
    }
}

extern "C" cn_status cn_shard_prologue(cn_plan *p, void *psi_, const void *edges_all, void *step_send, void *stream_)
{
    if (!p || !psi_ || (((uintptr_t)psi_) & 15) != 0) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    cudaStream_t stream = (cudaStream_t)stream_;
    cn_status st;
    if (p->nshards == 1) { // degenerate: behaves like the first third of cn_step
        if ((st = shard_map_psi(p, psi_)) != CN_OK) return st;
        if ((st = launch_pass(p, (cplx *)psi_, 0, 1, stream)) != CN_OK) return st;
        p->sh_out = 1;
        return CN_OK;
    }
    if (!step_send || (p->above && !edges_all)) return CN_EINVAL;
    if ((st = shard_map_psi(p, psi_)) != CN_OK) return st;
    if (p->above) // psi^0 on the last row of the preceding shard: the old value of "the joint line above" for block 0
        CN_CUDA(p, cudaMemcpyAsync(p->sup[0] - 1, (const cplx *)edges_all + (p->shard - 1), sizeof(cplx),
                                   cudaMemcpyDeviceToDevice, stream));
    shard_bind_record(p, (cplx *)step_send);
    if ((st = launch_pass(p, (cplx *)psi_, 0, /*cur=*/1, stream)) != CN_OK) return st;
    p->sh_out = 1;
    return launch_rs(p, p->sh_out, stream, 1, (cplx *)step_send);
}

extern "C" cn_status cn_shard_advance(cn_plan *p, void *psi_, const void *step_all, void *step_send, void *stream_)
{
    if (!p || !psi_) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    cudaStream_t stream = (cudaStream_t)stream_;
    cn_status st;
    if (p->tmPsiFor != psi_) return CN_EINVAL; // cn_shard_prologue starts a run on this vector
    if (p->nshards == 1) {
        if ((st = launch_rs(p, p->sh_out, stream)) != CN_OK) return st;
        const int cur = p->sh_out;
        p->sh_out = cur ^ 1;
        return launch_pass(p, (cplx *)psi_, 1, cur, stream);
    }
    if (!step_all || !step_send) return CN_EINVAL;
    if ((st = launch_rs(p, p->sh_out, stream, 2, (cplx *)step_all)) != CN_OK) return st;
    const int cur = p->sh_out;
    shard_bind_record(p, (cplx *)step_send);
    if ((st = launch_pass(p, (cplx *)psi_, 1, cur, stream)) != CN_OK) return st;
    p->sh_out = cur ^ 1;
    return launch_rs(p, p->sh_out, stream, 1, (cplx *)step_send);
}

extern "C" cn_status cn_shard_epilogue(cn_plan *p, void *psi_, const void *step_all, void *stream_)
{
    if (!p || !psi_) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    cudaStream_t stream = (cudaStream_t)stream_;
    cn_status st;
    if (p->tmPsiFor != psi_) return CN_EINVAL;
    if (p->nshards == 1) {
        if ((st = launch_rs(p, p->sh_out, stream)) != CN_OK) return st;
    } else {
        if (!step_all) return CN_EINVAL;
        if ((st = launch_rs(p, p->sh_out, stream, 2, (cplx *)step_all)) != CN_OK) return st;
    }
    return launch_pass(p, (cplx *)psi_, 2, p->sh_out, stream);
}

// ---- the same protocol driven by the library, the exchange left to a callback (one shard per process / thread) ------------
// send / recv records are device buffers the plan owns (allocated once, here); the callback enqueues an all-gather of
// `count` complex128 values per shard, in rank order, on `stream` and returns CN_OK.
struct cn_shard_bufs {
    cplx *msend = nullptr, *mrecv = nullptr, *esend = nullptr, *erecv = nullptr, *ssend[2] = {nullptr, nullptr}, *srecv = nullptr;
};

static cn_status shard_buffers(cn_plan *p, cn_shard_bufs *b)
{
    int64_t mc = 0, sc = 0;
    cn_status st = cn_shard_counts(p, &mc, &sc);
    if (st != CN_OK) return st;
    const size_t S = (size_t)p->nshards;
    if (!p->xbuf) {
        const size_t total = (size_t)mc * (1 + S) + (1 + S) + (size_t)sc * (2 + S);
        CN_CUDA(p, cudaMalloc((void **)&p->xbuf, sizeof(cplx) * total));
        CN_CUDA(p, cudaMemset(p->xbuf, 0, sizeof(cplx) * total));
    }
    cplx *q = p->xbuf;
    b->msend = q; q += mc;
    b->mrecv = q; q += (size_t)mc * S;
    b->esend = q; q += 1;
    b->erecv = q; q += S;
    b->ssend[0] = q; q += sc;
    b->ssend[1] = q; q += sc;
    b->srecv = q;
    return CN_OK;
}

extern "C" cn_status cn_shard_factorize(cn_plan *p, cn_exchange_fn exchange, void *ctx, void *stream)
{
    if (!p || (p->nshards > 1 && !exchange)) return CN_EINVAL;
    if (p->xbuf) { cudaFree(p->xbuf); p->xbuf = nullptr; } // options may have changed the record sizes
    cn_shard_bufs b;
    cn_status st = shard_buffers(p, &b);
    if (st != CN_OK) return st;
    int64_t mc = 0, sc = 0;
    cn_shard_counts(p, &mc, &sc);
    if ((st = cn_shard_factorize_local(p, b.msend, stream)) != CN_OK) return st;
    if (p->nshards > 1 && (st = exchange(ctx, b.msend, b.mrecv, mc, stream)) != CN_OK) return st;
    return cn_shard_factorize_finish(p, b.mrecv, stream);
}

extern "C" cn_status cn_shard_run(cn_plan *p, void *psi, int64_t nsteps, cn_exchange_fn exchange, void *ctx, void *stream)
{
    if (!p || !psi || nsteps < 0 || (p->nshards > 1 && !exchange)) return CN_EINVAL;
    if (!p->factorized) return CN_ENOTFACTORIZED;
    if (nsteps == 0) return CN_OK;
    cn_shard_bufs b;
    cn_status st = shard_buffers(p, &b);
    if (st != CN_OK) return st;
    int64_t mc = 0, sc = 0;
    cn_shard_counts(p, &mc, &sc);
    const bool many = p->nshards > 1;
    if (many) {
        if ((st = cn_shard_edge(p, psi, b.esend, stream)) != CN_OK) return st;
        if ((st = exchange(ctx, b.esend, b.erecv, 1, stream)) != CN_OK) return st;
    }
    if ((st = cn_shard_prologue(p, psi, b.erecv, b.ssend[0], stream)) != CN_OK) return st;
    for (int64_t k = 1; k <= nsteps; ++k) {
        if (many && (st = exchange(ctx, b.ssend[(k - 1) & 1], b.srecv, sc, stream)) != CN_OK) return st;
        st = (k < nsteps) ? cn_shard_advance(p, psi, b.srecv, b.ssend[k & 1], stream) : cn_shard_epilogue(p, psi, b.srecv, stream);
        if (st != CN_OK) return st;
    }
    return CN_OK;
}

// ---- cn_step_static: a stepper that allocates NOTHING ------------------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it): no plan, no cudaMalloc / cudaFree / allocating library routine on this path.  What a plan keeps in device
// memory it allocated -- gamma and the inverse pivots of the whole-system downward elimination,
// the scratch of the on-chip stepper of cn_onchip.cuh -- lives in ONE file-scope device array of fixed size
// (CN_STATIC_NMAX rows: 96 KB + a flag; every GPU that loads the library holds it until the process exits).
//   * every call shares the array: it keeps the last call's contents, so every call rewrites all it reads (gamma and
//     pivots of ITS N rows) and clears the breakdown flag first; two calls that overlap on the GPU (different streams,
//     different host threads) RACE on it -- the caller serialises them;
//   * in host code `cn_static_scratch` is a host-side stand-in, not a device address: the kernels get the address
//     cudaGetSymbolAddress returns, fetched once per device with that device current (static_setup).
#define CN_STATIC_BYTES ((size_t)CN_STATIC_NMAX * (sizeof(cplx) + sizeof(double)) + 256)
static __device__ __align__(256) unsigned char cn_static_scratch[CN_STATIC_BYTES];
static_assert(CN_STATIC_NMAX <= CN_ONCHIP_NMAX, "cn_step_static runs on the on-chip stepper");

// layout of the scratch: [qB: NMAX complex][gamma: NMAX double][flag: int, padded]
struct cn_static_view {
    cplx *qB;
    double *gam;
    int *flag;
};
static cn_static_view static_view(unsigned char *base)
{
    cn_static_view v;
    v.qB = (cplx *)base;
    v.gam = (double *)(base + (size_t)CN_STATIC_NMAX * sizeof(cplx));
    v.flag = (int *)(base + (size_t)CN_STATIC_NMAX * (sizeof(cplx) + sizeof(double)));
    return v;
}

// Variant of k_factor_whole (cn_batched.cuh) that owns no plan memory: gamma_i = 2 + 2 dx^2 V_i and the inverse pivots
// p_0 = mu_0, p_i = mu_i - q_{i-1}, q_i = 1 / p_i of the whole system, both into the static scratch.  Same arithmetic,
// same order as cn_factorize for an on-chip plan, so psi agrees with cn_step to the last bit.  flag := 0 / 1 (breakdown).
__global__ void k_static_factor(int64_t N, double two_dx2, double rho, const double *__restrict__ V,
                                cplx *__restrict__ qB, double *__restrict__ gam, int *__restrict__ flag)
{
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) gam[i] = fma(two_dx2, V[i], 2.0);
    __syncthreads();
    if (threadIdx.x != 0) return;
    cplx qprev = cmake(0.0, 0.0);
    bool bad = false;
    for (int64_t i = 0; i < N; ++i) {
        cplx p = cmake(-gam[i] - qprev.x, rho - qprev.y);
        if (!cfinite_nonzero(p)) bad = true;
        qprev = crecip(p);
        qB[i] = qprev;
    }
    *flag = bad ? 1 : 0; // cleared on every call: the array keeps the last call's contents
}

// the asynchronous call cannot return CN_EBREAKDOWN: a zero or non-finite pivot (non-finite V) turns psi into NaN
__global__ void k_static_poison(int64_t N, cplx *__restrict__ psi, const int *__restrict__ flag)
{
    if (*flag == 0) return;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
        psi[i] = cmake(nan, nan);
}

// set-up, once per device, with that device current: the DEVICE address of the scratch and the shared-memory opt-in of
// the on-chip kernels (neither allocates).  A table indexed by the device ordinal; a spin lock of plain atomics keeps
// concurrent first calls from several host threads apart (no allocating C++ runtime object on this path).
#define CN_STATIC_MAXDEV 64
static unsigned char *g_static_ptr[CN_STATIC_MAXDEV];
static int g_static_ready[CN_STATIC_MAXDEV];
static int g_static_lock;

// there is no plan to keep the CUDA error in: it is cleared and reported as CN_ECUDA
static cn_status static_fail(cudaError_t)
{
    (void)cudaGetLastError();
    return CN_ECUDA;
}

static cn_status static_setup(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(e);
    if (dev < 0 || dev >= CN_STATIC_MAXDEV) return CN_EINVAL;
    if (!__atomic_load_n(&g_static_ready[dev], __ATOMIC_ACQUIRE)) {
        while (__atomic_exchange_n(&g_static_lock, 1, __ATOMIC_ACQUIRE)) {}
        cn_status st = CN_OK;
        if (!g_static_ready[dev]) {
            void *ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, cn_static_scratch);
            if (e == cudaSuccess && (!ptr || ((uintptr_t)ptr & 255u) != 0)) e = cudaErrorInvalidSymbol;
#define CN_STATIC_ATTR(T)                                                                                     \
    if (e == cudaSuccess)                                                                                     \
        e = cudaFuncSetAttribute((const void *)k_onchip_steps<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                 (int)onchip_smem_bytes<T>());
            CN_STATIC_ATTR(32)
            CN_STATIC_ATTR(64)
            CN_STATIC_ATTR(128)
            CN_STATIC_ATTR(256)
            CN_STATIC_ATTR(512)
#undef CN_STATIC_ATTR
            if (e == cudaSuccess) {
                g_static_ptr[dev] = (unsigned char *)ptr;
                __atomic_store_n(&g_static_ready[dev], 1, __ATOMIC_RELEASE);
            } else {
                st = static_fail(e);
            }
        }
        __atomic_store_n(&g_static_lock, 0, __ATOMIC_RELEASE);
        if (st != CN_OK) return st;
    }
    *out = g_static_ptr[dev];
    return CN_OK;
}

extern "C" cn_status cn_step_static(int64_t N, double dx, double dt, const double *V, void *psi_, int64_t nsteps,
                                    void *stream_)
{
    if (N > CN_STATIC_NMAX) return CN_ETOOLARGE; // beyond the static scratch: use a plan (cn_plan_create / cn_step)
    if (!V || !psi_ || N < 2 || nsteps < 0) return CN_EINVAL;
    if (!std::isfinite(dx) || !std::isfinite(dt) || dx <= 0.0 || dt == 0.0) return CN_EINVAL;
    if (((uintptr_t)psi_ & 15u) != 0 || ((uintptr_t)V & 7u) != 0) return CN_EINVAL;
    if (nsteps == 0) return CN_OK;
    unsigned char *base = nullptr;
    cn_status st = static_setup(&base);
    if (st != CN_OK) return st;
    const cn_static_view sv = static_view(base);
    cudaStream_t stream = (cudaStream_t)stream_;
    cplx *psi = (cplx *)psi_;
    const double rho = 4.0 * dx * dx / dt, two_dx2 = 2.0 * dx * dx; // as cn_plan_create
    cudaError_t e = launch_k(k_static_factor, 1u, 256u, 0, stream, false, N, two_dx2, rho, V, sv.qB, sv.gam, sv.flag);
    if (e != cudaSuccess) return static_fail(e);
    const int64_t chunks = (N + 7) / 8;
#define CN_ONCHIP(T)                                                                                 \
    launch_k(k_onchip_steps<T>, 1u, (unsigned)T, onchip_smem_bytes<T>(), stream, false, N, nsteps, rho, psi, \
             (const cplx *)sv.qB, (const double *)sv.gam)
    if (chunks <= 32) e = CN_ONCHIP(32);
    else if (chunks <= 64) e = CN_ONCHIP(64);
    else if (chunks <= 128) e = CN_ONCHIP(128);
    else if (chunks <= 256) e = CN_ONCHIP(256);
    else e = CN_ONCHIP(512);
#undef CN_ONCHIP
    if (e != cudaSuccess) return static_fail(e);
    e = launch_k(k_static_poison, 4u, 256u, 0, stream, false, N, psi, (const int *)sv.flag);
    if (e != cudaSuccess) return static_fail(e);
    return CN_OK;
}
