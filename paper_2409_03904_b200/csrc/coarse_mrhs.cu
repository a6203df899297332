// C ABI of the B200-native coarse multi-RHS operator and block CG (include/coarse_mrhs.h).
// Host-side orchestration only: argument checks, kernel selection, launches.  All arithmetic of the
// path runs in the CUDA kernels of this directory.  No CPU fallback exists.
#include <chrono>
#include <cstdarg>
#include <cstring>
#include <atomic>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>
#include <cmath>

#include "blockcg_kernels.cuh"
#include "common.cuh"
#include "setup_kernels.cuh"
#include "stencil_generic.cuh"
#include "stencil_simt.cuh"
#include "stencil_tc.cuh"
#include "stencil_dmma.cuh"
#include "stencil_h16.cuh"
#include "stencil_h16x.cuh"
#include "peaks.cuh"
#include "blockla_tc.cuh"

namespace cmrhs {

thread_local char g_err[512] = "";
static std::atomic<int64_t> g_launches{0};

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

cudaError_t ensure_dyn_smem(const void *func, size_t bytes)
{
    if (bytes <= 16 * 1024) return cudaSuccess;                 // far below the default limit even with the kernel's static part
    struct Seen { size_t static_bytes = 0, have = 0; bool known = false; };
    static std::mutex mu;
    static std::map<std::pair<int, const void *>, Seen> seen;    // (device, kernel) -> static bytes, dynamic bytes already granted
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    Seen &k = seen[{dev, func}];
    if (!k.known) {
        cudaFuncAttributes fa;
        e = cudaFuncGetAttributes(&fa, func);
        if (e != cudaSuccess) return e;
        k.static_bytes = fa.sharedSizeBytes;
        k.known = true;
    }
    // without opt-in, static + dynamic shared memory together must fit the default 48 KB
    if (k.have >= bytes || (k.have == 0 && k.static_bytes + bytes <= 48 * 1024)) return cudaSuccess;
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) k.have = bytes;
    return e;
}

// ---- tiled SIMT variants: (dtype, nbasis, nrhs) -> kernel ---------------------------------------------
//                      T      NB TM TN GC KSPLIT STAGES WARPS
using V_f32_s64 = SimtConfig<float, 32, 8, 8, 8, 4, 4, 8>;
using V_f32_s32 = SimtConfig<float, 32, 8, 4, 8, 4, 4, 12>;
using V_f32_s16 = SimtConfig<float, 32, 4, 4, 4, 4, 4, 16>;
using V_f32_s8 = SimtConfig<float, 32, 4, 2, 4, 4, 5, 16>;
using V_f32_s4 = SimtConfig<float, 32, 4, 1, 4, 4, 5, 16>;
using V_f32_s1 = SimtConfig<float, 32, 1, 1, 1, 4, 6, 16>;
using V_f24_s64 = SimtConfig<float, 24, 6, 8, 8, 3, 5, 8>;
using V_f24_s16 = SimtConfig<float, 24, 6, 2, 8, 3, 5, 16>;
using V_d24_s8 = SimtConfig<double, 24, 3, 2, 4, 3, 3, 16>;
using V_d8_s4 = SimtConfig<double, 8, 1, 1, 4, 1, 8, 16>;
using V_d32_s16 = SimtConfig<double, 32, 4, 4, 4, 4, 4, 8>;
// complex128 on the FP64 tensor path (DMMA):   NB  S KSPLIT STAGES WARPS
using D_d24_s8 = DmmaConfig<24, 8, 1, 2, 8>;       // (whole stencil matrices per stage: 0.614 ms at configs[1], 0.538 with the balanced partition; KSPLIT 3 with 16 warps: 0.71, SIMT: 0.624)
using D_d32_s16 = DmmaConfig<32, 16, 4, 4, 8>;
using D_d24_s16 = DmmaConfig<24, 16, 3, 4, 8>;
using D_d32_s8 = DmmaConfig<32, 8, 4, 3, 12>;
using D_d16_s16 = DmmaConfig<16, 16, 2, 4, 8>;
using D_d16_s8 = DmmaConfig<16, 8, 2, 4, 16>;
using D_d8_s8 = DmmaConfig<8, 8, 1, 6, 16>;

struct SimtVariant {
    int dtype, nb, s;
    const char *name;
    int (*launch)(const void *, const int32_t *, const void *, void *, int64_t, int, cudaStream_t);
};
#define CMRHS_VARIANT(DT, CFG) {DT, CFG::NB, CFG::S, "stencil_simt<" #CFG ">", &launch_stencil_simt<CFG>}
#define CMRHS_DMMA_VARIANT(CFG) {COARSE_C128, CFG::NB, CFG::S, "stencil_dmma<" #CFG ">", &launch_stencil_dmma<CFG>}
static const SimtVariant kSimtVariants[] = {         // (first match wins: the DMMA variants come before the SIMT ones of the same shape)
    CMRHS_DMMA_VARIANT(D_d24_s8), CMRHS_DMMA_VARIANT(D_d32_s16), CMRHS_DMMA_VARIANT(D_d24_s16), CMRHS_DMMA_VARIANT(D_d32_s8),
    CMRHS_DMMA_VARIANT(D_d16_s16), CMRHS_DMMA_VARIANT(D_d16_s8), CMRHS_DMMA_VARIANT(D_d8_s8),
    CMRHS_VARIANT(COARSE_C64, V_f32_s64), CMRHS_VARIANT(COARSE_C64, V_f32_s32), CMRHS_VARIANT(COARSE_C64, V_f32_s16),
    CMRHS_VARIANT(COARSE_C64, V_f32_s8),  CMRHS_VARIANT(COARSE_C64, V_f32_s4),  CMRHS_VARIANT(COARSE_C64, V_f32_s1),
    CMRHS_VARIANT(COARSE_C64, V_f24_s64), CMRHS_VARIANT(COARSE_C64, V_f24_s16), CMRHS_VARIANT(COARSE_C128, V_d24_s8),
    CMRHS_VARIANT(COARSE_C128, V_d8_s4),  CMRHS_VARIANT(COARSE_C128, V_d32_s16),
};

static const SimtVariant *find_variant(int dtype, int nb, int s, bool allow_dmma = true)
{
    for (const auto &v : kSimtVariants)
        if (v.dtype == dtype && v.nb == nb && v.s == s && (allow_dmma || v.name[8] != 'd')) return &v;      // "stencil_dmma<..."
    return nullptr;
}

}  // namespace cmrhs

using namespace cmrhs;

// ---- the handle ---------------------------------------------------------------------------------------
struct coarse_op {
    LatticeDims dims;
    int nb = 0, nrhs_max = 0, dtype = 0;
    uint32_t flags = 0;
    int num_sms = 0;
    int device = 0;              // the CUDA device the handle (its memory, its kernel attributes) belongs to
    size_t esize = 0;            // bytes per complex element
    void *At = nullptr;          // [V][81][nb(k)][nb(i)]
    float *Ak = nullptr;         // planar k-major [V][81][part][nb(k)][nb(i)] for the tensor path (complex64 only)
    bool tc_ok = false;
    unsigned char *Ah = nullptr; // pre-split FP16 tiles [V][81][hi 4 KB | lo 4 KB] for the FP16-split tensor kernel (complex64, nbasis 32)
    bool h16_ok = false;
    unsigned char *Ax = nullptr; // pre-split FP16 tiles, K-major core-matrix image [V][81][8 nb^2 bytes] (stencil_h16x.cuh: any nbasis in {8,16,24,32})
    bool h16x_ok = false;
    bool x_wide_only = false;    // both split-FP16 layouts are kept (COARSE_FLAG_H16X_WIDE): Ax serves nrhs > 48 only
    float inv_sA = 1.0f;         // 1 / (power-of-two operator scale of Ah)
    unsigned char *Xh = nullptr; // [V] split operand tiles of the current X (pre-pass of the FP16-split kernel)
    cudaStream_t copy_stream = nullptr;   // device->host copy of the solution overlapping the true-residual apply (block_cg_solve_host*)
    cudaEvent_t copy_event = nullptr;
    bool d_colmax_ready = false; // inside a begin/step/end solve: op->amax holds the column maxima of D (written by fused pass 2)
    uint32_t *amax = nullptr;    // [64] per-column max |x| bit patterns (pre-pass of the FP16-split kernel) + [64] scratch
    int32_t *nbr = nullptr;      // [V][81]
    void *pblk[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};           // q, Q, D, z, Z of pblock_cg_solve (allocated on first use)
    void *blk[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // Q, D, Z, T, and two staging blocks for the *_host entry points
    zdouble *gram_partial = nullptr;
    zdouble *defl_partial = nullptr, *defl_C = nullptr;      // deflation: 64 x nrhs_max coefficients and their per-CTA partials (allocated by the first coarse_deflate)
    int gram_blocks = 0;
    zdouble *small = nullptr;    // 6 s x s matrices
    double *dscal = nullptr;     // bnorm[64] relres[64] stop[2] truerel[64]
    int32_t *dinfo = nullptr;
    double *hpin = nullptr;      // pinned host mirror of relres/stop/truerel
    const void *bcg_B = nullptr; // state of a begin/step/end solve
    void *bcg_X = nullptr;
    int bcg_s = 0, bcg_its = 0;
    bool bcg_active = false;
    // optional per-launch timing of the stencil kernel (coarse_op_profile): event pairs recorded on the launch stream
    bool prof_on = false;
    int prof_n = 0;
    cudaEvent_t prof_ev[2 * 64] = {};
    int64_t device_bytes = 0;
    // one BlockCGrQ iteration as a CUDA graph (launch-bound small lattices: 9-14 launches per iteration; the paper loses ~50 % of its
    // coarse operator to launch synchronisation).  Captured at the second iteration of a solve (the first differs in one
    // pre-pass) and replayed while the block X, the width and the pre-pass state are the same; any capture error turns it off.
    cudaGraphExec_t step_graph = nullptr;
    cudaStream_t graph_stream = nullptr;      // the handle's own (blocking) stream: a capture cannot run on the legacy default stream
    const void *graph_X = nullptr, *graph_cand_X = nullptr;
    int graph_cand_s = 0, graph_seen = 0;
    int graph_s = 0, graph_launches = 0;
    bool graph_colmax_in = false, graph_colmax_out = false, graph_off = false;
};

static int alloc_dev(coarse_op *op, void **p, size_t bytes)
{
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        set_error("cudaMalloc of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? COARSE_OUT_OF_MEMORY : COARSE_CUDA_ERROR;
    }
    op->device_bytes += (int64_t)bytes;
    return COARSE_OK;
}

static BcgSmall small_view(const coarse_op *op)
{
    const size_t m = (size_t)COARSE_MAX_NRHS * COARSE_MAX_NRHS;
    BcgSmall w;
    w.G = op->small;
    w.C = op->small + m;
    w.K1 = op->small + 2 * m;
    w.K2 = op->small + 3 * m;
    w.K3 = op->small + 4 * m;
    w.K4 = op->small + 5 * m;
    w.bnorm = op->dscal;
    w.relres = op->dscal + 64;
    w.stop = op->dscal + 128;
    return w;
}

extern "C" const char *coarse_last_error(void) { return g_err; }
extern "C" int64_t coarse_launch_count(void) { return g_launches.load(); }

static int check_shape(const int32_t dims[4], int nb, int s, int dtype)
{
    if (!dims) { set_error("dims is NULL"); return COARSE_INVALID_ARG; }
    for (int k = 0; k < 4; ++k)
        if (dims[k] < 1) { set_error("dims[%d] = %d < 1", k, dims[k]); return COARSE_INVALID_ARG; }
    if (dtype != COARSE_C64 && dtype != COARSE_C128) { set_error("unknown dtype %d", dtype); return COARSE_INVALID_ARG; }
    if (nb < 1 || s < 1) { set_error("nbasis and nrhs must be >= 1"); return COARSE_INVALID_ARG; }
    if (nb > COARSE_MAX_NBASIS || s > COARSE_MAX_NRHS) {
        set_error("nbasis %d / nrhs %d outside the supported range (<= %d / <= %d)", nb, s, COARSE_MAX_NBASIS, COARSE_MAX_NRHS);
        return COARSE_UNSUPPORTED;
    }
    const int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    if (V > 0x7fffffffLL) { set_error("lattice volume %lld exceeds int32 site indices", (long long)V); return COARSE_UNSUPPORTED; }
    return COARSE_OK;
}

extern "C" int coarse_op_destroy(coarse_op_t *op)
{
    if (!op) return COARSE_OK;
    cudaFree(op->At);
    cudaFree(op->Ak);
    if (op->copy_stream) cudaStreamDestroy(op->copy_stream);
    if (op->copy_event) cudaEventDestroy(op->copy_event);
    for (int b = 0; b < 5; ++b) cudaFree(op->pblk[b]);
    cudaFree(op->Ah);
    cudaFree(op->Ax);
    cudaFree(op->Xh);
    cudaFree(op->amax);
    cudaFree(op->nbr);
    for (void *b : op->blk) cudaFree(b);
    cudaFree(op->gram_partial);
    cudaFree(op->defl_partial);
    cudaFree(op->defl_C);
    cudaFree(op->small);
    cudaFree(op->dscal);
    cudaFree(op->dinfo);
    if (op->hpin) cudaFreeHost(op->hpin);
    for (cudaEvent_t e : op->prof_ev) if (e) cudaEventDestroy(e);
    if (op->step_graph) cudaGraphExecDestroy(op->step_graph);
    if (op->graph_stream) cudaStreamDestroy(op->graph_stream);
    delete op;
    return COARSE_OK;
}

extern "C" int coarse_op_create(coarse_op_t **out, const int32_t dims[4], int32_t nbasis, int32_t nrhs_max, int32_t dtype,
                                const void *A_dev, uint32_t flags, void *stream_v)
{
    if (!out) { set_error("out is NULL"); return COARSE_INVALID_ARG; }
    *out = nullptr;
    int st = check_shape(dims, nbasis, nrhs_max, dtype);
    if (st != COARSE_OK) return st;
    if (!A_dev) { set_error("A_dev is NULL"); return COARSE_INVALID_ARG; }
    cudaStream_t stream = (cudaStream_t)stream_v;
    int dev = 0;
    CMRHS_CUDA(cudaGetDevice(&dev));
    coarse_op *op = new (std::nothrow) coarse_op;
    if (!op) { set_error("host allocation failed"); return COARSE_OUT_OF_MEMORY; }
    for (int k = 0; k < 4; ++k) op->dims.L[k] = dims[k];
    op->dims.V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    op->nb = nbasis;
    op->nrhs_max = nrhs_max;
    op->dtype = dtype;
    op->flags = flags;
    op->esize = dtype == COARSE_C64 ? sizeof(cplx<float>) : sizeof(cplx<double>);
    op->device = dev;
    cudaError_t ce = cudaDeviceGetAttribute(&op->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (ce != cudaSuccess) { set_error("cudaDeviceGetAttribute: %s", cudaGetErrorString(ce)); delete op; return COARSE_CUDA_ERROR; }

    const int64_t V = op->dims.V;
    const int64_t ntiles = V * kNPoint;
    const size_t a_bytes = (size_t)ntiles * nbasis * nbasis * op->esize;
    const size_t blk_bytes = (size_t)V * nbasis * nrhs_max * op->esize;
    op->gram_blocks = op->num_sms * 8;
#define CMRHS_TRY(expr)                      \
    do {                                     \
        int _s = (expr);                     \
        if (_s != COARSE_OK) {               \
            coarse_op_destroy(op);           \
            return _s;                       \
        }                                    \
    } while (0)
    const bool want_tc = dtype == COARSE_C64 && !(flags & (COARSE_FLAG_NO_TENSOR | COARSE_FLAG_FORCE_GENERIC)) && tc_supported(nbasis, 8);
    const bool want_split16 = want_tc && !(flags & COARSE_FLAG_TF32);
    // nbasis 32: the paired-site kernel (stencil_h16) by default; COARSE_FLAG_H16X: the X-in-tensor-memory kernel instead;
    // COARSE_FLAG_H16X_WIDE: BOTH layouts, the latter serving nrhs > 48 where it is the faster one
    const bool both16 = want_split16 && nbasis == 32 && (flags & COARSE_FLAG_H16X_WIDE) && !(flags & COARSE_FLAG_H16X) && nrhs_max > 48;
    const bool want_h16x = want_split16 && h16x_supported(nbasis, 8) && (nbasis != 32 || (flags & COARSE_FLAG_H16X) || both16);
    const bool want_h16 = want_split16 && (!want_h16x || both16) && h16_supported(nbasis, 8);
    op->x_wide_only = both16;
    const bool want_simt = !(want_tc && (flags & COARSE_FLAG_TENSOR_ONLY));
    if (want_simt) CMRHS_TRY(alloc_dev(op, &op->At, a_bytes));
    CMRHS_TRY(alloc_dev(op, (void **)&op->nbr, (size_t)ntiles * sizeof(int32_t)));
    if (want_tc && !want_h16 && !want_h16x) CMRHS_TRY(alloc_dev(op, (void **)&op->Ak, a_bytes));
    if (want_h16x) CMRHS_TRY(alloc_dev(op, (void **)&op->Ax, a_bytes));
    if (want_h16) CMRHS_TRY(alloc_dev(op, (void **)&op->Ah, a_bytes));
    if (want_h16 || want_h16x) {
        CMRHS_TRY(alloc_dev(op, (void **)&op->amax, 128 * sizeof(uint32_t)));
        // scratch block of the split X tiles (padding rows / columns of a tile are never written again: zeroed once).  A handle with
        // both layouts uses it in either format: the two kernels serve disjoint widths and every apply rewrites the rows it reads
        size_t xh_bytes = want_h16x ? (size_t)V * h16x_site_bytes(nbasis, nrhs_max) : 0;
        const size_t xh2 = want_h16 ? (size_t)V * h16_xo_bytes(nrhs_max < 8 ? 8 : nrhs_max) : 0;
        if (xh2 > xh_bytes) xh_bytes = xh2;
        CMRHS_TRY(alloc_dev(op, (void **)&op->Xh, xh_bytes));
        CMRHS_CUDA(cudaMemsetAsync(op->Xh, 0, xh_bytes, stream));
    }
    for (int b = 0; b < 6; ++b) CMRHS_TRY(alloc_dev(op, &op->blk[b], blk_bytes));
    CMRHS_TRY(alloc_dev(op, (void **)&op->gram_partial, (size_t)op->gram_blocks * nrhs_max * nrhs_max * sizeof(zdouble)));
    CMRHS_TRY(alloc_dev(op, (void **)&op->small, (size_t)6 * COARSE_MAX_NRHS * COARSE_MAX_NRHS * sizeof(zdouble)));
    CMRHS_TRY(alloc_dev(op, (void **)&op->dscal, 256 * sizeof(double)));
    CMRHS_TRY(alloc_dev(op, (void **)&op->dinfo, 4 * sizeof(int32_t)));
    ce = cudaMallocHost((void **)&op->hpin, 256 * sizeof(double));
    if (ce != cudaSuccess) { set_error("cudaMallocHost: %s", cudaGetErrorString(ce)); coarse_op_destroy(op); return COARSE_CUDA_ERROR; }
#undef CMRHS_TRY

    // a1: neighbour table, once ("The pointers are precomputed")
    {
        const int grid = (int)(ceil_div(ntiles, 256) < 65535 ? ceil_div(ntiles, 256) : 65535);
        neighbour_table_kernel<<<grid, 256, 0, stream>>>(op->dims, op->nbr);
        count_launch();
    }
    // re-layout A into k-major tiles (SIMT kernels: interleaved complex; tensor kernel: planar float32)
    const int rgrid = (int)(ntiles < 1048576 ? ntiles : 1048576);
    if (want_simt) {
        if (dtype == COARSE_C64)
            relayout_transpose_kernel<float><<<rgrid, 128, 0, stream>>>((const cplx<float> *)A_dev, (cplx<float> *)op->At, ntiles, nbasis);
        else
            relayout_transpose_kernel<double><<<rgrid, 128, 0, stream>>>((const cplx<double> *)A_dev, (cplx<double> *)op->At, ntiles, nbasis);
        count_launch();
    }
    if (want_tc && !want_h16 && !want_h16x) {
        relayout_planar_kernel<<<rgrid, 128, 0, stream>>>((const cplx<float> *)A_dev, op->Ak, ntiles, nbasis);
        count_launch();
        op->tc_ok = true;
    }
    if (want_h16 || want_h16x) {
        // operator scale: the power of two that maps max |Re a|, |Im a| into [2^14, 2^15) (stencil_h16.cuh)
        uint32_t bits = 0;
        ce = cudaMemsetAsync(op->amax, 0, 128 * sizeof(uint32_t), stream);
        if (ce == cudaSuccess) {
            absmax_kernel<<<op->num_sms * 8, 256, 0, stream>>>((const float *)A_dev, (int64_t)ntiles * nbasis * nbasis * 2, op->amax + 64);
            count_launch();
            ce = cudaMemcpyAsync(&bits, op->amax + 64, sizeof(uint32_t), cudaMemcpyDeviceToHost, stream);
        }
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(stream);
        if (ce != cudaSuccess) {
            set_error("operator scale pass failed: %s", cudaGetErrorString(ce));
            coarse_op_destroy(op);
            return COARSE_CUDA_ERROR;
        }
        const float sA = h_scale_from_bits(bits);
        op->inv_sA = 1.0f / sA;
        if (want_h16) {
            relayout_h16_kernel<<<rgrid, 256, 0, stream>>>((const cplx<float> *)A_dev, op->Ah, ntiles, sA);
            op->h16_ok = true;
            count_launch();
        }
        if (want_h16x) {
            relayout_h16x_kernel<<<rgrid, 256, 0, stream>>>((const cplx<float> *)A_dev, op->Ax, ntiles, nbasis, sA);
            op->h16x_ok = true;
            count_launch();
        }
    }
    ce = cudaGetLastError();
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(stream);
    if (ce != cudaSuccess) {
        set_error("operator setup kernels failed: %s", cudaGetErrorString(ce));
        coarse_op_destroy(op);
        return COARSE_CUDA_ERROR;
    }
    *out = op;
    return COARSE_OK;
}

extern "C" int64_t coarse_op_device_bytes(const coarse_op_t *op) { return op ? op->device_bytes : 0; }

static const SimtVariant *select_variant(const coarse_op *op, int nrhs)
{
    if (op->flags & COARSE_FLAG_FORCE_GENERIC) return nullptr;
    return find_variant(op->dtype, op->nb, nrhs, !(op->flags & COARSE_FLAG_NO_TENSOR));
}

static bool use_tc(const coarse_op *op, int nrhs) { return op->tc_ok && tc_supported(op->nb, nrhs); }
static bool use_h16(const coarse_op *op, int nrhs) { return op->h16_ok && h16_supported(op->nb, nrhs) && !(op->x_wide_only && nrhs > 48); }
// the X-in-tensor-memory kernel covers every nrhs; a single column (or a pair) is left to a tuned SIMT variant when there is one
static bool use_h16x(const coarse_op *op, int nrhs)
{
    if (!op->h16x_ok || !h16x_supported(op->nb, nrhs)) return false;
    if (op->x_wide_only) return nrhs > 48;
    return nrhs >= 4 || !op->At || !find_variant(op->dtype, op->nb, nrhs);
}
// the kernels whose X operand is scaled by per-column powers of two (column maxima in op->amax)
static bool use_split16(const coarse_op *op, int nrhs) { return use_h16(op, nrhs) || use_h16x(op, nrhs); }

extern "C" const char *coarse_op_kernel_name(const coarse_op_t *op, int32_t nrhs)
{
    if (!op) return "";
    if (use_h16(op, nrhs)) return "stencil_h16<fp16x3>";
    if (use_h16x(op, nrhs)) return "stencil_h16x<fp16x3>";
    if (use_tc(op, nrhs)) return "stencil_tc<tf32x3>";
    if (!op->At) return "unsupported";
    const SimtVariant *v = select_variant(op, nrhs);
    return v ? v->name : (op->dtype == COARSE_C64 ? "stencil_generic<float>" : "stencil_generic<double>");
}

static int apply_launch(const coarse_op *op, const void *X, void *Y, int nrhs, cudaStream_t stream, bool have_colmax);

// have_colmax: the caller guarantees that op->amax holds the column maxima of X (only bcg_step, for D after fused pass 2)
static int apply_impl(const coarse_op *op_c, const void *X, void *Y, int nrhs, cudaStream_t stream, bool have_colmax = false)
{
    coarse_op *op = const_cast<coarse_op *>(op_c);
    if (!op->prof_on || op->prof_n >= 64) return apply_launch(op, X, Y, nrhs, stream, have_colmax);
    const int k = op->prof_n;
    CMRHS_CUDA(cudaEventRecord(op->prof_ev[2 * k], stream));
    int st = apply_launch(op, X, Y, nrhs, stream, have_colmax);
    CMRHS_CUDA(cudaEventRecord(op->prof_ev[2 * k + 1], stream));
    op->prof_n = k + 1;
    return st;
}

static int apply_launch(const coarse_op *op, const void *X, void *Y, int nrhs, cudaStream_t stream, bool have_colmax)
{
    if (use_h16(op, nrhs)) {
        if (!have_colmax) const_cast<coarse_op *>(op)->d_colmax_ready = false;     // this apply's own pre-pass overwrites op->amax
        return launch_stencil_h16(op->Ah, op->inv_sA, op->amax, op->Xh, op->dims, X, Y, nrhs, op->num_sms, stream, have_colmax);
    }
    if (use_h16x(op, nrhs)) {
        if (!have_colmax) const_cast<coarse_op *>(op)->d_colmax_ready = false;
        switch (op->nb) {
        case 8: return launch_stencil_h16x<8>(op->Ax, op->inv_sA, op->amax, op->Xh, op->dims, X, Y, nrhs, op->num_sms, stream, have_colmax);
        case 16: return launch_stencil_h16x<16>(op->Ax, op->inv_sA, op->amax, op->Xh, op->dims, X, Y, nrhs, op->num_sms, stream, have_colmax);
        case 24: return launch_stencil_h16x<24>(op->Ax, op->inv_sA, op->amax, op->Xh, op->dims, X, Y, nrhs, op->num_sms, stream, have_colmax);
        default: return launch_stencil_h16x<32>(op->Ax, op->inv_sA, op->amax, op->Xh, op->dims, X, Y, nrhs, op->num_sms, stream, have_colmax);
        }
    }
    if (use_tc(op, nrhs)) {
        switch (op->nb) {
        case 8: return launch_stencil_tc<8>(op->Ak, op->dims, X, Y, nrhs, op->num_sms, stream);
        case 16: return launch_stencil_tc<16>(op->Ak, op->dims, X, Y, nrhs, op->num_sms, stream);
        case 24: return launch_stencil_tc<24>(op->Ak, op->dims, X, Y, nrhs, op->num_sms, stream);
        default: return launch_stencil_tc<32>(op->Ak, op->dims, X, Y, nrhs, op->num_sms, stream);
        }
    }
    if (!op->At) {
        set_error("COARSE_FLAG_TENSOR_ONLY: nrhs %d is not covered by the tensor-core kernel (multiples of 8)", nrhs);
        return COARSE_UNSUPPORTED;
    }
    const SimtVariant *v = select_variant(op, nrhs);
    if (v) return v->launch(op->At, op->nbr, X, Y, op->dims.V, op->num_sms, stream);
    if (op->dtype == COARSE_C64)
        return launch_stencil_generic<float>((const cplx<float> *)op->At, op->nbr, (const cplx<float> *)X, (cplx<float> *)Y,
                                             op->dims.V, op->nb, nrhs, op->num_sms, stream);
    return launch_stencil_generic<double>((const cplx<double> *)op->At, op->nbr, (const cplx<double> *)X, (cplx<double> *)Y,
                                          op->dims.V, op->nb, nrhs, op->num_sms, stream);
}

// the handle's device must be the current one (its buffers and kernel attributes live there)
static int check_device(const coarse_op *op)
{
    int dev = -1;
    CMRHS_CUDA(cudaGetDevice(&dev));
    if (dev != op->device) { set_error("handle was created on device %d, current device is %d", op->device, dev); return COARSE_INVALID_ARG; }
    return COARSE_OK;
}

// device blocks must be 16-byte aligned: bulk-TMA loads, cp.async and float4 accesses (coarse_mrhs.h)
static bool misaligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

static int check_apply_args(const coarse_op *op, const void *X, const void *Y, int nrhs, bool device_ptrs = true)
{
    if (!op || !X || !Y) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (nrhs < 1 || nrhs > op->nrhs_max) { set_error("nrhs %d outside 1..nrhs_max=%d", nrhs, op->nrhs_max); return COARSE_INVALID_ARG; }
    if (X == Y) { set_error("Y must not alias X"); return COARSE_INVALID_ARG; }
    if (device_ptrs && (misaligned16(X) || misaligned16(Y))) { set_error("X and Y must be 16-byte aligned"); return COARSE_INVALID_ARG; }
    return check_device(op);
}

extern "C" int coarse_op_apply(const coarse_op_t *op, const void *X_dev, void *Y_dev, int32_t nrhs, void *stream)
{
    int st = check_apply_args(op, X_dev, Y_dev, nrhs);
    if (st != COARSE_OK) return st;
    return apply_impl(op, X_dev, Y_dev, nrhs, (cudaStream_t)stream);
}

extern "C" int coarse_op_apply_host(coarse_op_t *op, const void *X_host, void *Y_host, int32_t nrhs, void *stream_v)
{
    int st = check_apply_args(op, X_host, Y_host, nrhs, false);
    if (st != COARSE_OK) return st;
    cudaStream_t stream = (cudaStream_t)stream_v;
    const size_t bytes = (size_t)op->dims.V * op->nb * nrhs * op->esize;
    CMRHS_CUDA(cudaMemcpyAsync(op->blk[4], X_host, bytes, cudaMemcpyHostToDevice, stream));
    st = apply_impl(op, op->blk[4], op->blk[5], nrhs, stream);
    if (st != COARSE_OK) return st;
    CMRHS_CUDA(cudaMemcpyAsync(Y_host, op->blk[5], bytes, cudaMemcpyDeviceToHost, stream));
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    return COARSE_OK;
}

// ---- block-CG building blocks --------------------------------------------------------------------------
static bool use_tla(const coarse_op *op, int s);

template <typename T>
static int gram_impl(const coarse_op *op, const void *U, const void *W, zdouble *G, int64_t n, int s, cudaStream_t stream)
{
    if (sizeof(T) == 4 && use_tla(op, s)) {               // wide complex64 blocks: split-FP16 Gram on the tensor cores (blockla_tc.cuh)
        int blocks = 0;
        const int st_tg = launch_tgram(U, W, op->gram_partial, op->gram_blocks, n, s, op->num_sms, stream, &blocks);
        if (st_tg != COARSE_OK) return st_tg;
        gram_reduce_kernel<<<(s * s * 32 + 127) / 128, 128, 0, stream>>>(op->gram_partial, blocks, s * s, G);
        CMRHS_LAUNCH_CHECK();
        return COARSE_OK;
    }
#ifndef CMRHS_NO_GRAM_PIPE      // (A/B builds: the staged kernel below for every width)
    if constexpr (sizeof(T) == 4) if ((s == 16 || s == 32) && n >= 4096) {       // complex64 at the widths block CG runs at: bulk-copy pipeline (gram_pipe_kernel)
        constexpr int kTT = 4;
        const int RGp = kLaThreads / ((s / kTT) * (s / kTT));          // 16 / 4 row groups
        const int rows = 12288 / (s * (int)sizeof(cplx<T>));           // 12 KB per operand and stage: 96 / 48 rows
        const int flush = 36 / (rows / RGp);                           // runs of 36 rows in T between flushes to double
        const size_t smem = (size_t)kGramPipeStages * 2 * rows * s * sizeof(cplx<T>) + kGramPipeStages * sizeof(uint64_t);
        int blocks = 2 * op->num_sms;
        if (blocks > op->gram_blocks) blocks = op->gram_blocks;
        if ((int64_t)blocks > ceil_div(n, rows)) blocks = (int)ceil_div(n, rows);
        const cplx<T> *u = (const cplx<T> *)U, *w = (const cplx<T> *)W;
        if (s == 16) {
            auto kern = gram_pipe_kernel<T, kTT, 16>;
            CMRHS_SMEM_ATTR(kern, smem);
            kern<<<blocks, kLaThreads, smem, stream>>>(u, w, n, rows, flush, op->gram_partial);
        } else {
            auto kern = gram_pipe_kernel<T, kTT, 32>;
            CMRHS_SMEM_ATTR(kern, smem);
            kern<<<blocks, kLaThreads, smem, stream>>>(u, w, n, rows, flush, op->gram_partial);
        }
        CMRHS_LAUNCH_CHECK();
        gram_reduce_kernel<<<(s * s * 32 + 127) / 128, 128, 0, stream>>>(op->gram_partial, blocks, s * s, G);
        CMRHS_LAUNCH_CHECK();
        return COARSE_OK;
    }
#endif
    int TT = s > 32 ? 4 : (s >= 8 ? 2 : 1);
    const int nt = (s + TT - 1) / TT;
    const int RG = kLaThreads / (nt * nt);
    size_t tile_bytes = 40960;            // (20-80 KB measured equal on B200)
    int rows = (int)(tile_bytes / (2 * (size_t)s * sizeof(cplx<T>)));
    rows = rows / RG * RG;
    if (rows < RG) rows = RG;
    size_t smem = (size_t)rows * s * 2 * sizeof(cplx<T>);
    if (RG > 1 && smem < (size_t)s * s * sizeof(zdouble)) smem = (size_t)s * s * sizeof(zdouble);
    int blocks = op->gram_blocks;
    if ((int64_t)blocks > ceil_div(n, rows)) blocks = (int)ceil_div(n, rows);
    if (blocks < 1) blocks = 1;
    const cplx<T> *u = (const cplx<T> *)U, *w = (const cplx<T> *)W;
#define CMRHS_GRAM_CASE(TTV, ...)                                                                                \
    {                                                                                                            \
        auto kern = gram_partial_kernel<T, TTV, ##__VA_ARGS__>;                                                  \
        CMRHS_SMEM_ATTR(kern, smem); \
        kern<<<blocks, kLaThreads, smem, stream>>>(u, w, n, s, rows, op->gram_partial);                          \
    }
    if (TT == 4 && s == 64) CMRHS_GRAM_CASE(4, 64)
    else if (TT == 2 && s == 32) CMRHS_GRAM_CASE(2, 32)
    else if (TT == 2 && s == 16) CMRHS_GRAM_CASE(2, 16)
    else if (TT == 2 && s == 8) CMRHS_GRAM_CASE(2, 8)
    else
    switch (TT) {
    case 1: CMRHS_GRAM_CASE(1) break;
    case 2: CMRHS_GRAM_CASE(2) break;
    case 3: CMRHS_GRAM_CASE(3) break;
    default: CMRHS_GRAM_CASE(4) break;
    }
#undef CMRHS_GRAM_CASE
    CMRHS_LAUNCH_CHECK();
    gram_reduce_kernel<<<(s * s * 32 + 127) / 128, 128, 0, stream>>>(op->gram_partial, blocks, s * s, G);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

static int gram_dispatch(const coarse_op *op, const void *U, const void *W, zdouble *G, int64_t n, int s, cudaStream_t stream)
{
    return op->dtype == COARSE_C64 ? gram_impl<float>(op, U, W, G, n, s, stream) : gram_impl<double>(op, U, W, G, n, s, stream);
}

template <typename T>
static int rotate_impl(const coarse_op *op, const void *U, const zdouble *K, const void *Vin, void *out, double beta, int64_t n,
                       int s, cudaStream_t stream)
{
    const int TC = (s + 15) / 16;
    const int ncg = (s + TC - 1) / TC;
    const int RL = kLaThreads / ncg;
    int rows = RL * 4;
    const size_t smem = ((size_t)s * s + (size_t)rows * (s + 1)) * sizeof(cplx<T>);
    const int64_t ntiles = ceil_div(n, rows);
    const int grid = (int)(ntiles < (int64_t)op->num_sms * 4 ? ntiles : (int64_t)op->num_sms * 4);
#define CMRHS_ROT_CASE(TCV)                                                                                      \
    {                                                                                                            \
        auto kern = rotate_kernel<T, TCV>;                                                                       \
        CMRHS_SMEM_ATTR(kern, smem); \
        kern<<<grid, kLaThreads, smem, stream>>>((const cplx<T> *)U, K, (const cplx<T> *)Vin, (cplx<T> *)out, (T)beta, n, s, rows); \
    }
    switch (TC) {
    case 1: CMRHS_ROT_CASE(1) break;
    case 2: CMRHS_ROT_CASE(2) break;
    case 3: CMRHS_ROT_CASE(3) break;
    default: CMRHS_ROT_CASE(4) break;
    }
#undef CMRHS_ROT_CASE
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// complex64 blocks of width >= 32 (or >= 16 with COARSE_FLAG_TENSOR_LINALG): rotations and Gram products on the tensor cores
static bool use_tla(const coarse_op *op, int s)
{
    if (op->dtype != COARSE_C64 || (op->flags & (COARSE_FLAG_NO_TENSOR | COARSE_FLAG_FORCE_GENERIC)) || !tla_supported(s)) return false;
    return s >= 40 || (op->flags & COARSE_FLAG_TENSOR_LINALG);      // (measured at configs[3]: at width 32 the fused SIMT passes are still faster: 2.4 vs 2.9 ms)
}

static int rotate_dispatch(const coarse_op *op, const void *U, const zdouble *K, const void *Vin, void *out, double beta, int64_t n,
                           int s, cudaStream_t stream)
{
    if (use_tla(op, s)) return launch_trot(U, K, beta != 0.0 ? Vin : nullptr, out, beta, n, s, op->num_sms, stream);
    return op->dtype == COARSE_C64 ? rotate_impl<float>(op, U, K, Vin, out, beta, n, s, stream)
                                   : rotate_impl<double>(op, U, K, Vin, out, beta, n, s, stream);
}

// ---- the two fused passes of a BlockCGrQ iteration (blockcg_kernels.cuh) ---------------------------------
struct FusedPlan { int W, TR, rows, grid; size_t smem; };
// shared-memory budget of one CTA of the fused passes: the tile height TR is halved until the two K matrices and the
// double-buffered row tiles fit.  Measured at nrhs 64 (config 4): 100 KB (TR 1) 15.8 ms, 140 KB (TR 2) 11.0 ms, 210 KB (TR 4,
// one CTA per SM) 9.0 ms per iteration of linear algebra -- the wider register tile beats the second CTA.
#ifndef LA_W4_FROM
#define LA_W4_FROM 33
#endif
#ifndef LA_CAP
#define LA_CAP 210
#endif

template <typename T>
static FusedPlan fused_plan(const coarse_op *op, int64_t n, int s)
{
    FusedPlan p;
    p.W = s >= LA_W4_FROM ? 4 : (s >= 8 ? 2 : 1);
    if ((s + p.W - 1) / p.W > 16) p.W = 4;
    const int ncg = (s + p.W - 1) / p.W, RL = kLaThreads / ncg, su = s + LaPad<T>::v;
#ifndef LA_TR0
#define LA_TR0 2      // complex64, width 16: 64-row tiles, 4 CTAs per SM (other_ms 0.693 -> 0.675 against TR 4 with 2 CTAs; TR 8: 0.765; W 4: 0.97)
#endif
    int tr0 = (s == 16 && sizeof(T) == 4) ? LA_TR0 : 4;
    for (p.TR = tr0; ; p.TR /= 2) {
        p.rows = RL * p.TR;
        size_t tiles = (size_t)4 * p.rows * su * sizeof(cplx<T>);      // two operands x two stages
        const size_t red = (size_t)s * s * sizeof(zdouble);
        if (tiles < red) tiles = red;
        p.smem = (size_t)2 * s * s * sizeof(cplx<T>) + tiles;
        if (p.smem <= LA_CAP * 1024 || p.TR == 1) break;
    }
    int per_sm = p.smem <= 27 * 1024 ? 8 : (p.smem <= 56 * 1024 ? 4 : (p.smem <= 113 * 1024 ? 2 : 1));
    const int64_t ntiles = ceil_div(n, p.rows);
    int64_t g = (int64_t)op->num_sms * per_sm;
    if (g > op->gram_blocks) g = op->gram_blocks;
    p.grid = (int)(ntiles < g ? ntiles : g);
    return p;
}

template <typename T, int TR, int W, int S = 0>
static int fused1_launch(const coarse_op *op, const FusedPlan &p, const void *D, const void *Z, const void *Q, void *X, void *Tout,
                         const zdouble *K1, const zdouble *K2, int64_t n, int s, cudaStream_t stream)
{
    auto kern = bcg_fused1_kernel<T, TR, W, S>;
    CMRHS_SMEM_ATTR(kern, p.smem);
    kern<<<p.grid, kLaThreads, p.smem, stream>>>((const cplx<T> *)D, (const cplx<T> *)Z, (const cplx<T> *)Q, (cplx<T> *)X, (cplx<T> *)Tout, K1, K2,
                                                  n, s, op->gram_partial);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}
template <typename T, int TR, int W, int S = 0>
static int fused2_launch(const coarse_op *op, const FusedPlan &p, const void *Tin, void *D, void *Qout, const zdouble *K3, const zdouble *K4,
                         int64_t n, int s, cudaStream_t stream)
{
    auto kern = bcg_fused2_kernel<T, TR, W, S>;
    CMRHS_SMEM_ATTR(kern, p.smem);
    // the next reader of D is the stencil kernel: if that is the FP16-split one, its column-maxima pre-pass is done here
    uint32_t *colmax = (sizeof(T) == 4 && use_split16(op, s)) ? op->amax : nullptr;
    if (colmax) CMRHS_CUDA(cudaMemsetAsync(colmax, 0, 64 * sizeof(uint32_t), stream));
    kern<<<p.grid, kLaThreads, p.smem, stream>>>((const cplx<T> *)Tin, (cplx<T> *)D, (cplx<T> *)Qout, K3, K4, n, s, colmax);
    const_cast<coarse_op *>(op)->d_colmax_ready = colmax != nullptr;
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// the common block widths run kernels with s as a compile-time constant (plan TR 4, W 2)
#define CMRHS_FUSED_SWITCH(CALL)                                         \
    if (p.TR == 4 && p.W == 2) {                                         \
        if (s == 8) return CALL(4, 2, 8); if (s == 16) return CALL(4, 2, 16); if (s == 32) return CALL(4, 2, 32); \
        if (s == 64) return CALL(4, 2, 64);                              \
    }                                                                    \
    if (p.W == 4 && s == 64) {                                           \
        if (p.TR == 4) return CALL(4, 4, 64); if (p.TR == 2) return CALL(2, 4, 64); return CALL(1, 4, 64); \
    }                                                                    \
    if (p.W == 4 && p.TR == 4 && s == 32) return CALL(4, 4, 32);         \
    if (p.W == 4 && p.TR == 4 && s == 16) return CALL(4, 4, 16);         \
    if (p.W == 2 && p.TR == 2 && s == 16) return CALL(2, 2, 16);         \
    if (p.W == 2 && p.TR == 8 && s == 16) return CALL(8, 2, 16);         \
    if (p.TR == 4) {                                                     \
        if (p.W == 4) return CALL(4, 4); if (p.W == 2) return CALL(4, 2); return CALL(4, 1); \
    }                                                                    \
    if (p.TR == 2) {                                                     \
        if (p.W == 4) return CALL(2, 4); if (p.W == 2) return CALL(2, 2); return CALL(2, 1); \
    }                                                                    \
    if (p.W == 4) return CALL(1, 4); if (p.W == 2) return CALL(1, 2); return CALL(1, 1);

// X += D K1 ; T = Q + Z K2 ; G = T^H T   (G through the deterministic two-stage reduction)
template <typename T>
static int fused1_impl(const coarse_op *op, const void *D, const void *Z, const void *Q, void *X, void *Tout, const zdouble *K1,
                       const zdouble *K2, zdouble *G, int64_t n, int s, cudaStream_t stream)
{
    const FusedPlan p = fused_plan<T>(op, n, s);
    auto run = [&]() -> int {
#define CMRHS_F1(TRV, WV, ...) fused1_launch<T, TRV, WV, ##__VA_ARGS__>(op, p, D, Z, Q, X, Tout, K1, K2, n, s, stream)
        CMRHS_FUSED_SWITCH(CMRHS_F1)
#undef CMRHS_F1
    };
    int st = run();
    if (st != COARSE_OK) return st;
    gram_reduce_kernel<<<(s * s * 32 + 127) / 128, 128, 0, stream>>>(op->gram_partial, p.grid, s * s, G);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}
// Q = T K3 ; D = Q + D K4
template <typename T>
static int fused2_impl(const coarse_op *op, const void *Tin, void *D, void *Qout, const zdouble *K3, const zdouble *K4, int64_t n, int s,
                       cudaStream_t stream)
{
    const FusedPlan p = fused_plan<T>(op, n, s);
#define CMRHS_F2(TRV, WV, ...) fused2_launch<T, TRV, WV, ##__VA_ARGS__>(op, p, Tin, D, Qout, K3, K4, n, s, stream)
    CMRHS_FUSED_SWITCH(CMRHS_F2)
#undef CMRHS_F2
}

static int axpby_dispatch(const coarse_op *op, const void *U, const void *W, void *out, double a, double b, int64_t total,
                          cudaStream_t stream)
{
    const int grid = (int)(ceil_div(total, 256) < (int64_t)op->num_sms * 16 ? ceil_div(total, 256) : (int64_t)op->num_sms * 16);
    if (op->dtype == COARSE_C64)
        axpby_kernel<float><<<grid, 256, 0, stream>>>((const cplx<float> *)U, (const cplx<float> *)W, (cplx<float> *)out, (float)a, (float)b, total);
    else
        axpby_kernel<double><<<grid, 256, 0, stream>>>((const cplx<double> *)U, (const cplx<double> *)W, (cplx<double> *)out, a, b, total);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

static int small_smem_attr(const void *kern, int s, int nmat, size_t *smem)
{
    *smem = (size_t)nmat * s * s * sizeof(zdouble);
    CMRHS_SMEM_ATTR(kern, *smem);
    return COARSE_OK;
}

extern "C" int coarse_block_gram(coarse_op_t *op, const void *U_dev, const void *W_dev, void *G_dev, int64_t n, int32_t s, void *stream)
{
    if (!op || !U_dev || !W_dev || !G_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (s < 1 || s > op->nrhs_max || n < 1) { set_error("bad n/s"); return COARSE_INVALID_ARG; }
    return gram_dispatch(op, U_dev, W_dev, (zdouble *)G_dev, n, s, (cudaStream_t)stream);
}

extern "C" int coarse_block_rotate(coarse_op_t *op, const void *U_dev, const void *K_dev, void *W_dev, double beta, int64_t n, int32_t s,
                                   void *stream)
{
    if (!op || !U_dev || !K_dev || !W_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (s < 1 || s > COARSE_MAX_NRHS || n < 1) { set_error("bad n/s"); return COARSE_INVALID_ARG; }
    if (U_dev == W_dev) { set_error("W must not alias U"); return COARSE_INVALID_ARG; }
    return rotate_dispatch(op, U_dev, (const zdouble *)K_dev, W_dev, W_dev, beta, n, s, (cudaStream_t)stream);
}

extern "C" int coarse_small_cholesky(const void *G_dev, void *S_dev, void *Sinv_dev, int32_t s, int32_t *info_dev, void *stream)
{
    if (!G_dev || !S_dev || !info_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (s < 1 || s > COARSE_MAX_NRHS) { set_error("bad s"); return COARSE_INVALID_ARG; }
    size_t smem;
    int st = small_smem_attr((const void *)small_cholesky_kernel, s, 2, &smem);
    if (st != COARSE_OK) return st;
    small_cholesky_kernel<<<1, kLaThreads, smem, (cudaStream_t)stream>>>((const zdouble *)G_dev, (zdouble *)S_dev, (zdouble *)Sinv_dev, s, info_dev);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

extern "C" int coarse_small_hpd_inverse(const void *G_dev, void *M_dev, int32_t s, int32_t *info_dev, void *stream)
{
    if (!G_dev || !M_dev || !info_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (s < 1 || s > COARSE_MAX_NRHS) { set_error("bad s"); return COARSE_INVALID_ARG; }
    size_t smem;
    int st = small_smem_attr((const void *)small_hpd_inverse_kernel, s, 2, &smem);
    if (st != COARSE_OK) return st;
    small_hpd_inverse_kernel<<<1, kLaThreads, smem, (cudaStream_t)stream>>>((const zdouble *)G_dev, (zdouble *)M_dev, s, info_dev);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// ---- BlockCGrQ (Fig. 2 left) ----------------------------------------------------------
static int small_launch(void (*kern)(BcgSmall, int), const coarse_op *op, int s, int nmat, cudaStream_t stream)
{
    size_t smem;
    int st = small_smem_attr((const void *)kern, s, nmat, &smem);
    if (st != COARSE_OK) return st;
    kern<<<1, kLaThreads, smem, stream>>>(small_view(op), s);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// copies relres[64] | stop[2] | truerel[64] (device doubles 64..193) to the pinned mirror and synchronises
static int fetch_scalars(const coarse_op *op, cudaStream_t stream)
{
    CMRHS_CUDA(cudaMemcpyAsync(op->hpin, op->dscal + 64, 130 * sizeof(double), cudaMemcpyDeviceToHost, stream));
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    return COARSE_OK;
}

#define CMRHS_STEP(expr)                   \
    do {                                   \
        int _s = (expr);                   \
        if (_s != COARSE_OK) return _s;    \
    } while (0)

// The solve is split into begin / step / poll / end so that a caller (bench.py) can time exactly K iterations
// on the device without the per-iteration host read of block_cg_solve.  State lives in the handle.
static int bcg_begin(coarse_op *op, const void *B, void *X, int s, double tol, cudaStream_t stream, bool zero_guess = false)
{
    const int64_t n = op->dims.V * op->nb, total = n * s;
    const size_t blk_bytes = (size_t)total * op->esize;
    void *Q = op->blk[0], *D = op->blk[1], *Z = op->blk[2], *T = op->blk[3];
    BcgSmall w = small_view(op);
    op->bcg_B = B; op->bcg_X = X; op->bcg_s = s; op->bcg_its = 0; op->bcg_active = false;
    op->d_colmax_ready = false;
    // ||B[:,r]||
    CMRHS_STEP(gram_dispatch(op, B, B, w.G, n, s, stream));
    bcg_bnorm_kernel<<<1, 64, 0, stream>>>(w, s);
    CMRHS_LAUNCH_CHECK();
    // R_0 = B - H X_0  (held in T); with a zero initial guess R_0 = B and the apply is skipped
    if (zero_guess) {
        CMRHS_CUDA(cudaMemsetAsync(X, 0, blk_bytes, stream));
        CMRHS_CUDA(cudaMemcpyAsync(T, B, blk_bytes, cudaMemcpyDeviceToDevice, stream));
    } else {
        CMRHS_STEP(apply_impl(op, X, Z, s, stream));
        CMRHS_STEP(axpby_dispatch(op, B, Z, T, 1.0, -1.0, total, stream));
    }
    // Q_0 C_0 = R_0 by Cholesky of R^H R
    CMRHS_STEP(gram_dispatch(op, T, T, w.G, n, s, stream));
    {
        size_t smem;
        CMRHS_STEP(small_smem_attr((const void *)bcg_init_kernel, s, 2, &smem));
        bcg_init_kernel<<<1, kLaThreads, smem, stream>>>(w, s, tol);
        CMRHS_LAUNCH_CHECK();
    }
    CMRHS_STEP(fetch_scalars(op, stream));
    const double *h_stop = op->hpin + 64;
    if (h_stop[1] != 0.0) return COARSE_BREAKDOWN;
    if (h_stop[0] <= tol) return COARSE_OK;                                             // X_0 already solves the system
    CMRHS_STEP(rotate_dispatch(op, T, w.K1, nullptr, Q, 0.0, n, s, stream));           // Q_0 = R_0 C_0^-1
    CMRHS_CUDA(cudaMemcpyAsync(D, Q, blk_bytes, cudaMemcpyDeviceToDevice, stream));    // D_0 = Q_0
    op->bcg_active = true;
    return COARSE_NOT_CONVERGED;
}

// one iteration k -> k+1 of Fig. 2 (left), statements 8-13; asynchronous, no host read
static int bcg_step(coarse_op *op, cudaStream_t stream)
{
    const int s = op->bcg_s;
    const int64_t n = op->dims.V * op->nb;
    void *Q = op->blk[0], *D = op->blk[1], *Z = op->blk[2], *T = op->blk[3], *X = op->bcg_X;
    BcgSmall w = small_view(op);
    CMRHS_STEP(apply_impl(op, D, Z, s, stream, op->d_colmax_ready));               // Z_k = H D_k
    op->d_colmax_ready = false;
    CMRHS_STEP(gram_dispatch(op, D, Z, w.G, n, s, stream));                        // D^H Z
    CMRHS_STEP(small_launch(bcg_step1_kernel, op, s, 3, stream));                  // M, K1 = M C, K2 = -M
    if ((op->flags & COARSE_FLAG_UNFUSED_LINALG) || use_tla(op, s)) {       // (wide complex64 blocks: every product on the tensor cores)
        CMRHS_STEP(rotate_dispatch(op, D, w.K1, X, X, 1.0, n, s, stream));             // X += D M C
        CMRHS_STEP(rotate_dispatch(op, Z, w.K2, Q, T, 1.0, n, s, stream));             // T = Q - Z M
        CMRHS_STEP(gram_dispatch(op, T, T, w.G, n, s, stream));                        // T^H T
        CMRHS_STEP(small_launch(bcg_step2_kernel, op, s, 3, stream));                  // S, K3 = S^-1, K4 = S^H, C = S C
        CMRHS_STEP(rotate_dispatch(op, T, w.K3, nullptr, Q, 0.0, n, s, stream));       // Q = T S^-1
        CMRHS_STEP(rotate_dispatch(op, D, w.K4, Q, D, 1.0, n, s, stream));             // D = Q + D S^H
    } else if (op->dtype == COARSE_C64) {
        CMRHS_STEP(fused1_impl<float>(op, D, Z, Q, X, T, w.K1, w.K2, w.G, n, s, stream));   // X += D M C ; T = Q - Z M ; T^H T
        CMRHS_STEP(small_launch(bcg_step2_kernel, op, s, 3, stream));                        // S, K3 = S^-1, K4 = S^H, C = S C
        CMRHS_STEP(fused2_impl<float>(op, T, D, Q, w.K3, w.K4, n, s, stream));               // Q = T S^-1 ; D = Q + D S^H
    } else {
        CMRHS_STEP(fused1_impl<double>(op, D, Z, Q, X, T, w.K1, w.K2, w.G, n, s, stream));
        CMRHS_STEP(small_launch(bcg_step2_kernel, op, s, 3, stream));
        CMRHS_STEP(fused2_impl<double>(op, T, D, Q, w.K3, w.K4, n, s, stream));
    }
    op->bcg_its += 1;
    return COARSE_OK;
}

// bcg_step through a CUDA graph where that pays (the iteration is launch-bound: small lattices) and is possible
static int bcg_step_fast(coarse_op *op, cudaStream_t stream)
{
    const int64_t n_elems = op->dims.V * op->nb * (int64_t)op->bcg_s;
    if (op->graph_off || op->prof_on || n_elems > (1ll << 22) || (op->flags & COARSE_FLAG_NO_GRAPH)) return bcg_step(op, stream);
    if (op->step_graph && op->graph_X == op->bcg_X && op->graph_s == op->bcg_s && op->graph_colmax_in == op->d_colmax_ready) {
        cudaStream_t gs = stream ? stream : op->graph_stream;
        CMRHS_CUDA(cudaGraphLaunch(op->step_graph, gs));
        count_launch(op->graph_launches);
        op->d_colmax_ready = op->graph_colmax_out;
        op->bcg_its += 1;
        return COARSE_OK;
    }
    if (op->bcg_its < 1) return bcg_step(op, stream);          // (the first iteration of a solve runs the column-maxima pre-pass itself)
    // capturing and instantiating costs ~0.15 ms: only once the same block and width have run a few iterations without a graph
    if (op->graph_cand_X != op->bcg_X || op->graph_cand_s != op->bcg_s) { op->graph_cand_X = op->bcg_X; op->graph_cand_s = op->bcg_s; op->graph_seen = 0; }
    if (++op->graph_seen <= 5) return bcg_step(op, stream);
    if (!op->graph_stream && cudaStreamCreate(&op->graph_stream) != cudaSuccess) { op->graph_off = true; cudaGetLastError(); return bcg_step(op, stream); }
    cudaStream_t gs = stream ? stream : op->graph_stream;
    const bool colmax_in = op->d_colmax_ready;
    const int its0 = op->bcg_its;
    const int64_t l0 = g_launches.load();
    if (cudaStreamBeginCapture(gs, cudaStreamCaptureModeRelaxed) != cudaSuccess) { op->graph_off = true; cudaGetLastError(); return bcg_step(op, stream); }
    const int st = bcg_step(op, gs);
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(gs, &graph);
    const int launches = (int)(g_launches.load() - l0);
    g_launches.fetch_sub(launches);                             // (counted when the graph is launched)
    op->bcg_its = its0;
    if (st != COARSE_OK || ce != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        op->graph_off = true;
        op->d_colmax_ready = colmax_in;
        return bcg_step(op, stream);
    }
    if (op->step_graph) { cudaGraphExecDestroy(op->step_graph); op->step_graph = nullptr; }
    const cudaError_t ie = cudaGraphInstantiate(&op->step_graph, graph, 0);
    cudaGraphDestroy(graph);
    if (ie != cudaSuccess) { cudaGetLastError(); op->step_graph = nullptr; op->graph_off = true; op->d_colmax_ready = colmax_in; return bcg_step(op, stream); }
    op->graph_X = op->bcg_X;
    op->graph_s = op->bcg_s;
    op->graph_colmax_in = colmax_in;
    op->graph_colmax_out = op->d_colmax_ready;
    op->graph_launches = launches;
    op->d_colmax_ready = colmax_in;
    return bcg_step_fast(op, stream);                           // now replays it
}

// true residual from one extra apply; fills res (iterations, residuals); synchronises
static int bcg_end(coarse_op *op, block_cg_result *res, cudaStream_t stream)
{
    const int s = op->bcg_s;
    const int64_t n = op->dims.V * op->nb, total = n * s;
    void *Z = op->blk[2], *T = op->blk[3];
    BcgSmall w = small_view(op);
    CMRHS_STEP(apply_impl(op, op->bcg_X, Z, s, stream));
    CMRHS_STEP(axpby_dispatch(op, op->bcg_B, Z, T, 1.0, -1.0, total, stream));
    CMRHS_STEP(gram_dispatch(op, T, T, w.G, n, s, stream));
    bcg_truerel_kernel<<<1, 64, 0, stream>>>(w, s, op->dscal + 130);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(fetch_scalars(op, stream));
    for (int r = 0; r < s; ++r) {
        res->rel_res_recursive[r] = op->hpin[r];
        res->rel_res_true[r] = op->hpin[66 + r];
    }
    res->iterations = op->bcg_its;
    op->bcg_active = false;
    return COARSE_OK;
}

// X_host_out (optional): the solution is final when the loop ends, so its copy to the host is started then, on the handle's
// copy stream, and overlaps the extra apply that evaluates the true residual
static int block_cg_impl(coarse_op *op, const void *B, void *X, int s, double tol, int maxiter, block_cg_result *res,
                         cudaStream_t stream, bool zero_guess = false, void *X_host_out = nullptr)
{
    const double *h_stop = op->hpin + 64;
    memset(res, 0, sizeof(*res));
    for (int k = 0; k < COARSE_MAX_HISTORY; ++k) res->history[k] = -1.0;
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    const auto t0 = std::chrono::steady_clock::now();
    int status = bcg_begin(op, B, X, s, tol, stream, zero_guess);
    if (status != COARSE_OK && status != COARSE_NOT_CONVERGED && status != COARSE_BREAKDOWN) return status;
    res->history[0] = h_stop[0];
    if (status == COARSE_NOT_CONVERGED) {
        for (int k = 0; k < maxiter; ++k) {
            CMRHS_STEP(bcg_step_fast(op, stream));
            CMRHS_STEP(fetch_scalars(op, stream));                                         // stop scalar -> host
            if (h_stop[1] != 0.0) {
                // D^H Z failed (statement 9): the iteration did nothing (the s x s kernels froze X, blockcg_kernels.cuh): it does not count
                if (h_stop[1] == 2.0) op->bcg_its -= 1;
                status = COARSE_BREAKDOWN;
                break;
            }
            if (op->bcg_its < COARSE_MAX_HISTORY) res->history[op->bcg_its] = h_stop[0];
            if (h_stop[0] <= tol) { status = COARSE_OK; break; }
        }
    }
    if (X_host_out) {
        if (!op->copy_stream) {
            CMRHS_CUDA(cudaStreamCreateWithFlags(&op->copy_stream, cudaStreamNonBlocking));
            CMRHS_CUDA(cudaEventCreateWithFlags(&op->copy_event, cudaEventDisableTiming));
        }
        CMRHS_CUDA(cudaEventRecord(op->copy_event, stream));
        CMRHS_CUDA(cudaStreamWaitEvent(op->copy_stream, op->copy_event, 0));
        CMRHS_CUDA(cudaMemcpyAsync(X_host_out, X, (size_t)op->dims.V * op->nb * s * op->esize, cudaMemcpyDeviceToHost, op->copy_stream));
    }
    CMRHS_STEP(bcg_end(op, res, stream));                                                  // reads X only
    if (X_host_out) CMRHS_CUDA(cudaStreamSynchronize(op->copy_stream));
    res->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    res->status = status;
    return status;
}

static int check_solve_args(const coarse_op *op, const void *B, const void *X, int nrhs, double tol, int maxiter,
                            const block_cg_result *res, bool device_ptrs = true)
{
    if (!op || !B || !X || !res) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (nrhs < 1 || nrhs > op->nrhs_max) { set_error("nrhs %d outside 1..nrhs_max=%d", nrhs, op->nrhs_max); return COARSE_INVALID_ARG; }
    if (!(tol > 0.0) || maxiter < 0) { set_error("tol must be > 0 and maxiter >= 0"); return COARSE_INVALID_ARG; }
    if (B == X) { set_error("X must not alias B"); return COARSE_INVALID_ARG; }
    if (device_ptrs && (misaligned16(B) || misaligned16(X))) { set_error("B and X must be 16-byte aligned"); return COARSE_INVALID_ARG; }
    if (op->bcg_active) { set_error("a block_cg_begin/step/end solve is active on this handle"); return COARSE_INVALID_ARG; }
    return check_device(op);
}

extern "C" int block_cg_solve(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter,
                              block_cg_result *res, void *stream)
{
    int st = check_solve_args(op, B_dev, X_dev, nrhs, tol, maxiter, res);
    if (st != COARSE_OK) return st;
    return block_cg_impl(op, B_dev, X_dev, nrhs, tol, maxiter, res, (cudaStream_t)stream);
}

extern "C" int block_cg_solve_host_ex(coarse_op_t *op, const void *B_host, void *X_host, int32_t nrhs, double tol, int32_t maxiter,
                                      uint32_t flags, block_cg_result *res, void *stream_v)
{
    int st = check_solve_args(op, B_host, X_host, nrhs, tol, maxiter, res, false);
    if (st != COARSE_OK) return st;
    if (flags & ~(uint32_t)COARSE_SOLVE_ZERO_GUESS) { set_error("unknown solve flags 0x%x", flags); return COARSE_INVALID_ARG; }
    const bool zero = (flags & COARSE_SOLVE_ZERO_GUESS) != 0;
    cudaStream_t stream = (cudaStream_t)stream_v;
    const size_t bytes = (size_t)op->dims.V * op->nb * nrhs * op->esize;
    CMRHS_CUDA(cudaMemcpyAsync(op->blk[4], B_host, bytes, cudaMemcpyHostToDevice, stream));
    if (!zero) CMRHS_CUDA(cudaMemcpyAsync(op->blk[5], X_host, bytes, cudaMemcpyHostToDevice, stream));
    st = block_cg_impl(op, op->blk[4], op->blk[5], nrhs, tol, maxiter, res, stream, zero, X_host);      // copies X back itself
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    return st;
}

extern "C" int block_cg_solve_host(coarse_op_t *op, const void *B_host, void *X_host, int32_t nrhs, double tol,
                                   int32_t maxiter, block_cg_result *res, void *stream)
{
    return block_cg_solve_host_ex(op, B_host, X_host, nrhs, tol, maxiter, 0u, res, stream);
}

extern "C" int block_cg_solve_ex(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter, uint32_t flags,
                                 block_cg_result *res, void *stream)
{
    int st = check_solve_args(op, B_dev, X_dev, nrhs, tol, maxiter, res);
    if (st != COARSE_OK) return st;
    if (flags & ~(uint32_t)COARSE_SOLVE_ZERO_GUESS) { set_error("unknown solve flags 0x%x", flags); return COARSE_INVALID_ARG; }
    return block_cg_impl(op, B_dev, X_dev, nrhs, tol, maxiter, res, (cudaStream_t)stream, (flags & COARSE_SOLVE_ZERO_GUESS) != 0);
}

// ---- synthetic inputs (bench convenience) --------------------------------
template <typename T>
static int fill_synthetic_impl(void *A_dev, const LatticeDims &d, int nb, uint64_t seed, double c_factor, double *c_out,
                               cudaStream_t stream)
{
    const int64_t total = d.V * kNPoint * nb * nb;
    const int grid = (int)(ceil_div(total, 256) < 148 * 32 ? ceil_div(total, 256) : 148 * 32);
    synth_fill_kernel<T><<<grid, 256, 0, stream>>>((cplx<T> *)A_dev, d, nb, synth_key(seed, SYNTH_TAG_A), synth_key(seed, SYNTH_TAG_G));
    CMRHS_LAUNCH_CHECK();
    double c = 0.0;
    if (c_factor != 0.0) {
        double *bound = nullptr;
        CMRHS_CUDA(cudaMalloc((void **)&bound, (size_t)(d.V + 1) * sizeof(double)));
        const int bgrid = (int)(ceil_div(d.V * 32, 256) < 148 * 16 ? ceil_div(d.V * 32, 256) : 148 * 16);
        synth_bound_kernel<T><<<bgrid, 256, 0, stream>>>((const cplx<T> *)A_dev, d.V, nb, bound);
        count_launch();
        max_reduce_kernel<<<1, 256, 0, stream>>>(bound, d.V, bound + d.V);
        count_launch();
        double best = 0.0;
        cudaError_t e = cudaMemcpyAsync(&best, bound + d.V, sizeof(double), cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        cudaFree(bound);
        if (e != cudaSuccess) { set_error("synthetic bound pass failed: %s", cudaGetErrorString(e)); return COARSE_CUDA_ERROR; }
        c = (double)(float)(c_factor * best);
        const int sgrid = (int)ceil_div(d.V * nb, 256);
        synth_shift_kernel<T><<<sgrid, 256, 0, stream>>>((cplx<T> *)A_dev, d.V, nb, (float)c);
        CMRHS_LAUNCH_CHECK();
    }
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    if (c_out) *c_out = c;
    return COARSE_OK;
}

extern "C" int coarse_op_fill_synthetic(void *A_dev, const int32_t dims[4], int32_t nbasis, int32_t dtype, uint64_t seed,
                                        double c_factor, double *c_out, void *stream)
{
    int st = check_shape(dims, nbasis, 1, dtype);
    if (st != COARSE_OK) return st;
    if (!A_dev) { set_error("A_dev is NULL"); return COARSE_INVALID_ARG; }
    LatticeDims d;
    for (int k = 0; k < 4; ++k) d.L[k] = dims[k];
    d.V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    return dtype == COARSE_C64 ? fill_synthetic_impl<float>(A_dev, d, nbasis, seed, c_factor, c_out, (cudaStream_t)stream)
                               : fill_synthetic_impl<double>(A_dev, d, nbasis, seed, c_factor, c_out, (cudaStream_t)stream);
}

extern "C" int coarse_fill_block(void *X_dev, const int32_t dims[4], int32_t nbasis, int32_t nrhs, int32_t dtype, uint64_t seed,
                                 int32_t tag, void *stream_v)
{
    int st = check_shape(dims, nbasis, nrhs, dtype);
    if (st != COARSE_OK) return st;
    if (!X_dev) { set_error("X_dev is NULL"); return COARSE_INVALID_ARG; }
    cudaStream_t stream = (cudaStream_t)stream_v;
    const int64_t total = (int64_t)dims[0] * dims[1] * dims[2] * dims[3] * nbasis * nrhs;
    const int grid = (int)(ceil_div(total, 256) < 148 * 32 ? ceil_div(total, 256) : 148 * 32);
    const uint64_t key = synth_key(seed, (uint64_t)tag);
    if (dtype == COARSE_C64) synth_block_kernel<float><<<grid, 256, 0, stream>>>((cplx<float> *)X_dev, total, key);
    else synth_block_kernel<double><<<grid, 256, 0, stream>>>((cplx<double> *)X_dev, total, key);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

extern "C" int block_cg_begin(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, double *rel_res0,
                              void *stream)
{
    block_cg_result dummy;
    if (op) op->bcg_active = false;                      // a new begin abandons an unfinished begin/step/end solve
    int st = check_solve_args(op, B_dev, X_dev, nrhs, tol, 0, &dummy);
    if (st != COARSE_OK) return st;
    st = bcg_begin(op, B_dev, X_dev, nrhs, tol, (cudaStream_t)stream);
    if (rel_res0 && (st == COARSE_OK || st == COARSE_NOT_CONVERGED)) *rel_res0 = op->hpin[64];
    return st;
}

extern "C" int block_cg_step(coarse_op_t *op, int32_t count, void *stream)
{
    if (!op || count < 0) { set_error("bad argument"); return COARSE_INVALID_ARG; }
    if (!op->bcg_active) { set_error("block_cg_step without an active block_cg_begin"); return COARSE_INVALID_ARG; }
    for (int k = 0; k < count; ++k) CMRHS_STEP(bcg_step_fast(op, (cudaStream_t)stream));
    return COARSE_OK;
}

extern "C" int block_cg_end(coarse_op_t *op, block_cg_result *res, void *stream)
{
    if (!op || !res) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (!op->bcg_B) { set_error("block_cg_end without block_cg_begin"); return COARSE_INVALID_ARG; }
    memset(res, 0, sizeof(*res));
    for (int k = 0; k < COARSE_MAX_HISTORY; ++k) res->history[k] = -1.0;
    CMRHS_STEP(bcg_end(op, res, (cudaStream_t)stream));
    double worst = 0.0;
    for (int r = 0; r < op->bcg_s; ++r) worst = worst > res->rel_res_recursive[r] ? worst : res->rel_res_recursive[r];
    if (op->bcg_its < COARSE_MAX_HISTORY) res->history[op->bcg_its] = worst;
    res->status = op->hpin[65] != 0.0 ? COARSE_BREAKDOWN : COARSE_OK;
    return res->status;
}

// ---- per-launch timing of the stencil kernel, for bench.py's roofline object --------------------------------
// ---- Chebyshev polynomial coarse solve ------------------------------------------------
static int cheby_check(const coarse_op *op, const void *B_dev, const void *X_dev, int nrhs, double lo, double hi, int order)
{
    if (!op || !B_dev || !X_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (B_dev == X_dev) { set_error("X must not alias B"); return COARSE_INVALID_ARG; }
    if (nrhs < 1 || nrhs > op->nrhs_max) { set_error("nrhs %d outside 1..%d", nrhs, op->nrhs_max); return COARSE_INVALID_ARG; }
    if (!(lo > 0.0) || !(hi > lo) || order < 1 || order > 100000) { set_error("need 0 < lo < hi and 1 <= order <= 100000"); return COARSE_INVALID_ARG; }
    if (op->bcg_active) { set_error("polynomial solve inside an active block_cg_begin/end solve"); return COARSE_INVALID_ARG; }
    return COARSE_OK;
}

// X = (accumulate ? X : 0) + P(H) B
static int cheby_impl(coarse_op *op, const void *B_dev, void *X_dev, int nrhs, double lo, double hi, int order, bool accumulate,
                      cudaStream_t stream)
{
    // c_j = (2/n) sum_k f(x_k) cos(pi j (k + 1/2) / n), f = 1/x at the first-kind Chebyshev points of [lo, hi]
    const int n = order;
    std::vector<double> c((size_t)n), fk((size_t)n);
    const double PI = 3.14159265358979323846;
    for (int k = 0; k < n; ++k) fk[(size_t)k] = 1.0 / (0.5 * (hi + lo) + 0.5 * (hi - lo) * cos(PI * (k + 0.5) / n));
    for (int j = 0; j < n; ++j) {
        double acc = 0.0;
        for (int k = 0; k < n; ++k) acc += fk[(size_t)k] * cos(PI * j * (k + 0.5) / n);
        c[(size_t)j] = 2.0 * acc / n;
    }
    const double alpha = 2.0 / (hi - lo), beta = -(hi + lo) / (hi - lo);      // y(H) = alpha H + beta
    const int64_t total = op->dims.V * op->nb * (int64_t)nrhs;
    const size_t blk_bytes = (size_t)total * op->esize;
    void *Z = op->blk[2], *Ta = op->blk[0], *Tb = op->blk[1];
    const int64_t cvec = ceil_div(total, (int64_t)(32 / op->esize) * 256);
    const int grid = (int)(cvec < (int64_t)op->num_sms * 8 ? (cvec < 1 ? 1 : cvec) : (int64_t)op->num_sms * 8);
    // the split-FP16 apply scales every column of its input by a power of two: the step that writes T_{j+1} also finds its column maxima
    uint32_t *colmax = (op->dtype == COARSE_C64 && use_split16(op, nrhs)) ? op->amax : nullptr;
    auto step = [&](const void *z, const void *tc, void *tp, double ca, double cb, double cp, double cx, double cn) -> int {
        if (colmax) CMRHS_CUDA(cudaMemsetAsync(colmax, 0, 64 * sizeof(uint32_t), stream));
        if (op->dtype == COARSE_C64)
            cheby_step_kernel<float><<<grid, 256, 0, stream>>>((const cplx<float> *)z, (const cplx<float> *)tc, (cplx<float> *)tp,
                                                               (cplx<float> *)X_dev, (float)ca, (float)cb, (float)cp, (float)cx, (float)cn, total, nrhs, colmax);
        else
            cheby_step_kernel<double><<<grid, 256, 0, stream>>>((const cplx<double> *)z, (const cplx<double> *)tc, (cplx<double> *)tp,
                                                                (cplx<double> *)X_dev, ca, cb, cp, cx, cn, total, nrhs, nullptr);
        CMRHS_LAUNCH_CHECK();
        return COARSE_OK;
    };
    const void *x_in = accumulate ? X_dev : B_dev;                  // (with b = 0 the second operand is only read)
    const double keep = accumulate ? 1.0 : 0.0;
    if (n == 1) return axpby_dispatch(op, B_dev, x_in, X_dev, 0.5 * c[0], keep, total, stream);          // X = (c_0 / 2) B [+ X]
    // T_0 = B ;  T_1 = y(H) B -> Ta ;  X = (c_0/2) T_0 + c_1 T_1 [+ X]
    CMRHS_STEP(apply_impl(op, B_dev, Z, nrhs, stream));
    CMRHS_STEP(axpby_dispatch(op, B_dev, x_in, X_dev, 0.5 * c[0], keep, total, stream));
    CMRHS_STEP(step(Z, B_dev, Ta, alpha, beta, 0.0, 1.0, c[1]));
    if (n == 2) return COARSE_OK;
    CMRHS_CUDA(cudaMemcpyAsync(Tb, B_dev, blk_bytes, cudaMemcpyDeviceToDevice, stream));               // T_prev = T_0
    void *tc = Ta, *tp = Tb;
    for (int j = 1; j < n - 1; ++j) {
        CMRHS_STEP(apply_impl(op, tc, Z, nrhs, stream, colmax != nullptr));                            // Z = H T_j (column maxima of T_j: from the step that wrote it)
        CMRHS_STEP(step(Z, tc, tp, 2.0 * alpha, 2.0 * beta, 1.0, 1.0, c[(size_t)j + 1]));              // T_{j+1} -> tp ; X += c_{j+1} T_{j+1}
        void *t = tc; tc = tp; tp = t;
    }
    return COARSE_OK;
}

extern "C" int coarse_cheby_apply(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double lo, double hi, int32_t order,
                                  void *stream)
{
    CMRHS_STEP(cheby_check(op, B_dev, X_dev, nrhs, lo, hi, order));
    return cheby_impl(op, B_dev, X_dev, nrhs, lo, hi, order, false, (cudaStream_t)stream);
}

// ---- multi-RHS deflation and the composite Defl + Cheby coarse solve (Eq. 7-12) ------------------
static int deflate_check(const coarse_op *op, const void *Vev, const double *lambda, int nev, int nrhs)
{
    if (!Vev || !lambda) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (nev < 1 || nev > COARSE_MAX_NEV) { set_error("nev %d outside 1..%d", nev, COARSE_MAX_NEV); return COARSE_INVALID_ARG; }
    if (nrhs < 1 || nrhs > op->nrhs_max) { set_error("nrhs %d outside 1..%d", nrhs, op->nrhs_max); return COARSE_INVALID_ARG; }
    for (int i = 0; i < nev; ++i)
        if (!(lambda[i] > 0.0)) { set_error("lambda[%d] is not positive", i); return COARSE_INVALID_ARG; }
    return COARSE_OK;
}

template <typename T>
static int deflate_impl(coarse_op *op, const void *Vev, const double *lambda, int nev, const void *B, void *QBpar, void *Bperp, int s,
                        cudaStream_t stream)
{
    // The eigenvectors are taken in chunks of m <= 64 columns (the paper deflates with several hundred): chunk j
    // projects the running b_perp (orthonormal vectors: <i|b_perp> = <i|b> for the vectors still to come), so one pass over a chunk
    // and the block per stage, and b_perp may alias B.  Every chunk costs five passes over the block: wide chunks whatever nrhs_max is
    // (chunks of nrhs_max = 16 vectors: 9.5 ms at nev 192; the scratch for 64 x nrhs_max coefficients comes with the first call).
    const int64_t n = op->dims.V * op->nb;
    const int mc = COARSE_MAX_NRHS;
    if (!op->defl_partial) {
        CMRHS_STEP(alloc_dev(op, (void **)&op->defl_partial, (size_t)op->gram_blocks * mc * op->nrhs_max * sizeof(zdouble)));
        CMRHS_STEP(alloc_dev(op, (void **)&op->defl_C, (size_t)mc * op->nrhs_max * sizeof(zdouble)));
    }
    zdouble *Cm = op->defl_C;                           // m x s <= 64 x nrhs_max complex128
    for (int j0 = 0; j0 < nev; j0 += mc) {
        const int m = nev - j0 < mc ? nev - j0 : mc;
        const cplx<T> *Vj = (const cplx<T> *)Vev + j0;
        const cplx<T> *Bin = j0 == 0 ? (const cplx<T> *)B : (const cplx<T> *)Bperp;
        // stage 1: C = V_j^H b_perp
        int rows = (int)(32768 / ((size_t)(m + s) * sizeof(cplx<T>)));
        if (rows < 1) rows = 1;
        int blocks = op->gram_blocks;
        if ((int64_t)blocks > ceil_div(n, rows)) blocks = (int)ceil_div(n, rows);
        size_t smem1 = (size_t)rows * (m + s) * sizeof(cplx<T>);
        // register-tiled kernels: m and s multiples of 4, rows of the eigenvector block 16-byte aligned
        const bool tiled = m % 4 == 0 && s % 4 == 0 && (m / 4) * (s / 4) <= kLaThreads && (sizeof(T) == 8 || nev % 2 == 0);
        if (tiled) {
            if ((m / 4) * (s / 4) * 2 <= kLaThreads && smem1 < (size_t)m * s * sizeof(zdouble)) smem1 = (size_t)m * s * sizeof(zdouble);   // (several row groups: <= 32 KB)
            rgram_tiled_kernel<T><<<blocks, kLaThreads, smem1, stream>>>(Vj, nev, Bin, n, m, s, rows, op->defl_partial);
        } else {
            rgram_partial_kernel<T><<<blocks, kLaThreads, smem1, stream>>>(Vj, nev, Bin, n, m, s, rows, op->defl_partial);
        }
        CMRHS_LAUNCH_CHECK();
        gram_reduce_kernel<<<(m * s * 32 + 127) / 128, 128, 0, stream>>>(op->defl_partial, blocks, m * s, Cm);
        CMRHS_LAUNCH_CHECK();
        // stage 2: Qb_par (+)= V_j (C / lambda), b_perp -= V_j C
        DeflLambda lam;
        for (int i = 0; i < COARSE_MAX_NRHS; ++i) lam.inv[i] = i < m ? 1.0 / lambda[j0 + i] : 0.0;
        if (tiled && s / 4 <= 16) {
            int RL = kLaThreads / (s / 4);
            if (RL > 64) RL = 64;
            const int TR = (s >= 32 && sizeof(T) == 4) ? 4 : 2;              // wide blocks have few row lanes: more rows per thread
            const size_t smem2 = ((size_t)2 * m * s + (size_t)RL * TR * (m + LaPad<T>::v)) * sizeof(cplx<T>);
            const int64_t ntiles = ceil_div(n, (int64_t)RL * TR);
            const int grid = (int)(ntiles < (int64_t)op->num_sms * 4 ? ntiles : (int64_t)op->num_sms * 4);
            if (TR == 4) {
                auto kern = deflate_update_tiled_kernel<T, 4>;
                CMRHS_SMEM_ATTR(kern, smem2);
                kern<<<grid, kLaThreads, smem2, stream>>>(Vj, nev, Bin, Cm, lam, (cplx<T> *)QBpar, (cplx<T> *)Bperp, n, m, s, RL, j0 > 0 ? 1 : 0);
            } else {
                auto kern = deflate_update_tiled_kernel<T, 2>;
                CMRHS_SMEM_ATTR(kern, smem2);
                kern<<<grid, kLaThreads, smem2, stream>>>(Vj, nev, Bin, Cm, lam, (cplx<T> *)QBpar, (cplx<T> *)Bperp, n, m, s, RL, j0 > 0 ? 1 : 0);
            }
        } else {
            const int rows2 = 64;
            const size_t smem2 = ((size_t)2 * m * s + (size_t)rows2 * m) * sizeof(cplx<T>);
            auto kern = deflate_update_kernel<T>;
            CMRHS_SMEM_ATTR(kern, smem2);
            const int64_t ntiles = ceil_div(n, rows2);
            const int grid = (int)(ntiles < (int64_t)op->num_sms * 4 ? ntiles : (int64_t)op->num_sms * 4);
            kern<<<grid, kLaThreads, smem2, stream>>>(Vj, nev, Bin, Cm, lam, (cplx<T> *)QBpar, (cplx<T> *)Bperp, n, m, s, rows2, j0 > 0 ? 1 : 0);
        }
        CMRHS_LAUNCH_CHECK();
    }
    return COARSE_OK;
}

extern "C" int coarse_deflate(coarse_op_t *op, const void *Vev_dev, const double *lambda_host, int32_t nev, const void *B_dev,
                              void *QBpar_dev, void *Bperp_dev, int32_t nrhs, void *stream)
{
    if (!op || !B_dev || !QBpar_dev || !Bperp_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (B_dev == QBpar_dev || QBpar_dev == Bperp_dev) { set_error("outputs must not alias each other or B's first output"); return COARSE_INVALID_ARG; }
    CMRHS_STEP(deflate_check(op, Vev_dev, lambda_host, nev, nrhs));
    if (op->bcg_active) { set_error("coarse_deflate inside an active block_cg_begin/end solve"); return COARSE_INVALID_ARG; }
    return op->dtype == COARSE_C64 ? deflate_impl<float>(op, Vev_dev, lambda_host, nev, B_dev, QBpar_dev, Bperp_dev, nrhs, (cudaStream_t)stream)
                                   : deflate_impl<double>(op, Vev_dev, lambda_host, nev, B_dev, QBpar_dev, Bperp_dev, nrhs, (cudaStream_t)stream);
}

// X = Defl(b_par) + P(H) b_perp  (Eq. 12); b_perp goes through workspace block 3
static int cheby_defl_impl(coarse_op *op, const void *Vev_dev, const double *lambda_host, int nev, const void *B_dev, void *X_dev, int nrhs,
                           double lo, double hi, int order, cudaStream_t stream)
{
    void *Bperp = op->blk[3];
    if (op->dtype == COARSE_C64) CMRHS_STEP(deflate_impl<float>(op, Vev_dev, lambda_host, nev, B_dev, X_dev, Bperp, nrhs, stream));
    else CMRHS_STEP(deflate_impl<double>(op, Vev_dev, lambda_host, nev, B_dev, X_dev, Bperp, nrhs, stream));
    return cheby_impl(op, Bperp, X_dev, nrhs, lo, hi, order, true, stream);
}

extern "C" int coarse_cheby_defl_solve(coarse_op_t *op, const void *Vev_dev, const double *lambda_host, int32_t nev, const void *B_dev,
                                       void *X_dev, int32_t nrhs, double lo, double hi, int32_t order, void *stream)
{
    CMRHS_STEP(cheby_check(op, B_dev, X_dev, nrhs, lo, hi, order));
    CMRHS_STEP(deflate_check(op, Vev_dev, lambda_host, nev, nrhs));
    return cheby_defl_impl(op, Vev_dev, lambda_host, nev, B_dev, X_dev, nrhs, lo, hi, order, (cudaStream_t)stream);
}

// ---- Preconditioned BlockCGrQ (Fig. 2 right) with a stationary preconditioner -----------------
static int precond_apply(coarse_op *op, const coarse_precond *M, const void *z, void *Z, int s, cudaStream_t stream)
{
    if (M->kind == COARSE_PRECOND_CHEBY) return cheby_impl(op, z, Z, s, M->lo, M->hi, M->order, false, stream);
    return cheby_defl_impl(op, M->Vev_dev, M->lambda_host, M->nev, z, Z, s, M->lo, M->hi, M->order, stream);
}

extern "C" int pblock_cg_solve(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter,
                               const coarse_precond *M, block_cg_result *res, void *stream_v)
{
    if (!op || !B_dev || !X_dev || !M || !res) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (B_dev == X_dev) { set_error("X must not alias B"); return COARSE_INVALID_ARG; }
    if (nrhs < 1 || nrhs > op->nrhs_max) { set_error("nrhs %d outside 1..%d", nrhs, op->nrhs_max); return COARSE_INVALID_ARG; }
    if (!(tol >= 0.0) || maxiter < 0) { set_error("bad tol / maxiter"); return COARSE_INVALID_ARG; }
    if (M->kind != COARSE_PRECOND_CHEBY && M->kind != COARSE_PRECOND_DEFL_CHEBY) { set_error("unknown preconditioner kind %d", M->kind); return COARSE_INVALID_ARG; }
    if (!(M->lo > 0.0) || !(M->hi > M->lo) || M->order < 1 || M->order > 100000) { set_error("preconditioner: need 0 < lo < hi and 1 <= order <= 100000"); return COARSE_INVALID_ARG; }
    if (M->kind == COARSE_PRECOND_DEFL_CHEBY) CMRHS_STEP(deflate_check(op, M->Vev_dev, M->lambda_host, M->nev, nrhs));
    if (op->bcg_active) { set_error("pblock_cg_solve inside an active block_cg_begin/end solve"); return COARSE_INVALID_ARG; }
    cudaStream_t stream = (cudaStream_t)stream_v;
    const int s = nrhs;
    const int64_t n = op->dims.V * op->nb, total = n * s;
    const size_t blk_bytes_max = (size_t)n * op->nrhs_max * op->esize;
    for (int b = 0; b < 5; ++b)                     // q, Q, D, z, Z: allocated on first use (blocks 0-3 belong to the preconditioner)
        if (!op->pblk[b]) CMRHS_STEP(alloc_dev(op, &op->pblk[b], blk_bytes_max));
    void *q = op->pblk[0], *Q = op->pblk[1], *D = op->pblk[2], *z = op->pblk[3], *Z = op->pblk[4];
    BcgSmall w = small_view(op);
    const double *h_stop = op->hpin + 64;
    memset(res, 0, sizeof(*res));
    for (int k = 0; k < COARSE_MAX_HISTORY; ++k) res->history[k] = -1.0;
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    const auto t0 = std::chrono::steady_clock::now();
    auto small3 = [&](void (*kern)(BcgSmall, int)) -> int { return small_launch(kern, op, s, 3, stream); };
    // ||B[:,r]|| ;  z_0 = B - H X_0 ;  relative residual of the start
    CMRHS_STEP(gram_dispatch(op, B_dev, B_dev, w.G, n, s, stream));
    bcg_bnorm_kernel<<<1, 64, 0, stream>>>(w, s);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(apply_impl(op, X_dev, Z, s, stream));
    CMRHS_STEP(axpby_dispatch(op, B_dev, Z, z, 1.0, -1.0, total, stream));
    CMRHS_STEP(gram_dispatch(op, z, z, w.G, n, s, stream));
    pbcg_rel0_kernel<<<1, 32, 0, stream>>>(w, s);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(fetch_scalars(op, stream));
    res->history[0] = h_stop[0];
    int status = COARSE_NOT_CONVERGED, its = 0;
    if (h_stop[0] <= tol) status = COARSE_OK;
    else {
        // Z_0 = M^-1 z_0 ;  C_0^H C_0 = Z_0^H z_0 ;  q_0 = z_0 C_0^-1 ;  Q_0 = Z_0 C_0^-1 ;  D_0 = Q_0
        CMRHS_STEP(precond_apply(op, M, z, Z, s, stream));
        CMRHS_STEP(gram_dispatch(op, Z, z, w.G, n, s, stream));
        CMRHS_STEP(small3(pbcg_init_kernel));
        CMRHS_STEP(rotate_dispatch(op, z, w.K1, nullptr, q, 0.0, n, s, stream));
        CMRHS_STEP(rotate_dispatch(op, Z, w.K1, nullptr, Q, 0.0, n, s, stream));
        CMRHS_CUDA(cudaMemcpyAsync(D, Q, (size_t)total * op->esize, cudaMemcpyDeviceToDevice, stream));
        for (int k = 0; k < maxiter; ++k) {
            CMRHS_STEP(apply_impl(op, D, z, s, stream));                                   // z_k = H D_k
            CMRHS_STEP(precond_apply(op, M, z, Z, s, stream));                             // Z_k = M^-1 z_k
            CMRHS_STEP(gram_dispatch(op, D, z, w.G, n, s, stream));                        // D^H z
            CMRHS_STEP(small3(bcg_step1_kernel));                                          // N ; K1 = N C ; K2 = -N
            CMRHS_STEP(rotate_dispatch(op, D, w.K1, X_dev, X_dev, 1.0, n, s, stream));     // X += D N C
            CMRHS_STEP(rotate_dispatch(op, z, w.K2, q, q, 1.0, n, s, stream));             // t = q - z N   (in place)
            CMRHS_STEP(rotate_dispatch(op, Z, w.K2, Q, Q, 1.0, n, s, stream));             // T = Q - Z N   (in place)
            // stop test first: the residual of X_{k+1} is r_{k+1} = q_{k+1} C_{k+1} = t_k C_k, so it is available before the
            // factorisation (near convergence T^H t is dominated by rounding and need not be positive definite any more)
            CMRHS_STEP(gram_dispatch(op, q, q, w.G, n, s, stream));                        // t^H t -> ||t C_k|| column norms
            CMRHS_STEP(small3(pbcg_resid_kernel));
            CMRHS_STEP(fetch_scalars(op, stream));
            its = k + 1;
            if (h_stop[1] != 0.0) { status = COARSE_BREAKDOWN; break; }
            if (its < COARSE_MAX_HISTORY) res->history[its] = h_stop[0];
            for (int r = 0; r < s; ++r) res->rel_res_recursive[r] = op->hpin[r];
            if (h_stop[0] <= tol) { status = COARSE_OK; break; }
            if (its == maxiter) break;
            CMRHS_STEP(gram_dispatch(op, Q, q, w.G, n, s, stream));                        // T^H t = <T|T>_M
            CMRHS_STEP(small3(bcg_step2_kernel));                                          // S ; K3 = S^-1 ; K4 = S^H ; C = S C
            CMRHS_STEP(rotate_dispatch(op, q, w.K3, nullptr, q, 0.0, n, s, stream));       // q = t S^-1    (in place)
            CMRHS_STEP(rotate_dispatch(op, Q, w.K3, nullptr, Q, 0.0, n, s, stream));       // Q = T S^-1    (in place)
            CMRHS_STEP(rotate_dispatch(op, D, w.K4, Q, D, 1.0, n, s, stream));             // D = Q + D S^H
        }
        if (status == COARSE_NOT_CONVERGED || status == COARSE_OK) {                       // a breakdown inside step1 / step2 shows up here
            CMRHS_STEP(fetch_scalars(op, stream));
            if (h_stop[1] != 0.0) status = COARSE_BREAKDOWN;
        }
    }
    if (its == 0) for (int r = 0; r < s; ++r) res->rel_res_recursive[r] = op->hpin[r];
    // true residual from one extra apply
    CMRHS_STEP(apply_impl(op, X_dev, Z, s, stream));
    CMRHS_STEP(axpby_dispatch(op, B_dev, Z, z, 1.0, -1.0, total, stream));
    CMRHS_STEP(gram_dispatch(op, z, z, w.G, n, s, stream));
    bcg_truerel_kernel<<<1, 64, 0, stream>>>(w, s, op->dscal + 130);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(fetch_scalars(op, stream));
    for (int r = 0; r < s; ++r) res->rel_res_true[r] = op->hpin[66 + r];
    res->iterations = its;
    res->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    res->status = status;
    return status;
}

// ---- stacked single-Krylov CG ---------------------------------------------------------------
template <typename T>
static int stacked_cg_impl(coarse_op *op, const void *B_dev, void *X_dev, int s, double tol, int maxiter, block_cg_result *res, cudaStream_t stream)
{
    const int64_t n = op->dims.V * op->nb, total = n * s;
    cplx<T> *R = (cplx<T> *)op->blk[0], *P = (cplx<T> *)op->blk[1], *Z = (cplx<T> *)op->blk[2];
    const cplx<T> *B = (const cplx<T> *)B_dev;
    cplx<T> *X = (cplx<T> *)X_dev;
    double *partial = reinterpret_cast<double *>(op->gram_partial), *sc = op->dscal + 200;
    const int nblk = op->gram_blocks;
    const int egrid = (int)(ceil_div(total, 256) < (int64_t)op->num_sms * 16 ? ceil_div(total, 256) : (int64_t)op->num_sms * 16);
    BcgSmall w = small_view(op);
    auto fetch_stop = [&](double *out) -> int {
        CMRHS_CUDA(cudaMemcpyAsync(op->hpin + 200, sc, 5 * sizeof(double), cudaMemcpyDeviceToHost, stream));
        CMRHS_CUDA(cudaStreamSynchronize(stream));
        *out = op->hpin[204];
        return COARSE_OK;
    };
    // ||B||_F^2 ;  R = B - H X_0 ;  rho_0
    fdot_partial_kernel<T><<<nblk, kLaThreads, 0, stream>>>(B, B, total, partial);
    CMRHS_LAUNCH_CHECK();
    scg_scalar_kernel<<<1, 32, 0, stream>>>(0, partial, nblk, sc);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(apply_impl(op, X, Z, s, stream));
    CMRHS_STEP(axpby_dispatch(op, B, Z, R, 1.0, -1.0, total, stream));
    fdot_partial_kernel<T><<<nblk, kLaThreads, 0, stream>>>(R, R, total, partial);
    CMRHS_LAUNCH_CHECK();
    scg_scalar_kernel<<<1, 32, 0, stream>>>(1, partial, nblk, sc);
    CMRHS_LAUNCH_CHECK();
    double stop = 0.0;
    CMRHS_STEP(fetch_stop(&stop));
    res->history[0] = stop;
    int status = COARSE_NOT_CONVERGED, its = 0;
    if (stop <= tol) status = COARSE_OK;
    else {
        CMRHS_CUDA(cudaMemcpyAsync(P, R, (size_t)total * sizeof(cplx<T>), cudaMemcpyDeviceToDevice, stream));
        for (int k = 0; k < maxiter; ++k) {
            CMRHS_STEP(apply_impl(op, P, Z, s, stream));                                        // Z = H P
            fdot_partial_kernel<T><<<nblk, kLaThreads, 0, stream>>>(P, Z, total, partial);
            CMRHS_LAUNCH_CHECK();
            scg_scalar_kernel<<<1, 32, 0, stream>>>(2, partial, nblk, sc);                       // alpha
            CMRHS_LAUNCH_CHECK();
            scg_update1_kernel<T><<<nblk, kLaThreads, 0, stream>>>(P, Z, X, R, sc, total, partial);   // X, R, <R, R>
            CMRHS_LAUNCH_CHECK();
            scg_scalar_kernel<<<1, 32, 0, stream>>>(3, partial, nblk, sc);                       // beta, rho, stop
            CMRHS_LAUNCH_CHECK();
            CMRHS_STEP(fetch_stop(&stop));
            its = k + 1;
            if (its < COARSE_MAX_HISTORY) res->history[its] = stop;
            if (!(stop == stop)) { status = COARSE_BREAKDOWN; break; }
            if (stop <= tol) { status = COARSE_OK; break; }
            scg_update2_kernel<T><<<egrid, 256, 0, stream>>>(R, P, sc, total);                   // P = R + beta P
            CMRHS_LAUNCH_CHECK();
        }
    }
    for (int r = 0; r < s; ++r) res->rel_res_recursive[r] = stop;
    // per-column true residuals from one extra apply
    CMRHS_STEP(gram_dispatch(op, B, B, w.G, n, s, stream));
    bcg_bnorm_kernel<<<1, 64, 0, stream>>>(w, s);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(apply_impl(op, X, Z, s, stream));
    CMRHS_STEP(axpby_dispatch(op, B, Z, R, 1.0, -1.0, total, stream));
    CMRHS_STEP(gram_dispatch(op, R, R, w.G, n, s, stream));
    bcg_truerel_kernel<<<1, 64, 0, stream>>>(w, s, op->dscal + 130);
    CMRHS_LAUNCH_CHECK();
    CMRHS_STEP(fetch_scalars(op, stream));
    for (int r = 0; r < s; ++r) res->rel_res_true[r] = op->hpin[66 + r];
    res->iterations = its;
    res->status = status;
    return status;
}

extern "C" int stacked_cg_solve(coarse_op_t *op, const void *B_dev, void *X_dev, int32_t nrhs, double tol, int32_t maxiter,
                                block_cg_result *res, void *stream_v)
{
    if (!op || !B_dev || !X_dev || !res) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (B_dev == X_dev) { set_error("X must not alias B"); return COARSE_INVALID_ARG; }
    if (nrhs < 1 || nrhs > op->nrhs_max) { set_error("nrhs %d outside 1..%d", nrhs, op->nrhs_max); return COARSE_INVALID_ARG; }
    if (!(tol >= 0.0) || maxiter < 0) { set_error("bad tol / maxiter"); return COARSE_INVALID_ARG; }
    if (op->bcg_active) { set_error("stacked_cg_solve inside an active block_cg_begin/end solve"); return COARSE_INVALID_ARG; }
    cudaStream_t stream = (cudaStream_t)stream_v;
    memset(res, 0, sizeof(*res));
    for (int k = 0; k < COARSE_MAX_HISTORY; ++k) res->history[k] = -1.0;
    CMRHS_CUDA(cudaStreamSynchronize(stream));
    const auto t0 = std::chrono::steady_clock::now();
    const int st = op->dtype == COARSE_C64 ? stacked_cg_impl<float>(op, B_dev, X_dev, nrhs, tol, maxiter, res, stream)
                                           : stacked_cg_impl<double>(op, B_dev, X_dev, nrhs, tol, maxiter, res, stream);
    res->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    return st;
}

// ---- multi-RHS block project / promote (Eq. 14-15) -----------------------------------------------------
static int transfer_check(const void *a, const void *b, const void *c, int64_t Vc, int vb, int nb, int s, int dtype)
{
    if (!a || !b || !c) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (dtype != COARSE_C64 && dtype != COARSE_C128) { set_error("dtype must be COARSE_C64 or COARSE_C128"); return COARSE_INVALID_ARG; }
    if (Vc < 1 || vb < 1 || nb < 1 || nb > COARSE_MAX_NBASIS || s < 1 || s > COARSE_MAX_NRHS) { set_error("bad Vc / vblock / nbasis / nrhs"); return COARSE_INVALID_ARG; }
    return COARSE_OK;
}

template <typename T>
static int transfer_launch(bool project, const void *Bas, const void *in, void *out, int64_t Vc, int vb, int nb, int s, cudaStream_t stream)
{
    int dev = 0, sms = 0;
    CMRHS_CUDA(cudaGetDevice(&dev));
    CMRHS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = (int)(Vc < (int64_t)sms * 4 ? Vc : (int64_t)sms * 4);
    const bool tuned = nb % 4 == 0 && s % 4 == 0 && (nb / 4) * (s / 4) <= kXferConsumers;       // 4 x 4 register tiles, 7 consumer warps
    if (project && tuned) {
        // G sites at a time (one group of (nb/4)(s/4) threads each, at most 8), stages of about 24 KB, a site's rows cut into equal tiles
        const int ntile = (nb / 4) * (s / 4);
        int G = kXferConsumers / ntile;
        if (G > 8) G = 8;
        if ((int64_t)G > Vc) G = (int)Vc;
        int rows = (int)(24576 / ((size_t)G * (nb + s) * sizeof(cplx<T>)));
        if (rows < 1) rows = 1;
        if (rows > 32) rows = 32;
        const int tps = (vb + rows - 1) / rows;
        rows = (vb + tps - 1) / tps;
        const int flush = rows >= 32 ? 1 : 32 / rows;                  // runs of <= 32 rows between flushes
        const size_t smem = (size_t)kGramPipeStages * G * rows * (nb + s) * sizeof(cplx<T>) + 2 * kGramPipeStages * sizeof(uint64_t);
        const int64_t nchunk = (Vc + G - 1) / G;
        const int pgrid = (int)(nchunk < (int64_t)sms * 2 ? nchunk : (int64_t)sms * 2);
        auto kern = block_project_pipe_kernel<T>;
        CMRHS_SMEM_ATTR(kern, smem);
        kern<<<pgrid, kLaThreads, smem, stream>>>((const cplx<T> *)Bas, (const cplx<T> *)in, (cplx<T> *)out, Vc, vb, nb, s, rows, G, flush);
    } else if (project) {
        int rows = (int)(32768 / ((size_t)(nb + s) * sizeof(cplx<T>)));
        if (rows > vb) rows = vb;
        if (rows < 1) rows = 1;
        const size_t smem = (size_t)rows * (nb + s) * sizeof(cplx<T>);
        block_project_kernel<T><<<grid, kLaThreads, smem, stream>>>((const cplx<T> *)Bas, (const cplx<T> *)in, (cplx<T> *)out, Vc, vb, nb, s, rows);
    } else if (tuned && s / 4 <= 16) {
        // lanes along the rows: RL row lanes x s/4 column groups; TR = 2 rows per thread; two row tiles and two coarse blocks in shared memory
        constexpr int TR = 2;
        const int ncg = s / 4;
        int RL = kLaThreads / ncg;
        if (RL > 64) RL = 64;
        const int ld = nb + LaPad<T>::v;
        auto smem_of = [&](int rl) { return ((size_t)2 * nb * s + (size_t)2 * rl * TR * ld) * sizeof(cplx<T>); };
        while (smem_of(RL) > 200 * 1024 && RL > 8) RL /= 2;          // (complex128 at nbasis 64: 64-row tiles)
        const size_t smem = smem_of(RL);
        const int per_sm = smem <= 110 * 1024 ? 2 : 1;
        const int pgrid = (int)(Vc < (int64_t)sms * per_sm ? Vc : (int64_t)sms * per_sm);
        auto kern = block_promote_tiled_kernel<T, TR>;
        CMRHS_SMEM_ATTR(kern, smem);
        kern<<<pgrid, kLaThreads, smem, stream>>>((const cplx<T> *)Bas, (const cplx<T> *)in, (cplx<T> *)out, Vc, vb, nb, s, RL);
    } else {
        int rows = 32;
        if (rows > vb) rows = vb;
        const size_t smem = ((size_t)nb * s + (size_t)rows * (nb + 1)) * sizeof(cplx<T>);
        auto kern = block_promote_kernel<T>;
        CMRHS_SMEM_ATTR(kern, smem);
        kern<<<grid, kLaThreads, smem, stream>>>((const cplx<T> *)Bas, (const cplx<T> *)in, (cplx<T> *)out, Vc, vb, nb, s, rows);
    }
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

extern "C" int coarse_block_project(const void *Basis_dev, const void *F_dev, void *C_dev, int64_t Vc, int32_t vblock, int32_t nbasis, int32_t nrhs,
                                    int32_t dtype, void *stream)
{
    CMRHS_STEP(transfer_check(Basis_dev, F_dev, C_dev, Vc, vblock, nbasis, nrhs, dtype));
    return dtype == COARSE_C64 ? transfer_launch<float>(true, Basis_dev, F_dev, C_dev, Vc, vblock, nbasis, nrhs, (cudaStream_t)stream)
                               : transfer_launch<double>(true, Basis_dev, F_dev, C_dev, Vc, vblock, nbasis, nrhs, (cudaStream_t)stream);
}

extern "C" int coarse_block_promote(const void *Basis_dev, const void *C_dev, void *F_dev, int64_t Vc, int32_t vblock, int32_t nbasis, int32_t nrhs,
                                    int32_t dtype, void *stream)
{
    CMRHS_STEP(transfer_check(Basis_dev, C_dev, F_dev, Vc, vblock, nbasis, nrhs, dtype));
    return dtype == COARSE_C64 ? transfer_launch<float>(false, Basis_dev, C_dev, F_dev, Vc, vblock, nbasis, nrhs, (cudaStream_t)stream)
                               : transfer_launch<double>(false, Basis_dev, C_dev, F_dev, Vc, vblock, nbasis, nrhs, (cudaStream_t)stream);
}

// ---- roofline denominators measured on this device (bench helper) -----------------------------------
template <int KIND>
static int time_alu_peak(int num_sms, double flops_per_thread_iter, double *sink_dev, cudaStream_t stream, cudaEvent_t e0, cudaEvent_t e1, double *tflops)
{
    const int iters = 4096, grid = num_sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        CMRHS_CUDA(cudaEventRecord(e0, stream));
        peak_alu_kernel<KIND><<<grid, threads, 0, stream>>>(iters, 1.0f + rep, sink_dev);
        CMRHS_LAUNCH_CHECK();
        CMRHS_CUDA(cudaEventRecord(e1, stream));
        CMRHS_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        CMRHS_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double tf = flops_per_thread_iter * iters * (double)grid * threads / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    *tflops = best;
    return COARSE_OK;
}

extern "C" int coarse_measure_peaks(double *out_host, int32_t nout, void *scratch_dev, int64_t scratch_bytes, void *stream_v)
{
    if (!out_host || nout < 5 || !scratch_dev || scratch_bytes < (int64_t)1 << 28) {
        set_error("coarse_measure_peaks: need out[>=5] and a device scratch block of at least 256 MiB");
        return COARSE_INVALID_ARG;
    }
    cudaStream_t stream = (cudaStream_t)stream_v;
    int dev = 0, num_sms = 0;
    CMRHS_CUDA(cudaGetDevice(&dev));
    CMRHS_CUDA(cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev));
    cudaEvent_t e0, e1;
    CMRHS_CUDA(cudaEventCreate(&e0));
    CMRHS_CUDA(cudaEventCreate(&e1));
    uint32_t *sink = static_cast<uint32_t *>(scratch_dev);               // first 256 bytes: sinks of the kernels
    const uint4 *buf = reinterpret_cast<const uint4 *>(static_cast<unsigned char *>(scratch_dev) + 256);
    const int64_t n16 = (scratch_bytes - 256) / 16;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {                                   // read-only stream, best of 5 after one warm-up
        CMRHS_CUDA(cudaEventRecord(e0, stream));
        peak_read_kernel<<<num_sms * 16, 256, 0, stream>>>(buf, n16, sink);
        CMRHS_LAUNCH_CHECK();
        CMRHS_CUDA(cudaEventRecord(e1, stream));
        CMRHS_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        CMRHS_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        const double gbs = (double)n16 * 16.0 / (ms * 1e-3) / 1e9;
        if (rep > 0 && gbs > best) best = gbs;
    }
    out_host[0] = best;
    double *dsink = reinterpret_cast<double *>(sink) + 8;
    int st = time_alu_peak<0>(num_sms, 16 * 2.0, dsink, stream, e0, e1, &out_host[1]);                      // FFMA
    if (st == COARSE_OK) st = time_alu_peak<1>(num_sms, 16 * 4.0, dsink, stream, e0, e1, &out_host[2]);     // FFMA2
    if (st == COARSE_OK) st = time_alu_peak<2>(num_sms, 16 * 2.0, dsink, stream, e0, e1, &out_host[3]);     // DFMA
    if (st == COARSE_OK) st = time_alu_peak<3>(num_sms, 16 * 512.0 / 32.0, dsink, stream, e0, e1, &out_host[4]);   // DMMA m8n8k4: 512 flops per warp
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return st;
}

extern "C" int coarse_op_profile(coarse_op_t *op, int32_t enable)
{
    if (!op) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (enable && !op->prof_ev[0])
        for (cudaEvent_t &e : op->prof_ev) CMRHS_CUDA(cudaEventCreate(&e));
    op->prof_on = enable != 0;
    op->prof_n = 0;
    return COARSE_OK;
}

extern "C" int coarse_op_profile_read(coarse_op_t *op, double *ms, int32_t capacity, int32_t *count)
{
    if (!op || !ms || !count) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    int n = op->prof_n < capacity ? op->prof_n : capacity;
    for (int k = 0; k < n; ++k) {
        CMRHS_CUDA(cudaEventSynchronize(op->prof_ev[2 * k + 1]));
        float t = 0.f;
        CMRHS_CUDA(cudaEventElapsedTime(&t, op->prof_ev[2 * k], op->prof_ev[2 * k + 1]));
        ms[k] = (double)t;
    }
    *count = n;
    op->prof_n = 0;
    return COARSE_OK;
}

// ---- Gram product without any allocation (coarse_mrhs.h: coarse_block_gram_noalloc) -----------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and
// therefore cannot hold a coarse_op handle, whose create allocates the scratch of coarse_block_gram.  The per-CTA partial
// sums of stage 1 live in a file-scope device array instead: every GPU that loads the library holds these 4 MiB until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the address a kernel may be given comes from
// cudaGetSymbolAddress, asked once per device with that device current (below).  Every call shares the array: calls that
// overlap on the GPU (two streams, two host threads) race.  Every CTA of stage 1 writes its whole partial and stage 2 reads
// only the partials of this launch, so nothing has to start at zero and the last call's contents do not matter.
constexpr int kNoallocMaxS = COARSE_NOALLOC_MAX_NRHS;        // 32
constexpr int kNoallocBlocks = 256;                          // CTAs of stage 1 (>= 1 per SM on B200)
static __device__ __align__(256) unsigned char g_noalloc_gram_scratch[(size_t)kNoallocBlocks * kNoallocMaxS * kNoallocMaxS * sizeof(zdouble)];
static_assert(sizeof(g_noalloc_gram_scratch) == COARSE_NOALLOC_SCRATCH_BYTES, "coarse_mrhs.h states the size of the static scratch");

constexpr int kNoallocMaxDev = 64;
static std::mutex g_noalloc_mu;
static zdouble *g_noalloc_ptr[kNoallocMaxDev];               // device address of the array on device d (nullptr: not asked yet)

static int noalloc_scratch(zdouble **out)
{
    int dev = 0;
    CMRHS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoallocMaxDev) { set_error("coarse_block_gram_noalloc: device index %d beyond %d", dev, kNoallocMaxDev - 1); return COARSE_UNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        CMRHS_CUDA(cudaGetSymbolAddress(&ptr, g_noalloc_gram_scratch));       // of the CURRENT device's copy of the array
        if (!ptr) { set_error("cudaGetSymbolAddress returned a null address"); return COARSE_CUDA_ERROR; }
        g_noalloc_ptr[dev] = static_cast<zdouble *>(ptr);
    }
    *out = g_noalloc_ptr[dev];
    return COARSE_OK;
}

template <typename T>
static int gram_noalloc_impl(const void *U, const void *W, zdouble *G, int64_t n, int s, zdouble *partial, cudaStream_t stream)
{
    // stage 1 as gram_impl's SIMT path, with the run-time-width kernels and a row tile of 32 KB: static + dynamic shared memory stay
    // below the 48 KB every kernel may use without an attribute call
    const int TT = s >= 8 ? 2 : 1;
    const int nt = (s + TT - 1) / TT;
    const int RG = kLaThreads / (nt * nt);
    int rows = (int)(32768 / (2 * (size_t)s * sizeof(cplx<T>)));
    rows = rows / RG * RG;
    if (rows < RG) rows = RG;
    size_t smem = (size_t)rows * s * 2 * sizeof(cplx<T>);
    if (RG > 1 && smem < (size_t)s * s * sizeof(zdouble)) smem = (size_t)s * s * sizeof(zdouble);
    int blocks = kNoallocBlocks;
    if ((int64_t)blocks > ceil_div(n, rows)) blocks = (int)ceil_div(n, rows);
    if (blocks < 1) blocks = 1;
    const cplx<T> *u = static_cast<const cplx<T> *>(U), *w = static_cast<const cplx<T> *>(W);
    if (TT == 2) gram_partial_kernel<T, 2><<<blocks, kLaThreads, smem, stream>>>(u, w, n, s, rows, partial);
    else gram_partial_kernel<T, 1><<<blocks, kLaThreads, smem, stream>>>(u, w, n, s, rows, partial);
    CMRHS_LAUNCH_CHECK();
    gram_reduce_kernel<<<(s * s * 32 + 127) / 128, 128, 0, stream>>>(partial, blocks, s * s, G);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

extern "C" int coarse_block_gram_noalloc(int32_t dtype, const void *U_dev, const void *W_dev, void *G_dev, int64_t n, int32_t s, void *stream)
{
    if (!U_dev || !W_dev || !G_dev) { set_error("NULL argument"); return COARSE_INVALID_ARG; }
    if (dtype != COARSE_C64 && dtype != COARSE_C128) { set_error("dtype must be COARSE_C64 or COARSE_C128"); return COARSE_INVALID_ARG; }
    if (n < 1 || s < 1) { set_error("bad n/s"); return COARSE_INVALID_ARG; }
    if (s > kNoallocMaxS) {
        set_error("coarse_block_gram_noalloc: nrhs %d beyond COARSE_NOALLOC_MAX_NRHS = %d (the static scratch holds %d partials of %d x %d); use coarse_block_gram",
                  (int)s, kNoallocMaxS, kNoallocBlocks, kNoallocMaxS, kNoallocMaxS);
        return COARSE_UNSUPPORTED;
    }
    if (misaligned16(U_dev) || misaligned16(W_dev) || misaligned16(G_dev)) { set_error("U, W and G must be 16-byte aligned"); return COARSE_INVALID_ARG; }
    zdouble *partial = nullptr;
    const int st = noalloc_scratch(&partial);
    if (st != COARSE_OK) return st;
    return dtype == COARSE_C64 ? gram_noalloc_impl<float>(U_dev, W_dev, static_cast<zdouble *>(G_dev), n, s, partial, (cudaStream_t)stream)
                               : gram_noalloc_impl<double>(U_dev, W_dev, static_cast<zdouble *>(G_dev), n, s, partial, (cudaStream_t)stream);
}

#ifdef CMRHS_TC_TRACE
// developer diagnostic (not part of the ABI): per-CTA, per-warp cycle counters of the last tensor-kernel launch
extern "C" int coarse_debug_trace_read(long long *out)
{
    return (int)cudaMemcpyFromSymbol(out, cmrhs::g_tc_trace, sizeof(cmrhs::g_tc_trace));
}
#endif
