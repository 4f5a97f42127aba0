// C ABI (include/dode.h) and host logic of the DODE SPGD library.  sm_100a only; no CPU fallback.
#include "../../include/dode.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "kernels_dense.cuh"
#include "kernels_csr.cuh"
#include <cub/device/device_reduce.cuh>
#include <cuda/std/functional>
#include "kernels_tc.cuh"
#include "kernels_tc2.cuh"
#include "kernels_dar.cuh"
#include "kernels_probe.cuh"

using namespace dode;

// Minibatch panels and their tensor maps for the tensor-core path, one set per issue stream
struct TcBuf {
    float *Qg_full = nullptr, *Qg_lo = nullptr;   // [cap][T*Np]
    float *rp_full = nullptr, *rp_lo = nullptr;   // [cap][T*Lp]
    int cap = 0, bn = 0;
    float* part = nullptr;                        // split-K partial sums [ksplit][T][tiles*128][bn]
    size_t part_cap = 0;                          // floats
    CUtensorMap mapQ_f, mapQ_l, mapR_f, mapR_l;   // boxes of bn days
    int bh = 0;                                   // CTA-pair kernel (kernels_tc2.cuh): boxes of bh = bn / 2 days
    CUtensorMap mapQ_f2, mapQ_l2, mapR_f2, mapR_l2;
};

// Two internal streams that plain dode_spgd_step calls alternate on (tensor-core path): consecutive iterations touch
// disjoint days (chunks of a permutation) and read-only operators, so iteration i+1 may start while
// iteration i drains.  A kernel of one lane then fills the SM slots the other lane's kernel leaves at its prologue,
// dependency wait and tail — the short kernels of small networks (corridor: 288 CTAs = one wave) are otherwise
// serialised by the grid-wide dependency between forward and gradient.
struct Lane {
    cudaStream_t st = nullptr;
    cudaEvent_t done = nullptr, entry = nullptr;
    TcBuf buf;
    int64_t last_id = 0;          // id of the latest step issued on this lane
    int64_t seen_other = 0;       // latest step id of the OTHER lane that this lane has already waited for
};

struct dode_ctx {
    dode_dims dm{};
    int Np = 0, Lp = 0;          // padded N / L (dense: 128-byte rows when that costs <= 3 %, else 32- or 16-byte)
    cudaStream_t stream = nullptr;
    // dense storage (layouts: kernels_dense.cuh)
    float* Ag = nullptr;         // [C][T][H+1][Lp][Np]  departure-major, a3
    float* Af = nullptr;         // [C][T][H+1][Np][Lp]  arrival-major (lag-merged), a2
    // CSR storage (a6)
    CsrStore csr{};
    // state
    float* q = nullptr;          // [D][T][Np]
    float* G = nullptr;          // [D][T][Np] Adagrad accumulator (NEXT-1), allocated by the first dode_adagrad_step
    float* x = nullptr;          // [D][T][L]
    float* r = nullptr;          // [T*Lp][bp] residual panel (FFMA / CSR paths)
    size_t r_cap = 0;            // floats
    float* Qb = nullptr;         // [T*Np][bp] gathered state panel (FFMA path, 1 < b)
    size_t qb_cap = 0;
    double* d_part = nullptr;    // objective partials
    size_t part_cap = 0;
    double* d_obj = nullptr;     // [D] per-day objective + 2 scalars
    double* d_mom = nullptr;     // [2*D] per-day sum and sum of squares of x (dode_r2), allocated by its first call
    float *pu = nullptr, *pv = nullptr, *pw = nullptr;   // apply / power-iteration scratch: [T][Np], [T][Lp], [T][N]
    std::vector<int32_t> labels;
    std::vector<int32_t> stamp;  // distinctness check
    int32_t stamp_id = 0;
    int64_t launches = 0;
    std::string path;
    char err[512] = {0};
    bool sm_opt_in[16] = {false};
    // tensor-core path (kernels_tc.cuh)
    TcBuf tcb;                                     // panels of the ctx stream
    Lane lane[2];
    bool lanes_on = true, lanes_dirty = false;     // dirty: lane work not yet joined into the ctx stream
    int lane_next = 0;
    unsigned lanes_used = 0;                       // lanes the latest step_impl call issued work on (bit per lane)
    int64_t lane_step_id = 0;
    std::vector<int64_t> day_last_id;              // [D] id of the last lane step that touched the day
    std::vector<int8_t> day_last_lane;             // [D] and its lane (-1: none)
    long rpitch = 0;
    // kernel-selection options (dode_set_option)
    int tc_min_b = 8, opt_ksplit = 0, opt_bstages = 0;
    int opt_pair = 1;                              // 0 = single-CTA kernels only, 1 = CTA pairs + single-CTA odd tile, 2 = pairs only
    bool opt_pdl = true;
    bool tc_ready = false, tc_attr = false;
    CUtensorMap mapA_fwd, mapA_fwd64, mapA_grad, mapA_grad64;
    // streaming steps (dode_spgd_step_host): copy streams, staging buffers, ping-pong events
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr, s_sc = nullptr, s_ga = nullptr;   // copies only / scatter into x / gather of q
    cudaEvent_t ev_h2d = nullptr, ev_step[2] = {nullptr, nullptr}, ev_d2h[2] = {nullptr, nullptr};
    cudaEvent_t ev_scat[2] = {nullptr, nullptr}, ev_gath[2] = {nullptr, nullptr};
    std::vector<int32_t> prev_days;
    float *stage_x = nullptr, *stage_q = nullptr;
    size_t stage_x_cap = 0, stage_q_cap = 0;
    int64_t host_calls = 0;
    cudaEvent_t ev_fence = nullptr;
    bool plain_since_host = true;   // non-streaming work was issued on the ctx stream since the last streaming step
    // optional per-kernel event timing (dode_timing_enable / dode_timing_read)
    bool timing = false;
    std::vector<cudaEvent_t> ev_pool;
    struct Pending { int kind; cudaEvent_t a, b; };
    std::vector<Pending> ev_pending;
    double t_total[3] = {0, 0, 0};
    int64_t t_count[3] = {0, 0, 0};
};

enum { KIND_FWD = 0, KIND_GRAD = 1, KIND_OTHER = 2 };

// NEXT-1, Alg. 1 as printed: optional row-chunk mask on the residual and Adagrad in the update
struct StepOpt {
    const uint8_t* mask = nullptr;   // device [n][T][L] by position in the day list; null = every row
    float* G = nullptr;              // Adagrad accumulator [D][T][Np]; null = plain projected step
    float eps = 0.f;
};

struct KernelTimer {      // records an event pair around one launch when timing is on
    dode_ctx* c; cudaEvent_t a = nullptr, b = nullptr; int kind;
    KernelTimer(dode_ctx* ctx, int k) : c(ctx), kind(k) {
        if (!c->timing) return;
        for (cudaEvent_t* e : {&a, &b}) {
            if (!c->ev_pool.empty()) { *e = c->ev_pool.back(); c->ev_pool.pop_back(); }
            else if (cudaEventCreate(e) != cudaSuccess) { *e = nullptr; }
        }
        if (a && b) cudaEventRecord(a, c->stream);
    }
    ~KernelTimer() {
        if (!c->timing || !a || !b) return;
        cudaEventRecord(b, c->stream);
        c->ev_pending.push_back({kind, a, b});
    }
};

static thread_local char g_create_err[512] = {0};

static int fail(dode_ctx* c, int code, const char* fmt, ...) {
    char* dst = c ? c->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? DODE_ENOMEM : DODE_ECUDA,      \
                        "%s: %s", #call, cudaGetErrorString(e_));                             \
    } while (0)

static inline int ceil_div(long a, long b) { return (int)((a + b - 1) / b); }
static inline int round_up(int a, int b) { return (a + b - 1) / b * b; }

// Padded extent of an operator dimension: whole 128-byte lines per row when that costs at most 3 % more bytes, else
// whole 32-byte sectors (8 floats).  8 is also what the tensor path needs: the K windows of the bf16 correction panels
// start at multiples of the padded dimension, and a TMA box must start on a 16-byte boundary (8 bf16).
static int pad_dim(int n) {
    const int p = round_up(n, 32);
    if ((long)p * 100 <= (long)n * 103) return p;
    return round_up(n, 8);
}

static int ensure_buf(dode_ctx* ctx, float** buf, size_t* cap, size_t floats) {
    if (*cap >= floats) return DODE_OK;
    if (*buf) { CU(cudaStreamSynchronize(ctx->stream)); CU(cudaFree(*buf)); *buf = nullptr; *cap = 0; }
    CU(cudaMalloc(buf, floats * sizeof(float)));
    *cap = floats;
    return DODE_OK;
}

static int pick_bt(int n) { return n <= 1 ? 1 : n <= 2 ? 2 : n <= 4 ? 4 : n <= 8 ? 8 : 16; }

static size_t cluster_floats(const dode_ctx* ctx) {
    const dode_dims& d = ctx->dm;
    return (size_t)d.T * (d.H + 1) * ctx->Lp * ctx->Np;
}

// ---- dense FFMA launches ------------------------------------------------------------------------
template <int BT, int EPI>
static int launch_band(dode_ctx* ctx, int slot, const BandArgs& a, int nbt, const DayList& dl, int kind) {
    int cwlog2 = 0;
    while ((1 << cwlog2) < a.M4 && cwlog2 < 5) ++cwlog2;
    // short time axes (T = 1 on the Fig. 12 shape): narrower column groups give more CTAs; 8 column threads still read
    // whole 128-byte lines per K row
    while (cwlog2 > 2 && (long)ceil_div(a.M4, 1 << cwlog2) * a.T * nbt < 2 * 148) --cwlog2;
    const size_t smem = (size_t)kThreads * 4 * BT * sizeof(float);
    if (smem > 48 * 1024 && !ctx->sm_opt_in[slot]) {
        CU(cudaFuncSetAttribute(band_coldot<BT, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->sm_opt_in[slot] = true;
    }
    dim3 grid(ceil_div(a.M4, 1 << cwlog2), a.T, nbt);
    KernelTimer kt(ctx, kind);
    band_coldot<BT, EPI><<<grid, kThreads, smem, ctx->stream>>>(a, cwlog2, dl);
    ctx->launches++;
    return DODE_OK;
}

template <int EPI>
static int launch_band_bt(dode_ctx* ctx, int bt, const BandArgs& a, const DayList& dl, int kind) {
    const int nbt = a.bp / bt;
    switch (bt) {
        case 1: return launch_band<1, EPI>(ctx, EPI * 5 + 0, a, nbt, dl, kind);
        case 2: return launch_band<2, EPI>(ctx, EPI * 5 + 1, a, nbt, dl, kind);
        case 4: return launch_band<4, EPI>(ctx, EPI * 5 + 2, a, nbt, dl, kind);
        case 8: return launch_band<8, EPI>(ctx, EPI * 5 + 3, a, nbt, dl, kind);
        default: return launch_band<16, EPI>(ctx, EPI * 5 + 4, a, nbt, dl, kind);
    }
}

static BandArgs band_args(const dode_ctx* ctx, int c, bool forward, int bp) {
    const dode_dims& d = ctx->dm;
    BandArgs a{};
    a.A = (forward ? ctx->Af : ctx->Ag) + (size_t)c * cluster_floats(ctx);
    a.M = forward ? d.L : d.N;
    a.M4 = (forward ? ctx->Lp : ctx->Np) / 4;
    a.kunit = forward ? ctx->Np : ctx->Lp;
    a.T = d.T; a.H = d.H; a.bp = bp; a.forward = forward ? 1 : 0;
    return a;
}

// a2 on the FFMA / CSR paths: residual panel of one sub-batch (<= kMaxDays days of cluster c) into ctx->r
// ([T*Lp][bp], day fastest); returns the day tile bt and the panel stride bp
static int forward_batch(dode_ctx* ctx, int c, const DayList& dl, int* bt_out, int* bp_out, const uint8_t* mask = nullptr) {
    const dode_dims& d = ctx->dm;
    const bool csr = d.storage == DODE_CSR;
    const int bt = csr ? 32 : pick_bt(dl.n);
    const int bp = csr ? csr_bp(dl.n) : ceil_div(dl.n, bt) * bt;
    const size_t dayStride = (size_t)d.T * ctx->Np;
    int rc = ensure_buf(ctx, &ctx->r, &ctx->r_cap, (size_t)d.T * ctx->Lp * bp);
    if (rc) return rc;
    if (!csr) {
        const float* panel = ctx->q + (size_t)dl.day[0] * dayStride;      // b = 1: the day's state IS the panel
        if (bp > 1) {
            if ((rc = ensure_buf(ctx, &ctx->Qb, &ctx->qb_cap, dayStride * bp))) return rc;
            KernelTimer kt(ctx, KIND_OTHER);
            gather_panel<<<dim3(ceil_div((long)dayStride, 32), ceil_div(bp, 32)), 256, 0, ctx->stream>>>(
                ctx->q, dayStride, (long)dayStride, ctx->Qb, bp, dl);
            ctx->launches++;
            panel = ctx->Qb;
        }
        BandArgs a = band_args(ctx, c, true, bp);
        a.B = panel; a.x = ctx->x; a.out = ctx->r; a.mask = mask;
        if ((rc = launch_band_bt<EPI_RESID>(ctx, bt, a, dl, KIND_FWD))) return rc;
    } else {
        KernelTimer kt(ctx, KIND_FWD);
        rc = csr_forward(ctx->csr, c, ctx->q, dayStride, ctx->x, ctx->r, bp, bp, dl, d, ctx->Np, ctx->stream,
                         &ctx->launches, mask);
        if (rc) return fail(ctx, rc, "CSR scratch allocation failed");
    }
    *bt_out = bt; *bp_out = bp;
    return DODE_OK;
}

// waits for the compute stream and for the copy streams of the streaming step
static cudaError_t sync_all(dode_ctx* ctx) {
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (ctx->s_h2d) { cudaError_t e2 = cudaStreamSynchronize(ctx->s_h2d); if (e == cudaSuccess) e = e2; }
    if (ctx->s_d2h) { cudaError_t e2 = cudaStreamSynchronize(ctx->s_d2h); if (e == cudaSuccess) e = e2; }
    for (cudaStream_t st : {ctx->s_sc, ctx->s_ga})
        if (st) { cudaError_t e2 = cudaStreamSynchronize(st); if (e == cudaSuccess) e = e2; }
    for (Lane& ln : ctx->lane)
        if (ln.st) { cudaError_t e2 = cudaStreamSynchronize(ln.st); if (e == cudaSuccess) e = e2; }
    ctx->lanes_dirty = false;
    return e;
}

static int validate_days(dode_ctx* ctx, const int32_t* days, int32_t n, bool same_cluster, int* cluster) {
    if (!days || n <= 0) return fail(ctx, DODE_EINVAL, "days is null or n <= 0");
    const dode_dims& d = ctx->dm;
    if (++ctx->stamp_id == INT32_MAX) { std::fill(ctx->stamp.begin(), ctx->stamp.end(), 0); ctx->stamp_id = 1; }
    for (int i = 0; i < n; ++i) {
        const int day = days[i];
        if (day < 0 || day >= d.D) return fail(ctx, DODE_EINVAL, "day %d out of range [0,%d)", day, d.D);
        if (ctx->stamp[day] == ctx->stamp_id) return fail(ctx, DODE_EINVAL, "day %d listed twice", day);
        ctx->stamp[day] = ctx->stamp_id;
        if (same_cluster && ctx->labels[day] != ctx->labels[days[0]])
            return fail(ctx, DODE_EINVAL, "days %d and %d belong to different clusters", days[0], day);
    }
    if (cluster) *cluster = ctx->labels[days[0]];
    return DODE_OK;
}


// ---- tensor-core path: tensor maps, panels, launches ---------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode() {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (PFN_encodeTiled)p;
    }
    return fn;
}

// fp32 tensor, innermost dim first; out-of-bounds elements read as zero
static int make_map(dode_ctx* ctx, CUtensorMap* m, const void* base, int rank, const uint64_t* dims,
                    const uint64_t* strides_bytes, const uint32_t* box, bool swizzle128, bool bf16_sw64 = false) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) return fail(ctx, DODE_ECUDA, "cuTensorMapEncodeTiled is unavailable");
    cuuint64_t gd[3]; cuuint64_t gs[2]; cuuint32_t bx[3]; cuuint32_t es[3] = {1, 1, 1};
    for (int i = 0; i < rank; ++i) { gd[i] = dims[i]; bx[i] = box[i]; }
    for (int i = 0; i + 1 < rank; ++i) gs[i] = strides_bytes[i];
    CUresult r = enc(m, bf16_sw64 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, (cuuint32_t)rank,
                     const_cast<void*>(base), gd, gs, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     bf16_sw64 ? CU_TENSOR_MAP_SWIZZLE_64B : swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, DODE_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return DODE_OK;
}

// create-time: the A maps over Af / Ag, one (cluster, time) slab per index of the outer dimension so that K rows
// beyond the slab read as zero
static int tc_setup(dode_ctx* ctx) {
    const dode_dims& d = ctx->dm;
    ctx->rpitch = (long)d.T * ctx->Lp;
    const uint64_t slabs = (uint64_t)d.C * d.T;
    for (int fwd = 0; fwd < 2; ++fwd) {
        const uint64_t Mp = fwd ? ctx->Lp : ctx->Np, krows = (uint64_t)(d.H + 1) * (fwd ? ctx->Np : ctx->Lp);
        const uint64_t dims[3] = {Mp, krows, slabs};
        const uint64_t str[2] = {Mp * 4, krows * Mp * 4};
        const uint32_t box[3] = {(uint32_t)tc::kTileM, (uint32_t)tc::kTileK, 1}, box64[3] = {(uint32_t)tc::kTileM / 2, (uint32_t)tc::kTileK, 1};
        const float* base = fwd ? ctx->Af : ctx->Ag;
        int rc = make_map(ctx, fwd ? &ctx->mapA_fwd : &ctx->mapA_grad, base, 3, dims, str, box, false);
        if (rc) return rc;
        if ((rc = make_map(ctx, fwd ? &ctx->mapA_fwd64 : &ctx->mapA_grad64, base, 3, dims, str, box64, false))) return rc;
    }
    ctx->tc_ready = true;
    return DODE_OK;
}

// B tensor maps over the minibatch panels with boxes of `boxdays` days
static int tc_make_bmaps(dode_ctx* ctx, TcBuf& tb, int boxdays, CUtensorMap* mQf, CUtensorMap* mQl, CUtensorMap* mRf, CUtensorMap* mRl) {
    const size_t qlen = (size_t)ctx->dm.T * ctx->Np;
    // B operands: K-major windows of the per-day vectors, SWIZZLE_128B tiles of {32 floats, boxdays days}
    const uint64_t qd[2] = {(uint64_t)qlen, (uint64_t)tb.cap};
    const uint64_t qs[1] = {(uint64_t)qlen * 4};
    const uint32_t bb[2] = {(uint32_t)tc::kTileK, (uint32_t)boxdays};
    int rc;
    if ((rc = make_map(ctx, mQf, tb.Qg_full, 2, qd, qs, bb, true))) return rc;
    // the correction operands: two bf16 planes (bf16(v) | bf16(v - tf32(v))) of tb.cap rows each in the same allocation
    const uint64_t qd16[2] = {(uint64_t)qlen, (uint64_t)2 * tb.cap};
    const uint64_t qs16[1] = {(uint64_t)qlen * 2};
    if ((rc = make_map(ctx, mQl, tb.Qg_lo, 2, qd16, qs16, bb, false, true))) return rc;
    const uint64_t rd[2] = {(uint64_t)ctx->rpitch, (uint64_t)tb.cap};
    const uint64_t rs[1] = {(uint64_t)ctx->rpitch * 4};
    if ((rc = make_map(ctx, mRf, tb.rp_full, 2, rd, rs, bb, true))) return rc;
    const uint64_t rd16[2] = {(uint64_t)ctx->rpitch, (uint64_t)2 * tb.cap};
    const uint64_t rs16[1] = {(uint64_t)ctx->rpitch * 2};
    return make_map(ctx, mRl, tb.rp_lo, 2, rd16, rs16, bb, false, true);
}

// panels for `rows` minibatch days (>= dsplit * bn) and B tensor maps with boxes of bn days
static int tc_ensure(dode_ctx* ctx, TcBuf& tb, cudaStream_t st, int bn, int rows) {
    const dode_dims& d = ctx->dm;
    const size_t qlen = (size_t)d.T * ctx->Np;
    if (tb.cap < rows) {
        const int bn_alloc = rows;
        CU(cudaStreamSynchronize(st));
        cudaFree(tb.Qg_full); cudaFree(tb.Qg_lo); cudaFree(tb.rp_full); cudaFree(tb.rp_lo);
        tb.Qg_full = tb.Qg_lo = tb.rp_full = tb.rp_lo = nullptr;
        tb.cap = 0; tb.bn = 0; tb.bh = 0;
        CU(cudaMalloc(&tb.Qg_full, bn_alloc * qlen * 4)); CU(cudaMalloc(&tb.Qg_lo, bn_alloc * qlen * 4));
        CU(cudaMalloc(&tb.rp_full, (size_t)bn_alloc * ctx->rpitch * 4)); CU(cudaMalloc(&tb.rp_lo, (size_t)bn_alloc * ctx->rpitch * 4));
        CU(cudaMemsetAsync(tb.Qg_full, 0, bn_alloc * qlen * 4, st)); CU(cudaMemsetAsync(tb.Qg_lo, 0, bn_alloc * qlen * 4, st));
        CU(cudaMemsetAsync(tb.rp_full, 0, (size_t)bn_alloc * ctx->rpitch * 4, st));
        CU(cudaMemsetAsync(tb.rp_lo, 0, (size_t)bn_alloc * ctx->rpitch * 4, st));
        tb.cap = bn_alloc;
    }
    if (tb.bn != bn) {
        int rc;
        if ((rc = tc_make_bmaps(ctx, tb, bn, &tb.mapQ_f, &tb.mapQ_l, &tb.mapR_f, &tb.mapR_l))) return rc;
        tb.bn = bn;
    }
    if (!ctx->tc_attr) {
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32<false, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32<false, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32<false, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32<true, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32<true, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32<true, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32_pair<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        CU(cudaFuncSetAttribute(tc::banded_gemm_3xtf32_pair<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        ctx->tc_attr = true;
    }
    return DODE_OK;
}

// Launch geometry of the tensor-core kernels for a minibatch of bn (multiple of 16) days
struct TcGeom { int stages, bstages, nring; size_t smem; int ks_f, ks_g; size_t part_floats; };

// minibatch of n days -> day groups per tile (1, or 2 above 128 days) and days per group (MMA N, multiple of 16)
// (wider than 64 days: the CTA-pair kernel, whose two CTAs stage bn / 2 days each, so bn is a multiple of 32)
static bool tc_pair_width(const dode_ctx* ctx, int n) { return ctx->opt_pair != 0 && n > 64; }
static void tc_day_groups(const dode_ctx* ctx, int n, int* dsplit, int* bn) {
    *dsplit = n > 128 ? 2 : 1;
    *bn = round_up(ceil_div(n, *dsplit), tc_pair_width(ctx, n) ? 32 : 16);
}

// shared-memory geometry of the CTA-pair kernel: B stages of bn / 2 days, one CTA per SM
static TcGeom tc_pair_geometry(const dode_ctx* ctx, int bn) {
    TcGeom g{};
    const int bStage = bn * tc::kTileK * 4;        // (bn / 2 days) x (fp32 + two bf16 planes)
    const int fixed = 512;
    const int budget = 227 * 1024 - fixed;
    // 4 B stages and 4 TMEM A buffers, fixed: the issue loop of the kernel is unrolled for them (DODE_OPT_TC_BSTAGES steers
    // the single-CTA kernels only).  Measured on large_dense b = 256: 3 -> 55.7, 4 -> 55.1, 5 -> 56.0 ms per epoch.
    const int sb = 4;
    const int sa = std::max(2, std::min((budget - sb * bStage) / tc::kABytes, 16));
    g.stages = sa; g.bstages = sb;
    g.nring = 4;                                   // 2 * bn <= 256 accumulator columns + 4 x 64
    g.smem = (size_t)sa * tc::kABytes + (size_t)sb * bStage + fixed;
    g.ks_f = g.ks_g = 1;
    return g;
}

static TcGeom tc_geometry(const dode_ctx* ctx, int bn, int dsplit) {
    const dode_dims& d = ctx->dm;
    TcGeom g{};
    // Two TMA rings (kernels_tc.cuh): B stages of B_full + bf16(B) + bf16(B_lo) tiles — the panels sit in L2, a shallow
    // ring covers them — and A stages of one 16 KB tile each, as many as the rest of the shared memory holds (the A
    // bytes in flight per SM are what hides the HBM latency).  Two CTAs per SM when 256 TMEM columns suffice.
    // An SM has 228 KB of shared memory, 1 KB of it reserved per resident CTA; a CTA may use up to 227 KB.
    const int bStage = 2 * bn * tc::kTileK * 4;
    const int fixed = 512;                         // barriers (2*SA + 2*SB + 10 of them, SA <= 16, SB <= 8) + the TMEM slot
    const int acc_cols = 2 * bn;
    const bool two = acc_cols + 128 <= 256;
    const int budget = (two ? 228 * 1024 / 2 - 1024 : 227 * 1024) - fixed;
    int sb = ctx->opt_bstages > 0 ? ctx->opt_bstages : 3;      // measured: 2 starves the MMA warp at every width, 4 = 3
    int sa = (budget - sb * bStage) / tc::kABytes;
    sa = std::max(2, std::min(sa, 16));
    sb = std::max(2, std::min(sb, sa));
    g.stages = sa;
    g.bstages = sb;
    g.nring = two ? 2 : (acc_cols + 256 <= 512 ? 4 : 2);
    g.smem = (size_t)sa * tc::kABytes + (size_t)sb * bStage + fixed;
    // split-K when the time axis is too short to fill the machine (T * tiles CTAs for 148 SMs x 1-2 CTAs): e.g. the
    // Fig. 12 workload, T = 1.  Each pass then runs ksplit CTAs per tile and a small epilogue kernel.
    const int slots = 148 * (g.smem * 2 + 2048 <= 227 * 1024 ? 2 : 1);
    auto pick_split = [&](int M, int kunit) {
        const long ctas = (long)ceil_div(M, tc::kTileM) * d.T * dsplit;
        const int nk_max = ceil_div((long)(d.H + 1) * kunit, tc::kTileK);
        int ks = (int)std::min<long>(slots / std::max<long>(ctas, 1), nk_max / 8);
        if (ctx->opt_ksplit > 0) ks = ctx->opt_ksplit;
        return std::max(1, std::min(ks, 32));
    };
    g.ks_f = pick_split(d.L, ctx->Np);
    g.ks_g = pick_split(d.N, ctx->Lp);
    g.part_floats = (g.ks_f > 1 || g.ks_g > 1)
        ? (size_t)std::max(g.ks_f * ceil_div(d.L, tc::kTileM), g.ks_g * ceil_div(d.N, tc::kTileM)) * tc::kTileM * d.T * bn * dsplit : 0;
    return g;
}

static int tc_ensure_part(dode_ctx* ctx, TcBuf& tb, cudaStream_t st, size_t need) {
    if (tb.part_cap >= need) return DODE_OK;
    CU(cudaStreamSynchronize(st));
    cudaFree(tb.part); tb.part = nullptr; tb.part_cap = 0;
    CU(cudaMalloc(&tb.part, need * sizeof(float)));
    tb.part_cap = need;
    return DODE_OK;
}

// Launch with programmatic stream serialization (PDL): the kernel may start while its predecessor drains; it
// calls griddepcontrol.wait before touching anything the predecessor wrote.  Per-kernel event timing records
// events between launches, which serialises them again — timing mode therefore shows un-overlapped durations.
template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(bool pdl, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// one SPGD iteration of a sub-batch (8 <= n <= 256 days) on the tensor cores
static int tc_step(dode_ctx* ctx, int c, const DayList& dl, float eta, const StepOpt& opt, TcBuf& tb, cudaStream_t st) {
    const dode_dims& d = ctx->dm;
    int dsplit, bn;
    tc_day_groups(ctx, dl.n, &dsplit, &bn);
    int rc = tc_ensure(ctx, tb, st, bn, dsplit * bn);
    if (rc) return rc;
    const TcGeom geo0 = tc_geometry(ctx, bn, dsplit);
    const int stages = geo0.stages, nring = geo0.nring;
    const size_t smem = geo0.smem;
    const size_t dayStride = (size_t)d.T * ctx->Np;
    {
        KernelTimer kt(ctx, KIND_OTHER);
        CU(launch_pdl(ctx->opt_pdl, tc::gather_split, dim3(std::min<long>(64, ceil_div((long)dayStride / 4, 256)), dl.n), dim3(256), 0,
                      st, ctx->q, dayStride, (long)dayStride / 4, tb.Qg_full, reinterpret_cast<__nv_bfloat16*>(tb.Qg_lo), tb.cap, dl));
        ctx->launches++;
    }
    tc::TcParams p{};
    p.T = d.T; p.H = d.H; p.Lp = ctx->Lp; p.Np = ctx->Np; p.bn = bn; p.dsplit = dsplit; p.bnt = dsplit * bn;
    p.stages = stages; p.bstages = geo0.bstages; p.nring = nring;
    p.slab0 = c * d.T;
    p.x = ctx->x; p.rp_full = tb.rp_full; p.rp_lo = reinterpret_cast<__nv_bfloat16*>(tb.rp_lo); p.pcap = tb.cap; p.rpitch = ctx->rpitch;
    p.q = ctx->q; p.dayStride = dayStride; p.eta = eta;
    p.mask = opt.mask; p.G = opt.G; p.eps = opt.eps;
    const bool ada = opt.mask || opt.G;
    auto kern = bn <= 32 ? (ada ? tc::banded_gemm_3xtf32<true, 16> : tc::banded_gemm_3xtf32<false, 16>)
              : bn <= 64 ? (ada ? tc::banded_gemm_3xtf32<true, 32> : tc::banded_gemm_3xtf32<false, 32>)
                         : (ada ? tc::banded_gemm_3xtf32<true, 64> : tc::banded_gemm_3xtf32<false, 64>);
    const TcGeom& geo = geo0;
    const int ks_f = geo.ks_f, ks_g = geo.ks_g;
    if ((rc = tc_ensure_part(ctx, tb, st, geo.part_floats))) return rc;
    p.part = tb.part;
    // CTA pairs (kernels_tc2.cuh) for minibatches wider than 64 days, unless the pass is split along K
    const bool pair = tc_pair_width(ctx, dl.n) && ks_f == 1 && ks_g == 1;
    TcGeom pgeo{};
    if (pair) {
        pgeo = tc_pair_geometry(ctx, bn);
        if (tb.bh != bn / 2) {
            if ((rc = tc_make_bmaps(ctx, tb, bn / 2, &tb.mapQ_f2, &tb.mapQ_l2, &tb.mapR_f2, &tb.mapR_l2))) return rc;
            tb.bh = bn / 2;
        }
    }
    auto pkern = ada ? tc::banded_gemm_3xtf32_pair<true> : tc::banded_gemm_3xtf32_pair<false>;
    auto epilogue = [&](int Mt) -> int {           // second half of a split-K pass
        const dim3 g(ceil_div((long)Mt * (p.bnt / 4), 256), d.T);
        if (ada) tc::splitk_epilogue<true><<<g, 256, 0, st>>>(p, Mt, dl);
        else tc::splitk_epilogue<false><<<g, 256, 0, st>>>(p, Mt, dl);
        ctx->launches++;
        return DODE_OK;
    };
    // one pass over all output tiles: pairs of tiles on the pair kernel, an odd last tile (or everything, when pairs are
    // not used) on the single-CTA kernel
    auto run_pass = [&](int M, int ks, const CUtensorMap& mA, const CUtensorMap& mA64, const CUtensorMap& mBf, const CUtensorMap& mBl,
                        const CUtensorMap& mBf2, const CUtensorMap& mBl2) -> int {
        const int tiles = ceil_div(M, tc::kTileM);
        int done = 0;
        if (pair) {
            const int npairs = ctx->opt_pair == 2 ? ceil_div(tiles, 2) : tiles / 2;
            if (npairs > 0) {
                p.mtile0 = 0; p.ksplit = 1; p.stages = pgeo.stages; p.bstages = pgeo.bstages; p.nring = pgeo.nring;
                CU(launch_pdl(ctx->opt_pdl, pkern, dim3(2 * dsplit * npairs, d.T, 1), dim3(tc::kThreadsTC), pgeo.smem, st,
                              mA, mA64, mBf2, mBl2, p, dl));
                ctx->launches++;
                done = 2 * npairs;
            }
        }
        if (done < tiles) {
            p.mtile0 = done; p.ksplit = ks; p.stages = geo.stages; p.bstages = geo.bstages; p.nring = geo.nring;
            CU(launch_pdl(ctx->opt_pdl, kern, dim3((tiles - done) * dsplit, d.T, ks), dim3(tc::kThreadsTC), smem, st,
                          mA, mA64, mBf, mBl, p, dl));
            ctx->launches++;
            if (ks > 1) epilogue(tiles * tc::kTileM);
        }
        return DODE_OK;
    };
    {
        KernelTimer kt(ctx, KIND_FWD);
        p.mode = 0; p.M = d.L; p.kunit = ctx->Np;
        if ((rc = run_pass(d.L, ks_f, ctx->mapA_fwd, ctx->mapA_fwd64, tb.mapQ_f, tb.mapQ_l, tb.mapQ_f2, tb.mapQ_l2))) return rc;
    }
    {
        KernelTimer kt(ctx, KIND_GRAD);
        p.mode = 1; p.M = d.N; p.kunit = ctx->Lp;
        if ((rc = run_pass(d.N, ks_g, ctx->mapA_grad, ctx->mapA_grad64, tb.mapR_f, tb.mapR_l, tb.mapR_f2, tb.mapR_l2))) return rc;
    }
    char buf[96];
    snprintf(buf, sizeof buf, dsplit > 1 ? "tcgen05%s_3xtf32_fwd_bn%dx2+tcgen05%s_3xtf32_grad_bn%dx2"
                                         : "tcgen05%s_3xtf32_fwd_bn%d+tcgen05%s_3xtf32_grad_bn%d",
             pair ? "_pair" : "", bn, pair ? "_pair" : "", bn);
    ctx->path = buf;
    return DODE_OK;
}

// ---- lanes ------------------------------------------------------------------------------------------
// makes the ctx stream wait for everything issued on the lanes so far (asynchronous; no host wait)
static int join_lanes(dode_ctx* ctx) {
    if (!ctx->lanes_dirty) return DODE_OK;
    for (Lane& ln : ctx->lane)
        if (ln.st && ln.last_id) CU(cudaStreamWaitEvent(ctx->stream, ln.done, 0));
    ctx->lanes_dirty = false;
    return DODE_OK;
}

static int lane_init(dode_ctx* ctx, Lane& ln) {
    if (ln.st) return DODE_OK;
    CU(cudaStreamCreateWithFlags(&ln.st, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&ln.done, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&ln.entry, cudaEventDisableTiming));
    return DODE_OK;
}

// picks the lane of the next step, forks it from the ctx stream and orders it after earlier steps on its days
static int lane_begin(dode_ctx* ctx, const DayList& dl, Lane** out) {
    const int li = ctx->lane_next;
    ctx->lane_next ^= 1;
    Lane& ln = ctx->lane[li];
    Lane& ot = ctx->lane[li ^ 1];
    if (int rc = lane_init(ctx, ln)) return rc;
    // fork: whatever is on the ctx stream now (the caller's work, earlier non-lane calls) precedes this step
    CU(cudaEventRecord(ln.entry, ctx->stream));
    CU(cudaStreamWaitEvent(ln.st, ln.entry, 0));
    // a day last stepped on the other lane by a step this lane has not waited for yet (steps of this lane: stream order)
    bool conflict = false;
    for (int i = 0; i < dl.n; ++i)
        conflict |= ctx->day_last_lane[dl.day[i]] == (li ^ 1) && ctx->day_last_id[dl.day[i]] > ln.seen_other;
    if (conflict) {
        CU(cudaStreamWaitEvent(ln.st, ot.done, 0));
        ln.seen_other = ot.last_id;
    }
    const int64_t id = ++ctx->lane_step_id;
    for (int i = 0; i < dl.n; ++i) { ctx->day_last_lane[dl.day[i]] = (int8_t)li; ctx->day_last_id[dl.day[i]] = id; }
    ln.last_id = id;
    *out = &ln;
    return DODE_OK;
}

static int lane_end(dode_ctx* ctx, Lane* ln) {
    CU(cudaEventRecord(ln->done, ln->st));
    ctx->lanes_dirty = true;
    return DODE_OK;
}

static int step_impl(dode_ctx* ctx, const int32_t* days, int32_t n, float eta, int c, const StepOpt& opt0 = StepOpt(),
                     bool allow_lanes = false) {
    const dode_dims& d = ctx->dm;
    const size_t dayStride = (size_t)d.T * ctx->Np;
    const int chunk = d.storage == DODE_CSR ? kCsrMaxDays : kMaxDays;
    ctx->lanes_used = 0;
    for (int off = 0; off < n; off += chunk) {          // days are independent units
        DayList dl;
        dl.n = std::min(chunk, n - off);
        std::memcpy(dl.day, days + off, sizeof(int) * dl.n);
        int bt, bp, rc;
        StepOpt opt = opt0;
        if (opt.mask) opt.mask += (size_t)off * d.T * d.L;
        const bool tcp = ctx->tc_ready && ctx->tc_min_b > 0 && dl.n >= ctx->tc_min_b;
        if (tcp && allow_lanes && ctx->lanes_on && !ctx->timing && !opt.mask && !opt.G) {
            Lane* ln = nullptr;
            if ((rc = lane_begin(ctx, dl, &ln))) return rc;
            if ((rc = tc_step(ctx, c, dl, eta, opt, ln->buf, ln->st))) return rc;
            if ((rc = lane_end(ctx, ln))) return rc;
            ctx->lanes_used |= 1u << (ln - ctx->lane);
            continue;
        }
        if ((rc = join_lanes(ctx))) return rc;
        if (tcp) {
            if ((rc = tc_step(ctx, c, dl, eta, opt, ctx->tcb, ctx->stream))) return rc;
            continue;
        }
        if ((rc = forward_batch(ctx, c, dl, &bt, &bp, opt.mask))) return rc;
        if (d.storage == DODE_DENSE) {
            BandArgs a = band_args(ctx, c, false, bp);
            a.B = ctx->r; a.q = ctx->q; a.dayStride = dayStride; a.eta = eta; a.G = opt.G; a.eps = opt.eps;
            if ((rc = launch_band_bt<EPI_UPDATE>(ctx, bt, a, dl, KIND_GRAD))) return rc;
            char buf[96];
            snprintf(buf, sizeof buf, "ffma_coldot_fwd_bt%d+ffma_coldot_grad_bt%d", bt, bt);
            ctx->path = buf;
        } else {
            {
                KernelTimer kt(ctx, KIND_GRAD);
                rc = csr_gradient(ctx->csr, c, ctx->r, ctx->q, dayStride, nullptr, eta, bp, bp, dl, d, ctx->Np,
                                  ctx->stream, &ctx->launches, opt.G, opt.eps);
            }
            if (rc) return fail(ctx, rc, "CSR scratch allocation failed");
            char buf[96];
            snprintf(buf, sizeof buf, "csr_fwd_bp%d+csr_grad_bp%d", bp, bp);
            ctx->path = buf;
        }
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(ctx, DODE_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
    return DODE_OK;
}

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

void dode_destroy(dode_ctx* ctx) {
    if (!ctx) return;
    sync_all(ctx);
    if (ctx->s_h2d) cudaStreamDestroy(ctx->s_h2d);
    if (ctx->s_d2h) cudaStreamDestroy(ctx->s_d2h);
    if (ctx->s_sc) cudaStreamDestroy(ctx->s_sc);
    if (ctx->s_ga) cudaStreamDestroy(ctx->s_ga);
    for (int i = 0; i < 2; ++i) { if (ctx->ev_scat[i]) cudaEventDestroy(ctx->ev_scat[i]); if (ctx->ev_gath[i]) cudaEventDestroy(ctx->ev_gath[i]); }
    if (ctx->ev_h2d) cudaEventDestroy(ctx->ev_h2d);
    if (ctx->ev_fence) cudaEventDestroy(ctx->ev_fence);
    for (int i = 0; i < 2; ++i) { if (ctx->ev_step[i]) cudaEventDestroy(ctx->ev_step[i]); if (ctx->ev_d2h[i]) cudaEventDestroy(ctx->ev_d2h[i]); }
    cudaFree(ctx->stage_x); cudaFree(ctx->stage_q);
    for (TcBuf* tb : {&ctx->tcb, &ctx->lane[0].buf, &ctx->lane[1].buf}) {
        cudaFree(tb->part);
        cudaFree(tb->Qg_full); cudaFree(tb->Qg_lo); cudaFree(tb->rp_full); cudaFree(tb->rp_lo);
    }
    for (Lane& ln : ctx->lane) {
        if (ln.st) cudaStreamDestroy(ln.st);
        if (ln.done) cudaEventDestroy(ln.done);
        if (ln.entry) cudaEventDestroy(ln.entry);
    }
    cudaFree(ctx->Ag); cudaFree(ctx->Af); cudaFree(ctx->G); cudaFree(ctx->q); cudaFree(ctx->x); cudaFree(ctx->r); cudaFree(ctx->Qb);
    for (auto& p : ctx->ev_pending) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    for (auto e : ctx->ev_pool) cudaEventDestroy(e);
    cudaFree(ctx->d_part); cudaFree(ctx->d_obj); cudaFree(ctx->d_mom); cudaFree(ctx->pu); cudaFree(ctx->pv); cudaFree(ctx->pw);
    csr_free(ctx->csr);
    delete ctx;
}

int dode_create(dode_ctx** out, const dode_dims* dims, const dode_dar* R, const int32_t* labels, const float* x,
                float q0, void* stream) {
    dode_ctx* ctx = nullptr;   // errors before allocation go to the thread-local buffer
    if (!out) return fail(ctx, DODE_EINVAL, "out is null");
    *out = nullptr;
    if (!dims || !R || !labels || !x) return fail(ctx, DODE_EINVAL, "null argument");
    const dode_dims d = *dims;
    if (d.N < 1 || d.L < 1 || d.T < 1 || d.H < 0 || d.C < 1 || d.D < 1)
        return fail(ctx, DODE_EINVAL, "dims must be positive (N=%d L=%d T=%d H=%d C=%d D=%d)", d.N, d.L, d.T, d.H, d.C, d.D);
    if (d.storage != DODE_DENSE && d.storage != DODE_CSR) return fail(ctx, DODE_EINVAL, "unknown storage %d", d.storage);
    if (d.T > 65535) return fail(ctx, DODE_EINVAL, "T=%d exceeds 65535 (the time index rides on grid.y)", d.T);
    if (d.storage == DODE_DENSE && !R->dense) return fail(ctx, DODE_EINVAL, "R->dense is null");
    if (d.storage == DODE_CSR && (!R->blk_off || !R->row_ptr || (R->nnz > 0 && (!R->col_idx || !R->val)) || R->nnz < 0))
        return fail(ctx, DODE_EINVAL, "CSR arrays are null or nnz < 0");
    for (int i = 0; i < d.D; ++i)
        if (labels[i] < 0 || labels[i] >= d.C) return fail(ctx, DODE_EINVAL, "labels[%d]=%d not in [0,%d)", i, labels[i], d.C);
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail(ctx, DODE_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
    if (major != 10) return fail(ctx, DODE_ECUDA, "this library is built for sm_100a only (device is sm_%d0)", major);

    dode_ctx* c = new (std::nothrow) dode_ctx();
    if (!c) return fail(ctx, DODE_ENOMEM, "host allocation failed");
    c->dm = d;
    c->Np = d.storage == DODE_DENSE ? pad_dim(d.N) : round_up(d.N, 4);
    c->Lp = d.storage == DODE_DENSE ? pad_dim(d.L) : d.L;
    c->stream = (cudaStream_t)stream;
    c->labels.assign(labels, labels + d.D);
    c->stamp.assign(d.D, 0);
    c->day_last_id.assign(d.D, 0);
    c->day_last_lane.assign(d.D, -1);
    ctx = c;
#define CUC(call)                                                                                          \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess) {                                                                           \
            int code_ = fail(nullptr, e_ == cudaErrorMemoryAllocation ? DODE_ENOMEM : DODE_ECUDA, "%s: %s", \
                             #call, cudaGetErrorString(e_));                                               \
            dode_destroy(c);                                                                               \
            cudaGetLastError();                                                                            \
            return code_;                                                                                  \
        }                                                                                                  \
    } while (0)
    const size_t TNp = (size_t)d.T * c->Np, TL = (size_t)d.T * d.L;
    CUC(cudaMalloc(&c->q, (size_t)d.D * TNp * sizeof(float)));
    CUC(cudaMalloc(&c->x, (size_t)d.D * TL * sizeof(float)));
    CUC(cudaMalloc(&c->d_obj, ((size_t)d.D + 8) * sizeof(double)));
    CUC(cudaMalloc(&c->pu, TNp * sizeof(float)));
    CUC(cudaMalloc(&c->pv, (size_t)d.T * c->Lp * sizeof(float)));
    CUC(cudaMalloc(&c->pw, (size_t)d.T * d.N * sizeof(float)));
    CUC(cudaMemcpyAsync(c->x, x, (size_t)d.D * TL * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    fill_state<<<1184, 256, 0, c->stream>>>(c->q, (size_t)d.D * d.T, d.N, c->Np, q0);
    c->launches++;
    if (d.storage == DODE_DENSE) {
        // a0: the two packed copies of the operator (kernels_dense.cuh); the caller's tensor is not kept
        const size_t total = (size_t)d.C * cluster_floats(c);
        const long blocks = (long)d.C * d.T * (d.H + 1);
        CUC(cudaMalloc(&c->Ag, total * sizeof(float)));
        CUC(cudaMalloc(&c->Af, total * sizeof(float)));
        pack_departure_major<<<148 * 16, 256, 0, c->stream>>>(R->dense, c->Ag, blocks, d.T, d.H, d.L, d.N, c->Lp, c->Np);
        pack_arrival_major<<<dim3((unsigned)blocks, ceil_div(c->Lp, 32), ceil_div(c->Np, 32)), 256, 0, c->stream>>>(
            R->dense, c->Af, d.T, d.H, d.L, d.N, c->Lp, c->Np);
        c->launches += 2;
        int rc = tc_setup(c);
        if (rc) { snprintf(g_create_err, 512, "%s", c->err); dode_destroy(c); cudaGetLastError(); return rc; }
    } else {
        int rc = csr_build(c->csr, d, *R, c->stream, g_create_err);
        if (rc) { dode_destroy(c); cudaGetLastError(); return rc; }
    }
    CUC(cudaStreamSynchronize(c->stream));   // caller may free its buffers on return
    CUC(cudaGetLastError());
#undef CUC
    *out = c;
    return DODE_OK;
}

// a plain step after streaming steps: the gathers of q on s_ga (beside the ctx stream) must have read their days first
static int fence_streaming(dode_ctx* ctx) {
    if (!ctx->plain_since_host && ctx->s_ga)
        for (int i = 0; i < 2; ++i) CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_gath[i], 0));
    ctx->plain_since_host = true;
    return DODE_OK;
}

int dode_spgd_step(dode_ctx* ctx, const int32_t* days, int32_t n, float eta) {
    if (!ctx) return DODE_EINVAL;
    int c = 0, rc;
    if ((rc = validate_days(ctx, days, n, true, &c))) return rc;
    if ((rc = fence_streaming(ctx))) return rc;
    return step_impl(ctx, days, n, eta, c, StepOpt(), true);
}

int dode_join(dode_ctx* ctx) {
    if (!ctx) return DODE_EINVAL;
    return join_lanes(ctx);
}

int dode_set_option(dode_ctx* ctx, int32_t option, int32_t value) {
    if (!ctx) return DODE_EINVAL;
    switch (option) {
        case DODE_OPT_TC_MIN_B:
            if (value < 0) return fail(ctx, DODE_EINVAL, "DODE_OPT_TC_MIN_B must be >= 0");
            ctx->tc_min_b = value;
            return DODE_OK;
        case DODE_OPT_LANES:
            if (value != 0 && value != 1) return fail(ctx, DODE_EINVAL, "DODE_OPT_LANES must be 0 or 1");
            ctx->lanes_on = value != 0;
            return join_lanes(ctx);
        case DODE_OPT_TC_KSPLIT:
            if (value < 0 || value > 32) return fail(ctx, DODE_EINVAL, "DODE_OPT_TC_KSPLIT must be in [0, 32]");
            ctx->opt_ksplit = value;
            return DODE_OK;
        case DODE_OPT_TC_BSTAGES:
            if (value != 0 && (value < 2 || value > 8)) return fail(ctx, DODE_EINVAL, "DODE_OPT_TC_BSTAGES must be 0 or in [2, 8]");
            ctx->opt_bstages = value;
            return DODE_OK;
        case DODE_OPT_TC_PAIR:
            if (value < 0 || value > 2) return fail(ctx, DODE_EINVAL, "DODE_OPT_TC_PAIR must be 0, 1 or 2");
            ctx->opt_pair = value;
            return DODE_OK;
        case DODE_OPT_PDL:
            if (value != 0 && value != 1) return fail(ctx, DODE_EINVAL, "DODE_OPT_PDL must be 0 or 1");
            ctx->opt_pdl = value != 0;
            return DODE_OK;
        default:
            return fail(ctx, DODE_EINVAL, "unknown option %d", option);
    }
}

int dode_reserve(dode_ctx* ctx, int32_t max_days) {
    if (!ctx) return DODE_EINVAL;
    if (max_days < 1) return fail(ctx, DODE_EINVAL, "max_days must be >= 1");
    const dode_dims& d = ctx->dm;
    int rc;
    if (d.storage == DODE_CSR) {
        const int bp = csr_bp(std::min<int>(max_days, kCsrMaxDays));
        if ((rc = ensure_buf(ctx, &ctx->r, &ctx->r_cap, (size_t)d.T * ctx->Lp * std::max(bp, 64)))) return rc;
        if ((rc = csr_ensure(ctx->csr, d, ctx->Np, std::max(bp, 64), ctx->stream))) return fail(ctx, rc, "CSR scratch allocation failed");
    } else {
        const int w = round_up(std::min<int>(max_days, kMaxDays), 16);
        const size_t dayStride = (size_t)d.T * ctx->Np;
        // FFMA panels (b < DODE_OPT_TC_MIN_B, and dode_objective's sub-batches of 64 days)
        if ((rc = ensure_buf(ctx, &ctx->r, &ctx->r_cap, (size_t)d.T * ctx->Lp * std::max(w, 64)))) return rc;
        if ((rc = ensure_buf(ctx, &ctx->Qb, &ctx->qb_cap, dayStride * std::max(w, 64)))) return rc;
        if (ctx->tc_ready && ctx->tc_min_b > 0 && max_days >= ctx->tc_min_b) {
            for (Lane& ln : ctx->lane)
                if ((rc = lane_init(ctx, ln))) return rc;
            size_t part = 0;
            int rows = 0, bn_max = 16;
            for (int n = 1; n <= std::min<int>(max_days, kMaxDays); ++n) {
                int ds, bn;
                tc_day_groups(ctx, n, &ds, &bn);
                part = std::max(part, tc_geometry(ctx, bn, ds).part_floats);
                rows = std::max(rows, ds * bn);
                bn_max = std::max(bn_max, bn);
            }
            struct { TcBuf* tb; cudaStream_t st; } bufs[3] = {{&ctx->tcb, ctx->stream}, {&ctx->lane[0].buf, ctx->lane[0].st},
                                                              {&ctx->lane[1].buf, ctx->lane[1].st}};
            for (auto& b : bufs) {
                if ((rc = tc_ensure(ctx, *b.tb, b.st, bn_max, rows))) return rc;
                if ((rc = tc_ensure_part(ctx, *b.tb, b.st, part))) return rc;
            }
        }
    }
    CU(sync_all(ctx));
    CU(cudaGetLastError());
    return DODE_OK;
}

int dode_adagrad_step(dode_ctx* ctx, const int32_t* days, int32_t n, float eta, float eps, const uint8_t* row_mask) {
    if (!ctx) return DODE_EINVAL;
    int c = 0, rc;
    if ((rc = validate_days(ctx, days, n, true, &c))) return rc;
    if (!(eps > 0.f) || !(eta > 0.f)) return fail(ctx, DODE_EINVAL, "eta and eps must be positive");
    const dode_dims& d = ctx->dm;
    if (!ctx->G) {
        const size_t bytes = (size_t)d.D * d.T * ctx->Np * sizeof(float);
        CU(cudaMalloc(&ctx->G, bytes));
        CU(cudaMemsetAsync(ctx->G, 0, bytes, ctx->stream));
    }
    StepOpt opt;
    opt.mask = row_mask; opt.G = ctx->G; opt.eps = eps;
    if ((rc = fence_streaming(ctx))) return rc;
    return step_impl(ctx, days, n, eta, c, opt);
}

int dode_adagrad_reset(dode_ctx* ctx) {
    if (!ctx) return DODE_EINVAL;
    if (ctx->G) CU(cudaMemsetAsync(ctx->G, 0, (size_t)ctx->dm.D * ctx->dm.T * ctx->Np * sizeof(float), ctx->stream));
    return DODE_OK;
}

// staging <-> state for the streaming step: x[day_i] <- stage[i] (scatter) / stage[i] <- q[day_i] without the pad columns
__global__ void __launch_bounds__(256)
stage_scatter_x(const float* __restrict__ stage, float* __restrict__ x, long TL, const __grid_constant__ DayList dl) {
    const float* src = stage + (size_t)blockIdx.y * TL;
    float* dst = x + (size_t)dl.day[blockIdx.y] * TL;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < TL; i += (long)gridDim.x * blockDim.x) dst[i] = src[i];
}
__global__ void __launch_bounds__(256)
stage_gather_q(const float* __restrict__ q, float* __restrict__ stage, int T, int N, int Np, const __grid_constant__ DayList dl) {
    const float* src = q + (size_t)dl.day[blockIdx.y] * T * Np;
    float* dst = stage + (size_t)blockIdx.y * T * N;
    const long total = (long)T * N;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const long t = i / N;
        dst[i] = src[t * Np + (i - t * N)];
    }
}

// device staging of the streaming step: two halves each, ping-pong over calls
static int ensure_staging(dode_ctx* ctx, int n) {
    const dode_dims& d = ctx->dm;
    const size_t TL = (size_t)d.T * d.L, TN = (size_t)d.T * d.N;
    if (ctx->stage_x_cap >= TL * n && ctx->stage_q_cap >= TN * n) return DODE_OK;
    CU(sync_all(ctx));
    cudaFree(ctx->stage_x); cudaFree(ctx->stage_q);
    ctx->stage_x = ctx->stage_q = nullptr; ctx->stage_x_cap = ctx->stage_q_cap = 0;
    CU(cudaMalloc(&ctx->stage_x, 2 * TL * n * sizeof(float)));
    CU(cudaMalloc(&ctx->stage_q, 2 * TN * n * sizeof(float)));
    ctx->stage_x_cap = TL * n; ctx->stage_q_cap = TN * n;
    return DODE_OK;
}

int dode_spgd_step_host(dode_ctx* ctx, const int32_t* days, int32_t n, float eta, const float* x_host, float* q_host) {
    if (!ctx) return DODE_EINVAL;
    int c = 0, rc;
    if ((rc = validate_days(ctx, days, n, true, &c))) return rc;
    if (!x_host || !q_host) return fail(ctx, DODE_EINVAL, "x_host or q_host is null");
    // (consecutive streaming steps keep alternating on the internal step streams like plain ones; the lanes are joined
    // into the ctx stream only at the transition from plain calls, for the fence below)
    if (ctx->plain_since_host && (rc = join_lanes(ctx))) return rc;
    const dode_dims& d = ctx->dm;
    const size_t TL = (size_t)d.T * d.L, TN = (size_t)d.T * d.N;
    if (!ctx->s_h2d) {
        CU(cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->s_sc, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->s_ga, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&ctx->ev_h2d, cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&ctx->ev_step[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_d2h[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_scat[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_gath[i], cudaEventDisableTiming));
        }
        CU(cudaEventCreateWithFlags(&ctx->ev_fence, cudaEventDisableTiming));
    }
    if (ctx->plain_since_host) {      // earlier steps on the ctx stream / the lanes may still read x or write q of these days
        CU(cudaEventRecord(ctx->ev_fence, ctx->stream));
        CU(cudaStreamWaitEvent(ctx->s_sc, ctx->ev_fence, 0));
        ctx->plain_since_host = false;
    }
    if ((rc = ensure_staging(ctx, n))) return rc;
    // One-deep software pipeline over calls i: upload(i+1) || step(i) || download(i-1), on five streams:
    //   s_h2d / s_d2h  carry ONLY the PCIe copies, so each copy engine runs them back to back (a kernel between two copies
    //                  on a copy stream left the engine idle for the kernel plus two engine hand-overs per call)
    //   s_sc / s_ga    scatter of the uploaded counts into x / gather of the updated q into the download buffer: small
    //                  kernels beside the steps, off the ctx stream, which carries only the SPGD kernels
    // Staging buffers ping-pong over calls (half `me` = call parity).  Orderings (events in stream order cover every
    // earlier call of the same parity):
    //   upload(i)   after scatter(i-2), the last reader of x-staging half `me`
    //   scatter(i)  after upload(i); after step(i-2); after step(i-1) if the calls share a day (it still reads that x)
    //   step(i)     after scatter(i); after gather(i-2); after gather(i-1) if the calls share a day (it still reads that q)
    //   gather(i)   after step(i); after download(i-2), the last reader of q-staging half `me`
    //   download(i) after gather(i)
    const int me = (int)(ctx->host_calls & 1), other = me ^ 1;
    const bool two = ctx->host_calls >= 2;
    bool shares_day = false;                       // validate_days stamped this call's days with stamp_id
    for (int32_t pd : ctx->prev_days) shares_day |= ctx->stamp[pd] == ctx->stamp_id;
    float* sx = ctx->stage_x + (size_t)me * ctx->stage_x_cap;
    float* sq = ctx->stage_q + (size_t)me * ctx->stage_q_cap;
    if (two) CU(cudaStreamWaitEvent(ctx->s_h2d, ctx->ev_scat[me], 0));
    CU(cudaMemcpyAsync(sx, x_host, TL * n * sizeof(float), cudaMemcpyHostToDevice, ctx->s_h2d));
    CU(cudaEventRecord(ctx->ev_h2d, ctx->s_h2d));
    CU(cudaStreamWaitEvent(ctx->s_sc, ctx->ev_h2d, 0));
    if (two) CU(cudaStreamWaitEvent(ctx->s_sc, ctx->ev_step[me], 0));
    if (shares_day) CU(cudaStreamWaitEvent(ctx->s_sc, ctx->ev_step[other], 0));
    for (int off = 0; off < n; off += kMaxDays) {
        DayList dl; dl.n = std::min(kMaxDays, n - off);
        std::memcpy(dl.day, days + off, sizeof(int) * dl.n);
        stage_scatter_x<<<dim3(std::min<long>(64, ceil_div((long)TL, 256)), dl.n), 256, 0, ctx->s_sc>>>(
            sx + TL * off, ctx->x, (long)TL, dl);
        ctx->launches++;
    }
    CU(cudaEventRecord(ctx->ev_scat[me], ctx->s_sc));
    CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_scat[me], 0));
    if (two) CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_gath[me], 0));
    if (shares_day) CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_gath[other], 0));
    if ((rc = step_impl(ctx, days, n, eta, c, StepOpt(), true))) return rc;
    if (ctx->lanes_used) {                        // the step ran on internal step streams: the gather follows those
        for (int li = 0; li < 2; ++li)
            if (ctx->lanes_used & (1u << li)) CU(cudaStreamWaitEvent(ctx->s_ga, ctx->lane[li].done, 0));
        CU(cudaEventRecord(ctx->ev_step[me], ctx->s_ga));
    } else {
        CU(cudaEventRecord(ctx->ev_step[me], ctx->stream));
        CU(cudaStreamWaitEvent(ctx->s_ga, ctx->ev_step[me], 0));
    }
    if (two) CU(cudaStreamWaitEvent(ctx->s_ga, ctx->ev_d2h[me], 0));
    for (int off = 0; off < n; off += kMaxDays) {
        DayList dl; dl.n = std::min(kMaxDays, n - off);
        std::memcpy(dl.day, days + off, sizeof(int) * dl.n);
        stage_gather_q<<<dim3(std::min<long>(64, ceil_div((long)TN, 256)), dl.n), 256, 0, ctx->s_ga>>>(
            ctx->q, sq + TN * off, d.T, d.N, ctx->Np, dl);
        ctx->launches++;
    }
    CU(cudaEventRecord(ctx->ev_gath[me], ctx->s_ga));
    CU(cudaStreamWaitEvent(ctx->s_d2h, ctx->ev_gath[me], 0));
    CU(cudaMemcpyAsync(q_host, sq, TN * n * sizeof(float), cudaMemcpyDeviceToHost, ctx->s_d2h));
    CU(cudaEventRecord(ctx->ev_d2h[me], ctx->s_d2h));
    ctx->prev_days.assign(days, days + n);
    ctx->host_calls++;
    CU(cudaGetLastError());
    return DODE_OK;
}

int dode_objective(dode_ctx* ctx, const int32_t* days, int32_t n, double* per_day, double* total) {
    if (!ctx) return DODE_EINVAL;
    const dode_dims& d = ctx->dm;
    std::vector<int32_t> all;
    if (!days) {
        all.resize(d.D);
        for (int i = 0; i < d.D; ++i) all[i] = i;
        days = all.data();
        n = d.D;
    }
    int rc;
    if ((rc = validate_days(ctx, days, n, false, nullptr))) return rc;
    CU(sync_all(ctx));                        // pending streamed uploads of x belong to the state being evaluated
    // group positions by cluster, evaluate in sub-batches; d_obj[i] receives f of days[i]
    constexpr int kObjBatch = 64;
    const long rows = (long)d.T * ctx->Lp;
    const int rowsPerBlock = 2048, nchunks = ceil_div(rows, rowsPerBlock);
    if (ctx->part_cap < (size_t)nchunks * kObjBatch) {
        if (ctx->d_part) CU(cudaFree(ctx->d_part));
        ctx->d_part = nullptr;
        CU(cudaMalloc(&ctx->d_part, (size_t)nchunks * kObjBatch * sizeof(double)));
        ctx->part_cap = (size_t)nchunks * kObjBatch;
    }
    std::vector<double> host(n), tmp(n);
    std::vector<int> pos, order;                 // order[k] = position in `days` of the k-th result on the device
    order.reserve(n);
    for (int c = 0; c < d.C; ++c) {
        pos.clear();
        for (int i = 0; i < n; ++i)
            if (ctx->labels[days[i]] == c) pos.push_back(i);
        for (size_t off = 0; off < pos.size(); off += kObjBatch) {
            DayList dl;
            dl.n = (int)std::min<size_t>(kObjBatch, pos.size() - off);
            for (int j = 0; j < dl.n; ++j) dl.day[j] = days[pos[off + j]];
            int bt, bp;
            if ((rc = forward_batch(ctx, c, dl, &bt, &bp))) return rc;
            sumsq_partial<<<dim3(nchunks, ceil_div(dl.n, 32)), kThreads, 0, ctx->stream>>>(ctx->r, ctx->d_part, rows, bp,
                                                                                         dl.n, rowsPerBlock);
            sumsq_final<<<ceil_div(dl.n, 64), 64, 0, ctx->stream>>>(ctx->d_part, ctx->d_obj + order.size(), nchunks, dl.n);
            ctx->launches += 2;
            for (int j = 0; j < dl.n; ++j) order.push_back(pos[off + j]);
        }
    }
    // one download and one host synchronisation for the whole list (d_obj holds D + 8 doubles, n <= D)
    CU(cudaMemcpyAsync(tmp.data(), ctx->d_obj, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    for (int k = 0; k < n; ++k) host[order[k]] = tmp[k];
    CU(cudaGetLastError());
    double tot = 0.0;
    for (int i = 0; i < n; ++i) tot += host[i];
    if (per_day) std::memcpy(per_day, host.data(), sizeof(double) * n);
    if (total) *total = tot;
    return DODE_OK;
}

int dode_r2(dode_ctx* ctx, const int32_t* days, int32_t n, double* per_day, double* mean) {
    if (!ctx) return DODE_EINVAL;
    const dode_dims& d = ctx->dm;
    std::vector<int32_t> all;
    if (!days) {
        all.resize(d.D);
        for (int i = 0; i < d.D; ++i) all[i] = i;
        days = all.data();
        n = d.D;
    }
    if (n <= 0) return fail(ctx, DODE_EINVAL, "n <= 0");
    std::vector<double> f(n), mom(2 * (size_t)n);
    int rc = dode_objective(ctx, days, n, f.data(), nullptr);            // validates the list (distinct: n <= D), SS_res per day
    if (rc) return rc;
    if (!ctx->d_mom) CU(cudaMalloc(&ctx->d_mom, 2 * (size_t)d.D * sizeof(double)));
    const long TL = (long)d.T * d.L;
    for (int off = 0; off < n; off += kMaxDays) {
        DayList dl; dl.n = std::min(kMaxDays, n - off);
        std::memcpy(dl.day, days + off, sizeof(int) * dl.n);
        x_moments<<<dl.n, kThreads, 0, ctx->stream>>>(ctx->x, TL, ctx->d_mom + 2 * (size_t)off, dl);
        ctx->launches++;
    }
    CU(cudaMemcpyAsync(mom.data(), ctx->d_mom, sizeof(double) * 2 * n, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));              // one host round trip for the whole list
    double acc = 0.0;
    for (int i = 0; i < n; ++i) {
        const double ss_tot = mom[2 * i + 1] - mom[2 * i] * mom[2 * i] / (double)TL;
        const double r2 = 1.0 - f[i] / ss_tot;
        if (per_day) per_day[i] = r2;
        acc += r2;
    }
    CU(cudaGetLastError());
    if (mean) *mean = acc / n;
    return DODE_OK;
}

static int copy_q(dode_ctx* ctx, int32_t day, float* out, const float* in, int32_t is_device) {
    const dode_dims& d = ctx->dm;
    if (day < 0 || day >= d.D) return fail(ctx, DODE_EINVAL, "day %d out of range [0,%d)", day, d.D);
    if (!out && !in) return fail(ctx, DODE_EINVAL, "null buffer");
    CU(sync_all(ctx));
    float* qd = ctx->q + (size_t)day * d.T * ctx->Np;
    if (out)
        CU(cudaMemcpy2DAsync(out, d.N * sizeof(float), qd, ctx->Np * sizeof(float), d.N * sizeof(float), d.T,
                             is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    else
        CU(cudaMemcpy2DAsync(qd, ctx->Np * sizeof(float), in, d.N * sizeof(float), d.N * sizeof(float), d.T,
                             is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return DODE_OK;
}

int dode_get_q(dode_ctx* ctx, int32_t day, float* out, int32_t is_device) {
    if (!ctx) return DODE_EINVAL;
    if (!out) return fail(ctx, DODE_EINVAL, "out is null");
    return copy_q(ctx, day, out, nullptr, is_device);
}

int dode_set_q(dode_ctx* ctx, int32_t day, const float* in, int32_t is_device) {
    if (!ctx) return DODE_EINVAL;
    if (!in) return fail(ctx, DODE_EINVAL, "in is null");
    return copy_q(ctx, day, nullptr, in, is_device);
}

// v[T][opitch] = rho_c * (padded u in ctx->pu), minibatch 1 through the production kernels
static int apply_padded(dode_ctx* ctx, int c, float* v, int opitch) {
    const dode_dims& d = ctx->dm;
    DayList dl; dl.n = 1; dl.day[0] = 0;
    if (d.storage == DODE_DENSE) {
        BandArgs a = band_args(ctx, c, true, 1);
        a.B = ctx->pu; a.out = v; a.opitch = opitch;
        return launch_band<1, EPI_STORE>(ctx, 15, a, 1, dl, KIND_FWD);
    }
    int rc = csr_forward(ctx->csr, c, ctx->pu, 0, nullptr, v, 32, 1, dl, d, ctx->Np, ctx->stream, &ctx->launches);
    return rc ? fail(ctx, rc, "CSR scratch allocation failed") : DODE_OK;
}

// u[T][N] = rho_c^T * (padded v in ctx->pv, [T][Lp])
static int apply_t_padded(dode_ctx* ctx, int c, float* u) {
    const dode_dims& d = ctx->dm;
    DayList dl; dl.n = 1; dl.day[0] = 0;
    if (d.storage == DODE_DENSE) {
        BandArgs a = band_args(ctx, c, false, 1);
        a.B = ctx->pv; a.out = u; a.opitch = d.N;
        return launch_band<1, EPI_STORE>(ctx, 15, a, 1, dl, KIND_GRAD);
    }
    int rc = csr_gradient(ctx->csr, c, ctx->pv, nullptr, 0, u, 0.f, 32, 1, dl, d, ctx->Np, ctx->stream, &ctx->launches);
    return rc ? fail(ctx, rc, "CSR scratch allocation failed") : DODE_OK;
}

int dode_apply(dode_ctx* ctx, int32_t c, const float* u, float* v) {
    if (!ctx) return DODE_EINVAL;
    const dode_dims& d = ctx->dm;
    if (c < 0 || c >= d.C || !u || !v) return fail(ctx, DODE_EINVAL, "bad cluster or null buffer");
    if (int rj = join_lanes(ctx)) return rj;
    scale_pad<<<592, 256, 0, ctx->stream>>>(u, ctx->pu, (size_t)d.T, d.N, ctx->Np, nullptr);
    ctx->launches++;
    int rc = apply_padded(ctx, c, v, d.L);
    if (rc) return rc;
    CU(cudaGetLastError());
    return DODE_OK;
}

int dode_apply_t(dode_ctx* ctx, int32_t c, const float* v, float* u) {
    if (!ctx) return DODE_EINVAL;
    const dode_dims& d = ctx->dm;
    if (c < 0 || c >= d.C || !u || !v) return fail(ctx, DODE_EINVAL, "bad cluster or null buffer");
    if (int rj = join_lanes(ctx)) return rj;
    scale_pad<<<592, 256, 0, ctx->stream>>>(v, ctx->pv, (size_t)d.T, d.L, ctx->Lp, nullptr);
    ctx->launches++;
    int rc = apply_t_padded(ctx, c, u);
    if (rc) return rc;
    CU(cudaGetLastError());
    return DODE_OK;
}

int dode_lipschitz(dode_ctx* ctx, int32_t c, int32_t iters, double* L_out) {
    if (!ctx) return DODE_EINVAL;
    const dode_dims& d = ctx->dm;
    if (c < 0 || c >= d.C || iters < 1 || !L_out) return fail(ctx, DODE_EINVAL, "bad cluster, iters or null output");
    if (int rj = join_lanes(ctx)) return rj;
    double* nrm = ctx->d_obj + d.D;       // [0] = |w|^2, [1] = |v|^2
    const size_t TN = (size_t)d.T * d.N, TLp = (size_t)d.T * ctx->Lp;
    fill_f32<<<592, 256, 0, ctx->stream>>>(ctx->pw, TN, 1.f);
    ctx->launches++;
    for (int it = 0; it < iters; ++it) {
        sumsq_single<<<1, 1024, 0, ctx->stream>>>(ctx->pw, TN, nrm);
        scale_pad<<<592, 256, 0, ctx->stream>>>(ctx->pw, ctx->pu, (size_t)d.T, d.N, ctx->Np, nrm);
        ctx->launches += 2;
        int rc = apply_padded(ctx, c, ctx->pv, ctx->Lp);          // pad columns come out as 0
        if (rc) return rc;
        sumsq_single<<<1, 1024, 0, ctx->stream>>>(ctx->pv, TLp, nrm + 1);
        ctx->launches++;
        if ((rc = apply_t_padded(ctx, c, ctx->pw))) return rc;
    }
    CU(cudaMemcpyAsync(L_out, nrm + 1, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(sync_all(ctx));
    CU(cudaGetLastError());
    return DODE_OK;
}

// shared by dode_dar_build (od_ptr == nullptr: one path per OD, p = 1) and dode_assignment_build
static int build_operator(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* od_ptr, const int32_t* path_ptr,
                          const int32_t* path_links, const float* link_len, const float* speed, double dt, double theta,
                          float* R_out, void* stream) {
    dode_ctx* ctx = nullptr;                   // no ctx: errors go to the thread-local buffer (dode_last_error(NULL))
    if (N < 1 || L < 1 || T < 1 || H < 0 || !(dt > 0.0)) return fail(ctx, DODE_EINVAL, "dims must be positive and dt > 0");
    if (!path_ptr || !path_links || !link_len || !speed || !R_out) return fail(ctx, DODE_EINVAL, "null argument");
    if (!(theta >= 0.0)) return fail(ctx, DODE_EINVAL, "theta must be >= 0");
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail(ctx, DODE_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
    if (major != 10) return fail(ctx, DODE_ECUDA, "this library is built for sm_100a only (device is sm_%d0)", major);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)T * (H + 1) * L * N * sizeof(float);
    CU(cudaMemsetAsync(R_out, 0, bytes, st));
    const long total = (long)T * N;
    // few, long, dependent double-precision walks per thread: small blocks spread them over all SMs
    const int threads = 64;
    const int blocks = (int)std::min<long>((total + threads - 1) / threads, 148L * 64);
    if (od_ptr)
        assignment_build_dense<<<blocks, threads, 0, st>>>(N, L, T, H, od_ptr, path_ptr, path_links, link_len, speed, dt, theta, R_out);
    else
        dar_build_dense<<<blocks, threads, 0, st>>>(N, L, T, H, path_ptr, path_links, link_len, speed, dt, R_out);
    CU(cudaGetLastError());
    return DODE_OK;
}

int dode_dar_build(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* path_ptr, const int32_t* path_links,
                   const float* link_len, const float* speed, double dt, float* R_out, void* stream) {
    return build_operator(N, L, T, H, nullptr, path_ptr, path_links, link_len, speed, dt, 0.0, R_out, stream);
}

int dode_assignment_build(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* od_ptr, const int32_t* path_ptr,
                          const int32_t* path_links, const float* link_len, const float* speed, double dt, double theta,
                          float* R_out, void* stream) {
    if (!od_ptr) return fail(nullptr, DODE_EINVAL, "od_ptr is null");
    return build_operator(N, L, T, H, od_ptr, path_ptr, path_links, link_len, speed, dt, theta, R_out, stream);
}

int dode_assignment_build_csr(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* od_ptr, const int32_t* path_ptr,
                              const int32_t* path_links, const float* link_len, const float* speed, double dt, double theta,
                              int64_t* blk_off_out, int32_t* row_ptr_out, int32_t* col_idx_out, float* val_out,
                              int64_t cap, int64_t* nnz_out, void* stream) {
    dode_ctx* ctx = nullptr;
    if (N < 1 || L < 1 || T < 1 || H < 0 || !(dt > 0.0)) return fail(ctx, DODE_EINVAL, "dims must be positive and dt > 0");
    if (!path_ptr || !path_links || !link_len || !speed || !nnz_out) return fail(ctx, DODE_EINVAL, "null argument");
    if (!(theta >= 0.0)) return fail(ctx, DODE_EINVAL, "theta must be >= 0");
    if (cap > 0 && (!blk_off_out || !row_ptr_out || !col_idx_out || !val_out)) return fail(ctx, DODE_EINVAL, "null output");
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail(ctx, DODE_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
    if (major != 10) return fail(ctx, DODE_ECUDA, "this library is built for sm_100a only (device is sm_%d0)", major);
    cudaStream_t st = (cudaStream_t)stream;
    const long total = (long)T * N, blocks_sh = (long)T * (H + 1);
    const int threads = 64;
    const int grid = (int)std::min<long>((total + threads - 1) / threads, 148L * 64);
    int32_t* cnt = nullptr; int64_t* offs = nullptr; void* tmp = nullptr; int64_t* d_nu = nullptr;
    unsigned long long *k0 = nullptr, *k1 = nullptr; float *v0 = nullptr, *v1 = nullptr;
    int rc = DODE_OK;
    int64_t nt = 0, nu = 0;
    auto cleanup = [&]() { cudaFree(cnt); cudaFree(offs); cudaFree(tmp); cudaFree(d_nu); cudaFree(k0); cudaFree(k1); cudaFree(v0); cudaFree(v1); };
#define BCU(call)                                                                                                     \
    do {                                                                                                              \
        cudaError_t e_ = (call);                                                                                      \
        if (e_ != cudaSuccess) {                                                                                      \
            rc = fail(ctx, e_ == cudaErrorMemoryAllocation ? DODE_ENOMEM : DODE_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
            cleanup(); cudaGetLastError();                                                                            \
            return rc;                                                                                                \
        }                                                                                                             \
    } while (0)
    BCU(cudaMalloc(&cnt, (size_t)total * 4));
    BCU(cudaMalloc(&offs, (size_t)(total + 1) * 8));
    BCU(cudaMalloc(&d_nu, 8));
    assignment_tuples<<<grid, threads, 0, st>>>(N, L, T, H, od_ptr, path_ptr, path_links, link_len, speed, dt, theta, cnt,
                                                nullptr, nullptr, nullptr);
    size_t tb_scan = 0;
    cub::DeviceScan::ExclusiveSum(nullptr, tb_scan, cnt, offs, (int)total, st);
    BCU(cudaMalloc(&tmp, tb_scan));
    BCU(cub::DeviceScan::ExclusiveSum(tmp, tb_scan, cnt, offs, (int)total, st));
    int64_t last_off = 0; int32_t last_cnt = 0;
    BCU(cudaMemcpyAsync(&last_off, offs + total - 1, 8, cudaMemcpyDeviceToHost, st));
    BCU(cudaMemcpyAsync(&last_cnt, cnt + total - 1, 4, cudaMemcpyDeviceToHost, st));
    BCU(cudaStreamSynchronize(st));
    nt = last_off + last_cnt;
    if (cap < nt) {                               // the caller sizes its arrays from this
        *nnz_out = nt;
        cleanup();
        return fail(ctx, DODE_ENOMEM, "output capacity %lld is below the %lld shares to emit", (long long)cap, (long long)nt);
    }
    cudaFree(tmp); tmp = nullptr;
    if (!blk_off_out || !row_ptr_out) {           // sizing call on an operator without a single share
        *nnz_out = 0;
        cleanup();
        return DODE_OK;
    }
    if (nt > 0) {
        BCU(cudaMalloc(&k0, (size_t)nt * 8)); BCU(cudaMalloc(&k1, (size_t)nt * 8));
        BCU(cudaMalloc(&v0, (size_t)nt * 4)); BCU(cudaMalloc(&v1, (size_t)nt * 4));
        assignment_tuples<<<grid, threads, 0, st>>>(N, L, T, H, od_ptr, path_ptr, path_links, link_len, speed, dt, theta, cnt,
                                                    offs, k0, v0);
        int bits = 1;
        while (bits < 64 && ((unsigned long long)1 << bits) < (unsigned long long)blocks_sh * L * N) ++bits;
        size_t tb_sort = 0, tb_red = 0;
        cub::DeviceRadixSort::SortPairs(nullptr, tb_sort, k0, k1, v0, v1, nt, 0, bits, st);
        cub::DeviceReduce::ReduceByKey(nullptr, tb_red, k1, k0, v1, val_out, d_nu, cuda::std::plus<>{}, nt, st);
        BCU(cudaMalloc(&tmp, std::max(tb_sort, tb_red)));
        BCU(cub::DeviceRadixSort::SortPairs(tmp, tb_sort, k0, k1, v0, v1, nt, 0, bits, st));
        // equal keys = several paths of one OD over one link in one lag: their shares add up (Eq. 41 summed over the OD's paths)
        BCU(cub::DeviceReduce::ReduceByKey(tmp, tb_red, k1, k0, v1, val_out, d_nu, cuda::std::plus<>{}, nt, st));
        BCU(cudaMemcpyAsync(&nu, d_nu, 8, cudaMemcpyDeviceToHost, st));
        BCU(cudaStreamSynchronize(st));
        csr_cols_from_keys<<<1184, 256, 0, st>>>(k0, nu, N, col_idx_out);
    }
    const long nb = blocks_sh * (L + 1);
    csr_bounds_from_keys<<<(unsigned)((nb + 255) / 256), 256, 0, st>>>(k0, nu, blocks_sh, L, N, blk_off_out, row_ptr_out);
    BCU(cudaStreamSynchronize(st));
    BCU(cudaGetLastError());
#undef BCU
    cleanup();
    *nnz_out = nu;
    return DODE_OK;
}

int dode_probe_fp32_peak(int32_t reps, double* tflops, void* stream) {
    dode_ctx* ctx = nullptr;
    if (reps < 1 || !tflops) return fail(ctx, DODE_EINVAL, "reps < 1 or null output");
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* buf = nullptr;
    CU(cudaMalloc(&buf, 4096));
    const float init[3] = {0.999f, 0.001f, 1.0f};
    cudaError_t e = cudaMemcpyAsync(buf, init, sizeof init, cudaMemcpyHostToDevice, st);
    cudaEvent_t a = nullptr, b = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    const int outer = 2048, blocks = sms * 2, threads = 1024;
    double best = 0.0;
    for (int r = 0; r <= reps && e == cudaSuccess; ++r) {                 // launch 0 is the warm-up
        cudaEventRecord(a, st);
        ffma_peak_probe<<<blocks, threads, 0, st>>>(buf, buf + 8, outer);
        cudaEventRecord(b, st);
        e = cudaEventSynchronize(b);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
        const double fl = 2.0 * kProbeChains * kProbeInner * (double)outer * threads * blocks;
        if (r > 0 && ms > 0.f) best = std::max(best, fl / (ms * 1e-3) / 1e12);
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(buf);
    if (e != cudaSuccess) return fail(ctx, DODE_ECUDA, "ffma_peak_probe: %s", cudaGetErrorString(e));
    *tflops = best;
    return DODE_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// dode_visit_static (include/dode.h): one visit of one day without any allocation.  The residual r [T][L] is the
// visit's only scratch; it lives in g_static_scratch below — one copy per GPU that loads this library, held until the
// process exits.  In HOST code the name g_static_scratch is a host-side stand-in, not a device address: the address a
// kernel can use comes from cudaGetSymbolAddress, looked up once per device with that device current.
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) float g_static_scratch[DODE_STATIC_SCRATCH_FLOATS];

// Alg. 1 line 9, inner part: r[t][l] = sum_{h <= min(H,t)} sum_n R[t-h][h][l][n] q[t-h][n] - x[t][l].
// One warp per (t, l): lanes stride the N columns of each of the (<= H+1) operator rows, then a shuffle reduction.
__global__ void __launch_bounds__(256)
visit_static_residual(int N, int L, int T, int H, const float* __restrict__ R, const float* __restrict__ q,
                      const float* __restrict__ x, float* __restrict__ r) {
    const long w = (long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (w >= (long)T * L) return;
    const int t = (int)(w / L), l = (int)(w % L);
    const int hmax = min(H, t);
    float acc0 = 0.f, acc1 = 0.f;
    for (int h = 0; h <= hmax; ++h) {
        const float* row = R + (((size_t)(t - h) * (H + 1) + h) * L + l) * (size_t)N;
        const float* qs = q + (size_t)(t - h) * N;
        int n = lane;
        for (; n + 32 < N; n += 64) {
            acc0 = fmaf(__ldg(row + n), qs[n], acc0);
            acc1 = fmaf(__ldg(row + n + 32), qs[n + 32], acc1);
        }
        if (n < N) acc0 = fmaf(__ldg(row + n), qs[n], acc0);
    }
    float acc = acc0 + acc1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) r[w] = acc - x[w];
}

// Alg. 1 lines 9-11: g[s][n] = sum_{h <= min(H,T-1-s)} sum_l R[s][h][l][n] r[s+h][l];
// q[s][n] <- max(0, q[s][n] - eta g[s][n]).  The rows (h, l) of departure s are one contiguous slab of R and meet the
// contiguous window r[s*L ..]: row k = h*L + l <-> r[s*L + k].  CTA = 32 columns x 8 row slices, grid (ceil(N/32), T).
__global__ void __launch_bounds__(256)
visit_static_update(int N, int L, int T, int H, const float* __restrict__ R, const float* __restrict__ r,
                    float* __restrict__ q, float eta) {
    __shared__ float part[8][33];
    const int col = threadIdx.x & 31, ks = threadIdx.x >> 5;
    const int s = blockIdx.y, n = blockIdx.x * 32 + col;
    const int K = (min(H, T - 1 - s) + 1) * L;
    const float* Rs = R + (size_t)s * (H + 1) * L * (size_t)N + n;
    const float* rs = r + (size_t)s * L;
    float acc0 = 0.f, acc1 = 0.f;
    if (n < N) {
        int k = ks;
        for (; k + 8 < K; k += 16) {
            acc0 = fmaf(__ldg(Rs + (size_t)k * N), rs[k], acc0);
            acc1 = fmaf(__ldg(Rs + (size_t)(k + 8) * N), rs[k + 8], acc1);
        }
        if (k < K) acc0 = fmaf(__ldg(Rs + (size_t)k * N), rs[k], acc0);
    }
    part[ks][col] = acc0 + acc1;
    __syncthreads();
    if (ks == 0 && n < N) {
        float g = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) g += part[j][col];
        float* qp = q + (size_t)s * N + n;
        *qp = fmaxf(0.f, *qp - eta * g);
    }
}

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mu;
static float* g_static_ptr[kStaticMaxDevices] = {nullptr};

// Device address of the current device's copy of g_static_scratch (looked up once per device).
static int static_scratch(float** out) {
    dode_ctx* ctx = nullptr;
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(ctx, DODE_EINVAL, "device ordinal %d outside [0, %d)", dev, kStaticMaxDevices);
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return fail(ctx, DODE_ECUDA, "cudaGetSymbolAddress returned a null address on device %d", dev);
        g_static_ptr[dev] = static_cast<float*>(p);
    }
    *out = g_static_ptr[dev];
    return DODE_OK;
}

extern "C" {

int dode_visit_static(int32_t N, int32_t L, int32_t T, int32_t H, const float* R, float* q, const float* x, float eta,
                      void* stream) {
    dode_ctx* ctx = nullptr;
    if (N < 1 || L < 1 || T < 1 || H < 0) return fail(ctx, DODE_EINVAL, "N, L, T must be positive and H >= 0");
    if (!R || !q || !x) return fail(ctx, DODE_EINVAL, "null R, q or x");
    if (!(eta > 0.f)) return fail(ctx, DODE_EINVAL, "eta must be > 0");
    if ((long)T * L > (long)DODE_STATIC_SCRATCH_FLOATS || T > 65535)
        return fail(ctx, DODE_EINVAL,
                    "dode_visit_static: T*L = %ld residual floats (T = %d) exceed the static scratch of %d floats / the "
                    "limit T <= 65535; this entry point allocates nothing — use dode_create + dode_spgd_step",
                    (long)T * L, (int)T, (int)DODE_STATIC_SCRATCH_FLOATS);
    float* r = nullptr;
    const int rc = static_scratch(&r);
    if (rc != DODE_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    visit_static_residual<<<ceil_div((long)T * L, 8), 256, 0, st>>>(N, L, T, H, R, q, x, r);
    visit_static_update<<<dim3(ceil_div(N, 32), T), 256, 0, st>>>(N, L, T, H, R, r, q, eta);
    CU(cudaGetLastError());
    return DODE_OK;
}

int dode_timing_enable(dode_ctx* ctx, int32_t on) {
    if (!ctx) return DODE_EINVAL;
    ctx->timing = on != 0;
    return join_lanes(ctx);
}

int dode_timing_read(dode_ctx* ctx, int32_t kind, double* total_ms, int64_t* launches, int32_t reset) {
    if (!ctx) return DODE_EINVAL;
    if (kind < 0 || kind > 2) return fail(ctx, DODE_EINVAL, "kind must be 0 (forward), 1 (gradient+update) or 2");
    CU(sync_all(ctx));
    for (auto& p : ctx->ev_pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p.a, p.b) == cudaSuccess) { ctx->t_total[p.kind] += ms; ctx->t_count[p.kind]++; }
        ctx->ev_pool.push_back(p.a); ctx->ev_pool.push_back(p.b);
    }
    ctx->ev_pending.clear();
    if (total_ms) *total_ms = ctx->t_total[kind];
    if (launches) *launches = ctx->t_count[kind];
    if (reset) { ctx->t_total[kind] = 0; ctx->t_count[kind] = 0; }
    return DODE_OK;
}

#ifdef DODE_BRINGUP
// bring-up only: the record of waits that gave up (kernels_tc.cuh); not declared in include/dode.h
int dode_bringup_wait_record(int* host64) {
    int z = 0;
    cudaError_t e = cudaMemcpyFromSymbol(host64, tc::g_wait_rec, sizeof(int) * 64);
    cudaMemcpyToSymbol(tc::g_wait_abort, &z, sizeof(int));
    return (int)e;
}
#endif

int64_t dode_launch_count(const dode_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* dode_last_path(const dode_ctx* ctx) { return ctx ? ctx->path.c_str() : ""; }

int dode_sync(dode_ctx* ctx) {
    if (!ctx) return DODE_EINVAL;
    CU(sync_all(ctx));
    CU(cudaGetLastError());
    return DODE_OK;
}

const char* dode_last_error(const dode_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

}  // extern "C"
