/* dode.h — C ABI of the B200-native SPGD/NNLS hot path of Ma & Qian (arXiv 1901.09266).
 *
 * The library solves, day by day, the non-negative least squares problem
 *     min  sum_d || rho_{c(d)} q_d - x_d ||^2   s.t.  q_d >= 0          (Eq. 40/42)
 * by stochastic projected gradient descent (Alg. 1) with the re-scoping of
 * BASELINE.json:north_star (minibatch = days of one cluster; plain projected step; one DAR
 * operator per cluster — DESIGN.md readings A2, A3, A7).
 *
 * Notation: N OD pairs, L observed links, T intervals per day, H max lag,
 * C clusters, D days.  R[c][s][h] is the L x N block that maps departures in interval s to link
 * counts in interval s+h (Table 2: rho entry [(h2-1)|A|+a, (h1-1)Pi+k] with
 * s = h1-1, h = h2-h1).  Blocks with s+h >= T may be present; they are ignored.
 *
 * Conventions: plain C types; every function returns DODE_OK (0) or a negative dode_status;
 * nothing is written to stdout/stderr; no global state (one stated exception: the static scratch array of
 * dode_visit_static); no CPU fallback — every call fails with
 * DODE_ECUDA if no usable sm_100 device/context exists.  "device" pointers are CUDA device
 * pointers valid in the current context (e.g. torch-allocated); "host" pointers are ordinary
 * host memory.  All work is issued on the stream given to dode_create or ordered with it as dode_spgd_step states.  A sticky CUDA error is
 * reported by the next synchronising call.
 */
#ifndef DODE_H_
#define DODE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dode_ctx dode_ctx;

typedef enum dode_status {
    DODE_OK = 0,
    DODE_EINVAL = -1,  /* bad argument; state untouched */
    DODE_ENOMEM = -2,  /* device or host allocation failed */
    DODE_ECUDA = -3    /* CUDA runtime error (text in dode_last_error) */
} dode_status;

enum { DODE_DENSE = 0, DODE_CSR = 1 };

typedef struct dode_dims {
    int32_t N, L, T, H, C, D;
    int32_t storage; /* DODE_DENSE or DODE_CSR */
} dode_dims;

/* The DAR operator of every cluster (the paper's assignment matrix B = delta.rho.p, Eq. 41,
 * PAPER.md:337-340, shared by a cluster's days).
 *   DENSE: dense = device fp32 [C][T][H+1][L][N], n fastest.
 *   CSR  : per (c,s,h) block, rows = links, columns = OD pairs, blocks concatenated in [c][s][h]
 *          order ("coordinate format sparse representation"):
 *            blk_off  device int64 [C*T*(H+1) + 1]  first nnz of each block (blk_off[last] = nnz)
 *            row_ptr  device int32 [C*T*(H+1)][L+1]  row offsets relative to the block start
 *            col_idx  device int32 [nnz]             OD index n, ascending within a row
 *            val      device fp32  [nnz]
 * The library copies/re-packs what it needs during dode_create and keeps no caller pointer. */
typedef struct dode_dar {
    const float* dense;
    const int64_t* blk_off;
    const int32_t* row_ptr;
    const int32_t* col_idx;
    const float* val;
    int64_t nnz;
} dode_dar;

/* a0: store R, labels, x; q[d][s][n] <- q0 ("Initialize x", Alg. 1 line 3).
 *   labels  host   int32 [D], each in [0, C)
 *   x       device fp32  [D][T][L]  (Table 2 link-flow order: entry t*L + l)
 *   stream  cudaStream_t (NULL = legacy default stream)
 * On failure *out is NULL. */
int dode_create(dode_ctx** out, const dode_dims* dims, const dode_dar* R, const int32_t* labels,
                const float* x, float q0, void* stream);

/* a1-a4: one SPGD iteration on the listed days (Alg. 1 lines 8-11):
 *   r = rho_c Q_B - X_B ;  g = rho_c^T r ;  q_d <- max(0, q_d - eta g_d)  for d in days.
 *   days  host int32 [n]; all in [0, D), distinct, same cluster — else DODE_EINVAL, state untouched.
 * Asynchronous; no device->host traffic.  No host synchronisation once the minibatch panels exist: the first step of
 * a given width allocates them (cudaMalloc + a stream synchronisation) unless dode_reserve was called before.
 * Ordering: a step starts after everything that was on the ctx stream when it was called and after every earlier
 * step that shares a day with it.  Steps on disjoint days (the chunks of one epoch) may overlap
 * each other: the library alternates them on two internal streams.  Every other library call is ordered after all
 * earlier steps by itself; work that the CALLER puts on the ctx stream (an event record, a kernel) is ordered after
 * them only once dode_join has been called. */
int dode_spgd_step(dode_ctx* ctx, const int32_t* days, int32_t n, float eta);

/* Makes the ctx stream wait for every step issued so far (asynchronous, no host wait). */
int dode_join(dode_ctx* ctx);

/* Pre-allocates the per-step scratch buffers of dode_spgd_step (minibatch panels of the kernel families the current
 * options select, on the ctx stream and on the two internal step streams) for minibatches of up to max_days days, so
 * that no later dode_spgd_step with n <= max_days allocates or synchronises.  (dode_adagrad_step's accumulator and
 * dode_spgd_step_host's staging halves are allocated by their own first call.)  Synchronises once itself.
 * max_days >= 1. */
int dode_reserve(dode_ctx* ctx, int32_t max_days);

/* Per-ctx kernel-selection options (no process-wide state, nothing is read from the environment).  All of them keep
 * results valid; they exist so that tests and benchmarks can steer every kernel family over every shape.
 *   DODE_OPT_TC_MIN_B   minibatch width from which dense steps use the tcgen05 3xTF32 kernels; 0 = never
 *                       (FFMA kernels for every width).  Default 8.
 *   DODE_OPT_LANES      1 = consecutive plain steps alternate on two internal streams (default), 0 = ctx stream only.
 *   DODE_OPT_TC_KSPLIT  split-K factor of the tcgen05 kernels, 1..32; 0 = automatic (default: split only when the time
 *                       axis is too short to fill the machine).
 *   DODE_OPT_PDL        1 = kernels of a step are chained by programmatic dependent launch (default), 0 = plain
 *                       stream order.
 *   DODE_OPT_TC_BSTAGES stages of the tcgen05 kernels' minibatch-panel (B) ring, 2..8; 0 = automatic (default).  The
 *                       operator (A) ring takes the rest of the shared memory.  (Single-CTA kernels only: the CTA-pair
 *                       kernel's ring geometry is fixed at 4 B stages.)
 *   DODE_OPT_TC_PAIR    tcgen05 kernels for minibatches wider than 64 days: 1 = pairs of CTAs on the two SMs of a TPC
 *                       (tcgen05.mma.cta_group::2 on 256-output tiles, each CTA staging half of the minibatch panel
 *                       tile), an odd last 128-output tile on the single-CTA kernel (default); 2 = pairs only (an odd
 *                       last tile is paired with an idle CTA); 0 = single-CTA kernels only.
 * Unknown option or out-of-range value: DODE_EINVAL, nothing changes.  Asynchronous (orders later steps after earlier
 * ones where the option changes the stream they run on). */
enum { DODE_OPT_TC_MIN_B = 0, DODE_OPT_LANES = 1, DODE_OPT_TC_KSPLIT = 2, DODE_OPT_PDL = 3, DODE_OPT_TC_BSTAGES = 4,
       DODE_OPT_TC_PAIR = 5 };
int dode_set_option(dode_ctx* ctx, int32_t option, int32_t value);

/* NEXT-1 — Alg. 1 as the paper prints it, on the listed days of one cluster:
 *   line 8   B_o = the rows of each day's system selected by row_mask (a chunk of the permuted row range, 398-404)
 *   line 9   g = B_o^T (B_o x - y_o)          == rho^T (mask .* (rho q - x))
 *   line 10  x = Adagrad(x, g, eta)           G += g^2 ; q -= eta g / (sqrt(G) + eps)   ([14]; reading A18)
 *   line 11  x = max(x, 0)
 *   row_mask  device uint8 [n][T][L] indexed by the POSITION in `days` (entry t*L + l, Table 2 link-flow order),
 *             non-zero = row belongs to the chunk; NULL = every row (full-batch Adagrad).  Read during the call's
 *             kernels: keep it alive and unmodified until they have run (stream order is enough).
 *   eta, eps  > 0, else DODE_EINVAL.
 * The accumulator G ([D][T][N] fp32, zero at first use) lives in the ctx; dode_adagrad_reset zeroes it.
 * Same validation, asynchrony and kernels as dode_spgd_step (the mask and the accumulator ride in the epilogues). */
int dode_adagrad_step(dode_ctx* ctx, const int32_t* days, int32_t n, float eta, float eps, const uint8_t* row_mask);
int dode_adagrad_reset(dode_ctx* ctx);

/* The same iteration for a streaming caller (bench.py's end-to-end leg): uploads the n days' counts from x_host
 * ([n][T][L], host; pinned memory makes the copies asynchronous), runs the step, and downloads the n days' updated q
 * into q_host ([n][T][N], host).  ASYNCHRONOUS and pipelined over consecutive calls on two internal copy streams
 * (PCIe copies only) and two helper streams (scatter into x, gather of q):
 * the upload of call i+1 and the download of call i-1 overlap the kernels of call i (calls that share a day are
 * ordered).  x_host must stay valid and q_host is defined only after the next synchronising call (dode_sync,
 * dode_objective, dode_r2, dode_get_q, dode_set_q, dode_lipschitz, dode_timing_read, dode_reserve, dode_destroy): each
 * of them waits for the ctx stream AND for the library's internal step and copy streams. */
int dode_spgd_step_host(dode_ctx* ctx, const int32_t* days, int32_t n, float eta,
                        const float* x_host, float* q_host);

/* a5: f_d = sum_t sum_l r_d[t][l]^2 — no 1/2, no mean (Eq. 42).
 *   days     host int32 [n], or NULL for all D days (then n is ignored); any mix of clusters
 *   per_day  host double [n] (or [D]), nullable
 *   total    host double, nullable
 * fp32 products, fp64 sums.  Synchronises. */
int dode_objective(dode_ctx* ctx, const int32_t* days, int32_t n, double* per_day, double* total);

/* Step 6 "quality check" ("R-square between the observed link flow and estimated link flow",
 * PAPER.md:553): coefficient of determination of the fitted counts of each listed day, observed counts as reference,
 *     R2_d = 1 - sum_t sum_l (x_d - rho q_d)^2 / sum_t sum_l (x_d - mean(x_d))^2      (reading A17).
 *   days     host int32 [n], or NULL for all D days (then n is ignored)
 *   per_day  host double [n] (or [D]), nullable;   mean  host double (average over the listed days), nullable
 * SS_res is dode_objective's value; sums in fp64.  Synchronises. */
int dode_r2(dode_ctx* ctx, const int32_t* days, int32_t n, double* per_day, double* mean);

/* Export / import one day's state in Table 2 order (entry s*N + n).
 * out/in: fp32 [T][N]; is_device != 0 means a device pointer.  Synchronises. */
int dode_get_q(dode_ctx* ctx, int32_t day, float* out, int32_t is_device);
int dode_set_q(dode_ctx* ctx, int32_t day, const float* in, int32_t is_device);

/* v = rho_c u and u = rho_c^T v through the production kernels with minibatch 1.
 *   u device fp32 [T][N];  v device fp32 [T][L].  Asynchronous on the ctx stream. */
int dode_apply(dode_ctx* ctx, int32_t c, const float* u, float* v);
int dode_apply_t(dode_ctx* ctx, int32_t c, const float* v, float* u);

/* a7: L_c ~ lambda_max(rho_c^T rho_c): Rayleigh quotient after `iters` power iterations from the
 * all-ones vector, run through dode_apply/dode_apply_t's kernels (fp32 products, fp64 norms).
 * eta_c = 1/L_c is the step "dependent on the problem scale".  Synchronises. */
int dode_lipschitz(dode_ctx* ctx, int32_t c, int32_t iters, double* L_out);

/* NEXT-4 — Step 1 of the framework: the DAR blocks of ONE day / traffic pattern from link speeds (Eq. 17-18 and
 * Example 3; "iterating over departure time intervals and paths").  Needs no ctx.
 *   path_ptr    device int32 [N+1]      links of OD n's path: path_links[path_ptr[n] .. path_ptr[n+1]) in travel order
 *   path_links  device int32 [path_ptr[N]], each in [0, L)   (one path per OD: route share p = 1 in Eq. 41)
 *   link_len    device fp32 [L]         link lengths
 *   speed       device fp32 [T][L]      link speed in each interval, length units per second, > 0
 *   dt          interval length |H| in seconds (300 for the paper's 5-minute data)
 *   R_out       device fp32 [T][H+1][L][N]  (one cluster's slab of dode_dar.dense); fully overwritten
 * The flow departing in interval s is bracketed by the trajectories leaving at s*dt and (s+1)*dt, each crossing a link at
 * the speed of the interval in which it enters it; at the tail of link a it arrives evenly spread over [a1, a2) and
 *     R[s][h2-s][a][n] = |[a1,a2) ∩ H_h2| / (a2 - a1).
 * Shares with h2-s > H or h2 >= T are dropped.  Asynchronous on `stream`; errors of this call are read
 * with dode_last_error(NULL). */
int dode_dar_build(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* path_ptr, const int32_t* path_links,
                   const float* link_len, const float* speed, double dt, float* R_out, void* stream);

/* NEXT-4, with route choice: the assignment matrix B = delta * rho * p of one pattern (Eq. 41) for
 * several paths per OD and Logit route shares p_k(s) = exp(-theta c_k(s)) / sum_k' exp(-theta c_k'(s)) (Eq. 37,
 * PAPER.md:309-312), c_k(s) = travel time of path k for the vehicle leaving at the start of interval s, from the
 * pattern's speeds.  R_out[s][h][l][n] = sum over the OD's paths k of rho_k(s, s+h; l) p_k(s).
 *   od_ptr    device int32 [N+1]   paths of OD n: od_ptr[n] .. od_ptr[n+1])  (at least one each)
 *   path_ptr  device int32 [P+1], path_links, link_len, speed, dt, R_out, stream: as dode_dar_build, P = od_ptr[N]
 *   theta     Logit dispersion factor, >= 0 (per second of travel time)
 * With one path per OD this is dode_dar_build. */
int dode_assignment_build(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* od_ptr, const int32_t* path_ptr,
                          const int32_t* path_links, const float* link_len, const float* speed, double dt, double theta,
                          float* R_out, void* stream);

/* NEXT-4 for large networks: the same operator as dode_assignment_build (od_ptr == NULL: dode_dar_build, one path per OD),
 * emitted directly in the boundary CSR format of dode_dar for ONE cluster / pattern ("coordinate format sparse
 * representation"; Table 2 "Sparse") — the dense slab of a config-4-sized network would be
 * terabytes.  Blocks in [s][h] order, rows = links, columns = OD pairs ascending; several paths of one OD through the same
 * link and lag are merged (their shares add up, Eq. 41); shares with h > H or s+h >= T are dropped.
 *   blk_off_out  device int64 [T*(H+1) + 1];  row_ptr_out  device int32 [T*(H+1)][L+1]
 *   col_idx_out  device int32 [cap];          val_out      device fp32 [cap]
 *   cap          entries the two arrays can hold;  nnz_out  host int64
 * If cap is smaller than the number of shares the walk emits (before merging), nothing is written, *nnz_out receives that
 * number and DODE_ENOMEM is returned: call once with cap = 0 to size the arrays.  On success *nnz_out = entries written.
 * Uses temporary device memory of about 24 bytes per share.  Synchronises `stream`.  Errors: dode_last_error(NULL). */
int dode_assignment_build_csr(int32_t N, int32_t L, int32_t T, int32_t H, const int32_t* od_ptr, const int32_t* path_ptr,
                              const int32_t* path_links, const float* link_len, const float* speed, double dt, double theta,
                              int64_t* blk_off_out, int32_t* row_ptr_out, int32_t* col_idx_out, float* val_out,
                              int64_t cap, int64_t* nnz_out, void* stream);

/* Optional per-kernel timing for roofline reports: while enabled, every forward (kind 0) and
 * gradient+update (kind 1) launch is bracketed by CUDA events on the ctx stream.  dode_timing_read
 * synchronises, folds finished event pairs into the running totals and returns the total device
 * time (ms) and launch count of one kind; reset != 0 clears that kind's totals afterwards. */
int dode_timing_enable(dode_ctx* ctx, int32_t on);
int dode_timing_read(dode_ctx* ctx, int32_t kind, double* total_ms, int64_t* launches, int32_t reset);

/* Measurement helper (needs no ctx, not on the SPGD path): the device's FP32 FFMA rate from a register-only kernel of
 * independent fused multiply-add chains (2 CTAs x 1024 threads per SM, 8 chains per thread), best of `reps` timed
 * launches after one warm-up, in TFLOP/s (2 flops per FFMA).  bench.py uses it as the denominator of every "alu"
 * roofline instead of the nominal SMs x 128 lanes x 2 x clock.  Synchronises `stream`.  Errors: dode_last_error(NULL). */
int dode_probe_fp32_peak(int32_t reps, double* tflops, void* stream);

/* One visit of ONE day (Alg. 1 lines 9-11 on a single-day minibatch; the same r = rho q - x,
 * g = rho^T r, q <- max(0, q - eta g) as dode_spgd_step with n = 1) for callers that may not allocate: code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Needs no ctx and calls no cudaMalloc, cudaFree
 * or allocating library routine: the day's residual r [T][L] — the only scratch of a visit — lives in a file-scope
 * device array of DODE_STATIC_SCRATCH_FLOATS floats (1 MiB) that every GPU loading the library holds until exit.
 *   R    device fp32 [T][H+1][L][N], the boundary order of dode_dar.dense for one cluster (n fastest), read only
 *   q    device fp32 [T][N], updated in place;   x  device fp32 [T][L], read only;   eta > 0
 *   stream  the cudaStream_t (as void*) both kernels are launched on; asynchronous, nothing is synchronised
 * Limits: T*L <= DODE_STATIC_SCRATCH_FLOATS and T <= 65535, else DODE_EINVAL with the sizes in dode_last_error(NULL)
 * and nothing launched (use dode_create + dode_spgd_step for larger days: they allocate at create / first use).
 * Every call on a device shares that device's array.  The forward kernel writes every element the gradient kernel reads,
 * so nothing has to start at zero and no call sees the previous call's contents; but two calls that OVERLAP on one GPU
 * (different streams, or several host threads each on its own stream) race on r: keep calls on a device in one stream
 * or order them with events.  The first call on each device looks up the array's device address
 * (cudaGetSymbolAddress with that device current, once per device, under a mutex); later calls only launch.
 * Plain FP32 FFMA kernels (one warp per residual element; 32 OD columns x 8 row slices per gradient CTA) on the
 * unpadded boundary layout — a convenience path, not the tuned one; results agree with dode_spgd_step within the
 * tolerance of DESIGN.md §4 (different FP32 summation order). */
#define DODE_STATIC_SCRATCH_FLOATS (1 << 18)
int dode_visit_static(int32_t N, int32_t L, int32_t T, int32_t H, const float* R, float* q, const float* x, float eta,
                      void* stream);

/* Number of kernels this ctx has launched so far (bench.py's gpu_launches). */
int64_t dode_launch_count(const dode_ctx* ctx);

/* Which kernel family the last step used: "<forward kernel>+<gradient kernel>", e.g.
 * "ffma_coldot_fwd_bt4+ffma_coldot_grad_bt4", "tcgen05_3xtf32_fwd_bn64+tcgen05_3xtf32_grad_bn64",
 * "csr_fwd_bp128+csr_grad_bp128". */
const char* dode_last_path(const dode_ctx* ctx);

/* Waits for all work issued on the ctx stream and on the library's internal streams; returns a pending CUDA error if
 * any. */
int dode_sync(dode_ctx* ctx);

void dode_destroy(dode_ctx* ctx);

/* Text of the last error on this ctx ("" if none).  With ctx == NULL: the text of the last
 * failed dode_create on this thread. */
const char* dode_last_error(const dode_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* DODE_H_ */
