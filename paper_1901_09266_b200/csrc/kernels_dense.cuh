// Dense FP32-FFMA kernels of the SPGD hot path, sm_100a.
//
// Regime: minibatch b < 8, where streaming R from HBM bounds the step (arithmetic intensity b/2 flop per
// byte of R per pass).  Every element of R is needed by exactly ONE output row (a2) / output column (a3),
// so R goes HBM -> registers directly with 128-bit coalesced loads (no shared-memory staging: there is no
// reuse to capture); the only reused operand is the minibatch panel (Q or r), which is small and lives in L1/L2.
//
// The library keeps the operator twice, each copy with the OUTPUT index contiguous, so that both passes are
// the same "column dot" stream (thread = 4 output columns, walks K rows, no cross-lane reduction):
//   Ag [C][T][H+1][Lp][Np]  departure-major (the boundary order, zero padded): for departure s the K rows are
//                           (h,l) and n is contiguous            -> a3, g[s][n] = sum_k Ag[s][k][n] r[s*Lp + k]
//   Af [C][T][H+1][Np][Lp]  arrival-major, lag-merged at create: for arrival t the K rows are (j,n), j-th lag
//                           slot = departure s = t-hmax+j (hmax = min(H,t)), and l is contiguous
//                                                                -> a2, r[t][l] = sum_k Af[t][k][l] q[(t-hmax)*Np + k]
// In both cases the second operand is a contiguous window of the day's state vector.
//   q    [D][T][Np]   state; x [D][T][L]
//   panels (FFMA path): [rows][bp], day index fastest (bp = b rounded up to BT)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dode {

constexpr int kMaxDays = 256;      // days per launch (larger minibatches are split; days are independent)
constexpr int kThreads = 256;

struct DayList {
    int n;
    int day[kMaxDays];
};

__device__ __forceinline__ float4 ldg_stream(const float4* p) {     // R: read once, keep it out of L1
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// Alg. 1 lines 10-11: x = Adagrad(x, g, eta); x = max(x, 0).  Adagrad [14] as the paper's PyTorch
// implementation has it: G += g^2, x -= eta g / (sqrt(G) + eps)  (reading A18).
__device__ __forceinline__ float adagrad_update(float q, float g, float* Gp, float eta, float eps) {
    const float Gn = fmaf(g, g, __ldcg(Gp));      // through L2: under PDL the previous step may have written it (kernels_tc.cuh)
    *Gp = Gn;
    return fmaxf(0.f, q - eta * g / (sqrtf(Gn) + eps));
}

template <int BT> struct RVec;
template <> struct RVec<1> { using type = float; };
template <> struct RVec<2> { using type = float2; };
template <> struct RVec<4> { using type = float4; };

enum { EPI_RESID = 0, EPI_UPDATE = 1, EPI_STORE = 2 };

struct BandArgs {
    const float* A;      // one cluster's copy (Af for a2, Ag for a3): [T][krows][M4*4]
    const float* B;      // panel [T*kunit][bp]: window rows w0(tt) .. w0(tt)+Kc
    int M;               // valid outputs per time index (L for a2, N for a3)
    int M4;              // padded outputs / 4
    int kunit;           // K rows per lag (Np for a2, Lp for a3)
    int T, H, bp;
    int forward;         // 1: a2 (window ends at tt), 0: a3 (window starts at tt)
    // epilogues
    const float* x;      // EPI_RESID: [D][T][M]
    float* out;          // EPI_RESID: r panel [T*M4*4][bp]; EPI_STORE: [T][opitch]
    int opitch;
    float* q;            // EPI_UPDATE: state, in place
    size_t dayStride;
    float eta;
    // NEXT-1, Alg. 1 as printed: row-chunk minibatch and Adagrad
    const uint8_t* mask; // EPI_RESID: [n][T][M] bytes by position in the day list, 0 = row not in the chunk B_o (r = 0); nullable
    float* G;            // EPI_UPDATE: Adagrad accumulator [D][T][Mp], nullable = plain projected step
    float eps;
};

// ---------------------------------------------------------------------------------------------
// a2 / a3 (+a4): out[tt][m][d] = sum_{k < Kc} A[tt][k][m] * B[w0 + k][d]
//   a2 ("B_o x - y", Alg. 1 line 9): Kc = (min(H,tt)+1)*Np, w0 = (tt-min(H,tt))*Np, EPI_RESID subtracts x
//   a3 ("g = B_o^T(...)"):            Kc = (min(H,T-1-tt)+1)*Lp, w0 = tt*Lp, EPI_UPDATE applies
//        q <- max(0, q - eta g) ("x = max(x,0)") in place
// A thread owns one float4 of outputs and walks K rows; 256 threads = CW column-threads x KS row-slices;
// partial sums meet in shared memory, then the CTA runs the epilogue with coalesced accesses.
// grid = (ceil(M4/CW), T, ceil(b/BT)), block = 256, dynamic smem = 256*4*BT*4 bytes.
// ---------------------------------------------------------------------------------------------
template <int BT, int EPI>
__global__ void __launch_bounds__(kThreads)
band_coldot(const __grid_constant__ BandArgs a, int cwlog2, const __grid_constant__ DayList dl) {
    extern __shared__ float sm[];
    const int CW = 1 << cwlog2, KS = kThreads >> cwlog2;
    const int col = threadIdx.x & (CW - 1), ks = threadIdx.x >> cwlog2;
    const int tt = blockIdx.y, d0 = blockIdx.z * BT;
    const int m4 = min((int)blockIdx.x * CW + col, a.M4 - 1);
    const int lags = (a.forward ? min(a.H, tt) : min(a.H, a.T - 1 - tt)) + 1;
    const int Kc = lags * a.kunit;
    const long w0 = a.forward ? (long)(tt - lags + 1) * a.kunit : (long)tt * a.kunit;
    const int bp = a.bp;

    const float4* Ap = reinterpret_cast<const float4*>(a.A) + (size_t)tt * (a.H + 1) * a.kunit * a.M4 + m4;
    const float* Bp = a.B + (size_t)w0 * bp + d0;

    float acc[4][BT];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int j = 0; j < BT; ++j) acc[c][j] = 0.f;

    constexpr int VW = BT >= 4 ? 4 : BT;           // days per panel load
    using rvec = typename RVec<VW>::type;
    constexpr int U = 4;
    int k = ks;
    for (; k + (U - 1) * KS < Kc; k += U * KS) {
        float4 av[U];
#pragma unroll
        for (int u = 0; u < U; ++u) av[u] = ldg_stream(Ap + (size_t)(k + u * KS) * a.M4);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const rvec* rr = reinterpret_cast<const rvec*>(Bp + (size_t)(k + u * KS) * bp);
#pragma unroll
            for (int jv = 0; jv < BT / VW; ++jv) {
                const rvec rv = __ldg(rr + jv);
                const float* rf = reinterpret_cast<const float*>(&rv);
#pragma unroll
                for (int e = 0; e < VW; ++e) {
                    const int j = jv * VW + e;
                    acc[0][j] = fmaf(av[u].x, rf[e], acc[0][j]);
                    acc[1][j] = fmaf(av[u].y, rf[e], acc[1][j]);
                    acc[2][j] = fmaf(av[u].z, rf[e], acc[2][j]);
                    acc[3][j] = fmaf(av[u].w, rf[e], acc[3][j]);
                }
            }
        }
    }
    for (; k < Kc; k += KS) {
        const float4 av = ldg_stream(Ap + (size_t)k * a.M4);
        const rvec* rr = reinterpret_cast<const rvec*>(Bp + (size_t)k * bp);
#pragma unroll
        for (int jv = 0; jv < BT / VW; ++jv) {
            const rvec rv = __ldg(rr + jv);
            const float* rf = reinterpret_cast<const float*>(&rv);
#pragma unroll
            for (int e = 0; e < VW; ++e) {
                const int j = jv * VW + e;
                acc[0][j] = fmaf(av.x, rf[e], acc[0][j]);
                acc[1][j] = fmaf(av.y, rf[e], acc[1][j]);
                acc[2][j] = fmaf(av.z, rf[e], acc[2][j]);
                acc[3][j] = fmaf(av.w, rf[e], acc[3][j]);
            }
        }
    }

    // partials: sm[ks][j][col*4 + c]
    const int O = BT * CW * 4;
#pragma unroll
    for (int j = 0; j < BT; ++j)
        *reinterpret_cast<float4*>(sm + (size_t)ks * O + j * CW * 4 + col * 4) =
            make_float4(acc[0][j], acc[1][j], acc[2][j], acc[3][j]);
    __syncthreads();
    const int Mp = a.M4 * 4;
    for (int o = threadIdx.x; o < O; o += kThreads) {
        float g = 0.f;
        for (int q = 0; q < KS; ++q) g += sm[(size_t)q * O + o];
        const int j = o >> (cwlog2 + 2), mm = o & (CW * 4 - 1);
        const int m = blockIdx.x * CW * 4 + mm;
        if (m >= Mp) continue;
        if (EPI == EPI_RESID) {
            // pad days (d0+j >= n) repeat the last day; pad rows (m >= M) are written as 0
            float v = 0.f;
            if (m < a.M) {
                const int pos = min(d0 + j, dl.n - 1);
                v = g - __ldg(a.x + ((size_t)dl.day[pos] * a.T + tt) * a.M + m);
                if (a.mask != nullptr && a.mask[((size_t)pos * a.T + tt) * a.M + m] == 0) v = 0.f;   // row outside B_o
            }
            a.out[((size_t)tt * Mp + m) * bp + d0 + j] = v;
        } else if (EPI == EPI_UPDATE) {
            if (m < a.M && d0 + j < dl.n) {
                const size_t qi = (size_t)dl.day[d0 + j] * a.dayStride + (size_t)tt * Mp + m;
                float* qp = a.q + qi;
                if (a.G != nullptr) *qp = adagrad_update(*qp, g, a.G + qi, a.eta, a.eps);
                else *qp = fmaxf(0.f, fmaf(-a.eta, g, *qp));
            }
        } else {
            if (m < a.opitch && j == 0) a.out[(size_t)tt * a.opitch + m] = g;
        }
    }
}

// ---- create-time packing (a0) -------------------------------------------------------------------
// Ag[c][s][h][l][n] = R[c][s][h][l][n] for l < L, n < N and s+h < T; everything else 0.
// (blocks with s+h >= T "may be present; they are ignored" — include/dode.h)
__global__ void __launch_bounds__(256)
pack_departure_major(const float* __restrict__ R, float* __restrict__ Ag, long blocks, int T, int H, int L, int N,
                     int Lp, int Np) {
    const long total = blocks * Lp * (Np / 4);
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int n4 = (int)(i % (Np / 4));
        const long rowi = i / (Np / 4);
        const int l = (int)(rowi % Lp);
        const long blk = rowi / Lp;                       // (c*T + s)*(H+1) + h
        const int h = (int)(blk % (H + 1)), s = (int)((blk / (H + 1)) % T);
        float v[4] = {0.f, 0.f, 0.f, 0.f};
        if (l < L && s + h < T) {
            const float* src = R + (blk * L + l) * (size_t)N + n4 * 4;
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (n4 * 4 + e < N) v[e] = __ldg(src + e);
        }
        reinterpret_cast<float4*>(Ag)[i] = make_float4(v[0], v[1], v[2], v[3]);
    }
}

// Af[c][t][j][n][l] = R[c][s][h][l][n] with s = t-hmax+j, h = hmax-j, hmax = min(H,t), for j <= hmax; 0 otherwise.
// One 32x32 (l x n) transpose tile per block; grid = (C*T*(H+1), ceil(Lp/32), ceil(Np/32)) — the block count can
// exceed the 65535 limit of grid.y/z, so it rides on grid.x.
__global__ void __launch_bounds__(256)
pack_arrival_major(const float* __restrict__ R, float* __restrict__ Af, int T, int H, int L, int N, int Lp, int Np) {
    __shared__ float tile[32][33];
    const long ctj = blockIdx.x;                          // (c*T + t)*(H+1) + j
    const int j = (int)(ctj % (H + 1));
    const long ct = ctj / (H + 1);
    const int t = (int)(ct % T);
    const long c = ct / T;
    const int hmax = min(H, t);
    const int l0 = blockIdx.y * 32, n0 = blockIdx.z * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const bool valid = j <= hmax;
    if (valid) {
        const int s = t - hmax + j, h = hmax - j;
        const float* src = R + (((c * T + s) * (H + 1) + h) * (size_t)L) * N;
        for (int ll = ty; ll < 32; ll += 8) {
            const int l = l0 + ll, n = n0 + tx;
            tile[ll][tx] = (l < L && n < N) ? __ldg(src + (size_t)l * N + n) : 0.f;
        }
    }
    __syncthreads();
    float* dst = Af + ctj * (size_t)Np * Lp;
    for (int nn = ty; nn < 32; nn += 8) {
        const int n = n0 + nn, l = l0 + tx;
        if (n < Np && l < Lp) dst[(size_t)n * Lp + l] = valid ? tile[tx][nn] : 0.f;
    }
}

// dst[i*bp + d] = src[day_d*dayStride + i] for i < rowLen, d < bp (pad days repeat the last day). 32x32 smem transpose.
__global__ void __launch_bounds__(256)
gather_panel(const float* __restrict__ src, size_t dayStride, long rowLen, float* __restrict__ dst, int bp,
             const __grid_constant__ DayList dl) {
    __shared__ float tile[32][33];
    const long i0 = (long)blockIdx.x * 32;
    const int d0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int dd = ty; dd < 32; dd += 8) {
        const int d = min(d0 + dd, dl.n - 1);
        const long i = i0 + tx;
        tile[dd][tx] = i < rowLen ? __ldg(src + (size_t)dl.day[d] * dayStride + i) : 0.f;
    }
    __syncthreads();
    for (int ii = ty; ii < 32; ii += 8) {
        const long i = i0 + ii;
        if (i < rowLen && d0 + tx < bp) dst[i * bp + d0 + tx] = tile[tx][ii];
    }
}

// ---------------------------------------------------------------------------------------------
// a5: per-day sum of squares of r[T][L][bp] in double.  Stage 1: block (chunk, day-tile) sums a
// slab of (t,l) rows; stage 2: one warp per day adds the chunk partials in a fixed order.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads)
sumsq_partial(const float* __restrict__ r, double* __restrict__ part, long rows, int bp, int nb, int rowsPerBlock) {
    __shared__ double red[kThreads];
    const int dt = threadIdx.x & 31, rt = threadIdx.x >> 5;     // 32 days x 8 row lanes
    const int d = blockIdx.y * 32 + dt;
    const long r0 = (long)blockIdx.x * rowsPerBlock, r1 = min(rows, r0 + rowsPerBlock);
    double acc = 0.0;
    if (d < nb)
        for (long k = r0 + rt; k < r1; k += 8) {
            const float v = r[k * bp + d];
            acc += (double)v * (double)v;
        }
    red[threadIdx.x] = acc;
    __syncthreads();
    if (rt == 0 && d < nb) {
        double sacc = 0.0;
        for (int q = 0; q < 8; ++q) sacc += red[q * 32 + dt];
        part[(size_t)blockIdx.x * nb + d] = sacc;
    }
}

__global__ void sumsq_final(const double* __restrict__ part, double* __restrict__ out, int nchunks, int nb) {
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= nb) return;
    double acc = 0.0;
    for (int c = 0; c < nchunks; ++c) acc += part[(size_t)c * nb + d];
    out[d] = acc;
}

// Step 6 quality check: per-day sum and sum of squares of the observed counts x[day][T*L] in double
// (for SS_tot of the coefficient of determination).  One block per listed day.
__global__ void __launch_bounds__(kThreads)
x_moments(const float* __restrict__ x, long TL, double* __restrict__ out, const __grid_constant__ DayList dl) {
    __shared__ double s1[kThreads], s2[kThreads];
    const float* xd = x + (size_t)dl.day[blockIdx.x] * TL;
    double a = 0.0, b = 0.0;
    for (long i = threadIdx.x; i < TL; i += kThreads) {
        const double v = (double)xd[i];
        a += v; b += v * v;
    }
    s1[threadIdx.x] = a; s2[threadIdx.x] = b;
    __syncthreads();
    for (int s = kThreads / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) { s1[threadIdx.x] += s1[threadIdx.x + s]; s2[threadIdx.x] += s2[threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[2 * blockIdx.x] = s1[0]; out[2 * blockIdx.x + 1] = s2[0]; }
}

// ---- small helpers for a7 (power iteration) and state init ----
__global__ void fill_f32(float* p, size_t n, float v) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = v;
}

// q[d][s][n] = v for n < N, 0 in the pad columns
__global__ void fill_state(float* q, size_t rows, int N, int Np, float v) {
    const size_t total = rows * Np;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x)
        q[i] = ((int)(i % Np) < N) ? v : 0.f;
}

// out[0] = sum v^2 (double), single block (vectors here are T*N or T*L long)
__global__ void __launch_bounds__(1024) sumsq_single(const float* __restrict__ v, size_t n, double* __restrict__ out) {
    __shared__ double red[1024];
    double acc = 0.0;
    for (size_t i = threadIdx.x; i < n; i += 1024) acc += (double)v[i] * (double)v[i];
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = red[0];
}

// dst[row][0..Np) = src[row][0..N) * (1/sqrt(*nrm2)), pad columns 0  (src stride N, dst stride Np)
__global__ void scale_pad(const float* __restrict__ src, float* __restrict__ dst, size_t rows, int N, int Np,
                          const double* __restrict__ nrm2) {
    const float sc = nrm2 ? (float)(1.0 / sqrt(*nrm2)) : 1.f;
    const size_t total = rows * Np;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / Np;
        const int n = (int)(i - row * Np);
        dst[i] = n < N ? src[row * N + n] * sc : 0.f;
    }
}

}  // namespace dode
