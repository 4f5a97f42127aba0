// Dense FP32-FFMA kernels of the SPGD hot path, sm_100a.
//
// Regime: minibatch b small enough that streaming R from HBM bounds the step
// (arithmetic intensity b/2 flop per byte of R per pass).  Every element of R is needed by
// exactly ONE output row (a2) / output column (a3), so R goes HBM -> registers directly with
// 128-bit coalesced loads (no shared-memory staging: there is no reuse to capture); the only
// reused operand is the minibatch state (Q or r), which is small and lives in L1/L2.
//
// Layouts (device, fp32):
//   Rc   [T][H+1][L][Np]    one cluster's blocks, Np = N rounded up to 4 (pad columns are 0)
//   q    [D][T][Np]         state; day d at q + d*T*Np
//   x    [D][T][L]
//   r    [T][L][bp]         residual of the current minibatch, day index fastest (bp = b rounded up to BT)
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

// Sum V (power of two <= 32) per-lane values across the warp with V-1 + log2(32/V) shuffles.
// Returns, in every lane, the total of value index (lane & (V-1)).
template <int V>
__device__ __forceinline__ float warp_reduce_multi(float (&v)[V], int lane) {
#pragma unroll
    for (int n = V / 2; n >= 1; n >>= 1) {
        const bool up = (lane & n) != 0;
#pragma unroll
        for (int i = 0; i < n; ++i) {
            const float send = up ? v[i] : v[i + n];
            const float keep = up ? v[i + n] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, n);
        }
    }
    float s = v[0];
#pragma unroll
    for (int off = V; off < 32; off <<= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    return s;
}

// ---------------------------------------------------------------------------------------------
// a2: forward residual  r[t][l][d] = sum_{h<=min(H,t)} sum_n R[t-h][h][l][n] q_d[t-h][n] - x_d[t][l]
// ("B_o x - y", Alg. 1 line 9).  One warp owns RL link rows of one arrival interval
// t for BT days; lanes run along the contiguous OD index (the reduction index), so the K loop is
// the flattened (h, n/4) float4 index and the sum over lanes is a shuffle reduction at the end.
// grid = (ceil(L / (8*RL)), T, ceil(b/BT)), block = 256.
// ---------------------------------------------------------------------------------------------
template <int BT, int RL>
__global__ void __launch_bounds__(kThreads)
fwd_rowdot(const float* __restrict__ Rc, const float* __restrict__ qbase, size_t dayStride,
           const float* __restrict__ xbase, float* __restrict__ r,
           int N4, int L, int T, int H, int bp, const __grid_constant__ DayList dl) {
    static_assert(BT * RL <= 32, "one shuffle-reduction group");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int t = blockIdx.y;
    const int l0 = (blockIdx.x * (kThreads / 32) + warp) * RL;
    if (l0 >= L) return;
    const int d0 = blockIdx.z * BT;

    const float4* Rrow[RL];
#pragma unroll
    for (int i = 0; i < RL; ++i) {
        const int l = min(l0 + i, L - 1);
        Rrow[i] = reinterpret_cast<const float4*>(Rc) + ((size_t)t * (H + 1) * L + l) * N4;
    }
    const float4* qd[BT];
#pragma unroll
    for (int j = 0; j < BT; ++j) {
        const int day = dl.day[min(d0 + j, dl.n - 1)];
        qd[j] = reinterpret_cast<const float4*>(qbase + (size_t)day * dayStride) + (size_t)t * N4;
    }
    // block (s = t-h, h) sits H*L*N4 float4 before block (t-h+1, h-1); q[t-h] sits N4 before q[t-h+1]
    const long hstepR = (long)H * L * N4;
    const int F = (min(H, t) + 1) * N4;
    const int dh = 32 / N4, dn = 32 - dh * N4;
    int h = lane / N4, n4 = lane - h * N4;

    float acc[RL][BT];
#pragma unroll
    for (int i = 0; i < RL; ++i)
#pragma unroll
        for (int j = 0; j < BT; ++j) acc[i][j] = 0.f;

#pragma unroll 2
    for (int f = lane; f < F; f += 32) {
        const long ro = (long)n4 - (long)h * hstepR;
        const long qo = (long)n4 - (long)h * N4;
        float4 a[RL];
#pragma unroll
        for (int i = 0; i < RL; ++i) a[i] = ldg_stream(Rrow[i] + ro);
#pragma unroll
        for (int j = 0; j < BT; ++j) {
            const float4 qv = __ldg(qd[j] + qo);
#pragma unroll
            for (int i = 0; i < RL; ++i) {
                acc[i][j] = fmaf(a[i].x, qv.x, acc[i][j]);
                acc[i][j] = fmaf(a[i].y, qv.y, acc[i][j]);
                acc[i][j] = fmaf(a[i].z, qv.z, acc[i][j]);
                acc[i][j] = fmaf(a[i].w, qv.w, acc[i][j]);
            }
        }
        n4 += dn; h += dh;
        if (n4 >= N4) { n4 -= N4; ++h; }
    }

    float v[RL * BT];
#pragma unroll
    for (int i = 0; i < RL; ++i)
#pragma unroll
        for (int j = 0; j < BT; ++j) v[i * BT + j] = acc[i][j];
    const float tot = warp_reduce_multi<RL * BT>(v, lane);
    if (lane < RL * BT) {
        const int i = lane / BT, j = lane - i * BT;
        const int l = l0 + i;
        if (l < L) {
            float xv = 0.f;
            if (xbase != nullptr) {
                const int day = dl.day[min(d0 + j, dl.n - 1)];
                xv = __ldg(xbase + ((size_t)day * T + t) * L + l);
            }
            r[((size_t)t * L + l) * bp + d0 + j] = tot - xv;   // pad days (d0+j >= n) repeat the last day
        }
    }
}

template <int BT> struct RVec;
template <> struct RVec<1> { using type = float; };
template <> struct RVec<2> { using type = float2; };
template <> struct RVec<4> { using type = float4; };

// ---------------------------------------------------------------------------------------------
// a3 + a4: transpose gradient g[s][n][d] = sum_{h<=min(H,T-1-s)} sum_l R[s][h][l][n] r[s+h][l][d]
// ("g = B_o^T(...)") with the projected update q <- max(0, q - eta g) in the epilogue
// ("x = max(x,0)").  The (h,l) rows of R[s] are contiguous, so a thread owns one
// float4 of OD columns and walks rows; 256 threads = CW column-threads x KS row-slices; partial
// sums meet in shared memory, then the CTA applies the update with coalesced q accesses.
// grid = (ceil(N4/CW), T, ceil(b/BT)), block = 256, dynamic smem = 256*4*BT*4 bytes.
// UPDATE = false stores g to gout[s][n] (minibatch 1; dode_apply_t).
// ---------------------------------------------------------------------------------------------
template <int BT, bool UPDATE>
__global__ void __launch_bounds__(kThreads)
grad_coldot(const float* __restrict__ Rc, const float* __restrict__ r, float* __restrict__ qbase,
            size_t dayStride, float* __restrict__ gout, float eta,
            int N, int N4, int L, int T, int H, int bp, int cwlog2, const __grid_constant__ DayList dl) {
    extern __shared__ float sm[];
    const int CW = 1 << cwlog2, KS = kThreads >> cwlog2;
    const int col = threadIdx.x & (CW - 1), ks = threadIdx.x >> cwlog2;
    const int s = blockIdx.y, d0 = blockIdx.z * BT;
    const int n4 = min((int)blockIdx.x * CW + col, N4 - 1);
    const int Kc = (min(H, T - 1 - s) + 1) * L;

    const float4* Rp = reinterpret_cast<const float4*>(Rc) + (size_t)s * (H + 1) * L * N4 + n4;
    const float* rp = r + (size_t)s * L * bp + d0;

    float acc[4][BT];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int j = 0; j < BT; ++j) acc[c][j] = 0.f;

    constexpr int VW = BT >= 4 ? 4 : BT;           // days per r load
    using rvec = typename RVec<VW>::type;
    constexpr int U = 4;
    int k = ks;
    for (; k + (U - 1) * KS < Kc; k += U * KS) {
        float4 a[U];
#pragma unroll
        for (int u = 0; u < U; ++u) a[u] = ldg_stream(Rp + (size_t)(k + u * KS) * N4);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const rvec* rr = reinterpret_cast<const rvec*>(rp + (size_t)(k + u * KS) * bp);
#pragma unroll
            for (int jv = 0; jv < BT / VW; ++jv) {
                const rvec rv = __ldg(rr + jv);
                const float* rf = reinterpret_cast<const float*>(&rv);
#pragma unroll
                for (int e = 0; e < VW; ++e) {
                    const int j = jv * VW + e;
                    acc[0][j] = fmaf(a[u].x, rf[e], acc[0][j]);
                    acc[1][j] = fmaf(a[u].y, rf[e], acc[1][j]);
                    acc[2][j] = fmaf(a[u].z, rf[e], acc[2][j]);
                    acc[3][j] = fmaf(a[u].w, rf[e], acc[3][j]);
                }
            }
        }
    }
    for (; k < Kc; k += KS) {
        const float4 a = ldg_stream(Rp + (size_t)k * N4);
        const rvec* rr = reinterpret_cast<const rvec*>(rp + (size_t)k * bp);
#pragma unroll
        for (int jv = 0; jv < BT / VW; ++jv) {
            const rvec rv = __ldg(rr + jv);
            const float* rf = reinterpret_cast<const float*>(&rv);
#pragma unroll
            for (int e = 0; e < VW; ++e) {
                const int j = jv * VW + e;
                acc[0][j] = fmaf(a.x, rf[e], acc[0][j]);
                acc[1][j] = fmaf(a.y, rf[e], acc[1][j]);
                acc[2][j] = fmaf(a.z, rf[e], acc[2][j]);
                acc[3][j] = fmaf(a.w, rf[e], acc[3][j]);
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
    const int Np = N4 * 4;
    for (int o = threadIdx.x; o < O; o += kThreads) {
        float g = 0.f;
        for (int q = 0; q < KS; ++q) g += sm[(size_t)q * O + o];
        const int j = o >> (cwlog2 + 2), nn = o & (CW * 4 - 1);
        const int n = blockIdx.x * CW * 4 + nn;
        if (n < N && d0 + j < dl.n) {
            if (UPDATE) {
                float* qp = qbase + (size_t)dl.day[d0 + j] * dayStride + (size_t)s * Np + n;
                *qp = fmaxf(0.f, fmaf(-eta, g, *qp));
            } else {
                gout[(size_t)s * N + n] = g;
            }
        }
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
