// a6: block-sparse CSR variant of a2-a4 for large networks (BASELINE.json configs[4]).
//
// The boundary format is one CSR per (c,s,h) block (include/dode.h).  At create time each cluster is
// re-packed, on the device, into two lag-merged ROW-BLOCKED sparse matrices so that both passes stream their
// non-zeros contiguously and deterministically (no atomics on the hot path) and so that one gathered panel row
// feeds up to kRB output rows:
//   F (forward):  row block (t/2, l/4) — 4 links x 2 arrival intervals = 8 output rows — holds one entry per distinct
//                 state row (s,n) that feeds any of them: payload (s - (2*(t/2) - H))*Np + n, values val[8] by
//                 (t%2)*4 + l%4 (0 where an output has no entry) -> operand Qb[(s*Np + n)*bp + d].  Paths are
//                 contiguous link runs with slowly growing lag and 2-4 adjacent lags per link, so
//                 adjacent links AND adjacent arrival intervals share most (s,n): 3.7 products per gathered row
//                 against 1 for plain CSR and 2.3 for 4 links x 1 interval (the gathers, not the FMAs, bound the pass).
//   G (gradient): row block (s/4, n) holds one entry per distinct residual row (t,l), t = s+h, reached from any of
//                 its 4 departure intervals: payload kl = (t - 4*(s/4))*L + l, values val[4] by s%4
//                 -> operand r[((4*(s/4))*L + kl)*bp + d].  The lag window of a (link, OD) pair spans 2-4 adjacent
//                 lags, so consecutive departure intervals share most residual rows: ~2x fewer gathers.
// Entries with s+h >= T are dropped.  The re-pack is a radix sort of 64-bit keys, a head-flag scan
// and a scatter (CUB, create-time only).
//
// Hot path: the minibatch state is gathered once per step into the day-fastest panel Qb[T*Np][bp]
// (a coalesced transpose), so that one entry pulls bp contiguous floats; a warp owns one
// row block and its lanes run along the days.  The update q <- max(0, q - eta g) is applied to Qb in the
// gradient kernel's epilogue and scattered back to q[d][s][n].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "../../include/dode.h"
#include "kernels_dense.cuh"

namespace dode {

constexpr int kCsrMaxDays = 128;
constexpr int kRB = 4;            // links (forward) / departure intervals (gradient) per row block
constexpr int kFT = 2;            // arrival intervals per forward row block
constexpr int kFS = kRB * kFT;    // output rows (value slots) of a forward entry
// Gathered panel rows a warp keeps in flight: both passes stall on the latency of the gathers (ncu: long-scoreboard stalls
// dominate), so more loads in flight pay until the registers run out (measured on configs[4]: forward 7.92 / 7.48 / 7.43 /
// 7.08 ms at 2 / 4 / 6 / 8; gradient, which runs 4 CTAs of 64 registers per SM, 9.77 / 9.46 / 13.3 / 16.9 ms).
constexpr int kInFlightF = 8, kInFlightG = 4;     // (gradient with 3 CTAs per SM and 6 / 8 in flight: 10.8 / 12.3 ms)

struct CsrCluster {
    int64_t* rowptrF = nullptr;   // [ceil(T/2)*ceil(L/4) + 1]
    int32_t* payF = nullptr;      // [nuF]  (s - (2*(t/2) - H))*Np + n
    float4* valF = nullptr;       // [2*nuF] eight values per entry, slot (t%2)*4 + l%4
    int64_t* rowptrG = nullptr;   // [ceil(T/4)*Np + 1]
    int32_t* payG = nullptr;      // [nuG]  (t - 4*(s/4))*L + l
    float4* valG = nullptr;       // [nuG]  by s%4
    int32_t* permG = nullptr;     // [Np]   OD indices ordered by the first link of their path (processing order of a3)
    int64_t nnz = 0;              // valid entries (s+h < T)
    int64_t nuF = 0, nuG = 0;     // distinct (row block, payload) entries
};

struct CsrStore {
    bool ready = false;
    int C = 0;
    CsrCluster* cl = nullptr;     // host array [C]
    float* Qb = nullptr;          // [T*Np][bp]
    int cap_bp = 0;
    // NEXT-1 (row-chunk + Adagrad), allocated on first use
    float* Mb = nullptr;          // [T*L][bp]  row mask as 0/1 floats
    float* Gb = nullptr;          // [T*Np][bp] Adagrad accumulator panel
    int cap_bp_ada = 0;
};

// ---- create-time re-pack ---------------------------------------------------------------------------
// one warp per input CSR row (s,h,l) of cluster c; key = ((row block * K + payload) << slot bits) | slot
__global__ void csr_expand_keys(const int64_t* __restrict__ blk_off, const int32_t* __restrict__ row_ptr,
                                const int32_t* __restrict__ col_idx, int c, int N, int Np, int L, int T, int H,
                                int64_t base, unsigned long long* __restrict__ keyF,
                                unsigned long long* __restrict__ keyG) {
    const long warp = (blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    const long rows = (long)T * (H + 1) * L;
    if (warp >= rows) return;
    const int l = (int)(warp % L);
    const long sh = warp / L;
    const int h = (int)(sh % (H + 1)), s = (int)(sh / (H + 1));
    const long b = (long)c * T * (H + 1) + sh;
    const int32_t* rp = row_ptr + b * (L + 1);
    const int64_t k0 = blk_off[b] + rp[l], k1 = blk_off[b] + rp[l + 1];
    const unsigned long long KF = (unsigned long long)(H + kFT) * Np, KG = (unsigned long long)(H + kRB) * L;
    const unsigned long long LB = (unsigned long long)(L + kRB - 1) / kRB;
    const bool valid = s + h < T;
    const int t = s + h, sb = s / kRB, tb = t / kFT;
    for (int64_t k = k0 + lane; k < k1; k += 32) {
        const int n = col_idx[k];
        const unsigned long long rbF = (unsigned long long)tb * LB + l / kRB;
        const unsigned long long payF = (unsigned long long)(s - (tb * kFT - H)) * Np + n;       // s >= t - H >= tb*kFT - H
        const unsigned long long rbG = (unsigned long long)sb * Np + n, payG = (unsigned long long)(t - sb * kRB) * L + l;
        keyF[k - base] = valid ? ((rbF * KF + payF) << 3) | (unsigned)((t % kFT) * kRB + l % kRB) : ~0ull;
        keyG[k - base] = valid ? ((rbG * KG + payG) << 2) | (unsigned)(s % kRB) : ~0ull;
    }
}

// head[i] = 1 where a new (row block, payload) starts in the sorted key array
__global__ void csr_heads(const unsigned long long* __restrict__ keys, int64_t n, int shift, int32_t* __restrict__ head) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        head[i] = (i == 0 || (keys[i] >> shift) != (keys[i - 1] >> shift)) ? 1 : 0;
}

// uidx = inclusive scan of head; entry u = uidx[i]-1 receives val[i] in slot key & (2^shift - 1); heads also write
// payload and key
__global__ void csr_scatter_unique(const unsigned long long* __restrict__ keys, const float* __restrict__ val,
                                   const int32_t* __restrict__ uidx, int64_t n, unsigned long long K, int L, int shift,
                                   float* __restrict__ val4, int32_t* __restrict__ pay, unsigned long long* __restrict__ ukey) {
    const bool forward = shift == 3;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long key = keys[i], kk = key >> shift;
        const int64_t u = (int64_t)uidx[i] - 1;
        val4[(u << shift) + (int)(key & ((1u << shift) - 1))] = val[i];
        if (i == 0 || kk != (keys[i - 1] >> shift)) {
            const unsigned long long rem = kk % K;
            if (forward) {
                pay[u] = (int32_t)rem;                                             // s_rel * Np + n
            } else {
                pay[u] = (int32_t)rem;
            }
            ukey[u] = kk;
        }
    }
}

// rowptr[rb] = lower_bound(ukey, rb*K)
__global__ void csr_rowptr(const unsigned long long* __restrict__ ukey, int64_t nu, long rows,
                           unsigned long long K, int64_t* __restrict__ rowptr) {
    const long row = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (row > rows) return;
    const unsigned long long target = (unsigned long long)row * K;
    int64_t lo = 0, hi = nu;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (ukey[mid] < target) lo = mid + 1; else hi = mid;
    }
    rowptr[row] = lo;
}

// first link of OD n's path = smallest link index among the entries of its first non-empty row block (L if none)
__global__ void csr_first_link(const int64_t* __restrict__ rowptrG, const int32_t* __restrict__ payG, int Np, long SB, int L,
                               int32_t* __restrict__ first, int32_t* __restrict__ ident) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= Np) return;
    int best = L;
    for (long sb = 0; sb < SB && best == L; ++sb) {
        const int64_t k0 = rowptrG[sb * Np + n], k1 = rowptrG[sb * Np + n + 1];
        for (int64_t k = k0; k < k1; ++k) best = min(best, payG[k] % L);
    }
    first[n] = best;
    ident[n] = n;
}

__global__ void count_invalid(const unsigned long long* __restrict__ keys, int64_t n, unsigned long long* cnt) {
    unsigned long long local = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        local += keys[i] == ~0ull;
    for (int o = 16; o; o >>= 1) local += __shfl_xor_sync(0xffffffffu, local, o);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(cnt, local);
}

inline void csr_free(CsrStore& st) {
    if (st.cl) {
        for (int c = 0; c < st.C; ++c) {
            cudaFree(st.cl[c].rowptrF); cudaFree(st.cl[c].payF); cudaFree(st.cl[c].valF);
            cudaFree(st.cl[c].rowptrG); cudaFree(st.cl[c].payG); cudaFree(st.cl[c].valG); cudaFree(st.cl[c].permG);
        }
        delete[] st.cl;
        st.cl = nullptr;
    }
    cudaFree(st.Qb); cudaFree(st.Mb); cudaFree(st.Gb);
    st.Qb = st.Mb = st.Gb = nullptr;
    st.ready = false;
}

inline int csr_build(CsrStore& st, const dode_dims& d, const dode_dar& R, cudaStream_t stream, char* err) {
#define CSR_CU(call)                                                                             \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            snprintf(err, 512, "%s: %s", #call, cudaGetErrorString(e_));                         \
            cudaFree(kF); cudaFree(kG); cudaFree(kS); cudaFree(vS); cudaFree(tmp); cudaFree(dcnt); \
            cudaFree(head); cudaFree(ukey);                                                      \
            return e_ == cudaErrorMemoryAllocation ? DODE_ENOMEM : DODE_ECUDA;                   \
        }                                                                                        \
    } while (0)
    const int Np = (d.N + 3) / 4 * 4;
    st.C = d.C;
    st.cl = new CsrCluster[d.C];
    const long nblk = (long)d.T * (d.H + 1);
    std::vector<int64_t> off(d.C + 1);
    unsigned long long *kF = nullptr, *kG = nullptr, *kS = nullptr, *dcnt = nullptr, *ukey = nullptr;
    float* vS = nullptr;
    int32_t* head = nullptr;
    void* tmp = nullptr;
    for (int c = 0; c <= d.C; ++c)
        CSR_CU(cudaMemcpyAsync(&off[c], R.blk_off + (long)c * nblk, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
    CSR_CU(cudaStreamSynchronize(stream));
    if (off[d.C] != R.nnz) { snprintf(err, 512, "blk_off[last]=%lld but nnz=%lld", (long long)off[d.C], (long long)R.nnz); return DODE_EINVAL; }
    int64_t maxn = 1;
    for (int c = 0; c < d.C; ++c) maxn = std::max<int64_t>(maxn, off[c + 1] - off[c]);
    if (maxn >= (int64_t)1 << 31) { snprintf(err, 512, "more than 2^31 non-zeros in one cluster"); return DODE_EINVAL; }
    CSR_CU(cudaMalloc(&kF, maxn * 8)); CSR_CU(cudaMalloc(&kG, maxn * 8)); CSR_CU(cudaMalloc(&kS, maxn * 8));
    CSR_CU(cudaMalloc(&ukey, maxn * 8)); CSR_CU(cudaMalloc(&head, maxn * 4));
    CSR_CU(cudaMalloc(&vS, maxn * 4)); CSR_CU(cudaMalloc(&dcnt, 8));
    size_t tmp_sort = 0, tmp_scan = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tmp_sort, kF, kS, (const float*)nullptr, vS, maxn, 0, 64, stream);
    cub::DeviceScan::InclusiveSum(nullptr, tmp_scan, head, head, (int)maxn, stream);
    const size_t tmp_bytes = std::max(tmp_sort, tmp_scan);
    CSR_CU(cudaMalloc(&tmp, tmp_bytes));
    const unsigned long long KF = (unsigned long long)(d.H + kFT) * Np, KG = (unsigned long long)(d.H + kRB) * d.L;
    const long LB = (d.L + kRB - 1) / kRB, SB = (d.T + kRB - 1) / kRB, TB = (d.T + kFT - 1) / kFT;
    for (int c = 0; c < d.C; ++c) {
        CsrCluster& cl = st.cl[c];
        const int64_t n = off[c + 1] - off[c];
        const long rows_in = nblk * d.L;
        unsigned long long ninv = 0;
        if (n > 0) {
            csr_expand_keys<<<(unsigned)((rows_in * 32 + 255) / 256), 256, 0, stream>>>(
                R.blk_off, R.row_ptr, R.col_idx, c, d.N, Np, d.L, d.T, d.H, off[c], kF, kG);
            CSR_CU(cudaMemsetAsync(dcnt, 0, 8, stream));
            count_invalid<<<1184, 256, 0, stream>>>(kF, n, dcnt);
            CSR_CU(cudaMemcpyAsync(&ninv, dcnt, 8, cudaMemcpyDeviceToHost, stream));
        }
        CSR_CU(cudaStreamSynchronize(stream));
        const int64_t nv = n - (int64_t)ninv;
        cl.nnz = nv;
        for (int pass = 0; pass < 2; ++pass) {
            unsigned long long* kin = pass == 0 ? kF : kG;
            const unsigned long long K = pass == 0 ? KF : KG;
            const long rows = pass == 0 ? TB * LB : SB * Np;                 // row blocks
            const int shift = pass == 0 ? 3 : 2;                             // log2(value slots per entry)
            int64_t nu = 0;
            if (nv > 0) {
                // invalid keys are all-ones: sort on all 64 bits so they land at the end
                CSR_CU(cub::DeviceRadixSort::SortPairs(tmp, tmp_sort, kin, kS, R.val + off[c], vS, n, 0, 64, stream));
                csr_heads<<<1184, 256, 0, stream>>>(kS, nv, shift, head);
                CSR_CU(cub::DeviceScan::InclusiveSum(tmp, tmp_scan, head, head, (int)nv, stream));
                int32_t last = 0;
                CSR_CU(cudaMemcpyAsync(&last, head + nv - 1, 4, cudaMemcpyDeviceToHost, stream));
                CSR_CU(cudaStreamSynchronize(stream));
                nu = last;
            }
            int32_t** pay = pass == 0 ? &cl.payF : &cl.payG;
            float4** val4 = pass == 0 ? &cl.valF : &cl.valG;
            int64_t** rowptr = pass == 0 ? &cl.rowptrF : &cl.rowptrG;
            (pass == 0 ? cl.nuF : cl.nuG) = nu;
            CSR_CU(cudaMalloc(pay, std::max<int64_t>(nu, 1) * 4));
            CSR_CU(cudaMalloc(val4, (std::max<int64_t>(nu, 1) * 4) << shift));
            CSR_CU(cudaMalloc(rowptr, (rows + 1) * 8));
            if (nu > 0) {
                CSR_CU(cudaMemsetAsync(*val4, 0, (nu * 4) << shift, stream));
                csr_scatter_unique<<<1184, 256, 0, stream>>>(kS, vS, head, nv, K, d.L, shift,
                                                             reinterpret_cast<float*>(*val4), *pay, ukey);
            }
            csr_rowptr<<<(unsigned)((rows + 1 + 255) / 256), 256, 0, stream>>>(ukey, nu, rows, K, *rowptr);
        }
        // processing order of the gradient rows: ODs sorted by the first link of their path
        {
            int32_t* sc = nullptr;                       // [Np] keys in | [Np] keys out | [Np] identity
            CSR_CU(cudaMalloc(&sc, (size_t)3 * Np * 4));
            CSR_CU(cudaMalloc(&cl.permG, (size_t)Np * 4));
            csr_first_link<<<(Np + 255) / 256, 256, 0, stream>>>(cl.rowptrG, cl.payG, Np, SB, d.L, sc, sc + 2 * Np);
            size_t need = 0;
            void* t2 = nullptr;
            cub::DeviceRadixSort::SortPairs(nullptr, need, sc, sc + Np, sc + 2 * Np, cl.permG, Np, 0, 32, stream);
            cudaError_t e2 = cudaMalloc(&t2, need);
            if (e2 == cudaSuccess) e2 = cub::DeviceRadixSort::SortPairs(t2, need, sc, sc + Np, sc + 2 * Np, cl.permG, Np, 0, 32, stream);
            if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(stream);
            cudaFree(t2); cudaFree(sc);
            CSR_CU(e2);
        }
        CSR_CU(cudaStreamSynchronize(stream));
    }
    CSR_CU(cudaGetLastError());
    cudaFree(kF); cudaFree(kG); cudaFree(kS); cudaFree(vS); cudaFree(tmp); cudaFree(dcnt); cudaFree(head); cudaFree(ukey);
    st.ready = true;
    return DODE_OK;
#undef CSR_CU
}

// ---- hot path ------------------------------------------------------------------------------------
// dst[i*bp + d] = src[day_d*dayStride + i] for i < rowLen, d < bp (pad days -> 0).  32x32 smem transpose.
// BYPOS: the source is indexed by the position in the day list (a caller's per-step buffer) instead of the day id.
template <typename SrcT, bool BYPOS>
__global__ void __launch_bounds__(256)
gather_days(const SrcT* __restrict__ src, size_t dayStride, long rowLen, float* __restrict__ dst, int bp,
            const __grid_constant__ DayList dl) {
    __shared__ float tile[32][33];
    const long i0 = (long)blockIdx.x * 32;
    const int d0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int dd = ty; dd < 32; dd += 8) {
        const int d = d0 + dd;
        const long i = i0 + tx;
        tile[dd][tx] = (d < dl.n && i < rowLen) ? (float)__ldg(src + (size_t)(BYPOS ? d : dl.day[d]) * dayStride + i) : 0.f;
    }
    __syncthreads();
    for (int ii = ty; ii < 32; ii += 8) {
        const long i = i0 + ii;
        if (i < rowLen && d0 + tx < bp) dst[i * bp + d0 + tx] = tile[tx][ii];
    }
}

// q[day_d*dayStride + i] = src[i*bp + d] for d < n
__global__ void __launch_bounds__(256)
scatter_days(const float* __restrict__ src, int bp, long rowLen, float* __restrict__ dst, size_t dayStride,
             const __grid_constant__ DayList dl) {
    __shared__ float tile[32][33];
    const long i0 = (long)blockIdx.x * 32;
    const int d0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int ii = ty; ii < 32; ii += 8) {
        const long i = i0 + ii;
        tile[ii][tx] = (i < rowLen && d0 + tx < bp) ? src[i * bp + d0 + tx] : 0.f;
    }
    __syncthreads();
    for (int dd = ty; dd < 32; dd += 8) {
        const int d = d0 + dd;
        const long i = i0 + tx;
        if (d < dl.n && i < rowLen) dst[(size_t)dl.day[d] * dayStride + i] = tile[tx][dd];
    }
}

// A lane owns DV consecutive days of a panel row (day = lane*DV + e): one 16-byte vector access per lane and row.  (The
// other mapping, day = lane + 32*e with one 128-byte line per load instruction, was measured 8 % slower on configs[4].)
template <int DV> struct DVec;
template <> struct DVec<1> { using type = float; };
template <> struct DVec<2> { using type = float2; };
template <> struct DVec<4> { using type = float4; };
template <int DV> __device__ __forceinline__ int day_of(int lane, int e) { return lane * DV + e; }

// Accumulator of one output row over a lane's DV days.  Both CSR passes are bound by instruction issue (about 28 per
// gathered row at an IPC near 2), so the multiply-adds are issued as packed pairs: fma.rn.f32x2 (sm_100) does two fp32 FMAs
// per instruction, and ptxas takes the duplicated scalar factor as a broadcast operand (SASS: FFMA2 Rd, Ra.F32,
// Rb.F32x2.HI_LO, Rc.F32x2.HI_LO) — half the FMA instructions, same arithmetic (each half is an ordinary fp32 fma.rn).
__device__ __forceinline__ unsigned long long pack2(float a, float b) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
template <int DV> struct DayAcc;
template <> struct DayAcc<1> {
    float a = 0.f;
    __device__ __forceinline__ void fma(float v, const float* q) { a = fmaf(v, q[0], a); }
    __device__ __forceinline__ void get(float* o) const { o[0] = a; }
};
template <> struct DayAcc<2> {
    unsigned long long p = 0ull;
    __device__ __forceinline__ void fma(float v, const float* q) { p = ffma2(pack2(v, v), pack2(q[0], q[1]), p); }
    __device__ __forceinline__ void get(float* o) const { asm("mov.b64 {%0, %1}, %2;" : "=f"(o[0]), "=f"(o[1]) : "l"(p)); }
};
template <> struct DayAcc<4> {
    unsigned long long p0 = 0ull, p1 = 0ull;
    __device__ __forceinline__ void fma(float v, const float* q) {
        const unsigned long long vv = pack2(v, v);
        p0 = ffma2(vv, pack2(q[0], q[1]), p0);
        p1 = ffma2(vv, pack2(q[2], q[3]), p1);
    }
    __device__ __forceinline__ void get(float* o) const {
        asm("mov.b64 {%0, %1}, %2;" : "=f"(o[0]), "=f"(o[1]) : "l"(p0));
        asm("mov.b64 {%0, %1}, %2;" : "=f"(o[2]), "=f"(o[3]) : "l"(p1));
    }
};
template <int DV> __device__ __forceinline__ void ld_days(const float* __restrict__ row, int lane, float* v) {
    const typename DVec<DV>::type t = *reinterpret_cast<const typename DVec<DV>::type*>(row + lane * DV);
#pragma unroll
    for (int e = 0; e < DV; ++e) v[e] = reinterpret_cast<const float*>(&t)[e];
}
template <int DV> __device__ __forceinline__ void st_days(float* __restrict__ row, int lane, const float* v) {
    typename DVec<DV>::type t;
#pragma unroll
    for (int e = 0; e < DV; ++e) reinterpret_cast<float*>(&t)[e] = v[e];
    *reinterpret_cast<typename DVec<DV>::type*>(row + lane * DV) = t;
}


// a2 (CSR): one warp per row block (t/2, l/4) of F = 8 output rows; lanes along days (DV days per lane, bp = 32*DV).
//   r[(t*L+l)*rbp + d] = sum_k val_k[(t%2)*4 + l%4] * Qb[(base + pay_k)*bp + d] - x[day_d][t][l]    for d < rbp,
//   base = (2*(t/2) - H)*Np.  The counts are read straight from x[D][T][L] (one scalar per output and day).
// A chunk of 32 entries is fetched by the whole warp with coalesced loads; the eight values of an entry are then
// broadcast from shared memory (two LDS.128 at a warp-uniform address) and its payload by one shuffle — nine shuffles
// per entry would cost more LSU slots than the 512-byte gather they accompany.
template <int DV>
__global__ void __launch_bounds__(256, 3)
csr_fwd(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ pay, const float4* __restrict__ val,
        const float* __restrict__ Qb, const float* __restrict__ x, const float* __restrict__ Mb, float* __restrict__ r,
        long rblocks, int T, int H, int L, int LB, int Np, int rbp, const __grid_constant__ DayList dl) {
    constexpr int bp = 32 * DV;
    __shared__ float4 sval[8][64];                   // per warp: 32 entries x 2 float4
    // Warps walk the row blocks LINK-BLOCK-major, time-minor: the warps in flight then cover a few dozen neighbouring
    // link blocks over all t, whose OD sets overlap (paths are link runs), so the panel rows they gather (~100 MB) stay
    // in L2; time-major order would sweep the whole 25-lag window of every OD (256 MB) for every t.
    const long w = (blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    if (w >= rblocks) return;
    const int TB = (int)(rblocks / LB);
    const long lb = w / TB, tb = w - lb * TB;
    const long rb = tb * LB + lb;
    const int l0 = (int)lb * kRB;
    const int64_t k0 = rowptr[rb], k1 = rowptr[rb + 1];
    const float* qrow = Qb + ((long)tb * kFT - H) * Np * bp;                  // entries only reach rows >= 0
    DayAcc<DV> accp[kFS];
    for (int64_t kb = k0; kb < k1; kb += 32) {
        const int cnt = (int)min((int64_t)32, k1 - kb);
        const int o = lane < cnt ? __ldg(pay + kb + lane) : 0;
        __syncwarp();                                // the previous chunk's values have been read
        if (lane < 2 * cnt) sval[wib][lane] = __ldg(val + 2 * kb + lane);
        if (lane + 32 < 2 * cnt) sval[wib][lane + 32] = __ldg(val + 2 * kb + lane + 32);
        __syncwarp();
        int j = 0;
        for (; j + kInFlightF <= cnt; j += kInFlightF) {
            float qv[kInFlightF][DV];
#pragma unroll
            for (int u = 0; u < kInFlightF; ++u) {
                const int oo = __shfl_sync(0xffffffffu, o, j + u);
                ld_days<DV>(qrow + (long)oo * bp, lane, qv[u]);
            }
#pragma unroll
            for (int u = 0; u < kInFlightF; ++u) {
                const float4 va = sval[wib][2 * (j + u)], vb = sval[wib][2 * (j + u) + 1];
                const float vv[kFS] = {va.x, va.y, va.z, va.w, vb.x, vb.y, vb.z, vb.w};
#pragma unroll
                for (int i = 0; i < kFS; ++i) accp[i].fma(vv[i], qv[u]);
            }
        }
        for (; j < cnt; ++j) {
            const int oo = __shfl_sync(0xffffffffu, o, j);
            float qf[DV];
            ld_days<DV>(qrow + (long)oo * bp, lane, qf);
            const float4 va = sval[wib][2 * j], vb = sval[wib][2 * j + 1];
            const float vv[kFS] = {va.x, va.y, va.z, va.w, vb.x, vb.y, vb.z, vb.w};
#pragma unroll
            for (int i = 0; i < kFS; ++i) accp[i].fma(vv[i], qf);
        }
    }
    float acc[kFS][DV];
#pragma unroll
    for (int i = 0; i < kFS; ++i) accp[i].get(acc[i]);
#pragma unroll
    for (int i = 0; i < kFS; ++i) {
        const int l = l0 + (i & (kRB - 1));
        const long t = tb * kFT + (i >> 2);
        if (l >= L || t >= T) continue;
        const size_t row = (size_t)t * L + l;
        if (x != nullptr) {
#pragma unroll
            for (int e = 0; e < DV; ++e) {
                const int d = day_of<DV>(lane, e);
                acc[i][e] = d < dl.n ? acc[i][e] - __ldg(x + ((size_t)dl.day[d] * T + t) * L + l) : 0.f;   // pad days: r = 0
            }
        }
        if (Mb != nullptr) {                      // rows outside the chunk B_o contribute no residual
            float mf[DV];
            ld_days<DV>(Mb + row * bp, lane, mf);
#pragma unroll
            for (int e = 0; e < DV; ++e) acc[i][e] = mf[e] != 0.f ? acc[i][e] : 0.f;
        }
        if (rbp == bp) {
            st_days<DV>(r + row * bp, lane, acc[i]);
        } else {
#pragma unroll
            for (int e = 0; e < DV; ++e)
                if (day_of<DV>(lane, e) < rbp) r[row * rbp + day_of<DV>(lane, e)] = acc[i][e];
        }
    }
}

// a3+a4 (CSR): one warp per row block (s/4, n) of G.  g_i[d] = sum_k val_k[i] * r[((4*sb)*L + kl_k)*rbp + d], s = 4*sb+i;
// UPDATE: Qb[(s*Np+n)*bp + d] = max(0, Qb - eta g_i); else gout[s*N + n] = g_i[0].
template <int DV, bool UPDATE>
__global__ void __launch_bounds__(256, 4)
csr_grad(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ kl, const float4* __restrict__ val,
         const int32_t* __restrict__ perm, const float* __restrict__ r, float* __restrict__ Qb, float* __restrict__ gout, float eta,
         float* __restrict__ Gb, float eps, long rblocks, int T, int L, int N, int Np, int rbp) {
    constexpr int bp = 32 * DV;
    // Warps walk the row blocks OD-major in path order (perm: ODs sorted by the first link of their path), time-minor:
    // the warps in flight then gather residual rows of a few dozen neighbouring links over all t (~10 MB, L2-resident)
    // instead of the 28-interval window of every link (72 MB, which thrashes a 63 MB L2 partition).
    const long w = (blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= rblocks) return;
    const long SB = rblocks / Np;
    const long i = w / SB, sb = w - i * SB;
    const int n = __ldg(perm + i);
    if (n >= N) return;
    const long rb = sb * Np + n;
    const int64_t k0 = rowptr[rb], k1 = rowptr[rb + 1];
    const bool full = rbp == bp;
    const float* rrow = r + (size_t)sb * kRB * L * rbp;
    // A chunk of 32 entries is fetched by the whole warp with coalesced loads and parked in shared memory; an entry's
    // payload and its four values are then read back at a warp-uniform address (one LDS.32 + one LDS.128, one wavefront
    // each) instead of five shuffles per gathered row: the pass is bound by the LSU/MIO pipe, which the 512-byte gathers
    // already keep busy.
    __shared__ float4 sval[8][32];
    __shared__ int sidx[8][32];
    const int wib = threadIdx.x >> 5;
    DayAcc<DV> accp[kRB];
    for (int64_t kb = k0; kb < k1; kb += 32) {
        const int64_t k = kb + lane;
        const int cnt = (int)min((int64_t)32, k1 - kb);
        __syncwarp();                                // the previous chunk has been read
        sidx[wib][lane] = k < k1 ? __ldg(kl + k) : 0;
        sval[wib][lane] = k < k1 ? __ldg(val + k) : make_float4(0.f, 0.f, 0.f, 0.f);
        __syncwarp();
        int j = 0;
        if (full) {
            for (; j + kInFlightG <= cnt; j += kInFlightG) {
                float rv[kInFlightG][DV];
#pragma unroll
                for (int u = 0; u < kInFlightG; ++u) ld_days<DV>(rrow + (long)sidx[wib][j + u] * bp, lane, rv[u]);
#pragma unroll
                for (int u = 0; u < kInFlightG; ++u) {
                    const float4 v = sval[wib][j + u];
                    const float vv[kRB] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int i = 0; i < kRB; ++i) accp[i].fma(vv[i], rv[u]);
                }
            }
        }
        for (; j < cnt; ++j) {
            const int oo = sidx[wib][j];
            const float4 v = sval[wib][j];
            const float v4[kRB] = {v.x, v.y, v.z, v.w};
            float rf[DV];
            if (full) {
                ld_days<DV>(rrow + (long)oo * bp, lane, rf);
            } else {
#pragma unroll
                for (int e = 0; e < DV; ++e)
                    rf[e] = day_of<DV>(lane, e) < rbp ? rrow[(long)oo * rbp + day_of<DV>(lane, e)] : 0.f;
            }
#pragma unroll
            for (int i = 0; i < kRB; ++i) accp[i].fma(v4[i], rf);
        }
    }
    float acc[kRB][DV];
#pragma unroll
    for (int i = 0; i < kRB; ++i) accp[i].get(acc[i]);
#pragma unroll
    for (int i = 0; i < kRB; ++i) {
        const long s = sb * kRB + i;
        if (s >= T) break;
        if (UPDATE) {
            float* qp = Qb + ((size_t)s * Np + n) * bp;
            float qf[DV];
            ld_days<DV>(qp, lane, qf);
#pragma unroll
            for (int e = 0; e < DV; ++e) {
                if (Gb != nullptr) qf[e] = adagrad_update(qf[e], acc[i][e], Gb + ((size_t)s * Np + n) * bp + day_of<DV>(lane, e), eta, eps);
                else qf[e] = fmaxf(0.f, fmaf(-eta, acc[i][e], qf[e]));
            }
            st_days<DV>(qp, lane, qf);
        } else if (lane == 0) {
            gout[(size_t)s * N + n] = acc[i][0];
        }
    }
}

inline int csr_bp(int n) { return n <= 32 ? 32 : n <= 64 ? 64 : 128; }

inline int csr_ensure(CsrStore& st, const dode_dims& d, int Np, int bp, cudaStream_t stream) {
    if (st.cap_bp >= bp) return DODE_OK;
    cudaStreamSynchronize(stream);
    cudaFree(st.Qb);
    st.Qb = nullptr; st.cap_bp = 0;
    if (cudaMalloc(&st.Qb, (size_t)d.T * Np * bp * 4) != cudaSuccess) return DODE_ENOMEM;
    st.cap_bp = bp;
    return DODE_OK;
}

// state gather + forward.  rbp: stride of r (== bp for steps/objective, 1 for dode_apply).
inline int csr_ensure_ada(CsrStore& st, const dode_dims& d, int Np, int bp, cudaStream_t stream) {
    if (st.cap_bp_ada >= bp) return DODE_OK;
    cudaStreamSynchronize(stream);
    cudaFree(st.Mb); cudaFree(st.Gb);
    st.Mb = st.Gb = nullptr; st.cap_bp_ada = 0;
    if (cudaMalloc(&st.Mb, (size_t)d.T * d.L * bp * 4) != cudaSuccess) return DODE_ENOMEM;
    if (cudaMalloc(&st.Gb, (size_t)d.T * Np * bp * 4) != cudaSuccess) return DODE_ENOMEM;
    st.cap_bp_ada = bp;
    return DODE_OK;
}

// mask (nullable): device bytes [n][T][L] by position in the day list
inline int csr_forward(CsrStore& st, int c, const float* qbase, size_t dayStride, const float* xbase, float* r,
                       int bp, int rbp, const DayList& dl, const dode_dims& d, int Np, cudaStream_t stream,
                       int64_t* launches, const uint8_t* mask = nullptr) {
    int rc = csr_ensure(st, d, Np, bp, stream);
    if (rc) return rc;
    if (mask && (rc = csr_ensure_ada(st, d, Np, bp, stream))) return rc;
    const CsrCluster& cl = st.cl[c];
    const long qlen = (long)d.T * Np, xlen = (long)d.T * d.L;
    gather_days<float, false><<<dim3((unsigned)((qlen + 31) / 32), bp / 32), 256, 0, stream>>>(qbase, dayStride, qlen, st.Qb, bp, dl);
    if (mask) {
        gather_days<uint8_t, true><<<dim3((unsigned)((xlen + 31) / 32), bp / 32), 256, 0, stream>>>(mask, (size_t)d.T * d.L, xlen, st.Mb, bp, dl);
        *launches += 1;
    }
    const float* Mb = mask ? st.Mb : nullptr;
    const int LB = (d.L + kRB - 1) / kRB;
    const long rblocks = (long)((d.T + kFT - 1) / kFT) * LB;
    const unsigned grid = (unsigned)((rblocks * 32 + 255) / 256);
    switch (bp) {
        case 32: csr_fwd<1><<<grid, 256, 0, stream>>>(cl.rowptrF, cl.payF, cl.valF, st.Qb, xbase, Mb, r, rblocks, d.T, d.H, d.L, LB, Np, rbp, dl); break;
        case 64: csr_fwd<2><<<grid, 256, 0, stream>>>(cl.rowptrF, cl.payF, cl.valF, st.Qb, xbase, Mb, r, rblocks, d.T, d.H, d.L, LB, Np, rbp, dl); break;
        default: csr_fwd<4><<<grid, 256, 0, stream>>>(cl.rowptrF, cl.payF, cl.valF, st.Qb, xbase, Mb, r, rblocks, d.T, d.H, d.L, LB, Np, rbp, dl); break;
    }
    *launches += 2;
    return DODE_OK;
}

// gradient + update on Qb + scatter back to q (UPDATE), or g -> gout for minibatch 1 (dode_apply_t, rbp = 1)
inline int csr_gradient(CsrStore& st, int c, const float* r, float* qbase, size_t dayStride, float* gout, float eta,
                        int bp, int rbp, const DayList& dl, const dode_dims& d, int Np, cudaStream_t stream,
                        int64_t* launches, float* Gbase = nullptr, float eps = 0.f) {
    int rc = csr_ensure(st, d, Np, bp, stream);
    if (rc) return rc;
    if (Gbase && (rc = csr_ensure_ada(st, d, Np, bp, stream))) return rc;
    const CsrCluster& cl = st.cl[c];
    const long rows = (long)d.T * Np;
    const long rblocks = (long)((d.T + kRB - 1) / kRB) * Np;
    const unsigned grid = (unsigned)((rblocks * 32 + 255) / 256);
    if (gout) {
        csr_grad<1, false><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.payG, cl.valG, cl.permG, r, nullptr, gout, eta, nullptr, 0.f, rblocks, d.T, d.L, d.N, Np, rbp);
        *launches += 1;
        return DODE_OK;
    }
    float* Gb = nullptr;
    if (Gbase) {                      // Adagrad accumulator of the minibatch days as a day-fastest panel, like Qb
        gather_days<float, false><<<dim3((unsigned)((rows + 31) / 32), bp / 32), 256, 0, stream>>>(Gbase, dayStride, rows, st.Gb, bp, dl);
        Gb = st.Gb;
        *launches += 1;
    }
    switch (bp) {
        case 32: csr_grad<1, true><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.payG, cl.valG, cl.permG, r, st.Qb, nullptr, eta, Gb, eps, rblocks, d.T, d.L, d.N, Np, rbp); break;
        case 64: csr_grad<2, true><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.payG, cl.valG, cl.permG, r, st.Qb, nullptr, eta, Gb, eps, rblocks, d.T, d.L, d.N, Np, rbp); break;
        default: csr_grad<4, true><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.payG, cl.valG, cl.permG, r, st.Qb, nullptr, eta, Gb, eps, rblocks, d.T, d.L, d.N, Np, rbp); break;
    }
    scatter_days<<<dim3((unsigned)((rows + 31) / 32), bp / 32), 256, 0, stream>>>(st.Qb, bp, rows, qbase, dayStride, dl);
    if (Gbase) {
        scatter_days<<<dim3((unsigned)((rows + 31) / 32), bp / 32), 256, 0, stream>>>(st.Gb, bp, rows, Gbase, dayStride, dl);
        *launches += 1;
    }
    *launches += 2;
    return DODE_OK;
}

}  // namespace dode
