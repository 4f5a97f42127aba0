// a6: block-sparse CSR variant of a2-a4 for large networks (BASELINE.json configs[4]).
//
// The boundary format is one CSR per (c,s,h) block (include/dode.h).  At create time each cluster is
// re-packed, on the device, into two lag-merged CSR matrices so that both passes stream their non-zeros
// contiguously and deterministically (no atomics on the hot path):
//   F (forward):  row (t,l) holds every entry of blocks (t-h,h), h<=min(H,t):  (off = n - h*Np, val)
//                 so that the operand is Qb[(t*Np + off)*bp + d]
//   G (gradient): row (s,n) holds every entry of blocks (s,h), s+h<T:           (kl = h*L + l, val)
//                 so that the operand is r[(s*L + kl)*bp + d]
// Entries with s+h >= T are dropped.  The re-pack is a stable radix sort of 64-bit keys
// (CUB, create-time only).
//
// Hot path: the minibatch state is gathered once per step into day-fastest panels Qb[T*Np][bp] and
// Xb[T*L][bp] (coalesced transposes), so that one non-zero pulls bp contiguous floats; a warp owns one
// CSR row and its lanes run along the days.  The update q <- max(0, q - eta g) is applied to Qb in the
// gradient kernel's epilogue and scattered back to q[d][s][n].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <cub/device/device_radix_sort.cuh>

#include "../../include/dode.h"
#include "kernels_dense.cuh"

namespace dode {

constexpr int kCsrMaxDays = 128;

struct CsrCluster {
    int64_t* rowptrF = nullptr;   // [T*L + 1]
    int32_t* offF = nullptr;      // [nnzF]
    float* valF = nullptr;
    int64_t* rowptrG = nullptr;   // [T*N + 1]
    int32_t* klG = nullptr;       // [nnzG]
    float* valG = nullptr;
    int64_t nnz = 0;              // valid entries (s+h < T)
};

struct CsrStore {
    bool ready = false;
    int C = 0;
    CsrCluster* cl = nullptr;     // host array [C]
    float* Qb = nullptr;          // [T*Np][bp]
    float* Xb = nullptr;          // [T*L][bp]
    int cap_bp = 0;
};

// ---- create-time re-pack ---------------------------------------------------------------------------
// one warp per input CSR row (s,h,l) of cluster c
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
    const unsigned long long KF = (unsigned long long)(H + 1) * Np, KG = (unsigned long long)(H + 1) * L;
    const bool valid = s + h < T;
    for (int64_t k = k0 + lane; k < k1; k += 32) {
        const int n = col_idx[k];
        keyF[k - base] = valid ? ((unsigned long long)(s + h) * L + l) * KF + (unsigned long long)h * Np + n : ~0ull;
        keyG[k - base] = valid ? ((unsigned long long)s * Np + n) * KG + (unsigned long long)h * L + l : ~0ull;
    }
}

// rowptr[row] = lower_bound(keys, row*K); decoded payload: F -> n - h*Np, G -> h*L + l
__global__ void csr_rowptr(const unsigned long long* __restrict__ keys, int64_t nvalid, long rows,
                           unsigned long long K, int64_t* __restrict__ rowptr) {
    const long row = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (row > rows) return;
    const unsigned long long target = (unsigned long long)row * K;
    int64_t lo = 0, hi = nvalid;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (keys[mid] < target) lo = mid + 1; else hi = mid;
    }
    rowptr[row] = lo;
}

__global__ void csr_decode(const unsigned long long* __restrict__ keys, int64_t nvalid, unsigned long long K,
                           int Np, int forward, int32_t* __restrict__ out) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < nvalid; i += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long rem = keys[i] % K;
        if (forward) {
            const int h = (int)(rem / Np), n = (int)(rem - (unsigned long long)h * Np);
            out[i] = n - h * Np;
        } else {
            out[i] = (int32_t)rem;
        }
    }
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
            cudaFree(st.cl[c].rowptrF); cudaFree(st.cl[c].offF); cudaFree(st.cl[c].valF);
            cudaFree(st.cl[c].rowptrG); cudaFree(st.cl[c].klG); cudaFree(st.cl[c].valG);
        }
        delete[] st.cl;
        st.cl = nullptr;
    }
    cudaFree(st.Qb); cudaFree(st.Xb);
    st.Qb = st.Xb = nullptr;
    st.ready = false;
}

inline int csr_build(CsrStore& st, const dode_dims& d, const dode_dar& R, cudaStream_t stream, char* err) {
#define CSR_CU(call)                                                                             \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            snprintf(err, 512, "%s: %s", #call, cudaGetErrorString(e_));                         \
            cudaFree(kF); cudaFree(kG); cudaFree(kS); cudaFree(vS); cudaFree(tmp); cudaFree(dcnt); \
            return e_ == cudaErrorMemoryAllocation ? DODE_ENOMEM : DODE_ECUDA;                   \
        }                                                                                        \
    } while (0)
    const int Np = (d.N + 3) / 4 * 4;
    st.C = d.C;
    st.cl = new CsrCluster[d.C];
    const long nblk = (long)d.T * (d.H + 1);
    std::vector<int64_t> off(d.C + 1);
    unsigned long long *kF = nullptr, *kG = nullptr, *kS = nullptr, *dcnt = nullptr;
    float* vS = nullptr;
    void* tmp = nullptr;
    for (int c = 0; c <= d.C; ++c)
        CSR_CU(cudaMemcpyAsync(&off[c], R.blk_off + (long)c * nblk, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
    CSR_CU(cudaStreamSynchronize(stream));
    if (off[d.C] != R.nnz) { snprintf(err, 512, "blk_off[last]=%lld but nnz=%lld", (long long)off[d.C], (long long)R.nnz); return DODE_EINVAL; }
    int64_t maxn = 1;
    for (int c = 0; c < d.C; ++c) maxn = std::max<int64_t>(maxn, off[c + 1] - off[c]);
    CSR_CU(cudaMalloc(&kF, maxn * 8)); CSR_CU(cudaMalloc(&kG, maxn * 8)); CSR_CU(cudaMalloc(&kS, maxn * 8));
    CSR_CU(cudaMalloc(&vS, maxn * 4)); CSR_CU(cudaMalloc(&dcnt, 8));
    size_t tmp_bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, kF, kS, (const float*)nullptr, vS, maxn, 0, 64, stream);
    CSR_CU(cudaMalloc(&tmp, tmp_bytes));
    const unsigned long long KF = (unsigned long long)(d.H + 1) * Np, KG = (unsigned long long)(d.H + 1) * d.L;
    for (int c = 0; c < d.C; ++c) {
        CsrCluster& cl = st.cl[c];
        const int64_t n = off[c + 1] - off[c];
        const long rows_in = nblk * d.L;
        if (n > 0) {
            csr_expand_keys<<<(unsigned)((rows_in * 32 + 255) / 256), 256, 0, stream>>>(
                R.blk_off, R.row_ptr, R.col_idx, c, d.N, Np, d.L, d.T, d.H, off[c], kF, kG);
            CSR_CU(cudaMemsetAsync(dcnt, 0, 8, stream));
            count_invalid<<<1184, 256, 0, stream>>>(kF, n, dcnt);
        }
        unsigned long long ninv = 0;
        if (n > 0) CSR_CU(cudaMemcpyAsync(&ninv, dcnt, 8, cudaMemcpyDeviceToHost, stream));
        CSR_CU(cudaStreamSynchronize(stream));
        const int64_t nv = n - (int64_t)ninv;
        cl.nnz = nv;
        const long rowsF = (long)d.T * d.L, rowsG = (long)d.T * Np;
        CSR_CU(cudaMalloc(&cl.rowptrF, (rowsF + 1) * 8)); CSR_CU(cudaMalloc(&cl.rowptrG, (rowsG + 1) * 8));
        CSR_CU(cudaMalloc(&cl.offF, std::max<int64_t>(nv, 1) * 4)); CSR_CU(cudaMalloc(&cl.valF, std::max<int64_t>(nv, 1) * 4));
        CSR_CU(cudaMalloc(&cl.klG, std::max<int64_t>(nv, 1) * 4)); CSR_CU(cudaMalloc(&cl.valG, std::max<int64_t>(nv, 1) * 4));
        for (int pass = 0; pass < 2; ++pass) {
            unsigned long long* kin = pass == 0 ? kF : kG;
            const unsigned long long K = pass == 0 ? KF : KG;
            const long rows = pass == 0 ? rowsF : rowsG;
            float* vout = pass == 0 ? cl.valF : cl.valG;
            if (n > 0) {
                // invalid keys are all-ones: sort on all 64 bits so they land at the end
                CSR_CU(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, kin, kS, R.val + off[c], vS, n, 0, 64, stream));
                CSR_CU(cudaMemcpyAsync(vout, vS, nv * 4, cudaMemcpyDeviceToDevice, stream));
                csr_decode<<<1184, 256, 0, stream>>>(kS, nv, K, Np, pass == 0, pass == 0 ? cl.offF : cl.klG);
            }
            csr_rowptr<<<(unsigned)((rows + 1 + 255) / 256), 256, 0, stream>>>(kS, nv, rows, K, pass == 0 ? cl.rowptrF : cl.rowptrG);
        }
        CSR_CU(cudaStreamSynchronize(stream));
    }
    CSR_CU(cudaGetLastError());
    cudaFree(kF); cudaFree(kG); cudaFree(kS); cudaFree(vS); cudaFree(tmp); cudaFree(dcnt);
    st.ready = true;
    return DODE_OK;
#undef CSR_CU
}

// ---- hot path ------------------------------------------------------------------------------------
// dst[i*bp + d] = src[day_d*dayStride + i] for i < rowLen, d < bp (pad days -> 0).  32x32 smem transpose.
__global__ void __launch_bounds__(256)
gather_days(const float* __restrict__ src, size_t dayStride, long rowLen, float* __restrict__ dst, int bp,
            const __grid_constant__ DayList dl) {
    __shared__ float tile[32][33];
    const long i0 = (long)blockIdx.x * 32;
    const int d0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int dd = ty; dd < 32; dd += 8) {
        const int d = d0 + dd;
        const long i = i0 + tx;
        tile[dd][tx] = (d < dl.n && i < rowLen) ? __ldg(src + (size_t)dl.day[d] * dayStride + i) : 0.f;
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

template <int DV> struct DVec;
template <> struct DVec<1> { using type = float; };
template <> struct DVec<2> { using type = float2; };
template <> struct DVec<4> { using type = float4; };

// a2 (CSR): one warp per row (t,l) of F; lanes along days (DV days per lane, bp = 32*DV).
// r[(t*L+l)*rbp + d] = sum_k val_k * Qb[(t*Np + off_k)*bp + d] - Xb[(t*L+l)*bp + d]   for d < rbp
template <int DV>
__global__ void __launch_bounds__(256)
csr_fwd(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ off, const float* __restrict__ val,
        const float* __restrict__ Qb, const float* __restrict__ Xb, float* __restrict__ r,
        long rows, int L, int Np, int rbp) {
    constexpr int bp = 32 * DV;
    using vec = typename DVec<DV>::type;
    const long row = (blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (row >= rows) return;
    const long t = row / L;
    const int64_t k0 = rowptr[row], k1 = rowptr[row + 1];
    const float* qrow = Qb + (size_t)t * Np * bp + lane * DV;
    float acc[DV];
#pragma unroll
    for (int e = 0; e < DV; ++e) acc[e] = 0.f;
    for (int64_t kb = k0; kb < k1; kb += 32) {
        const int64_t k = kb + lane;
        const int o = k < k1 ? __ldg(off + k) : 0;
        const float v = k < k1 ? __ldg(val + k) : 0.f;
        const int cnt = (int)min((int64_t)32, k1 - kb);
        int j = 0;
        for (; j + 4 <= cnt; j += 4) {
            vec qv[4]; float vv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int oo = __shfl_sync(0xffffffffu, o, j + u);
                vv[u] = __shfl_sync(0xffffffffu, v, j + u);
                qv[u] = *reinterpret_cast<const vec*>(qrow + (long)oo * bp);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float* qf = reinterpret_cast<const float*>(&qv[u]);
#pragma unroll
                for (int e = 0; e < DV; ++e) acc[e] = fmaf(vv[u], qf[e], acc[e]);
            }
        }
        for (; j < cnt; ++j) {
            const int oo = __shfl_sync(0xffffffffu, o, j);
            const float vv = __shfl_sync(0xffffffffu, v, j);
            const vec qv = *reinterpret_cast<const vec*>(qrow + (long)oo * bp);
            const float* qf = reinterpret_cast<const float*>(&qv);
#pragma unroll
            for (int e = 0; e < DV; ++e) acc[e] = fmaf(vv, qf[e], acc[e]);
        }
    }
    if (Xb != nullptr) {
        const vec xv = *reinterpret_cast<const vec*>(Xb + (size_t)row * bp + lane * DV);
        const float* xf = reinterpret_cast<const float*>(&xv);
#pragma unroll
        for (int e = 0; e < DV; ++e) acc[e] -= xf[e];
    }
    if (rbp == bp) {
        vec out;
        float* of = reinterpret_cast<float*>(&out);
#pragma unroll
        for (int e = 0; e < DV; ++e) of[e] = acc[e];
        *reinterpret_cast<vec*>(r + (size_t)row * bp + lane * DV) = out;
    } else {
#pragma unroll
        for (int e = 0; e < DV; ++e)
            if (lane * DV + e < rbp) r[(size_t)row * rbp + lane * DV + e] = acc[e];
    }
}

// a3+a4 (CSR): one warp per row (s,n) of G.  g[d] = sum_k val_k * r[(s*L + kl_k)*rbp + d];
// UPDATE: Qb[(s*Np+n)*bp + d] = max(0, Qb - eta g); else gout[s*N + n] = g[0].
template <int DV, bool UPDATE>
__global__ void __launch_bounds__(256)
csr_grad(const int64_t* __restrict__ rowptr, const int32_t* __restrict__ kl, const float* __restrict__ val,
         const float* __restrict__ r, float* __restrict__ Qb, float* __restrict__ gout, float eta,
         long rows, int L, int N, int Np, int rbp) {
    constexpr int bp = 32 * DV;
    using vec = typename DVec<DV>::type;
    const long row = (blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (row >= rows) return;
    const long s = row / Np;
    const int n = (int)(row - s * Np);
    if (n >= N) return;
    const int64_t k0 = rowptr[row], k1 = rowptr[row + 1];
    const bool full = rbp == bp;
    const float* rrow = r + (size_t)s * L * rbp + lane * DV;
    float acc[DV];
#pragma unroll
    for (int e = 0; e < DV; ++e) acc[e] = 0.f;
    for (int64_t kb = k0; kb < k1; kb += 32) {
        const int64_t k = kb + lane;
        const int o = k < k1 ? __ldg(kl + k) : 0;
        const float v = k < k1 ? __ldg(val + k) : 0.f;
        const int cnt = (int)min((int64_t)32, k1 - kb);
        int j = 0;
        if (full) {
            for (; j + 4 <= cnt; j += 4) {
                vec rv[4]; float vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int oo = __shfl_sync(0xffffffffu, o, j + u);
                    vv[u] = __shfl_sync(0xffffffffu, v, j + u);
                    rv[u] = *reinterpret_cast<const vec*>(rrow + (long)oo * bp);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float* rf = reinterpret_cast<const float*>(&rv[u]);
#pragma unroll
                    for (int e = 0; e < DV; ++e) acc[e] = fmaf(vv[u], rf[e], acc[e]);
                }
            }
        }
        for (; j < cnt; ++j) {
            const int oo = __shfl_sync(0xffffffffu, o, j);
            const float vv = __shfl_sync(0xffffffffu, v, j);
#pragma unroll
            for (int e = 0; e < DV; ++e)
                if (full || lane * DV + e < rbp) acc[e] = fmaf(vv, rrow[(long)oo * rbp + e], acc[e]);
        }
    }
    if (UPDATE) {
        vec* qp = reinterpret_cast<vec*>(Qb + (size_t)row * bp + lane * DV);
        vec qv = *qp;
        float* qf = reinterpret_cast<float*>(&qv);
#pragma unroll
        for (int e = 0; e < DV; ++e) qf[e] = fmaxf(0.f, fmaf(-eta, acc[e], qf[e]));
        *qp = qv;
    } else if (lane == 0) {
        gout[(size_t)s * N + n] = acc[0];
    }
}

inline int csr_bp(int n) { return n <= 32 ? 32 : n <= 64 ? 64 : 128; }

inline int csr_ensure(CsrStore& st, const dode_dims& d, int Np, int bp, cudaStream_t stream) {
    if (st.cap_bp >= bp) return DODE_OK;
    cudaStreamSynchronize(stream);
    cudaFree(st.Qb); cudaFree(st.Xb);
    st.Qb = st.Xb = nullptr; st.cap_bp = 0;
    if (cudaMalloc(&st.Qb, (size_t)d.T * Np * bp * 4) != cudaSuccess) return DODE_ENOMEM;
    if (cudaMalloc(&st.Xb, (size_t)d.T * d.L * bp * 4) != cudaSuccess) return DODE_ENOMEM;
    st.cap_bp = bp;
    return DODE_OK;
}

// gathers + forward.  rbp: stride of r (== bp for steps/objective, 1 for dode_apply).
inline int csr_forward(CsrStore& st, int c, const float* qbase, size_t dayStride, const float* xbase, float* r,
                       int bp, int rbp, const DayList& dl, const dode_dims& d, int Np, cudaStream_t stream,
                       int64_t* launches) {
    int rc = csr_ensure(st, d, Np, bp, stream);
    if (rc) return rc;
    const CsrCluster& cl = st.cl[c];
    const long qlen = (long)d.T * Np, xlen = (long)d.T * d.L;
    gather_days<<<dim3((unsigned)((qlen + 31) / 32), bp / 32), 256, 0, stream>>>(qbase, dayStride, qlen, st.Qb, bp, dl);
    if (xbase)
        gather_days<<<dim3((unsigned)((xlen + 31) / 32), bp / 32), 256, 0, stream>>>(xbase, (size_t)d.T * d.L, xlen, st.Xb, bp, dl);
    const unsigned grid = (unsigned)((xlen * 32 + 255) / 256);
    const float* Xb = xbase ? st.Xb : nullptr;
    switch (bp) {
        case 32: csr_fwd<1><<<grid, 256, 0, stream>>>(cl.rowptrF, cl.offF, cl.valF, st.Qb, Xb, r, xlen, d.L, Np, rbp); break;
        case 64: csr_fwd<2><<<grid, 256, 0, stream>>>(cl.rowptrF, cl.offF, cl.valF, st.Qb, Xb, r, xlen, d.L, Np, rbp); break;
        default: csr_fwd<4><<<grid, 256, 0, stream>>>(cl.rowptrF, cl.offF, cl.valF, st.Qb, Xb, r, xlen, d.L, Np, rbp); break;
    }
    *launches += xbase ? 3 : 2;
    return DODE_OK;
}

// gradient + update on Qb + scatter back to q (UPDATE), or g -> gout for minibatch 1 (dode_apply_t, rbp = 1)
inline int csr_gradient(CsrStore& st, int c, const float* r, float* qbase, size_t dayStride, float* gout, float eta,
                        int bp, int rbp, const DayList& dl, const dode_dims& d, int Np, cudaStream_t stream,
                        int64_t* launches) {
    int rc = csr_ensure(st, d, Np, bp, stream);
    if (rc) return rc;
    const CsrCluster& cl = st.cl[c];
    const long rows = (long)d.T * Np;
    const unsigned grid = (unsigned)((rows * 32 + 255) / 256);
    if (gout) {
        csr_grad<1, false><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.klG, cl.valG, r, nullptr, gout, eta, rows, d.L, d.N, Np, rbp);
        *launches += 1;
        return DODE_OK;
    }
    switch (bp) {
        case 32: csr_grad<1, true><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.klG, cl.valG, r, st.Qb, nullptr, eta, rows, d.L, d.N, Np, rbp); break;
        case 64: csr_grad<2, true><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.klG, cl.valG, r, st.Qb, nullptr, eta, rows, d.L, d.N, Np, rbp); break;
        default: csr_grad<4, true><<<grid, 256, 0, stream>>>(cl.rowptrG, cl.klG, cl.valG, r, st.Qb, nullptr, eta, rows, d.L, d.N, Np, rbp); break;
    }
    scatter_days<<<dim3((unsigned)((rows + 31) / 32), bp / 32), 256, 0, stream>>>(st.Qb, bp, rows, qbase, dayStride, dl);
    *launches += 2;
    return DODE_OK;
}

}  // namespace dode
