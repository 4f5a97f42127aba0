// NEXT-4: Step 1 of the framework, the DAR blocks of one day / one traffic pattern from link speeds
// (Eq. 17-18 and Example 3).  The paper calls this construction "the most time-consuming part in the
// DODE framework" and iterates "over departure time intervals and paths", walking the links of a path and computing
// the arrival time at each.  Here that double loop is the thread grid: one thread per (departure
// interval s, OD n) carries the leading (t = s dt) and the trailing (t = (s+1) dt) trajectory down the path; at the tail
// of every link the window [a1, a2) between them is cut at the interval boundaries and the shares
// |[a1,a2) ∩ H_h2| / (a2 - a1) go to R[s][h2 - s][l][n] (boundary layout of include/dode.h).  A trajectory crosses a link
// at the speed of the interval in which it enters it (reading A20).  Times are doubles: a day is 86 400 s and
// the shares need ~1e-7 of an interval.  R is zero-filled by the caller (cudaMemsetAsync) — the fill, not this kernel's
// scattered non-zeros, is what moves the bytes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dode {

__global__ void __launch_bounds__(256)
dar_build_dense(int N, int L, int T, int H, const int32_t* __restrict__ path_ptr, const int32_t* __restrict__ path_links,
                const float* __restrict__ len, const float* __restrict__ speed, double dt, float* __restrict__ R) {
    const long total = (long)T * N;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int s = (int)(i / N), n = (int)(i - (long)s * N);
        double a1 = (double)s * dt, a2 = (double)(s + 1) * dt;
        const int j1 = __ldg(path_ptr + n + 1);
        for (int j = __ldg(path_ptr + n); j < j1; ++j) {
            const int l = __ldg(path_links + j);
            const int h_first = (int)floor(a1 / dt);
            if (a2 > a1) {
                const int h_last = (int)floor(a2 / dt);
                const double inv = 1.0 / (a2 - a1);
                for (int h2 = h_first; h2 <= h_last; ++h2) {
                    const double lo = fmax(a1, (double)h2 * dt), hi = fmin(a2, (double)(h2 + 1) * dt);
                    const int h = h2 - s;
                    if (hi > lo && h <= H && h2 < T)
                        R[(((size_t)s * (H + 1) + h) * L + l) * N + n] = (float)((hi - lo) * inv);
                }
            } else if (h_first - s <= H && h_first < T) {
                R[(((size_t)s * (H + 1) + (h_first - s)) * L + l) * N + n] = 1.f;     // FIFO violated: all in one interval
            }
            const int i1 = min(T - 1, h_first), i2 = min(T - 1, (int)floor(a2 / dt));
            const double ll = (double)__ldg(len + l);
            a1 += ll / (double)__ldg(speed + (size_t)i1 * L + l);
            a2 += ll / (double)__ldg(speed + (size_t)i2 * L + l);
        }
    }
}

// Travel time of path k for the vehicle that leaves at time t0 (entry-interval speeds).
__device__ __forceinline__ double path_travel_time(int k, double t0, int L, int T, double dt, const int32_t* __restrict__ path_ptr,
                                                   const int32_t* __restrict__ path_links, const float* __restrict__ len,
                                                   const float* __restrict__ speed) {
    double t = t0;
    const int j1 = __ldg(path_ptr + k + 1);
    for (int j = __ldg(path_ptr + k); j < j1; ++j) {
        const int l = __ldg(path_links + j);
        const int i = min(T - 1, (int)floor(t / dt));
        t += (double)__ldg(len + l) / (double)__ldg(speed + (size_t)i * L + l);
    }
    return t - t0;
}

// B = delta * rho * p (Eq. 41) with several paths per OD and Logit route shares (Eq. 37,
// PAPER.md:309-312): thread (s, n) first evaluates the path travel times c_k(s) of the OD's paths for the vehicle leaving
// at s dt (kept in registers for up to 8 paths, re-walked beyond that), then walks every path once more
// as dar_build_dense does and ADDS share * rho into R[s][h][l][n].  Only this thread touches column (s, n), so the
// accumulation over paths that share a link is deterministic; the adds are issued as fire-and-forget reductions
// (atomicAdd with the result unused -> RED) because a plain `+=` is a dependent global load per entry and made the
// kernel a chain of memory latencies.  R zero-filled by the caller.
__global__ void __launch_bounds__(256)
assignment_build_dense(int N, int L, int T, int H, const int32_t* __restrict__ od_ptr, const int32_t* __restrict__ path_ptr,
                       const int32_t* __restrict__ path_links, const float* __restrict__ len,
                       const float* __restrict__ speed, double dt, double theta, float* __restrict__ R) {
    const long total = (long)T * N;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int s = (int)(i / N), n = (int)(i - (long)s * N);
        const int k0 = __ldg(od_ptr + n), k1 = __ldg(od_ptr + n + 1);
        const double t0 = (double)s * dt;
        constexpr int kCache = 8;                  // travel times of up to 8 paths stay in registers; beyond that they are re-walked
        double cc[kCache] = {};
        const bool cached = k1 - k0 <= kCache;
        auto ctime = [&](int k) {
            return cached ? cc[k - k0] : path_travel_time(k, t0, L, T, dt, path_ptr, path_links, len, speed);
        };
        double cmin = 1e300, z = 0.0;
        for (int k = k0; k < k1; ++k) {
            const double c = path_travel_time(k, t0, L, T, dt, path_ptr, path_links, len, speed);
            if (cached) cc[k - k0] = c;
            cmin = fmin(cmin, c);
        }
        for (int k = k0; k < k1; ++k) z += exp(-theta * (ctime(k) - cmin));
        for (int k = k0; k < k1; ++k) {
            const double share = exp(-theta * (ctime(k) - cmin)) / z;
            double a1 = t0, a2 = (double)(s + 1) * dt;
            const int j1 = __ldg(path_ptr + k + 1);
            for (int j = __ldg(path_ptr + k); j < j1; ++j) {
                const int l = __ldg(path_links + j);
                const int h_first = (int)floor(a1 / dt);
                if (a2 > a1) {
                    const int h_last = (int)floor(a2 / dt);
                    const double inv = share / (a2 - a1);
                    for (int h2 = h_first; h2 <= h_last; ++h2) {
                        const double lo = fmax(a1, (double)h2 * dt), hi = fmin(a2, (double)(h2 + 1) * dt);
                        const int h = h2 - s;
                        if (hi > lo && h <= H && h2 < T)
                            atomicAdd(R + (((size_t)s * (H + 1) + h) * L + l) * N + n, (float)((hi - lo) * inv));
                    }
                } else if (h_first - s <= H && h_first < T) {
                    atomicAdd(R + (((size_t)s * (H + 1) + (h_first - s)) * L + l) * N + n, (float)share);
                }
                const int i1 = min(T - 1, h_first), i2 = min(T - 1, (int)floor(a2 / dt));
                const double ll = (double)__ldg(len + l);
                a1 += ll / (double)__ldg(speed + (size_t)i1 * L + l);
                a2 += ll / (double)__ldg(speed + (size_t)i2 * L + l);
            }
        }
    }
}

// ---- CSR output (the paper stores rho and B sparse: "coordinate format sparse representation", Table 2
// "Sparse") — what makes Step 1 possible for large networks, whose dense slab would be terabytes.
// Thread (s, n) walks its OD's paths exactly as the dense kernels do and emits one (key, value) tuple per share, key =
// ((s*(H+1) + h)*L + l)*N + n, i.e. the boundary CSR order [s][h][l][n] of include/dode.h.  Pass 1 (out == nullptr) only
// counts the tuples of each thread; after an exclusive scan pass 2 writes them at the thread's offset.  The host then
// sorts by key, adds up tuples with equal keys (several paths of one OD over one link) and derives the row pointers.
template <typename Emit>
__device__ __forceinline__ void walk_paths(int s, int n, int L, int T, int H, const int32_t* __restrict__ od_ptr,
                                           const int32_t* __restrict__ path_ptr, const int32_t* __restrict__ path_links,
                                           const float* __restrict__ len, const float* __restrict__ speed, double dt,
                                           double theta, Emit emit) {
    const int k0 = od_ptr ? __ldg(od_ptr + n) : n, k1 = od_ptr ? __ldg(od_ptr + n + 1) : n + 1;
    const double t0 = (double)s * dt;
    double cmin = 1e300, z = 1.0;
    if (k1 - k0 > 1) {                             // Logit shares (Eq. 37); one path: p = 1
        z = 0.0;
        for (int k = k0; k < k1; ++k) cmin = fmin(cmin, path_travel_time(k, t0, L, T, dt, path_ptr, path_links, len, speed));
        for (int k = k0; k < k1; ++k) z += exp(-theta * (path_travel_time(k, t0, L, T, dt, path_ptr, path_links, len, speed) - cmin));
    }
    for (int k = k0; k < k1; ++k) {
        const double share = k1 - k0 > 1 ? exp(-theta * (path_travel_time(k, t0, L, T, dt, path_ptr, path_links, len, speed) - cmin)) / z : 1.0;
        double a1 = t0, a2 = (double)(s + 1) * dt;
        const int j1 = __ldg(path_ptr + k + 1);
        for (int j = __ldg(path_ptr + k); j < j1; ++j) {
            const int l = __ldg(path_links + j);
            const int h_first = (int)floor(a1 / dt);
            if (a2 > a1) {
                const int h_last = (int)floor(a2 / dt);
                const double inv = share / (a2 - a1);
                for (int h2 = h_first; h2 <= h_last; ++h2) {
                    const double lo = fmax(a1, (double)h2 * dt), hi = fmin(a2, (double)(h2 + 1) * dt);
                    const int h = h2 - s;
                    if (hi > lo && h <= H && h2 < T) emit(h, l, (float)((hi - lo) * inv));
                }
            } else if (h_first - s <= H && h_first < T) {
                emit(h_first - s, l, (float)share);                       // FIFO violated: all in one interval
            }
            const int i1 = min(T - 1, h_first), i2 = min(T - 1, (int)floor(a2 / dt));
            const double ll = (double)__ldg(len + l);
            a1 += ll / (double)__ldg(speed + (size_t)i1 * L + l);
            a2 += ll / (double)__ldg(speed + (size_t)i2 * L + l);
        }
    }
}

// pass 1: cnt[i] = tuples of thread i = (s, n);  pass 2 (keys != nullptr): writes them from offs[i] on
__global__ void __launch_bounds__(64)
assignment_tuples(int N, int L, int T, int H, const int32_t* __restrict__ od_ptr, const int32_t* __restrict__ path_ptr,
                  const int32_t* __restrict__ path_links, const float* __restrict__ len, const float* __restrict__ speed,
                  double dt, double theta, int32_t* __restrict__ cnt, const int64_t* __restrict__ offs,
                  unsigned long long* __restrict__ keys, float* __restrict__ vals) {
    const long total = (long)T * N;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int s = (int)(i / N), n = (int)(i - (long)s * N);
        if (keys == nullptr) {
            int c = 0;
            walk_paths(s, n, L, T, H, od_ptr, path_ptr, path_links, len, speed, dt, theta, [&](int, int, float) { ++c; });
            cnt[i] = c;
        } else {
            int64_t o = offs[i];
            walk_paths(s, n, L, T, H, od_ptr, path_ptr, path_links, len, speed, dt, theta, [&](int h, int l, float v) {
                keys[o] = (((unsigned long long)s * (H + 1) + h) * L + l) * N + n;
                vals[o] = v;
                ++o;
            });
        }
    }
}

// row_ptr[b][l] (relative to the block's first entry) and blk_off[b] from the sorted unique keys: one thread per (b, l)
// boundary, lower bound of key (b*L + l)*N.  rows = blocks * L.
__global__ void csr_bounds_from_keys(const unsigned long long* __restrict__ ukey, int64_t nu, long blocks, int L, int N,
                                     int64_t* __restrict__ blk_off, int32_t* __restrict__ row_ptr) {
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;          // over blocks * (L + 1)
    if (i >= blocks * (L + 1)) return;
    const long b = i / (L + 1);
    const int l = (int)(i - b * (L + 1));
    auto lower = [&](unsigned long long target) {
        int64_t lo = 0, hi = nu;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (ukey[mid] < target) lo = mid + 1; else hi = mid;
        }
        return lo;
    };
    const int64_t first = lower((unsigned long long)b * L * N);
    const int64_t here = l == 0 ? first : lower(((unsigned long long)b * L + l) * N);
    row_ptr[i] = (int32_t)(here - first);
    if (l == 0) blk_off[b] = first;
    if (i == 0) blk_off[blocks] = nu;
}

__global__ void csr_cols_from_keys(const unsigned long long* __restrict__ ukey, int64_t nu, int N, int32_t* __restrict__ col) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < nu; i += (int64_t)gridDim.x * blockDim.x)
        col[i] = (int32_t)(ukey[i] % (unsigned long long)N);
}

}  // namespace dode
