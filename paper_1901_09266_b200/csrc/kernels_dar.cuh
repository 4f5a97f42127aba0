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

}  // namespace dode
