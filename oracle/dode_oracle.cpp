// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded C++ loops for the SPGD/NNLS hot path of
// Ma & Qian (arXiv 1901.09266), written from the paper under the
// readings of SURVEY.md §8(c) / DESIGN.md.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load this file.  It
// shares no code, header, table or helper with the CUDA path
// (paper_1901_09266_b200/csrc) and neither side includes the other.
//
// What is computed (per day d of cluster c, all sums in double, storage fp32):
//   O2a  r[t][l] = sum_{h=0..min(H,t)} sum_n R[c][t-h][h][l][n] q[t-h][n] - x[t][l]
//        -- "B_o x - y", PAPER.md:406 (Alg. 1 line 9); Eq. 40/42;
//           entry layout of Table 2: q entry (h1-1)|K|+k,
//           x entry (h2-1)|A|+a, rho entry [(h2-1)|A|+a, (h1-1)Pi+k];
//           block (h2,h1) with lag h = h2-h1 >= 0 (FIFO);
//           cross-midnight flow dropped: no s+h >= T term.
//   O2b  g[s][n] = sum_{h=0..min(H,T-1-s)} sum_l R[c][s][h][l][n] r[s+h][l]
//        -- "g = B_o^T (B_o x - y)".  No factor 2 (reading A1).
//   O2c  q[s][n] = max(0, q[s][n] - eta g[s][n])
//        -- "x = max(x,0)"; plain step instead of Adagrad (reading A3,
//           BASELINE.json north_star).  r is complete before any q changes.
//   O3   f = sum_t sum_l r[t][l]^2, no 1/2, no mean -- Eq. 42.
//   O5   R2_d = 1 - sum r^2 / sum (x - mean x)^2 -- Step 6 quality check (reading A17).
//   O4   L_c = lambda_max(rho_c^T rho_c) by power iteration from the all-ones
//        vector (reading A10; PAPER.md:416 only says the rate depends on scale).
//
// Pins (tests/test_oracle_pins.py): P1 active-set NNLS on the T=12 instance,
// P2 KKT, P3 finite differences, P4 planted recovery, P5 closed-form linear
// iteration, P6 Example 1, P8 adjoint, P9 descent,
// P10 separability, P12 dense assembly by Table 2, P13 dense-vs-CSR, P14 R2 closed forms,
// P15 row-chunk Adagrad against torch.optim.Adagrad on the assembled matrix, P16 DAR construction (O7): the paper's
// Example 3 worked by hand, the constant-speed closed form, unit row sums, vehicle conservation through O2a,
// P10b run_schedule with several clusters and a different step per iteration against per-day visit replays,
// P18 the multi-visit day replays (oracle_replay_day / _csr: the same loops with the OUTPUT rows of a pass handed to
// several threads, every output element accumulated in the same order) bit for bit against repeated oracle_visit.
// No function here is "parity unpinned".
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <chrono>
#include <cstring>
#include <functional>
#include <thread>
#include <vector>

namespace {

struct Dims { int N, L, T, H; };

inline size_t blk(const Dims& d, int s, int h) {            // offset of R_c[s][h] (L x N, n fastest)
    return ((size_t)s * (d.H + 1) + h) * (size_t)d.L * d.N;
}

// O2a in double (no rounding of r) for the output rows t0 <= t < t1; x may be null (then r = rho q).
void forward_rows(const Dims& d, const float* Rc, const float* q, const float* x, double* r, int t0, int t1) {
    for (int t = t0; t < t1; ++t)
        for (int l = 0; l < d.L; ++l) {
            double acc = 0.0;
            const int hmax = d.H < t ? d.H : t;
            for (int h = 0; h <= hmax; ++h) {
                const float* row = Rc + blk(d, t - h, h) + (size_t)l * d.N;
                const float* qs = q + (size_t)(t - h) * d.N;
                for (int n = 0; n < d.N; ++n) acc += (double)row[n] * (double)qs[n];
            }
            r[(size_t)t * d.L + l] = acc - (x ? (double)x[(size_t)t * d.L + l] : 0.0);
        }
}

void forward_d(const Dims& d, const float* Rc, const float* q, const float* x, double* r) {
    forward_rows(d, Rc, q, x, r, 0, d.T);
}

// O2b: g = rho^T r, r given in fp32 storage, for the output rows s0 <= s < s1.
void gradient_rows(const Dims& d, const float* Rc, const float* r, double* g, int s0, int s1) {
    for (int s = s0; s < s1; ++s)
        for (int n = 0; n < d.N; ++n) {
            double acc = 0.0;
            const int hmax = d.H < d.T - 1 - s ? d.H : d.T - 1 - s;
            for (int h = 0; h <= hmax; ++h) {
                const float* B = Rc + blk(d, s, h);
                const float* rt = r + (size_t)(s + h) * d.L;
                for (int l = 0; l < d.L; ++l) acc += (double)B[(size_t)l * d.N + n] * (double)rt[l];
            }
            g[(size_t)s * d.N + n] = acc;
        }
}

void gradient_f(const Dims& d, const float* Rc, const float* r, double* g) {
    gradient_rows(d, Rc, r, g, 0, d.T);
}

// fn(i0, i1) over a partition of [0, n) into `threads` contiguous ranges, one std::thread each (threads <= 1: inline).
// Used only to hand DIFFERENT OUTPUT ROWS of one pass to different threads: no output element is shared, and the
// order in which each element's sum is accumulated does not depend on the partition.
void parallel_rows(int n, int threads, const std::function<void(int, int)>& fn) {
    if (threads <= 1 || n <= 1) { fn(0, n); return; }
    threads = std::min(threads, n);
    std::vector<std::thread> pool;
    for (int k = 0; k < threads; ++k) {
        const int i0 = (int)((long)n * k / threads), i1 = (int)((long)n * (k + 1) / threads);
        pool.emplace_back(fn, i0, i1);
    }
    for (auto& th : pool) th.join();
}

void visit(const Dims& d, const float* Rc, float* q, const float* x, float eta,
           std::vector<double>& rd, std::vector<float>& rf, std::vector<double>& g) {
    const size_t TL = (size_t)d.T * d.L, TN = (size_t)d.T * d.N;
    rd.resize(TL); rf.resize(TL); g.resize(TN);
    forward_d(d, Rc, q, x, rd.data());
    for (size_t i = 0; i < TL; ++i) rf[i] = (float)rd[i];                 // r stored fp32 (O2a)
    gradient_f(d, Rc, rf.data(), g.data());
    for (size_t i = 0; i < TN; ++i) {                                     // O2c
        const double v = (double)q[i] - (double)eta * g[i];
        q[i] = (float)(v > 0.0 ? v : 0.0);
    }
}

}  // namespace

extern "C" {

// r[t][l] (fp32) for one day; Rc = R[c] as [T][H+1][L][N].
void oracle_forward_residual(int N, int L, int T, int H, const float* Rc, const float* q,
                             const float* x, float* r) {
    Dims d{N, L, T, H};
    std::vector<double> rd((size_t)T * L);
    forward_d(d, Rc, q, x, rd.data());
    for (size_t i = 0; i < rd.size(); ++i) r[i] = (float)rd[i];
}

// g[s][n] (double) = rho_c^T r.
void oracle_gradient(int N, int L, int T, int H, const float* Rc, const float* r, double* g) {
    Dims d{N, L, T, H};
    gradient_f(d, Rc, r, g);
}

// One SPGD visit of one day, in place on q (O2a-O2c).
void oracle_visit(int N, int L, int T, int H, const float* Rc, float* q, const float* x, float eta) {
    Dims d{N, L, T, H};
    std::vector<double> rd, g; std::vector<float> rf;
    visit(d, Rc, q, x, eta, rd, rf, g);
}

// O3: f = sum r^2 with r in double from the current q.
double oracle_objective_day(int N, int L, int T, int H, const float* Rc, const float* q, const float* x) {
    Dims d{N, L, T, H};
    std::vector<double> rd((size_t)T * L);
    forward_d(d, Rc, q, x, rd.data());
    double f = 0.0;
    for (double v : rd) f += v * v;
    return f;
}

// O3 with the rows of the forward pass split over `threads` threads; the squares are summed in index order afterwards,
// so the value equals oracle_objective_day bit for bit (pin P18).
double oracle_objective_day_mt(int N, int L, int T, int H, const float* Rc, const float* q, const float* x, int threads) {
    Dims d{N, L, T, H};
    std::vector<double> rd((size_t)T * L);
    parallel_rows(T, threads, [&](int t0, int t1) { forward_rows(d, Rc, q, x, rd.data(), t0, t1); });
    double f = 0.0;
    for (double v : rd) f += v * v;
    return f;
}

// O5 (Step 6 "quality check"; "R-square between the observed link flow and estimated link flow",
// PAPER.md:553): coefficient of determination of one day's fitted counts, observed counts as the reference
// (reading A17):  R2 = 1 - sum (x - rho q)^2 / sum (x - mean(x))^2  over the day's T*L entries, all in double.
double oracle_r2_day(int N, int L, int T, int H, const float* Rc, const float* q, const float* x) {
    Dims d{N, L, T, H};
    const size_t TL = (size_t)T * L;
    std::vector<double> rd(TL);
    forward_d(d, Rc, q, x, rd.data());
    double ss_res = 0.0, mean = 0.0, ss_tot = 0.0;
    for (double v : rd) ss_res += v * v;
    for (size_t i = 0; i < TL; ++i) mean += (double)x[i];
    mean /= (double)TL;
    for (size_t i = 0; i < TL; ++i) ss_tot += ((double)x[i] - mean) * ((double)x[i] - mean);
    return 1.0 - ss_res / ss_tot;
}

// O6 (NEXT-1): one iteration of Alg. 1 as the paper states it on one day:
//   line 8  B_o = rows `mask` of the day's system (a chunk of the permuted row range),
//   line 9  g = B_o^T (B_o x - y_o)   == rho^T (mask .* (rho q - x)),
//   line 10 x = Adagrad(x, g, eta)    -- accumulate G += g^2, step eta * g / (sqrt(G) + eps)  ([14]; the paper's
//                                        implementation is PyTorch, whose Adagrad is exactly this with eps = 1e-10;
//                                        reading A18),
//   line 11 x = max(x, 0).
// mask is [T][L] bytes (nullable = every row); G is the fp32 accumulator state [T][N], updated in place.
void oracle_visit_adagrad(int N, int L, int T, int H, const float* Rc, float* q, float* G, const float* x,
                          const uint8_t* mask, float eta, float eps) {
    Dims d{N, L, T, H};
    const size_t TL = (size_t)T * L, TN = (size_t)T * N;
    std::vector<double> rd(TL), g(TN);
    std::vector<float> rf(TL);
    forward_d(d, Rc, q, x, rd.data());
    for (size_t i = 0; i < TL; ++i) rf[i] = (mask && !mask[i]) ? 0.f : (float)rd[i];
    gradient_f(d, Rc, rf.data(), g.data());
    for (size_t i = 0; i < TN; ++i) {
        const double Gd = (double)G[i] + g[i] * g[i];
        G[i] = (float)Gd;
        const double v = (double)q[i] - (double)eta * g[i] / (std::sqrt(Gd) + (double)eps);
        q[i] = (float)(v > 0.0 ? v : 0.0);
    }
}

// Replays a schedule: iteration k visits days sched_days[sched_ptr[k] .. sched_ptr[k+1])
// with step eta[k].  R is [C][T][H+1][L][N]; labels[D]; x [D][T][L]; q [D][T][N] in place.
// day_mask (nullable, [D]): days with mask 0 are skipped -- valid because days
// are independent units (pin P10).
void oracle_run_schedule(int N, int L, int T, int H, int C, int D, const float* R,
                         const int32_t* labels, const float* x, float* q,
                         const int32_t* sched_days, const int64_t* sched_ptr, const float* sched_eta,
                         int K, const uint8_t* day_mask) {
    (void)C;
    Dims d{N, L, T, H};
    const size_t Rc_sz = (size_t)T * (H + 1) * L * N, TL = (size_t)T * L, TN = (size_t)T * N;
    std::vector<double> rd, g; std::vector<float> rf;
    for (int k = 0; k < K; ++k)
        for (int64_t i = sched_ptr[k]; i < sched_ptr[k + 1]; ++i) {
            const int day = sched_days[i];
            if (day < 0 || day >= D) continue;
            if (day_mask && !day_mask[day]) continue;
            visit(d, R + Rc_sz * labels[day], q + TN * day, x + TL * day, sched_eta[k], rd, rf, g);
        }
}

// O4: Rayleigh quotient of rho_c^T rho_c after `iters` power iterations from all-ones, in double.
double oracle_power_iteration(int N, int L, int T, int H, const float* Rc, int iters) {
    Dims d{N, L, T, H};
    const size_t TL = (size_t)T * L, TN = (size_t)T * N;
    std::vector<double> u(TN, 1.0), v(TL), w(TN);
    double lam = 0.0;
    for (int it = 0; it < iters; ++it) {
        double nu = 0.0;
        for (double a : u) nu += a * a;
        nu = std::sqrt(nu);
        for (double& a : u) a /= nu;
        // v = rho u
        for (int t = 0; t < T; ++t)
            for (int l = 0; l < L; ++l) {
                double acc = 0.0;
                const int hmax = H < t ? H : t;
                for (int h = 0; h <= hmax; ++h) {
                    const float* row = Rc + blk(d, t - h, h) + (size_t)l * N;
                    const double* us = u.data() + (size_t)(t - h) * N;
                    for (int n = 0; n < N; ++n) acc += (double)row[n] * us[n];
                }
                v[(size_t)t * L + l] = acc;
            }
        lam = 0.0;
        for (double a : v) lam += a * a;          // u^T rho^T rho u with |u| = 1
        // w = rho^T v
        for (int s = 0; s < T; ++s)
            for (int n = 0; n < N; ++n) {
                double acc = 0.0;
                const int hmax = H < T - 1 - s ? H : T - 1 - s;
                for (int h = 0; h <= hmax; ++h) {
                    const float* B = Rc + blk(d, s, h);
                    const double* vt = v.data() + (size_t)(s + h) * L;
                    for (int l = 0; l < L; ++l) acc += (double)B[(size_t)l * N + n] * vt[l];
                }
                w[(size_t)s * N + n] = acc;
            }
        u = w;
    }
    return lam;
}

// ---- a6: the same O2a-O2c with R_c given as CSR per (s,h) block ("coordinate format
// sparse representation"; Table 2 "Sparse").
// blk_off[(s*(H+1)+h)] = first nnz of block (s,h) (int64, T*(H+1)+1 entries, for this cluster);
// row_ptr[(s*(H+1)+h)*(L+1) + l] = offset of row l relative to the block start; col = OD index n.
static void csr_forward_rows(int N, int L, int T, int H, const int64_t* blk_off, const int32_t* row_ptr,
                             const int32_t* col_idx, const float* val, const float* q, const float* x, float* rf,
                             int t0, int t1) {
    (void)T;
    for (int t = t0; t < t1; ++t)
        for (int l = 0; l < L; ++l) {
            double acc = 0.0;
            const int hmax = H < t ? H : t;
            for (int h = 0; h <= hmax; ++h) {
                const size_t b = (size_t)(t - h) * (H + 1) + h;
                const int32_t* rp = row_ptr + b * (L + 1);
                for (int64_t k = blk_off[b] + rp[l]; k < blk_off[b] + rp[l + 1]; ++k)
                    acc += (double)val[k] * (double)q[(size_t)(t - h) * N + col_idx[k]];
            }
            rf[(size_t)t * L + l] = (float)(acc - (double)x[(size_t)t * L + l]);
        }
}

// g rows s0 <= s < s1 (g zeroed by the caller); every entry of block (s,h) adds into row s only
static void csr_gradient_rows(int N, int L, int T, int H, const int64_t* blk_off, const int32_t* row_ptr,
                              const int32_t* col_idx, const float* val, const float* rf, double* g, int s0, int s1) {
    for (int s = s0; s < s1; ++s) {
        const int hmax = H < T - 1 - s ? H : T - 1 - s;
        for (int h = 0; h <= hmax; ++h) {
            const size_t b = (size_t)s * (H + 1) + h;
            const int32_t* rp = row_ptr + b * (L + 1);
            for (int l = 0; l < L; ++l)
                for (int64_t k = blk_off[b] + rp[l]; k < blk_off[b] + rp[l + 1]; ++k)
                    g[(size_t)s * N + col_idx[k]] += (double)val[k] * (double)rf[(size_t)(s + h) * L + l];
        }
    }
}

void oracle_visit_csr(int N, int L, int T, int H, const int64_t* blk_off, const int32_t* row_ptr,
                      const int32_t* col_idx, const float* val, float* q, const float* x, float eta) {
    const size_t TL = (size_t)T * L, TN = (size_t)T * N;
    std::vector<float> rf(TL);
    std::vector<double> g(TN, 0.0);
    csr_forward_rows(N, L, T, H, blk_off, row_ptr, col_idx, val, q, x, rf.data(), 0, T);
    csr_gradient_rows(N, L, T, H, blk_off, row_ptr, col_idx, val, rf.data(), g.data(), 0, T);
    for (size_t i = 0; i < TN; ++i) {
        const double v = (double)q[i] - (double)eta * g[i];
        q[i] = (float)(v > 0.0 ? v : 0.0);
    }
}

// Multi-visit replay of ONE day for the full-K parity tests ("the oracle replays the full K-iteration
// schedule for a seeded sample of days"; days are independent units).  `visits` consecutive visits with
// the same operator and step — O2a, O2b, O2c exactly as oracle_visit / oracle_visit_csr compute them (the same row
// functions; r complete before any q changes) — with the output rows of each pass split over `threads` threads.
// After visit number ckpt[j] (1-based, ascending) q is copied to out[j].  The replay stops early once `budget_s`
// seconds have passed (checked between visits; <= 0: no limit); the number of visits done is returned.
int oracle_replay_day(int N, int L, int T, int H, const float* Rc, float* q, const float* x, float eta, int visits,
                      const int32_t* ckpt, int nckpt, float* out, int threads, double budget_s) {
    Dims d{N, L, T, H};
    const size_t TL = (size_t)T * L, TN = (size_t)T * N;
    std::vector<double> rd(TL), g(TN);
    std::vector<float> rf(TL);
    const auto t_start = std::chrono::steady_clock::now();
    int j = 0, v = 0;
    for (; v < visits; ++v) {
        if (budget_s > 0 && v > 0 &&
            std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count() > budget_s) break;
        parallel_rows(T, threads, [&](int t0, int t1) { forward_rows(d, Rc, q, x, rd.data(), t0, t1); });
        for (size_t i = 0; i < TL; ++i) rf[i] = (float)rd[i];                 // r stored fp32 (O2a)
        parallel_rows(T, threads, [&](int s0, int s1) { gradient_rows(d, Rc, rf.data(), g.data(), s0, s1); });
        for (size_t i = 0; i < TN; ++i) {                                     // O2c
            const double w = (double)q[i] - (double)eta * g[i];
            q[i] = (float)(w > 0.0 ? w : 0.0);
        }
        while (j < nckpt && ckpt[j] == v + 1) { std::memcpy(out + (size_t)j * TN, q, TN * sizeof(float)); ++j; }
    }
    return v;
}

int oracle_replay_day_csr(int N, int L, int T, int H, const int64_t* blk_off, const int32_t* row_ptr,
                          const int32_t* col_idx, const float* val, float* q, const float* x, float eta, int visits,
                          const int32_t* ckpt, int nckpt, float* out, int threads, double budget_s) {
    const size_t TL = (size_t)T * L, TN = (size_t)T * N;
    std::vector<float> rf(TL);
    std::vector<double> g(TN);
    const auto t_start = std::chrono::steady_clock::now();
    int j = 0, v = 0;
    for (; v < visits; ++v) {
        if (budget_s > 0 && v > 0 &&
            std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count() > budget_s) break;
        std::fill(g.begin(), g.end(), 0.0);
        parallel_rows(T, threads, [&](int t0, int t1) {
            csr_forward_rows(N, L, T, H, blk_off, row_ptr, col_idx, val, q, x, rf.data(), t0, t1); });
        parallel_rows(T, threads, [&](int s0, int s1) {
            csr_gradient_rows(N, L, T, H, blk_off, row_ptr, col_idx, val, rf.data(), g.data(), s0, s1); });
        for (size_t i = 0; i < TN; ++i) {
            const double w = (double)q[i] - (double)eta * g[i];
            q[i] = (float)(w > 0.0 ? w : 0.0);
        }
        while (j < nckpt && ckpt[j] == v + 1) { std::memcpy(out + (size_t)j * TN, q, TN * sizeof(float)); ++j; }
    }
    return v;
}

double oracle_objective_day_csr(int N, int L, int T, int H, const int64_t* blk_off, const int32_t* row_ptr,
                                const int32_t* col_idx, const float* val, const float* q, const float* x) {
    double f = 0.0;
    for (int t = 0; t < T; ++t)
        for (int l = 0; l < L; ++l) {
            double acc = 0.0;
            const int hmax = H < t ? H : t;
            for (int h = 0; h <= hmax; ++h) {
                const size_t b = (size_t)(t - h) * (H + 1) + h;
                const int32_t* rp = row_ptr + b * (L + 1);
                for (int64_t k = blk_off[b] + rp[l]; k < blk_off[b] + rp[l + 1]; ++k)
                    acc += (double)val[k] * (double)q[(size_t)(t - h) * N + col_idx[k]];
            }
            const double r = acc - (double)x[(size_t)t * L + l];
            f += r * r;
        }
    return f;
}

// O7 (NEXT-4): Step 1 of the framework, the DAR matrix of one day / one pattern from link speeds (PAPER.md:187-228,
// Eq. 17-18 and Example 3; loop order of PAPER.md:377: "iterating over departure time intervals and paths ... we iterate
// over all the links in the path from origin to destination and compute the arrival time of each link").
//   path of OD n: links path_links[path_ptr[n] .. path_ptr[n+1]) in travel order (one path per OD: p = 1, Eq. 41);
//   speed[t][l]: the link's speed in interval t (length units per second), len[l] its length, dt = |H| in seconds.
//   The vehicles departing in H_s = [s dt, (s+1) dt) are bracketed by a leading (t1 = s dt) and a trailing
//   (t2 = (s+1) dt) trajectory; a trajectory crosses a link at the speed of the interval in which it ENTERS the link
//   ("the speeds of links are the slopes of the trajectory"; reading A20).  At the tail of link a the
//   flow of H_s arrives spread evenly over [a1, a2) = [tau_a(t1), tau_a(t2)) (Eq. 16), so (Eq. 18)
//       rho(s, h2) = |[a1, a2) ∩ H_h2| / (a2 - a1)           -> R[s][h2 - s][l][n]
//   Entries with h2 - s > H or h2 >= T are dropped (reading A6).  If a2 <= a1 (FIFO violated by a speed
//   jump between the two entries) the whole flow is put in the interval of a1.
// R is [T][H+1][L][N], zeroed here.  All times in double.
void oracle_dar_build(int N, int L, int T, int H, const int32_t* path_ptr, const int32_t* path_links, const float* len,
                      const float* speed, double dt, float* R) {
    const size_t total = (size_t)T * (H + 1) * L * N;
    for (size_t i = 0; i < total; ++i) R[i] = 0.f;
    for (int s = 0; s < T; ++s)
        for (int n = 0; n < N; ++n) {
            double a1 = (double)s * dt, a2 = (double)(s + 1) * dt;       // arrival of the two trajectories at the next link
            for (int j = path_ptr[n]; j < path_ptr[n + 1]; ++j) {
                const int l = path_links[j];
                // the share of H_s that reaches the tail of link l within each interval h2
                const int h_first = (int)std::floor(a1 / dt);
                if (a2 > a1) {
                    const int h_last = (int)std::floor(a2 / dt);
                    for (int h2 = h_first; h2 <= h_last; ++h2) {
                        const double lo = std::max(a1, (double)h2 * dt), hi = std::min(a2, (double)(h2 + 1) * dt);
                        if (hi <= lo) continue;
                        const int h = h2 - s;
                        if (h <= H && h2 < T) R[(((size_t)s * (H + 1) + h) * L + l) * N + n] = (float)((hi - lo) / (a2 - a1));
                    }
                } else if (h_first - s <= H && h_first < T) {
                    R[(((size_t)s * (H + 1) + (h_first - s)) * L + l) * N + n] = 1.f;
                }
                // cross the link at the speed of the interval of entry
                const int i1 = std::min(T - 1, (int)std::floor(a1 / dt)), i2 = std::min(T - 1, (int)std::floor(a2 / dt));
                a1 += (double)len[l] / (double)speed[(size_t)i1 * L + l];
                a2 += (double)len[l] / (double)speed[(size_t)i2 * L + l];
            }
        }
}

// O8 (NEXT-4, second half): the assignment matrix B = delta * rho * p of one pattern (Eq. 41) with
// several paths per OD and Logit route shares (Eq. 37):
//   paths of OD n: od_ptr[n] .. od_ptr[n+1]);  links of path k: path_links[path_ptr[k] .. path_ptr[k+1]) in travel order;
//   c_k(s) = travel time of path k for the vehicle leaving at the start of interval s (entry-interval speeds, reading
//            A20; one speed table per pattern = the pattern's mean speeds, reading A22);
//   p_k(s) = exp(-theta c_k(s)) / sum_{k' in K_n} exp(-theta c_k'(s))       (Eq. 37; constant within the interval, Eq. 38);
//   R[s][h][l][n] = sum_{k in K_n} rho_k(s, s+h; l) p_k(s)                  (Eq. 41 summed over the OD's paths, as Eq. 40 does).
// rho_k as in O7.  R is [T][H+1][L][N], zeroed here.
void oracle_assignment_build(int N, int L, int T, int H, const int32_t* od_ptr, const int32_t* path_ptr,
                             const int32_t* path_links, const float* len, const float* speed, double dt, double theta,
                             float* R) {
    const size_t total = (size_t)T * (H + 1) * L * N;
    std::vector<double> acc(total, 0.0);
    for (int s = 0; s < T; ++s)
        for (int n = 0; n < N; ++n) {
            const int k0 = od_ptr[n], k1 = od_ptr[n + 1];
            // route shares from the leading vehicle's path travel times
            std::vector<double> c(k1 - k0), pk(k1 - k0);
            double cmin = 1e300;
            for (int k = k0; k < k1; ++k) {
                double t = (double)s * dt;
                for (int j = path_ptr[k]; j < path_ptr[k + 1]; ++j) {
                    const int l = path_links[j];
                    const int i = std::min(T - 1, (int)std::floor(t / dt));
                    t += (double)len[l] / (double)speed[(size_t)i * L + l];
                }
                c[k - k0] = t - (double)s * dt;
                cmin = std::min(cmin, c[k - k0]);
            }
            double z = 0.0;
            for (int k = k0; k < k1; ++k) { pk[k - k0] = std::exp(-theta * (c[k - k0] - cmin)); z += pk[k - k0]; }
            for (int k = k0; k < k1; ++k) {
                const double share = pk[k - k0] / z;
                double a1 = (double)s * dt, a2 = (double)(s + 1) * dt;
                for (int j = path_ptr[k]; j < path_ptr[k + 1]; ++j) {
                    const int l = path_links[j];
                    const int h_first = (int)std::floor(a1 / dt);
                    if (a2 > a1) {
                        const int h_last = (int)std::floor(a2 / dt);
                        for (int h2 = h_first; h2 <= h_last; ++h2) {
                            const double lo = std::max(a1, (double)h2 * dt), hi = std::min(a2, (double)(h2 + 1) * dt);
                            if (hi <= lo) continue;
                            const int h = h2 - s;
                            if (h <= H && h2 < T) acc[(((size_t)s * (H + 1) + h) * L + l) * N + n] += share * (hi - lo) / (a2 - a1);
                        }
                    } else if (h_first - s <= H && h_first < T) {
                        acc[(((size_t)s * (H + 1) + (h_first - s)) * L + l) * N + n] += share;
                    }
                    const int i1 = std::min(T - 1, (int)std::floor(a1 / dt)), i2 = std::min(T - 1, (int)std::floor(a2 / dt));
                    a1 += (double)len[l] / (double)speed[(size_t)i1 * L + l];
                    a2 += (double)len[l] / (double)speed[(size_t)i2 * L + l];
                }
            }
        }
    for (size_t i = 0; i < total; ++i) R[i] = (float)acc[i];
}

}  // extern "C"
