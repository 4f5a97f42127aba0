// CTA-pair form of the tensor-core pass (kernels_tc.cuh) for minibatches wider than 64 days: two CTAs of a cluster, on the
// two SMs of one TPC, run ONE tcgen05.mma.cta_group::2 per instruction slot on a 256-output tile (two vertically
// adjacent 128-output tiles of the same time index and day group).
//
// Why: at bn = 128 the single-CTA kernel is bound by shared-memory bandwidth, not by the tensor pipe: per
// 16 KB chunk of A it moves 48 KB in by TMA (A, fp32 B, two bf16 B planes), 16 KB out to the splitters and 32 KB out to
// the MMAs' B operand = 96 KB ~ 768 cycles at 128 B/cycle against 512 tensor cycles.  In a pair each CTA stages only HALF
// of the B tile (bn/2 days) and the instruction reads the two halves from the two SMs: 32 KB in, 16 KB to the splitters,
// 16 KB to the MMAs = 64 KB ~ 512 cycles per chunk, the tensor time; the L2 -> SM traffic of the panels halves as well.
//
// Arithmetic is that of kernels_tc.cuh, instruction for instruction per output row (3xTF32 with bf16 correction
// products in their own accumulator, drains every kFlushChunks chunks): each CTA's 128 accumulator rows receive the
// same sequence of additions as in the single-CTA kernel.
//
// Protocol (rank 0 = leader, the only CTA that issues MMAs; "mc" = tcgen05.commit multicast to both CTAs):
//   fullA[2][SA]  local    TMA landed an A tile                       waited by the local splitter group
//   fullB[SB]     leader   both CTAs' B halves landed (2 arrivals with expect_tx, cta_group::2 TMA from the peer)
//   split[nring]  leader   both CTAs' splitters stored A_hi / bf16 planes into their TMEM (8 warp arrivals)
//   emptyB[SB]    mc       MMAs of the chunk in this B stage retired   waited by both TMA producers
//   a_empty[nring] mc      MMAs that read this TMEM A buffer retired   waited by both CTAs' splitters
//   accum         mc       all MMAs so far retired (drains and the end)
//   drained       leader   both CTAs' threads have read the accumulators of a drain (16 warp arrivals)
#pragma once
#include "kernels_tc.cuh"

namespace dode {
namespace tc {

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// address of the same shared-memory location in CTA `rank` of the cluster (shared::cluster window)
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank) {
    uint32_t d;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(d) : "r"(saddr), "r"(rank));
    return d;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n"
                 "barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// Arrivals on a barrier of the pair's leader carry no generic-proxy data: what they order is tensor-memory traffic
// (tcgen05.st / tcgen05.ld, completed by tcgen05.wait and fenced by tcgen05.fence) and TMA bytes, so the default
// (.release.cta) form is enough.  The cluster-scope release / acquire forms were measured: 92 ms instead of 56 ms per
// large_dense b = 256 epoch — every arrival then pays a cluster-wide fence on the critical handshake loop.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t caddr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(caddr) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_cluster(uint32_t caddr, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cluster.b64 _, [%0], %1;" ::"r"(caddr), "r"(bytes) : "memory");
}
// wait on a barrier that the other CTA of the pair (or a multicast tcgen05.commit) arrives on
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity, int tag = 0, int aux = 0) {
    uint32_t done;
#ifdef DODE_BRINGUP
    long spins = 0;
#endif
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.b32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
#ifdef DODE_BRINGUP
        if (!done && ((++spins & 0xffff) == 0)) {
            const bool aborted = *(volatile int*)&g_wait_abort != 0;
            if (aborted || spins > (1L << 24)) {
                if (!aborted && atomicAdd(&g_wait_abort, 1) == 0) {
                    g_wait_rec[60] = blockIdx.x; g_wait_rec[61] = blockIdx.y; g_wait_rec[62] = blockIdx.z;
                    __threadfence();
                }
                __threadfence();
                if ((threadIdx.x & 31) == 0 && (int)(blockIdx.x >> 1) == (*(volatile int*)&g_wait_rec[60] >> 1) &&
                    (int)blockIdx.y == *(volatile int*)&g_wait_rec[61]) {
                    const int k = atomicAdd(&g_wait_rec[59], 1);
                    if (k < 14) { int* r = g_wait_rec + 4 * k; r[0] = tag + 100 * (blockIdx.x & 1); r[1] = aux; r[2] = threadIdx.x >> 5; r[3] = (int)parity; }
                }
                return;
            }
        }
#else
        (void)tag; (void)aux;
#endif
    } while (!done);
}
// TMA load into THIS CTA's shared memory whose bytes are counted on a barrier of the pair's leader
__device__ __forceinline__ void tma_load_2d_pair(void* dst, const CUtensorMap* map, uint32_t bar_caddr, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(bar_caddr), "r"(c0), "r"(c1) : "memory");
}
// arrives on the barrier at this offset in BOTH CTAs once every MMA issued so far has retired
__device__ __forceinline__ void umma_commit_pair(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void umma_tf32_ts_pair(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::tf32 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_bf16_ts_pair(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// instruction descriptors of the pair: M = 256 (128 rows in each CTA), N = bn
__host__ __device__ constexpr uint32_t umma_idesc_tf32_pair(int bn) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}
__host__ __device__ constexpr uint32_t umma_idesc_bf16_pair(int bn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}

constexpr int kPairPart = 64;      // fp32 partial sums per splitter thread: bn / 2 <= 64 day columns

// grid.x = 2 (rank) x dsplit x pairs of output tiles; cluster (2, 1, 1).  p.bn is a multiple of 32, 64 < bn <= 128;
// p.ksplit == 1.  mapBf / mapBl have boxes of bn / 2 days.
template <bool ADA>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreadsTC, 1)
banded_gemm_3xtf32_pair(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapA64,
                        const __grid_constant__ CUtensorMap mapBf, const __grid_constant__ CUtensorMap mapBl,
                        const __grid_constant__ TcParams p, const __grid_constant__ DayList dl) {
    extern __shared__ __align__(1024) uint8_t smem[];
    if ((smem_u32(smem) & 1023u) != 0u) __trap();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = (int)cluster_ctarank();                      // == blockIdx.x & 1
    const bool leader = rank == 0;
    const int tt = blockIdx.y;
    const int pairIdx = ((int)blockIdx.x >> 1) / p.dsplit;
    const int m0 = (p.mtile0 + 2 * pairIdx + rank) * kTileM;
    const int d0 = (((int)blockIdx.x >> 1) % p.dsplit) * p.bn;  // first day (position in the list) of the pair's group
    const int bh = p.bn >> 1;                                     // days whose B rows THIS CTA stages
    const int dh = d0 + rank * bh;
    const int bBytes = bh * kTileK * 4;                           // this CTA's half of the fp32 B tile
    const int SA = p.stages, SB = p.bstages;
    const int bStage = 2 * bBytes;                                // B_full | bf16(B) | bf16(B_lo), bh days each
    uint8_t* ringB = smem + (size_t)SA * kABytes;
    const int nring = p.nring;
    const bool dummy = m0 >= p.M;                                 // second CTA of an odd last pair: stages B only
    const bool half = p.M - m0 <= 64;
    const int BM = half ? kTileM / 2 : kTileM;
    const int aBytes = BM * kTileK * 4;
    const CUtensorMap* mA = half ? &mapA64 : &mapA;
    uint64_t* bars = reinterpret_cast<uint64_t*>(ringB + (size_t)SB * bStage);
    uint64_t* fullA = bars;                       // [2][SA]
    uint64_t* fullB = bars + 2 * SA;              // [SB]   (the leader's copy is used)
    uint64_t* emptyB = fullB + SB;                // [SB]
    uint64_t* split = emptyB + SB;                // [4]    (leader's)
    uint64_t* a_empty = split + 4;                // [4]
    uint64_t* accum = a_empty + 4;
    uint64_t* drained = accum + 1;                // (leader's)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(drained + 1);

    const int lags = (p.mode == 0 ? min(p.H, tt) : min(p.H, p.T - 1 - tt)) + 1;
    const int nk = (lags * p.kunit + kTileK - 1) / kTileK;
    const int w0 = p.mode == 0 ? (tt - lags + 1) * p.kunit : tt * p.kunit;    // first element of the B window

    const int acc_cols = 2 * p.bn;
    uint32_t tmem_cols = 32;
    while ((int)tmem_cols < acc_cols + 64 * nring) tmem_cols <<= 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < 2 * SA; ++s) mbar_init(&fullA[s], 1);
        for (int s = 0; s < SB; ++s) { mbar_init(&fullB[s], 2); mbar_init(&emptyB[s], 1); }
        for (int j = 0; j < nring; ++j) { mbar_init(&split[j], 8); mbar_init(&a_empty[j], 1); }
        mbar_init(accum, 1);
        mbar_init(drained, 16);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(mA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapBf) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapBl) : "memory");
    }
    cluster_sync_all();                           // both CTAs' barriers exist before anything arrives on them remotely
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = *tmem_slot;
    const uint32_t tmem_ring = tmem_d + (uint32_t)acc_cols;
    const int per_group = nring >> 1;
    if (SB != 4 || nring != 4) __trap();          // the MMA issue loop below is unrolled for this geometry
    // the leader's copies of the barriers the peer arrives on
    const uint32_t fullB_l = mapa_u32(smem_u32(fullB), 0), split_l = mapa_u32(smem_u32(split), 0);
    const uint32_t drained_l = mapa_u32(smem_u32(drained), 0);

    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // the operator is static: the first ring round of A is requested before the dependency wait (kernels_tc.cuh)
    const int npre = dummy ? 0 : min(SA, nk);
    if (warp == 0) {
        if (elect_one()) {
            for (int kc = 0; kc < npre; ++kc) {
                uint64_t* fb = &fullA[(kc & 1) * SA + kc];
                mbar_expect_tx(fb, aBytes);
                tma_load_3d(smem + (size_t)kc * kABytes, mA, fb, m0, kc * kTileK, p.slab0 + tt);
            }
        }
        __syncwarp();
    }
    float pre[16];
    const int erow = ((warp & 3) << 5) + lane, em = m0 + erow;
    const int egroup = warp >= 2 ? (warp - 2) >> 2 : 0;
    const int emc = max(0, min(em, p.M - 1));
    const float* ebase = p.mode == 0 ? p.x + ((size_t)tt * p.M + emc) : p.q + ((size_t)tt * p.Np + emc);
    const size_t estride = p.mode == 0 ? (size_t)p.T * p.M : p.dayStride;
    auto prefetch = [&](int c0) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int d = min(d0 + c0 + j, dl.n - 1);
            pre[j] = __ldcg(ebase + (size_t)dl.day[d] * estride);
        }
    };
    uint32_t keep = 0xffffu;
    auto prefetch_mask = [&](int c0) {
        keep = 0;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int d = d0 + c0 + j;
            if (em < p.M && d < dl.n && __ldg(p.mask + ((size_t)d * p.T + tt) * p.M + em) != 0) keep |= 1u << j;
        }
    };
    if (p.mode == 0 && warp >= 2) prefetch(16 * egroup);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (ADA && p.mode == 0 && p.mask != nullptr && warp >= 2) prefetch_mask(16 * egroup);
    if (p.mode == 1 && warp >= 2) prefetch(16 * egroup);

    if (warp == 0) {
        // ===== TMA producer (both CTAs): own A tile, own half of the B tiles =====
        int sb = 0, ph = 1;
        int sa = 0;
        for (int kc = 0; kc < nk; ++kc) {
            if (kc >= SB) mbar_wait_cluster(&emptyB[sb], ph, 1, kc);     // chunk kc - SB retired (arrival from the leader's commit)
            if (elect_one()) {
                const int ka = kc - SB + SA;
                if (!dummy && kc >= SB && ka < nk) {
                    int sk = sa - SB; if (sk < 0) sk += SA;
                    uint64_t* fa = &fullA[(ka & 1) * SA + sk];
                    mbar_expect_tx(fa, aBytes);
                    tma_load_3d(smem + (size_t)sk * kABytes, mA, fa, m0, ka * kTileK, p.slab0 + tt);
                }
                uint8_t* st = ringB + (size_t)sb * bStage;
                const uint32_t fb = fullB_l + (uint32_t)sb * 8u;
                mbar_expect_tx_cluster(fb, (uint32_t)bStage);
                tma_load_2d_pair(st, &mapBf, fb, w0 + kc * kTileK, dh);
                tma_load_2d_pair(st + bBytes, &mapBl, fb, w0 + kc * kTileK, dh);                        // bf16(B)
                tma_load_2d_pair(st + bBytes + bBytes / 2, &mapBl, fb, w0 + kc * kTileK, p.pcap + dh);  // bf16(B_lo)
            }
            __syncwarp();
            if (++sb == SB) { sb = 0; ph ^= 1; }
            if (++sa == SA) sa = 0;
        }
    } else if (warp == 1) {
        if (leader) {
            // ===== MMA issuer (leader only) =====
            const uint32_t idesc1 = umma_idesc_tf32_pair(p.bn), idesc16 = umma_idesc_bf16_pair(p.bn);
            // Shared-memory descriptors: the high words are constants of the layout, the low word is the tile address in
            // 16-byte units (+ the LBO bit), so a K slice or a ring stage is ONE 32-bit add away from the ring's base.
            // (Building every descriptor from its byte address cost ~90 uniform-datapath instructions per chunk, and
            // the issuing warp — not the tensor pipe — set the pace: 930 cycles per chunk against 512 of tensor work.)
            constexpr uint32_t hi128 = (uint32_t)(umma_desc_k_sw128_c(0) >> 32), hi64 = (uint32_t)(umma_desc_k_sw64_c(0) >> 32);
            const uint32_t ring16 = (((smem_u32(ringB) & 0x3FFFFu) >> 4) | (1u << 16));
            const uint32_t st16 = (uint32_t)bStage >> 4, bB16 = (uint32_t)bBytes >> 4;
            // The ring geometry of the pair kernel is fixed (4 B stages, 4 TMEM A buffers), so chunk kc uses B stage kc % 4
            // and TMEM buffer ((kc & 1) << 1) | ((kc >> 1) & 1), both static after unrolling by 4, and all barriers
            // of a group of 4 chunks are in the same phase.
            for (int kc0 = 0; kc0 < nk; kc0 += 4) {
                const uint32_t par = ((uint32_t)kc0 >> 2) & 1u;
                const bool restart = (kc0 & (kFlushChunks - 1)) == 0;   // first chunk of a segment: the accumulators start over
                if (restart && kc0 > 0) {                               // drain: the splitter threads read the sums so far
                    if (elect_one()) umma_commit_pair(accum);
                    __syncwarp();
                    mbar_wait_cluster(drained, (kc0 / kFlushChunks - 1) & 1, 2, kc0);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int kc = kc0 + j;
                    if (kc >= nk) break;                                // warp-uniform
                    const int jr = ((j & 1) << 1) | (j >> 1);
                    mbar_wait_cluster(&fullB[j], par, 3, kc);
                    mbar_wait_cluster(&split[jr], par, 4, kc);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t f16 = ring16 + (uint32_t)j * st16;   // fp32 B | bf16(B) | bf16(B_lo)
                    const uint32_t h16 = f16 + bB16, l16 = h16 + (bB16 >> 1);
                    const uint32_t afull = tmem_ring + (uint32_t)jr * 64, a16 = afull + 32, alo16 = afull + 48;
                    if (elect_one()) {
#pragma unroll
                        for (int k = 0; k < kTileK / 8; ++k)
                            umma_tf32_ts_pair(tmem_d, afull + k * 8, desc_pack(f16 + 2 * k, hi128), idesc1, !(restart && j == 0 && k == 0));
#pragma unroll
                        for (int k = 0; k < kTileK / 16; ++k) {
                            umma_bf16_ts_pair(tmem_d + (uint32_t)p.bn, alo16 + k * 8, desc_pack(h16 + 2 * k, hi64), idesc16, !(restart && j == 0 && k == 0));
                            umma_bf16_ts_pair(tmem_d + (uint32_t)p.bn, a16 + k * 8, desc_pack(l16 + 2 * k, hi64), idesc16, 1);
                        }
                        umma_commit_pair(&emptyB[j]);
                        umma_commit_pair(&a_empty[jr]);
                    }
                    __syncwarp();
                }
            }
            if (elect_one()) {
                if (nk == 0) { mbar_arrive(accum); mbar_arrive_cluster(mapa_u32(smem_u32(accum), 1)); }
                else umma_commit_pair(accum);
            }
            __syncwarp();
        }
    } else {
        // ===== splitters (both CTAs): smem column -> registers -> own TMEM; group g takes chunks kc = g, g+2, ... =====
        const int group = (warp - 2) >> 2;
        const int lane_base = (warp & 3) * 32;
        const int row = lane_base + lane;
        const uint32_t tacc = tmem_d + ((uint32_t)lane_base << 16);
        float part[kPairPart];
#pragma unroll
        for (int j = 0; j < kPairPart; ++j) part[j] = 0.f;
        int s = -1;
        uint32_t fph = 0u;
        for (int kc = 0; kc < nk; ++kc) {
            if (kc > 0 && kc % kFlushChunks == 0) {
                mbar_wait_cluster(accum, (kc / kFlushChunks - 1) & 1, 5, kc);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                __syncwarp();
#pragma unroll
                for (int i = 0; i < kPairPart / 16; ++i) {
                    const int c0 = 16 * group + 32 * i;
                    if (c0 < p.bn) {
                        uint32_t v[16], w[16];
                        tmem_ld16x2_wait(tacc + (uint32_t)c0, tacc + (uint32_t)(c0 + p.bn), v, w);
#pragma unroll
                        for (int j = 0; j < 16; ++j) part[i * 16 + j] += __uint_as_float(v[j]) + __uint_as_float(w[j]);
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(drained_l);
            }
            if (++s == SA) s = 0;
            if ((kc & 1) != group) continue;
            const int use = kc >> 1;
            const int jr = group * per_group + (use & (per_group - 1));     // per_group is 1 or 2
            const bool work = !dummy && lane_base < BM;              // rows that are stored at the end
            if (!dummy) {
                mbar_wait(&fullA[group * SA + s], (fph >> s) & 1u, 6, kc);
                fph ^= 1u << s;
            }
            if (use >= per_group) mbar_wait_cluster(&a_empty[jr], ((use >> (per_group >> 1)) - 1) & 1, 7, kc);
            if (work) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const float* A = reinterpret_cast<const float*>(smem + (size_t)s * kABytes) + row;
                const uint32_t t0 = tmem_ring + (uint32_t)jr * 64 + ((uint32_t)lane_base << 16);
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    uint32_t hi[16], h16[8], l16[8];
#pragma unroll
                    for (int k = 0; k < 16; ++k) hi[k] = __float_as_uint(A[(hf * 16 + k) * BM]);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float a0 = __uint_as_float(hi[2 * i]), a1 = __uint_as_float(hi[2 * i + 1]);
                        h16[i] = pack_bf16(a0, a1);
                        l16[i] = pack_bf16(tf32_lo(a0), tf32_lo(a1));
                    }
                    __syncwarp();
                    tmem_st16(t0 + hf * 16, hi);
                    tmem_st8(t0 + 32 + hf * 8, h16);
                    tmem_st8(t0 + 48 + hf * 8, l16);
                }
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(split_l + (uint32_t)jr * 8u);
        }
        // ---- epilogue: every CTA stores its own 128 output rows ----
        mbar_wait_cluster(accum, (nk > 0 ? (nk - 1) / kFlushChunks : 0) & 1, 8, nk);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int m = m0 + row;
#pragma unroll
        for (int i = 0; i < kPairPart / 16; ++i) {
            const int c0 = 16 * group + 32 * i;
            if (c0 >= p.bn) break;
            uint32_t v[16], w[16];
            float cur[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) cur[j] = pre[j];
            const uint32_t curkeep = keep;
            if (c0 + 32 < p.bn) {
                prefetch(c0 + 32);
                if (ADA && p.mode == 0 && p.mask != nullptr) prefetch_mask(c0 + 32);
            }
            __syncwarp();
            tmem_ld16x2_wait(tacc + (uint32_t)c0, tacc + (uint32_t)(c0 + p.bn), v, w);
            if (m < p.M) {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int d = d0 + c0 + j;
                    if (d < dl.n) {
                        const float acc = nk ? part[i * 16 + j] + (__uint_as_float(v[j]) + __uint_as_float(w[j])) : 0.f;
                        if (p.mode == 0) {
                            const float r = (!ADA || ((curkeep >> j) & 1u)) ? acc - cur[j] : 0.f;
                            p.rp_full[(size_t)d * p.rpitch + (size_t)tt * p.Lp + m] = r;
                            p.rp_lo[(size_t)d * p.rpitch + (size_t)tt * p.Lp + m] = __float2bfloat16_rn(r);
                            p.rp_lo[(size_t)(p.pcap + d) * p.rpitch + (size_t)tt * p.Lp + m] = __float2bfloat16_rn(tf32_lo(r));
                        } else {
                            const size_t qi = (size_t)dl.day[d] * p.dayStride + (size_t)tt * p.Np + m;
                            if (ADA && p.G != nullptr) p.q[qi] = adagrad_update(cur[j], acc, p.G + qi, p.eta, p.eps);
                            else p.q[qi] = fmaxf(0.f, fmaf(-p.eta, acc, cur[j]));
                        }
                    }
                }
            }
        }
        __syncwarp();
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    // neither CTA may leave while the other can still reach its shared memory (multicast arrivals, the peer half of B)
    cluster_sync_all();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"(tmem_cols) : "memory");
    }
}

}  // namespace tc
}  // namespace dode
