// Tensor-core path of a2-a4 for minibatch b >= 8: banded block GEMMs on tcgen05 (5th-gen tensor
// cores, FP32 accumulators in TMEM) with 3xTF32 split arithmetic (bf16 correction terms), TMA-staged operands.
//
// Per output tile (time index tt, 128 outputs m0..m0+127) the pass is one GEMM
//        D[128 x BN] = sum_k A[k][m] * B[k][d]             (BN = b rounded up to 16 days)
//   forward  (a2): A = Af[tt] (K rows (j,n), outputs l contiguous),  B[k][d] = Qg[d][(tt-hmax)*Np + k]
//   gradient (a3): A = Ag[tt] (K rows (h,l), outputs n contiguous),  B[k][d] = rp[d][tt*Lp + k]
// (layouts: kernels_dense.cuh).  In both passes B is a contiguous window of a per-day vector, K-major, and A
// arrives "M-major" (the output index contiguous in HBM, so TMA moves 512-byte runs).  That is fine because
// A never feeds the tensor core from shared memory: 3xTF32 has to split A = A_hi + A_lo anyway, so splitter
// threads (thread = output row = TMEM lane) read their COLUMN of the landed tile (consecutive lanes ->
// consecutive words, conflict-free), and write A_hi / A_lo into tensor memory with tcgen05.st; tcgen05.mma
// then takes A from TMEM (TS form) and B from shared memory (K-major descriptors: SWIZZLE_128B fp32, SWIZZLE_64B bf16).
// Truncation at the day boundary falls out of zero rows packed at create time and of TMA's
// zero fill beyond the end of the per-day vector / of the K rows of a slab.
//
// 3xTF32 (north_star: "3xTF32 tensor-core emulation ... where the tolerance still holds"):
//   a = a_hi + a_lo with a_hi = a truncated to TF32 (what the tensor core reads from an fp32 container),
//   a_lo = a - a_hi (exact in fp32);   a*b ~= a_hi*b_hi + a_lo*b + a*b_lo   (a_lo*b_lo ~ 2^-22 dropped).
//   The MAIN product a_hi*b_hi runs as kind::tf32 on the fp32 data itself (K = 8 per instruction) into D[:, 0:bn].
//   The two CORRECTION products are 2^-11 of it, so their factors need only bf16 precision (rounding a 2^-11-sized
//   factor to 8 bits costs 2^-19 of the product, unbiased): they run as kind::f16 on bf16 operands (K = 16 per
//   instruction, i.e. half the tensor time of a TF32 instruction per K) into their own accumulator D[:, bn:2bn]:
//       D_corr += bf16(a_lo) * bf16(b)  +  bf16(a) * bf16(b_lo).
//   Per 32-row K chunk: 4 TF32 + 4 bf16 instructions = the tensor time of 2 TF32 products per fp32 product, not 3.
//   B operands per minibatch: one fp32 plane and two bf16 planes (bf16(v), bf16(v - tf32(v))), produced where B is
//   produced (gather kernel / forward epilogue) — the same bytes as fp32 v and v_lo.  A: the splitters store the fp32
//   values (32 TMEM columns) and the two bf16 planes packed two per column (16 + 16 columns).  bn <= 128 days per CTA;
//   wider minibatches are split into two day groups (blockIdx.x & 1).  The epilogue adds main and correction halves.
// Accumulation accuracy (measured): tcgen05 adds into its FP32 accumulator with round-toward-zero, so
//   every accumulating instruction loses ~half an ulp of the running sum, always in the same direction: a relative bias
//   of about -n * 2^-24 after n instructions on same-signed data (-1.5e-5 at K = 2048, -2e-4 at K = 13312 with every
//   MMA landing in one accumulator).  Two measures bound it independently of K: (1) the small correction products never
//   touch the main accumulator (above), (2) every kFlushChunks K chunks the accumulators are DRAINED by the splitter
//   threads into fp32 registers (round-to-nearest adds) and restarted, so that no accumulator ever takes more than
//   4 * kFlushChunks additions (bias <= ~4e-6 relative, whatever K).
// TMEM columns: [0, 2*bn) accumulators, then nring x (32 cols A fp32 | 16 cols bf16(A) | 16 cols bf16(A_lo)).
//
// Warp roles (320 threads): warp 0 = TMA producer, warp 1 = MMA issuer + TMEM owner, warps 2-5 and 6-9 = two
// groups of splitters that take alternate K chunks, then the epilogue (TMEM -> registers -> global, fused
// -x / projected update), column chunks interleaved between the groups.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels_dense.cuh"

namespace dode {
namespace tc {

constexpr int kThreadsTC = 320;
constexpr int kTileM = 128;
constexpr int kTileK = 32;                       // 32 fp32 = 128 B = one SWIZZLE_128B span
constexpr int kABytes = kTileM * kTileK * 4;     // 16 KB
constexpr int kFlushChunks = 16;                 // K chunks between two drains of the TMEM accumulators (see above)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
#ifdef DODE_BRINGUP
// bring-up only (never in the default build): a wait that gives up after ~1e7 polls, records who waited for what, and
// raises a flag that makes every other wait give up too, so that a deadlocked kernel ends and the record can be read
__device__ int g_wait_abort = 0;
__device__ int g_wait_rec[64];
#endif
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, int tag = 0, int aux = 0) {
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
                if (!aborted && atomicAdd(&g_wait_abort, 1) == 0) {          // first to give up names the block to report
                    g_wait_rec[60] = blockIdx.x; g_wait_rec[61] = blockIdx.y; g_wait_rec[62] = blockIdx.z;
                    __threadfence();
                }
                __threadfence();
                if ((threadIdx.x & 31) == 0 && (int)blockIdx.x == *(volatile int*)&g_wait_rec[60] &&
                    (int)blockIdx.y == *(volatile int*)&g_wait_rec[61] && (int)blockIdx.z == *(volatile int*)&g_wait_rec[62]) {
                    const int k = atomicAdd(&g_wait_rec[59], 1);
                    if (k < 14) { int* r = g_wait_rec + 4 * k; r[0] = tag; r[1] = aux; r[2] = threadIdx.x >> 5; r[3] = (int)parity; }
                }
                return;
            }
        }
#else
        (void)tag; (void)aux;
#endif
    } while (!done);
}

// One lane of a converged warp (elect.sync).  Inside a warp-uniform branch this lets ptxas emit the uniform-datapath
// instructions (UTMALDG, UTCHMMA, UTCBAR) once, predicated, instead of an ELECT/BRA.U.ANY loop per instruction.
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "elect.sync _|p, 0xffffffff;\n"
        "selp.b32 %0, 1, 0, p;\n"
        "}\n" : "=r"(pred));
    return pred != 0;
}

__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// K-major SWIZZLE_128B shared-memory matrix descriptor (sm_100 format): rows of 128 B, 8-row groups 1024 B apart.
__device__ __forceinline__ uint64_t umma_desc_k_sw128(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);          // start address, 16-byte units
    d |= (uint64_t)1 << 16;                            // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024 >> 4) << 32;                  // stride byte offset: 8 rows x 128 B
    d |= (uint64_t)1 << 46;                            // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;                            // layout type SWIZZLE_128B
    return d;
}

// K-major SWIZZLE_64B descriptor for the bf16 tiles (rows of 32 bf16 = 64 B, 8-row groups 512 B apart).
__device__ __forceinline__ uint64_t umma_desc_k_sw64(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(512 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)4 << 61;                            // layout type SWIZZLE_64B
    return d;
}

// The same two descriptors as compile-time constants of the layout (address 0), and a descriptor assembled from its
// two 32-bit words: high word = layout constants, low word = address in 16-byte units | LBO bit.
__host__ __device__ constexpr uint64_t umma_desc_k_sw128_c(uint32_t a16) {
    return (uint64_t)a16 | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__host__ __device__ constexpr uint64_t umma_desc_k_sw64_c(uint32_t a16) {
    return (uint64_t)a16 | ((uint64_t)1 << 16) | ((uint64_t)(512 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)4 << 61);
}
__device__ __forceinline__ uint64_t desc_pack(uint32_t lo, uint32_t hi) {
    uint64_t d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "r"(lo), "r"(hi));
    return d;
}

// kind::f16 instruction descriptor: D = F32, A = B = BF16, both K-major, M = 128, N = bn.
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int bn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
}

// kind::tf32 instruction descriptor: D = F32, A = B = TF32, both K-major, M = 128, N = bn.
__host__ __device__ constexpr uint32_t umma_idesc_tf32(int bn) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
}

__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

struct TcParams {
    int mode;            // 0 = forward (a2), 1 = gradient (a3 + a4)
    int M;               // valid outputs per time index (L forward, N gradient)
    int T, H;
    int kunit;           // K rows per lag (Np forward, Lp gradient)
    int slab0;           // c*T: first (cluster, time) slab of the A tensor map
    int mtile0;          // first 128-output tile of this launch (a pass may be split between the pair and the single-CTA kernel)
    int Lp, Np;
    int bn;              // days per CTA (MMA N of the main product), a multiple of 16, <= 128
    int dsplit;          // day groups per output tile (1, or 2 for minibatches wider than 128 days): blockIdx.x % dsplit
    int bnt;             // dsplit * bn: padded minibatch width (row stride of the split-K partial sums)
    int stages;          // A ring: stages of one 16 KB A tile each (HBM latency: as deep as shared memory allows)
    int bstages;         // B ring: stages of B_full | bf16(B) | bf16(B_lo) (panels live in L2: 2-3 suffice), <= stages
    int nring;           // TMEM A buffers (2 or 4), half per splitter group
    // epilogue
    const float* x;      // [D][T][L]        (forward)
    float* rp_full;      // [bcap][rpitch]   (forward output / gradient B operand)
    __nv_bfloat16* rp_lo;   // [2][pcap][rpitch] bf16: bf16(r) then bf16(r - tf32(r))
    int pcap;               // rows of the minibatch panels (second bf16 plane starts at row pcap)
    long rpitch;
    float* q;            // [D][T][Np]       (gradient, in place)
    size_t dayStride;
    float eta;
    // NEXT-1 (Alg. 1 as printed); both nullable
    const uint8_t* mask; // forward: [n][T][L] bytes by position in the day list, 0 = row outside the chunk B_o (r = 0)
    float* G;            // gradient: Adagrad accumulator [D][T][Np], in place
    float eps;
    // split-K (short time axes: T * tiles CTAs would not fill the machine): blockIdx.z takes a
    // contiguous range of K chunks and stores its raw accumulators to part[ks][tt][m][bn]; splitk_epilogue sums the
    // ranges in a fixed order and applies the pass's epilogue.  ksplit = 1: the fused epilogue below.
    int ksplit;
    float* part;
};

__device__ __forceinline__ void umma_tf32_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

__device__ __forceinline__ void umma_bf16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}
// two fp32 -> one word of two bf16 (round to nearest even): `lo` in bits 0-15 (the lower K index), `hi` in bits 16-31
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    uint32_t d;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
__device__ __forceinline__ float tf32_lo(float v) { return v - __uint_as_float(__float_as_uint(v) & 0xffffe000u); }

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
          "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}

// tcgen05.ld is asynchronous: its destination registers are written some time after the instruction issues and may be
// read only after tcgen05.wait::ld.  Load and wait therefore live in ONE asm statement: with them in separate
// statements the compiler is free to spill a destination register in between (it believes the value is there) and to
// hand the register to another variable, which the late write then clobbers — seen as an intermittent hang of the
// kernel variant that spills (ADA, 96 registers).
__device__ __forceinline__ void tmem_ld16_wait(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld16x2_wait(uint32_t t0, uint32_t t1, uint32_t* v, uint32_t* w) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%32];\n"
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%33];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]),
          "=r"(w[8]), "=r"(w[9]), "=r"(w[10]), "=r"(w[11]), "=r"(w[12]), "=r"(w[13]), "=r"(w[14]), "=r"(w[15])
        : "r"(t0), "r"(t1) : "memory");
}


// ADA = true compiles in the NEXT-1 epilogues (row mask on r, Adagrad accumulator).  It is a template parameter, not a
// run-time branch, because the extra live values cost 25 registers: 117 x 320 threads no longer fits two CTAs per SM.
// PART = fp32 partial sums a splitter thread carries across drains = its share of the bn day columns (bn <= 2 * PART):
// 16 / 32 for the two-CTAs-per-SM shapes (bn <= 32 / 64), 64 for bn <= 128 (one CTA per SM).
template <bool ADA, int PART>
__global__ void __launch_bounds__(kThreadsTC, PART <= 32 ? 2 : 1)
banded_gemm_3xtf32(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapA64,
                   const __grid_constant__ CUtensorMap mapBf, const __grid_constant__ CUtensorMap mapBl,
                   const __grid_constant__ TcParams p, const __grid_constant__ DayList dl) {
    // SWIZZLE_128B tiles need 1024-byte alignment: the declared alignment places the dynamic shared memory (the kernel
    // has no static shared memory) on such a boundary of the CTA's window; no slack is allocated for a manual round-up.
    extern __shared__ __align__(1024) uint8_t smem[];
    if ((smem_u32(smem) & 1023u) != 0u) __trap();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tt = blockIdx.y;                    // arrival interval t (forward) / departure interval s (gradient)
    const int m0 = ((int)blockIdx.x / p.dsplit + p.mtile0) * kTileM;
    const int d0 = ((int)blockIdx.x % p.dsplit) * p.bn;       // first day (position in the list) of this CTA's group
    const int bBytes = p.bn * kTileK * 4;
    // Two rings, because the two operands have different latencies to hide: A streams from HBM (deep ring), the B
    // panels sit in L2 (shallow ring).  Chunk kc uses A stage kc % SA and B stage kc % SB; MMAs retire in order, so
    // "chunk kc - SB retired" frees B stage kc % SB for chunk kc AND the A stage of chunk kc - SB for chunk kc - SB + SA.
    const int SA = p.stages, SB = p.bstages;
    const int bStage = 2 * bBytes;                               // B_full (fp32) | bf16(B) | bf16(B_lo)   (half a B tile each)
    uint8_t* ringB = smem + (size_t)SA * kABytes;
    const int nring = p.nring;
    // a tile with <= 64 valid outputs (small networks, ragged last tile) fetches and splits a 64-wide A box; the
    // MMA still runs M = 128 and the upper accumulator rows are never stored
    const bool half = p.M - m0 <= 64;
    const int BM = half ? kTileM / 2 : kTileM;                   // A tile in smem: [kTileK rows][BM floats], no swizzle
    const int aBytes = BM * kTileK * 4;
    const CUtensorMap* mA = half ? &mapA64 : &mapA;
    uint64_t* bars = reinterpret_cast<uint64_t*>(ringB + (size_t)SB * bStage);
    // full: TMA landed an A tile.  One barrier per (splitter group, A stage): chunk kc completes
    // full[(kc & 1) * SA + kc % SA], and only that group's splitters wait on it, so every waiter of a barrier sees EVERY
    // one of its phases in turn.  (With one barrier per stage a group would have to watch the other group's chunks go by
    // just to keep count, and a warp that is slow to start could fall two phases behind and wait for ever — seen once in
    // ~300 steps on the multiyear shape.)  fullB: the B tiles of a chunk landed; only the MMA warp waits on it.  (One
    // barrier for both made the splitters wait for the B tiles, which are requested three chunks later than the A tile.)
    uint64_t* full = bars;                        // [2][SA]
    uint64_t* fullB = bars + 2 * SA;              // [SB]
    uint64_t* empty = fullB + SB;                 // [SB] MMAs of the chunk in this B stage retired
    uint64_t* split = empty + SB;                 // [nring] A_hi/A_lo in TMEM
    uint64_t* a_empty = split + 4;                // [nring] MMAs that read this TMEM buffer retired
    uint64_t* accum = a_empty + 4;                // all MMAs issued so far retired (every drain and the end)
    uint64_t* drained = accum + 1;                // the splitter threads have read the accumulators of a drain
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(drained + 1);

    const int lags = (p.mode == 0 ? min(p.H, tt) : min(p.H, p.T - 1 - tt)) + 1;
    const int nk_all = (lags * p.kunit + kTileK - 1) / kTileK;
    const int cps = (nk_all + p.ksplit - 1) / p.ksplit;                         // chunks per split
    const int kbase = (int)blockIdx.z * cps;                                    // first chunk of this CTA's range
    const int nk = max(0, min(nk_all, kbase + cps) - kbase);
    const int w0 = (p.mode == 0 ? (tt - lags + 1) * p.kunit : tt * p.kunit) + kbase * kTileK;   // first element of the B window

    const int acc_cols = 2 * p.bn;
    uint32_t tmem_cols = 32;
    while ((int)tmem_cols < acc_cols + 64 * nring) tmem_cols <<= 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < SA; ++s) { mbar_init(&full[s], 1); mbar_init(&full[SA + s], 1); }
        for (int s = 0; s < SB; ++s) { mbar_init(&fullB[s], 1); mbar_init(&empty[s], 1); }
        for (int j = 0; j < nring; ++j) { mbar_init(&split[j], 128); mbar_init(&a_empty[j], 1); }
        mbar_init(accum, 1);
        mbar_init(drained, 256);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(mA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapBf) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapBl) : "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_d = *tmem_slot;
    const uint32_t tmem_ring = tmem_d + (uint32_t)acc_cols;
    const int per_group = nring >> 1;

    // Programmatic dependent launch: everything above overlapped the previous kernel's tail.  The next kernel in
    // the stream may start its own prologue now; nothing produced by the previous kernel is touched before the wait.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // The operator is static: the A tiles of the first ring round are requested NOW, before the dependency wait — a CTA
    // that gets its SM slot while the previous kernel's slower CTAs are still running streams its first SA chunks
    // under that kernel's tail.  The B tiles (panels written by the previous kernel) follow after the wait; the stage's
    // barrier expects the bytes of all three loads from the start.
    const int npre = min(SA, nk);
    if (warp == 0) {
        if (elect_one()) {
            for (int kc = 0; kc < npre; ++kc) {                  // (kc < SA: the stage index is kc)
                uint64_t* fb = &full[(kc & 1) * SA + kc];
                mbar_expect_tx(fb, aBytes);
                tma_load_3d(smem + (size_t)kc * kABytes, mA, fb, m0, (kbase + kc) * kTileK, p.slab0 + tt);
            }
        }
        __syncwarp();
    }
    // Epilogue operands (x for the forward pass, the old q for the update) are fetched by the epilogue threads
    // BEFORE the main loop so that their DRAM/L2 latency is hidden behind it: 16 values per thread.
    float pre[16];
    const int erow = ((warp & 3) << 5) + lane, em = m0 + erow;
    const int egroup = warp >= 2 ? (warp - 2) >> 2 : 0;
    // One base pointer and one day stride for both passes, rows and days clamped instead of predicated: the loads are
    // unconditional, nothing reads their registers before the epilogue (which applies m < M, d < n), and the address
    // is one multiply-add per element.  (Predicated per-mode loads with the full index expression were ~2400 SASS
    // instructions ahead of the main loop — 3800 cycles before a CTA's first split in the per-chunk trace.)
    const int emc = min(em, p.M - 1);
    const float* ebase = p.mode == 0 ? p.x + ((size_t)tt * p.M + emc) : p.q + ((size_t)tt * p.Np + emc);
    const size_t estride = p.mode == 0 ? (size_t)p.T * p.M : p.dayStride;
    auto prefetch = [&](int c0) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int d = min(d0 + c0 + j, dl.n - 1);
            pre[j] = __ldcg(ebase + (size_t)dl.day[d] * estride);    // through L2: q may have been written under PDL
        }
    };
    uint32_t keep = 0xffffu;                                          // bit j: row (em, day c0+j) belongs to the chunk B_o
    auto prefetch_mask = [&](int c0) {
        keep = 0;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int d = d0 + c0 + j;
            if (em < p.M && d < dl.n && __ldg(p.mask + ((size_t)d * p.T + tt) * p.M + em) != 0) keep |= 1u << j;
        }
    };
    const bool fused_epi = p.ksplit == 1;
    if (fused_epi && p.mode == 0 && warp >= 2) prefetch(16 * egroup);             // x is a static input
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (ADA && p.mode == 0 && p.mask != nullptr && warp >= 2) prefetch_mask(16 * egroup);   // the caller's buffer: after the wait
    // q was written by the previous step's kernel, which may still have been running on this SM when this CTA was
    // launched (PDL): the launch-time L1 invalidation does not cover it, so q is read through L2 (ld.global.cg)
    if (fused_epi && p.mode == 1 && warp >= 2) prefetch(16 * egroup);

    if (warp == 0) {
        // ===== TMA producer =====
        int sb = 0, ph = 1;                                      // ph: parity of the previous round of B slot sb
        int sa = 0;                                              // A stage of chunk kc (== that of chunk kc - SB + SA ... + SB)
        for (int kc = 0; kc < nk; ++kc) {
            if (kc >= SB) mbar_wait(&empty[sb], ph, 1, kc);      // chunk kc - SB retired
            if (elect_one()) {
                const int ka = kc - SB + SA;                     // the A stage that chunk kc - SB leaves takes chunk ka
                if (kc >= SB && ka < nk) {                       // (ka >= SA >= npre: the first round was requested before the wait)
                    int sk = sa - SB; if (sk < 0) sk += SA;      // ka % SA == (kc - SB) % SA
                    uint64_t* fa = &full[(ka & 1) * SA + sk];
                    mbar_expect_tx(fa, aBytes);
                    tma_load_3d(smem + (size_t)sk * kABytes, mA, fa, m0, (kbase + ka) * kTileK, p.slab0 + tt);
                }
                uint8_t* st = ringB + (size_t)sb * bStage;
                uint64_t* fb = &fullB[sb];
                mbar_expect_tx(fb, 2 * bBytes);
                tma_load_2d(st, &mapBf, fb, w0 + kc * kTileK, d0);
                tma_load_2d(st + bBytes, &mapBl, fb, w0 + kc * kTileK, d0);                       // bf16(B)
                tma_load_2d(st + bBytes + bBytes / 2, &mapBl, fb, w0 + kc * kTileK, p.pcap + d0);   // bf16(B_lo)
            }
            __syncwarp();
            if (++sb == SB) { sb = 0; ph ^= 1; }
            if (++sa == SA) sa = 0;
        }
    } else if (warp == 1) {
        // ===== MMA issuer: the whole warp walks the loop, one elected lane issues =====
        const uint32_t idesc1 = umma_idesc_tf32(p.bn), idesc16 = umma_idesc_bf16(p.bn);
        // Shared-memory descriptors: the high words are constants of the layout, the low word is the tile address in
        // 16-byte units (+ the LBO bit), so a K slice or a ring stage is ONE 32-bit add away from the ring's base.
        // (Building every descriptor from its byte address cost ~90 uniform-datapath instructions per chunk; with
        // them the issuing warp — not the tensor pipe or the stream — set the pace of the wide-minibatch kernels.)
        constexpr uint32_t hi128 = (uint32_t)(umma_desc_k_sw128_c(0) >> 32), hi64 = (uint32_t)(umma_desc_k_sw64_c(0) >> 32);
        const uint32_t ring16 = ((smem_u32(ringB) & 0x3FFFFu) >> 4) | (1u << 16);
        const uint32_t st16 = (uint32_t)bStage >> 4, bB16 = (uint32_t)bBytes >> 4;
        const int pg_mask = per_group - 1, pg_shift = per_group >> 1;   // per_group is 1 or 2
        int sb = 0;                                             // B stage
        uint32_t bph = 0u;                                      // parity of the next phase of fullB[sb], bit sb
        for (int kc = 0; kc < nk; ++kc) {
            const int g = kc & 1, use = kc >> 1;
            const int jr = g * per_group + (use & pg_mask);
            const bool restart = kc % kFlushChunks == 0;        // first chunk of a segment: the accumulators start over
            if (restart && kc > 0) {                            // drain: the splitter threads read the sums so far
                if (elect_one()) umma_commit(accum);
                __syncwarp();
                mbar_wait(drained, (kc / kFlushChunks - 1) & 1, 2, kc);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            }
            mbar_wait(&fullB[sb], (bph >> sb) & 1u, 3, kc);
            bph ^= 1u << sb;
            mbar_wait(&split[jr], (use >> pg_shift) & 1, 4, kc);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t f16 = ring16 + (uint32_t)sb * st16;                  // fp32 B | bf16(B) | bf16(B_lo)
            const uint32_t h16 = f16 + bB16, l16 = h16 + (bB16 >> 1);
            const uint32_t afull = tmem_ring + (uint32_t)jr * 64, a16 = afull + 32, alo16 = afull + 48;
            if (elect_one()) {
#pragma unroll
                for (int k = 0; k < kTileK / 8; ++k)             // main product, UMMA_K = 8 for tf32 (32 bytes of the 128-byte rows)
                    umma_tf32_ts(tmem_d, afull + k * 8, desc_pack(f16 + 2 * k, hi128), idesc1, !(restart && k == 0));
#pragma unroll
                for (int k = 0; k < kTileK / 16; ++k) {          // corrections in bf16, UMMA_K = 16 (32 bytes of the 64-byte rows)
                    umma_bf16_ts(tmem_d + (uint32_t)p.bn, alo16 + k * 8, desc_pack(h16 + 2 * k, hi64), idesc16, !(restart && k == 0));  // a_lo * b
                    umma_bf16_ts(tmem_d + (uint32_t)p.bn, a16 + k * 8, desc_pack(l16 + 2 * k, hi64), idesc16, 1);                       // a * b_lo
                }
                umma_commit(&empty[sb]);
                umma_commit(&a_empty[jr]);
            }
            __syncwarp();
            if (++sb == SB) sb = 0;
        }
        if (elect_one()) { if (nk == 0) mbar_arrive(accum); else umma_commit(accum); }
        __syncwarp();
    } else {
        // ===== splitters: smem column -> registers -> TMEM (A_hi, A_lo); group g takes chunks kc = g, g+2, ... =====
        const int group = (warp - 2) >> 2;
        const int lane_base = (warp & 3) * 32;                  // TMEM lanes this warp may touch
        const int row = lane_base + lane;                       // output row within the tile == TMEM lane
        const uint32_t tacc = tmem_d + ((uint32_t)lane_base << 16);
        // partial sums of this thread's day columns (chunks c0 = 16*group + 32*i), filled by the drains
        float part[PART];
#pragma unroll
        for (int j = 0; j < PART; ++j) part[j] = 0.f;
        int s = -1;
        uint32_t fph = 0u;                                      // parity of the next phase of this group's full[s], bit s
        for (int kc = 0; kc < nk; ++kc) {
            if (kc > 0 && kc % kFlushChunks == 0) {
                // ---- drain (both groups, every thread its own columns): main + correction halves into registers ----
                mbar_wait(accum, (kc / kFlushChunks - 1) & 1, 5, kc);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                __syncwarp();
#pragma unroll
                for (int i = 0; i < PART / 16; ++i) {
                    const int c0 = 16 * group + 32 * i;
                    if (c0 < p.bn) {                            // warp-uniform
                        uint32_t v[16], w[16];
                        tmem_ld16x2_wait(tacc + (uint32_t)c0, tacc + (uint32_t)(c0 + p.bn), v, w);
#pragma unroll
                        for (int j = 0; j < 16; ++j) part[i * 16 + j] += __uint_as_float(v[j]) + __uint_as_float(w[j]);
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                mbar_arrive(drained);
            }
            if (++s == SA) s = 0;
            if ((kc & 1) != group) continue;
            const int use = kc >> 1;
            const int jr = group * per_group + (use & (per_group - 1));       // per_group is 1 or 2
            mbar_wait(&full[group * SA + s], (fph >> s) & 1u, 6, kc);
            fph ^= 1u << s;
            if (use >= per_group) mbar_wait(&a_empty[jr], ((use >> (per_group >> 1)) - 1) & 1, 7, kc);
            if (lane_base >= BM) { mbar_arrive(&split[jr]); continue; }    // rows never stored
            const float* A = reinterpret_cast<const float*>(smem + (size_t)s * kABytes) + row;
            const uint32_t t0 = tmem_ring + (uint32_t)jr * 64 + ((uint32_t)lane_base << 16);
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {                    // two halves of the 32 K rows: 32 live registers, not 64
                uint32_t hi[16], h16[8], l16[8];                // (one 32-wide pass spills beside the partial sums: measured slower)
#pragma unroll
                for (int k = 0; k < 16; ++k) hi[k] = __float_as_uint(A[(hf * 16 + k) * BM]);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float a0 = __uint_as_float(hi[2 * i]), a1 = __uint_as_float(hi[2 * i + 1]);
                    h16[i] = pack_bf16(a0, a1);
                    l16[i] = pack_bf16(tf32_lo(a0), tf32_lo(a1));
                }
                __syncwarp();                                   // tcgen05.st is .sync.aligned
                tmem_st16(t0 + hf * 16, hi);                    // fp32 as it is: the tensor core reads its TF32 part
                tmem_st8(t0 + 32 + hf * 8, h16);
                tmem_st8(t0 + 48 + hf * 8, l16);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            mbar_arrive(&split[jr]);
        }
        // ---- epilogue ----
        mbar_wait(accum, (nk > 0 ? (nk - 1) / kFlushChunks : 0) & 1, 8, nk);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int m = m0 + row;
#pragma unroll
        for (int i = 0; i < PART / 16; ++i) {
            const int c0 = 16 * group + 32 * i;
            if (c0 >= p.bn) break;
            uint32_t v[16], w[16];
            float cur[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) cur[j] = pre[j];
            const uint32_t curkeep = keep;
            if (fused_epi && c0 + 32 < p.bn) {                  // next chunk's operands: in flight across this chunk's stores
                prefetch(c0 + 32);
                if (ADA && p.mode == 0 && p.mask != nullptr) prefetch_mask(c0 + 32);
            }
            __syncwarp();                                       // tcgen05.ld / wait::ld are .sync.aligned
            tmem_ld16x2_wait(tacc + (uint32_t)c0, tacc + (uint32_t)(c0 + p.bn), v, w);
            float sum[16];
#pragma unroll
            for (int j = 0; j < 16; ++j)
                sum[j] = nk ? part[i * 16 + j] + (__uint_as_float(v[j]) + __uint_as_float(w[j])) : 0.f;
            if (!fused_epi) {                                   // split-K: raw partial sums, 16 consecutive days per thread
                if (m < p.M) {
                    float4* dst = reinterpret_cast<float4*>(
                        p.part + (((size_t)blockIdx.z * gridDim.y + tt) * ((size_t)(gridDim.x / p.dsplit) * kTileM) + m) * p.bnt + d0 + c0);   // (split-K launches cover all tiles: mtile0 = 0)
#pragma unroll
                    for (int j = 0; j < 16; j += 4) dst[j >> 2] = make_float4(sum[j], sum[j + 1], sum[j + 2], sum[j + 3]);
                }
                continue;
            }
            if (m < p.M) {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int d = d0 + c0 + j;
                    if (d < dl.n) {
                        const float acc = sum[j];
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
    __syncthreads();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"(tmem_cols) : "memory");
    }
}

// Second half of a split-K pass: out[tt][m][d] = sum_ks part[ks][tt][m][d] in a fixed order, then the pass's epilogue
// (the same arithmetic as the fused one).  Thread = (m, 4 days); grid = (ceil(Mt*bn/4 / 256), T).
template <bool ADA>
__global__ void __launch_bounds__(256)
splitk_epilogue(const __grid_constant__ TcParams p, int Mt, const __grid_constant__ DayList dl) {
    const int tt = blockIdx.y;
    const int q4 = p.bnt >> 2;
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= (long)Mt * q4) return;
    const int m = (int)(i / q4), d0 = (int)(i - (long)m * q4) * 4;
    if (m >= p.M) return;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int ks = 0; ks < p.ksplit; ++ks) {
        const float4 v = __ldcg(reinterpret_cast<const float4*>(p.part + (((size_t)ks * p.T + tt) * Mt + m) * p.bnt + d0));
        acc[0] += v.x; acc[1] += v.y; acc[2] += v.z; acc[3] += v.w;
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int d = d0 + e;
        if (d >= dl.n) break;
        if (p.mode == 0) {
            float r = acc[e] - __ldg(p.x + ((size_t)dl.day[d] * p.T + tt) * p.M + m);
            if (ADA && p.mask != nullptr && p.mask[((size_t)d * p.T + tt) * p.M + m] == 0) r = 0.f;
            p.rp_full[(size_t)d * p.rpitch + (size_t)tt * p.Lp + m] = r;
            p.rp_lo[(size_t)d * p.rpitch + (size_t)tt * p.Lp + m] = __float2bfloat16_rn(r);
            p.rp_lo[(size_t)(p.pcap + d) * p.rpitch + (size_t)tt * p.Lp + m] = __float2bfloat16_rn(tf32_lo(r));
        } else {
            const size_t qi = (size_t)dl.day[d] * p.dayStride + (size_t)tt * p.Np + m;
            const float qv = __ldcg(p.q + qi);
            if (ADA && p.G != nullptr) p.q[qi] = adagrad_update(qv, acc[e], p.G + qi, p.eta, p.eps);
            else p.q[qi] = fmaxf(0.f, fmaf(-p.eta, acc[e], qv));
        }
    }
}

// a1 for the tensor path: Qg_full[d][i] = q[day_d][i] (fp32) and the two bf16 planes of the correction operands,
// g16[d][i] = bf16(q), g16[pcap + d][i] = bf16(q - trunc_tf32(q)), i over T*Np (float4 wide)
__global__ void __launch_bounds__(256)
gather_split(const float* __restrict__ q, size_t dayStride, long len4, float* __restrict__ gfull, __nv_bfloat16* __restrict__ g16,
             int pcap, const __grid_constant__ DayList dl) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");          // q is written by the previous step's update
    const int d = blockIdx.y;
    const float4* src = reinterpret_cast<const float4*>(q + (size_t)dl.day[d] * dayStride);
    float4* f = reinterpret_cast<float4*>(gfull + (size_t)d * dayStride);
    uint2* h = reinterpret_cast<uint2*>(g16 + (size_t)d * dayStride);
    uint2* l = reinterpret_cast<uint2*>(g16 + (size_t)(pcap + d) * dayStride);
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < len4; i += (long)gridDim.x * blockDim.x) {
        const float4 v = __ldcg(src + i);          // through L2: see the note on PDL and L1 in banded_gemm_3xtf32
        f[i] = v;
        h[i] = make_uint2(pack_bf16(v.x, v.y), pack_bf16(v.z, v.w));
        l[i] = make_uint2(pack_bf16(tf32_lo(v.x), tf32_lo(v.y)), pack_bf16(tf32_lo(v.z), tf32_lo(v.w)));
    }
}

}  // namespace tc
}  // namespace dode
