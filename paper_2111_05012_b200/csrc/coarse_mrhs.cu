// coarse_mrhs.cu -- row F4 of SURVEY.md section 8(f): the coarse operator applied to K right-hand sides at once,
//   out_k(X) = A_0(X) in_k(X) + sum_mu [ A_{+mu}(X) in_k(X+mu) + A_{-mu}(X) in_k(X-mu) ],   k = 0 .. K-1
// (Eqs. 4, 7; many right-hand sides are "a typical situation").
//
// With K right-hand sides every block A_d(X) is re-used K times: the arithmetic intensity is K flop/byte and the
// operation per coarse site is a dense contraction (N x 9N complex) . (9N x K complex) -- the one place of this path
// where tensor cores belong.  Per site, in REAL arithmetic on the interleaved (re, im)
// storage:  C[r][(k,re)] = sum_j (a_r[2j] b_kj.re - a_r[2j+1] b_kj.im),  C[r][(k,im)] = sum_j (a_r[2j] b_kj.im +
// a_r[2j+1] b_kj.re), i.e. C (64 x 2K) = A (64 x 1152, the rows of the nine blocks as stored) . B' (1152 x 2K) with
// B'[(2j, 2j+1)][(k,re)] = (b.re, -b.im), B'[(2j, 2j+1)][(k,im)] = (b.im, b.re).
//
// tcgen05 (5th-generation tensor cores): kind::tf32 MMAs with fp32 accumulators in TMEM.  TF32 alone (10-bit mantissa)
// would miss the fp32 bar of 2e-6 by two orders of magnitude, so every fp32 operand is split into hi + lo
// (hi = x rounded to the nearest TF32 value, i.e. 13 low mantissa bits cleared; lo = x - hi, exact, either sign) and each
// product is formed from the hi / lo pieces ("3xTF32"; with the stacked operands below all four terms come out).  The split is done
// by the producer warps on the way from HBM to shared memory, so A is still read from HBM exactly once, as fp32.
//
// One persistent CTA per SM, warp-specialised (704 threads):
//   warps 0-3   epilogue: tcgen05.ld each accumulator chain, add it in registers (fp32, round-to-nearest), store out_k(X)
//   warps 4-5   MMA issuers (one elected lane each, accumulator chains in turn); warp 4 allocates / frees TMEM
//   warps 6-21  producers, four groups of four warps that take the stages in turn: stream A (whole 128-byte lines,
//               L1 no-allocate), build B' from the neighbours' input vectors (L2-resident), split into hi / lo, store
//               both in the 128-byte-swizzled K-major layout UMMA reads (conflict-free stores)
// Shared-memory ring of 4 stages (one stage = half a block: A as 128 rows (hi | lo) x 64 reals, B' as 4K rows
// (hi | lo) x 64 reals), a ring of TMEM accumulator slots (one per chain of two stages); mbarriers full[] (producers ->
// issuer), done[] (tcgen05.commit -> producers), tfull[] (tcgen05.commit -> epilogue), tfree[] (epilogue -> issuer).
#include "common.cuh"
#include "knobs.h"

namespace lqcd {

constexpr int MR_ROWS = 64;          // N = 2 nvec = 64 rows per block; hi and lo stacked: UMMA M = 128
constexpr int MR_KT = 64;            // reals of the contraction index per stage (half a block)
constexpr int MR_HALVES = 18;        // 9 blocks x 2 halves per coarse site
constexpr int MR_AS = 2;             // pipeline stages accumulated into one TMEM slot (chain of MR_AS * 8 MMAs)
constexpr int MR_EPI_WARPS = 4, MR_PROD_GROUPS = 4, MR_PROD_WARPS = 4 * MR_PROD_GROUPS;
constexpr int MR_ISSUERS = 2;         // MMA-issuing warps (one elected lane each); stages in turn, like the producers
constexpr int MR_THREADS = (MR_EPI_WARPS + MR_ISSUERS + MR_PROD_WARPS) * 32;  // 704
constexpr int MR_TMEM_COLS = 512;    // all of TMEM: one accumulator slot of 2 NCOL columns per pipeline stage

struct MrhsParams {
    int Lc[4];
    FastDiv dLc[3];  // division by Lc[0..2] as a multiply-high
    int Vc;
    int nrhs;     // K
    int stages;      // shared-memory pipeline stages
    int slots;       // TMEM accumulator slots (2 NCOL columns each); a multiple of groups
    long long vstride;  // reals between consecutive right-hand sides: Vc * 128
};

// ---- PTX wrappers -----------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// Developer aid (compiled only with -DLQCD_MRHS_TRACE): clock64 stamps of CTA 0's three roles for the first 128 stages.
#ifdef LQCD_MRHS_TRACE
__device__ long long g_mr_trace[3][128][6];
#define MR_TRACE(role, idx, which)                                                                \
    do {                                                                                          \
        if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && (idx) < 128) g_mr_trace[role][idx][which] = clock64(); \
    } while (0)
#else
#define MR_TRACE(role, idx, which)
#endif
// spin on the phase parity (one lane; see mbar_wait)
#ifdef LQCD_MRHS_TRACE
__device__ int g_mr_hang[64][4];
__device__ int g_mr_hang_n;
__device__ __forceinline__ void mbar_wait_lane(unsigned long long* bar, unsigned parity, int tag = 0, int g = 0) {
    for (int n = 0; n < (1 << 22); n++) {
        unsigned ok;
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (ok) return;
    }
    const int i = atomicAdd(&g_mr_hang_n, 1);
    if (i < 64) {
        g_mr_hang[i][0] = blockIdx.x * 1000 + (threadIdx.x >> 5);
        g_mr_hang[i][1] = tag;
        g_mr_hang[i][2] = g;
        g_mr_hang[i][3] = (int)parity;
    }
}
#else
__device__ __forceinline__ void mbar_wait_lane(unsigned long long* bar, unsigned parity, int tag = 0, int g = 0) {
    unsigned ok;
    do {  // try_wait suspends the thread for a bounded time; no asm labels (they clash when inlined repeatedly)
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
#endif
// the whole warp waits: lane 0 polls, __syncwarp orders its acquire before the other lanes' later accesses
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity, int tag = 0, int g = 0) {
    if ((threadIdx.x & 31) == 0) mbar_wait_lane(bar, parity, tag, g);
    __syncwarp();
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(unsigned long long* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
// D[tmem] (+)= A[smem] . B[smem]^T, kind::tf32, K = 8 reals per instruction
__device__ __forceinline__ void tc_mma_tf32(unsigned tmem_d, unsigned long long desc_a, unsigned long long desc_b,
                                            unsigned idesc, unsigned accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// Shared-memory matrix descriptor, K-major, 128-byte swizzle: the tile is stored as rows of 128 bytes (32 reals of
// the contraction index); inside each group of 8 rows (1024 bytes, 1024-byte aligned) the 16-byte chunk c of row r
// sits at chunk position c ^ (r & 7).  SBO = 1024 bytes between 8-row groups; LBO is not used by this mode.
// A k-step of 8 reals advances the start address by 32 bytes inside the 128-byte row.
__device__ __forceinline__ unsigned long long umma_desc_sw128(unsigned saddr) {
    unsigned long long d = 0;
    d |= (unsigned long long)((saddr & 0x3FFFFu) >> 4);
    d |= 1ull << 16;                           // LBO field (ignored for swizzled K-major layouts)
    d |= (unsigned long long)(1024 >> 4) << 32;  // SBO
    d |= 1ull << 46;                           // descriptor version of sm_100
    d |= 2ull << 61;                           // layout type SWIZZLE_128B
    return d;
}
// byte offset of 16-byte chunk kc (0..15) of row r in a [2 K-atoms][rows][128 B] swizzled tile
__device__ __forceinline__ int sw128_off(int rows, int r, int kc) {
    return (kc >> 3) * rows * 128 + r * 128 + (((kc & 7) ^ (r & 7)) << 4);
}
__device__ __forceinline__ V16<float> ldg_stream(const float* p) {
    V16<float> v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.r[0]), "=f"(v.r[1]), "=f"(v.r[2]), "=f"(v.r[3])
                 : "l"(p));
    return v;
}
__device__ __forceinline__ void split_tf32(const V16<float>& x, V16<float>& hi, V16<float>& lo) {
#pragma unroll
    for (int q = 0; q < 4; q++) {
        hi.r[q] = __uint_as_float((__float_as_uint(x.r[q]) + 0x1000u) & 0xFFFFE000u);  // nearest TF32
        lo.r[q] = x.r[q] - hi.r[q];
    }
}

// neighbour of coarse site X for block d (0 diag, 1+2mu forward, 2+2mu backward), periodic.  No dynamic indexing of
// the parameter struct (that would put it in local memory) and no run-time division: this sits on the producers'
// critical path (with a generic version the address arithmetic took longer than the loads it precedes).
__device__ __forceinline__ int coarse_neighbour(const MrhsParams& P, int X, int d) {
    if (d == 0) return X;
    const int mu = (d - 1) >> 1;
    const int q0 = P.dLc[0].div(X), x0 = X - q0 * P.Lc[0];
    const int q1 = P.dLc[1].div(q0), x1 = q0 - q1 * P.Lc[1];
    const int q2 = P.dLc[2].div(q1), x2 = q1 - q2 * P.Lc[2];
    const int s1 = P.Lc[0], s2 = s1 * P.Lc[1], s3 = s2 * P.Lc[2];
    const int c = mu == 0 ? x0 : mu == 1 ? x1 : mu == 2 ? x2 : q2;
    const int L = mu == 0 ? P.Lc[0] : mu == 1 ? P.Lc[1] : mu == 2 ? P.Lc[2] : P.Lc[3];
    const int stride = mu == 0 ? 1 : mu == 1 ? s1 : mu == 2 ? s2 : s3;
    if ((d - 1) & 1) return c == 0 ? X + (L - 1) * stride : X - stride;  // backward
    return c == L - 1 ? X - (L - 1) * stride : X + stride;               // forward
}

// shared memory: [stages][ A: 128 rows (hi, lo) x 64 reals = 32 KB | B_hi ncol*256 B | B_lo ncol*256 B ], then the
// exchange buffer of the epilogue (64 x ncol floats), then the mbarriers
__host__ __device__ constexpr unsigned mr_stage_bytes(int ncol) {
    return 2u * MR_ROWS * MR_KT * 4u + 2u * (unsigned)ncol * MR_KT * 4u;
}
__host__ __device__ constexpr int mr_max_stages(int ncol) {  // one TMEM slot of 2 ncol columns per stage
    return MR_TMEM_COLS / (2 * ncol) < 8 ? MR_TMEM_COLS / (2 * ncol) : 8;
}

// What shaped this kernel (all measured on B200):
//  * The tensor core adds into its fp32 accumulator with TRUNCATION: a chain of n accumulating MMAs shrinks the result
//    by about n * 2^-25 (432 MMAs per output -> 1.4e-5 relative, far above the 2e-6 bar).  So chains are short: every
//    pipeline stage (8 k-steps) starts FRESH accumulators in its own TMEM slot, and the epilogue warps add the slots
//    into registers in IEEE round-to-nearest fp32 (2.4e-7 relative L2 against the fp64 oracle).
//  * UMMA with M = 64 and both operands in shared memory exposes the A-read latency (~60-80 cycles per MMA instead of
//    N/2).  So hi and lo of A are STACKED to M = 128 rows: one MMA with B_hi gives hi.hi (rows 0-63) and lo.hi
//    (rows 64-127), one with B_lo gives hi.lo and lo.lo -- two full-rate MMAs per k-step instead of three slow ones,
//    and the fourth product term comes for free.  The small products sit in other TMEM lanes/columns than hi.hi, so
//    their truncation does not touch the main chain.
//  * After a tcgen05.commit the issuing thread stalls for several hundred cycles, and the MMAs here are tiny (16
//    cycles), so one issuer cannot keep up: MR_ISSUERS warps take the stages round-robin (stages are independent: fresh
//    accumulators), and ONE commit per stage signals both the producers (stage free) and the epilogue (slot ready).
template <int NCOL>
__global__ void __launch_bounds__(MR_THREADS, 1)
    k_coarse_mrhs(float* __restrict__ out, const float* __restrict__ in, const float* __restrict__ A, MrhsParams P) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = P.stages;
    constexpr int ncol = NCOL;
    constexpr unsigned stage_bytes = mr_stage_bytes(NCOL);
    float* xbuf = reinterpret_cast<float*>(smem + (size_t)S * stage_bytes);           // [64][NCOL]
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(xbuf + MR_ROWS * NCOL);
    const int T = P.slots;
    unsigned long long* full = bars;               // [S] producers -> issuer: operands of the stage are in shared memory
    unsigned long long* done = bars + S;           // [S] tcgen05.commit -> producers: the MMAs have read the stage
    unsigned long long* tfull = bars + 2 * S;      // [T] tcgen05.commit -> epilogue: the slot's accumulators are complete
    unsigned long long* tfree = bars + 2 * S + T;  // [T] epilogue -> issuer: the slot has been read
    unsigned* tmem_slot = reinterpret_cast<unsigned*>(bars + 2 * S + 2 * T);

    if (threadIdx.x == 0) {
        for (int i = 0; i < S; i++) {
            mbar_init(&full[i], 4);  // one arrival per warp of the producer group that owns the stage
            mbar_init(&done[i], 1);  // one tcgen05.commit
        }
        for (int i = 0; i < T; i++) {
            mbar_init(&tfull[i], 1);              // one tcgen05.commit
            mbar_init(&tfree[i], MR_EPI_WARPS);   // one arrival per epilogue warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == MR_EPI_WARPS) {  // the first issuer warp owns the tensor memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "n"(MR_TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem_base = *tmem_slot;
    const int nsites = (P.Vc - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;  // sites of this CTA
    const int G = nsites * MR_HALVES;                                                   // stages of this CTA

    if (warp < MR_EPI_WARPS) {
        // ===== epilogue: accumulator row 32 w + t lives in TMEM lane 32 w + t (UMMA M = 128) =====
        int g = 0;
        for (int it = 0; it < nsites; it++) {
            const int X = blockIdx.x + it * gridDim.x;
            float acc[NCOL];
#pragma unroll
            for (int q = 0; q < NCOL; q++) acc[q] = 0.f;
            for (int ch = 0; ch < MR_HALVES / MR_AS; ch++, g++) {  // g counts accumulator chains here
                const int st = g % T;  // TMEM slot
                if (warp == 0) MR_TRACE(2, g, 0);
                mbar_wait(&tfull[st], (g / T) & 1, 1, g);
                if (warp == 0) MR_TRACE(2, g, 1);
                tc_fence_after();
                const unsigned taddr = tmem_base + ((unsigned)(32 * warp) << 16) + (unsigned)(st * 2 * NCOL);
#pragma unroll
                for (int c0 = 0; c0 < 2 * NCOL; c0 += 32) {  // 32 columns per round trip
                    unsigned v[32];
#pragma unroll
                    for (int h = 0; h < 2; h++)
                        asm volatile(
                            "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                            "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                            : "=r"(v[16 * h + 0]), "=r"(v[16 * h + 1]), "=r"(v[16 * h + 2]), "=r"(v[16 * h + 3]),
                              "=r"(v[16 * h + 4]), "=r"(v[16 * h + 5]), "=r"(v[16 * h + 6]), "=r"(v[16 * h + 7]),
                              "=r"(v[16 * h + 8]), "=r"(v[16 * h + 9]), "=r"(v[16 * h + 10]), "=r"(v[16 * h + 11]),
                              "=r"(v[16 * h + 12]), "=r"(v[16 * h + 13]), "=r"(v[16 * h + 14]), "=r"(v[16 * h + 15])
                            : "r"(taddr + c0 + 16 * h));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int q = 0; q < 32; q++) acc[(c0 + q) % NCOL] += __uint_as_float(v[q]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tfree[st]);
                if (warp == 0) MR_TRACE(2, g, 2);
            }
            // rows 64..127 hold the lo(A) products of rows 0..63: add them across warps through shared memory
            if (warp >= 2) {
                const int row = 32 * (warp - 2) + lane;
#pragma unroll
                for (int q = 0; q < NCOL; q++) xbuf[q * MR_ROWS + row] = acc[q];
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (warp < 2) {
                const int row = 32 * warp + lane;
#pragma unroll
                for (int k = 0; k < NCOL / 2; k++)
                    if (k < P.nrhs)
                        *reinterpret_cast<float2*>(out + k * P.vstride + ((long long)X * MR_ROWS + row) * 2) =
                            make_float2(acc[2 * k] + xbuf[(2 * k) * MR_ROWS + row],
                                        acc[2 * k + 1] + xbuf[(2 * k + 1) * MR_ROWS + row]);
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
        }
    } else if (warp < MR_EPI_WARPS + MR_ISSUERS) {
        // ===== MMA issuers (one elected lane per warp) =====
        // instruction descriptor: D fp32, A and B TF32, both K-major, M = 128 (hi rows | lo rows of A),
        // N = 2 ncol (B'_hi rows | B'_lo rows): ONE MMA per k-step yields all four products hi.hi, lo.hi, hi.lo, lo.lo
        const unsigned idesc =
            (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)((2 * ncol) >> 3) << 17) | ((128u >> 4) << 24);
        const unsigned s0 = smem_u32(smem);
        const unsigned long long dA = umma_desc_sw128(s0);
        const unsigned long long dB = umma_desc_sw128(s0 + 2 * MR_ROWS * MR_KT * 4);
        // Issuer warp m takes the stages g = m, m + NG, ... (NG = P.groups divides S and T: a stage and a slot always
        // have the same issuer).  A wait on a ready mbarrier still costs ~300 cycles of shared-memory latency under the producers'
        // store traffic, a commit as much again: one issuer alone paced the kernel at ~1700 cycles per stage.
        // Issuer warp m takes the accumulator chains c = m, m + MR_ISSUERS, ... (MR_AS stages each).  MR_ISSUERS * MR_AS
        // divides S and MR_ISSUERS divides T, so a stage and a slot always have the same issuer (a parity wait cannot
        // tell one completed phase from the one two phases earlier).  One issuer alone cannot keep up: a wait on a ready
        // mbarrier costs ~300 cycles under the producers' store traffic, issuing 8 small MMAs ~500, a commit ~100.
        const int mi = warp - MR_EPI_WARPS;
        if (lane == 0) {
            for (int c = mi; c < G / MR_AS; c += MR_ISSUERS) {
                const int sl = c % T;
                MR_TRACE(1, c * MR_AS, 0);
                mbar_wait_lane(&tfree[sl], ((c / T) & 1) ^ 1, 2, c);
                MR_TRACE(1, c * MR_AS, 1);
                const unsigned tmem_d = tmem_base + (unsigned)(sl * 2 * NCOL);
#pragma unroll
                for (int hs = 0; hs < MR_AS; hs++) {
                    const int g = c * MR_AS + hs, st = g % S;
                    mbar_wait_lane(&full[st], (g / S) & 1, 3, g);
                    MR_TRACE(1, g, 2);
                    tc_fence_after();
                    // descriptors differ from those of (stage 0, k-step 0) only in the 14-bit address field
                    const unsigned long long so = (unsigned long long)(((unsigned)st * stage_bytes) >> 4);
#pragma unroll
                    for (int ks = 0; ks < MR_KT / 8; ks++) {  // 8 reals = 32 bytes of the 128-byte swizzled row
                        const unsigned long long ao =
                            so + (unsigned long long)(((ks >> 2) * 2 * MR_ROWS * 128 + (ks & 3) * 32) >> 4);
                        const unsigned long long bo =
                            so + (unsigned long long)(((ks >> 2) * 2 * ncol * 128 + (ks & 3) * 32) >> 4);
                        tc_mma_tf32(tmem_d, dA + ao, dB + bo, idesc, (hs | ks) != 0);
                    }
                    MR_TRACE(1, g, 3);
                    tc_commit(&done[st]);
                    MR_TRACE(1, g, 4);
                }
                tc_commit(&tfull[sl]);
            }
        }
        __syncwarp();
    } else {
        // ===== producers: MR_PROD_GROUPS groups of 4 warps, group pg takes the stages g = pg, pg + MR_PROD_GROUPS, ... =====
        // A group loads its NEXT stage into registers right after handing over the current one, and converts it a
        // full round (MR_PROD_GROUPS stage times, > the HBM latency) later.  Why not a deeper register prefetch inside
        // one group: fence.proxy.async / the releasing mbarrier arrive drain every outstanding load of the thread,
        // so loads in flight across a hand-over serialise the pipeline (measured: ~2000 cycles per stage).
        // Stage ownership: MR_PROD_GROUPS divides S, so a stage is always filled by the same group (a parity wait
        // cannot tell one completed phase from the one two phases earlier).
        const int pw = warp - MR_EPI_WARPS - MR_ISSUERS;  // 0..15
        const int pg = pw >> 2, wq = pw & 3;              // group, warp in group
        const int ptg = wq * 32 + lane;                   // 0..127
        // A: a warp instruction reads 2 rows x 256 contiguous bytes (whole 128-byte lines); 8 consecutive lanes then
        // store 8 chunks of ONE swizzled 128-byte row: conflict-free
        const int rl = lane >> 4, kcA = lane & 15;
        constexpr int kpad = NCOL / 2;
        constexpr int NA = MR_ROWS * (MR_KT / 4) / 128;              // 8 A loads per thread
        constexpr int NB = (kpad * (MR_KT / 4) + 127) / 128;          // B loads per thread
        const int rowA = wq * 2 + rl;                                 // rows rowA + 8 i
        const long long a_thr = (long long)rowA * 128 + kcA * 4;      // + i * 8 * 128 reals
        const int offA = sw128_off(2 * MR_ROWS, rowA, kcA);           // + i * 8 * 128 bytes; lo: + 64 * 128 bytes
        int kB[NB], offB[NB];
        long long b_thr[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) {
            const int q = ptg + j * 128;
            kB[j] = q >> 4;
            offB[j] = sw128_off(2 * ncol, 2 * kB[j], q & 15);
            b_thr[j] = (long long)kB[j] * P.vstride + (q & 15) * 4;
        }
        V16<float> a[NA], bq[NB];
        auto issue = [&](int g) {  // global loads of stage g
            const int it = g / MR_HALVES, hb = g - it * MR_HALVES, d = hb >> 1, half = hb & 1;
            const int X = blockIdx.x + it * gridDim.x;
            const float* Ab = A + ((long long)X * 9 + d) * (MR_ROWS * 128) + half * MR_KT + a_thr;
#pragma unroll
            for (int i = 0; i < NA; i++) a[i] = ldg_stream(Ab + i * 8 * 128);
            const float* Bb = in + (long long)coarse_neighbour(P, X, d) * 128 + half * MR_KT;
#pragma unroll
            for (int j = 0; j < NB; j++) {  // 16 consecutive lanes read the 256 contiguous bytes of one right-hand side
                if (kB[j] < kpad && kB[j] < P.nrhs)
                    bq[j] = *reinterpret_cast<const V16<float>*>(Bb + b_thr[j]);
                else
                    bq[j].r[0] = bq[j].r[1] = bq[j].r[2] = bq[j].r[3] = 0.f;
            }
        };
        constexpr int NG = MR_PROD_GROUPS;
        if (pg < G) issue(pg);
        for (int g = pg; g < G; g += NG) {
            const int st = g % S;
            if (wq == 0) MR_TRACE(0, g, 0);
            mbar_wait(&done[st], ((g / S) & 1) ^ 1, 4, g);
            if (wq == 0) MR_TRACE(0, g, 1);
            unsigned char* sA = smem + (size_t)st * stage_bytes;       // 128 rows: hi 0..63, lo 64..127
            unsigned char* sB = sA + 2 * MR_ROWS * MR_KT * 4;          // 2 ncol rows: hi 0..ncol-1, lo ncol..
#pragma unroll
            for (int i = 0; i < NA; i++) {
                V16<float> hi, lo;
                split_tf32(a[i], hi, lo);
                *reinterpret_cast<V16<float>*>(sA + offA + i * 8 * 128) = hi;
                *reinterpret_cast<V16<float>*>(sA + offA + i * 8 * 128 + MR_ROWS * 128) = lo;
            }
            // B': rows (k, re) = (b.re, -b.im), (k, im) = (b.im, b.re) per complex entry; 16 chunks of 2 complex
#pragma unroll
            for (int j = 0; j < NB; j++) {
                if (kB[j] < kpad) {
                    const V16<float> b = bq[j];
                    V16<float> re, im, hi, lo;
                    re.r[0] = b.r[0]; re.r[1] = -b.r[1]; re.r[2] = b.r[2]; re.r[3] = -b.r[3];
                    im.r[0] = b.r[1]; im.r[1] = b.r[0]; im.r[2] = b.r[3]; im.r[3] = b.r[2];
                    // row 2k+1 = row 2k + 128 bytes with the swizzle bit 0 flipped (2k is even)
                    split_tf32(re, hi, lo);
                    *reinterpret_cast<V16<float>*>(sB + offB[j]) = hi;
                    *reinterpret_cast<V16<float>*>(sB + offB[j] + ncol * 128) = lo;
                    split_tf32(im, hi, lo);
                    *reinterpret_cast<V16<float>*>(sB + (offB[j] ^ 16) + 128) = hi;
                    *reinterpret_cast<V16<float>*>(sB + (offB[j] ^ 16) + 128 + ncol * 128) = lo;
                }
            }
            if (wq == 0) MR_TRACE(0, g, 2);
            fence_proxy_async();  // generic-proxy stores -> visible to the tensor core's async-proxy reads
            __syncwarp();
            if (lane == 0) mbar_arrive(&full[st]);
            if (wq == 0) MR_TRACE(0, g, 3);
            if (g + NG < G) issue(g + NG);
            if (wq == 0) MR_TRACE(0, g, 4);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == MR_EPI_WARPS) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(MR_TMEM_COLS)
                     : "memory");
    }
}

static int mrhs_max_smem() { return max_optin_smem(); }
static int mrhs_sm_count() { return sm_count(); }

// one tensor-core launch for up to 16 right-hand sides
template <int NCOL>
static int mrhs_launch_ncol(float* out, const float* in, const float* A, MrhsParams P, cudaStream_t st, const char* what) {
    constexpr size_t stage = mr_stage_bytes(NCOL);
    // S = 4 stages: a multiple of the producer groups and of MR_ISSUERS * MR_AS (stage ownership, see the kernel)
    const int S = 4;
    static_assert(4 % MR_PROD_GROUPS == 0 && 4 % (MR_ISSUERS * MR_AS) == 0, "stage ownership");
    if ((size_t)mrhs_max_smem() < S * stage + MR_ROWS * NCOL * 4 + 1024) {
        set_error("%s: not enough shared memory for the pipeline", what);
        return LQCD_EUNSUPPORTED;
    }
    P.slots = mr_max_stages(NCOL) / MR_ISSUERS * MR_ISSUERS;
    P.stages = S;
    const size_t smem = S * stage + MR_ROWS * NCOL * 4 + (2 * S + 2 * 8) * 8 + 16;
    static unsigned long long attr = 0;
    ensure_dynamic_smem(k_coarse_mrhs<NCOL>, mrhs_max_smem(), attr);
    const int grid = P.Vc < mrhs_sm_count() ? P.Vc : mrhs_sm_count();
    k_coarse_mrhs<NCOL><<<grid, MR_THREADS, smem, st>>>(out, in, A, P);
    count_launch();
    return check_launch(what);
}

static int mrhs_tensor_launch(float* out, const float* in, const float* A, const int cdims[4], int nrhs, long long vstride,
                              cudaStream_t st, const char* what) {
    MrhsParams P;
    for (int mu = 0; mu < 4; mu++) P.Lc[mu] = cdims[mu];
    for (int mu = 0; mu < 3; mu++) P.dLc[mu].set(cdims[mu]);
    P.Vc = (int)volume(cdims);
    P.nrhs = nrhs;
    P.vstride = vstride;
    P.stages = 0;
    if (nrhs <= 8)  // UMMA with M = 128 needs N to be a multiple of 16 return mrhs_launch_ncol<16>(out, in, A, P, st, what);
    return mrhs_launch_ncol<32>(out, in, A, P, st, what);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {
#ifdef LQCD_MRHS_TRACE
int lqcd_debug_mrhs_trace(long long* host) {
    return cudaMemcpyFromSymbol(host, g_mr_trace, sizeof(g_mr_trace)) == cudaSuccess ? 0 : -3;
}
int lqcd_debug_mrhs_hang(int* host) {
    int n = 0;
    cudaMemcpyFromSymbol(&n, g_mr_hang_n, sizeof(int));
    cudaMemcpyFromSymbol(host, g_mr_hang, sizeof(g_mr_hang));
    int z = 0;
    cudaMemcpyToSymbol(g_mr_hang_n, &z, sizeof(int));
    return n;
}
#endif


int lqcd_coarse_mult_mrhs_f32(float* out, const float* in, const float* A, const int cdims[4], int nvec, int nrhs,
                              unsigned flags, void* stream) {
    const char* what = "lqcd_coarse_mult_mrhs_f32";
    clear_error();
    if (!out || !in || !A || check_dims(cdims) || nvec < 1 || nrhs < 1) {
        set_error("%s: null pointer, non-positive dim, nvec < 1 or nrhs < 1", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(out) || !aligned16(in) || !aligned16(A) || out == in) {
        set_error("%s: pointers must be 16-byte aligned and out must not alias in", what);
        return LQCD_EINVAL;
    }
    if (flags & ~LQCD_DAGGER) {
        set_error("%s: unknown flag bits 0x%x", what, flags);
        return LQCD_EINVAL;
    }
    for (int mu = 0; mu < 4; mu++)
        if (cdims[mu] < 2) {
            set_error("%s: coarse extent < 2", what);
            return LQCD_EINVAL;
        }
    if (volume(cdims) * 9 * 64 * 64 > 0x7fffffffffffLL || volume(cdims) > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    const long long vstride = volume(cdims) * 4 * nvec;  // reals per coarse vector
    if (nvec == 32 && flags == 0 && g_knobs.mrhs_tensor >= 0) {
        for (int k0 = 0; k0 < nrhs; k0 += 16) {  // 16 right-hand sides per launch (TMEM slots and registers)
            const int kn = nrhs - k0 < 16 ? nrhs - k0 : 16;
            int rc = mrhs_tensor_launch(out + k0 * vstride, in + k0 * vstride, A, cdims, kn, vstride,
                                        (cudaStream_t)stream, what);
            if (rc) return rc;
        }
        return LQCD_OK;
    }
    // other sizes, and the dagger form: one single-right-hand-side application per vector
    for (int k = 0; k < nrhs; k++) {
        int rc = lqcd_coarse_mult_f32(out + k * vstride, in + k * vstride, A, cdims, nvec, flags, stream);
        if (rc) return rc;
    }
    return LQCD_OK;
}

int lqcd_coarse_mult_mrhs_f64(double* out, const double* in, const double* A, const int cdims[4], int nvec, int nrhs,
                              unsigned flags, void* stream) {
    const char* what = "lqcd_coarse_mult_mrhs_f64";
    clear_error();
    if (!out || !in || !A || check_dims(cdims) || nvec < 1 || nrhs < 1) {
        set_error("%s: null pointer, non-positive dim, nvec < 1 or nrhs < 1", what);
        return LQCD_EINVAL;
    }
    const long long vstride = volume(cdims) * 4 * nvec;
    for (int k = 0; k < nrhs; k++) {
        int rc = lqcd_coarse_mult_f64(out + k * vstride, in + k * vstride, A, cdims, nvec, flags, stream);
        if (rc) return rc;
    }
    return LQCD_OK;
}
}
