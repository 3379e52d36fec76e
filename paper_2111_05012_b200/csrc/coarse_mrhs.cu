// coarse_mrhs.cu -- row F4 of SURVEY.md section 8(f): the coarse operator applied to K right-hand sides at once,
//   out_k(X) = A_0(X) in_k(X) + sum_mu [ A_{+mu}(X) in_k(X+mu) + A_{-mu}(X) in_k(X-mu) ],   k = 0 .. K-1
// (Eqs. 4, 7; many right-hand sides are "a typical situation").
//
// With K right-hand sides every block A_d(X) is re-used K times: the arithmetic intensity is K flop/byte and the
// operation per coarse site is a dense contraction (N x 9N complex) . (9N x K complex) -- the one place of this path
// where tensor cores belong.  Per block, in REAL arithmetic on the interleaved (re, im)
// storage:  C[r][(k,re)] = sum_j (a_r[2j] b_kj.re - a_r[2j+1] b_kj.im),  C[r][(k,im)] = sum_j (a_r[2j] b_kj.im +
// a_r[2j+1] b_kj.re), i.e. C (64 x 2K) = A (64 x 128, the rows of the block as stored) . B' (128 x 2K) with
// B'[(2j, 2j+1)][(k,re)] = (b.re, -b.im), B'[(2j, 2j+1)][(k,im)] = (b.im, b.re).
//
// tcgen05 (5th-generation tensor cores): kind::tf32 MMAs with fp32 accumulators in TMEM.  TF32 alone (10-bit mantissa)
// would miss the fp32 bar of 2e-6 by two orders of magnitude, so every fp32 operand is split into hi + lo
// (hi = x rounded to the nearest TF32 value; lo = x - hi, exact) and the product is hi.hi + lo.hi + hi.lo (lo.lo,
// 2^-22 relative, is dropped) -- "3xTF32".
//
// Data path of the matrix (DESIGN.md section 6.8 -- why not "split into shared memory"): at the HBM rate an SM takes
// in ~28 B/clk of A; shared memory moves 128 B/clk.  A split written back to shared memory costs 5 bytes of
// shared-memory traffic per byte of A (TMA write, read, lo write, two operand reads by the tensor core) plus the
// traffic of B' -- more than the pipe has.  Here A goes  HBM --TMA--> shared memory (raw fp32, 128B-swizzled, a ring
// of whole blocks, no register ever holds a load across a hand-over) --ld.shared--> registers (split) --tcgen05.st-->
// TENSOR MEMORY, and the MMAs take their A operand from tensor memory (hi in columns 0-63, lo in columns 64-127 of
// the same lane): 2 bytes of shared-memory traffic per byte of A.  Only B' (built from the L2-resident input
// vectors) is a shared-memory operand.
//
// UMMA shape: a block has 64 rows but M = 64 runs at half rate, so the two halves of the contraction index are
// stacked: TMEM lane 64 h + r holds row r, reals 64 h .. 64 h + 63 (h = 0, 1), and B' carries the rows of both halves
// side by side (N index = h * NCOL + (k, re|im)); the accumulator is then block-diagonal -- lanes of half h use the
// columns of half h, the other half of the products is discarded (the tensor pipe has the room: 64 % busy at the
// HBM roofline for K = 16) -- and the two halves are added by the epilogue.
//
// One persistent CTA per SM, warp-specialised (704 threads):
//   warps 0-3    epilogue: tcgen05.ld the accumulators of every block, add them in registers (fp32, round to
//                nearest: the tensor core adds by truncation, so chains are kept to one block), store out_k(X)
//   warps 4-11   converters: raw A block -> (hi, lo) -> tensor memory (warp w owns TMEM lanes 32 (w % 4) ..)
//   warps 12-19  B' builders, two groups of four (one per B' slot, taking the blocks in turn): neighbour's input
//                vectors (L2, prefetched two blocks ahead) -> rows (b.re, -b.im), (b.im, b.re), hi / lo, swizzled
//   warp 20      MMA issuer: the whole warp runs the loop, the lane chosen by elect.sync issues (under `lane == 0`
//                ptxas wraps every tcgen05.mma in an ELECT / BRA.U.ANY loop, ~60 cycles per instruction -- more than
//                these MMAs take to execute).  Allocates / frees tensor memory
//   warp 21      TMA producer: cp.async.bulk.tensor of the next block as soon as a ring slot is free
// Hand-overs: mbarriers where hardware arrives -- raw_full[S] (TMA complete_tx -> converters), done[2] / bdone[2]
// (tcgen05.commit -> converters, epilogue / builders); named barriers (bar.arrive / bar.sync) between warps --
// converters -> TMA producer (ring slot read), converters -> issuer (A slot written), builders -> issuer (B' slot
// written), epilogue -> issuer (accumulators read).  An mbarrier operation queues behind the LDS / STS / tensor-core
// traffic of the shared-memory pipe (300-550 cycles per wait here, even when the phase is complete); a named barrier
// lives in the barrier unit.
// Measured (c5, K = 16, 1965 MHz): 2.54 ms = 0.79 of the measured copy peak; K <= 8: 0.95-1.0.  What bounds K = 16 is
// the shared-memory pipe (per block: 32 KB TMA write + 32 KB LDS + 32 KB B' STS + 48 KB tensor-core operand reads =
// 1125 cycles at 128 B/clk against ~1200-1500 for the block at the HBM rate) -- DESIGN.md section 6.8.
#include <cuda.h>  // CUtensorMap and its enums only: the encoder is fetched through cudaGetDriverEntryPoint

#include "common.cuh"
#include "knobs.h"

namespace lqcd {

constexpr int MR_ROWS = 64;     // N = 2 nvec = 64 rows per block
constexpr int MR_REALS = 128;   // reals per row of a block
constexpr int MR_BLOCKS = 9;    // blocks per coarse site
constexpr int MR_EPI_WARPS = 4, MR_CONV_WARPS = 8, MR_B_WARPS = 8;  // B' builders: two groups of four
constexpr int MR_WARP_CONV = MR_EPI_WARPS, MR_WARP_B = MR_WARP_CONV + MR_CONV_WARPS;
constexpr int MR_B_GROUP = 4;                       // warps per B' builder group (one group per B' slot)
constexpr int MR_B_SLOTS = 2;                       // B' ring: the builders run a block ahead of the slot the MMAs read
constexpr int MR_A_THREADS = (MR_CONV_WARPS + 1) * 32;  // named barrier: converters + issuer
constexpr int MR_B_THREADS = (MR_B_GROUP + 1) * 32;     // named barrier: one builder group + issuer
constexpr int MR_B_AHEAD = 2;                       // blocks the B' builders' L2 prefetch runs ahead
constexpr int MR_WARP_MMA = MR_WARP_B + MR_B_WARPS, MR_WARP_TMA = MR_WARP_MMA + 1;
constexpr int MR_THREADS = (MR_WARP_TMA + 1) * 32;  // 704
constexpr int MR_TMEM_COLS = 512;                   // all of tensor memory
constexpr int MR_A_COLS = 128;                      // one A slot: hi (64 columns) | lo (64 columns), 128 lanes
constexpr unsigned MR_RAW_BYTES = MR_ROWS * MR_REALS * 4;  // 32 KB: one raw block
static_assert(MR_WARP_CONV % 4 == 0 && MR_CONV_WARPS % 4 == 0, "a warp reaches TMEM lanes 32 (warp % 4) .. only");

struct MrhsParams {
    int Lc[4];
    FastDiv dLc[3];  // division by Lc[0..2] as a multiply-high
    int Vc;
    int nrhs;           // K
    int stages;         // raw-block ring slots
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
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// One lane waits for the phase of parity `parity` to complete (try_wait suspends the thread for a bounded time, so
// this is not a hot spin).  A wait that lasts longer than ~2 s of SM clock can only be a protocol error: trap, so that
// the launch fails with an error instead of hanging the device.
__device__ __forceinline__ void mbar_wait_lane(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    long long t0 = 0;
    for (unsigned n = 0;; n++) {
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
        if ((n & 1023u) == 1023u) {
            const long long t = clock64();
            if (t0 == 0) t0 = t;
            else if (t - t0 > 4000000000ll) __trap();
        }
    }
}
// the whole warp waits: lane 0 polls, __syncwarp orders its acquire before the other lanes' later accesses
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    if ((threadIdx.x & 31) == 0) mbar_wait_lane(bar, parity);
    __syncwarp();
}
// one lane of the (converged) warp, chosen by the hardware.  ptxas knows that exactly one thread passes an elect.sync
// predicate and issues the tcgen05 instructions under it directly; under `lane == 0` it wraps every one of them in an
// ELECT / BRA.U.ANY loop (~60 cycles per MMA, measured)
__device__ __forceinline__ bool elect_one() {
    unsigned pred;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "elect.sync _|p, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(pred));
    return pred != 0;
}
// Named (hardware) barriers for the hand-overs between warps: producers bar.arrive and go on, the consumer warp
// bar.syncs.  They live in the barrier unit, not in shared memory: an mbarrier operation queues behind the LDS / STS /
// tensor-core traffic of the shared-memory pipe (300-550 cycles per wait in this kernel, measured, even when the phase
// is already complete), these take ~50.  mbarriers remain where hardware arrives: TMA complete_tx and tcgen05.commit.
__device__ __forceinline__ void nbar_arrive(int id, int threads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ void nbar_sync(int id, int threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
constexpr int MR_BAR_EPI = 1;        // the epilogue's exchange of the two halves (128 threads)
constexpr int MR_BAR_A = 2;          // + A slot: converters -> issuer (A slot in tensor memory written)
constexpr int MR_BAR_ACC = 4;        // + slot: epilogue -> issuer (accumulator slot read)
constexpr int MR_BAR_B = 6;          // + B' slot: builders -> issuer (B' slot written)
constexpr int MR_BAR_RAW = 9;        // + ring slot: converters -> TMA producer (raw block read)
constexpr int MR_MAX_STAGES = 6;     // barrier ids 9 .. 14
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(unsigned long long* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
// D[tmem] (+)= A[tmem] . B[smem]^T, kind::tf32, K = 8 reals per instruction.  A: lane = row, 8 consecutive 32-bit
// columns = the 8 reals; B: K-major shared-memory tile (descriptor); D: lane = row of A, column = row of B.
__device__ __forceinline__ void tc_mma_tf32_ts(unsigned tmem_d, unsigned tmem_a, unsigned long long desc_b, unsigned idesc,
                                               unsigned accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d),
        "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// 2-D tiled TMA load: box (32 reals x 64 rows) of the matrix viewed as [rows][128 reals] into 8 KB of shared memory
// (128-byte swizzle), completion counted in bytes on `bar`; L2 evict-first (A is streamed exactly once).
__device__ __forceinline__ void tma_load_2d(void* dst, const void* tmap, unsigned long long* bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(smem_u32(dst)),
        "l"(reinterpret_cast<unsigned long long>(tmap)), "r"(smem_u32(bar)), "r"(c0), "r"(c1),
        "l"(0x12F0000000000000ull)
        : "memory");
}
// Shared-memory matrix descriptor, K-major, 128-byte swizzle: the tile is stored as rows of 128 bytes (32 reals of
// the contraction index); inside each group of 8 rows (1024 bytes, 1024-byte aligned) the 16-byte chunk c of row r
// sits at chunk position c ^ (r & 7).  SBO = 1024 bytes between 8-row groups; LBO is not used by this mode.
// A k-step of 8 reals advances the start address by 32 bytes inside the 128-byte row.
__device__ __forceinline__ unsigned long long umma_desc_sw128(unsigned saddr) {
    unsigned long long d = 0;
    d |= (unsigned long long)((saddr & 0x3FFFFu) >> 4);
    d |= 1ull << 16;                             // LBO field (ignored for swizzled K-major layouts)
    d |= (unsigned long long)(1024 >> 4) << 32;  // SBO
    d |= 1ull << 46;                             // descriptor version of sm_100
    d |= 2ull << 61;                             // layout type SWIZZLE_128B
    return d;
}
// byte offset of 16-byte chunk kc (0..15) of row r in a [2 K-atoms][rows][128 B] swizzled tile
__device__ __forceinline__ int sw128_off(int rows, int r, int kc) {
    return (kc >> 3) * rows * 128 + r * 128 + (((kc & 7) ^ (r & 7)) << 4);
}
__device__ __forceinline__ void split_tf32(const V16<float>& x, V16<float>& hi, V16<float>& lo) {
#pragma unroll
    for (int q = 0; q < 4; q++) {
        hi.r[q] = __uint_as_float((__float_as_uint(x.r[q]) + 0x1000u) & 0xFFFFE000u);  // nearest TF32
        lo.r[q] = x.r[q] - hi.r[q];
    }
}
// 16 consecutive 32-bit columns of this thread's TMEM lane <- 16 registers / and back
__device__ __forceinline__ void tmem_st16(unsigned taddr, const float* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
        "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
        "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
        "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
        "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15]))
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(unsigned taddr, unsigned* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}

// neighbour of coarse site X for block d (0 diag, 1+2mu forward, 2+2mu backward), periodic.  No dynamic indexing of
// the parameter struct (that would put it in local memory) and no run-time division.
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

// shared memory: [S raw blocks of 32 KB (TMA destination, 1024-byte aligned)] [2 B' slots] [epilogue exchange
// buffer 64 x NCOL floats] [mbarriers].  One B' slot: 2 K-atoms x (4 NCOL rows: hi rows of half 0, of half 1, then the
// lo rows) x 128 B.
__host__ __device__ constexpr unsigned mr_bslot_bytes(int ncol) { return 2u * 4u * (unsigned)ncol * 128u; }
__host__ __device__ constexpr size_t mr_smem_bytes(int ncol, int stages) {
    return (size_t)stages * MR_RAW_BYTES + MR_B_SLOTS * mr_bslot_bytes(ncol) + (size_t)MR_ROWS * ncol * 4 + 16 * 8 + 16;
}

// NCOL = 2 Kp: accumulator columns per half of the contraction index (Kp = 8 or 16 right-hand sides, zero-padded)
template <int NCOL>
__global__ void __launch_bounds__(MR_THREADS, 1)
    k_coarse_mrhs(float* __restrict__ out, const float* __restrict__ in, const __grid_constant__ CUtensorMap tmA,
                  MrhsParams P) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = P.stages;
    constexpr unsigned bslot = mr_bslot_bytes(NCOL);
    constexpr int BROWS = 4 * NCOL;     // rows of a B' slot per K-atom: hi (half 0 | half 1), lo (half 0 | half 1)
    constexpr int ACC_COLS = 4 * NCOL;  // one accumulator slot: main (2 NCOL columns) | small (2 NCOL columns)
    constexpr int KP = NCOL / 2;
    static_assert(2 * MR_A_COLS + 2 * ACC_COLS <= MR_TMEM_COLS, "tensor memory: two A slots and two accumulator slots");
    unsigned char* sB = smem + (size_t)S * MR_RAW_BYTES;
    float* xbuf = reinterpret_cast<float*>(sB + MR_B_SLOTS * bslot);  // [NCOL][64]
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(xbuf + MR_ROWS * NCOL);
    unsigned long long* raw_full = bars;   // [<= 8] TMA complete_tx -> converters: the raw block has landed
    unsigned long long* done = bars + 8;   // [2] tcgen05.commit: the MMAs of the block have completed (A / accumulator slot)
    unsigned long long* bdone = bars + 10; // [3] the same event per B' slot (a parity wait cannot look two phases back)
    unsigned* tmem_slot = reinterpret_cast<unsigned*>(bars + 14);

    if (threadIdx.x == 0) {
        for (int i = 0; i < S; i++) mbar_init(&raw_full[i], 1);  // the producer's arrive.expect_tx
        for (int i = 0; i < 2; i++) mbar_init(&done[i], 1);      // one tcgen05.commit
        for (int i = 0; i < MR_B_SLOTS; i++) mbar_init(&bdone[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // rows of B' beyond the right-hand sides present stay zero for the whole kernel
    for (unsigned i = threadIdx.x; i < MR_B_SLOTS * bslot / 16; i += MR_THREADS)
        reinterpret_cast<float4*>(sB)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    fence_proxy_async();
    if (warp == MR_WARP_MMA) {  // the issuer warp owns the tensor memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "n"(MR_TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem_base = *tmem_slot;
    const unsigned tmem_acc = tmem_base + 2 * MR_A_COLS;
    const int nsites = (P.Vc - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;  // sites of this CTA
    const int G = nsites * MR_BLOCKS;                                                   // blocks of this CTA

    if (warp < MR_EPI_WARPS) {
        // ===== epilogue: TMEM lane 64 h + r = row r of half h; warp q reads lanes 32 q .. 32 q + 31 =====
        const int q = warp, h = q >> 1, row = 32 * (q & 1) + lane;
        int g = 0;
        for (int it = 0; it < nsites; it++) {
            const int X = blockIdx.x + it * gridDim.x;
            float acc[NCOL];
#pragma unroll
            for (int c = 0; c < NCOL; c++) acc[c] = 0.f;
            for (int d = 0; d < MR_BLOCKS; d++, g++) {
                const int a = g & 1;
                mbar_wait(&done[a], (unsigned)(g >> 1) & 1u);
                tc_fence_after();
                // the columns of this half: main at h NCOL, small (lo.hi + hi.lo) at 2 NCOL + h NCOL
                const unsigned taddr = tmem_acc + ((unsigned)(32 * q) << 16) + (unsigned)(a * ACC_COLS + h * NCOL);
#pragma unroll
                for (int c0 = 0; c0 < NCOL; c0 += 16) {  // 16 columns of main and of small per round trip
                    unsigned vm[16], vs[16];
                    tmem_ld16(taddr + c0, vm);
                    tmem_ld16(taddr + 2 * NCOL + c0, vs);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int c = 0; c < 16; c++) acc[c0 + c] += __uint_as_float(vm[c]) + __uint_as_float(vs[c]);
                }
                tc_fence_before();
                nbar_arrive(MR_BAR_ACC + a, (MR_EPI_WARPS + 1) * 32);
            }
            // the two halves of the contraction index meet through shared memory
            if (h == 1) {
#pragma unroll
                for (int c = 0; c < NCOL; c++) xbuf[c * MR_ROWS + row] = acc[c];
            }
            nbar_sync(MR_BAR_EPI, MR_EPI_WARPS * 32);
            if (h == 0) {
#pragma unroll
                for (int k = 0; k < KP; k++)
                    if (k < P.nrhs)
                        *reinterpret_cast<float2*>(out + k * P.vstride + ((long long)X * MR_ROWS + row) * 2) =
                            make_float2(acc[2 * k] + xbuf[(2 * k) * MR_ROWS + row],
                                        acc[2 * k + 1] + xbuf[(2 * k + 1) * MR_ROWS + row]);
            }
            nbar_sync(MR_BAR_EPI, MR_EPI_WARPS * 32);
        }
    } else if (warp < MR_WARP_B) {
        // ===== converters: raw block (shared memory, as TMA wrote it) -> hi | lo -> tensor memory =====
        // thread = one TMEM lane (64 h + r) and 32 of its 64 reals: segment seg = 2 h + ch of the 128-real row.  The
        // TMA box of segment seg is [64 rows][128 B] at seg * 8 KB with chunk c of row r at c ^ (r & 7): 8 consecutive
        // lanes (rows) read 8 different chunk positions -- conflict-free 128-bit loads.
        const int cw = warp - MR_WARP_CONV, q = warp & 3, ch = cw >> 2, h = q >> 1, r = 32 * (q & 1) + lane;
        const unsigned src_off = (unsigned)((2 * h + ch) * 8192 + r * 128);
        const unsigned tlane = tmem_base + ((unsigned)(32 * q) << 16) + (unsigned)(32 * ch);
        int s = 0, ph = 0;
        for (int g = 0; g < G; g++) {
            const int a = g & 1;
            mbar_wait(&raw_full[s], (unsigned)ph);
            mbar_wait(&done[a], ((unsigned)(g >> 1) & 1u) ^ 1u);  // the MMAs of block g - 2 have read A slot a
            tc_fence_after();
            const unsigned char* src = smem + (size_t)s * MR_RAW_BYTES + src_off;
            const unsigned taddr = tlane + (unsigned)(a * MR_A_COLS);
#pragma unroll
            for (int part = 0; part < 2; part++) {
                float hi[16], lo[16];
#pragma unroll
                for (int c = 0; c < 4; c++) {
                    const int chunk = part * 4 + c;
                    const V16<float> x = *reinterpret_cast<const V16<float>*>(src + ((chunk ^ (r & 7)) << 4));
                    V16<float> xh, xl;
                    split_tf32(x, xh, xl);
#pragma unroll
                    for (int e = 0; e < 4; e++) {
                        hi[4 * c + e] = xh.r[e];
                        lo[4 * c + e] = xl.r[e];
                    }
                }
                tmem_st16(taddr + 16 * part, hi);
                tmem_st16(taddr + 64 + 16 * part, lo);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            tc_fence_before();
            nbar_arrive(MR_BAR_RAW + s, (MR_CONV_WARPS + 1) * 32);
            nbar_arrive(MR_BAR_A + a, MR_A_THREADS);
            if (++s == S) {
                s = 0;
                ph ^= 1;
            }
        }
    } else if (warp < MR_WARP_MMA) {
        // ===== B' builders: warp bw takes the right-hand sides k = bw, bw + 4, ...; lane = 16-byte chunk of the 512-byte
        // neighbour vector (2 complex): half h = lane >> 4, chunk kc = lane & 15 of that half's 64 reals =====
        // Two groups of four warps: group m builds B' slot m, i.e. the blocks g = m, m + 2, ... -- a group's loop (wait
        // for the slot, convert, proxy fence, arrive, next loads) takes longer than one block period, two run in turn.
        const int bw = warp - MR_WARP_B, grp = bw / MR_B_GROUP, wq = bw % MR_B_GROUP;
        constexpr int NB = KP / MR_B_GROUP;  // right-hand sides per warp: k = wq, wq + 4, ...
        const int hB = lane >> 4, kc = lane & 15;
        int offB[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) offB[j] = sw128_off(BROWS, hB * NCOL + 2 * (wq + MR_B_GROUP * j), kc);
        V16<float> bq[NB];
        struct Walk {  // (site iteration, block) of the group's blocks g = grp, grp + 2, ...
            int it, d, g;
            __device__ void next() {
                g += 2;
                d += 2;
                if (d >= MR_BLOCKS) {
                    d -= MR_BLOCKS;
                    it++;
                }
            }
        } ld{0, grp, grp}, pf{0, grp, grp};
        // the vectors of a block into L2, MR_B_AHEAD of the group's blocks before they are loaded: a neighbour in a
        // direction the CTA has not visited lately comes from HBM, and the register loads run only one block ahead
        auto prefetch = [&]() {
            if (pf.g < G) {
                const int X = blockIdx.x + pf.it * gridDim.x;
                const float* Bb = in + (long long)coarse_neighbour(P, X, pf.d) * MR_REALS + lane * 4;
#pragma unroll
                for (int j = 0; j < NB; j++)
                    if (wq + MR_B_GROUP * j < P.nrhs && (lane & 7) == 0)
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(Bb + (long long)(wq + MR_B_GROUP * j) * P.vstride));
            }
            pf.next();
        };
        // address of the group's next block's vectors (this lane's 16 bytes of right-hand side 0), computed ahead of
        // the hand-over so that only the load instructions themselves follow it
        auto next_src = [&]() -> const float* {
            const int X = blockIdx.x + ld.it * gridDim.x;
            const float* Bb = in + (long long)coarse_neighbour(P, X, ld.d) * MR_REALS + lane * 4;
            ld.next();
            return Bb;
        };
        auto issue = [&](const float* Bb) {
#pragma unroll
            for (int j = 0; j < NB; j++)
                if (wq + MR_B_GROUP * j < P.nrhs)
                    bq[j] = *reinterpret_cast<const V16<float>*>(Bb + (long long)(wq + MR_B_GROUP * j) * P.vstride);
        };
        for (int i = 0; i < MR_B_AHEAD; i++) prefetch();
        if (grp < G) issue(next_src());
        int sl = grp, ph = 0;  // B' slot g % 3 and the parity of its use count g / 3
        for (int g = grp; g < G; g += 2) {
            prefetch();
            const float* nxt = g + 2 < G ? next_src() : in;  // while the slot is still busy
            mbar_wait(&bdone[sl], (unsigned)ph ^ 1u);  // the MMAs of block g - 3 have read B' slot sl
            unsigned char* dst = sB + (size_t)sl * bslot;
#pragma unroll
            for (int j = 0; j < NB; j++) {
                if (wq + MR_B_GROUP * j < P.nrhs) {
                    V16<float> h, l, t;
                    split_tf32(bq[j], h, l);  // once per element: rounding to nearest is symmetric, hi(-x) = -hi(x)
                    // row (k, re) = (b.re, -b.im), row (k, im) = (b.im, b.re) per complex entry; row 2k+1 = row 2k + 128
                    // bytes with the swizzle bit 0 flipped (2k is even); the lo rows are 2 NCOL rows further
                    t.r[0] = h.r[0]; t.r[1] = -h.r[1]; t.r[2] = h.r[2]; t.r[3] = -h.r[3];
                    *reinterpret_cast<V16<float>*>(dst + offB[j]) = t;
                    t.r[0] = l.r[0]; t.r[1] = -l.r[1]; t.r[2] = l.r[2]; t.r[3] = -l.r[3];
                    *reinterpret_cast<V16<float>*>(dst + offB[j] + 2 * NCOL * 128) = t;
                    t.r[0] = h.r[1]; t.r[1] = h.r[0]; t.r[2] = h.r[3]; t.r[3] = h.r[2];
                    *reinterpret_cast<V16<float>*>(dst + (offB[j] ^ 16) + 128) = t;
                    t.r[0] = l.r[1]; t.r[1] = l.r[0]; t.r[2] = l.r[3]; t.r[3] = l.r[2];
                    *reinterpret_cast<V16<float>*>(dst + (offB[j] ^ 16) + 128 + 2 * NCOL * 128) = t;
                }
            }
            fence_proxy_async();  // generic-proxy stores -> visible to the tensor core's async-proxy reads
            nbar_arrive(MR_BAR_B + sl, MR_B_THREADS);
            if (g + 2 < G) issue(nxt);  // after the hand-over: the fence and the arrive would wait for loads in flight
            sl += 2;  // g + 2
            if (sl >= MR_B_SLOTS) {
                sl -= MR_B_SLOTS;
                ph ^= 1;
            }
        }
    } else if (warp < MR_WARP_TMA) {
        // ===== MMA issuers (one lane each; issuer m = slot m).  Per k-step of 8 reals (of both halves at once):
        //   [main | small] (+)= A_hi . [B'_hi | B'_lo]^T   (M = 128, N = 4 NCOL)
        //   small           += A_lo . B'_hi^T              (M = 128, N = 2 NCOL)
        // instruction descriptor: D fp32, A and B TF32, K-major, N >> 3 at bit 17, M >> 4 at bit 24 =====
        const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((128u >> 4) << 24);
        const unsigned idesc1 = idesc | ((unsigned)((4 * NCOL) >> 3) << 17);
        const unsigned idesc2 = idesc | ((unsigned)((2 * NCOL) >> 3) << 17);
        const unsigned long long dB0 = umma_desc_sw128(smem_u32(sB));
        int sl = 0;  // B' slot g % 3
        for (int g = 0; g < G; g++) {  // the whole warp runs the loop; one elected lane issues
            const int a = g & 1;
            if (g >= 2) nbar_sync(MR_BAR_ACC + a, (MR_EPI_WARPS + 1) * 32);  // the epilogue has read block g - 2
            nbar_sync(MR_BAR_A + a, MR_A_THREADS);
            nbar_sync(MR_BAR_B + sl, MR_B_THREADS);
            tc_fence_after();
            const unsigned ta = tmem_base + (unsigned)(a * MR_A_COLS), td = tmem_acc + (unsigned)(a * ACC_COLS);
            const unsigned long long db = dB0 + (unsigned long long)((sl * bslot) >> 4);
            if (elect_one()) {
#pragma unroll
                for (int ks = 0; ks < 8; ks++) {  // 8 reals = 32 bytes of the 128-byte swizzled row
                    const unsigned long long bo = db + (unsigned long long)(((ks >> 2) * BROWS * 128 + (ks & 3) * 32) >> 4);
                    tc_mma_tf32_ts(td, ta + 8 * ks, bo, idesc1, ks != 0);
                    tc_mma_tf32_ts(td + 2 * NCOL, ta + 64 + 8 * ks, bo, idesc2, 1u);
                }
                tc_commit(&done[a]);
                tc_commit(&bdone[sl]);
            }
            __syncwarp();
            if (++sl == MR_B_SLOTS) sl = 0;
        }
        __syncwarp();
    } else {
        // ===== TMA producer (one lane): four boxes of 32 reals x 64 rows per block, one transaction barrier =====
        int s = 0, ph = 0, it = 0, d = 0;
        for (int g = 0; g < G; g++) {
            if (g >= S) nbar_sync(MR_BAR_RAW + s, (MR_CONV_WARPS + 1) * 32);  // the converters have read block g - S
            if (elect_one()) {
                mbar_arrive_expect_tx(&raw_full[s], MR_RAW_BYTES);
                const int X = blockIdx.x + it * gridDim.x;
                const int row0 = (X * MR_BLOCKS + d) * MR_ROWS;
                unsigned char* dst = smem + (size_t)s * MR_RAW_BYTES;
#pragma unroll
                for (int seg = 0; seg < 4; seg++) tma_load_2d(dst + seg * 8192, &tmA, &raw_full[s], seg * 32, row0);
            }
            __syncwarp();
            if (++d == MR_BLOCKS) {
                d = 0;
                it++;
            }
            if (++s == S) {
                s = 0;
                ph ^= 1;
            }
        }
        __syncwarp();
    }

    tc_fence_before();
    __syncthreads();
    if (warp == MR_WARP_MMA) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(MR_TMEM_COLS)
                     : "memory");
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
// cuTensorMapEncodeTiled through the runtime's driver entry-point query: the library does not link libcuda, so it
// still loads (and answers size queries) on a box without a driver.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            p = nullptr;
        cudaGetLastError();
        fn = (EncodeTiledFn)p;
    }
    return fn;
}
// The coarse matrix as a 2-D tensor [Vc * 9 * 64 rows][128 reals]; box = 32 reals x 64 rows (a quarter of a block),
// written to shared memory with the 128-byte swizzle the converters read it with.
static int make_matrix_tensor_map(CUtensorMap* tm, const float* A, long long Vc, const char* what) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) {
        set_error("%s: cuTensorMapEncodeTiled is not available from this driver", what);
        return LQCD_EUNSUPPORTED;
    }
    const cuuint64_t gdim[2] = {(cuuint64_t)MR_REALS, (cuuint64_t)Vc * MR_BLOCKS * MR_ROWS};
    const cuuint64_t gstride[1] = {(cuuint64_t)MR_REALS * sizeof(float)};
    const cuuint32_t box[2] = {32, (cuuint32_t)MR_ROWS};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(A), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("%s: cuTensorMapEncodeTiled failed (CUresult %d)", what, (int)r);
        return LQCD_ECUDA;
    }
    return LQCD_OK;
}

// one tensor-core launch for up to NCOL / 2 right-hand sides
template <int NCOL>
static int mrhs_launch_ncol(float* out, const float* in, const CUtensorMap& tm, MrhsParams P, cudaStream_t st,
                            const char* what) {
    const size_t fixed = mr_smem_bytes(NCOL, 0);
    int S = (int)(((size_t)max_optin_smem() - fixed) / MR_RAW_BYTES);
    if ((size_t)max_optin_smem() < fixed + 2 * (size_t)MR_RAW_BYTES) {
        set_error("%s: not enough shared memory for the pipeline", what);
        return LQCD_EUNSUPPORTED;
    }
    if (S > MR_MAX_STAGES) S = MR_MAX_STAGES;
    if (g_knobs.mrhs_stages >= 2 && g_knobs.mrhs_stages < S) S = g_knobs.mrhs_stages;
    P.stages = S;
    static unsigned long long attr = 0;
    ensure_dynamic_smem(k_coarse_mrhs<NCOL>, max_optin_smem(), attr);
    const int grid = P.Vc < sm_count() ? P.Vc : sm_count();
    k_coarse_mrhs<NCOL><<<grid, MR_THREADS, mr_smem_bytes(NCOL, S), st>>>(out, in, tm, P);
    count_launch();
    return check_launch(what);
}

static int mrhs_tensor_launch(float* out, const float* in, const CUtensorMap& tm, const int cdims[4], int nrhs,
                              long long vstride, cudaStream_t st, const char* what) {
    MrhsParams P;
    for (int mu = 0; mu < 4; mu++) P.Lc[mu] = cdims[mu];
    for (int mu = 0; mu < 3; mu++) P.dLc[mu].set(cdims[mu]);
    P.Vc = (int)volume(cdims);
    P.nrhs = nrhs;
    P.vstride = vstride;
    P.stages = 0;
    if (nrhs <= 8) return mrhs_launch_ncol<16>(out, in, tm, P, st, what);
    return mrhs_launch_ncol<32>(out, in, tm, P, st, what);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {

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
    if (volume(cdims) * 9 * 64 * 64 > 0x7fffffffffffLL || volume(cdims) * 9 * 64 > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    const long long vstride = volume(cdims) * 4 * nvec;  // reals per coarse vector
    if (nvec == 32 && flags == 0 && g_knobs.mrhs_tensor >= 0) {
        CUtensorMap tm;
        int rc = make_matrix_tensor_map(&tm, A, volume(cdims), what);
        if (rc) return rc;
        for (int k0 = 0; k0 < nrhs; k0 += 16) {  // 16 right-hand sides per launch (tensor-memory columns)
            const int kn = nrhs - k0 < 16 ? nrhs - k0 : 16;
            rc = mrhs_tensor_launch(out + k0 * vstride, in + k0 * vstride, tm, cdims, kn, vstride, (cudaStream_t)stream,
                                    what);
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
