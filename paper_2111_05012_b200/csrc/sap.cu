// sap.cu -- row F3 of SURVEY.md section 8(f): blocked BLAS-1, the inner-domain solver
// M_SAP^(e/o) ~ (D_SAP^(e/o))^-1 ("MINRES algorithm with fixed number of iterations, 6"; reading Q17
// of DESIGN.md: the minimal-residual iteration, run independently in every domain) and the Schwarz alternating
// procedure with fixed iterations (listing PAPER.md:127-131).
//
// B200 design: a 4^4 domain's residual, links and clover term are 168 KB in fp32 -- they
// fit the 227 KB of shared memory of one SM (192 KB with the exchange buffer of the two-threads-per-site split).
// k_mr_domain therefore runs ALL n_mr iterations of one domain inside one CTA: the operator fields are read from
// HBM once per half sweep instead of once per iteration, the blocked dot products are CTA reductions, the blocked
// axpys are register updates, and nothing but the solution goes back to HBM.  Domains that do not fit (fp64 4^4, 8x4^3) take the generic path: D_SAP^(e/o) by k_wilson_clover and
// one fused blocked dotc/dotc/axpy/axpy kernel per iteration.
#include "common.cuh"
#include "fermion.cuh"
#include "knobs.h"
#include "layout.cuh"

namespace lqcd {

template <typename T>
int wilson_clover_call(T* out, const T* in, const T* U, const T* clover, const T* rhs, T kappa, const int dims[4],
                       const int bc[4], const int* domain, unsigned flags, void* stream, const char* what);

// (wilson_clover.cu) out_k = rhs_k - D in_k for nrhs vectors back to back, pairs sharing the links and the clover term
template <typename T>
int wilson_clover_residual_group_call(T* r, const T* x, const T* U, const T* clover, const T* b, T kappa,
                                      const int dims[4], const int bc[4], const int domain[4], unsigned flags,
                                      void* stream, const char* what);
template <typename T>
int wilson_clover_mrhs_call(T* out, const T* in, const T* U, const T* clover, const T* rhs, T kappa, const int dims[4],
                            const int bc[4], int nrhs, unsigned flags, void* stream, const char* what,
                            const int* domain, unsigned group);

struct DomParams {
    int L[4], dom[4], Lc[4], bc[4], multi[4];
    int bv, Vc;
    int parity;    // 0 = all domains, 1 = even, 2 = odd
    int halfgrid;  // 1: the grid enumerates only the domains of the selected group (needs Lc[0] even)
    FastDiv d_Lc[3], d_half, d_dom[3];  // reciprocals of Lc[0..2], Lc[0] / 2 and dom[0..2] for the index decode
    SiteOrder ord; // native position of a site (layout.cuh)
};

// Coarse coordinates of the domain of CTA b; false if that domain is not in the selected group.
__device__ __forceinline__ bool domain_of_cta(const DomParams& P, int b, int Xc[4]) {
    // (divisions by run-time extents as multiply-high with host-computed reciprocals: the decode with hardware-less
    // integer division was 1.6 k issue cycles per CTA of 16 warps)
    int q;
    if (P.halfgrid) {
        const int h = P.Lc[0] >> 1;
        q = P.d_half.div(b);
        const int hx = b - q * h;
        b = q;
        q = P.d_Lc[1].div(b); Xc[1] = b - q * P.Lc[1]; b = q;
        q = P.d_Lc[2].div(b); Xc[2] = b - q * P.Lc[2];
        Xc[3] = q;
        Xc[0] = 2 * hx + ((Xc[1] + Xc[2] + Xc[3] + P.parity - 1) & 1);
        return true;
    }
    q = P.d_Lc[0].div(b); Xc[0] = b - q * P.Lc[0]; b = q;
    q = P.d_Lc[1].div(b); Xc[1] = b - q * P.Lc[1]; b = q;
    q = P.d_Lc[2].div(b); Xc[2] = b - q * P.Lc[2];
    Xc[3] = q;
    return P.parity == 0 || ((Xc[0] + Xc[1] + Xc[2] + Xc[3]) & 1) == P.parity - 1;
}

// local coordinates of local index l (x fastest) and the NATIVE position of that fine site
__device__ __forceinline__ int domain_site(const DomParams& P, const int Xc[4], int l, int lx[4]) {
    int x[4];
#pragma unroll
    for (int mu = 0; mu < 3; mu++) {
        const int q = P.d_dom[mu].div(l);
        lx[mu] = l - q * P.dom[mu];
        l = q;
        x[mu] = Xc[mu] * P.dom[mu] + lx[mu];
    }
    lx[3] = l;
    x[3] = Xc[3] * P.dom[3] + l;
    return P.ord.index(x);
}

// Sum of NRED partial sums per thread over the CTA, same bits in every thread; fixed order (warp tree, then warps in
// index order).  red: shared scratch of (blockDim.x / 32) * NRED values.  Contains one __syncthreads().
template <int NRED, typename T> __device__ __forceinline__ void cta_sum(T v[NRED], T* red) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int q = 0; q < NRED; q++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
        if (lane == 0) red[w * NRED + q] = v[q];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NRED; q++) {
        T s = red[q];
        for (int i = 1; i < nw; i++) s += red[i * NRED + q];
        v[q] = s;
    }
}
// The same for a CTA of NW warps known at compile time, fp32: the second stage reads the NW * NRED partial sums as
// broadcast 128-bit loads (12 LDS.128 instead of 48 LDS.32 at NW = 16, NRED = 3) and adds them in the SAME order as
// cta_sum (warps in index order), so the two give the same bits.  red must be 16-byte aligned.
template <int NRED, int NW> __device__ __forceinline__ void cta_sum_v(float v[NRED], float* red) {
    static_assert((NRED * NW) % 4 == 0, "partials must fill whole float4s");
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < NRED; q++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
        if (lane == 0) red[w * NRED + q] = v[q];
    }
    __syncthreads();
    float t[NRED * NW];
#pragma unroll
    for (int j = 0; j < NRED * NW / 4; j++) {
        const float4 f = reinterpret_cast<const float4*>(red)[j];
        t[4 * j] = f.x, t[4 * j + 1] = f.y, t[4 * j + 2] = f.z, t[4 * j + 3] = f.w;
    }
#pragma unroll
    for (int q = 0; q < NRED; q++) {
        float s = t[q];
#pragma unroll
        for (int i = 1; i < NW; i++) s += t[i * NRED + q];
        v[q] = s;
    }
}

// ---- the shared-memory-resident inner-domain solver ------------------------------------------------------
// Shared-memory image of one domain (bv sites, local index l, x fastest):
//   rho_s [NJ][bv]  vec16            the current residual (every thread reads its neighbours' from here)
//   U_s   [mu][NFULL][bv] vec16      the four forward links of site l, laid out as in HBM:
//   U_t   [mu][bv] float2 (fp32)     18 reals = NFULL full vec16 rows (+ one 8-byte tail in fp32)
//   C_s   [NR][bv]  vec16            the clover term (Hermitian storage, 72 reals)
//   xch_s [NJ/2][2 bvp] vec16        exchange of the partial hop sums between the two threads of a site
// fp32, 4^4: 24 + 72 + 72 + 24 KB = 192 KB of the SM's 227 KB.
//
// TWO threads per site (l, h): with one thread per site the kernel needs 255 registers, i.e. 8 warps per SM, and
// was latency-bound on shared-memory loads (ncu: 2 warps per scheduler, issue slots 41 % busy).  Thread h = 0
// computes the x and y hops, h = 1 the z and t hops (h is warp-uniform: threads l and l + bvp, so the direction
// templates do not diverge); the halves of the two partial sums are exchanged through xch_s, after which thread h
// owns the chirality block chi = h of the site (spin components 2h, 2h+1): its clover block, its 12 reals of rho, z
// and p, its share of the blocked dot products.  128 registers, 16 warps per SM.
template <typename T> __device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global.L2::64B [%0], [%1], 8;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_group() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

template <typename T> struct MrSmem {
    static constexpr int NV = VecOf<T>::NV, NJ = 24 / NV, NR = 72 / NV, NFULL = 18 / NV, TAIL = 18 - NFULL * NV;
    static __host__ __device__ size_t bytes(int bv, int bvp) {
        return (size_t)bv * (NJ + 4 * NFULL + NR) * 16 + (size_t)bv * 4 * TAIL * sizeof(T) +
               (size_t)bvp * 2 * (NJ / 2) * 16 + 16 * 3 * sizeof(T);
    }
};

// One directed hop of D_SAP with every operand in shared memory.
template <int MU, bool FWD, int SGN, typename T>
__device__ __forceinline__ void hop_smem(T acc[24], const V16<T>* __restrict__ rho_s, const V16<T>* __restrict__ U_s,
                                         const T* __restrict__ U_t, int bv, int l_link, int l_nb, T ph) {
    using S = MrSmem<T>;
    constexpr int NV = S::NV;
    T p[24], h[12], u[18], g[12];
#pragma unroll
    for (int j = 0; j < S::NJ; j++) {
        const V16<T> v = rho_s[j * bv + l_nb];
#pragma unroll
        for (int q = 0; q < NV; q++) p[j * NV + q] = v.r[q];
    }
#pragma unroll
    for (int j = 0; j < S::NFULL; j++) {
        const V16<T> v = U_s[(MU * S::NFULL + j) * bv + l_link];
#pragma unroll
        for (int q = 0; q < NV; q++) u[j * NV + q] = v.r[q];
    }
    if (S::TAIL) {
        const float2 v = *reinterpret_cast<const float2*>(U_t + (MU * bv + l_link) * 2);
        u[16] = (T)v.x;
        u[17] = (T)v.y;
    }
    project<MU, SGN, T>(h, p);
    su3_mult<FWD, T, false>(g, u, h);  // scalar arithmetic here: see fermion.cuh
    reconstruct<MU, SGN, T, false>(acc, g, ph);
}

// x (+)= M_SAP^(g) r: one domain per CTA, two threads per site (see above); ACC: accumulate into x.
// BVC: sites per domain as a compile-time constant (a multiple of 32; every shared-memory row offset then folds into
// the immediate field of LDS/STS: -12 % instructions), 0 = run-time P.bv.
template <typename T, bool ACC, int BVC>
__global__ void __launch_bounds__(sizeof(T) == 4 ? 512 : 320, 1)  // fp64 fits at most 151 sites (320 threads)
    k_mr_domain(T* __restrict__ x, const T* __restrict__ r, const T* __restrict__ U, const T* __restrict__ clover,
                T kappa, DomParams P, int niter, int nrhs, long long rstride) {
    using S = MrSmem<T>;
    constexpr int NV = S::NV, NJ = S::NJ, NH = S::NJ / 2, NR = S::NR, NFULL = S::NFULL;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int bv = BVC ? BVC : P.bv, bvp = BVC ? BVC : (int)(blockDim.x >> 1), tid = threadIdx.x;
    V16<T>* rho_s = reinterpret_cast<V16<T>*>(smem_raw);
    V16<T>* U_s = rho_s + NJ * bv;
    V16<T>* C_s = U_s + 4 * NFULL * bv;
    V16<T>* xch_s = C_s + NR * bv;
    T* U_t = reinterpret_cast<T*>(xch_s + NH * 2 * bvp);
    T* red = U_t + 4 * bv * S::TAIL;

    const int h = tid >= bvp;  // warp-uniform (bvp is a multiple of 32)
    const int l0 = tid - h * bvp;
    const bool active = l0 < bv;
    const int l = active ? l0 : 0;
    int Xc[4], lx[4];
    const bool selected = domain_of_cta(P, blockIdx.x, Xc);
    const int s = domain_site(P, Xc, l, lx);
    const int lane = s & 31;
    const long long chunk = s >> 5;
    const long long sp_off = (chunk * NJ * CH + lane) * NV;  // native spinor row 0 of site s
    if (!selected) {  // M^(g) r vanishes outside the group: zero without ACC, x untouched with ACC (reached with ACC
                      // only when Lc[0] is odd and the grid therefore enumerates all domains)
        if (!ACC && active) {
            V16<T> zero;
#pragma unroll
            for (int q = 0; q < NV; q++) zero.r[q] = 0;
#pragma unroll
            for (int k = 0; k < nrhs; k++)
#pragma unroll
                for (int j = 0; j < NH; j++)
                    st16_stream(x + k * rstride + sp_off + (long long)(NH * h + j) * CH * NV, zero);
        }
        return;
    }

    // ---- stage the domain (every operand is read ONCE from HBM): links and clover straight into shared memory
    // (cp.async, 64-byte L2 granularity: a 4-site x-run of a domain is half a 128-byte line)
    if (active) {
#pragma unroll
        for (int m = 0; m < 2; m++) {
            const int mu = 2 * h + m;
            const T* g = U + (chunk * 4 + mu) * (18LL * CH);
#pragma unroll
            for (int j = 0; j < NFULL; j++) cp_async16<T>(&U_s[(mu * NFULL + j) * bv + l], g + (j * CH + lane) * NV);
            if (S::TAIL) cp_async8(U_t + (mu * bv + l) * 2, g + NFULL * NV * CH + lane * 2);
        }
    }
    cp_async_commit();  // group "links": needed by the first hop phase
    if (active) {
        const T* cbase = clover + (chunk * NR * CH + lane) * NV;
#pragma unroll
        for (int j = 0; j < NR / 2; j++) {
            const int row = h * (NR / 2) + j;
            cp_async16<T>(&C_s[row * bv + l], cbase + (long long)row * CH * NV);
        }
    }
    cp_async_commit();  // group "clover": first needed AFTER the hop phase of the first iteration, and only by the
                        // thread that staged it (thread (l, h) stages and reads rows h * NR/2 ... of site l)
    T rho[12];  // my half of the residual; the first right-hand side's is requested before any wait
#pragma unroll
    for (int j = 0; j < NH; j++) {
        const V16<T> v = ld16_g64(r + sp_off + (long long)(NH * h + j) * CH * NV);
#pragma unroll
        for (int q = 0; q < NV; q++) rho[j * NV + q] = v.r[q];
    }
    if (ACC && active) {
#pragma unroll
        for (int j = 0; j < NH; j++)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(x + sp_off + (long long)(NH * h + j) * CH * NV));
    }

    // neighbours inside the domain (local index, wrapped) and hop phases: a hop that leaves the domain is cut
    // (phase 0); in a direction spanned by ONE domain the wrap is the lattice's own and carries bc[mu].
    int nf[4], nb[4];
    T pf[4], pb[4];
    {
        int ls = 1;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const bool wf = lx[mu] == P.dom[mu] - 1, wb = lx[mu] == 0;
            nf[mu] = wf ? l - (P.dom[mu] - 1) * ls : l + ls;
            nb[mu] = wb ? l + (P.dom[mu] - 1) * ls : l - ls;
            const T wrap = P.multi[mu] ? (T)0 : (T)P.bc[mu];
            pf[mu] = wf ? wrap : (T)1;
            pb[mu] = wb ? wrap : (T)1;
            ls *= P.dom[mu];
        }
    }
    const int partner = h ? tid - bvp : tid + bvp;

    // Right-hand sides one after the other on the resident operator: links and clover (86 % of the staged bytes) are
    // read from HBM once for all of them.
    cp_async_wait_group<1>();  // my links have landed (everybody's after the first barrier below)
    for (int krhs = 0; krhs < nrhs; krhs++) {
    const T* rk = r + krhs * rstride;
    T* xk = x + krhs * rstride;
    if (krhs > 0) {
#pragma unroll
        for (int j = 0; j < NH; j++) {
            const V16<T> v = ld16_g64(rk + sp_off + (long long)(NH * h + j) * CH * NV);
#pragma unroll
            for (int q = 0; q < NV; q++) rho[j * NV + q] = v.r[q];
        }
    }
    T z[12];
#pragma unroll
    for (int q = 0; q < 12; q++) z[q] = 0;

    for (int it = 0; it < niter; it++) {
        if (active) {
#pragma unroll
            for (int j = 0; j < NH; j++) {
                V16<T> v;
#pragma unroll
                for (int q = 0; q < NV; q++) v.r[q] = rho[j * NV + q];
                rho_s[(NH * h + j) * bv + l] = v;
            }
        }
        __syncthreads();  // rho_s complete (first pass: also the cp.async data of every thread)
        // my four hops of D_SAP rho; the half of the partial sum that belongs to the other chirality goes to the partner
        T mine[12];
        {
            T acc[24];
#pragma unroll
            for (int q = 0; q < 24; q++) acc[q] = 0;
            if (h == 0) {
                hop_smem<0, true, -1, T>(acc, rho_s, U_s, U_t, bv, l, nf[0], pf[0]);
                hop_smem<0, false, +1, T>(acc, rho_s, U_s, U_t, bv, nb[0], nb[0], pb[0]);
                hop_smem<1, true, -1, T>(acc, rho_s, U_s, U_t, bv, l, nf[1], pf[1]);
                hop_smem<1, false, +1, T>(acc, rho_s, U_s, U_t, bv, nb[1], nb[1], pb[1]);
#pragma unroll
                for (int j = 0; j < NH; j++) {
                    V16<T> v;
#pragma unroll
                    for (int q = 0; q < NV; q++) {
                        v.r[q] = acc[12 + j * NV + q];
                        mine[j * NV + q] = acc[j * NV + q];
                    }
                    xch_s[j * 2 * bvp + tid] = v;
                }
            } else {
                hop_smem<2, true, -1, T>(acc, rho_s, U_s, U_t, bv, l, nf[2], pf[2]);
                hop_smem<2, false, +1, T>(acc, rho_s, U_s, U_t, bv, nb[2], nb[2], pb[2]);
                hop_smem<3, true, -1, T>(acc, rho_s, U_s, U_t, bv, l, nf[3], pf[3]);
                hop_smem<3, false, +1, T>(acc, rho_s, U_s, U_t, bv, nb[3], nb[3], pb[3]);
#pragma unroll
                for (int j = 0; j < NH; j++) {
                    V16<T> v;
#pragma unroll
                    for (int q = 0; q < NV; q++) {
                        v.r[q] = acc[j * NV + q];
                        mine[j * NV + q] = acc[12 + j * NV + q];
                    }
                    xch_s[j * 2 * bvp + tid] = v;
                }
            }
        }
        __syncthreads();
        T p[12];
#pragma unroll
        for (int j = 0; j < NH; j++) {
            const V16<T> v = xch_s[j * 2 * bvp + partner];
#pragma unroll
            for (int q = 0; q < NV; q++) p[j * NV + q] = fma(-kappa, mine[j * NV + q] + v.r[q], rho[j * NV + q]);
        }
        {
            cp_async_wait_group<0>();  // my clover rows (a no-op after the first iteration)
            T cl[36];
#pragma unroll
            for (int j = 0; j < 36 / NV; j++) {
                const V16<T> v = C_s[(h * (36 / NV) + j) * bv + l];
#pragma unroll
                for (int q = 0; q < NV; q++) cl[j * NV + q] = v.r[q];
            }
            herm6_madd<T, false>(p, cl, rho);
        }
        // alpha = <p|rho>_X / <p|p>_X  (blocked dotc)
        T d[3] = {0, 0, 0};
        if (active) {
#pragma unroll
            for (int k = 0; k < 6; k++) {
                d[0] = fma(p[2 * k], rho[2 * k], d[0]);
                d[0] = fma(p[2 * k + 1], rho[2 * k + 1], d[0]);
                d[1] = fma(p[2 * k], rho[2 * k + 1], d[1]);
                d[1] = fma(-p[2 * k + 1], rho[2 * k], d[1]);
                d[2] = fma(p[2 * k], p[2 * k], d[2]);
                d[2] = fma(p[2 * k + 1], p[2 * k + 1], d[2]);
            }
        }
        if constexpr (BVC == 256 && sizeof(T) == 4) cta_sum_v<3, 16>(d, red);
        else cta_sum<3, T>(d, red);
        const T ar = d[2] > 0 ? d[0] / d[2] : (T)0, ai = d[2] > 0 ? d[1] / d[2] : (T)0;
        // z += alpha rho ; rho -= alpha p  (blocked axpy)
#pragma unroll
        for (int k = 0; k < 6; k++) {
            const T rr = rho[2 * k], ri = rho[2 * k + 1];
            z[2 * k] = fma(ar, rr, z[2 * k]);
            z[2 * k] = fma(-ai, ri, z[2 * k]);
            z[2 * k + 1] = fma(ar, ri, z[2 * k + 1]);
            z[2 * k + 1] = fma(ai, rr, z[2 * k + 1]);
            rho[2 * k] = fma(-ar, p[2 * k], rho[2 * k]);
            rho[2 * k] = fma(ai, p[2 * k + 1], rho[2 * k]);
            rho[2 * k + 1] = fma(-ar, p[2 * k + 1], rho[2 * k + 1]);
            rho[2 * k + 1] = fma(-ai, p[2 * k], rho[2 * k + 1]);
        }
        // hazards: rho_s and xch_s are rewritten only after the barrier in cta_sum (all reads done) and, for
        // red, after the two barriers of the next iteration.
    }

    if (active) {
#pragma unroll
        for (int j = 0; j < NH; j++) {
            T* px = xk + sp_off + (long long)(NH * h + j) * CH * NV;
            V16<T> v;
#pragma unroll
            for (int q = 0; q < NV; q++) v.r[q] = z[j * NV + q];
            if (ACC) {
                const V16<T> xo = ld16_g64(px);
#pragma unroll
                for (int q = 0; q < NV; q++) v.r[q] += xo.r[q];
            }
            st16(px, v);
        }
    }
    }  // right-hand sides
}

// ---- the persistent tensor-memory form of the resident solver (fp32, 4^4 domains, tiled site order) ----------
// k_mr_domain is bound by the shared-memory pipe (ncu: LDS wavefronts 68 % of the pipe's peak, short-scoreboard and
// MIO-throttle stalls on top), and 55 % of its LDS traffic are operands that are PRIVATE to a thread and constant over
// the n_mr iterations: the four links of its four hops and its clover block.  Blackwell's tensor memory (256 KB per
// SM, 128 lanes x 512 columns of 32 bits, read by tcgen05.ld on a datapath of its own: measured 870 B/clk/SM against
// the shared-memory pipe's 128) is addressed exactly that way -- lane = thread of a warp quarter, column = register
// index -- so this kernel parks them there: the first iteration of a domain reads them from shared memory and stores
// them with tcgen05.st, the others read them back with tcgen05.ld (shared-memory pipe 68 -> 47 % busy).  No
// tensor-core instruction is issued; the parked bits are the staged fp32 values.
// One CTA per SM walks the domains b = blockIdx.x, blockIdx.x + gridDim.x, ...; tensor memory is allocated once.  From
// the second iteration on the staging buffers are idle, so the NEXT domain is staged under the remaining iterations:
// on the tiled site order a 4^4 domain is 8 whole chunks, i.e. 8 contiguous 9216-byte blocks of links, 8 of clover
// term, requested as 16 bulk copies (cp.async.bulk, completion on two mbarriers: links, clover) instead of 22 cp.async
// instructions in every thread, and the HBM reads that the one-CTA-per-domain kernel exposes at the start of every
// CTA disappear behind the arithmetic.
// Shared memory mirrors the native chunk layouts (local site l = 32 c + lane, c = (z >> 1) + 2 t).
// Columns of a thread in tensor memory (warp w: lanes 32 (w % 4) ..., column block 128 (w / 4)): hop k's link at 20 k
// (18 reals), clover block at 80 (36 reals).
// Preconditions (host): tiled site order, every enumerated domain selected (all domains, or the half grid of one
// group), niter >= 2.  Same arithmetic in the same order as k_mr_domain: bit-identical results (tested).
__device__ __forceinline__ void tm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// tcgen05.ld is asynchronous: its destination registers are valid after tcgen05.wait::ld.  The registers are in/out
// operands of the wait, so no use of them can be scheduled above it.
__device__ __forceinline__ void tm_wait_ld18(float* v) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3]), "+f"(v[4]), "+f"(v[5]), "+f"(v[6]), "+f"(v[7]), "+f"(v[8]),
                   "+f"(v[9]), "+f"(v[10]), "+f"(v[11]), "+f"(v[12]), "+f"(v[13]), "+f"(v[14]), "+f"(v[15]), "+f"(v[16]),
                   "+f"(v[17])::"memory");
}
__device__ __forceinline__ void tm_wait_ld36(float* v) {
    tm_wait_ld18(v);  // (the second half is ordered behind the first wait by the same mechanism)
    asm volatile("" : "+f"(v[18]), "+f"(v[19]), "+f"(v[20]), "+f"(v[21]), "+f"(v[22]), "+f"(v[23]), "+f"(v[24]), "+f"(v[25]),
                 "+f"(v[26]), "+f"(v[27]), "+f"(v[28]), "+f"(v[29]), "+f"(v[30]), "+f"(v[31]), "+f"(v[32]), "+f"(v[33]),
                 "+f"(v[34]), "+f"(v[35])::"memory");
}
__device__ __forceinline__ void tm_st16(unsigned ta, const float* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(ta),
        "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]), "f"(v[8]), "f"(v[9]),
        "f"(v[10]), "f"(v[11]), "f"(v[12]), "f"(v[13]), "f"(v[14]), "f"(v[15])
        : "memory");
}
__device__ __forceinline__ void tm_st4(unsigned ta, const float* v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(ta), "f"(v[0]), "f"(v[1]), "f"(v[2]),
                 "f"(v[3])
                 : "memory");
}
__device__ __forceinline__ void tm_st2(unsigned ta, const float* v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(ta), "f"(v[0]), "f"(v[1]) : "memory");
}
__device__ __forceinline__ void tm_ld16(float* v, unsigned ta) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]), "=f"(v[8]),
          "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15])
        : "r"(ta));
}
__device__ __forceinline__ void tm_ld4(float* v, unsigned ta) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3])
                 : "r"(ta));
}
__device__ __forceinline__ void tm_ld2(float* v, unsigned ta) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "r"(ta));
}
constexpr int TM_COLS = 512, TM_LINK = 20, TM_CLOVER = 80;

// mbarrier + bulk-copy plumbing of the staging
__device__ __forceinline__ unsigned sm_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(sm_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void sbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(sm_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void sbar_wait(unsigned long long* bar, unsigned parity) {
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
            : "r"(sm_u32(bar)), "r"(parity)
            : "memory");
        if (ok) return;
        if ((n & 1023u) == 1023u) {  // a wait of seconds can only be a protocol error: fail the launch, do not hang
            const long long t = clock64();
            if (t0 == 0) t0 = t;
            else if (t - t0 > 4000000000ll) __trap();
        }
    }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(sm_u32(dst)),
                 "l"(src), "r"(bytes), "r"(sm_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

// Shared-memory image of the persistent kernel (offsets in floats): chunk-major copies of the native layouts
struct TmSmem {
    static constexpr int RHO = 0;                    // [6][256] float4: the current residual (as in k_mr_domain)
    static constexpr int LINKS = RHO + 6 * 256 * 4;  // [8 chunks][4 mu][576]: rows 0..3 [lane] float4, tail [lane] float2
    static constexpr int CLOVER = LINKS + 8 * 2304;  // [8][18 rows][32] float4
    static constexpr int RNEXT = CLOVER + 8 * 2304;  // [8][6 rows][32] float4: first residual of the staged domain
    static constexpr int XCH = RNEXT + 8 * 768;      // [3][512] float4
    static constexpr int RED = XCH + 3 * 512 * 4;    // 48 partial sums
    static constexpr int SLOT = RED + 48;            // tensor-memory base address (+ pad)
    static constexpr int BARS = SLOT + 4;            // two mbarriers (16 bytes)
    static constexpr int FLOATS = BARS + 4;
    static constexpr size_t BYTES = (size_t)FLOATS * 4;
};

// The first iteration's hop: operands from shared memory (chunk layout), the link parked in tensor memory on the way.
template <int MU, bool FWD, int SGN>
__device__ __forceinline__ void hop_chunk_park(float acc[24], const V16<float>* __restrict__ rho_s,
                                               const float* __restrict__ links_s, int l_link, int l_nb, float ph,
                                               unsigned ta) {
    float p[24], h[12], u[18], g[12];
#pragma unroll
    for (int j = 0; j < 6; j++) {
        const V16<float> v = rho_s[j * 256 + l_nb];
#pragma unroll
        for (int q = 0; q < 4; q++) p[j * 4 + q] = v.r[q];
    }
    const float* lk = links_s + ((l_link >> 5) * 4 + MU) * 576;
    const int lane = l_link & 31;
#pragma unroll
    for (int j = 0; j < 4; j++) {
        const V16<float> v = *reinterpret_cast<const V16<float>*>(lk + j * 128 + lane * 4);
#pragma unroll
        for (int q = 0; q < 4; q++) u[j * 4 + q] = v.r[q];
    }
    const float2 v = *reinterpret_cast<const float2*>(lk + 512 + lane * 2);
    u[16] = v.x;
    u[17] = v.y;
    tm_st16(ta, u);
    tm_st2(ta + 16, u + 16);
    project<MU, SGN, float>(h, p);
    su3_mult<FWD, float, false>(g, u, h);
    reconstruct<MU, SGN, float, false>(acc, g, ph);
}
// The other iterations' hop: the neighbour spinor from shared memory, the link from tensor memory.  un holds the link
// requested one hop ahead; NEXT: request the following hop's link (at ta_next) before the arithmetic of this one.
template <int MU, bool FWD, int SGN, bool NEXT>
__device__ __forceinline__ void hop_tm(float acc[24], const V16<float>* __restrict__ rho_s, int l_nb, float ph,
                                       float un[18], unsigned ta_next) {
    float p[24], h[12], u[18], g[12];
#pragma unroll
    for (int j = 0; j < 6; j++) {
        const V16<float> v = rho_s[j * 256 + l_nb];
#pragma unroll
        for (int q = 0; q < 4; q++) p[j * 4 + q] = v.r[q];
    }
    tm_wait_ld18(un);
#pragma unroll
    for (int q = 0; q < 18; q++) u[q] = un[q];
    if (NEXT) {
        tm_ld16(un, ta_next);
        tm_ld2(un + 16, ta_next + 16);
    }
    project<MU, SGN, float>(h, p);
    su3_mult<FWD, float, false>(g, u, h);
    reconstruct<MU, SGN, float, false>(acc, g, ph);
}

template <bool ACC>
__global__ void __launch_bounds__(512, 1)
    k_mr_domain_tm(float* __restrict__ x, const float* __restrict__ r, const float* __restrict__ U,
                   const float* __restrict__ clover, float kappa, DomParams P, int niter, int nrhs, long long rstride,
                   int ndom) {
    using T = float;
    constexpr int NV = 4, NH = 3, bv = 256, bvp = 256;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* sm = reinterpret_cast<float*>(smem_raw);
    const int tid = threadIdx.x;
    V16<T>* rho_s = reinterpret_cast<V16<T>*>(sm + TmSmem::RHO);
    const float* links_s = sm + TmSmem::LINKS;
    const float* clover_s = sm + TmSmem::CLOVER;
    const float* rnext_s = sm + TmSmem::RNEXT;
    V16<T>* xch_s = reinterpret_cast<V16<T>*>(sm + TmSmem::XCH);
    T* red = sm + TmSmem::RED;
    unsigned& tm_slot = *reinterpret_cast<unsigned*>(sm + TmSmem::SLOT);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(sm + TmSmem::BARS);  // [0] links + residual, [1] clover

    const int h = tid >= bvp;  // warp-uniform
    const int l = tid - h * bvp;
    const int partner = h ? tid - bvp : tid + bvp;
    const int lc = l >> 5, lane = l & 31;  // my chunk of the domain and my lane in it (= native lane: tiled order)
    const int cstep_z = P.ord.T[2] >> 5, cstep_t = P.ord.T[3] >> 5;  // chunk stride between z pairs / time slices

    // first chunk of domain b
    auto chunk0 = [&](int b) {
        int Xc[4];
        domain_of_cta(P, b, Xc);
        return P.ord.index(Xc[0] * 4, Xc[1] * 4, Xc[2] * 4, Xc[3] * 4) >> 5;
    };
    // staging of domain b.  Links and clover term: 16 bulk copies on two mbarriers, one per warp (lane 0) -- the SM
    // accepts one bulk request per ~80 cycles and its issuer waits for it, so their number is what counts: with the
    // residual and the L2 prefetch of the solution as bulk requests too (32) they were 2.6 k cycles on the critical
    // path of every domain.  Those two are per-thread instead: cp.async of my half of the (first) residual, which only I
    // read, and prefetch.global.L2 of my lines of the solution.
    // (The copies of the other warps may complete before thread 0's expect_tx: the phase cannot, it needs that arrival.)
    auto stage = [&](int b) {
        const long long c0 = chunk0(b);
        {
            const long long so = ((c0 + (lc & 1) * cstep_z + (lc >> 1) * cstep_t) * 6 * CH + lane) * NV;
#pragma unroll
            for (int j = 0; j < NH; j++) {
                cp_async16<T>(sm + TmSmem::RNEXT + lc * 768 + (NH * h + j) * 128 + lane * 4,
                              r + so + (long long)(NH * h + j) * CH * NV);
                if (ACC) asm volatile("prefetch.global.L2 [%0];" ::"l"(x + so + (long long)(NH * h + j) * CH * NV));
            }
            cp_async_commit();
        }
        if (tid == 0) {
            sbar_expect_tx(&bars[0], 8 * 9216);
            sbar_expect_tx(&bars[1], 8 * 9216);
        }
        if ((tid & 31) == 0) {
            // (the buffers were last READ through the generic proxy, before the CTA barrier that precedes this call;
            // the fence orders those accesses before the async-proxy writes of the copies -- cheap insurance)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const int i = tid >> 5, c = i & 7;
            const long long ch = c0 + (c & 1) * cstep_z + (c >> 1) * cstep_t;
            if (i < 8) bulk_g2s(sm + TmSmem::LINKS + c * 2304, U + ch * 2304, 9216, &bars[0]);
            else bulk_g2s(sm + TmSmem::CLOVER + c * 2304, clover + ch * 2304, 9216, &bars[1]);
        }
    };
    if (tid == 0) {
        sbar_init(&bars[0], 1);
        sbar_init(&bars[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sm_u32(&tm_slot)),
                     "n"(TM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tm_fence_before();
    __syncthreads();
    tm_fence_after();
    const unsigned tm_base = tm_slot + ((unsigned)(32 * ((tid >> 5) & 3)) << 16) + (unsigned)((tid >> 7) * 128);
    int b = blockIdx.x;
    if (b < ndom) stage(b);

    // neighbours inside the domain and hop phases: the same for every domain
    int nf[4], nb[4];
    T pf[4], pb[4];
    {
        const int lxm[4] = {l & 3, (l >> 2) & 3, (l >> 4) & 3, l >> 6};
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int ls = 1 << (2 * mu);
            const bool wf = lxm[mu] == 3, wb = lxm[mu] == 0;
            nf[mu] = wf ? l - 3 * ls : l + ls;
            nb[mu] = wb ? l + 3 * ls : l - ls;
            const T wrap = P.multi[mu] ? (T)0 : (T)P.bc[mu];
            pf[mu] = wf ? wrap : (T)1;
            pb[mu] = wb ? wrap : (T)1;
        }
    }
    unsigned phase = 0;
    for (; b < ndom; b += gridDim.x, phase ^= 1u) {
        const long long ch = chunk0(b) + (lc & 1) * cstep_z + (lc >> 1) * cstep_t;  // my native chunk
        const long long sp_off = (ch * 6 * CH + lane) * NV;
        sbar_wait(&bars[0], phase);  // the links of this domain have landed
        cp_async_wait_group<0>();    // ... and my half of its first residual
        T rho[12];
#pragma unroll
        for (int j = 0; j < NH; j++) {
            const V16<T> v = *reinterpret_cast<const V16<T>*>(rnext_s + lc * 768 + (NH * h + j) * 128 + lane * 4);
#pragma unroll
            for (int q = 0; q < NV; q++) rho[j * NV + q] = v.r[q];
        }
        for (int krhs = 0; krhs < nrhs; krhs++) {
            const T* rk = r + krhs * rstride;
            T* xk = x + krhs * rstride;
            if (krhs > 0) {
#pragma unroll
                for (int j = 0; j < NH; j++) {
                    const V16<T> v = ld16_g64(rk + sp_off + (long long)(NH * h + j) * CH * NV);
#pragma unroll
                    for (int q = 0; q < NV; q++) rho[j * NV + q] = v.r[q];
                }
            }
            T z[12];
#pragma unroll
            for (int q = 0; q < 12; q++) z[q] = 0;
            for (int it = 0; it < niter; it++) {
                const bool first = krhs == 0 && it == 0;  // operands still only in shared memory
#pragma unroll
                for (int j = 0; j < NH; j++) {
                    V16<T> v;
#pragma unroll
                    for (int q = 0; q < NV; q++) v.r[q] = rho[j * NV + q];
                    rho_s[(NH * h + j) * bv + l] = v;
                }
                __syncthreads();
                T mine[12];
                {
                    T acc[24];
#pragma unroll
                    for (int q = 0; q < 24; q++) acc[q] = 0;
                    if (first) {
                        if (h == 0) {
                            hop_chunk_park<0, true, -1>(acc, rho_s, links_s, l, nf[0], pf[0], tm_base);
                            hop_chunk_park<0, false, +1>(acc, rho_s, links_s, nb[0], nb[0], pb[0], tm_base + TM_LINK);
                            hop_chunk_park<1, true, -1>(acc, rho_s, links_s, l, nf[1], pf[1], tm_base + 2 * TM_LINK);
                            hop_chunk_park<1, false, +1>(acc, rho_s, links_s, nb[1], nb[1], pb[1], tm_base + 3 * TM_LINK);
                        } else {
                            hop_chunk_park<2, true, -1>(acc, rho_s, links_s, l, nf[2], pf[2], tm_base);
                            hop_chunk_park<2, false, +1>(acc, rho_s, links_s, nb[2], nb[2], pb[2], tm_base + TM_LINK);
                            hop_chunk_park<3, true, -1>(acc, rho_s, links_s, l, nf[3], pf[3], tm_base + 2 * TM_LINK);
                            hop_chunk_park<3, false, +1>(acc, rho_s, links_s, nb[3], nb[3], pb[3], tm_base + 3 * TM_LINK);
                        }
                        tm_wait_st();
                    } else {
                        float un[18];
                        tm_ld16(un, tm_base);
                        tm_ld2(un + 16, tm_base + 16);
                        if (h == 0) {
                            hop_tm<0, true, -1, true>(acc, rho_s, nf[0], pf[0], un, tm_base + TM_LINK);
                            hop_tm<0, false, +1, true>(acc, rho_s, nb[0], pb[0], un, tm_base + 2 * TM_LINK);
                            hop_tm<1, true, -1, true>(acc, rho_s, nf[1], pf[1], un, tm_base + 3 * TM_LINK);
                            hop_tm<1, false, +1, false>(acc, rho_s, nb[1], pb[1], un, 0u);
                        } else {
                            hop_tm<2, true, -1, true>(acc, rho_s, nf[2], pf[2], un, tm_base + TM_LINK);
                            hop_tm<2, false, +1, true>(acc, rho_s, nb[2], pb[2], un, tm_base + 2 * TM_LINK);
                            hop_tm<3, true, -1, true>(acc, rho_s, nf[3], pf[3], un, tm_base + 3 * TM_LINK);
                            hop_tm<3, false, +1, false>(acc, rho_s, nb[3], pb[3], un, 0u);
                        }
                    }
#pragma unroll
                    for (int j = 0; j < NH; j++) {
                        V16<T> v;
#pragma unroll
                        for (int q = 0; q < NV; q++) {
                            v.r[q] = h ? acc[j * NV + q] : acc[12 + j * NV + q];
                            mine[j * NV + q] = h ? acc[12 + j * NV + q] : acc[j * NV + q];
                        }
                        xch_s[j * 2 * bvp + tid] = v;
                    }
                }
                __syncthreads();
                T p[12];
#pragma unroll
                for (int j = 0; j < NH; j++) {
                    const V16<T> v = xch_s[j * 2 * bvp + partner];
#pragma unroll
                    for (int q = 0; q < NV; q++) p[j * NV + q] = fma(-kappa, mine[j * NV + q] + v.r[q], rho[j * NV + q]);
                }
                {
                    T cl[36];
                    if (first) {
                        sbar_wait(&bars[1], phase);  // the clover term of this domain has landed
#pragma unroll
                        for (int j = 0; j < 9; j++) {
                            const V16<T> v =
                                *reinterpret_cast<const V16<T>*>(clover_s + lc * 2304 + (h * 9 + j) * 128 + lane * 4);
#pragma unroll
                            for (int q = 0; q < NV; q++) cl[j * NV + q] = v.r[q];
                        }
                        tm_st16(tm_base + TM_CLOVER, cl);
                        tm_st16(tm_base + TM_CLOVER + 16, cl + 16);
                        tm_st4(tm_base + TM_CLOVER + 32, cl + 32);
                        tm_wait_st();
                    } else {
                        tm_ld16(cl, tm_base + TM_CLOVER);
                        tm_ld16(cl + 16, tm_base + TM_CLOVER + 16);
                        tm_ld4(cl + 32, tm_base + TM_CLOVER + 32);
                        tm_wait_ld36(cl);
                    }
                    herm6_madd<T, false>(p, cl, rho);
                }
                T d[3] = {0, 0, 0};
#pragma unroll
                for (int k = 0; k < 6; k++) {
                    d[0] = fma(p[2 * k], rho[2 * k], d[0]);
                    d[0] = fma(p[2 * k + 1], rho[2 * k + 1], d[0]);
                    d[1] = fma(p[2 * k], rho[2 * k + 1], d[1]);
                    d[1] = fma(-p[2 * k + 1], rho[2 * k], d[1]);
                    d[2] = fma(p[2 * k], p[2 * k], d[2]);
                    d[2] = fma(p[2 * k + 1], p[2 * k + 1], d[2]);
                }
                cta_sum_v<3, 16>(d, red);
                // every thread is past its last read of the staging buffers of this domain: stage the next one
                if (first && b + (int)gridDim.x < ndom) stage(b + gridDim.x);
                const T ar = d[2] > 0 ? d[0] / d[2] : (T)0, ai = d[2] > 0 ? d[1] / d[2] : (T)0;
#pragma unroll
                for (int k = 0; k < 6; k++) {
                    const T rr = rho[2 * k], ri = rho[2 * k + 1];
                    z[2 * k] = fma(ar, rr, z[2 * k]);
                    z[2 * k] = fma(-ai, ri, z[2 * k]);
                    z[2 * k + 1] = fma(ar, ri, z[2 * k + 1]);
                    z[2 * k + 1] = fma(ai, rr, z[2 * k + 1]);
                    rho[2 * k] = fma(-ar, p[2 * k], rho[2 * k]);
                    rho[2 * k] = fma(ai, p[2 * k + 1], rho[2 * k]);
                    rho[2 * k + 1] = fma(-ar, p[2 * k + 1], rho[2 * k + 1]);
                    rho[2 * k + 1] = fma(-ai, p[2 * k], rho[2 * k + 1]);
                }
            }
#pragma unroll
            for (int j = 0; j < NH; j++) {
                T* px = xk + sp_off + (long long)(NH * h + j) * CH * NV;
                V16<T> v;
#pragma unroll
                for (int q = 0; q < NV; q++) v.r[q] = z[j * NV + q];
                if (ACC) {
                    const V16<T> xo = ld16_g64(px);
#pragma unroll
                    for (int q = 0; q < NV; q++) v.r[q] += xo.r[q];
                }
                st16(px, v);
            }
        }  // right-hand sides
    }  // domains
    tm_fence_before();
    __syncthreads();
    if (tid < 32)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm_slot), "n"(TM_COLS) : "memory");
}

// ---- blocked BLAS-1: one CTA per domain, sites strided over the threads ------------------------
// native spinor row j of site s
template <typename T> __device__ __forceinline__ const T* srow(const T* f, int s, int j) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
    return f + (((long long)(s >> 5) * NJ + j) * CH + (s & 31)) * NV;
}
template <typename T> __device__ __forceinline__ T* srow(T* f, int s, int j) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
    return f + (((long long)(s >> 5) * NJ + j) * CH + (s & 31)) * NV;
}

// out[X] = <a|b>_X = sum over the sites of domain X of conj(a) b   (complex, interleaved)
template <typename T>
__global__ void __launch_bounds__(128) k_block_dotc(T* __restrict__ out, const T* __restrict__ a,
                                                     const T* __restrict__ b, DomParams P) {
    __shared__ T red[4 * 2];
    int Xc[4], lx[4];
    domain_of_cta(P, blockIdx.x, Xc);
    T d[2] = {0, 0};
    for (int l = threadIdx.x; l < P.bv; l += blockDim.x) {
        const int s = domain_site(P, Xc, l, lx);
        T va[24], vb[24];
        load_spinor<T>(va, a, s);
        load_spinor<T>(vb, b, s);
#pragma unroll
        for (int k = 0; k < 12; k++) {
            d[0] = fma(va[2 * k], vb[2 * k], d[0]);
            d[0] = fma(va[2 * k + 1], vb[2 * k + 1], d[0]);
            d[1] = fma(va[2 * k], vb[2 * k + 1], d[1]);
            d[1] = fma(-va[2 * k + 1], vb[2 * k], d[1]);
        }
    }
    cta_sum<2, T>(d, red);
    if (threadIdx.x == 0) {
        out[2 * blockIdx.x] = d[0];
        out[2 * blockIdx.x + 1] = d[1];
    }
}

// y(x) += coef[X(x)] a(x)
template <typename T>
__global__ void __launch_bounds__(128) k_block_caxpy(T* __restrict__ y, const T* __restrict__ coef,
                                                      const T* __restrict__ a, DomParams P) {
    int Xc[4], lx[4];
    domain_of_cta(P, blockIdx.x, Xc);
    const T cr = coef[2 * blockIdx.x], ci = coef[2 * blockIdx.x + 1];
    for (int l = threadIdx.x; l < P.bv; l += blockDim.x) {
        const int s = domain_site(P, Xc, l, lx);
        T va[24], vy[24];
        load_spinor<T>(va, a, s);
        load_spinor<T>(vy, y, s);
#pragma unroll
        for (int k = 0; k < 12; k++) {
            vy[2 * k] = fma(cr, va[2 * k], vy[2 * k]);
            vy[2 * k] = fma(-ci, va[2 * k + 1], vy[2 * k]);
            vy[2 * k + 1] = fma(cr, va[2 * k + 1], vy[2 * k + 1]);
            vy[2 * k + 1] = fma(ci, va[2 * k], vy[2 * k + 1]);
        }
        constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
#pragma unroll
        for (int j = 0; j < NJ; j++) {
            V16<T> v;
#pragma unroll
            for (int q = 0; q < NV; q++) v.r[q] = vy[j * NV + q];
            st16(srow(y, s, j), v);
        }
    }
}

// ---- generic inner-domain solver (domains that do not fit in shared memory) ------------------------------------
// rho = P_g r; z = 0 (when z != nullptr)
template <typename T>
__global__ void __launch_bounds__(128) k_mr_init(T* __restrict__ rho, T* __restrict__ z, const T* __restrict__ r,
                                                  DomParams P) {
    int Xc[4], lx[4];
    const bool selected = domain_of_cta(P, blockIdx.x, Xc);
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
    for (int l = threadIdx.x; l < P.bv; l += blockDim.x) {
        const int s = domain_site(P, Xc, l, lx);
#pragma unroll
        for (int j = 0; j < NJ; j++) {
            V16<T> v = ld16(srow(r, s, j));
            V16<T> zero;
#pragma unroll
            for (int q = 0; q < NV; q++) {
                zero.r[q] = 0;
                if (!selected) v.r[q] = 0;
            }
            st16(srow(rho, s, j), v);
            if (z) st16(srow(z, s, j), zero);
        }
    }
}

// one minimal-residual update per domain: alpha = <p|rho>_X / <p|p>_X; z += alpha rho; rho -= alpha p
template <typename T>
__global__ void __launch_bounds__(128) k_mr_update(T* __restrict__ z, T* __restrict__ rho, const T* __restrict__ p,
                                                    DomParams P) {
    __shared__ T red[4 * 3];
    int Xc[4], lx[4];
    if (!domain_of_cta(P, blockIdx.x, Xc)) return;
    T d[3] = {0, 0, 0};
    for (int l = threadIdx.x; l < P.bv; l += blockDim.x) {
        const int s = domain_site(P, Xc, l, lx);
        T vp[24], vr[24];
        load_spinor<T>(vp, p, s);
        load_spinor<T>(vr, rho, s);
#pragma unroll
        for (int k = 0; k < 12; k++) {
            d[0] = fma(vp[2 * k], vr[2 * k], d[0]);
            d[0] = fma(vp[2 * k + 1], vr[2 * k + 1], d[0]);
            d[1] = fma(vp[2 * k], vr[2 * k + 1], d[1]);
            d[1] = fma(-vp[2 * k + 1], vr[2 * k], d[1]);
            d[2] = fma(vp[2 * k], vp[2 * k], d[2]);
            d[2] = fma(vp[2 * k + 1], vp[2 * k + 1], d[2]);
        }
    }
    cta_sum<3, T>(d, red);
    const T ar = d[2] > 0 ? d[0] / d[2] : (T)0, ai = d[2] > 0 ? d[1] / d[2] : (T)0;
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
    for (int l = threadIdx.x; l < P.bv; l += blockDim.x) {
        const int s = domain_site(P, Xc, l, lx);
        T vp[24], vr[24], vz[24];
        load_spinor<T>(vp, p, s);
        load_spinor<T>(vr, rho, s);
        load_spinor<T>(vz, z, s);
#pragma unroll
        for (int k = 0; k < 12; k++) {
            const T rr = vr[2 * k], ri = vr[2 * k + 1];
            vz[2 * k] = fma(ar, rr, vz[2 * k]);
            vz[2 * k] = fma(-ai, ri, vz[2 * k]);
            vz[2 * k + 1] = fma(ar, ri, vz[2 * k + 1]);
            vz[2 * k + 1] = fma(ai, rr, vz[2 * k + 1]);
            vr[2 * k] = fma(-ar, vp[2 * k], vr[2 * k]);
            vr[2 * k] = fma(ai, vp[2 * k + 1], vr[2 * k]);
            vr[2 * k + 1] = fma(-ar, vp[2 * k + 1], vr[2 * k + 1]);
            vr[2 * k + 1] = fma(-ai, vp[2 * k], vr[2 * k + 1]);
        }
#pragma unroll
        for (int j = 0; j < NJ; j++) {
            V16<T> a, b;
#pragma unroll
            for (int q = 0; q < NV; q++) {
                a.r[q] = vz[j * NV + q];
                b.r[q] = vr[j * NV + q];
            }
            st16(srow(z, s, j), a);
            st16(srow(rho, s, j), b);
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
static int dom_setup(DomParams& P, const int dims[4], const int bc[4], const int domain[4], const char* what) {
    if (check_dims(dims) || !domain) {
        set_error("%s: null or non-positive dims/domain", what);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) {
        set_error("%s: volume exceeds 2^31-1 sites", what);
        return LQCD_EUNSUPPORTED;
    }
    P.bv = 1;
    P.Vc = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (domain[mu] < 1 || dims[mu] % domain[mu]) {
            set_error("%s: domain[%d] = %d does not divide dims[%d] = %d", what, mu, domain[mu], mu, dims[mu]);
            return LQCD_EINVAL;
        }
        if (bc && bc[mu] != 1 && bc[mu] != -1) {
            set_error("%s: bc[%d] = %d not in {+1,-1}", what, mu, bc[mu]);
            return LQCD_EINVAL;
        }
        P.L[mu] = dims[mu];
        P.dom[mu] = domain[mu];
        P.Lc[mu] = dims[mu] / domain[mu];
        P.bc[mu] = bc ? bc[mu] : 1;
        P.multi[mu] = P.Lc[mu] > 1;
        P.bv *= domain[mu];
        P.Vc *= P.Lc[mu];
    }
    P.parity = 0;
    P.halfgrid = 0;
    P.ord.set(dims);
    {  // reciprocals of the index decode: exact while (CTA or site index) * divisor < 2^32
        long long dmax = 1;
        for (int mu = 0; mu < 3; mu++) dmax = P.Lc[mu] > dmax ? P.Lc[mu] : dmax;
        if ((long long)P.Vc * dmax >= 0x100000000LL || (long long)P.bv * P.bv >= 0x100000000LL) {
            set_error("%s: lattice too large for the 32-bit index decode", what);
            return LQCD_EUNSUPPORTED;
        }
        for (int mu = 0; mu < 3; mu++) {
            P.d_Lc[mu].set(P.Lc[mu]);
            P.d_dom[mu].set(P.dom[mu]);
        }
        P.d_half.set(P.Lc[0] > 1 ? P.Lc[0] / 2 : 1);
    }
    return LQCD_OK;
}

template <typename T> static size_t mr_smem_bytes(int bv) { return MrSmem<T>::bytes(bv, (bv + 31) / 32 * 32); }

template <typename T> static bool mr_fits_smem(int bv) {
    return g_knobs.sap_fused >= 0 && bv <= 256 && mr_smem_bytes<T>(bv) <= (size_t)max_optin_smem();
}

// z (+)= M_SAP^(g) r.  ws: two native spinors of scratch (rho, p) when the generic path is taken.
template <typename T>
static int mr_domain_call(T* z, const T* r, const T* U, const T* clover, T kappa, const int dims[4], const int bc[4],
                          const int domain[4], unsigned flags, int niter, int K, void* ws, void* stream,
                          const char* what) {
    clear_error();
    if (!z || !r || !U || !clover || !bc || K < 1) {
        set_error("%s: null pointer", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(z) || !aligned16(r) || !aligned16(U) || !aligned16(clover) || !aligned16(ws)) {
        set_error("%s: pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    if (z == r) {
        set_error("%s: z must not alias r", what);
        return LQCD_EINVAL;
    }
    if ((flags & ~(LQCD_DOMAIN_EVEN | LQCD_DOMAIN_ODD | LQCD_ACCUMULATE)) ||
        ((flags & LQCD_DOMAIN_EVEN) && (flags & LQCD_DOMAIN_ODD)) || niter < 0) {
        set_error("%s: bad flags 0x%x or niter %d", what, flags, niter);
        return LQCD_EINVAL;
    }
    DomParams P;
    int rc = dom_setup(P, dims, bc, domain, what);
    if (rc) return rc;
    P.parity = (flags & LQCD_DOMAIN_EVEN) ? 1 : (flags & LQCD_DOMAIN_ODD) ? 2 : 0;
    const bool acc = flags & LQCD_ACCUMULATE;
    cudaStream_t st = (cudaStream_t)stream;

    if (mr_fits_smem<T>(P.bv)) {
        const size_t smem = mr_smem_bytes<T>(P.bv);
        const int threads = 2 * ((P.bv + 31) / 32 * 32);  // two threads per site
        unsigned grid = (unsigned)P.Vc;
        if (acc && P.parity != 0 && P.Lc[0] % 2 == 0) {  // no CTA for the domains of the other group
            P.halfgrid = 1;
            grid = (unsigned)(P.Vc / 2);
        }
        const long long rstride = (long long)nchunks(dims) * CH * 24;  // right-hand sides back to back
        if constexpr (sizeof(T) == 4) {
            if (g_knobs.sap_tmem >= 0 && niter >= 2 && (P.parity == 0 || P.halfgrid) && P.ord.tiled && domain[0] == 4 &&
                domain[1] == 4 && domain[2] == 4 && domain[3] == 4 && TmSmem::BYTES <= (size_t)max_optin_smem()) {
                // persistent form: one CTA per SM walks the domains, links and clover blocks parked in tensor memory
                const int ndom = (int)grid;
                const unsigned g = grid < (unsigned)sm_count() ? grid : (unsigned)sm_count();
                static unsigned long long attr_a = 0, attr_b = 0;
                if (acc) {
                    ensure_dynamic_smem(k_mr_domain_tm<true>, (int)TmSmem::BYTES, attr_a);
                    k_mr_domain_tm<true><<<g, 512, TmSmem::BYTES, st>>>(z, r, U, clover, kappa, P, niter, K, rstride, ndom);
                } else {
                    ensure_dynamic_smem(k_mr_domain_tm<false>, (int)TmSmem::BYTES, attr_b);
                    k_mr_domain_tm<false><<<g, 512, TmSmem::BYTES, st>>>(z, r, U, clover, kappa, P, niter, K, rstride, ndom);
                }
                count_launch();
                return check_launch(what);
            }
        }
#define LAUNCH_MR(ACC, BVC)                                                                                   \
    do {                                                                                                      \
        static unsigned long long attr = 0;                                                                   \
        ensure_dynamic_smem(k_mr_domain<T, ACC, BVC>, max_optin_smem(), attr);                                \
        k_mr_domain<T, ACC, BVC><<<grid, threads, smem, st>>>(z, r, U, clover, kappa, P, niter, K, rstride);   \
    } while (0)
        if (sizeof(T) == 4 && P.bv == 256) {  // the paper's typical 4^4 domain
            if (acc) LAUNCH_MR(true, (sizeof(T) == 4 ? 256 : 0));
            else LAUNCH_MR(false, (sizeof(T) == 4 ? 256 : 0));
        } else {
            if (acc) LAUNCH_MR(true, 0);
            else LAUNCH_MR(false, 0);
        }
#undef LAUNCH_MR
        count_launch();
        return check_launch(what);
    }

    // generic path
    if (!ws) {
        set_error("%s: this domain size needs the workspace of lqcd_mr_workspace_bytes()", what);
        return LQCD_EINVAL;
    }
    const size_t nreal = (size_t)nchunks(dims) * CH * 24;
    T* rho = reinterpret_cast<T*>(ws);
    T* p = rho + nreal;
    const unsigned ddflags = flags & (LQCD_DOMAIN_EVEN | LQCD_DOMAIN_ODD);
    for (int k = 0; k < K; k++) {  // one right-hand side after the other
        T* zk = z + k * nreal;
        k_mr_init<T><<<(unsigned)P.Vc, 128, 0, st>>>(rho, acc ? nullptr : zk, r + k * nreal, P);
        count_launch();
        for (int it = 0; it < niter; it++) {
            rc = wilson_clover_call<T>(p, rho, U, clover, nullptr, kappa, dims, bc, domain, ddflags, stream, what);
            if (rc) return rc;
            k_mr_update<T><<<(unsigned)P.Vc, 128, 0, st>>>(zk, rho, p, P);
            count_launch();
        }
    }
    return check_launch(what);
}

// SAP with fixed iterations.  x: solution; r: scratch, receives the residual; b: right-hand side.
template <typename T>
static int sap_call(T* x, T* r, const T* b, const T* U, const T* clover, T kappa, const int dims[4], const int bc[4],
                    const int domain[4], int n_sap, int n_mr, int K, unsigned flags, void* ws, void* stream,
                    const char* what) {
    clear_error();
    if (!x || !r || !b || !U || !clover || !bc || check_dims(dims) || !domain || K < 1) {
        set_error("%s: null pointer or non-positive dim", what);
        return LQCD_EINVAL;
    }
    if (x == r || x == b || r == b) {
        set_error("%s: x, r and b must be distinct", what);
        return LQCD_EINVAL;
    }
    if ((flags & ~(LQCD_SAP_INITIAL_GUESS | LQCD_SAP_NO_FINAL_RESIDUAL)) || n_sap < 0 || n_mr < 0) {
        set_error("%s: bad flags 0x%x, n_sap %d or n_mr %d", what, flags, n_sap, n_mr);
        return LQCD_EINVAL;
    }
    {  // validate everything before the first enqueue ("nothing enqueued on error")
        DomParams P;
        int rc = dom_setup(P, dims, bc, domain, what);
        if (rc) return rc;
        if (!aligned16(x) || !aligned16(r) || !aligned16(b) || !aligned16(U) || !aligned16(clover) || !aligned16(ws)) {
            set_error("%s: pointers must be 16-byte aligned", what);
            return LQCD_EINVAL;
        }
        if (!mr_fits_smem<T>(P.bv) && !ws) {
            set_error("%s: this domain size needs the workspace of lqcd_mr_workspace_bytes()", what);
            return LQCD_EINVAL;
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    const long long nreal = (long long)nchunks(dims) * CH * 24;  // K vectors back to back
    const size_t bytes = (size_t)nreal * sizeof(T) * K;
    int rc;
    // |r_k> := |b_k> - D|x_k>; right-hand sides in pairs (links, clover read once).  Between two half sweeps only
    // the group solved NEXT reads the residual, so it is computed on that group's domains alone (`next` =
    // LQCD_DOMAIN_EVEN / ODD; about 0.6 of the traffic of the full pass); next = 0: all sites.
    auto residual = [&](unsigned next) -> int {
        if (g_knobs.sap_group_residual < 0) next = 0;
        if (K == 1 && next)
            return wilson_clover_residual_group_call<T>(r, x, U, clover, b, kappa, dims, bc, domain, next, stream,
                                                        what);
        if (K == 1) return wilson_clover_call<T>(r, x, U, clover, b, kappa, dims, bc, nullptr, 0, stream, what);
        return wilson_clover_mrhs_call<T>(r, x, U, clover, b, kappa, dims, bc, K, 0, stream, what, domain, next);
    };
    const T* res = r;
    if (flags & LQCD_SAP_INITIAL_GUESS) {
        if ((rc = residual(n_sap > 0 ? LQCD_DOMAIN_EVEN : 0u))) return rc;
    } else {  // |x> := 0, |r> := |b>: the first half sweep reads b itself
        if (cudaMemsetAsync(x, 0, bytes, st) != cudaSuccess) return check_launch(what);
        res = b;
        if (n_sap == 0 && !(flags & LQCD_SAP_NO_FINAL_RESIDUAL))
            if (cudaMemcpyAsync(r, b, bytes, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return check_launch(what);
    }
    for (int i = 0; i < n_sap; i++)
        for (int g = 0; g < 2; g++) {
            // |x_k> := |x_k> + M_SAP^(e/o)|r_k>, all k on the resident operator of each domain
            rc = mr_domain_call<T>(x, res, U, clover, kappa, dims, bc, domain,
                                   (g == 0 ? LQCD_DOMAIN_EVEN : LQCD_DOMAIN_ODD) | LQCD_ACCUMULATE, n_mr, K, ws, stream,
                                   what);
            if (rc) return rc;
            const bool last = (i == n_sap - 1 && g == 1);
            if (last && (flags & LQCD_SAP_NO_FINAL_RESIDUAL)) break;
            if ((rc = residual(last ? 0u : g == 0 ? LQCD_DOMAIN_ODD : LQCD_DOMAIN_EVEN))) return rc;
            res = r;
        }
    return LQCD_OK;
}

template <typename T>
static int block_blas_call(int which, T* out, const T* a, const T* b, const int dims[4], const int domain[4],
                           void* stream, const char* what) {
    clear_error();
    if (!out || !a || !b) {
        set_error("%s: null pointer", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(a) || !aligned16(b) || (which == 1 && !aligned16(out))) {
        set_error("%s: spinor pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    DomParams P;
    int rc = dom_setup(P, dims, nullptr, domain, what);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (which == 0) k_block_dotc<T><<<(unsigned)P.Vc, 128, 0, st>>>(out, a, b, P);
    else k_block_caxpy<T><<<(unsigned)P.Vc, 128, 0, st>>>(out, a, b, P);
    count_launch();
    return check_launch(what);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {

size_t lqcd_mr_workspace_bytes(const int dims[4], const int domain[4], int real_bytes) {
    DomParams P;
    if (dom_setup(P, dims, nullptr, domain, "lqcd_mr_workspace_bytes")) return 0;
    if (real_bytes != 4 && real_bytes != 8) return 0;
    const bool fits = real_bytes == 4 ? mr_fits_smem<float>(P.bv) : mr_fits_smem<double>(P.bv);
    return fits ? 0 : 2 * (size_t)nchunks(dims) * CH * 24 * (size_t)real_bytes;
}

int lqcd_block_dotc_f32(float* out, const float* a, const float* b, const int dims[4], const int domain[4],
                        void* stream) {
    return block_blas_call<float>(0, out, a, b, dims, domain, stream, "lqcd_block_dotc_f32");
}
int lqcd_block_dotc_f64(double* out, const double* a, const double* b, const int dims[4], const int domain[4],
                        void* stream) {
    return block_blas_call<double>(0, out, a, b, dims, domain, stream, "lqcd_block_dotc_f64");
}
int lqcd_block_caxpy_f32(float* y, const float* coef, const float* a, const int dims[4], const int domain[4],
                         void* stream) {
    return block_blas_call<float>(1, y, coef, a, dims, domain, stream, "lqcd_block_caxpy_f32");
}
int lqcd_block_caxpy_f64(double* y, const double* coef, const double* a, const int dims[4], const int domain[4],
                         void* stream) {
    return block_blas_call<double>(1, y, coef, a, dims, domain, stream, "lqcd_block_caxpy_f64");
}

int lqcd_mr_domain_solve_f32(float* z, const float* r, const float* U, const float* clover, float kappa,
                             const int dims[4], const int bc[4], const int domain[4], unsigned flags, int niter,
                             void* ws_dev, void* stream) {
    return mr_domain_call<float>(z, r, U, clover, kappa, dims, bc, domain, flags, niter, 1, ws_dev, stream,
                                 "lqcd_mr_domain_solve_f32");
}
int lqcd_mr_domain_solve_f64(double* z, const double* r, const double* U, const double* clover, double kappa,
                             const int dims[4], const int bc[4], const int domain[4], unsigned flags, int niter,
                             void* ws_dev, void* stream) {
    return mr_domain_call<double>(z, r, U, clover, kappa, dims, bc, domain, flags, niter, 1, ws_dev, stream,
                                  "lqcd_mr_domain_solve_f64");
}

int lqcd_sap_f32(float* x, float* r, const float* b, const float* U, const float* clover, float kappa,
                 const int dims[4], const int bc[4], const int domain[4], int n_sap, int n_mr, unsigned flags,
                 void* ws_dev, void* stream) {
    return sap_call<float>(x, r, b, U, clover, kappa, dims, bc, domain, n_sap, n_mr, 1, flags, ws_dev, stream,
                           "lqcd_sap_f32");
}
int lqcd_sap_f64(double* x, double* r, const double* b, const double* U, const double* clover, double kappa,
                 const int dims[4], const int bc[4], const int domain[4], int n_sap, int n_mr, unsigned flags,
                 void* ws_dev, void* stream) {
    return sap_call<double>(x, r, b, U, clover, kappa, dims, bc, domain, n_sap, n_mr, 1, flags, ws_dev, stream,
                            "lqcd_sap_f64");
}
int lqcd_sap_mrhs_f32(float* x, float* r, const float* b, const float* U, const float* clover, float kappa,
                      const int dims[4], const int bc[4], const int domain[4], int nrhs, int n_sap, int n_mr,
                      unsigned flags, void* ws_dev, void* stream) {
    return sap_call<float>(x, r, b, U, clover, kappa, dims, bc, domain, n_sap, n_mr, nrhs, flags, ws_dev, stream,
                           "lqcd_sap_mrhs_f32");
}
int lqcd_sap_mrhs_f64(double* x, double* r, const double* b, const double* U, const double* clover, double kappa,
                      const int dims[4], const int bc[4], const int domain[4], int nrhs, int n_sap, int n_mr,
                      unsigned flags, void* ws_dev, void* stream) {
    return sap_call<double>(x, r, b, U, clover, kappa, dims, bc, domain, n_sap, n_mr, nrhs, flags, ws_dev, stream,
                            "lqcd_sap_mrhs_f64");
}
}
