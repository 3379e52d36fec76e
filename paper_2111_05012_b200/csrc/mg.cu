// mg.cu -- row F3 of SURVEY.md section 8(f), second half: one V-cycle of the multigrid preconditioner,
//   "Each step is a Richardson refinement |x> + M_i(|b> - D|x>) -> |x>"
//   (1) M_1 = prolong o coarse solver o restrict   (1a)-(1c)
//   (2) M_2 = SAP with fixed iterations
// and the coarse solver (1b): BiCGStab (listing PAPER.md:71 with M = 1, x_0 = 0) with a FIXED number of iterations
// (reading Q18 of DESIGN.md).
//
// B200 design: the whole V-cycle is enqueued on one stream with no host synchronisation and no host copies (the
// paper's GPU version bounced restriction/prolongation through the host).  The Krylov scalars never
// leave the device: every dot product is a two-stage reduction with a fixed order (per-CTA partial sums, then each
// consumer CTA re-adds the partials in index order), the quotients alpha, omega, beta are recomputed redundantly by
// every CTA of the kernel that needs them, and each vector update is fused with the dot product that follows it.
// A coarse vector at config 5 is 21 MB -- it lives in the 126 MB L2, so the BLAS-1 kernels cost microseconds next to
// the two D_c applications per iteration.
#include "common.cuh"
#include "knobs.h"

namespace lqcd {

constexpr int RED_CTAS = 296;  // 2 x 148 SMs: partial sums per dot product
constexpr int RED_THREADS = 256;

// scalars on the device (complex as 2 reals): rho[2] (double-buffered by iteration parity), alpha, omega
enum { SC_RHO = 0, SC_ALPHA = 4, SC_OMEGA = 6, SC_COUNT = 8 };

template <typename T> struct Cx {
    T re, im;
};
template <typename T> __device__ __forceinline__ Cx<T> cmul(Cx<T> a, Cx<T> b) {
    return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
// num / den, 0 if den == 0 (the iteration then stalls instead of producing NaN; same rule as the oracle)
template <typename T> __device__ __forceinline__ Cx<T> cquot(Cx<T> n, Cx<T> d) {
    const T m = d.re * d.re + d.im * d.im;
    if (m == 0) return {0, 0};
    return {(n.re * d.re + n.im * d.im) / m, (n.im * d.re - n.re * d.im) / m};
}

// Batched form: every kernel below is launched with grid (nred, K): blockIdx.y is the right-hand side, whose vectors
// lie K-fold back to back (2 n reals apart), whose partial sums are part + y * nred * 3 and whose scalars sc + y * 8.
// Sum of the gridDim.x partial triples of this right-hand side in a fixed order, same bits in every thread of every
// CTA.  Must be called by all threads of the CTA.  scratch: 3 values of shared memory.
template <typename T>
__device__ __forceinline__ void sum_partials(T out[3], const T* __restrict__ part, T* scratch, int nred) {
    part += (long long)blockIdx.y * nred * 3;
    if (threadIdx.x < 32) {
        T s[3] = {0, 0, 0};
        for (int i = threadIdx.x; i < nred; i += 32) {
            s[0] += part[3 * i];
            s[1] += part[3 * i + 1];
            s[2] += part[3 * i + 2];
        }
#pragma unroll
        for (int q = 0; q < 3; q++) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s[q] += __shfl_xor_sync(0xffffffffu, s[q], o);
            if (threadIdx.x == 0) scratch[q] = s[q];
        }
    }
    __syncthreads();
    out[0] = scratch[0];
    out[1] = scratch[1];
    out[2] = scratch[2];
    __syncthreads();
}

// CTA reduction of 3 values, thread 0 writes the CTA's partial triple
template <typename T> __device__ __forceinline__ void write_partial(T d[3], T* __restrict__ part, T* red) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < 3; q++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) d[q] += __shfl_xor_sync(0xffffffffu, d[q], o);
        if (lane == 0) red[w * 3 + q] = d[q];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < 3; q++) {
            T s = 0;
            for (int i = 0; i < RED_THREADS / 32; i++) s += red[i * 3 + q];
            part[3 * ((long long)blockIdx.y * gridDim.x + blockIdx.x) + q] = s;
        }
    }
}

// part[cta] = partial of ( <a|b> (complex), <a|a> (real) ); n complex elements
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_cdot(T* __restrict__ part, const T* __restrict__ a,
                                                       const T* __restrict__ b, long long n) {
    __shared__ T red[RED_THREADS / 32 * 3];
    T d[3] = {0, 0, 0};
    a += (long long)blockIdx.y * 2 * n;
    b += (long long)blockIdx.y * 2 * n;
    for (long long k = blockIdx.x * (long long)RED_THREADS + threadIdx.x; k < n; k += (long long)gridDim.x * RED_THREADS) {
        const T ar = a[2 * k], ai = a[2 * k + 1], br = b[2 * k], bi = b[2 * k + 1];
        d[0] = fma(ar, br, d[0]);
        d[0] = fma(ai, bi, d[0]);
        d[1] = fma(ar, bi, d[1]);
        d[1] = fma(-ai, br, d[1]);
        d[2] = fma(ar, ar, d[2]);
        d[2] = fma(ai, ai, d[2]);
    }
    write_partial<T>(d, part, red);
}

// rho[0] = sum of the partials (one CTA)
template <typename T>
__global__ void __launch_bounds__(32) k_set_rho(T* __restrict__ sc, const T* __restrict__ part, int nred) {
    __shared__ T scratch[3];
    T s[3];
    sum_partials<T>(s, part, scratch, nred);
    sc += blockIdx.y * SC_COUNT;
    if (threadIdx.x == 0) {
        sc[SC_RHO] = s[0];
        sc[SC_RHO + 1] = s[1];
    }
}

// alpha = rho / <rt|v>;  s = r - alpha v
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_bicg_s(T* __restrict__ s, const T* __restrict__ r,
                                                         const T* __restrict__ v, const T* __restrict__ part,
                                                         T* __restrict__ sc, int it, long long n) {
    __shared__ T scratch[3];
    T d[3];
    sum_partials<T>(d, part, scratch, gridDim.x);
    sc += blockIdx.y * SC_COUNT;
    s += (long long)blockIdx.y * 2 * n;
    r += (long long)blockIdx.y * 2 * n;
    v += (long long)blockIdx.y * 2 * n;
    const Cx<T> rho = {sc[SC_RHO + 2 * (it & 1)], sc[SC_RHO + 2 * (it & 1) + 1]};
    const Cx<T> alpha = cquot<T>(rho, {d[0], d[1]});
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc[SC_ALPHA] = alpha.re;
        sc[SC_ALPHA + 1] = alpha.im;
    }
    for (long long k = blockIdx.x * (long long)RED_THREADS + threadIdx.x; k < n; k += (long long)gridDim.x * RED_THREADS) {
        const Cx<T> av = cmul<T>(alpha, {v[2 * k], v[2 * k + 1]});
        s[2 * k] = r[2 * k] - av.re;
        s[2 * k + 1] = r[2 * k + 1] - av.im;
    }
}

// omega = <t|s> / <t|t>;  x (+)= alpha p + omega s;  r = s - omega t;  partial of <rt|r>
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_bicg_xr(T* __restrict__ x, T* __restrict__ r, const T* __restrict__ p,
                                                          const T* __restrict__ s, const T* __restrict__ t,
                                                          const T* __restrict__ rt, const T* __restrict__ part_in,
                                                          T* __restrict__ part_out, T* __restrict__ sc, int first,
                                                          long long n) {
    __shared__ T scratch[3];
    __shared__ T red[RED_THREADS / 32 * 3];
    T d[3];
    sum_partials<T>(d, part_in, scratch, gridDim.x);
    sc += blockIdx.y * SC_COUNT;
    {
        const long long bo = (long long)blockIdx.y * 2 * n;
        x += bo; r += bo; p += bo; s += bo; t += bo; rt += bo;
    }
    const Cx<T> omega = cquot<T>({d[0], d[1]}, {d[2], 0});
    const Cx<T> alpha = {sc[SC_ALPHA], sc[SC_ALPHA + 1]};
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc[SC_OMEGA] = omega.re;
        sc[SC_OMEGA + 1] = omega.im;
    }
    T q[3] = {0, 0, 0};
    for (long long k = blockIdx.x * (long long)RED_THREADS + threadIdx.x; k < n; k += (long long)gridDim.x * RED_THREADS) {
        const Cx<T> sk = {s[2 * k], s[2 * k + 1]};
        const Cx<T> ap = cmul<T>(alpha, {p[2 * k], p[2 * k + 1]}), os = cmul<T>(omega, sk);
        const Cx<T> ot = cmul<T>(omega, {t[2 * k], t[2 * k + 1]});
        const T xr = first ? (T)0 : x[2 * k], xi = first ? (T)0 : x[2 * k + 1];
        x[2 * k] = xr + (ap.re + os.re);
        x[2 * k + 1] = xi + (ap.im + os.im);
        const T rr = sk.re - ot.re, ri = sk.im - ot.im;
        r[2 * k] = rr;
        r[2 * k + 1] = ri;
        const T ar = rt[2 * k], ai = rt[2 * k + 1];
        q[0] = fma(ar, rr, q[0]);
        q[0] = fma(ai, ri, q[0]);
        q[1] = fma(ar, ri, q[1]);
        q[1] = fma(-ai, rr, q[1]);
    }
    write_partial<T>(q, part_out, red);
}

// rho' = <rt|r>;  beta = (alpha / omega) (rho' / rho);  p = r + beta (p - omega v);  rho := rho'
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_bicg_p(T* p_out, const T* p_in,  // may alias (p updated in place)
                                                         const T* __restrict__ r, const T* __restrict__ v,
                                                         const T* __restrict__ part, T* __restrict__ sc, int it,
                                                         long long n) {
    __shared__ T scratch[3];
    T d[3];
    sum_partials<T>(d, part, scratch, gridDim.x);
    sc += blockIdx.y * SC_COUNT;
    {
        const long long bo = (long long)blockIdx.y * 2 * n;
        p_out += bo; p_in += bo; r += bo; v += bo;
    }
    const Cx<T> rho = {sc[SC_RHO + 2 * (it & 1)], sc[SC_RHO + 2 * (it & 1) + 1]};
    const Cx<T> alpha = {sc[SC_ALPHA], sc[SC_ALPHA + 1]}, omega = {sc[SC_OMEGA], sc[SC_OMEGA + 1]};
    const Cx<T> rho_new = {d[0], d[1]};
    const Cx<T> beta = cmul<T>(cquot<T>(alpha, omega), cquot<T>(rho_new, rho));
    if (blockIdx.x == 0 && threadIdx.x == 0) {  // the other parity slot: nobody reads it in this kernel
        sc[SC_RHO + 2 * ((it + 1) & 1)] = rho_new.re;
        sc[SC_RHO + 2 * ((it + 1) & 1) + 1] = rho_new.im;
    }
    for (long long k = blockIdx.x * (long long)RED_THREADS + threadIdx.x; k < n; k += (long long)gridDim.x * RED_THREADS) {
        const Cx<T> ov = cmul<T>(omega, {v[2 * k], v[2 * k + 1]});
        const Cx<T> bp = cmul<T>(beta, {p_in[2 * k] - ov.re, p_in[2 * k + 1] - ov.im});
        p_out[2 * k] = r[2 * k] + bp.re;
        p_out[2 * k + 1] = r[2 * k + 1] + bp.im;
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
static size_t align256(size_t b) { return (b + 255) / 256 * 256; }

// partial sums per dot product and right-hand side: 2 x 148 CTAs for one vector, fewer each for a batch
static int red_ctas(int nrhs) {
    int n = 2 * RED_CTAS / nrhs;
    if (n > RED_CTAS) n = RED_CTAS;
    if (n < 8) n = 8;
    return n;
}

template <typename T> struct BicgWs {  // carve-up of the caller's scratch (K vectors back to back each)
    T *v, *s, *t, *p, *r, *part_a, *part_b, *sc, *half;
    static size_t bytes(long long n, int K) {  // (+ the four scratch vectors of the half-storage operator)
        return 5 * align256((size_t)n * 2 * sizeof(T) * K) + 2 * align256((size_t)red_ctas(K) * K * 3 * sizeof(T)) +
               align256((size_t)SC_COUNT * K * sizeof(T)) + align256((size_t)n * 2 * sizeof(T) * 4);
    }
    void carve(void* ws, long long n, int K) {
        char* c = reinterpret_cast<char*>(ws);
        const size_t vb = align256((size_t)n * 2 * sizeof(T) * K), pb = align256((size_t)red_ctas(K) * K * 3 * sizeof(T));
        v = (T*)c; c += vb;
        s = (T*)c; c += vb;
        t = (T*)c; c += vb;
        p = (T*)c; c += vb;
        r = (T*)c; c += vb;
        part_a = (T*)c; c += pb;
        part_b = (T*)c; c += pb;
        sc = (T*)c; c += align256((size_t)SC_COUNT * K * sizeof(T));
        half = (T*)c;
    }
};

// out_k = D_c in_k for K vectors back to back: one pass over A on the tensor cores where that applies (coarse_mrhs.cu)
template <typename T>
static int coarse_mult_any(T* out, const T* in, const T* A, const int cdims[4], int nvec, int K, void* st);
template <typename T>
static int coarse_mult_half_any(T* out, const T* in, const T* Ah, const int cdims[4], int nvec, void* ws, void* st);
template <>
int coarse_mult_half_any<float>(float* out, const float* in, const float* Ah, const int cdims[4], int nvec, void* ws,
                                void* st) {
    return lqcd_coarse_mult_half_f32(out, in, Ah, cdims, nvec, 0, ws, st);
}
template <>
int coarse_mult_half_any<double>(double* out, const double* in, const double* Ah, const int cdims[4], int nvec, void* ws,
                                 void* st) {
    return lqcd_coarse_mult_half_f64(out, in, Ah, cdims, nvec, 0, ws, st);
}
template <>
int coarse_mult_any<float>(float* out, const float* in, const float* A, const int cdims[4], int nvec, int K, void* st) {
    if (K == 1) return lqcd_coarse_mult_f32(out, in, A, cdims, nvec, 0, st);
    return lqcd_coarse_mult_mrhs_f32(out, in, A, cdims, nvec, K, 0, st);
}
template <>
int coarse_mult_any<double>(double* out, const double* in, const double* A, const int cdims[4], int nvec, int K,
                            void* st) {
    if (K == 1) return lqcd_coarse_mult_f64(out, in, A, cdims, nvec, 0, st);
    return lqcd_coarse_mult_mrhs_f64(out, in, A, cdims, nvec, K, 0, st);
}

// x_k = niter BiCGStab iterations for D_c x_k = b_k from x_k = 0 (PAPER.md:71 with M = 1), k = 0 .. K-1: K independent
// recurrences (own scalars each) that share the applications of D_c; r_out may be NULL
// Hooks (sharded solve, lqcd_coarse_bicgstab_hooks): `apply` replaces the application of D_c (A may then be NULL),
// `reduce` sums an array of per-CTA partial sums element by element over the ranks, in place, stream-ordered.
struct BicgHooks {
    lqcd_apply_fn apply;
    lqcd_reduce_fn reduce;
    void* user;
};

template <typename T>
static int bicgstab_call(T* x, T* r_out, const T* b, const T* A, const int cdims[4], int nvec, int K, int niter,
                         void* ws, void* stream, const char* what, const BicgHooks* H = nullptr, bool half = false) {
    // half: A is the half storage of the coarse matrix (lqcd_coarse_mult_half); single right-hand side only
    clear_error();
    if (half && (K != 1 || (H && H->apply))) {
        set_error("%s: half storage takes one right-hand side and no apply hook", what);
        return LQCD_EINVAL;
    }
    if (H && H->apply && !A) A = b;  // never read: the hook applies the operator
    if (!x || !b || !A || !ws || check_dims(cdims) || nvec < 1 || niter < 0 || K < 1 || K > 65535) {
        set_error("%s: null pointer, non-positive dim, nvec < 1, niter < 0 or nrhs outside 1..65535", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(x) || !aligned16(b) || !aligned16(A) || !aligned16(ws) || !aligned16(r_out)) {
        set_error("%s: pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    if (x == b || r_out == b || (r_out && r_out == x)) {
        set_error("%s: x, r_out and b must be distinct", what);
        return LQCD_EINVAL;
    }
    for (int mu = 0; mu < 4; mu++)
        if (cdims[mu] < 2 && !(H && H->apply)) {  // (a rank's part of a sharded lattice may be one site thick)
            set_error("%s: coarse extent < 2", what);
            return LQCD_EINVAL;
        }
    const long long n = volume(cdims) * 2 * nvec;
    const size_t vbytes = (size_t)n * 2 * sizeof(T) * K;
    cudaStream_t st = (cudaStream_t)stream;
    BicgWs<T> W;
    W.carve(ws, n, K);
    int rc;
    const size_t npart = (size_t)red_ctas(K) * K * 3;
    auto Dc = [&](T* out, const T* in) -> int {
        if (H && H->apply) {
            if (H->apply(out, in, stream, H->user)) {
                set_error("%s: the apply hook failed", what);
                return LQCD_ECUDA;
            }
            return LQCD_OK;
        }
        if (half) return coarse_mult_half_any<T>(out, in, A, cdims, nvec, W.half, stream);
        return coarse_mult_any<T>(out, in, A, cdims, nvec, K, stream);
    };
    auto allreduce = [&](T* part) -> int {  // the partial sums of every rank, element by element
        if (H && H->reduce && H->reduce(part, npart, (int)sizeof(T), stream, H->user)) {
            set_error("%s: the reduce hook failed", what);
            return LQCD_ECUDA;
        }
        return LQCD_OK;
    };
    if (niter == 0) {
        if (cudaMemsetAsync(x, 0, vbytes, st) != cudaSuccess) return check_launch(what);
        if (r_out && cudaMemcpyAsync(r_out, b, vbytes, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
            return check_launch(what);
        return LQCD_OK;
    }
    const dim3 grid((unsigned)red_ctas(K), (unsigned)K);
    // r := b, rt := b, p := b, x := 0 -- without copies: the first iteration reads b in their place
    k_cdot<T><<<grid, RED_THREADS, 0, st>>>(W.part_a, b, b, n);
    if ((rc = allreduce(W.part_a))) return rc;
    k_set_rho<T><<<dim3(1, (unsigned)K), 32, 0, st>>>(W.sc, W.part_a, (int)grid.x);
    count_launch(2);
    for (int it = 0; it < niter; it++) {
        const T* p = it == 0 ? b : W.p;
        const T* r = it == 0 ? b : W.r;
        if ((rc = Dc(W.v, p))) return rc;                                                        // v = D_c p
        k_cdot<T><<<grid, RED_THREADS, 0, st>>>(W.part_a, b, W.v, n);                           // <rt|v>
        if ((rc = allreduce(W.part_a))) return rc;
        k_bicg_s<T><<<grid, RED_THREADS, 0, st>>>(W.s, r, W.v, W.part_a, W.sc, it, n);          // s = r - alpha v
        if ((rc = Dc(W.t, W.s))) return rc;                                                      // t = D_c s
        k_cdot<T><<<grid, RED_THREADS, 0, st>>>(W.part_a, W.t, W.s, n);                         // <t|s>, <t|t>
        if ((rc = allreduce(W.part_a))) return rc;
        k_bicg_xr<T><<<grid, RED_THREADS, 0, st>>>(x, W.r, p, W.s, W.t, b, W.part_a, W.part_b, W.sc, it == 0, n);
        count_launch(4);
        if (it + 1 < niter) {  // the last p is never used
            if ((rc = allreduce(W.part_b))) return rc;
            k_bicg_p<T><<<grid, RED_THREADS, 0, st>>>(W.p, p, W.r, W.v, W.part_b, W.sc, it, n);
            count_launch();
        }
    }
    if (r_out && cudaMemcpyAsync(r_out, W.r, vbytes, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return check_launch(what);
    return check_launch(what);
}

template <typename T> struct FineCalls;
template <> struct FineCalls<float> {
    static int restrict_(float* o, const float* i, const float* v, const int* d, const int* b, int nv, void* st) {
        return lqcd_restrict_f32(o, i, v, d, b, nv, st);
    }
    static int prolong_(float* o, const float* i, const float* v, const int* d, const int* b, int nv, void* st) {
        return lqcd_prolong_f32(o, i, v, d, b, nv, st);
    }
    static int restrict_mrhs_(float* o, const float* i, const float* v, const int* d, const int* b, int nv, int K,
                              void* st) {
        return lqcd_restrict_mrhs_f32(o, i, v, d, b, nv, K, st);
    }
    static int prolong_mrhs_(float* o, const float* i, const float* v, const int* d, const int* b, int nv, int K,
                             void* st) {
        return lqcd_prolong_mrhs_f32(o, i, v, d, b, nv, K, st);
    }
    static int sap_(float* x, float* r, const float* b, const float* U, const float* c, float k, const int* d,
                    const int* bc, const int* dom, int K, int ns, int nm, unsigned fl, void* ws, void* st) {
        return lqcd_sap_mrhs_f32(x, r, b, U, c, k, d, bc, dom, K, ns, nm, fl, ws, st);
    }
};
template <> struct FineCalls<double> {
    static int restrict_(double* o, const double* i, const double* v, const int* d, const int* b, int nv, void* st) {
        return lqcd_restrict_f64(o, i, v, d, b, nv, st);
    }
    static int prolong_(double* o, const double* i, const double* v, const int* d, const int* b, int nv, void* st) {
        return lqcd_prolong_f64(o, i, v, d, b, nv, st);
    }
    static int restrict_mrhs_(double* o, const double* i, const double* v, const int* d, const int* b, int nv, int K,
                              void* st) {
        return lqcd_restrict_mrhs_f64(o, i, v, d, b, nv, K, st);
    }
    static int prolong_mrhs_(double* o, const double* i, const double* v, const int* d, const int* b, int nv, int K,
                             void* st) {
        return lqcd_prolong_mrhs_f64(o, i, v, d, b, nv, K, st);
    }
    static int sap_(double* x, double* r, const double* b, const double* U, const double* c, double k, const int* d,
                    const int* bc, const int* dom, int K, int ns, int nm, unsigned fl, void* ws, void* st) {
        return lqcd_sap_mrhs_f64(x, r, b, U, c, k, d, bc, dom, K, ns, nm, fl, ws, st);
    }
};

static size_t mg_ws_bytes(const int dims[4], const int block[4], int nvec, int K, int real_bytes) {
    int cd[4];
    if (check_block(dims, block, nvec, cd)) return 0;
    const long long n = volume(cd) * 2 * nvec;
    const size_t fine = align256((size_t)nchunks(dims) * CH * 24 * real_bytes * K);  // one residual per right-hand side
    const size_t cvec = align256((size_t)n * 2 * real_bytes * K);
    const size_t bicg = real_bytes == 4 ? BicgWs<float>::bytes(n, K) : BicgWs<double>::bytes(n, K);
    return fine + 2 * cvec + bicg + align256(lqcd_mr_workspace_bytes(dims, block, real_bytes));
}

// x = M b: one V-cycle
template <typename T>
static int vcycle_call(T* x, const T* b, const T* U, const T* clover, T kappa, const int dims[4], const int bc[4],
                       const int block[4], int nvec, const T* nullvecs, const T* A, int K, int n_coarse, int n_sap,
                       int n_mr, void* ws, void* stream, const char* what, bool half = false) {
    clear_error();
    int cd[4];
    if (!x || !b || !U || !clover || !nullvecs || !A || !ws || !bc || check_block(dims, block, nvec, cd)) {
        set_error("%s: null pointer or bad dims/block/nvec", what);
        return LQCD_EINVAL;
    }
    if (x == b || n_coarse < 0 || n_sap < 0 || n_mr < 0 || K < 1 || !aligned16(ws)) {
        set_error("%s: x must not alias b; iteration counts must be >= 0; nrhs >= 1; ws 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    for (int mu = 0; mu < 4; mu++)
        if (bc[mu] != 1 && bc[mu] != -1) {
            set_error("%s: bc[%d] = %d not in {+1,-1}", what, mu, bc[mu]);
            return LQCD_EINVAL;
        }
    if (!aligned16(x) || !aligned16(b) || !aligned16(U) || !aligned16(clover) || !aligned16(nullvecs) || !aligned16(A)) {
        set_error("%s: pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    const long long n = volume(cd) * 2 * nvec;
    char* c = reinterpret_cast<char*>(ws);
    T* r = (T*)c;
    c += align256((size_t)nchunks(dims) * CH * 24 * sizeof(T) * K);
    T* bcv = (T*)c;
    c += align256((size_t)n * 2 * sizeof(T) * K);
    T* xcv = (T*)c;
    c += align256((size_t)n * 2 * sizeof(T) * K);
    void* bicg_ws = c;
    c += BicgWs<T>::bytes(n, K);
    void* mr_ws = lqcd_mr_workspace_bytes(dims, block, (int)sizeof(T)) ? (void*)c : nullptr;
    int rc;
    // (1) |x> := M_1 |b>   (|x> = 0, so the first residual is |b> itself); all right-hand sides together
    if (K == 1) {
        if ((rc = FineCalls<T>::restrict_(bcv, b, nullvecs, dims, block, nvec, stream))) return rc;        // (1a) Eq. 5
    } else if ((rc = FineCalls<T>::restrict_mrhs_(bcv, b, nullvecs, dims, block, nvec, K, stream))) {
        return rc;
    }
    if ((rc = bicgstab_call<T>(xcv, nullptr, bcv, A, cd, nvec, K, n_coarse, bicg_ws, stream, what, nullptr, half)))
        return rc;  // (1b)
    if (K == 1) {
        if ((rc = FineCalls<T>::prolong_(x, xcv, nullvecs, dims, block, nvec, stream))) return rc;         // (1c) Eq. 6
    } else if ((rc = FineCalls<T>::prolong_mrhs_(x, xcv, nullvecs, dims, block, nvec, K, stream))) {
        return rc;
    }
    // (2) |x> := |x> + M_2 (|b> - D|x>): SAP started from |x> (its first step is the residual |b> - D|x>)
    return FineCalls<T>::sap_(x, r, b, U, clover, kappa, dims, bc, block, K, n_sap, n_mr,
                              LQCD_SAP_INITIAL_GUESS | LQCD_SAP_NO_FINAL_RESIDUAL, mr_ws, stream);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {

size_t lqcd_coarse_bicgstab_workspace_bytes(const int cdims[4], int nvec, int real_bytes) {
    if (check_dims(cdims) || nvec < 1 || (real_bytes != 4 && real_bytes != 8)) return 0;
    const long long n = volume(cdims) * 2 * nvec;
    return real_bytes == 4 ? BicgWs<float>::bytes(n, 1) : BicgWs<double>::bytes(n, 1);
}
size_t lqcd_coarse_bicgstab_mrhs_workspace_bytes(const int cdims[4], int nvec, int nrhs, int real_bytes) {
    if (check_dims(cdims) || nvec < 1 || nrhs < 1 || (real_bytes != 4 && real_bytes != 8)) return 0;
    const long long n = volume(cdims) * 2 * nvec;
    return real_bytes == 4 ? BicgWs<float>::bytes(n, nrhs) : BicgWs<double>::bytes(n, nrhs);
}
int lqcd_coarse_bicgstab_mrhs_f32(float* x, float* r_out, const float* b, const float* A, const int cdims[4], int nvec,
                                  int nrhs, int niter, void* ws_dev, void* stream) {
    return bicgstab_call<float>(x, r_out, b, A, cdims, nvec, nrhs, niter, ws_dev, stream,
                                "lqcd_coarse_bicgstab_mrhs_f32");
}
int lqcd_coarse_bicgstab_mrhs_f64(double* x, double* r_out, const double* b, const double* A, const int cdims[4],
                                  int nvec, int nrhs, int niter, void* ws_dev, void* stream) {
    return bicgstab_call<double>(x, r_out, b, A, cdims, nvec, nrhs, niter, ws_dev, stream,
                                 "lqcd_coarse_bicgstab_mrhs_f64");
}
int lqcd_coarse_bicgstab_hooks_f32(float* x, float* r_out, const float* b, const int cdims[4], int nvec, int niter,
                                   lqcd_apply_fn apply, lqcd_reduce_fn reduce, void* user, void* ws_dev, void* stream) {
    if (!apply) {
        clear_error();
        set_error("lqcd_coarse_bicgstab_hooks_f32: null apply hook");
        return LQCD_EINVAL;
    }
    const BicgHooks H = {apply, reduce, user};
    return bicgstab_call<float>(x, r_out, b, nullptr, cdims, nvec, 1, niter, ws_dev, stream,
                                "lqcd_coarse_bicgstab_hooks_f32", &H);
}
int lqcd_coarse_bicgstab_hooks_f64(double* x, double* r_out, const double* b, const int cdims[4], int nvec, int niter,
                                   lqcd_apply_fn apply, lqcd_reduce_fn reduce, void* user, void* ws_dev,
                                   void* stream) {
    if (!apply) {
        clear_error();
        set_error("lqcd_coarse_bicgstab_hooks_f64: null apply hook");
        return LQCD_EINVAL;
    }
    const BicgHooks H = {apply, reduce, user};
    return bicgstab_call<double>(x, r_out, b, nullptr, cdims, nvec, 1, niter, ws_dev, stream,
                                 "lqcd_coarse_bicgstab_hooks_f64", &H);
}
int lqcd_coarse_bicgstab_f32(float* x, float* r_out, const float* b, const float* A, const int cdims[4], int nvec,
                             int niter, void* ws_dev, void* stream) {
    return bicgstab_call<float>(x, r_out, b, A, cdims, nvec, 1, niter, ws_dev, stream, "lqcd_coarse_bicgstab_f32");
}
int lqcd_coarse_bicgstab_f64(double* x, double* r_out, const double* b, const double* A, const int cdims[4], int nvec,
                             int niter, void* ws_dev, void* stream) {
    return bicgstab_call<double>(x, r_out, b, A, cdims, nvec, 1, niter, ws_dev, stream, "lqcd_coarse_bicgstab_f64");
}

int lqcd_coarse_bicgstab_half_f32(float* x, float* r_out, const float* b, const float* Ah, const int cdims[4], int nvec,
                                  int niter, void* ws_dev, void* stream) {
    return bicgstab_call<float>(x, r_out, b, Ah, cdims, nvec, 1, niter, ws_dev, stream, "lqcd_coarse_bicgstab_half_f32",
                                nullptr, true);
}
int lqcd_coarse_bicgstab_half_f64(double* x, double* r_out, const double* b, const double* Ah, const int cdims[4],
                                  int nvec, int niter, void* ws_dev, void* stream) {
    return bicgstab_call<double>(x, r_out, b, Ah, cdims, nvec, 1, niter, ws_dev, stream, "lqcd_coarse_bicgstab_half_f64",
                                 nullptr, true);
}

size_t lqcd_mg_workspace_bytes(const int dims[4], const int block[4], int nvec, int real_bytes) {
    if (real_bytes != 4 && real_bytes != 8) return 0;
    return mg_ws_bytes(dims, block, nvec, 1, real_bytes);
}
size_t lqcd_mg_mrhs_workspace_bytes(const int dims[4], const int block[4], int nvec, int nrhs, int real_bytes) {
    if ((real_bytes != 4 && real_bytes != 8) || nrhs < 1) return 0;
    return mg_ws_bytes(dims, block, nvec, nrhs, real_bytes);
}
int lqcd_mg_vcycle_mrhs_f32(float* x, const float* b, const float* U, const float* clover, float kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const float* nullvecs,
                            const float* A, int nrhs, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream) {
    return vcycle_call<float>(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, A, nrhs, n_coarse, n_sap, n_mr,
                              ws_dev, stream, "lqcd_mg_vcycle_mrhs_f32");
}
int lqcd_mg_vcycle_mrhs_f64(double* x, const double* b, const double* U, const double* clover, double kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const double* nullvecs,
                            const double* A, int nrhs, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream) {
    return vcycle_call<double>(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, A, nrhs, n_coarse, n_sap, n_mr,
                               ws_dev, stream, "lqcd_mg_vcycle_mrhs_f64");
}
int lqcd_mg_vcycle_f32(float* x, const float* b, const float* U, const float* clover, float kappa, const int dims[4],
                       const int bc[4], const int block[4], int nvec, const float* nullvecs, const float* A,
                       int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream) {
    return vcycle_call<float>(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, A, 1, n_coarse, n_sap, n_mr,
                              ws_dev, stream, "lqcd_mg_vcycle_f32");
}
int lqcd_mg_vcycle_f64(double* x, const double* b, const double* U, const double* clover, double kappa,
                       const int dims[4], const int bc[4], const int block[4], int nvec, const double* nullvecs,
                       const double* A, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream) {
    return vcycle_call<double>(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, A, 1, n_coarse, n_sap, n_mr,
                               ws_dev, stream, "lqcd_mg_vcycle_f64");
}
int lqcd_mg_vcycle_half_f32(float* x, const float* b, const float* U, const float* clover, float kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const float* nullvecs,
                            const float* Ah, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream) {
    return vcycle_call<float>(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, Ah, 1, n_coarse, n_sap, n_mr,
                              ws_dev, stream, "lqcd_mg_vcycle_half_f32", true);
}
int lqcd_mg_vcycle_half_f64(double* x, const double* b, const double* U, const double* clover, double kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const double* nullvecs,
                            const double* Ah, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream) {
    return vcycle_call<double>(x, b, U, clover, kappa, dims, bc, block, nvec, nullvecs, Ah, 1, n_coarse, n_sap, n_mr,
                               ws_dev, stream, "lqcd_mg_vcycle_half_f64", true);
}
}
