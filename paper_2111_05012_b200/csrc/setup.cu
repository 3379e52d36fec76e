// setup.cu -- F2 of SURVEY.md 8(f): the set-up steps of the multigrid hierarchy on the device, so that the operator
// fields the hot path consumes never have to be built on the host:
//   * lqcd_clover_from_links   F(x) from the plaquette leaves of the links ("12x12 Hermitian matrix made
//                              of link variables"; formula = DESIGN.md reading Q1), written in the native clover layout;
//   * lqcd_orthonormalize_blocks   block- and chirality-wise orthonormalisation of the null vectors;
//   * lqcd_galerkin_coarse     the nine dense blocks <I|D|J> of the coarse operator (Eq. 7).
// These run once per gauge configuration (the paper's set-up takes 5.6-893 s, Table 1); they are written for clarity and
// reasonable speed, not to a roofline.  Parity against the oracle's O3 / O4 / O6 is tested like the hot path.
#include "aggregate.cuh"
#include "common.cuh"
#include "fermion.cuh"
#include "layout.cuh"

namespace lqcd {

// ------------------------------------------------------------------------------------------------------------
// 3x3 complex matrices in registers: m[2*(3a+b)+reim]
// ------------------------------------------------------------------------------------------------------------
template <typename T> struct M3 {
    T m[18];
};

template <typename T> __device__ __forceinline__ M3<T> load_m3(const T* __restrict__ U, int s, int mu) {
    M3<T> r;
#pragma unroll
    for (int k = 0; k < 18; k++) r.m[k] = U[gauge18_off<T>(s, mu, k)];
    return r;
}

// C = op(A) op(B), op = identity or Hermitian conjugate
template <bool ADJA, bool ADJB, typename T> __device__ __forceinline__ M3<T> mul(const M3<T>& A, const M3<T>& B) {
    M3<T> C;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            T cr = 0, ci = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const T ar = ADJA ? A.m[2 * (3 * k + i)] : A.m[2 * (3 * i + k)];
                const T ai = ADJA ? -A.m[2 * (3 * k + i) + 1] : A.m[2 * (3 * i + k) + 1];
                const T br = ADJB ? B.m[2 * (3 * j + k)] : B.m[2 * (3 * k + j)];
                const T bi = ADJB ? -B.m[2 * (3 * j + k) + 1] : B.m[2 * (3 * k + j) + 1];
                cr = fma(ar, br, cr);
                cr = fma(-ai, bi, cr);
                ci = fma(ar, bi, ci);
                ci = fma(ai, br, ci);
            }
            C.m[2 * (3 * i + j)] = cr;
            C.m[2 * (3 * i + j) + 1] = ci;
        }
    return C;
}

struct CloverParams {
    int L[4];
    int V;
    SiteOrder ord;  // native position of a site (layout.cuh)
};

__device__ __forceinline__ int shifted(const CloverParams& P, const int x[4], int mu, int dmu, int nu, int dnu) {
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] += dmu;
    if (y[mu] >= P.L[mu]) y[mu] -= P.L[mu];
    if (y[mu] < 0) y[mu] += P.L[mu];
    y[nu] += dnu;
    if (y[nu] >= P.L[nu]) y[nu] -= P.L[nu];
    if (y[nu] < 0) y[nu] += P.L[nu];
    return P.ord.index(y);  // native position
}

// Hermitian 3x3 F_{mu nu}(x) = (Q - Q^dag) / (8 i), Q = sum of the four plaquette leaves in the mu-nu plane that
// start and end at x, all with the same orientation (links periodic).  f[2*(3a+b)+reim].
template <typename T>
__device__ void field_strength(T f[18], const T* __restrict__ U, const CloverParams& P, const int x[4], int s, int mu,
                               int nu) {
    T q[18];
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] = 0;
    M3<T> a, b, c, d, t;
    // leaf 1: U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)
    a = load_m3(U, s, mu);
    b = load_m3(U, shifted(P, x, mu, +1, nu, 0), nu);
    c = load_m3(U, shifted(P, x, mu, 0, nu, +1), mu);
    d = load_m3(U, s, nu);
    t = mul<false, true>(mul<false, true>(mul<false, false>(a, b), c), d);
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] += t.m[k];
    // leaf 2: U_nu(x) U_mu^dag(x-mu+nu) U_nu^dag(x-mu) U_mu(x-mu)
    a = load_m3(U, s, nu);
    b = load_m3(U, shifted(P, x, mu, -1, nu, +1), mu);
    c = load_m3(U, shifted(P, x, mu, -1, nu, 0), nu);
    d = load_m3(U, shifted(P, x, mu, -1, nu, 0), mu);
    t = mul<false, false>(mul<false, true>(mul<false, true>(a, b), c), d);
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] += t.m[k];
    // leaf 3: U_mu^dag(x-mu) U_nu^dag(x-mu-nu) U_mu(x-mu-nu) U_nu(x-nu)
    a = load_m3(U, shifted(P, x, mu, -1, nu, 0), mu);
    b = load_m3(U, shifted(P, x, mu, -1, nu, -1), nu);
    c = load_m3(U, shifted(P, x, mu, -1, nu, -1), mu);
    d = load_m3(U, shifted(P, x, mu, 0, nu, -1), nu);
    t = mul<false, false>(mul<false, false>(mul<true, true>(a, b), c), d);
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] += t.m[k];
    // leaf 4: U_nu^dag(x-nu) U_mu(x-nu) U_nu(x+mu-nu) U_mu^dag(x)
    a = load_m3(U, shifted(P, x, mu, 0, nu, -1), nu);
    b = load_m3(U, shifted(P, x, mu, 0, nu, -1), mu);
    c = load_m3(U, shifted(P, x, mu, +1, nu, -1), nu);
    d = load_m3(U, s, mu);
    t = mul<false, true>(mul<false, false>(mul<true, false>(a, b), c), d);
#pragma unroll
    for (int k = 0; k < 18; k++) q[k] += t.m[k];
    // (Q - Q^dag) / (8 i): with D = Q_ab - conj(Q_ba), F_ab = -i D / 8 = (Im D, -Re D) / 8
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const T dr = q[2 * (3 * i + j)] - q[2 * (3 * j + i)];
            const T di = q[2 * (3 * i + j) + 1] + q[2 * (3 * j + i) + 1];
            f[2 * (3 * i + j)] = di * (T)0.125;
            f[2 * (3 * i + j) + 1] = -dr * (T)0.125;
        }
}

// F(x) = kappa csw sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x).  In the chiral basis of DESIGN.md sigma_{mu nu} is block
// diagonal with Pauli matrices on the two spin components of each chirality block (upper block, lower block):
//   s_xy = (t3, t3)  s_xz = (-t2, -t2)  s_yz = (t1, t1)  s_xt = (-t1, +t1)  s_yt = (-t2, +t2)  s_zt = (-t3, +t3),
// so block chi is  kappa csw [ t1 (x) W1 + t2 (x) W2 + t3 (x) W3 ],  W1 = F_yz -+ F_xt, W2 = -F_xz -+ F_yt,
// W3 = F_xy -+ F_zt (upper sign: chi = 0), i.e. the 6x6 matrix [[W3, W1 - i W2], [W1 + i W2, -W3]], k = 3 spin + colour.
template <typename T>
__global__ void __launch_bounds__(128) k_clover_from_links(T* __restrict__ clover, const T* __restrict__ U, T coef,
                                                           CloverParams P) {
    const int sc = blockIdx.x * blockDim.x + threadIdx.x;  // canonical site index
    if (sc >= P.V) return;
    int x[4], r = sc;
    x[0] = r % P.L[0]; r /= P.L[0];
    x[1] = r % P.L[1]; r /= P.L[1];
    x[2] = r % P.L[2]; r /= P.L[2];
    x[3] = r;
    const int s = P.ord.index(x);  // native position: what every field access below takes
    T B1[18], B2[18], B3[18], E[18];
    field_strength(B3, U, P, x, s, 0, 1);  // xy
    field_strength(B2, U, P, x, s, 0, 2);  // xz (enters with a minus sign)
    field_strength(B1, U, P, x, s, 1, 2);  // yz
#pragma unroll
    for (int k = 0; k < 18; k++) B2[k] = -B2[k];
    T W1[2][18], W2[2][18], W3[2][18];
    field_strength(E, U, P, x, s, 0, 3);  // xt
#pragma unroll
    for (int k = 0; k < 18; k++) {
        W1[0][k] = B1[k] - E[k];
        W1[1][k] = B1[k] + E[k];
    }
    field_strength(E, U, P, x, s, 1, 3);  // yt
#pragma unroll
    for (int k = 0; k < 18; k++) {
        W2[0][k] = B2[k] - E[k];
        W2[1][k] = B2[k] + E[k];
    }
    field_strength(E, U, P, x, s, 2, 3);  // zt
#pragma unroll
    for (int k = 0; k < 18; k++) {
        W3[0][k] = B3[k] - E[k];
        W3[1][k] = B3[k] + E[k];
    }
#pragma unroll
    for (int chi = 0; chi < 2; chi++) {
        // diagonal: W3_ii for spin 0, -W3_ii for spin 1 (real: W3 is Hermitian)
#pragma unroll
        for (int i = 0; i < 3; i++) {
            clover[clover_off<T>(s, clover_diag_r(chi, i))] = coef * W3[chi][2 * (3 * i + i)];
            clover[clover_off<T>(s, clover_diag_r(chi, 3 + i))] = -coef * W3[chi][2 * (3 * i + i)];
        }
        // strictly lower triangle (k > l), k = 3a + i, l = 3b + j
#pragma unroll
        for (int k = 1; k < 6; k++)
#pragma unroll
            for (int l = 0; l < k; l++) {
                const int a = k / 3, i = k % 3, b = l / 3, j = l % 3;
                T vr, vi;
                if (a == b) {  // +-W3_ij
                    const T sg = a == 0 ? (T)1 : (T)-1;
                    vr = sg * W3[chi][2 * (3 * i + j)];
                    vi = sg * W3[chi][2 * (3 * i + j) + 1];
                } else {  // a = 1, b = 0: (W1 + i W2)_ij
                    vr = W1[chi][2 * (3 * i + j)] - W2[chi][2 * (3 * i + j) + 1];
                    vi = W1[chi][2 * (3 * i + j) + 1] + W2[chi][2 * (3 * i + j)];
                }
                clover[clover_off<T>(s, clover_low_r(chi, k, l, 0))] = coef * vr;
                clover[clover_off<T>(s, clover_low_r(chi, k, l, 1))] = coef * vi;
            }
    }
}

template <typename T>
static int clover_from_links_call(T* clover, const T* U, T kappa, T csw, const int dims[4], void* stream,
                                  const char* what) {
    clear_error();
    if (!clover || !U || check_dims(dims) || !aligned16(clover) || !aligned16(U) || (const void*)clover == (const void*)U) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    CloverParams P;
    for (int mu = 0; mu < 4; mu++) P.L[mu] = dims[mu];
    P.V = (int)volume(dims);
    P.ord.set(dims);
    k_clover_from_links<T><<<(P.V + 127) / 128, 128, 0, (cudaStream_t)stream>>>(clover, U, kappa * csw, P);
    count_launch();
    return check_launch(what);
}

// ------------------------------------------------------------------------------------------------------------
// Block orthonormalisation: within every aggregate (X, chi) the nvec null vectors, restricted to
// the aggregate, are orthonormalised in index order (Gram-Schmidt; the result -- the Q of a QR with positive
// diagonal -- is unique, so it is compared with the oracle's modified Gram-Schmidt up to rounding).
// One CTA per aggregate; the vector being processed lives in shared memory; every vector is projected twice
// against its predecessors ("twice is enough"), all predecessors of one pass at once: warps own predecessors j for
// the dot products <w_j|w_i>, threads own 16-byte slices for the update w_i -= sum_j r_j w_j.
// ------------------------------------------------------------------------------------------------------------
// aggregates whose vector had no component left after the projections (zero or non-finite norm): such a vector is
// written as ZERO instead of Inf/NaN, and counted here (lqcd_orthonormalize_degenerate_count)
__device__ unsigned long long g_ortho_degenerate;

template <typename T>
__global__ void __launch_bounds__(256) k_orthonormalize(T* __restrict__ v, TransferParams P) {
    constexpr int NV = VecOf<T>::NV, CPV = NV / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* wi = reinterpret_cast<T*>(smem_raw);  // LV vec16
    T* rj = wi + (size_t)P.LV * NV;          // 2 * nvec reals: the dots of this pass
    T* red = rj + 2 * P.nvec;                // 8 partial norms
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, W = blockDim.x >> 5;
    T* vagg = v + (long long)blockIdx.x * P.nvec * P.LV * NV;
    for (int i = 0; i < P.nvec; i++) {
        T* vi = vagg + (long long)i * P.LV * NV;
        for (int p = threadIdx.x; p < P.LV; p += blockDim.x) st16(wi + (size_t)p * NV, ld16(vi + (size_t)p * NV));
        __syncthreads();
        for (int pass = 0; pass < 2; pass++) {
            for (int j = w; j < i; j += W) {  // r_j = <w_j | w_i>
                const T* vj = vagg + (long long)j * P.LV * NV;
                T sr = 0, si = 0;
                for (int p = lane; p < P.LV; p += 32) {
                    const V16<T> a = ld16(vj + (size_t)p * NV);
                    const V16<T> x = *reinterpret_cast<const V16<T>*>(wi + (size_t)p * NV);
#pragma unroll
                    for (int e = 0; e < CPV; e++) {
                        sr = fma(a.r[2 * e], x.r[2 * e], sr);
                        sr = fma(a.r[2 * e + 1], x.r[2 * e + 1], sr);
                        si = fma(a.r[2 * e], x.r[2 * e + 1], si);
                        si = fma(-a.r[2 * e + 1], x.r[2 * e], si);
                    }
                }
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) {
                    sr += __shfl_xor_sync(0xffffffffu, sr, off);
                    si += __shfl_xor_sync(0xffffffffu, si, off);
                }
                if (lane == 0) {
                    rj[2 * j] = sr;
                    rj[2 * j + 1] = si;
                }
            }
            __syncthreads();
            for (int p = threadIdx.x; p < P.LV; p += blockDim.x) {  // w_i -= sum_j r_j w_j
                V16<T> acc = *reinterpret_cast<const V16<T>*>(wi + (size_t)p * NV);
                for (int j = 0; j < i; j++) {
                    const V16<T> a = ld16(vagg + ((long long)j * P.LV + p) * NV);
                    const T cr = rj[2 * j], ci = rj[2 * j + 1];
#pragma unroll
                    for (int e = 0; e < CPV; e++) {
                        acc.r[2 * e] = fma(-cr, a.r[2 * e], acc.r[2 * e]);
                        acc.r[2 * e] = fma(ci, a.r[2 * e + 1], acc.r[2 * e]);
                        acc.r[2 * e + 1] = fma(-cr, a.r[2 * e + 1], acc.r[2 * e + 1]);
                        acc.r[2 * e + 1] = fma(-ci, a.r[2 * e], acc.r[2 * e + 1]);
                    }
                }
                *reinterpret_cast<V16<T>*>(wi + (size_t)p * NV) = acc;
            }
            __syncthreads();
        }
        // normalise and write back
        T n2 = 0;
        for (int p = threadIdx.x; p < P.LV; p += blockDim.x) {
            const V16<T> x = *reinterpret_cast<const V16<T>*>(wi + (size_t)p * NV);
#pragma unroll
            for (int e = 0; e < NV; e++) n2 = fma(x.r[e], x.r[e], n2);
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, off);
        if (lane == 0) red[w] = n2;
        __syncthreads();
        T tot = 0;
        for (int k = 0; k < W; k++) tot += red[k];
        const bool ok = tot > (T)0 && tot < (T)INFINITY;  // false for 0, Inf and NaN
        const T inv = ok ? (T)1 / sqrt(tot) : (T)0;
        if (!ok && threadIdx.x == 0) atomicAdd(&g_ortho_degenerate, 1ull);
        for (int p = threadIdx.x; p < P.LV; p += blockDim.x) {
            V16<T> x = *reinterpret_cast<const V16<T>*>(wi + (size_t)p * NV);
#pragma unroll
            for (int e = 0; e < NV; e++) x.r[e] *= inv;
            st16(vi + (size_t)p * NV, x);
        }
        __syncthreads();  // vi is complete (and red, wi are free) before the next vector reads it
    }
}

template <typename T>
static int orthonormalize_call(T* v, const int dims[4], const int block[4], int nvec, void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, v, v, v, dims, block, nvec, what);
    if (rc) return rc;
    if ((long long)P.bv * 6 < nvec) {
        set_error("%s: %d vectors cannot be independent on aggregates of %d complex components", what, nvec, P.bv * 6);
        return LQCD_EINVAL;
    }
    const size_t smem = ((size_t)P.bv * 12 + 2 * (size_t)nvec + 8) * sizeof(T);
    if (smem > 200 * 1024) {
        set_error("%s: block of %d sites does not fit in shared memory", what, P.bv);
        return LQCD_EUNSUPPORTED;
    }
    auto kern = k_orthonormalize<T>;
    static unsigned long long attr = 0;
    if (smem > 48 * 1024) ensure_dynamic_smem(kern, 200 * 1024, attr);
    kern<<<(unsigned)(2 * volume(P.Lc)), 256, smem, (cudaStream_t)stream>>>(v, P);
    count_launch();
    return check_launch(what);
}

// ------------------------------------------------------------------------------------------------------------
// Galerkin coarse operator, Eq. 7: A[X][d][I][J] = <I| D_d |J> with D split into its part inside the
// aggregates (d = 0: site-diagonal term and hops with both ends in X -- this is D_SAP with domain = block) and the
// eight directed hops that leave the aggregate (d = 1 + 2 mu forward, 2 + 2 mu backward).
// Column by column, with the hot-path kernels: for J = (chi_J, i_J) the fine vector P e_J that carries column J of P
// on EVERY aggregate at once is written, one piece of D is applied to it, and the restriction of the result is column
// J of A[.][d] at every coarse site (a directed hop out of X reaches exactly one neighbour aggregate, so the columns
// of different aggregates never mix -- also when the coarse extent is 2 and X+mu = X-mu).
// ------------------------------------------------------------------------------------------------------------
// fine native spinor <- column (chi_J, i_J) of P on every aggregate (zero on the other chirality)
template <typename T>
__global__ void __launch_bounds__(256) k_prolongator_column(T* __restrict__ out_f, const T* __restrict__ v, int chiJ,
                                                            int iJ, TransferParams P) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV, JH = 12 / NV;
    const int X = blockIdx.x;
    for (int q = threadIdx.x; q < 2 * P.LV; q += blockDim.x) {
        const int chi = q / P.LV, p = q % P.LV;
        V16<T> val;
#pragma unroll
        for (int e = 0; e < NV; e++) val.r[e] = 0;
        if (chi == chiJ) val = ld16(v + ((((long long)X * 2 + chi) * P.nvec + iJ) * P.LV + p) * NV);
        const int l = p / JH, jj = p % JH;
        const int s = fine_site(P, X, l);
        st16(out_f + (((long long)(s >> 5) * NJ + chi * JH + jj) * CH + (s & 31)) * NV, val);
    }
}

struct HopParams {
    int L[4], b[4], multi[4], bc[4];
    int V;
    SiteOrder ord;  // native position of a site (layout.cuh)
};

// out(x) = -kappa beta (1 -+ g_mu) U in(x +- mu) if that hop leaves the aggregate of x, else 0
template <typename T, int MU, bool FWD>
__global__ void __launch_bounds__(128) k_hop_cross(T* __restrict__ out, const T* __restrict__ in, const T* __restrict__ U,
                                                   T kappa, HopParams P) {
    const int sc = blockIdx.x * blockDim.x + threadIdx.x;  // canonical site index
    if (sc >= P.V) return;
    int x[4], r = sc;
    x[0] = r % P.L[0]; r /= P.L[0];
    x[1] = r % P.L[1]; r /= P.L[1];
    x[2] = r % P.L[2]; r /= P.L[2];
    x[3] = r;
    const int s = P.ord.index(x);  // native position
    T acc[24];
#pragma unroll
    for (int k = 0; k < 24; k++) acc[k] = 0;
    const int lx = x[MU] % P.b[MU];
    const bool crosses = P.multi[MU] && (FWD ? lx == P.b[MU] - 1 : lx == 0);
    if (crosses) {
        const bool wraps = FWD ? x[MU] == P.L[MU] - 1 : x[MU] == 0;
        const int nb = FWD ? P.ord.fwd(s, MU, x[MU]) : P.ord.bwd(s, MU, x[MU]);
        const T ph = -kappa * (wraps ? (T)P.bc[MU] : (T)1);
        T p[24], h[12], u[18], g[12];
        load_spinor<T>(p, in, nb);
        load_link<T, false>(u, U, FWD ? s : nb, MU);
        constexpr int SGN = FWD ? -1 : +1;  // (1 - g_mu) forward, (1 + g_mu) backward (Eq. 1)
        project<MU, SGN, T>(h, p);
        su3_mult<FWD, T>(g, u, h);
        reconstruct<MU, SGN, T>(acc, g, ph);
    }
    store_spinor<T>(out, s, acc);
}

// A[X][d][I][J] <- xc[X][I] for every X, I
template <typename T>
__global__ void k_scatter_column(T* __restrict__ A, const T* __restrict__ xc, int d, int J, int N, long long Vc) {
    const long long n = Vc * N;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long X = idx / N;
        const int I = (int)(idx % N);
        T* dst = A + ((((X * 9 + d) * N + I) * N) + J) * 2;
        dst[0] = xc[idx * 2];
        dst[1] = xc[idx * 2 + 1];
    }
}

static inline size_t up256(size_t n) { return (n + 255) & ~(size_t)255; }

template <typename T> static size_t galerkin_ws_bytes(const int dims[4], const int block[4], int nvec) {
    int cd[4];
    if (check_block(dims, block, nvec, cd)) return 0;
    // one column of P, its nine images under the pieces of D, their nine restrictions
    return up256(10 * (size_t)nchunks(dims) * CH * 24 * sizeof(T) + 9 * (size_t)volume(cd) * 4 * nvec * sizeof(T));
}

template <typename T> int dd_mult(T*, const T*, const T*, const T*, T, const int*, const int*, const int*, void*);
template <> int dd_mult<float>(float* o, const float* i, const float* U, const float* c, float k, const int* d,
                               const int* bc, const int* b, void* st) {
    return lqcd_wilson_clover_dd_mult_f32(o, i, U, c, k, d, bc, b, 0, st);
}
template <> int dd_mult<double>(double* o, const double* i, const double* U, const double* c, double k, const int* d,
                                const int* bc, const int* b, void* st) {
    return lqcd_wilson_clover_dd_mult_f64(o, i, U, c, k, d, bc, b, 0, st);
}
// (transfer.cu) nrhs fine vectors back to back -> nrhs coarse vectors back to back, null vectors streamed once per group
template <typename T>
int restrict_mrhs_call(T* out_c, const T* in_f, const T* v, const int dims[4], const int block[4], int nvec, int nrhs,
                       void* stream, const char* what);

template <typename T>
static int galerkin_call(T* A, const T* U, const T* clover, const T* v, T kappa, const int dims[4], const int bc[4],
                         const int block[4], int nvec, void* ws, void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, A, U, v, dims, block, nvec, what);
    if (rc) return rc;
    for (int mu = 0; mu < 4; mu++)
        if (P.Lc[mu] < 2) {  // the 9-point stencil of directed blocks needs two coarse sites per direction (Q8)
            set_error("%s: coarse extent < 2 in direction %d", what, mu);
            return LQCD_EINVAL;
        }
    if (!clover || !ws || !bc || !aligned16(clover) || !aligned16(ws)) {
        set_error("%s: null or misaligned pointer", what);
        return LQCD_EINVAL;
    }
    HopParams H;
    for (int mu = 0; mu < 4; mu++) {
        if (bc[mu] != 1 && bc[mu] != -1) {
            set_error("%s: bc[%d] = %d not in {+1,-1}", what, mu, bc[mu]);
            return LQCD_EINVAL;
        }
        H.L[mu] = dims[mu];
        H.b[mu] = block[mu];
        H.multi[mu] = 1;  // coarse extents are >= 2 (check_block)
        H.bc[mu] = bc[mu];
    }
    H.V = (int)volume(dims);
    H.ord.set(dims);
    cudaStream_t st = (cudaStream_t)stream;
    const long long Vc = volume(P.Lc);
    // vectors back to back, as restrict_mrhs_call expects them (every size is a multiple of 16 bytes)
    const long long fstride = (long long)nchunks(dims) * CH * 24, cstride = Vc * 4 * nvec;
    T* col = (T*)ws;
    T* img = col + fstride;        // nine images
    T* xc = col + 10 * fstride;    // nine restrictions
    const int N = 2 * nvec;
    const unsigned hop_grid = (unsigned)((H.V + 127) / 128);
    long long sgrid = (Vc * N + 255) / 256;
    if (sgrid > 148 * 32) sgrid = 148 * 32;
    for (int J = 0; J < N; J++) {
        k_prolongator_column<T><<<(unsigned)Vc, 256, 0, st>>>(col, v, J / nvec, J % nvec, P);
        count_launch();
        if ((rc = dd_mult<T>(img, col, U, clover, kappa, dims, bc, block, stream))) return rc;
        k_hop_cross<T, 0, true><<<hop_grid, 128, 0, st>>>(img + 1 * fstride, col, U, kappa, H);
        k_hop_cross<T, 0, false><<<hop_grid, 128, 0, st>>>(img + 2 * fstride, col, U, kappa, H);
        k_hop_cross<T, 1, true><<<hop_grid, 128, 0, st>>>(img + 3 * fstride, col, U, kappa, H);
        k_hop_cross<T, 1, false><<<hop_grid, 128, 0, st>>>(img + 4 * fstride, col, U, kappa, H);
        k_hop_cross<T, 2, true><<<hop_grid, 128, 0, st>>>(img + 5 * fstride, col, U, kappa, H);
        k_hop_cross<T, 2, false><<<hop_grid, 128, 0, st>>>(img + 6 * fstride, col, U, kappa, H);
        k_hop_cross<T, 3, true><<<hop_grid, 128, 0, st>>>(img + 7 * fstride, col, U, kappa, H);
        k_hop_cross<T, 3, false><<<hop_grid, 128, 0, st>>>(img + 8 * fstride, col, U, kappa, H);
        count_launch(8);
        // the nine restrictions in one pass over the null vectors (they are 97 % of a restriction's traffic)
        if ((rc = restrict_mrhs_call<T>(xc, img, v, dims, block, nvec, 9, stream, what))) return rc;
        for (int d = 0; d < 9; d++) k_scatter_column<T><<<(unsigned)sgrid, 256, 0, st>>>(A, xc + d * cstride, d, J, N, Vc);
        count_launch(9);
    }
    return check_launch(what);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {
int lqcd_orthonormalize_blocks_f32(float* nullvecs, const int dims[4], const int block[4], int nvec, void* stream) {
    return orthonormalize_call<float>(nullvecs, dims, block, nvec, stream, "lqcd_orthonormalize_blocks_f32");
}
int lqcd_orthonormalize_blocks_f64(double* nullvecs, const int dims[4], const int block[4], int nvec, void* stream) {
    return orthonormalize_call<double>(nullvecs, dims, block, nvec, stream, "lqcd_orthonormalize_blocks_f64");
}
long long lqcd_orthonormalize_degenerate_count(void* stream) {
    unsigned long long n = 0, zero = 0;
    if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess ||
        cudaMemcpyFromSymbol(&n, g_ortho_degenerate, sizeof(n)) != cudaSuccess ||
        cudaMemcpyToSymbol(g_ortho_degenerate, &zero, sizeof(zero)) != cudaSuccess) {
        set_error("lqcd_orthonormalize_degenerate_count: %s", cudaGetErrorString(cudaGetLastError()));
        return LQCD_ECUDA;
    }
    return (long long)n;
}
size_t lqcd_galerkin_workspace_bytes(const int dims[4], const int block[4], int nvec, int real_bytes) {
    return real_bytes == 8 ? galerkin_ws_bytes<double>(dims, block, nvec) : galerkin_ws_bytes<float>(dims, block, nvec);
}
int lqcd_galerkin_coarse_f32(float* A, const float* U, const float* clover, const float* nullvecs, float kappa,
                             const int dims[4], const int bc[4], const int block[4], int nvec, void* ws_dev,
                             void* stream) {
    return galerkin_call<float>(A, U, clover, nullvecs, kappa, dims, bc, block, nvec, ws_dev, stream,
                                "lqcd_galerkin_coarse_f32");
}
int lqcd_galerkin_coarse_f64(double* A, const double* U, const double* clover, const double* nullvecs, double kappa,
                             const int dims[4], const int bc[4], const int block[4], int nvec, void* ws_dev,
                             void* stream) {
    return galerkin_call<double>(A, U, clover, nullvecs, kappa, dims, bc, block, nvec, ws_dev, stream,
                                 "lqcd_galerkin_coarse_f64");
}
int lqcd_clover_from_links_f32(float* clover_native, const float* U_native18, float kappa, float csw, const int dims[4],
                               void* stream) {
    return clover_from_links_call<float>(clover_native, U_native18, kappa, csw, dims, stream,
                                         "lqcd_clover_from_links_f32");
}
int lqcd_clover_from_links_f64(double* clover_native, const double* U_native18, double kappa, double csw,
                               const int dims[4], void* stream) {
    return clover_from_links_call<double>(clover_native, U_native18, kappa, csw, dims, stream,
                                          "lqcd_clover_from_links_f64");
}
}
