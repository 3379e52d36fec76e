// transfer.cu -- rows A4/A5 of the hot path: block restriction and prolongation with chirality-split null
// vectors (Eqs. 5, 6):
//   restrict:  out_c[X][chi][i]    = sum_{x in X} sum_{alpha in chi, c} conj(v_i(x,alpha,c)) in_f(x,alpha,c)
//   prolong:   out_f(x,alpha,c)    = sum_i v_i(x,alpha,c) in_c[X(x)][chi(alpha)][i]
//
// Design: both are a single pass over the null vectors (nvec*96 B per fine site
// in fp32 -- 97% of the traffic), so the native null-vector layout [X][chi][i][l][k] makes the part of v_i
// that belongs to one aggregate (X, chi) ONE contiguous vector of |block|*6 complex, read with full-width
// 128-bit coalesced, L1::no_allocate / L2 evict-first loads by both kernels.  One CTA per aggregate (X, chi):
//   restrict: the aggregate's slice of in_f is staged once in shared memory; each warp owns null vectors
//             i = w, w+W, ... and finishes its dot product with a warp-shuffle tree (fixed order, no atomics);
//   prolong:  the nvec coarse coefficients sit in shared memory; each thread owns 16-byte slices of the
//             aggregate and accumulates over i, no reduction across threads.
// The paper's GPU version bounced these two steps through the host; here they stay on the device.
#include "aggregate.cuh"
#include "common.cuh"
#include "knobs.h"

namespace lqcd {

template <typename T> __device__ __forceinline__ void cdot_acc(T& sr, T& si, const V16<T>& a, const V16<T>& x);
// sum conj(a) x over the complex entries of one vec16
template <> __device__ __forceinline__ void cdot_acc<float>(float& sr, float& si, const V16<float>& a,
                                                            const V16<float>& x) {
    sr = fmaf(a.r[0], x.r[0], sr);
    sr = fmaf(a.r[1], x.r[1], sr);
    si = fmaf(a.r[0], x.r[1], si);
    si = fmaf(-a.r[1], x.r[0], si);
    sr = fmaf(a.r[2], x.r[2], sr);
    sr = fmaf(a.r[3], x.r[3], sr);
    si = fmaf(a.r[2], x.r[3], si);
    si = fmaf(-a.r[3], x.r[2], si);
}
template <> __device__ __forceinline__ void cdot_acc<double>(double& sr, double& si, const V16<double>& a,
                                                             const V16<double>& x) {
    sr = fma(a.r[0], x.r[0], sr);
    sr = fma(a.r[1], x.r[1], sr);
    si = fma(a.r[0], x.r[1], si);
    si = fma(-a.r[1], x.r[0], si);
}

// acc += a * (cr + i ci) for each complex entry of the vec16
template <typename T> __device__ __forceinline__ void caxpy(V16<T>& acc, const V16<T>& a, T cr, T ci) {
    constexpr int NV = VecOf<T>::NV;
#pragma unroll
    for (int e = 0; e < NV / 2; e++) {
        acc.r[2 * e] = fma(a.r[2 * e], cr, acc.r[2 * e]);
        acc.r[2 * e] = fma(-a.r[2 * e + 1], ci, acc.r[2 * e]);
        acc.r[2 * e + 1] = fma(a.r[2 * e], ci, acc.r[2 * e + 1]);
        acc.r[2 * e + 1] = fma(a.r[2 * e + 1], cr, acc.r[2 * e + 1]);
    }
}

// Dependency fence of a batch of streaming loads.  ptxas sinks the later loads of a batch below the arithmetic on the
// earlier ones (SASS of k_restrict: 4 LDG, then FFMA and LDG interleaved: 3-4 requests in flight per lane instead of
// UNROLL).  fence_batch() returns 0, computed from one register of EVERY load of the batch (ptxas also reorders the loads
// among themselves, so the last one alone is not enough) and a zero that is only known at run time; it is added to the
// shared-memory index from which every product of the batch reads its other operand: no product can start before the
// whole batch has returned, so its UNROLL loads are issued back to back.  UNROLL / 2 LOP3 per batch; the arithmetic
// and its order are unchanged (bit-identical results).  Measured at c5 on the power-capped box (1.5 GHz): k_restrict
// fp32 4998 -> 4674 us (7.2 TB/s), fp64 9715 -> 9346 us.  The same fence in k_prolong changes nothing (fp32 4915 -> 4920
// us: at 95 % occupancy enough requests are in flight without it) and is not used there.
template <int N> __device__ __forceinline__ int fence_batch(const V16<float> (&a)[N], int zero) {
    int m = 0;
#pragma unroll
    for (int u = 0; u < N; u++) m |= __float_as_int(a[u].r[0]);
    return m & zero;
}
template <int N> __device__ __forceinline__ int fence_batch(const V16<double> (&a)[N], int zero) {
    int m = 0;
#pragma unroll
    for (int u = 0; u < N; u++) m |= __double2loint(a[u].r[0]);
    return m & zero;
}

template <typename T, int UNROLL>
__global__ void __launch_bounds__(256) k_restrict(T* __restrict__ out_c, const T* __restrict__ in_f,
                                                  const T* __restrict__ v, TransferParams P) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV, JH = 12 / NV;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);  // [l][12 reals of chirality chi]
    const int agg = blockIdx.x + P.agg_off;  // (X, chi)
    const int X = agg >> 1, chi = agg & 1;
    // stage the aggregate's slice of in_f
    for (int idx = threadIdx.x; idx < P.LV; idx += blockDim.x) {
        const int l = idx / JH, jj = idx % JH;
        const int s = fine_site(P, X, l);
        const T* src = in_f + (((long long)(s >> 5) * NJ + chi * JH + jj) * CH + (s & 31)) * NV;
        st16(sm + (long long)idx * NV, ld16(src));
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, W = blockDim.x >> 5;
    const T* vagg = v + (long long)agg * P.nvec * P.LV * NV;
    for (int i = w; i < P.nvec; i += W) {
        const T* vi = vagg + (long long)i * P.LV * NV;
        T sr[UNROLL], si[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; u++) sr[u] = si[u] = 0;
        int p = lane;
        for (; p + 32 * (UNROLL - 1) < P.LV; p += 32 * UNROLL) {
            V16<T> a[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; u++) a[u] = ld16_stream(vi + (long long)(p + 32 * u) * NV);
            const int z = fence_batch(a, P.zero);
#pragma unroll
            for (int u = 0; u < UNROLL; u++)
                cdot_acc<T>(sr[u], si[u], a[u], *reinterpret_cast<const V16<T>*>(sm + (p + 32 * u + z) * NV));
        }
        for (; p < P.LV; p += 32)
            cdot_acc<T>(sr[0], si[0], ld16_stream(vi + (long long)p * NV), *reinterpret_cast<const V16<T>*>(sm + p * NV));
        T tr = 0, ti = 0;
#pragma unroll
        for (int u = 0; u < UNROLL; u++) {
            tr += sr[u];
            ti += si[u];
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            tr += __shfl_xor_sync(0xffffffffu, tr, off);
            ti += __shfl_xor_sync(0xffffffffu, ti, off);
        }
        if (lane == 0) {
            T* o = out_c + ((long long)agg * P.nvec + i) * 2;
            o[0] = tr;
            o[1] = ti;
        }
    }
}

// restrict for up to NRMAX fine vectors at once (F4 for the transfer: the null vectors -- 97 % of the traffic -- are
// streamed ONCE for all of them).  in_f + r * fstride is the r-th fine vector, out_c + r * cstride the r-th result.
template <typename T, int UNROLL, int NRMAX>
__global__ void __launch_bounds__(256) k_restrict_mrhs(T* __restrict__ out_c, long long cstride,
                                                       const T* __restrict__ in_f, long long fstride, int nr,
                                                       const T* __restrict__ v, TransferParams P) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV, JH = 12 / NV;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);  // [r][l][12 reals of chirality chi]
    const int agg = blockIdx.x + P.agg_off;  // (X, chi)
    const int X = agg >> 1, chi = agg & 1;
    for (int idx = threadIdx.x; idx < P.LV; idx += blockDim.x) {
        const int l = idx / JH, jj = idx % JH;
        const int s = fine_site(P, X, l);
        const long long off = (((long long)(s >> 5) * NJ + chi * JH + jj) * CH + (s & 31)) * NV;
        for (int r = 0; r < nr; r++) st16(sm + ((long long)r * P.LV + idx) * NV, ld16(in_f + r * fstride + off));
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, W = blockDim.x >> 5;
    const T* vagg = v + (long long)agg * P.nvec * P.LV * NV;
    for (int i = w; i < P.nvec; i += W) {
        const T* vi = vagg + (long long)i * P.LV * NV;
        T sr[NRMAX], si[NRMAX];
#pragma unroll
        for (int r = 0; r < NRMAX; r++) sr[r] = si[r] = 0;
        int p = lane;
        for (; p + 32 * (UNROLL - 1) < P.LV; p += 32 * UNROLL) {
            V16<T> a[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; u++) a[u] = ld16_stream(vi + (long long)(p + 32 * u) * NV);
#pragma unroll
            for (int r = 0; r < NRMAX; r++)
                if (r < nr) {
#pragma unroll
                    for (int u = 0; u < UNROLL; u++)
                        cdot_acc<T>(sr[r], si[r], a[u],
                                    *reinterpret_cast<const V16<T>*>(sm + ((long long)r * P.LV + p + 32 * u) * NV));
                }
        }
        for (; p < P.LV; p += 32) {
            const V16<T> a = ld16_stream(vi + (long long)p * NV);
#pragma unroll
            for (int r = 0; r < NRMAX; r++)
                if (r < nr) cdot_acc<T>(sr[r], si[r], a, *reinterpret_cast<const V16<T>*>(sm + ((long long)r * P.LV + p) * NV));
        }
#pragma unroll
        for (int r = 0; r < NRMAX; r++) {
            if (r < nr) {
                T tr = sr[r], ti = si[r];
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) {
                    tr += __shfl_xor_sync(0xffffffffu, tr, off);
                    ti += __shfl_xor_sync(0xffffffffu, ti, off);
                }
                if (lane == 0) {
                    T* o = out_c + r * cstride + ((long long)agg * P.nvec + i) * 2;
                    o[0] = tr;
                    o[1] = ti;
                }
            }
        }
    }
}

template <typename T, int UNROLL>
__global__ void __launch_bounds__(256) k_prolong(T* __restrict__ out_f, const T* __restrict__ in_c,
                                                 const T* __restrict__ v, TransferParams P) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV, JH = 12 / NV;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* xc = reinterpret_cast<T*>(smem_raw);  // nvec complex
    const int agg = blockIdx.x + P.agg_off;
    const int X = agg >> 1, chi = agg & 1;
    for (int i = threadIdx.x; i < 2 * P.nvec; i += blockDim.x) xc[i] = in_c[(long long)agg * P.nvec * 2 + i];
    __syncthreads();
    const T* vagg = v + (long long)agg * P.nvec * P.LV * NV;
    for (int p = threadIdx.x; p < P.LV; p += blockDim.x) {
        V16<T> acc;
#pragma unroll
        for (int e = 0; e < NV; e++) acc.r[e] = 0;
        const T* vp = vagg + (long long)p * NV;
        int i = 0;
        for (; i + UNROLL <= P.nvec; i += UNROLL) {
            V16<T> a[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; u++) a[u] = ld16_stream(vp + (long long)(i + u) * P.LV * NV);
#pragma unroll
            for (int u = 0; u < UNROLL; u++) caxpy<T>(acc, a[u], xc[2 * (i + u)], xc[2 * (i + u) + 1]);
        }
        for (; i < P.nvec; i++) caxpy<T>(acc, ld16_stream(vp + (long long)i * P.LV * NV), xc[2 * i], xc[2 * i + 1]);
        const int l = p / JH, jj = p % JH;
        const int s = fine_site(P, X, l);
        T* dst = out_f + (((long long)(s >> 5) * NJ + chi * JH + jj) * CH + (s & 31)) * NV;
        st16_stream(dst, acc);
    }
}

// prolong for up to NRMAX coarse vectors at once: the null vectors are streamed once, every thread keeps NRMAX
// accumulators for its 16-byte slice of the aggregate
template <typename T, int UNROLL, int NRMAX>
__global__ void __launch_bounds__(256) k_prolong_mrhs(T* __restrict__ out_f, long long fstride,
                                                      const T* __restrict__ in_c, long long cstride, int nr,
                                                      const T* __restrict__ v, TransferParams P) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV, JH = 12 / NV;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* xc = reinterpret_cast<T*>(smem_raw);  // [r][nvec] complex
    const int agg = blockIdx.x + P.agg_off;
    const int X = agg >> 1, chi = agg & 1;
    for (int q = threadIdx.x; q < nr * 2 * P.nvec; q += blockDim.x) {
        const int r = q / (2 * P.nvec), i = q % (2 * P.nvec);
        xc[q] = in_c[r * cstride + (long long)agg * P.nvec * 2 + i];
    }
    __syncthreads();
    const T* vagg = v + (long long)agg * P.nvec * P.LV * NV;
    for (int p = threadIdx.x; p < P.LV; p += blockDim.x) {
        V16<T> acc[NRMAX];
#pragma unroll
        for (int r = 0; r < NRMAX; r++)
#pragma unroll
            for (int e = 0; e < NV; e++) acc[r].r[e] = 0;
        const T* vp = vagg + (long long)p * NV;
        int i = 0;
        for (; i + UNROLL <= P.nvec; i += UNROLL) {
            V16<T> a[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; u++) a[u] = ld16_stream(vp + (long long)(i + u) * P.LV * NV);
#pragma unroll
            for (int r = 0; r < NRMAX; r++)
                if (r < nr) {
#pragma unroll
                    for (int u = 0; u < UNROLL; u++)
                        caxpy<T>(acc[r], a[u], xc[(r * P.nvec + i + u) * 2], xc[(r * P.nvec + i + u) * 2 + 1]);
                }
        }
        for (; i < P.nvec; i++) {
            const V16<T> a = ld16_stream(vp + (long long)i * P.LV * NV);
#pragma unroll
            for (int r = 0; r < NRMAX; r++)
                if (r < nr) caxpy<T>(acc[r], a, xc[(r * P.nvec + i) * 2], xc[(r * P.nvec + i) * 2 + 1]);
        }
        const int l = p / JH, jj = p % JH;
        const int s = fine_site(P, X, l);
        const long long off = (((long long)(s >> 5) * NJ + chi * JH + jj) * CH + (s & 31)) * NV;
#pragma unroll
        for (int r = 0; r < NRMAX; r++)
            if (r < nr) st16_stream(out_f + r * fstride + off, acc[r]);
    }
}

template <typename T>
static int restrict_call(T* out_c, const T* in_f, const T* v, const int dims[4], const int block[4], int nvec,
                         void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, out_c, in_f, v, dims, block, nvec, what);
    if (rc) return rc;
    const size_t smem = (size_t)P.bv * 12 * sizeof(T);
    if (smem > 200 * 1024) {
        set_error("%s: block of %d sites does not fit in shared memory", what, P.bv);
        return LQCD_EUNSUPPORTED;
    }
    auto kern = k_restrict<T, 8>;
    if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int warps = g_knobs.transfer_warps > 0 ? g_knobs.transfer_warps : 8;
    if (warps > 8) warps = 8;
    if (warps > nvec) warps = nvec;
    const long long nagg = 2 * volume(P.Lc);
    kern<<<(unsigned)nagg, warps * 32, smem, (cudaStream_t)stream>>>(out_c, in_f, v, P);
    count_launch();
    return check_launch(what);
}

// restrict on the aggregates of the coarse sites [X0, X1) only (host_api.cu: under the upload of the next slab)
template <typename T>
int restrict_range_call(T* out_c, const T* in_f, const T* v, const int dims[4], const int block[4], int nvec, long long X0,
                        long long X1, void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, out_c, in_f, v, dims, block, nvec, what);
    if (rc) return rc;
    const size_t smem = (size_t)P.bv * 12 * sizeof(T);
    if (smem > 200 * 1024) {
        set_error("%s: block of %d sites does not fit in shared memory", what, P.bv);
        return LQCD_EUNSUPPORTED;
    }
    if (X1 <= X0) return LQCD_OK;
    auto kern = k_restrict<T, 8>;
    if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int warps = g_knobs.transfer_warps > 0 ? g_knobs.transfer_warps : 8;
    if (warps > 8) warps = 8;
    if (warps > nvec) warps = nvec;
    P.agg_off = (int)(2 * X0);
    kern<<<(unsigned)(2 * (X1 - X0)), warps * 32, smem, (cudaStream_t)stream>>>(out_c, in_f, v, P);
    count_launch();
    return check_launch(what);
}
template int restrict_range_call<float>(float*, const float*, const float*, const int*, const int*, int, long long,
                                        long long, void*, const char*);
template int restrict_range_call<double>(double*, const double*, const double*, const int*, const int*, int, long long,
                                         long long, void*, const char*);

// nrhs fine vectors back to back -> nrhs coarse vectors back to back; the null vectors are read once per group of
// NRMAX vectors (as many as fit in shared memory next to each other: 9 in fp32, 4 in fp64 for 4^4 blocks)
template <typename T>
int restrict_mrhs_call(T* out_c, const T* in_f, const T* v, const int dims[4], const int block[4], int nvec, int nrhs,
                       void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, out_c, in_f, v, dims, block, nvec, what);
    if (rc) return rc;
    if (nrhs < 1) {
        set_error("%s: nrhs < 1", what);
        return LQCD_EINVAL;
    }
    constexpr int NRMAX = 9;
    const size_t one = (size_t)P.bv * 12 * sizeof(T);
    int per = (int)((108 * 1024) / one);  // nine 12-KB slices of a 4^4 aggregate in fp32; two CTAs per SM
    if (per > NRMAX) per = NRMAX;
    const long long fstride = (long long)nchunks(dims) * CH * 24, cstride = volume(P.Lc) * 4 * nvec;
    if (per < 2) {  // block too large to hold two slices: one vector at a time
        for (int k = 0; k < nrhs; k++)
            if ((rc = restrict_call<T>(out_c + k * cstride, in_f + k * fstride, v, dims, block, nvec, stream, what))) return rc;
        return LQCD_OK;
    }
    auto kern = k_restrict_mrhs<T, 4, NRMAX>;
    static unsigned long long attr = 0;
    ensure_dynamic_smem(kern, 108 * 1024, attr);
    int warps = nvec < 8 ? nvec : 8;
    const long long nagg = 2 * volume(P.Lc);
    for (int k = 0; k < nrhs; k += per) {
        const int nr = nrhs - k < per ? nrhs - k : per;
        kern<<<(unsigned)nagg, warps * 32, nr * one, (cudaStream_t)stream>>>(out_c + k * cstride, cstride,
                                                                             in_f + k * fstride, fstride, nr, v, P);
        count_launch();
    }
    return check_launch(what);
}
template int restrict_mrhs_call<float>(float*, const float*, const float*, const int*, const int*, int, int, void*,
                                       const char*);
template int restrict_mrhs_call<double>(double*, const double*, const double*, const int*, const int*, int, int, void*,
                                        const char*);

template <typename T>
static int prolong_call(T* out_f, const T* in_c, const T* v, const int dims[4], const int block[4], int nvec,
                        void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, out_f, in_c, v, dims, block, nvec, what);
    if (rc) return rc;
    const size_t smem = (size_t)nvec * 2 * sizeof(T);
    if (smem > 48 * 1024) {
        set_error("%s: nvec = %d outside the compiled range", what, nvec);
        return LQCD_EUNSUPPORTED;
    }
    int threads = P.LV >= 256 ? 256 : (P.LV + 31) / 32 * 32;
    const long long nagg = 2 * volume(P.Lc);
    k_prolong<T, 8><<<(unsigned)nagg, threads, smem, (cudaStream_t)stream>>>(out_f, in_c, v, P);
    count_launch();
    return check_launch(what);
}

// prolong on the aggregates of the coarse sites [X0, X1) only (host_api.cu: the download of a slab runs under the
// prolongation of the next)
template <typename T>
int prolong_range_call(T* out_f, const T* in_c, const T* v, const int dims[4], const int block[4], int nvec, long long X0,
                       long long X1, void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, out_f, in_c, v, dims, block, nvec, what);
    if (rc) return rc;
    const size_t smem = (size_t)nvec * 2 * sizeof(T);
    if (smem > 48 * 1024) {
        set_error("%s: nvec = %d outside the compiled range", what, nvec);
        return LQCD_EUNSUPPORTED;
    }
    if (X1 <= X0) return LQCD_OK;
    const int threads = P.LV >= 256 ? 256 : (P.LV + 31) / 32 * 32;
    P.agg_off = (int)(2 * X0);
    k_prolong<T, 8><<<(unsigned)(2 * (X1 - X0)), threads, smem, (cudaStream_t)stream>>>(out_f, in_c, v, P);
    count_launch();
    return check_launch(what);
}
template int prolong_range_call<float>(float*, const float*, const float*, const int*, const int*, int, long long,
                                       long long, void*, const char*);
template int prolong_range_call<double>(double*, const double*, const double*, const int*, const int*, int, long long,
                                        long long, void*, const char*);

// nrhs coarse vectors back to back -> nrhs fine vectors back to back, null vectors read once per group of 8
template <typename T>
int prolong_mrhs_call(T* out_f, const T* in_c, const T* v, const int dims[4], const int block[4], int nvec, int nrhs,
                      void* stream, const char* what) {
    TransferParams P;
    int rc = transfer_setup<T>(P, out_f, in_c, v, dims, block, nvec, what);
    if (rc) return rc;
    if (nrhs < 1) {
        set_error("%s: nrhs < 1", what);
        return LQCD_EINVAL;
    }
    constexpr int NRMAX = 8;
    const size_t one = (size_t)nvec * 2 * sizeof(T);
    if (NRMAX * one > 48 * 1024) {
        set_error("%s: nvec = %d outside the compiled range", what, nvec);
        return LQCD_EUNSUPPORTED;
    }
    const long long fstride = (long long)nchunks(dims) * CH * 24, cstride = volume(P.Lc) * 4 * nvec;
    const int threads = P.LV >= 256 ? 256 : (P.LV + 31) / 32 * 32;
    const long long nagg = 2 * volume(P.Lc);
    for (int k = 0; k < nrhs; k += NRMAX) {
        const int nr = nrhs - k < NRMAX ? nrhs - k : NRMAX;
        k_prolong_mrhs<T, 4, NRMAX><<<(unsigned)nagg, threads, nr * one, (cudaStream_t)stream>>>(
            out_f + k * fstride, fstride, in_c + k * cstride, cstride, nr, v, P);
        count_launch();
    }
    return check_launch(what);
}
template int prolong_mrhs_call<float>(float*, const float*, const float*, const int*, const int*, int, int, void*,
                                      const char*);
template int prolong_mrhs_call<double>(double*, const double*, const double*, const int*, const int*, int, int, void*,
                                       const char*);

}  // namespace lqcd

using namespace lqcd;

extern "C" {
int lqcd_restrict_f32(float* o, const float* i, const float* v, const int dims[4], const int block[4], int nvec,
                      void* st) {
    return restrict_call<float>(o, i, v, dims, block, nvec, st, "lqcd_restrict_f32");
}
int lqcd_restrict_f64(double* o, const double* i, const double* v, const int dims[4], const int block[4], int nvec,
                      void* st) {
    return restrict_call<double>(o, i, v, dims, block, nvec, st, "lqcd_restrict_f64");
}
int lqcd_prolong_f32(float* o, const float* i, const float* v, const int dims[4], const int block[4], int nvec,
                     void* st) {
    return prolong_call<float>(o, i, v, dims, block, nvec, st, "lqcd_prolong_f32");
}
int lqcd_prolong_f64(double* o, const double* i, const double* v, const int dims[4], const int block[4], int nvec,
                     void* st) {
    return prolong_call<double>(o, i, v, dims, block, nvec, st, "lqcd_prolong_f64");
}
int lqcd_restrict_mrhs_f32(float* o, const float* i, const float* v, const int dims[4], const int block[4], int nvec,
                           int nrhs, void* st) {
    return restrict_mrhs_call<float>(o, i, v, dims, block, nvec, nrhs, st, "lqcd_restrict_mrhs_f32");
}
int lqcd_restrict_mrhs_f64(double* o, const double* i, const double* v, const int dims[4], const int block[4],
                           int nvec, int nrhs, void* st) {
    return restrict_mrhs_call<double>(o, i, v, dims, block, nvec, nrhs, st, "lqcd_restrict_mrhs_f64");
}
int lqcd_prolong_mrhs_f32(float* o, const float* i, const float* v, const int dims[4], const int block[4], int nvec,
                          int nrhs, void* st) {
    return prolong_mrhs_call<float>(o, i, v, dims, block, nvec, nrhs, st, "lqcd_prolong_mrhs_f32");
}
int lqcd_prolong_mrhs_f64(double* o, const double* i, const double* v, const int dims[4], const int block[4],
                          int nvec, int nrhs, void* st) {
    return prolong_mrhs_call<double>(o, i, v, dims, block, nvec, nrhs, st, "lqcd_prolong_mrhs_f64");
}
}
