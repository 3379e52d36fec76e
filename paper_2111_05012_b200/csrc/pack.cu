// pack.cu -- device->device re-layout kernels between the canonical interchange layouts and the native
// layouts of include/lqcd_b200.h.  Not on the timed path.  One thread per (site, real): canonical side
// is read/written fully coalesced.
#include "common.cuh"
#include "layout.cuh"

namespace lqcd {

template <typename T, bool UNPACK>
__global__ void k_spinor(T* __restrict__ dst, const T* __restrict__ src, long long n0, long long n, SiteOrder ord) {
    // canonical reals [n0, n) (24 per site)
    for (long long idx = n0 + blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long s = ord.from_canonical((int)(idx / 24));  // native position of canonical site idx / 24
        const int r = (int)(idx % 24);
        if (UNPACK) dst[idx] = src[spinor_off<T>(s, r)];
        else dst[spinor_off<T>(s, r)] = src[idx];
    }
}

// canonical U[mu][s][a][b] -> native [chunk][mu][...]
template <typename T, bool L12>
__global__ void k_gauge(T* __restrict__ dst, const T* __restrict__ src, long long V, SiteOrder ord) {
    const long long n = 4 * V * 18;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(idx % 18);
        const long long ms = idx / 18;
        const long long s = ord.from_canonical((int)(ms % V));
        const int mu = (int)(ms / V);
        if (L12) {
            if (r < 12) dst[gauge12_off<T>(s, mu, r)] = src[idx];
        } else {
            dst[gauge18_off<T>(s, mu, r)] = src[idx];
        }
    }
}

// canonical F[s][chi][k][l] complex -> native 72 reals: diagonal real parts, strictly-lower entries.
// The Hermitian part (F + F^dag)/2 of the input is what is stored.
template <typename T>
__global__ void k_clover(T* __restrict__ dst, const T* __restrict__ src, long long V, SiteOrder ord) {
    const long long n = V * 72;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long s = idx / 72;
        const int r = (int)(idx % 72);
        const int chi = r / 36, q = r % 36;
        const T* blk = src + (s * 2 + chi) * 72;  // [k][l][reim]
        T val;
        if (q < 6) {
            val = blk[(q * 6 + q) * 2];
        } else {
            const int t = (q - 6) / 2, reim = (q - 6) % 2;
            int k = 1;
            while (tri(k + 1, 0) <= t) k++;
            const int l = t - tri(k, 0);
            const T lo = blk[(k * 6 + l) * 2 + reim];
            const T up = blk[(l * 6 + k) * 2 + reim];
            val = reim ? (T)0.5 * (lo - up) : (T)0.5 * (lo + up);
        }
        dst[clover_off<T>((long long)ord.from_canonical((int)s), r)] = val;
    }
}

// native 72 reals -> canonical full Hermitian blocks F[s][chi][k][l] complex
template <typename T>
__global__ void k_clover_unpack(T* __restrict__ dst, const T* __restrict__ src, long long V, SiteOrder ord) {
    const long long n = V * 72;  // one thread per (site, chi, k, l)
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long s = ord.from_canonical((int)(idx / 72));
        const int e = (int)(idx % 72), chi = e / 36, k = (e % 36) / 6, l = e % 6;
        T re, im;
        if (k == l) {
            re = src[clover_off<T>(s, clover_diag_r(chi, k))];
            im = 0;
        } else if (k > l) {
            re = src[clover_off<T>(s, clover_low_r(chi, k, l, 0))];
            im = src[clover_off<T>(s, clover_low_r(chi, k, l, 1))];
        } else {
            re = src[clover_off<T>(s, clover_low_r(chi, l, k, 0))];
            im = -src[clover_off<T>(s, clover_low_r(chi, l, k, 1))];
        }
        dst[idx * 2] = re;
        dst[idx * 2 + 1] = im;
    }
}

struct BlockGeom {
    int L[4], b[4], Lc[4];
    int bv;
};

template <typename T, bool UNPACK>
__global__ void k_nullvec(T* __restrict__ native, T* __restrict__ canon, int i, int nvec, BlockGeom g, long long V) {
    const long long n = V * 24;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n;
         idx += (long long)gridDim.x * blockDim.x) {
        long long s = idx / 24;
        const int r = (int)(idx % 24);
        const int alpha = r / 6, c = (r % 6) / 2, reim = r % 2;
        int x[4];
        x[0] = (int)(s % g.L[0]); s /= g.L[0];
        x[1] = (int)(s % g.L[1]); s /= g.L[1];
        x[2] = (int)(s % g.L[2]); s /= g.L[2];
        x[3] = (int)s;
        long long X = 0;
        int l = 0;
        for (int mu = 3; mu >= 0; mu--) {
            X = X * g.Lc[mu] + x[mu] / g.b[mu];
            l = l * g.b[mu] + x[mu] % g.b[mu];
        }
        const long long off = nullvec_off(X, alpha / 2, i, l, 3 * (alpha % 2) + c, reim, nvec, g.bv);
        if (UNPACK) canon[idx] = native[off];
        else native[off] = canon[idx];
    }
}

static int grid_for(long long n) {
    long long g = (n + 255) / 256;
    if (g > 148LL * 64) g = 148LL * 64;
    if (g < 1) g = 1;
    return (int)g;
}

template <typename T, bool UNPACK>
static int spinor_call(T* dst, const T* src, const int dims[4], void* stream, const char* what) {
    clear_error();
    if (!dst || !src || check_dims(dims) || !aligned16(dst) || !aligned16(src) || dst == src) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    const long long V = volume(dims);
    if (V > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    SiteOrder ord;
    ord.set(dims);
    k_spinor<T, UNPACK><<<grid_for(V * 24), 256, 0, (cudaStream_t)stream>>>(dst, src, 0, V * 24, ord);
    count_launch();
    return check_launch(what);
}

// the sites [s0, s1) only (arguments validated by the caller, host_api.cu)
template <typename T, bool UNPACK>
int spinor_range_call(T* dst, const T* src, const int dims[4], long long s0, long long s1, void* stream, const char* what) {
    if (s1 <= s0) return LQCD_OK;
    SiteOrder ord;
    ord.set(dims);
    k_spinor<T, UNPACK><<<grid_for((s1 - s0) * 24), 256, 0, (cudaStream_t)stream>>>(dst, src, s0 * 24, s1 * 24, ord);
    count_launch();
    return check_launch(what);
}
template int spinor_range_call<float, false>(float*, const float*, const int*, long long, long long, void*, const char*);
template int spinor_range_call<float, true>(float*, const float*, const int*, long long, long long, void*, const char*);
template int spinor_range_call<double, false>(double*, const double*, const int*, long long, long long, void*, const char*);
template int spinor_range_call<double, true>(double*, const double*, const int*, long long, long long, void*, const char*);

template <typename T>
static int gauge_call(T* dst, const T* src, const int dims[4], unsigned flags, void* stream, const char* what) {
    clear_error();
    if (!dst || !src || check_dims(dims) || !aligned16(dst) || !aligned16(src) || dst == src ||
        (flags & ~LQCD_LINKS_12)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    const long long V = volume(dims);
    if (V > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    SiteOrder ord;
    ord.set(dims);
    if (flags & LQCD_LINKS_12)
        k_gauge<T, true><<<grid_for(V * 72), 256, 0, (cudaStream_t)stream>>>(dst, src, V, ord);
    else
        k_gauge<T, false><<<grid_for(V * 72), 256, 0, (cudaStream_t)stream>>>(dst, src, V, ord);
    count_launch();
    return check_launch(what);
}

template <typename T> static int clover_call(T* dst, const T* src, const int dims[4], void* stream, const char* what) {
    clear_error();
    if (!dst || !src || check_dims(dims) || !aligned16(dst) || !aligned16(src) || dst == src) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    const long long V = volume(dims);
    if (V > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    SiteOrder ord;
    ord.set(dims);
    k_clover<T><<<grid_for(V * 72), 256, 0, (cudaStream_t)stream>>>(dst, src, V, ord);
    count_launch();
    return check_launch(what);
}

template <typename T>
static int clover_unpack_call(T* dst, const T* src, const int dims[4], void* stream, const char* what) {
    clear_error();
    if (!dst || !src || check_dims(dims) || !aligned16(dst) || !aligned16(src) || dst == src) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    const long long V = volume(dims);
    if (V > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    SiteOrder ord;
    ord.set(dims);
    k_clover_unpack<T><<<grid_for(V * 72), 256, 0, (cudaStream_t)stream>>>(dst, src, V, ord);
    count_launch();
    return check_launch(what);
}

template <typename T, bool UNPACK>
static int nullvec_call(T* native, T* canon, int i, const int dims[4], const int block[4], int nvec, void* stream,
                        const char* what) {
    clear_error();
    BlockGeom g;
    if (!native || !canon || check_block_local(dims, block, nvec, g.Lc) || i < 0 || i >= nvec || !aligned16(native) ||
        !aligned16(canon)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    g.bv = 1;
    for (int mu = 0; mu < 4; mu++) {
        g.L[mu] = dims[mu];
        g.b[mu] = block[mu];
        g.bv *= block[mu];
    }
    const long long V = volume(dims);
    k_nullvec<T, UNPACK><<<grid_for(V * 24), 256, 0, (cudaStream_t)stream>>>(native, canon, i, nvec, g, V);
    count_launch();
    return check_launch(what);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {
int lqcd_pack_spinor_f32(float* d, const float* s, const int dims[4], void* st) {
    return spinor_call<float, false>(d, s, dims, st, "lqcd_pack_spinor_f32");
}
int lqcd_pack_spinor_f64(double* d, const double* s, const int dims[4], void* st) {
    return spinor_call<double, false>(d, s, dims, st, "lqcd_pack_spinor_f64");
}
int lqcd_unpack_spinor_f32(float* d, const float* s, const int dims[4], void* st) {
    return spinor_call<float, true>(d, s, dims, st, "lqcd_unpack_spinor_f32");
}
int lqcd_unpack_spinor_f64(double* d, const double* s, const int dims[4], void* st) {
    return spinor_call<double, true>(d, s, dims, st, "lqcd_unpack_spinor_f64");
}
int lqcd_pack_gauge_f32(float* d, const float* s, const int dims[4], unsigned flags, void* st) {
    return gauge_call<float>(d, s, dims, flags, st, "lqcd_pack_gauge_f32");
}
int lqcd_pack_gauge_f64(double* d, const double* s, const int dims[4], unsigned flags, void* st) {
    return gauge_call<double>(d, s, dims, flags, st, "lqcd_pack_gauge_f64");
}
int lqcd_pack_clover_f32(float* d, const float* s, const int dims[4], void* st) {
    return clover_call<float>(d, s, dims, st, "lqcd_pack_clover_f32");
}
int lqcd_pack_clover_f64(double* d, const double* s, const int dims[4], void* st) {
    return clover_call<double>(d, s, dims, st, "lqcd_pack_clover_f64");
}
int lqcd_unpack_clover_f32(float* d, const float* s, const int dims[4], void* st) {
    return clover_unpack_call<float>(d, s, dims, st, "lqcd_unpack_clover_f32");
}
int lqcd_unpack_clover_f64(double* d, const double* s, const int dims[4], void* st) {
    return clover_unpack_call<double>(d, s, dims, st, "lqcd_unpack_clover_f64");
}
int lqcd_pack_nullvec_f32(float* d, const float* s, int i, const int dims[4], const int block[4], int nvec, void* st) {
    return nullvec_call<float, false>(d, const_cast<float*>(s), i, dims, block, nvec, st, "lqcd_pack_nullvec_f32");
}
int lqcd_pack_nullvec_f64(double* d, const double* s, int i, const int dims[4], const int block[4], int nvec,
                          void* st) {
    return nullvec_call<double, false>(d, const_cast<double*>(s), i, dims, block, nvec, st, "lqcd_pack_nullvec_f64");
}
int lqcd_unpack_nullvec_f32(float* d, const float* s, int i, const int dims[4], const int block[4], int nvec,
                            void* st) {
    return nullvec_call<float, true>(const_cast<float*>(s), d, i, dims, block, nvec, st, "lqcd_unpack_nullvec_f32");
}
int lqcd_unpack_nullvec_f64(double* d, const double* s, int i, const int dims[4], const int block[4], int nvec,
                            void* st) {
    return nullvec_call<double, true>(const_cast<double*>(s), d, i, dims, block, nvec, st, "lqcd_unpack_nullvec_f64");
}
}
