// coarse_half.cu -- the coarse operator (row A3, Eqs. 4, 7) on HALF storage.
//
// gamma5-hermiticity of D (Eq. 2) carries over to the Galerkin blocks (Eq. 7):
//     A_{-mu}(X) = G5c  A_{+mu}(X - mu)^dag  G5c,        G5c = diag(+1 (chi = 0), -1 (chi = 1)) (x) 1_nvec
// (pinned on the oracle side, tests/test_oracle_pins.py), so only A_0 and the four FORWARD blocks need to be stored:
// 5 instead of 9 blocks per coarse site -- 5 N^2 + 2 N instead of 9 N^2 + 2 N complex of compulsory traffic.
//
//   out(X) = A_0(X) in(X) + sum_mu A_{+mu}(X) in(X + mu)  +  sum_mu G5c A_{+mu}(X - mu)^dag G5c in(X - mu)
//
// Every stored block is read from HBM exactly ONCE and serves both sites it couples: the warp that owns site Y streams
// the rows of A_{+mu}(Y); a row r gives (i) the forward dot product  <row r | in(Y + mu)>  for out(Y), reduced over
// the lanes by a shuffle tree as in coarse.cu, and (ii) the column-wise contribution  conj(A[r][c]) s_r in_r(Y)  to
// out(Y + mu)[c] -- the transposed product.  Because one warp walks ALL rows of the block and a lane keeps its
// 16-byte slice of the row, the transposed sums are lane-local: no shuffle, no atomics.  They are written to a scratch
// vector bw[mu][Y + mu] and a second, tiny pass adds   out(X) += bw[0][X] + bw[1][X] + bw[2][X] + bw[3][X]   in that
// fixed order: results are bit-reproducible.  Two launches; scratch = 4 coarse vectors.
// Coarse extent 2 (X + mu == X - mu) needs no special case: the block of Y still reaches Y + mu exactly once each way.
// LQCD_DAGGER (G5c D_c G5c): the two G5c of the transposed term cancel, the forward terms take them as in coarse.cu.
#include <mutex>
#include "common.cuh"
#include "knobs.h"

namespace lqcd {

struct CoarseHalfParams {
    int Lc[4];
    int Vc;
    int nvec;
    int N;   // 2 nvec
    int RV;  // vec16 per matrix row
    int dagger;
};

// sr + i si += a . x (complex, 16 bytes of each) / bacc += conj(a) w for the complex scalar w = (wr, wi)
template <typename T> __device__ __forceinline__ void cdot16(T& sr, T& si, const V16<T>& a, const V16<T>& x) {
#pragma unroll
    for (int e = 0; e < VecOf<T>::NV / 2; e++) {
        sr = fma(a.r[2 * e], x.r[2 * e], sr);
        sr = fma(-a.r[2 * e + 1], x.r[2 * e + 1], sr);
        si = fma(a.r[2 * e], x.r[2 * e + 1], si);
        si = fma(a.r[2 * e + 1], x.r[2 * e], si);
    }
}
template <typename T> __device__ __forceinline__ void conj_axpy16(V16<T>& acc, const V16<T>& a, T wr, T wi) {
#pragma unroll
    for (int e = 0; e < VecOf<T>::NV / 2; e++) {
        acc.r[2 * e] = fma(a.r[2 * e], wr, acc.r[2 * e]);
        acc.r[2 * e] = fma(a.r[2 * e + 1], wi, acc.r[2 * e]);
        acc.r[2 * e + 1] = fma(a.r[2 * e], wi, acc.r[2 * e + 1]);
        acc.r[2 * e + 1] = fma(-a.r[2 * e + 1], wr, acc.r[2 * e + 1]);
    }
}

// One warp per coarse site; a row is spread over the 32 lanes, CPL vec16 per lane; R rows in flight.
// FULL: the row is exactly 32 CPL vec16 and N is a multiple of R (no predicates: the loads stay batched).
template <typename T, int CPL, int R, bool FULL>
__global__ void __launch_bounds__(128, 4)
    k_coarse_half(T* __restrict__ out, T* __restrict__ bw, const T* __restrict__ in, const T* __restrict__ Ah,
                  CoarseHalfParams P) {
    constexpr int NV = VecOf<T>::NV;
    constexpr int CPV = NV / 2;  // complex per vec16
    const int lane = threadIdx.x & 31;
    const int X = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (X >= P.Vc) return;
    int fwd[4];
    {
        int rem = X, xc[4];
        xc[0] = rem % P.Lc[0]; rem /= P.Lc[0];
        xc[1] = rem % P.Lc[1]; rem /= P.Lc[1];
        xc[2] = rem % P.Lc[2]; rem /= P.Lc[2];
        xc[3] = rem;
        const int stride[4] = {1, P.Lc[0], P.Lc[0] * P.Lc[1], P.Lc[0] * P.Lc[1] * P.Lc[2]};
#pragma unroll
        for (int mu = 0; mu < 4; mu++)
            fwd[mu] = (xc[mu] == P.Lc[mu] - 1) ? X - (P.Lc[mu] - 1) * stride[mu] : X + stride[mu];
    }
    // my slices of the five source vectors of the forward terms (G5c in for the dagger form), of the source of the
    // transposed terms (G5c in(X), or in(X) for the dagger form), and the G5c signs of my columns
    V16<T> xv[5][CPL], wsrc[CPL], sgn[CPL];
#pragma unroll
    for (int c = 0; c < CPL; c++) {
        const int v = lane + 32 * c;
        const bool ok = FULL || v < P.RV;
#pragma unroll
        for (int e = 0; e < CPV; e++) {
            const T s = (v * CPV + e >= P.nvec) ? (T)-1 : (T)1;
            sgn[c].r[2 * e] = sgn[c].r[2 * e + 1] = s;
        }
#pragma unroll
        for (int d = 0; d < 5; d++) {
            if (ok) {
                xv[d][c] = ld16(in + ((long long)(d == 0 ? X : fwd[d - 1]) * P.RV + v) * NV);
            } else {
#pragma unroll
                for (int e = 0; e < NV; e++) xv[d][c].r[e] = 0;
            }
        }
#pragma unroll
        for (int e = 0; e < NV; e++) {
            const T plain = xv[0][c].r[e], signed_ = plain * sgn[c].r[e];
            wsrc[c].r[e] = P.dagger ? plain : signed_;
            if (P.dagger) {
                xv[0][c].r[e] = signed_;
#pragma unroll
                for (int d = 1; d < 5; d++) xv[d][c].r[e] *= sgn[c].r[e];
            }
        }
    }
    V16<T> bacc[4][CPL];
#pragma unroll
    for (int mu = 0; mu < 4; mu++)
#pragma unroll
        for (int c = 0; c < CPL; c++)
#pragma unroll
            for (int e = 0; e < NV; e++) bacc[mu][c].r[e] = 0;

    const T* Asite = Ah + (long long)X * 5 * P.N * P.RV * NV;
    for (int row0 = 0; row0 < P.N; row0 += R) {
        // all loads of the R rows first: R * 5 * CPL independent streaming 16-byte requests per lane
        V16<T> a[R][5][CPL];
#pragma unroll
        for (int r = 0; r < R; r++)
#pragma unroll
            for (int d = 0; d < 5; d++)
#pragma unroll
                for (int c = 0; c < CPL; c++) {
                    const int v = lane + 32 * c;
                    if (FULL || (row0 + r < P.N && v < P.RV))
                        a[r][d][c] = ld16_stream(Asite + (((long long)d * P.N + row0 + r) * P.RV + v) * NV);
                    else {
#pragma unroll
                        for (int e = 0; e < NV; e++) a[r][d][c].r[e] = 0;
                    }
                }
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int row = row0 + r;
            // (i) forward: out(X)[row] = sum_d <row of block d | source d>
            T sr = 0, si = 0;
#pragma unroll
            for (int d = 0; d < 5; d++)
#pragma unroll
                for (int c = 0; c < CPL; c++) cdot16<T>(sr, si, a[r][d][c], xv[d][c]);
            // (ii) transposed: the scalar s_row in_row(X) lives in vec16 row / CPV of the source: lane (row / CPV) % 32
            const int vrow = row / CPV, erow = row - vrow * CPV, crow = vrow >> 5;
            T cr = 0, ci = 0;
#pragma unroll
            for (int c = 0; c < CPL; c++)
#pragma unroll
                for (int e = 0; e < CPV; e++)
                    if (c == crow && e == erow) {
                        cr = wsrc[c].r[2 * e];
                        ci = wsrc[c].r[2 * e + 1];
                    }
            const T wr = __shfl_sync(0xffffffffu, cr, vrow & 31), wi = __shfl_sync(0xffffffffu, ci, vrow & 31);
#pragma unroll
            for (int mu = 0; mu < 4; mu++)
#pragma unroll
                for (int c = 0; c < CPL; c++) conj_axpy16<T>(bacc[mu][c], a[r][1 + mu][c], wr, wi);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                sr += __shfl_xor_sync(0xffffffffu, sr, off);
                si += __shfl_xor_sync(0xffffffffu, si, off);
            }
            if (lane == 0 && (FULL || row < P.N)) {
                const T s = (P.dagger && row >= P.nvec) ? (T)-1 : (T)1;
                T* o = out + ((long long)X * P.N + row) * 2;
                o[0] = s * sr;
                o[1] = s * si;
            }
        }
    }
    // the transposed products go to the scratch vector of their direction at the site they belong to
#pragma unroll
    for (int mu = 0; mu < 4; mu++)
#pragma unroll
        for (int c = 0; c < CPL; c++) {
            const int v = lane + 32 * c;
            if (FULL || v < P.RV) {
                V16<T> o = bacc[mu][c];
                if (!P.dagger) {
#pragma unroll
                    for (int e = 0; e < NV; e++) o.r[e] *= sgn[c].r[e];
                }
                st16(bw + (((long long)mu * P.Vc + fwd[mu]) * P.RV + v) * NV, o);
            }
        }
}

// out += bw[0] + bw[1] + bw[2] + bw[3], in this order (n vec16 per vector)
template <typename T>
__global__ void __launch_bounds__(256) k_coarse_half_sum(T* __restrict__ out, const T* __restrict__ bw, long long n) {
    constexpr int NV = VecOf<T>::NV;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        V16<T> o = ld16(out + i * NV);
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const V16<T> b = ld16(bw + ((long long)mu * n + i) * NV);
#pragma unroll
            for (int e = 0; e < NV; e++) o.r[e] += b.r[e];
        }
        st16(out + i * NV, o);
    }
}

// Ah[X][0] = A[X][0], Ah[X][1 + mu] = A[X][1 + 2 mu]  (nb = vec16 per block)
template <typename T>
__global__ void __launch_bounds__(256) k_pack_coarse_half(T* __restrict__ Ah, const T* __restrict__ A, long long Vc,
                                                          long long nb) {
    constexpr int NV = VecOf<T>::NV;
    const long long n = Vc * 5 * nb;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long X = i / (5 * nb), rem = i - X * 5 * nb;
        const int h = (int)(rem / nb);
        const long long k = rem - h * nb;
        const int d = h == 0 ? 0 : 2 * h - 1;
        st16(Ah + i * NV, ld16_stream(A + ((X * 9 + d) * nb + k) * NV));
    }
}

template <typename T> static int half_geometry(CoarseHalfParams& P, const int cdims[4], int nvec, const char* what) {
    if (check_dims(cdims) || nvec < 1) {
        set_error("%s: non-positive dim or nvec < 1", what);
        return LQCD_EINVAL;
    }
    for (int mu = 0; mu < 4; mu++) {
        if (cdims[mu] < 2) {
            set_error("%s: coarse extent %d < 2 in direction %d", what, cdims[mu], mu);
            return LQCD_EINVAL;
        }
        P.Lc[mu] = cdims[mu];
    }
    if (volume(cdims) > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    P.Vc = (int)volume(cdims);
    P.nvec = nvec;
    P.N = 2 * nvec;
    P.RV = 2 * P.N / VecOf<T>::NV;
    if (P.RV > 128) {
        set_error("%s: nvec = %d outside the compiled range (row longer than 128 vec16)", what, nvec);
        return LQCD_EUNSUPPORTED;
    }
    return LQCD_OK;
}

template <typename T, int CPL>
static void launch_half(T* out, T* bw, const T* in, const T* Ah, const CoarseHalfParams& P, cudaStream_t st) {
    constexpr int R = CPL == 1 ? 2 : 1;
    const int warps = 4;
    const unsigned grid = (unsigned)((P.Vc + warps - 1) / warps);
    const bool full = P.RV == 32 * CPL && P.N % R == 0;
    if (full) k_coarse_half<T, CPL, R, true><<<grid, warps * 32, 0, st>>>(out, bw, in, Ah, P);
    else k_coarse_half<T, CPL, R, false><<<grid, warps * 32, 0, st>>>(out, bw, in, Ah, P);
}

template <typename T>
static int coarse_half_call(T* out, const T* in, const T* Ah, const int cdims[4], int nvec, unsigned flags, void* ws,
                            void* stream, const char* what) {
    clear_error();
    if (!out || !in || !Ah || !ws) {
        set_error("%s: null pointer", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(out) || !aligned16(in) || !aligned16(Ah) || !aligned16(ws) || out == in) {
        set_error("%s: pointers must be 16-byte aligned and out must not alias in", what);
        return LQCD_EINVAL;
    }
    if (flags & ~LQCD_DAGGER) {
        set_error("%s: unknown flag bits 0x%x", what, flags);
        return LQCD_EINVAL;
    }
    CoarseHalfParams P;
    int rc = half_geometry<T>(P, cdims, nvec, what);
    if (rc) return rc;
    P.dagger = (flags & LQCD_DAGGER) ? 1 : 0;
    cudaStream_t st = (cudaStream_t)stream;
    T* bw = static_cast<T*>(ws);
    if (P.RV <= 32) launch_half<T, 1>(out, bw, in, Ah, P, st);
    else if (P.RV <= 64) launch_half<T, 2>(out, bw, in, Ah, P, st);
    else if (P.RV <= 96) launch_half<T, 3>(out, bw, in, Ah, P, st);
    else launch_half<T, 4>(out, bw, in, Ah, P, st);
    const long long n = (long long)P.Vc * P.RV;
    long long grid = (n + 255) / 256;
    if (grid > 148 * 16) grid = 148 * 16;
    k_coarse_half_sum<T><<<(unsigned)grid, 256, 0, st>>>(out, bw, n);
    count_launch(2);
    return check_launch(what);
}

template <typename T>
static int pack_half_call(T* Ah, const T* A, const int cdims[4], int nvec, void* stream, const char* what) {
    clear_error();
    if (!Ah || !A || !aligned16(Ah) || !aligned16(A) || Ah == A) {
        set_error("%s: null, misaligned or aliasing pointer", what);
        return LQCD_EINVAL;
    }
    CoarseHalfParams P;
    int rc = half_geometry<T>(P, cdims, nvec, what);
    if (rc) return rc;
    const long long nb = (long long)P.N * P.RV;
    long long grid = ((long long)P.Vc * 5 * nb + 255) / 256;
    if (grid > 148 * 32) grid = 148 * 32;
    k_pack_coarse_half<T><<<(unsigned)grid, 256, 0, (cudaStream_t)stream>>>(Ah, A, P.Vc, nb);
    count_launch();
    return check_launch(what);
}

// ---- the variant that allocates nothing ----------------------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it): the four scratch vectors bw[0..3] live in a file-scope device array instead of a caller-supplied workspace.
// Every GPU that loads the library holds these LQCD_NOALLOC_SCRATCH_BYTES until the process exits.
//
// In HOST code the name g_half_scratch is the host-side stand-in of the symbol, NOT a device address (a kernel handed
// &g_half_scratch[0] from the host would fault or, where the GPU can reach host memory, quietly use the wrong memory):
// the device address is asked for once per device with cudaGetSymbolAddress, with that device current, and cached.
static __device__ __align__(256) unsigned char g_half_scratch[LQCD_NOALLOC_SCRATCH_BYTES];
static void* g_half_scratch_addr[64] = {};  // per device ordinal; written once, under g_half_scratch_mutex
static std::mutex g_half_scratch_mutex;

static int half_scratch_ptr(void** out, const char* what) {
    const int d = current_device();
    if (d < 0 || d >= 64) {
        set_error("%s: no current CUDA device (or ordinal %d >= 64)", what, d);
        return LQCD_ECUDA;
    }
    std::lock_guard<std::mutex> lock(g_half_scratch_mutex);
    if (!g_half_scratch_addr[d]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_half_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            set_error("%s: cudaGetSymbolAddress of the static scratch failed on device %d: %s", what, d,
                      cudaGetErrorString(e));
            return LQCD_ECUDA;
        }
        g_half_scratch_addr[d] = p;
    }
    *out = g_half_scratch_addr[d];
    return LQCD_OK;
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {
size_t lqcd_native_coarse_half_reals(const int cdims[4], int nvec) {
    if (check_dims(cdims) || nvec < 1) return 0;
    return (size_t)volume(cdims) * 5 * 8 * (size_t)nvec * (size_t)nvec;
}
size_t lqcd_coarse_half_workspace_bytes(const int cdims[4], int nvec, int real_bytes) {
    if (check_dims(cdims) || nvec < 1 || (real_bytes != 4 && real_bytes != 8)) return 0;
    return (size_t)volume(cdims) * 4 * 4 * (size_t)nvec * (size_t)real_bytes;
}
int lqcd_pack_coarse_half_f32(float* Ah, const float* A, const int cdims[4], int nvec, void* stream) {
    return pack_half_call<float>(Ah, A, cdims, nvec, stream, "lqcd_pack_coarse_half_f32");
}
int lqcd_pack_coarse_half_f64(double* Ah, const double* A, const int cdims[4], int nvec, void* stream) {
    return pack_half_call<double>(Ah, A, cdims, nvec, stream, "lqcd_pack_coarse_half_f64");
}
int lqcd_coarse_mult_half_f32(float* out, const float* in, const float* Ah, const int cdims[4], int nvec,
                              unsigned flags, void* ws_dev, void* stream) {
    return coarse_half_call<float>(out, in, Ah, cdims, nvec, flags, ws_dev, stream, "lqcd_coarse_mult_half_f32");
}
int lqcd_coarse_mult_half_f64(double* out, const double* in, const double* Ah, const int cdims[4], int nvec,
                              unsigned flags, void* ws_dev, void* stream) {
    return coarse_half_call<double>(out, in, Ah, cdims, nvec, flags, ws_dev, stream, "lqcd_coarse_mult_half_f64");
}
int lqcd_coarse_mult_half_noalloc_f32(float* out, const float* in, const float* Ah, const int cdims[4], int nvec,
                                      unsigned flags, void* stream) {
    const char* what = "lqcd_coarse_mult_half_noalloc_f32";
    clear_error();
    const size_t need = lqcd_coarse_half_workspace_bytes(cdims, nvec, (int)sizeof(float));
    if (need == 0) {
        set_error("%s: non-positive dim or nvec < 1", what);
        return LQCD_EINVAL;
    }
    if (need > (size_t)LQCD_NOALLOC_SCRATCH_BYTES) {
        set_error("%s: the problem needs %zu bytes of scratch (4 coarse vectors of %lld sites x %d complex), the static "
                  "array holds LQCD_NOALLOC_SCRATCH_BYTES = %zu: use lqcd_coarse_mult_half_f32 with a caller-owned "
                  "workspace", what, need, volume(cdims), 2 * nvec, (size_t)LQCD_NOALLOC_SCRATCH_BYTES);
        return LQCD_EUNSUPPORTED;
    }
    void* ws = nullptr;
    const int rc = half_scratch_ptr(&ws, what);
    if (rc) return rc;
    // Nothing has to start at zero: k_coarse_half writes every element of bw[0..3] of THIS problem (each site Y stores
    // the whole vector bw[mu][Y + mu], and every site is some Y + mu) before k_coarse_half_sum reads it, so whatever
    // an earlier call left in the array, of this or another size, is overwritten or never read.
    return coarse_half_call<float>(out, in, Ah, cdims, nvec, flags, ws, stream, what);
}
}
