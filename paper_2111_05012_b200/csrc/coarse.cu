// coarse.cu -- row A3 of the hot path: the coarse-lattice operator, a 9-point stencil of dense N x N complex
// blocks, N = 2 nvec (Eqs. 4, 7):
//   out(X) = A[X][0] in(X) + sum_mu ( A[X][1+2mu] in(X+mu) + A[X][2+2mu] in(X-mu) ),   neighbours modulo Lc.
//
// Design: the operator is a pure stream of A (9 N^2 complex per coarse site, read
// exactly once); the vectors are ~N/(9 N^2) of the traffic and live in L2.  A stays in its canonical row-major
// layout: one matrix row is N complex = one contiguous run of vec16.  A group of LPR lanes owns a row (LPR = 32
// for N = 64 in fp32: one 512-byte coalesced request per row per block), each lane multiplies its 16-byte slice
// of the row with the matching slice of the neighbour vector -- held in registers for all nine neighbours and
// reused across the rows the warp walks -- accumulates over the nine blocks, and the row's dot product is
// finished by a warp-shuffle tree (the paper's GPU mapping is one thread per row; here a row is
// spread across lanes so that every request is a full-width coalesced 128-bit access).  R rows per lane are in
// flight at once (R*9 independent 16-byte loads per lane), A is loaded with L1::no_allocate / L2 evict-first.
// Reduction order is fixed (no atomics) so results are reproducible.
#include "common.cuh"
#include "knobs.h"

namespace lqcd {

struct CoarseParams {
    int Lc[4];
    int Vc;
    int nvec;
    int N;          // 2 nvec
    int RV;         // vec16 per matrix row
    int ntile;      // row tiles per site
    int tpw;        // row tiles per warp (divides ntile)
    long long ntask;  // Vc * ntile / tpw warp tasks
    int dagger;
};

template <typename T> __device__ __forceinline__ void cmadd(T& sr, T& si, const V16<T>& a, const V16<T>& x);
template <> __device__ __forceinline__ void cmadd<float>(float& sr, float& si, const V16<float>& a, const V16<float>& x) {
    sr = fmaf(a.r[0], x.r[0], sr);
    sr = fmaf(-a.r[1], x.r[1], sr);
    si = fmaf(a.r[0], x.r[1], si);
    si = fmaf(a.r[1], x.r[0], si);
    sr = fmaf(a.r[2], x.r[2], sr);
    sr = fmaf(-a.r[3], x.r[3], sr);
    si = fmaf(a.r[2], x.r[3], si);
    si = fmaf(a.r[3], x.r[2], si);
}
template <> __device__ __forceinline__ void cmadd<double>(double& sr, double& si, const V16<double>& a,
                                                          const V16<double>& x) {
    sr = fma(a.r[0], x.r[0], sr);
    sr = fma(-a.r[1], x.r[1], sr);
    si = fma(a.r[0], x.r[1], si);
    si = fma(a.r[1], x.r[0], si);
}

// LPR lanes per row (power of two <= 32), CPL vec16 per lane per row, R rows in flight per lane.
// FULL: N is a multiple of the row tile and a row is exactly LPR*CPL vec16 -- no bounds predicates, so the loads of
// a tile are unconditional and stay batched at the top of the tile.
template <typename T, int LPR, int CPL, int R, bool FULL>
__global__ void __launch_bounds__(256, 2) k_coarse(T* __restrict__ out, const T* __restrict__ in, const T* __restrict__ A,
                                                CoarseParams P) {
    constexpr int NV = VecOf<T>::NV;
    constexpr int CPV = NV / 2;  // complex per vec16
    constexpr int G = 32 / LPR;  // rows side by side in a warp
    const int lane = threadIdx.x & 31;
    const int g = lane / LPR, q = lane % LPR;
    const long long task = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (task >= P.ntask) return;
    const int wps = P.ntile / P.tpw;  // warps per site
    const int X = (int)(task / wps);
    const int tile0 = (int)(task % wps) * P.tpw;

    // the nine source sites
    int src[9];
    {
        int xc[4], rem = X;
        xc[0] = rem % P.Lc[0]; rem /= P.Lc[0];
        xc[1] = rem % P.Lc[1]; rem /= P.Lc[1];
        xc[2] = rem % P.Lc[2]; rem /= P.Lc[2];
        xc[3] = rem;
        const int stride[4] = {1, P.Lc[0], P.Lc[0] * P.Lc[1], P.Lc[0] * P.Lc[1] * P.Lc[2]};
        src[0] = X;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            src[1 + 2 * mu] = (xc[mu] == P.Lc[mu] - 1) ? X - (P.Lc[mu] - 1) * stride[mu] : X + stride[mu];
            src[2 + 2 * mu] = (xc[mu] == 0) ? X + (P.Lc[mu] - 1) * stride[mu] : X - stride[mu];
        }
    }
    // my slices of the nine source vectors (with the Gamma5c sign of the column for the dagger variant)
    V16<T> xv[9][CPL];
#pragma unroll
    for (int d = 0; d < 9; d++)
#pragma unroll
        for (int c = 0; c < CPL; c++) {
            const int v = q + LPR * c;
            if (FULL || v < P.RV) {
                xv[d][c] = ld16(in + ((long long)src[d] * P.RV + v) * NV);
                if (P.dagger) {
#pragma unroll
                    for (int e = 0; e < CPV; e++)
                        if (v * CPV + e >= P.nvec) {
                            xv[d][c].r[2 * e] = -xv[d][c].r[2 * e];
                            xv[d][c].r[2 * e + 1] = -xv[d][c].r[2 * e + 1];
                        }
                }
            } else {
#pragma unroll
                for (int e = 0; e < NV; e++) xv[d][c].r[e] = 0;
            }
        }

    const T* Asite = A + (long long)X * 9 * P.N * P.RV * NV;
    for (int t = 0; t < P.tpw; t++) {
        const int rbase = (tile0 + t) * (G * R);
        T sr[R], si[R];
#pragma unroll
        for (int r = 0; r < R; r++) sr[r] = si[r] = 0;
        // issue all loads of the tile first (R * 9 * CPL independent 16-byte requests per lane)
        V16<T> a[R][9][CPL];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int row = rbase + r * G + g;
#pragma unroll
            for (int d = 0; d < 9; d++)
#pragma unroll
                for (int c = 0; c < CPL; c++) {
                    const int v = q + LPR * c;
                    if (FULL || (row < P.N && v < P.RV))
                        a[r][d][c] = ld16_stream(Asite + (((long long)d * P.N + row) * P.RV + v) * NV);
                    else {
#pragma unroll
                        for (int e = 0; e < NV; e++) a[r][d][c].r[e] = 0;
                    }
                }
        }
#pragma unroll
        for (int r = 0; r < R; r++)
#pragma unroll
            for (int d = 0; d < 9; d++)
#pragma unroll
                for (int c = 0; c < CPL; c++) cmadd<T>(sr[r], si[r], a[r][d][c], xv[d][c]);
        // finish the row dot products across the LPR lanes of each group
#pragma unroll
        for (int r = 0; r < R; r++) {
#pragma unroll
            for (int off = LPR / 2; off > 0; off >>= 1) {
                sr[r] += __shfl_xor_sync(0xffffffffu, sr[r], off);
                si[r] += __shfl_xor_sync(0xffffffffu, si[r], off);
            }
            const int row = rbase + r * G + g;
            if (q == 0 && (FULL || row < P.N)) {
                T s = (P.dagger && row >= P.nvec) ? (T)-1 : (T)1;
                T* o = out + ((long long)X * P.N + row) * 2;
                o[0] = s * sr[r];
                o[1] = s * si[r];
            }
        }
    }
}

template <typename T, int LPR, int CPL, int R>
static void launch_coarse(T* out, const T* in, const T* A, CoarseParams P, cudaStream_t st) {
    constexpr int G = 32 / LPR;
    P.ntile = (P.N + G * R - 1) / (G * R);
    // row tiles per warp: as many as possible (the nine source slices are loaded once per warp) while the grid
    // still has several waves of warps (>= 148 SMs x 256 warp tasks)
    int tpw = g_knobs.coarse_rows_per_warp > 0 ? g_knobs.coarse_rows_per_warp : P.ntile;
    if (tpw > P.ntile) tpw = P.ntile;
    while (tpw > 1 && (P.ntile % tpw != 0 ||
                       (g_knobs.coarse_rows_per_warp <= 0 && (long long)P.Vc * (P.ntile / tpw) < 148LL * 256)))
        tpw--;
    P.tpw = tpw;
    P.ntask = (long long)P.Vc * (P.ntile / tpw);
    int warps = g_knobs.coarse_warps > 0 ? g_knobs.coarse_warps : 4;
    if (warps > 8) warps = 8;
    const long long grid = (P.ntask + warps - 1) / warps;
    const bool full = (P.N % (G * R) == 0) && (P.RV == LPR * CPL);
    if (full) k_coarse<T, LPR, CPL, R, true><<<(unsigned)grid, warps * 32, 0, st>>>(out, in, A, P);
    else k_coarse<T, LPR, CPL, R, false><<<(unsigned)grid, warps * 32, 0, st>>>(out, in, A, P);
}

template <typename T>
static int coarse_call(T* out, const T* in, const T* A, const int cdims[4], int nvec, unsigned flags, void* stream,
                       const char* what) {
    clear_error();
    if (!out || !in || !A || check_dims(cdims) || nvec < 1) {
        set_error("%s: null pointer, non-positive dim or nvec < 1", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(out) || !aligned16(in) || !aligned16(A)) {
        set_error("%s: pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    if (out == in) {
        set_error("%s: out must not alias in", what);
        return LQCD_EINVAL;
    }
    if (flags & ~LQCD_DAGGER) {
        set_error("%s: unknown flag bits 0x%x", what, flags);
        return LQCD_EINVAL;
    }
    CoarseParams P;
    for (int mu = 0; mu < 4; mu++) {
        if (cdims[mu] < 2) {
            set_error("%s: coarse extent %d < 2 in direction %d", what, cdims[mu], mu);
            return LQCD_EINVAL;
        }
        P.Lc[mu] = cdims[mu];
    }
    if (volume(cdims) > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    constexpr int NV = VecOf<T>::NV;
    P.Vc = (int)volume(cdims);
    P.nvec = nvec;
    P.N = 2 * nvec;
    P.RV = 2 * P.N / NV;
    P.dagger = (flags & LQCD_DAGGER) ? 1 : 0;
    cudaStream_t st = (cudaStream_t)stream;
    const int RV = P.RV;
    if (RV > 128) {
        set_error("%s: nvec = %d outside the compiled range (row longer than 128 vec16)", what, nvec);
        return LQCD_EUNSUPPORTED;
    }
    if (RV <= 1) launch_coarse<T, 1, 1, 2>(out, in, A, P, st);
    else if (RV <= 2) launch_coarse<T, 2, 1, 2>(out, in, A, P, st);
    else if (RV <= 4) launch_coarse<T, 4, 1, 2>(out, in, A, P, st);
    else if (RV <= 8) launch_coarse<T, 8, 1, 2>(out, in, A, P, st);
    else if (RV <= 16) launch_coarse<T, 16, 1, 2>(out, in, A, P, st);
    else if (RV <= 32) {
        if (g_knobs.coarse_R == 1) launch_coarse<T, 32, 1, 1>(out, in, A, P, st);
        else if (g_knobs.coarse_R == 4) launch_coarse<T, 32, 1, 4>(out, in, A, P, st);
        else launch_coarse<T, 32, 1, 2>(out, in, A, P, st);
    }
    else if (RV <= 64) launch_coarse<T, 32, 2, 1>(out, in, A, P, st);
    else if (RV <= 96) launch_coarse<T, 32, 3, 1>(out, in, A, P, st);
    else launch_coarse<T, 32, 4, 1>(out, in, A, P, st);
    count_launch();
    return check_launch(what);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {
int lqcd_coarse_mult_f32(float* out, const float* in, const float* A, const int cdims[4], int nvec, unsigned flags,
                         void* stream) {
    return coarse_call<float>(out, in, A, cdims, nvec, flags, stream, "lqcd_coarse_mult_f32");
}
int lqcd_coarse_mult_f64(double* out, const double* in, const double* A, const int cdims[4], int nvec, unsigned flags,
                         void* stream) {
    return coarse_call<double>(out, in, A, cdims, nvec, flags, stream, "lqcd_coarse_mult_f64");
}
}
