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
    unsigned part_mask;  // sharded variants only: bit mu = direction mu is partitioned over ranks
    int nsites;          // sites the grid enumerates: Vc, or the face volume in MODE 2
    int face;            // MODE 2: the face 2 mu + dir this launch completes
};

// received faces of the sharded operator (MODE 2): face 2 mu + dir, [face site][N complex]
struct CoarseFaces {
    const void* p[8];
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
// MODE 0: the operator.  Sharded variants (halo exchange on the coarse lattice): MODE 1 = interior
// pass, the blocks of hops that leave the local lattice in a partitioned direction act on zero (the source is not
// read); MODE 2 = boundary completion, one launch per face over its sites only: out += the block of the hop that leaves
// through that face, applied to the received face.
template <typename T, int LPR, int CPL, int R, bool FULL, int MODE = 0>
__global__ void __launch_bounds__(256, 2) k_coarse(T* __restrict__ out, const T* __restrict__ in, const T* __restrict__ A,
                                                CoarseParams P, CoarseFaces F = CoarseFaces()) {
    constexpr int NV = VecOf<T>::NV;
    constexpr int CPV = NV / 2;  // complex per vec16
    constexpr int G = 32 / LPR;  // rows side by side in a warp
    const int lane = threadIdx.x & 31;
    const int g = lane / LPR, q = lane % LPR;
    const long long task = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (task >= P.ntask) return;
    const int wps = P.ntile / P.tpw;  // warps per site
    int X = (int)(task / wps);  // MODE 2: the face site
    const int tile0 = (int)(task % wps) * P.tpw;

    // the nine source sites
    int src[9];
    unsigned cut = 0;  // MODE 1: bit d = hop d leaves the local lattice in a partitioned direction
    int blk0 = 0;      // MODE 2: the one block this launch applies (slot 0 of the arrays below)
    {
        int xc[4];
        const int stride[4] = {1, P.Lc[0], P.Lc[0] * P.Lc[1], P.Lc[0] * P.Lc[1] * P.Lc[2]};
        if (MODE == 2) {
            // one launch per face: site from the face index; the only live block is the hop that leaves through it
            // (X_mu = Lc - 1: forward hop d = 1 + 2 mu, served by face 2 mu + 1; X_mu = 0: d = 2 + 2 mu, face 2 mu)
            const int mu = P.face >> 1, dir = P.face & 1, f = X;
            int rem = f;
            X = 0;
#pragma unroll
            for (int nu = 0; nu < 4; nu++) {
                if (nu == mu) {
                    xc[nu] = dir ? P.Lc[nu] - 1 : 0;
                } else {
                    xc[nu] = rem % P.Lc[nu];
                    rem /= P.Lc[nu];
                }
                X += xc[nu] * stride[nu];
            }
            blk0 = dir ? 1 + 2 * mu : 2 + 2 * mu;
            src[0] = f;
        } else {
            int rem = X;
            xc[0] = rem % P.Lc[0]; rem /= P.Lc[0];
            xc[1] = rem % P.Lc[1]; rem /= P.Lc[1];
            xc[2] = rem % P.Lc[2]; rem /= P.Lc[2];
            xc[3] = rem;
            src[0] = X;
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                src[1 + 2 * mu] = (xc[mu] == P.Lc[mu] - 1) ? X - (P.Lc[mu] - 1) * stride[mu] : X + stride[mu];
                src[2 + 2 * mu] = (xc[mu] == 0) ? X + (P.Lc[mu] - 1) * stride[mu] : X - stride[mu];
            }
        }
        if (MODE == 1) {
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                if (!((P.part_mask >> mu) & 1)) continue;
                if (xc[mu] == P.Lc[mu] - 1) cut |= 1u << (1 + 2 * mu);
                if (xc[mu] == 0) cut |= 1u << (2 + 2 * mu);
            }
        }
    }
    constexpr int ND = MODE == 2 ? 1 : 9;  // blocks per site in this pass
    // does the source of slot d take part in this pass?
    auto live = [&](int d) -> bool { return MODE == 1 ? !((cut >> d) & 1) : true; };
    // my slices of the source vectors (with the Gamma5c sign of the column for the dagger variant)
    V16<T> xv[ND][CPL];
#pragma unroll
    for (int d = 0; d < ND; d++)
#pragma unroll
        for (int c = 0; c < CPL; c++) {
            const int v = q + LPR * c;
            if ((FULL || v < P.RV) && live(d)) {
                const T* from = MODE == 2 ? static_cast<const T*>(F.p[0]) : in;  // the launch's face
                xv[d][c] = ld16(from + ((long long)src[d] * P.RV + v) * NV);
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

    const T* Asite = A + ((long long)X * 9 + blk0) * P.N * P.RV * NV;
    for (int t = 0; t < P.tpw; t++) {
        const int rbase = (tile0 + t) * (G * R);
        T sr[R], si[R];
#pragma unroll
        for (int r = 0; r < R; r++) sr[r] = si[r] = 0;
        // issue all loads of the tile first (R * 9 * CPL independent 16-byte requests per lane)
        V16<T> a[R][ND][CPL];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int row = rbase + r * G + g;
#pragma unroll
            for (int d = 0; d < ND; d++)
#pragma unroll
                for (int c = 0; c < CPL; c++) {
                    const int v = q + LPR * c;
                    // (MODE 1 streams the blocks of cut hops too -- their sources are zero: a per-block predicate
                    // breaks the batch of unconditional loads and costs 12 %, the skipped bytes would save < 1 %)
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
            for (int d = 0; d < ND; d++)
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
                if (MODE == 2) {
                    o[0] += s * sr[r];
                    o[1] += s * si[r];
                } else {
                    o[0] = s * sr[r];
                    o[1] = s * si[r];
                }
            }
        }
    }
}

template <typename T, int LPR, int CPL, int R, int MODE>
static void launch_coarse_mode(T* out, const T* in, const T* A, CoarseParams P, cudaStream_t st,
                               const CoarseFaces& F) {
    constexpr int G = 32 / LPR;
    P.ntile = (P.N + G * R - 1) / (G * R);
    // row tiles per warp: as many as possible (the nine source slices are loaded once per warp) while the grid
    // still has several waves of warps (>= 148 SMs x 256 warp tasks)
    // (the thin per-face launches of MODE 2 amortise the per-warp set-up over more rows: one wave of 32 warps per SM)
    const long long min_tasks = MODE == 2 ? 148LL * 32 : 148LL * 256;
    int tpw = g_knobs.coarse_rows_per_warp > 0 ? g_knobs.coarse_rows_per_warp : P.ntile;
    if (tpw > P.ntile) tpw = P.ntile;
    while (tpw > 1 && (P.ntile % tpw != 0 ||
                       (g_knobs.coarse_rows_per_warp <= 0 && (long long)P.nsites * (P.ntile / tpw) < min_tasks)))
        tpw--;
    P.tpw = tpw;
    P.ntask = (long long)P.nsites * (P.ntile / tpw);
    int warps = g_knobs.coarse_warps > 0 ? g_knobs.coarse_warps : 4;
    if (warps > 8) warps = 8;
    const long long grid = (P.ntask + warps - 1) / warps;
    const bool full = (P.N % (G * R) == 0) && (P.RV == LPR * CPL);
    if (full) k_coarse<T, LPR, CPL, R, true, MODE><<<(unsigned)grid, warps * 32, 0, st>>>(out, in, A, P, F);
    else k_coarse<T, LPR, CPL, R, false, MODE><<<(unsigned)grid, warps * 32, 0, st>>>(out, in, A, P, F);
}

template <typename T, int LPR, int CPL, int R>
static void launch_coarse(T* out, const T* in, const T* A, const CoarseParams& P, cudaStream_t st, int mode,
                          const CoarseFaces& F) {
    if (mode == 0) launch_coarse_mode<T, LPR, CPL, R, 0>(out, in, A, P, st, F);
    else if (mode == 1) launch_coarse_mode<T, LPR, CPL, R, 1>(out, in, A, P, st, F);
    else launch_coarse_mode<T, LPR, CPL, R, 2>(out, in, A, P, st, F);
}

// mode 0: D_c; mode 1: interior pass of the sharded operator; mode 2: its boundary completion (in = NULL, sources from
// recv[8], out accumulated)
template <typename T>
static int coarse_call(T* out, const T* in, const T* A, const int cdims[4], int nvec, unsigned flags, void* stream,
                       const char* what, int mode = 0, unsigned part_mask = 0, const T* const* recv = nullptr) {
    clear_error();
    if (mode == 2 && !in) in = A;  // never read in mode 2; keeps the checks below uniform
    if (part_mask > 15u || (mode == 2 && !recv)) {
        set_error("%s: bad part_mask 0x%x or null recv", what, part_mask);
        return LQCD_EINVAL;
    }
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
    CoarseFaces F;
    for (int i = 0; i < 8; i++) F.p[i] = nullptr;
    for (int mu = 0; mu < 4; mu++) {
        const bool part = (part_mask >> mu) & 1;
        if (cdims[mu] < 2 && !part) {  // (a partitioned direction may be one site thick: both hops leave)
            set_error("%s: coarse extent %d < 2 in direction %d", what, cdims[mu], mu);
            return LQCD_EINVAL;
        }
        P.Lc[mu] = cdims[mu];
        if (mode == 2 && part)
            for (int dir = 0; dir < 2; dir++) {
                if (!recv[2 * mu + dir] || !aligned16(recv[2 * mu + dir])) {
                    set_error("%s: recv[%d] is null or not 16-byte aligned", what, 2 * mu + dir);
                    return LQCD_EINVAL;
                }
                F.p[2 * mu + dir] = recv[2 * mu + dir];
            }
    }
    P.part_mask = part_mask;
    if (mode == 2 && !part_mask) return LQCD_OK;
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
    CoarseFaces Fl = F;  // MODE 2: slot 0 = the face of the launch
    auto launch = [&]() {
        if (RV <= 1) launch_coarse<T, 1, 1, 2>(out, in, A, P, st, mode, Fl);
        else if (RV <= 2) launch_coarse<T, 2, 1, 2>(out, in, A, P, st, mode, Fl);
        else if (RV <= 4) launch_coarse<T, 4, 1, 2>(out, in, A, P, st, mode, Fl);
        else if (RV <= 8) launch_coarse<T, 8, 1, 2>(out, in, A, P, st, mode, Fl);
        else if (RV <= 16) launch_coarse<T, 16, 1, 2>(out, in, A, P, st, mode, Fl);
        else if (RV <= 32) {
            if (g_knobs.coarse_R == 1) launch_coarse<T, 32, 1, 1>(out, in, A, P, st, mode, Fl);
            else if (g_knobs.coarse_R == 4 || (mode == 2 && g_knobs.coarse_R == 0))  // thin launch: more rows in flight
                launch_coarse<T, 32, 1, 4>(out, in, A, P, st, mode, Fl);
            else launch_coarse<T, 32, 1, 2>(out, in, A, P, st, mode, Fl);
        }
        else if (RV <= 64) launch_coarse<T, 32, 2, 1>(out, in, A, P, st, mode, Fl);
        else if (RV <= 96) launch_coarse<T, 32, 3, 1>(out, in, A, P, st, mode, Fl);
        else launch_coarse<T, 32, 4, 1>(out, in, A, P, st, mode, Fl);
        count_launch();
    };
    P.nsites = P.Vc;
    P.face = 0;
    if (mode != 2) {
        launch();
    } else {  // one launch per face, in face order (a site on several faces is completed in a fixed order)
        for (int face = 0; face < 8; face++) {
            if (!((part_mask >> (face >> 1)) & 1)) continue;
            P.face = face;
            Fl.p[0] = F.p[face];
            P.nsites = P.Vc / P.Lc[face >> 1];
            launch();
        }
    }
    return check_launch(what);
}

// ---- sharded coarse operator: the faces ("same pattern on the coarse lattice, N complex per face
// site") -- face 2 mu + dir = the coarse vectors of the sites with X_mu = 0 (dir 0) / Lc_mu - 1 (dir 1), face site =
// lexicographic index of the other three coordinates, [face site][N complex].
template <typename T>
__global__ void __launch_bounds__(256) k_coarse_halo_pack(CoarseFaces send_c, const T* __restrict__ in, CoarseParams P) {
    constexpr int NV = VecOf<T>::NV;
    const int face = blockIdx.y, mu = face >> 1, dir = face & 1;
    if (!((P.part_mask >> mu) & 1)) return;
    T* buf = static_cast<T*>(const_cast<void*>(send_c.p[face]));
    const long long n = (long long)(P.Vc / P.Lc[mu]) * P.RV;  // vec16 of this face
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        int f = (int)(i / P.RV);
        const int v = (int)(i - (long long)f * P.RV);
        int X = 0, stride = 1;
#pragma unroll
        for (int nu = 0; nu < 4; nu++) {
            int c;
            if (nu == mu) {
                c = dir ? P.Lc[mu] - 1 : 0;
            } else {
                c = f % P.Lc[nu];
                f /= P.Lc[nu];
            }
            X += c * stride;
            stride *= P.Lc[nu];
        }
        st16(buf + i * NV, ld16(in + ((long long)X * P.RV + v) * NV));
    }
}

template <typename T>
static int coarse_halo_pack_call(T* const send[8], const T* in, const int cdims[4], int nvec, unsigned part_mask,
                                 void* stream, const char* what) {
    clear_error();
    if (!send || !in || check_dims(cdims) || nvec < 1 || part_mask > 15u || !aligned16(in)) {
        set_error("%s: null or misaligned pointer, non-positive dim, nvec < 1 or part_mask 0x%x", what, part_mask);
        return LQCD_EINVAL;
    }
    if (volume(cdims) > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    constexpr int NV = VecOf<T>::NV;
    CoarseParams P;
    CoarseFaces F;
    P.Vc = (int)volume(cdims);
    P.nvec = nvec;
    P.N = 2 * nvec;
    P.RV = 2 * P.N / NV;
    P.part_mask = part_mask;
    long long nmax = 0;
    for (int mu = 0; mu < 4; mu++) {
        P.Lc[mu] = cdims[mu];
        for (int dir = 0; dir < 2; dir++) {
            F.p[2 * mu + dir] = nullptr;
            if (!((part_mask >> mu) & 1)) continue;
            if (!send[2 * mu + dir] || !aligned16(send[2 * mu + dir])) {
                set_error("%s: send[%d] is null or not 16-byte aligned", what, 2 * mu + dir);
                return LQCD_EINVAL;
            }
            F.p[2 * mu + dir] = send[2 * mu + dir];
            const long long n = (long long)(P.Vc / cdims[mu]) * P.RV;
            nmax = n > nmax ? n : nmax;
        }
    }
    if (!part_mask) return LQCD_OK;
    long long gx = (nmax + 255) / 256;
    if (gx > 148 * 8) gx = 148 * 8;
    k_coarse_halo_pack<T><<<dim3((unsigned)gx, 8), 256, 0, (cudaStream_t)stream>>>(F, in, P);
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

size_t lqcd_coarse_halo_face_reals(const int cdims[4], int nvec, int mu) {
    if (check_dims(cdims) || nvec < 1 || mu < 0 || mu > 3) return 0;
    return (size_t)(volume(cdims) / cdims[mu]) * 4 * (size_t)nvec;
}
int lqcd_coarse_halo_pack_f32(float* const send[8], const float* in, const int cdims[4], int nvec, unsigned part_mask,
                              void* stream) {
    return coarse_halo_pack_call<float>(send, in, cdims, nvec, part_mask, stream, "lqcd_coarse_halo_pack_f32");
}
int lqcd_coarse_halo_pack_f64(double* const send[8], const double* in, const int cdims[4], int nvec,
                              unsigned part_mask, void* stream) {
    return coarse_halo_pack_call<double>(send, in, cdims, nvec, part_mask, stream, "lqcd_coarse_halo_pack_f64");
}
int lqcd_coarse_mult_interior_f32(float* out, const float* in, const float* A, const int cdims[4], int nvec,
                                  unsigned part_mask, unsigned flags, void* stream) {
    return coarse_call<float>(out, in, A, cdims, nvec, flags, stream, "lqcd_coarse_mult_interior_f32", 1, part_mask);
}
int lqcd_coarse_mult_interior_f64(double* out, const double* in, const double* A, const int cdims[4], int nvec,
                                  unsigned part_mask, unsigned flags, void* stream) {
    return coarse_call<double>(out, in, A, cdims, nvec, flags, stream, "lqcd_coarse_mult_interior_f64", 1, part_mask);
}
int lqcd_coarse_halo_add_f32(float* out, const float* const recv[8], const float* A, const int cdims[4], int nvec,
                             unsigned part_mask, unsigned flags, void* stream) {
    return coarse_call<float>(out, nullptr, A, cdims, nvec, flags, stream, "lqcd_coarse_halo_add_f32", 2, part_mask,
                              recv);
}
int lqcd_coarse_halo_add_f64(double* out, const double* const recv[8], const double* A, const int cdims[4], int nvec,
                             unsigned part_mask, unsigned flags, void* stream) {
    return coarse_call<double>(out, nullptr, A, cdims, nvec, flags, stream, "lqcd_coarse_halo_add_f64", 2, part_mask,
                               recv);
}
}
