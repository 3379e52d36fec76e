// fermion.cuh -- device building blocks shared by the fine-operator kernels (wilson_clover.cu) and the set-up
// kernels (setup.cu): native spinor / link access, spin projection and reconstruction in the chiral basis of
// DESIGN.md, SU(3) times half-spinor.
#pragma once
#include "common.cuh"
#include "layout.cuh"

namespace lqcd {

// ---- loads --------------------------------------------------------------------------------------------
// G64: 64-byte L2 fetch granularity (even/odd-domain mode, see common.cuh)
template <typename T, bool G64 = false>
__device__ __forceinline__ void load_spinor(T p[24], const T* __restrict__ f, int s) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
    const T* base = f + ((long long)(s >> 5) * NJ * CH + (s & 31)) * NV;
#pragma unroll
    for (int j = 0; j < NJ; j++) {
        V16<T> v = G64 ? ld16_g64(base + (long long)j * CH * NV) : ld16(base + (long long)j * CH * NV);
#pragma unroll
        for (int q = 0; q < NV; q++) p[j * NV + q] = v.r[q];
    }
}

template <typename T> __device__ __forceinline__ void store_spinor(T* __restrict__ f, int s, const T p[24]) {
    constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
    T* base = f + ((long long)(s >> 5) * NJ * CH + (s & 31)) * NV;
#pragma unroll
    for (int j = 0; j < NJ; j++) {
        V16<T> v;
#pragma unroll
        for (int q = 0; q < NV; q++) v.r[q] = p[j * NV + q];
        st16_stream(base + (long long)j * CH * NV, v);
    }
}

// link U_mu(s) as 18 reals u[2*(3a+b)+reim]; with L12 the third row is conj(row0 x row1)
template <typename T, bool L12, bool G64 = false>
__device__ __forceinline__ void load_link(T u[18], const T* __restrict__ U, int s, int mu) {
    constexpr int NV = VecOf<T>::NV;
    const long long chunk = s >> 5;
    const int lane = s & 31;
    if (L12) {
        const T* base = U + (chunk * 4 + mu) * (12LL * CH) + lane * NV;
#pragma unroll
        for (int j = 0; j < 12 / NV; j++) {
            V16<T> v = G64 ? ld16_g64(base + j * CH * NV) : ld16(base + j * CH * NV);
#pragma unroll
            for (int q = 0; q < NV; q++) u[j * NV + q] = v.r[q];
        }
        // row2 = conj(row0 x row1)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
            const T ar = u[2 * c1], ai = u[2 * c1 + 1];          // row0[c1]
            const T br = u[6 + 2 * c2], bi = u[6 + 2 * c2 + 1];  // row1[c2]
            const T cr = u[2 * c2], ci = u[2 * c2 + 1];          // row0[c2]
            const T dr = u[6 + 2 * c1], di = u[6 + 2 * c1 + 1];  // row1[c1]
            u[12 + 2 * c] = (ar * br - ai * bi) - (cr * dr - ci * di);
            u[12 + 2 * c + 1] = -((ar * bi + ai * br) - (cr * di + ci * dr));
        }
    } else {
        constexpr int NFULL = 18 / NV;
        const T* base = U + (chunk * 4 + mu) * (18LL * CH);
#pragma unroll
        for (int j = 0; j < NFULL; j++) {
            V16<T> v = G64 ? ld16_g64(base + (j * CH + lane) * NV) : ld16(base + (j * CH + lane) * NV);
#pragma unroll
            for (int q = 0; q < NV; q++) u[j * NV + q] = v.r[q];
        }
        if (NFULL * NV < 18) {  // f32: reals 16, 17 in a float2 row
            const T* tail = base + NFULL * NV * CH + lane * 2;
            const float2 v = *reinterpret_cast<const float2*>(tail);
            u[16] = (T)v.x;
            u[17] = (T)v.y;
        }
    }
}

// ---- spin projection / reconstruction (chiral basis; table in DESIGN.md "Spin projectors") ------------
// SGN = -1: (1 - g_mu), SGN = +1: (1 + g_mu).  h[2][3] complex stored as h[sp*6 + 2c + reim].
template <int MU, int SGN, typename T> __device__ __forceinline__ void project(T h[12], const T p[24]) {
    constexpr T sg = (T)SGN;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const T p0r = p[2 * c], p0i = p[2 * c + 1];
        const T p1r = p[6 + 2 * c], p1i = p[6 + 2 * c + 1];
        const T p2r = p[12 + 2 * c], p2i = p[12 + 2 * c + 1];
        const T p3r = p[18 + 2 * c], p3i = p[18 + 2 * c + 1];
        if (MU == 0) {  // h0 = p0 - sg i p3 ; h1 = p1 - sg i p2
            h[2 * c] = p0r + sg * p3i;
            h[2 * c + 1] = p0i - sg * p3r;
            h[6 + 2 * c] = p1r + sg * p2i;
            h[6 + 2 * c + 1] = p1i - sg * p2r;
        } else if (MU == 1) {  // h0 = p0 - sg p3 ; h1 = p1 + sg p2
            h[2 * c] = p0r - sg * p3r;
            h[2 * c + 1] = p0i - sg * p3i;
            h[6 + 2 * c] = p1r + sg * p2r;
            h[6 + 2 * c + 1] = p1i + sg * p2i;
        } else if (MU == 2) {  // h0 = p0 - sg i p2 ; h1 = p1 + sg i p3
            h[2 * c] = p0r + sg * p2i;
            h[2 * c + 1] = p0i - sg * p2r;
            h[6 + 2 * c] = p1r - sg * p3i;
            h[6 + 2 * c + 1] = p1i + sg * p3r;
        } else {  // h0 = p0 + sg p2 ; h1 = p1 + sg p3
            h[2 * c] = p0r + sg * p2r;
            h[2 * c + 1] = p0i + sg * p2i;
            h[6 + 2 * c] = p1r + sg * p3r;
            h[6 + 2 * c + 1] = p1i + sg * p3i;
        }
    }
}

// acc += ph * (1 + SGN g_mu)-reconstruction of g (g = link times projected half spinor)
template <int MU, int SGN, typename T> __device__ __forceinline__ void reconstruct(T acc[24], const T g[12], T ph) {
    const T sp = (T)SGN * ph;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const T g0r = g[2 * c], g0i = g[2 * c + 1], g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        acc[2 * c] = fma(ph, g0r, acc[2 * c]);
        acc[2 * c + 1] = fma(ph, g0i, acc[2 * c + 1]);
        acc[6 + 2 * c] = fma(ph, g1r, acc[6 + 2 * c]);
        acc[6 + 2 * c + 1] = fma(ph, g1i, acc[6 + 2 * c + 1]);
        if (MU == 0) {  // r2 = sg i g1 ; r3 = sg i g0
            acc[12 + 2 * c] = fma(-sp, g1i, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(sp, g1r, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(-sp, g0i, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(sp, g0r, acc[18 + 2 * c + 1]);
        } else if (MU == 1) {  // r2 = sg g1 ; r3 = -sg g0
            acc[12 + 2 * c] = fma(sp, g1r, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(sp, g1i, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(-sp, g0r, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(-sp, g0i, acc[18 + 2 * c + 1]);
        } else if (MU == 2) {  // r2 = sg i g0 ; r3 = -sg i g1
            acc[12 + 2 * c] = fma(-sp, g0i, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(sp, g0r, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(sp, g1i, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(-sp, g1r, acc[18 + 2 * c + 1]);
        } else {  // r2 = sg g0 ; r3 = sg g1
            acc[12 + 2 * c] = fma(sp, g0r, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(sp, g0i, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(sp, g1r, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(sp, g1i, acc[18 + 2 * c + 1]);
        }
    }
}

// g = U h (FWD) or U^dag h (!FWD) for the two colour vectors of the half spinor
template <bool FWD, typename T> __device__ __forceinline__ void su3_mult(T g[12], const T u[18], const T h[12]) {
#pragma unroll
    for (int sp = 0; sp < 2; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            T gr = 0, gi = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const T hr = h[sp * 6 + 2 * b], hi = h[sp * 6 + 2 * b + 1];
                if (FWD) {
                    const T ur = u[2 * (3 * a + b)], ui = u[2 * (3 * a + b) + 1];
                    gr = fma(ur, hr, gr);
                    gr = fma(-ui, hi, gr);
                    gi = fma(ur, hi, gi);
                    gi = fma(ui, hr, gi);
                } else {  // conj(U_ba)
                    const T ur = u[2 * (3 * b + a)], ui = u[2 * (3 * b + a) + 1];
                    gr = fma(ur, hr, gr);
                    gr = fma(ui, hi, gr);
                    gi = fma(ur, hi, gi);
                    gi = fma(-ui, hr, gi);
                }
            }
            g[sp * 6 + 2 * a] = gr;
            g[sp * 6 + 2 * a + 1] = gi;
        }
}

// out6 += Hermitian 6x6 block (36 reals: 6 diagonal, 15 complex strictly-lower row-major) times in6
template <typename T> __device__ __forceinline__ void herm6_madd(T out[12], const T cl[36], const T in[12]) {
#pragma unroll
    for (int k = 0; k < 6; k++) {
        T sr = fma(cl[k], in[2 * k], out[2 * k]);
        T si = fma(cl[k], in[2 * k + 1], out[2 * k + 1]);
#pragma unroll
        for (int l = 0; l < 6; l++) {
            if (l == k) continue;
            const T xr = in[2 * l], xi = in[2 * l + 1];
            if (l < k) {  // L_kl
                const T ar = cl[6 + 2 * tri(k, l)], ai = cl[6 + 2 * tri(k, l) + 1];
                sr = fma(ar, xr, sr);
                sr = fma(-ai, xi, sr);
                si = fma(ar, xi, si);
                si = fma(ai, xr, si);
            } else {  // conj(L_lk)
                const T ar = cl[6 + 2 * tri(l, k)], ai = cl[6 + 2 * tri(l, k) + 1];
                sr = fma(ar, xr, sr);
                sr = fma(ai, xi, sr);
                si = fma(ar, xi, si);
                si = fma(-ai, xr, si);
            }
        }
        out[2 * k] = sr;
        out[2 * k + 1] = si;
    }
}

template <typename T, bool G64 = false>
__device__ __forceinline__ void load_clover_block(T cl[36], const T* __restrict__ C, int s, int chi) {
    constexpr int NV = VecOf<T>::NV, NJ = 72 / NV;
    const T* base = C + (((long long)(s >> 5) * NJ + chi * (36 / NV)) * CH + (s & 31)) * NV;
#pragma unroll
    for (int j = 0; j < 36 / NV; j++) {
        V16<T> v = G64 ? ld16_stream_g64(base + (long long)j * CH * NV) : ld16_stream(base + (long long)j * CH * NV);
#pragma unroll
        for (int q = 0; q < NV; q++) cl[j * NV + q] = v.r[q];
    }
}

}  // namespace lqcd
