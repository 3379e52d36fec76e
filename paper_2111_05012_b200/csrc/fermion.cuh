// fermion.cuh -- device building blocks shared by the fine-operator kernels (wilson_clover.cu) and the set-up
// kernels (setup.cu): native spinor / link access, spin projection and reconstruction in the chiral basis of
// DESIGN.md, SU(3) times half-spinor.
#pragma once
#include "common.cuh"
#include "layout.cuh"

namespace lqcd {

// ---- packed fp32 arithmetic (sm_100a: fma.rn.f32x2 = SASS FFMA2) ---------------------------------------------
// One FFMA2 does two IEEE fp32 FMAs (same rounding as two scalar fma()) for ONE issue slot; the FMA pipe's rate in
// flops is unchanged (measured: 73 TFLOP/s either way), so this halves the ISSUE cost of the complex arithmetic below,
// which is what the fp32 fine kernels are short of under a power-capped clock.  ptxas folds a scalar
// broadcast (a, a), a negated broadcast and a swapped pair (hi, lo) into operand modifiers of FFMA2 (R.F32, -R.F32,
// R.F32x2.LO_HI), so none of the pair constructors below costs an instruction as long as the two halves of a pair
// are produced and consumed consistently.  fp64 keeps the scalar code, and so does a kernel that asks for it with
// PACK = false: the shared-memory-resident domain solver, bound by LDS traffic at 4 warps per scheduler, was 1.5-2 %
// SLOWER packed (half the independent FMA chains per thread to cover the pipe latency with).
__device__ __forceinline__ float2 pk2(float lo, float hi) { return make_float2(lo, hi); }
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 sw2(float2 v) { return make_float2(v.y, v.x); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
template <typename T> struct is_f32 { static constexpr bool value = false; };
template <> struct is_f32<float> { static constexpr bool value = true; };

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
template <int MU, int SGN, typename T, bool PACK = true>
__device__ __forceinline__ void reconstruct(T acc[24], const T g[12], T ph) {
    const T sp = (T)SGN * ph;
    if constexpr (PACK && is_f32<T>::value) {
        // pairs over the two spin components of a chirality half: (acc[2c+ri], acc[6+2c+ri]) and (acc[12+2c+ri],
        // acc[18+2c+ri]); g comes from su3_mult in the same pairing, so every line is one FFMA2; lane by lane the
        // same fma as the scalar code below
        const float2 PH = bc2(ph), SP = bc2(sp), SN = bc2(-sp), SPN = pk2(sp, -sp), SNP = pk2(-sp, sp);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const float2 GR = pk2(g[2 * c], g[6 + 2 * c]), GI = pk2(g[2 * c + 1], g[6 + 2 * c + 1]);
            float2 A01r = pk2(acc[2 * c], acc[6 + 2 * c]), A01i = pk2(acc[2 * c + 1], acc[6 + 2 * c + 1]);
            float2 A23r = pk2(acc[12 + 2 * c], acc[18 + 2 * c]), A23i = pk2(acc[12 + 2 * c + 1], acc[18 + 2 * c + 1]);
            A01r = fma2(PH, GR, A01r);
            A01i = fma2(PH, GI, A01i);
            if (MU == 0) {  // r2 = sg i g1 ; r3 = sg i g0
                A23r = fma2(SN, sw2(GI), A23r);
                A23i = fma2(SP, sw2(GR), A23i);
            } else if (MU == 1) {  // r2 = sg g1 ; r3 = -sg g0
                A23r = fma2(SPN, sw2(GR), A23r);
                A23i = fma2(SPN, sw2(GI), A23i);
            } else if (MU == 2) {  // r2 = sg i g0 ; r3 = -sg i g1
                A23r = fma2(SNP, GI, A23r);
                A23i = fma2(SPN, GR, A23i);
            } else {  // r2 = sg g0 ; r3 = sg g1
                A23r = fma2(SP, GR, A23r);
                A23i = fma2(SP, GI, A23i);
            }
            acc[2 * c] = A01r.x, acc[6 + 2 * c] = A01r.y, acc[2 * c + 1] = A01i.x, acc[6 + 2 * c + 1] = A01i.y;
            acc[12 + 2 * c] = A23r.x, acc[18 + 2 * c] = A23r.y, acc[12 + 2 * c + 1] = A23i.x, acc[18 + 2 * c + 1] = A23i.y;
        }
        return;
    }
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
template <bool FWD, typename T, bool PACK = true>
__device__ __forceinline__ void su3_mult(T g[12], const T u[18], const T h[12]) {
    if constexpr (PACK && is_f32<T>::value) {
        // the two colour vectors of the half spinor ride in the two lanes: a link element is a broadcast operand, no
        // swap and no sign fix-up; lane by lane the same fma chain as the scalar code below
        float2 HR[3], HI[3];
#pragma unroll
        for (int b = 0; b < 3; b++) HR[b] = pk2(h[2 * b], h[6 + 2 * b]), HI[b] = pk2(h[2 * b + 1], h[6 + 2 * b + 1]);
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float2 GR = pk2(0.f, 0.f), GI = pk2(0.f, 0.f);
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const float ur = FWD ? u[2 * (3 * a + b)] : u[2 * (3 * b + a)];
                const float ui = FWD ? u[2 * (3 * a + b) + 1] : -u[2 * (3 * b + a) + 1];
                GR = fma2(bc2(ur), HR[b], GR);
                GR = fma2(bc2(-ui), HI[b], GR);
                GI = fma2(bc2(ur), HI[b], GI);
                GI = fma2(bc2(ui), HR[b], GI);
            }
            g[2 * a] = GR.x, g[6 + 2 * a] = GR.y, g[2 * a + 1] = GI.x, g[6 + 2 * a + 1] = GI.y;
        }
        return;
    }
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
template <typename T, bool PACK = true>
__device__ __forceinline__ void herm6_madd(T out[12], const T cl[36], const T in[12]) {
    if constexpr (PACK && is_f32<T>::value) {
        // (re, im) pairs: S collects a_r (x_r, x_i), Q collects +-a_i (x_i, x_r) (the swapped pair is an operand
        // modifier); out = (S.re - Q.re, S.im + Q.im).  13 instructions per row instead of 22; the two partial sums are
        // added at the end, so the rounding order differs from the scalar code (both are within the parity bars).
        float2 X[6];
#pragma unroll
        for (int l = 0; l < 6; l++) X[l] = pk2(in[2 * l], in[2 * l + 1]);
#pragma unroll
        for (int k = 0; k < 6; k++) {
            float2 S = fma2(bc2(cl[k]), X[k], pk2(out[2 * k], out[2 * k + 1]));
            float2 Q = pk2(0.f, 0.f);
#pragma unroll
            for (int l = 0; l < 6; l++) {
                if (l == k) continue;
                const int t = l < k ? tri(k, l) : tri(l, k);
                const float ar = cl[6 + 2 * t], ai = cl[6 + 2 * t + 1];
                S = fma2(bc2(ar), X[l], S);
                Q = fma2(bc2(l < k ? ai : -ai), sw2(X[l]), Q);
            }
            out[2 * k] = S.x - Q.x;
            out[2 * k + 1] = S.y + Q.y;
        }
        return;
    }
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
