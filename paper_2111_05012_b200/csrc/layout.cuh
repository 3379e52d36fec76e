// layout.cuh -- offsets (in reals) into the native device layouts documented in include/lqcd_b200.h.
// Used by the pack/unpack kernels with run-time indices and by the mult kernels with compile-time
// indices (everything folds to constants there).
#pragma once
#include "common.cuh"

namespace lqcd {

// ---- spinor: [chunk][j][lane] vec16 over 24 reals r = 2*(3 alpha + c) + reim -------------------------
template <typename T> __host__ __device__ __forceinline__ long long spinor_off(long long s, int r) {
    constexpr int NV = VecOf<T>::NV;
    const long long chunk = s >> 5;
    const int lane = (int)(s & 31);
    return ((chunk * (24 / NV) + r / NV) * CH + lane) * NV + r % NV;
}

// ---- gauge, 18 reals r = 2*(3a+b)+reim per (site, mu): [chunk][mu][rows] ---------------------------
// f32: 4 float4 rows (reals 0..15) then one float2 row (reals 16,17); f64: 9 double2 rows.
template <typename T> __host__ __device__ __forceinline__ long long gauge18_off(long long s, int mu, int r) {
    constexpr int NV = VecOf<T>::NV;
    constexpr int NFULL = 18 / NV;
    const long long chunk = s >> 5;
    const int lane = (int)(s & 31);
    const long long base = (chunk * 4 + mu) * (18LL * CH);
    if (r < NFULL * NV) return base + ((long long)(r / NV) * CH + lane) * NV + r % NV;
    return base + (long long)NFULL * NV * CH + lane * 2 + (r - NFULL * NV);
}
// ---- gauge, 12 reals (rows a = 0, 1): [chunk][mu][j][lane] vec16 -------------------------------------
template <typename T> __host__ __device__ __forceinline__ long long gauge12_off(long long s, int mu, int r) {
    constexpr int NV = VecOf<T>::NV;
    const long long chunk = s >> 5;
    const int lane = (int)(s & 31);
    const long long base = (chunk * 4 + mu) * (12LL * CH);
    return base + ((long long)(r / NV) * CH + lane) * NV + r % NV;
}

// ---- clover: 72 reals per site; per chi: 6 real diagonal, then 15 complex strictly-lower entries ----
// position of the lower-triangle entry (k, l), k > l, in row-major order
__host__ __device__ __forceinline__ constexpr int tri(int k, int l) { return k * (k - 1) / 2 + l; }
__host__ __device__ __forceinline__ constexpr int clover_diag_r(int chi, int k) { return 36 * chi + k; }
__host__ __device__ __forceinline__ constexpr int clover_low_r(int chi, int k, int l, int reim) {
    return 36 * chi + 6 + 2 * tri(k, l) + reim;
}
template <typename T> __host__ __device__ __forceinline__ long long clover_off(long long s, int r) {
    constexpr int NV = VecOf<T>::NV;
    const long long chunk = s >> 5;
    const int lane = (int)(s & 31);
    return ((chunk * (72 / NV) + r / NV) * CH + lane) * NV + r % NV;
}

// ---- null vectors: [X][chi][i][l][k] complex -----------------------------------------------------------
__host__ __device__ __forceinline__ long long nullvec_off(long long X, int chi, int i, int l, int k, int reim,
                                                          int nvec, int bv) {
    return (((((X * 2 + chi) * nvec + i) * (long long)bv + l) * 6 + k) * 2) + reim;
}

}  // namespace lqcd
