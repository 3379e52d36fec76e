// layout.cuh -- offsets (in reals) into the native device layouts documented in include/lqcd_b200.h.
// Used by the pack/unpack kernels with run-time indices and by the mult kernels with compile-time
// indices (everything folds to constants there).
#pragma once
#include "common.cuh"

#include "knobs.h"

namespace lqcd {

// ---- site order: the native position n of a lattice site; chunk = n >> 5, lane = n & 31 in every fine layout below ----
// Canonical order n = x + Lx (y + Ly (z + Lz t)) puts 32 consecutive x-sites (and their continuation in y) into a chunk:
// with 4-site-wide domains the sites of ONE domain are then alternate 64-byte halves of every 128-byte line, and a pass
// over the even (or odd) domains -- SAP's half sweeps and the residuals between them -- fetches half lines (DESIGN.md
// section 6.4).  TILED order makes a chunk a 4 x 4 x 2 tile of sites (x, y, z), tiles in lexicographic order (x tiles
// fastest): n = 32 (Tx + ntx (Ty + nty (Tz + ntz t))) + (x & 3) + 4 (y & 3) + 16 (z & 1).  A 4^4 domain is 8 whole
// chunks, every 512-byte row of a chunk belongs to one domain, and a warp that owns a tile reads whole lines.
// Used whenever Lx % 4 == Ly % 4 == Lz % 2 == 0 (all BASELINE configs); canonical order otherwise.  One parametrisation
// covers both (canonical = one tile as large as the lattice).  Layout-opaque to callers: only pack / unpack speak it.
struct SiteOrder {
    int w[4];       // n(x + mu) - n(x) inside a tile
    int T[4];       // ... from a tile to the next tile in direction mu
    int lmask[4];   // x & lmask = coordinate inside the tile
    int lmax[4];    // its largest value
    int lshift[4];  // x >> lshift = tile coordinate
    int edgef[4];   // n(x + mu) - n(x) across a tile edge
    int wrapf[4];   // n(x) - n(x + mu) across the lattice edge (periodic wrap)
    int Lm1[4];     // L - 1
    int L[3];
    int tiled;

    __host__ void set(const int dims[4]) {
        tiled = g_knobs.site_order >= 0 && dims[0] % 4 == 0 && dims[1] % 4 == 0 && dims[2] % 2 == 0;
        const int te[4] = {tiled ? 4 : dims[0], tiled ? 4 : dims[1], tiled ? 2 : dims[2], tiled ? 1 : dims[3]};
        int wacc = 1, tacc = tiled ? 32 : 0;
        for (int mu = 0; mu < 4; mu++) {
            const int nt = dims[mu] / te[mu];
            w[mu] = wacc;
            T[mu] = tacc;
            lmax[mu] = te[mu] - 1;
            lmask[mu] = tiled ? te[mu] - 1 : 0x7fffffff;
            lshift[mu] = tiled ? (te[mu] == 4 ? 2 : te[mu] == 2 ? 1 : 0) : 31;
            edgef[mu] = T[mu] - (te[mu] - 1) * w[mu];
            wrapf[mu] = (te[mu] - 1) * w[mu] + (nt - 1) * T[mu];
            Lm1[mu] = dims[mu] - 1;
            wacc *= te[mu];
            tacc *= nt;
        }
        for (int mu = 0; mu < 3; mu++) L[mu] = dims[mu];
    }
    __device__ __forceinline__ int index(int x0, int x1, int x2, int x3) const {
        return (x0 & lmask[0]) * w[0] + (x0 >> lshift[0]) * T[0] + (x1 & lmask[1]) * w[1] + (x1 >> lshift[1]) * T[1] +
               (x2 & lmask[2]) * w[2] + (x2 >> lshift[2]) * T[2] + (x3 & lmask[3]) * w[3] + (x3 >> lshift[3]) * T[3];
    }
    __device__ __forceinline__ int index(const int x[4]) const { return index(x[0], x[1], x[2], x[3]); }
    // position of the neighbour in direction +mu / -mu of the site at position n whose mu-coordinate is xmu
    __device__ __forceinline__ int fwd(int n, int mu, int xmu) const {
        return (xmu & lmask[mu]) != lmax[mu] ? n + w[mu] : (xmu == Lm1[mu] ? n - wrapf[mu] : n + edgef[mu]);
    }
    __device__ __forceinline__ int bwd(int n, int mu, int xmu) const {
        return (xmu & lmask[mu]) != 0 ? n - w[mu] : (xmu == 0 ? n + wrapf[mu] : n - edgef[mu]);
    }
    // from the canonical index s = x + Lx (y + Ly (z + Lz t)); exact divisions: for the kernels off the hot path
    __device__ __forceinline__ int from_canonical(int s) const {
        if (!tiled) return s;
        const int q0 = s / L[0], x0 = s - q0 * L[0];
        const int q1 = q0 / L[1], x1 = q0 - q1 * L[1];
        const int q2 = q1 / L[2], x2 = q1 - q2 * L[2];
        return index(x0, x1, x2, q2);
    }
};

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
