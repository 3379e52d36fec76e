// common.cuh -- shared plumbing of the sm_100a kernels: error reporting, argument checks,
// the 16-byte vector type per precision, cache-hinted loads/stores, lattice geometry.
// Product code: never includes or links anything under oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdarg.h>

#include "../../include/lqcd_b200.h"

namespace lqcd {

constexpr int CH = 32;  // sites per native chunk (one warp-wide row of vec16)

// ---- error reporting -------------------------------------------------------------------------
void set_error(const char* fmt, ...);
void clear_error();
void count_launch(int n = 1);
int check_launch(const char* what);  // cudaGetLastError -> LQCD_ECUDA / LQCD_OK

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline int check_dims(const int dims[4]) {
    if (!dims) return LQCD_EINVAL;
    for (int mu = 0; mu < 4; mu++)
        if (dims[mu] < 1) return LQCD_EINVAL;
    return LQCD_OK;
}
inline long long volume(const int d[4]) { return (long long)d[0] * d[1] * d[2] * d[3]; }
inline long long nchunks(const int d[4]) { return (volume(d) + CH - 1) / CH; }

// block must divide dims.  The aggregate-local operations (restrict, prolong, null-vector packing and
// orthonormalisation) accept any coarse extent >= 1 -- a rank of a sharded lattice may be one aggregate thick;
// whatever applies the periodic 9-point coarse stencil needs coarse extents >= 2 (reading Q8).
inline int check_block_local(const int dims[4], const int block[4], int nvec, int cdims[4]) {
    if (check_dims(dims) || !block || nvec < 1) return LQCD_EINVAL;
    for (int mu = 0; mu < 4; mu++) {
        if (block[mu] < 1 || dims[mu] % block[mu]) return LQCD_EINVAL;
        cdims[mu] = dims[mu] / block[mu];
    }
    return LQCD_OK;
}
inline int check_block(const int dims[4], const int block[4], int nvec, int cdims[4]) {
    if (check_block_local(dims, block, nvec, cdims)) return LQCD_EINVAL;
    for (int mu = 0; mu < 4; mu++)
        if (cdims[mu] < 2) return LQCD_EINVAL;
    return LQCD_OK;
}

// ---- per-device facts and one-time kernel attributes (a process may drive several devices) -----------
int max_optin_smem();  // cudaDevAttrMaxSharedMemoryPerBlockOptin of the current device
int sm_count();        // cudaDevAttrMultiProcessorCount of the current device
int current_device();
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (kernel instantiation, device): `done` is the call
// site's static bit mask of devices already served
template <typename Kern> inline void ensure_dynamic_smem(Kern kern, int bytes, unsigned long long& done) {
    const int d = current_device();
    if (d >= 0 && d < 64 && ((done >> d) & 1ull)) return;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (d >= 0 && d < 64) done |= 1ull << d;
}

// ---- 16-byte vectors ----------------------------------------------------------------------------
template <typename T> struct VecOf;
template <> struct VecOf<float> {
    typedef float4 type;
    static constexpr int NV = 4;
};
template <> struct VecOf<double> {
    typedef double2 type;
    static constexpr int NV = 2;
};

// A 16-byte register bundle addressable by compile-time index.
template <typename T> struct V16;
template <> struct alignas(16) V16<float> {
    float r[4];
};
template <> struct alignas(16) V16<double> {
    double r[2];
};

// Default-cached 128-bit load (L1 + L2): data with reuse (spinors, links).
template <typename T> __device__ __forceinline__ V16<T> ld16(const T* p) {
    return *reinterpret_cast<const V16<T>*>(p);
}
// The same with a 64-byte L2 fetch granularity.  By default a miss pulls the whole 128-byte line from HBM; when
// only alternate 64-byte halves of the lines are wanted (even/odd domains of 4 sites in x: 4 sites x 16 B) that
// doubles the DRAM traffic (measured: 713 -> 563 -> ~400 B/site as the loads are switched to .L2::64B).
template <typename T> __device__ __forceinline__ V16<T> ld16_g64(const T* p) {
    V16<T> v;
    if constexpr (sizeof(T) == 4)
        asm volatile("ld.global.L2::64B.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(v.r[0]), "=f"(v.r[1]), "=f"(v.r[2]), "=f"(v.r[3])
                     : "l"(p)
                     : "memory");  // an ordinary (coherent) load of memory the kernel may also store to
    else
        asm volatile("ld.global.L2::64B.v2.f64 {%0,%1}, [%2];" : "=d"(v.r[0]), "=d"(v.r[1]) : "l"(p) : "memory");
    return v;
}
template <typename T> __device__ __forceinline__ V16<T> ld16_stream_g64(const T* p) {
    V16<T> v;
    if constexpr (sizeof(T) == 4)
        asm volatile("ld.global.nc.L1::no_allocate.L2::64B.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(v.r[0]), "=f"(v.r[1]), "=f"(v.r[2]), "=f"(v.r[3])
                     : "l"(p));
    else
        asm volatile("ld.global.nc.L1::no_allocate.L2::64B.v2.f64 {%0,%1}, [%2];"
                     : "=d"(v.r[0]), "=d"(v.r[1])
                     : "l"(p));
    return v;
}
// Read-only, L1 no-allocate, L2 evict-first: data streamed exactly once (clover, coarse blocks, null vectors).
// (The plain .L2::evict_first qualifier exists only for 256-bit loads on sm_100a, hence the policy operand;
// createpolicy is loop-invariant and gets hoisted.)  The loads are `volatile` so that a batch of them written
// back to back stays back to back (front-loaded memory-level parallelism) instead of being sunk to their uses.
template <typename T> __device__ __forceinline__ V16<T> ld16_stream(const T* p);
__device__ __forceinline__ uint64_t evict_first_policy() {
    uint64_t pol;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
template <> __device__ __forceinline__ V16<float> ld16_stream<float>(const float* p) {
    V16<float> v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(v.r[0]), "=f"(v.r[1]), "=f"(v.r[2]), "=f"(v.r[3])
                 : "l"(p), "l"(evict_first_policy()));
    return v;
}
template <> __device__ __forceinline__ V16<double> ld16_stream<double>(const double* p) {
    V16<double> v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(v.r[0]), "=d"(v.r[1])
                 : "l"(p), "l"(evict_first_policy()));
    return v;
}
// Streaming store (written once, not re-read by this kernel).
template <typename T> __device__ __forceinline__ void st16_stream(T* p, const V16<T>& v);
template <> __device__ __forceinline__ void st16_stream<float>(float* p, const V16<float>& v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.r[0]), "f"(v.r[1]), "f"(v.r[2]),
                 "f"(v.r[3])
                 : "memory");
}
template <> __device__ __forceinline__ void st16_stream<double>(double* p, const V16<double>& v) {
    asm volatile("st.global.cs.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.r[0]), "d"(v.r[1]) : "memory");
}
template <typename T> __device__ __forceinline__ void st16(T* p, const V16<T>& v) {
    *reinterpret_cast<V16<T>*>(p) = v;
}

// ---- division by a run-time constant: q = n / d for 0 <= n with n * d < 2^32 (block and thread indices by lattice
// extents), as one multiply-high (+ one multiply-add for d = 1) instead of the ~20-instruction integer division.
// m = ceil(2^32 / d); floor(n m / 2^32) = floor(n / d) whenever n (m d - 2^32) < 2^32, which n d < 2^32 implies.
struct FastDiv {
    unsigned m;    // ceil(2^32 / d) for d >= 2, 0 for d = 1
    unsigned one;  // 1 if d == 1
    __host__ void set(int d) {
        one = d == 1;
        m = d == 1 ? 0u : (unsigned)((0x100000000ull + (unsigned)d - 1) / (unsigned)d);
    }
    __device__ __forceinline__ int div(int n) const { return (int)(__umulhi((unsigned)n, m) + (unsigned)n * one); }
};

// ---- internal range forms of the hot-path calls (host_api.cu pipelines a host vector through them slab by slab) -----
// canonical <-> native re-layout of the sites [s0, s1) (canonical index) of a spinor
template <typename T, bool UNPACK>
int spinor_range_call(T* dst, const T* src, const int dims[4], long long s0, long long s1, void* stream, const char* what);
// D (or D^dag) on the time slices [t0, t1) only; both multiples of fine_tile_extent_t(); canonical tile traversal
template <typename T>
int wilson_clover_slab_call(T* out, const T* in, const T* U, const T* clover, T kappa, const int dims[4], const int bc[4],
                            unsigned flags, int t0, int t1, void* stream, const char* what);
int fine_tile_extent_t(const int dims[4], const int bc[4], int real_bytes);  // extent in t of the fine kernel's CTA tile
// restrict / prolong on the aggregates (X, chi) with X in [X0, X1) only
template <typename T>
int restrict_range_call(T* out_c, const T* in_f, const T* v, const int dims[4], const int block[4], int nvec, long long X0,
                        long long X1, void* stream, const char* what);
template <typename T>
int prolong_range_call(T* out_f, const T* in_c, const T* v, const int dims[4], const int block[4], int nvec, long long X0,
                       long long X1, void* stream, const char* what);

// ---- geometry passed to kernels by value ---------------------------------------------------------
struct Geom {
    int L[4];        // fine dims
    int V;           // volume (fits in int: the largest supported lattice is < 2^31 sites)
};

}  // namespace lqcd
