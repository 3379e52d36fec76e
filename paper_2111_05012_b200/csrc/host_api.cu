// host_api.cu -- end-to-end entry points on HOST right-hand sides (include/lqcd_b200.h, "end-to-end entry
// points"): H2D copy of the canonical vector, pack, the mult kernel, unpack, D2H copy, stream synchronise.
// The operator fields stay resident on the device in native layout.  fp32 (the multigrid parts of the paper run in
// single precision) and fp64 (the outer solver's precision).
#include "common.cuh"

namespace lqcd {
static inline size_t up256(size_t n) { return (n + 255) & ~(size_t)255; }
static int sync_or_error(cudaStream_t st, const char* what) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        set_error("%s: %s", what, cudaGetErrorString(e));
        return LQCD_ECUDA;
    }
    return LQCD_OK;
}
static int copy_or_error(void* dst, const void* src, size_t n, cudaMemcpyKind kind, cudaStream_t st, const char* what) {
    cudaError_t e = cudaMemcpyAsync(dst, src, n, kind, st);
    if (e != cudaSuccess) {
        set_error("%s: cudaMemcpyAsync: %s", what, cudaGetErrorString(e));
        return LQCD_ECUDA;
    }
    return LQCD_OK;
}
}  // namespace lqcd

using namespace lqcd;

namespace {
// the device calls of one precision
template <typename T> struct Dev;
template <> struct Dev<float> {
    static int pack(float* d, const float* s, const int* dims, void* st) { return lqcd_pack_spinor_f32(d, s, dims, st); }
    static int unpack(float* d, const float* s, const int* dims, void* st) { return lqcd_unpack_spinor_f32(d, s, dims, st); }
    static int fine(float* o, const float* i, const float* U, const float* cl, float k, const int* dims, const int* bc,
                    unsigned fl, void* st) { return lqcd_wilson_clover_mult_f32(o, i, U, cl, k, dims, bc, fl, st); }
    static int coarse(float* o, const float* i, const float* A, const int* cd, int nv, unsigned fl, void* st) {
        return lqcd_coarse_mult_f32(o, i, A, cd, nv, fl, st);
    }
    static int restrict_(float* o, const float* i, const float* v, const int* dims, const int* b, int nv, void* st) {
        return lqcd_restrict_f32(o, i, v, dims, b, nv, st);
    }
    static int prolong(float* o, const float* i, const float* v, const int* dims, const int* b, int nv, void* st) {
        return lqcd_prolong_f32(o, i, v, dims, b, nv, st);
    }
};
template <> struct Dev<double> {
    static int pack(double* d, const double* s, const int* dims, void* st) { return lqcd_pack_spinor_f64(d, s, dims, st); }
    static int unpack(double* d, const double* s, const int* dims, void* st) { return lqcd_unpack_spinor_f64(d, s, dims, st); }
    static int fine(double* o, const double* i, const double* U, const double* cl, double k, const int* dims,
                    const int* bc, unsigned fl, void* st) { return lqcd_wilson_clover_mult_f64(o, i, U, cl, k, dims, bc, fl, st); }
    static int coarse(double* o, const double* i, const double* A, const int* cd, int nv, unsigned fl, void* st) {
        return lqcd_coarse_mult_f64(o, i, A, cd, nv, fl, st);
    }
    static int restrict_(double* o, const double* i, const double* v, const int* dims, const int* b, int nv, void* st) {
        return lqcd_restrict_f64(o, i, v, dims, b, nv, st);
    }
    static int prolong(double* o, const double* i, const double* v, const int* dims, const int* b, int nv, void* st) {
        return lqcd_prolong_f64(o, i, v, dims, b, nv, st);
    }
};

// Workspace: [fine canonical][fine native A][fine native B][coarse A][coarse B], each rounded up to 256 B.
// coarse_mult_host only needs the two coarse slots and may be given a workspace of 2 * up256(Vc*N*2*sizeof(T)) bytes.
size_t host_ws_bytes(const int dims[4], const int block[4], int nvec, size_t rb) {
    if (check_dims(dims)) return 0;
    size_t fine_c = up256((size_t)volume(dims) * 24 * rb);
    size_t fine_n = up256(lqcd_native_spinor_reals(dims) * rb);
    size_t coarse = 0;
    int cd[4];
    if (block && nvec >= 1 && check_block_local(dims, block, nvec, cd) == LQCD_OK)
        coarse = up256((size_t)volume(cd) * 4 * nvec * rb);
    return fine_c + 2 * fine_n + 2 * coarse;
}

template <typename T>
int fine_host(const char* what, T* out_host, const T* in_host, const T* U, const T* clover, T kappa, const int dims[4],
              const int bc[4], unsigned flags, void* ws_dev, void* stream) {
    clear_error();
    if (!out_host || !in_host || !ws_dev || check_dims(dims) || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb_c = (size_t)volume(dims) * 24 * sizeof(T);
    const size_t fine_c = up256(nb_c), fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(T));
    char* ws = (char*)ws_dev;
    T* canon = (T*)ws;
    T* natA = (T*)(ws + fine_c);
    T* natB = (T*)(ws + fine_c + fine_n);
    int rc;
    if ((rc = copy_or_error(canon, in_host, nb_c, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = Dev<T>::pack(natA, canon, dims, stream))) return rc;
    if ((rc = Dev<T>::fine(natB, natA, U, clover, kappa, dims, bc, flags, stream))) return rc;
    if ((rc = Dev<T>::unpack(canon, natB, dims, stream))) return rc;
    if ((rc = copy_or_error(out_host, canon, nb_c, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}

template <typename T>
int coarse_host(const char* what, T* out_host, const T* in_host, const T* A, const int cdims[4], int nvec,
                unsigned flags, void* ws_dev, void* stream) {
    clear_error();
    if (!out_host || !in_host || !ws_dev || check_dims(cdims) || nvec < 1 || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb = (size_t)volume(cdims) * 4 * nvec * sizeof(T);
    T* a = (T*)ws_dev;
    T* b = (T*)((char*)ws_dev + up256(nb));
    int rc;
    if ((rc = copy_or_error(a, in_host, nb, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = Dev<T>::coarse(b, a, A, cdims, nvec, flags, stream))) return rc;
    if ((rc = copy_or_error(out_host, b, nb, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}

template <typename T>
int restrict_host(const char* what, T* out_c_host, const T* in_f_host, const T* nullvecs, const int dims[4],
                  const int block[4], int nvec, void* ws_dev, void* stream) {
    clear_error();
    int cd[4];
    if (!out_c_host || !in_f_host || !ws_dev || check_block_local(dims, block, nvec, cd) || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb_c = (size_t)volume(dims) * 24 * sizeof(T);
    const size_t fine_c = up256(nb_c), fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(T));
    const size_t nb_coarse = (size_t)volume(cd) * 4 * nvec * sizeof(T);
    char* ws = (char*)ws_dev;
    T* canon = (T*)ws;
    T* natA = (T*)(ws + fine_c);
    T* cvec = (T*)(ws + fine_c + 2 * fine_n);
    int rc;
    if ((rc = copy_or_error(canon, in_f_host, nb_c, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = Dev<T>::pack(natA, canon, dims, stream))) return rc;
    if ((rc = Dev<T>::restrict_(cvec, natA, nullvecs, dims, block, nvec, stream))) return rc;
    if ((rc = copy_or_error(out_c_host, cvec, nb_coarse, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}

template <typename T>
int prolong_host(const char* what, T* out_f_host, const T* in_c_host, const T* nullvecs, const int dims[4],
                 const int block[4], int nvec, void* ws_dev, void* stream) {
    clear_error();
    int cd[4];
    if (!out_f_host || !in_c_host || !ws_dev || check_block_local(dims, block, nvec, cd) || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb_c = (size_t)volume(dims) * 24 * sizeof(T);
    const size_t fine_c = up256(nb_c), fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(T));
    const size_t nb_coarse = (size_t)volume(cd) * 4 * nvec * sizeof(T);
    char* ws = (char*)ws_dev;
    T* canon = (T*)ws;
    T* natA = (T*)(ws + fine_c);
    T* cvec = (T*)(ws + fine_c + 2 * fine_n);
    int rc;
    if ((rc = copy_or_error(cvec, in_c_host, nb_coarse, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = Dev<T>::prolong(natA, cvec, nullvecs, dims, block, nvec, stream))) return rc;
    if ((rc = Dev<T>::unpack(canon, natA, dims, stream))) return rc;
    if ((rc = copy_or_error(out_f_host, canon, nb_c, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}
}  // namespace

extern "C" {

size_t lqcd_host_workspace_bytes(const int dims[4], const int block[4], int nvec) {
    return host_ws_bytes(dims, block, nvec, sizeof(float));
}
size_t lqcd_host_workspace_bytes_f64(const int dims[4], const int block[4], int nvec) {
    return host_ws_bytes(dims, block, nvec, sizeof(double));
}

#define LQCD_HOST_API(SFX, T)                                                                                        \
    int lqcd_wilson_clover_mult_host_##SFX(T* out_host, const T* in_host, const T* U, const T* clover, T kappa,      \
                                           const int dims[4], const int bc[4], unsigned flags, void* ws_dev,         \
                                           void* stream) {                                                           \
        return fine_host<T>("lqcd_wilson_clover_mult_host_" #SFX, out_host, in_host, U, clover, kappa, dims, bc,     \
                            flags, ws_dev, stream);                                                                  \
    }                                                                                                                \
    int lqcd_coarse_mult_host_##SFX(T* out_host, const T* in_host, const T* A, const int cdims[4], int nvec,         \
                                    unsigned flags, void* ws_dev, void* stream) {                                    \
        return coarse_host<T>("lqcd_coarse_mult_host_" #SFX, out_host, in_host, A, cdims, nvec, flags, ws_dev,       \
                              stream);                                                                               \
    }                                                                                                                \
    int lqcd_restrict_host_##SFX(T* out_c_host, const T* in_f_host, const T* nullvecs, const int dims[4],            \
                                 const int block[4], int nvec, void* ws_dev, void* stream) {                         \
        return restrict_host<T>("lqcd_restrict_host_" #SFX, out_c_host, in_f_host, nullvecs, dims, block, nvec,      \
                                ws_dev, stream);                                                                     \
    }                                                                                                                \
    int lqcd_prolong_host_##SFX(T* out_f_host, const T* in_c_host, const T* nullvecs, const int dims[4],             \
                                const int block[4], int nvec, void* ws_dev, void* stream) {                          \
        return prolong_host<T>("lqcd_prolong_host_" #SFX, out_f_host, in_c_host, nullvecs, dims, block, nvec,        \
                               ws_dev, stream);                                                                      \
    }
LQCD_HOST_API(f32, float)
LQCD_HOST_API(f64, double)
#undef LQCD_HOST_API
}
