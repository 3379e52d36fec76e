// host_api.cu -- end-to-end entry points on HOST right-hand sides (include/lqcd_b200.h, "end-to-end entry
// points"): H2D copy of the canonical vector, pack, the mult kernel, unpack, D2H copy, stream synchronise.
// The operator fields stay resident on the device in native layout.  fp32 (the multigrid parts of the paper run in
// single precision) and fp64 (the outer solver's precision).
//
// A call is PCIe-bound (a fine vector of config 5 is 1 GB each way against 1.4-5 ms of kernels), and PCIe is full
// duplex: so a fine vector travels in SLABS of time slices -- upload of slab k+1 (copy stream) under pack / kernel /
// unpack of slab k (the caller's stream) under the download of slab k-1 (second copy stream).  The kernels are the same
// ones on a range of tiles / aggregates (common.cuh "internal range forms"), so the results are bit-identical with
// the one-shot path, which small lattices (fewer than three slabs of ~16 MB) still take.  The two copy streams and the
// events are created once per host thread and device and kept.
#include "common.cuh"
#include "knobs.h"

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

// ---- slab pipeline plumbing ---------------------------------------------------------------------------------------
constexpr int MAX_SLABS = 64;
struct HostPipe {
    int dev = -1;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_in[MAX_SLABS], ev_cmp[MAX_SLABS], ev_start = nullptr, ev_done = nullptr;
    bool ok = false;
};
// the calling thread's pipe for the current device (created on first use; a thread that changes device gets a new one
// and leaks the old -- a handful of handles per thread)
static HostPipe* host_pipe() {
    static thread_local HostPipe pipe;
    const int d = current_device();
    if (pipe.ok && pipe.dev == d) return &pipe;
    HostPipe np;
    np.dev = d;
    bool good = cudaStreamCreateWithFlags(&np.s_in, cudaStreamNonBlocking) == cudaSuccess &&
                cudaStreamCreateWithFlags(&np.s_out, cudaStreamNonBlocking) == cudaSuccess &&
                cudaEventCreateWithFlags(&np.ev_start, cudaEventDisableTiming) == cudaSuccess &&
                cudaEventCreateWithFlags(&np.ev_done, cudaEventDisableTiming) == cudaSuccess;
    for (int k = 0; good && k < MAX_SLABS; k++)
        good = cudaEventCreateWithFlags(&np.ev_in[k], cudaEventDisableTiming) == cudaSuccess &&
               cudaEventCreateWithFlags(&np.ev_cmp[k], cudaEventDisableTiming) == cudaSuccess;
    if (!good) {
        cudaGetLastError();
        return nullptr;  // the caller falls back to the one-shot path
    }
    np.ok = true;
    pipe = np;
    return &pipe;
}
// time slices per slab: a multiple of `unit` dividing Lt with >= ~16 MB per slab and 3 ... MAX_SLABS slabs; 0 = do not
// pipeline (small lattice)
static int slab_extent(const int dims[4], int unit, size_t real_bytes) {
    if (unit < 1 || dims[3] % unit || g_knobs.host_slab_mb < 0) return 0;
    const size_t least = (size_t)(g_knobs.host_slab_mb > 0 ? g_knobs.host_slab_mb : 16) << 20;
    const size_t slice = (size_t)dims[0] * dims[1] * dims[2] * 24 * real_bytes;
    for (int m = unit; m <= dims[3] / 3; m += unit) {
        if (dims[3] % m) continue;
        if (slice * m >= least && dims[3] / m <= MAX_SLABS) return m;
    }
    return 0;
}
#define CUDA_OR_FAIL(expr)                                                          \
    do {                                                                            \
        cudaError_t e_ = (expr);                                                    \
        if (e_ != cudaSuccess) {                                                    \
            set_error("%s: %s: %s", what, #expr, cudaGetErrorString(e_));            \
            return LQCD_ECUDA;                                                      \
        }                                                                           \
    } while (0)
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
    // slab pipeline (see the top of the file).  Slab k of D needs the input slabs k - 1, k, k + 1 (periodic in t), so
    // the LAST slab is uploaded first and the operator runs on slab k once slab k + 1 is packed.
    const bool plain = U && clover && bc && aligned16(U) && aligned16(clover) && !(flags & ~(LQCD_DAGGER | LQCD_LINKS_12)) &&
                       out_host != in_host;
    const int mt = plain ? slab_extent(dims, fine_tile_extent_t(dims, bc, (int)sizeof(T)), sizeof(T)) : 0;
    HostPipe* hp = mt ? host_pipe() : nullptr;
    if (hp) {
        const int ns = dims[3] / mt;
        const long long V3 = (long long)dims[0] * dims[1] * dims[2], slab_sites = V3 * mt;
        const size_t slab_reals = (size_t)slab_sites * 24, slab_b = slab_reals * sizeof(T);
        CUDA_OR_FAIL(cudaEventRecord(hp->ev_start, st));
        CUDA_OR_FAIL(cudaStreamWaitEvent(hp->s_in, hp->ev_start, 0));
        CUDA_OR_FAIL(cudaStreamWaitEvent(hp->s_out, hp->ev_start, 0));
        for (int i = 0; i < ns; i++) {  // uploads: ns - 1, 0, 1, ..., ns - 2
            const int k = i == 0 ? ns - 1 : i - 1;
            CUDA_OR_FAIL(cudaMemcpyAsync(canon + k * slab_reals, in_host + k * slab_reals, slab_b, cudaMemcpyHostToDevice,
                                         hp->s_in));
            CUDA_OR_FAIL(cudaEventRecord(hp->ev_in[k], hp->s_in));
        }
        auto pack_slab = [&](int k) -> int {
            cudaError_t e = cudaStreamWaitEvent(st, hp->ev_in[k], 0);
            if (e != cudaSuccess) {
                set_error("%s: cudaStreamWaitEvent: %s", what, cudaGetErrorString(e));
                return LQCD_ECUDA;
            }
            return spinor_range_call<T, false>(natA, canon, dims, k * slab_sites, (k + 1) * slab_sites, stream, what);
        };
        if ((rc = pack_slab(ns - 1))) return rc;
        if ((rc = pack_slab(0))) return rc;
        for (int k = 0; k < ns; k++) {
            if (k + 1 <= ns - 2 && (rc = pack_slab(k + 1))) return rc;
            if ((rc = wilson_clover_slab_call<T>(natB, natA, U, clover, kappa, dims, bc, flags, k * mt, (k + 1) * mt, stream,
                                                 what)))
                return rc;
            // the canonical slab k is dead since pack(k): it takes the result
            if ((rc = spinor_range_call<T, true>(canon, natB, dims, k * slab_sites, (k + 1) * slab_sites, stream, what)))
                return rc;
            CUDA_OR_FAIL(cudaEventRecord(hp->ev_cmp[k], st));
            CUDA_OR_FAIL(cudaStreamWaitEvent(hp->s_out, hp->ev_cmp[k], 0));
            CUDA_OR_FAIL(cudaMemcpyAsync(out_host + k * slab_reals, canon + k * slab_reals, slab_b, cudaMemcpyDeviceToHost,
                                         hp->s_out));
        }
        CUDA_OR_FAIL(cudaEventRecord(hp->ev_done, hp->s_out));
        CUDA_OR_FAIL(cudaStreamWaitEvent(st, hp->ev_done, 0));
        return sync_or_error(st, what);
    }
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
    // slab pipeline: slabs of whole aggregates in t; restriction of slab k under the upload of slab k + 1
    const int mt = (nullvecs && aligned16(nullvecs)) ? slab_extent(dims, block[3], sizeof(T)) : 0;
    HostPipe* hp = mt ? host_pipe() : nullptr;
    if (hp) {
        const int ns = dims[3] / mt;
        const long long V3 = (long long)dims[0] * dims[1] * dims[2], slab_sites = V3 * mt;
        const long long slab_X = (long long)cd[0] * cd[1] * cd[2] * (mt / block[3]);
        const size_t slab_reals = (size_t)slab_sites * 24, slab_b = slab_reals * sizeof(T);
        CUDA_OR_FAIL(cudaEventRecord(hp->ev_start, st));
        CUDA_OR_FAIL(cudaStreamWaitEvent(hp->s_in, hp->ev_start, 0));
        for (int k = 0; k < ns; k++) {
            CUDA_OR_FAIL(cudaMemcpyAsync(canon + k * slab_reals, in_f_host + k * slab_reals, slab_b,
                                         cudaMemcpyHostToDevice, hp->s_in));
            CUDA_OR_FAIL(cudaEventRecord(hp->ev_in[k], hp->s_in));
        }
        for (int k = 0; k < ns; k++) {
            CUDA_OR_FAIL(cudaStreamWaitEvent(st, hp->ev_in[k], 0));
            if ((rc = spinor_range_call<T, false>(natA, canon, dims, k * slab_sites, (k + 1) * slab_sites, stream, what)))
                return rc;
            if ((rc = restrict_range_call<T>(cvec, natA, nullvecs, dims, block, nvec, k * slab_X, (k + 1) * slab_X, stream,
                                             what)))
                return rc;
        }
        if ((rc = copy_or_error(out_c_host, cvec, nb_coarse, cudaMemcpyDeviceToHost, st, what))) return rc;
        return sync_or_error(st, what);
    }
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
    // slab pipeline: the download of slab k under the prolongation of slab k + 1
    const int mt = (nullvecs && aligned16(nullvecs)) ? slab_extent(dims, block[3], sizeof(T)) : 0;
    HostPipe* hp = mt ? host_pipe() : nullptr;
    if (hp) {
        const int ns = dims[3] / mt;
        const long long V3 = (long long)dims[0] * dims[1] * dims[2], slab_sites = V3 * mt;
        const long long slab_X = (long long)cd[0] * cd[1] * cd[2] * (mt / block[3]);
        const size_t slab_reals = (size_t)slab_sites * 24, slab_b = slab_reals * sizeof(T);
        if ((rc = copy_or_error(cvec, in_c_host, nb_coarse, cudaMemcpyHostToDevice, st, what))) return rc;
        CUDA_OR_FAIL(cudaEventRecord(hp->ev_start, st));
        CUDA_OR_FAIL(cudaStreamWaitEvent(hp->s_out, hp->ev_start, 0));
        for (int k = 0; k < ns; k++) {
            if ((rc = prolong_range_call<T>(natA, cvec, nullvecs, dims, block, nvec, k * slab_X, (k + 1) * slab_X, stream,
                                            what)))
                return rc;
            if ((rc = spinor_range_call<T, true>(canon, natA, dims, k * slab_sites, (k + 1) * slab_sites, stream, what)))
                return rc;
            CUDA_OR_FAIL(cudaEventRecord(hp->ev_cmp[k], st));
            CUDA_OR_FAIL(cudaStreamWaitEvent(hp->s_out, hp->ev_cmp[k], 0));
            CUDA_OR_FAIL(cudaMemcpyAsync(out_f_host + k * slab_reals, canon + k * slab_reals, slab_b,
                                         cudaMemcpyDeviceToHost, hp->s_out));
        }
        CUDA_OR_FAIL(cudaEventRecord(hp->ev_done, hp->s_out));
        CUDA_OR_FAIL(cudaStreamWaitEvent(st, hp->ev_done, 0));
        return sync_or_error(st, what);
    }
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
