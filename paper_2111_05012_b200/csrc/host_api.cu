// host_api.cu -- end-to-end entry points on HOST right-hand sides (include/lqcd_b200.h, "end-to-end entry
// points"): H2D copy of the canonical vector, pack, the mult kernel, unpack, D2H copy, stream synchronise.
// The operator fields stay resident on the device in native layout.  fp32 only (the multigrid parts of the
// paper run in single precision).
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

extern "C" {

// Workspace: [fine canonical][fine native A][fine native B][coarse A][coarse B], each rounded up to 256 B.
// coarse_mult_host only needs the two coarse slots and may be given a workspace of 2 * up256(Vc*N*8) bytes.
size_t lqcd_host_workspace_bytes(const int dims[4], const int block[4], int nvec) {
    if (check_dims(dims)) return 0;
    size_t fine_c = up256((size_t)volume(dims) * 24 * sizeof(float));
    size_t fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(float));
    size_t coarse = 0;
    int cd[4];
    if (block && nvec >= 1 && check_block(dims, block, nvec, cd) == LQCD_OK)
        coarse = up256((size_t)volume(cd) * 4 * nvec * sizeof(float));
    return fine_c + 2 * fine_n + 2 * coarse;
}

int lqcd_wilson_clover_mult_host_f32(float* out_host, const float* in_host, const float* U, const float* clover,
                                     float kappa, const int dims[4], const int bc[4], unsigned flags, void* ws_dev,
                                     void* stream) {
    const char* what = "lqcd_wilson_clover_mult_host_f32";
    clear_error();
    if (!out_host || !in_host || !ws_dev || check_dims(dims) || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb_c = (size_t)volume(dims) * 24 * sizeof(float);
    const size_t fine_c = up256(nb_c), fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(float));
    char* ws = (char*)ws_dev;
    float* canon = (float*)ws;
    float* natA = (float*)(ws + fine_c);
    float* natB = (float*)(ws + fine_c + fine_n);
    int rc;
    if ((rc = copy_or_error(canon, in_host, nb_c, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = lqcd_pack_spinor_f32(natA, canon, dims, stream))) return rc;
    if ((rc = lqcd_wilson_clover_mult_f32(natB, natA, U, clover, kappa, dims, bc, flags, stream))) return rc;
    if ((rc = lqcd_unpack_spinor_f32(canon, natB, dims, stream))) return rc;
    if ((rc = copy_or_error(out_host, canon, nb_c, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}

int lqcd_coarse_mult_host_f32(float* out_host, const float* in_host, const float* A, const int cdims[4], int nvec,
                              unsigned flags, void* ws_dev, void* stream) {
    const char* what = "lqcd_coarse_mult_host_f32";
    clear_error();
    if (!out_host || !in_host || !ws_dev || check_dims(cdims) || nvec < 1 || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb = (size_t)volume(cdims) * 4 * nvec * sizeof(float);
    float* a = (float*)ws_dev;
    float* b = (float*)((char*)ws_dev + up256(nb));
    int rc;
    if ((rc = copy_or_error(a, in_host, nb, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = lqcd_coarse_mult_f32(b, a, A, cdims, nvec, flags, stream))) return rc;
    if ((rc = copy_or_error(out_host, b, nb, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}

int lqcd_restrict_host_f32(float* out_c_host, const float* in_f_host, const float* nullvecs, const int dims[4],
                           const int block[4], int nvec, void* ws_dev, void* stream) {
    const char* what = "lqcd_restrict_host_f32";
    clear_error();
    int cd[4];
    if (!out_c_host || !in_f_host || !ws_dev || check_block(dims, block, nvec, cd) || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb_c = (size_t)volume(dims) * 24 * sizeof(float);
    const size_t fine_c = up256(nb_c), fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(float));
    const size_t nb_coarse = (size_t)volume(cd) * 4 * nvec * sizeof(float);
    char* ws = (char*)ws_dev;
    float* canon = (float*)ws;
    float* natA = (float*)(ws + fine_c);
    float* cvec = (float*)(ws + fine_c + 2 * fine_n);
    int rc;
    if ((rc = copy_or_error(canon, in_f_host, nb_c, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = lqcd_pack_spinor_f32(natA, canon, dims, stream))) return rc;
    if ((rc = lqcd_restrict_f32(cvec, natA, nullvecs, dims, block, nvec, stream))) return rc;
    if ((rc = copy_or_error(out_c_host, cvec, nb_coarse, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}

int lqcd_prolong_host_f32(float* out_f_host, const float* in_c_host, const float* nullvecs, const int dims[4],
                          const int block[4], int nvec, void* ws_dev, void* stream) {
    const char* what = "lqcd_prolong_host_f32";
    clear_error();
    int cd[4];
    if (!out_f_host || !in_c_host || !ws_dev || check_block(dims, block, nvec, cd) || !aligned16(ws_dev)) {
        set_error("%s: invalid argument", what);
        return LQCD_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb_c = (size_t)volume(dims) * 24 * sizeof(float);
    const size_t fine_c = up256(nb_c), fine_n = up256(lqcd_native_spinor_reals(dims) * sizeof(float));
    const size_t nb_coarse = (size_t)volume(cd) * 4 * nvec * sizeof(float);
    char* ws = (char*)ws_dev;
    float* canon = (float*)ws;
    float* natA = (float*)(ws + fine_c);
    float* cvec = (float*)(ws + fine_c + 2 * fine_n);
    int rc;
    if ((rc = copy_or_error(cvec, in_c_host, nb_coarse, cudaMemcpyHostToDevice, st, what))) return rc;
    if ((rc = lqcd_prolong_f32(natA, cvec, nullvecs, dims, block, nvec, stream))) return rc;
    if ((rc = lqcd_unpack_spinor_f32(canon, natA, dims, stream))) return rc;
    if ((rc = copy_or_error(out_f_host, canon, nb_c, cudaMemcpyDeviceToHost, st, what))) return rc;
    return sync_or_error(st, what);
}
}
