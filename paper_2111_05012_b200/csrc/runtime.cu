// runtime.cu -- diagnostics, tuning knobs and native-size queries of the C ABI (include/lqcd_b200.h).
#include <atomic>
#include <string.h>

#include "common.cuh"
#include "knobs.h"

namespace lqcd {

static thread_local char g_err[512] = "";
static std::atomic<unsigned long long> g_launches{0};

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
void clear_error() { g_err[0] = 0; }
void count_launch(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("%s: %s", what, cudaGetErrorString(e));
        return LQCD_ECUDA;
    }
    return LQCD_OK;
}

thread_local Knobs g_knobs;

int current_device() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    return d;
}
static int device_attr(cudaDeviceAttr which, int* cache, int fallback) {
    const int d = current_device();
    if (d < 0) return fallback;
    if (d < 64 && cache[d] > 0) return cache[d];
    int v = 0;
    if (cudaDeviceGetAttribute(&v, which, d) != cudaSuccess || v < 1) {
        cudaGetLastError();
        return fallback;
    }
    if (d < 64) cache[d] = v;  // racing writers store the same value
    return v;
}
int max_optin_smem() {
    static int cache[64];
    return device_attr(cudaDevAttrMaxSharedMemoryPerBlockOptin, cache, 0);
}
int sm_count() {
    static int cache[64];
    return device_attr(cudaDevAttrMultiProcessorCount, cache, 148);
}

}  // namespace lqcd

using namespace lqcd;

extern "C" {

int lqcd_version(void) { return 100; }
const char* lqcd_last_error(void) { return g_err; }
unsigned long long lqcd_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int lqcd_set_fine_tile(const int tile[4]) {
    if (!tile || tile[0] == 0) {
        for (int mu = 0; mu < 4; mu++) g_knobs.fine_tile[mu] = 0;
        return LQCD_OK;
    }
    long long p = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (tile[mu] < 1) {
            set_error("lqcd_set_fine_tile: tile[%d] = %d", mu, tile[mu]);
            return LQCD_EINVAL;
        }
        p *= tile[mu];
    }
    if (p > 256) {
        set_error("lqcd_set_fine_tile: %lld threads per CTA > 256", p);
        return LQCD_EINVAL;
    }
    for (int mu = 0; mu < 4; mu++) g_knobs.fine_tile[mu] = tile[mu];
    return LQCD_OK;
}

int lqcd_set_knob(const char* name, int value) {
    if (!name) return LQCD_EINVAL;
    if (!strcmp(name, "coarse_rows_per_warp")) g_knobs.coarse_rows_per_warp = value;
    else if (!strcmp(name, "coarse_R")) g_knobs.coarse_R = value;
    else if (!strcmp(name, "coarse_warps")) g_knobs.coarse_warps = value;
    else if (!strcmp(name, "transfer_warps")) g_knobs.transfer_warps = value;
    else if (!strcmp(name, "fine_tslab")) g_knobs.fine_tslab = value;
    else if (!strcmp(name, "sap_fused")) g_knobs.sap_fused = value;
    else if (!strcmp(name, "sap_group_residual")) g_knobs.sap_group_residual = value;
    else if (!strcmp(name, "sap_tmem")) g_knobs.sap_tmem = value;
    else if (!strcmp(name, "host_slab_mb")) g_knobs.host_slab_mb = value;
    else if (!strcmp(name, "fine_mrhs")) g_knobs.fine_mrhs = value;
    else if (!strcmp(name, "mrhs_tensor")) g_knobs.mrhs_tensor = value;
    else if (!strcmp(name, "site_order")) g_knobs.site_order = value;
    else if (!strcmp(name, "mrhs_stages")) g_knobs.mrhs_stages = value;
    else {
        set_error("lqcd_set_knob: unknown knob '%s'", name);
        return LQCD_EINVAL;
    }
    return LQCD_OK;
}

size_t lqcd_native_spinor_reals(const int dims[4]) {
    if (check_dims(dims)) return 0;
    return (size_t)nchunks(dims) * CH * 24;
}
size_t lqcd_native_gauge_reals(const int dims[4], unsigned flags) {
    if (check_dims(dims)) return 0;
    return (size_t)nchunks(dims) * CH * 4 * ((flags & LQCD_LINKS_12) ? 12 : 18);
}
size_t lqcd_native_clover_reals(const int dims[4]) {
    if (check_dims(dims)) return 0;
    return (size_t)nchunks(dims) * CH * 72;
}
size_t lqcd_native_nullvecs_reals(const int dims[4], const int block[4], int nvec) {
    int cd[4];
    if (check_block_local(dims, block, nvec, cd)) return 0;
    return (size_t)volume(dims) * 24 * (size_t)nvec;
}
size_t lqcd_native_coarse_vec_reals(const int cdims[4], int nvec) {
    if (check_dims(cdims) || nvec < 1) return 0;
    return (size_t)volume(cdims) * 4 * (size_t)nvec;
}
size_t lqcd_native_coarse_mat_reals(const int cdims[4], int nvec) {
    if (check_dims(cdims) || nvec < 1) return 0;
    return (size_t)volume(cdims) * 9 * 8 * (size_t)nvec * (size_t)nvec;
}

}  // extern "C"
