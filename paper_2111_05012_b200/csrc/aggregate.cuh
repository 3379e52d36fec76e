// aggregate.cuh -- geometry of the aggregates (blocks x chirality) shared by the transfer kernels (transfer.cu) and
// the set-up kernels (setup.cu): the native null-vector layout is [X][chi][i][l][k], one contiguous vector of
// |block|*6 complex per (X, chi, i).
#pragma once
#include "common.cuh"
#include "layout.cuh"

namespace lqcd {

struct TransferParams {
    int L[4], b[4], Lc[4];
    int bv;    // sites per block
    int nvec;
    int LV;    // vec16 per (X, chi, i) vector = bv * 12 / NV
    int agg_off;  // first aggregate (X, chi) of the launch (range forms of restrict / prolong; 0 otherwise)
    int zero;     // always 0, but only known at run time: the dependency fence of the streaming batches (transfer.cu)
    SiteOrder ord;  // native position of a fine site (layout.cuh)
};

// native position of the fine site with local index l inside coarse site X
__device__ __forceinline__ int fine_site(const TransferParams& P, int X, int l) {
    int x[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const int Xmu = X % P.Lc[mu];
        X /= P.Lc[mu];
        const int lmu = l % P.b[mu];
        l /= P.b[mu];
        x[mu] = Xmu * P.b[mu] + lmu;
    }
    return P.ord.index(x);
}

template <typename T>
inline int transfer_setup(TransferParams& P, const void* a, const void* b, const void* c, const int dims[4],
                          const int block[4], int nvec, const char* what) {
    clear_error();
    if (!a || !b || !c) {
        set_error("%s: null pointer", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(a) || !aligned16(b) || !aligned16(c)) {
        set_error("%s: pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    if (check_block_local(dims, block, nvec, P.Lc)) {  // aggregate-local: any coarse extent >= 1
        set_error("%s: bad dims/block/nvec (block must divide dims, nvec >= 1)", what);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) return LQCD_EUNSUPPORTED;
    P.bv = 1;
    for (int mu = 0; mu < 4; mu++) {
        P.L[mu] = dims[mu];
        P.b[mu] = block[mu];
        P.bv *= block[mu];
    }
    P.nvec = nvec;
    P.agg_off = 0;
    P.zero = 0;
    P.LV = P.bv * 12 / VecOf<T>::NV;
    P.ord.set(dims);
    return LQCD_OK;
}

}  // namespace lqcd
