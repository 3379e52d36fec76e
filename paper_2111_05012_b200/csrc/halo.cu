// halo.cu -- the exchange step of the SHARDED fine operator (the paper runs D on a 4-D
// domain decomposition over the nodes with one halo exchange per application).
//
// One rank owns a local lattice dims[4]; in every PARTITIONED direction mu (bit mu of part_mask) the hops that
// leave the local lattice are served by the neighbouring rank.  One application of D (Eq. 1) is
//   1. lqcd_wilson_clover_halo_pack:   the 2 faces per partitioned direction, as spin-PROJECTED half spinors
//        (12 reals per face site instead of 24: the rank-2 structure of (1 -+ g_mu)); the face that feeds the
//        neighbour's BACKWARD hop is multiplied by U_mu^dag(x) here, because the link lives on the sender;
//   2. the exchange (torch.distributed / NCCL send-recv, or peer copies; not in this library: plain buffers);
//   3. lqcd_wilson_clover_mult_interior (wilson_clover.cu): D with the leaving hops switched off -- independent of
//        2, so it overlaps the exchange on another stream;
//   4. lqcd_wilson_clover_halo_add:    out(x) -= kappa * [reconstructed received half spinors], forward faces
//        multiplied by the local link U_mu(x), with the boundary phase of a hop that wraps the GLOBAL lattice.
//
// Face buffers: face (mu, dir), dir 0: x_mu = 0, dir 1: x_mu = L_mu - 1; face site f = lexicographic index of the other
// three coordinates (x fastest); 12 reals per site as rows of one 16-byte vector, buf[(j * Fv + f) * NV + q].
#include "common.cuh"
#include "fermion.cuh"
#include "layout.cuh"

namespace lqcd {

struct HaloParams {
    int L[4];
    int fv[4];        // face volume V / L[mu]
    int phase[8];     // +1 / -1 per receive face (2 mu + dir)
    unsigned mask;    // partitioned directions
    SiteOrder ord;    // native position of a site (layout.cuh)
};

// face site f of direction mu at x_mu = xm -> native position of that site
__device__ __forceinline__ int face_site(const HaloParams& P, int mu, int f, int xm) {
    int x[4];
#pragma unroll
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) {
            x[nu] = xm;
        } else {
            x[nu] = f % P.L[nu];
            f /= P.L[nu];
        }
    }
    return P.ord.index(x);
}

template <typename T> __device__ __forceinline__ void store_half(T* __restrict__ buf, int fv, int f, const T h[12]) {
    constexpr int NV = VecOf<T>::NV;
#pragma unroll
    for (int j = 0; j < 12 / NV; j++) {
        V16<T> v;
#pragma unroll
        for (int q = 0; q < NV; q++) v.r[q] = h[j * NV + q];
        st16(buf + ((long long)j * fv + f) * NV, v);
    }
}
template <typename T> __device__ __forceinline__ void load_half(T h[12], const T* __restrict__ buf, int fv, int f) {
    constexpr int NV = VecOf<T>::NV;
#pragma unroll
    for (int j = 0; j < 12 / NV; j++) {
        const V16<T> v = ld16(buf + ((long long)j * fv + f) * NV);
#pragma unroll
        for (int q = 0; q < NV; q++) h[j * NV + q] = v.r[q];
    }
}

struct FacePtrs {
    void* p[8];
};

template <int MU, bool DAG, bool L12, typename T>
__device__ __forceinline__ void pack_face(const HaloParams& P, int dir, T* __restrict__ buf, const T* __restrict__ in,
                                          const T* __restrict__ U) {
    // D: forward hops carry (1 - g_mu), backward (1 + g_mu); D^dag: swapped (wilson_clover.cu)
    constexpr int SF = DAG ? +1 : -1, SB = DAG ? -1 : +1;
    const int fv = P.fv[MU];
    for (int f = blockIdx.x * blockDim.x + threadIdx.x; f < fv; f += gridDim.x * blockDim.x) {
        const int s = face_site(P, MU, f, dir ? P.L[MU] - 1 : 0);
        T p[24], h[12];
        load_spinor<T>(p, in, s);
        if (dir) {  // feeds the backward hop of the +mu neighbour: U_mu^dag(x) (1 + g_mu) in(x)
            T u[18], g[12];
            load_link<T, L12>(u, U, s, MU);
            project<MU, SB, T>(h, p);
            su3_mult<false, T>(g, u, h);
            store_half<T>(buf, fv, f, g);
        } else {  // feeds the forward hop of the -mu neighbour, who owns the link: (1 - g_mu) in(x)
            project<MU, SF, T>(h, p);
            store_half<T>(buf, fv, f, h);
        }
    }
}

template <typename T, bool DAG, bool L12>
__global__ void __launch_bounds__(128) k_halo_pack(FacePtrs send, const T* __restrict__ in, const T* __restrict__ U,
                                                   HaloParams P) {
    const int face = blockIdx.y, mu = face >> 1, dir = face & 1;
    if (!((P.mask >> mu) & 1)) return;
    T* buf = static_cast<T*>(send.p[face]);
    switch (mu) {
        case 0: pack_face<0, DAG, L12, T>(P, dir, buf, in, U); break;
        case 1: pack_face<1, DAG, L12, T>(P, dir, buf, in, U); break;
        case 2: pack_face<2, DAG, L12, T>(P, dir, buf, in, U); break;
        default: pack_face<3, DAG, L12, T>(P, dir, buf, in, U); break;
    }
}

// One thread per face site of direction MU adds BOTH received faces of that direction (x_mu = 0, then x_mu = L - 1:
// the same site when L_mu = 1), so that no two threads of a launch touch the same output site; the four directions
// are four launches in stream order.  Fixed order -> bit-reproducible.
template <int MU, typename T, bool DAG, bool L12>
__global__ void __launch_bounds__(128) k_halo_add(T* __restrict__ out, const T* __restrict__ from_minus,
                                                  const T* __restrict__ from_plus, const T* __restrict__ U, T kappa,
                                                  HaloParams P) {
    constexpr int SF = DAG ? +1 : -1, SB = DAG ? -1 : +1;
    const int fv = P.fv[MU];
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= fv) return;
    {  // backward hop at x_mu = 0: the -mu neighbour sent U^dag (1 + g_mu) in
        const int s = face_site(P, MU, f, 0);
        T g[12], acc[24], o[24];
        load_half<T>(g, from_minus, fv, f);
#pragma unroll
        for (int r = 0; r < 24; r++) acc[r] = 0;
        reconstruct<MU, SB, T>(acc, g, (T)P.phase[2 * MU]);
        load_spinor<T>(o, out, s);
#pragma unroll
        for (int r = 0; r < 24; r++) o[r] = fma(-kappa, acc[r], o[r]);
        store_spinor<T>(out, s, o);
    }
    {  // forward hop at x_mu = L - 1: the +mu neighbour sent (1 - g_mu) in; the link is mine
        const int s = face_site(P, MU, f, P.L[MU] - 1);
        T h[12], u[18], g[12], acc[24], o[24];
        load_half<T>(h, from_plus, fv, f);
        load_link<T, L12>(u, U, s, MU);
        su3_mult<true, T>(g, u, h);
#pragma unroll
        for (int r = 0; r < 24; r++) acc[r] = 0;
        reconstruct<MU, SF, T>(acc, g, (T)P.phase[2 * MU + 1]);
        load_spinor<T>(o, out, s);
#pragma unroll
        for (int r = 0; r < 24; r++) o[r] = fma(-kappa, acc[r], o[r]);
        store_spinor<T>(out, s, o);
    }
}

static int halo_setup(HaloParams& P, const int dims[4], unsigned part_mask, unsigned flags, const char* what) {
    if (check_dims(dims)) {
        set_error("%s: non-positive dim", what);
        return LQCD_EINVAL;
    }
    if ((flags & ~(LQCD_DAGGER | LQCD_LINKS_12)) || part_mask > 15u) {
        set_error("%s: bad flags 0x%x or part_mask 0x%x", what, flags, part_mask);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) {
        set_error("%s: volume exceeds 2^31-1 sites", what);
        return LQCD_EUNSUPPORTED;
    }
    const long long V = volume(dims);
    for (int mu = 0; mu < 4; mu++) {
        P.L[mu] = dims[mu];
        P.fv[mu] = (int)(V / dims[mu]);
    }
    for (int i = 0; i < 8; i++) P.phase[i] = 1;
    P.mask = part_mask;
    P.ord.set(dims);
    return LQCD_OK;
}

template <typename T>
static int halo_pack_call(T* const send[8], const T* in, const T* U, const int dims[4], unsigned part_mask,
                          unsigned flags, void* stream, const char* what) {
    clear_error();
    HaloParams P;
    int rc = halo_setup(P, dims, part_mask, flags, what);
    if (rc) return rc;
    if (!send || !in || !U || !aligned16(in) || !aligned16(U)) {
        set_error("%s: null or misaligned pointer", what);
        return LQCD_EINVAL;
    }
    FacePtrs fp;
    int fvmax = 0;
    for (int i = 0; i < 8; i++) {
        fp.p[i] = nullptr;
        if (!((part_mask >> (i >> 1)) & 1)) continue;
        if (!send[i] || !aligned16(send[i])) {
            set_error("%s: send[%d] is null or not 16-byte aligned", what, i);
            return LQCD_EINVAL;
        }
        fp.p[i] = send[i];
        fvmax = P.fv[i >> 1] > fvmax ? P.fv[i >> 1] : fvmax;
    }
    if (!part_mask) return LQCD_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const dim3 grid((unsigned)((fvmax + 127) / 128), 8);
    const bool dag = flags & LQCD_DAGGER, l12 = flags & LQCD_LINKS_12;
    if (dag && l12) k_halo_pack<T, true, true><<<grid, 128, 0, st>>>(fp, in, U, P);
    else if (dag) k_halo_pack<T, true, false><<<grid, 128, 0, st>>>(fp, in, U, P);
    else if (l12) k_halo_pack<T, false, true><<<grid, 128, 0, st>>>(fp, in, U, P);
    else k_halo_pack<T, false, false><<<grid, 128, 0, st>>>(fp, in, U, P);
    count_launch();
    return check_launch(what);
}

template <int MU, typename T>
static void halo_add_launch(T* out, const T* fm, const T* fp, const T* U, T kappa, const HaloParams& P, bool dag,
                            bool l12, cudaStream_t st) {
    const unsigned grid = (unsigned)((P.fv[MU] + 127) / 128);
    if (dag && l12) k_halo_add<MU, T, true, true><<<grid, 128, 0, st>>>(out, fm, fp, U, kappa, P);
    else if (dag) k_halo_add<MU, T, true, false><<<grid, 128, 0, st>>>(out, fm, fp, U, kappa, P);
    else if (l12) k_halo_add<MU, T, false, true><<<grid, 128, 0, st>>>(out, fm, fp, U, kappa, P);
    else k_halo_add<MU, T, false, false><<<grid, 128, 0, st>>>(out, fm, fp, U, kappa, P);
    count_launch();
}

template <typename T>
static int halo_add_call(T* out, const T* const recv[8], const T* U, T kappa, const int dims[4],
                         const int face_phase[8], unsigned part_mask, unsigned flags, void* stream, const char* what) {
    clear_error();
    HaloParams P;
    int rc = halo_setup(P, dims, part_mask, flags, what);
    if (rc) return rc;
    if (!out || !recv || !U || !face_phase || !aligned16(out) || !aligned16(U)) {
        set_error("%s: null or misaligned pointer", what);
        return LQCD_EINVAL;
    }
    for (int i = 0; i < 8; i++) {
        if (!((part_mask >> (i >> 1)) & 1)) continue;
        if (face_phase[i] != 1 && face_phase[i] != -1) {
            set_error("%s: face_phase[%d] = %d not in {+1,-1}", what, i, face_phase[i]);
            return LQCD_EINVAL;
        }
        if (!recv[i] || !aligned16(recv[i])) {
            set_error("%s: recv[%d] is null or not 16-byte aligned", what, i);
            return LQCD_EINVAL;
        }
        P.phase[i] = face_phase[i];
    }
    cudaStream_t st = (cudaStream_t)stream;
    const bool dag = flags & LQCD_DAGGER, l12 = flags & LQCD_LINKS_12;
    if (part_mask & 1u) halo_add_launch<0, T>(out, recv[0], recv[1], U, kappa, P, dag, l12, st);
    if (part_mask & 2u) halo_add_launch<1, T>(out, recv[2], recv[3], U, kappa, P, dag, l12, st);
    if (part_mask & 4u) halo_add_launch<2, T>(out, recv[4], recv[5], U, kappa, P, dag, l12, st);
    if (part_mask & 8u) halo_add_launch<3, T>(out, recv[6], recv[7], U, kappa, P, dag, l12, st);
    return check_launch(what);
}

template <typename T>
int wilson_clover_interior_call(T* out, const T* in, const T* U, const T* clover, const T* rhs, T kappa,
                                const int dims[4], const int bc[4], unsigned part_mask, unsigned flags, void* stream,
                                const char* what, const int* domain);

}  // namespace lqcd

using namespace lqcd;

extern "C" {

size_t lqcd_halo_face_reals(const int dims[4], int mu) {
    if (check_dims(dims) || mu < 0 || mu > 3) return 0;
    return (size_t)(volume(dims) / dims[mu]) * 12;
}

int lqcd_wilson_clover_halo_pack_f32(float* const send[8], const float* in, const float* U, const int dims[4],
                                     unsigned part_mask, unsigned flags, void* stream) {
    return halo_pack_call<float>(send, in, U, dims, part_mask, flags, stream, "lqcd_wilson_clover_halo_pack_f32");
}
int lqcd_wilson_clover_halo_pack_f64(double* const send[8], const double* in, const double* U, const int dims[4],
                                     unsigned part_mask, unsigned flags, void* stream) {
    return halo_pack_call<double>(send, in, U, dims, part_mask, flags, stream, "lqcd_wilson_clover_halo_pack_f64");
}
int lqcd_wilson_clover_mult_interior_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                         const int dims[4], const int bc[4], unsigned part_mask, unsigned flags,
                                         void* stream) {
    return wilson_clover_interior_call<float>(out, in, U, clover, nullptr, kappa, dims, bc, part_mask, flags, stream,
                                              "lqcd_wilson_clover_mult_interior_f32", nullptr);
}
int lqcd_wilson_clover_mult_interior_f64(double* out, const double* in, const double* U, const double* clover,
                                         double kappa, const int dims[4], const int bc[4], unsigned part_mask,
                                         unsigned flags, void* stream) {
    return wilson_clover_interior_call<double>(out, in, U, clover, nullptr, kappa, dims, bc, part_mask, flags, stream,
                                               "lqcd_wilson_clover_mult_interior_f64", nullptr);
}
int lqcd_wilson_clover_residual_interior_f32(float* r, const float* b, const float* x, const float* U,
                                             const float* clover, float kappa, const int dims[4], const int bc[4],
                                             const int* domain, unsigned part_mask, unsigned flags, void* stream) {
    if (!b) {
        clear_error();
        set_error("lqcd_wilson_clover_residual_interior_f32: null rhs");
        return LQCD_EINVAL;
    }
    return wilson_clover_interior_call<float>(r, x, U, clover, b, kappa, dims, bc, part_mask, flags, stream,
                                              "lqcd_wilson_clover_residual_interior_f32", domain);
}
int lqcd_wilson_clover_residual_interior_f64(double* r, const double* b, const double* x, const double* U,
                                             const double* clover, double kappa, const int dims[4], const int bc[4],
                                             const int* domain, unsigned part_mask, unsigned flags, void* stream) {
    if (!b) {
        clear_error();
        set_error("lqcd_wilson_clover_residual_interior_f64: null rhs");
        return LQCD_EINVAL;
    }
    return wilson_clover_interior_call<double>(r, x, U, clover, b, kappa, dims, bc, part_mask, flags, stream,
                                               "lqcd_wilson_clover_residual_interior_f64", domain);
}
int lqcd_wilson_clover_halo_add_f32(float* out, const float* const recv[8], const float* U, float kappa,
                                    const int dims[4], const int face_phase[8], unsigned part_mask, unsigned flags,
                                    void* stream) {
    return halo_add_call<float>(out, recv, U, kappa, dims, face_phase, part_mask, flags, stream,
                                "lqcd_wilson_clover_halo_add_f32");
}
int lqcd_wilson_clover_halo_add_f64(double* out, const double* const recv[8], const double* U, double kappa,
                                    const int dims[4], const int face_phase[8], unsigned part_mask, unsigned flags,
                                    void* stream) {
    return halo_add_call<double>(out, recv, U, kappa, dims, face_phase, part_mask, flags, stream,
                                 "lqcd_wilson_clover_halo_add_f64");
}

}  // extern "C"
