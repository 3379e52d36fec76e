// wilson_clover.cu -- rows A1/A2 of the hot path: the fine-lattice Wilson-clover operator,
//   out(x) = in(x) + F(x) in(x) - kappa sum_mu [ (1 - g_mu) U_mu(x) in(x+mu) + (1 + g_mu) U_mu^dag(x-mu) in(x-mu) ]
// (Eq. 1) and its gamma5-conjugate D^dag = gamma5 D gamma5 (Eq. 2).
//
// Design: one thread per lattice site (as the paper's GPU mapping),
// but each CTA owns a compact 4-D tile of sites so that most neighbour spinors and backward links are
// served by L1/L2 rather than HBM; native chunk-of-32 SoA layouts give 128-bit fully coalesced accesses;
// the clover term and the output are streamed with evict-first / streaming hints so that they do not
// displace the spinor and link lines that still have reuse; halo-free neighbour indexing modulo L with the
// boundary phase bc[mu] applied on hops that wrap.  Spin projection uses the rank-2 structure of
// (1 -+ g_mu) in the chiral basis: only two colour vectors per hop are multiplied by the link.
// The dagger variant swaps the two projectors (gamma5 (1 -+ g_mu) gamma5 = (1 +- g_mu), [F, gamma5] = 0),
// so it costs exactly the same traffic and arithmetic.
#include "common.cuh"
#include "fermion.cuh"
#include "knobs.h"
#include "layout.cuh"

namespace lqcd {

struct FineParams {
    int L[4];      // lattice extents
    int tile[4];   // sites per CTA per direction
    int ntile[4];  // tiles per direction
    int bc[4];     // +1 / -1
    int tilevol;   // threads that own a site (<= blockDim.x)
    int tile_off;  // first tile of the launch (slab form: the grid covers a range of time slices; 0 otherwise)
    int warp_tiles;  // 1: tiled site order and a CTA tile made of whole 4 x 4 x 2 layout tiles: a warp owns one of them
    int wt[3];       // ... layout tiles per CTA tile in x, y, z
    FastDiv d_wt[3];
    int zslab;     // traversal slab extent in z tiles (0 = canonical tile order)
    int per_slab, nslab_full;  // zslab * ntile[3]; number of slabs of full height
    FastDiv d_ntile[3], d_tile[3], d_per_slab, d_zslab, d_dom[4];
    // domain-decomposed variant D_SAP; unused by the plain operator
    int dom[4];    // domain extents (the aggregation block)
    int multi[4];  // 1 if there is more than one domain in that direction (else no hop is ever cut)
    int parity;    // 0 = all domains, 1 = even domains only, 2 = odd domains only
    int keep;      // with parity != 0: 1 = leave the sites of the other group untouched instead of zeroing them
    int cut_lat;   // 1 = hops are cut where they leave the LATTICE (sharded interior pass), not where they leave a domain
    SiteOrder ord;  // native position of a site (layout.cuh)
};

// Which site is mine: CTA -> tile (x tiles fastest; optionally z-slabbed traversal), thread -> site in tile.  All
// divisions by run-time extents are multiply-high with host-computed reciprocals (the index decode was a quarter of
// the integer work of the fine kernel).  False for the padding threads of a CTA.
__device__ __forceinline__ bool fine_decode(const FineParams& P, int x[4], int& s_out) {
    int tid = threadIdx.x;
    if (tid >= P.tilevol) return false;
    int b = blockIdx.x + P.tile_off, q;
    int tc[4];
    q = P.d_ntile[0].div(b); tc[0] = b - q * P.ntile[0]; b = q;
    q = P.d_ntile[1].div(b); tc[1] = b - q * P.ntile[1]; b = q;
    if (P.zslab > 0) {
        // order: x, y, z within slab, t, slab  (keeps the +-t neighbours of a slab resident in L2)
        const int slab = P.d_per_slab.div(b);
        const int r = b - slab * P.per_slab;
        if (slab >= P.nslab_full) {  // ragged last slab (rare: slabs are chosen of equal height when possible)
            const int zs = P.ntile[2] - P.nslab_full * P.zslab;
            const int rr = b - P.nslab_full * P.per_slab;
            tc[2] = P.nslab_full * P.zslab + rr % zs;
            tc[3] = rr / zs;
        } else {
            tc[3] = P.d_zslab.div(r);
            tc[2] = slab * P.zslab + (r - tc[3] * P.zslab);
        }
    } else {
        tc[3] = P.d_ntile[2].div(b);
        tc[2] = b - tc[3] * P.ntile[2];
    }
    if (P.warp_tiles) {
        // lane = position inside a 4 x 4 x 2 layout tile (= chunk of the native layouts): every 128-bit access of the
        // warp is one contiguous 512-byte row; warps enumerate the layout tiles of the CTA tile, x fastest
        int w = tid >> 5;
        q = P.d_wt[0].div(w); const int wx = w - q * P.wt[0]; w = q;
        q = P.d_wt[1].div(w); const int wy = w - q * P.wt[1]; w = q;
        q = P.d_wt[2].div(w); const int wz = w - q * P.wt[2]; w = q;
        x[0] = tc[0] * P.tile[0] + 4 * wx + (tid & 3);
        x[1] = tc[1] * P.tile[1] + 4 * wy + ((tid >> 2) & 3);
        x[2] = tc[2] * P.tile[2] + 2 * wz + ((tid >> 4) & 1);
        x[3] = tc[3] * P.tile[3] + w;
    } else {
        q = P.d_tile[0].div(tid); x[0] = tc[0] * P.tile[0] + (tid - q * P.tile[0]); tid = q;
        q = P.d_tile[1].div(tid); x[1] = tc[1] * P.tile[1] + (tid - q * P.tile[1]); tid = q;
        q = P.d_tile[2].div(tid); x[2] = tc[2] * P.tile[2] + (tid - q * P.tile[2]); tid = q;
        x[3] = tc[3] * P.tile[3] + tid;
    }
    s_out = P.ord.index(x);  // native position: chunk = s >> 5, lane = s & 31
    return true;

}

// one directed hop: FWD: (1 + SGN g_mu) U_mu(x) in(x+mu);  !FWD: (1 + SGN g_mu) U_mu^dag(x-mu) in(x-mu)
template <int MU, bool FWD, int SGN, bool L12, bool G64, typename T>
__device__ __forceinline__ void hop(T acc[24], const T* __restrict__ in, const T* __restrict__ U, int s_link, int s_nb,
                                    T ph) {
    T p[24], h[12], u[18], g[12];
    load_spinor<T, G64>(p, in, s_nb);
    load_link<T, L12, G64>(u, U, s_link, MU);
    project<MU, SGN, T>(h, p);
    su3_mult<FWD, T>(g, u, h);
    reconstruct<MU, SGN, T>(acc, g, ph);
}

// DD: the domain-decomposed operator D_SAP -- hops whose two ends lie in different domains are switched off
// (no load is issued for them), and with P.parity != 0 only the sites of even (odd) domains are computed, the
// others are set to zero (D_SAP^(e/o) = P_e/o D_SAP P_e/o).
// DD = 2: the even/odd mode; active data then comes in alternate 64-byte half lines -> 64-byte L2 granularity.
// RES: the Richardson residual out = rhs - D in in the same pass: one more streamed read.
template <typename T, bool DAG, bool L12, int DD, bool RES, int MAXTHREADS, int MINBLOCKS>
__global__ void __launch_bounds__(MAXTHREADS, MINBLOCKS)
    k_wilson_clover(T* __restrict__ out, const T* __restrict__ in, const T* __restrict__ U, const T* __restrict__ clover,
                    const T* __restrict__ rhs, T kappa, FineParams P) {
    int x[4], s;
    if (!fine_decode(P, x, s)) return;

    // neighbour sites (halo-free, modulo L; native positions) and wrap phases
    int sf[4], sb[4];
    T pf[4], pb[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const bool wf = (x[mu] == P.L[mu] - 1), wb = (x[mu] == 0);
        sf[mu] = P.ord.fwd(s, mu, x[mu]);
        sb[mu] = P.ord.bwd(s, mu, x[mu]);
        pf[mu] = wf ? (T)P.bc[mu] : (T)1;
        pb[mu] = wb ? (T)P.bc[mu] : (T)1;
    }

    T acc[24];
#pragma unroll
    for (int r = 0; r < 24; r++) acc[r] = 0;

    // link sites: U_mu(x) for the forward hop, U_mu(x - mu) for the backward hop
    int lf[4] = {s, s, s, s}, lb[4] = {sb[0], sb[1], sb[2], sb[3]};
    // Domain decomposition: a hop that leaves my domain is switched off.  Control flow stays uniform (the eight
    // hops are one straight-line, software-pipelined instruction stream, as in D): a cut hop gets phase 0 and is
    // redirected to operands this thread needs anyway -- its own spinor and the link of the opposite hop of the
    // same direction -- so it costs L1 hits and idle flops but no DRAM traffic (the links and neighbour spinors
    // across a domain face are never touched).
    if (DD) {
        int par = 0;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const int X = P.d_dom[mu].div(x[mu]), lx = x[mu] - X * P.dom[mu];
            par += X;
            const bool ef = P.cut_lat ? x[mu] == P.L[mu] - 1 : lx == P.dom[mu] - 1;
            const bool eb = P.cut_lat ? x[mu] == 0 : lx == 0;
            if (P.multi[mu] && ef) {  // forward hop leaves the domain
                sf[mu] = s;
                lf[mu] = sb[mu];
                pf[mu] = 0;
            }
            if (P.multi[mu] && eb) {  // backward hop leaves the domain
                lb[mu] = s;
                sb[mu] = s;
                pb[mu] = 0;
            }
        }
        if (P.parity != 0 && (par & 1) != P.parity - 1) {  // my domain is not in the selected group: zero
            if (!P.keep) store_spinor<T>(out, s, acc);
            return;
        }
    }

    // D: forward hops carry (1 - g_mu), backward (1 + g_mu); D^dag: the two are swapped.
    constexpr int SF = DAG ? +1 : -1, SB = DAG ? -1 : +1;
    constexpr bool G64 = (DD == 2);
    hop<0, true, SF, L12, G64, T>(acc, in, U, lf[0], sf[0], pf[0]);
    hop<0, false, SB, L12, G64, T>(acc, in, U, lb[0], sb[0], pb[0]);
    hop<1, true, SF, L12, G64, T>(acc, in, U, lf[1], sf[1], pf[1]);
    hop<1, false, SB, L12, G64, T>(acc, in, U, lb[1], sb[1], pb[1]);
    hop<2, true, SF, L12, G64, T>(acc, in, U, lf[2], sf[2], pf[2]);
    hop<2, false, SB, L12, G64, T>(acc, in, U, lb[2], sb[2], pb[2]);
    hop<3, true, SF, L12, G64, T>(acc, in, U, lf[3], sf[3], pf[3]);
    hop<3, false, SB, L12, G64, T>(acc, in, U, lb[3], sb[3], pb[3]);

    // site-diagonal part: (1 + F) in, then out = that - kappa * hops
    T p[24], o[24];
    load_spinor<T, (DD == 2)>(p, in, s);
#pragma unroll
    for (int r = 0; r < 24; r++) o[r] = fma(-kappa, acc[r], p[r]);
#pragma unroll
    for (int chi = 0; chi < 2; chi++) {
        T cl[36];
        load_clover_block<T, (DD == 2)>(cl, clover, s, chi);
        herm6_madd<T>(o + 12 * chi, cl, p + 12 * chi);
    }
    if (RES) {
        constexpr int NV = VecOf<T>::NV, NJ = 24 / NV;
        const T* base = rhs + ((long long)(s >> 5) * NJ * CH + (s & 31)) * NV;
#pragma unroll
        for (int j = 0; j < NJ; j++) {
            const V16<T> v = ld16_stream(base + (long long)j * CH * NV);
#pragma unroll
            for (int q = 0; q < NV; q++) o[j * NV + q] = v.r[q] - o[j * NV + q];
        }
    }
    store_spinor<T>(out, s, o);
}

// Automatic CTA tile: powers of two dividing L, x first (128-byte lines hold 8 consecutive x sites of one
// vec16 row), up to 128 threads.
static void auto_tile(const int L[4], int tile[4]) {
    const int cap[4] = {8, 4, 4, 4};
    int vol = 1;
    for (int mu = 0; mu < 4; mu++) {
        int t = 1;
        while (t * 2 <= cap[mu] && L[mu] % (t * 2) == 0 && vol * t * 2 <= 128) t *= 2;
        tile[mu] = t;
        vol *= t;
    }
    // use left-over thread budget (small or odd lattices)
    for (int mu = 0; mu < 4 && vol < 128; mu++)
        while (L[mu] % (tile[mu] * 2) == 0 && vol * 2 <= 128) {
            tile[mu] *= 2;
            vol *= 2;
        }
}

// Launch geometry of the fine kernels: CTA tile, tile traversal, reciprocals of the index decode.  real_bytes = 4 / 8.
static int fine_setup(FineParams& P, long long& ntiles_out, const int dims[4], const int bc[4], const int* domain,
                      unsigned flags, int real_bytes, const char* what) {
    for (int mu = 0; mu < 4; mu++) {
        if (bc[mu] != 1 && bc[mu] != -1) {
            set_error("%s: bc[%d] = %d not in {+1,-1}", what, mu, bc[mu]);
            return LQCD_EINVAL;
        }
        P.L[mu] = dims[mu];
        P.bc[mu] = bc[mu];
        P.dom[mu] = dims[mu];
        P.multi[mu] = 0;
        if (domain) {
            if (domain[mu] < 1 || dims[mu] % domain[mu]) {
                set_error("%s: domain[%d] = %d does not divide dims[%d] = %d", what, mu, domain[mu], mu, dims[mu]);
                return LQCD_EINVAL;
            }
            P.dom[mu] = domain[mu];
            P.multi[mu] = dims[mu] / domain[mu] > 1;
        }
    }
    P.parity = (flags & LQCD_DOMAIN_EVEN) ? 1 : (flags & LQCD_DOMAIN_ODD) ? 2 : 0;
    P.keep = 0;
    P.cut_lat = 0;
    P.tile_off = 0;
    P.ord.set(dims);
    bool user_ok = g_knobs.fine_tile[0] > 0;
    for (int mu = 0; mu < 4 && user_ok; mu++) user_ok = dims[mu] % g_knobs.fine_tile[mu] == 0;
    if (user_ok)
        for (int mu = 0; mu < 4; mu++) P.tile[mu] = g_knobs.fine_tile[mu];
    else if (P.parity != 0)
        auto_tile(P.dom, P.tile);  // tiles inside one domain: a whole CTA is either computed or zero-filled
    else
        auto_tile(dims, P.tile);
    P.tilevol = 1;
    long long ntiles = 1;
    for (int mu = 0; mu < 4; mu++) {
        P.ntile[mu] = dims[mu] / P.tile[mu];
        P.tilevol *= P.tile[mu];
        ntiles *= P.ntile[mu];
    }
    P.warp_tiles = P.ord.tiled && P.tile[0] % 4 == 0 && P.tile[1] % 4 == 0 && P.tile[2] % 2 == 0;
    P.wt[0] = P.warp_tiles ? P.tile[0] / 4 : 1;
    P.wt[1] = P.warp_tiles ? P.tile[1] / 4 : 1;
    P.wt[2] = P.warp_tiles ? P.tile[2] / 2 : 1;
    for (int mu = 0; mu < 3; mu++) P.d_wt[mu].set(P.wt[mu]);
    // Traversal: canonical tile order keeps the +-t neighbours in L2 only while one time-slice of operands
    // (V3 * bytes/site) is well below the L2 capacity; beyond that, walk the lattice in z-slabs whose
    // per-time-slice footprint is <= ~32 MB (z faces of a slab are re-read: +2-3% traffic).
    if (g_knobs.fine_tslab > 0) {
        P.zslab = g_knobs.fine_tslab;
    } else if (g_knobs.fine_tslab < 0) {
        P.zslab = 0;
    } else {
        const double site_bytes = 192.0 * real_bytes;
        const double slice = (double)dims[0] * dims[1] * dims[2] * site_bytes;
        P.zslab = 0;
        if (slice > 40e6) {
            const double layer = (double)dims[0] * dims[1] * P.tile[2] * site_bytes;  // one z-tile layer
            int zs = (int)(32e6 / layer);
            if (zs < 1) zs = 1;
            while (zs > 1 && P.ntile[2] % zs) zs--;  // prefer slabs of equal height
            P.zslab = zs;
        }
    }
    if (P.zslab >= P.ntile[2]) P.zslab = 0;
    // reciprocals for the index decode (exact while n * d < 2^32: n is a tile index or a thread index)
    P.per_slab = (P.zslab > 0 ? P.zslab : 1) * P.ntile[3];
    P.nslab_full = P.zslab > 0 ? P.ntile[2] / P.zslab : 0;
    {
        long long dmax = P.per_slab;
        for (int mu = 0; mu < 3; mu++) dmax = P.ntile[mu] > dmax ? P.ntile[mu] : dmax;
        if (ntiles * dmax >= 0x100000000LL) {
            set_error("%s: lattice too large for the 32-bit index decode", what);
            return LQCD_EUNSUPPORTED;
        }
    }
    for (int mu = 0; mu < 3; mu++) {
        P.d_ntile[mu].set(P.ntile[mu]);
        P.d_tile[mu].set(P.tile[mu]);
    }
    P.d_per_slab.set(P.per_slab);
    P.d_zslab.set(P.zslab > 0 ? P.zslab : 1);
    for (int mu = 0; mu < 4; mu++) P.d_dom[mu].set(P.dom[mu]);
    ntiles_out = ntiles;
    return LQCD_OK;
}

// domain == NULL: the plain operator D; otherwise D_SAP with those domains
template <typename T>
int wilson_clover_call(T* out, const T* in, const T* U, const T* clover, const T* rhs, T kappa, const int dims[4],
                       const int bc[4], const int* domain, unsigned flags, void* stream, const char* what) {
    clear_error();
    if (!out || !in || !U || !clover || check_dims(dims) || !bc) {
        set_error("%s: null pointer or non-positive dim", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(out) || !aligned16(in) || !aligned16(U) || !aligned16(clover)) {
        set_error("%s: pointers must be 16-byte aligned", what);
        return LQCD_EINVAL;
    }
    if (out == in) {
        set_error("%s: out must not alias in", what);
        return LQCD_EINVAL;
    }
    if (rhs && (!aligned16(rhs) || domain || (flags & LQCD_DAGGER) || rhs == out)) {  // rhs is read through the
        // read-only path (ld.global.nc) and out is written: the two must not overlap
        set_error("%s: the residual form needs an aligned rhs distinct from out and takes neither a domain nor "
                  "LQCD_DAGGER", what);
        return LQCD_EINVAL;
    }
    const unsigned allowed = LQCD_DAGGER | LQCD_LINKS_12 | (domain ? (LQCD_DOMAIN_EVEN | LQCD_DOMAIN_ODD) : 0u);
    if ((flags & ~allowed) || ((flags & LQCD_DOMAIN_EVEN) && (flags & LQCD_DOMAIN_ODD))) {
        set_error("%s: unknown or contradictory flag bits 0x%x", what, flags);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) {
        set_error("%s: volume exceeds 2^31-1 sites", what);
        return LQCD_EUNSUPPORTED;
    }
    FineParams P;
    long long ntiles = 0;
    {
        const int rc = fine_setup(P, ntiles, dims, bc, domain, flags, (int)sizeof(T), what);
        if (rc) return rc;
    }
    int threads = (P.tilevol + 31) / 32 * 32;
    const bool dag = flags & LQCD_DAGGER, l12 = flags & LQCD_LINKS_12;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = (unsigned)ntiles;
    // registers per thread: fp32 128 (4 CTAs/SM), fp64 168 (3 CTAs/SM) -- measured best on B200
#define LAUNCH_R(DAG, L12, DD, RES)                                                                          \
    do {                                                                                                     \
        if (threads <= 128)                                                                                  \
            k_wilson_clover<T, DAG, L12, DD, RES, 128, (sizeof(T) == 4 ? 4 : 3)>                             \
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);                               \
        else                                                                                                 \
            k_wilson_clover<T, DAG, L12, DD, RES, 256, (sizeof(T) == 4 ? 2 : 1)>                             \
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);                               \
    } while (0)
#define LAUNCH(DAG, L12, DD) LAUNCH_R(DAG, L12, DD, false)
#define LAUNCH_DD(DAG, L12)                                                                                  \
    do {                                                                                                     \
        if (domain && P.parity != 0) LAUNCH(DAG, L12, 2);                                                    \
        else if (domain) LAUNCH(DAG, L12, 1);                                                                \
        else LAUNCH(DAG, L12, 0);                                                                            \
    } while (0)
    if (rhs && l12) LAUNCH_R(false, true, 0, true);
    else if (rhs) LAUNCH_R(false, false, 0, true);
    else if (dag && l12) LAUNCH_DD(true, true);
    else if (dag) LAUNCH_DD(true, false);
    else if (l12) LAUNCH_DD(false, true);
    else LAUNCH_DD(false, false);
#undef LAUNCH_DD
#undef LAUNCH
#undef LAUNCH_R
    count_launch();
    return check_launch(what);
}
// D (D^dag) on the time slices [t0, t1) only: the tiles of those slices in canonical tile order (tiles of one time
// slice are then consecutive), as host_api.cu needs to run the operator slab by slab under the upload of the next
// slab.  Arguments were validated by the caller; t0, t1 multiples of the CTA tile's extent in t.
int fine_tile_extent_t(const int dims[4], const int bc[4], int real_bytes) {
    FineParams P;
    long long ntiles = 0;
    if (fine_setup(P, ntiles, dims, bc, nullptr, 0u, real_bytes, "fine_tile_extent_t")) return 0;
    return P.tile[3];
}
template <typename T>
int wilson_clover_slab_call(T* out, const T* in, const T* U, const T* clover, T kappa, const int dims[4], const int bc[4],
                            unsigned flags, int t0, int t1, void* stream, const char* what) {
    FineParams P;
    long long ntiles = 0;
    {
        const int rc = fine_setup(P, ntiles, dims, bc, nullptr, 0u, (int)sizeof(T), what);
        if (rc) return rc;
    }
    if (t0 % P.tile[3] || t1 % P.tile[3] || t0 < 0 || t1 > dims[3] || t1 <= t0) {
        set_error("%s: slab [%d, %d) is not made of whole tiles", what, t0, t1);
        return LQCD_EINVAL;
    }
    P.zslab = 0;  // canonical tile order: x, y, z, t
    P.per_slab = P.ntile[3];
    P.nslab_full = 0;
    const long long per_t = (long long)P.ntile[0] * P.ntile[1] * P.ntile[2];
    P.tile_off = (int)(per_t * (t0 / P.tile[3]));
    const unsigned grid = (unsigned)(per_t * ((t1 - t0) / P.tile[3]));
    const int threads = (P.tilevol + 31) / 32 * 32;
    const bool dag = flags & LQCD_DAGGER, l12 = flags & LQCD_LINKS_12;
    cudaStream_t st = (cudaStream_t)stream;
    const T* rhs = nullptr;
#define LAUNCH_S(DAG, L12)                                                                                   \
    do {                                                                                                     \
        if (threads <= 128)                                                                                  \
            k_wilson_clover<T, DAG, L12, 0, false, 128, (sizeof(T) == 4 ? 4 : 3)>                            \
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);                               \
        else                                                                                                 \
            k_wilson_clover<T, DAG, L12, 0, false, 256, (sizeof(T) == 4 ? 2 : 1)>                            \
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);                               \
    } while (0)
    if (dag && l12) LAUNCH_S(true, true);
    else if (dag) LAUNCH_S(true, false);
    else if (l12) LAUNCH_S(false, true);
    else LAUNCH_S(false, false);
#undef LAUNCH_S
    count_launch();
    return check_launch(what);
}
template int wilson_clover_slab_call<float>(float*, const float*, const float*, const float*, float, const int*,
                                            const int*, unsigned, int, int, void*, const char*);
template int wilson_clover_slab_call<double>(double*, const double*, const double*, const double*, double, const int*,
                                             const int*, unsigned, int, int, void*, const char*);

// r := b - D x on the domains of ONE group only (flags: LQCD_DOMAIN_EVEN / ODD), the other sites of r untouched: what
// SAP needs between two half sweeps, where only the group solved next reads the residual (sap.cu).  The full operator
// (no hop is cut): the even/odd kernel variant with the cut switched off, the residual epilogue and no zero fill.
template <typename T>
int wilson_clover_residual_group_call(T* r, const T* x, const T* U, const T* clover, const T* b, T kappa,
                                      const int dims[4], const int bc[4], const int domain[4], unsigned flags,
                                      void* stream, const char* what) {
    // (arguments were validated by the caller, sap_call)
    FineParams P;
    long long ntiles = 0;
    {
        const int rc = fine_setup(P, ntiles, dims, bc, domain, flags & (LQCD_DOMAIN_EVEN | LQCD_DOMAIN_ODD),
                                  (int)sizeof(T), what);
        if (rc) return rc;
    }
    for (int mu = 0; mu < 4; mu++) P.multi[mu] = 0;
    P.keep = 1;
    const int threads = (P.tilevol + 31) / 32 * 32;
    const bool l12 = flags & LQCD_LINKS_12;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = (unsigned)ntiles;
#define LAUNCH_G(L12)                                                                                        \
    do {                                                                                                     \
        if (threads <= 128)                                                                                  \
            k_wilson_clover<T, false, L12, 2, true, 128, (sizeof(T) == 4 ? 4 : 3)>                           \
                <<<grid, threads, 0, st>>>(r, x, U, clover, b, kappa, P);                                    \
        else                                                                                                 \
            k_wilson_clover<T, false, L12, 2, true, 256, (sizeof(T) == 4 ? 2 : 1)>                           \
                <<<grid, threads, 0, st>>>(r, x, U, clover, b, kappa, P);                                    \
    } while (0)
    if (l12) LAUNCH_G(true);
    else LAUNCH_G(false);
#undef LAUNCH_G
    count_launch();
    return check_launch(what);
}
template int wilson_clover_residual_group_call<float>(float*, const float*, const float*, const float*, const float*,
                                                      float, const int*, const int*, const int*, unsigned, void*,
                                                      const char*);
template int wilson_clover_residual_group_call<double>(double*, const double*, const double*, const double*,
                                                       const double*, double, const int*, const int*, const int*,
                                                       unsigned, void*, const char*);

// The interior pass of the sharded operator (halo.cu): D on the LOCAL lattice with every hop that leaves it in a
// partitioned direction (bit mu of part_mask) switched off -- the D_SAP kernel with the local lattice as its one
// domain and the cut forced in those directions; the other directions wrap with bc[mu] as in D.
// rhs != NULL: the residual form out = rhs - (that operator) in.
template <typename T>
int wilson_clover_interior_call(T* out, const T* in, const T* U, const T* clover, const T* rhs, T kappa,
                                const int dims[4], const int bc[4], unsigned part_mask, unsigned flags, void* stream,
                                const char* what, const int* domain) {
    // flags may carry LQCD_DOMAIN_EVEN / ODD with rhs and domain: the residual on that group of domains only, the
    // other sites untouched (the sharded SAP's intermediate residuals)
    clear_error();
    const unsigned group = flags & (LQCD_DOMAIN_EVEN | LQCD_DOMAIN_ODD);
    flags &= ~group;
    if (group && (!rhs || !domain || group == (LQCD_DOMAIN_EVEN | LQCD_DOMAIN_ODD))) {
        set_error("%s: a domain group needs the residual form, a domain and ONE of LQCD_DOMAIN_EVEN / ODD", what);
        return LQCD_EINVAL;
    }
    if (!out || !in || !U || !clover || check_dims(dims) || !bc) {
        set_error("%s: null pointer or non-positive dim", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(out) || !aligned16(in) || !aligned16(U) || !aligned16(clover) || out == in) {
        set_error("%s: pointers must be 16-byte aligned and out must not alias in", what);
        return LQCD_EINVAL;
    }
    if ((flags & ~(LQCD_DAGGER | LQCD_LINKS_12)) || part_mask > 15u) {
        set_error("%s: bad flags 0x%x or part_mask 0x%x", what, flags, part_mask);
        return LQCD_EINVAL;
    }
    if (rhs && (!aligned16(rhs) || (flags & LQCD_DAGGER) || rhs == out)) {
        set_error("%s: the residual form needs an aligned rhs distinct from out and does not take LQCD_DAGGER", what);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) {
        set_error("%s: volume exceeds 2^31-1 sites", what);
        return LQCD_EUNSUPPORTED;
    }
    FineParams P;
    long long ntiles = 0;
    {
        const int rc = fine_setup(P, ntiles, dims, bc, group ? domain : dims, group, (int)sizeof(T), what);
        if (rc) return rc;
    }
    for (int mu = 0; mu < 4; mu++) P.multi[mu] = (part_mask >> mu) & 1;
    P.cut_lat = 1;
    P.keep = group ? 1 : 0;
    const int threads = (P.tilevol + 31) / 32 * 32;
    const bool dag = flags & LQCD_DAGGER, l12 = flags & LQCD_LINKS_12;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = (unsigned)ntiles;
#define LAUNCH_I(DAG, L12, RES)                                                                              \
    do {                                                                                                     \
        if (threads <= 128)                                                                                  \
            k_wilson_clover<T, DAG, L12, 1, RES, 128, (sizeof(T) == 4 ? 4 : 3)>                              \
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);                               \
        else                                                                                                 \
            k_wilson_clover<T, DAG, L12, 1, RES, 256, (sizeof(T) == 4 ? 2 : 1)>                              \
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);                               \
    } while (0)
    if (group && l12) {
        if (threads <= 128)
            k_wilson_clover<T, false, true, 2, true, 128, (sizeof(T) == 4 ? 4 : 3)>
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);
        else
            k_wilson_clover<T, false, true, 2, true, 256, (sizeof(T) == 4 ? 2 : 1)>
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);
    } else if (group) {
        if (threads <= 128)
            k_wilson_clover<T, false, false, 2, true, 128, (sizeof(T) == 4 ? 4 : 3)>
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);
        else
            k_wilson_clover<T, false, false, 2, true, 256, (sizeof(T) == 4 ? 2 : 1)>
                <<<grid, threads, 0, st>>>(out, in, U, clover, rhs, kappa, P);
    }
    else if (rhs && l12) LAUNCH_I(false, true, true);
    else if (rhs) LAUNCH_I(false, false, true);
    else if (dag && l12) LAUNCH_I(true, true, false);
    else if (dag) LAUNCH_I(true, false, false);
    else if (l12) LAUNCH_I(false, true, false);
    else LAUNCH_I(false, false, false);
#undef LAUNCH_I
    count_launch();
    return check_launch(what);
}
template int wilson_clover_interior_call<float>(float*, const float*, const float*, const float*, const float*, float,
                                                const int*, const int*, unsigned, unsigned, void*, const char*,
                                                const int*);
template int wilson_clover_interior_call<double>(double*, const double*, const double*, const double*, const double*,
                                                 double, const int*, const int*, unsigned, unsigned, void*,
                                                 const char*, const int*);

template int wilson_clover_call<float>(float*, const float*, const float*, const float*, const float*, float,
                                       const int*, const int*, const int*, unsigned, void*, const char*);
template int wilson_clover_call<double>(double*, const double*, const double*, const double*, const double*, double,
                                        const int*, const int*, const int*, unsigned, void*, const char*);


// ---- F4 (fine half): D on NRHS right-hand sides at once ---------------------------------------------------
// Every link and clover block is loaded ONCE per site and applied to NRHS spinors: compulsory traffic per site drops
// from NRHS * 768 B to 576 + NRHS * 192 B (18-real links): 1.6x less at NRHS = 2.  One thread per site as in
// k_wilson_clover, same tile / traversal geometry; registers, not bandwidth, limit NRHS (24 accumulators per
// right-hand side).  Right-hand side k lives at in + k * rstride (native spinors back to back).
template <int MU, bool FWD, int SGN, bool L12, int NRHS, typename T>
__device__ __forceinline__ void hop_mrhs(T (&acc)[NRHS][24], const T* __restrict__ in, long long rstride,
                                         const T* __restrict__ U, int s_link, int s_nb, T ph) {
    T u[18];
    load_link<T, L12>(u, U, s_link, MU);
#pragma unroll
    for (int k = 0; k < NRHS; k++) {
        T p[24], h[12], g[12];
        load_spinor<T>(p, in + k * rstride, s_nb);
        project<MU, SGN, T>(h, p);
        su3_mult<FWD, T>(g, u, h);
        reconstruct<MU, SGN, T>(acc[k], g, ph);
    }
}

// RES: out_k = rhs_k - D in_k (the residual of SAP / of a Richardson step), rhs_k = rhs + k * rstride
template <typename T, bool DAG, bool L12, int NRHS, bool RES>
__global__ void __launch_bounds__(128, sizeof(T) == 4 ? 3 : 2)
    k_wilson_clover_mrhs(T* __restrict__ out, const T* __restrict__ in, long long rstride, const T* __restrict__ U,
                         const T* __restrict__ clover, const T* __restrict__ rhs, T kappa, FineParams P) {
    int x[4], s;
    if (!fine_decode(P, x, s)) return;
    if (P.parity != 0) {  // one group of domains only, the other sites untouched (SAP's intermediate residuals)
        int par = 0;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) par += P.d_dom[mu].div(x[mu]);
        if ((par & 1) != P.parity - 1) return;
    }
    int sf[4], sb[4];
    T pf[4], pb[4];
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        const bool wf = (x[mu] == P.L[mu] - 1), wb = (x[mu] == 0);
        sf[mu] = P.ord.fwd(s, mu, x[mu]);
        sb[mu] = P.ord.bwd(s, mu, x[mu]);
        pf[mu] = wf ? (T)P.bc[mu] : (T)1;
        pb[mu] = wb ? (T)P.bc[mu] : (T)1;
    }
    T acc[NRHS][24];
#pragma unroll
    for (int k = 0; k < NRHS; k++)
#pragma unroll
        for (int r = 0; r < 24; r++) acc[k][r] = 0;
    constexpr int SF = DAG ? +1 : -1, SB = DAG ? -1 : +1;
    hop_mrhs<0, true, SF, L12, NRHS, T>(acc, in, rstride, U, s, sf[0], pf[0]);
    hop_mrhs<0, false, SB, L12, NRHS, T>(acc, in, rstride, U, sb[0], sb[0], pb[0]);
    hop_mrhs<1, true, SF, L12, NRHS, T>(acc, in, rstride, U, s, sf[1], pf[1]);
    hop_mrhs<1, false, SB, L12, NRHS, T>(acc, in, rstride, U, sb[1], sb[1], pb[1]);
    hop_mrhs<2, true, SF, L12, NRHS, T>(acc, in, rstride, U, s, sf[2], pf[2]);
    hop_mrhs<2, false, SB, L12, NRHS, T>(acc, in, rstride, U, sb[2], sb[2], pb[2]);
    hop_mrhs<3, true, SF, L12, NRHS, T>(acc, in, rstride, U, s, sf[3], pf[3]);
    hop_mrhs<3, false, SB, L12, NRHS, T>(acc, in, rstride, U, sb[3], sb[3], pb[3]);

    // site-diagonal part, one chirality block of the clover term at a time (loaded once for all right-hand sides)
    constexpr int NV = VecOf<T>::NV, NH = 12 / NV;  // vec16 rows per chirality half of a spinor
    const long long sp_off = ((long long)(s >> 5) * (24 / NV) * CH + (s & 31)) * NV;
#pragma unroll
    for (int chi = 0; chi < 2; chi++) {
        T cl[36];
        load_clover_block<T>(cl, clover, s, chi);
#pragma unroll
        for (int k = 0; k < NRHS; k++) {
            T p[12], o[12];
#pragma unroll
            for (int j = 0; j < NH; j++) {
                const V16<T> v = ld16(in + k * rstride + sp_off + (long long)(NH * chi + j) * CH * NV);
#pragma unroll
                for (int q = 0; q < NV; q++) p[j * NV + q] = v.r[q];
            }
#pragma unroll
            for (int r = 0; r < 12; r++) o[r] = fma(-kappa, acc[k][12 * chi + r], p[r]);
            herm6_madd<T>(o, cl, p);
#pragma unroll
            for (int j = 0; j < NH; j++) {
                V16<T> v;
#pragma unroll
                for (int q = 0; q < NV; q++) v.r[q] = o[j * NV + q];
                if (RES) {
                    const V16<T> bb = ld16_stream(rhs + k * rstride + sp_off + (long long)(NH * chi + j) * CH * NV);
#pragma unroll
                    for (int q = 0; q < NV; q++) v.r[q] = bb.r[q] - v.r[q];
                }
                st16_stream(out + k * rstride + sp_off + (long long)(NH * chi + j) * CH * NV, v);
            }
        }
    }
}

template <typename T>
int wilson_clover_mrhs_call(T* out, const T* in, const T* U, const T* clover, const T* rhs, T kappa, const int dims[4],
                            const int bc[4], int nrhs, unsigned flags, void* stream, const char* what,
                            const int* domain, unsigned group) {
    // domain != NULL and group = LQCD_DOMAIN_EVEN / ODD: only the sites of that group of domains are computed, the
    // others are left as they are (internal: the residual form between SAP's half sweeps)
    clear_error();
    if (!out || !in || !U || !clover || check_dims(dims) || !bc || nrhs < 1) {
        set_error("%s: null pointer, non-positive dim or nrhs < 1", what);
        return LQCD_EINVAL;
    }
    if (!aligned16(out) || !aligned16(in) || !aligned16(U) || !aligned16(clover) || out == in) {
        set_error("%s: pointers must be 16-byte aligned and out must not alias in", what);
        return LQCD_EINVAL;
    }
    if ((flags & ~(LQCD_DAGGER | LQCD_LINKS_12)) || (rhs && ((flags & LQCD_DAGGER) || !aligned16(rhs) || rhs == out))) {
        set_error("%s: unknown flag bits 0x%x (the residual form takes no LQCD_DAGGER and needs rhs distinct from out)",
                  what, flags);
        return LQCD_EINVAL;
    }
    if (volume(dims) > 0x7fffffffLL) {
        set_error("%s: volume exceeds 2^31-1 sites", what);
        return LQCD_EUNSUPPORTED;
    }
    FineParams P;
    long long ntiles = 0;
    {
        // tiles of at most 128 sites: the kernel is compiled for 128 threads
        const int rc = fine_setup(P, ntiles, dims, bc, group ? domain : nullptr, group, (int)sizeof(T), what);
        if (rc) return rc;
        for (int mu = 0; mu < 4; mu++) P.multi[mu] = 0;  // the full operator: no hop is cut
    }
    const long long rstride = (long long)nchunks(dims) * CH * 24;
    const int threads = (P.tilevol + 31) / 32 * 32;
    const bool dag = flags & LQCD_DAGGER, l12 = flags & LQCD_LINKS_12;
    cudaStream_t st = (cudaStream_t)stream;
    int k = 0;
    if (threads <= 128 && g_knobs.fine_mrhs >= 0) {
        for (; k + 2 <= nrhs; k += 2) {  // pairs of right-hand sides
            T* o = out + k * rstride;
            const T* i = in + k * rstride;
            const T* bk = rhs ? rhs + k * rstride : nullptr;
            const unsigned g = (unsigned)ntiles;
            if (rhs && l12) k_wilson_clover_mrhs<T, false, true, 2, true><<<g, threads, 0, st>>>(o, i, rstride, U, clover, bk, kappa, P);
            else if (rhs) k_wilson_clover_mrhs<T, false, false, 2, true><<<g, threads, 0, st>>>(o, i, rstride, U, clover, bk, kappa, P);
            else if (dag && l12) k_wilson_clover_mrhs<T, true, true, 2, false><<<g, threads, 0, st>>>(o, i, rstride, U, clover, bk, kappa, P);
            else if (dag) k_wilson_clover_mrhs<T, true, false, 2, false><<<g, threads, 0, st>>>(o, i, rstride, U, clover, bk, kappa, P);
            else if (l12) k_wilson_clover_mrhs<T, false, true, 2, false><<<g, threads, 0, st>>>(o, i, rstride, U, clover, bk, kappa, P);
            else k_wilson_clover_mrhs<T, false, false, 2, false><<<g, threads, 0, st>>>(o, i, rstride, U, clover, bk, kappa, P);
            count_launch();
        }
        const int rc = check_launch(what);
        if (rc) return rc;
    }
    for (; k < nrhs; k++) {  // an odd one out (or a user tile of more than 128 sites): the single-right-hand-side kernel
        const int rc = group ? wilson_clover_residual_group_call<T>(out + k * rstride, in + k * rstride, U, clover,
                                                                    rhs + k * rstride, kappa, dims, bc, domain,
                                                                    group | (flags & LQCD_LINKS_12), stream, what)
                             : wilson_clover_call<T>(out + k * rstride, in + k * rstride, U, clover,
                                                     rhs ? rhs + k * rstride : nullptr, kappa, dims, bc, nullptr,
                                                     flags, stream, what);
        if (rc) return rc;
    }
    return LQCD_OK;
}

template int wilson_clover_mrhs_call<float>(float*, const float*, const float*, const float*, const float*, float,
                                            const int*, const int*, int, unsigned, void*, const char*, const int*,
                                            unsigned);
template int wilson_clover_mrhs_call<double>(double*, const double*, const double*, const double*, const double*,
                                             double, const int*, const int*, int, unsigned, void*, const char*,
                                             const int*, unsigned);

}  // namespace lqcd

using namespace lqcd;

extern "C" {
int lqcd_wilson_clover_mult_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                const int dims[4], const int bc[4], unsigned flags, void* stream) {
    return wilson_clover_call<float>(out, in, U, clover, nullptr, kappa, dims, bc, nullptr, flags, stream,
                                     "lqcd_wilson_clover_mult_f32");
}
int lqcd_wilson_clover_mult_f64(double* out, const double* in, const double* U, const double* clover, double kappa,
                                const int dims[4], const int bc[4], unsigned flags, void* stream) {
    return wilson_clover_call<double>(out, in, U, clover, nullptr, kappa, dims, bc, nullptr, flags, stream,
                                      "lqcd_wilson_clover_mult_f64");
}
int lqcd_wilson_clover_dd_mult_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                   const int dims[4], const int bc[4], const int domain[4], unsigned flags,
                                   void* stream) {
    if (!domain) {
        set_error("lqcd_wilson_clover_dd_mult_f32: null domain");
        return LQCD_EINVAL;
    }
    return wilson_clover_call<float>(out, in, U, clover, nullptr, kappa, dims, bc, domain, flags, stream,
                                     "lqcd_wilson_clover_dd_mult_f32");
}
int lqcd_wilson_clover_dd_mult_f64(double* out, const double* in, const double* U, const double* clover, double kappa,
                                   const int dims[4], const int bc[4], const int domain[4], unsigned flags,
                                   void* stream) {
    if (!domain) {
        set_error("lqcd_wilson_clover_dd_mult_f64: null domain");
        return LQCD_EINVAL;
    }
    return wilson_clover_call<double>(out, in, U, clover, nullptr, kappa, dims, bc, domain, flags, stream,
                                      "lqcd_wilson_clover_dd_mult_f64");
}
}

extern "C" {
int lqcd_wilson_clover_residual_f32(float* r, const float* b, const float* x, const float* U, const float* clover,
                                    float kappa, const int dims[4], const int bc[4], unsigned flags, void* stream) {
    if (!b) {
        set_error("lqcd_wilson_clover_residual_f32: null rhs");
        return LQCD_EINVAL;
    }
    return wilson_clover_call<float>(r, x, U, clover, b, kappa, dims, bc, nullptr, flags, stream,
                                     "lqcd_wilson_clover_residual_f32");
}
int lqcd_wilson_clover_residual_f64(double* r, const double* b, const double* x, const double* U,
                                    const double* clover, double kappa, const int dims[4], const int bc[4],
                                    unsigned flags, void* stream) {
    if (!b) {
        set_error("lqcd_wilson_clover_residual_f64: null rhs");
        return LQCD_EINVAL;
    }
    return wilson_clover_call<double>(r, x, U, clover, b, kappa, dims, bc, nullptr, flags, stream,
                                      "lqcd_wilson_clover_residual_f64");
}
}

extern "C" {
int lqcd_wilson_clover_mult_mrhs_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                     const int dims[4], const int bc[4], int nrhs, unsigned flags, void* stream) {
    return wilson_clover_mrhs_call<float>(out, in, U, clover, nullptr, kappa, dims, bc, nrhs, flags, stream,
                                          "lqcd_wilson_clover_mult_mrhs_f32", nullptr, 0u);
}
int lqcd_wilson_clover_mult_mrhs_f64(double* out, const double* in, const double* U, const double* clover,
                                     double kappa, const int dims[4], const int bc[4], int nrhs, unsigned flags,
                                     void* stream) {
    return wilson_clover_mrhs_call<double>(out, in, U, clover, nullptr, kappa, dims, bc, nrhs, flags, stream,
                                           "lqcd_wilson_clover_mult_mrhs_f64", nullptr, 0u);
}
}
