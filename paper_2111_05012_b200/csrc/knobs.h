// knobs.h -- tuning knobs (lqcd_set_fine_tile / lqcd_set_knob), one set per calling host thread like the last-error
// string: two threads with different settings do not race.  Results never depend on them.
#pragma once
namespace lqcd {
struct Knobs {
    int fine_tile[4] = {0, 0, 0, 0};  // 0 = automatic
    int fine_tslab = 0;               // 0 = automatic; >0 = z tiles per traversal slab; <0 = canonical order
    int coarse_rows_per_warp = 0;     // row tiles per warp, 0 = automatic
    int coarse_R = 0;                 // rows in flight per lane (1, 2, 4), 0 = automatic (2)
    int coarse_warps = 0;             // warps per CTA of the coarse kernel, 0 = automatic
    int transfer_warps = 0;           // warps per CTA of restrict, 0 = automatic
    int mrhs_tensor = 0;              // 0 = tcgen05 path of coarse_mult_mrhs when it applies; -1 = never
    int mrhs_stages = 0;              // pipeline stages of coarse_mult_mrhs, 0 = as many as fit
    int fine_mrhs = 0;                // -1 = wilson_clover_mult_mrhs applies the single-right-hand-side kernel per vector
    int sap_fused = 0;                // 0 = shared-memory-resident inner-domain solver when it fits; -1 = never
    int site_order = 0;               // 0 = tiled site order (4 x 4 x 2 chunks) when the extents allow; -1 = canonical.
                                      // Changes the NATIVE layout: every native field must be packed after setting it
    int sap_group_residual = 0;       // 0 = SAP's intermediate residuals on the next group's domains only; -1 = all sites
    int host_slab_mb = 0;             // host-vector calls: smallest slab of the upload / compute / download pipeline in MB;
                                      // 0 = 16; -1 = never pipeline (one-shot path)
    int sap_tmem = 0;                 // 0 = the resident solver parks links and clover blocks in tensor memory (fp32 4^4
                                      // domains); -1 = shared memory only
};
extern thread_local Knobs g_knobs;
}  // namespace lqcd
