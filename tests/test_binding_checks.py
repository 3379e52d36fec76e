"""The binding refuses tensors whose size does not match the geometry BEFORE the C call (the C ABI
sees raw pointers, only the binding knows the sizes).  No GPU needed: the checks precede every device access, so a
wrong size raises ValueError("... needs N") and a right size reaches the "expected a CUDA tensor" guard."""
import pytest
import torch

import paper_2111_05012_b200 as lq

DIMS, BLOCK, BC, NV = (4, 4, 4, 8), (2, 2, 2, 4), (1, 1, 1, -1), 4
CD = tuple(l // b for l, b in zip(DIMS, BLOCK))


def fields():
    z = lambda n: torch.zeros(n, dtype=torch.float32)
    return dict(x=z(lq.native_spinor_reals(DIMS)), y=z(lq.native_spinor_reals(DIMS)),
                U=z(lq.native_gauge_reals(DIMS)), U12=z(lq.native_gauge_reals(DIMS, True)),
                cl=z(lq.native_clover_reals(DIMS)), v=z(lq.native_nullvecs_reals(DIMS, BLOCK, NV)),
                xc=z(lq.native_coarse_vec_reals(CD, NV)), yc=z(lq.native_coarse_vec_reals(CD, NV)),
                A=z(lq.native_coarse_mat_reals(CD, NV)))


def size_error(fn, *a, **k):
    with pytest.raises(ValueError, match="needs"):
        fn(*a, **k)


def reaches_device_guard(fn, *a, **k):
    with pytest.raises(ValueError, match="CUDA tensor"):
        fn(*a, **k)


def test_fine_operator_sizes():
    f = fields()
    reaches_device_guard(lq.wilson_clover_mult, f["y"], f["x"], f["U"], f["cl"], 0.1, DIMS, BC)
    reaches_device_guard(lq.wilson_clover_mult, f["y"], f["x"], f["U12"], f["cl"], 0.1, DIMS, BC, links12=True)
    size_error(lq.wilson_clover_mult, f["y"], f["x"], f["U12"], f["cl"], 0.1, DIMS, BC)                 # 12 as 18
    size_error(lq.wilson_clover_mult, f["y"], f["x"], f["U"], f["cl"], 0.1, DIMS, BC, links12=True)     # 18 as 12
    size_error(lq.wilson_clover_mult, f["y"][:-4], f["x"], f["U"], f["cl"], 0.1, DIMS, BC)              # short out
    size_error(lq.wilson_clover_mult, f["y"], f["x"][4:], f["U"], f["cl"], 0.1, DIMS, BC)
    size_error(lq.wilson_clover_mult, f["y"], f["x"], f["U"], f["cl"][:-4], 0.1, DIMS, BC)
    size_error(lq.wilson_clover_dd_mult, f["y"], f["x"], f["U12"], f["cl"], 0.1, DIMS, BC, BLOCK)
    size_error(lq.wilson_clover_residual, f["y"], f["x"][:-4], f["x"], f["U"], f["cl"], 0.1, DIMS, BC)
    size_error(lq.wilson_clover_mult_interior, f["y"], f["x"], f["U"], f["cl"][:-4], 0.1, DIMS, BC, 8)


def test_coarse_and_transfer_sizes():
    f = fields()
    reaches_device_guard(lq.coarse_mult, f["yc"], f["xc"], f["A"], CD, NV)
    size_error(lq.coarse_mult, f["yc"], f["xc"], f["A"][:-2], CD, NV)
    size_error(lq.coarse_mult, f["yc"], f["xc"], f["A"], CD, NV + 1)          # nvec mismatch
    size_error(lq.coarse_mult, f["yc"][:-2], f["xc"], f["A"], CD, NV)
    reaches_device_guard(lq.restrict, f["xc"], f["x"], f["v"], DIMS, BLOCK, NV)
    size_error(lq.restrict, f["xc"], f["x"], f["v"][:-2], DIMS, BLOCK, NV)
    size_error(lq.restrict, f["xc"], f["x"], f["v"], DIMS, (4, 2, 2, 4), NV)     # block mismatch: other coarse size
    size_error(lq.prolong, f["y"], f["xc"][:-2], f["v"], DIMS, BLOCK, NV)
    size_error(lq.prolong, f["y"][:-4], f["xc"], f["v"], DIMS, BLOCK, NV)
    size_error(lq.orthonormalize_blocks, f["v"][:-2], DIMS, BLOCK, NV)
    size_error(lq.galerkin_coarse, f["U12"], f["cl"], f["v"], 0.1, DIMS, BC, BLOCK, NV)


def test_multi_rhs_sizes_are_per_vector():
    f = fields()
    K = 3
    xk, yk = torch.stack([f["xc"]] * K), torch.stack([f["yc"]] * K)
    reaches_device_guard(lq.coarse_mult_mrhs, yk, xk, f["A"], CD, NV)
    size_error(lq.coarse_mult_mrhs, yk[:2], xk, f["A"], CD, NV)                  # K from in; out holds only 2
    size_error(lq.coarse_mult_mrhs, yk, xk[:, :-2], f["A"], CD, NV)
    fk = torch.stack([f["x"]] * K)
    size_error(lq.wilson_clover_mult_mrhs, fk[:2], fk, f["U"], f["cl"], 0.1, DIMS, BC)
    size_error(lq.restrict_mrhs, yk[:1], fk, f["v"], DIMS, BLOCK, NV)
    size_error(lq.prolong_mrhs, fk, xk[:2].contiguous()[:, :-2], f["v"], DIMS, BLOCK, NV)


def test_solver_and_workspace_sizes():
    f = fields()
    size_error(lq.mr_domain_solve, f["y"], f["x"], f["U12"], f["cl"], 0.1, DIMS, BC, BLOCK)
    size_error(lq.sap, f["y"], f["y"].clone(), f["x"][:-4], f["U"], f["cl"], 0.1, DIMS, BC, BLOCK)
    size_error(lq.coarse_bicgstab, f["yc"], f["xc"], f["A"][:-2], CD, NV, 2, ws=torch.zeros(16, dtype=torch.uint8))
    size_error(lq.mg_vcycle, f["y"], f["x"], f["U"], f["cl"], 0.1, DIMS, BC, BLOCK, NV, f["v"], f["A"][:-2],
               ws=torch.zeros(16, dtype=torch.uint8))
    # a domain too large for the shared-memory-resident solver needs scratch: None or a short one is refused
    big = (8, 8, 8, 8)
    g = dict(x=torch.zeros(lq.native_spinor_reals(big)), U=torch.zeros(lq.native_gauge_reals(big)),
             cl=torch.zeros(lq.native_clover_reals(big)))
    need = lq.mr_workspace(big, big, device="cpu")
    assert need is not None and need.numel() > 0
    size_error(lq.mr_domain_solve, g["x"].clone(), g["x"], g["U"], g["cl"], 0.1, big, BC, big, ws=None)
    size_error(lq.mr_domain_solve, g["x"].clone(), g["x"], g["U"], g["cl"], 0.1, big, BC, big, ws=need[:-16])
    reaches_device_guard(lq.mr_domain_solve, g["x"].clone(), g["x"], g["U"], g["cl"], 0.1, big, BC, big, ws=need)


def test_halo_faces_and_host_calls():
    f = fields()
    faces = [torch.zeros(lq.halo_face_reals(DIMS, fc >> 1)) if (fc >> 1) == 3 else None for fc in range(8)]
    reaches_device_guard(lq.wilson_clover_halo_pack, faces, f["x"], f["U"], DIMS, 8)
    short = list(faces)
    short[6] = faces[6][:-4]
    size_error(lq.wilson_clover_halo_pack, short, f["x"], f["U"], DIMS, 8)
    missing = list(faces)
    missing[7] = None
    with pytest.raises(ValueError, match="missing face"):
        lq.wilson_clover_halo_add(f["y"], missing, f["U"], 0.1, DIMS, [1] * 8, 8)
    cf = [torch.zeros(lq.coarse_halo_face_reals(CD, NV, fc >> 1)) if (fc >> 1) == 3 else None for fc in range(8)]
    cshort = list(cf)
    cshort[7] = cf[7][:-2]
    size_error(lq.coarse_halo_add, f["yc"], cshort, f["A"], CD, NV, 8)
    # host entry points: host vectors of the canonical size, device scratch of the advertised size
    V = DIMS[0] * DIMS[1] * DIMS[2] * DIMS[3]
    h = torch.zeros((V, 4, 3, 2))
    ws = torch.zeros(lq.host_workspace_bytes(DIMS, BLOCK, NV), dtype=torch.uint8)
    size_error(lq.wilson_clover_mult_host, h, h[:-1], f["U"], f["cl"], 0.1, DIMS, BC, ws)
    size_error(lq.wilson_clover_mult_host, h, h, f["U"], f["cl"], 0.1, DIMS, BC, ws[:64])
    size_error(lq.restrict_host, torch.zeros_like(f["xc"])[:-2], h, f["v"], DIMS, BLOCK, NV, ws)
    size_error(lq.prolong_host, h, torch.zeros_like(f["xc"]), f["v"], DIMS, BLOCK, NV, ws[:64])
    size_error(lq.coarse_mult_host, torch.zeros_like(f["xc"]), torch.zeros_like(f["xc"]), f["A"], CD, NV, ws[:64])
