#!/usr/bin/env python
"""bench.py -- throughput of the hot path on synthetic lattices shaped like the
paper's workloads.

    python bench.py --gpus N --steps K --warmup W [--workload c5|c4|c3|c2] [--precision f32|f64] [--impl ours|reference]

One "step" = one pass of the whole hot path over one right-hand side:
    D x (A1, 18-real links), D^dag x (A2), restrict x (A4), coarse_mult (A3), prolong (A5)  [A4->A3->A5 chained = A6]
Metric (BASELINE.json): fp32 Wilson-clover & coarse mat-vec GB/s and GFLOP/s; % of HBM roofline.  `value` is the
ALGORITHMIC GB/s of the whole step (compulsory bytes of section 8(d) / measured time), inputs resident in HBM;
`kernels` carries sites/s, GFLOP/s, GB/s and roofline fraction per kernel; `e2e` is the same metric through the
host-vector C-ABI calls with the H2D/D2H copies inside the timed region.

Multi-GPU: the path is single-GPU by the north_star ("replicas only"): --gpus N runs N independent
replicas, one process per GPU under torchrun, barrier + max-over-ranks timing, no data-path collective.
Opt-in: --sharded makes the ranks share ONE lattice instead (each holds a sub-lattice of the config's size) with a
halo exchange inside D, D^dag and D_c (--sharded-transport p2p | peer).

--impl reference times the CPU oracle as it stands on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import lqcd_inputs as li

METRIC = "fp32 Wilson-clover & coarse mat-vec GB/s and GFLOP/s; % of HBM roofline"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent
HBM_PIN_RATE_GBS = 3996e6 * 2 * 8192 / 8 / 1e9  # 8184 GB/s: memory clock x DDR x bus width (what ncu's DRAM % refers to)


# ----------------------------------------------------------------------------------------------------------
# algorithmic bytes / nominal flops per launch (restated in DESIGN.md "Roofline model")
# ----------------------------------------------------------------------------------------------------------
def model(cfg: li.Config, links12: bool = False, real_bytes: int = 4) -> dict:
    """real_bytes: 4 for the fp32 kernels (the figures of SURVEY 8(d)), 8 for the fp64 variants (twice the bytes)."""
    V, Vc, N, nv = cfg.volume, cfg.cvolume, 2 * cfg.nvec, cfg.nvec
    bv = V // Vc
    w = real_bytes // 4
    fine_b = (96 + 96 + (192 if links12 else 288) + 288) * V * w
    fine_f = 1872 * V
    coarse_b = (9 * N * N * 8 + 2 * N * 8) * Vc * w
    coarse_f = 9 * N * N * 8 * Vc
    tr_b = ((nv * 96 + 96) * V + N * 8 * Vc) * w
    tr_f = nv * 96 * V
    return {
        "wilson_clover": {"bytes": fine_b, "flops": fine_f, "units": V},
        "wilson_clover_dagger": {"bytes": fine_b, "flops": fine_f, "units": V},
        "restrict": {"bytes": tr_b, "flops": tr_f, "units": V},
        "coarse_mult": {"bytes": coarse_b, "flops": coarse_f, "units": Vc},
        "prolong": {"bytes": tr_b, "flops": tr_f, "units": V},
        "_block_sites": bv,
    }


def model_dsap(cfg: li.Config, parity: int = 0) -> dict:
    """F1, D_SAP with the aggregation block as domain: links and hops that cross a domain face are never touched."""
    V = cfg.volume
    kept = [(b - 1) / b if l // b > 1 else 1.0 for l, b in zip(cfg.dims, cfg.block)]   # per direction
    link_b = sum(72 * k for k in kept)
    hop_f = sum(2 * 165 * k for k in kept)
    active_b, active_f = 96 + 96 + link_b + 288, hop_f + 504 + 48
    if parity == 0:
        return {"bytes": active_b * V, "flops": active_f * V, "units": V}
    return {"bytes": (active_b + 96) * V / 2, "flops": active_f * V / 2, "units": V}   # other group: zeros written


def model_sap(cfg: li.Config, n_sap: int = 4, n_mr: int = 6) -> dict:
    """F3: the inner-domain solver on one domain group (x += M^(g) r, the operator read once for all n_mr iterations)
    and SAP(n_sap) = 2 n_sap half sweeps, each one solver launch and one residual r = b - D x."""
    V = cfg.volume
    d = model_dsap(cfg, 0)
    site_b = d["bytes"] / V + 96           # r, links inside the domain, clover, x read + x written
    site_f = n_mr * (d["flops"] / V + 336)  # D_SAP + two blocked dots (96 + 48) + two blocked axpys (2 x 96)
    mr = {"bytes": site_b * V / 2, "flops": site_f * V / 2, "units": V / 2}
    res = {"bytes": (768 + 96) * V, "flops": (1872 + 24) * V}
    return {"mr": mr, "sap": {"bytes": 2 * n_sap * (mr["bytes"] + res["bytes"]),
                              "flops": 2 * n_sap * (mr["flops"] + res["flops"]), "units": V}}


STEP_ORDER = ["wilson_clover", "wilson_clover_dagger", "restrict", "coarse_mult", "prolong"]
KERNEL_SYMBOL = {  # the __global__ each row launches (for the ncu launch list)
    "wilson_clover": "k_wilson_clover", "wilson_clover_dagger": "k_wilson_clover", "restrict": "k_restrict",
    "coarse_mult": "k_coarse", "prolong": "k_prolong",
}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def recorded_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture
    (profiles/ncu_traffic.csv: workload,kernel,dram_bytes_per_launch,...), or None if that row is absent."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["kernel"] == kernel:
                    return float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


# ----------------------------------------------------------------------------------------------------------
# ranks: one process per GPU, replicas only
# ----------------------------------------------------------------------------------------------------------
class Ranks:
    """torch.distributed plumbing: barrier and max-over-ranks.  backend nccl on GPUs, gloo in the CPU tests."""

    def __init__(self, backend: str | None = None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            self.backend = backend or "nccl"
            if self.backend == "nccl":
                import torch
                torch.cuda.set_device(self.local_rank)
            dist.init_process_group(self.backend, rank=self.rank, world_size=self.world)
            self.dist = dist

    def _tensor(self, x):
        import torch
        dev = "cuda" if (self.dist is not None and self.backend == "nccl") else "cpu"
        return torch.tensor([float(x)], dtype=torch.float64, device=dev)

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max(self, x: float) -> float:
        if self.dist is None:
            return float(x)
        t = self._tensor(x)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum(self, x: float) -> float:
        if self.dist is None:
            return float(x)
        t = self._tensor(x)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return float(t.item())

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


def default_rank_grid(world: int):
    """Split t first, then z, y, x, by factors of two (an odd remainder goes to t): 2 -> 1x1x1x2, 8 -> 1x2x2x2."""
    r = [1, 1, 1, 1]
    mu = 3
    while world % 2 == 0:
        r[mu] *= 2
        world //= 2
        mu = (mu - 1) % 4
    r[3] *= world
    return tuple(r)


def whole_job_value(units_per_rank: float, world: int, max_seconds: float) -> float:
    """weak scaling, replicas: every rank processes units_per_rank in (at most) max_seconds."""
    return units_per_rank * world / max_seconds


# ----------------------------------------------------------------------------------------------------------
# clocks during the timed region
# ----------------------------------------------------------------------------------------------------------
_REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}


SETTLE_S = 0.5  # untimed run-in of a single-kernel extra row (time_single)


class ClockSampler(threading.Thread):
    def __init__(self, device_index: int, period_s: float = 0.004):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.max_mhz = period_s, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(device_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.nv = pynvml
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    bits = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for b, name in _REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "nvml unavailable"}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------------------
# the workload on the device (synthetic, seeded)
# ----------------------------------------------------------------------------------------------------------
class Workload:
    """Device-resident native operator fields + rotating right-hand sides of one config."""

    NBUF = 4  # distinct input/output buffer sets rotated across steps (and every buffer is >> L2 at c4/c5)

    def __init__(self, cfg: li.Config, device, seed: int, synthetic_operators: bool = False, precision: str = "f32"):
        import torch
        import paper_2111_05012_b200 as lq
        self.cfg, self.lq, self.dev = cfg, lq, device
        rdt, cdt = (torch.float32, torch.complex64) if precision == "f32" else (torch.float64, torch.complex128)
        self.sh_fine = self.sh_coarse = None
        gen = torch.Generator(device=device)
        gen.manual_seed(seed)
        V, Vc, nv = cfg.volume, cfg.cvolume, cfg.nvec
        # gauge: the config's recipe, fp64 on the device, rounded to fp32 once, packed (18-real and 12-real)
        U = li.t_gauge_field(cfg, gen, device).to(cdt)
        self.U18 = lq.pack_gauge(U, cfg.dims)
        self.U12 = lq.pack_gauge(U, cfg.dims, links12=True)
        del U
        self.setup_ms = {}

        def timed(name, fn):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            r = fn()
            torch.cuda.synchronize()
            self.setup_ms[name] = (time.perf_counter() - t0) * 1e3
            return r

        if synthetic_operators:
            cl = li.t_clover_synthetic(gen, V, device).to(cdt)
            self.clover = lq.pack_clover(cl, cfg.dims)
            del cl
        else:  # the true clover term of these links, built by the device set-up kernel (F2)
            self.clover = timed("clover_from_links", lambda: lq.clover_from_links(self.U18, cfg.kappa, cfg.csw, cfg.dims))
        self.x = [lq.pack_spinor(li.t_spinor(gen, V, device, rdt), cfg.dims) for _ in range(self.NBUF)]
        self.y = [lq.empty_spinor(cfg.dims, dtype=rdt) for _ in range(self.NBUF)]
        self.yd = [lq.empty_spinor(cfg.dims, dtype=rdt) for _ in range(self.NBUF)]
        self.z = [lq.empty_spinor(cfg.dims, dtype=rdt) for _ in range(self.NBUF)]
        self.xc = [torch.empty((Vc, 2, nv), dtype=cdt, device=device) for _ in range(self.NBUF)]
        self.yc = [torch.empty((Vc, 2, nv), dtype=cdt, device=device) for _ in range(self.NBUF)]
        # null vectors: Gaussian, one canonical vector at a time into its native slot (never twice in HBM)
        self.v = torch.empty(lq.native_nullvecs_reals(cfg.dims, cfg.block, nv), dtype=rdt, device=device)
        scale = 1.0 / np.sqrt(2.0 * 6 * (V // Vc))  # unit-norm aggregates on average, like orthonormal ones
        for i in range(nv):
            vi = li.t_spinor(gen, V, device, rdt) * scale
            lq.pack_nullvec(self.v, vi, i, cfg.dims, cfg.block, nv)
            del vi
        if synthetic_operators:
            self.A = li.t_coarse_matrix_synthetic(gen, Vc, nv, device).to(cdt)
        else:  # block-orthonormal null vectors and the true Galerkin coarse operator P^dag D P (F2)
            timed("orthonormalize_blocks", lambda: lq.orthonormalize_blocks(self.v, cfg.dims, cfg.block, nv))
            self.A = timed("galerkin_coarse", lambda: lq.galerkin_coarse(self.U18, self.clover, self.v, cfg.kappa,
                                                                          cfg.dims, cfg.bc, cfg.block, nv))
        torch.cuda.synchronize()

    def enable_sharded(self, grid, part_mask, transport="p2p"):
        """--sharded: this rank's fields are one sub-lattice of a lattice split over `grid`; D, D^dag and D_c then run
        as pack -> [exchange || interior] -> add (paper_2111_05012_b200/sharded.py); restrict / prolong are block-local."""
        from paper_2111_05012_b200 import sharded as sh
        c = self.cfg
        self.sh_fine = sh.ShardedWilsonClover(self.U18, self.clover, c.kappa, c.dims, c.bc, grid, part_mask=part_mask,
                                              transport=transport)
        self.sh_coarse = sh.ShardedCoarse(self.A, c.cdims, c.nvec, grid, part_mask=part_mask, transport=transport)

    # one launch per row; `i` picks the buffer set
    def wilson_clover(self, i):
        c = self.cfg
        if self.sh_fine is not None:
            return self.sh_fine.apply(self.y[i], self.x[i])
        self.lq.wilson_clover_mult(self.y[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc)

    def wilson_clover_dagger(self, i):
        c = self.cfg
        if self.sh_fine is not None:
            return self.sh_fine.apply(self.yd[i], self.x[i], dagger=True)
        self.lq.wilson_clover_mult(self.yd[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, dagger=True)

    def wilson_clover_12(self, i):
        c = self.cfg
        self.lq.wilson_clover_mult(self.y[i], self.x[i], self.U12, self.clover, c.kappa, c.dims, c.bc, links12=True)

    def wilson_clover_dd(self, i):
        c = self.cfg
        self.lq.wilson_clover_dd_mult(self.y[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, c.block)

    def wilson_clover_dd_even(self, i):
        c = self.cfg
        self.lq.wilson_clover_dd_mult(self.y[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, c.block,
                                      parity=1)

    def mr_even(self, i):
        c = self.cfg
        self.lq.mr_domain_solve(self.y[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, c.block, parity=1,
                                niter=6, accumulate=True, ws=getattr(self, "mr_ws", None))

    def sap(self, i):
        c = self.cfg
        self.lq.sap(self.y[i], self.z[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, c.block, n_sap=4,
                    n_mr=6, ws=getattr(self, "mr_ws", None))

    def fine_mrhs(self, i):
        c = self.cfg
        self.lq.wilson_clover_mult_mrhs(self.y2[i % 2], self.x2[i % 2], self.U18, self.clover, c.kappa, c.dims, c.bc)

    def sharded_self(self, i):
        self.sharded_op.apply(self.y[i], self.x[i])

    def sharded_vcycle(self, i):
        self.sharded_op.apply(self.y[i], self.x[i])

    def sharded_sap(self, i):
        self.sharded_op.apply(self.y[i], self.z[i], self.x[i])

    def sharded_self_coarse(self, i):
        self.sharded_op.apply(self.yc[i], self.xc[i])

    def coarse_mrhs(self, i):
        c = self.cfg
        self.lq.coarse_mult_mrhs(self.ycK, self.xcK, self.A, c.cdims, c.nvec)

    def vcycle_mrhs(self, i):
        c = self.cfg
        self.lq.mg_vcycle_mrhs(self.yK, self.xK, self.U18, self.clover, c.kappa, c.dims, c.bc, c.block, c.nvec, self.v,
                               self.A, n_coarse=8, n_sap=4, n_mr=6, ws=self.mg_ws)

    def bicg_mrhs(self, i):
        c = self.cfg
        self.lq.coarse_bicgstab_mrhs(self.ycK, self.xcK, self.A, c.cdims, c.nvec, 8, ws=self.bicg_ws)

    def bicg_single(self, i):
        c = self.cfg
        self.lq.coarse_bicgstab(self.ycK[i % 4], self.xcK[i % 4], self.A, c.cdims, c.nvec, 8, ws=self.bicg_ws)

    def vcycle(self, i):
        c = self.cfg
        self.lq.mg_vcycle(self.y[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, c.block, c.nvec, self.v,
                          self.A, n_coarse=8, n_sap=4, n_mr=6, ws=self.mg_ws)

    def vcycle_half(self, i):
        c = self.cfg
        self.lq.mg_vcycle(self.y[i], self.x[i], self.U18, self.clover, c.kappa, c.dims, c.bc, c.block, c.nvec, self.v,
                          self.Ah, n_coarse=8, n_sap=4, n_mr=6, ws=self.mg_ws, half=True)

    def restrict(self, i):
        c = self.cfg
        self.lq.restrict(self.xc[i], self.x[i], self.v, c.dims, c.block, c.nvec)

    def coarse_mult(self, i):
        c = self.cfg
        if self.sh_coarse is not None:
            return self.sh_coarse.apply(self.yc[i], self.xc[i])
        self.lq.coarse_mult(self.yc[i], self.xc[i], self.A, c.cdims, c.nvec)

    def prolong(self, i):
        c = self.cfg
        self.lq.prolong(self.z[i], self.yc[i], self.v, c.dims, c.block, c.nvec)

    def coarse_mult_half(self, i):
        c = self.cfg
        self.lq.coarse_mult_half(self.yc[i], self.xc[i], self.Ah, c.cdims, c.nvec, ws=self.half_ws)


def time_steps(W: Workload, steps: int, warmup: int, ranks: Ranks):
    """K steps between one pair of events (whole-step time) with an event after every launch (per-kernel times)."""
    import torch
    fns = [getattr(W, n) for n in STEP_ORDER]
    for k in range(warmup):
        for f in fns:
            f(k % W.NBUF)
    torch.cuda.synchronize()
    ranks.barrier()
    torch.cuda.synchronize()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(len(fns) + 1)] for _ in range(steps)]
    n0 = W.lq.launch_count()
    for k in range(steps):
        ev[k][0].record()
        for j, f in enumerate(fns):
            f(k % W.NBUF)
            ev[k][j + 1].record()
    torch.cuda.synchronize()
    launches = W.lq.launch_count() - n0
    ranks.barrier()
    total_s = ev[0][0].elapsed_time(ev[-1][-1]) * 1e-3
    per_kernel = {}
    for j, name in enumerate(STEP_ORDER):
        per_kernel[name] = [ev[k][j].elapsed_time(ev[k][j + 1]) * 1e-3 for k in range(steps)]
    return total_s, per_kernel, launches


def time_single(W: Workload, name: str, reps: int, warmup: int = 3, settle_s: float = 0.0, clocks: dict = None):
    """one row alone, rotating buffers (used for the 12-real-link variant and the sweep).
    settle_s > 0: the row is first run back to back for that long, untimed, so that the SM clock of the power-capped
    box has settled on THIS row's load (after a tensor-core row it stays near 1.3 GHz for > 100 ms, which made the
    next bandwidth row read 10-15 % slow: profiles/r02c_fine_c5.md); clocks: a dict that receives the SM clock sampled
    during the timed launches."""
    import torch
    f = getattr(W, name)
    for k in range(warmup):
        f(k % W.NBUF)
    if settle_s > 0:
        t_end, k = time.perf_counter() + settle_s, 0
        while time.perf_counter() < t_end:
            for _ in range(4):
                f(k % W.NBUF)
                k += 1
            torch.cuda.synchronize()
    torch.cuda.synchronize()
    sampler = ClockSampler(torch.cuda.current_device()) if clocks is not None else None
    if sampler:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(reps):
        f(k % W.NBUF)
    e1.record()
    torch.cuda.synchronize()
    if sampler:
        c = sampler.stop()
        clocks.update({"sm_mhz": c.get("sm_mhz"), "clock_reasons": c.get("reasons", [])})
    return e0.elapsed_time(e1) * 1e-3 / reps


def measure_pcie(device, nbytes: int = 1 << 30, reps: int = 3) -> dict:
    """Pinned-memory copy rates of this box, the ceiling of the e2e figure: H2D alone, D2H alone, and both directions at
    once on two streams (PCIe is full duplex).  GB/s per direction, best of `reps`, CUDA events."""
    import torch
    h_in = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    h_out = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d_a = torch.empty(nbytes, dtype=torch.uint8, device=device)
    d_b = torch.empty(nbytes, dtype=torch.uint8, device=device)
    s1, s2 = torch.cuda.Stream(device=device), torch.cuda.Stream(device=device)

    def run(h2d: bool, d2h: bool) -> float:
        best = float("inf")
        for _ in range(reps):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            s1.wait_event(e0)
            s2.wait_event(e0)
            if h2d:
                with torch.cuda.stream(s1):
                    d_a.copy_(h_in, non_blocking=True)
            if d2h:
                with torch.cuda.stream(s2):
                    h_out.copy_(d_b, non_blocking=True)
            torch.cuda.current_stream().wait_stream(s1)
            torch.cuda.current_stream().wait_stream(s2)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) * 1e-3)
        return nbytes / best / 1e9

    return {"h2d_GBps": run(True, False), "d2h_GBps": run(False, True), "duplex_GBps_per_direction": run(True, True),
            "bytes": nbytes}


def time_e2e(W: Workload, steps: int, warmup: int, ranks: Ranks):
    """The same step through the host-vector C-ABI calls: canonical fp32 vectors in pinned host memory, H2D and D2H
    inside the timed region, every call synchronising."""
    import torch
    c, lq = W.cfg, W.lq
    V, Vc, nv = c.volume, c.cvolume, c.nvec
    # Three independent chains of the step -- D x;  D^dag x;  restrict -> coarse_mult -> prolong -- each on its own stream
    # with its own scratch, driven by its own host thread (the C calls release the GIL and synchronise their stream):
    # uploads of one chain overlap downloads of another, PCIe being full duplex.
    from concurrent.futures import ThreadPoolExecutor
    nws = lq.host_workspace_bytes(c.dims, c.block, nv, dtype=W.v.dtype)
    ws = [torch.empty(nws, dtype=torch.uint8, device=W.dev) for _ in range(3)]
    streams = [torch.cuda.Stream(device=W.dev) for _ in range(3)]
    g = torch.Generator()
    g.manual_seed(99)
    rdt = W.v.dtype
    x_h = torch.randn((V, 4, 3, 2), generator=g, dtype=rdt).pin_memory()
    y_h = [torch.empty((V, 4, 3, 2), dtype=rdt).pin_memory() for _ in range(3)]
    xc_h = torch.empty((Vc, 2, nv, 2), dtype=rdt).pin_memory()
    yc_h = torch.empty((Vc, 2, nv, 2), dtype=rdt).pin_memory()

    def chain_d():
        torch.cuda.set_device(W.dev)  # worker threads start on device 0
        lq.wilson_clover_mult_host(y_h[0], x_h, W.U18, W.clover, c.kappa, c.dims, c.bc, ws[0], stream=streams[0])

    def chain_ddag():
        torch.cuda.set_device(W.dev)
        lq.wilson_clover_mult_host(y_h[1], x_h, W.U18, W.clover, c.kappa, c.dims, c.bc, ws[1], dagger=True,
                                   stream=streams[1])

    def chain_transfer():
        torch.cuda.set_device(W.dev)
        lq.restrict_host(xc_h, x_h, W.v, c.dims, c.block, nv, ws[2], stream=streams[2])
        lq.coarse_mult_host(yc_h, xc_h, W.A, c.cdims, nv, ws[2], stream=streams[2])
        lq.prolong_host(y_h[2], yc_h, W.v, c.dims, c.block, nv, ws[2], stream=streams[2])

    pool = ThreadPoolExecutor(max_workers=3)

    def one():
        futs = [pool.submit(f) for f in (chain_d, chain_ddag, chain_transfer)]
        for f in futs:
            f.result()

    fine_b, coarse_b = V * 24 * x_h.element_size(), Vc * 2 * nv * 2 * x_h.element_size()
    h2d = 3 * fine_b + 2 * coarse_b          # x (three times), xc, yc
    d2h = 3 * fine_b + 2 * coarse_b          # D x, D^dag x, prolong out, xc, yc
    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    ranks.barrier()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        one()
    e1.record()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    dev_s = e0.elapsed_time(e1) * 1e-3
    pool.shutdown()
    return max(wall, dev_s) / steps, h2d, d2h


# ----------------------------------------------------------------------------------------------------------
# the CPU oracle as a baseline (the only place outside tests/ and smoke() that executes oracle/)
# ----------------------------------------------------------------------------------------------------------
def sample_config(cfg: li.Config) -> li.Config:
    """The bounded sample of a workload the oracle is timed on: the same recipe (links, kappa, c_sw, block, nvec,
    boundary conditions) on a lattice of at most 16^3 x 32 sites."""
    cap = (16, 16, 16, 32)
    dims = tuple(min(l, c) for l, c in zip(cfg.dims, cap))
    return li.Config(cfg.name + "-sample", dims, cfg.block, cfg.nvec, cfg.gauge, cfg.eps, cfg.kappa, cfg.csw,
                     seed=cfg.seed, bc=cfg.bc)


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    import platform
    return platform.processor() or "unknown"


class OracleSample:
    """Host fields of the sample, fp32-rounded (the oracle promotes them and computes in fp64)."""

    def __init__(self, cfg: li.Config):
        import oracle
        self.oracle = oracle
        self.scfg = s = sample_config(cfg)
        rng = np.random.default_rng(s.seed)
        c64 = lambda a: np.ascontiguousarray(a.astype(np.complex64))
        self.U = c64(li.gauge_field(s, rng))
        self.psi = c64(li.spinor(rng, s.volume))
        g = li._cgauss(rng, (s.volume, 2, 6, 6))
        self.clover = c64(0.025 * (g + np.conj(np.swapaxes(g, -1, -2))))
        self.v = c64(li.null_vectors(rng, s.nvec, s.volume) / np.sqrt(2.0 * 6 * (s.volume // s.cvolume)))
        self.A = c64(li.coarse_matrix_synthetic(rng, s.cvolume, s.nvec))
        self.cores = os.cpu_count() or 1
        self.threads = oracle.set_threads(self.cores)

    def step(self):
        o, s = self.oracle, self.scfg
        o.wilson_clover_mult(self.psi, self.U, self.clover, s.kappa, s.dims, s.bc)
        o.wilson_clover_mult(self.psi, self.U, self.clover, s.kappa, s.dims, s.bc, dagger=True)
        xc = o.restrict(self.psi, self.v, s.dims, s.block)
        yc = o.coarse_mult(np.ascontiguousarray(xc.astype(np.complex64)), self.A, s.cdims)
        o.prolong(np.ascontiguousarray(yc.astype(np.complex64)), self.v, s.dims, s.block)

    def time(self, steps: int, warmup: int) -> float:
        for _ in range(warmup):
            self.step()
        t0 = time.perf_counter()
        for _ in range(steps):
            self.step()
        return (time.perf_counter() - t0) / steps

    def describe(self) -> str:
        s = self.scfg
        return (f"whole 5-row step on a {'x'.join(map(str, s.dims))} lattice ({s.volume} sites) of the same recipe, "
                f"block {'x'.join(map(str, s.block))}, nvec {s.nvec}, fp32-rounded inputs, fp64 arithmetic")


def oracle_full_rows(name: str = "c4") -> dict:
    """SURVEY 8(d) "oracle beside it": the oracle's D, D^dag and coarse_mult at the FULL size of config 4 (32^3 x 64 fine,
    8^3 x 16 coarse, N = 64), once with 1 thread (1 repeat) and with all cores (best of 3).  The fields have config 4's
    shapes and fp32 storage but are plain Gaussian numbers: the oracle has no data-dependent control flow, and the exact
    SU(3) recipe at 2 M sites costs minutes of host time for no change in what is measured.  Transfers (restrict,
    prolong) are not timed at this size: their null vectors are 6.4 GB of host memory -- the sample above has them."""
    import oracle
    cfg = li.CONFIGS[name]
    V, Vc, nv, n = cfg.volume, cfg.cvolume, cfg.nvec, 2 * cfg.nvec
    rng = np.random.default_rng(cfg.seed)

    def gauss(shape, scale=1.0):
        a = rng.standard_normal(shape + (2,), dtype=np.float32)
        if scale != 1.0:
            a *= np.float32(scale)
        return a.view(np.complex64).reshape(shape)

    U, psi, clover = gauss((4, V, 3, 3), 0.5), gauss((V, 4, 3)), gauss((V, 2, 6, 6), 0.05)
    A, xc = gauss((Vc, 9, n, n), 0.05), gauss((Vc, 2, nv))
    m = model(cfg)
    cores = os.cpu_count() or 1
    rows = {
        "wilson_clover": lambda: oracle.wilson_clover_mult(psi, U, clover, cfg.kappa, cfg.dims, cfg.bc),
        "wilson_clover_dagger": lambda: oracle.wilson_clover_mult(psi, U, clover, cfg.kappa, cfg.dims, cfg.bc, dagger=True),
        "coarse_mult": lambda: oracle.coarse_mult(xc, A, cfg.cdims),
    }
    out = {"workload": f"{name}: fine {'x'.join(map(str, cfg.dims))}, coarse {'x'.join(map(str, cfg.cdims))}, N = {n}; "
                       "Gaussian fields of the config's shapes, fp32 storage, fp64 arithmetic", "rows": {}}
    for label, fn in rows.items():
        r = {}
        for threads, reps in ((1, 1), (cores, 3)):
            used = oracle.set_threads(threads)
            best = min(_timed(fn) for _ in range(reps))
            r[f"threads_{used}"] = {"s": best, "repeats": reps, "units_per_s": m[label]["units"] / best,
                                    "GFLOPs": m[label]["flops"] / best / 1e9, "GBps": m[label]["bytes"] / best / 1e9}
        out["rows"][label] = r
    oracle.set_threads(cores)
    return out


def _timed(fn) -> float:
    t0 = time.perf_counter()
    fn()
    return time.perf_counter() - t0


def cpu_baseline_dict(cfg: li.Config, steps: int = 3, warmup: int = 1, full_rows: bool = True):
    """The oracle as it stands on this box's host cores: the bounded sample of the workload (the line's value) and, per
    SURVEY 8(d), the metric's rows at full config-4 size with 1 thread and with all cores."""
    smp = OracleSample(cfg)
    sec = smp.time(steps, warmup)
    d = {"value": step_bytes(smp.scfg) / sec / 1e9, "unit": "GB/s", "cores": smp.threads, "kind": "oracle",
         "sample": smp.describe(), "ms_per_step": sec * 1e3, "gflops": step_flops(smp.scfg) / sec / 1e9,
         "cpu_model": cpu_model(), "host_cores": smp.cores}
    if full_rows:
        d["full_size_rows"] = oracle_full_rows("c4")
    return d, smp, sec


def step_bytes(cfg: li.Config) -> int:
    m = model(cfg)
    return sum(m[k]["bytes"] for k in STEP_ORDER)


def step_flops(cfg: li.Config) -> int:
    m = model(cfg)
    return sum(m[k]["flops"] for k in STEP_ORDER)


def config_dict(cfg: li.Config, n_gpus: int, sample_of: str | None = None) -> dict:
    return {
        "workload": (("" if sample_of is None else f"bounded SAMPLE of {sample_of} -- what this line ran is ") +
                     f"{cfg.name}: fine {'x'.join(map(str, cfg.dims))} ({cfg.volume} sites), block "
                     f"{'x'.join(map(str, cfg.block))} -> coarse {'x'.join(map(str, cfg.cdims))}, nvec {cfg.nvec} "
                     f"(N={2 * cfg.nvec}), {cfg.gauge} links, kappa {cfg.kappa}, bc {list(cfg.bc)}; step = D, D^dag, "
                     f"restrict, coarse_mult, prolong on one right-hand side"),
        "replicas": n_gpus, "parallelism": "replicas only (single-GPU path)",
        "l2": "every operand stream of the timed kernels is larger than L2 at c4/c5; 4 rotating buffer sets",
    }


def run_reference(args, cfg: li.Config, ranks: Ranks):
    if ranks.rank != 0:
        return
    smp = OracleSample(cfg)
    sec = smp.time(args.steps, args.warmup)
    val = step_bytes(smp.scfg) / sec / 1e9
    cb = {"value": val, "unit": "GB/s", "cores": smp.threads, "kind": "oracle", "sample": smp.describe(),
          "cpu_model": cpu_model(), "host_cores": smp.cores}
    if not args.no_extras:
        cb["full_size_rows"] = oracle_full_rows("c4")
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the line states what ran: the oracle is timed on a bounded sample (same recipe, smaller lattice), so this is
        # NOT the same configuration as the GPU arm's line -- GB/s is intensive, but a 131 072-site lattice sits far
        # better in the host caches than the full workload would
        "config": config_dict(smp.scfg, args.gpus, sample_of=cfg.name), "same_config_as_gpu_arm": False,
        "gflops": step_flops(smp.scfg) / sec / 1e9,
        "cpu_baseline": cb,
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, cfg: li.Config, ranks: Ranks):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    dev_index = ranks.local_rank if ranks.world > 1 else 0
    torch.cuda.set_device(dev_index)
    device = torch.device("cuda", dev_index)
    import paper_2111_05012_b200 as lq
    f64 = args.precision == "f64"
    rb = 8 if f64 else 4
    W = Workload(cfg, device, seed=cfg.seed + 17 * ranks.rank, synthetic_operators=args.synthetic_operators,
                 precision=args.precision)
    m = model(cfg, real_bytes=rb)
    peak, peak_src = measured_peak()
    sharded = None
    if args.sharded is not None:
        from paper_2111_05012_b200 import sharded as sh
        rg = tuple(int(v) for v in args.sharded.split(",")) if args.sharded else default_rank_grid(ranks.world)
        grid = sh.RankGrid(rg, ranks.rank)
        if grid.world != ranks.world:
            raise SystemExit(f"--sharded {rg}: {grid.world} ranks, but WORLD_SIZE = {ranks.world}")
        mask = grid.part_mask | args.sharded_mask
        if args.sharded_transport == "peer" and ranks.dist is None:  # symmetric memory rendezvous needs a group
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29512")
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=device)
        W.enable_sharded(grid, mask, args.sharded_transport)
        sharded = {"rank_grid": list(rg), "part_mask": mask, "transport": args.sharded_transport,
                   "global_dims": [cfg.dims[mu] * rg[mu] for mu in range(4)],
                   "halo_bytes_sent_per_D": 2 * 4 * sum(lq.halo_face_reals(cfg.dims, mu) for mu in range(4)
                                                        if (mask >> mu) & 1),
                   "halo_bytes_sent_per_Dc": 2 * 4 * sum(lq.coarse_halo_face_reals(cfg.cdims, cfg.nvec, mu)
                                                         for mu in range(4) if (mask >> mu) & 1)}

    sampler = ClockSampler(dev_index)
    sampler.start()
    total_s, per_kernel, launches = time_steps(W, args.steps, args.warmup, ranks)
    clocks = sampler.stop()
    max_s = ranks.max(total_s)
    sec_per_step = max_s / args.steps
    sbytes, sflops = step_bytes(cfg) * (rb // 4), step_flops(cfg)
    value = whole_job_value(sbytes, ranks.world, sec_per_step) / 1e9

    kernels = {}
    for name in STEP_ORDER:
        t = statistics.mean(per_kernel[name])
        kernels[name] = {
            "us": t * 1e6, "us_min": min(per_kernel[name]) * 1e6, "share": t * args.steps / total_s,
            "GBps": m[name]["bytes"] / t / 1e9, "GFLOPs": m[name]["flops"] / t / 1e9,
            "units_per_s": m[name]["units"] / t, "frac_of_hbm_peak": m[name]["bytes"] / t / 1e9 / peak,
            "bytes_per_launch": m[name]["bytes"], "symbol": KERNEL_SYMBOL[name],
            "frac_of_pin_rate": m[name]["bytes"] / t / 1e9 / HBM_PIN_RATE_GBS,
        }
    dominant = max(STEP_ORDER, key=lambda n: kernels[n]["us"])
    roofline = {
        "bound": "hbm", "kernel": dominant, "achieved": kernels[dominant]["GBps"], "peak": peak, "unit": "GB/s",
        "frac": kernels[dominant]["GBps"] / peak, "traffic": recorded_traffic(cfg.name + (":f64" if f64 else ""), dominant),
        "peak_source": peak_src, "algorithmic_bytes_per_launch": m[dominant]["bytes"],
        "frac_of_pin_rate": kernels[dominant]["GBps"] / HBM_PIN_RATE_GBS, "pin_rate": HBM_PIN_RATE_GBS,
        # the two kernels the metric names, next to the dominant one (restrict / prolong carry 70 % of the step's bytes)
        "metric_kernels": {
            n: {"us": kernels[n]["us"], "achieved": kernels[n]["GBps"], "frac": kernels[n]["GBps"] / peak,
                "frac_of_pin_rate": kernels[n]["GBps"] / HBM_PIN_RATE_GBS, "GFLOPs": kernels[n]["GFLOPs"],
                "traffic": recorded_traffic(cfg.name + (":f64" if f64 else ""), n),
                "algorithmic_bytes_per_launch": m[n]["bytes"]}
            for n in ("wilson_clover", "wilson_clover_dagger", "coarse_mult")},
    }
    # the 12-real-link variant of A1 (config 4 asks for both storages), timed alone
    extra = {}
    if not args.no_extras and sharded is None:
        c12 = {}
        t12 = time_single(W, "wilson_clover_12", reps=max(50, args.steps), settle_s=SETTLE_S, clocks=c12)
        m12 = model(cfg, links12=True, real_bytes=rb)["wilson_clover"]
        extra["wilson_clover_links12"] = {"us": t12 * 1e6, "GBps": m12["bytes"] / t12 / 1e9,
                                          "GFLOPs": m12["flops"] / t12 / 1e9, "units_per_s": m12["units"] / t12,
                                          "frac_of_hbm_peak": m12["bytes"] / t12 / 1e9 / peak, **c12}
    if not args.no_extras and sharded is None and not f64:
        # F1 (next row of SURVEY 8(f)): the domain-decomposed operator D_SAP, all domains and the even group
        for name, par in (("wilson_clover_dd", 0), ("wilson_clover_dd_even", 1)):
            cr = {}
            t = time_single(W, name, reps=max(50, args.steps), settle_s=SETTLE_S, clocks=cr)
            md = model_dsap(cfg, par)
            extra[name] = {"us": t * 1e6, "GBps": md["bytes"] / t / 1e9, "GFLOPs": md["flops"] / t / 1e9,
                           "units_per_s": md["units"] / t, "frac_of_hbm_peak": md["bytes"] / t / 1e9 / peak,
                           "bytes_per_launch": md["bytes"], **cr}

        # F3: the inner-domain solver (6 minimal-residual iterations, even domains), shared-memory-resident and
        # generic, and the SAP smoother with the paper's parameters (n = 4, 6 inner iterations)
        import torch
        ms = model_sap(cfg)
        for name, knob, key in (("mr_even", 0, "mr"), ("mr_even", -1, "mr"), ("sap", 0, "sap")):
            W.lq.set_knob("sap_fused", knob)
            nb = int(W.lq.lib().lqcd_mr_workspace_bytes(W.lq._i4(cfg.dims), W.lq._i4(cfg.block), 4))
            W.mr_ws = torch.empty(nb, dtype=torch.uint8, device=W.dev) if nb else None
            row_sampler = ClockSampler(0)  # this row's own clock: an ALU-bound kernel runs into the power cap
            row_sampler.start()
            t = time_single(W, name, reps=max(3, min(10, args.steps)) * (3 if key == "mr" else 1), warmup=1)
            row_clocks = row_sampler.stop()
            W.mr_ws = None
            md = ms[key]
            label = {("mr_even", 0): "mr_domain_solve_even", ("mr_even", -1): "mr_domain_solve_even_generic",
                     ("sap", 0): "sap_4_6"}[(name, knob)]
            extra[label] = {"us": t * 1e6, "GBps": md["bytes"] / t / 1e9, "GFLOPs": md["flops"] / t / 1e9,
                            "units_per_s": md["units"] / t, "frac_of_hbm_peak": md["bytes"] / t / 1e9 / peak,
                            "bytes_per_launch": md["bytes"],
                            "path": "generic" if nb else "shared-memory-resident"}
            if label == "mr_domain_solve_even" and not nb and row_clocks.get("sm_mhz"):
                # The resident solver is bound on the SM, not by HBM.  With the links and clover blocks
                # parked in tensor memory (fp32 4^4 domains on the tiled site order: persistent kernel) the binding
                # roof is the fp32 pipe: 1472 FFMA / FADD per site and iteration (SASS count of the iteration body,
                # two threads per site) against 128 lanes/clk/SM x 148 SMs x SM clock; the shared-memory pipe carries
                # 8 neighbour spinors (96 B) + the store and the exchange of rho (96 + 192 B) = 1056 B per site and
                # iteration (1824 B when links and clover term are read from shared memory too) at 128 B/clk/SM.
                tm = cfg.block == (4, 4, 4, 4) and all(d % 4 == 0 for d in cfg.dims[:2]) and cfg.dims[2] % 2 == 0
                sites_it = (cfg.volume / 2) * 6
                clk = row_clocks["sm_mhz"] * 1e6
                alu_roof, smem_roof = 128.0 * 148 * clk, 128.0 * 148 * clk
                smem_b = (1056.0 if tm else 1824.0) * sites_it
                extra[label]["path"] = "persistent, operands in tensor memory" if tm else "shared-memory-resident"
                extra[label]["roofline"] = {
                    "bound": "alu" if tm else "shared-memory bandwidth",
                    "achieved": (1472.0 * sites_it / t / 1e12) if tm else smem_b / t / 1e12,
                    "peak": (alu_roof if tm else smem_roof) / 1e12,
                    "unit": "T fp32 lane-instructions/s" if tm else "TB/s",
                    "frac": (1472.0 * sites_it / t / alu_roof) if tm else smem_b / t / smem_roof,
                    "fp32_instructions_per_site_iteration": 1472,
                    "shared_memory": {"bytes_per_site_iteration": 1056 if tm else 1824,
                                      "achieved_TBps": smem_b / t / 1e12, "frac": smem_b / t / smem_roof},
                    "sm_mhz": row_clocks["sm_mhz"], "clock_reasons": row_clocks.get("reasons", [])}
        W.lq.set_knob("sap_fused", 0)
        # one V-cycle x = M b of the preconditioner: restrict, 8 BiCGStab iterations on D_c,
        # prolong, SAP(4, 6) -- everything on one stream, no host synchronisation
        W.mg_ws = W.lq.mg_workspace(cfg.dims, cfg.block, cfg.nvec, device=W.dev)
        n0 = W.lq.launch_count()
        t = time_single(W, "vcycle", reps=3, warmup=1)
        nl = (W.lq.launch_count() - n0) // 4
        mvc = {"bytes": 2 * m["restrict"]["bytes"] + 16 * m["coarse_mult"]["bytes"] + ms["sap"]["bytes"],
               "flops": 2 * m["restrict"]["flops"] + 16 * m["coarse_mult"]["flops"] + ms["sap"]["flops"]}
        extra["mg_vcycle_8_4_6"] = {"us": t * 1e6, "GBps": mvc["bytes"] / t / 1e9, "GFLOPs": mvc["flops"] / t / 1e9,
                                    "units_per_s": cfg.volume / t, "launches": int(nl),
                                    "frac_of_hbm_peak": mvc["bytes"] / t / 1e9 / peak, "bytes_per_launch": mvc["bytes"]}
        # ... and on 8 right-hand sides at once: restrictions, coarse solves (tensor cores) and prolongations shared
        KV = 8
        W.xK = torch.stack([W.x[k % W.NBUF] for k in range(KV)])
        W.yK = torch.empty_like(W.xK)
        nbk = int(W.lq.lib().lqcd_mg_mrhs_workspace_bytes(W.lq._i4(cfg.dims), W.lq._i4(cfg.block), cfg.nvec, KV, 4))
        W.mg_ws = torch.empty(nbk, dtype=torch.uint8, device=W.dev)
        tk = time_single(W, "vcycle_mrhs", reps=2, warmup=1)
        extra["mg_vcycle_mrhs_8"] = {"us": tk * 1e6, "us_per_rhs": tk * 1e6 / KV,
                                     "speedup_vs_8_single_vcycles": KV * t / tk}
        del W.xK, W.yK
        W.mg_ws = None
        # F4: the coarse operator on 16 right-hand sides at once (tcgen05, 3xTF32): A is read from HBM once
        K = 16
        gk = torch.Generator(device=W.dev)
        gk.manual_seed(4242)
        W.xcK = torch.view_as_complex(torch.randn((K, cfg.cvolume, 2, cfg.nvec, 2), generator=gk, device=W.dev,
                                                  dtype=torch.float32))
        W.ycK = torch.empty_like(W.xcK)
        ck, ckb = {}, {}
        # burst (the row's first launches, the box still at the clock of whatever ran before) and sustained (after
        # the run-in: this kernel alone pulls the power-capped box down to ~1.3 GHz)
        t_burst = time_single(W, "coarse_mrhs", reps=max(30, args.steps), warmup=3, clocks=ckb)
        t = time_single(W, "coarse_mrhs", reps=max(30, args.steps), warmup=3, settle_s=SETTLE_S, clocks=ck)
        mc = m["coarse_mult"]
        vec_b = 2 * K * cfg.cvolume * 2 * cfg.nvec * 8
        extra["coarse_mult_mrhs_16"] = {
            "us": t * 1e6, "us_per_rhs": t * 1e6 / K, "GBps": (mc["bytes"] + vec_b) / t / 1e9,
            "GFLOPs": K * mc["flops"] / t / 1e9, "units_per_s": K * cfg.cvolume / t,
            "speedup_vs_16_single_applications": K * kernels["coarse_mult"]["us"] * 1e-6 / t,
            "frac_of_hbm_peak": (mc["bytes"] + vec_b) / t / 1e9 / peak, "bytes_per_launch": mc["bytes"] + vec_b,
            "path": "tcgen05 kind::tf32, hi/lo split of both operands (3xTF32), fp32 accumulation", **ck,
            "burst": {"us": t_burst * 1e6, "frac_of_hbm_peak": (mc["bytes"] + vec_b) / t_burst / 1e9 / peak,
                      "sm_mhz": ckb.get("sm_mhz")}}
        # the coarse operator on half storage (A_0 and the forward blocks; the backward blocks are
        # G5c A_+mu(X - mu)^dag G5c): 5/9 of the matrix traffic, every stored block read once for both sites it couples
        prepare_row(W, "coarse_mult_half")
        ch = {}
        t = time_single(W, "coarse_mult_half", reps=max(50, args.steps), settle_s=SETTLE_S, clocks=ch)
        mh = model_coarse_half(cfg)
        yh, y9 = torch.empty_like(W.xc[0]), torch.empty_like(W.xc[0])
        W.lq.coarse_mult_half(yh, W.xc[0], W.Ah, cfg.cdims, cfg.nvec, ws=W.half_ws)
        W.lq.coarse_mult(y9, W.xc[0], W.A, cfg.cdims, cfg.nvec)
        dev = (torch.linalg.vector_norm((yh - y9).to(torch.complex128)) /
               torch.linalg.vector_norm(y9.to(torch.complex128))).item()
        extra["coarse_mult_half_storage"] = {
            "us": t * 1e6, "GBps": mh["bytes"] / t / 1e9, "GFLOPs": mh["flops"] / t / 1e9, "units_per_s": cfg.cvolume / t,
            "frac_of_hbm_peak": mh["bytes"] / t / 1e9 / peak, "bytes_per_launch": mh["bytes"], "launches": 2,
            "speedup_vs_nine_block_storage": kernels["coarse_mult"]["us"] * 1e-6 / t,
            "rel_l2_vs_nine_block_kernel_on_this_operator": dev, **ch}
        # ... and the V-cycle with its coarse solve on the half storage (16 applications of D_c at 5/9 of the bytes)
        W.mg_ws = W.lq.mg_workspace(cfg.dims, cfg.block, cfg.nvec, device=W.dev)
        tvh = time_single(W, "vcycle_half", reps=3, warmup=1)
        extra["mg_vcycle_8_4_6_half_storage"] = {
            "us": tvh * 1e6, "speedup_vs_mg_vcycle_8_4_6": extra["mg_vcycle_8_4_6"]["us"] * 1e-6 / tvh}
        W.mg_ws = None
        del W.Ah, W.half_ws, yh, y9
        # the coarse solver (1b) on the same 16 right-hand sides: 8 BiCGStab iterations, batched (D_c through the
        # tensor-core kernel) against one right-hand side at a time
        nb = int(W.lq.lib().lqcd_coarse_bicgstab_mrhs_workspace_bytes(W.lq._i4(cfg.cdims), cfg.nvec, K, 4))
        W.bicg_ws = torch.empty(nb, dtype=torch.uint8, device=W.dev)
        t1 = time_single(W, "bicg_single", reps=3, warmup=1)
        tk = time_single(W, "bicg_mrhs", reps=3, warmup=1)
        extra["coarse_bicgstab_mrhs_16x8"] = {"us": tk * 1e6, "us_single_rhs": t1 * 1e6,
                                               "speedup_vs_16_single_solves": K * t1 / tk,
                                               "GFLOPs": K * 16 * mc["flops"] / tk / 1e9}
        del W.xcK, W.ycK, W.bicg_ws
        # F4, fine half: D on two right-hand sides at once (links and clover read once for both)
        W.x2 = [torch.stack([W.x[0], W.x[1]]), torch.stack([W.x[2], W.x[3]])]
        W.y2 = [torch.empty_like(W.x2[0]), torch.empty_like(W.x2[1])]
        cf = {}
        t = time_single(W, "fine_mrhs", reps=max(50, args.steps), settle_s=SETTLE_S, clocks=cf)
        fb, ff = (576 + 2 * 192) * cfg.volume, 2 * m["wilson_clover"]["flops"]
        extra["wilson_clover_mrhs_2"] = {
            "us": t * 1e6, "us_per_rhs": t * 1e6 / 2, "GBps": fb / t / 1e9, "GFLOPs": ff / t / 1e9,
            "units_per_s": 2 * cfg.volume / t,
            "speedup_vs_2_single_applications": 2 * kernels["wilson_clover"]["us"] * 1e-6 / t,
            "frac_of_hbm_peak": fb / t / 1e9 / peak, "bytes_per_launch": fb, **cf}
        del W.x2, W.y2
        # SURVEY 8(e), the sharded operators' own cost on one GPU: directions marked partitioned with the rank as its
        # own neighbour (pack -> interior -> add; nothing crosses a link, so this is the kernels' overhead over the
        # plain operator; a multi-GPU run adds only the transfer of the halo bytes, overlapped with the interior pass)
        from paper_2111_05012_b200 import sharded as sh
        one = sh.RankGrid((1, 1, 1, 1))
        sd = {"note": "one rank exchanging with itself; masks: t, z+t, all four directions"}
        for tag, mask in (("t", 8), ("zt", 12), ("xyzt", 15)):
            W.sharded_op = sh.ShardedWilsonClover(W.U18, W.clover, cfg.kappa, cfg.dims, cfg.bc, one, part_mask=mask)
            t = time_single(W, "sharded_self", reps=max(10, args.steps))
            sd[tag] = {"us": t * 1e6, "overhead_vs_plain": t / (kernels["wilson_clover"]["us"] * 1e-6),
                       "halo_bytes_sent": 2 * 4 * sum(W.lq.halo_face_reals(cfg.dims, mu) for mu in range(4)
                                                      if (mask >> mu) & 1),
                       "launches": 2 + bin(mask).count("1")}
        extra["wilson_clover_sharded_selfhalo"] = sd
        sc = {}
        for tag, mask in (("t", 8), ("zt", 12), ("xyzt", 15)):
            W.sharded_op = sh.ShardedCoarse(W.A, cfg.cdims, cfg.nvec, one, part_mask=mask)
            t = time_single(W, "sharded_self_coarse", reps=max(10, args.steps))
            sc[tag] = {"us": t * 1e6, "overhead_vs_plain": t / (kernels["coarse_mult"]["us"] * 1e-6),
                       "halo_bytes_sent": 2 * 4 * sum(W.lq.coarse_halo_face_reals(cfg.cdims, cfg.nvec, mu)
                                                      for mu in range(4) if (mask >> mu) & 1), "launches": 3}
        extra["coarse_mult_sharded_selfhalo"] = sc
        # the smoother on a sharded lattice (t partitioned): local domain solves, halo exchange in the residuals only
        W.sharded_op = sh.ShardedSAP(sh.ShardedWilsonClover(W.U18, W.clover, cfg.kappa, cfg.dims, cfg.bc, one,
                                                            part_mask=8), cfg.block, n_sap=4, n_mr=6)
        t = time_single(W, "sharded_sap", reps=5, warmup=1)
        extra["sap_4_6_sharded_selfhalo_t"] = {"us": t * 1e6, "overhead_vs_sap_4_6": t * 1e6 / extra["sap_4_6"]["us"],
                                               "launches": 8 + 8 * 3}
        # ... and the whole V-cycle (restrict, 8 BiCGStab iterations on the sharded D_c through the solver's hooks,
        # prolong, sharded SAP(4, 6)); one rank: the cross-rank sum of the dot products is the identity
        W.sharded_op = sh.ShardedVcycle(W.sharded_op.op, sh.ShardedCoarse(W.A, cfg.cdims, cfg.nvec, one, part_mask=8),
                                        W.v, cfg.block, cfg.nvec, n_coarse=8, n_sap=4, n_mr=6)
        t = time_single(W, "sharded_vcycle", reps=3, warmup=1)
        extra["mg_vcycle_8_4_6_sharded_selfhalo_t"] = {
            "us": t * 1e6, "overhead_vs_mg_vcycle_8_4_6": t * 1e6 / extra["mg_vcycle_8_4_6"]["us"]}
        del W.sharded_op

    if not args.no_extras and sharded is None and not f64:
        # the fp64 variants of the five rows (north_star: "fp64 and fp32 kernel variants"), on config 4's lattice when
        # the workload is larger (the fp64 fields of config 5 do not fit beside its fp32 ones): twice the bytes
        c64 = cfg if cfg.volume <= li.CONFIGS["c4"].volume else li.CONFIGS["c4"]
        W64 = Workload(c64, device, seed=c64.seed + 5, synthetic_operators=args.synthetic_operators, precision="f64")
        m64 = model(c64, real_bytes=8)
        _, pk64, _ = time_steps(W64, max(5, min(20, args.steps)), 3, ranks)
        rows = {}
        for name in STEP_ORDER:
            t = statistics.mean(pk64[name])
            rows[name] = {"us": t * 1e6, "GBps": m64[name]["bytes"] / t / 1e9, "GFLOPs": m64[name]["flops"] / t / 1e9,
                          "units_per_s": m64[name]["units"] / t, "frac_of_hbm_peak": m64[name]["bytes"] / t / 1e9 / peak}
        t64 = sum(r["us"] for r in rows.values()) * 1e-6
        extra["fp64_five_rows"] = {"workload": c64.name, "dtype": "f64", "ms_per_step": t64 * 1e3,
                                   "GBps": sum(m64[n]["bytes"] for n in STEP_ORDER) / t64 / 1e9,
                                   "frac_of_hbm_peak": sum(m64[n]["bytes"] for n in STEP_ORDER) / t64 / 1e9 / peak,
                                   "kernels": rows}
        del W64
        torch.cuda.empty_cache()

    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    e2e_s, h2d, d2h = time_e2e(W, e2e_steps, 1, ranks)
    e2e_s = ranks.max(e2e_s)
    pcie = measure_pcie(device)
    # Ceilings of one e2e step.  (i) Both directions perfectly overlapped.  (ii) The dependency-aware bound: inside a call
    # the vector travels in slabs (upload of slab k+1 under the kernels of slab k under the download of slab k-1,
    # host_api.cu), so the two operator chains keep both directions busy; but prolong's result (one fine vector) can
    # only leave after restrict's input (one fine vector) has arrived, and while that input occupies a share s of the
    # upload link the operator chains' uploads -- hence their downloads -- lose exactly that share: whatever the
    # interleaving, the download link idles for one fine-vector upload:  t >= t_duplex + fine_bytes / h2d rate.
    t_duplex = max(h2d, d2h) / (pcie["duplex_GBps_per_direction"] * 1e9)
    fine_bytes = cfg.volume * 24 * (8 if f64 else 4)
    t_chain = t_duplex + fine_bytes / (pcie["h2d_GBps"] * 1e9)
    e2e = {"value": whole_job_value(sbytes, ranks.world, e2e_s) / 1e9, "unit": "GB/s", "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3, "steps": e2e_steps,
           "pcie_measured": pcie, "ms_if_full_duplex": t_duplex * 1e3, "frac_of_full_duplex_pcie": t_duplex / e2e_s,
           "ms_dependency_bound": t_chain * 1e3, "frac_of_dependency_bound": t_chain / e2e_s,
           "GBps_per_direction": max(h2d, d2h) / e2e_s / 1e9,
           "note": "host-vector C-ABI calls, pinned canonical vectors, three independent chains on three streams; PCIe "
                   "copies dominate.  Inside a call the vector travels in slabs of time slices: upload of slab k+1 under "
                   "pack / kernel / unpack of slab k under the download of slab k-1.  The transfer chain (restrict -> "
                   "coarse operator -> prolong) has its one-vector download strictly after its one-vector upload, which "
                   "leaves the download link idle for one upload whatever the interleaving: ms_dependency_bound = "
                   "ms_if_full_duplex + one fine vector / h2d rate"}

    line = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": ranks.world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec_per_step * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.precision, "data": "synthetic", "config": config_dict(cfg, ranks.world),
        "gflops": whole_job_value(sflops, ranks.world, sec_per_step) / 1e9,
        "fine_sites_per_s": whole_job_value(2 * cfg.volume, ranks.world, sec_per_step),
        "frac_of_hbm_peak": value / ranks.world / peak,
        "kernels": kernels, "extra": extra, "setup_ms": W.setup_ms,
        "operators": "synthetic" if args.synthetic_operators else "device-built (clover from links, Galerkin P^dag D P)", "roofline": roofline, "e2e": e2e, "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if sharded is not None:  # one lattice over all ranks: the per-rank sub-lattice is the config's lattice (weak)
        line["config"]["parallelism"] = ("sharded: one lattice of %s over a %s grid of ranks; halo exchange per D, "
                                         "D^dag, D_c" % ("x".join(map(str, sharded["global_dims"])),
                                                         "x".join(map(str, sharded["rank_grid"]))))
        line["sharded"] = sharded
    if ranks.rank == 0 and ranks.world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"], _, _ = cpu_baseline_dict(cfg, steps=3, warmup=1, full_rows=not args.no_extras)
    if ranks.rank == 0:
        print(json.dumps(line), flush=True)


ROW_MODELS = {  # rows that --rows can time alone -> (Workload method, model of its algorithmic bytes / flops)
    "wilson_clover": lambda c, m: m["wilson_clover"], "wilson_clover_dagger": lambda c, m: m["wilson_clover"],
    "restrict": lambda c, m: m["restrict"], "coarse_mult": lambda c, m: m["coarse_mult"],
    "prolong": lambda c, m: m["prolong"],
    "wilson_clover_12": lambda c, m: model(c, links12=True)["wilson_clover"],
    "wilson_clover_dd": lambda c, m: model_dsap(c, 0), "wilson_clover_dd_even": lambda c, m: model_dsap(c, 1),
    "mr_even": lambda c, m: model_sap(c)["mr"], "sap": lambda c, m: model_sap(c)["sap"],
    "fine_mrhs": lambda c, m: {"bytes": (576 + 2 * 192) * c.volume, "flops": 2 * m["wilson_clover"]["flops"]},
    "coarse_mrhs": lambda c, m: {"bytes": m["coarse_mult"]["bytes"] + 2 * 16 * c.cvolume * 2 * c.nvec * 8,
                                 "flops": 16 * m["coarse_mult"]["flops"]},
    "coarse_mult_half": lambda c, m: model_coarse_half(c),
}


def model_coarse_half(cfg: li.Config, real_bytes: int = 4) -> dict:
    """Half-storage coarse operator: A_0 and the four forward blocks are stored, the backward blocks
    come from the neighbour's forward block (A_-mu(X) = G5c A_+mu(X-mu)^dag G5c): 5 blocks per coarse site."""
    Vc, N = cfg.cvolume, 2 * cfg.nvec
    w = real_bytes // 4
    return {"bytes": (5 * N * N * 8 + 2 * N * 8) * Vc * w, "flops": 9 * N * N * 8 * Vc, "units": Vc}


def prepare_row(W: Workload, name: str):
    """Buffers that some rows need beside the Workload's own (fp32)."""
    import torch
    cfg = W.cfg
    if name == "fine_mrhs" and not hasattr(W, "x2"):
        W.x2 = [torch.stack([W.x[0], W.x[1]]), torch.stack([W.x[2], W.x[3]])]
        W.y2 = [torch.empty_like(W.x2[0]), torch.empty_like(W.x2[1])]
    if name == "coarse_mult_half" and not hasattr(W, "Ah"):
        W.Ah = W.lq.pack_coarse_half(W.A, cfg.cdims, cfg.nvec)
        W.half_ws = W.lq.coarse_half_workspace(cfg.cdims, cfg.nvec, dtype=W.v.dtype, device=W.dev)
        for xc in W.xc:  # the rows that feed coarse_mult in the step are outputs of restrict; alone they need data
            xc.copy_(torch.view_as_complex(torch.randn(xc.shape + (2,), device=W.dev, dtype=W.v.dtype)))
    if name == "coarse_mrhs" and not hasattr(W, "xcK"):
        gk = torch.Generator(device=W.dev)
        gk.manual_seed(4242)
        W.xcK = torch.view_as_complex(torch.randn((16, cfg.cvolume, 2, cfg.nvec, 2), generator=gk, device=W.dev,
                                                  dtype=torch.float32))
        W.ycK = torch.empty_like(W.xcK)


def run_rows(args, cfg: li.Config):
    """--rows a,b,...: each named row timed alone (CUDA events, rotating buffers); one JSON line.  This is the command
    the per-kernel ncu captures under profiles/ run."""
    import torch
    torch.cuda.set_device(0)
    device = torch.device("cuda", 0)
    W = Workload(cfg, device, seed=cfg.seed, synthetic_operators=args.synthetic_operators, precision=args.precision)
    m = model(cfg, real_bytes=8 if args.precision == "f64" else 4)
    peak, peak_src = measured_peak()
    # tuning knobs of the library for this run (results never depend on them)
    if args.fine_tile:
        W.lq.set_fine_tile(tuple(int(v) for v in args.fine_tile.split("x")))
    for kv in args.knob or []:
        k, v = kv.split("=")
        W.lq.set_knob(k, int(v))
    sampler = ClockSampler(0)
    sampler.start()
    out = {}
    for name in args.rows.split(","):
        prepare_row(W, name)
        t = time_single(W, name, reps=args.steps, warmup=args.warmup)
        md = ROW_MODELS[name](cfg, m)
        out[name] = {"us": t * 1e6, "GBps": md["bytes"] / t / 1e9, "GFLOPs": md["flops"] / t / 1e9,
                     "frac_of_hbm_peak": md["bytes"] / t / 1e9 / peak, "bytes_per_launch": md["bytes"]}
    clocks = sampler.stop()
    print(json.dumps({"metric": METRIC, "rows": out, "unit": "GB/s", "peak": peak, "peak_source": peak_src,
                      "workload": cfg.name, "dtype": args.precision, "data": "synthetic", "steps": args.steps,
                      "warmup": args.warmup, "clocks": clocks, "fine_tile": args.fine_tile or "auto",
                      "knobs": args.knob or []}), flush=True)


def run_sweep(args):
    """Config 5's bandwidth-roofline sweep: the fp32 fine operator (and D^dag) and the coarse operator over volumes
    8^3x16 ... 48^3x96 (and the matching coarse lattices, block 4^4, nvec 32): algorithmic GB/s versus footprint,
    showing the L2 -> HBM transition.  Operator fields are random numbers written straight into the native layouts
    (throughput does not depend on values); two buffer sets alternate.  One JSON line."""
    import torch
    import paper_2111_05012_b200 as lq
    torch.cuda.set_device(0)
    peak, peak_src = measured_peak()
    gen = torch.Generator(device="cuda")
    gen.manual_seed(5)
    rnd = lambda n, s=1.0: torch.randn(n, device="cuda", dtype=torch.float32, generator=gen) * s
    out = []
    for l in (8, 16, 24, 32, 40, 48):
        dims, cd, nv = (l, l, l, 2 * l), (l // 4, l // 4, l // 4, l // 2), 32
        cfg = li.Config(f"sweep{l}", dims, (4, 4, 4, 4), nv, "haar", 0.0, 0.1372, 1.7)
        m = model(cfg)
        U, cl = rnd(lq.native_gauge_reals(dims)), rnd(lq.native_clover_reals(dims), 0.05)
        x = [rnd(lq.native_spinor_reals(dims)) for _ in range(2)]
        y = [torch.empty_like(x[0]) for _ in range(2)]
        A = rnd(lq.native_coarse_mat_reals(cd, nv), 0.05)
        xc = [rnd(lq.native_coarse_vec_reals(cd, nv)) for _ in range(2)]
        yc = [torch.empty_like(xc[0]) for _ in range(2)]
        reps = max(20, min(400, int(2e9 / m["wilson_clover"]["bytes"]) * 10))

        def timed(f):
            for k in range(5):
                f(k % 2)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for k in range(reps):
                f(k % 2)
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) * 1e-3 / reps

        t_d = timed(lambda i: lq.wilson_clover_mult(y[i], x[i], U, cl, cfg.kappa, dims, cfg.bc))
        t_dd = timed(lambda i: lq.wilson_clover_mult(y[i], x[i], U, cl, cfg.kappa, dims, cfg.bc, dagger=True))
        t_c = timed(lambda i: lq.coarse_mult(yc[i], xc[i], A, cd, nv))
        fb, cb = m["wilson_clover"]["bytes"], m["coarse_mult"]["bytes"]
        out.append({
            "fine_dims": list(dims), "coarse_dims": list(cd), "reps": reps,
            "fine_footprint_MB": (fb + 96 * cfg.volume) / 1e6, "coarse_footprint_MB": cb / 1e6,
            "wilson_clover": {"us": t_d * 1e6, "GBps": fb / t_d / 1e9, "GFLOPs": m["wilson_clover"]["flops"] / t_d / 1e9,
                              "frac_of_hbm_peak": fb / t_d / 1e9 / peak},
            "wilson_clover_dagger": {"us": t_dd * 1e6, "GBps": fb / t_dd / 1e9, "frac_of_hbm_peak": fb / t_dd / 1e9 / peak},
            "coarse_mult": {"us": t_c * 1e6, "GBps": cb / t_c / 1e9, "GFLOPs": m["coarse_mult"]["flops"] / t_c / 1e9,
                            "frac_of_hbm_peak": cb / t_c / 1e9 / peak},
        })
        del U, cl, x, y, A, xc, yc
    print(json.dumps({"metric": METRIC, "sweep": out, "unit": "GB/s", "peak": peak, "peak_source": peak_src,
                      "dtype": "f32", "data": "synthetic",
                      "note": "footprints below ~126 MB are L2-resident across repetitions: GB/s there is not an HBM figure"}),
          flush=True)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=sorted(li.CONFIGS), default="c5")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--precision", choices=("f32", "f64"), default="f32",
                    help="f64: the fp64 kernel variants on the same step (twice the algorithmic bytes; the headline "
                         "metric is fp32)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--sharded", nargs="?", const="", default=None, metavar="R0,R1,R2,R3",
                    help="opt-in: the ranks share ONE lattice (each holds a sub-lattice of the config's size) and "
                         "exchange halos; default grid splits t, z, y, x in turn")
    ap.add_argument("--sharded-transport", choices=("p2p", "peer"), default="p2p",
                    help="with --sharded: p2p = pack, then torch.distributed send/recv; peer = the pack kernels store "
                         "into the neighbours' receive buffers over NVLink peer memory (symmetric memory)")
    ap.add_argument("--sharded-mask", type=int, default=0,
                    help="with --sharded: also treat these directions (bit mu) as partitioned, the rank being its own "
                         "neighbour there (exercises the whole exchange path on one GPU)")
    ap.add_argument("--synthetic-operators", action="store_true",
                    help="random clover term and coarse matrix instead of the device-built ones (DESIGN.md section 4)")
    ap.add_argument("--sweep", action="store_true", help="config 5's bandwidth-roofline sweep over volumes (1 GPU)")
    ap.add_argument("--rows", default=None, metavar="ROW[,ROW...]",
                    help="time the named rows alone (1 GPU; %s)" % ", ".join(sorted(ROW_MODELS)))
    ap.add_argument("--fine-tile", default=None, metavar="AxBxCxD",
                    help="with --rows: sites per CTA of the fine kernels (lqcd_set_fine_tile), e.g. 4x4x4x2")
    ap.add_argument("--knob", action="append", metavar="NAME=VALUE",
                    help="with --rows: lqcd_set_knob(NAME, VALUE) before timing; may be repeated")
    args = ap.parse_args()
    cfg = li.CONFIGS[args.workload]
    if args.sweep:
        run_sweep(args)
        return
    if args.rows:
        run_rows(args, cfg)
        return
    if args.impl == "reference":
        # rank 0 alone runs the oracle; the other ranks exit 0 without work (no process group needed)
        if int(os.environ.get("RANK", "0")) == 0:
            r = Ranks.__new__(Ranks)
            r.rank, r.world, r.local_rank, r.dist = 0, 1, 0, None
            run_reference(args, cfg, r)
        return
    ranks = Ranks()
    if ranks.world != args.gpus and ranks.rank == 0:
        print(f"[bench] note: --gpus {args.gpus} but WORLD_SIZE={ranks.world}; using WORLD_SIZE", file=sys.stderr)
    try:
        run_ours(args, cfg, ranks)
    finally:
        ranks.close()


if __name__ == "__main__":
    main()
