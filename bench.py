#!/usr/bin/env python
"""bench.py -- headline benchmark of the tropical transfer sweep (BASELINE.json metric:
"Sweep time per instance & achieved HBM GB/s (frac. of peak), LxL tropical sweep").

Workload at N=1: BASELINE.json configs[3] -- 32x32 +-J Ising, h=0, Tropical<f32> energy, the
2^32-entry state vector swept in place row by row -- the configuration north_star's ">= 60 % of
the HBM roofline on the 2^28..2^32-entry sweeps" is quoted on.  With h = 0 the library stores the
flip-symmetric half of that vector (2^31 elements, 8 GiB; include/ttn.h);
north_star's full-vector bytes appear only as `algorithmic_equivalent_frac`.  A "step" is one whole
sweep (every pass kernel + the final reduction) of one instance per GPU.  With N GPUs each rank sweeps its own
instance (seed 4000 + rank): replicas, no data-path collective, "scaling": "weak".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--L 32] [--impl ours|reference]

`value`  : ms per instance, device-timed with CUDA events on the launching stream, couplings
           already resident in HBM (ttn_plan_launch only), max over ranks / instances per step.
`e2e`    : the same through the one-call C ABI (ttn_sweep_energy) with HOST coupling buffers:
           plan + host->device upload + sweep + device->host result, timed on the host clock
           around the synchronising call.
`roofline`: the roof that binds.  The sweep is bound by the FMNMX issue rate of the alu pipe, not by HBM:
           `roofline` = executed max-plus updates per second against 148 SMs x 64 lanes/clk x the sampled
           SM clock ("bound": "alu").  `hbm_roofline` beside it: `achieved` = the bytes the sweep really
           moves (one read + one write of the STORED state per pass, first pass write-only, last
           read-only) over the measured time against the measured copy bandwidth in MEASURED_PEAKS.json;
           `algorithmic_equivalent_frac` = north_star's figure, (L-1)*2*4*2^L bytes per sweep (one read +
           one write of the FULL vector per row) over the same time and peak -- a statement
           about time saved against a one-pass-per-row sweep, not a bandwidth, and allowed to exceed 1.
`cpu_baseline`: the CPU oracle (oracle/, unmodified) timed on the host cores on a bounded
           sample: one full sweep of a smaller lattice, reported UNSCALED next to the GPU time for
           that same lattice; `value` is its extrapolation to the workload by the update count
           (L-1)*L*2^L and is labelled as such.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from ttn_inputs import make_batch  # noqa: E402

METRIC = "sweep_time_per_instance"
UNIT = "ms"


def updates(L: int) -> float:
    """el-gate updates of one sweep: (L-1) rows x L gates x 2^L elements."""
    return float(L - 1) * L * 2.0 ** L


def bytes_min(L: int) -> float:
    """north_star's minimum traffic: one read + one write of the f32 state per row, row 0
    write-only and the last row read-only."""
    return float(L - 1) * 2 * 4 * 2.0 ** L


def bytes_moved(elem_bytes: float, state_elements: float, passes: int, batch: int = 1) -> float:
    """What the passes of one sweep really move through HBM (computed, not measured): every pass reads and
    writes the stored state once, the first pass only writes, the last only reads."""
    return float(batch) * (2 * passes - 2) * elem_bytes * state_elements


ALU_LANES = 64            # FMNMX / VIADDMNMX lanes per clock and SM (profiles/r01_ubench.md)
SMS = 148


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def rank_env():
    """(rank, local_rank, world) from the torchrun environment (1 process per GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def seed_for_rank(rank: int) -> int:
    """Replicas only: rank r sweeps its own cfg-4 instance."""
    return 4000 + rank


def max_over_ranks(x: float, dist, device="cpu") -> float:
    """Device-timed numbers are reported as the MAX over ranks (the contract's timing rule)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_ms_per_instance(ms_per_step: float, world: int) -> float:
    """Each rank sweeps one instance per step: `value` = step time / instances in flight."""
    return ms_per_step / world


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (nvidia-smi, 200 ms)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._stop_evt.is_set():
            try:
                out = subprocess.check_output(
                    ["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                    text=True, timeout=5).strip().split(",")
                self.samples.append(float(out[0]))
                self.max_mhz = float(out[1])
                for n, v in zip(names, out[2:]):
                    if v.strip().lower() == "active":
                        self.reasons.add(n)
            except Exception:
                pass
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=10)
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def workload_name(L: int) -> str:
    return (f"{L}x{L} +-J Ising (p=0.5, h=0) Tropical<f32> energy sweep, "
            f"2^{L}-entry state in place, 1 instance per GPU (seed 4000+rank)")


# The oracle's one full-size run: 32x32 +-J seed 4000, O-dp, 34 GB frontier.
ORACLE_FULL_32 = {"seconds": 4776, "cores": 6, "where": "build box, round 1 (tests/golden/oracle_values.txt ising_energy 32 4000)"}


def ncu_traffic_per_launch(summary_csv: str, kernel_substr: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch, averaged over the launches of the
    kernel in a committed `ncu --set full` summary (profiles/*.csv: one row per metric -- name, unit,
    one column per captured launch; units byte / Kbyte / Mbyte / Gbyte).  None when the file is
    absent: the number is never a literal in this script."""
    path = os.path.join(ROOT, "profiles", summary_csv)
    if not os.path.exists(path):
        return None, None
    import csv
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    rows = {r[0]: r for r in csv.reader(open(path)) if r}
    names = rows.get("Kernel Name")
    rd, wr = rows.get("dram__bytes_read.sum"), rows.get("dram__bytes_write.sum")
    if not (names and rd and wr):
        return None, None
    vals = [float(rd[i]) * scale[rd[1]] + float(wr[i]) * scale[wr[1]]
            for i in range(2, len(names)) if kernel_substr in names[i]]
    return (sum(vals) / len(vals) if vals else None), "profiles/" + summary_csv


def time_plan(torch, plan, reps=3, warm=1):
    for _ in range(warm):
        plan.launch()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        plan.launch()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores.  Each step is a bounded
    sample (a full sweep of a smaller lattice of the same +-J distribution), scaled to the
    32x32 metric by the update count."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    Ls = args.ref_L
    Jh, Jv, _ = make_batch(Ls, [4000], "pmj")
    times = []
    for i in range(args.warmup + args.steps):
        t = time.perf_counter()
        oracle.dp_ising(Ls, Jh[0], Jv[0], None, count=False)
        if i >= args.warmup:
            times.append(time.perf_counter() - t)
    per_update = float(np.mean(times)) / updates(Ls)
    val = per_update * updates(args.L) * 1e3
    cores = oracle.num_threads()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(times)) * 1e3,
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        # the same workload key as the CUDA arm; what one step actually ran is in cpu_baseline.sample
        # state_bytes as the CUDA arm prints it: with h = 0 it stores the flip-symmetric half of the vector (L >= 14)
        "config": {"workload": workload_name(args.L), "L": args.L,
                   "state_bytes": 4 * 2 ** (args.L - 1 if args.L >= 14 else args.L)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"full O-dp sweep of a {Ls}x{Ls} +-J instance per step, scaled by "
                                   f"(L-1)L2^L updates to {args.L}x{args.L}"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def other_configs(torch):
    """cfg 2, 3, 5 of BASELINE.json through the plan API; bytes_min as in
    BASELINE.md section 2 (north_star roofline: (L-1) * 2 * B_e * q^L per instance)."""
    import paper_2008_06888_b200 as ttn
    from ttn_inputs import CONFIGS, config_batch
    peak, _ = measured_peaks()
    rows = {}
    for name, cfg, q, call, be in (("cfg2_16x16_gauss_ground_config_batch256", 2, 2, ttn.CALL_CONFIG, 4),
                                   ("cfg3_24x24_pmj_count_batch16", 3, 2, ttn.CALL_COUNT, 12),
                                   ("cfg5_potts_18x18_pmj_count_batch4", 5, 3, ttn.CALL_COUNT, 12)):
        try:
            Jh, Jv, h = config_batch(cfg)
            plan = ttn.Plan(q, call, Jh, Jv, h)
            plan.launch()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(3):
                plan.launch()
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b) / 3
            B, Lc = Jh.shape[0], CONFIGS[cfg]["L"]
            bmin = B * (Lc - 1) * 2 * be * q ** Lc      # cfg 2: = the checkpoints written once and read back once
            moved = bytes_moved(be, plan.state_elements, plan.num_passes, B)
            if call == ttn.CALL_CONFIG:                 # every pass reads and writes (checkpoints); the backward pass reads them once
                moved = float(B) * (2 * plan.num_passes - 1 + Lc) * be * plan.state_elements
            rows[name] = {"ms_total": ms, "ms_per_instance": ms / B, "batch": B, "hbm_passes": plan.num_passes,
                          "launches": plan.num_launches,
                          # q^L, or the part of it the sweep stores: half (h = 0 flip symmetry, cfg 3), a third
                          # (Potts colour rotation, cfg 5)
                          "state_elements_stored": plan.state_elements,
                          # bytes the passes move (computed from the pass count) over time and measured peak
                          "bytes_moved_computed": moved,
                          "hbm_roofline_frac": moved / (peak * 1e9) / (ms * 1e-3),
                          # north_star's figure: one read + write of the FULL q^L vector per row; may exceed 1
                          "algorithmic_equivalent_frac": bmin / (peak * 1e9) / (ms * 1e-3)}
            plan.close()
            del plan
            torch.cuda.empty_cache()
        except ttn.TTNError as e:
            rows[name] = {"unavailable": str(e)}
    # the rest of north_star's "2^28..2^32-entry" band (f32, +-J, h = 0: flip-reduced like the headline) and
    # the paper's own headline workload, 32x32 GAUSSIAN couplings and fields in Float32 (PAPER.md:118, 282:
    # 590 s on its GPU): fields break the flip symmetry, so this leg sweeps the full 2^32-entry state
    for name, Lc, kind, seed in (("band_28x28_pmj_f32", 28, "pmj", 4000), ("band_30x30_pmj_f32", 30, "pmj", 4000),
                                 ("paper_32x32_gauss_J_and_h_f32", 32, "gauss", 2032)):
        try:
            Jh, Jv, h = make_batch(Lc, [seed], kind, fields=(kind == "gauss"))
            plan = ttn.Plan(2, ttn.CALL_ENERGY, Jh, Jv, h)
            ms = time_plan(torch, plan, reps=3)
            E = float(plan.read()[0][0])
            rows[name] = {"ms_per_instance": ms, "E0": E, "hbm_passes": plan.num_passes, "launches": plan.num_launches,
                          "state_elements_stored": plan.state_elements,
                          "bound": "alu",
                          "alu_roofline_frac": float(Lc) * (Lc - 1) * plan.state_elements / (ms * 1e-3) / (SMS * ALU_LANES * 1.965e9),
                          "hbm_roofline_frac": bytes_moved(4, plan.state_elements, plan.num_passes) / (peak * 1e9) / (ms * 1e-3),
                          "algorithmic_equivalent_frac": bytes_min(Lc) / (peak * 1e9) / (ms * 1e-3)}
            plan.close()
            del plan
            torch.cuda.empty_cache()
        except (ttn.TTNError, RuntimeError) as e:
            rows[name] = {"unavailable": str(e).splitlines()[0][:200]}
            torch.cuda.empty_cache()
    # +-J chimera graph, L x L unit cells (8 L^2 spins), Tropical<i16>, through the
    # one-call C ABI (host couplings; table upload and the read-back of E0 are inside the timed region).
    # State: the paper's 16^L, 2^(4L) int16, no ancilla in HBM (ttn_chimera2.cuh).  Roofline
    # denominator = the paper's formulation: one read + one write of that state per unit cell (each cell is
    # one 16 x 16 tensor applied to the state), the first one write-only.  The sweep itself makes 4 passes
    # per COLUMN of cells (3 gate-row passes + the column's vertical chain), i.e. fewer bytes than that.
    from ttn_inputs import make_chimera_instance
    for Lc, reps in ((7, 3), (8, 3)):
        name = f"next3_chimera_{Lc}x{Lc}_cells_{8 * Lc * Lc}_spins_i16"
        try:
            I = make_chimera_instance(Lc, Lc, 7000 + Lc)
            wsc = ttn.alloc_workspace(ttn.chimera_workspace_bytes(Lc, Lc))
            E = ttn.chimera_sweep_energy_i16(I.K, I.Jv, I.Jh, workspace=wsc)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                E2 = ttn.chimera_sweep_energy_i16(I.K, I.Jv, I.Jh, workspace=wsc)
            b.record()
            torch.cuda.synchronize()
            assert E2 == E
            ms = a.elapsed_time(b) / reps
            state_bytes = 2 * 2 ** (4 * Lc)
            passes = 4 * Lc - 3                         # column 0: the chain kernel alone (write-only)
            rows[name] = {"ms_total": ms, "E0": E, "state_bytes": state_bytes, "hbm_passes": passes,
                          "launches": passes + 1,
                          "bytes_moved": (2 * passes - 2) * state_bytes,      # first pass write-only, last read-only
                          "hbm_roofline_frac": (2 * passes - 2) * state_bytes / (peak * 1e9) / (ms * 1e-3),
                          "algorithmic_equivalent_frac": (2 * Lc * Lc - 1) * state_bytes / (peak * 1e9) / (ms * 1e-3),
                          "algorithmic_equivalent_note": "denominator: one read + write of the 16^L int16 state per unit cell "
                                               "(the paper's tensor-by-tensor evolution); round 1 kept a 4-spin "
                                               "ancilla in HBM (16 x the state) and took 2686 ms at 8 x 8 cells"}
            del wsc
            torch.cuda.empty_cache()
        except (ttn.TTNError, RuntimeError) as e:      # RuntimeError: torch could not allocate the state
            rows[name] = {"unavailable": str(e).splitlines()[0][:200]}
            torch.cuda.empty_cache()
    # chimera counting (Fig. 3: residual entropies): CountingTropical on the same column front
    try:
        Lc = 8
        I = make_chimera_instance(Lc, Lc, 7000 + Lc)
        wsc = ttn.alloc_workspace(ttn.chimera_count_workspace_bytes(Lc, Lc))
        E, g = ttn.chimera_sweep_count(I.K, I.Jv, I.Jh, workspace=wsc)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        E2, g2 = ttn.chimera_sweep_count(I.K, I.Jv, I.Jh, workspace=wsc)
        b.record()
        torch.cuda.synchronize()
        assert (E2, g2) == (E, g)
        rows["next3_chimera_8x8_cells_512_spins_count"] = {
            "ms_total": a.elapsed_time(b), "E0": E, "degeneracy": g, "state_bytes": 12 * 2 ** (4 * Lc),
            "entropy_per_spin": float(np.log(g) / (8 * Lc * Lc))}
        del wsc
        torch.cuda.empty_cache()
    except (ttn.TTNError, RuntimeError) as e:
        rows["next3_chimera_8x8_cells_512_spins_count"] = {"unavailable": str(e).splitlines()[0][:200]}
        torch.cuda.empty_cache()
    return rows


def cpu_baseline(L_target: int, L_sample: int, gpu_ms_same_L=None):
    """O-dp as it stands on the host cores: ONE full sweep of an L_sample x L_sample +-J instance
    (a measurement), next to the GPU time for the same instance; `value` extrapolates it to the
    workload by the update count -- an under-estimate, since the 32x32 frontier (34 GB) is far out
    of cache while the sample's is not: the one measured full-size run is quoted beside it."""
    import oracle
    Jh, Jv, _ = make_batch(L_sample, [4000], "pmj")
    t = time.perf_counter()
    E = oracle.dp_ising(L_sample, Jh[0], Jv[0], None, count=False)[0]
    dt = time.perf_counter() - t
    val = dt / updates(L_sample) * updates(L_target) * 1e3
    return {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "extrapolated": True,
            "sample": f"one full O-dp sweep of a {L_sample}x{L_sample} +-J instance (seed 4000), measured {dt:.1f} s; "
                      f"`value` scales it by (L-1)L2^L updates to {L_target}x{L_target}",
            "measured": {"L": L_sample, "ms": dt * 1e3, "E0": E, "gpu_ms_same_instance": gpu_ms_same_L},
            "full_size_oracle_run": ORACLE_FULL_32 if L_target == 32 else None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--L", type=int, default=32)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-L", type=int, default=24, dest="ref_L")
    ap.add_argument("--cpu-L", type=int, default=28, dest="cpu_L")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", dest="no_other_configs")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                   # timing rule: W >= 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2008_06888_b200 as ttn

    rank, local_rank, world = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the sweep has no CPU path)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    L = args.L
    Jh, Jv, _ = make_batch(L, [seed_for_rank(rank)], "pmj")
    ws = ttn.alloc_workspace(ttn.workspace_bytes(2, L, ttn.TROPICAL_F32, 1), f"cuda:{local_rank}")
    plan = ttn.Plan(2, ttn.CALL_ENERGY, Jh, Jv, None, workspace=ws)
    torch.cuda.synchronize()

    for _ in range(args.warmup):
        plan.launch()
    torch.cuda.synchronize()
    E_dev = plan.read()[0][0]

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank) if rank == 0 else None
    barrier()
    if sampler:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record()
    for k in range(args.steps):
        plan.launch()
        ev[k + 1].record()
    barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = ev[0].elapsed_time(ev[-1])
    step_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / args.steps

    # ---- end to end through the one-call C ABI with host buffers -----------------------------
    e2e_times = []
    for i in range(2 + min(args.steps, 3)):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        E_host = ttn.sweep_energy(Jh, Jv, workspace=ws)[0]
        if i >= 2:
            e2e_times.append((time.perf_counter() - t0) * 1e3)
    e2e_ms = float(np.mean(e2e_times))
    e2e_ms = max_over_ranks(e2e_ms, dist, "cuda")
    assert E_host == E_dev, (E_host, E_dev)

    # ---- NEXT-1 beside it: the same instance in Tropical<i16> (exact for integer couplings) ------
    i16 = None
    try:
        p16 = ttn.Plan(2, ttn.CALL_ENERGY_I16, Jh, Jv, None, workspace=ws)
        for _ in range(2):
            p16.launch()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(3):
            p16.launch()
        b.record()
        torch.cuda.synchronize()
        E16 = p16.read()[0][0]
        assert E16 == E_dev, (E16, E_dev)
        i16 = {"ms_per_instance": a.elapsed_time(b) / 3, "hbm_passes": p16.num_passes, "state_bytes": 2 * p16.state_elements,
               "note": "ttn_sweep_energy_i16 (SURVEY.md NEXT-1), same instance, E0 identical; not the headline metric"}
        p16.close()
    except ttn.TTNError as e:      # e.g. L below the i16 path's limits
        i16 = {"unavailable": str(e)}

    # ---- the GPU time for the very instance the CPU baseline sweeps (same L, same seed)
    gpu_same = None
    if rank == 0 and not args.no_cpu_baseline:
        Jc, Jd, _ = make_batch(args.cpu_L, [4000], "pmj")
        pc = ttn.Plan(2, ttn.CALL_ENERGY, Jc, Jd, None, workspace=ws if args.cpu_L <= L else None)
        gpu_same = time_plan(torch, pc, reps=3)
        pc.close()

    # ---- the other BASELINE.json configs, timed beside the headline (rank 0, one GPU; they are parity
    # cases, not the metric: device time of ttn_plan_launch, couplings resident, mean of 3 launches)
    others = None
    if rank == 0 and world == 1 and L == 32 and not args.no_other_configs:
        others = other_configs(torch)

    if rank == 0:
        peak, peak_src = measured_peaks()
        traffic, traffic_src = ncu_traffic_per_launch("r03b_ncu_full_sweep_summary.csv", "fused_pass_kernel") if L == 32 else (None, None)
        per_inst_ms = whole_job_ms_per_instance(ms_per_step, world)
        moved = bytes_moved(4, plan.state_elements, plan.num_passes)    # bytes one sweep really moves (computed)
        achieved = moved / (ms_per_step * 1e-3) / 1e9                   # GB/s per GPU
        alg_equiv = bytes_min(L) / (ms_per_step * 1e-3) / 1e9           # north_star's full-vector, pass-per-row bytes
        sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
        alu_peak = SMS * ALU_LANES * sm_mhz * 1e6                       # FMNMX: 64 lanes/clk/SM (alu pipe)
        # max-plus updates the sweep executes: L (L-1) gates (L-1 of them flip gates under the h = 0
        # reduction) over the stored state
        upd_exec = float(L) * (L - 1) * plan.state_elements
        out = {
            "metric": METRIC, "value": per_inst_ms, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(L),
                       "L": L, "state_bytes": 4 * plan.state_elements, "hbm_passes": plan.num_passes,
                       "symmetry": "h = 0: the flip-symmetric half-state (column 0 up) is stored and swept"
                       if plan.state_elements < 2 ** L else "none",
                       "l2_policy": "state (>= 1 GiB) far larger than the 126 MB L2; no flush needed"
                       if L >= 28 else "state fits L2: flush not applied, number is L2-resident",
                       "E0": E_dev},
            "e2e": {"value": e2e_ms / world, "unit": UNIT,
                    "h2d_bytes_per_step": int(Jh.nbytes + Jv.nbytes), "d2h_bytes_per_step": 4},
            "gpu_launches": plan.num_launches * args.steps,
            # the roof that binds: FMNMX issue on the alu pipe (the sweep moves ~0.3 TB in ~0.18 s, a quarter of the HBM peak)
            "roofline": {"bound": "alu", "achieved": upd_exec / (ms_per_step * 1e-3) / 1e9,
                         "peak": alu_peak / 1e9, "unit": "G max-plus updates/s",
                         "frac": upd_exec / (ms_per_step * 1e-3) / alu_peak,
                         "updates_per_sweep": upd_exec,
                         "peak_source": "148 SMs x 64 FMNMX lanes/clk/SM (profiles/r01_ubench.md) x the SM clock sampled "
                                        "during the timed region (DESIGN.md section 6)",
                         # dram__bytes_read.sum + dram__bytes_write.sum per pass launch, mean over ALL 19 pass launches of
                         # one sweep, read from the committed ncu --set full summary (None if absent / other L)
                         "traffic": traffic, "traffic_source": traffic_src,
                         "traffic_computed_per_launch": moved / plan.num_passes,
                         "note": "1 FMNMX per EXECUTED update: L(L-1) gates over the stored state (half of north_star's "
                                 "full-vector count under the h = 0 flip reduction)",
                         "kernel": "ttn::fused_pass_kernel<LOW|HIGH> (all %d pass launches of one sweep)" % plan.num_passes},
            "hbm_roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                             "frac": achieved / peak, "peak_source": peak_src,
                             "bytes_moved_per_sweep_computed": moved,
                             "note": "achieved = bytes the %d passes move (read + write of the STORED state per pass, first "
                                     "write-only, last read-only) / time" % plan.num_passes,
                             # north_star's yardstick: (L-1)*2*4*2^L bytes (FULL vector, one pass per row) over the same
                             # time; not a bandwidth -- the sweep stores half the vector and fuses rows -- may exceed 1
                             "algorithmic_bytes_per_sweep": bytes_min(L),
                             "algorithmic_equivalent_GBs": alg_equiv,
                             "algorithmic_equivalent_frac": alg_equiv / peak,
                             "algorithmic_equivalent_frac_vs_nominal_8TBs": alg_equiv / 8000.0},
            "step_ms_median": float(np.median(step_ms)), "step_ms_best": float(np.min(step_ms)),
            "step_ms": step_ms, "clocks": clocks, "tropical_i16": i16,
        }
        if others is not None:
            out["other_configs"] = others
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(L, args.cpu_L, gpu_same)
        print(json.dumps(out))
    plan.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
