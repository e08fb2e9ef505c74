#!/usr/bin/env python
"""bench.py -- one JSON line for the KBMOD shift-and-stack hot path on B200.

A "step" is one pass of the whole hot path (S1..S6: kbmod_make_psi_phi + kbmod_search) over one
synthetic DECam-shaped stack.  Default workload = BASELINE.json configs[2], the configuration the
metric is quoted on (15 x 4096 x 4096, 640 velocities, K=8, min_obs=8; 1.07e10 trajectories,
1.61e11 trajectory-evals).  `value` = trajectory-evals/s of the whole step with inputs resident in
HBM; `e2e` = the same through the public API from pinned HOST buffers (H2D of sci/var/mask and D2H
of the result planes inside the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 3] [--kernel 0]

--kernel 0 (default): the library's default search kernel (KBMOD_KERNEL_AUTO), the one the GPU test
suite validates against the oracle; the same kernel every run.  --kernel k (1 direct, 2 tiled,
3 TMA-staged, 4 tiled + queued top-K) times that kernel instead; 3 and 4 are opt-in until they have
passed the GPU suite on hardware.  The kernel and its knobs travel in
kbmod_search_options; the host plan (kbmod_plan: it depends on times / grid / shape only) is built
once before the timed region, as a survey pipeline searching many stacks of one cadence would.

--mode threshold: the paper's own retention rule (row N4): kbmod_search_threshold with nu >= --nu-min
(default 10) in place of the per-pixel top-K; `--config 6` is the paper's production
grid (128 x 250 = 32 000 velocities on 13 images).  Not the driver's default workload.

N > 1 (torchrun): every rank searches its own independent stack (the survey's fields/CCDs are
independent searches) -- weak scaling, no data-path collective.  --bands (N > 1):
ONE stack replicated on every rank, each rank searching its band of start rows through
kbmod_search_rows -- strong scaling, still no data-path collective.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1901_02492_b200 import shard, synth  # noqa: E402

METRIC = "trajectory-evals/s"
UNIT = "trajectory-evals/s"
SM_COUNT = 148
LDS_BYTES_PER_CLK_PER_SM = 128          # shared-memory crossbar (B300_MICROARCH.md "LDS/STS")
SAMPLE_BYTES = 8                        # one float2 (psi, phi) per trajectory-eval
KERNEL_NAMES = {0: "search_tiled_kernel (automatic)", 1: "search_direct_kernel", 2: "search_tiled_kernel",
                3: "search_staged_kernel", 4: "search_tiledq_kernel"}


def last_capture(kernel):
    """The last committed `ncu --set full` capture of this search kernel at the bench workload
    (profiles/ncu_captures.csv, hand-copied from the summaries it cites).  It describes the commit
    it names, not this run: it is reported beside the roofline, never as `traffic`."""
    import csv
    p = os.path.join(ROOT, "profiles", "ncu_captures.csv")
    if not os.path.exists(p):
        return None
    name = KERNEL_NAMES.get(kernel, "").split(" ")[0]
    for row in csv.DictReader(open(p)):
        if row["kernel"] == name:
            out = {}
            for k, v in row.items():
                try:
                    out[k] = float(v) if k not in ("kernel", "commit", "source", "note") else v
                except ValueError:
                    out[k] = v or None
            out["l2_to_sm_bytes_per_sample_byte"] = (out["l2_to_l1_bytes"] / (15 * 4096 * 4096 * 640 * 8.0)
                                                     if out.get("l2_to_l1_bytes") else None)
            return out
    return None


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d.get("hbm_gbs", 6650.0)), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def workload(args):
    over = {}
    if args.rows:
        over["H"] = args.rows
    cfg = synth.config(args.config, **over)
    return cfg


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True,
                                     text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 7
                          for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(self.rows)}


# ----------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle as it stands, on the host cores, bounded sample
# ----------------------------------------------------------------------------------------------
def oracle_prepare(cfg, st):
    """A full-height psi/phi stack for the oracle's search sample, made outside any timed region
    by repeating a 32-row band built by the oracle (the oracle's work per evaluation does not
    depend on the values; building all 2.5e8 pixels on the CPU would take minutes)."""
    import oracle
    band = min(cfg.H, 32)
    pp_band = oracle.make_psi_phi(st.sci[:, :band], st.var[:, :band], st.mask[:, :band], st.psf)
    reps = int(math.ceil(cfg.H / band))
    return np.ascontiguousarray(np.tile(pp_band, (1, reps, 1, 1))[:, :cfg.H])


def oracle_sample(cfg, st, pp_full, rows):
    """One bounded sample of the step through the oracle as it stands: psi/phi of `rows` rows of
    every image, then the full-grid search of `rows` start rows (full images, all velocities).
    Returns (trajectory-evals, seconds)."""
    import oracle
    rows = min(rows, cfg.H)
    y0 = cfg.H // 2 - rows // 2
    t0 = time.perf_counter()
    oracle.make_psi_phi(st.sci[:, y0:y0 + rows], st.var[:, y0:y0 + rows],
                        st.mask[:, y0:y0 + rows], st.psf)
    oracle.search(pp_full, st.times, st.vel_grid, cfg.K, cfg.min_obs, mode=oracle.MODE_F32SEQ,
                  y_begin=y0, y_end=y0 + rows)
    return rows * cfg.W * cfg.V * cfg.N, time.perf_counter() - t0


def sample_text(cfg, rows):
    return (f"{min(rows, cfg.H)} of {cfg.H} start rows per step: psi/phi of those rows of all "
            f"{cfg.N} images + search of {min(rows, cfg.H)} x {cfg.W} start pixels x {cfg.V} "
            f"velocities x {cfg.N} images; oracle f32seq mode, OpenMP over rows")


def run_reference(args, cfg, st):
    import oracle
    oracle.build()
    pp_full = oracle_prepare(cfg, st)
    for _ in range(args.warmup):
        oracle_sample(cfg, st, pp_full, max(1, args.ref_rows // 8))
    tot_e, tot_s = 0, 0.0
    for _ in range(args.steps):
        e, s = oracle_sample(cfg, st, pp_full, args.ref_rows)
        tot_e += e
        tot_s += s
    val = tot_e / tot_s
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": config_dict(cfg, args),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(),
                         "kind": "oracle", "sample": sample_text(cfg, args.ref_rows)},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def evals_per_step(cfg, world):
    return cfg.evals * world


def config_dict(cfg, args):
    return {"workload": f"BASELINE.json configs[{args.config - 1}] {cfg.name}: N={cfg.N} "
                        f"{cfg.H}x{cfg.W} fp32, V={cfg.V} ({cfg.n_angles}x{cfg.n_speeds}), "
                        f"K={cfg.K}, min_obs={cfg.min_obs}, seed={cfg.seed}",
            "trajectories": cfg.trajectories, "trajectory_evals": cfg.evals,
            "step": ("kbmod_make_psi_phi + kbmod_search_threshold (S1..S5 + nu >= %g, row N4)" % args.nu_min
                     if getattr(args, "mode", "topk") == "threshold" else "kbmod_make_psi_phi + kbmod_search (S1..S6)"),
            "l2": "inputs larger than L2 (stack 2.0 GB+ vs 126 MB); no flush needed",
            "parallelism": (f"one stack: psi/phi sharded by image + one NCCL all-gather, then start-row bands x{args.gpus} "
                            "(kbmod_search_rows)" if getattr(args, "bands", False)
                            and args.gpus > 1 else f"independent stacks x{args.gpus}")}


# ----------------------------------------------------------------------------------------------
# GPU arm
# ----------------------------------------------------------------------------------------------
def run_gpu(args, cfg, st, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_1901_02492_b200 import binding, build
    build.build()
    binding.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    kernel = args.kernel
    N, H, W, V, K = cfg.N, cfg.H, cfg.W, cfg.V, cfg.K
    # the host plan depends on (times, grid, shape, K, options) only: built once, outside the timed region
    plan = binding.Plan(st.times, N, H, W, st.vel_grid, K, kernel=kernel, tile_group_w=args.group_w,
                        staged_geom=args.staged_geom)

    # pinned host inputs and outputs (for e2e), resident device copies (for value)
    h_sci = torch.from_numpy(st.sci).pin_memory()
    h_var = torch.from_numpy(st.var).pin_memory()
    h_mask = torch.from_numpy(st.mask).pin_memory()
    d_sci, d_var, d_mask = h_sci.to(dev), h_var.to(dev), h_mask.to(dev)
    psiphi = torch.empty((N, H, W, 2), dtype=torch.float32, device=dev)
    bands = bool(args.bands) and world > 1
    y0, y1 = shard.row_bands(H, world)[rank] if bands else (0, H)
    out = binding.alloc_result(y1 - y0, W, K, dev)
    ws = binding.alloc_workspace(binding.search_workspace(N, H, W, V, K), dev)
    h_out = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.items()}
    e_sci, e_var, e_mask = torch.empty_like(d_sci), torch.empty_like(d_var), torch.empty_like(d_mask)
    h_count = torch.zeros(1, dtype=torch.int64).pin_memory()

    def search_step():
        if args.mode == "threshold":
            return binding.search_threshold(psiphi, st.times, st.vel_grid, cfg.min_obs, args.nu_min, args.capacity,
                                            y_begin=y0, y_end=y1, kernel=kernel, tile_group_w=args.group_w, workspace=ws)
        return binding.search(psiphi, None, None, K, cfg.min_obs, out=out, workspace=ws, plan=plan, y_begin=y0, y_end=y1)

    def build_psi_phi(a, b, c):
        if bands:       # one stack on all ranks: S2 sharded by image, one all-gather (NCCL), then the row-band search
            psiphi.copy_(shard.make_psi_phi_sharded(a, b, c, st.psf))
        else:
            binding.make_psi_phi(a, b, c, st.psf, out=psiphi)

    def step_resident():
        build_psi_phi(d_sci, d_var, d_mask)
        search_step()

    def step_e2e():
        e_sci.copy_(h_sci, non_blocking=True)
        e_var.copy_(h_var, non_blocking=True)
        e_mask.copy_(h_mask, non_blocking=True)
        build_psi_phi(e_sci, e_var, e_mask)
        r = search_step()
        if args.mode == "threshold":
            h_count.copy_(r[0], non_blocking=True)          # the candidate list stays on the device for N1/N2
            return
        for k in out:
            h_out[k].copy_(out[k], non_blocking=True)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, sampler=None):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        barrier()
        if sampler:
            sampler.start()
        ev[0].record()
        for s in range(steps):
            fn()
            ev[s + 1].record()
        barrier()
        if sampler:
            sampler.stop_flag.set()
        return shard.max_over_ranks(ev[0].elapsed_time(ev[-1]), dev)

    for _ in range(max(3, args.warmup)):
        step_resident()
    binding.search_status(ws)               # raises if a kernel gave up (never times a broken run)
    sampler = ClockSampler(local_rank)
    n0 = binding.launch_count()
    total_ms = timed(step_resident, args.steps, sampler)
    launches = binding.launch_count() - n0
    clocks = sampler.summary()

    # per-phase device times (same stream, CUDA events), median over the timed count
    def phase(fn, reps):
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))
    reps = max(3, min(args.steps, 10))
    ms_psiphi = phase(lambda: binding.make_psi_phi(d_sci, d_var, d_mask, st.psf, out=psiphi), reps)
    ms_search = phase(search_step, reps)

    binding.search_status(ws)
    step_e2e()
    e2e_steps = max(1, min(args.steps, 5))
    e2e_ms = timed(step_e2e, e2e_steps)

    # the same step through the single C-ABI call that takes HOST buffers (kbmod_search_host);
    # reported beside `e2e`, and only if its result planes equal the resident run's
    host_abi = None
    try:
        if world > 1 or args.mode == "threshold":
            raise RuntimeError("measured at N=1 in top-K mode only")
        ws_h = binding.alloc_workspace(binding.search_host_workspace(N, H, W, V, K), dev)
        run_h = lambda: binding.search_host(h_sci, h_var, h_mask, st.psf, st.times, st.vel_grid, K,
                                            cfg.min_obs, h_out, ws_h, kernel=kernel)
        run_h()
        binding.search_status(ws_h)
        same = all(torch.equal(h_out[k], out[k].cpu()) or k in ("nu", "alpha", "psi", "phi") and
                   torch.equal(h_out[k].view(torch.int32), out[k].cpu().view(torch.int32)) for k in out)
        if same:
            ms = timed(run_h, e2e_steps) / e2e_steps
            host_abi = {"value": evals_per_step(cfg, world) / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms,
                        "call": "kbmod_search_host", "verified_equal_to_resident_run": True}
        else:
            host_abi = {"error": "result planes differ from the resident run"}
        del ws_h
    except Exception as exc:                                   # never costs the main line
        host_abi = {"error": f"{type(exc).__name__}: {exc}"[:200]}

    if rank != 0:
        return
    hbm_gbs, sm_max_mhz, peak_src = load_peaks()
    evals = cfg.evals * (1 if bands else world)        # --bands: one stack shared by all ranks
    ms_per_step = total_ms / args.steps
    value = evals / (ms_per_step * 1e-3)
    # roofline of the dominant kernel (the search): algorithmic shared-memory sample bytes
    # (8 B per trajectory-eval) against the LSU peak 148 SM x 128 B/clk x max SM clock
    lsu_peak = SM_COUNT * LDS_BYTES_PER_CLK_PER_SM * sm_max_mhz * 1e6 / 1e9       # GB/s
    band_evals = cfg.evals * (y1 - y0) // H           # what THIS rank's search launch processed
    achieved = band_evals * SAMPLE_BYTES / (ms_search * 1e-3) / 1e9
    hbm_bytes = N * H * W * 8 + H * W * K * 24
    # e2e: host buffers in, host result planes out, transfers inside the timed region.  The headline
    # is the single C-ABI call on HOST buffers (kbmod_search_host) when its planes were verified
    # equal to the resident run's; the same step driven from Python (torch pinned-memory copies
    # around kbmod_make_psi_phi + kbmod_search) is reported beside it and is the fallback.
    xfer = {"h2d_bytes_per_step": int(h_sci.numel() * 4 + h_var.numel() * 4 + h_mask.numel()),
            "d2h_bytes_per_step": (8 if args.mode == "threshold" else
                                   int(sum(v.numel() * v.element_size() for v in h_out.values())))}
    e2e_binding = {"value": evals / (e2e_ms / e2e_steps * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / e2e_steps,
                   "path": "torch pinned H2D copies + kbmod_make_psi_phi + kbmod_search + torch D2H copies", **xfer}
    if host_abi and "value" in host_abi and world == 1:
        e2e = {"value": host_abi["value"], "unit": UNIT, "ms_per_step": host_abi["ms_per_step"],
               "path": "kbmod_search_host: one C-ABI call, HOST buffers in and out", **xfer}
    else:
        e2e = dict(e2e_binding)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "strong" if bands else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(cfg, args),
        "trajectories_per_s": cfg.trajectories * (1 if bands else world) / (ms_per_step * 1e-3),
        "phases_ms": {"make_psi_phi": ms_psiphi, "search": ms_search},
        "search_only": {"trajectory_evals_per_s": cfg.evals / (ms_search * 1e-3),
                        "trajectories_per_s": cfg.trajectories / (ms_search * 1e-3)},
        "roofline": {"bound": "smem", "achieved": achieved, "peak": lsu_peak, "unit": "GB/s",
                     "frac": achieved / lsu_peak,
                     # dram bytes of THIS build's kernel need an ncu capture of this commit; none exists
                     # until one is taken (profiles/), so none is claimed
                     "traffic": None,
                     "last_capture": (last_capture(kernel) if args.config == 3 and not args.rows else None),
                     "kernel": f"kbmod_search -> {KERNEL_NAMES.get(kernel, kernel)}",
                     "peak_source": f"148 SM x 128 B/clk x {sm_max_mhz:.0f} MHz ({peak_src} max "
                                    "SM clock); north_star roofline = slower of HBM and LSU",
                     "hbm": {"compulsory_bytes": hbm_bytes, "peak": hbm_gbs,
                             "achieved": hbm_bytes / (ms_search * 1e-3) / 1e9,
                             "floor_ms": hbm_bytes / (hbm_gbs * 1e9) * 1e3},
                     "lsu_floor_ms": band_evals * SAMPLE_BYTES / (lsu_peak * 1e9) * 1e3},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": e2e,
        "e2e_binding_copies": e2e_binding,
        "e2e_host_abi": host_abi,
        "search_kernel": KERNEL_NAMES.get(kernel, str(kernel)),
        "search_options": {"kernel": kernel, "tile_group_w": args.group_w, "staged_geom": args.staged_geom,
                           "plan": "kbmod_plan built once before the timed region"},
    }
    if world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        del d_sci, d_var, d_mask
        pp_full = oracle_prepare(cfg, st)
        oracle_sample(cfg, st, pp_full, 1)
        e, s = oracle_sample(cfg, st, pp_full, args.ref_rows)
        line["cpu_baseline"] = {"value": e / s, "unit": UNIT, "cores": oracle.num_threads(),
                                "kind": "oracle", "sample": sample_text(cfg, args.ref_rows),
                                "seconds": s}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--rows", type=int, default=0, help="override H (debug only)")
    ap.add_argument("--kernel", type=int, default=0, choices=[0, 1, 2, 3, 4],
                    help="0 library default (the kernel the GPU test suite validates), 1 direct, 2 tiled, "
                         "3 TMA-staged, 4 tiled + queued top-K (3 and 4: opt-in, see DESIGN.md section 8)")
    ap.add_argument("--group-w", type=int, default=0, help="kbmod_search_options.tile_group_w (0 = default)")
    ap.add_argument("--staged-geom", type=int, default=0, help="kbmod_search_options.staged_geom (kernel 3)")
    ap.add_argument("--mode", default="topk", choices=["topk", "threshold"],
                    help="topk: kbmod_search (BASELINE.json's metric); threshold: kbmod_search_threshold (row N4)")
    ap.add_argument("--nu-min", type=float, default=10.0, help="--mode threshold: detection threshold (PAPER.md:237)")
    ap.add_argument("--capacity", type=int, default=1 << 24, help="--mode threshold: candidate list capacity")
    ap.add_argument("--bands", action="store_true",
                    help="N > 1: one replicated stack, one band of start rows per rank (strong scaling)")
    ap.add_argument("--ref-rows", type=int, default=256, help="start rows per oracle sample")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = workload(args)

    if args.impl == "reference":
        if rank != 0:
            return
        st = synth.make_stack(cfg)
        run_reference(args, cfg, st)
        return

    import torch.distributed as dist
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")
    # an independent stack per rank (weak scaling), or the same stack on every rank (--bands)
    st = synth.make_stack(cfg, seed=cfg.seed if args.bands else shard.rank_seed(cfg.seed, rank))
    run_gpu(args, cfg, st, rank, world, local_rank)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
