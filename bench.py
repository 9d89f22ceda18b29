#!/usr/bin/env python
"""bench.py — one JSON line for the radiance-cascades hot path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A "step" is one full J solve (every cascade: pack, march, boundary, merge, J) of one synthetic
atmosphere.  Default workload: BASELINE.json configs[2] (1024x1024 cells, 64 wavelengths, 8 cascades),
the configuration the metric's target is quoted on.  value = probe-ray-wavelength segments per second,
whole job, inputs resident in HBM; e2e = the same through rc_solve_J_host with pinned HOST buffers
(H2D of chi, eta and D2H of J inside the timed region).  N > 1: one process per GPU, each solving its
wavelength block of the SAME atmosphere (the path shards by wavelength with no exchange; Jbar: one NCCL
all-reduce) - strong scaling; without a launcher `--gpus N` starts the N ranks itself.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2408_14425_b200 import atmospheres  # noqa: E402

METRIC = "probe-ray-wavelength segments/sec"
UNIT = "seg-lambda/s"
SM_COUNT, MUFU_PER_CLK_SM = 148, 16  # one ex2 per segment-wavelength; DESIGN.md §7
# ncu --set full captures of the dominant launch that are committed under profiles/, keyed by (mode, config, cascade):
# dram__bytes_read.sum + dram__bytes_write.sum per launch, l1tex__m_xbar2l1tex_read_bytes.sum (bytes that really came over
# the L2 -> SM path; the algorithmic bytes also count what L1 served), lts__t_sectors % of peak, and where the capture is.
# A run whose mode / config / launch plan has no entry reports traffic = null.  Every entry names the kernel it is a capture
# of and the sha of that kernel's source text at the capture's commit (kernel_text_sha): when HEAD's text differs the
# capture describes another kernel, and the line reports its figures under `stale_capture` only, with traffic = null.
NCU_CAPTURES = {
    ("flat", 2, 5): {"kernel": "march_kernel", "sha": "e6187b462936d78b", "commit": "e582544", "capture_ms": 30.78,
                     "dram_bytes": 2.027300e9 + 0.269690e9, "l2_to_sm_bytes": 484.840640e9, "lts_pct": 46.02,
                     "source": "profiles/ncu_r3.md: ncu --set full of march_kernel<8,1,3,8,2,0,0>, cascade 5 of config 2, "
                               "commit e582544 (30.78 ms under ncu)"},
    ("flat", 4, 5): {"kernel": "march_list_kernel", "sha": "7b7b5b40dbc40a63", "commit": "e582544", "capture_ms": 47.67,
                     "dram_bytes": 149.293018e9 + 3.933113e9, "l2_to_sm_bytes": 348.052288e9, "lts_pct": 30.28,
                     "source": "profiles/ncu_r3.md: ncu --set full of march_list_kernel<8,1,8,4,6,0> (hit lists), cascade 5 of config 4, "
                               "commit e582544 (47.67 ms under ncu)"},
    ("flat_incl8", 2, 5): {"kernel": "march_kernel", "sha": "e6187b462936d78b", "commit": "e43f0bd", "capture_ms": 223.63,
                           "dram_bytes": 5.754840e9 + 2.158622e9, "l2_to_sm_bytes": 1119.340e9, "lts_pct": 14.64,
                           "source": "profiles/ncu_r3.md: ncu --set full of march_kernel<8,8,2,8,3,0,0>, cascade 5 of config 2 x 8 "
                                     "inclinations, commit e43f0bd (223.6 ms under ncu)"},
    ("line_incl8", 2, 5): {"kernel": "march_kernel", "sha": "e6187b462936d78b", "commit": "e43f0bd", "capture_ms": 497.19,
                           "dram_bytes": 5.784382e9 + 2.636249e9, "l2_to_sm_bytes": 1878.842e9, "lts_pct": 11.05,
                           "source": "profiles/ncu_r3.md: ncu --set full of march_kernel<8,8,2,8,3,0,1>, cascade 5 of the "
                                     "moving line x 8 inclinations on the config-2 grid, commit e43f0bd (497.2 ms under ncu)"},
}


def kernel_text_sha(kernel: str):
    """sha256 (16 hex digits) of the source text of one kernel of csrc/rc_kernels.cu together with the device helpers in front
    of the march kernels (packed arithmetic, cell updates, warp -> probe mapping): what an ncu capture describes.  An entry
    of NCU_CAPTURES whose sha differs from HEAD's text is a capture of another kernel and its numbers are not used."""
    import hashlib
    lines = (ROOT / "paper_2408_14425_b200" / "csrc" / "rc_kernels.cu").read_text().splitlines()
    k = next((i for i, l in enumerate(lines) if l.startswith("__global__") and f" {kernel}(" in l), None)
    if k is None:
        return None
    h0 = next(i for i, l in enumerate(lines) if "f32x2 pk2(" in l)
    m = next(i for i, l in enumerate(lines) if l.startswith("__global__") and " march_kernel(" in l) - 1
    b0 = k - 1 if lines[k - 1].startswith("template") else k
    b1 = next(i for i in range(k, len(lines)) if lines[i] == "}")
    return hashlib.sha256("\n".join(lines[h0:m] + lines[b0:b1 + 1]).encode()).hexdigest()[:16]


def secondary_wanted(args, world):
    """Only the plain default run (config 2, one GPU, no mode flags) carries the other configs along."""
    return (world == 1 and args.config == 2 and not args.no_secondary and not args.line and not args.bilinear_fix
            and args.inclinations == 1 and not args.active and not args.tune and not args.analyse and not args.no_analyse)


def secondary_runs(configs=(0, 1, 3, 4), steps=3, warmup=3, timeout=420):
    """The other BASELINE.json configs in the same driver run, so that each has a number under the driver's clock: this
    script again, one child process per config (the GPU is idle while they run: the parent has finished timing), `steps`
    timed steps each.  A child that fails or overruns leaves its error text, never an exception."""
    out = {"note": f"bench.py --config N --steps {steps} --warmup {warmup} --no-cpu-baseline as child processes after the timed "
                   "region of this line; ms are device-timed solves / end-to-end rc_solve_J_host steps as in the main line"}
    for cfg in configs:
        cmd = [sys.executable, str(Path(__file__).resolve()), "--config", str(cfg), "--steps", str(steps), "--warmup", str(warmup),
               "--no-cpu-baseline", "--no-secondary"]
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout)
            d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
            out[f"config{cfg}"] = {"workload": d["config"]["workload"], "solve_ms": d["solve_ms"], "e2e_ms": d["e2e"]["ms_per_step"],
                                   "value": d["value"], "value_walked": d.get("value_walked"), "unit": d["unit"],
                                   "walked_fraction": d["config"]["walked_fraction"], "e2e_matches_device_path": d["e2e"]["matches_device_path"],
                                   "gpu_launches": d["gpu_launches"], "sm_mhz": d["clocks"].get("sm_mhz"), "reasons": d["clocks"].get("reasons")}
        except Exception as ex:  # noqa: BLE001 - reported in the line
            out[f"config{cfg}"] = {"error": f"{type(ex).__name__}: {str(ex)[:200]}"}
    return out


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True).start()
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(self.NAMES, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(atm, nwin, size=8, seed=0):
    """Time the fp64 oracle, as it stands, on `nwin` windows of size x size cells (all wavelengths)."""
    from oracle import rc_oracle
    rc_oracle.build()
    rng = np.random.default_rng(seed)
    segl, secs = 0, 0.0
    for _ in range(nwin):
        x0 = int(rng.integers(0, atm.nx - size + 1))
        y0 = int(rng.integers(0, atm.ny - size + 1))
        t = time.perf_counter()
        out = rc_oracle.solve_atmosphere(atm, window=(x0, x0 + size, y0, y0 + size), want_counts=True)
        secs += time.perf_counter() - t
        segl += int(out["segments"].sum()) * atm.nlambda * (1 if atm.mu is None else len(atm.mu))
    return segl, secs, rc_oracle.num_threads()


def run_reference(args, atm, workload):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    oracle_sample(atm, args.warmup, seed=99)
    segl, secs, cores = oracle_sample(atm, args.steps, seed=7)
    v = segl / secs
    sample = f"{args.steps} windows of 8x8 cells x {atm.nlambda} wavelengths (all cascades they depend on), one per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": workload},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start N ranks of this very command line (one per GPU) and wait."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
    sys.exit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lambda-batch", type=int, default=0)
    ap.add_argument("--line", action="store_true",
                    help="velocity-dependent line mode (SURVEY §8(f) f1): configs[2]'s recipe as a moving-line "
                         "atmosphere, opacities evaluated per ray (rc_set_line_atmosphere)")
    ap.add_argument("--bilinear-fix", action="store_true",
                    help="RC_BILINEAR_FIX (SURVEY §8(f) f3): 4 sub-rays per interval below the top cascade")
    ap.add_argument("--inclinations", type=int, default=1,
                    help="2.5D: N Gauss-Radau inclined rays per flatland ray (SURVEY §8(f) f2); the unit count "
                         "becomes segment-wavelength-inclinations")
    ap.add_argument("--active", default="",
                    help="sparsity as the paper defines it (PAPER.md:380, SURVEY §8(f) f4): 'occupied' flags the cells that hold "
                         "opacity, a number in (0, 1) the densest fraction of the cells (0.25: the paper's production run)")
    ap.add_argument("--no-analyse", action="store_true",
                    help="skip rc_analyse_atmosphere (free-space acceleration of mostly-empty atmospheres: by default called for "
                         "config 4, whose recipe is > 90 %% empty, and with --active, where the unflagged cells count as empty)")
    ap.add_argument("--analyse", action="store_true", help="call rc_analyse_atmosphere whatever the workload")
    ap.add_argument("--tune", default="", help="rc_set_tuning knobs, e.g. march_variant=0,bands=3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the `secondary` object (the other BASELINE configs, 3 steps each, run as child processes of the default bench)")
    ap.add_argument("--cpu-baseline-whole", action="store_true",
                    help="also time the oracle on ONE WHOLE solve of the workload (config 2: ~3 minutes on 16 cores) and check "
                         "the GPU J against it on every cell")
    ap.add_argument("--e2e-steps", type=int, default=0, help="end-to-end steps (default: the same as --steps)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    e2e_steps = args.e2e_steps or args.steps

    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    fx, fy, fl, fc = atmospheres.FULL_SHAPES[args.config]
    workload = (f"BASELINE.json configs[{args.config}]: {fx}x{fy} cells, {fl} wavelengths, {fc} cascades, "
                f"seeded synthetic atmosphere (DESIGN.md §4)")
    atm = atmospheres.make_config(args.config)      # ONE atmosphere for the whole job; ranks take wavelength blocks of it
    if args.line:
        atm = atmospheres.line_config2()
        fx, fy, fl, fc = atm.nx, atm.ny, atm.nlambda, atm.ncascades
        workload = (f"moving-line variant of BASELINE.json configs[2]: {fx}x{fy} cells, {fl} wavelengths, {fc} cascades, "
                    "line opacity evaluated per ray from the projected velocity (SURVEY §8(f) f1)")
    if args.inclinations > 1:
        atm = atmospheres.with_inclinations(atm, args.inclinations)
        workload += f", 2.5D with {args.inclinations} Gauss-Radau inclinations per ray (value counts segment-wavelength-inclinations)"
    if args.active:
        atm = (atmospheres.with_active_cells(atm) if args.active == "occupied" else
               atmospheres.with_active_cells(atm, mode="fraction", fraction=float(args.active)))
        workload += (f", cells of interest: {args.active} ({100 * atm.meta['active_fraction']:.1f} % of the cells flagged; "
                     "value counts the segments of flagged probes only)")
    if args.impl == "reference":
        run_reference(args, atm, workload)
        return

    import torch
    import torch.distributed as dist
    from paper_2408_14425_b200 import binding, sharding
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    hbm_peak, sm_max_mhz, peak_src = peaks()
    nlambda_job = atm.nlambda
    if world > 1:
        # the path shards by wavelength: rank r solves its contiguous block of the SAME
        # atmosphere; per-wavelength J needs no exchange, Jbar one all-reduce of nx ny floats (inside the timed region)
        # (the moving line shards the same way: every rank holds the six line parameters, its block is a slice of x_lambda)
        atm = sharding.shard_atmosphere(atm, rank, world)
        assert atm.nlambda > 0, f"{nlambda_job} wavelengths do not cover {world} ranks"

    flags = binding.RC_ACCUM_J if atm.accumulate else 0
    if args.bilinear_fix:
        flags |= binding.RC_BILINEAR_FIX
        workload += ", bilinear fix (the unit count includes the 4 sub-rays of every interval)"
    rc = binding.RadianceCascades(atm.ncascades, atm.c0_interval, local_rank, args.lambda_batch, flags)
    if args.tune:
        rc.set_tuning(**{k: float(v) for k, v in (kv.split("=") for kv in args.tune.split(","))})
    if atm.mu is not None:
        rc.set_inclinations(atm.mu, atm.w_mu)
    rc.ensure_workspace(atm.nx, atm.ny, atm.nlambda, host_io=True)
    if rc._ws.numel() < (80 << 20):  # room for the 64 MB region of the gather-bandwidth probe
        rc.set_workspace(torch.empty(80 << 20, dtype=torch.uint8, device=dev))
    active_d = None if atm.active is None else torch.from_numpy(np.ascontiguousarray(atm.active)).to(dev)
    if atm.line is not None:
        line_h = torch.from_numpy(atm.line).pin_memory()
        line_d = line_h.to(dev)
        rc.set_line_atmosphere(line_d, atm.xl)
    else:
        chi_h = torch.from_numpy(atm.chi).pin_memory()
        eta_h = torch.from_numpy(atm.eta).pin_memory()
        chi, eta = chi_h.to(dev), eta_h.to(dev)
        rc.set_atmosphere(chi, eta)

    def configure():
        rc.set_boundary(atm.I_below, atm.I_above)
        rc.set_lambda_weights(atm.weights)
        if active_d is not None:
            rc.set_active_cells(active_d)
    configure()
    analysed = None
    if not args.no_analyse and (args.analyse or (args.config == 4 and atm.line is None) or args.active):
        analysed = rc.analyse_atmosphere()   # empty-cell scan; switches the distance-field march on when > 2/3 is empty
    seg = rc.count_segments()
    l2_gather_gbs = rc.probe_gather_bandwidth(64)      # L2 -> SM ceiling of the gather pattern (64 MB region)
    tma_bulk_gbs = rc.probe_bulk_copy_bandwidth(64)    # the same pattern through TMA bulk copies + shared memory
    nincl = 1 if atm.mu is None else len(atm.mu)
    segl_job = sum(seg) * nlambda_job * nincl          # the whole job's units per step (every rank has the same geometry)
    J = rc.solve_J()
    walked = rc.count_walked(out=J)                    # segments actually integrated (early exit, sparsity, free-space jumps)

    def step():
        rc.solve_J(out=J)
        if world > 1 and atm.accumulate:
            sharding.allreduce_jbar(J)                  # NCCL all-reduce of the ranks' weighted partial sums
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    rc.set_timing(args.steps)

    def barrier():
        if world > 1:
            dist.barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize(); barrier()
    clocks = sampler.stop()
    ms = torch.tensor([e0.elapsed_time(e1)], device=dev)
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_total = float(ms.item())
    st = rc.get_stats()
    launches = (st.kernel_launches + (1 if world > 1 and atm.accumulate else 0)) * args.steps
    rc.set_timing(0)

    # end to end through the C ABI with HOST buffers: H2D of the inputs, solve, D2H of J, every step
    out_h = torch.empty(J.shape, dtype=torch.float32, pin_memory=True)
    if atm.line is not None:
        h2d_bytes = int(atm.line.nbytes)

        def e2e_step():
            rc.solve_J_line_host(line_h, atm.xl, out_h)
    else:
        h2d_bytes = int(2 * atm.chi.nbytes)

        def e2e_step():
            rc.solve_J_host(chi_h, eta_h, out_h)
            if world > 1 and atm.accumulate:
                Jd = out_h.to(dev, non_blocking=True)
                sharding.allreduce_jbar(Jd)
                out_h.copy_(Jd)
    e2e_step()
    configure()      # the host path may have moved the atmosphere inside the workspace: boundary, weights, flags again
    e2e_step()
    barrier(); torch.cuda.synchronize()
    e0.record()
    for _ in range(e2e_steps):
        e2e_step()
    e1.record()
    torch.cuda.synchronize(); barrier()
    ms2 = torch.tensor([e0.elapsed_time(e1)], device=dev)
    if world > 1:
        dist.all_reduce(ms2, op=dist.ReduceOp.MAX)
    e2e_ms = float(ms2.item()) / e2e_steps
    same = bool(torch.equal(out_h, J.cpu()))

    if rank == 0:
        ms_step = ms_total / args.steps
        value = segl_job / (ms_step * 1e-3)
        # dominant kernel: the march+merge launch of the heaviest cascade (of this rank's wavelength block)
        ms_march = [st.ms_march[i] for i in range(atm.ncascades)]
        dom = int(np.argmax(ms_march))
        casc_bytes = 2 * 4 * atm.nx * atm.ny * atm.nlambda * nincl  # read merged cascade i+1, write cascade i
        # chi+eta gather: 8 B per segment-wavelength; where segments are left out by construction (flagged probes
        # only, free-space jumps) the roofline counts the segments the launch really integrates, `value` stays geometric
        sparse_run = atm.active is not None or (analysed is not None and bool(analysed.sparse_march))
        seg_dom = walked[dom] if sparse_run else seg[dom]
        alg_bytes = 8 * seg_dom * atm.nlambda + casc_bytes
        ach = alg_bytes / (ms_march[dom] * 1e-3) / 1e9
        mode = ("line" if atm.line is not None else "flat") + (f"_incl{nincl}" if nincl > 1 else "") + ("_fix" if args.bilinear_fix else "")
        cap = NCU_CAPTURES.get((mode, args.config, dom)) if world == 1 and not args.active and not args.tune else None
        stale_cap = None
        if cap is not None and kernel_text_sha(cap["kernel"]) != cap["sha"]:
            stale_cap, cap = cap, None      # a capture of an earlier version of the kernel: reported, not used
        dram = None if cap is None else cap["dram_bytes"]
        mufu_per_unit = 3 if atm.line is not None else 1  # line mode: ex2 (profile), rcp (eta/chi), ex2 (transmittance)
        sfu_peak = SM_COUNT * MUFU_PER_CLK_SM * sm_max_mhz * 1e6 / mufu_per_unit
        ach_alu = seg_dom * atm.nlambda * nincl / (ms_march[dom] * 1e-3)
        mufu_bound = ach_alu / sfu_peak > ach / l2_gather_gbs
        l2_meas = None if cap is None else cap["l2_to_sm_bytes"] / (ms_march[dom] * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if world > 1 else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload, "seg_lambda_per_step": segl_job, "lambda_batch": st.lambda_batch,
                       "l2": ("inputs (chi+eta %.0f MB per rank) larger than L2" % (h2d_bytes / 1e6)) if atm.line is None else
                             "line parameters (%.0f MB) fit L2; merged cascades (2 x %.0f MB per cascade) stream through it"
                             % (h2d_bytes / 1e6, 4 * atm.nx * atm.ny * atm.nlambda / 1e6),
                       "parallelism": (f"1 GPU" if world == 1 else
                                       f"{world} ranks x {atm.nlambda} of the {nlambda_job} wavelengths of one atmosphere (contiguous blocks, "
                                       f"no exchange during the solve" + ("; Jbar: one NCCL all-reduce of nx ny floats per step)" if atm.accumulate else ")")),
                       "early_exit": True,
                       "segments_geometric_per_wavelength": sum(seg), "segments_walked_per_wavelength": sum(walked),
                       "walked_fraction": sum(walked) / max(sum(seg), 1),
                       "empty_cell_fraction": None if analysed is None else analysed.empty_cells / (atm.nx * atm.ny),
                       "distance_field_march": None if analysed is None else bool(analysed.sparse_march),
                       "hit_lists": None if analysed is None else bool(analysed.sparse_lists),
                       "hit_list_bytes": None if analysed is None else int(analysed.sparse_list_bytes),
                       "active_cell_fraction": None if atm.active is None else atm.meta["active_fraction"]},
            "solve_ms": ms_step,
            # The binding roof of the dominant kernel.  HBM is NOT it: the gathers (8 B per segment-wavelength, each cell
            # crossed ~5 x 4^i times per cascade) are served by L2 and L1, DRAM sees 0.4 % of them (the `hbm` object).
            # bound "l2": algorithmic gather bytes over the L2 -> SM gather ceiling measured in this very run by
            # rc_probe_gather_bandwidth (the march's access pattern alone: random 1 KB warp-wide runs, LDG.256, 48 warps/SM,
            # 64 MB L2-resident region) - an achieved figure of a micro-kernel, not a data-sheet peak (the guides give none);
            # part of the algorithmic bytes is served by L1 (the children of a direction group share cells), which is why
            # `l2_measured` (ncu: bytes that crossed L2 -> SM / this run's launch time) is reported beside it.
            # bound "alu": the MUFU pipe (16 ex2/clk/SM), where one gather feeds several exponentials (inclinations, line).
            "roofline": ({"bound": "alu", "pipe": f"MUFU, 16/clk/SM x 148 SMs at sm_max_mhz, {mufu_per_unit} per unit",
                          "kernel": f"march_kernel<{st.lambda_batch * nincl}> cascade {dom}", "achieved": ach_alu, "peak": sfu_peak,
                          "unit": UNIT, "frac": ach_alu / sfu_peak} if mufu_bound else
                         {"bound": "l2", "kernel": f"march_kernel<{st.lambda_batch}> cascade {dom}", "achieved": ach, "peak": l2_gather_gbs,
                          "unit": "GB/s", "frac": ach / l2_gather_gbs,
                          "peak_source": "measured in this run by rc_probe_gather_bandwidth(64 MB): the march's gather pattern alone from "
                                         "L2; achieved by a micro-kernel, not a hardware peak",
                          "l2_measured": {"achieved": l2_meas, "frac": None if l2_meas is None else l2_meas / l2_gather_gbs,
                                          "ncu_lts_t_sectors_pct": None if cap is None else cap.get("lts_pct"),
                                          "note": "ncu l1tex__m_xbar2l1tex_read_bytes.sum of the committed capture / this run's launch time"}}),
            "roofline_l2_probe": {"bound": "l2", "achieved": ach, "peak": l2_gather_gbs, "unit": "GB/s", "frac": ach / l2_gather_gbs,
                                  "peak_source": "achieved by a micro-kernel (rc_probe_gather_bandwidth(64 MB), this run: random 1 KB "
                                                 "warp-wide runs, LDG.256, 48 warps/SM, region L2-resident), not a hardware peak",
                                  "ncu_lts_t_sectors_pct": None if cap is None else cap.get("lts_pct"),
                                  "tma_bulk_copy_gbs_same_pattern": tma_bulk_gbs},
            "roofline_alu": {"bound": "alu", "pipe": f"MUFU, 16/clk/SM x 148 SMs at sm_max_mhz, {mufu_per_unit} per unit", "achieved": ach_alu,
                             "peak": sfu_peak, "unit": UNIT, "frac": ach_alu / sfu_peak},
            "hbm": {"peak": hbm_peak, "peak_source": peak_src, "unit": "GB/s", "algorithmic_bytes": alg_bytes,
                    "algorithmic_over_hbm": ach / hbm_peak,
                    "solve_algorithmic_over_hbm": (8 * sum(seg) * atm.nlambda * world + 2 * casc_bytes * world * atm.ncascades) / (ms_step * 1e-3) / 1e9 / hbm_peak,
                    "traffic": dram, "dram_gbs": None if dram is None else dram / (ms_march[dom] * 1e-3) / 1e9,
                    "frac": None if dram is None else dram / (ms_march[dom] * 1e-3) / 1e9 / hbm_peak,
                    "traffic_source": ("no ncu capture of this mode, config and launch plan is committed" if cap is None else cap["source"]),
                    "note": "traffic = dram__bytes_read.sum + dram__bytes_write.sum of the dominant launch (ncu --set full); "
                            "algorithmic = 8 B per segment-wavelength + merged cascade read/write"},
            "ms_per_launch": ms_march[dom],
            "per_cascade_ms": {"march": ms_march, "pack": [st.ms_pack[i] for i in range(atm.ncascades)]},
            "segments_per_cascade": seg, "segments_walked_per_cascade": walked,
            "e2e": {"value": segl_job / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps,
                    "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": int(out_h.numel() * 4),
                    "call": "rc_solve_J_line_host" if atm.line is not None else "rc_solve_J_host",
                    "matches_device_path": same},
            "gpu_launches": launches, "clocks": clocks,
        }
        line["roofline"]["traffic"] = dram
        # the tier's own figure beside `frac`: algorithmic bytes (8 B per segment-wavelength the launch integrates + the merged
        # cascade read and written) / launch time / the measured HBM copy peak; above 1 because L2 and L1 serve the gathers
        line["roofline"]["algorithmic_over_hbm"] = ach / hbm_peak
        line["roofline"]["hbm_peak_gbs"] = hbm_peak
        if cap is not None:
            line["hbm"]["capture"] = {k: cap[k] for k in ("kernel", "sha", "commit", "capture_ms")}
        if stale_cap is not None:
            line["hbm"]["stale_capture"] = {**{k: stale_cap[k] for k in ("kernel", "sha", "commit", "capture_ms", "dram_bytes")},
                                            "head_sha": kernel_text_sha(stale_cap["kernel"]),
                                            "note": "the kernel's source changed after this capture: no traffic or derived fraction is reported from it"}
        # `value` counts GEOMETRIC segments - every in-box cell segment of every ray, whether or not the march had to
        # integrate it (early exit of opaque rays, unflagged probes, jumps over free space); `value_walked` counts only
        # the segments the kernels really integrated.  They differ by `walked_fraction`; dense runs: ~1.
        wf = sum(walked) / max(sum(seg), 1)
        line["value_kind"] = "geometric segments x wavelengths / time"
        line["value_walked"] = value * wf
        line["e2e"]["value_walked"] = line["e2e"]["value"] * wf
        if world == 1 and not args.no_cpu_baseline:
            nwin = 3
            segl, secs, cores = oracle_sample(atm, nwin)
            line["cpu_baseline"] = {"value": segl / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{nwin} windows of 8x8 cells x {atm.nlambda} wavelengths, "
                                              f"{segl:.3e} segment-wavelengths in {secs:.1f} s"}
            if args.cpu_baseline_whole:
                from oracle import rc_oracle
                t0 = time.perf_counter()
                ref = rc_oracle.solve_atmosphere(atm)
                secs = time.perf_counter() - t0
                Jo = ref["Jbar"] if atm.accumulate else ref["J"]
                Jg = J.cpu().numpy().astype(np.float64)
                m = Jo > 1e-6 * Jo.max(axis=(0, 1), keepdims=True) if Jo.ndim == 3 else Jo > 1e-6 * Jo.max()
                line["cpu_baseline"]["whole_solve"] = {"seconds": secs, "value": segl_job / secs, "unit": UNIT,
                                                       "gpu_max_rel_err_all_cells": float(np.max(np.abs(Jg[m] - Jo[m]) / Jo[m]))}
        rc.close()
        rc = None
        if secondary_wanted(args, world):
            del J, out_h
            torch.cuda.empty_cache()
            line["secondary"] = secondary_runs()
        print(json.dumps(line))
    if rc is not None:
        rc.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
