#!/usr/bin/env python
"""bench.py -- SFFT difference images/s at 4088^2 (L=11, DK=2), and % of HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" = one pass of the whole hot path (sfft_build_system,
sfft_solve, sfft_subtract) over ONE synthetic 4088 x 4088 science/template pair, L=11, DK=2, DB=2
(BASELINE.json configs[2], the configuration `metric` is quoted on).  Nothing is reused between
steps.  `value` is timed with the inputs resident in HBM; `e2e` is the same metric through
sfft_difference_host with pinned HOST buffers (H2D of S and R, D2H of D and the coefficients inside
the timed region).  N > 1: replicas only -- every rank runs the same
independent problem on its own GPU, no data-path collective; value = N / max-over-ranks step time.

Extra objects on the JSON line: `roofline` (dominant kernel, timed live with CUDA events through
the library's per-launch timers on the plan's stream), `path_roofline` (the metric's "% of HBM
roofline": 34 r of algorithmic bytes over the a1+a2+a3+a5 time), `stages_ms`, `kernels_ms`,
`batched` (configs[3]: template-side work once, per-science-image throughput), `cross_convolve`
(f2: both PSF cross-convolutions of the pair, device time, 16 r of algorithmic bytes), `decorrelate`
(f1: decorrelation stamp build + one application), `align` (f3: affine resampling of one
frame and its mask), `constant_ratio` (f4: the step under the constant-photometric-ratio constraint), `stamp_mode`
(f4: the path on a 1000 x 1000 cut-out), `cpu_baseline`
(the oracle on this box's host cores, bounded sample), `clocks`.

--impl reference times the CPU oracle (oracle/, as it stands) on the same config and metric.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "sfft_difference_images_per_sec_4088sq_L11_DK2"
UNIT = "images/s"
WORKLOAD = dict(workload="BASELINE.json configs[2]: single 4088x4088 fp64 pair, 60k stars, L=11, DK=2, DB=2 (n=732)",
                nx=4088, ny=4088, L=11, DK=2, DB=2, n=732)
NOMINAL_HBM_GBS = 7700.0
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            d = json.loads(f.read_text())
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def algorithmic_bytes(nx, ny, DK, NK):
    """SURVEY.md 8(d) / DESIGN.md: bytes the canonical 2-D-FFT formulation must move, in units of
    r = nx*ny*8 (one FP64 image; a half spectrum is ~r).  Per kernel and per stage group."""
    r = nx * ny * 8.0
    k = {
        "row_fwd_R": (1 + (DK + 1)) * r,        # read R, write DK+1 row-transformed intermediates
        "col_fwd_R": ((DK + 1) + NK) * r,       # read them, write NK spectra
        "row_fwd_S": 2 * r, "col_fwd_S": 2 * r,
        "lagcol_omega": NK * r,                 # NK template spectra, once
        "lagcol_theta": (NK + 1) * r,           # + the science spectrum
        "col_inv": (NK + 1) * r,                # NK spectra in, one intermediate out
        "row_inv": 3 * r,                       # intermediate + S in, D out
    }
    path = (1 + 2 * (DK + 1) + NK) * r + 4 * r + (NK + 1) * r + (NK + 4) * r   # 13 + 4 + 7 + 10 = 34 r at DK=2
    return k, path


class ClockSampler:
    """Samples SM clock, power and throttle reasons of one GPU every 100 ms (NVML) while running."""

    def __init__(self, index):
        self.index, self.samples, self.reasons, self._stop, self._t = index, [], set(), threading.Event(), None
        self.max_mhz, self.ok = None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def _loop(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop.is_set():
            try:
                self.samples.append((int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)),
                                     nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0))
                try:
                    bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for b, nm in names.items():
                    if bits & b:
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop.wait(0.1)

    def start(self):
        if self.ok:
            self._t = threading.Thread(target=self._loop, daemon=True)
            self._t.start()

    def stop(self):
        if self._t:
            self._stop.set()
            self._t.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        mhz = sorted(s[0] for s in self.samples)
        return {"sm_mhz": mhz[len(mhz) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "power_w_max": round(max(s[1] for s in self.samples), 1), "samples": len(mhz)}


# ------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------
def oracle_step(S, R, L, DK, DB):
    """The oracle's whole path (direct-sum build_system, textbook Cholesky, real-space subtract) on the full pair,
    as it stands.  Returns seconds of (build, solve, subtract)."""
    import oracle
    t0 = time.perf_counter()
    G, h = oracle.build_system(S, R, None, L, DK, DB)
    t1 = time.perf_counter()
    c = oracle.solve(G, h)
    t2 = time.perf_counter()
    oracle.subtract(S, R, L, DK, DB, c)
    t3 = time.perf_counter()
    return t1 - t0, t2 - t1, t3 - t2


def config_dict(cfg, world):
    """The `config` object of the JSON line: identical for both arms (the driver compares them)."""
    return dict(cfg, parallelism=f"replicas x{world}" if world > 1 else "single GPU",
                l2="inputs larger than L2: S, R 134 MB each, ~5 GB streamed per step vs 126 MB L2; no flush")


def cpu_baseline(S, R, cfg):
    """One FULL oracle step on the same pair (about 15 s on 16 cores: the bounded sample is the whole workload)."""
    import oracle
    tb, ts, tsub = oracle_step(S, R, cfg["L"], cfg["DK"], cfg["DB"])
    full = tb + ts + tsub
    return {"value": 1.0 / full, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"one full step (oracle build_system {tb:.2f} s + solve {ts:.2f} s + subtract {tsub:.2f} s) on the "
                      f"same 4088x4088 pair; nothing scaled",
            "seconds_full_frame": round(full, 3)}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config/metric, the full step every step; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    import oracle
    from paper_2509_18544_b200 import starfield
    cfg = dict(WORKLOAD)
    pair = starfield.make_pair(2)
    S, R = pair["S"], pair["R"]
    for _ in range(args.warmup):
        oracle_step(S, R, cfg["L"], cfg["DK"], cfg["DB"])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(S, R, cfg["L"], cfg["DK"], cfg["DB"])
    sec = (time.perf_counter() - t0) / args.steps
    val = 1.0 / sec
    sample = f"each step = the full oracle build_system+solve+subtract on the 4088x4088 pair ({sec:.2f} s measured); nothing scaled"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, int(os.environ.get("WORLD_SIZE", str(args.gpus)))),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------
# multi-GPU host logic: replicas only -- no data-path collective
# ------------------------------------------------------------------------------------------
def max_over_ranks(values, device):
    """Element-wise MAX over all ranks of a list of floats (device times); identity when not distributed."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def replica_throughput(world, ms_per_step):
    """Whole-job images/s of `world` independent replicas that each finish one image per step."""
    return world * 1e3 / ms_per_step


def ncu_traffic(kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture (profiles/ncu_traffic.json).  The
    capture is stamped with the hash of the kernel sources it was taken from; a different tree gets null, not a stale
    number."""
    f = ROOT / "profiles" / "ncu_traffic.json"
    try:
        from paper_2509_18544_b200.build import source_hash
        d = json.loads(f.read_text())
        if d.get("csrc_sha256") != source_hash():
            return None
        return d["kernels"][kernel]["dram_bytes_per_launch"]
    except Exception:
        return None


# ------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2509_18544_b200 import SfftPlan, sfft, starfield

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libsfft has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = dict(WORKLOAD)
    nx, ny, L, DK, DB = cfg["nx"], cfg["ny"], cfg["L"], cfg["DK"], cfg["DB"]
    NK = (DK + 1) * (DK + 2) // 2
    pair = starfield.make_pair(2)                      # same seeded pair on every replica
    S_np, R_np = pair["S"], pair["R"]
    dS, dR = torch.from_numpy(S_np).cuda(), torch.from_numpy(R_np).cuda()
    D = torch.empty_like(dS)
    coeffs = torch.empty(cfg["n"], dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    plan = SfftPlan(nx, ny, L, DK, DB, stream=stream)

    def step():
        plan.build_system(dS, dR)
        plan.solve()
        plan.subtract(D, coeffs)

    # ---- headline: K steps, device-resident inputs --------------------------------------------
    for _ in range(max(args.warmup, 3)):
        step()
    plan.sync_status()
    clocks = ClockSampler(local)
    barrier()
    clocks.start()
    n0 = plan.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = plan.launch_count - n0
    plan.sync_status()

    # ---- e2e: host buffers through sfft_difference_host ---------------------------------------
    hS, hR = torch.from_numpy(S_np).pin_memory(), torch.from_numpy(R_np).pin_memory()
    hD = torch.empty((ny, nx), dtype=torch.float64).pin_memory()
    hc = torch.empty(cfg["n"], dtype=torch.float64).pin_memory()
    for _ in range(2):
        plan.difference_host(hS, hR, None, hD, hc)
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(stream)
    for _ in range(args.steps):
        plan.difference_host(hS, hR, None, hD, hc)
    f1.record(stream)
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    clk = clocks.stop()

    ms_total, ms_e2e = max_over_ranks([ms_total, ms_e2e], "cuda")
    ms_step = ms_total / args.steps
    value = replica_throughput(world, ms_step)
    e2e_value = replica_throughput(world, ms_e2e / args.steps)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, world),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(2 * nx * ny * 8),
                    "d2h_bytes_per_step": int(nx * ny * 8 + cfg["n"] * 8), "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": int(launches), "clocks": clk, "library": sfft.version(),
            "workspace_gb": round(plan.workspace_bytes / 1e9, 3)}

    if rank == 0:
        line.update(detail_rank0(plan, step, args, cfg, NK, dS, dR, pair, torch))
        if world == 1:
            line["cpu_baseline"] = cpu_baseline(S_np, R_np, cfg)
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def detail_rank0(plan, step, args, cfg, NK, dS, dR, pair, torch):
    """Per-stage and per-kernel times (live, CUDA events on the plan's stream), the rooflines, the
    batched variant and the measured FP64 rates.  Runs after the headline region, on rank 0."""
    from paper_2509_18544_b200 import sfft, starfield
    nx, ny, DK = cfg["nx"], cfg["ny"], cfg["DK"]
    peak, peak_src = measured_peaks()
    kbytes, path_bytes = algorithmic_bytes(nx, ny, DK, NK)
    K = max(3, min(args.steps, 10))
    ws_fp64 = plan.workspace_bytes          # before the host-batch call adds its staging buffers

    # per stage
    stages = {}
    for _ in range(K):
        plan.enable_timings(1)
        step()
        for k, v in plan.get_timings().items():
            stages.setdefault(k, []).append(v)
    stages = {k: float(np.median(v)) for k, v in stages.items()}
    # per kernel launch
    ksum, kcnt = {}, {}
    for _ in range(K):
        plan.enable_timings(2)
        step()
        per = {}
        for name, ms in plan.kernel_timings():
            per[name] = per.get(name, 0.0) + ms
            kcnt[name] = kcnt.get(name, 0) + 1
        for name, ms in per.items():
            ksum.setdefault(name, []).append(ms)
    plan.enable_timings(0)
    kernels = {k: float(np.median(v)) for k, v in ksum.items()}          # ms per step, all launches of that kernel
    kcnt = {k: v // K for k, v in kcnt.items()}

    out = {"stages_ms": {k: round(v, 4) for k, v in stages.items()},
           "kernels_ms": {k: round(v, 4) for k, v in sorted(kernels.items(), key=lambda kv: -kv[1])},
           "kernel_launches_per_step": kcnt}

    # FP64 rates of this box (the ALU roofline of a2 and a4)
    try:
        out["fp64_probe_tflops"] = {"dfma": round(sfft.probe_fp64(0), 2), "dmma_m8n8k4": round(sfft.probe_fp64(1), 2)}
    except Exception as e:  # pragma: no cover
        out["fp64_probe_tflops"] = {"error": str(e)}
    # dominant kernel among those that stream images/spectra.  The Omega lag pass is bound by FP64 instruction issue, not
    # by HBM (21 pairs x (16 products + 16-point DFT + 21 folded lags) per 16 spectrum elements =
    # 308/16 FP64 instructions per element and pair, counted as 2 flop each against the probed DFMA rate): if it is the
    # dominant kernel the line says "alu"; the dominant HBM-bound kernel is reported beside it either way.
    hbm_kernels = {k: v for k, v in kernels.items() if k in kbytes}
    dom = max(hbm_kernels, key=hbm_kernels.get)

    def hbm_line(kn):
        per_launch_ms = kernels[kn] / kcnt[kn]
        ach = kbytes[kn] / (per_launch_ms * 1e-3) / 1e9
        return {"kernel": kn, "bound": "hbm", "achieved": round(ach, 1), "peak": peak, "unit": "GB/s",
                "frac": round(ach / peak, 4), "traffic": ncu_traffic(kn), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": kbytes[kn], "ms_per_launch": round(per_launch_ms, 4),
                "share_of_step": round(kernels[kn] / sum(kernels.values()), 3)}
    if dom == "lagcol_omega" and "dfma" in out["fp64_probe_tflops"]:
        npair = NK * (NK + 1) // 2
        flop = npair * 4096.0 * 2049.0 * (64 + 160 + 84) / 16.0 * 2.0
        ms_l = kernels[dom] / kcnt[dom]
        pk = out["fp64_probe_tflops"]["dfma"]
        out["roofline"] = {"kernel": dom, "bound": "alu", "achieved": round(flop / ms_l / 1e9, 2), "peak": pk, "unit": "TFLOP/s",
                           "frac": round(flop / ms_l / 1e9 / pk, 4), "traffic": ncu_traffic(dom),
                           "peak_source": "measured (sfft_probe_fp64: register-resident DFMA loop on every SM)",
                           "algorithmic_flop_per_launch": flop, "ms_per_launch": round(ms_l, 4),
                           "share_of_step": round(kernels[dom] / sum(kernels.values()), 3),
                           "hbm_view": hbm_line(dom)}
        rest = {k: v for k, v in hbm_kernels.items() if k != dom}
        out["roofline_hbm_dominant"] = hbm_line(max(rest, key=rest.get))
    else:
        out["roofline"] = hbm_line(dom)
    out["kernel_rooflines"] = {k: {"ms": round(kernels[k] / kcnt[k], 4), "frac_of_measured_hbm": round(kbytes[k] / (kernels[k] / kcnt[k]) / 1e6 / peak, 4)}
                               for k in hbm_kernels}
    t_path = sum(stages[k] for k in ("a1_template", "a1_science", "a2_omega", "a2_theta", "a3_gather", "a5_subtract"))
    out["path_roofline"] = {"what": "a1+a2+a3+a5 (BASELINE.json target: >= 0.60)", "algorithmic_bytes": path_bytes,
                            "ms": round(t_path, 4), "achieved_gbs": round(path_bytes / t_path / 1e6, 1),
                            "frac_of_measured": round(path_bytes / t_path / 1e6 / peak, 4),
                            "frac_of_nominal_7.7TBs": round(path_bytes / t_path / 1e6 / NOMINAL_HBM_GBS, 4),
                            "a4_ms": round(stages["a4_factor"] + stages["a4_solve"], 4)}
    # f2: cross-convolution S (*) psf_R, R (*) psf_S with L x L stamps on the same plan.
    # Algorithmic bytes per convolution: image 1 r + row intermediate 1 r written and read + spectrum 1 r written and
    # read + inverse intermediate 1 r written and read + output 1 r = 8 r.  The oracle is timed on a bounded crop.
    try:
        import oracle
        import time as _time
        L = cfg["L"]
        w = (L - 1) // 2
        yy, xx = np.mgrid[-w:w + 1, -w:w + 1]
        psfs = []
        for sg in (1.0, 0.85):
            st = np.exp(-0.5 * (xx * xx + yy * yy) / (sg * sg)); psfs.append(st / st.sum())
        dpS, dpR = (torch.from_numpy(a).cuda() for a in psfs)
        oS, oR = torch.empty_like(dS), torch.empty_like(dR)
        stream = torch.cuda.current_stream()
        for _ in range(3):
            plan.convolve_stamp(dS, dpR, oS); plan.convolve_stamp(dR, dpS, oR)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            plan.convolve_stamp(dS, dpR, oS); plan.convolve_stamp(dR, dpS, oR)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / K
        crop = 1022 if ny >= 1022 and nx >= 1022 else min(nx, ny)
        t0 = _time.perf_counter()
        ref = oracle.convolve_stamp(pair["S"][:crop, :crop], psfs[1])
        t_cpu = _time.perf_counter() - t0
        got = oS[:crop - w, :crop - w].cpu().numpy()[w:, w:]          # interior of the crop: same taps on both sides
        err = float(np.max(np.abs(got - ref[w:crop - w, w:crop - w])))
        r = nx * ny * 8.0
        out["cross_convolve"] = {"workload": f"S (*) psf_R and R (*) psf_S, {L} x {L} stamps, {nx} x {ny} (PAPER.md:86)",
                                 "ms": round(ms, 4), "pairs_per_s": round(1e3 / ms, 1),
                                 "algorithmic_bytes": 16 * r, "achieved_gbs": round(16 * r / ms / 1e6, 1),
                                 "frac_of_measured_hbm": round(16 * r / ms / 1e6 / peak, 4),
                                 "oracle_check_max_abs_err": err,
                                 "cpu_oracle": {"seconds_sample": round(t_cpu, 3), "sample": f"one convolution of the top-left {crop} x {crop} crop",
                                                "pairs_per_s_full_frame_est": round(1.0 / (2 * t_cpu * (nx * ny) / (crop * crop)), 4)}}
    except Exception as ex:  # pragma: no cover
        out["cross_convolve"] = {"error": str(ex)}

    # f3: Lanczos-3 resampling of the template under a small rotation + shift (2 r of
    # algorithmic bytes: the frame read once, written once) and the nearest-neighbour mask.  Oracle check on the
    # top-left crop (same pixel coordinates, so every pixel whose footprint lies inside the crop must agree).
    try:
        from oracle import alignment as _al
        cx, cy, th = (nx - 1) / 2.0, (ny - 1) / 2.0, 2e-4
        co, si = float(np.cos(th)), float(np.sin(th))
        Maff = [co, -si, cx - co * cx + si * cy + 0.37, si, co, cy - si * cx - co * cy - 0.21]
        oA = torch.empty_like(dR)
        dM = (torch.rand((ny, nx), device="cuda") > 0.02).to(torch.uint8)
        oM = torch.empty_like(dM)
        res = {}
        for name, fn in (("lanczos3", lambda: plan.resample_affine(dR, Maff, 3, float("nan"), oA)),
                         ("bilinear", lambda: plan.resample_affine(dR, Maff, 1, float("nan"), oA)),
                         ("mask_nearest", lambda: plan.resample_affine_mask(dM, Maff, 0, oM))):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            stream = torch.cuda.current_stream()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(K):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            res[name] = e0.elapsed_time(e1) / K
        plan.resample_affine(dR, Maff, 3, float("nan"), oA)
        crop = 1022 if ny >= 1022 and nx >= 1022 else min(nx, ny)
        ref = _al.resample_affine(pair["R"][:crop, :crop], Maff, _al.LANCZOS3, np.nan)
        got = oA[:crop, :crop].cpu().numpy()
        okm = ~np.isnan(ref) & ~np.isnan(got)
        r = nx * ny * 8.0
        out["align"] = {"workload": f"affine resampling of one {nx} x {ny} frame, rotation 2e-4 rad + sub-pixel shift (PAPER.md:85)",
                        "lanczos3_ms": round(res["lanczos3"], 4), "bilinear_ms": round(res["bilinear"], 4),
                        "mask_nearest_ms": round(res["mask_nearest"], 4),
                        "lanczos3_achieved_gbs": round(2 * r / res["lanczos3"] / 1e6, 1),
                        "lanczos3_frac_of_measured_hbm": round(2 * r / res["lanczos3"] / 1e6 / peak, 4),
                        "bilinear_frac_of_measured_hbm": round(2 * r / res["bilinear"] / 1e6 / peak, 4),
                        "oracle_check_pixels": int(okm.sum()),
                        "oracle_check_max_abs_err": float(np.max(np.abs(got[okm] - ref[okm])))}
    except Exception as ex:  # pragma: no cover
        out["align"] = {"error": str(ex)}

    # f1: the decorrelation kernel from a local kernel stamp and the two PSF stamps on an
    # N = 64 grid (sfft_decorrelation_stamp synchronises: host clock), then applied to a frame (8 r, like one
    # cross-convolution).  K is a fixed synthetic stamp so that the oracle sees no CUDA-path value.
    try:
        import oracle
        from oracle import decorrelation as _deco
        import time as _time
        L = cfg["L"]
        w = (L - 1) // 2
        yy, xx = np.mgrid[-w:w + 1, -w:w + 1]

        def _g(sg, dx=0.0):
            st = np.exp(-0.5 * ((xx - dx) ** 2 + yy * yy) / (sg * sg)); return st / st.sum()
        Kst, pS, pR = 1.05 * _g(0.6, 0.1), _g(1.0), _g(0.85)
        vS, vR, Ng = 64.0, 64.0 / 9.0, 64
        dK, dpS, dpR = (torch.from_numpy(a).cuda() for a in (Kst, pS, pR))
        dW = torch.empty((L, L), dtype=torch.float64, device="cuda")
        oW = torch.empty_like(dS)
        for _ in range(3):
            plan.decorrelation_stamp(dK, dpS, dpR, vS, vR, Ng, dW)
            plan.convolve_stamp(dS, dW, oW)
        torch.cuda.synchronize()
        t0 = _time.perf_counter()
        for _ in range(K):
            plan.decorrelation_stamp(dK, dpS, dpR, vS, vR, Ng, dW)
        ms_build = (_time.perf_counter() - t0) * 1e3 / K
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            plan.convolve_stamp(dS, dW, oW)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_apply = e0.elapsed_time(e1) / K
        W0 = _deco.decorrelation_stamp(Kst, pS, pR, vS, vR, Ng, L)
        crop = 1022 if ny >= 1022 and nx >= 1022 else min(nx, ny)
        ref = oracle.convolve_stamp(pair["S"][:crop, :crop], W0)
        got = oW[:crop - w, :crop - w].cpu().numpy()[w:, w:]
        r = nx * ny * 8.0
        out["decorrelate"] = {"workload": f"decorrelation stamp {L} x {L} on a {Ng} x {Ng} grid, applied to one {nx} x {ny} frame (PAPER.md:88)",
                              "stamp_build_ms_host_clock": round(ms_build, 4), "apply_ms": round(ms_apply, 4),
                              "apply_achieved_gbs": round(8 * r / ms_apply / 1e6, 1),
                              "apply_frac_of_measured_hbm": round(8 * r / ms_apply / 1e6 / peak, 4),
                              "oracle_check_stamp_max_abs_err": float(np.max(np.abs(dW.cpu().numpy() - W0))),
                              "oracle_check_image_max_abs_err": float(np.max(np.abs(got - ref[w:crop - w, w:crop - w])))}
    except Exception as ex:  # pragma: no cover
        out["decorrelate"] = {"error": str(ex)}

    # f4 variant: the same step with the constant-photometric-ratio solve (NK - 1 more triangular solves).
    try:
        oD = torch.empty_like(dS); oc = torch.empty(plan.n, dtype=torch.float64, device="cuda")

        def rstep():
            plan.build_system(dS, dR); plan.solve(); plan.subtract(oD, oc)
        plan.set_constant_ratio(True)            # plan mode: the auxiliary solves run behind the factor, beside the science side
        for _ in range(3):
            rstep()
        plan.sync_status()
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            rstep()
        e1.record(stream)
        torch.cuda.synchronize()
        plan.sync_status()
        rms_ = e0.elapsed_time(e1) / K
        LLb = cfg["L"] ** 2
        sums = [float(oc[t * LLb:(t + 1) * LLb].sum()) for t in range(NK)]
        plan.set_constant_ratio(False)
        out["constant_ratio"] = {"workload": "the headline step in the sfft_set_constant_ratio(1) plan mode",
                                 "ms_per_step": round(rms_, 4), "images_per_s": round(1e3 / rms_, 1),
                                 "tap_sums_per_term": sums}
        step()                                   # leave the plan with the free solution
    except Exception as ex:  # pragma: no cover
        plan.set_constant_ratio(False)
        out["constant_ratio"] = {"error": str(ex)}

    # f4: "decrease the processed stamp size ... down to a minimum size of 1000 x 1000 px": the same path
    # on a contiguous 1000 x 1000 cut-out of the pair (a second, small plan; same L, DK, DB).
    try:
        from paper_2509_18544_b200 import SfftPlan as _Plan
        sn = 1000
        y0, x0 = (ny - sn) // 2, (nx - sn) // 2
        cS, cR = dS[y0:y0 + sn, x0:x0 + sn].contiguous(), dR[y0:y0 + sn, x0:x0 + sn].contiguous()
        sp = _Plan(sn, sn, cfg["L"], cfg["DK"], cfg["DB"])
        cD = torch.empty_like(cS); cc = torch.empty(sp.n, dtype=torch.float64, device="cuda")
        def sstep():
            sp.build_system(cS, cR); sp.solve(); sp.subtract(cD, cc)
        for _ in range(3):
            sstep()
        sp.sync_status()
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            sstep()
        e1.record(stream)
        torch.cuda.synchronize()
        sp.sync_status()
        sms = e0.elapsed_time(e1) / K
        out["stamp_mode"] = {"workload": f"{sn} x {sn} cut-out of the same pair, L={cfg['L']}, DK={cfg['DK']}, DB={cfg['DB']} (PAPER.md:105)",
                             "ms_per_step": round(sms, 4), "stamps_per_s": round(1e3 / sms, 1),
                             "workspace_gb": round(sp.workspace_bytes / 1e9, 3)}
        sp.destroy()
    except Exception as ex:  # pragma: no cover
        out["stamp_mode"] = {"error": str(ex)}

    # batched variant (BASELINE.json configs[3]): template once, B science images
    B = args.batch
    if B > 0:
        tmpl = dict(pair)
        Ss = [dS] + [torch.from_numpy(starfield.make_batch_science(tmpl, b)).cuda() for b in range(1, min(B, 4))]
        S_list = [Ss[b % len(Ss)] for b in range(B)]          # B launches over 4 distinct seeded images
        D_list = [torch.empty_like(dS) for _ in range(min(B, 4))]
        D_arg = [D_list[b % len(D_list)] for b in range(B)]
        cb = torch.empty((B, cfg["n"]), dtype=torch.float64, device="cuda")
        stream = torch.cuda.current_stream()
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]

        def batch_once():
            e[0].record(stream)
            plan.set_template(dR)
            e[1].record(stream)
            plan.subtract_batch(S_list, D_arg, cb)
            e[2].record(stream)
            torch.cuda.synchronize()
            plan.sync_status()
            return e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2])
        batch_once()                                           # warm-up with the FULL batch (nothing is allocated after
        reps = [batch_once() for _ in range(5)]                # plan creation, but clocks and caches settle)
        t_t, t_b = float(np.median([a for a, _ in reps])), float(np.median([b for _, b in reps]))
        r = nx * ny * 8.0
        # per image: a1 of S 4 r, Theta (NK + 4)/4 r (four images share one pass over the NK template spectra), a5 (NK + 4) r
        per_img_bytes = (4 + (NK + 4) / 4.0 + (NK + 4)) * r + (13 + NK) * r / B
        out["batched"] = {"workload": f"BASELINE.json configs[3]: one template, B={B} science images "
                                      f"({len(Ss)} distinct seeded images cycled)",
                          "B": B, "repetitions": 5, "template_ms": round(t_t, 3), "per_image_ms": round(t_b / B, 4),
                          "per_image_ms_all_reps": [round(b / B, 4) for _, b in reps],
                          "images_per_s": round(B * 1e3 / (t_t + t_b), 1),
                          "frac_of_measured_hbm": round(per_img_bytes / ((t_t + t_b) / B) / 1e6 / peak, 4)}
        # the same batch in the constant-photometric-ratio plan mode (f4): auxiliary solves once per template
        try:
            plan.set_constant_ratio(True)
            batch_once()
            reps2 = [batch_once() for _ in range(5)]
            t_t2, t_b2 = float(np.median([a for a, _ in reps2])), float(np.median([b for _, b in reps2]))
            out["batched"]["constant_ratio_mode"] = {"template_ms": round(t_t2, 3), "per_image_ms": round(t_b2 / B, 4),
                                                     "images_per_s": round(B * 1e3 / (t_t2 + t_b2), 1)}
        except Exception as ex:  # pragma: no cover
            out["batched"]["constant_ratio_mode"] = {"error": str(ex)}
        plan.set_constant_ratio(False)

        # the same batch from HOST memory (sfft_difference_host_batch): template up once, three-deep upload | compute |
        # download pipeline; 4 pinned science buffers and 4 pinned outputs cycled
        try:
            hR = torch.from_numpy(pair["R"]).pin_memory()
            hS = [t_.cpu().pin_memory() for t_ in Ss]
            hD = [torch.empty((ny, nx), dtype=torch.float64).pin_memory() for _ in range(len(Ss))]
            hc = torch.empty((B, cfg["n"]), dtype=torch.float64).pin_memory()
            S_h = [hS[b % len(hS)] for b in range(B)]; D_h = [hD[b % len(hD)] for b in range(B)]
            plan.difference_host_batch(hR, S_h, None, D_h, hc)
            th = []
            for _ in range(3):
                t0 = time.perf_counter()
                plan.difference_host_batch(hR, S_h, None, D_h, hc)
                th.append((time.perf_counter() - t0) * 1e3)
            ms_h = float(np.median(th))
            out["batched"]["e2e"] = {"what": "sfft_difference_host_batch: R up once, per image 134 MB up and 134 MB down over PCIe inside the timed region (host clock, the call synchronises)",
                                     "ms_per_image": round(ms_h / B, 4), "images_per_s": round(B * 1e3 / ms_h, 1),
                                     "h2d_bytes_per_image": int(nx * ny * 8), "d2h_bytes_per_image": int(nx * ny * 8 + cfg["n"] * 8),
                                     "pcie_gbs_each_way": round(nx * ny * 8 / (ms_h / B) / 1e6, 1)}
            del hS, hD
        except Exception as ex:  # pragma: no cover
            out["batched"]["e2e"] = {"error": str(ex)}

    # f4, reduced-memory mode (SFFT_PLAN_FP32_SPECTRA): spectra stored as complex64 -- workspace and speed beside the FP64 plan
    try:
        from paper_2509_18544_b200 import SfftPlan as _Plan
        p32 = _Plan(nx, ny, cfg["L"], cfg["DK"], cfg["DB"], flags=_Plan.FP32_SPECTRA)
        o32 = torch.empty_like(dS)

        def step32():
            p32.build_system(dS, dR); p32.solve(); p32.subtract(o32)
        for _ in range(3):
            step32()
        p32.sync_status()
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            step32()
        e1.record(stream)
        torch.cuda.synchronize()
        ms32 = e0.elapsed_time(e1) / K
        p32.enable_timings(2); step32()
        k32 = {}
        for name, ms in p32.kernel_timings():
            k32[name] = k32.get(name, 0.0) + ms
        p32.enable_timings(0)
        rm = {"workload": "the headline step on a plan created with SFFT_PLAN_FP32_SPECTRA (complex64 spectra, FP64 arithmetic)",
              "ms_per_step": round(ms32, 4), "images_per_s": round(1e3 / ms32, 1), "workspace_gb": round(p32.workspace_bytes / 1e9, 3),
              "fp64_plan_workspace_gb": round(ws_fp64 / 1e9, 3),
              "kernels_ms": {k_: round(v_, 4) for k_, v_ in sorted(k32.items(), key=lambda kv: -kv[1])[:8]},
              "tolerances": "G, h 2e-7; kernel coefficients 1e-4; background 5e-3; D 3e-3 sigma (tests/test_gpu_fp32_spectra.py; measured 8e-8, 5e-8, 1e-5, 6e-4, 5e-4)"}
        if B > 0:
            cb32 = torch.empty((B, cfg["n"]), dtype=torch.float64, device="cuda")
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            tt = []
            for _ in range(4):
                ev[0].record(stream); p32.set_template(dR); ev[1].record(stream); p32.subtract_batch(S_list, D_arg, cb32); ev[2].record(stream)
                torch.cuda.synchronize()
                tt.append((ev[0].elapsed_time(ev[1]), ev[1].elapsed_time(ev[2])))
            tt = tt[1:]
            a_, b_ = float(np.median([x for x, _ in tt])), float(np.median([y for _, y in tt]))
            rm["batched"] = {"B": B, "template_ms": round(a_, 3), "per_image_ms": round(b_ / B, 4), "images_per_s": round(B * 1e3 / (a_ + b_), 1)}
        out["reduced_memory"] = rm
        p32.destroy()
        del o32
    except Exception as ex:  # pragma: no cover
        out["reduced_memory"] = {"error": str(ex)}

    # a4 on its own (BASELINE.json north_star: "FP64 tensor-pipe utilisation for the solve"): the factorisation of the
    # n = 732 system as sfft_set_template runs it (alone on the machine, stage timer), n^3/3 flop against the probed DMMA rate
    try:
        dmma = out.get("fp64_probe_tflops", {}).get("dmma_m8n8k4")
        fa = []
        for _ in range(5):
            plan.enable_timings(1)
            plan.set_template(dR)
            fa.append(plan.get_timings()["a4_factor"])
        plan.enable_timings(0)
        step()
        n = cfg["n"]
        ms_f = float(np.median(fa))
        out["a4"] = {"n": n, "flops": n ** 3 / 3.0, "factor_ms_alone": round(ms_f, 4),
                     "factor_ms_beside_science_side": out["stages_ms"]["a4_factor"], "solve_ms": out["stages_ms"]["a4_solve"],
                     "achieved_tflops": round(n ** 3 / 3.0 / ms_f / 1e9, 3),
                     "frac_of_dmma_probe": round(n ** 3 / 3.0 / ms_f / 1e9 / dmma, 4) if dmma else None,
                     "bound": "latency (a 732-step dependent chain; 0.13 GFLOP)"}
    except Exception as ex:  # pragma: no cover
        out["a4"] = {"error": str(ex)}

    # cuFFT beside the product's transforms (BASELINE.json north_star: "cuFFT timed only as a comparison, never on the product
    # path"): torch.fft.rfft2 / irfft2 of one zero-padded 4096 x 4096 FP64 frame against row_fwd_S + col_fwd_S and col_inv + row_inv
    try:
        pad = torch.zeros((4096, 4096), dtype=torch.float64, device="cuda"); pad[:ny, :nx] = dS
        for _ in range(3):
            sp_ = torch.fft.rfft2(pad); back = torch.fft.irfft2(sp_, s=pad.shape)
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        tf, ti = [], []
        for _ in range(K):
            ev[0].record(stream); sp_ = torch.fft.rfft2(pad); ev[1].record(stream); back = torch.fft.irfft2(sp_, s=pad.shape); ev[2].record(stream)
            torch.cuda.synchronize()
            tf.append(ev[0].elapsed_time(ev[1])); ti.append(ev[1].elapsed_time(ev[2]))
        del pad, sp_, back
        r = nx * ny * 8.0
        ours_f = kernels.get("row_fwd_S", 0.0) + kernels.get("col_fwd_S", 0.0)
        ours_i = kernels.get("col_inv", 0.0) + kernels.get("row_inv", 0.0)
        out["cufft_compare"] = {"what": "comparison only, never on the product path: torch.fft (cuFFT) FP64 rfft2 / irfft2 of one 4096 x 4096 frame",
                                "cufft_rfft2_ms": round(float(np.median(tf)), 4), "cufft_irfft2_ms": round(float(np.median(ti)), 4),
                                "cufft_rfft2_frac_of_measured_hbm_4r": round(4 * r / float(np.median(tf)) / 1e6 / peak, 4),
                                "ours_row_fwd_S_plus_col_fwd_S_ms": round(ours_f, 4),
                                "ours_fwd_frac_of_measured_hbm_4r": round(4 * r / ours_f / 1e6 / peak, 4) if ours_f else None,
                                "ours_col_inv_plus_row_inv_ms": round(ours_i, 4),
                                "note": "ours inverse = NK = 6 spectra combined with the synthesised kernel spectra + the fused subtraction (10 r), cuFFT inverse = one plain transform (4 r)"}
    except Exception as ex:  # pragma: no cover
        out["cufft_compare"] = {"error": str(ex)}

    # BASELINE.json configs[4] (large kernel: L = 21, DK = 3, n = 4416): one more plan, the seeded pair of the config
    if args.large:
        try:
            from paper_2509_18544_b200 import SfftPlan as _Plan
            c4 = starfield.make_pair(4)
            d4S, d4R = torch.from_numpy(c4["S"]).cuda(), torch.from_numpy(c4["R"]).cuda()
            p4 = _Plan(nx, ny, c4["L"], c4["DK"], c4["DB"])
            o4 = torch.empty_like(d4S)

            def step4():
                p4.build_system(d4S, d4R); p4.solve(); p4.subtract(o4)
            for _ in range(2):
                step4()
            p4.sync_status()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(5):
                step4()
            e1.record(stream)
            torch.cuda.synchronize()
            ms4 = e0.elapsed_time(e1) / 5
            st4 = {}
            for _ in range(3):
                p4.enable_timings(1); step4()
                for k_, v_ in p4.get_timings().items():
                    st4.setdefault(k_, []).append(v_)
            st4 = {k_: round(float(np.median(v_)), 4) for k_, v_ in st4.items()}
            p4.enable_timings(2); step4()
            k4 = {}
            for name, ms in p4.kernel_timings():
                k4[name] = k4.get(name, 0.0) + ms
            p4.enable_timings(0)
            n4 = p4.n
            NK4, W4 = 10, 20
            dfma = out.get("fp64_probe_tflops", {}).get("dfma"); dmma = out.get("fp64_probe_tflops", {}).get("dmma_m8n8k4")
            # Omega pass: 55 pairs x 4096 x 2049 elements, two lag halves; per 16 elements and half: 16 products (64) +
            # 16-point DFT (160) + 21 lags folded (84) FP64 instructions, 2 flop each
            om_flop = 55 * 4096.0 * 2049 * 2 * (64 + 160 + 84) / 16.0 * 2
            om_ms = k4.get("lagcol_omega", 0.0)
            fac_ms = st4.get("a4_factor", 0.0)
            out["large_kernel"] = {"workload": "BASELINE.json configs[4]: 4088x4088 pair, L=21, DK=3, DB=2 (n=4416)", "n": n4,
                                   "ms_per_step": round(ms4, 4), "images_per_s": round(1e3 / ms4, 2), "stages_ms": st4,
                                   "kernels_ms": {k_: round(v_, 4) for k_, v_ in sorted(k4.items(), key=lambda kv: -kv[1])[:10]},
                                   "a2_omega_lagcol": {"ms": round(om_ms, 4), "fp64_flop": om_flop,
                                                       "frac_of_dfma_probe": round(om_flop / om_ms / 1e9 / dfma, 4) if dfma and om_ms else None},
                                   "a4_factor": {"ms": fac_ms, "flops": n4 ** 3 / 3.0,
                                                 "achieved_tflops": round(n4 ** 3 / 3.0 / fac_ms / 1e9, 3) if fac_ms else None,
                                                 "frac_of_dmma_probe": round(n4 ** 3 / 3.0 / fac_ms / 1e9 / dmma, 4) if dmma and fac_ms else None},
                                   "workspace_gb": round(p4.workspace_bytes / 1e9, 3)}
            p4.destroy()
            del d4S, d4R, o4
        except Exception as ex:  # pragma: no cover
            out["large_kernel"] = {"error": str(ex)}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=32, help="science images of the batched (configs[3]) extra; 0 = skip")
    ap.add_argument("--large", type=int, default=1, help="1: also run BASELINE.json configs[4] (n = 4416) as the `large_kernel` extra")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
