#!/usr/bin/env python
"""bench.py -- IM columns/s of the synthetic Shack-Hartmann interaction matrix on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]
                  [--slope-mode nd|gtilt] [--repair] [--dictionary MODES_PER_LAYER]

A "step" is one pass of the whole hot path (S1-S4 of SURVEY.md sec. 8(a)) over one synthetic
workload: BASELINE.json config C (default 3: ELT MCAO ground DM, 5065 actuators x 6 LGS WFS =
30,390 columns).  One JSON line is printed by rank 0.

  value     columns/s, inputs resident in HBM, COLD L2: every timed step has its own CUDA-event pair and a
            256 MiB scratch buffer is overwritten between steps, outside the timed windows (SURVEY.md
            sec. 8(d), H7); the mean over the K steps is the headline.  config.warm_ms_per_step is the same
            K steps back to back without the flush, reported beside it.
  e2e       columns/s through synim_interaction_matrix_host: pinned HOST cube/bboxes in, HOST IM out,
            copies inside the timed region
  roofline  algorithmic bytes (IF bytes that must be read + IM bytes written) / mean cold step
            time, against the measured HBM copy bandwidth (frac) and the 8 TB/s datasheet figure
            (frac_datasheet)
  cpu_baseline  the float64 oracle, as it stands, on the host cores, on a bounded sample of modes

--repair times synim_interaction_matrix_repaired (edge repair) on the config's modes cut by a
source-frame mask; --dictionary M (default 64; 0 to skip) adds, at N=1, the 12-layer dictionary of PAPER.md:132 (M modes per
layer) through synim_dictionary_host under config.dictionary.
--extra (default "5,4,2,3p,4p,3g,3r", most wanted first): at N=1 the line also carries, under config.other_configs, short device-resident runs
of the other configurations, each in its own process.
config.ablation (and other_configs[*].ablation; --no-ablate to skip): after everything else, a few cold steps each of a plain
fill of the matrix (the write stream alone), half the modes and one wave of CTAs, and every class of sensors on its own --
what a step's time is made of, measured on the box that ran the line.
--impl reference times the oracle only (rank 0; other ranks exit).  N > 1: every rank holds its own
workload of the same shape (independent problems, no data-path collective): weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "IM columns/s (actuator x WFS)"
UNIT = "columns/s"
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent
DATASHEET_HBM_GBS = 8000.0    # B200 datasheet HBM3e figure (the "strict" denominator)
FLUSH_BYTES = 256 << 20       # scratch buffer overwritten between timed steps (2x the 126 MB L2)


def algorithmic_bytes(wl) -> dict:
    """IF bytes that must be read once (32-byte sectors of each bbox row; the whole mode when dense)
    plus IM bytes written."""
    if wl.bbox is not None:
        b = wl.bbox.astype(np.int64)
        w = np.maximum(b[:, 2] - b[:, 0] + 1, 0)
        h = np.maximum(b[:, 3] - b[:, 1] + 1, 0)
        read = int((h * ((w * 4 + 31) // 32) * 32).sum())
    else:
        read = int(wl.n_modes) * wl.ny * wl.nx * 4
    write = int(wl.n_rows) * int(wl.n_modes) * 4
    return {"read": read, "write": write, "total": read + write}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth, burst)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def profile_traffic(cfg: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu summary."""
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        best = None
        for line in open(p):
            f = [x.strip() for x in line.split(",")]
            if f and f[0] == f"cfg{cfg}":
                best = float(f[1]) + float(f[2])      # the last matching line is the newest round
        return best
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for nme, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_throughput(wl, target_s: float, n_threads: int = 0):
    """Time the oracle (as it stands, OpenMP over modes) on a seeded sample of modes sized for about
    ``target_s`` seconds.  Returns (columns/s, cores, description)."""
    from oracle import oracle as O
    cores = O.num_threads() if n_threads <= 0 else n_threads
    rng = np.random.default_rng(7759)
    probe = np.sort(rng.choice(wl.n_modes, size=min(wl.n_modes, max(cores, 8)), replace=False))
    t0 = time.perf_counter()
    O.interaction_matrix(wl, modes=probe, n_threads=n_threads)
    dt = time.perf_counter() - t0
    n = int(min(wl.n_modes, max(len(probe), round(len(probe) * target_s / max(dt, 1e-6)))))
    sel = np.sort(rng.choice(wl.n_modes, size=n, replace=False))
    t0 = time.perf_counter()
    O.interaction_matrix(wl, modes=sel, n_threads=n_threads)
    dt = time.perf_counter() - t0
    cols = n * len(wl.wfs)
    return cols / dt, cores, f"{n} of {wl.n_modes} modes (seeded draw) x {len(wl.wfs)} WFS = {cols} columns in {dt:.1f} s"


def config_dict(wl, extra=None):
    d = {"workload": f"BASELINE.json configs[{wl.cfg - 1}]: {wl.name}", "n_modes": wl.n_modes, "n_wfs": len(wl.wfs),
         "columns": wl.n_columns, "im_rows": wl.n_rows, "grid": [wl.ny, wl.nx],
         "l2": f"flushed: a {FLUSH_BYTES >> 20} MiB scratch buffer is overwritten between timed steps, outside the "
               "per-step event pairs"}
    if extra:
        d.update(extra)
    return d


T_START = time.time()


def other_configs(spec: str, budget_s: float) -> dict:
    """Short device-resident runs of the other configurations (cold-L2 protocol, 10 steps), one process each so that
    nothing they do can take the headline run down; what the line keeps of each: step time, columns/s, roofline
    fractions, the dominant kernel and the parity spot check."""
    out = {}
    for tag in [t.strip() for t in spec.split(",") if t.strip()]:
        cfg = tag.rstrip("rgp")
        if cfg not in ("1", "2", "3", "4", "5"):
            out[tag] = {"error": "unknown tag"}
            continue
        if time.time() - T_START > budget_s:      # the default run must end within minutes whatever the box is like
            out[tag] = {"skipped": f"time budget: {budget_s:.0f} s since the start of bench.py were spent (--extra-budget-s)"}
            continue
        cmd = [sys.executable, os.path.abspath(__file__), "--config", cfg, "--steps", "10", "--warmup", "3", "--no-e2e",
               "--no-cpu-baseline", "--parity-modes", "32", "--extra", "none"]
        if tag.endswith("r"):
            cmd.append("--repair")
        if tag.endswith("g"):
            cmd += ["--slope-mode", "gtilt"]
        env = dict(os.environ, SYNIM_BENCH_CHILD="1")
        if tag.endswith("p"):
            env["SYNIM_ZONAL_PACKED"] = "1"
        try:
            res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
            last = [ln for ln in res.stdout.strip().splitlines() if ln.startswith("{")]
            if res.returncode != 0 or not last:
                out[tag] = {"error": (res.stderr or res.stdout)[-400:]}
                continue
            d = json.loads(last[-1])
            out[tag] = {"workload": d["config"]["workload"], "columns": d["config"]["columns"], "ms_per_step": d["ms_per_step"],
                        "cold_ms_min_med_max": d["config"]["cold_ms_min_med_max"], "warm_ms_per_step": d["config"]["warm_ms_per_step"],
                        "columns_per_s": d["value"], "frac": d["roofline"]["frac"], "frac_datasheet": d["roofline"]["frac_datasheet"],
                        "algorithmic_bytes": d["roofline"]["algorithmic_bytes"]["total"], "kernel": d["roofline"]["kernel"],
                        "gpu_launches": d["gpu_launches"], "parity_spot_check": d["parity_spot_check"],
                        "clocks": d["clocks"], "slope_mode": d["config"].get("slope_mode"),
                        "edge_repair": d["config"].get("edge_repair"), "ablation": d["config"].get("ablation"),
                        "packed_zonal_walk": tag.endswith("p")}
        except Exception as exc:
            out[tag] = {"error": f"{type(exc).__name__}: {exc}"}
    return out


def ablate(synim, wl, geom, cube, bbox, diag, bmax, affines, scales, out, scratch, stream, smode, full_ms, k=5):
    """Measured decomposition of a step (cold-L2 protocol, mean of k steps each): the write stream alone, fewer modes
    (is the grid's tail or the launch what is paid for?), and every class of sensors on its own."""
    import torch

    def cold_ms(fn):
        fn(); fn()
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(k)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(k)]
        for i in range(k):
            scratch.fill_(i & 0xff)
            e0[i].record(stream); fn(); e1[i].record(stream)
        torch.cuda.synchronize()
        return float(np.mean([e0[i].elapsed_time(e1[i]) for i in range(k)]))

    def run(g, n, o, aff, sc):
        synim.interaction_matrix(g, cube[:n], None if bbox is None else bbox[:n], aff, sc, out=o, bbox_max=bmax, stream=stream,
                                 diag=None if diag is None else diag[:n], mode=smode)

    res = {"protocol": f"cold L2, mean of {k} steps each", "full_step_ms": full_ms,
           "im_fill_ms": cold_ms(lambda: out.zero_()),
           "im_fill_note": "torch fill of the whole matrix buffer: the write stream alone, no sampling"}
    n = wl.n_modes
    counts = {"half_modes": n // 2}
    if bbox is not None:
        counts["one_wave_1036_ctas"] = min(n, 148 * 7)      # synim_strip_kernel: one CTA per mode, 7 CTAs per SM
    res["fewer_modes"] = {tag: {"n_modes": c, "ms": cold_ms(lambda c=c: run(geom, c, out[:c], affines, scales))}
                          for tag, c in counts.items() if 0 < c < n}
    # sensors: every class (same subaperture grid) on its own, and the first sensor alone
    classes = {}
    for i, w in enumerate(wl.wfs):
        classes.setdefault((w.n_subap, w.n_pix), []).append(i)
    groups = {f"{ns}x{ns} subapertures of {npx} px ({len(ix)} sensors)": ix for (ns, npx), ix in classes.items() if len(classes) > 1}
    if len(wl.wfs) > 1:
        groups["first sensor alone"] = [0]
        groups["second sensor alone"] = [1]
    res["sensors"] = {}
    for tag, ix in groups.items():
        sub = [wl.wfs[i] for i in ix]
        g = synim.create_geometry(wl.ny, wl.nx, sub)
        o = torch.empty((n, g.num_rows), dtype=torch.float32, device=out.device)
        aff, sc = [affines[i] for i in ix], [scales[i] for i in ix]
        res["sensors"][tag] = {"columns": n * len(ix), "im_bytes": int(o.numel() * 4), "ms": cold_ms(lambda: run(g, n, o, aff, sc))}
        torch.cuda.synchronize()
        g.destroy()
        del o
    return res


def run_reference(args, rank: int):
    if rank != 0:
        return
    from paper_2606_07759_b200 import workloads
    wl = workloads.make_config(args.config)
    per_step_s = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    vals, desc, cores = [], "", 0
    for k in range(args.warmup + args.steps):
        v, cores, desc = oracle_throughput(wl, per_step_s)
        if k >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wl.n_columns / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(wl, {"note": "float64 CPU oracle; each step is a bounded sample, ms_per_step extrapolated"}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--parity-modes", type=int, default=256)
    ap.add_argument("--repair", action="store_true",
                    help="time synim_interaction_matrix_repaired (edge repair, PAPER.md:69-76) on the config's modes cut by "
                         "a source-frame pupil mask instead of the plain hot path")
    ap.add_argument("--dictionary", type=int, default=64, metavar="MODES_PER_LAYER",
                    help="at N=1 also run the 12-layer dictionary of PAPER.md:132 (workloads.make_dictionary, this many modes per "
                         "layer) through synim_dictionary_host and report it under config.dictionary (0: skip)")
    ap.add_argument("--extra", default="5,4,2,3p,4p,3g,3r",
                    help="at N=1, after the timed run: short device-resident runs of these other configurations, each in its "
                         "own process, reported under config.other_configs ('3r' = config 3 with edge repair, '3g' = config 3 "
                         "with the G-tilt estimator, '3p' / '4p' = config 3 / 4 through the opt-in packed zonal walk, SYNIM_ZONAL_PACKED=1; "
                         "'none' to skip)")
    ap.add_argument("--extra-budget-s", type=float, default=200.0,
                    help="no further --extra child is started once bench.py has been running this long (reported as skipped)")
    ap.add_argument("--no-ablate", action="store_true",
                    help="skip config.ablation: after the timed run, a few cold steps each of (a) a plain fill of the matrix "
                         "(the write stream alone), (b) half the modes, and one wave of CTAs for zonal modes, (c) every class of "
                         "sensors (and a single sensor) on its own -- what the step time is made of, measured, not inferred")
    ap.add_argument("--slope-mode", default="nd", choices=["nd", "gtilt"],
                    help="nd = the paper's numerical-derivative engine (the metric); gtilt = the comparison estimator")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    from paper_2606_07759_b200 import build, sharding, synim, workloads
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0 and not os.environ.get("SYNIM_BENCH_CHILD"):      # (a child of other_configs: the parent has built it)
        build.build_library()
    if dist is not None:
        dist.barrier()
    synim.lib()
    warmup = max(args.warmup, 3)

    # every rank: its own workload of the same shape (independent problems -> weak scaling)
    wl = workloads.make_config(args.config)
    repair_mask = None
    if args.repair:
        if args.slope_mode != "nd":
            raise SystemExit("bench.py: --repair belongs to the numerical-derivative engine")
        # the modes cut by a round mask in the source frame, 1 % inside the grid's edge (a DM / pupil mask)
        wl = workloads.masked(wl, workloads.make_pupil(wl.nx, 0.99 * wl.nx, 0.0) if wl.ny == wl.nx else np.ones((wl.ny, wl.nx), np.float32))
        repair_mask = torch.from_numpy(wl.mask).cuda()
    affines = synim.affines_of(wl)
    scales = [w.slope_scale for w in wl.wfs]
    stream = torch.cuda.current_stream()
    cube = torch.from_numpy(wl.cube).cuda()
    out = torch.empty((wl.n_modes, wl.n_rows), dtype=torch.float32, device="cuda")
    scratch = torch.empty(FLUSH_BYTES, dtype=torch.uint8, device="cuda")

    # the very first call of a session: geometry, supports (one pass over the cube) and the IM, timed together
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_first0 = time.perf_counter()
    e0.record(stream)
    geom = synim.create_geometry(wl.ny, wl.nx, wl.wfs)
    bbox, diag, bmax = None, None, (0, 0)
    if wl.bbox is not None:
        bbox, diag = synim.compute_supports(cube)
        bmax = synim.bbox_extent(bbox)
    smode = synim.SLOPES_GTILT if args.slope_mode == "gtilt" else synim.SLOPES_ND
    synim.interaction_matrix(geom, cube, bbox, affines, scales, out=out, bbox_max=bmax, stream=stream, diag=diag, mode=smode,
                             repair_mask=repair_mask)
    e1.record(stream)
    torch.cuda.synchronize()
    first_call = {"wall_ms": 1e3 * (time.perf_counter() - t_first0), "device_ms": e0.elapsed_time(e1),
                  "includes": "synim_create_geometry + synim_compute_bboxes + synim_bbox_extent + synim_interaction_matrix"
                              " (first launch: module load, shared-memory opt-in)"}
    assert geom.num_rows == wl.n_rows

    def step(o=out, c=cube, b=bbox, d=diag):
        synim.interaction_matrix(geom, c, b, affines, scales, out=o, bbox_max=bmax, stream=stream, diag=d, mode=smode,
                                 repair_mask=repair_mask)

    launches0 = synim.launch_count()
    step()
    launches_per_step = synim.launch_count() - launches0
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    K = args.steps
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    scratch.fill_(1)
    step()   # one more untimed step: the GPU sat idle while the clock sampler started
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t_wall0 = time.time()
    for k in range(K):     # COLD: flush, then one step inside its own event pair
        scratch.fill_(k & 0xff)
        ev0[k].record(stream)
        step()
        ev1[k].record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    cold = np.array([ev0[k].elapsed_time(ev1[k]) for k in range(K)])
    # WARM: the same K steps back to back (what round 1 reported)
    wv = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    wv[0].record(stream)
    for k in range(K):
        step()
        wv[k + 1].record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t_wall1 = time.time()
    warm = np.array([wv[k].elapsed_time(wv[k + 1]) for k in range(K)])
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None

    # strong scaling beside it: ONE cube, rank r computes the columns of its
    # sharding.partition_modes range into its block of the matrix; no exchange
    strong_ms = 0.0
    if world > 1:
        b, e = sharding.partition_modes(wl.n_modes, world)[rank]
        sub = (out[b:e], cube[b:e], None if bbox is None else bbox[b:e], None if diag is None else diag[b:e])
        if e > b:
            for _ in range(3):
                step(*sub)
        torch.cuda.synchronize()
        dist.barrier()
        sv0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        sv1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        for k in range(K):
            scratch.fill_(k & 0xff)
            sv0[k].record(stream)
            if e > b:
                step(*sub)
            sv1[k].record(stream)
        torch.cuda.synchronize()
        strong_ms = float(np.mean([sv0[k].elapsed_time(sv1[k]) for k in range(K)]))
        step()       # the whole matrix again, for the checks below

    # the timed launch configuration against the oracle on >= 256 sampled modes (rank 0)
    parity = None
    if rank == 0:
        from oracle import oracle as O
        rng = np.random.default_rng(7759 + 100)
        sel = np.sort(rng.choice(wl.n_modes, size=min(args.parity_modes, wl.n_modes), replace=False))
        ref = O.interaction_matrix(wl, modes=sel, mode=O.GTILT if args.slope_mode == "gtilt" else O.ND,
                                   repair_mask=wl.mask if args.repair else None)
        got = out[torch.from_numpy(sel).cuda()].cpu().numpy().T.astype(np.float64)
        amp = np.abs(wl.cube[sel]).reshape(len(sel), -1).max(axis=1)
        l2w = elw = 0.0
        r0 = 0
        for w in wl.wfs:       # per (mode, WFS) column; columns that are pure cancellation (R17) left out
            r1 = r0 + 2 * w.n_valid
            cm = np.abs(ref[r0:r1]).max(axis=0)
            live = cm > 100 * 2.0 ** -24 * abs(w.slope_scale) * amp
            d = got[r0:r1][:, live] - ref[r0:r1][:, live]
            l2w = max(l2w, float((np.linalg.norm(d, axis=0) / np.linalg.norm(ref[r0:r1][:, live], axis=0)).max()))
            elw = max(elw, float((np.abs(d).max(axis=0) / cm[live]).max()))
            r0 = r1
        parity = {"sampled_modes": int(len(sel)), "max_rel_l2": l2w, "max_elementwise": elw}

    # end to end through the HOST-buffer entry point (pinned host memory, copies inside the timing)
    e2e = None
    if args.repair:
        args.no_e2e = True     # the host-buffer entry points have no repaired variant
    e2e_error = None
    if not args.no_e2e:
        h_cube = torch.from_numpy(wl.cube).pin_memory()
        h_bbox = None if wl.bbox is None else torch.from_numpy(wl.bbox).pin_memory()
        h_out = torch.empty((wl.n_modes, geom.num_rows), dtype=torch.float32).pin_memory()

        def host_step():
            synim.interaction_matrix_host(geom, h_cube, h_bbox, affines, scales, out_host=h_out, stream=stream, mode=smode)
        try:
            host_step()
            torch.cuda.synchronize()
        except Exception as exc:        # reported in the line; the device-resident numbers stand on their own
            e2e_error = f"{type(exc).__name__}: {exc}"
        if dist is not None:
            dist.barrier()
        e2e_ms = 0.0
        if e2e_error is None:
            t0 = time.perf_counter()
            try:
                for _ in range(args.e2e_steps):
                    host_step()
                torch.cuda.synchronize()
            except Exception as exc:
                e2e_error = f"{type(exc).__name__}: {exc}"
            e2e_ms = 1e3 * (time.perf_counter() - t0) / args.e2e_steps
        host_in = h_cube.numel() * 4 + (0 if h_bbox is None else h_bbox.numel() * 4)
        if h_bbox is None:
            h2d = host_in
        else:
            # the library packs each mode's bbox (plus the ring the kernel stages with it) into a pinned
            # buffer and copies only that: [n][bh+2][roundup4(bw+5)] floats + bboxes and origins (include/synim.h)
            bwm = int((wl.bbox[:, 2] - wl.bbox[:, 0] + 1).max()); bhm = int((wl.bbox[:, 3] - wl.bbox[:, 1] + 1).max())
            h2d = wl.n_modes * max(8, (bwm + 8) & ~3) * max(4, bhm + 2) * 4 + wl.n_modes * 24
        d2h = h_out.numel() * 4
        e2e_parity = None
        if rank == 0 and e2e_error is None:
            got_h = h_out[torch.from_numpy(sel)].numpy().T.astype(np.float64)
            cmx = np.abs(ref).max(axis=0)
            e2e_parity = float((np.abs(got_h - got).max(axis=0) / np.maximum(cmx, 1e-30)).max())
        if e2e_error is None:
            e2e = (e2e_ms, h2d, d2h, host_in, e2e_parity)

    # what the step time is made of (N = 1; a side leg: reported, never fatal)
    ablation = None
    if world == 1 and not args.no_ablate and not args.repair:
        try:
            ablation = ablate(synim, wl, geom, cube, bbox, diag, bmax, affines, scales, out, scratch, stream, smode,
                              float(cold.mean()))
        except Exception as exc:
            ablation = {"error": f"{type(exc).__name__}: {exc}"}

    # the multi-layer dictionary of PAPER.md:132-138, end to end through host buffers (the very last device work: a
    # side leg that fails here can hurt nothing else)
    dictionary = None
    if args.dictionary > 0 and world == 1 and not os.environ.get("SYNIM_BENCH_CHILD"):
        try:
            layers = workloads.make_dictionary(n_layers=12, max_modes=args.dictionary)
            dgeom = synim.create_geometry(layers[0].ny, layers[0].nx, layers[0].wfs)
            spec = [dict(cube=torch.from_numpy(l.cube).pin_memory(), bbox=torch.from_numpy(l.bbox).pin_memory(),
                         affines=synim.affines_of(l),
                         out=torch.empty((l.n_modes, dgeom.num_rows), dtype=torch.float32).pin_memory()) for l in layers]
            synim.dictionary_host(dgeom, spec, stream=stream)      # warm-up: buffers, module load
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            synim.dictionary_host(dgeom, spec, stream=stream)
            torch.cuda.synchronize()
            d_ms = 1e3 * (time.perf_counter() - t0)
            n_cols = sum(l.n_columns for l in layers)
            d2h = sum(l.n_modes for l in layers) * dgeom.num_rows * 4
            from oracle import oracle as O2
            l0 = layers[-1]
            pick = np.arange(min(4, l0.n_modes))
            refd = O2.interaction_matrix(l0, modes=pick)
            gotd = spec[-1]["out"][: len(pick)].numpy().T.astype(np.float64)
            dictionary = {"layers": len(layers), "grids": [l.ny for l in layers], "modes_per_layer": [l.n_modes for l in layers],
                          "columns": n_cols, "ms": d_ms, "columns_per_s": n_cols / (d_ms * 1e-3),
                          "host_cube_bytes": int(sum(l.cube.nbytes for l in layers)), "d2h_bytes": int(d2h),
                          "d2h_gbs": d2h / (d_ms * 1e-3) / 1e9,
                          "top_layer_max_abs_err_vs_oracle": float(np.abs(gotd - refd).max() / np.abs(refd).max()),
                          "api": "synim_dictionary_host (pinned host buffers, chunks of 64 MB of matrix, two in flight)"}
            dgeom.destroy()
        except Exception as exc:       # (a side leg: reported, never fatal)
            dictionary = {"error": f"{type(exc).__name__}: {exc}"}

    # max over ranks (one process: no device work here, so that a side leg that failed above cannot take the line down)
    times = [float(cold.mean()), e2e[0] if e2e else 0.0, float(warm.mean()), strong_ms]
    if dist is not None:
        t = torch.tensor(times, dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        times = [float(x) for x in t]
    cold_ms, e2e_ms, warm_ms, strong_ms = times
    plan = sharding.weak_scaling_plan(wl.n_columns, world)

    if rank == 0:
        value = plan["total_units"] / (cold_ms * 1e-3)
        ab = algorithmic_bytes(wl)
        peak, peak_src = measured_peak()
        kernel_ms = float(cold.mean())
        achieved = ab["total"] / (kernel_ms * 1e-3) / 1e9
        traffic = profile_traffic(args.config)
        extra = {"parallelism": f"{world} independent workloads, one per GPU, no collective",
                 "timing": "cold L2: one CUDA-event pair per step, scratch flush between steps outside the pairs; "
                           "value and ms_per_step are the MEAN over the steps",
                 "cold_ms_min_med_max": [float(cold.min()), float(np.median(cold)), float(cold.max())],
                 "warm_ms_per_step": warm_ms, "warm_ms_min_med_max": [float(warm.min()), float(np.median(warm)), float(warm.max())],
                 "first_call": first_call}
        if dictionary:
            extra["dictionary"] = dictionary
        if ablation:
            extra["ablation"] = ablation
        if args.repair:
            extra["edge_repair"] = "synim_interaction_matrix_repaired, threshold 0.999999, modes cut by a round source-frame mask"
        if world > 1:
            extra["strong_scaling"] = {"what": "ONE cube sharded by contiguous mode ranges (sharding.partition_modes), cold L2, "
                                               "max over ranks", "ms_per_step": strong_ms,
                                       "columns_per_s": wl.n_columns / (strong_ms * 1e-3) if strong_ms > 0 else None}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warmup, "ms_per_step": cold_ms, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": config_dict(wl, dict(extra, slope_mode=args.slope_mode)),
                "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                             "frac": achieved / peak, "frac_datasheet": achieved / DATASHEET_HBM_GBS,
                             "traffic": traffic,
                             "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of the committed ncu capture "
                                               "(profiles/dram_traffic.csv), not measured in this run",
                             "peak_source": peak_src, "algorithmic_bytes": ab,
                             "kernel": synim.hot_kernel_name(wl.bbox is None, args.slope_mode == "gtilt", args.repair), "kernel_ms": kernel_ms,
                             "warm_frac": ab["total"] / (float(warm.mean()) * 1e-3) / 1e9 / peak},
                "clocks": clocks, "gpu_launches": 2 * args.steps * launches_per_step,
                "gpu_launches_note": f"{launches_per_step} launch(es) of this library's kernels per step (counted by the library), "
                                     f"{args.steps} cold + {args.steps} warm timed steps",
                "parity_spot_check": parity}
        if e2e:
            line["e2e"] = {"value": plan["total_units"] / (e2e_ms * 1e-3), "unit": UNIT,
                           "h2d_bytes_per_step": e2e[1], "d2h_bytes_per_step": e2e[2], "ms_per_step": e2e_ms,
                           "host_input_bytes": e2e[3], "max_elementwise_vs_device_path": e2e[4],
                           "api": "synim_interaction_matrix_host (pinned host buffers; compact supports are packed "
                                  "on the host and only they cross the bus; chunks of modes pipelined: pack | H2D + kernel | D2H)"}
        if e2e_error:
            line["e2e"] = {"value": None, "unit": UNIT, "error": e2e_error}
        if world == 1 and args.extra.strip().lower() != "none":
            line["config"]["other_configs"] = other_configs(args.extra, args.extra_budget_s)
        if world == 1 and not args.no_cpu_baseline:
            v, cores, desc = oracle_throughput(wl, 10.0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
            v1, _, desc1 = oracle_throughput(wl, 6.0, n_threads=1)
            line["cpu_baseline_1thread"] = {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc1}
        print(json.dumps(line), flush=True)
    try:
        geom.destroy()
    except Exception:
        pass
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
