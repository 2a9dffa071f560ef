#!/usr/bin/env python
"""bench.py -- strain-seconds/s of the gwi hot path on B200 (BASELINE.json metric), one JSON line on stdout.

Workload at N=1 (BASELINE.json configs[1]): one paper-scale model (2 branches x 20 gated dilated blocks, 64 residual /
128 skip channels, k=2) in FP16 mode on a batch of 1024 windows x 4096 samples x 2 detectors of seeded N(0,1) noise
with 10 % of windows carrying a chirp.  One "step" = one pass of the whole hot path over one batch:
gwi_infer (lift, 40 block-layers, head) -> gwi_ensemble_triggers (mean, threshold 0.5, runs >= 2048) -> trigger count.
1 window = 1 s of two-detector strain, so value = windows / s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--windows B] [--impl reference] [--scaling weak|strong]

Multi-GPU (one process per GPU; with --gpus N > 1 and no launcher the ranks are started here through
torch.distributed.run): --scaling weak (default): every rank runs the same per-GPU batch (the path shards over windows;
no collective on the data path), value = all ranks' windows / max-over-ranks time.  --scaling strong: the configs[4]
stream (--stream-chunks one-hour chunks) is time-sharded over the ranks (gwi_stream_set_shard), the shard-edge runs are
gathered and joined on rank 0; value = stream seconds / max-over-ranks wall time.
"""
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

import gwsynth as gs  # noqa: E402

METRIC = "strain-seconds/s (2 detectors, ensemble) on 1 B200; % FP16 tensor peak"
UNIT = "strain-seconds/s"
T = 4096
THETA, LMIN = 0.5, 2048
NROT = 8  # rotating input/output buffers: 8 x (16.8 MB in + 16.8 MB out) > 126 MB L2


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


PROFILE_CSV = os.path.join("profiles", "r2_k_stack_raw.csv")   # `ncu -i ... --page raw --csv` of the committed capture


def profile_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum of k_stack per launch, read from the committed ncu capture
    (profiles/r2_k_stack.md names the command).  None if the file is missing."""
    import csv
    path = os.path.join(ROOT, PROFILE_CSV)
    if not os.path.exists(path):
        return None
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    rows = list(csv.reader(open(path)))
    hdr, units = rows[0], rows[1]
    best = None
    for r in rows[2:]:
        name = r[hdr.index("Kernel Name")] if "Kernel Name" in hdr else ""
        if "k_stack" not in name:
            continue
        tot = 0.0
        for col in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            i = hdr.index(col)
            tot += float(r[i].replace(",", "")) * scale.get(units[i], 1.0)
        best = tot if best is None else max(best, tot)
    return best


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            time.sleep(0.02)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows for n, v in zip(names, r[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def stream_bench(dev, work, rank, n_chunks=744, paper_month=False):
    """Extra, reported beside the headline: the streaming ensemble path (gwi_stream_*) on the config-1 architecture.
    hour  = BASELINE.json configs[2]: 4-model ensemble, 1 h two-detector stream resident in HBM, one push + finish.
    month = configs[4]: 744 one-hour chunks pushed from pinned host buffers (H2D on the side stream inside the timed
            region), triggers read back at the end.  Two distinct seeded hour chunks rotate as the host source."""
    import torch
    import paper_2201_11133_b200 as gwi
    N1 = 3600 * gs.FS
    models = []
    for sd in range(4):
        pth = os.path.join(work, f"bench_cfg1_seed{sd}_r{rank}.gwim")
        gs.make_model_file(pth, gs.CFG1_ARCH, seed=sd)
        models.append(gwi.load_model(pth, gwi.FP16, dev.index))
    host = [torch.from_numpy(gs.stream_noise(1, c * N1, N1)).pin_memory() for c in range(2)]
    xd = host[0].to(dev)
    out = {}
    # ---- hour, device resident
    times = []
    for rep in range(5):
        st = gwi.Stream(models, N1, N1, THETA, LMIN, capacity=4096)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        st.push(xd[0], xd[1])
        e1.record()
        n, _ = st.finish()
        times.append(e0.elapsed_time(e1))
        st.close()
    ms = float(np.median(times[2:]))
    mufu_ops = N1 * 4 * (gs.CFG1_ARCH.tanh_per_timestep() if hasattr(gs.CFG1_ARCH, "tanh_per_timestep") else 256)
    floor_ms = mufu_ops / (16 * 148 * 1.965e9) * 1e3
    out["hour"] = {"workload": "configs[2]: 4 models (config-1 arch), 1 h stream, FP16, resident in HBM", "ms": ms,
                   "strain_seconds_per_s": 3600 / (ms * 1e-3), "triggers": n,
                   "bound": "alu (MUFU tanh: 256 per sample per model at 16/clk/SM x 148 SMs x 1.965 GHz)",
                   "mufu_floor_ms": floor_ms, "frac_of_mufu_floor": floor_ms / ms}
    # ---- hour, 4 paper-scale models (SURVEY.md 8(f) NEXT-2 in the small): tensor-core stream back end
    try:
        pm = []
        for sd in range(4):
            pth = os.path.join(work, f"bench_paper_seed{sd}_s{rank}.gwim")
            gs.make_model_file(pth, gs.PAPER_ARCH, seed=sd)
            pm.append(gwi.load_model(pth, gwi.FP16, dev.index))
        times = []
        for rep in range(3):
            st = gwi.Stream(pm, N1, N1, THETA, LMIN, capacity=4096)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            st.push(xd[0], xd[1])
            e1.record()
            n, _ = st.finish()
            times.append(e0.elapsed_time(e1))
            st.close()
        ms = float(np.median(times[1:]))
        out["hour_paper_scale"] = {"workload": "4 paper-scale models (2x20 blocks, R64/S128), 1 h stream, FP16, resident in HBM; "
                                               "148 segments of 99714 outputs + 2046 recomputed warm-up samples through k_stack in one launch per model",
                                   "ms": ms, "strain_seconds_per_s": 3600 / (ms * 1e-3), "triggers": n,
                                   "tflops_algorithmic": gs.PAPER_ARCH.flops_per_timestep() * N1 * 4 / (ms * 1e-3) / 1e12}
        # the same with 32 one-second time slides (paper-scale background estimation)
        lags = [gs.FS * k for k in range(1, 33)]
        for nl in (32, 60):
            # 60 one-second lags = the paper's 5 yr of time-slid background per month of data
            lg = [gs.FS * k for k in range(1, nl + 1)]
            times = []
            for rep in range(2):
                st = gwi.Stream(pm, N1, N1, THETA, LMIN, lags=lg, capacity=4096)
                tail = xd[1, N1 - st.tail_samples:].contiguous()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                st.prime(tail, sync=False)                       # the priming pass is part of the timed region
                st.push(xd[0], xd[1])
                e1.record()
                n, _ = st.finish()
                times.append(e0.elapsed_time(e1))
                st.close()
            ms = float(times[-1])
            out[f"hour_paper_scale_{nl}_slides"] = {"workload": f"4 paper-scale models, 1 h stream, zero lag + {nl} circular lags of k x 1 s, FP16 "
                                                                "(priming pass included)",
                                                    "ms": ms, "strain_seconds_per_s": 3600 / (ms * 1e-3),
                                                    "slid_strain_seconds_per_s": (nl + 1) * 3600 / (ms * 1e-3), "triggers": n}
        # NEXT-2 scaled to the default run: 24 one-hour chunks from pinned host memory through the 4 x paper-scale ensemble
        # (the whole month, 744 chunks, is --paper-month: about 2.5 minutes without slides)
        nh = min(24, n_chunks)
        st = gwi.Stream(pm, nh * N1, N1, THETA, LMIN, capacity=65536)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for c in range(nh):
            h = host[c & 1]
            st.push(h[0], h[1])
        n, _ = st.finish()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        st.close()
        out["day_paper_scale"] = {"workload": f"{nh} one-hour chunks from pinned host memory (H2D on the side stream inside the timed region), "
                                              "4 paper-scale models, zero lag, FP16; the month (744 chunks) is this x 31 (--paper-month runs it)",
                                  "wall_s": dt, "strain_seconds_per_s": nh * 3600 / dt, "triggers": n,
                                  "tflops_algorithmic": gs.PAPER_ARCH.flops_per_timestep() * N1 * nh * 4 / dt / 1e12}
        if paper_month:
            # the month through the 4 x paper-scale ensemble, streamed from pinned host memory
            for name, lg in (("month_paper_scale", []), ("month_paper_scale_32_slides", lags)):
                st = gwi.Stream(pm, n_chunks * N1, N1, THETA, LMIN, lags=lg, capacity=65536)
                if lg:
                    st.prime(host[(n_chunks - 1) & 1][1, N1 - st.tail_samples:].contiguous())
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for c in range(n_chunks):
                    h = host[c & 1]
                    st.push(h[0], h[1])
                n, _ = st.finish()
                torch.cuda.synchronize()
                dt = time.perf_counter() - t0
                st.close()
                out[name] = {"workload": f"{n_chunks} one-hour chunks from pinned host memory, 4 paper-scale models, "
                                         f"{1 + len(lg)} slide(s), FP16", "wall_s": dt,
                             "strain_seconds_per_s": n_chunks * 3600 / dt,
                             "slid_strain_seconds_per_s": (1 + len(lg)) * n_chunks * 3600 / dt, "triggers": n}
        del pm
    except Exception as ex:
        out["hour_paper_scale"] = {"error": repr(ex)}
    # ---- configs[3]: 1 day, 32 circular one-second slides, all lags in one pass (slid-strain-seconds/s)
    try:
        n_hours = 24 if n_chunks >= 24 else max(n_chunks, 1)
        xc = torch.from_numpy(np.stack([gs.coloured_whitened_noise(2 + d, d, N1, seg_len=N1) for d in range(2)])).to(dev)
        lags = [gs.FS * k for k in range(1, 33)]
        st = gwi.Stream(models, n_hours * N1, N1, THETA, LMIN, lags=lags, capacity=65536)
        tail = xc[1, N1 - st.tail_samples:].contiguous()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        st.prime(tail, sync=False)                               # the priming pass is part of the timed region
        for c in range(n_hours):
            st.push(xc[0], xc[1])
        e1.record()
        n, _ = st.finish()
        ms = e0.elapsed_time(e1)
        st.close()
        out["day_32_slides"] = {"workload": f"configs[3]: {n_hours} h of coloured-then-whitened noise (reading A27; one seeded hour per detector "
                                            "pushed repeatedly, resident in HBM), 4 models (config-1 arch), zero lag + 32 circular lags of "
                                            "k x 1 s, all lags in one pass", "ms": ms,
                                "strain_seconds_per_s": n_hours * 3600 / (ms * 1e-3),
                                "slid_strain_seconds_per_s": 33 * n_hours * 3600 / (ms * 1e-3), "triggers": n}
        del xc
    except Exception as ex:
        out["day_32_slides"] = {"error": repr(ex)}
    # ---- standalone post-processing (a-8..a-10) on materialised probabilities: HBM-bound, algorithmic bytes = M x N x 4
    try:
        Np = 1 << 27
        g = torch.Generator(device=dev)
        g.manual_seed(7)
        probs = [torch.rand(Np, generator=g, device=dev, dtype=torch.float32) * 0.45 for _ in range(4)]
        for k in range(16):                                    # 16 plateaus of 1 s above the threshold -> 16 triggers
            for pm_ in probs:
                pm_[(k + 1) * 7_000_003:(k + 1) * 7_000_003 + gs.FS] = 0.9
        times = []
        for rep in range(6):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            cnt, _, _ = gwi.ensemble_triggers(probs, THETA, LMIN, capacity=4096, sync=False)
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1))
        ms = float(np.median(times[2:]))
        hbm = peaks()[0].get("hbm_gbs", 6650.0)
        gbs = 4 * Np * 4 / (ms * 1e-3) / 1e9
        out["post"] = {"workload": "gwi_ensemble_triggers on 4 x 2^27 float32 probabilities (2.1 GB > L2): mean, threshold, run clustering",
                       "ms": ms, "triggers": int(cnt.item()), "bound": "hbm", "achieved_gb_per_s": gbs, "peak_gb_per_s": hbm,
                       "frac": gbs / hbm, "samples_per_s": Np / (ms * 1e-3)}
        del probs
    except Exception as ex:
        out["post"] = {"error": repr(ex)}
    # ---- NEXT-1 legs: the paper's peak rule on one model's probabilities, and the one-pass threshold sweep (both HBM-bound)
    try:
        Nf = 1 << 26
        g = torch.Generator(device=dev)
        g.manual_seed(8)
        xs = [torch.rand(Nf, generator=g, device=dev, dtype=torch.float32) * 0.45 for _ in range(4)]
        for k in range(16):                                    # 16 plateaus of 1 s: flat-top peaks of width 4096
            for x_ in xs:
                x_[(k + 1) * 3_500_003:(k + 1) * 3_500_003 + gs.FS] = 0.9
        hbm = peaks()[0].get("hbm_gbs", 6650.0)
        times = []
        for rep in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            npk, _ = gwi.find_peaks(xs[0], THETA, float(LMIN), capacity=4096, sync=False)
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1))
            npk = int(npk.item())
        ms = float(np.median(times[1:]))
        gbs = Nf * 4 / (ms * 1e-3) / 1e9
        out["find_peaks"] = {"workload": "gwi_find_peaks (SciPy find_peaks(height, width) rule) on 2^26 float32 probabilities of one model "
                                         "(268 MB > L2), height 0.5, width >= 2048",
                             "ms": ms, "peaks": npk, "bound": "hbm", "algorithmic_bytes": Nf * 4, "achieved_gb_per_s": gbs,
                             "peak_gb_per_s": hbm, "frac": gbs / hbm,
                             "note": "algorithmic bytes = one read of the array (level 1 of the pyramids and the candidate mask come from "
                                     "the same pass); the rest is 3-6 small launches on 3 % of the data"}
        ths = [0.30 + 0.01 * k for k in range(64)]
        gwi.threshold_sweep(xs, ths, LMIN)
        times = []
        for rep in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            cnts = gwi.threshold_sweep(xs, ths, LMIN)
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1))
        ms = float(np.median(times[1:]))
        gbs = 4 * Nf * 4 / (ms * 1e-3) / 1e9
        out["sweep"] = {"workload": "gwi_threshold_sweep: trigger counts at 64 thresholds in one pass over 4 x 2^26 float32 probabilities "
                                    "(1.07 GB > L2), L_min 2048", "ms": ms, "counts_at_0.5": int(cnts[20].item()), "bound": "hbm",
                        "algorithmic_bytes": 4 * Nf * 4, "achieved_gb_per_s": gbs, "peak_gb_per_s": hbm, "frac": gbs / hbm}
        del xs
    except Exception as ex:
        out["find_peaks"] = {"error": repr(ex)}
    # ---- whitening front end (NEXT-4): one 4096 s segment (2^24 samples) of one detector, raw fp32 -> fp16
    try:
        nw, nper = 1 << 24, 2 * gs.FS
        g = torch.Generator(device=dev)
        g.manual_seed(9)
        raw = torch.randn(nw, generator=g, device=dev, dtype=torch.float32) * 1e-21
        gwi.whiten(raw, nper)                                      # builds and caches the FFT plans
        times = []
        for rep in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            w = gwi.whiten(raw, nper)
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1))
        ms = float(np.median(times[1:]))
        hbm = peaks()[0].get("hbm_gbs", 6650.0)
        gbs = nw * (4 + 2) / (ms * 1e-3) / 1e9
        out["whiten"] = {"workload": "gwi_whiten: 2^24 raw fp32 samples (4096 s of one detector) -> whitened unit-variance fp16; Welch PSD "
                                     "(2 s Hann frames, 50 % overlap), division in the frequency domain (three cuFFT transforms, plans cached)",
                         "ms": ms, "strain_seconds_per_s": nw / gs.FS / (ms * 1e-3), "bound": "hbm",
                         "algorithmic_bytes": nw * 6, "achieved_gb_per_s": gbs, "peak_gb_per_s": hbm, "frac": gbs / hbm,
                         "note": "algorithmic bytes = 4 B in + 2 B out per sample; the path makes about 9 passes over the segment (statistics, "
                                 "framing, three transforms, division, scaling), so the fraction of a single-pass roofline is small by construction"}
        del raw, w
    except Exception as ex:
        out["whiten"] = {"error": repr(ex)}
    # ---- month, host -> device streaming
    st = gwi.Stream(models, n_chunks * N1, N1, THETA, LMIN, capacity=65536)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for c in range(n_chunks):
        h = host[c & 1]
        st.push(h[0], h[1])
    n, _ = st.finish()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    st.close()
    # the same chunk copies alone (no compute): what the pinned-buffer path can deliver
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage = torch.empty_like(xd)
    stage.copy_(host[0], non_blocking=True)
    torch.cuda.synchronize()
    e0.record()
    for c in range(10):
        stage.copy_(host[c & 1], non_blocking=True)
    e1.record()
    torch.cuda.synchronize()
    h2d_alone = 10 * N1 * 4 / (e0.elapsed_time(e1) * 1e-3) / 1e9
    out["month"] = {"workload": f"configs[4]: {n_chunks / 24:.0f} days x 4096 Hz x 2 detectors FP16 in {n_chunks} one-hour chunks from pinned host "
                                "memory (2 distinct seeded chunks rotating), 4-model ensemble + trigger clustering",
                    "wall_s": dt, "strain_seconds_per_s": n_chunks * 3600 / dt, "h2d_bytes": n_chunks * N1 * 2 * 2,
                    "h2d_gb_per_s": n_chunks * N1 * 4 / dt / 1e9,
                    "h2d_gb_per_s_copies_alone": h2d_alone,
                    "note": "compute-bound: the copies run on the stream handle's side stream under the kernels", "triggers": n}
    return out


def strong_bench(args, dev, work, rank, world):
    """--scaling strong: BASELINE.json configs[4] time-sharded over the ranks: the
    stream of --stream-chunks one-hour chunks is cut into `world` contiguous spans; rank r runs its span through its own
    gwi_stream handle in shard mode (R_f - 1 warm-up samples in front, chunks pushed from pinned host memory), the
    records that touch a span edge are gathered and joined on rank 0.  No collective on the data path.  Time = max over
    ranks of the wall time from the first push to the records on the host."""
    import torch
    import paper_2201_11133_b200 as gwi
    from paper_2201_11133_b200 import shard
    N1 = 3600 * gs.FS
    models = []
    for sd in range(4):
        pth = os.path.join(work, f"bench_cfg1_seed{sd}_r{rank}.gwim")
        gs.make_model_file(pth, gs.CFG1_ARCH, seed=sd)
        models.append(gwi.load_model(pth, gwi.FP16, dev.index))
    host = [torch.from_numpy(gs.stream_noise(1, c * N1, N1)).pin_memory() for c in range(2)]
    n_chunks = args.stream_chunks
    c0, c1 = shard.plan_windows(n_chunks, world)[rank]
    rf = models[0].receptive_field
    a = shard.shard_stream_args(n_chunks * N1, c0 * N1, c1 * N1, rf)
    warm = a["shard"][1]

    def run():
        st = gwi.Stream(models, a["n_total"], N1, THETA, LMIN, capacity=65536, shard=a["shard"])
        torch.cuda.synchronize()
        if world > 1:
            torch.distributed.barrier()
        t0 = time.perf_counter()
        if warm:
            prev = host[(c0 - 1) & 1]
            st.push(prev[0, N1 - warm:].contiguous().pin_memory(), prev[1, N1 - warm:].contiguous().pin_memory())
        for c in range(c0, c1):
            h = host[c & 1]
            st.push(h[0], h[1])
        n, recs = st.finish()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        st.close()
        return dt, [(r.slide, r.start, r.end, r.peak_p, r.mean_p, r.model_mask) for r in recs]

    run() if c1 - c0 <= 4 else None                                # warm-up pass only when it is cheap
    dt, recs = run()
    if world > 1:
        import torch.distributed as dist
        tt = torch.tensor([dt], device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        dt = float(tt.item())
        allrecs = [r for part in shard.gather_objects(recs, dist) for r in part]
    else:
        allrecs = recs
    if rank != 0:
        return
    merged = shard.merge_edge_records(allrecs, LMIN)
    line = {"metric": METRIC, "value": n_chunks * 3600 / dt, "unit": UNIT, "n_gpus": world, "steps": 1, "warmup": 0,
            "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f16",
            "data": "synthetic",
            "config": {"workload": f"configs[4] time-sharded: {n_chunks} one-hour chunks x 4096 Hz x 2 detectors FP16 from pinned host "
                                   "memory, 4-model ensemble (config-1 arch) + trigger clustering; contiguous spans per rank with "
                                   f"{rf - 1} warm-up samples, shard-edge runs joined on rank 0",
                       "chunks_per_rank": [c1_ - c0_ for c0_, c1_ in shard.plan_windows(n_chunks, world)],
                       "l2": "every chunk (59 MB) is streamed from host memory", "parallelism": f"time shards x{world} (strong)"},
            "triggers": len(merged)}
    print(json.dumps(line), flush=True)


def oracle_sample(model_path, x16, n_windows):
    """Times the oracle as it stands on the host cores over `n_windows` windows of the workload."""
    from oracle import gwo
    om = gwo.Model(model_path, round_fp16=True)
    xs = x16[:n_windows].astype(np.float64)
    t0 = time.perf_counter()
    p = om.infer_windows(xs)
    pb = gwo.ensemble_mean([p.reshape(-1)])
    gwo.triggers(pb, THETA, LMIN)
    dt = time.perf_counter() - t0
    return n_windows / dt, dt, gwo.num_threads()


def run_reference(args, model_path, x16):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import gwo
    nthreads = gwo.num_threads()
    nwin = max(1, min(nthreads, 16))
    times = []
    for i in range(args.warmup + args.steps):
        rate, dt, _ = oracle_sample(model_path, x16[(i * nwin) % 64:], nwin)
        if i >= args.warmup:
            times.append(dt)
    dt = float(np.mean(times))
    val = nwin / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[1] paper-scale single model, bounded sample", "windows_per_step": nwin, "T": T},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": nthreads, "kind": "oracle",
                             "sample": f"{nwin} windows x {T} samples per step (of the 1024-window batch)"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--windows", type=int, default=1024)
    ap.add_argument("--impl", default="gwi")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stream", action="store_true", help="skip the extra streaming-ensemble measurements")
    ap.add_argument("--stream-chunks", type=int, default=744, help="one-hour chunks of the month-long stream leg")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: every rank runs the configs[1] batch (headline); strong: the configs[4] stream time-sharded over the ranks")
    ap.add_argument("--paper-month", action="store_true",
                    help="also stream the month through the 4 x paper-scale ensemble, without and with 32 slides (about 7 minutes)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started without a launcher: start the N ranks here (one process per GPU, NCCL over NVLink for the plumbing)
        import socket
        sk = socket.socket()
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
        sk.close()
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])

    work = os.path.join(ROOT, "gpurun_out") if os.access(ROOT, os.W_OK) else "/tmp"
    os.makedirs(work, exist_ok=True)
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    model_path = os.path.join(work, f"bench_paper_seed0_r{rank}.gwim")
    gs.make_model_file(model_path, gs.PAPER_ARCH, seed=0)
    B = args.windows

    if args.impl == "reference":
        x16, _ = gs.cfg2_windows(seed=1, B=64, T=T)
        run_reference(args, model_path, x16)
        return

    import torch
    import paper_2201_11133_b200 as gwi
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the gwi library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    if args.scaling == "strong":
        strong_bench(args, dev, work, rank, world)
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- inputs: NROT different seeded batches so that the rotating working set exceeds L2 -------------------
    x_host = []
    for r in range(NROT):
        x, _ = gs.cfg2_windows(seed=1 + r + 100 * rank, B=B, T=T)
        x_host.append(torch.from_numpy(x).pin_memory())
    x_dev = [x.to(dev) for x in x_host]
    p_dev = [torch.empty((B, T), dtype=torch.float32, device=dev) for _ in range(NROT)]
    model = gwi.load_model(model_path, gwi.FP16, local_rank)
    flops_per_step = gs.PAPER_ARCH.flops_per_timestep() * B * T

    def step(i, timing=None):
        x, p = x_dev[i % NROT], p_dev[i % NROT]
        if timing is not None:
            timing[0].record()
        model.infer(x, out=p)
        if timing is not None:
            timing[1].record()
        cnt, trig, _ = gwi.ensemble_triggers([p.view(-1)], THETA, LMIN, capacity=4096, sync=False)
        return cnt

    def e2e_run(nsteps):
        """nsteps steps from pinned host buffers through the public API: every step's strain is copied host -> device on a
        side stream into one of two device buffers (the copy of step i+1 overlaps the compute of step i), and every
        step's trigger count and records are read back to the host before the next step's compute is enqueued."""
        cur = torch.cuda.current_stream()

        def issue_copy(i):
            b = i & 1
            with torch.cuda.stream(copy_stream):
                copy_stream.wait_event(buf_free[b])             # the compute that last read this buffer has finished
                xd2[b].copy_(x_host[i % NROT], non_blocking=True)
                h2d_done[b].record(copy_stream)

        for b in range(2):
            buf_free[b].record(cur)
        issue_copy(0)
        tot = 0
        for i in range(nsteps):
            b = i & 1
            if i + 1 < nsteps:
                issue_copy(i + 1)
            cur.wait_event(h2d_done[b])
            model.infer(xd2[b], out=pd2[b])
            buf_free[b].record(cur)
            cnt, trig, _ = gwi.ensemble_triggers([pd2[b].view(-1)], THETA, LMIN, capacity=4096, sync=False)
            cnt_host.copy_(cnt, non_blocking=True)              # D2H of the result
            trig_host.copy_(trig, non_blocking=True)
            cur.synchronize()
            tot += int(cnt_host.item())
        return tot

    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = gwi.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t_start.record()
    for i in range(args.steps):
        step(i, ev[i])
    t_end.record()
    torch.cuda.synchronize()
    launches = gwi.launch_count() - l0
    total_ms = t_start.elapsed_time(t_end)
    infer_ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    if world > 1:
        tt = torch.tensor([total_ms], device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())

    # ---- end to end through the public API with host buffers ------------------------------------------------
    xd2 = [torch.empty_like(x_dev[0]) for _ in range(2)]
    pd2 = [torch.empty_like(p_dev[0]) for _ in range(2)]
    copy_stream = torch.cuda.Stream(device=dev)
    h2d_done = [torch.cuda.Event() for _ in range(2)]
    buf_free = [torch.cuda.Event() for _ in range(2)]
    cnt_host = torch.zeros(1, dtype=torch.int32).pin_memory()
    trig_host = torch.zeros(4096 * 32, dtype=torch.uint8).pin_memory()
    e2e_run(2)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    e2e_run(args.steps)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    if world > 1:
        tt = torch.tensor([e2e_s], device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s = float(tt.item())
    sampler.stop_flag = True
    sampler.join(timeout=3)
    stream_extra = None
    if not args.no_stream and world == 1:
        try:
            stream_extra = stream_bench(dev, work, rank, args.stream_chunks, args.paper_month)
        except Exception as ex:  # the headline line must still come out
            stream_extra = {"error": repr(ex)}

    if rank != 0:
        return
    pk, pk_kind = peaks()
    ms_per_step = total_ms / args.steps
    value = world * B * args.steps / (total_ms * 1e-3)
    tflops = flops_per_step / (infer_ms * 1e-3) / 1e12
    # the timed region is a fraction of a second at near-maximum clocks: the burst figure is the denominator;
    # the sustained and the nominal ones are reported beside it
    peak_tf = pk["bf16_tflops"]
    traffic = profile_traffic()
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16",
        "data": "synthetic",
        "config": {"workload": "configs[1]: paper-scale SINGLE model (2x20 blocks, R64/S128, k2), FP16 operands / FP32 "
                               "accumulate, batch of windows x 4096 x 2, then mean/threshold/cluster; `value` is this model's "
                               "windows/s (1 window = 1 strain-second); the 4-model ensemble strain-seconds/s of configs[2]-[4] "
                               "are in `stream`",
                   "windows_per_gpu": B, "T": T, "threshold": THETA, "min_len": LMIN,
                   "l2": f"rotating {NROT} input+output buffer pairs ({NROT * B * T * 8 / 1e6:.0f} MB) > 126 MB L2",
                   "tensor_core_kernel": bool(model.uses_tensor_cores), "parallelism": f"replicas x{world} (weak)"},
        "clocks": sampler.summary(),
        "e2e": {"value": world * B * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": B * T * 2 * 2,
                "d2h_bytes_per_step": 4 + 4096 * 32,
                "how": "public API from pinned host buffers, wall clock; H2D of step i+1 on a side stream overlaps the compute of "
                       "step i (two device buffers); count + records read back every step"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "tensor", "achieved": tflops, "peak": peak_tf, "unit": "TFLOP/s", "frac": tflops / peak_tf,
                     "traffic": traffic, "traffic_note": f"dram__bytes_read.sum + dram__bytes_write.sum of k_stack per launch, read from {PROFILE_CSV} "
                     "(ncu --set full capture of this command, profiles/r2_k_stack.md)",
                     "peak_kind": f"bf16 cuBLAS burst (best of 10), {pk_kind}; fp16 = same tensor rate",
                     "frac_of_sustained": tflops / pk.get("bf16_tflops_sustained", peak_tf),
                     "peak_sustained": pk.get("bf16_tflops_sustained"), "frac_of_nominal_2250": tflops / 2250.0,
                     "kernel": "gwi_infer (k_stack + k_head_tc of one call)", "flops_per_launch": flops_per_step,
                     "infer_ms": infer_ms},
    }
    if stream_extra is not None:
        line["stream"] = stream_extra
    if not args.no_cpu_baseline and world == 1:
        nthreads = os.cpu_count() or 1
        nwin = max(1, min(3 * nthreads, 48))
        rate, dt, cores = oracle_sample(model_path, x_host[0].numpy(), nwin)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{nwin} windows x {T} samples of the same batch, {dt:.1f} s"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
