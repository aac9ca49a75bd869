#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

A "step" is one pass of the whole hot path (tred_drift, tred_blockbin, tred_effq,
tred_convolve_plan, tred_convolve, tred_gather_waveforms) over one synthetic spill.
N = 1 workload: BASELINE.json's third config, the full beam spill in one module that the
metric "ms per spill" is quoted on (~0.93 M 1-mm segments, 230x230 pixels x 5000 ticks,
4-point Gauss-Legendre, blocks 16x16x128, response 11x11 x 100 phases x 400 ticks); it fits
one GPU (56 GB).  `--config 1|2|4` select the other workloads, `--config 5` the
representation sweep with the dense-grid comparison.  N > 1: every rank simulates its own
spill of the same recipe (seed 1003 + rank): the path shards over independent events with
no collective ("weak").
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample instead.
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
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import gen  # noqa: E402

METRIC = "segments_per_s"
UNIT = "segments/s"
FMA_LANES_PER_SM = 128          # fp32 FMA lanes per SM (4 SMSPs x 32), B300_MICROARCH.md


def _env_int(k, d):
    try:
        return int(os.environ.get(k, d))
    except ValueError:
        return d


def workload(cfg_id: int, rank: int):
    from paper_2602_12052_b200.shard import event_seed
    cfg, segs = gen.make_segments(cfg_id, seed=event_seed(cfg_id, rank))
    R = gen.make_response(cfg, 2000 + cfg_id)
    seg = np.ascontiguousarray(np.stack([segs[k] for k in gen.SEG_FIELDS]).astype(np.float32))
    return cfg, segs, seg, R


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi sampled during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100", "-i", str(self.index)],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=2)
        except Exception:
            self.p.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def _load_traffic(workload_name: str) -> dict:
    """DRAM bytes per step and stage from the committed ncu --set full capture
    (profiles/traffic.csv: workload,stage,dram_bytes_per_step); {} if there is none."""
    out = {}
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 3 and p[0] == workload_name:
                    out[p[1]] = float(p[2])
    except (OSError, ValueError):
        pass
    return out


# --------------------------------------------------------------------------- oracle legs
def oracle_sample(cfg, segs, R, n_sample: int):
    """The oracle as it stands on the first n_sample segments: whole path, every pixel of
    its output footprint.  Returns (segments, seconds, threads)."""
    import oracle as o
    sub = {k: v[:n_sample] for k, v in segs.items()}
    t0 = time.perf_counter()
    aug = o.drift(cfg, sub)
    keys = o.blocks(cfg, aug)
    payload = o.effq(cfg, aug, keys)
    tiles = o.out_tiles(cfg, keys)
    pix = np.unique(tiles % (cfg.npix_x * cfg.npix_y))
    o.conv_fft(cfg, keys, payload, R, pix)
    dt = time.perf_counter() - t0
    return len(sub["q"]), dt, os.cpu_count()


REF_SEGMENTS = {1: 60, 2: 40, 3: 8, 4: 8}      # ~20 s of oracle work on 8-16 host cores


def _ref_segments(args):
    return args.ref_segments or REF_SEGMENTS.get(args.config, 8)


def run_reference(args):
    rank = _env_int("RANK", 0)
    if rank != 0:
        return 0
    cfg, segs, seg, R = workload(args.config, 0)
    n_sample = _ref_segments(args)
    for _ in range(args.warmup and 1):
        oracle_sample(cfg, segs, R, max(2, n_sample // 8))
    times = []
    for _ in range(args.steps):
        n, dt, cores = oracle_sample(cfg, segs, R, n_sample)
        times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = n / (ms * 1e-3)
    sample = f"first {n} segments of config {args.config}, whole path, all pixels of their footprint"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2602_12052_b200 import Tred

    world = _env_int("WORLD_SIZE", 1)
    rank = _env_int("RANK", 0)
    local = _env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg, segs, seg_h, R = workload(args.config, rank)
    if args.mac_mode:
        cfg = cfg.with_(mac_mode=args.mac_mode)
    nseg = seg_h.shape[1]
    sim = Tred(cfg, device=dev, conv_work_bytes=args.work_gb << 30 if args.work_gb else None)
    rhat = sim.prepare_response(torch.from_numpy(R).to(dev))       # once per response
    seg_d = torch.from_numpy(seg_h).to(dev)
    seg_pinned = torch.from_numpy(seg_h).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # config 4: device-memory-bounded chunks of occupied blocks (peak <= 40 GB)
    if args.config == 4:
        sim.conv_work_bytes = (args.work_gb or 5) << 30

        def simulate(s):
            return sim.simulate_chunked(s, rhat, payload_budget_bytes=args.budget_gb << 30)
    else:
        def simulate(s):
            return sim.simulate(s, rhat)

    # ---- warm-up
    out = None
    for _ in range(max(args.warmup, 3)):
        out = None                          # a step's outputs are released before the next step
        out = simulate(seg_d)
    barrier()
    info = {k: out[k] for k in ("npairs", "nblocks", "ncp", "nsp", "ntiles", "nrt")}
    # Gauss-Legendre node evaluations of one step = cuboids of every bounding box x n^3
    _, augi0, _ = sim.drift(seg_d)
    ext = (augi0[3:6] - augi0[0:3] + 1).to(torch.float64)
    info["gl_nodes"] = float((ext[0] * ext[1] * ext[2]).sum().item()) * cfg.gl_n ** 3

    # ---- timed region 1: inputs resident in HBM, device time by CUDA events
    sampler = ClockSampler(local)
    sampler.start()
    sim.profile_begin(events=False)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_wall0 = time.perf_counter()
    torch.cuda.reset_peak_memory_stats(dev)
    for a, b in ev:
        out = None
        flush.zero_()                       # flush L2 between timed iterations
        a.record()
        out = simulate(seg_d)
        b.record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    peak_mem = torch.cuda.max_memory_allocated(dev)
    nchunks = len(out.get("chunks", [])) or 1
    out = None
    launches = sum(v[1] for v in sim.profile_end().values())
    ms_steps = [a.elapsed_time(b) for a, b in ev]
    ms = float(np.mean(ms_steps))

    # ---- timed region 2: per-stage events (roofline of the dominant kernel)
    stage_ms = {}
    stage_prof_last = {}
    for _ in range(args.steps):
        flush.zero_()
        sim.profile_begin(events=True)
        simulate(seg_d)
        torch.cuda.synchronize()
        stage_prof_last = sim.profile_end()
        for k, (m, n) in stage_prof_last.items():
            stage_ms[k] = stage_ms.get(k, 0.0) + m / args.steps
    barrier()

    # ---- timed region 3: end to end through the public API with HOST buffers: segments from
    # pinned host memory in, tile keys and waveform tiles back to pinned host memory
    e2e_ms = []
    h2d = seg_pinned.numel() * 4
    d2h = 0
    o2 = None
    nt_cap = int(info["ntiles"] * 1.05) + 1024
    keys_h = torch.empty((nt_cap,), dtype=torch.int64).pin_memory()
    data_h = torch.empty((nt_cap, cfg.block[2]), dtype=torch.float32).pin_memory()
    for i in range(args.steps + 1):
        o2 = None
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sd = seg_pinned.to(dev, non_blocking=True)
        o2 = simulate(sd)
        nt = o2["ntiles"]
        if nt > nt_cap:                     # cannot happen for a fixed workload; keep the copy honest anyway
            keys_h = torch.empty((nt,), dtype=torch.int64).pin_memory()
            data_h = torch.empty((nt, cfg.block[2]), dtype=torch.float32).pin_memory()
            nt_cap = nt
        keys_h[:nt].copy_(o2["tile_keys"], non_blocking=True)
        data_h[:nt].copy_(o2["tile_data"], non_blocking=True)
        torch.cuda.synchronize()
        if i > 0:
            e2e_ms.append(1e3 * (time.perf_counter() - t0))
        d2h = nt * 8 + nt * cfg.block[2] * 4
    e2e = float(np.mean(e2e_ms))
    o2 = None
    barrier()

    # ---- max over ranks of the times, sum of the units (paper_2602_12052_b200/shard.py)
    from paper_2602_12052_b200.shard import reduce_timing
    (ms_max, e2e_max), total_seg = reduce_timing([ms, e2e], nseg, device=dev)

    if rank == 0:
        d = sim.dims
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        # per-stage rooflines: algorithmic work of the METHOD per step
        # / CUDA-event time of the stage, against the measured peaks
        nb = info["nblocks"]
        ncols = cfg.block[0] * cfg.block[1]
        K = 2 * cfg.resp_half + 1
        nf, L = d.n_freq, d.fft_len
        sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        hbm = peaks.get("hbm_gbs", 6650.0)
        hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650"
        alu_peak = 148 * FMA_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12          # fp32 TFLOP/s at max clock
        tf32_peak = peaks.get("bf16_tflops", 1590.0) * 0.5                     # guide: tf32 = bf16 / 2 nominal
        fftf = 2.5 * L * np.log2(L)                                            # flops of one real FFT of length L
        payload_b = nb * d.block_floats * 4.0
        spd_b = info["nsp"] * d.n_over * cfg.block[2] * 4.0
        work = {
            "effq": ("hbm", payload_b + nseg * 104.0),
            "fft_fwd": ("alu", nb * ncols * fftf),
            "mac": ("tensor" if sim.cfg.mac_mode != 1 else "alu", nb * ncols * K * K * (8.0 * (nf - 1) + 4.0)),
            "accum": ("hbm", info["nsp"] * nf * 8.0),
            "ifft": ("alu", info["nsp"] * fftf),
            "gather": ("hbm", spd_b + info["ntiles"] * cfg.block[2] * 4.0),
        }
        pk = {"hbm": (hbm, "GB/s", 1e9, hbm_src),
              "alu": (alu_peak, "TFLOP/s", 1e12, "derived: 148 SM x 128 lanes x 2 x sm_max_mhz (DESIGN.md)"),
              "tensor": (tf32_peak, "TFLOP/s", 1e12,
                         "tf32 dense = measured bf16_tflops x 1/2 (nominal ratio); the kernel executes one tf32 "
                         "and two bf16 products per algorithmic fp32 product (2 tf32-equivalents), so 1/2 "
                         "is its ceiling")}
        nlaunch = {k: v[1] for k, v in stage_prof_last.items()}
        traffic = _load_traffic(cfg.name)
        stage_roof = {}
        for k, (bound, w) in work.items():
            if stage_ms.get(k, 0.0) <= 0:
                continue
            peak, unit, sc, src = pk[bound]
            nl = max(nlaunch.get(k, 1), 1)
            ach = w / (stage_ms[k] * 1e-3) / sc
            tr = traffic.get(k)
            stage_roof[k] = {"kernel": k, "bound": bound, "achieved": ach, "peak": peak, "unit": unit,
                             "frac": ach / peak, "ms_per_launch": stage_ms[k] / nl, "launches_per_step": nl,
                             "work_per_launch": w / nl, "peak_source": src,
                             "traffic": (tr / nl) if tr else None}
        if "mac" in stage_roof and stage_roof["mac"]["bound"] == "tensor":
            # what the tensor cores execute: 3 products per fp32 product (tf32-equivalent: the two
            # bf16 correction products of the default mode run at twice the tf32 rate and count
            # half), row tiles of 128 rows (partly filled), 2 x 128 output columns for 2 x 121 offsets
            nprod = 3.0 if sim.cfg.mac_mode in (2, 3, 4, 5) else 2.0
            ex = nprod * 2.0 * info["nrt"] * 128 * (2 * d.n_off_pad) * (2 * d.n_phase) * nf
            stage_roof["mac"]["executed_tflops"] = ex / (stage_ms["mac"] * 1e-3) / 1e12
            stage_roof["mac"]["executed_frac"] = stage_roof["mac"]["executed_tflops"] / tf32_peak
        dom = max(stage_roof, key=lambda k: stage_ms[k])
        roof = dict(stage_roof[dom])
        payload_gb = nb * d.block_floats * 4 / 1e9
        line = {"metric": METRIC, "value": total_seg / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_max,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": cfg.name, "segments_per_event": nseg, "events": world,
                           "pixels": [cfg.npix_x, cfg.npix_y], "nticks": cfg.nticks, "gl_n": cfg.gl_n,
                           "block": list(cfg.block), "resp_nticks": cfg.resp_nticks, "fft_len": d.fft_len,
                           "l2": "flushed between timed iterations (256 MiB write)",
                           "parallelism": f"events x{world}, no collective",
                           "chunks": nchunks, **info},
                "e2e": {"value": total_seg / (e2e_max * 1e-3), "unit": UNIT, "ms_per_step": e2e_max,
                        "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
                "gpu_launches": int(launches),
                "clocks": clocks,
                "stage_ms": {k: round(v, 4) for k, v in stage_ms.items() if v > 0},
                "roofline": roof,
                "stage_roofline": {k: {kk: (round(vv, 6) if isinstance(vv, float) else vv)
                                       for kk, vv in v.items() if kk in ("bound", "achieved", "peak", "unit", "frac",
                                                                          "traffic", "executed_tflops",
                                                                          "executed_frac")}
                                   for k, v in stage_roof.items()},
                "peak_mem_gb": peak_mem / 1e9,
                "payload_gb": payload_gb,
                "wall_s_timed_region": t_wall}
        if not args.no_cpu_baseline and world == 1:
            n, dt, cores = oracle_sample(cfg, segs, R, _ref_segments(args))
            line["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"first {n} segments of config {args.config}, whole path, "
                                              f"all pixels of their footprint ({dt:.1f} s)"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# --------------------------------------------------------------------------- config 5
def dense_grid_convolution(torch, cfg, keys, payload, R_d, pix_ids):
    """Comparison point of BASELINE config 5: FFT convolution of the WHOLE plane on the
    dense grid (no block sparsity), one sub-pixel phase at a time (Eq. (14) with the 3-D
    FFT over pixel x pixel x time), with torch.fft (cuFFT): a timed
    comparison only, not the product path.  Returns (dense rows for pix_ids, ms, peak bytes)."""
    dev = payload.device
    S, H, Tr = cfg.sub, cfg.resp_half, cfg.resp_nticks
    Bx, By, Bt = cfg.block
    NBx, NBy = -(-cfg.npix_x * S // Bx), -(-cfg.npix_y * S // By)
    NBt = -(-cfg.nticks // Bt)
    K = 2 * H + 1
    nx, ny, nt = cfg.npix_x + K - 1, cfg.npix_y + K - 1, NBt * Bt + Tr - 1
    nt += nt & 1
    torch.cuda.reset_peak_memory_stats(dev)
    base = torch.cuda.memory_allocated(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    nb = keys.numel()
    bmap = torch.full((NBt * NBx * NBy,), nb, dtype=torch.int64, device=dev)      # nb = the zero block
    bmap[keys] = torch.arange(nb, device=dev)
    bmap = bmap.view(NBt, NBx, NBy)
    pay = torch.cat([payload.view(nb, Bx, By, Bt), torch.zeros((1, Bx, By, Bt), device=dev)])
    px = torch.arange(cfg.npix_x, device=dev)
    py = torch.arange(cfg.npix_y, device=dev)
    acc = None
    for jx in range(S):
        ix = px * S + jx
        for jy in range(S):
            iy = py * S + jy
            slot = bmap[:, (ix // Bx)[:, None], (iy // By)[None, :]]                # [NBt][npx][npy]
            q = pay[slot, (ix % Bx)[None, :, None], (iy % By)[None, None, :], :]     # [NBt][npx][npy][Bt]
            q = q.permute(1, 2, 0, 3).reshape(cfg.npix_x, cfg.npix_y, NBt * Bt)
            qh = torch.fft.rfftn(q, s=(nx, ny, nt))
            rh = torch.fft.rfftn(R_d[jx, jy], s=(nx, ny, nt))
            acc = qh * rh if acc is None else acc.addcmul_(qh, rh)
            del q, qh, rh, slot
    out = torch.fft.irfftn(acc, s=(nx, ny, nt))[H:H + cfg.npix_x, H:H + cfg.npix_y, :cfg.nticks]
    rows = out.reshape(cfg.npix_x * cfg.npix_y, cfg.nticks)[pix_ids.long()].contiguous()
    e1.record()
    torch.cuda.synchronize()
    return rows, e0.elapsed_time(e1), torch.cuda.max_memory_allocated(dev) - base


def run_sweep(args):
    """BASELINE config 5: block shapes x Gauss-Legendre orders on config-3 inputs, one JSON
    line each (ms per spill, peak GB, occupied-block fraction), then the dense-grid line."""
    import torch
    from paper_2602_12052_b200 import Tred
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    cfg0, segs, seg_h, R = workload(3, 0)
    seg_d = torch.from_numpy(seg_h).to(dev)
    R_d = torch.from_numpy(R).to(dev)
    steps = max(1, min(args.steps, 3))
    for block in ((4, 4, 32), (8, 8, 64), (16, 16, 128), (32, 32, 256)):
        for n in (1, 2, 3, 4):
            cfg = cfg0.with_(block=block, gl_n=n)
            torch.cuda.empty_cache()
            torch.cuda.reset_peak_memory_stats(dev)
            sim = Tred(cfg, device=dev)
            rhat = sim.prepare_response(R_d)
            out = sim.simulate(seg_d, rhat)                      # warm-up
            ms = []
            for _ in range(steps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                out = sim.simulate(seg_d, rhat)
                b.record()
                torch.cuda.synchronize()
                ms.append(a.elapsed_time(b))
            d = sim.dims
            nb_all = int(d.NB[0] * d.NB[1] * d.NB[2])
            print(json.dumps({"sweep": "block x gl_n", "workload": cfg0.name, "block": list(block), "gl_n": n,
                              "fft_len": d.fft_len, "ms_per_spill": float(np.mean(ms)),
                              "segments_per_s": seg_h.shape[1] / (float(np.mean(ms)) * 1e-3),
                              "nblocks": out["nblocks"], "occupied_block_fraction": out["nblocks"] / nb_all,
                              "payload_gb": out["nblocks"] * d.block_floats * 4 / 1e9,
                              "peak_gb": torch.cuda.max_memory_allocated(dev) / 1e9}), flush=True)
            del sim, rhat, out
    # dense-grid comparison on the config-3 representation
    cfg = cfg0
    torch.cuda.empty_cache()
    sim = Tred(cfg, device=dev)
    rhat = sim.prepare_response(R_d)
    rng = np.random.default_rng(5)
    pix = torch.from_numpy(np.sort(rng.choice(cfg.npix_x * cfg.npix_y, 64, replace=False)).astype(np.int32)).to(dev)
    out = sim.simulate(seg_d, rhat, pix_ids=pix, keep=True)
    sparse_rows = out["dense"]
    keys, payload = out["keys"].clone(), out["payload"].clone()
    del out, rhat
    sim._work.clear()
    torch.cuda.empty_cache()
    rows, ms, peak = dense_grid_convolution(torch, cfg, keys, payload, R_d, pix)      # warm-up (cuFFT plans)
    rows, ms, peak = dense_grid_convolution(torch, cfg, keys, payload, R_d, pix)
    err = float((rows - sparse_rows).abs().max() / sparse_rows.abs().max())
    print(json.dumps({"sweep": "dense grid", "workload": cfg.name, "impl": "torch.fft (cuFFT), comparison only",
                      "ms_per_spill_convolution_only": ms, "peak_gb_convolution_only": peak / 1e9,
                      "dense_fine_grid_gb_if_materialised": cfg.npix_x * cfg.npix_y * cfg.sub ** 2 * cfg.nticks * 4 / 1e9,
                      "max_abs_diff_vs_block_sparse_over_max": err, "pixels_compared": int(pix.numel())}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--ref-segments", type=int, default=0, help="oracle sample size (0 = per config)")
    ap.add_argument("--work-gb", type=int, default=0, help="tred_convolve workspace cap (GiB), 0 = default")
    ap.add_argument("--budget-gb", type=int, default=7, help="config 4: block payload per chunk (GiB)")
    ap.add_argument("--mac-mode", type=int, default=0, help="tred_config.mac_mode (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.config == 5:
        return run_sweep(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
