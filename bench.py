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


def csrc_sha() -> str:
    """sha1 over the CUDA sources and the header: the code state a profile belongs to."""
    import hashlib
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2602_12052_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    h.update(open(os.path.join(ROOT, "include", "tred.h"), "rb").read())
    return h.hexdigest()[:16]


def _load_traffic(workload_name: str):
    """DRAM bytes per step and stage from the committed ncu --set full capture
    (profiles/traffic.csv: a `# csrc_sha=<hash>` line, then workload,stage,dram_bytes_per_step).
    The capture belongs to one state of the kernels: if csrc/ has changed since, the numbers
    are refused ({} and the reason)."""
    out, sha = {}, None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                if line.startswith("#"):
                    if "csrc_sha=" in line:
                        sha = line.split("csrc_sha=")[1].split()[0]
                    continue
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 3 and p[0] == workload_name:
                    out[p[1]] = float(p[2])
    except (OSError, ValueError):
        return {}, "no profiles/traffic.csv"
    if sha != csrc_sha():
        return {}, f"profiles/traffic.csv was captured at csrc_sha {sha}, the sources are now {csrc_sha()}: refused"
    return out, f"ncu --set full capture at csrc_sha {sha} (profiles/traffic.csv)"


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
MAC_KERNELS = {   # tred_last_mac_mode -> (arithmetic of the spectrum product, tensor-core products per fp32 product,
                  #                        rate of those products relative to the bf16 / fp16 dense peak)
    1: ("fp32 FMA", 0, 0.0),
    2: ("3xTF32 split (tf32 tensor cores, fp32 accumulate), products in memory", 3.0, 0.5),
    3: ("3xTF32 split (tf32 tensor cores, fp32 accumulate)", 3.0, 0.5),
    4: ("3xTF32 split on mirror-pair sums / differences", 1.5, 0.5),
    5: ("3xTF32 split (tf32 tensor cores, fp32 accumulate)", 3.0, 0.5),
    6: ("tf32 + 2 x bf16 split (fp32 accumulate)", 2.0, 0.5),
    7: ("3 x fp16 split, x = s (hi + lo) with power-of-two scales (fp32 accumulate)", 3.0, 1.0),
}


def measure(args, cfg_id, rank, world, dev, steps, stages: bool):
    """Times one workload: device-resident inputs (CUDA events), per-stage events, and end to
    end through tred_simulate with pinned HOST buffers on both sides."""
    import torch
    import torch.distributed as dist
    from paper_2602_12052_b200 import Tred

    cfg, segs, seg_h, R = workload(cfg_id, rank)
    if args.mac_mode:
        cfg = cfg.with_(mac_mode=args.mac_mode)
    nseg = seg_h.shape[1]
    conv_cap = None
    budget = 0
    if cfg_id == 4:                         # device-memory-bounded chunks of occupied blocks (peak <= 40 GB)
        conv_cap = (args.work_gb or 5) << 30
        budget = args.budget_gb << 30
    elif args.work_gb:
        conv_cap = args.work_gb << 30
    sim = Tred(cfg, device=dev, conv_work_bytes=conv_cap)
    rhat = sim.prepare_response(torch.from_numpy(R).to(dev))       # once per response
    seg_d = torch.from_numpy(seg_h).to(dev)
    seg_pinned = torch.from_numpy(seg_h).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def simulate(s, **kw):
        return sim.simulate(s, rhat, payload_budget_bytes=budget, **kw)

    out = None
    for _ in range(max(args.warmup, 3)):
        out = None                          # a step's outputs are released before the next step
        out = simulate(seg_d)
    barrier()
    info = {k: out[k] for k in ("npairs", "nblocks", "ncp", "nsp", "ntiles", "nrt", "nchunks", "host_reads")}
    mac_mode = out["mac_mode"]

    # ---- timed region 1: inputs resident in HBM, device time by CUDA events
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    sim.profile_begin(events=False)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
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
    out = None
    launches = sum(v[1] for v in sim.profile_end().values())
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))

    # ---- timed region 2: per-stage events
    stage_ms, stage_n = {}, {}
    if stages:
        for _ in range(steps):
            flush.zero_()
            sim.profile_begin(events=True)
            simulate(seg_d)
            torch.cuda.synchronize()
            for k, (m, n) in sim.profile_end().items():
                stage_ms[k] = stage_ms.get(k, 0.0) + m / steps
                stage_n[k] = n
        barrier()

    # ---- timed region 3: end to end through the C-ABI call with HOST buffers: segments from
    # pinned host memory in, tile keys and waveform tiles written to pinned host memory
    nt_cap = int(info["ntiles"] * 1.05) + 1024
    keys_h = torch.empty((nt_cap,), dtype=torch.int64).pin_memory()
    data_h = torch.empty((nt_cap, cfg.block[2]), dtype=torch.float32).pin_memory()
    e2e_ms = []
    for i in range(steps + 1):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        o2 = simulate(seg_pinned, host_out=(keys_h, data_h))
        torch.cuda.synchronize()
        if i > 0:
            e2e_ms.append(1e3 * (time.perf_counter() - t0))
    e2e = float(np.mean(e2e_ms))
    h2d = seg_pinned.numel() * 4
    d2h = o2["ntiles"] * 8 + o2["ntiles"] * cfg.block[2] * 4
    barrier()
    return dict(cfg=cfg, segs=segs, R=R, sim=sim, nseg=nseg, info=info, mac_mode=mac_mode, ms=ms, e2e=e2e, h2d=h2d,
                d2h=d2h, launches=int(launches) // max(steps, 1), clocks=clocks, peak_mem=peak_mem, t_wall=t_wall,
                stage_ms=stage_ms, stage_n=stage_n, seg_d=seg_d, rhat=rhat)


def cufft_s4_comparison(torch, m, rows_sample: int = 8192):
    """Timed comparison only (north_star (d); PAPER.md:L230, L264 is this form): S4 with library
    FFTs -- torch.fft.rfft (cuFFT) of the zero-padded time columns of a sample of charge pixels,
    the per-frequency product with the precomputed response spectrum as a batched complex
    matrix product (cuBLAS), the inverse cuFFT of the products -- extrapolated to the event by
    the number of charge pixels.  The overlap-add over the offsets is not included (lower bound)."""
    cfg, sim, info = m["cfg"], m["sim"], m["info"]
    dev = m["seg_d"].device
    d = sim.dims
    L, nph, noff = d.fft_len, d.n_phase, d.n_off
    n = min(rows_sample, max(info["ncp"], 1))
    q = torch.rand((n, nph, cfg.block[2]), dtype=torch.float32, device=dev)       # same shape as the payload columns
    W = torch.randn((L // 2 + 1, nph, noff), dtype=torch.complex64, device=dev)    # stands in for FFT(R^j), precomputed
    ms = []
    for i in range(4):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        qh = torch.fft.rfft(q, n=L, dim=2)                            # [n][phase][f]
        T = torch.matmul(qh.permute(2, 0, 1), W)                      # [f][n][off]
        o = torch.fft.irfft(T.permute(1, 2, 0), n=L, dim=2)          # [n][off][L]
        b.record()
        torch.cuda.synchronize()
        if i > 0:
            ms.append(a.elapsed_time(b))
        del qh, T, o
    per_row = float(np.mean(ms)) / n
    return {"impl": "torch.fft.rfft (cuFFT) + batched complex matmul (cuBLAS) + torch.fft.irfft, comparison only",
            "rows_sampled": n, "ms_sample": float(np.mean(ms)), "ms_per_spill_extrapolated": per_row * info["ncp"],
            "not_included": "overlap-add over the offsets, gather of the payload columns"}


def next_rows_overhead(torch, m, ms_step):
    """SURVEY 8(f) rows timed on the same workload, as overhead over one step (context: the paper
    quotes +5-10 % for truth provenance): the truth record of every segment
    (tred_truth, counting pass + fill) and the trigger-reset readout of the whole pixel plane."""
    from paper_2602_12052_b200 import readout
    sim, cfg = m["sim"], m["cfg"]
    augf, augi, _ = sim.drift(m["seg_d"])

    def timed(fn, n=3):
        fn()
        ms = []
        for _ in range(n):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); b.synchronize()
            ms.append(a.elapsed_time(b))
        return float(np.mean(ms))
    nrec = [0]

    def truth():
        nrec[0] = int(sim.truth(augf, augi)[3].item())
    t_truth = timed(truth)
    out = {"truth_record_ms": t_truth, "truth_records": nrec[0], "truth_overhead": t_truth / ms_step}
    del augf, augi
    npix = cfg.npix_x * cfg.npix_y
    if npix * cfg.nticks * 4 <= (8 << 30):
        pix = torch.arange(npix, dtype=torch.int32, device=m["seg_d"].device)
        dense = sim.simulate(m["seg_d"], m["rhat"], pix)["dense"]
        par = dict(threshold_e=5000.0, n_integ=16, n_reset=8, max_hits=16, adc_lsb_e=0.0)
        hits = [0]

        def ro():
            hits[0] = int(readout(dense, par)[0].sum().item())
        t_ro = timed(ro)
        out.update({"readout_ms": t_ro, "readout_channels": npix, "readout_hits": hits[0], "readout_overhead": t_ro / ms_step})
        del dense
    return out


def slab_pair_statistics(torch, m):
    """Plan statistics for the transform length (PAPER.md:L264 pads every
    block on its own): the share of charge pixels (time slab bt, pixel) whose pixel is also
    occupied in slab bt + 1.  Greedily pairing such neighbours into one transform of 2 Bt ticks
    (L2 = fft length of 2 Bt + Tr - 1) instead of two of L would change the spectrum bytes and
    product flops by the factor reported.  Integer work on the plan's keys only."""
    sim, cfg = m["sim"], m["cfg"]
    augf, augi, npairs = sim.drift(m["seg_d"])
    k, blk_off, pair_seg, slab_off, nblocks = sim.blockbin(augi, int(npairs.item()))
    nb = int(nblocks.item())
    p = sim.convolve_plan(nb, k)
    ncp = int(p["ncp"].item())
    cp = p["cp_keys"][:ncp]
    npix = cfg.npix_x * cfg.npix_y
    has_next = torch.isin(cp + npix, cp)
    # greedy pairing along time per pixel: runs of consecutive slabs of one pixel, floor(len / 2) pairs
    pix, bt = cp % npix, cp // npix
    order = torch.argsort(pix * (int(sim.dims.NB[2]) + 1) + bt)
    ps, bs = pix[order], bt[order]
    brk = torch.ones_like(ps, dtype=torch.bool)
    brk[1:] = (ps[1:] != ps[:-1]) | (bs[1:] != bs[:-1] + 1)
    run_id = torch.cumsum(brk.to(torch.int64), 0) - 1
    run_len = torch.bincount(run_id)
    pairs = int((run_len // 2).sum().item())
    singles = ncp - 2 * pairs

    def fft_len(n):
        best = None
        a = 8
        while a < 4 * n:
            b = a
            while b < 4 * n:
                if b >= n and (best is None or b < best):
                    best = b
                b *= 3
            a *= 2
        return best
    Bt, Tr = cfg.block[2], cfg.resp_nticks
    L1, L2 = fft_len(Bt + Tr - 1), fft_len(2 * Bt + Tr - 1)
    return {"charge_pixels": ncp, "with_occupied_next_slab": float(has_next.float().mean().item()),
            "greedy_pairs": pairs, "singles": singles, "L": L1, "L_two_slabs": L2,
            "spectrum_bytes_factor_if_paired": (pairs * L2 + singles * L1) / (ncp * L1)}


def run_cuda(args):
    import torch
    import torch.distributed as dist

    world = _env_int("WORLD_SIZE", 1)
    rank = _env_int("RANK", 0)
    local = _env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    m = measure(args, args.config, rank, world, dev, args.steps, stages=True)
    cfg, sim, info, nseg = m["cfg"], m["sim"], m["info"], m["nseg"]
    stage_ms, clocks = m["stage_ms"], m["clocks"]
    fma_tflops = sim.bench_fma()                                   # measured fp32 FMA rate of this device
    # Gauss-Legendre node evaluations of one step = cuboids of every bounding box x n^3
    _, augi0, _ = sim.drift(m["seg_d"])
    ext = (augi0[3:6] - augi0[0:3] + 1).to(torch.float64)
    info["gl_nodes"] = float((ext[0] * ext[1] * ext[2]).sum().item()) * cfg.gl_n ** 3
    del augi0, ext

    # ---- max over ranks of the times, sum of the units (paper_2602_12052_b200/shard.py)
    from paper_2602_12052_b200.shard import reduce_timing
    (ms_max, e2e_max), total_seg = reduce_timing([m["ms"], m["e2e"]], nseg, device=dev)

    if rank == 0:
        d = sim.dims
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        # per-stage rooflines: ALGORITHMIC work of the method per step
        # / CUDA-event time of the stage, against the measured peaks; `own_*`:
        # the bytes this design moves in the stage (its intermediates included)
        nb = info["nblocks"]
        ncols = cfg.block[0] * cfg.block[1]
        K = 2 * cfg.resp_half + 1
        nf, L, Bt = d.n_freq, d.fft_len, cfg.block[2]
        hbm = peaks.get("hbm_gbs", 6650.0)
        hbm_src = "measured copy bandwidth (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"
        # tensor peak of the dtype the product runs in; the kernel is timed inside a long step: sustained figure
        bf16 = peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops", 1590.0))
        bf16_src = ("measured cuBLAS bf16, sustained (MEASURED_PEAKS.json bf16_tflops_sustained)"
                    if "bf16_tflops_sustained" in peaks else "fallback")
        mac_name, nprod, rel_rate = MAC_KERNELS.get(m["mac_mode"], ("?", 0, 0.0))
        fftf = 2.5 * L * np.log2(L)                                            # flops of one real FFT of length L
        payload_b = nb * d.block_floats * 4.0
        rows_pad = info["nrt"] * 128
        row_b = max(d.n_phase * 8, ((2 * d.n_phase + 15) // 16) * 32 * 2)      # a row of spectra: fp32 complex or fp16 hi/lo
        qhat_b = rows_pad * nf * row_b * 1.0
        opart_b = info["nrt"] * nf * (8 + 2 * cfg.resp_half) * 64 * 8.0
        ohat_b = info["nsp"] * nf * 8.0
        spd_b = info["nsp"] * d.n_over * Bt * 4.0
        tiles_b = info["ntiles"] * Bt * 4.0
        mac_flops = nb * ncols * K * K * (8.0 * (nf - 1) + 4.0)
        work = {   # stage: (bound, algorithmic work, own bytes)
            "effq": ("hbm", payload_b + nseg * 104.0, payload_b + nseg * 104.0),
            "fft_fwd": ("hbm", payload_b, payload_b + qhat_b),
            "mac": ("tensor" if nprod else "alu", mac_flops, qhat_b + opart_b),
            "accum": ("hbm", ohat_b, opart_b + 2 * ohat_b),
            "ifft": ("hbm", ohat_b + spd_b, ohat_b + spd_b),
            "gather": ("hbm", spd_b + tiles_b, spd_b + tiles_b),
        }
        pk = {"hbm": (hbm, "GB/s", 1e9, hbm_src),
              "alu": (fma_tflops, "TFLOP/s", 1e12, "measured in this run: tred_bench_fma (independent fp32 FMA chains)"),
              "tensor": (bf16 * rel_rate, "TFLOP/s", 1e12,
                         f"{bf16_src} x {rel_rate} (rate of the product's tensor-core dtype relative to bf16 / fp16)")}
        traffic, traffic_src = _load_traffic(cfg.name)
        stage_roof = {}
        for k, (bound, w, own) in work.items():
            if stage_ms.get(k, 0.0) <= 0:
                continue
            peak, unit, sc, src = pk[bound]
            nl = max(m["stage_n"].get(k, 1), 1)
            sec = stage_ms[k] * 1e-3
            ach = w / sec / sc
            tr = traffic.get(k)
            stage_roof[k] = {"kernel": k, "bound": bound, "achieved": ach, "peak": peak, "unit": unit,
                             "frac": ach / peak if peak else None, "ms_per_launch": stage_ms[k] / nl,
                             "launches_per_step": nl, "work_per_launch": w / nl, "peak_source": src,
                             "traffic": (tr / nl) if tr else None, "traffic_source": traffic_src,
                             "own_gbs": own / sec / 1e9, "own_frac_of_hbm": own / sec / 1e9 / hbm}
        if "mac" in stage_roof and nprod:
            # what the tensor cores execute: `nprod` products per fp32 product, row tiles of 128 rows
            # (partly filled), 2 x kp columns for 2 x noff offsets, K padded to the MMA step
            kpad = ((2 * d.n_phase + 15) // 16) * 16 if m["mac_mode"] == 7 else 2 * d.n_phase
            ex = nprod * 2.0 * rows_pad * (2 * d.n_off_pad) * kpad * nf
            r = stage_roof["mac"]
            r["executed_tflops"] = ex / (stage_ms["mac"] * 1e-3) / 1e12
            r["executed_frac"] = r["executed_tflops"] / r["peak"]
            r["ceiling"] = mac_flops / ex
            r["arithmetic"] = mac_name
        # SURVEY 8(d)'s own S4 floor: all of S4's flops on the fp32 FMA pipes
        s4_ms = sum(stage_ms.get(k, 0.0) for k in ("fft_fwd", "conv_misc", "mac", "accum", "ifft"))
        s4_flops = nb * ncols * fftf + mac_flops + info["nsp"] * fftf
        s4 = {"ms": s4_ms, "algorithmic_tflop": s4_flops / 1e12, "fma_floor_ms": s4_flops / (fma_tflops * 1e12) * 1e3,
              "algorithmic_bytes_gb": (payload_b + spd_b) / 1e9,
              "hbm_floor_ms": (payload_b + spd_b) / (hbm * 1e9) * 1e3}
        dom = max(stage_roof, key=lambda k: stage_ms[k])
        roof = dict(stage_roof[dom])
        payload_gb = payload_b / 1e9
        line = {"metric": METRIC, "value": total_seg / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_max,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": f"f32 (spectrum product: {mac_name}; index path f64)",
                "data": "synthetic",
                "config": {"workload": cfg.name, "segments_per_event": nseg, "events": world,
                           "pixels": [cfg.npix_x, cfg.npix_y], "nticks": cfg.nticks, "gl_n": cfg.gl_n,
                           "block": list(cfg.block), "resp_nticks": cfg.resp_nticks, "fft_len": d.fft_len,
                           "l2": "flushed between timed iterations (256 MiB write)",
                           "parallelism": f"events x{world}, no collective",
                           "mac_mode_ran": m["mac_mode"], **info},
                "e2e": {"value": total_seg / (e2e_max * 1e-3), "unit": UNIT, "ms_per_step": e2e_max,
                        "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"],
                        "through": "tred_simulate (C ABI) with pinned host buffers for segments and tiles"},
                "gpu_launches": m["launches"] * args.steps,
                "gpu_launches_per_step": m["launches"],
                "clocks": clocks,
                "fma_tflops_measured": fma_tflops,
                "stage_ms": {k: round(v, 4) for k, v in stage_ms.items() if v > 0},
                "roofline": roof,
                "stage_roofline": {k: {kk: (round(vv, 6) if isinstance(vv, float) else vv)
                                       for kk, vv in v.items() if kk in ("bound", "achieved", "peak", "unit", "frac",
                                                                          "traffic", "own_gbs", "own_frac_of_hbm",
                                                                          "executed_tflops", "executed_frac",
                                                                          "ceiling")}
                                   for k, v in stage_roof.items()},
                "s4": s4,
                "peak_mem_gb": m["peak_mem"] / 1e9,
                "payload_gb": payload_gb,
                "wall_s_timed_region": m["t_wall"]}
        if world == 1 and not args.no_extras:
            line["cufft_s4_comparison"] = cufft_s4_comparison(torch, m)
            line["next_rows"] = next_rows_overhead(torch, m, ms_max)
            line["s4"]["two_slab_statistics"] = slab_pair_statistics(torch, m)
        segs, R = m["segs"], m["R"]
        # release the main workload before the other configurations are timed
        m.clear(); sim = None
        torch.cuda.empty_cache()
        if world == 1 and not args.no_extras and args.config == 3:
            extra = {}
            for cid in (1, 2, 4):
                x = measure(args, cid, 0, 1, dev, 10 if cid < 4 else 2, stages=False)
                extra[x["cfg"].name] = {"segments": x["nseg"], "ms_per_step": x["ms"],
                                        "segments_per_s": x["nseg"] / (x["ms"] * 1e-3), "e2e_ms_per_step": x["e2e"],
                                        "gpu_launches_per_step": x["launches"], "host_reads_per_step": x["info"]["host_reads"],
                                        "chunks": x["info"]["nchunks"], "nblocks": x["info"]["nblocks"],
                                        "peak_mem_gb": x["peak_mem"] / 1e9, "mac_mode_ran": x["mac_mode"]}
                x.clear()
                torch.cuda.empty_cache()
            # BASELINE config 5 (Fig. 11): the representation sweep, one timed
            # spill per cell, and the dense-grid comparison
            t_sw = time.perf_counter()
            extra["cfg5_sweep"] = list(sweep_cells(dev, 1))
            extra["cfg5_sweep_wall_s"] = time.perf_counter() - t_sw
            line["extra"] = extra
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


def sweep_cells(dev, steps: int, with_dense: bool = True):
    """BASELINE config 5: block shapes x Gauss-Legendre orders on config-3 inputs -- one record per
    cell (ms per spill, peak GB, occupied-block fraction, the kernels that ran), then the
    dense-grid comparison.  A generator: `--config 5` prints the records one per line, the
    default run stores them under "extra"."""
    import torch
    from paper_2602_12052_b200 import Tred
    cfg0, segs, seg_h, R = workload(3, 0)
    seg_d = torch.from_numpy(seg_h).to(dev)
    R_d = torch.from_numpy(R).to(dev)
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
            yield {"sweep": "block x gl_n", "workload": cfg0.name, "block": list(block), "gl_n": n,
                   "fft_len": d.fft_len, "ms_per_spill": float(np.mean(ms)), "steps": steps,
                   "segments_per_s": seg_h.shape[1] / (float(np.mean(ms)) * 1e-3),
                   "nblocks": out["nblocks"], "occupied_block_fraction": out["nblocks"] / nb_all,
                   "payload_gb": out["nblocks"] * d.block_floats * 4 / 1e9,
                   "peak_gb": torch.cuda.max_memory_allocated(dev) / 1e9,
                   "mac_mode_ran": sim.last_mac_mode()}
            del sim, rhat, out
    if not with_dense:
        return
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
    yield {"sweep": "dense grid", "workload": cfg.name, "impl": "torch.fft (cuFFT), comparison only",
           "ms_per_spill_convolution_only": ms, "peak_gb_convolution_only": peak / 1e9,
           "dense_fine_grid_gb_if_materialised": cfg.npix_x * cfg.npix_y * cfg.sub ** 2 * cfg.nticks * 4 / 1e9,
           "max_abs_diff_vs_block_sparse_over_max": err, "pixels_compared": int(pix.numel())}


def run_sweep(args):
    import torch
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    for rec in sweep_cells(dev, max(1, min(args.steps, 3))):
        print(json.dumps(rec), flush=True)
    return 0


def _spawn_ranks(n: int) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks here (one process per GPU,
    replicas of the spill: PAPER.md:L256-260, drift volumes are independent), exactly as the
    driver would: torch.distributed.run on this node, rendezvous on 127.0.0.1."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--ref-segments", type=int, default=0, help="oracle sample size (0 = per config)")
    ap.add_argument("--work-gb", type=int, default=0, help="tred_convolve workspace cap (GiB), 0 = default")
    ap.add_argument("--budget-gb", type=int, default=5, help="config 4: block payload per chunk (GiB)")
    ap.add_argument("--mac-mode", type=int, default=0, help="tred_config.mac_mode (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip configs 1, 2, 4 and the cuFFT comparison")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return _spawn_ranks(args.gpus)
    if args.gpus != _env_int("WORLD_SIZE", 1):
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={_env_int('WORLD_SIZE', 1)}", file=sys.stderr)
        return 2
    if args.impl == "reference":
        return run_reference(args)
    if args.config == 5:
        return run_sweep(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
