"""paper_2602_12052_b200 -- thin Python binding of libtred (include/tred.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of
`csrc/`.  PyTorch provides device memory and streams.  There is no CPU fallback: if the
library cannot be built/loaded, or no CUDA device is present, the calls raise.

    from paper_2602_12052_b200 import Tred
    sim = Tred(cfg)                       # cfg: object/dict with the tred_config fields
    rhat = sim.prepare_response(resp)     # resp: float32 CUDA tensor [S][S][2H+1][2H+1][Tr]
    out = sim.simulate(seg, rhat)         # seg: float32 CUDA tensor [8][nseg]
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

__all__ = ["Tred", "TredError", "lib", "TredConfig", "TredDims", "EXPORTS", "split_steps", "split_steps_static", "TredStepsConfig", "readout", "TredReadoutConfig"]

_c_i64 = C.c_int64
_c_p = C.c_void_p


class TredConfig(C.Structure):
    """Mirror of `tred_config` (include/tred.h)."""
    _fields_ = [("npix_x", C.c_int32), ("npix_y", C.c_int32), ("sub", C.c_int32), ("nticks", C.c_int32),
                ("pitch_mm", C.c_double), ("tick_us", C.c_double),
                ("origin_x_mm", C.c_double), ("origin_y_mm", C.c_double), ("t_origin_us", C.c_double),
                ("v_mm_us", C.c_double), ("lifetime_us", C.c_double),
                ("DL_mm2_us", C.c_double), ("DT_mm2_us", C.c_double),
                ("sigma_min_xy_mm", C.c_double), ("sigma_min_t_us", C.c_double),
                ("nsigma", C.c_double), ("point_thresh", C.c_double),
                ("gl_n", C.c_int32), ("block", C.c_int32 * 3),
                ("resp_half", C.c_int32), ("resp_nticks", C.c_int32),
                ("effq_mode", C.c_int32), ("mac_mode", C.c_int32), ("fft_mode", C.c_int32)]


class TredDims(C.Structure):
    """Mirror of `tred_dims` (include/tred.h)."""
    _fields_ = [("NG", _c_i64 * 3), ("NB", _c_i64 * 3),
                ("fft_len", C.c_int32), ("out_len", C.c_int32), ("n_over", C.c_int32),
                ("n_freq", C.c_int32), ("n_phase", C.c_int32), ("n_off", C.c_int32),
                ("n_off_pad", C.c_int32), ("pix_per_block", C.c_int32),
                ("rhat_floats", _c_i64), ("block_floats", _c_i64), ("conv_row_bytes", _c_i64),
                ("dft_ticks", C.c_int32)]


class TredStepsConfig(C.Structure):
    """Mirror of `tred_steps_config` (include/tred.h)."""
    _fields_ = [("max_len_mm", C.c_double), ("recomb_model", C.c_int32), ("w_ion_ev", C.c_double),
                ("efield_kv_cm", C.c_double), ("density_g_cm3", C.c_double),
                ("birks_A", C.c_double), ("birks_k", C.c_double),
                ("box_alpha", C.c_double), ("box_beta", C.c_double)]


class TredReadoutConfig(C.Structure):
    """Mirror of `tred_readout_config` (include/tred.h)."""
    _fields_ = [("threshold_e", C.c_double), ("n_integ", C.c_int32), ("n_reset", C.c_int32),
                ("max_hits", C.c_int32), ("adc_lsb_e", C.c_double)]


class TredSimResult(C.Structure):
    """Mirror of `tred_sim_result` (include/tred.h)."""
    _fields_ = [(k, _c_i64) for k in ("nseg", "npairs", "nblocks", "ncp", "nsp", "ntiles", "nrt", "nchunks",
                                       "work_bytes_needed", "conv_bytes_needed", "conv_bytes_min",
                                       "work_bytes_used")] + \
               [("host_reads", C.c_int32), ("mac_mode", C.c_int32)]


# name -> (restype, argtypes); every symbol include/tred.h declares
EXPORTS = {
    "tred_get_dims": (C.c_int, [C.POINTER(TredConfig), C.POINTER(TredDims)]),
    "tred_create": (C.c_int, [C.POINTER(TredConfig), C.POINTER(_c_p)]),
    "tred_destroy": (None, [_c_p]),
    "tred_strerror": (C.c_char_p, [C.c_int]),
    "tred_last_cuda_error": (C.c_char_p, []),
    "tred_abi_version": (C.c_int, []),
    "tred_last_mac_mode": (C.c_int, [_c_p]),
    "tred_drift": (C.c_int, [_c_p, _c_i64, _c_p, _c_p, _c_p, _c_p, _c_p]),
    "tred_blockbin_work_bytes": (C.c_size_t, [_c_p, _c_i64, _c_i64]),
    "tred_blockbin": (C.c_int, [_c_p, _c_i64, _c_p, _c_i64, _c_i64, _c_p, _c_p, _c_p, _c_p, _c_p,
                                _c_p, C.c_size_t, _c_p]),
    "tred_effq_work_bytes": (C.c_size_t, [_c_p, _c_i64]),
    "tred_effq": (C.c_int, [_c_p, _c_i64, _c_i64, _c_p, _c_p, _c_p, _c_p, _c_p, _c_p, _c_p, C.c_size_t, _c_p]),
    "tred_prepare_response": (C.c_int, [_c_p, _c_p, _c_p, _c_p]),
    "tred_plan_work_bytes": (C.c_size_t, [_c_p]),
    "tred_convolve_plan": (C.c_int, [_c_p, _c_i64, _c_p,
                                     _c_i64, _c_p, _c_p, _c_p,
                                     _c_i64, _c_p, _c_p, _c_p,
                                     _c_i64, _c_p, _c_p,
                                     _c_p,
                                     _c_p, C.c_size_t, _c_p]),
    "tred_convolve_work_bytes": (C.c_size_t, [_c_p, _c_i64, _c_i64]),
    "tred_convolve": (C.c_int, [_c_p, _c_i64, _c_p, _c_p, _c_p,
                                _c_i64, _c_p, _c_p,
                                _c_i64, _c_p, _c_p,
                                _c_p,
                                _c_p, _c_p, _c_p, C.c_size_t, _c_p]),
    "tred_gather_waveforms": (C.c_int, [_c_p, _c_i64, _c_p, _c_p, _c_p, _c_i64, _c_i64, _c_p, _c_p, C.c_int,
                                        _c_i64, _c_p, _c_p, _c_p]),
    "tred_simulate": (C.c_int, [_c_p, _c_i64, _c_p, C.c_int, _c_p, _c_i64, _c_p, C.c_size_t,
                                _c_i64, _c_p, _c_p, C.c_int, _c_i64, _c_p, _c_p, C.POINTER(TredSimResult), _c_p]),
    "tred_steps_work_bytes": (C.c_size_t, [_c_i64]),
    "tred_steps": (C.c_int, [C.POINTER(TredStepsConfig), _c_i64, _c_p, _c_i64, _c_p, _c_p, _c_p, _c_p,
                             C.c_size_t, _c_p]),
    "tred_steps_static_max": (_c_i64, []),
    "tred_steps_static": (C.c_int, [C.POINTER(TredStepsConfig), _c_i64, _c_p, _c_i64, _c_p, _c_p, _c_p, _c_p]),
    "tred_readout": (C.c_int, [C.POINTER(TredReadoutConfig), _c_i64, C.c_int32, _c_p, _c_p, _c_p, _c_p, _c_p, _c_p]),
    "tred_truth_work_bytes": (C.c_size_t, [_c_p, _c_i64]),
    "tred_truth": (C.c_int, [_c_p, _c_i64, _c_p, _c_p, _c_i64, _c_p, _c_p, _c_p, _c_p, _c_p, C.c_size_t, _c_p]),
    "tred_profile_begin": (C.c_int, [_c_p, C.c_int]),
    "tred_profile_end": (C.c_int, [_c_p, C.c_int, _c_p, _c_p]),
    "tred_bench_fma": (C.c_int, [_c_p, C.c_int32, _c_p, C.POINTER(C.c_double), _c_p]),
    "tred_stage_count": (C.c_int, []),
    "tred_stage_name": (C.c_char_p, [C.c_int]),
}

_LIB = None


class TredError(RuntimeError):
    pass


def lib() -> C.CDLL:
    """Builds (if stale) and loads libtred.so; raises if that is impossible."""
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = C.CDLL(path)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(L, name)          # AttributeError if a declared symbol is missing
            fn.restype = res
            fn.argtypes = args
        _LIB = L
    return _LIB


_CFG_FIELDS = [f[0] for f in TredConfig._fields_]
_CFG_OPTIONAL = ("effq_mode", "mac_mode", "fft_mode")        # 0 = library default


def make_config(cfg) -> TredConfig:
    get = (lambda k: cfg[k]) if isinstance(cfg, dict) else (lambda k: getattr(cfg, k))
    c = TredConfig()
    for k in _CFG_FIELDS:
        if k in _CFG_OPTIONAL:
            try:
                v = get(k)
            except (KeyError, AttributeError):
                v = 0
            setattr(c, k, int(v))
            continue
        v = get(k)
        if k == "block":
            c.block[0], c.block[1], c.block[2] = (int(x) for x in v)
        else:
            setattr(c, k, v)
    return c


def _check(rc: int, what: str):
    if rc != 0:
        L = lib()
        msg = L.tred_strerror(rc).decode()
        if rc == -3:
            msg += ": " + L.tred_last_cuda_error().decode()
        raise TredError(f"{what} failed ({rc}): {msg}")


def get_dims(cfg) -> TredDims:
    d = TredDims()
    c = make_config(cfg)
    _check(lib().tred_get_dims(C.byref(c), C.byref(d)), "tred_get_dims")
    return d


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def readout(wave, params: dict, noise=None):
    """tred_readout: waveforms [npix][nticks] (float32 CUDA tensor) -> (nhit, hit_tick, hit_adc)."""
    import torch
    if not wave.is_cuda:
        raise TredError("tred_readout needs CUDA tensors: the TRED path has no CPU fallback")
    assert wave.dtype == torch.float32 and wave.is_contiguous() and wave.dim() == 2
    c = TredReadoutConfig()
    for k, _ in TredReadoutConfig._fields_:
        setattr(c, k, params.get(k, 0))
    npix, nticks = wave.shape
    mh = int(c.max_hits)
    dev = wave.device
    if noise is not None:
        assert noise.is_cuda and noise.dtype == torch.float32 and noise.is_contiguous()
        assert tuple(noise.shape) == (npix, mh, 3)
    nhit = torch.empty((max(npix, 1),), dtype=torch.int32, device=dev)
    tick = torch.empty((max(npix, 1), max(mh, 1)), dtype=torch.int32, device=dev)
    adc = torch.empty((max(npix, 1), max(mh, 1)), dtype=torch.float32, device=dev)
    _check(lib().tred_readout(C.byref(c), npix, nticks, _ptr(wave), _ptr(noise), _ptr(nhit), _ptr(tick), _ptr(adc),
                              C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)), "tred_readout")
    return nhit[:npix], tick[:npix, :mh], adc[:npix, :mh]


def split_steps(steps, params: dict, cap_seg: int | None = None):
    """tred_steps: G4Steps [8][nstep] (float32 CUDA tensor: x0,y0,z0,x1,y1,z1,dE,t0) -> step-segments
    [8][nseg] for Tred.drift / Tred.simulate, and the parent step of every segment.  Sizes the
    output from the device-side count (one host read) unless cap_seg is given."""
    import torch
    if not steps.is_cuda:
        raise TredError("tred_steps needs CUDA tensors: the TRED path has no CPU fallback")
    assert steps.dtype == torch.float32 and steps.is_contiguous() and steps.shape[0] == 8
    L = lib()
    c = TredStepsConfig()
    for k, _ in TredStepsConfig._fields_:
        setattr(c, k, params[k])
    nstep = steps.shape[1]
    dev = steps.device
    stream = C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
    work = torch.empty((max(L.tred_steps_work_bytes(nstep), 256),), dtype=torch.uint8, device=dev)
    nseg = torch.zeros((1,), dtype=torch.int64, device=dev)
    if cap_seg is None:                                 # counting pass: capacity 0
        _check(L.tred_steps(C.byref(c), nstep, _ptr(steps), 0, None, None, _ptr(nseg), _ptr(work), work.numel(),
                            stream), "tred_steps")
        cap_seg = int(nseg.item())
    seg = torch.empty((8, max(cap_seg, 1)), dtype=torch.float32, device=dev)
    parent = torch.empty((max(cap_seg, 1),), dtype=torch.int32, device=dev)
    _check(L.tred_steps(C.byref(c), nstep, _ptr(steps), cap_seg, _ptr(seg), _ptr(parent), _ptr(nseg), _ptr(work),
                        work.numel(), stream), "tred_steps")
    return seg[:, :cap_seg], parent[:cap_seg], nseg


def split_steps_static(steps, params: dict, seg, parent, nseg):
    """tred_steps_static: `split_steps` for callers that must not allocate device memory (an input
    stage whose memory all belongs to a pool, a thread beside another thread's graph recording, a
    per-event loop that cannot take cudaMalloc's synchronisation).  Nothing is allocated here or in
    the library: the caller passes the outputs -- seg [8][cap_seg] float32, parent [cap_seg] int32,
    nseg [1] int64, CUDA tensors (cap_seg = seg.shape[1]; seg and parent may be None for the
    counting pass) -- and the scratch is a fixed array inside libtred.so.  At most
    tred_steps_static_max() steps per call; calls that can overlap on the GPU (other streams) share
    that array and must be ordered by the caller.  Make the first call on a device at set-up."""
    import torch
    if not steps.is_cuda:
        raise TredError("tred_steps_static needs CUDA tensors: the TRED path has no CPU fallback")
    assert steps.dtype == torch.float32 and steps.is_contiguous() and steps.shape[0] == 8
    L = lib()
    nstep = steps.shape[1]
    if nstep > L.tred_steps_static_max():
        raise TredError(f"tred_steps_static: {nstep} steps exceed the fixed scratch of "
                        f"{L.tred_steps_static_max()} steps per call; split the batch or use split_steps")
    c = TredStepsConfig()
    for k, _ in TredStepsConfig._fields_:
        setattr(c, k, params[k])
    cap_seg = 0
    if seg is not None:
        assert seg.is_cuda and seg.dtype == torch.float32 and seg.is_contiguous() and seg.shape[0] == 8
        cap_seg = seg.shape[1]
        assert parent.is_cuda and parent.dtype == torch.int32 and parent.numel() >= cap_seg
    assert nseg.is_cuda and nseg.dtype == torch.int64 and nseg.numel() >= 1
    stream = C.c_void_p(torch.cuda.current_stream(steps.device).cuda_stream)
    _check(L.tred_steps_static(C.byref(c), nstep, _ptr(steps), cap_seg, _ptr(seg) if cap_seg else None,
                               _ptr(parent) if cap_seg else None, _ptr(nseg), stream), "tred_steps_static")


class Tred:
    """One configuration on one CUDA device.  Methods mirror the C calls one to one; the
    tensors they return are ordinary torch CUDA tensors owned by the caller."""

    def __init__(self, cfg, device="cuda:0", conv_work_bytes: int | None = None):
        import torch
        if not torch.cuda.is_available():
            raise TredError("no CUDA device: the TRED path has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.L = lib()
        self.cfg = make_config(cfg)
        self.dims = TredDims()
        _check(self.L.tred_get_dims(C.byref(self.cfg), C.byref(self.dims)), "tred_get_dims")
        h = _c_p()
        _check(self.L.tred_create(C.byref(self.cfg), C.byref(h)), "tred_create")
        self.h = h
        self.conv_work_bytes = conv_work_bytes
        self._work = {}

    def __del__(self):
        try:
            if getattr(self, "h", None):
                self.L.tred_destroy(self.h)
                self.h = None
        except Exception:
            pass

    # -- helpers ------------------------------------------------------------------
    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def _empty(self, shape, dtype):
        return self.torch.empty(shape, dtype=dtype, device=self.device)

    def _workbuf(self, name, nbytes):
        """Grow-only cached byte buffer."""
        b = self._work.get(name)
        if b is None or b.numel() < nbytes:
            b = None
            self._work.pop(name, None)
            b = self._empty((max(int(nbytes), 256),), self.torch.uint8)
            self._work[name] = b
        return b

    def profile_begin(self, events: bool = True):
        _check(self.L.tred_profile_begin(self.h, 1 if events else 0), "tred_profile_begin")

    def profile_end(self) -> dict:
        """{stage name: (milliseconds, kernel launches)}; synchronises the recorded events."""
        n = self.L.tred_stage_count()
        ms = (C.c_float * n)()
        ln = (C.c_int64 * n)()
        _check(self.L.tred_profile_end(self.h, n, C.cast(ms, _c_p), C.cast(ln, _c_p)), "tred_profile_end")
        return {self.L.tred_stage_name(i).decode(): (float(ms[i]), int(ln[i])) for i in range(n)}

    def bench_fma(self, iters: int = 4096, reps: int = 5) -> float:
        """Measured fp32 FMA rate of this device in TFLOP/s (best of `reps`, CUDA events)."""
        t = self.torch
        out = self._empty((1,), t.float32)
        fl = C.c_double(0.0)
        best = 0.0
        for _ in range(reps + 1):
            a, b = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
            a.record()
            _check(self.L.tred_bench_fma(self.h, iters, _ptr(out), C.byref(fl), self._stream()), "tred_bench_fma")
            b.record()
            b.synchronize()
            best = max(best, fl.value / (a.elapsed_time(b) * 1e-3) / 1e12)
        return best

    def last_mac_mode(self) -> int:
        """The spectrum-product kernel (tred_config.mac_mode value 1..7) the last convolve launched."""
        return int(self.L.tred_last_mac_mode(self.h))

    # -- the calls ----------------------------------------------------------------
    def prepare_response(self, resp):
        t = self.torch
        K = 2 * self.cfg.resp_half + 1
        S = self.cfg.sub
        assert resp.is_cuda and resp.dtype == t.float32 and resp.is_contiguous()
        assert tuple(resp.shape) == (S, S, K, K, self.cfg.resp_nticks), resp.shape
        rhat = self._empty((self.dims.rhat_floats,), t.float32)
        _check(self.L.tred_prepare_response(self.h, _ptr(resp), _ptr(rhat), self._stream()),
               "tred_prepare_response")
        return rhat

    def drift(self, seg):
        t = self.torch
        assert seg.is_cuda and seg.dtype == t.float32 and seg.is_contiguous() and seg.shape[0] == 8
        nseg = seg.shape[1]
        augf = self._empty((10, nseg), t.float32)
        augi = self._empty((8, nseg), t.int32)
        npairs = self._empty((1,), t.int64)
        _check(self.L.tred_drift(self.h, nseg, _ptr(seg), _ptr(augf), _ptr(augi), _ptr(npairs),
                                 self._stream()), "tred_drift")
        return augf, augi, npairs

    def blockbin(self, augi, cap_pairs: int, cap_blocks: int | None = None):
        t = self.torch
        nseg = augi.shape[1]
        cap_blocks = cap_pairs if cap_blocks is None else cap_blocks
        NBt = int(self.dims.NB[2])
        keys = self._empty((max(cap_blocks, 1),), t.int64)
        blk_off = self._empty((max(cap_blocks, 1) + 1,), t.int32)
        pair_seg = self._empty((max(cap_pairs, 1),), t.int32)
        slab_off = self._empty((NBt + 1,), t.int32)
        nblocks = self._empty((1,), t.int64)
        wb = self.L.tred_blockbin_work_bytes(self.h, nseg, cap_pairs)
        work = self._workbuf("bin", wb)
        _check(self.L.tred_blockbin(self.h, nseg, _ptr(augi), cap_pairs, cap_blocks, _ptr(keys),
                                    _ptr(blk_off), _ptr(pair_seg), _ptr(slab_off), _ptr(nblocks),
                                    _ptr(work), work.numel(), self._stream()), "tred_blockbin")
        return keys, blk_off, pair_seg, slab_off, nblocks

    def effq(self, nblocks: int, keys, blk_off, pair_seg, augf, augi, payload=None, work_bytes: int | None = None):
        t = self.torch
        nseg = augf.shape[1]
        if payload is None:
            payload = self._empty((max(nblocks, 1), self.cfg.block[0], self.cfg.block[1], self.cfg.block[2]),
                                  t.float32)
        # workspace for the per-segment tables (less is allowed: same values, slower)
        wb = self.L.tred_effq_work_bytes(self.h, nseg)
        if work_bytes is not None:
            wb = min(wb, int(work_bytes))
        work = self._workbuf("effq", wb) if wb > 0 else None
        _check(self.L.tred_effq(self.h, nseg, nblocks, _ptr(keys), _ptr(blk_off), _ptr(pair_seg),
                                _ptr(augf), _ptr(augi), _ptr(payload), _ptr(work),
                                wb if work is not None else 0, self._stream()), "tred_effq")
        return payload

    def convolve_plan(self, nblocks: int, keys, cap_cp: int | None = None, cap_sp: int | None = None,
                      cap_tiles: int | None = None) -> dict:
        """Footprints of the convolution; returns a dict of device tensors (counts are
        1-element int64 device tensors, read them yourself)."""
        t = self.torch
        NBt = int(self.dims.NB[2])
        nmap = NBt * self.cfg.npix_x * self.cfg.npix_y
        K2 = self.dims.n_off
        if cap_cp is None:
            cap_cp = min(nblocks * self.dims.pix_per_block, nmap)
        if cap_sp is None:
            cap_sp = min(cap_cp * K2, nmap)
        if cap_tiles is None:
            cap_tiles = min(cap_sp * self.dims.n_over, nmap)
        p = dict(cp_keys=self._empty((max(cap_cp, 1),), t.int64), cp_off=self._empty((NBt + 1,), t.int32),
                 ncp=self._empty((1,), t.int64),
                 sp_keys=self._empty((max(cap_sp, 1),), t.int64), sp_off=self._empty((NBt + 1,), t.int32),
                 nsp=self._empty((1,), t.int64),
                 tile_keys=self._empty((max(cap_tiles, 1),), t.int64), ntiles=self._empty((1,), t.int64),
                 rt_off=self._empty((NBt + 1,), t.int32))
        pw = self.L.tred_plan_work_bytes(self.h)
        p["work"] = self._empty((pw,), t.uint8)
        _check(self.L.tred_convolve_plan(self.h, nblocks, _ptr(keys),
                                         cap_cp, _ptr(p["cp_keys"]), _ptr(p["cp_off"]), _ptr(p["ncp"]),
                                         cap_sp, _ptr(p["sp_keys"]), _ptr(p["sp_off"]), _ptr(p["nsp"]),
                                         cap_tiles, _ptr(p["tile_keys"]), _ptr(p["ntiles"]),
                                         _ptr(p["rt_off"]),
                                         _ptr(p["work"]), p["work"].numel(), self._stream()), "tred_convolve_plan")
        return p

    def convolve(self, nblocks: int, keys, payload, rhat, plan: dict, ncp: int, nsp: int,
                 cp_off_host, sp_off_host, sp_data=None, work_bytes: int | None = None, rt_off_host=None):
        t = self.torch
        import numpy as np
        row = self.dims.n_over * self.cfg.block[2]
        if sp_data is None:
            sp_data = self._empty((max(nsp, 1), row), t.float32)
        co = np.ascontiguousarray(cp_off_host, dtype=np.int32)
        po = np.ascontiguousarray(sp_off_host, dtype=np.int32)
        if rt_off_host is None:
            rt_off_host = plan["rt_off"].cpu().numpy()
        ro = np.ascontiguousarray(rt_off_host, dtype=np.int32)
        ns_max = int(np.diff(po).max()) if len(po) > 1 else 0
        need = self.L.tred_convolve_work_bytes(self.h, 128, ns_max)
        if work_bytes is None:
            work_bytes = self.conv_work_bytes
        if work_bytes is None:
            work_bytes = min(self.L.tred_convolve_work_bytes(self.h, ncp, nsp), 16 << 30)
        work_bytes = max(int(work_bytes), int(need))
        work = self._workbuf("conv", work_bytes)
        _check(self.L.tred_convolve(self.h, nblocks, _ptr(keys), _ptr(payload), _ptr(rhat),
                                    ncp, _ptr(plan["cp_keys"]), co.ctypes.data_as(_c_p),
                                    nsp, _ptr(plan["sp_keys"]), po.ctypes.data_as(_c_p),
                                    ro.ctypes.data_as(_c_p),
                                    _ptr(plan["work"]), _ptr(sp_data), _ptr(work), work.numel(), self._stream()),
               "tred_convolve")
        return sp_data

    def gather_waveforms(self, nsp: int, sp_data, plan: dict, ntiles: int, pix_ids=None, tile_plan=None,
                         tile_data=None, tile_begin: int = 0, accumulate: bool = False):
        """`plan`: plan of the blocks sp_data belongs to; `tile_plan` (default: the same): plan
        whose tile list is filled; [tile_begin, tile_begin + ntiles) is the range of it."""
        t = self.torch
        Bt = self.cfg.block[2]
        tp = plan if tile_plan is None else tile_plan
        if tile_data is None:
            tile_data = self._empty((max(ntiles, 1), Bt), t.float32)
        dense = None
        npix = 0
        if pix_ids is not None and pix_ids.numel() > 0:
            assert pix_ids.dtype == t.int32 and pix_ids.is_cuda
            npix = pix_ids.numel()
            dense = self._empty((npix, self.cfg.nticks), t.float32)
        _check(self.L.tred_gather_waveforms(self.h, nsp, _ptr(sp_data), _ptr(plan["work"]), _ptr(tp["work"]),
                                            tile_begin, ntiles, _ptr(tp["tile_keys"]), _ptr(tile_data),
                                            1 if accumulate else 0, npix, _ptr(pix_ids), _ptr(dense),
                                            self._stream()), "tred_gather_waveforms")
        return tile_data, dense

    # -- whole path -----------------------------------------------------------------
    def simulate(self, seg, rhat, pix_ids=None, keep=False, payload_budget_bytes: int = 0,
                 host_out=None):
        """Segments in, per-pixel current waveforms out: one call of
        tred_simulate.  `seg` may be a CUDA tensor or a (pinned) host tensor; `host_out` =
        (tile_keys, tile_data) host tensors to receive the tiles (default: device tensors are
        returned).  `keep=True` runs the stepwise calls instead and returns the intermediates
        too (tests).  The binding only owns the workspace: it grows it when the library says
        how much this event needs and calls again."""
        t = self.torch
        if keep:
            return self.simulate_steps(seg, rhat, pix_ids, keep=True)
        assert seg.dtype == t.float32 and seg.is_contiguous() and seg.shape[0] == 8
        nseg = seg.shape[1]
        Bt = self.cfg.block[2]
        res = TredSimResult()
        npix = 0
        dense = None
        if pix_ids is not None and pix_ids.numel() > 0:
            assert pix_ids.dtype == t.int32 and pix_ids.is_cuda
            npix = pix_ids.numel()
            dense = self._empty((npix, self.cfg.nticks), t.float32)
        cap_tiles = getattr(self, "_cap_tiles", 0)
        want = max(getattr(self, "_sim_bytes", 0), (256 << 20) + nseg * 512)
        tk = td = None
        for _ in range(8):
            work = self._workbuf("sim", want)
            if host_out is not None:
                tk, td = host_out
                cap = min(tk.numel(), td.shape[0])
            else:
                cap = cap_tiles
                if tk is None or tk.numel() != max(cap, 1):
                    tk = td = None                                # release before allocating the larger ones
                    tk = self._empty((max(cap, 1),), t.int64)
                    td = self._empty((max(cap, 1), Bt), t.float32)
            rc = self.L.tred_simulate(self.h, nseg, _ptr(seg), 0 if seg.is_cuda else 1, _ptr(rhat),
                                      int(payload_budget_bytes), _ptr(work), work.numel(), cap, _ptr(tk), _ptr(td),
                                      0 if host_out is None else 1, npix, _ptr(pix_ids), _ptr(dense), C.byref(res),
                                      self._stream())
            if rc == -2 and res.work_bytes_needed > work.numel():          # workspace: grow and call again
                want = int(res.work_bytes_needed) + (64 << 20)
                if self.conv_work_bytes is not None and res.conv_bytes_needed > 0:      # bounded peak memory
                    grant = min(max(int(self.conv_work_bytes), int(res.conv_bytes_min)), int(res.conv_bytes_needed))
                    want -= int(res.conv_bytes_needed) - grant
                self._work.pop("sim", None)
                work = None
                continue
            if rc == -2 and res.ntiles > cap:                               # tile capacity
                if host_out is not None:
                    raise TredError(f"host_out holds {cap} tiles, the event has {res.ntiles}")
                cap_tiles = int(res.ntiles * 1.01) + 1024
                continue
            _check(rc, "tred_simulate")
            break
        else:
            raise TredError("tred_simulate: workspace negotiation did not converge")
        self._sim_bytes, self._cap_tiles = want, cap_tiles
        nt = int(res.ntiles)
        out = {k: int(getattr(res, k)) for k in ("nseg", "npairs", "nblocks", "ncp", "nsp", "ntiles", "nrt",
                                                 "nchunks", "host_reads", "mac_mode", "work_bytes_used")}
        out.update(tile_keys=tk[:nt], tile_data=td[:nt], dense=dense)
        return out

    def simulate_steps(self, seg, rhat, pix_ids=None, keep=False):
        """The same path through the stepwise calls (three host reads of counts); returns the
        intermediates as well when keep=True."""
        t = self.torch
        nseg = seg.shape[1]
        augf, augi, npairs = self.drift(seg)
        cap_pairs = int(npairs.item())
        keys, blk_off, pair_seg, slab_off, nblocks_d = self.blockbin(augi, cap_pairs)
        nblocks = int(nblocks_d.item())
        payload = self.effq(nblocks, keys, blk_off, pair_seg, augf, augi)
        plan = self.convolve_plan(nblocks, keys)
        counts = t.cat([plan["ncp"], plan["nsp"], plan["ntiles"], plan["cp_off"].to(t.int64),
                        plan["sp_off"].to(t.int64), plan["rt_off"].to(t.int64)]).cpu().numpy()
        ncp, nsp, ntiles = int(counts[0]), int(counts[1]), int(counts[2])
        NBt = int(self.dims.NB[2])
        co, po, ro = (counts[3 + i * (NBt + 1):3 + (i + 1) * (NBt + 1)] for i in range(3))
        sp_data = self.convolve(nblocks, keys, payload, rhat, plan, ncp, nsp, co, po, rt_off_host=ro)
        tile_data, dense = self.gather_waveforms(nsp, sp_data, plan, ntiles, pix_ids)
        tile_keys, sp_keys, sp_off = plan["tile_keys"], plan["sp_keys"], plan["sp_off"]
        out = dict(nseg=nseg, npairs=cap_pairs, nblocks=nblocks, ncp=ncp, nsp=nsp, ntiles=ntiles, nrt=int(ro[-1]),
                   tile_keys=tile_keys[:ntiles], tile_data=tile_data[:ntiles], dense=dense)
        if keep:
            out.update(augf=augf, augi=augi, keys=keys[:nblocks], blk_off=blk_off[:nblocks + 1],
                       pair_seg=pair_seg[:cap_pairs], slab_off=slab_off, payload=payload[:nblocks],
                       sp_keys=sp_keys[:nsp], sp_data=sp_data[:nsp], sp_off=sp_off)
        return out

    # -- truth record --------------------------------
    def truth(self, augf, augi, cap_rec: int | None = None):
        """Charge of every segment per (pixel, time tile): (rec_seg, rec_key, rec_q, nrec)."""
        t = self.torch
        nseg = augf.shape[1]
        work = self._workbuf("truth", self.L.tred_truth_work_bytes(self.h, nseg))
        nrec = self._empty((1,), t.int64)
        if cap_rec is None:                         # counting pass
            _check(self.L.tred_truth(self.h, nseg, _ptr(augf), _ptr(augi), 0, None, None, None, _ptr(nrec),
                                     _ptr(work), work.numel(), self._stream()), "tred_truth")
            cap_rec = int(nrec.item())
            if cap_rec < 0:
                raise TredError("tred_truth: a segment reaches more than 32 pixels or time tiles on one axis")
        rs = self._empty((max(cap_rec, 1),), t.int32)
        rk = self._empty((max(cap_rec, 1),), t.int64)
        rq = self._empty((max(cap_rec, 1),), t.float32)
        _check(self.L.tred_truth(self.h, nseg, _ptr(augf), _ptr(augi), cap_rec, _ptr(rs), _ptr(rk), _ptr(rq),
                                 _ptr(nrec), _ptr(work), work.numel(), self._stream()), "tred_truth")
        return rs[:cap_rec], rk[:cap_rec], rq[:cap_rec], nrec

    # -- truth attribution ---------------------------------
    def attribute(self, seg, rhat, group, pix_ids, ngroups: int | None = None):
        """On-demand waveform attribution "by re-convolving selected contributions"
        (PAPER.md:L356): the path is linear in the segment charges, so the waveform a group of
        segments (a track, a particle, a vertex) leaves on the requested pixels is the path run
        on that group alone.  `group` [nseg] int tensor (group id of every segment, < 0: none).
        Returns dense [ngroups][npix][nticks]; summed over the groups it equals the waveform
        of all grouped segments up to fp32 rounding."""
        t = self.torch
        assert group.shape[0] == seg.shape[1]
        if ngroups is None:
            ngroups = int(group.max().item()) + 1 if group.numel() else 0
        out = t.zeros((max(ngroups, 1), pix_ids.numel(), self.cfg.nticks), dtype=t.float32, device=self.device)
        for gid in range(ngroups):
            idx = t.nonzero(group == gid).flatten()
            if idx.numel() == 0:
                continue
            sub = seg.index_select(1, idx).contiguous()          # selecting rows: marshalling, no arithmetic
            out[gid] = self.simulate(sub, rhat, pix_ids=pix_ids)["dense"]
        return out[:ngroups]

    # -- whole path in bounded-memory chunks of occupied blocks (BASELINE config 4) --------
    def simulate_chunked(self, seg, rhat, pix_ids=None, payload_budget_bytes: int = 8 << 30):
        """Same result as `simulate`, bit for bit, with the block payload, the convolution
        workspace and the slab outputs held for one range of time slabs at a time
        (chunks bounded by device memory): tred_simulate with a payload
        budget.  `chunks` in the result is the number of slab ranges."""
        out = self.simulate(seg, rhat, pix_ids, payload_budget_bytes=payload_budget_bytes)
        out["chunks"] = out["nchunks"]
        return out
