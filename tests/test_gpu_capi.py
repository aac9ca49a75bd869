"""The C ABI as a C caller sees it: tred_create, tred_prepare_response, tred_simulate, tred_destroy
through ctypes, with HOST buffers for the segments and the waveform tiles (torch supplies device
memory only).  SURVEY.md Sec. 8(b); PAPER.md:L57-61 (segments in, waveforms out)."""
import ctypes as C

import numpy as np
import pytest

import gen
import oracle as o

pytestmark = pytest.mark.gpu


def test_simulate_through_the_c_abi_with_host_buffers():
    import torch
    import paper_2602_12052_b200 as pkg
    L = pkg.lib()
    cfg, segs = gen.make_segments(1)
    R = gen.make_response(cfg, 2001)
    c = pkg.make_config(cfg)
    h = C.c_void_p()
    assert L.tred_create(C.byref(c), C.byref(h)) == 0
    dims = pkg.TredDims()
    assert L.tred_get_dims(C.byref(c), C.byref(dims)) == 0
    try:
        resp = torch.from_numpy(R).cuda()
        rhat = torch.empty((dims.rhat_floats,), dtype=torch.float32, device="cuda")
        st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
        assert L.tred_prepare_response(h, C.c_void_p(resp.data_ptr()), C.c_void_p(rhat.data_ptr()), st) == 0
        seg = np.ascontiguousarray(np.stack([segs[k] for k in gen.SEG_FIELDS]).astype(np.float32))   # HOST [8][nseg]
        nseg = seg.shape[1]
        aug = o.drift(cfg, segs)
        keys = o.blocks(cfg, aug)
        tiles = o.out_tiles(cfg, keys)
        Bt = cfg.block[2]
        cap = len(tiles) + 7
        tk = np.full((cap,), -1, dtype=np.int64)                                       # HOST outputs
        td = np.zeros((cap, Bt), dtype=np.float32)
        res = pkg.TredSimResult()
        work = torch.empty((1 << 20,), dtype=torch.uint8, device="cuda")              # too small on purpose
        calls = 0
        while True:
            rc = L.tred_simulate(h, nseg, seg.ctypes.data_as(C.c_void_p), 1, C.c_void_p(rhat.data_ptr()), 0,
                                 C.c_void_p(work.data_ptr()), work.numel(), cap, tk.ctypes.data_as(C.c_void_p),
                                 td.ctypes.data_as(C.c_void_p), 1, 0, None, None, C.byref(res), st)
            calls += 1
            if rc == -2 and res.work_bytes_needed > work.numel():                      # TRED_ECAP: grow as told
                work = None
                work = torch.empty((int(res.work_bytes_needed),), dtype=torch.uint8, device="cuda")
                continue
            break
        assert rc == 0 and calls >= 2
        torch.cuda.synchronize()
        assert res.nseg == nseg and res.nblocks == len(keys) and res.ntiles == len(tiles)
        assert res.mac_mode == L.tred_last_mac_mode(h) and res.mac_mode in (1, 2, 3, 5, 6, 7)
        np.testing.assert_array_equal(tk[:len(tiles)], tiles)
        assert (tk[len(tiles):] == -1).all()
        # a second event on the same context needs ONE host read of the counts
        rc = L.tred_simulate(h, nseg, seg.ctypes.data_as(C.c_void_p), 1, C.c_void_p(rhat.data_ptr()), 0,
                             C.c_void_p(work.data_ptr()), work.numel(), cap, tk.ctypes.data_as(C.c_void_p),
                             td.ctypes.data_as(C.c_void_p), 1, 0, None, None, C.byref(res), st)
        torch.cuda.synchronize()
        assert rc == 0 and res.host_reads == 1
        # waveforms of a few pixels against the oracle's direct sum
        npix = cfg.npix_x * cfg.npix_y
        pix = np.unique(tiles % npix)[::9]
        ref = o.conv_direct(cfg, keys, o.effq(cfg, aug, keys), R, pix)
        got = np.zeros_like(ref)
        for r, p in enumerate(pix):
            for i in np.flatnonzero(tk[:len(tiles)] % npix == p):
                tb = tk[i] // npix
                n = min(Bt, cfg.nticks - tb * Bt)
                got[r, tb * Bt: tb * Bt + n] = td[i, :n]
        assert np.abs(got - ref).max() <= 1e-4 * np.abs(ref).max()
        # tile capacity too small: TRED_ECAP, the required count reported, nothing written
        tk2 = np.full((3,), -1, dtype=np.int64)
        rc = L.tred_simulate(h, nseg, seg.ctypes.data_as(C.c_void_p), 1, C.c_void_p(rhat.data_ptr()), 0,
                             C.c_void_p(work.data_ptr()), work.numel(), 3, tk2.ctypes.data_as(C.c_void_p),
                             td.ctypes.data_as(C.c_void_p), 1, 0, None, None, C.byref(res), st)
        torch.cuda.synchronize()
        assert rc == -2 and res.ntiles == len(tiles) and (tk2 == -1).all()
    finally:
        L.tred_destroy(h)
