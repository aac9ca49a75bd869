"""CPU-only checks of the boundary: libtred.so builds, loads, exports every symbol that
include/tred.h declares, and its host-side logic (derived sizes, argument checks,
"no GPU -> fail loudly") behaves.  No compute call is made here."""
import os
import re

import pytest

import gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "tred.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tred_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2602_12052_b200 as pkg
    L = pkg.lib()
    names = _declared_symbols()
    assert "tred_drift" in names and "tred_gather_waveforms" in names and len(names) >= 16
    for n in names:
        assert hasattr(L, n), f"libtred.so does not export {n}"
    assert set(names) == set(pkg.EXPORTS), set(names) ^ set(pkg.EXPORTS)
    assert L.tred_abi_version() == 2
    assert L.tred_strerror(-2).decode().startswith("capacity")


def test_five_north_star_calls_are_present():
    names = _declared_symbols()
    for n in ("tred_drift", "tred_effq", "tred_blockbin", "tred_convolve", "tred_gather_waveforms"):
        assert n in names


@pytest.mark.parametrize("cfg_id,L,nover,ppb", [(1, 288, 5, 4), (2, 512, 8, 4), (3, 576, 5, 9)])
def test_dims_host_logic(cfg_id, L, nover, ppb):
    """fft_len is the smallest 2^a 3^b (a >= 3) >= Bt + Tr - 1 (reading G20; the paper pads
    to a power of two, which this rule reproduces for its own block)."""
    import paper_2602_12052_b200 as pkg
    cfg = gen.make_config(cfg_id)
    d = pkg.get_dims(cfg)
    assert d.fft_len == L and d.out_len == cfg.block[2] + cfg.resp_nticks - 1
    assert d.fft_len >= d.out_len
    n = L
    while n % 2 == 0:
        n //= 2
    while n % 3 == 0:
        n //= 3
    assert n == 1 and L % 8 == 0
    assert d.n_over == nover and d.n_freq == L // 2 and d.pix_per_block == ppb
    assert list(d.NG) == [cfg.sub * cfg.npix_x, cfg.sub * cfg.npix_y, cfg.nticks]
    assert list(d.NB) == [-(-d.NG[a] // cfg.block[a]) for a in range(3)]
    assert (d.n_phase, d.n_off, d.n_off_pad) == (100, 121, 128)
    # fp32 spectrum + tf32 hi/lo matrices + the four mirror-symmetric half matrices + flag + the fp16
    # hi/lo matrix [f][256][13 blocks of 32 halves] and its scales + the DFT matrix [L][2 Bt] halves
    nf = L // 2
    assert d.rhat_floats == 14 * nf * 100 * 128 + 4 * nf * 128 * 100 + 8 + nf * 256 * 208 + (nf + 7) // 8 * 8 + \
        L * cfg.block[2]
    assert d.conv_row_bytes == (L // 2) * (100 + 128) * 8


def test_paper_block_shape_gives_paper_padding():
    """The paper's own block: 32 ticks with a ~2000-tick response pads to 2048."""
    import paper_2602_12052_b200 as pkg
    cfg = gen.make_config(1, block=(8, 8, 32), resp_nticks=2000, nticks=4096)
    assert pkg.get_dims(cfg).fft_len == 2048


def test_bad_config_is_rejected():
    import paper_2602_12052_b200 as pkg
    with pytest.raises(pkg.TredError):
        pkg.get_dims(gen.make_config(1, gl_n=5))
    with pytest.raises(pkg.TredError):
        pkg.get_dims(gen.make_config(1, block=(8, 8, 48)))       # not a power of two


def test_no_gpu_fails_loudly():
    import torch
    import paper_2602_12052_b200 as pkg
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(pkg.TredError):
        pkg.Tred(gen.make_config(1))
    # the C entry point itself refuses too (no fallback inside the library)
    import ctypes as C
    h = C.c_void_p()
    c = pkg.make_config(gen.make_config(1))
    assert pkg.lib().tred_create(C.byref(c), C.byref(h)) == -3
