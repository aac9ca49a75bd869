"""tred_steps_static: the step splitter for callers that cannot allocate device memory.

Some users of the step splitter have no workspace to pass and may not ask the CUDA runtime for
one: an input stage whose device memory all belongs to somebody else's pool, a thread working
beside another thread's CUDA-graph recording (cudaMalloc / cudaFree from any thread are errors
then), a per-event loop that cannot take the device-wide synchronisation an allocation implies.
For them `tred_steps_static` keeps its scratch in a fixed array inside libtred.so (about 4 MiB per
GPU, at most 2^20 steps per call) instead of in a caller's workspace.

This file checks that entry point against `tred_steps` (whose parity with the oracle is
tests/test_gpu_parity.py::test_steps_parity): same counts, parents and segment ends bit for bit,
charges within the 1e-6 that test uses -- on two calls in a row with different inputs, the second
one smaller, because all calls share the one scratch array and it keeps what the last call left.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

import gen


def _steps_tensor(torch, seed, n_tracks):
    steps = gen.make_steps(seed, n_tracks=n_tracks)
    return torch.from_numpy(np.ascontiguousarray(np.stack([steps[k] for k in gen.STEP_FIELDS]))).cuda()


@pytest.mark.gpu
def test_steps_static_matches_steps_on_two_calls_in_a_row():
    import torch
    from paper_2602_12052_b200 import split_steps, split_steps_static

    # the larger event first: its leftovers stay in the scratch the second call works in
    for call, (seed, n_tracks, model) in enumerate([(31, 60, 0), (32, 25, 1)]):
        par = dict(gen.STEP_PARAMS, recomb_model=model)
        st = _steps_tensor(torch, seed, n_tracks)
        seg_ref, parent_ref, nseg_ref = split_steps(st, par)            # existing path, own workspace
        n = int(nseg_ref.item())
        assert n > st.shape[1], "the workload must split some steps"

        # the caller of the static entry point brings every output buffer
        nseg = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        split_steps_static(st, par, None, None, nseg)                    # counting pass
        assert int(nseg.item()) == n, call
        seg = torch.full((8, n), float("nan"), dtype=torch.float32, device="cuda")
        parent = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        split_steps_static(st, par, seg, parent, nseg)
        torch.cuda.synchronize()
        assert int(nseg.item()) == n, call
        np.testing.assert_array_equal(parent.cpu().numpy(), parent_ref.cpu().numpy())
        got, ref = seg.cpu().numpy(), seg_ref.cpu().numpy()
        for i, k in enumerate(gen.SEG_FIELDS):
            if k == "q":
                np.testing.assert_allclose(got[i], ref[i], rtol=1e-6, err_msg=f"call {call}")
            else:
                np.testing.assert_array_equal(got[i], ref[i], err_msg=f"call {call}: {k}")

    # too small an output: the count is still reported, nothing is written past the capacity
    seg10 = torch.full((8, 10), float("nan"), dtype=torch.float32, device="cuda")
    parent12 = torch.full((12,), -1, dtype=torch.int32, device="cuda")
    split_steps_static(st, par, seg10, parent12, nseg)
    assert int(nseg.item()) == n
    np.testing.assert_array_equal(seg10.cpu().numpy(), ref[:, :10])
    assert parent12.cpu().numpy()[10:].tolist() == [-1, -1]


@pytest.mark.gpu
def test_steps_static_refuses_more_steps_than_its_scratch_holds():
    import torch
    import ctypes as C
    import paper_2602_12052_b200 as pkg

    L = pkg.lib()
    limit = L.tred_steps_static_max()
    assert limit == 1 << 20
    nseg = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    c = pkg.TredStepsConfig()
    for k, _ in pkg.TredStepsConfig._fields_:
        setattr(c, k, gen.STEP_PARAMS[k])
    # the size check comes before any access: no step data is needed to see the refusal
    rc = L.tred_steps_static(C.byref(c), limit + 1, None, 0, None, None, C.c_void_p(nseg.data_ptr()), None)
    assert rc == -2 and L.tred_strerror(rc).decode().startswith("capacity")
    torch.cuda.synchronize()
    assert int(nseg.item()) == -7                                        # outputs untouched
    big = torch.zeros((8, limit + 1), dtype=torch.float32, device="cuda")
    with pytest.raises(pkg.TredError, match="exceed the fixed scratch"):
        pkg.split_steps_static(big, gen.STEP_PARAMS, None, None, nseg)
    # exactly the limit is accepted (zero-length steps: one piece each)
    pkg.split_steps_static(big[:, :limit].contiguous(), gen.STEP_PARAMS, None, None, nseg)
    assert int(nseg.item()) == limit


def test_steps_static_header_numbers_agree():
    """CPU: the limit the header states is the one the library reports, and the stated size of the
    resident array follows from it (no GPU call)."""
    import os
    import re
    import paper_2602_12052_b200 as pkg

    text = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "tred.h")).read()
    mx = int(re.search(r"#define\s+TRED_STEPS_STATIC_MAX\s+(\d+)", text).group(1))
    nb = int(re.search(r"#define\s+TRED_STEPS_STATIC_BYTES\s+(\d+)", text).group(1))
    assert pkg.lib().tred_steps_static_max() == mx
    assert nb == ((mx + 1) * 4 + 255) // 256 * 256 + 2048 and nb < 8 << 20
