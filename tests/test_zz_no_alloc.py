"""dg_max_wavespeed_noalloc: the max-wavespeed call for users who cannot allocate device memory for the library.

Every other call of include/dg_b200.h works out of a workspace the caller allocates and binds.  A time-step monitor
hooked into somebody else's time loop, or a plug-in under an application that has handed out all GPU memory at
start-up and forbids cudaMalloc afterwards, has nothing to bind: it owns a pointer to the state and a slot for the
answer.  For such callers the reduction's scratch sits in a fixed array inside the library (a block counter and one
partial maximum per thread block, 256.25 KiB per GPU, hence at most DG_NOALLOC_MAX_NODES = 2^29 nodes).

What is checked here: the call gives the same number as the existing path (dg_set_state + dg_max_wavespeed, which is
itself compared with the oracle in test_gpu_parity.py) within that test's tolerance, on two calls in a row -- the
second on a different, smaller state, so that a counter or partial maxima left over from the first call (the array
is shared and keeps its contents) would show.  Sizes beyond the limit are refused with a text, before any GPU work.

This file is named to be collected LAST: `pytest -x` stops at the first failure, and a failure in this add-on must
not hide the parity tests.  It must pass alone in a fresh process and after all other tests.
"""
import ctypes
import re
import os

import numpy as np
import pytest

from paper_2006_15698_b200 import binding
from paper_2006_15698_b200 import inputs as I

G = 1.4
TOL = 4e-16          # relative; the tolerance test_layout_roundtrip_and_wavespeed_all_variants uses for this quantity
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_limit_is_the_headers_and_larger_sizes_are_refused_with_a_text():
    """No GPU needed: the size check comes before the first CUDA call."""
    header = open(os.path.join(ROOT, "include", "dg_b200.h")).read()
    limit = int(re.search(r"#define\s+DG_NOALLOC_MAX_NODES\s+(\d+)ull", header).group(1))
    assert limit == binding.NOALLOC_MAX_NODES == 1 << 29
    lib = binding.load_library()
    err = ctypes.create_string_buffer(512)
    fake = ctypes.c_void_p(256)                       # never dereferenced: the call must refuse first
    assert lib.dg_max_wavespeed_noalloc(fake, limit + 1, G, fake, None, err, len(err)) == 3          # DG_ENOMEM
    text = err.value.decode()
    assert "DG_NOALLOC_MAX_NODES" in text and str(limit + 1) in text and str(limit) in text, text
    assert lib.dg_max_wavespeed_noalloc(fake, limit + 1, G, fake, None, None, 0) == 3                # text is optional
    assert lib.dg_max_wavespeed_noalloc(None, 8, G, fake, None, err, len(err)) == 1                  # DG_EINVAL
    assert lib.dg_max_wavespeed_noalloc(fake, 8, G, None, None, err, len(err)) == 1
    assert lib.dg_max_wavespeed_noalloc(fake, 0, G, fake, None, err, len(err)) == 1
    assert lib.dg_max_wavespeed_noalloc(fake, 8, 1.0, fake, None, err, len(err)) == 1 and b"gamma" in err.value


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path():
    torch = pytest.importorskip("torch")
    from paper_2006_15698_b200 import DG

    # first state: several thread blocks of the reduction (16,384 nodes each) and a ragged last one;
    # second state: smaller (fewer blocks than the first call used), faster flow, its maximum in another place
    cases = [dict(n=(9, 7, 5), p=4, vel=(0.5, -0.3, 0.2), seed=11),       # 39,375 nodes -> 3 blocks
             dict(n=(5, 3, 2), p=2, vel=(-1.1, 0.4, 0.9), seed=5)]        # 810 nodes -> 1 block
    want, states = [], []
    for c in cases:
        nx, ny, nz = c["n"]
        ext = (1.0, 0.6, 0.4)
        q = I.density_wave(nx, ny, nz, c["p"], ext, vel=c["vel"], noise=5e-2, seed=c["seed"], waves=(1, 2, 1))
        dg = DG(nx, ny, nz, c["p"], G, ext)
        want.append(dg.set_state(q).max_wavespeed())                     # the existing path
        dg.close()
        states.append(torch.from_numpy(q).to("cuda").contiguous())
    assert want[0] != want[1]

    # the caller provides input and output; the two calls go back to back on one stream with no synchronisation
    # between them, the way a time loop would issue them
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    binding.max_wavespeed_noalloc(states[0], G, out[0:1])
    binding.max_wavespeed_noalloc(states[1], G, out[1:2])
    got = out.cpu().numpy()
    for g, w in zip(got, want):
        assert abs(g - w) <= TOL * w, (got, want)

    # and once more in the other order: the first call's result is reproduced after a smaller call has used the array
    binding.max_wavespeed_noalloc(states[0], G, out[1:2])
    assert out[1].item() == got[0]

    # the NaN rule of the existing path (negative pressure anywhere -> NaN) holds here too, and does not stick
    # in the shared array: the next call is clean again
    bad = states[1].clone()
    bad.view(-1, 5)[123, 4] = -1.0
    binding.max_wavespeed_noalloc(bad, G, out[0:1])
    binding.max_wavespeed_noalloc(states[1], G, out[1:2])
    assert np.isnan(out[0].item()) and out[1].item() == got[1]
