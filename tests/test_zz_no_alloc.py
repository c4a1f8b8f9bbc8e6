"""iqa_fused_tiles_static: the fused call for programs that are not allowed to allocate device memory.

Who needs it: a plug-in that lives inside somebody else's process (a telescope pipeline stage, a custom operator of an
inference server) and is given the device pointers of its inputs and outputs and nothing else, because the host program
handed out all device memory at start-up; a per-snapshot loop that must not run into the device-wide synchronisation
cudaMalloc / cudaFree bring along; a language binding without a CUDA allocator.  Such a caller cannot provide the
workspace iqa_fused_tiles asks for when tiles are wider than 64 pixels, so this entry point keeps the split-tile partial
sums in a fixed 1 MiB array inside the library (IQA_STATIC_WORKSPACE_BYTES) and refuses larger shapes.

What is checked (Eqs. 1-2, clamp PAPER.md:27):
  * CPU: the limit in the header and in the binding agree; shapes beyond it and bad arguments are refused before any
    CUDA call is made (so this part runs without a GPU);
  * GPU: two calls in a row (different shapes, so the second finds the first one's leftovers in the shared array) give
    what iqa_fused_tiles gives with a torch-allocated workspace -- inside the tolerance of the parity tests, and in
    fact bit for bit, since the kernels and the summation order are the same -- and match the CPU oracle; the calls
    leave torch's allocator statistics untouched.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide the
parity tests.  It passes alone in a fresh process (the first call does the per-device address look-up) and after the
rest of the suite.
"""
import os
import re

import numpy as np
import pytest

from paper_2501_10653_b200 import binding as B

ROOT = os.path.abspath(os.path.join(os.path.dirname(__file__), ".."))
FAKE = 0x1000   # non-NULL, aligned, never dereferenced: validation happens on the host
K = dict(C1=1e-6, C2=1e-6, C=1e-6, D=float(np.float32(1e-6)) / 2)


def _static(x=FAKE, y=FAKE, N=2048, N_T=128, C1=1e-6, C2=1e-6, C=1e-6, D=5e-7, lisi=FAKE, aug=FAKE, sx=FAKE, sy=FAKE):
    return B.iqa_fused_tiles_static(x, y, N, N_T, C1, C2, C, D, lisi, aug, sx, sy, None, None, None)


def test_limit_is_stated_once_and_enforced_before_any_cuda_call():
    header = open(os.path.join(ROOT, "include", "iqa_tiles.h")).read()
    m = re.search(r"#define\s+IQA_STATIC_WORKSPACE_BYTES\s+(\d+)", header)
    assert m and int(m.group(1)) == B.IQA_STATIC_WORKSPACE_BYTES == 1 << 20
    # every BASELINE.json configuration fits ...
    for N, N_T in [(256, 16), (2048, 64), (2048, 512), (8192, 64), (16384, 128)]:
        assert B.iqa_workspace_bytes(N, N_T) <= B.IQA_STATIC_WORKSPACE_BYTES
    # ... N = 32768 with 128-pixel tiles does not (4 MiB of partial sums): refused, with a status of its own
    assert B.iqa_workspace_bytes(32768, 128) > B.IQA_STATIC_WORKSPACE_BYTES
    assert _static(N=32768, N_T=128) == B.IQA_ERR_STATIC_LIMIT
    assert "IQA_STATIC_WORKSPACE_BYTES" in B.iqa_status_string(B.IQA_ERR_STATIC_LIMIT)
    # the other errors are those of iqa_fused_tiles, and they come first
    assert _static(x=None) == B.IQA_ERR_NULL
    assert _static(sy=None) == B.IQA_ERR_NULL
    assert _static(N=2048, N_T=100) == B.IQA_ERR_SHAPE
    assert _static(N=32768, N_T=100) == B.IQA_ERR_SHAPE
    assert _static(C1=0.0) == B.IQA_ERR_PARAM
    assert _static(N=32768, N_T=128, C=-1.0) == B.IQA_ERR_PARAM
    assert _static(x=FAKE + 2) == B.IQA_ERR_ALIGN


def _empty_outputs(torch, nt):
    return {k: torch.empty((nt, nt), dtype=torch.float32, device="cuda") for k in ("lisi", "auglisi", "X", "Y", "L", "A")}


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path_and_the_oracle():
    import torch

    import gpu_util as U
    from paper_2501_10653_b200 import synth

    # call 1: 256-pixel tiles (32 pieces per tile); call 2: 128-pixel tiles of a smaller image, whose partial sums land
    # on top of what call 1 left behind; call 3 repeats call 1 on top of call 2's leftovers.
    cases = []
    for N, N_T, seed in [(2048, 256, 11), (1024, 128, 12)]:
        cfg = synth.scaled(synth.CONFIGS[3], N, N_T)
        x, y, _ = synth.make_pair(cfg, seed=seed)
        assert 0 < B.iqa_workspace_bytes(N, N_T) <= B.IQA_STATIC_WORKSPACE_BYTES
        cases.append((N, N_T, x, y, U.to_dev(x), U.to_dev(y)))
    # outputs are the caller's: allocate them (and everything else torch needs) before the calls under test
    outs = [_empty_outputs(torch, N // N_T) for (N, N_T, *_rest) in cases] + [_empty_outputs(torch, cases[0][0] // cases[0][1])]
    refs = [B.fused_tiles(xd, yd, N_T, **K, numerators=True) for (_N, N_T, _x, _y, xd, yd) in cases]
    torch.cuda.synchronize()

    before = torch.cuda.memory_stats()["allocation.all.allocated"]
    order = [0, 1, 0]
    for slot, ci in enumerate(order):
        _N, N_T, _x, _y, xd, yd = cases[ci]
        B.fused_tiles_static(xd, yd, N_T, **K, out=outs[slot])       # same stream, back to back, no sync in between
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == before     # the binding allocated nothing either

    for slot, ci in enumerate(order):
        N, N_T, x, y, _xd, _yd = cases[ci]
        got = {k: v.cpu().numpy().astype(np.float64) for k, v in outs[slot].items()}
        ref = {k: v.cpu().numpy().astype(np.float64) for k, v in refs[ci].items()}
        U.assert_parity(got, ref, K["C"], f"static call {slot} vs iqa_fused_tiles (N={N}, N_T={N_T})")
        for k in got:                                                # same kernels, same order: bit for bit as well
            assert np.array_equal(got[k], ref[k]), (slot, k)
        U.assert_parity(got, U.run_oracle(x, y, N_T, K), K["C"], f"static call {slot} vs oracle")


@pytest.mark.gpu
def test_shapes_without_split_tiles_and_the_limit_on_a_device():
    import torch

    import gpu_util as U
    from paper_2501_10653_b200 import synth

    cfg = synth.CONFIGS[0]                      # N = 256, N_T = 16: no workspace at all, the array is not touched
    x, y, _ = synth.make_pair(cfg)
    xd, yd = U.to_dev(x), U.to_dev(y)
    out = B.fused_tiles_static(xd, yd, cfg.N_T, **K, out=_empty_outputs(torch, cfg.N // cfg.N_T))
    torch.cuda.synchronize()
    got = {k: v.cpu().numpy().astype(np.float64) for k, v in out.items()}
    U.assert_parity(got, U.run_oracle(x, y, cfg.N_T, K), K["C"], "static call, N_T = 16")
    # beyond the limit: refused with real device pointers too, outputs untouched
    marker = torch.full((4,), 7.0, device="cuda")
    rc = B.iqa_fused_tiles_static(xd, yd, 32768, 128, K["C1"], K["C2"], K["C"], K["D"], marker, marker, marker, marker)
    torch.cuda.synchronize()
    assert rc == B.IQA_ERR_STATIC_LIMIT and bool((marker == 7.0).all())
