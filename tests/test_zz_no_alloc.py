"""-m gpu: darts_gemm_bf16_static, the entry point that allocates nothing (include/darts.h) — the stream-K GEMM of the decode projections
with its fp32 pieces in the library's file-scope device array instead of a caller-provided buffer.  Checked against the existing path
(darts_debug_gemm_bf16, split_k = 0, scratch from torch) on calls in a row that share the array, against the oracle, and at the size limit.
The file name sorts last on purpose: a failure here must not hide another test under `pytest -x`."""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle.linear import linear
from paper_2605_30859_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _mk(shape, seed, scale=1.0):
    g = torch.Generator(device="cuda").manual_seed(seed)
    return (torch.randn(*shape, generator=g, device="cuda") * scale).to(torch.bfloat16)


def _tol(X, W, K):
    # tests/test_gpu_gemm.py's bound: bf16 products are exact in fp32, only the accumulation order differs
    return 4 * K * 2.0 ** -24 * float(np.max(np.abs(X.float().cpu().numpy()) @ np.abs(W.float().cpu().numpy()).T))


def test_static_scratch_gemm_matches_the_existing_path_on_calls_in_a_row():
    from paper_2605_30859_b200 import api
    d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=64, n_pages=64, max_rows=8, max_prompts=2, max_prompt_len=64, max_new=64)
    limit = C.c_size_t()
    assert api.darts_static_scratch_bytes(C.byref(limit)) == api.OK and limit.value == 32 << 20
    # different shapes back to back, then the first again: the shared array holds another shape's pieces and counts each time
    shapes = [(130, 2560, 9728), (37, 132, 192), (64, 6144, 2560), (300, 1000, 2560), (130, 2560, 9728), (130, 2560, 9728)]
    data = {s: (_mk((s[0], s[2]), s[0] + s[1]), _mk((s[1], s[2]), s[2], 0.05)) for s in set(shapes)}
    ref = {s: d.debug_gemm_bf16(X, W, split_k=0).clone() for s, (X, W) in data.items()}                 # the existing path
    outs = [torch.full((s[0], s[1]), float("nan"), dtype=torch.float32, device="cuda") for s in shapes]
    d.gemm_bf16_static(*data[shapes[0]], torch.empty_like(outs[0]))                                      # first call on the device: symbol lookup
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for s, out in zip(shapes, outs):
        d.gemm_bf16_static(*data[s], out)                                                                # no sync in between: stream order only
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory in use changed across calls that must not allocate"
    for s, out in zip(shapes, outs):
        X, W = data[s]
        got, want = out.cpu().numpy().astype(np.float64), ref[s].cpu().numpy().astype(np.float64)
        tol = _tol(X, W, s[2])
        assert np.max(np.abs(got - want)) <= tol, (s, float(np.max(np.abs(got - want))), tol)
        assert np.array_equal(got, want), s                        # same kernel, same plan, same summation order: the same bits
        assert np.max(np.abs(got - linear(X.float().cpu().numpy(), W.float().cpu().numpy()))) <= tol, s   # and the definition
    # beyond the limit: a clear error, nothing launched, the context stays usable
    X, W = _mk((512, 2560), 1), _mk((19456, 2560), 2, 0.05)
    with pytest.raises(api.DartsError) as e:
        d.gemm_bf16_static(X, W, torch.empty(512, 19456, dtype=torch.float32, device="cuda"))
    assert e.value.code == api.ERR_WORKSPACE_TOO_SMALL and "static scratch holds" in str(e.value)
    with pytest.raises(api.DartsError) as e:
        d.gemm_bf16_static(_mk((8, 100), 3), _mk((128, 100), 4), torch.empty(8, 128, dtype=torch.float32, device="cuda"))   # K % 64 != 0
    assert e.value.code == api.ERR_UNSUPPORTED
    s = shapes[1]
    out = d.gemm_bf16_static(*data[s], torch.empty(s[0], s[1], dtype=torch.float32, device="cuda"))
    assert torch.equal(out, ref[s])
    d.close()
