"""-m gpu parity of the tcgen05/TMEM GEMM (through the C-ABI hook darts_debug_gemm_bf16) against oracle.linear."""
import numpy as np
import pytest
import torch

from oracle.linear import linear
from paper_2605_30859_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2605_30859_b200 import api
    d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=64, n_pages=64, max_rows=8, max_prompts=2, max_prompt_len=64, max_new=64)
    yield d
    d.close()


@pytest.fixture(scope="module")
def ctx_pairs():
    from paper_2605_30859_b200 import api
    d = api.Darts(dict(cfg=dict(wl.CONFIGS["c2"]["model"])), page_size=64, n_pages=64, max_rows=8, max_prompts=2, max_prompt_len=64, max_new=64,
                  flags=api.FLAG_CTA_PAIRS)
    yield d
    d.close()


def _mk(shape, seed, scale=1.0):
    g = torch.Generator(device="cuda").manual_seed(seed)
    return (torch.randn(*shape, generator=g, device="cuda") * scale).to(torch.bfloat16)


@pytest.mark.parametrize("rows,N,K,S", [
    (1, 128, 64, 1),          # one row, one k-block
    (16, 256, 256, 1),
    (37, 132, 192, 3),        # ragged rows (3 boxes of 16), ragged N (tail tile, N % 128 != 0), ragged split
    (128, 384, 512, 2),       # full tile
    (200, 512, 1024, 4),      # two row tiles, second one ragged
    (300, 1000, 2560, 5),     # three row tiles, K of config 3
    (64, 6144, 2560, 4),      # config-3 QKV shape at 64 rows
    # S = 0: the stream-K weight-streaming kernel (swap-AB, persistent) the decode projections run on
    (1, 128, 64, 0),
    (16, 256, 256, 0),
    (37, 132, 192, 0),        # ragged rows, ragged N
    (200, 512, 1024, 0),      # 13 row boxes, pieces straddling CTAs
    (256, 384, 512, 0),       # one full 256-row block
    (300, 1000, 2560, 0),     # 257..512 rows: ONE 512-row block = two fused MMA N blocks (256 + 44) sharing the weight tile
    (512, 640, 512, 0),       # both fused N blocks full
    (289, 2560, 4096, 0),     # config-3 O projection at the row count of the profiled step
    (700, 640, 1024, 0),      # three row blocks
    (64, 6144, 2560, 0),      # config-3 QKV shape
    (130, 2560, 9728, 0),     # config-3 down projection: few tiles, long K (many pieces per tile)
    (2048, 19456, 256, 0),    # whole-tile mode (tiles >= 8 x SMs), prefill-like
])
def test_gemm_matches_oracle(ctx, rows, N, K, S):
    X, W = _mk((rows, K), rows + N), _mk((N, K), K + S, 0.05)
    got = ctx.debug_gemm_bf16(X, W, split_k=S).cpu().numpy().astype(np.float64)
    ref = linear(X.float().cpu().numpy(), W.float().cpu().numpy())
    # bf16 products are exact in fp32; only the fp32 accumulation order differs: ~K * 2^-24 relative to sum |x w|
    tol = 4 * K * 2.0 ** -24 * float(np.max(np.abs(X.float().cpu().numpy()) @ np.abs(W.float().cpu().numpy()).T))
    assert np.max(np.abs(got - ref)) <= tol, (np.max(np.abs(got - ref)), tol)


@pytest.mark.parametrize("rows,N,K", [
    (1, 128, 64), (16, 256, 256), (37, 132, 192), (200, 512, 1024), (256, 384, 512), (300, 1000, 2560), (512, 640, 512),
    (289, 2560, 4096), (700, 640, 1024), (64, 6144, 2560), (130, 2560, 9728), (512, 19456, 2560), (2048, 19456, 256),
])
def test_cta_pair_gemm_matches_oracle(ctx_pairs, rows, N, K):
    """The same shapes on the CTA-pair (tcgen05 cta_group::2) stream-K kernel: M = 256 weight rows per MMA, each CTA of the pair stages
    its own weight tile and half of the activation rows; odd tile counts (N = 132, 1000, 640 ...) leave the pair's second tile empty."""
    X, W = _mk((rows, K), rows + N), _mk((N, K), K + 3, 0.05)
    got = ctx_pairs.debug_gemm_bf16(X, W, split_k=0).cpu().numpy().astype(np.float64)
    ref = linear(X.float().cpu().numpy(), W.float().cpu().numpy())
    tol = 4 * K * 2.0 ** -24 * float(np.max(np.abs(X.float().cpu().numpy()) @ np.abs(W.float().cpu().numpy()).T))
    assert np.max(np.abs(got - ref)) <= tol, (np.max(np.abs(got - ref)), tol)
    assert torch.equal(ctx_pairs.debug_gemm_bf16(X, W, split_k=0).cpu(), torch.from_numpy(got).float())


@pytest.mark.parametrize("S", [4, 0])
def test_gemm_is_deterministic_and_split_order_fixed(ctx, S):
    X, W = _mk((50, 1024), 1), _mk((256, 1024), 2, 0.05)
    a = ctx.debug_gemm_bf16(X, W, split_k=S)
    b = ctx.debug_gemm_bf16(X, W, split_k=S)
    assert torch.equal(a, b)


def test_gemm_rejects_bad_shapes(ctx):
    from paper_2605_30859_b200 import api
    with pytest.raises(api.DartsError) as e:
        ctx.debug_gemm_bf16(_mk((4, 100), 0), _mk((8, 100), 1))
    assert e.value.code == api.ERR_UNSUPPORTED
