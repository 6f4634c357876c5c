"""-m gpu: token-level streaming hook (rollout side): the chunks delivered while the rollout runs
reassemble to exactly the tokens (and their log-probabilities) of the finished rollout, cover steps [0, n_steps) in order, and the
result equals the plain loop's."""
import numpy as np
import pytest

from paper_2605_30859_b200 import workloads as wl
from tests.gpu_util import make_ctx

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("chunk", [1, 5, 16, 64])
def test_chunks_reassemble_to_the_rollout(chunk):
    c = wl.CONFIGS["c1"]
    x = wl.rollout_inputs("c1", seed=1)
    d, _ = make_ctx(c["model"], 1, c["G"], c["Kp"], c["P"], c["max_new"], page=16)
    ref = d.rollout_host(x["prompts"], x["Kp"], x["K"], x["max_new"], 1.0, 3, forced_len=x["forced_len"])
    n_steps = d.counters()["n_steps"]
    got = []
    d.prefill(list(x["prompts"]), x["Kp"], x["K"], temperature=1.0, seed=3, forced_len=x["forced_len"])
    d.run_to_completion_streaming(chunk, lambda s0, s1, t, lp: got.append((s0, s1, t, lp)))
    res = d.results()
    for k in ("tokens", "len", "status", "sel", "logprob"):
        assert np.array_equal(res[k], ref[k]), k
    assert got[0][0] == 0 and all(a[1] == b[0] for a, b in zip(got, got[1:]))          # contiguous, in step order
    assert all(0 < s1 - s0 <= chunk and t.shape == (32, s1 - s0) and lp.shape == t.shape for s0, s1, t, lp in got)
    assert got[-1][1] >= n_steps
    stream = np.concatenate([g[2] for g in got], axis=1)
    stream_lp = np.concatenate([g[3] for g in got], axis=1)
    assert np.array_equal(stream[:, :n_steps], ref["tokens"][:, :n_steps])
    assert np.all(stream[:, n_steps:] == -1)
    assert np.array_equal(stream_lp[:, :n_steps], ref["logprob"][:, :n_steps])        # bitwise: same kernels, same order
    assert np.all(stream_lp[stream < 0] == 0.0) and np.all(stream_lp <= 0.0)
    d.close()
