"""Dense projection y = x W^T (oracle; test infrastructure only).

Every projection of the decoder (QKV, O, gate/up, down, LM head)
is this contraction with W stored [out_features, in_features] row-major:

    y[r, n] = sum_k x[r, k] * W[n, k]

evaluated in float64 after up-casting the stored bits.  `linear` is the library form (numpy
matmul); `linear_loops` is the same sum written out, used by the pin in
tests/test_oracle_transformer.py (brute force on tiny inputs, and the transposed-operand mistake
x @ W fails it because W is not square there).
"""
import numpy as np


def linear(x, W):
    return np.asarray(x, dtype=np.float64) @ np.asarray(W, dtype=np.float64).T


def linear_loops(x, W):
    x, W = np.asarray(x, dtype=np.float64), np.asarray(W, dtype=np.float64)
    R, K = x.shape
    N = W.shape[0]
    y = np.zeros((R, N))
    for r in range(R):
        for n in range(N):
            acc = 0.0
            for k in range(K):
                acc += x[r, k] * W[n, k]
            y[r, n] = acc
    return y
