"""Pins for oracle.philox: Random123 known-answer vectors, range of u, stream separation."""
import os

import numpy as np

from oracle import philox


def test_known_answer_vectors(golden_dir):
    n = 0
    for line in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        w = [int(x, 16) for x in line.split()]
        out = philox.philox4x32_10(w[0], w[1], w[2], w[3], w[4], w[5])
        assert [int(o) for o in out] == w[6:10], line
        n += 1
    assert n == 3


def test_vectorised_equals_scalar():
    c0 = np.arange(7, dtype=np.uint64) * 977
    a = philox.philox4x32_10(c0, 3, 2, 1, 11, 12)
    for t in range(7):
        b = philox.philox4x32_10(int(c0[t]), 3, 2, 1, 11, 12)
        assert [int(x[t]) for x in a] == [int(x) for x in b]


def test_uniform_open_interval_and_float32_exact():
    x = np.array([0, 0x1FF, 0x200, 0xFFFFFFFF], dtype=np.uint32)
    u = philox.uniform_from_bits(x)
    assert u[0] == 0.5 * 2.0 ** -23 and u[1] == u[0] and u[2] == 1.5 * 2.0 ** -23
    assert u[3] == 1.0 - 0.5 * 2.0 ** -23
    assert np.all(u.astype(np.float32).astype(np.float64) == u)      # exactly representable in fp32
    assert np.all((u > 0) & (u < 1))


def test_streams_differ_by_prompt_sample_step_seed():
    base = philox.gumbel_noise(64, 5, 1, 2, 3)
    assert np.array_equal(base, philox.gumbel_noise(64, 5, 1, 2, 3))
    for args in [(6, 1, 2, 3), (5, 0, 2, 3), (5, 1, 3, 3), (5, 1, 2, 4), (5 + (1 << 32), 1, 2, 3)]:
        assert not np.array_equal(base, philox.gumbel_noise(64, *args))


def test_gumbel_lane_assignment():
    # element v uses word (v & 3) of the block with counter c0 = v >> 2
    g = philox.gumbel_noise(8, 9, 4, 3, 2)
    w = philox.philox4x32_10(np.array([0, 1]), 2, 3, 4, 9, 0)
    for v in range(8):
        x = int(w[v & 3][v >> 2])
        u = ((x >> 9) + 0.5) / 8388608.0
        assert g[v] == -np.log(-np.log(u))


def test_gumbel_moments():
    g = np.concatenate([philox.gumbel_noise(4096, 123, i, 0, 0) for i in range(32)])
    assert abs(np.mean(g) - 0.5772156649) < 0.02                      # Euler-Mascheroni
    assert abs(np.var(g) - np.pi ** 2 / 6) < 0.05
