"""Pins for the oracle's Philox4x32-10 (oracle/rosen_oracle.cpp)."""
import numpy as np

import oracle


def test_known_answer_vectors(golden):
    rows = golden("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for row in rows:
        v = [int(x, 16) for x in row]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_counter_and_key_sensitivity():
    base = oracle.philox4x32_10((1, 2, 3, 4), (5, 6))
    seen = {base}
    for i in range(4):
        c = [1, 2, 3, 4]; c[i] ^= 1
        seen.add(oracle.philox4x32_10(c, (5, 6)))
    for i in range(2):
        k = [5, 6]; k[i] ^= 1
        seen.add(oracle.philox4x32_10((1, 2, 3, 4), k))
    assert len(seen) == 7  # every counter / key word matters


def test_word_uniformity():
    # 2^16 blocks: mean of the words / 2^32 is 1/2 within 5 s.e.; bit balance
    w = np.array([oracle.philox4x32_10((i, 0, 0, 0), (1, 0)) for i in range(1 << 14)], dtype=np.uint64)
    u = w.astype(np.float64).ravel() / 2.0 ** 32
    assert abs(u.mean() - 0.5) < 5 * np.sqrt(1 / 12 / u.size)
    bits = ((w.ravel()[:, None] >> np.arange(32, dtype=np.uint64)[None, :]) & np.uint64(1)).mean(axis=0)
    assert np.all(np.abs(bits - 0.5) < 5 * 0.5 / np.sqrt(w.size))
