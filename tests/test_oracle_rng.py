"""Pins for the oracle's RNG (pin E9)."""
import os

import numpy as np

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
GAMMA = 0x9E3779B97F4A7C15
MASK = (1 << 64) - 1


def _rows(name):
    with open(os.path.join(HERE, "golden", name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def test_philox_known_answers():
    for row in _rows("philox4x32_10_kat.txt"):
        w = [int(x, 16) for x in row]
        assert oracle.philox4x32_10(w[0:4], w[4:6]) == w[6:10]


def test_mix64_known_answers():
    for i, row in enumerate(_rows("splitmix64_kat.txt")):
        assert oracle.mix64(((i + 1) * GAMMA) & MASK) == int(row[0], 16)


def test_mix64_is_a_bijection_on_samples():
    # M is invertible: the three steps are xorshifts and odd multiplications.  Undo them in Python.
    def unxorshift(z, s):
        x = z
        for _ in range(64 // s + 1):
            x = z ^ (x >> s)
        return x & MASK

    inv1 = pow(0xBF58476D1CE4E5B9, -1, 1 << 64)
    inv2 = pow(0x94D049BB133111EB, -1, 1 << 64)
    rng = np.random.default_rng(1)
    for z in [0, 1, MASK, GAMMA] + [int(v) for v in rng.integers(0, 2 ** 63, 200)]:
        y = oracle.mix64(z)
        y = unxorshift(y, 31); y = (y * inv2) & MASK
        y = unxorshift(y, 27); y = (y * inv1) & MASK
        y = unxorshift(y, 30)
        assert y == z


def test_source_keys_distinct_and_definition():
    seed = 2409046680
    S = oracle.mix64((seed + GAMMA) & MASK)
    keys = [oracle.source_key(seed, h) for h in range(20000)]
    assert len(set(keys)) == len(keys)
    for h in (0, 1, 77, 19999):
        assert keys[h] == oracle.mix64(S ^ h)


def test_child_key_definition_and_distinct():
    kp = oracle.source_key(5, 9)
    seen = set()
    for c0 in (3, 4, 5, 200, 2 ** 24 + 1):
        for j in range(6):
            k = oracle.child_key(kp, c0, j)
            assert k == oracle.mix64((kp + GAMMA * ((c0 << 8) | (j + 1))) & MASK)
            seen.add(k)
    assert len(seen) == 30


def test_draw_layout_matches_block_words():
    # draw i uses block i>>1; even draws take (o1:o0), odd draws (o3:o2); u = ((x>>12)+0.5) 2^-52
    key = 0x0123456789ABCDEF
    u = oracle.draws(key, 0, 8)
    for i in range(8):
        o = oracle.philox4x32_10([i >> 1, 0, 0, 0], [key & 0xFFFFFFFF, key >> 32])
        x64 = (o[3] << 32 | o[2]) if (i & 1) else (o[1] << 32 | o[0])
        # exact: ((x>>12)+0.5)/2^52 is representable
        assert u[i] * 2.0 ** 52 - 0.5 == float(x64 >> 12)
    # first_ctr offsets the stream
    assert np.array_equal(oracle.draws(key, 3, 4), u[3:7])


def test_draws_open_interval_and_uniformity():
    n = 1_000_000
    u = oracle.draws(oracle.source_key(42, 7), 0, n)
    assert u.min() > 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 5 * np.sqrt(1 / 12 / n)
    assert abs(u.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
    hist, _ = np.histogram(u, bins=100, range=(0, 1))
    chi2 = ((hist - n / 100) ** 2 / (n / 100)).sum()
    assert chi2 < 99 + 5 * np.sqrt(2 * 99)
    # lag-1 serial correlation
    c = np.corrcoef(u[:-1], u[1:])[0, 1]
    assert abs(c) < 5 / np.sqrt(n)


def test_streams_of_different_keys_uncorrelated():
    a = oracle.draws(oracle.source_key(1, 0), 0, 200000)
    b = oracle.draws(oracle.source_key(1, 1), 0, 200000)
    assert abs(np.corrcoef(a, b)[0, 1]) < 5 / np.sqrt(200000)
