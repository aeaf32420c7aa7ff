"""Pins of the counter-based generator of the oracle (oracle/rng.py, reading S22): the published known-answer vectors of
Philox4x32-10, the counter/key layout, Box-Muller identities, and the statistics of the streams.  CPU only."""
import os

import numpy as np

from oracle import rng as R

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = R.philox4x32_10(np.array(v[0:4]), np.array(v[4:6]))
        assert [int(x) for x in out] == v[6:10], r


def test_counter_layout_and_stream_separation():
    """Element (i, j) depends on (seed, step, stream, i, j // 4) exactly as the header says: rebuilt from a single
    Philox call; changing any one of the five changes the block."""
    seed, step, sid = 0x1234567890ABCDEF, (7 << 32) + 5, 3
    x = R.draw_normal(seed, step, sid, 6, 11)
    w = R.philox4x32_10(np.array([step & 0xFFFFFFFF, step >> 32, 4, (sid << 24) + 2]),
                        np.array([seed & 0xFFFFFFFF, seed >> 32]))
    u = (w.astype(np.float64) + 0.5) / 2.0 ** 32
    r = np.sqrt(-2 * np.log(u[2])); want = np.float32(r * np.cos(2 * np.pi * u[3]))
    assert x[4, 10] == want                                             # element 10 = block 2, third value
    base = R.draw_normal(seed, step, sid, 6, 12)
    assert np.array_equal(base[:, :11], x)                              # a wider row extends, never reshuffles
    for other in (R.draw_normal(seed + 1, step, sid, 6, 12), R.draw_normal(seed, step + 1, sid, 6, 12),
                  R.draw_normal(seed, step, sid + 1, 6, 12), R.draw_normal(seed + (1 << 32), step, sid, 6, 12),
                  R.draw_normal(seed, step + (1 << 32), sid, 6, 12)):
        assert not np.any(other == base)
    assert not np.any(base[1:] == base[:-1])


def test_box_muller_pairs_and_uniform_range():
    u = R.uniform_of(np.array([0, 1, 2 ** 31, 2 ** 32 - 1], dtype=np.uint32))
    assert u[0] == 2.0 ** -33 and u[-1] == 1 - 2.0 ** -33 and np.all((u > 0) & (u < 1))
    x = R.draw_normal(11, 2, 0, 4000, 8).astype(np.float64)
    w = R._words(11, 2, 0, 4000, 2)
    ua = R.uniform_of(w)[..., 0]                                        # radius of the pair (0, 1) of each block
    r2 = x[:, 0::4] ** 2 + x[:, 1::4] ** 2
    assert np.allclose(r2, -2 * np.log(ua), rtol=1e-6)


def test_stream_statistics():
    x = R.draw_normal(2026, 1, 0, 20000, 22).astype(np.float64)
    n = x.size
    assert abs(x.mean()) < 4 / np.sqrt(n) and abs(x.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs((x ** 4).mean() - 3) < 4 * np.sqrt(96 / n) and abs((x ** 3).mean()) < 4 * np.sqrt(15 / n)
    c = np.corrcoef(x, rowvar=False)
    assert np.abs(c - np.eye(22)).max() < 5 / np.sqrt(20000)            # columns (blocks and pair members) uncorrelated
    assert abs(np.mean(x[1:] * x[:-1])) < 4 / np.sqrt(n)                # consecutive rows uncorrelated
    y = R.draw_normal(2026, 2, 0, 20000, 22).astype(np.float64)
    assert abs(np.mean(x * y)) < 4 / np.sqrt(n)                         # consecutive steps uncorrelated
    lu = R.draw_log_uniform(2026, 1, 1, 200000).astype(np.float64)
    u = np.exp(lu)
    h, _ = np.histogram(u, bins=50, range=(0, 1))
    chi2 = ((h - 4000.0) ** 2 / 4000.0).sum()
    assert chi2 < 49 + 5 * np.sqrt(98) and abs(lu.mean() + 1) < 4 / np.sqrt(200000)     # E ln u = -1, var = 1
