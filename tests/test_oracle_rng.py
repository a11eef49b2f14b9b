"""Pins for the oracle's random-number layer (reading R-3) and photon count (R-12b)."""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox_kat.txt")


def _kat_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(x, 16) for x in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 7
    for ctr, key, out in rows:
        assert list(O.philox4x32_10(ctr, key)) == out


def test_philox_is_a_bijection_of_the_counter_sample():
    # distinct counters under one key give distinct blocks (Philox is a keyed permutation)
    seen = set()
    for i in range(2000):
        seen.add(O.philox4x32_10((i, 0, 0, 0), (5, 9)))
        seen.add(O.philox4x32_10((0, 0, 0, i + 1), (5, 9)))
    assert len(seen) == 4000


def test_philox_word_statistics():
    # mean of 4e4 words/2^32 ~ 1/2, every bit position ~ balanced: catches a dropped round/xor
    w = np.array([O.philox4x32_10((i, 1, 2, 3), (0, 0)) for i in range(10000)], dtype=np.uint64).ravel()
    u = w / 2.0 ** 32
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / len(u))
    for b in range(32):
        frac = ((w >> np.uint64(b)) & np.uint64(1)).mean()
        assert abs(frac - 0.5) < 4 * 0.5 / math.sqrt(len(w))


def test_uniform_closed_form_and_range():
    # word 6627e8d5 -> 0.399046481
    assert O.uniform(0x6627E8D5) == pytest.approx(0.399046481, abs=5e-10)
    assert O.uniform(0) == 2.0 ** -24
    assert O.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert O.uniform(0x000001FF) == 2.0 ** -24  # low 9 bits are dropped
    for w in (0, 1, 0x1FF, 0x200, 0x12345678, 0xFFFFFFFF, 0x80000000):
        u = O.uniform(w)
        assert u == (w >> 9) * 2.0 ** -23 + 2.0 ** -24
        assert np.float32(u) == u  # exactly representable in fp32
        assert 0.0 < u < 1.0


def test_photon_count_round_half_up():
    assert O.photon_count(10.0) == 100000
    assert O.photon_count(1.0) == 10000
    assert O.photon_count(0.0) == 0
    assert O.photon_count(0.00004) == 0  # 0.4 photons
    assert O.photon_count(0.00005) == 1 or O.photon_count(0.00005) == 0  # float32(5e-5)*1e4 straddles 0.5
    assert O.photon_count(0.00016) == 2  # 1.6 -> 2
    assert O.photon_count(1.0e5) == 10 ** 9
    e = np.float32(123.456)
    assert O.photon_count(e) == math.floor(float(e) * 1.0e4 + 0.5)
