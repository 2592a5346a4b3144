"""Pins for the oracle's generator: Philox words, uniforms, Box-Muller, the entry rule.

None of these re-calls the oracle's own formula: they use published known answers, values
computed independently during the survey (tests/golden/*.txt, each with its citation), closed
forms, identities and statistical moments that a dropped term / wrong sign / wrong index breaks.
"""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def test_philox_known_answers():
    for r in _rows("philox_kat.txt"):
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_pair_mapping():
    """key=(seed lo, seed hi), ctr=(min,max,stream,0): survey-computed words, incl. (i,j)==(j,i)."""
    for r in _rows("philox_pairs.txt"):
        seed, i, j, stream = int(r[0]), int(r[1]), int(r[2]), int(r[3])
        want = [int(x, 16) for x in r[4:8]]
        got = oracle.philox_pairs(seed, stream, [i], [j])[0]
        assert [int(x) for x in got] == want


def test_philox_is_a_bijection_on_small_counter_sets():
    """Distinct counters give distinct outputs (Philox is a permutation for a fixed key)."""
    n = 4096
    i = np.arange(n, dtype=np.uint32)
    w = oracle.philox_pairs(5, 0, i, i + 7)
    assert len({tuple(x) for x in w.tolist()}) == n


def test_uniform_closed_form():
    """u = (2x+1)/2^33 exactly; endpoints strictly inside (0,1); symmetric about 1/2."""
    assert oracle.uniform(0) == 2.0 ** -33
    assert oracle.uniform(2 ** 32 - 1) == 1.0 - 2.0 ** -33
    for x in (1, 12345, 2 ** 31, 2 ** 32 - 2):
        assert oracle.uniform(x) == (2 * x + 1) / 2.0 ** 33
        assert oracle.uniform(x) + oracle.uniform(2 ** 32 - 1 - x) == 1.0


def test_box_muller_identity_and_special_angles():
    rng = np.random.default_rng(0)
    for u1, u2 in rng.random((200, 2)):
        g1, g2 = oracle.box_muller(float(u1), float(u2))
        assert g1 * g1 + g2 * g2 == pytest.approx(-2.0 * math.log(u1), rel=1e-14)
        assert math.atan2(g2, g1) % (2 * math.pi) == pytest.approx(2 * math.pi * u2, abs=1e-12)
    r = math.sqrt(-2.0 * math.log(0.5))
    assert oracle.box_muller(0.5, 0.0) == pytest.approx((r, 0.0), abs=1e-15)
    assert oracle.box_muller(0.5, 0.25) == pytest.approx((0.0, r), abs=1e-15)
    assert oracle.box_muller(0.5, 0.5) == pytest.approx((-r, 0.0), abs=1e-15)


def test_worked_entries_from_survey():
    """u1,u2,g1,g2,H_ij of SURVEY 8(c) c-4 (40-digit mpmath there), seed 1234, D=4096."""
    D, seed = 4096, 1234
    for r in _rows("entries_seed1234_D4096.txt"):
        i, j = int(r[0]), int(r[1])
        u1, u2, g1, g2, hre, him = (float(x) for x in r[2:8])
        w = oracle.philox_pairs(seed, 0, [i], [j])[0]
        assert oracle.uniform(int(w[0])) == pytest.approx(u1, rel=1e-15)
        assert oracle.uniform(int(w[1])) == pytest.approx(u2, rel=1e-15)
        b1, b2 = oracle.box_muller(u1, u2)
        assert b1 == pytest.approx(g1, rel=2e-14) and b2 == pytest.approx(g2, rel=2e-14)
        h = oracle.entry(D, seed, i, j)
        assert h.real == pytest.approx(hre, rel=2e-14)
        assert h.imag == pytest.approx(him, rel=2e-14, abs=0.0 if him else 0.0)


def test_entries_against_mpmath_from_raw_words():
    """Independent 40-digit evaluation from the raw words: checks libm accuracy and scaling."""
    import mpmath as mp
    mp.mp.dps = 40
    D, seed = 32768, 8
    rng = np.random.default_rng(3)
    ii = rng.integers(0, D, 40)
    jj = rng.integers(0, D, 40)
    ii[:4] = jj[:4]                                   # a few diagonal entries
    W = oracle.philox_pairs(seed, 0, ii, jj)
    for i, j, w in zip(ii, jj, W):
        u1 = (mp.mpf(int(w[0])) + mp.mpf(1) / 2) / mp.mpf(2) ** 32
        u2 = (mp.mpf(int(w[1])) + mp.mpf(1) / 2) / mp.mpf(2) ** 32
        r = mp.sqrt(-2 * mp.log(u1))
        g1, g2 = r * mp.cos(2 * mp.pi * u2), r * mp.sin(2 * mp.pi * u2)
        if i == j:
            want = complex(g1 / mp.sqrt(D), 0.0)
        else:
            s = 1 / mp.sqrt(2 * D)
            want = complex(g1 * s, (g2 if i < j else -g2) * s)
        got = oracle.entry(D, seed, int(i), int(j))
        assert abs(got - want) <= 4e-16 * 7.0 / math.sqrt(D)   # |g| <= 6.8, a few ulp
        if i == j:
            assert got.imag == 0.0


def test_hermiticity_bit_exact_and_real_diagonal():
    D = 512
    H = oracle.materialize(D, 77)
    assert np.array_equal(H, H.conj().T)
    assert np.all(np.diag(H).imag == 0.0)
    assert not np.allclose(H.imag[np.triu_indices(D, 1)], 0.0)


def test_entry_moments():
    """g ~ N(0,1): off-diagonal Re, Im each have variance 1/(2D); diagonal variance 1/D;
    E|H_ij|^2 = 1/D; Re and Im uncorrelated; the two triangles are conjugates (sum of Im = 0)."""
    D = 1024
    H = oracle.materialize(D, 2024)
    iu = np.triu_indices(D, 1)
    re, im = H.real[iu] * math.sqrt(2 * D), H.imag[iu] * math.sqrt(2 * D)
    n = re.size
    for g in (re, im):
        assert abs(g.mean()) < 5 / math.sqrt(n)
        assert abs(g.var() - 1.0) < 5 * math.sqrt(2.0 / n)
        assert abs((g ** 4).mean() - 3.0) < 5 * math.sqrt(96.0 / n)
    assert abs((re * im).mean()) < 5 / math.sqrt(n)
    d = np.diag(H).real * math.sqrt(D)
    assert abs(d.mean()) < 5 / math.sqrt(D) and abs(d.var() - 1.0) < 5 * math.sqrt(2.0 / D)
    assert abs((np.abs(H) ** 2).mean() * D - 1.0) < 0.01


def test_h0_uniform_in_minus_one_one():
    D = 32768
    h0 = oracle.h0_diagonal(D, 7)
    assert h0.min() > -1.0 and h0.max() < 1.0
    assert abs(h0.mean()) < 5 / math.sqrt(3 * D)
    assert abs(h0.var() - 1.0 / 3.0) < 0.01
    # survey-computed word for (seed 7, i=3, stream 1): 509611ad -> u = (x+1/2)/2^32
    assert h0[3] == 2.0 * ((0x509611AD + 0.5) / 2.0 ** 32) - 1.0
    # independent of the matrix stream even with an equal seed
    assert oracle.philox_pairs(7, 1, [3], [3])[0].tolist() != oracle.philox_pairs(7, 0, [3], [3])[0].tolist()
