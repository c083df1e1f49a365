"""Pins for the oracle's Philox block, RNG keying and integer thresholds (CPU only).

Each pin is something other than the oracle itself: published known answers, closed forms
evaluated in high-precision decimal arithmetic, or a keying recipe re-derived here from
DESIGN.md's "RNG keying" table with the block function treated as a black box.
"""
import math
import os
from decimal import Decimal, getcontext

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _kat_rows():
    rows = []
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(x, 16) for x in line.split()]
            rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, want in rows:
        got = oracle.philox4x32_10(ctr, key)
        assert [int(x) for x in got] == want


def test_philox_is_a_bijection_of_the_counter_on_a_sample():
    # a block cipher in counter mode: distinct counters -> distinct outputs
    outs = {tuple(int(x) for x in oracle.philox4x32_10([c, 0, 7, 1], [5, 9])) for c in range(4096)}
    assert len(outs) == 4096


def _ctr_word3(colour, tag, k):
    return colour | (tag << 8) | (k << 16)


@pytest.mark.parametrize("seed", [0, 2503146881, 0xDEADBEEF12345678])
def test_keying_scheme0_quad(seed):
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for P in [0, 1, 2, 3, 4, 127, 128, 1000003, (1 << 39) + 5]:
        for t, c in [(0, 0), (7, 1), (2**32 - 2, 1)]:
            unit = P >> 2
            blk = oracle.philox4x32_10([unit & 0xFFFFFFFF, unit >> 32, t, _ctr_word3(c, 2, 0)], key)
            assert oracle.u32(seed, 0, t, c, P) == int(blk[P & 3])


@pytest.mark.parametrize("seed", [1, 2503146884])
def test_keying_scheme1_plane_and_tail(seed):
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for P in [0, 31, 32, 127, 128, 129, 99999, (1 << 38) + 77]:
        for t, c in [(0, 0), (3, 1), (65, 0)]:
            G, lane = P >> 7, P & 127
            u = 0
            for k in range(8):
                blk = oracle.philox4x32_10([G & 0xFFFFFFFF, G >> 32, t, _ctr_word3(c, 3, k)], key)
                bit = (int(blk[lane >> 5]) >> (lane & 31)) & 1
                u |= bit << (31 - k)
            tail = oracle.philox4x32_10([P & 0xFFFFFFFF, P >> 32, t, _ctr_word3(c, 4, 0)], key)
            u |= int(tail[0]) >> 8
            assert oracle.u32(seed, 1, t, c, P) == u
            blk = oracle.philox4x32_10([G & 0xFFFFFFFF, G >> 32, t, _ctr_word3(c, 5, 0)], key)
            assert oracle.proposal_bit(seed, t, c, P) == (int(blk[lane >> 5]) >> (lane & 31)) & 1


@pytest.mark.parametrize("scheme", [0, 1])
def test_u32_is_uniform(scheme):
    # chi-square of the top byte and of a low byte over 2^16 sites; bits are fair
    n = 1 << 16
    u = np.array([oracle.u32(42, scheme, 5, 1, P) for P in range(n)], dtype=np.uint64)
    for shift in (24, 3):
        counts = np.bincount(((u >> shift) & 0xFF).astype(np.int64), minlength=256)
        chi2 = ((counts - n / 256) ** 2 / (n / 256)).sum()
        assert chi2 < 255 + 6 * math.sqrt(2 * 255)          # ~6 sigma
    ones = sum(int(((u >> b) & 1).sum()) for b in range(32))
    assert abs(ones - 16 * n) < 5 * math.sqrt(32 * n) / 2
    # different sweeps / colours / sites decorrelate
    v = np.array([oracle.u32(42, scheme, 6, 1, P) for P in range(4096)], dtype=np.float64)
    w = u[:4096].astype(np.float64)
    assert abs(np.corrcoef(v, w)[0, 1]) < 0.08


def test_initial_state_is_disordered_and_keyed():
    L = 256
    s = np.array([[oracle.lib().oracle_initial_spin(9, 0, L, i, j) for j in range(L)]
                  for i in range(L)])
    assert set(np.unique(s)) == {-1, 1}
    assert abs(s.mean()) < 5 / L                       # 5 sigma, sigma = 1/L
    # keying: Ising INIT plane, tag 0, unit P>>7
    for (i, j) in [(0, 0), (3, 77), (200, 255)]:
        c, P = (i + j) & 1, i * (L // 2) + (j >> 1)
        blk = oracle.philox4x32_10([P >> 7, 0, 0, _ctr_word3(c, 0, 0)], [9, 0])
        bit = (int(blk[(P & 127) >> 5]) >> (P & 31)) & 1
        assert s[i, j] == (1 if bit else -1)
    b = np.array([[oracle.lib().oracle_initial_spin(9, 1, L, i, j) for j in range(L)]
                  for i in range(L)])
    frac = [(b == v).mean() for v in (-1, 0, 1)]
    for f in frac:
        assert abs(f - 1 / 3) < 5 * math.sqrt(2 / 9) / L
    for (i, j) in [(0, 1), (17, 4), (255, 254)]:
        c, P = (i + j) & 1, i * (L // 2) + (j >> 1)
        blk = oracle.philox4x32_10([P >> 2, 0, 0, _ctr_word3(c, 1, 0)], [9, 0])
        assert b[i, j] == ((int(blk[P & 3]) * 3) >> 32) - 1


# ---------------------------------------------------------------------------- thresholds
getcontext().prec = 60


def _floor_2_32_exp(minus_x: Decimal) -> int:
    return int((Decimal(2) ** 32 * minus_x.exp()).to_integral_value(rounding="ROUND_FLOOR"))


def test_ising_thresholds_closed_form_at_beta_c():
    # exp(-4 beta_c) = (sqrt2 - 1)^2 exactly (Onsager beta_c = ln(1+sqrt2)/2)
    r = Decimal(2).sqrt() - 1
    want4 = int((Decimal(2) ** 32 * r ** 2).to_integral_value(rounding="ROUND_FLOOR"))
    want8 = int((Decimal(2) ** 32 * r ** 4).to_integral_value(rounding="ROUND_FLOOR"))
    assert (want4, want8) == (736899888, 126432032) == (0x2BEC3330, 0x07893320)
    beta_c = math.log(1 + math.sqrt(2)) / 2
    thr = oracle.thresholds(oracle.ISING, 0.0, beta_c)
    # fp64 exp may differ from the exact value in the last ulp: allow +-1 count of 2^32
    assert abs(int(thr[0]) - want4) <= 1 and abs(int(thr[1]) - want8) <= 1


def test_thresholds_limits():
    assert list(oracle.thresholds(oracle.ISING, 0.0, 0.0)) == [1 << 32, 1 << 32]
    assert list(oracle.thresholds(oracle.ISING, 0.0, math.inf)) == [0, 0]
    t0 = oracle.thresholds(oracle.BLUME_CAPEL, 0.3, 0.0)
    assert all(int(x) == 1 << 32 for x in t0)
    tinf = oracle.thresholds(oracle.BLUME_CAPEL, 0.0, math.inf).reshape(3, 2, 9)
    t1 = oracle.thresholds(oracle.BLUME_CAPEL, 0.0, 1.0).reshape(3, 2, 9)
    assert ((tinf == 0) | (tinf == 1 << 32)).all()
    assert ((tinf == 1 << 32) == (t1 == 1 << 32)).all()


@pytest.mark.parametrize("delta,beta", [(0.0, 1 / 1.6934), (1.0, 1.0), (-0.7, 0.37), (1.9, 2.5)])
def test_blume_capel_threshold_table(delta, beta):
    """Every entry against Eq. (1) evaluated independently in decimal arithmetic."""
    thr = oracle.thresholds(oracle.BLUME_CAPEL, delta, beta).reshape(3, 2, 9)
    others = {-1: (0, 1), 0: (1, -1), 1: (-1, 0)}      # code' = (code+1+b) mod 3, sigma = code-1
    for s in (-1, 0, 1):
        for b in (0, 1):
            s2 = others[s][b]
            assert s2 != s and (s2 + 1) == (s + 1 + 1 + b) % 3
            for h in range(-4, 5):
                # H = -s*h + Delta*s^2 for the terms that involve this site
                dE = Decimal(-(s2 - s) * h) + Decimal(repr(delta)) * (s2 * s2 - s * s)
                got = int(thr[s + 1, b, h + 4])
                if dE <= 0:
                    assert got == 1 << 32
                else:
                    want = _floor_2_32_exp(-(Decimal(repr(beta)) * dE))
                    assert abs(got - want) <= max(2, want >> 44)      # fp64 exp: ~1e-15 relative


def test_blume_capel_thresholds_quoted_values():
    # T = 1.6934, Delta = 0, dE = 1..8 (recomputed here in decimal)
    beta = Decimal(1) / Decimal("1.6934")
    want = [_floor_2_32_exp(-(beta * k)) for k in range(1, 9)]
    assert want == [2379560981, 1318359389, 730416868, 404676301, 224204719, 124217197,
                    68820639, 38129023]
    thr = oracle.thresholds(oracle.BLUME_CAPEL, 0.0, 1 / 1.6934).reshape(3, 2, 9)
    # sigma=+1 -> -1 (code 2, b 0): dE = 2h for h = 1..4
    assert [int(x) for x in thr[2, 0, 5:9]] == [want[1], want[3], want[5], want[7]]
    # sigma=+1 -> 0 (code 2, b 1): dE = h
    assert [int(x) for x in thr[2, 1, 5:9]] == want[0:4]


def test_detailed_balance_from_threshold_table_ising_4x4():
    """pi(x) p(x->x^s) = pi(x^s) p(x^s->x) for every state and site, p = thr/2^32.

    The half-sweep kernel factorises over the sites of one colour (their neighbours are of
    the other colour and frozen), so per-site balance implies balance of the half-sweep, and
    pi P_black P_white = pi for the sweep.  Residual: the 2^-32 floor of the thresholds."""
    import exact
    beta = math.log(1 + math.sqrt(2)) / 2
    ex = exact.ising_exact(4, beta)
    s = exact.enumerate_states(4, (-1, 1)).astype(np.int64)
    thr = oracle.thresholds(oracle.ISING, 0.0, beta).astype(np.float64) / 2.0 ** 32
    h = np.roll(s, 1, -1) + np.roll(s, -1, -1) + np.roll(s, 1, -2) + np.roll(s, -1, -2)
    dE = 2 * s * h
    p = np.where(dE <= 0, 1.0, np.where(dE == 4, thr[0], thr[1]))          # acceptance of x -> x^s
    p_back = np.where(-dE <= 0, 1.0, np.where(-dE == 4, thr[0], thr[1]))
    ratio = np.exp(-beta * dE)                                             # pi(x^s)/pi(x)
    assert np.allclose(p, ratio * p_back, rtol=2e-8, atol=0)
    # full sweep leaves pi invariant: apply P_black then P_white to pi by summing over flips
    pi = ex["prob"].copy()
    idx = np.arange(1 << 16)
    for colour in (0, 1):
        sites = [i * 4 + j for i in range(4) for j in range(4) if (i + j) % 2 == colour]
        acc = p.reshape(1 << 16, 16)
        new = np.zeros_like(pi)
        for mask in range(256):
            w = pi.copy()
            y = idx.copy()
            for b, site in enumerate(sites):
                if (mask >> b) & 1:
                    w = w * acc[:, site]
                    y = y ^ (1 << site)
                else:
                    w = w * (1.0 - acc[:, site])
            np.add.at(new, y, w)
        pi = new
    assert np.allclose(pi, ex["prob"], rtol=1e-7, atol=1e-15)


# ---- scheme 2: 56-bit tails and 64-bit thresholds ----------------------
BETA_C = math.log(1.0 + math.sqrt(2.0)) / 2.0
def test_scheme2_u64_extends_scheme1_u32():
    """u64 = top byte | 56 tail bits: its top 32 bits are scheme 1's u32, the next 32 bits are
    word 1 of the site's own tail block."""
    seed = 2503146884
    for t, c, P in [(0, 0, 0), (5, 1, 12345), (2 ** 31 + 7, 0, 2 ** 38 + 99), (17, 1, 127), (17, 1, 128)]:
        u = oracle.u64(seed, t, c, P)
        assert u >> 32 == oracle.u32(seed, 1, t, c, P)
        tail = oracle.philox4x32_10([P & 0xFFFFFFFF, P >> 32, t, c | (4 << 8)],
                                    [seed & 0xFFFFFFFF, seed >> 32])
        assert u & 0xFFFFFFFF == int(tail[1])


def test_thresholds64_refine_the_32_bit_table():
    """floor(thr64 / 2^32) == thr32 entry by entry (same fp64 exp, exact scaling), "always" flags
    agree except where only the 32-bit product rounds up, and closed forms at beta_c hold to the
    53 bits exp() carries."""
    import math
    from fractions import Fraction
    for model, delta, beta in [(oracle.ISING, 0.0, BETA_C), (oracle.BLUME_CAPEL, 0.0, 1 / 1.6934),
                               (oracle.BLUME_CAPEL, 0.7, 0.9), (oracle.ISING, 0.0, 1e-12)]:
        t32 = oracle.thresholds(model, delta, beta)
        t64, alw = oracle.thresholds64(model, delta, beta)
        for a, b, f in zip(t32, t64, alw):
            if f:
                assert int(a) == 2 ** 32
            elif int(a) < 2 ** 32:
                assert int(b) >> 32 == int(a)
    t64, alw = oracle.thresholds64(oracle.ISING, 0.0, BETA_C)
    r2 = Fraction(math.isqrt(2 * 10 ** 60), 10 ** 30)        # sqrt 2 to 30 digits
    for thr, power in zip(t64, (2, 4)):
        exact = (r2 - 1) ** power * 2 ** 64
        assert abs(int(thr) - exact) / exact < 2 ** -50
    # low temperature: the 32-bit table says "never", the 64-bit one still has a probability
    t32 = oracle.thresholds(oracle.ISING, 0.0, 3.0)
    t64, alw = oracle.thresholds64(oracle.ISING, 0.0, 3.0)
    assert int(t32[1]) == 0 and int(t64[1]) == math.floor(math.ldexp(math.exp(-24.0), 64)) > 0
    t64, alw = oracle.thresholds64(oracle.ISING, 0.0, 0.0)
    assert alw.tolist() == [1, 1]
    t64, alw = oracle.thresholds64(oracle.ISING, 0.0, math.inf)
    assert t64.tolist() == [0, 0] and alw.tolist() == [0, 0]


@pytest.mark.parametrize("model,beta", [(oracle.ISING, BETA_C), (oracle.BLUME_CAPEL, 1 / 1.6934)])
def test_scheme2_trajectory_equals_scheme1_when_no_32_bit_tie_occurs(model, beta):
    """The decisions of schemes 1 and 2 differ only if u32 == thr32 (probability 2^-32 per
    decision): on a small run the trajectories are identical, which pins the 64-bit path to the
    pinned 32-bit one."""
    a = oracle.OracleLattice(32, model, 0.0, seed=11, scheme=1)
    b = oracle.OracleLattice(32, model, 0.0, seed=11, scheme=2)
    a.sweep([beta] * 200)
    b.sweep([beta] * 200)
    assert np.array_equal(a.get_spins(), b.get_spins())
