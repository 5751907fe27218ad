"""Oracle interval primitives against exact rational arithmetic and mpmath.

Every arithmetic primitive must return the TIGHTEST enclosure (lower endpoint = RD of the exact
result, upper = RU): checked with python Fractions, which are exact.  Elementary functions must
contain the 50-digit mpmath value of every sampled point and stay within their stated pad.
"""
import math
import random
from fractions import Fraction as F

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as o

ADD, SUB, MUL, SQR, DIV, SQRT, SIN, COS, ATAN2, RECIP, SCALE = range(11)
INF = math.inf


def nxt(x, prec):
    return float(np.nextafter(np.float32(x), np.float32(INF))) if prec == 32 else math.nextafter(x, INF)


def prv(x, prec):
    return float(np.nextafter(np.float32(x), np.float32(-INF))) if prec == 32 else math.nextafter(x, -INF)


def assert_tight(lo, hi, exact_lo: F, exact_hi: F, prec=64):
    """lo = RD(exact_lo), hi = RU(exact_hi)."""
    assert F(lo) <= exact_lo and F(hi) >= exact_hi
    assert F(nxt(lo, prec)) > exact_lo, (lo, float(exact_lo))
    assert F(prv(hi, prec)) < exact_hi, (hi, float(exact_hi))


def rnd(rng, prec):
    m = rng.choice([1e-3, 1.0, 37.0, 450.0, 1e5])
    x = rng.uniform(-m, m)
    return float(np.float32(x)) if prec == 32 else x


def rnd_iv(rng, prec, positive=False):
    a, b = sorted((rnd(rng, prec), rnd(rng, prec)))
    kind = rng.random()
    if kind < 0.15:
        b = a                       # thin
    if positive:
        a, b = sorted((abs(a) + 1e-3, abs(b) + 1e-3))
        if prec == 32:
            a, b = float(np.float32(a)), float(np.float32(b))
            a, b = min(a, b), max(a, b)
    return a, b


@pytest.mark.parametrize("prec", [64, 32])
def test_add_sub_mul_sqr_scale_are_tight(prec):
    rng = random.Random(11 + prec)
    for _ in range(4000):
        a, b = rnd_iv(rng, prec), rnd_iv(rng, prec)
        lo, hi = o.prim(ADD, a, b, prec)
        assert_tight(lo, hi, F(a[0]) + F(b[0]), F(a[1]) + F(b[1]), prec)
        lo, hi = o.prim(SUB, a, b, prec)
        assert_tight(lo, hi, F(a[0]) - F(b[1]), F(a[1]) - F(b[0]), prec)
        prods = [F(x) * F(y) for x in a for y in b]
        lo, hi = o.prim(MUL, a, b, prec)
        assert_tight(lo, hi, min(prods), max(prods), prec)
        sq = [F(a[0]) ** 2, F(a[1]) ** 2]
        lo, hi = o.prim(SQR, a, prec=prec)
        if a[0] <= 0 <= a[1]:
            assert lo == 0.0
            assert_tight(0.0, hi, F(0), max(sq), prec)
        else:
            assert_tight(lo, hi, min(sq), max(sq), prec)
        c = rnd(rng, prec)
        lo, hi = o.prim(SCALE, a, (c, c), prec)
        sc = [F(c) * F(a[0]), F(c) * F(a[1])]
        assert_tight(lo, hi, min(sc), max(sc), prec)


@pytest.mark.parametrize("prec", [64, 32])
def test_mul_sign_cases(prec):
    """All nine sign combinations incl. zero endpoints and signed zeros."""
    pts = [-3.5, -1.25, -0.0, 0.0, 0.75, 2.5]
    ivs = [(x, y) for x in pts for y in pts if x <= y]
    for a in ivs:
        for b in ivs:
            prods = [F(x) * F(y) for x in a for y in b]
            lo, hi = o.prim(MUL, a, b, prec)
            assert F(lo) == min(prods) and F(hi) == max(prods)


@pytest.mark.parametrize("prec", [64, 32])
def test_div_recip_sqrt_are_tight(prec):
    rng = random.Random(5 + prec)
    for _ in range(3000):
        a, b = rnd_iv(rng, prec), rnd_iv(rng, prec, positive=True)
        lo, hi = o.prim(DIV, a, b, prec)
        q = [F(x) / F(y) for x in a for y in b]
        assert_tight(lo, hi, min(q), max(q), prec)
        lo, hi = o.prim(RECIP, b, prec=prec)
        assert_tight(lo, hi, 1 / F(b[1]), 1 / F(b[0]), prec)
        lo, hi = o.prim(SQRT, b, prec=prec)
        # RD(sqrt x): lo^2 <= x < next(lo)^2 ;  RU: prev(hi)^2 < x <= hi^2
        assert F(lo) ** 2 <= F(b[0]) < F(nxt(lo, prec)) ** 2
        assert F(prv(hi, prec)) ** 2 < F(b[1]) <= F(hi) ** 2
    # exact squares and the clamp of a negative lower endpoint
    assert o.prim(SQRT, (4.0, 9.0)) == (2.0, 3.0)
    assert o.prim(SQRT, (-1.0, 16.0)) == (0.0, 4.0)


def _ulp(x, prec):
    x = abs(x)
    return (nxt(x, prec) - x) if x > 0 else (5e-324 if prec == 64 else 1.4e-45)


@pytest.mark.parametrize("prec", [64, 32])
def test_sin_cos_enclose_and_are_narrow(prec):
    mp.mp.dps = 50
    rng = random.Random(3)
    pad = o.pad_ulps()
    for _ in range(1500):
        w = rng.choice([0.0, 1e-9, 1e-3, 0.1, 1.0, 3.0])
        c = rng.uniform(-4, 4)
        a = (max(c - w, -4.0), min(c + w, 4.0))
        if prec == 32:
            a = (float(np.float32(a[0])), float(np.float32(a[1])))
            if a[0] < -4 or a[1] > 4 or a[0] > a[1]:
                continue
        for op, fn, crit in ((SIN, mp.sin, [(mp.pi / 2, 1), (-mp.pi / 2, -1)]),
                             (COS, mp.cos, [(0, 1), (mp.pi, -1), (-mp.pi, -1)])):
            lo, hi = o.prim(op, a, prec=prec)
            vals = [fn(mp.mpf(a[0])), fn(mp.mpf(a[1]))] + [fn(mp.mpf(a[0]) + (mp.mpf(a[1]) - mp.mpf(a[0])) * t / 7) for t in range(1, 7)]
            ex_lo, ex_hi = min(vals), max(vals)
            for xc, v in crit:
                if a[0] <= xc <= a[1]:
                    ex_lo, ex_hi = min(ex_lo, v), max(ex_hi, v)
            assert mp.mpf(lo) <= ex_lo and mp.mpf(hi) >= ex_hi, (a, lo, hi)
            assert -1.0 <= lo and hi <= 1.0
            # narrow: within pad+1 ulps of the exact range (ulp taken at magnitude <= 1)
            tol = (pad + 1.5) * _ulp(1.0, prec)
            assert float(ex_lo - mp.mpf(lo)) <= tol and float(mp.mpf(hi) - ex_hi) <= tol, (a, lo, hi)
    # outside [-4,4] and NaN: whole range
    assert o.prim(SIN, (-5.0, 0.0), prec=prec) == (-1.0, 1.0)
    assert o.prim(COS, (0.0, 4.5), prec=prec) == (-1.0, 1.0)
    assert o.prim(SIN, (float("nan"), 0.0), prec=prec) == (-1.0, 1.0)
    # critical points
    assert o.prim(SIN, (1.0, 2.0), prec=prec)[1] == 1.0
    assert o.prim(SIN, (-2.0, -1.0), prec=prec)[0] == -1.0
    assert o.prim(COS, (-0.5, 0.25), prec=prec)[1] == 1.0
    assert o.prim(COS, (3.0, 3.5), prec=prec)[0] == -1.0
    assert o.prim(COS, (-3.5, -3.0), prec=prec)[0] == -1.0


@pytest.mark.parametrize("prec", [64, 32])
def test_atan2_encloses_rectangle(prec):
    mp.mp.dps = 50
    rng = random.Random(9)
    pad = o.pad_ulps()
    # smallest representable number >= pi: double(pi) < pi, float(pi) > pi
    PI_HI = math.nextafter(math.pi, 4.0) if prec == 64 else float(np.float32(math.pi))
    assert mp.mpf(PI_HI) > mp.pi > mp.mpf(prv(PI_HI, prec))
    for _ in range(1500):
        y, x = rnd_iv(rng, prec), rnd_iv(rng, prec)
        lo, hi = o.prim(ATAN2, y, x, prec)
        if x[0] <= 0 and y[0] <= 0 <= y[1]:
            assert (lo, hi) == (-PI_HI, PI_HI)       # cut or origin
            continue
        # dense boundary + interior sampling of the rectangle
        vals = []
        for s in range(9):
            for t in range(9):
                yy = mp.mpf(y[0]) + (mp.mpf(y[1]) - mp.mpf(y[0])) * s / 8
                xx = mp.mpf(x[0]) + (mp.mpf(x[1]) - mp.mpf(x[0])) * t / 8
                vals.append(mp.atan2(yy, xx))
        assert mp.mpf(lo) <= min(vals) and mp.mpf(hi) >= max(vals), (y, x, lo, hi)
        tol = (pad + 1.5) * _ulp(4.0, prec)
        assert float(min(vals) - mp.mpf(lo)) <= tol and float(mp.mpf(hi) - max(vals)) <= tol
