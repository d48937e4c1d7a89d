"""Host-side checks of the logarithm table of the heatbath's Kennedy-Pendleton draws (gauge_update.cu:kp_log;
no GPU): the committed header is what its generator writes, and the evaluation scheme the kernel uses -- exponent,
128-entry table, seven-term log1p series, split ln 2 -- re-done here step by step in exact rational arithmetic with one
rounding per fused multiply-add, agrees with the correctly rounded logarithm to 2.3e-16 max(|ln x|, 1) on the whole
range of a draw (multiples of 2^-53 in (0, 1]).  The oracle does not use the table (it calls std::log): this pins the
CUDA path's own constants, which the GPU parity tests then exercise through the heatbath."""
import math
import os
import random
import re
import subprocess
import sys
from fractions import Fraction

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1209_5942_b200", "csrc")


def _table():
    tab, hi, lo = [], None, None
    for line in open(os.path.join(CSRC, "kp_log_table.h")):
        m = re.match(r"\s*\{(\S+), (\S+)\},", line)
        if m:
            tab.append((float.fromhex(m.group(1)), float.fromhex(m.group(2))))
        m = re.match(r"constexpr double KP_LN2_HI = (\S+);", line)
        if m:
            hi = float.fromhex(m.group(1))
        m = re.match(r"constexpr double KP_LN2_LO = (\S+);", line)
        if m:
            lo = float.fromhex(m.group(1))
    return tab, hi, lo


def _fma(a, b, c):
    return float(Fraction(a) * Fraction(b) + Fraction(c))


def _kp_log(x, tab, hi, lo):
    mant, e = math.frexp(x)
    m, e = mant * 2.0, e - 1                   # x = m 2^e, m in [1, 2)
    inv_c, log_c = tab[int((m - 1.0) * 128.0)]
    eps = _fma(m, inv_c, -1.0)
    p = _fma(eps, 1.0 / 7.0, -1.0 / 6.0)
    for c in (0.2, -0.25, 1.0 / 3.0, -0.5):
        p = _fma(p, eps, c)
    p = _fma(p * eps, eps, eps)
    return _fma(float(e), hi, log_c) + _fma(float(e), lo, p)


def test_header_is_what_the_generator_writes():
    out = subprocess.run([sys.executable, os.path.join(CSRC, "gen_kp_log_table.py")], capture_output=True, text=True, check=True)
    assert out.stdout == open(os.path.join(CSRC, "kp_log_table.h")).read()


def test_table_entries_and_ln2_split():
    tab, hi, lo = _table()
    assert len(tab) == 128
    for i, (inv_c, log_c) in enumerate(tab):
        c = 1.0 + (i + 0.5) / 128.0
        assert abs(inv_c * c - 1.0) < 3e-16
        assert abs(log_c + math.log(inv_c)) <= 1.2e-16 * max(abs(log_c), 2.0 ** -8)
        for m in (1.0 + i / 128.0, math.nextafter(1.0 + (i + 1) / 128.0, 0.0)):     # the ends of the entry's interval
            assert abs(m * inv_c - 1.0) <= 2.0 ** -8
    assert math.frexp(hi)[0] * 2 ** 53 % 2 ** 11 == 0          # 11 trailing zero bits: e * KP_LN2_HI is exact
    from decimal import Decimal, getcontext
    getcontext().prec = 50
    ln2 = Fraction(Decimal(2).ln())                            # 50 digits
    assert abs(Fraction(hi) + Fraction(lo) - ln2) < Fraction(1, 2 ** 95)


def test_scheme_matches_the_correctly_rounded_logarithm():
    tab, hi, lo = _table()
    rng = random.Random(12095942)
    ks = [2 ** 53 - t for t in range(2000)] + list(range(1, 2001)) + [2 ** 52 + t for t in range(-1000, 1000)]
    ks += [rng.randrange(1, 2 ** 53 + 1) for _ in range(40000)]
    ks += [(128 + i) << 45 for i in range(128)] + [((128 + i) << 45) - 1 for i in range(1, 129)]   # table-interval ends
    worst = 0.0
    for k in ks:
        x = k * 2.0 ** -53
        want = math.log(x)
        worst = max(worst, abs(_kp_log(x, tab, hi, lo) - want) / max(abs(want), 1.0))
    assert worst <= 2.3e-16
    assert _kp_log(1.0, tab, hi, lo) == 0.0 or abs(_kp_log(1.0, tab, hi, lo)) < 1e-18
