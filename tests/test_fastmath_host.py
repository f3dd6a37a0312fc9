"""CPU-only check of the hand-built Psi evaluator of csrc/psi.cuh (host emulation of the same source, MUFU seeds
emulated at 2^-20) against the long-double oracle Psi: algorithm, tables and guards, with the 256-entry log table and
with the exponent-and-mantissa ("2-D") log table."""
import math

import numpy as np
import pytest

import oracle
from paper_2602_03857_b200 import binding

LN2 = math.log(2.0)


LOG2D = False      # log table under test (set by the autouse fixture: every test runs for both)


@pytest.fixture(autouse=True, params=[False, True], ids=["log256", "log2d"])
def _table(request):
    global LOG2D
    LOG2D = request.param
    yield


def _scaled_err(X, Y, Z, k0=0):
    got = binding.psi_eval_host(X, Y, Z, k0, LOG2D) - (X + Y) * k0 * LN2
    ref = oracle.psi(X, Y, Z, 1)
    R = math.sqrt(X * X + Y * Y + Z * Z)
    if R == 0:
        return abs(got - ref)
    # size of the three terms + amplification of the rounding of R in R+Y (R+X) when Y (X) is negative:
    # the plain double formula has the same sensitivity
    mag = abs(Z) * math.pi / 2 + abs(X * math.log(R + Y)) + abs(Y * math.log(R + X))
    amp = abs(X) * R / (R + Y) + abs(Y) * R / (R + X)
    return abs(got - ref) / (mag + amp + abs(X + Y) * abs(k0) * LN2 + 1e-300)


@pytest.mark.parametrize("scale", [1.0, 30.0, 1e3, 2e4, 3e6])
def test_psi_fast_random(scale):
    rng = np.random.default_rng(int(scale))
    worst = 0.0
    for _ in range(4000):
        X, Y = rng.uniform(-scale, scale, 2)
        Z = rng.uniform(-1, 1) * scale * rng.choice([1, 0.01, 1e-3])
        worst = max(worst, _scaled_err(X, Y, Z), _scaled_err(X, Y, Z, k0=13))
    assert worst <= 1e-15


def test_psi_fast_guards_and_special_points():
    pts = [(0, 0, 0), (0, -5, 0), (2, 3, 0), (0, 0, 5), (1, 1, 1), (3, -4, 0), (-3, 4, 1e-9), (0, 5, 2),
           (5, 0, 2), (-5, 0, -2), (1e-8, -1e4, 1e-8), (7, 7, 7), (7, -7, -7)]
    if LOG2D:         # the 2-D log table is only used when the geometry keeps R+Y, R+X inside its binades (never 0)
        pts = [a for a in pts if math.sqrt(sum(v * v for v in a)) + min(a[0], a[1]) > 1e-22]
    for args in pts:
        got = binding.psi_eval_host(*args, 0, LOG2D)
        assert math.isfinite(got)
        ref = oracle.psi(*args, 1)
        assert abs(got - ref) <= 1e-15 * max(1.0, abs(ref)) + 1e-12 * (args == (1e-8, -1e4, 1e-8))
    # every atan table interval and both table halves: ratio |XY|/(|Z|R) sweeps 1e-3 .. 1e3
    for q in np.logspace(-3, 3, 400):
        X = Y = 1.0
        # |XY|/(|Z| R) = q with R = sqrt(2 + Z^2): solve Z^2 (2 + Z^2) = 1/q^2
        Z = math.sqrt(-1 + math.sqrt(1 + 1 / q ** 2))
        assert _scaled_err(X, Y, Z) <= 1e-15
        assert _scaled_err(-X, Y, Z) <= 1e-15
        assert _scaled_err(X, Y, -Z) <= 1e-15
    # every log table interval: R + Y sweeps two octaves finely
    for a in np.linspace(1.0, 4.0, 1500):
        assert _scaled_err(0.5, a, 0.25) <= 1e-15
