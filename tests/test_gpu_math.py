"""gc_math.cuh: the branch-free divide / reciprocal / square root of the marching kernels must equal the IEEE
operators bit for bit wherever the fast path accepts the operands, and must refuse (fall back) elsewhere."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_fast_math_equals_ieee(gc):
    ctx = gc.Context(coord=0)
    rng = np.random.default_rng(190106798)
    n = 1 << 22
    # mantissas uniform, exponents spread over the window and beyond
    a = rng.uniform(1.0, 2.0, n) * 2.0 ** rng.integers(-520, 520, n) * rng.choice([-1.0, 1.0], n)
    b = rng.uniform(1.0, 2.0, n) * 2.0 ** rng.integers(-520, 520, n) * rng.choice([-1.0, 1.0], n)
    nm, nf = ctx.selftest_math(a, b)
    assert nm == 0
    assert 0 < nf < 3 * n
    # the scheme's range: depths, speeds, squares of tiny waves; positive a for sqrt
    a = np.abs(rng.standard_normal(n)) * 10.0 ** rng.uniform(-40, 8, n)
    b = rng.standard_normal(n) * 10.0 ** rng.uniform(-40, 8, n)
    nm, nf = ctx.selftest_math(a, b)
    assert nm == 0 and nf == 0
    # special operands: zeros of both signs, ones, powers of two, values next to powers of two, huge, tiny, inf, nan
    sp = np.array([0.0, -0.0, 1.0, -1.0, 2.0, 0.5, 3.0, 1.0 / 3.0, np.nextafter(1.0, 2.0), np.nextafter(1.0, 0.0),
                   np.nextafter(4.0, 5.0), np.nextafter(4.0, 3.0), 9.81, 4000.0, 1e-3, 1e-300, 1e300, 5e-324,
                   np.inf, -np.inf, np.nan, 2.0 ** -500, 2.0 ** 500, np.nextafter(2.0 ** -500, 0.0), 2.0 ** 501])
    A, B = np.meshgrid(sp, sp)
    nm, nf = ctx.selftest_math(A.ravel(), B.ravel())
    assert nm == 0 and nf > 0
    # hard cases of Newton reciprocals: mantissas next to a power of two from below (all ones) and from above,
    # with numerators that are powers of two, small integers and random
    k = np.concatenate([np.arange(1, 2049), rng.integers(1, 1 << 30, 4096)]).astype(np.float64)
    bs = np.concatenate([(1.0 - k * 2.0 ** -53), (1.0 + k * 2.0 ** -52), (2.0 - k * 2.0 ** -52)])
    bs = np.concatenate([bs, 4.0 * bs, -bs * 2.0 ** -7, bs * 2.0 ** 300])
    for a in (np.ones_like(bs), 2.0 ** rng.integers(-60, 60, bs.size), rng.integers(1, 1000, bs.size).astype(np.float64),
              rng.uniform(1.0, 2.0, bs.size), np.nextafter(bs, 0.0), np.nextafter(bs, 10.0), bs):
        nm, nf = ctx.selftest_math(np.abs(a), bs)
        assert nm == 0 and nf == 0
    # perfect squares and their neighbours (square-root rounding boundary cases)
    k = rng.integers(1, 1 << 26, n).astype(np.float64)
    sq = k * k
    for x in (sq, np.nextafter(sq, np.inf), np.nextafter(sq, 0.0)):
        nm, nf = ctx.selftest_math(x, k)
        assert nm == 0 and nf == 0
