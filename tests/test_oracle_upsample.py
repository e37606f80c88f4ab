"""Pins of the oracle's 10 s -> 5 s linear upsampling (orc_upsample2, reading A20)."""
import numpy as np


def test_linear_series_is_reproduced_exactly(orc):
    N, t0, dt = 64, 3.0, 5.0
    tc = t0 + 2 * dt * np.arange(N // 2 + 1)
    t = t0 + dt * np.arange(N)
    c = np.stack([2.0 - 0.25 * tc, 7.0 + 0.5 * tc])
    assert np.array_equal(orc.upsample2(c), np.stack([2.0 - 0.25 * t, 7.0 + 0.5 * t]))


def test_even_samples_are_the_coarse_samples(orc):
    rng = np.random.default_rng(0)
    c = rng.standard_normal((3, 33))
    f = orc.upsample2(c)
    assert f.shape == (3, 64)
    assert np.array_equal(f[:, 0::2], c[:, :-1])


def test_midpoint_error_of_a_quadratic(orc):
    """linear interpolation of t^2 over a step h overshoots the midpoint by exactly h^2 / 4"""
    h = 10.0
    tc = h * np.arange(17)
    f = orc.upsample2((tc ** 2)[None])[0]
    tm = tc[:-1] + h / 2
    assert np.allclose(f[1::2] - tm ** 2, h * h / 4, rtol=0, atol=1e-9)
