"""Seeded synthetic input generators (reading R13/R6).

This module holds none of the method's arithmetic: it only draws the random
initial states and per-element parameters that BOTH the CUDA path and the
oracle are handed.  Generator: numpy PCG64, ``default_rng([seed, stream])``,
always in float64; fp32 networks round these arrays once (``astype(float32)``).
"""
import math

import numpy as np

_STREAM_STATE, _STREAM_PARAM = 0, 1


def _u(n, seed, stream):
    return np.random.default_rng([int(seed), stream]).random(int(n))


def ks_phases(n, seed):
    """phi ~ U[-pi, pi)."""
    return -math.pi + 2.0 * math.pi * _u(n, seed, _STREAM_STATE)


def lorentzian_omega(n, seed, gamma=0.01, omega_max=1.0):
    """omega ~ Lorentzian(0, gamma) truncated to |omega| <= omega_max (reading R6).

    Inverse CDF on the sub-interval of u that maps inside the truncation:
    omega = gamma * tan(pi (u' - 1/2)),  u' = 1/2 + (2u - 1) * atan(omega_max/gamma)/pi.
    """
    u = _u(n, seed, _STREAM_PARAM)
    half = math.atan(omega_max / gamma) / math.pi
    return gamma * np.tan(math.pi * (2.0 * u - 1.0) * half)


def fhn_circle(n, seed, radius=2.0):
    """(u, v) on a circle of the given radius with seeded random angles; shape (2, n)."""
    th = 2.0 * math.pi * _u(n, seed, _STREAM_STATE)
    return np.stack([radius * np.cos(th), radius * np.sin(th)])


def hh_voltage(n, seed, lo=-70.0, hi=-50.0):
    """V ~ U[lo, hi) mV.  Gates are set to their steady state by the consumer."""
    return lo + (hi - lo) * _u(n, seed, _STREAM_STATE)


def hh_current(n, seed, lo=9.0, hi=11.0):
    """I_ext ~ U[lo, hi) uA/cm^2."""
    return lo + (hi - lo) * _u(n, seed, _STREAM_PARAM)
