"""Pins of the oracle's phaseless weight update (Eq. 7-12) by special cases that follow from the
equations without re-typing the formula."""
import cmath
import math

import numpy as np

from oracle import afqmc_oracle as orc


def test_no_force_bias_reduces_to_overlap_ratio():
    # xbar = 0: I = O, so w' = |O| max(0, cos arg O) w
    w = orc.phaseless_weight_update(2.0, complex(-3.0, 0.2), complex(-2.5, 0.5), np.ones(7), np.zeros(7))
    assert abs(w - 2.0 * math.exp(0.5) * math.cos(0.3)) < 1e-14


def test_phase_beyond_quarter_turn_kills_the_walker():
    for dphi in (math.pi / 2 + 1e-9, 2.0, math.pi, -2.5):
        assert orc.phaseless_weight_update(1.0, 0j, complex(0.3, dphi), np.zeros(3), np.zeros(3)) == 0.0
    assert orc.phaseless_weight_update(1.0, 0j, complex(0.3, 2 * math.pi - 0.1), np.zeros(3), np.zeros(3)) > 0.0   # wraps


def test_real_force_bias_gaussian_identity():
    # real xbar, O = 1: I = exp(x.xbar - xbar.xbar/2) = p(x - xbar)/p(x) for the normal density p (Eq. 4, 7)
    rng = np.random.default_rng(0)
    x, xb = rng.standard_normal(11), 0.3 * rng.standard_normal(11)
    ratio = math.exp(-0.5 * np.sum((x - xb) ** 2)) / math.exp(-0.5 * np.sum(x ** 2))
    assert abs(orc.phaseless_weight_update(1.5, 1 + 2j, 1 + 2j, x, xb) - 1.5 * ratio) < 1e-13


def test_imaginary_force_bias_only_changes_the_modulus_through_its_square():
    # purely imaginary xbar = i y: x.xbar is imaginary (a phase), -xbar.xbar/2 = +y.y/2 is real; theta = arg O is untouched
    x, y = np.array([0.5, -1.0, 2.0]), np.array([0.2, 0.1, -0.3])
    w = orc.phaseless_weight_update(1.0, 0j, complex(0.0, 0.4), x, 1j * y)
    assert abs(w - math.exp(0.5 * np.sum(y * y)) * math.cos(0.4)) < 1e-14


def test_linear_in_weight_and_multiplicative_in_overlap_modulus():
    rng = np.random.default_rng(1)
    x, xb = rng.standard_normal(5), rng.standard_normal(5) + 1j * rng.standard_normal(5)
    a = orc.phaseless_weight_update(1.0, complex(-4, 0.1), complex(-3, 0.3), x, xb)
    b = orc.phaseless_weight_update(3.0, complex(-4, 0.1), complex(-2, 0.3), x, xb)
    assert abs(b - 3.0 * math.e * a) < 1e-12 * abs(b)
    assert abs(cmath.phase(cmath.exp(1j * 0.2)) - 0.2) < 1e-15
