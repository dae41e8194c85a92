"""Pins of the oracle's steps a1-a2 (Philox, massless RAMBO, cuts): SURVEY.md 8(c) 'RAMBO' row.

What fixes them: Random123 known-answer vectors, four-momentum conservation, masslessness, the closed-form
two-body phase-space volume 1/(8 pi), isotropy moments, and the cut definitions of PAPER.md:118-135
(eqs. 14-15) in the BASELINE.json variant (reading A9).
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from golden_io import rows


def test_philox_known_answers():
    for c, k, e in rows("philox_kat.txt"):
        ctr = [int(x, 16) for x in c.split()]
        key = [int(x, 16) for x in k.split()]
        exp = [int(x, 16) for x in e.split()]
        assert list(O.philox4x32_10(ctr, key)) == exp


@pytest.mark.parametrize("n_final,sqrt_s,seed", [(2, 500.0, 0), (3, 1000.0, 1), (4, 1500.0, 3), (5, 2000.0, 4)])
def test_rambo_conservation_masslessness_cuts(n_final, sqrt_s, seed):
    n = 2048
    mom, w, tries = O.sample_momenta(n_final, sqrt_s, seed, n)
    assert mom.shape == (n_final + 2, 4, n)
    # beams: sqrt(s)/2 (1,0,0,+-1)
    h = 0.5 * sqrt_s
    assert np.all(mom[0] == np.array([h, 0, 0, h])[:, None])
    assert np.all(mom[1] == np.array([h, 0, 0, -h])[:, None])
    tot = mom[2:].sum(axis=0)
    assert np.max(np.abs(tot[0] - sqrt_s)) < 1e-10 * sqrt_s   # RAMBO divides by M = sqrt(Q^2): conditioning ~ eps Q0^2/M^2
    assert np.max(np.abs(tot[1:])) < 1e-10 * sqrt_s
    m2 = mom[2:, 0] ** 2 - (mom[2:, 1:] ** 2).sum(axis=1)
    assert np.max(np.abs(m2)) < 1e-10 * sqrt_s ** 2
    assert np.all(mom[2:, 0] > 0)
    # cuts, re-computed here with numpy from their definition (pT, eta, Delta R)
    pt = np.hypot(mom[2:, 1], mom[2:, 2])
    pabs = np.sqrt((mom[2:, 1:] ** 2).sum(axis=1))
    eta = np.arctanh(mom[2:, 3] / pabs)
    phi = np.arctan2(mom[2:, 2], mom[2:, 1])
    assert np.all(pt > 20.0) and np.all(np.abs(eta) < 2.5)
    for i in range(n_final):
        for j in range(i + 1, n_final):
            dphi = np.abs(phi[i] - phi[j])
            dphi = np.where(dphi > np.pi, 2 * np.pi - dphi, dphi)
            assert np.all(np.hypot(eta[i] - eta[j], dphi) > 0.4)
    assert np.all(tries >= 1) and np.all(w == O.rambo_weight(n_final, sqrt_s))


def test_rambo_two_body_weight_is_one_over_8pi():
    # closed form: massless two-body phase space  int dPhi_2 = 1/(8 pi)
    assert abs(O.rambo_weight(2, 500.0) - 1.0 / (8.0 * math.pi)) < 1e-16
    # three-body: s/(256 pi^3)
    s = 1000.0 ** 2
    assert abs(O.rambo_weight(3, 1000.0) / (s / (256.0 * math.pi ** 3)) - 1.0) < 1e-14


def test_rambo_isotropy_without_cuts():
    n = 200000
    mom, w, tries = O.sample_momenta(3, 1000.0, 11, n, pt_min=0.0, eta_max=0.0, dr_min=0.0)
    assert np.all(tries == 1)
    p = mom[2]                       # first final-state particle
    c = p[3] / p[0]
    # uniform cos(theta): <c> = 0, <c^2> = 1/3 ; uniform phi: <cos 2phi> = 0
    assert abs(c.mean()) < 5.0 / math.sqrt(3 * n)
    assert abs((c * c).mean() - 1.0 / 3.0) < 5.0 * math.sqrt(4.0 / 45.0 / n)
    phi = np.arctan2(p[2], p[1])
    assert abs(np.cos(2 * phi).mean()) < 5.0 / math.sqrt(2 * n)
    # energy spectrum of massless 3-body phase space: <E> = sqrt(s)/3 exactly by symmetry
    assert abs(mom[2:, 0].mean() - 1000.0 / 3.0) < 1e-9


def test_rambo_energy_law_three_body():
    """Flat massless 3-body phase space: x_i = 2 E_i / sqrt(s) has the marginal density 2x on [0, 1] (the Dalitz triangle
    x_1 + x_2 + x_3 = 2 is uniformly populated), so <E^2> = s/8 and, with sum E = sqrt(s), <E_i E_j> = 5 s / 48 for i != j.
    <E> = sqrt(s)/3 holds by symmetry for ANY q0 law, so it pins nothing; these second moments do: drawing q0 = -ln(u3)
    instead of -ln(u3 u4) (reading A7) gives <E^2> = 0.1313 s (and P(x < 1/2) = 0.277) -- about 39 sigma away at this sample size."""
    n = 200000
    s = 1000.0 ** 2
    mom, w, tries = O.sample_momenta(3, 1000.0, 12, n, pt_min=0.0, eta_max=0.0, dr_min=0.0)
    E = mom[2:, 0]                                  # [3, n]
    x = 2.0 * E / 1000.0
    # var(x^2) under density 2x: <x^4> - <x^2>^2 = 1/3 - 1/4 = 1/12
    for i in range(3):
        assert abs((E[i] ** 2).mean() - s / 8.0) < 5.0 * (s / 4.0) * math.sqrt(1.0 / 12.0 / n)
    for i in range(3):
        for j in range(i + 1, 3):
            prod = x[i] * x[j]
            assert abs(prod.mean() - 5.0 / 12.0) < 5.0 * prod.std() / math.sqrt(n)
    # the whole marginal, not only its moments: P(x < 1/2) = 1/4, P(x < 0.9) = 0.81
    for q, pr in [(0.5, 0.25), (0.9, 0.81)]:
        assert abs((x[0] < q).mean() - pr) < 5.0 * math.sqrt(pr * (1 - pr) / n)


def test_event_index_is_global_counter():
    # reading A17/A18: event e of a batch starting at first_event equals event first_event+e of a batch from 0
    a, wa, ta = O.sample_momenta(3, 1000.0, 1, 64, first_event=0)
    b, wb, tb = O.sample_momenta(3, 1000.0, 1, 16, first_event=40)
    assert np.array_equal(a[:, :, 40:56], b) and np.array_equal(ta[40:56], tb)
    c, _, _ = O.sample_momenta(3, 1000.0, 2, 64)
    assert not np.array_equal(a, c)


def test_cut_function_edges():
    # a 2-body back-to-back configuration at eta = 0 passes; same at pT just below threshold fails
    def two(pt, eta):
        pz = pt * math.sinh(eta)
        e = pt * math.cosh(eta)
        return np.array([[e, pt, 0.0, pz], [e, -pt, 0.0, -pz]])
    assert O.pass_cuts(two(50.0, 0.0))
    assert not O.pass_cuts(two(19.999, 0.0))
    assert O.pass_cuts(two(50.0, 2.49)) and not O.pass_cuts(two(50.0, 2.51))
    # Delta R: two nearly collinear particles
    e = 100.0
    a = np.array([[e, e * math.cos(0.0), e * math.sin(0.0), 0.0], [e, e * math.cos(0.39), e * math.sin(0.39), 0.0]])
    b = np.array([[e, e * math.cos(0.0), e * math.sin(0.0), 0.0], [e, e * math.cos(0.41), e * math.sin(0.41), 0.0]])
    assert not O.pass_cuts(a) and O.pass_cuts(b)
    # phi wrap-around: phi = +3.1 and -3.1 are 0.083 apart, not 6.2
    c = np.array([[e, e * math.cos(3.1), e * math.sin(3.1), 0.0], [e, e * math.cos(-3.1), e * math.sin(-3.1), 0.0]])
    assert not O.pass_cuts(c)
    assert O.pass_cuts(c, dr_min=0.0)
