"""Pins of the oracle's kinematics (wavefunctions, vertices, propagators, diagram signs) -- SURVEY.md 8(c).

Closed forms (textbook 2->2 QCD), Parke-Taylor / quark-line MHV partial amplitudes, Ward identity,
Lorentz invariance, parity, Bose symmetry, tier O1 (explicit colour sums, no basis) and tier O3
(Berends-Giele recursion, no diagrams).  A dropped diagram, a wrong relative sign, a wrong factor of the
four-gluon pieces or a transposed colour index fails at least one of them.
"""
import itertools

import numpy as np
import pytest

from oracle import oracle as O


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def sij(k, i, j):
    return mdot(k[i] + k[j], k[i] + k[j])


def mandelstam(mom, e):
    pa, pb, p1, p2 = [mom[i, :, e] for i in range(4)]
    return mdot(pa + pb, pa + pb), mdot(pa - p1, pa - p1), mdot(pa - p2, pa - p2)


CLOSED = {
    # BASELINE.json north_star: sum|M|^2 prop. to 32/27 (t^2+u^2)/(tu) - 8/3 (t^2+u^2)/s^2
    "u u~ > g g": lambda s, t, u: 32 / 27 * (t * t + u * u) / (t * u) - 8 / 3 * (t * t + u * u) / s ** 2,
    "g g > g g": lambda s, t, u: 9 / 2 * (3 - t * u / s ** 2 - s * u / t ** 2 - s * t / u ** 2),
    "u u > u u": lambda s, t, u: 4 / 9 * ((s * s + u * u) / t ** 2 + (s * s + t * t) / u ** 2) - 8 / 27 * s * s / (t * u),
    "u d > u d": lambda s, t, u: 4 / 9 * (s * s + u * u) / t ** 2,
    "u u~ > d d~": lambda s, t, u: 4 / 9 * (t * t + u * u) / s ** 2,
    "u u~ > u u~": lambda s, t, u: 4 / 9 * ((s * s + u * u) / t ** 2 + (t * t + u * u) / s ** 2) - 8 / 27 * u * u / (s * t),
    "g g > u u~": lambda s, t, u: 1 / 6 * (t * t + u * u) / (t * u) - 3 / 8 * (t * t + u * u) / s ** 2,
    "u g > u g": lambda s, t, u: -4 / 9 * (s * s + u * u) / (s * u) + (u * u + s * s) / t ** 2,
}


@pytest.mark.parametrize("name", sorted(CLOSED))
def test_two_to_two_closed_forms(oracle_process, name):
    P = oracle_process(name)
    mom, _, _ = O.sample_momenta(2, 500.0, 0, 64)
    me = P.me2(mom)
    for e in range(64):
        s, t, u = mandelstam(mom, e)
        ref = P.gs ** 4 * CLOSED[name](s, t, u)
        assert abs(me[e] / P.sym_factor / ref - 1.0) < 1e-12


# identical-particle factors 1/prod k! as BASELINE.json's config strings print them: "1/2!" (C1 by the closed form
# below), "1/3!", "1/2! 1/2!", "1/4!", "1/5!"; plus two processes that tell "u and u~ counted together" and "initial legs
# counted" apart.  Mutations this fails: counting u and u~ as identical (u u~ > u u~ would give 1/2), including the initial
# legs (g g > g g g would give 1/5!), forgetting the factor (1).
SYM_LITERALS = {
    "u u~ > g g": 1.0 / 2.0, "g g > g g g": 1.0 / 6.0, "u u > u u g g": 1.0 / 4.0, "g g > g g g g": 1.0 / 24.0,
    "u u~ > g g g g g": 1.0 / 120.0, "u u~ > u u~": 1.0, "u u > u u": 1.0 / 2.0, "u g > u g g": 1.0 / 2.0, "u u~ > d d~": 1.0,
}


@pytest.mark.parametrize("name", sorted(SYM_LITERALS))
def test_identical_particle_factor_literals(oracle_process, name):
    assert oracle_process(name).sym_factor == SYM_LITERALS[name]


def test_c1_absolute_value(oracle_process):
    """The oracle's me2 for BASELINE.json configs[0] itself -- factor included, nothing divided out:
    me2 = (1/2) g^4 [32/27 (t^2+u^2)/(tu) - 8/3 (t^2+u^2)/s^2] with g^2 = 4 pi 0.118 (the literal 1/2 is the 1/2! of P:66)."""
    P = oracle_process("u u~ > g g")
    mom, _, _ = O.sample_momenta(2, 500.0, 0, 256)
    me = P.me2(mom)
    g4 = (4.0 * np.pi * 0.118) ** 2
    for e in range(256):
        s, t, u = mandelstam(mom, e)
        ref = 0.5 * g4 * (32 / 27 * (t * t + u * u) / (t * u) - 8 / 3 * (t * t + u * u) / s ** 2)
        assert abs(me[e] / ref - 1.0) < 1e-12
    # and for identical quarks: 1/2! times the textbook u u -> u u result
    Q = oracle_process("u u > u u")
    mq = Q.me2(mom)
    for e in range(64):
        s, t, u = mandelstam(mom, e)
        ref = 0.5 * g4 * (4 / 9 * ((s * s + u * u) / t ** 2 + (s * s + t * t) / u ** 2) - 8 / 27 * s * s / (t * u))
        assert abs(mq[e] / ref - 1.0) < 1e-12


def all_outgoing(p):
    k = p.copy()
    k[:2] *= -1.0
    return k


@pytest.mark.parametrize("name", ["g g > g g", "g g > g g g", "g g > g g g g"])
def test_parke_taylor(oracle_process, name):
    # |J_sigma|^2 = 2^n g^(2n-4) s_ij^4 / prod s_{sigma_a sigma_a+1}; zero for <2 negative (or positive) helicities
    P = oracle_process(name)
    n = P.n_ext
    mom, _, _ = O.sample_momenta(n - 2, 1000.0, 7, 2)
    p = np.ascontiguousarray(mom[:, :, 1])
    k = all_outgoing(p)
    orders = [P.basis_element(al)[2][0] for al in range(P.n_color)]
    hels = list(itertools.product([-1, 1], repeat=n))
    if n == 6:
        hels = hels[::5]
    n_mhv = 0
    for hel in hels:
        hout = [-hel[i] if i < 2 else hel[i] for i in range(n)]
        neg = [i for i in range(n) if hout[i] < 0]
        _, J, _ = P.amplitudes(p, hel)
        scale = P.gs ** (n - 2) * 1e-9
        if len(neg) < 2 or len(neg) > n - 2:
            assert np.max(np.abs(J)) < scale
            continue
        if len(neg) != 2 and len(neg) != n - 2:
            continue
        pair = neg if len(neg) == 2 else [i for i in range(n) if hout[i] > 0]
        if len(pair) != 2:
            continue
        n_mhv += 1
        for al, o in enumerate(orders):
            den = 1.0
            for a in range(n):
                den *= sij(k, o[a], o[(a + 1) % n])
            pt = 2 ** n * P.gs ** (2 * n - 4) * sij(k, pair[0], pair[1]) ** 4 / abs(den)
            assert abs(abs(J[al]) ** 2 / pt - 1.0) < 1e-9
    assert n_mhv > 0


@pytest.mark.parametrize("name", ["u u~ > g g", "u u~ > g g g", "u u~ > g g g g"])
def test_quark_line_mhv(oracle_process, name):
    # |J_sigma|^2 = 2^k g^2k s_{q i}^3 s_{qb i} / (s_{qb q} s_{q s1} s_{s1 s2} ... s_{sk qb});  q = outgoing quark
    P = oracle_process(name)
    n = P.n_ext
    kg = n - 2
    mom, _, _ = O.sample_momenta(kg, 1000.0, 7, 2)
    p = np.ascontiguousarray(mom[:, :, 0])
    k = all_outgoing(p)
    q, qb = 1, 0        # incoming u~ (leg 1) = outgoing u ; incoming u (leg 0) = outgoing u~
    orders = [P.basis_element(al)[2][0] for al in range(P.n_color)]
    checked = 0
    for hel in itertools.product([-1, 1], repeat=n):
        hout = [-hel[i] if i < 2 else hel[i] for i in range(n)]
        _, J, _ = P.amplitudes(p, hel)
        if hel[0] == hel[1]:          # helicity not conserved along the massless quark line
            assert np.max(np.abs(J)) == 0.0 or np.max(np.abs(J)) < 1e-12
            continue
        neg = [i for i in range(2, n) if hout[i] < 0]
        pos = [i for i in range(2, n) if hout[i] > 0]
        if len(neg) == 0 or len(pos) == 0:
            assert np.max(np.abs(J)) < 1e-9 * P.gs ** kg
            continue
        if len(neg) == 1:
            i, hq = neg[0], hout[q]
        elif len(pos) == 1:
            i, hq = pos[0], -hout[q]
        else:
            continue
        for al, o in enumerate(orders):
            den = sij(k, qb, q) * sij(k, q, o[0]) * sij(k, o[-1], qb)
            for a in range(kg - 1):
                den *= sij(k, o[a], o[a + 1])
            num = sij(k, q, i) ** 3 * sij(k, qb, i) if hq < 0 else sij(k, qb, i) ** 3 * sij(k, q, i)
            pt = 2 ** kg * P.gs ** (2 * kg) * abs(num / den)
            assert abs(abs(J[al]) ** 2 / pt - 1.0) < 1e-9
            checked += 1
    assert checked > 0


@pytest.mark.parametrize("name", ["u u~ > g g", "g g > g g", "g g > g g g", "u u~ > g g g", "u u > u u g",
                                  "u u > u u g g", "u u~ > g g g g", "g g > g g g g"])
def test_ward_identity(oracle_process, name):
    # eps -> p for one external gluon: every colour-basis amplitude vanishes
    P = oracle_process(name)
    n = P.n_ext
    mom, _, _ = O.sample_momenta(n - 2, 1000.0, 5, 1)
    p = np.ascontiguousarray(mom[:, :, 0])
    gluons = [i for i, tok in enumerate(name.replace(">", "").split()) if tok == "g"]
    rng = np.random.default_rng(3)
    C = P.colour_matrix()
    for _ in range(4):
        hel = rng.choice([-1, 1], size=n)
        for wl in gluons:
            sw, Jw, Aw = P.amplitudes(p, hel, ward_leg=wl)
            # compare the colour-summed square with the incoherent diagram sum of the same configuration
            assert np.sqrt(abs(sw)) <= 1e-10 * np.abs(Aw).sum() * np.sqrt(np.abs(C).max())   # 0 <= 0 on helicity-violating lines


def boost_rotate(mom, rng):
    """random rotation + boost applied to all momenta mom[leg,4,E] (plain numpy Lorentz matrices)"""
    th, ph, ps = rng.uniform(0, np.pi), rng.uniform(0, 2 * np.pi), rng.uniform(0, 2 * np.pi)
    def rot(axis, a):
        R = np.eye(4)
        i, j = [(2, 3), (3, 1), (1, 2)][axis]
        R[i, i] = np.cos(a); R[j, j] = np.cos(a); R[i, j] = -np.sin(a); R[j, i] = np.sin(a)
        return R
    R = rot(2, ph) @ rot(1, th) @ rot(2, ps)
    beta = rng.uniform(-0.6, 0.6, size=3)
    b2 = beta @ beta
    g = 1.0 / np.sqrt(1.0 - b2)
    B = np.eye(4)
    B[0, 0] = g
    B[0, 1:] = g * beta
    B[1:, 0] = g * beta
    B[1:, 1:] += (g - 1.0) * np.outer(beta, beta) / b2
    L = B @ R
    return np.einsum("mn,lne->lme", L, mom)


@pytest.mark.parametrize("name,sqrt_s", [("u u~ > g g", 500.0), ("g g > g g g", 1000.0), ("u u > u u g g", 1000.0),
                                         ("u u~ > g g g g", 1000.0)])
def test_lorentz_invariance(oracle_process, name, sqrt_s):
    P = oracle_process(name)
    n_ev = 4
    mom, _, _ = O.sample_momenta(P.n_ext - 2, sqrt_s, 9, n_ev)
    me = P.me2(mom)
    me_b = P.me2(np.ascontiguousarray(boost_rotate(mom, np.random.default_rng(1))))
    assert np.max(np.abs(me_b / me - 1.0)) < 1e-10


@pytest.mark.parametrize("name", ["g g > g g g", "u u > u u g", "u u~ > g g g"])
def test_parity_and_bose_symmetry(oracle_process, name):
    P = oracle_process(name)
    n = P.n_ext
    mom, _, _ = O.sample_momenta(n - 2, 1000.0, 21, 2)
    p = np.ascontiguousarray(mom[:, :, 0])
    for hel in itertools.product([-1, 1], repeat=n):
        a = P.amplitudes(p, hel)[0]
        b = P.amplitudes(p, [-h for h in hel])[0]
        assert abs(a - b) <= 1e-11 * max(abs(a), abs(b)) + 1e-30
    # relabelling identical final-state particles leaves the summed |M|^2 unchanged
    toks = name.replace(">", "").split()
    finals = list(range(2, n))
    same = [(i, j) for i in finals for j in finals if i < j and toks[i] == toks[j]]
    me = P.me2(mom)
    for i, j in same:
        sw = mom.copy()
        sw[[i, j]] = sw[[j, i]]
        assert np.max(np.abs(P.me2(np.ascontiguousarray(sw)) / me - 1.0)) < 1e-11


@pytest.mark.parametrize("name", ["u u~ > g g", "g g > g g", "u u > u u", "g g > g g g", "u u~ > g g g", "u u > u u g"])
def test_colour_basis_vs_explicit_colour_sum(oracle_process, name):
    # tier O2 (eqs. 8-10) against tier O1 (eq. 4/7 summed colour by colour, no basis, no colour matrix)
    P = oracle_process(name, tier1=True)
    n = P.n_ext
    mom, _, _ = O.sample_momenta(n - 2, 1000.0, 2, 3)
    assert np.max(np.abs(P.me2(mom, tier=1) / P.me2(mom, tier=2) - 1.0)) < 1e-12


@pytest.mark.parametrize("name", ["g g > g g", "g g > g g g", "g g > g g g g"])
def test_berends_giele_cross_check(oracle_process, name):
    # tier O3: colour-ordered recursion (no diagram list) reproduces every diagram-built J_sigma
    P = oracle_process(name)
    n = P.n_ext
    mom, _, _ = O.sample_momenta(n - 2, 1000.0, 4, 1)
    p = np.ascontiguousarray(mom[:, :, 0])
    rng = np.random.default_rng(5)
    for _ in range(3):
        hel = rng.choice([-1, 1], size=n)
        _, J, _ = P.amplitudes(p, hel)
        for al in range(0, P.n_color, 1 if n < 6 else 7):
            bg = O.bg_gluon(p, hel, P.basis_element(al)[2][0], P.gs)
            assert abs(bg - J[al]) < 1e-10 * max(np.abs(J).max(), P.gs ** (n - 2))


@pytest.mark.parametrize("name,sqrt_s", [("g g > g g g", 1000.0), ("g g > g g g g", 1500.0)])
def test_explicit_colour_sum_over_bg_amplitudes(oracle_process, name, sqrt_s):
    """gluon_colour_sum_bg (explicit sum over all 8^n colour assignments of traces times Berends-Giele partial amplitudes: no
    diagrams, no colour matrix) against tier O2 (diagrams + colour basis + brute-force matrix) per helicity configuration.  This
    pins the routine that validates g g -> 5 g, where tier O2's colour build (8^7 x 720) is out of reach."""
    P = oracle_process(name)
    n = P.n_ext
    mom, _, _ = O.sample_momenta(n - 2, sqrt_s, 4, 2)
    # physical helicities; the incoming legs 0, 1 flip in the all-outgoing convention: MHV (two negative) and, for n = 6, NMHV
    hels = {5: [[1, 1, 1, 1, 1], [1, -1, 1, -1, 1]], 6: [[1, 1, 1, 1, 1, 1], [1, -1, -1, 1, -1, 1]]}[n]
    for e in range(2):
        p = np.ascontiguousarray(mom[:, :, e])
        for hel in hels:
            s2, _, _ = P.amplitudes(p, hel)
            s1 = O.gluon_colour_sum_bg(p, hel, P.gs)
            assert s2 > 0 and abs(s1 / s2 - 1.0) < 1e-11


def test_parke_taylor_seven_gluons():
    """Berends-Giele partial amplitudes of g g -> 5 g against Parke-Taylor for an MHV configuration (all-outgoing helicities
    with exactly two negative): |A_sigma|^2 = 2^n g^(2n-4) s_ij^4 / prod s_{sigma_a sigma_a+1}, and zero when fewer than two
    helicities differ from the rest."""
    n, gs = 7, np.sqrt(4 * np.pi * 0.118)
    mom, _, _ = O.sample_momenta(5, 2000.0, 13, 1)
    p = np.ascontiguousarray(mom[:, :, 0])
    k = all_outgoing(p)
    rng = np.random.default_rng(3)
    hel_out = np.array([-1, 1, 1, -1, 1, 1, 1])             # all-outgoing helicities: legs 0 and 3 negative
    hel = hel_out.copy(); hel[:2] *= -1                      # physical helicities of the two incoming gluons are flipped
    i, j = 0, 3
    for _ in range(12):
        order = [0] + list(rng.permutation(np.arange(1, n)))
        a = O.bg_gluon(p, hel, order, gs)
        den = 1.0
        for q in range(n):
            den *= sij(k, order[q], order[(q + 1) % n])
        ref = 2.0 ** n * gs ** (2 * n - 4) * sij(k, i, j) ** 4 / abs(den)
        assert abs(abs(a) ** 2 / ref - 1.0) < 1e-9
    # all-plus and one-minus (all-outgoing) vanish
    for hel_out in ([1] * 7, [-1] + [1] * 6):
        h = np.array(hel_out); h[:2] *= -1
        a = O.bg_gluon(p, h, list(range(n)), gs)
        assert abs(a) < 1e-9 * gs ** 5
