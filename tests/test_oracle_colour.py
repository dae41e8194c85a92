"""Pins of the oracle's colour machinery and diagram enumeration against the paper's printed tables
(Table 1, Table 4, colour statistics PAPER.md:215) and against closed-form
SU(3) results (Casimirs), SURVEY.md 8(c) pins.
"""
from fractions import Fraction

import numpy as np
import pytest

from golden_io import rows

TABLE1 = {r[0]: (int(r[1]), int(r[2])) for r in rows("table1_counts.txt")}
TABLE4 = {r[0]: int(r[1]) for r in rows("table4_distinct.txt")}

# processes the CPU suite can afford (g g > 5g and u u > u u g g g are NEXT-4: minutes to hours)
FAST = ["g g > g g", "g g > g g g", "u u~ > g g", "u u~ > g g g", "u u~ > g g g g", "u u > u u", "u u > u u g",
        "u u > u u g g"]
SLOW = ["g g > g g g g", "u u~ > g g g g g"]


def distinct_nonzero(C):
    v = C[np.abs(C) > 1e-9]
    return sorted(set(np.round(v, 8).tolist()))


@pytest.mark.parametrize("name", FAST + SLOW)
def test_table1_and_table4(oracle_process, name):
    P = oracle_process(name)
    assert (P.n_diagrams, P.n_color) == TABLE1[name]
    C = P.colour_matrix()
    assert len(distinct_nonzero(C)) == TABLE4[name]
    # PAPER.md:114 "symmetric"; real and positive semi-definite by construction of eq. 9
    assert P.C_max_asym < 1e-12 and P.C_max_imag < 1e-12
    assert P.colour_eigenvalues().min() > -1e-9
    # every diagram's colour factor is reproduced on EVERY colour assignment by its basis expansion
    assert P.max_residual < 1e-11


def test_topology_counts(oracle_process):
    # plain topologies (4-gluon vertex counted once): (2n-5)!!-type textbook numbers 4, 25, 220 for n gluons
    assert oracle_process("g g > g g").n_topologies == 4
    assert oracle_process("g g > g g g").n_topologies == 25
    assert oracle_process("g g > g g g g").n_topologies == 220
    assert oracle_process("u u~ > g g").n_topologies == 3
    assert oracle_process("u u~ > g g g").n_topologies == 16


def test_colour_matrix_closed_forms(oracle_process):
    # u u~ -> g g : Tr(T^a T^b T^b T^a) = C_F^2 N = 16/3,  Tr(T^a T^b T^a T^b) = C_F (C_F - N/2) N = -2/3
    C = oracle_process("u u~ > g g").colour_matrix()
    assert np.allclose(C, [[16 / 3, -2 / 3], [-2 / 3, 16 / 3]], atol=1e-13)
    # g g -> g g, 6 traces: diagonal 19/6, reflected trace 2/3, others -1/3 (Fierz)
    C = oracle_process("g g > g g").colour_matrix()
    for row in C:
        assert sorted(np.round(row, 10).tolist()) == sorted(np.round([19 / 6, 2 / 3] + [-1 / 3] * 4, 10).tolist())
    assert np.allclose(np.diag(C), 19 / 6)
    # u u -> u u : [[2, -2/3], [-2/3, 2]] for T^e_{j i1} T^e_{j' i2}: Tr(T^e T^f)^2 = (N^2-1)/4 = 2,
    # Tr(T^e T^f T^e T^f) = -2/3
    C = oracle_process("u u > u u").colour_matrix()
    assert np.allclose(C, [[2, -2 / 3], [-2 / 3, 2]], atol=1e-13)
    # u u~ -> k g: diagonal C_F^k N
    assert np.allclose(np.diag(oracle_process("u u~ > g g g").colour_matrix()), 64 / 9)
    assert np.allclose(np.diag(oracle_process("u u~ > g g g g").colour_matrix()), 256 / 27)


def test_colour_values_are_small_rationals(oracle_process):
    C = oracle_process("g g > g g g").colour_matrix()
    vals = [Fraction(v).limit_denominator(2000) for v in distinct_nonzero(C)]
    assert sorted(vals) == sorted(Fraction(a, b) for a, b in
                                  [(455, 108), (17, 27), (7, 54), (5, 108), (-1, 27), (-10, 27), (-29, 54)])
    # rank: full for gluon traces and quark strings, deficient for the two-quark-line set (reading A13)
    assert oracle_process("g g > g g g").color_rank == 24
    assert oracle_process("u u > u u g").color_rank == 4
    assert oracle_process("u u > u u g g").color_rank == 12


def test_colour_sum_rule_gg(oracle_process):
    # sum_alpha Tr(T^{a0} T^{s(a1)} ...) over all (n-1)! orderings is totally symmetric in colour; for n = 4
    # every row of C sums to 19/6 + 2/3 - 4/3 = 5/2
    C = oracle_process("g g > g g").colour_matrix()
    assert np.allclose(C.sum(axis=1), 2.5)
    C = oracle_process("g g > g g g g")
    assert np.allclose(C.colour_matrix().sum(axis=1), 2225 / 216)


def test_monte_carlo_colour_statistics(oracle_process):
    P = oracle_process("g g > g g g g")
    vals = {r[0]: (float(r[1]), float(r[2])) for r in rows("colour_stats_gg4g.txt")}
    assert abs(P.frac_nonzero_pairs - vals["frac_nonzero_pairs"][0]) < vals["frac_nonzero_pairs"][1]
    assert abs(P.frac_all_zero - vals["frac_all_zero"][0]) < vals["frac_all_zero"][1]
