"""Worked values printed in the paper (tests/golden/paper_values.txt), checked against the oracle
and the generators."""
import os

import numpy as np
import pytest

from workloads import generators as gen

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_two_particle_cell(orc):
    g = golden()
    for L in (1.0, 0.37):
        pm = np.array([[0.2, 0.1, 0.3, 1.5], [0.2 + L, 0.1, 0.3, 1.5]], np.float32)
        t = orc.Tree(pm, 16)
        b, _ = t.sph_cell_radii(np.zeros(2, np.float32))
        Lf = float(pm[1, 0]) - float(pm[0, 0])
        assert b[0] == pytest.approx(g["two_particle_cell_bmax_over_L"] * Lf, rel=1e-6)


def test_lane_emden_constant():
    xs, ths, ms = gen.lane_emden(1.5)
    assert xs[-1] == pytest.approx(golden()["lane_emden_n1.5_xi1"], rel=1e-5)
