"""the paper's second spin-1/2 systems (Fig. 3 c-f): the N = 20 ring and the N = 20
dodecahedron.  `-m "not gpu"`: the bond lists against textbook graph facts and the oracle's one-magnon sector against
its closed form; `-m gpu`: all M >= 0 sectors through ftlm_lanczos + ftlm_thermo (batched chains) against the oracle."""
import math

import numpy as np
import pytest

from oracle import ftlm_oracle as fo
from paper_2605_26261_b200 import workloads as W


def _adjacency(w):
    A = np.zeros((w.N, w.N))
    A[w.bond_i, w.bond_j] = 1.0
    return A + A.T


def test_dodecahedron_is_the_dodecahedral_graph():
    w = W.paper_workload("dodecahedron")
    assert (w.N, w.n_bonds, w.R, w.n_steps, w.sectors) == (20, 30, 100, 100, list(range(10, 21)))
    A = _adjacency(w)
    assert (A.sum(axis=0) == 3).all()
    # spectrum of the dodecahedral graph: 3, sqrt5 (x3), 1 (x5), 0 (x4), -2 (x4), -sqrt5 (x3)
    ev = np.sort(np.linalg.eigvalsh(A))
    ref = np.sort([3.0] + [math.sqrt(5)] * 3 + [1.0] * 5 + [0.0] * 4 + [-2.0] * 4 + [-math.sqrt(5)] * 3)
    assert np.abs(ev - ref).max() < 1e-12
    # girth 5 and twelve pentagons: closed walks tr A^3 = 0 (no triangles), tr A^4 counts only backtracking walks
    # (2 E + 4 sum_v C(deg, 2) = 60 + 240), and tr A^5 = 10 x (number of 5-cycles)
    assert round(np.trace(np.linalg.matrix_power(A, 3))) == 0
    assert round(np.trace(np.linalg.matrix_power(A, 4))) == 2 * 30 + 4 * 20 * 3
    assert round(np.trace(np.linalg.matrix_power(A, 5))) == 10 * 12


def test_ring20_definition():
    w = W.paper_workload("ring20")
    assert (w.N, w.n_bonds, w.R, w.n_steps, w.sectors) == (20, 20, 100, 100, list(range(10, 21)))
    A = _adjacency(w)
    assert (A.sum(axis=0) == 2).all() and round(np.trace(np.linalg.matrix_power(A, 20))) > 0
    assert np.abs(np.sort(np.linalg.eigvalsh(A)) - np.sort(2 * np.cos(2 * np.pi * np.arange(20) / 20))).max() < 1e-12


@pytest.mark.parametrize("name", ["ring20", "dodecahedron"])
def test_oracle_one_magnon_sector_closed_form(name):
    """One up spin (N_up = 1) hops on the graph: H = (sum_b J_b / 4 - deg / 2) 1 + A / 2 for J = 1 (Eq. 12-14 at s = 1/2):
    spectrum = N_B/4 - deg/2 + (adjacency eigenvalues)/2.  Pins the oracle on these bond lists; by the SU(2) nesting
    the same levels reappear in every sector down to M = 0."""
    w = W.paper_workload(name)
    deg = 2 if name == "ring20" else 3
    ev = np.linalg.eigvalsh(fo.dense_H(w.N, w.bond_i, w.bond_j, w.J, 0.0, 1))
    ref = np.sort(w.n_bonds / 4.0 - deg / 2.0 + np.linalg.eigvalsh(_adjacency(w)) / 2.0)
    assert np.abs(ev - ref).max() < 1e-12
    assert ev[-1] == pytest.approx(w.n_bonds / 4.0)                    # the ferromagnetic level sum_b J_b / 4
    ev2 = np.linalg.eigvalsh(fo.dense_H(w.N, w.bond_i, w.bond_j, w.J, 0.0, 2))
    for x in ev:                                                        # SU(2): sector N_up = 1 is contained in N_up = 2
        assert np.abs(ev2 - x).min() < 1e-9
