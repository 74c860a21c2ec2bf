"""Pins of the oracle's radial-distribution counts (oracle_rdf_counts; Eq. (11)) against
what the mathematics fixes: the coordination shells of the fcc lattice, the 13-atom icosahedron, the
Mackay shells, the total count, and a numpy brute force that shares no code with it."""
import math

import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W


def brute(pos, centre, r_select, bin_width, n_bins):
    pos = np.asarray(pos)
    sel = np.where(((pos - centre) ** 2).sum(axis=1) < r_select ** 2)[0]
    counts = np.zeros(n_bins, dtype=np.int64)
    for i in sel:
        d = np.sqrt(((pos - pos[i]) ** 2).sum(axis=1))
        d = np.delete(d, i)
        b = np.floor(d / bin_width).astype(np.int64)
        counts += np.bincount(b[b < n_bins], minlength=n_bins)[:n_bins]
    return counts, len(sel)


def test_fcc_coordination_shells(oracle_ld):
    """Central atom of an unjittered fcc sphere (a = 3.52): neighbours at a sqrt(k/2), k = 1..7, number
    12, 6, 24, 12, 24, 8, 48 (textbook fcc coordination sequence)."""
    a = 3.52
    pos = W.fcc_sphere(2000)
    width = 0.05
    counts, n_ref, centre = oracle_ld.rdf_counts(pos, 1.0, width, 140, centre=[0.0, 0.0, 0.0])
    assert n_ref == 1
    expect = [12, 6, 24, 12, 24, 8, 48]
    for k, z in enumerate(expect, start=1):
        r = a * math.sqrt(k / 2.0)
        assert counts[int(r / width)] == z, (k, r)
    assert counts[: int(a * math.sqrt(3.5) / width) + 1].sum() == sum(expect)      # nothing in between


def test_icosahedron_and_mackay_shells(oracle_ld):
    """Ni147 Mackay (radial spacing 2.49 A): the central atom sees 12 atoms at 2.49 A and the 12 vertices
    of shells 2 and 3 at 4.98 and 7.47 A; with the paper's 3 A selection the 13 innermost atoms are the
    reference set (centre of mass = the central atom)."""
    pos = W.mackay_icosahedron(3, 2.49)
    counts, n_ref, centre = oracle_ld.rdf_counts(pos, 3.0, 0.4, 40)
    assert n_ref == 13 and np.allclose(centre, 0.0, atol=1e-12)
    assert counts.sum() == 13 * 146                                   # 16 A covers the whole cluster
    only_centre, n1, _ = oracle_ld.rdf_counts(pos, 0.1, 0.01, 800)
    assert n1 == 1
    assert only_centre[int(2.49 / 0.01 - 0.5)] + only_centre[int(2.49 / 0.01 + 0.5)] >= 12
    assert only_centre[:245].sum() == 0 and only_centre[: int(2.6 / 0.01)].sum() == 12
    # a first-shell atom A d has 12 nearest neighbours: the centre, the shell-2 vertex 2 A d and the five shell-2
    # edge atoms (A + B) d at 2.49 A, and its five shell-1 neighbours B d at the tangential edge 1.0514622 * 2.49 A
    one, n1, _ = oracle_ld.rdf_counts(pos, 0.1, 0.01, 300, centre=pos[1])
    assert n1 == 1 and one[248:250].sum() == 7 and one[261:263].sum() == 5 and one[:300].sum() == 12


def test_dimer_and_total(oracle_ld):
    pos = np.array([[0.0, 0.0, 0.0], [0.0, 3.0, 4.0]])               # r = 5 exactly
    counts, n_ref, centre = oracle_ld.rdf_counts(pos, 100.0, 0.4, 20)
    assert n_ref == 2 and counts[12] == 2 and counts.sum() == 2       # 5 / 0.4 = 12.5
    assert np.allclose(centre, [0.0, 1.5, 2.0])
    counts, n_ref, _ = oracle_ld.rdf_counts(pos, 100.0, 0.4, 12)      # the bin lies beyond the histogram
    assert counts.sum() == 0
    counts, n_ref, _ = oracle_ld.rdf_counts(pos[:1], 1.0, 0.4, 5)     # N = 1
    assert n_ref == 1 and counts.sum() == 0


@pytest.mark.parametrize("seed", [1, 2])
def test_against_numpy_brute_force(oracle_ld, seed):
    w = W.fcc_cluster(700, 1500.0, seed=seed)
    centre = w.pos.mean(axis=0)
    counts, n_ref, c_used = oracle_ld.rdf_counts(w.pos, 6.0, 0.4, 30)
    assert np.allclose(c_used, centre, atol=1e-12)
    ref, n = brute(w.pos, centre, 6.0, 0.4, 30)
    assert n_ref == n and n > 40
    assert np.array_equal(counts, ref)
    # explicit centre, strict selection, selection of everything: total = N (N - 1)
    counts, n_ref, _ = oracle_ld.rdf_counts(w.pos, 1e3, 1.0, 100, centre=[1.0, -2.0, 0.5])
    assert n_ref == 700 and counts.sum() == 700 * 699
