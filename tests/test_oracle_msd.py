"""Pins of the oracle's aligned mean-square displacement (Oracle.msd_aligned; Eq. (12))
against what the mathematics fixes: rigid motions give zero, a dilation has a closed form, the fitted
rotation is a proper one and beats every other rotation (brute force), a single displaced atom, the fcc
shell counts of the selection, and a random walk with a known diffusion coefficient."""
import math

import numpy as np
import pytest

from oracle.sc_oracle import Oracle
from paper_1210_3559_b200 import workloads as W

msd = Oracle.msd_aligned


def rotation(rng):
    """uniform random proper rotation from a unit quaternion"""
    q = rng.normal(size=4)
    a, b, c, d = q / np.linalg.norm(q)
    return np.array([[a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)],
                     [2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)],
                     [2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d]])


def test_rigid_motion_gives_zero_and_recovers_the_rotation():
    rng = np.random.default_rng(5)
    ref = W.fcc_sphere(500) + rng.normal(scale=0.05, size=(500, 3))
    Q = rotation(rng)
    cur = ref @ Q.T + np.array([3.0, -7.0, 11.0])          # x_i = Q y_i + t
    m2, n2, R = msd(cur, ref, 0.0, 2)
    assert n2 == 500 and m2 < 1e-24
    assert np.abs(R @ Q - np.eye(3)).max() < 1e-13          # the fit undoes Q
    m1, _, _ = msd(cur, ref, 0.0, 1)
    m0, _, _ = msd(cur, ref, 0.0, 0)
    assert m1 > 1.0 and m0 > m1                              # without the rotation / the translation it is not zero
    # pure translation: align = 1 already gives zero, align = 0 gives |t|^2
    t = np.array([0.3, 0.4, 1.2])
    assert msd(ref + t, ref, 0.0, 1)[0] < 1e-26
    assert msd(ref + t, ref, 0.0, 0)[0] == pytest.approx(0.09 + 0.16 + 1.44, rel=1e-12)


def test_dilation_closed_form():
    """x_i' = s R0 y_i': the best rotation is R0^-1 and the residual is (s - 1)^2 <|y'|^2>."""
    rng = np.random.default_rng(6)
    ref = rng.normal(scale=4.0, size=(300, 3))
    yc = ref - ref.mean(axis=0)
    Q = rotation(rng)
    for s in (0.9, 1.0, 1.25):
        cur = s * (yc @ Q.T) + np.array([1.0, 2.0, 3.0])
        m, n, R = msd(cur, ref, 0.0, 2)
        assert m == pytest.approx((s - 1.0) ** 2 * (yc ** 2).sum(axis=1).mean(), rel=1e-11, abs=1e-24)
        assert np.abs(R @ Q - np.eye(3)).max() < 1e-12


def test_fit_is_a_proper_rotation_and_optimal_by_brute_force():
    rng = np.random.default_rng(7)
    ref = rng.normal(size=(12, 3))
    cur = ref @ rotation(rng).T + 0.3 * rng.normal(size=ref.shape)
    m, _, R = msd(cur, ref, 0.0, 2)
    assert np.abs(R @ R.T - np.eye(3)).max() < 1e-14 and np.linalg.det(R) == pytest.approx(1.0, abs=1e-13)
    xc, yc = cur - cur.mean(axis=0), ref - ref.mean(axis=0)

    def cost(Rt):
        return ((xc @ Rt.T - yc) ** 2).sum(axis=1).mean()

    assert cost(R) == pytest.approx(m, rel=1e-13)
    for _ in range(2000):                                    # anywhere on SO(3)
        assert cost(rotation(rng)) >= m - 1e-13
    for _ in range(2000):                                    # and in the neighbourhood of the optimum
        w = 1e-3 * rng.normal(size=3)
        th = np.linalg.norm(w)
        k = w / th
        Kx = np.array([[0, -k[2], k[1]], [k[2], 0, -k[0]], [-k[1], k[0], 0]])
        dR = np.eye(3) + math.sin(th) * Kx + (1 - math.cos(th)) * Kx @ Kx
        assert cost(dR @ R) >= m - 1e-13
    # mirror image of a chiral set: no proper rotation maps it back, the fit stays proper
    mir = ref * np.array([1.0, 1.0, -1.0])
    mm, _, Rm = msd(mir, ref, 0.0, 2)
    assert np.linalg.det(Rm) == pytest.approx(1.0, abs=1e-13) and mm > 1e-2
    xm = mir - mir.mean(axis=0)
    for _ in range(2000):
        assert ((xm @ rotation(rng).T - yc) ** 2).sum(axis=1).mean() >= mm - 1e-13


def test_selection_counts_and_one_displaced_atom():
    """fcc sphere about an atom (a = 3.52): 1, 13, 19, 43 atoms strictly within radii just above
    0, a/sqrt2, a, a*sqrt(3/2) (coordination 12, 6, 24); a single atom displaced by delta contributes
    |delta|^2 / n_sel when selected and nothing otherwise (align = 0)."""
    a = 3.52
    ref = W.fcc_sphere(3000)
    ref = ref[(ref ** 2).sum(axis=1) < 14.0 ** 2]            # complete shells about the atom at the origin:
    assert np.abs(ref.mean(axis=0)).max() < 1e-12            # symmetric, centroid = central atom
    n_all = len(ref)
    for r, n in ((0.1, 1), (a / math.sqrt(2) + 0.01, 13), (a + 0.01, 19), (a * math.sqrt(1.5) + 0.01, 43),
                 (a / math.sqrt(2) - 0.01, 1)):
        assert msd(ref, ref, r, 2)[1] == n
    d2 = (ref ** 2).sum(axis=1)
    inner = int(np.argmin(np.abs(d2 - a * a / 2)))           # a first-shell atom
    outer = int(np.argmax(d2))
    delta = np.array([0.3, -0.2, 0.6])
    for idx, hit in ((inner, True), (outer, False)):
        cur = ref.copy()
        cur[idx] += delta
        m, n, _ = msd(cur, ref, a + 0.01, 0)
        assert n == 19
        assert m == pytest.approx((delta ** 2).sum() / 19 if hit else 0.0, rel=1e-12, abs=1e-30)
    assert msd(ref, ref, 1e-6, 2)[1] == 1 and msd(ref + 5.0, ref, 0.0, 1)[1] == n_all
    far = ref + np.array([100.0, 0.0, 0.0])                  # selection uses the REFERENCE frame only
    assert msd(far, ref, a + 0.01, 0)[1] == 19


def test_random_walk_recovers_the_diffusion_coefficient():
    """Independent Gaussian steps of variance 2 D t per coordinate: <dr^2> = 2 z D t, z = 3 (Eq. (12));
    the rigid-body fit removes only O(1/N) of it."""
    rng = np.random.default_rng(8)
    n = 20000
    ref = W.fcc_sphere(n)
    D, t = 2.3e-6 / 0.1, 1.0e5                               # 2.3e-6 cm^2/s in A^2/fs, 100 ps
    cur = ref + rng.normal(scale=math.sqrt(2 * D * t), size=(n, 3))
    for align in (0, 1, 2):
        m, cnt, _ = msd(cur, ref, 0.0, align)
        assert cnt == n
        assert m / (2 * 3 * t) == pytest.approx(D, rel=0.03)
    m, cnt, _ = msd(cur, ref, 10.0, 2)                       # the paper's 10 A selection
    assert 300 < cnt < 400                                   # (4/3) pi 10^3 * 4 / a^3 = 384
    assert m / (2 * 3 * t) == pytest.approx(D, rel=0.15)


def test_degenerate_inputs():
    one = np.array([[1.0, 2.0, 3.0]])
    for align in (0, 1, 2):
        m, n, R = msd(one + (0.5 if align == 0 else 0.0), one, 0.0, align)
        assert n == 1 and m == pytest.approx(0.75 if align == 0 else 0.0, abs=1e-30)
    # two atoms: the rotation about their axis is free, the residual is not
    ref = np.array([[0.0, 0.0, 0.0], [2.0, 0.0, 0.0]])
    cur = np.array([[5.0, 5.0, 5.0], [5.0, 5.0, 8.0]])       # bond stretched from 2 to 3, turned to z
    m, n, R = msd(cur, ref, 0.0, 2)
    assert n == 2 and m == pytest.approx(0.25, rel=1e-12)    # each end 0.5 A from its reference
    assert np.linalg.det(R) == pytest.approx(1.0, abs=1e-13)
    assert msd(cur, ref, 1e-9, 2)[1] == 0 and msd(cur, ref, 1e-9, 2)[0] == 0.0
