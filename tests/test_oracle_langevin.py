"""Pins for the oracle's Langevin thermostat (reading Q18 of DESIGN.md; PAPER.md:145 gives only
"Langevin thermostat with a damping constant of 10 ps^-1").  All CPU, -m "not gpu".

What would fail where: a wrong Philox round / constant -> the known-answer vectors and the numpy
cross-check; a wrong counter layout, uniform mapping, Box-Muller pairing, c1 or c2 -> the N = 1
chain recomputed here from the definition with an independent Philox; a wrong place for the
thermostat in the step -> the gamma -> 0 and T = 0 limits; a wrong unit factor -> equipartition.
"""
import json
import math
from pathlib import Path

import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

KAT = json.loads((Path(__file__).parent / "golden" / "philox_kat.json").read_text())
ACC, KB, MASS = 9.648533215665e-3, 8.617333262e-5, 58.69      # retyped (reading Q4)


def philox_py(ctr, key, bits=32, rounds=10):
    """Philox-4xW written from Salmon et al. (SC'11), generic in the word width so that the W = 64
    instance can be checked against numpy's own Philox and the W = 32 one then differs only by its
    constants."""
    if bits == 32:
        m0, m1, w0, w1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    else:
        m0, m1, w0, w1 = 0xD2E7470EE14C6C93, 0xCA5A826395121157, 0x9E3779B97F4A7C15, 0xBB67AE8584CAA73B
    mask = (1 << bits) - 1
    c = list(ctr); k = list(key)
    for _ in range(rounds):
        p0, p1 = m0 * c[0], m1 * c[2]
        c = [(p1 >> bits) ^ c[1] ^ k[0], p1 & mask, (p0 >> bits) ^ c[3] ^ k[1], p0 & mask]
        k = [(k[0] + w0) & mask, (k[1] + w1) & mask]
    return c


def test_philox_known_answer_vectors(oracle_ld):
    for row in KAT["philox4x32_10"]:
        ctr = [int(x, 16) for x in row["ctr"]]; key = [int(x, 16) for x in row["key"]]
        out = [int(x, 16) for x in row["out"]]
        assert list(oracle_ld.philox4x32_10(ctr, key)) == out
        assert philox_py(ctr, key, 32) == out


def test_python_philox_structure_against_numpy():
    """numpy ships Philox4x64-10: same round function, other constants.  numpy increments the counter
    before each block."""
    key = [0x0123456789ABCDEF, 0xFEDCBA9876543210]
    ctr = [5, 7, 11, 13]
    bg = np.random.Philox(counter=np.array(ctr, dtype=np.uint64), key=np.array(key, dtype=np.uint64))
    raw = [int(x) for x in bg.random_raw(8)]
    assert raw[:4] == philox_py([6, 7, 11, 13], key, 64)
    assert raw[4:] == philox_py([7, 7, 11, 13], key, 64)


def test_python_philox_matches_oracle_on_random_inputs(oracle_ld):
    rng = np.random.default_rng(7)
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 2**32, 4)]; key = [int(x) for x in rng.integers(0, 2**32, 2)]
        assert list(oracle_ld.philox4x32_10(ctr, key)) == philox_py(ctr, key, 32)


def normals_py(seed, atom, step):
    w = philox_py([atom & 0xFFFFFFFF, step & 0xFFFFFFFF, step >> 32, 0], [seed & 0xFFFFFFFF, seed >> 32], 32)
    u = [(x + 0.5) / 2.0**32 for x in w]
    ra, rb = math.sqrt(-2.0 * math.log(u[0])), math.sqrt(-2.0 * math.log(u[2]))
    return np.array([ra * math.cos(2 * math.pi * u[1]), ra * math.sin(2 * math.pi * u[1]), rb * math.cos(2 * math.pi * u[3])])


def test_normals_definition_and_statistics(oracle_ld):
    for seed, atom, step in [(0, 0, 0), (1, 2, 3), (2**63 + 5, 2**31 + 1, 2**40 + 9), (12345, 1414, 9999)]:
        np.testing.assert_allclose(oracle_ld.langevin_normals(seed, atom, step), normals_py(seed, atom, step), rtol=0, atol=1e-14)
    xi = np.array([oracle_ld.langevin_normals(99, a, s) for a in range(200) for s in range(100)])
    n = xi.size
    assert abs(xi.mean()) < 4 / math.sqrt(n)
    assert abs(xi.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((xi**4).mean() - 3) < 4 * math.sqrt(96 / n)
    c = np.corrcoef(xi.T)                                   # the three components are uncorrelated
    assert np.abs(c - np.eye(3)).max() < 4 / math.sqrt(n / 3)
    # neighbouring counters are uncorrelated
    a = xi[:-1, 0] * xi[1:, 0]
    assert abs(a.mean()) < 4 / math.sqrt(a.size)


def test_single_atom_chain_from_the_definition(oracle_ld):
    """N = 1: no force, so v_k = c1 v_{k-1} + c2(T_k) xi(seed, 0, step0 + k - 1) and x_k = x_{k-1} + dt v
    where v is the velocity BEFORE the thermostat of step k (kick, drift, kick, then O)."""
    P = oracle_ld.params()
    dt, gamma, seed, step0, nsteps, T0, T1 = 2.0, 0.01, 4242, 17, 25, 300.0, 900.0
    x = np.array([[0.1, -0.2, 0.3]]); v = np.array([[1e-3, -2e-3, 5e-4]])
    out = oracle_ld.run(x, v, P, dt=dt, nsteps=nsteps, thermo_kind=2, T_start=T0, T_end=T1, gamma=gamma, seed=seed, step0=step0)
    xe, ve = x[0].copy(), v[0].copy()
    c1 = math.exp(-gamma * dt)
    for k in range(1, nsteps + 1):
        xe = xe + dt * ve
        Tk = T0 + (T1 - T0) * k / nsteps
        ve = c1 * ve + math.sqrt((1 - c1 * c1) * KB * Tk * ACC / MASS) * normals_py(seed, 0, step0 + k - 1)
    np.testing.assert_allclose(out["vel"][0], ve, rtol=1e-12, atol=1e-18)
    np.testing.assert_allclose(out["pos"][0], xe, rtol=1e-12, atol=1e-15)


def test_limits_gamma_zero_is_nve_and_zero_temperature_is_pure_damping(oracle_ld):
    w = W.config_c1()
    P = oracle_ld.params()
    nve = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=10)
    lg0 = oracle_ld.run(w.pos, w.vel, P, dt=1.0, nsteps=10, thermo_kind=2, T_start=500.0, T_end=500.0, gamma=0.0, seed=3)
    assert np.array_equal(nve["pos"], lg0["pos"]) and np.array_equal(nve["vel"], lg0["vel"])
    # T = 0, well separated atoms (negligible force): velocities decay by exp(-gamma t)
    pos = np.array([[0.0, 0, 0], [1e4, 0, 0], [0, 1e4, 0]]); vel = np.array([[1e-3, 0, 0], [0, 2e-3, 0], [0, 0, -3e-3]])
    out = oracle_ld.run(pos, vel, P, dt=1.0, nsteps=50, thermo_kind=2, T_start=0.0, T_end=0.0, gamma=0.02, seed=3)
    np.testing.assert_allclose(out["vel"], vel * math.exp(-0.02 * 50), rtol=1e-9, atol=1e-16)


def test_equipartition_of_free_particles(oracle_plain):
    """Fluctuation-dissipation: free particles (spacing 1e4 A, forces ~1e-30) relax to
    <v^2> = kB T ACC / m per component whatever gamma and dt are (the O step is exact)."""
    n = 4000
    pos = np.arange(n)[:, None] * np.array([[1e4, 0.0, 0.0]])
    vel = np.zeros((n, 3))
    P = oracle_plain.params(r_cut=5.0)          # keeps the CPU cost O(N^2) cheap rejections
    out = oracle_plain.run(pos, vel, P, dt=1.0, nsteps=12, thermo_kind=2, T_start=1000.0, T_end=1000.0, gamma=0.5, seed=11)
    var = out["vel"].var()
    expect = KB * 1000.0 * ACC / MASS * (1 - math.exp(-2 * 0.5 * 12))
    assert abs(var / expect - 1) < 4 * math.sqrt(2 / (3 * n))
    _, T = oracle_plain.kinetic(out["vel"])
    assert abs(T / 1000.0 - 1) < 0.06


def test_thermostatted_cluster_reaches_target_temperature(oracle_plain):
    """Ni147 at gamma = 10 ps^-1 started cold: the temperature climbs towards the
    bath's 600 K with time constant ~1/(2 gamma) = 50 fs for the kinetic part (equipartition with the
    potential energy halves the asymptote on this time scale: T(300 fs) in a broad window)."""
    w = W.config_c1()
    P = oracle_plain.params()
    out = oracle_plain.run(w.pos, 0.0 * w.vel, P, dt=1.0, nsteps=300, thermo_kind=2, T_start=600.0, T_end=600.0,
                           gamma=0.01, seed=5)
    _, T = oracle_plain.kinetic(out["vel"])
    assert 150.0 < T < 750.0
    # split runs continue the same noise stream when step0 advances
    a = oracle_plain.run(w.pos, w.vel, P, dt=1.0, nsteps=8, thermo_kind=2, T_start=600.0, T_end=600.0, gamma=0.01, seed=5)
    b1 = oracle_plain.run(w.pos, w.vel, P, dt=1.0, nsteps=3, thermo_kind=2, T_start=600.0, T_end=600.0, gamma=0.01, seed=5)
    b2 = oracle_plain.run(b1["pos"], b1["vel"], P, dt=1.0, nsteps=5, thermo_kind=2, T_start=600.0, T_end=600.0, gamma=0.01, seed=5, step0=3)
    np.testing.assert_allclose(b2["pos"], a["pos"], rtol=0, atol=1e-12)
