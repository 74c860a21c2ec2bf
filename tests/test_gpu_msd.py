"""sc_msd (aligned mean-square displacement for Eq. (12)) through the C ABI against the
oracle's Kabsch/SVD definition (Oracle.msd_aligned): the device solves the same minimisation by Horn's
quaternion matrix and Jacobi sweeps, so agreement is to rounding -- |dmsd| <= 1e-11 msd + 1e-22 <|y'|^2>,
rotation entries to 1e-12 where the minimiser is unique.  The selected-atom count is an integer: exact."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu


def rotation(rng):
    q = rng.normal(size=4)
    a, b, c, d = q / np.linalg.norm(q)
    return np.array([[a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)],
                     [2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)],
                     [2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d]])


def check(scmd, oracle_ld, cur, ref, r_centre, align, unique=True, **kw):
    import torch
    n = len(cur)
    sc = scmd.SuttonChen(n, **kw)
    sc.sc_set_state(torch.as_tensor(cur, device="cuda"), None)
    dref = torch.as_tensor(np.ascontiguousarray(ref), device="cuda")
    m, cnt, R = sc.sc_msd(dref, r_centre, align)
    mo, cnto, Ro = oracle_ld.msd_aligned(cur, ref, r_centre, align)
    scale = ((ref - ref.mean(axis=0)) ** 2).sum(axis=1).mean()
    assert cnt == cnto
    assert abs(m - mo) <= 1e-11 * mo + 1e-22 * scale + 1e-300, (m, mo)
    assert abs(np.linalg.det(R) - 1.0) < 1e-13 and np.abs(R @ R.T - np.eye(3)).max() < 1e-13
    if unique:
        assert np.abs(R - Ro).max() < 1e-12
    m2, cnt2, R2 = sc.sc_msd(dref, r_centre, align)             # fixed summation order: same bits
    assert m2 == m and cnt2 == cnt and np.array_equal(R, R2)
    sc.close()
    return m, cnt, R


@pytest.mark.parametrize("n_atoms", [3, 4, 149, 2057, 70000, 300000])
@pytest.mark.parametrize("align", [0, 1, 2])
def test_against_oracle(scmd, oracle_ld, n_atoms, align):
    """thermal displacements plus a rigid rotation and translation, several CTAs and a ragged tail
    (70000 = 274 CTAs; 300000 > 512 CTAs x 256: grid-stride), the paper's 10 A selection"""
    rng = np.random.default_rng(100 + n_atoms)
    ref = W.fcc_sphere(n_atoms) + rng.normal(scale=0.05, size=(n_atoms, 3))
    cur = (ref + rng.normal(scale=0.3, size=ref.shape)) @ rotation(rng).T + np.array([4.0, -2.0, 9.0])
    check(scmd, oracle_ld, cur, ref, 0.0, align)
    m, cnt, _ = check(scmd, oracle_ld, cur, ref, 10.0, align)
    assert 0 < cnt <= min(n_atoms, 420)


def test_rigid_motion_and_far_from_origin(scmd, oracle_ld):
    """exact rigid motion: msd is zero to rounding and the rotation comes back; a cluster 1e4 A from
    the origin loses nothing (centred covariance)"""
    rng = np.random.default_rng(7)
    ref = W.mackay_icosahedron(8)
    Q = rotation(rng)
    cur = ref @ Q.T + np.array([1.0, 2.0, 3.0])
    m, cnt, R = check(scmd, oracle_ld, cur, ref, 0.0, 2)
    assert cnt == 2057 and m < 1e-24 and np.abs(R @ Q - np.eye(3)).max() < 1e-13
    shift = np.array([1.0e4, -2.0e4, 3.0e4])
    m, _, R = check(scmd, oracle_ld, cur + shift, ref - shift, 10.0, 2)
    assert m < 1e-18 and np.abs(R @ Q - np.eye(3)).max() < 1e-11


def test_degenerate_inputs(scmd, oracle_ld):
    one = np.array([[1.0, 2.0, 3.0]])
    for align in (0, 1, 2):
        m, cnt, R = check(scmd, oracle_ld, one + (0.5 if align == 0 else 0.0), one, 0.0, align, unique=False)
        assert cnt == 1 and m == pytest.approx(0.75 if align == 0 else 0.0, abs=1e-30)
        assert np.array_equal(R, np.eye(3))
    ref = np.array([[0.0, 0.0, 0.0], [2.0, 0.0, 0.0]])
    cur = np.array([[5.0, 5.0, 5.0], [5.0, 5.0, 8.0]])
    m, cnt, _ = check(scmd, oracle_ld, cur, ref, 0.0, 2, unique=False)        # free rotation about the bond
    assert cnt == 2 and m == pytest.approx(0.25, rel=1e-12)
    m, cnt, _ = check(scmd, oracle_ld, cur, ref, 1e-9, 2, unique=False)       # nothing selected
    assert cnt == 0 and m == 0.0
    mir = np.random.default_rng(3).normal(size=(12, 3))
    check(scmd, oracle_ld, mir * np.array([1.0, 1.0, -1.0]), mir, 0.0, 2)     # mirror image: the fit stays proper


@pytest.mark.parametrize("mixed", [False, True])
def test_list_path_matches_the_reference_through_the_cell_sort(scmd, oracle_ld, mixed):
    """On the list path the resident records are re-sorted by cell at every build; the reference stays in the
    caller's order and is matched through the permutation.  Two builds with different sorts (state A, then a
    displaced and rotated state B), msd of B against A -- both synthetic, the oracle sees the same arrays."""
    import torch
    rng = np.random.default_rng(55)
    prec = dict(precision=scmd.SC_PREC_MIXED) if mixed else {}
    a = W.fcc_cluster(4000, 300.0, seed=77).pos
    b = (a + rng.normal(scale=0.4, size=a.shape)) @ rotation(rng).T + np.array([3.0, 1.0, -2.0])
    for kw in (dict(), dict(r_cut=7.0, skin=0.6)):
        sc = scmd.SuttonChen(len(a), **kw, **prec)
        d_a = torch.as_tensor(a, device="cuda")
        sc.sc_set_state(d_a, None)
        sc.sc_forces()                                            # first build: sorted by the cells of A
        assert sc.sc_msd(d_a, 0.0, 0)[0] == 0.0
        sc.sc_set_state(torch.as_tensor(b, device="cuda"), None)
        sc.sc_forces()                                            # second build: the cells of B
        if kw:
            assert sc.sc_stats()["n_rebuilds"] == 2
        for align, rc in ((0, 0.0), (1, 10.0), (2, 10.0), (2, 0.0)):
            m, cnt, R = sc.sc_msd(d_a, rc, align)
            mo, cnto, Ro = oracle_ld.msd_aligned(b, a, rc, align)
            assert cnt == cnto and abs(m - mo) <= 1e-11 * mo and np.abs(R - Ro).max() < 1e-12
        sc.close()


def test_after_md_steps(scmd, oracle_ld):
    """The reference is the initial structure; after 100 NVE steps the device msd of the device trajectory equals
    the oracle's msd of the ORACLE's trajectory (the two agree to 1e-8 A, i.e. to ~1e-7 of an msd of 0.05 A^2),
    through the multi-launch path, the list path (with re-sorts) and the one-launch loop."""
    import torch
    w = W.fcc_cluster(900, 1500.0, seed=78)
    for kw, persistent in ((dict(), 1), (dict(), 2), (dict(r_cut=6.5, skin=0.4), 0)):
        ref = oracle_ld.run(w.pos, w.vel, oracle_ld.params(r_cut=kw.get("r_cut", 0.0)), dt=1.0, nsteps=100)
        sc = scmd.SuttonChen(w.n_atoms, **kw)
        sc.sc_set_option(scmd.SC_OPT_PERSISTENT, persistent)
        d0 = torch.as_tensor(w.pos, device="cuda")
        sc.sc_set_state(d0, torch.as_tensor(w.vel, device="cuda"))
        sc.sc_step(1.0, 100)
        for align, rc in ((0, 0.0), (2, 10.0), (2, 0.0)):
            m, cnt, _ = sc.sc_msd(d0, rc, align)
            mo, cnto, _ = oracle_ld.msd_aligned(ref["pos"], w.pos, rc, align)
            assert cnt == cnto and abs(m - mo) <= 1e-6 * mo
            assert 0.005 < m < 1.0                                # 100 fs of thermal motion
        sc.close()


def test_argument_errors(scmd):
    import torch
    sc = scmd.SuttonChen(10)
    ref = torch.zeros(10, 3, dtype=torch.float64, device="cuda")
    with pytest.raises(scmd.ScError) as e:
        sc.sc_msd(ref)                                            # no positions yet
    assert e.value.status == scmd.SC_ERR_STATE
    sc.sc_set_state(torch.as_tensor(W.fcc_sphere(10), device="cuda"), None)
    for bad in (dict(align=3), dict(align=-1), dict(r_centre=float("nan"))):
        with pytest.raises(scmd.ScError) as e:
            sc.sc_msd(ref, **bad)
        assert e.value.status == scmd.SC_ERR_INVALID
    with pytest.raises(scmd.ScError):
        sc.sc_msd(ref[:5])                                        # wrong size is caught by the binding
    ref[3, 1] = float("inf")
    with pytest.raises(scmd.ScError) as e:
        sc.sc_msd(ref, 0.0, 1)
    assert e.value.status == scmd.SC_ERR_NONFINITE
    sc.close()
