"""sc_rdf (radial-distribution counts of the central atoms) against the oracle: integer
work, bit-exact."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu


def ctx(scmd, pos, vel=None, **kw):
    import torch
    sc = scmd.SuttonChen(len(pos), **kw)
    sc.sc_set_state(torch.as_tensor(np.ascontiguousarray(pos), device="cuda"),
                    None if vel is None else torch.as_tensor(np.ascontiguousarray(vel), device="cuda"))
    return sc


def test_paper_selection_on_mackay_clusters(scmd, oracle_ld):
    """The paper's procedure (3 A of the centre of mass, 0.4 A bins) on Ni147 and Ni2057."""
    for shells in (3, 8):
        pos = W.mackay_icosahedron(shells, 2.49)
        sc = ctx(scmd, pos)
        counts, n_ref, centre = sc.sc_rdf(3.0, 0.4, 60)
        sc.close()
        ref, n_o, c_o = oracle_ld.rdf_counts(pos, 3.0, 0.4, 60)
        assert n_ref == n_o == 13 and np.allclose(centre, c_o, atol=1e-12)
        assert np.array_equal(counts, ref) and counts.sum() > 0


@pytest.mark.parametrize("n_atoms,r_select,width,n_bins", [(1, 1.0, 0.4, 8), (2, 50.0, 0.4, 4096), (777, 7.5, 0.4, 50),
                                                          (2607, 1e3, 0.25, 200), (8000, 6.0, 0.1, 1000)])
def test_explicit_centre_bit_exact(scmd, oracle_ld, n_atoms, r_select, width, n_bins):
    """Explicit centre (so that the selection sees identical bits): few, many and all atoms as references,
    ragged sizes, one to 4096 bins, pairs beyond the last bin dropped."""
    w = W.liquid_droplet(n_atoms, 2000.0, seed=5) if n_atoms == 8000 else W.fcc_cluster(n_atoms, 1500.0, seed=40 + n_atoms)
    centre = w.pos.mean(axis=0) + 0.01
    sc = ctx(scmd, w.pos)
    counts, n_ref, used = sc.sc_rdf(r_select, width, n_bins, centre=centre)
    sc.close()
    ref, n_o, _ = oracle_ld.rdf_counts(w.pos, r_select, width, n_bins, centre=centre)
    assert np.array_equal(used, centre) and n_ref == n_o
    assert np.array_equal(counts, ref)
    if n_atoms == 2607:
        assert n_ref == 2607


def test_cell_sorted_order_and_mixed(scmd, oracle_ld):
    """The histogram works on the resident records whatever their internal order (the list path re-sorts them
    by cell at every build) and whatever the precision mode: two builds with different sorts, then the counts of
    the second (synthetic) state against the oracle on the same array."""
    rng = np.random.default_rng(19)
    a = W.fcc_cluster(3000, 1500.0, seed=9).pos
    b = a + rng.normal(scale=0.35, size=a.shape)                  # a hot, disordered state
    centre = b.mean(axis=0)
    ref, n_o, _ = oracle_ld.rdf_counts(b, 5.0, 0.4, 80, centre=centre)
    for kw in (dict(r_cut=8.0, skin=1.0), dict(r_cut=8.0, skin=1.0, precision=1), dict(precision=1), dict()):
        import torch
        sc = ctx(scmd, a, None, **kw)
        sc.sc_forces()                                            # build 1: cells of A
        sc.sc_set_state(torch.as_tensor(b, device="cuda"), None)
        sc.sc_forces()                                            # build 2: cells of B
        counts, n_ref, _ = sc.sc_rdf(5.0, 0.4, 80, centre=centre)
        sc.close()
        assert n_ref == n_o and np.array_equal(counts, ref)


def test_argument_validation(scmd):
    w = W.config_c1()
    sc = ctx(scmd, w.pos)
    for bad in (dict(n_bins=0), dict(n_bins=5000), dict(r_select=0.0), dict(bin_width=-1.0)):
        args = dict(r_select=3.0, bin_width=0.4, n_bins=10)
        args.update(bad)
        with pytest.raises(scmd.ScError):
            sc.sc_rdf(args["r_select"], args["bin_width"], args["n_bins"])
    sc.close()
    import torch
    sc = scmd.SuttonChen(10)
    with pytest.raises(scmd.ScError):
        sc.sc_rdf(3.0, 0.4, 10)                                        # no positions yet
    sc.close()
