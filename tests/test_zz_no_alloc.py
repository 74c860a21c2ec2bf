"""sc_density_noalloc (include/scmd.h; csrc/sc_noalloc.cu): the density sweep with its scratch in a static device array,
for callers that cannot call cudaMalloc.  Collected last on purpose (the suite runs with pytest -x).

Its output against the existing path's (sc_create + sc_set_state + sc_density, workspace-backed) within the tolerance the
other density tests use (1e-12 relative, tests/test_gpu_parity.py), on two calls in a row with DIFFERENT inputs -- the
array keeps the first call's contents --, then the first input again; and against the oracle; sizes beyond the maximum
are refused with a message."""
import numpy as np
import pytest

from paper_1210_3559_b200 import workloads as W

pytestmark = pytest.mark.gpu

RHO_TOL = 1e-12


def existing_path(scmd, pos):
    import torch
    sc = scmd.SuttonChen(len(pos))
    sc.sc_set_state(torch.as_tensor(pos, device="cuda"))
    rho = sc.sc_density().cpu().numpy()
    sc.close()
    return rho


def test_density_noalloc_two_calls_in_a_row(scmd, oracle_ld):
    import torch
    big = W.fcc_cluster(5003, 1500.0, seed=91)          # 40 CTAs, ragged last tile
    small = W.config_c1()                               # Ni147: 2 CTAs, leaves most of the array as the first call wrote it
    want_big, want_small = existing_path(scmd, big.pos), existing_path(scmd, small.pos)
    d_big, d_small = torch.as_tensor(big.pos, device="cuda"), torch.as_tensor(small.pos, device="cuda")
    rho_big = torch.full((big.n_atoms,), float("nan"), dtype=torch.float64, device="cuda")
    rho_small = torch.full((small.n_atoms,), float("nan"), dtype=torch.float64, device="cuda")
    s_big = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    s_small = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    scmd.sc_density_noalloc(d_big, rho_big, s_big)      # two calls in a row on one stream, no synchronisation between
    scmd.sc_density_noalloc(d_small, rho_small, s_small)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before      # nothing came from torch's allocator either
    for got, want, s in ((rho_big, want_big, s_big), (rho_small, want_small, s_small)):
        g = got.cpu().numpy()
        assert np.all(np.isfinite(g))
        assert np.max(np.abs(g - want) / want) < RHO_TOL
        assert abs(s.item() - np.sqrt(want).sum()) < 1e-12 * np.sqrt(want).sum()
    # the first input again: same bits as its first evaluation (fixed summation order, stale contents never read)
    again, s_again = torch.empty_like(rho_big), torch.empty_like(s_big)
    scmd.sc_density_noalloc(d_big, again, s_again)
    torch.cuda.synchronize()
    assert torch.equal(again, rho_big) and torch.equal(s_again, s_big)
    # and the oracle (long-double build) on the small cluster
    rho_o, _, _ = oracle_ld.energy_forces(small.pos, oracle_ld.params())
    assert np.max(np.abs(rho_small.cpu().numpy() - rho_o) / rho_o) < RHO_TOL


def test_density_noalloc_generic_exponents_and_limits(scmd):
    import torch
    w = W.fcc_cluster(700, 300.0, seed=92)
    kw = dict(n=7, m=3, eps=0.02, c=30.0, a=3.3)
    sc = scmd.SuttonChen(w.n_atoms, **kw)
    d_pos = torch.as_tensor(w.pos, device="cuda")
    sc.sc_set_state(d_pos)
    want = sc.sc_density().cpu().numpy()
    sc.close()
    rho = torch.empty(w.n_atoms, dtype=torch.float64, device="cuda")
    scmd.sc_density_noalloc(d_pos, rho, None, **kw)     # odd m: the reciprocal-square-root branch; no scalar wanted
    torch.cuda.synchronize()
    assert np.max(np.abs(rho.cpu().numpy() - want) / want) < RHO_TOL
    # the maximum itself works, one atom more is refused with a message that names the limit
    n_max = scmd.SC_NOALLOC_MAX_ATOMS
    top = W.fcc_cluster(n_max, 1500.0, seed=93)
    want_top = existing_path(scmd, top.pos)
    d_top = torch.as_tensor(top.pos, device="cuda")
    rho_top = torch.empty(n_max, dtype=torch.float64, device="cuda")
    scmd.sc_density_noalloc(d_top, rho_top)
    torch.cuda.synchronize()
    assert np.max(np.abs(rho_top.cpu().numpy() - want_top) / want_top) < RHO_TOL
    too_many = torch.zeros(n_max + 1, 3, dtype=torch.float64, device="cuda")
    out = torch.empty(n_max + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(scmd.ScError) as err:
        scmd.sc_density_noalloc(too_many, out)
    assert err.value.status == scmd.SC_ERR_NOMEM and "SC_NOALLOC_MAX_ATOMS" in str(err.value)
