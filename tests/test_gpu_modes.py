"""GPU parity of the iteration modes of SURVEY 8(f) N2 against the float64 oracle, through the C-ABI binding:
plain lambda iteration (loc_set_ali(0)) and the convergence-controlled loop (loc_iterate_until,
PAPER.md:77).  The oracle's plain-lambda arithmetic is pinned by tests/test_oracle_pins_1d.py (P1 with ali = False,
P8: ALI and lambda iteration share their fixed point)."""
import ctypes as C

import numpy as np
import pytest

import loc_workloads as W
import oracle as O
from parity import check_pops, rel_err, tex_all
from test_gpu_3d import small

pytestmark = pytest.mark.gpu

TOL_POP = 1e-3  # north_star: populations and T_ex within 1e-3 relative


def _model(m):
    from paper_2009_12609_b200 import LocModel
    return LocModel(m)


def _leaf(m):
    return (m.child < 0) if hasattr(m, "child") else np.ones(len(m.density), bool)


def _compare(m, sp, pg, pops_o):
    leaf = _leaf(m)
    worst, small_abs = check_pops(pg[:, leaf], pops_o[leaf])
    assert worst < TOL_POP and small_abs < 1e-10
    tg, to = tex_all(sp, pg.astype(np.float64).T[leaf], m.species), tex_all(sp, pops_o[leaf], m.species)
    big = pops_o[leaf][:, 1:] >= 1e-10 * pops_o[leaf].sum(axis=1, keepdims=True)
    assert rel_err(tg, to)[big].max() < TOL_POP


MODELS = [("1d-C1", lambda: W.shell_config(1), 8),
          ("1d-C2-small", lambda: W.shell_config(2, ns=90, nchannel=128, nsub=2), 5),
          ("3d-octree", lambda: small(nroot=4, nlev=3, nside=1, nch=40, frac=0.4), 4),
          ("3d-thick", lambda: small(nroot=6, nlev=1, nside=1, nch=48, dens=30.0), 4)]


@pytest.mark.parametrize("name,make,niter", MODELS, ids=[x[0] for x in MODELS])
def test_plain_lambda_iteration(name, make, niter):
    m = make()
    sp = O.OSpecies(m.species)
    pops_o, change_o = O.iterate(sp, m, niter, ali=False)
    g = _model(m)
    g.set_ali(False)
    g.init_lte()
    change_g = g.iterate(niter)
    pg = g.pops.cpu().numpy()
    g.close()
    _compare(m, sp, pg, pops_o)
    assert abs(change_g - change_o) <= 0.05 * change_o + 1e-5


def test_plain_lambda_differs_from_ali_before_convergence():
    """the switch does something: after 2 iterations of a thick model the two modes are apart by far more than the
    tolerance (they meet only at the fixed point, pin P8), and the GPU follows the oracle in each."""
    m = small(nroot=6, nlev=1, nside=1, nch=48, dens=30.0)
    sp = O.OSpecies(m.species)
    out = {}
    for ali in (True, False):
        g = _model(m)
        g.set_ali(ali)
        g.init_lte()
        g.iterate(2)
        out[ali] = g.pops.cpu().numpy()
        g.close()
        _compare(m, sp, out[ali], O.iterate(sp, m, 2, ali=ali)[0])
    assert np.max(np.abs(out[True][1] - out[False][1]) / out[True][1]) > 10 * TOL_POP


@pytest.mark.parametrize("ali", [True, False])
def test_iterate_until_stops_where_the_oracle_does(ali):
    m = W.shell_config(1)
    sp = O.OSpecies(m.species)
    _, changes, _ = O.iterate(sp, m, 12, ali=ali, history=True)
    changes = np.asarray(changes)
    # a tolerance midway (in log) between two successive oracle changes: the stopping iteration is not borderline
    k = 6
    assert changes[k] < changes[k - 1] and np.all(changes[:k] > changes[k])
    tol = float(np.sqrt(changes[k] * changes[k - 1]))
    g = _model(m)
    g.set_ali(ali)
    g.init_lte()
    n, ch = g.iterate_until(50, tol)
    pg = g.pops.cpu().numpy()
    assert n == k + 1 and ch <= tol
    assert abs(ch - changes[k]) <= 0.05 * changes[k] + 1e-5
    _compare(m, sp, pg, O.iterate(sp, m, k + 1, ali=ali)[0])
    # the cap: max_iter smaller than needed
    g.init_lte()
    n2, ch2 = g.iterate_until(3, tol)
    assert n2 == 3 and ch2 > tol
    # nothing to do
    assert g.iterate_until(0, tol) == (0, 0.0)
    g.close()


def test_mode_calls_reject_bad_arguments():
    from paper_2009_12609_b200 import binding as B
    m = W.shell_config(1, ns=8, nchannel=16)
    g = _model(m)
    lib = B.lib()
    assert lib.loc_set_ali(g.h, 2) == B.LOC_EINVAL
    assert lib.loc_set_ali(None, 1) == B.LOC_EINVAL
    assert lib.loc_iterate_until(g.h, -1, C.c_double(1e-3), None, None) == B.LOC_EINVAL
    assert lib.loc_iterate_until(g.h, 1, C.c_double(-1.0), None, None) == B.LOC_EINVAL
    g.close()


def test_tex_per_cell():
    """loc_tex against the oracle's T_ex (O.tex, pinned by the LTE limit P3): from LTE populations it returns T_kin, after
    iterations it follows the oracle's populations; refined cells and cells without gas give 0"""
    m = small(nroot=4, nlev=2, nside=1, nch=32, frac=0.4)
    leaf = m.child < 0
    empty = np.flatnonzero(leaf)[::5]
    m.density[empty] = 0.0
    gas = leaf & (m.density > 0)
    sp = O.OSpecies(m.species)
    g = _model(m)
    g.init_lte()
    for t in range(sp.ntrans):
        te = g.tex(t).cpu().numpy()
        assert np.max(np.abs(te[gas] - m.tkin[gas]) / m.tkin[gas]) < 2e-5  # float32 populations
        assert np.all(te[~gas] == 0.0)
    g.iterate(3)
    pops_o, _ = O.iterate(sp, m, 3)
    for t in range(sp.ntrans):
        u, l = m.species.upper[t], m.species.lower[t]
        ref = np.array([O.tex(sp, t, pops_o[c, u], pops_o[c, l]) for c in np.flatnonzero(gas)])
        te = g.tex(t).cpu().numpy()[gas]
        assert rel_err(te, ref).max() < TOL_POP
    from paper_2009_12609_b200 import binding as B
    with pytest.raises(B.LocError):
        g.tex(99)
    g.close()
