"""The three kernels of the statistical-equilibrium solve (loc_solve.cu) against the oracle's solve on the SAME counters,
and against each other: k_solve_f (float32 in registers, the default for <= 12 levels), k_solve_s (float64, shared memory),
k_solve (float64, local memory).  The counters come from one loc_simulate; the oracle's solve (O9: pivoted Gaussian
elimination in float64) is given those float32 counters converted back to its own units, so that only the solve differs."""
import numpy as np
import pytest

import loc_workloads as W
import oracle as O
from parity import check_pops, f32_pops_from_oracle_lte

pytestmark = pytest.mark.gpu
_C = 2.99792458e10


def _solve_all(m, sel=None, ali=True):
    """populations after ONE solve from the counters of one simulate, for solver option 0, 1, 2; and the oracle's"""
    from paper_2009_12609_b200 import LocModel, binding as B
    sp = O.OSpecies(m.species)
    pops64, pops32 = f32_pops_from_oracle_lte(sp, m)
    sel_arr = np.arange(sp.ntrans, dtype=np.int32) if sel is None else np.asarray(sel, np.int32)
    out = {}
    cnt = None
    for opt in (0, 1, 2):
        g = LocModel(m, ntrans_sim=len(sel_arr))
        g.set_option(B.LOC_OPT_SOLVER, opt)
        g.set_ali(1 if ali else 0)
        g.set_populations(pops32)
        g.simulate(sel)
        if cnt is None:
            sj, esc = g.counters()
            cnt = (sj.cpu().numpy().astype(np.float64), esc.cpu().numpy().astype(np.float64))
        g.solve()
        out[opt] = g.pops.cpu().numpy().copy()
        g.close()
    # the oracle's solve on the library's counters: P = SJ 8 pi nu^3 dv V_eff / c^3, LAM = 1 - ESC (tests/parity.py inverted)
    dv = 2.0 * m.band_half / m.nchannel
    is3d = hasattr(m, "child")
    n = len(m.density)
    veff = (m.root_cm / 2.0 ** np.asarray(m.level, np.int64)) ** 3 if is3d else np.ones(n)
    P = np.zeros((len(sel_arr), n))
    for k, t in enumerate(sel_arr):
        P[k] = cnt[0][:, k] * 8.0 * np.pi * sp.freq(int(t)) ** 3 * dv * veff / _C ** 3
    LAM = np.ascontiguousarray((1.0 - cnt[1][:, :len(sel_arr)]).T)
    po = pops64.copy()
    O.solve(sp, m.density, m.tkin, m.abundance, veff, sel_arr, P, LAM, dv, m.t_bg, po, ali)
    return out, po


@pytest.mark.parametrize("nlevel", [2, 3, 5, 8, 10, 12])
def test_register_solver_matches_oracle_solve_on_the_same_counters(nlevel):
    m = W.shell_config(2, ns=300, nchannel=128, nsub=2, nlevel=nlevel)
    out, po = _solve_all(m)
    for opt in (0, 1, 2):
        worst, small = check_pops(out[opt], po, tol=1e-3)
        # float32 registers: ~NL eps per population (GTH has no cancellation); the float64 kernels: rounding of the output only
        assert worst < (2e-5 if opt == 0 else 2e-6), (opt, worst)
        assert small < 1e-13


def test_register_solver_untraced_transitions_and_octree():
    """3 of 9 transitions traced (R23: the others see the background), refined cells skipped, T_kin varying per cell"""
    from test_gpu_3d import small
    m = small(which=4, nroot=4, nlev=3, nside=1, nch=64, frac=0.4, nls=10, seed=11)
    sel = np.array([0, 1, 2], np.int32)
    out, po = _solve_all(m, sel=sel)
    leaf = m.child < 0
    for opt in (0, 1, 2):
        worst, small_ = check_pops(out[opt][:, leaf], po[leaf], tol=1e-3)
        assert worst < (2e-5 if opt == 0 else 2e-6), (opt, worst)


def test_register_solver_plain_lambda_iteration():
    """loc_set_ali(0): the oracle's plain lambda mode carries the self term in its own counter, so the oracle solve cannot be
    fed the library's counters here; the float64 kernels are held to the oracle's lambda mode by tests/test_gpu_modes.py,
    and the register kernel is held to them"""
    m = W.shell_config(1, ns=40, nchannel=64)
    out, _ = _solve_all(m, ali=False)
    ref = np.ascontiguousarray(out[2].T.astype(np.float64))
    assert check_pops(out[1], ref, tol=1e-3)[0] < 2e-6
    assert check_pops(out[0], ref, tol=1e-3)[0] < 2e-5


def test_species_outside_the_pair_tables_takes_the_float64_solver():
    """levels listed in descending energy: every transition runs from the LOWER index to the higher one, which the dense
    pair tables of k_solve_f do not express: the library must fall back (same populations as the oracle)"""
    import copy
    m = W.shell_config(1, ns=24, nchannel=48)
    s = m.species
    nl = s.nlevel
    perm = np.arange(nl)[::-1]
    inv = np.argsort(perm)
    s2 = copy.copy(s)
    s2.energy_K, s2.g = s.energy_K[perm].copy(), s.g[perm].copy()
    s2.upper, s2.lower = inv[s.upper].astype(np.int32), inv[s.lower].astype(np.int32)
    s2.cu, s2.cl = inv[s.cu].astype(np.int32), inv[s.cl].astype(np.int32)
    m.species = s2
    out, po = _solve_all(m)
    for opt in (0, 1, 2):
        worst, _ = check_pops(out[opt], po, tol=1e-3)
        assert worst < 2e-6, (opt, worst)  # option 0 fell back to float64
