"""GPU parity with hyperfine structure (include/loc.h loc_set_hyperfine) against the
float64 oracle (pinned by tests/test_oracle_pins_hfs.py): first-simulate counters, populations / T_ex after ALI iterations, and
spectra, in 1D and on an octree; separated and overlapping components, mixed with transitions that have none."""
import copy

import numpy as np
import pytest

import loc_workloads as W
import oracle as O
from parity import check_pops, f32_pops_from_oracle_lte, oracle_SJ_ESC, rel_err, tex_all
from test_gpu_3d import small

pytestmark = pytest.mark.gpu
TOL_SJ = 1e-4
TOL_POP = 1e-3
KMS = 1e5


def _model(m, **kw):
    from paper_2009_12609_b200 import LocModel
    return LocModel(m, **kw)


def _hfs(m, table):
    m.species = copy.copy(m.species)
    m.species.hfs = {t: (np.asarray(d, float) * KMS, np.asarray(w, float)) for t, (d, w) in table.items()}
    return m


HFS_A = {0: ([-1.1, 0.05, 0.8], [0.2, 0.5, 0.3])}                                    # separated components, one transition
HFS_B = {0: ([-0.25, 0.0, 0.3], [0.3, 0.4, 0.3]), 2: ([-0.9, 0.9], [0.5, 0.5])}      # overlapping ones, and a doublet


@pytest.mark.parametrize("table,dens", [(HFS_A, 1.0), (HFS_B, 1.0), (HFS_A, 30.0)])
def test_1d_counters_and_iterations(table, dens):
    m = _hfs(W.shell_config(1, ns=40, nchannel=128), table)
    m.band_half = 3.0 * KMS
    m.density *= np.float32(dens)
    sp = O.OSpecies(m.species)
    pops64, pops32 = f32_pops_from_oracle_lte(sp, m)
    sel = np.arange(sp.ntrans, dtype=np.int32)
    ref = O.sim_1d(sp, m, pops64, sel)
    sj_o, esc_o = oracle_SJ_ESC(sp, m, ref, sel)
    g = _model(m)
    g.set_populations(pops32)
    g.simulate(geometry_counters=True)
    sj, esc = g.counters()
    sj, esc = sj.cpu().numpy(), esc.cpu().numpy()
    st = g.stats()
    assert rel_err(sj, sj_o).max() < TOL_SJ
    assert np.max(np.abs(esc - esc_o) / (np.abs(esc_o) + 3e-3)) < TOL_SJ
    # active updates: a transition with separated components has more channels within 5 sigma of a component than a single line
    assert st["active_updates"] > st["steps"] * sp.ntrans * 10
    pops_o, _ = O.iterate(sp, m, 6)
    g.init_lte()
    g.iterate(6)
    pg = g.pops.cpu().numpy()
    worst, small_abs = check_pops(pg, pops_o)
    assert worst < TOL_POP and small_abs < 1e-10
    assert rel_err(tex_all(sp, pg.astype(np.float64).T, m.species), tex_all(sp, pops_o, m.species)).max() < TOL_POP
    # spectra of the hyperfine transition and of a plain one, with the converged populations on both sides
    b = np.array([0.0, 0.4, 0.9]) * m.r_out[-1]
    for t in (0, 1):
        TA_o = O.spectra_1d(sp, m, pg.astype(np.float64).T, t, b)
        TA = g.spectra(t, len(b), offsets_cm=b).cpu().numpy()[0]
        assert np.max(np.abs(TA - TA_o)) < 2e-4 * np.max(np.abs(TA_o))
    g.close()


def test_1d_single_component_equals_no_structure():
    """one component at a negligible offset (1e-4 cm/s) takes the general path of the kernel and must give the plain kernel's
    counters (two code paths: 2e-5)"""
    m0 = W.shell_config(1, ns=30, nchannel=64)
    out = []
    for m in (m0, _hfs(copy.copy(m0), {1: ([1e-9], [1.0])})):
        g = _model(m)
        g.init_lte()
        g.simulate()
        sj, esc = g.counters()
        out.append((sj.cpu().numpy().copy(), esc.cpu().numpy().copy()))
        g.close()
    assert rel_err(out[1][0], out[0][0]).max() < 2e-5
    assert np.max(np.abs(out[1][1] - out[0][1])) < 2e-5


@pytest.mark.parametrize("table", [HFS_A, HFS_B])
def test_3d_counters_iterations_and_map(table):
    m = _hfs(small(which=4, nroot=4, nlev=3, nside=1, nch=128, frac=0.4, nls=4, seed=3, dens=10.0), table)
    sp = O.OSpecies(m.species)
    pops64, pops32 = f32_pops_from_oracle_lte(sp, m)
    sel = np.arange(sp.ntrans, dtype=np.int32)
    ref = O.sim_3d(sp, m, pops64, sel)
    sj_o, esc_o = oracle_SJ_ESC(sp, m, ref, sel)
    g = _model(m)
    g.set_populations(pops32)
    g.simulate(geometry_counters=True)
    sj, esc = g.counters()
    sj, esc = sj.cpu().numpy(), esc.cpu().numpy()
    vis, _ = g.geometry_counters()
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), ref["visits"])
    leaf = m.child < 0
    assert rel_err(sj[leaf], sj_o[leaf]).max() < TOL_SJ
    assert np.max(np.abs(esc[leaf] - esc_o[leaf]) / (np.abs(esc_o[leaf]) + 3e-3)) < TOL_SJ
    pops_o, _ = O.iterate(sp, m, 3)
    g.init_lte()
    g.iterate(3)
    pg = g.pops.cpu().numpy()
    worst, small_abs = check_pops(pg[:, leaf], pops_o[leaf])
    assert worst < TOL_POP and small_abs < 1e-10
    # map along +z, one pixel per finest cell
    nfine = m.nx << (m.nlev - 1)
    pix = (1 << 20) >> (m.nlev - 1)
    aff = np.array([pix // 2, pix // 2, pix, 0, 0, pix], np.int64)
    zdir = np.array([0.0, 0.0, 1.0])
    TA_o = O.spectra_3d(sp, m, pg.astype(np.float64).T, 0, zdir, nfine, nfine, aff)
    TA = g.spectra(0, nfine, nfine, dir=zdir, aff=aff).cpu().numpy()
    assert np.max(np.abs(TA - TA_o)) < 2e-4 * np.max(np.abs(TA_o))
    g.close()


def test_set_hyperfine_rejects_bad_arguments():
    import ctypes as C
    from paper_2009_12609_b200 import binding as B
    m = W.shell_config(1, ns=8, nchannel=32)
    g = _model(m)
    lib = B.lib()
    d = np.array([0.0, 1e4]); w = np.array([0.5, 0.6])
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    assert lib.loc_set_hyperfine(g.h, 0, 2, p(d), p(w)) == B.LOC_EINVAL          # weights do not sum to 1
    assert lib.loc_set_hyperfine(g.h, 99, 1, p(d), p(w)) == B.LOC_EINVAL         # no such transition
    assert lib.loc_set_hyperfine(g.h, 0, B.LOC_MAX_HFS + 1, p(d), p(w)) == B.LOC_EINVAL
    w = np.array([0.5, 0.5])
    assert lib.loc_set_hyperfine(g.h, 0, 2, p(d), p(w)) == B.LOC_OK
    assert lib.loc_set_hyperfine(g.h, 0, 0, None, None) == B.LOC_OK              # removed again
    g.close()
