"""GPU parity of the 1D shell-ray path (K1 + K8) against the float64 oracle, through the C-ABI binding."""
import numpy as np
import pytest

import loc_workloads as W
import oracle as O
from parity import check_pops, f32_pops_from_oracle_lte, oracle_SJ_ESC, rel_err, tex_all

pytestmark = pytest.mark.gpu

TOL_SJ = 1e-4   # north_star: per-cell absorbed-photon counts within 1e-4 relative
TOL_POP = 1e-3  # north_star: populations and T_ex within 1e-3 relative


def _model(m):
    from paper_2009_12609_b200 import LocModel
    return LocModel(m)


def _first_simulate(m, sel=None):
    sp = O.OSpecies(m.species)
    pops64, pops32 = f32_pops_from_oracle_lte(sp, m)
    sel = np.arange(sp.ntrans, dtype=np.int32) if sel is None else np.asarray(sel, np.int32)
    ref = O.sim_1d(sp, m, pops64, sel)
    sj_o, esc_o = oracle_SJ_ESC(sp, m, ref, sel)
    g = _model(m)
    g.set_populations(pops32)
    g.simulate(sel if len(sel) != sp.ntrans else None, geometry_counters=True)
    sj, esc = g.counters()
    vis, _ = g.geometry_counters()
    sj, esc, vis = sj.cpu().numpy(), esc.cpu().numpy(), vis.cpu().numpy()
    steps = g.stats()["steps"]
    g.close()
    return sj, esc, vis, steps, sj_o, esc_o, ref


@pytest.mark.parametrize("cfg", [dict(which=1), dict(which=1, ns=37, nchannel=50, nsub=3),
                                 dict(which=2, ns=150, nchannel=256, nsub=4), dict(which=2, ns=61, nchannel=97, nsub=2, nlevel=4)])
def test_first_simulate_counters(cfg):
    m = W.shell_config(**cfg)
    sj, esc, vis, steps, sj_o, esc_o, ref = _first_simulate(m)
    assert np.array_equal(vis.astype(np.int64), ref["visits"])  # bit-exact visit counts
    assert steps == ref["visits"].sum()
    assert rel_err(sj, sj_o).max() < TOL_SJ
    assert np.max(np.abs(esc - esc_o) / (np.abs(esc_o) + 3e-3)) < TOL_SJ


def test_selection_subset():
    m = W.shell_config(2, ns=40, nchannel=128, nsub=2)
    sj, esc, vis, steps, sj_o, esc_o, ref = _first_simulate(m, sel=[0, 2, 5])
    assert sj.shape[1] == 3
    assert rel_err(sj, sj_o).max() < TOL_SJ


def test_init_lte_matches_oracle():
    m = W.shell_config(2, ns=50, nsub=1, nchannel=32)
    sp = O.OSpecies(m.species)
    g = _model(m)
    g.init_lte()
    p = g.pops.cpu().numpy().astype(np.float64).T
    ref = O.lte(sp, m.density, m.tkin, m.abundance)
    assert rel_err(p, ref).max() < 2e-7
    g.close()


@pytest.mark.parametrize("cfg,niter", [(dict(which=1), 20), (dict(which=2, ns=120, nchannel=256, nsub=4), 8)])
def test_iterate_populations_and_tex(cfg, niter):
    m = W.shell_config(**cfg)
    sp = O.OSpecies(m.species)
    pops_o, change_o = O.iterate(sp, m, niter)
    g = _model(m)
    g.init_lte()
    change_g = g.iterate(niter)
    pg = g.pops.cpu().numpy()
    g.close()
    worst, small_abs = check_pops(pg, pops_o)
    assert worst < TOL_POP and small_abs < 1e-13 + 1e-10
    tg, to = tex_all(sp, pg.astype(np.float64).T, m.species), tex_all(sp, pops_o, m.species)
    big = pops_o[:, 1:] >= 1e-10 * pops_o.sum(axis=1, keepdims=True)
    assert rel_err(tg, to)[big].max() < TOL_POP
    assert abs(change_g - change_o) <= 0.05 * change_o + 1e-5


def test_solve_only_lte_limit():
    """high density: one solve from any counters must give Boltzmann populations (pin P3 through the GPU solver)."""
    m = W.shell_config(1, ns=16, nchannel=32)
    m.density[:] = 1e12
    sp = O.OSpecies(m.species)
    g = _model(m)
    g.init_lte()
    g.simulate()
    g.solve()
    p = g.pops.cpu().numpy().astype(np.float64).T
    ref = O.lte(sp, m.density, m.tkin, m.abundance)
    assert rel_err(p, ref).max() < 1e-5
    g.close()


def test_error_paths():
    from paper_2009_12609_b200 import binding as B
    m = W.shell_config(1, ns=8, nchannel=16)
    g = _model(m)
    with pytest.raises(B.LocError):
        g.simulate(sel=[99])
    with pytest.raises(B.LocError):
        g.set_directions(np.array([[0.0, 0.0, 1.0]]))
    g.close()
    bad = W.shell_config(1, ns=8, nchannel=16)
    bad.r_out = bad.r_out[::-1].copy()
    with pytest.raises(B.LocError):
        _model(bad)


def test_full_size_C2_invariants_and_enclosure():
    """BASELINE size, the launch configuration bench.py times (C2: 1000 shells, 4000 rays, 256 channels, 9 transitions,
    k_sim1d_w).  The oracle needs minutes per iteration at this size, so properties that hold at any size are checked:
      * every ray visits the shells of its path once in and once out: total visits = sum over rays of 2 (NS - 1 - k0) + 1
        = the library's step count, and shell k is visited by every ray whose tangent shell lies at or inside it;
      * pin P4 (blackbody enclosure): with T_bg = T_kin everywhere, one ALI iteration from LTE leaves the populations
        unchanged -- every normalisation of the ray weights, path lengths and counters enters;
      * escape fractions lie in (0, 1], counters are finite."""
    m = W.shell_config(2)
    m.tkin[:] = 10.0
    m.t_bg = 10.0
    g = _model(m)
    g.init_lte()
    g.simulate(geometry_counters=True)
    vis, _ = g.geometry_counters()
    vis = vis.cpu().numpy().astype(np.int64)
    st = g.stats()
    k0 = np.searchsorted(m.r_out, m.ray_p, side="right")  # tangent shell of each ray: first shell whose outer radius exceeds p
    ns = len(m.r_out)
    inside = k0 < ns
    expect = np.zeros(ns, np.int64)
    for k in k0[inside]:
        expect[k] += 1
        expect[k + 1:] += 2
    assert np.array_equal(vis, expect)
    assert vis.sum() == st["steps"] == int(np.sum(2 * (ns - 1 - k0[inside]) + 1))
    sj, esc = g.counters()
    sj, esc = sj.cpu().numpy(), esc.cpu().numpy()
    assert np.isfinite(sj).all() and np.isfinite(esc).all()
    assert esc.min() > 0 and esc.max() <= 1.0 + 1e-5
    p0 = g.pops.clone()
    change = g.iterate(1)
    p1, p0 = g.pops.cpu().numpy(), p0.cpu().numpy()
    g.close()
    big = p0 > 1e-10 * p0.sum(axis=0, keepdims=True)
    assert np.max(np.abs(p1 - p0)[big] / p0[big]) < 5e-5 and change < 5e-5
