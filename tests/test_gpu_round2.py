"""GPU parity cases added in round 2 ("paths and sizes not reached"), all against the float64 oracle through the
C-ABI: four hierarchy levels in the radiative kernel (C4's depth), 9 transitions x 256 channels (the transitions are split
over two launches), C5's shape (3 traced transitions x 256 channels, +-8 km/s), temperature-dependent collision rates
(ntemp = 3) in 1D and 3D, more than 256 directions, the caller-frame map loc_spectra_map, loc_set_option, and the
call-order / non-finite error paths of loc_solve / loc_iterate."""
import ctypes as C
import math

import numpy as np
import pytest

import loc_workloads as W
import oracle as O
from parity import check_pops, f32_pops_from_oracle_lte, oracle_SJ_ESC, rel_err, tex_all
from test_gpu_3d import small
from test_gpu_spectra import _close

pytestmark = pytest.mark.gpu
H0 = 1 << 20
TOL_SJ = 1e-4
TOL_POP = 1e-3


def _model(m, **kw):
    from paper_2009_12609_b200 import LocModel
    return LocModel(m, **kw)


def _leaf(m):
    return (m.child < 0) if hasattr(m, "child") else np.ones(len(m.density), bool)


def _first_simulate_3d(m, options=()):
    sp = O.OSpecies(m.species)
    sel = np.arange(sp.ntrans, dtype=np.int32) if m.sel is None else m.sel
    pops64, pops32 = f32_pops_from_oracle_lte(sp, m)
    ref = O.sim_3d(sp, m, pops64, sel)
    sj_o, esc_o = oracle_SJ_ESC(sp, m, ref, sel)
    g = _model(m, ntrans_sim=len(sel))
    for k, v in options:
        g.set_option(k, v)
    g.set_populations(pops32)
    g.simulate(None if m.sel is None else sel, geometry_counters=True)
    sj, esc = g.counters()
    sj, esc = sj.cpu().numpy(), esc.cpu().numpy()
    vis, pz = g.geometry_counters()
    launches = g.stats()["kernel_launches"]
    assert np.array_equal(vis.cpu().numpy().astype(np.int64), ref["visits"])
    assert np.array_equal(pz.cpu().numpy().astype(np.int64), ref["pathz"])
    g.close()
    leaf = m.child < 0
    assert np.all(sj[~leaf] == 0)
    assert rel_err(sj[leaf], sj_o[leaf]).max() < TOL_SJ
    assert np.max(np.abs(esc[leaf] - esc_o[leaf]) / (np.abs(esc_o[leaf]) + 3e-3)) < TOL_SJ
    return ref, launches


def test_four_hierarchy_levels_radiative():
    """C4's depth: root + 3 refinement levels = three donor-slot levels in the SAVE / LOAD discipline"""
    m = small(which=4, nroot=4, nlev=4, nside=1, nch=48, frac=0.45, nls=5, seed=4, dens=20.0)
    assert m.nlev == 4
    ref, _ = _first_simulate_3d(m)
    assert ref["ledger"]["created"] > 0 and ref["ledger"]["terminated"] > 0
    assert (m.level[m.child < 0] == 3).sum() > 100


def test_nine_transitions_256_channels_split_launches():
    """9 traced transitions x 256 channels = 36 KB of spectra per ray set > 24 KB: the transitions go through two launches
    (5 + 4) that share the counters' records; thick cells included"""
    m = small(which=4, nroot=5, nlev=2, nside=1, nch=256, frac=0.4, nls=10, dens=10.0)
    from paper_2009_12609_b200 import binding as B
    ref, launches_auto = _first_simulate_3d(m)
    # the same counters with the split forced further (3 launches) and a wider span reach: options change launches, not results
    _, launches_3 = _first_simulate_3d(m, options=((B.LOC_OPT_SIM3D_PARTS, 3), (B.LOC_OPT_SPAN_XCLIP, 3.8)))
    assert launches_3 == launches_auto + 1


@pytest.mark.parametrize("nls,warps", [(4, 1), (4, 2), (2, 1), (2, 2), (6, 1), (7, 1), (7, 2), (5, 2)])
def test_one_and_two_warp_ray_sets(nls, warps):
    """loc_set_option(LOC_OPT_SIM3D_WARPS): one warp per set of four rays carrying all transitions (the default up to 4
    traced transitions) and two warps splitting them give the oracle's counters alike; thick cells, 3 levels, 128 channels"""
    from paper_2009_12609_b200 import binding as B
    m = small(which=4, nroot=4, nlev=3, nside=1, nch=128, frac=0.4, nls=nls, seed=7, dens=15.0)
    _first_simulate_3d(m, options=((B.LOC_OPT_SIM3D_WARPS, warps),))


def test_C5_shape_three_of_nine_transitions_256_channels():
    """C5's shape: root + 2 levels, 3 of 9 transitions traced (R23), 256 channels over +-8 km/s, sigma_ln = 2, 2 km/s rms;
    first-simulate counters and 3 ALI iterations"""
    m = small(which=5, nroot=6, nlev=3, nside=1, nch=256, frac=0.38, nls=10, dens=5.0)
    assert m.band_half == 8e5 and list(m.sel) == [0, 1, 2] and m.nlev == 3
    _first_simulate_3d(m)
    sp = O.OSpecies(m.species)
    pops_o, _ = O.iterate(sp, m, 3, sel=m.sel)
    g = _model(m, ntrans_sim=3)
    g.init_lte()
    g.simulate(m.sel)
    g.init_lte()
    g.iterate(3)
    pg = g.pops.cpu().numpy()
    g.close()
    leaf = m.child < 0
    worst, small_abs = check_pops(pg[:, leaf], pops_o[leaf])
    assert worst < TOL_POP and small_abs < 1e-10


def _ntemp_species(nlevel, config):
    s = W.rotor_species(nlevel, config)
    rs = np.random.default_rng([91, nlevel])
    temps = np.array([8.0, 12.0, 18.0])
    s.rate_down = np.stack([s.rate_down[0] * rs.uniform(0.4, 2.5, size=s.rate_down.shape[1]) for _ in temps])
    s.temps_K = temps
    return s


@pytest.mark.parametrize("kind", ["1d", "3d", "3d-20levels"])
def test_temperature_dependent_collision_rates(kind):
    """ntemp = 3 table (R18): cells below, between and above the nodes; the oracle's interpolation is pinned
    by tests/test_oracle_pins_1d.py::test_coll_gamma_*.  The 20-level case takes the local-memory solver."""
    if kind == "1d":
        m = W.shell_config(2, ns=48, nchannel=96, nsub=2, nlevel=6)  # T_kin = 8 .. 15 K
        m.tkin[:] = np.linspace(5.0, 24.0, 48).astype(np.float32)
        m.species = _ntemp_species(6, 2)
        sel = None
    else:
        nls = 20 if kind.endswith("levels") else 5
        m = small(which=4, nroot=4, nlev=2, nside=1, nch=40, frac=0.4, nls=nls)  # T_kin = 10 .. 20 K per cell
        m.tkin[::7] = 6.0
        m.species = _ntemp_species(nls, 4)
        sel = np.arange(12, dtype=np.int32) if nls == 20 else None
    sp = O.OSpecies(m.species)
    assert (m.tkin < 8).any() and (m.tkin > 18).any() and ((m.tkin > 8) & (m.tkin < 18)).any()
    pops_o, _ = O.iterate(sp, m, 3, sel=sel)
    g = _model(m, ntrans_sim=(len(sel) if sel is not None else None))
    g.init_lte()
    if sel is not None:
        g.simulate(sel)
        g.init_lte()
    g.iterate(3)
    pg = g.pops.cpu().numpy()
    g.close()
    leaf = _leaf(m)
    worst, small_abs = check_pops(pg[:, leaf], pops_o[leaf])
    assert worst < TOL_POP and small_abs < 1e-10
    # the table matters: with the first row alone the oracle is off by far more than the tolerance
    s1 = W.rotor_species(len(m.species.energy_K), 2 if kind == "1d" else 4)
    s1.rate_down = m.species.rate_down[:1].copy()
    m1 = m
    m1.species = s1
    p1, _ = O.iterate(O.OSpecies(s1), m1, 3, sel=sel)
    assert np.max(np.abs(p1[leaf][:, 1] / pops_o[leaf][:, 1] - 1)) > 5 * TOL_POP


def test_more_than_256_directions():
    """768 directions (HEALPix Nside = 8) on a tiny octree: the task -> direction table holds 16-bit indices"""
    m = small(which=4, nroot=2, nlev=2, nside=8, nch=32, frac=0.5, nls=3)
    assert len(m.dirs) == 768
    ref, _ = _first_simulate_3d(m)
    assert ref["pathz"][m.child < 0].min() > 0


def test_spectra_map_caller_frame():
    """loc_spectra_map: pixel positions from the caller's frame (include/loc.h).  The expected start positions are written
    out here from the definition, with numpy, and the oracle integrates each pixel's line of sight on its own."""
    m = W.cloud_config(4, nroot=4, nlev=3, nchannel=40, nside=1, refine_frac=0.4, nlevel_species=4)
    m.abundance[:] = 3e-4
    sp = O.OSpecies(m.species)
    pops64, pops32 = f32_pops_from_oracle_lte(sp, m)
    g = _model(m)
    g.set_populations(pops32)
    L = m.nx * m.root_cm
    nfine = m.nx << (m.nlev - 1)
    pix_cm = m.root_cm / (1 << (m.nlev - 1))
    # (a) along +z, pixel = finest cell, centred: identical to the integer map of the bench (C5's map)
    pix = H0 >> (m.nlev - 1)
    for dz in (1.0, -1.0):
        d = np.array([0.0, 0.0, dz])
        ta = g.spectra_map(0, nfine, nfine, d, pix_cm, np.array([0.5 * L, 0.5 * L, 0.5 * L])).cpu().numpy()
        if dz > 0:
            ref = O.spectra_3d(sp, m, pops64, 0, d, nfine, nfine, np.array([pix // 2, pix // 2, pix, 0, 0, pix], np.int64))
        else:
            # from the other side: e1 = e2 x dir = y x (-z) = -x, so ix runs towards -x; working frame of -z: main axis z
            # mirrored, p = x, q = y not mirrored
            ref = O.spectra_3d(sp, m, pops64, 0, d, nfine, nfine, np.array([pix // 2, pix // 2, pix, 0, 0, pix], np.int64))[:, ::-1]
        _close(ta, ref)
    # (b) oblique direction, off-centre, pixel not commensurate with the cells: per-pixel start positions from the definition
    d = np.array([0.35, -0.5, 0.79])
    d /= np.linalg.norm(d)
    centre = np.array([0.47, 0.55, 0.52]) * L
    nx_, ny_, pcm = 7, 5, 0.37 * m.root_cm
    ta = g.spectra_map(1, nx_, ny_, d, pcm, centre).cpu().numpy()
    north = np.array([0.0, 0.0, 1.0])
    e2 = north - north.dot(d) * d
    e2 /= np.linalg.norm(e2)
    e1 = np.cross(e2, d)
    a = np.abs(d)
    ma = int(np.argmax(a >= a.max()))
    p, q = (ma + 1) % 3, (ma + 2) % 3
    sl = []
    for ax in (p, q):
        S = int(np.rint(a[ax] / a[ma] * 2 ** 20))
        sl.append(0.0 if S == 0 else 2.0 ** 32 / ((2 ** 52 + S // 2) // S))
    upc = H0 / m.root_cm
    Wd = m.nx * H0
    nonzero = 0
    for iy in range(ny_):
        for ix in range(nx_):
            X = centre + (ix - 0.5 * (nx_ - 1)) * pcm * e1 + (iy - 0.5 * (ny_ - 1)) * pcm * e2
            w = [Wd - upc * X[k] if d[k] < 0 else upc * X[k] for k in (ma, p, q)]
            bp, bq = math.floor(w[1] - sl[0] * w[0]), math.floor(w[2] - sl[1] * w[0])
            ref = O.spectra_3d(sp, m, pops64, 1, d, 1, 1, np.array([bp, bq, 0, 0, 0, 0], np.int64))[0, 0]
            # the library forms the same position from an affine map in double: allow the start to be one grid unit
            # (1e-6 of a root cell) off, which moves a spectrum by far less than the tolerance unless the line grazes a face
            _close(ta[iy, ix], ref)
            nonzero += bool(np.any(ref != 0))
    assert nonzero >= 20
    from paper_2009_12609_b200 import binding as B
    with pytest.raises(B.LocError):
        g.spectra_map(0, 4, 4, np.array([0.0, 0.0, 2.0]), pix_cm, centre)
    with pytest.raises(B.LocError):
        g.spectra_map(0, 4, 4, np.array([0.0, 0.0, 1.0]), -1.0, centre)
    g.close()


def test_options_and_error_paths():
    from paper_2009_12609_b200 import binding as B
    m = W.shell_config(1, ns=12, nchannel=32)
    sp = O.OSpecies(m.species)
    g = _model(m)
    lib = B.lib()
    assert lib.loc_set_option(g.h, 999, C.c_double(1.0)) == B.LOC_EINVAL
    assert lib.loc_set_option(g.h, B.LOC_OPT_WINDOW_XMIN, C.c_double(0.1)) == B.LOC_EINVAL
    assert lib.loc_set_option(g.h, B.LOC_OPT_SIM3D_PARTS, C.c_double(2.5)) == B.LOC_EINVAL
    assert lib.loc_set_option(None, B.LOC_OPT_WINDOW_XMIN, C.c_double(5.0)) == B.LOC_EINVAL
    # loc_solve before any loc_simulate: the counters hold nothing
    g.init_lte()
    assert lib.loc_solve(g.h, None) == B.LOC_ESTATE
    # niter = 0: nothing runs, change 0 (not the stale value of an earlier call)
    g.iterate(2)
    assert g.iterate(0) == 0.0
    # a narrower window is a different (worse) approximation; a wider one stays within tolerance: the option is live
    pops_o, _ = O.iterate(sp, m, 3)
    out = {}
    for x in (2.0, 6.0):
        g.set_option(B.LOC_OPT_WINDOW_XMIN, x)
        g.set_option(B.LOC_OPT_WINDOW_EPS_TAU, 1.0 if x == 2.0 else 1e-6)  # both rules of the window cut at 2 sigma / are default
        g.init_lte()
        g.iterate(3)
        out[x] = check_pops(g.pops.cpu().numpy(), pops_o)[0]
    assert out[6.0] < TOL_POP and out[2.0] > out[6.0]
    # the local-memory solver gives the same populations
    g.set_option(B.LOC_OPT_WINDOW_XMIN, 4.5)
    g.set_option(B.LOC_OPT_WINDOW_EPS_TAU, 1e-6)
    g.set_option(B.LOC_OPT_SOLVER_LOCAL, 1)
    g.init_lte()
    g.iterate(3)
    assert check_pops(g.pops.cpu().numpy(), pops_o)[0] < TOL_POP
    g.close()
    # non-finite populations are reported, not read as "converged"
    bad = W.shell_config(1, ns=12, nchannel=32)
    bad.tkin[3] = np.float32("nan")
    g = _model(bad)
    g.init_lte()
    with pytest.raises(B.LocError) as ei:
        g.iterate(1)
    assert ei.value.code == B.LOC_ENONFINITE
    with pytest.raises(B.LocError) as ei:
        g.iterate_until(5, 1e-3)
    assert ei.value.code == B.LOC_ENONFINITE
    g.close()


def test_state_guards_after_species_or_profile_change_and_no_collisions():
    """(a) loc_set_hyperfine / loc_set_species after a loc_simulate invalidate the counters -- loc_solve then
    returns LOC_ESTATE instead of solving on counters traced with another profile / species; (b) a species WITHOUT
    collisional pairs but WITH a temperature grid (ncoll = 0, ntemp > 1: legal) solves to finite populations (round 2 read
    uninitialised temperatures there) and gives what the oracle gives."""
    from paper_2009_12609_b200 import binding as B
    lib = B.lib()
    m = W.shell_config(1, ns=12, nchannel=32)
    g = _model(m)
    g.init_lte()
    g.simulate()
    assert lib.loc_solve(g.h, None) == B.LOC_OK
    g.simulate()
    B.loc_set_hyperfine(g.h, 0, [-0.3e5, 0.2e5], [0.4, 0.6])
    assert lib.loc_solve(g.h, None) == B.LOC_ESTATE
    g.simulate()
    assert lib.loc_solve(g.h, None) == B.LOC_OK
    B.loc_set_species(g.h, m.species)
    B.loc_set_populations(g.h, g.pops)
    assert lib.loc_solve(g.h, None) == B.LOC_ESTATE
    g.close()
    # (b) radiative-only species on a 3-node temperature grid
    m = W.shell_config(1, ns=12, nchannel=32)
    s = m.species
    s.cu, s.cl = np.zeros(0, np.int32), np.zeros(0, np.int32)
    s.temps_K = np.array([8.0, 12.0, 18.0])
    s.rate_down = np.zeros((3, 0))
    sp = O.OSpecies(s)
    pops_o, _ = O.iterate(sp, m, 2)
    g = _model(m)
    g.init_lte()
    g.iterate(2)
    pg = g.pops.cpu().numpy()
    g.close()
    assert np.all(np.isfinite(pg))
    assert check_pops(pg, pops_o)[0] < TOL_POP


def test_set_directions_invalid_arguments_keep_the_old_directions():
    """an invalid ARGUMENT (not a unit vector, more directions than ndir_max) is rejected before anything is touched: the
    model keeps its directions and step stream.  (A failure INSIDE the path set-up -- LOC_ENOMEM / LOC_ECUDA -- leaves the
    model without directions, include/loc.h; the workspace bound of 3 records per cell and direction is not reachable
    with a valid octree, so that branch has no test.)"""
    from paper_2009_12609_b200 import binding as B
    m = small(which=4, nroot=4, nlev=3, nside=1, nch=32, frac=0.5, nls=3)
    g = _model(m, ndir_max=12)
    g.init_lte()
    g.simulate()
    lib = B.lib()
    many = np.ascontiguousarray(np.tile(m.dirs, (1, 1)), np.float64)
    bad = many.copy()
    bad[5] *= 1.1
    assert lib.loc_set_directions(g.h, 12, bad.ctypes.data_as(C.c_void_p)) == B.LOC_EINVAL
    g.simulate()  # an invalid ARGUMENT leaves the old directions in place
    assert lib.loc_set_directions(g.h, 13, many.ctypes.data_as(C.c_void_p)) == B.LOC_EINVAL  # more than ndir_max
    g.close()


@pytest.mark.parametrize("case", ["octree", "C3", "1d"])
def test_counters_reproducible_run_to_run(case):
    """compute-sanitizer is closed on the GPU pool (profiles/r2_sanitizer.md), so a race between the lanes / warps that share a
    ray's spectra in shared memory is looked for by its symptom: two simulations from the same populations must give the same
    counters up to the order of the float32 atomic additions (observed ~1e-6; a lost or doubled update of a spectrum is
    orders of magnitude above that), and identical integer visit counts.  Thick octree with births, full-size C3, and 1D."""
    if case == "octree":
        m = small(which=4, nroot=6, nlev=3, nside=2, nch=128, frac=0.45, nls=10, seed=13, dens=20.0)
    elif case == "C3":
        m = W.cloud_config(3)
    else:
        m = W.shell_config(2, ns=400, nchannel=256, nsub=2)
    g = _model(m)
    g.init_lte()
    g.iterate(2)  # populations away from LTE
    out = []
    for _ in range(3):
        g.simulate(geometry_counters=True)
        sj, esc = g.counters()
        vis, _ = g.geometry_counters()
        out.append((sj.cpu().numpy().astype(np.float64), esc.cpu().numpy().astype(np.float64), vis.cpu().numpy().copy()))
    g.close()
    leaf = _leaf(m)
    for k in (1, 2):
        assert np.array_equal(out[k][2], out[0][2])
        assert rel_err(out[k][0][leaf], out[0][0][leaf]).max() < 2e-5
        assert np.max(np.abs(out[k][1][leaf] - out[0][1][leaf])) < 2e-5
