"""Pins of the oracle's hyperfine-structure profile ("assuming an LTE distribution
between the hyperfine components").  The definition: transition t has components k with velocity offsets dv_k and weights
w_k (sum 1); its profile is sum_k w_k Gaussian(v - v0 - dv_k); one population per level, so all components share one
source function.  Every expected value below comes from the single-component oracle (pinned elsewhere), from numpy, or
from a closed form -- never from the hyperfine code path itself."""
import copy
import math

import numpy as np
import pytest

import loc_workloads as W
import oracle as O

H, K, C = 6.62607015e-27, 1.380649e-16, 2.99792458e10


def _with_hfs(s, hfs):
    s2 = copy.copy(s)
    s2.hfs = dict(hfs)
    return s2


def test_one_component_is_the_plain_profile_bit_for_bit():
    """a single component at zero offset with weight 1 takes the hyperfine branch and must reproduce every counter"""
    m = W.shell_config(1, ns=10, nchannel=48)
    s0 = m.species
    o0 = O.OSpecies(s0)
    o1 = O.OSpecies(_with_hfs(s0, {0: ([0.0], [1.0]), 2: ([0.0], [1.0])}))
    pops = O.lte(o0, m.density, m.tkin, m.abundance)
    a, b = O.sim_1d(o0, m, pops), O.sim_1d(o1, m, pops)
    for k in ("ABS", "P", "LAM"):
        assert np.array_equal(a[k], b[k])
    m3 = W.cloud_config(4, nroot=3, nlev=2, nchannel=24, nside=1, refine_frac=0.4, nlevel_species=3)
    o0, o1 = O.OSpecies(m3.species), O.OSpecies(_with_hfs(m3.species, {1: ([0.0], [1.0])}))
    pops = O.lte(o0, m3.density, m3.tkin, m3.abundance)
    O.set_threads(1)  # (with several OpenMP threads the order of the atomic additions differs from run to run)
    try:
        a, b = O.sim_3d(o0, m3, pops), O.sim_3d(o1, m3, pops)
    finally:
        import os
        O.set_threads(os.cpu_count() or 1)
    for k in ("ABS", "P", "LAM"):
        assert np.array_equal(a[k], b[k])


def test_profile_is_the_weighted_sum_of_shifted_gaussians():
    """against numpy: weights, offsets and their sign (a component with dv_k > 0 sits at HIGHER channel velocity)"""
    s = W.rotor_species(3, 1)
    dvk, wk = np.array([-7.0e4, 0.0, 4.8e4]), np.array([0.2, 0.5, 0.3])
    o = O.OSpecies(_with_hfs(s, {0: (dvk, wk)}))
    nch, dv, sigma, v0 = 256, 62.5e2, 0.21e5, 0.13e5
    phi = O.profile_t(o, 0, nch, dv, sigma, v0)
    v = (np.arange(nch) - 0.5 * (nch - 1)) * dv
    expect = sum(w * dv / (sigma * math.sqrt(2 * math.pi)) * np.exp(-0.5 * ((v - v0 - d) / sigma) ** 2) for d, w in zip(dvk, wk))
    assert np.max(np.abs(phi - expect)) < 1e-15
    assert abs(phi.sum() - 1.0) < 1e-12  # all components inside the band: the weights keep the normalisation
    assert abs((phi * v).sum() - (v0 + (wk * dvk).sum())) < 1e-6 * sigma  # first moment: the weighted offset
    # the other transition has no hyperfine structure: the plain profile
    assert np.array_equal(O.profile_t(o, 1, nch, dv, sigma, v0), O.profile(nch, dv, sigma, v0))


def test_thin_limit_line_area_is_unchanged_and_components_carry_their_weight():
    """P2 with hyperfine structure: in the thin limit the integrated line is the column density of the upper level whatever
    the split, and with offsets of whole channels the spectrum is the weighted sum of shifted copies of the single line"""
    m = W.shell_config(1, ns=12, nchannel=256)
    m.band_half = 8e5
    m.t_bg = 0.0
    m.abundance[:] = 1e-12
    m.vrad[:] = 0
    dv = 2 * m.band_half / m.nchannel
    shifts, wk = np.array([-60, 0, 45]), np.array([0.15, 0.6, 0.25])
    s0 = m.species
    o0, o1 = O.OSpecies(s0), O.OSpecies(_with_hfs(s0, {0: (shifts * dv, wk)}))
    pops = O.lte(o0, m.density, m.tkin, m.abundance)
    b = np.array([0.0, 0.5]) * m.r_out[-1]
    T0, T1 = O.spectra_1d(o0, m, pops, 0, b), O.spectra_1d(o1, m, pops, 0, b)
    assert np.max(np.abs(T1.sum(axis=1) / T0.sum(axis=1) - 1)) < 1e-6  # (equal up to O(tau))
    expect = sum(w * np.roll(T0, sh, axis=1) for sh, w in zip(shifts, wk))
    assert np.max(np.abs(T1 - expect)) < 1e-6 * T0.max()  # (thin: tau ~ 1e-7; the residual is O(tau))
    # the counters of the simulation: without a background the only photons are the line's own; a photon emitted in
    # component k (fraction w_k) is absorbed by component k only (fraction w_k of the opacity): with separated components
    # the absorbed-photon counter is sum_k w_k^2 of the single line's, shell by shell
    a, h = O.sim_1d(o0, m, pops, np.array([0], np.int32)), O.sim_1d(o1, m, pops, np.array([0], np.int32))
    assert np.max(np.abs(h["P"] / a["P"] / (wk ** 2).sum() - 1)) < 1e-6


def test_slab_closed_form_with_overlapping_components():
    """P1 with hyperfine structure: I = B(T_bg) e^-tau + S (1 - e^-tau) per channel with tau from the summed profile (numpy)
    and the textbook Einstein-B absorption coefficient; components overlapping in velocity, thick and thin channels"""
    s = W.rotor_species(4, 1)
    dvk, wk = np.array([-0.3e5, 0.1e5, 0.5e5]), np.array([0.3, 0.45, 0.25])
    o = O.OSpecies(_with_hfs(s, {1: (dvk, wk)}))
    t, nch, band, tbg = 1, 96, 3e5, 2.73
    dv = 2 * band / nch
    a, steps, n_l, n_u, sigma, v0 = 2.2e30, np.array([2e15, 5e16, 9e14, 1e17]), 0.7, 0.3, 0.2e5, -0.2e5
    N, acc, _ = O.slab(o, t, nch, band, tbg, a, 1.0, steps, sigma, v0, n_u, n_l)
    v = (np.arange(nch) - 0.5 * (nch - 1)) * dv
    phi = sum(w * dv / (sigma * math.sqrt(2 * math.pi)) * np.exp(-0.5 * ((v - v0 - d) / sigma) ** 2) for d, w in zip(dvk, wk))
    u, l = s.upper[t], s.lower[t]
    nu = (s.energy_K[u] - s.energy_K[l]) * K / H
    Bul = C ** 2 * s.einstein_A[t] / (2 * H * nu ** 3)
    kap = H * nu / (4 * math.pi) * (n_l * s.g[u] / s.g[l] * Bul - n_u * Bul) * phi / (nu * dv / C)
    tau = kap * steps.sum()
    assert tau.max() > 1.0 and tau.min() < 1e-6
    Snu = 2 * H * nu ** 3 / C ** 2 / (n_l * s.g[u] / (n_u * s.g[l]) - 1)
    I_expect = O.planck(nu, tbg) * np.exp(-tau) + Snu * (-np.expm1(-tau))
    I = N / (a * 4 * math.pi * dv / (H * C))
    assert np.max(np.abs(I / I_expect - 1)) < 1e-13


def test_thick_components_saturate_at_the_same_source_function():
    """LTE between the components: one population per level, so every component that is optically thick
    reaches the SAME brightness (h nu / k)(S - n_bg) however small its weight -- a per-component source function or a
    weight applied to the emission alone would not"""
    s = W.rotor_species(3, 1)
    m = W.shell_config(1, ns=8, nchannel=256)
    m.band_half = 8e5
    dv = 2 * m.band_half / m.nchannel
    shifts, wk = np.array([-70, 0, 60]), np.array([0.1, 0.6, 0.3])
    m.species = _with_hfs(s, {0: (shifts * dv, wk)})
    o = O.OSpecies(m.species)
    m.density[:] = 1e5
    m.tkin[:] = 12.0
    m.vrad[:] = 0.0
    m.abundance[:] = 1e-3
    pops = O.lte(o, m.density, m.tkin, m.abundance)
    pops[:, 1] *= 0.7
    TA = O.spectra_1d(o, m, pops, 0, np.array([0.0]))[0]
    nu = o.freq(0)
    S_occ = 1.0 / (pops[0, 0] * s.g[1] / (pops[0, 1] * s.g[0]) - 1.0)
    plateau = H * nu / K * (S_occ - 1.0 / math.expm1(H * nu / (K * m.t_bg)))
    centre = (m.nchannel - 1) / 2
    for sh in shifts:
        c = int(round(centre + sh))
        assert abs(TA[c] / plateau - 1) < 1e-6, (sh, TA[c], plateau)


def test_blackbody_enclosure_and_mirror_with_hyperfine_structure():
    """P4 and P12 with a hyperfine transition: T_bg = T_kin keeps LTE (normalisation of the summed profile in every
    counter); mirroring the offsets and the velocities mirrors the channels and leaves the populations unchanged"""
    m = W.shell_config(1, ns=10, nchannel=128)
    m.band_half = 4e5
    m.tkin[:] = 11.0
    m.t_bg = 11.0
    m.density *= 30
    dvk, wk = np.array([-1.1e5, 0.2e5, 0.9e5]), np.array([0.25, 0.5, 0.25])
    m.species = _with_hfs(m.species, {0: (dvk, wk), 1: (0.5 * dvk, wk[::-1])})
    o = O.OSpecies(m.species)
    pops0 = O.lte(o, m.density, m.tkin, m.abundance)
    pops, _ = O.iterate(o, m, 1, pops=pops0.copy())
    assert np.max(np.abs(pops / pops0 - 1)) < 1e-11
    m.t_bg = 2.73
    m2 = copy.copy(m)
    m2.vrad = -m.vrad
    m2.species = _with_hfs(m.species, {0: (-dvk, wk), 1: (-0.5 * dvk, wk[::-1])})
    pa, _ = O.iterate(o, m, 2)
    pb, _ = O.iterate(O.OSpecies(m2.species), m2, 2)
    assert np.max(np.abs(pa / pb - 1)) < 1e-12
