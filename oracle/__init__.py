"""ctypes front end of the float64 CPU oracle (oracle/loc_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package (paper_2009_12609_b200) never imports this module, and this
module never imports the product package.  Argument marshalling only; all arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "loc_oracle.c")

LEDGER = ("injected", "emitted", "created", "absorbed", "selfabs", "escaped", "terminated", "rescale")


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"])
    return _SO


class _Species(C.Structure):
    _fields_ = [("nlevel", C.c_int), ("energy_K", C.c_void_p), ("g", C.c_void_p), ("ntrans", C.c_int),
                ("upper", C.c_void_p), ("lower", C.c_void_p), ("A", C.c_void_p), ("mass_amu", C.c_double),
                ("ncoll", C.c_int), ("cu", C.c_void_p), ("cl", C.c_void_p), ("ntemp", C.c_int),
                ("temps_K", C.c_void_p), ("rate_down", C.c_void_p), ("hf_off", C.c_void_p), ("hf_dv", C.c_void_p),
                ("hf_w", C.c_void_p)]


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("nlev", C.c_int), ("noff", C.c_void_p),
                ("child", C.c_void_p), ("root_cm", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_planck.restype = C.c_double
        _lib.orc_planck.argtypes = [C.c_double, C.c_double]
        _lib.orc_freq.restype = C.c_double
        _lib.orc_solve.restype = C.c_double
        _lib.orc_solve_sub.restype = C.c_double
        _lib.orc_tex.restype = C.c_double
    return _lib


def set_threads(n: int):
    os.environ["OMP_NUM_THREADS"] = str(n)
    try:
        omp = C.CDLL("libgomp.so.1")
        omp.omp_set_num_threads(int(n))
    except OSError:
        pass


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class OSpecies:
    """Holds contiguous arrays alive and the C struct that points at them."""

    def __init__(self, sp):
        self.e = _f64(sp.energy_K)
        self.g = _f64(sp.g)
        self.up = np.ascontiguousarray(sp.upper, np.int32)
        self.lo = np.ascontiguousarray(sp.lower, np.int32)
        self.A = _f64(sp.einstein_A)
        self.cu = np.ascontiguousarray(sp.cu, np.int32)
        self.cl = np.ascontiguousarray(sp.cl, np.int32)
        self.temps = _f64(sp.temps_K)
        self.rates = _f64(sp.rate_down)
        self.nlevel, self.ntrans = len(self.e), len(self.up)
        # hyperfine structure: sp.hfs = {transition: (offsets cm/s, weights)} (loc_workloads.Species), optional
        hfs = getattr(sp, "hfs", None) or {}
        if hfs:
            off = np.zeros(self.ntrans + 1, np.int32)
            dv, w = [], []
            for t in range(self.ntrans):
                if t in hfs:
                    dv += list(np.asarray(hfs[t][0], np.float64))
                    w += list(np.asarray(hfs[t][1], np.float64))
                off[t + 1] = len(dv)
            self.hf_off, self.hf_dv, self.hf_w = off, _f64(dv), _f64(w)
            hf = (_p(self.hf_off), _p(self.hf_dv), _p(self.hf_w))
        else:
            hf = (None, None, None)
        self.c = _Species(self.nlevel, _p(self.e), _p(self.g), self.ntrans, _p(self.up), _p(self.lo), _p(self.A),
                          float(sp.mass_amu), len(self.cu), _p(self.cu), _p(self.cl), len(self.temps), _p(self.temps),
                          _p(self.rates), *hf)

    def ref(self):
        return C.byref(self.c)

    def freq(self, t):
        return lib().orc_freq(self.ref(), C.c_int(t))


class OGrid:
    def __init__(self, m):
        self.noff = np.ascontiguousarray(m.noff, np.int64)
        self.child = np.ascontiguousarray(m.child, np.int32)
        self.c = _Grid(m.nx, m.ny, m.nz, int(m.nlev), _p(self.noff), _p(self.child), float(m.root_cm))
        self.ncell = int(self.noff[-1])

    def ref(self):
        return C.byref(self.c)


def planck(nu, T):
    return lib().orc_planck(float(nu), float(T))


def lte(sp: OSpecies, density, tkin, abundance):
    n = len(density)
    pops = np.zeros((n, sp.nlevel))
    d, t, a = _f64(density), _f64(tkin), _f64(abundance)
    lib().orc_lte(sp.ref(), C.c_int64(n), _p(d), _p(t), _p(a), _p(pops))
    return pops


def rate_matrix(sp: OSpecies, n, T, S, beta):
    R = np.zeros((sp.nlevel, sp.nlevel))
    S, beta = _f64(S), _f64(beta)
    lib().orc_rate_matrix(sp.ref(), C.c_double(n), C.c_double(T), _p(S), _p(beta), _p(R))
    return R


def solve_rates(R, ntot, method="ge"):
    NL = R.shape[0]
    x = np.zeros(NL)
    R = _f64(R)
    fn = lib().orc_solve_rates if method == "ge" else lib().orc_solve_gth
    rc = fn(C.c_int(NL), _p(R), C.c_double(ntot), _p(x))
    assert rc == 0, rc
    return x


def solve(sp: OSpecies, density, tkin, abundance, veff, sel, P, LAM, dv, tbg, pops, ali=True):
    """O9 over all cells; updates pops in place ([ncell][NL]); returns max relative change."""
    n = len(density)
    d, t, a, v = _f64(density), _f64(tkin), _f64(abundance), _f64(veff)
    sel = np.ascontiguousarray(sel, np.int32)
    P, LAM = _f64(P), _f64(LAM)
    assert pops.dtype == np.float64 and pops.flags.c_contiguous
    return lib().orc_solve(sp.ref(), C.c_int64(n), _p(d), _p(t), _p(a), _p(v), C.c_int(len(sel)), _p(sel), _p(P), _p(LAM),
                           C.c_double(dv), C.c_double(tbg), C.c_int(int(ali)), _p(pops))


def solve_sub(sp: OSpecies, density, tkin, abundance, veff, sel, P, LAM, dv, tbg, pops, nsub):
    """O9 with nsub sub-iterations between two ray passes (R26); nsub = 1 is solve()."""
    n = len(density)
    d, t, a, v = _f64(density), _f64(tkin), _f64(abundance), _f64(veff)
    sel = np.ascontiguousarray(sel, np.int32)
    P, LAM = _f64(P), _f64(LAM)
    assert pops.dtype == np.float64 and pops.flags.c_contiguous
    return lib().orc_solve_sub(sp.ref(), C.c_int64(n), _p(d), _p(t), _p(a), _p(v), C.c_int(len(sel)), _p(sel), _p(P), _p(LAM),
                               C.c_double(dv), C.c_double(tbg), C.c_int(int(nsub)), _p(pops))


def tex(sp: OSpecies, t, n_u, n_l):
    return lib().orc_tex(sp.ref(), C.c_int(t), C.c_double(n_u), C.c_double(n_l))


def veff_1d(r, p, w):
    r, p, w = _f64(r), _f64(p), _f64(w)
    v = np.zeros(len(r))
    lib().orc_veff_1d(C.c_int(len(r)), _p(r), C.c_int(len(p)), _p(p), _p(w), _p(v))
    return v


def path_1d(r, p):
    r = _f64(r)
    ns = len(r)
    sh = np.zeros(2 * ns, np.int32)
    s = np.zeros(2 * ns)
    mu = np.zeros(2 * ns)
    n = lib().orc_path_1d(C.c_int(ns), _p(r), C.c_double(p), _p(sh), _p(s), _p(mu))
    return sh[:n], s[:n], mu[:n]


def sim_1d(sp: OSpecies, m, pops, sel=None, ali=True, want_nout=False):
    """m: loc_workloads.ShellModel (float32 arrays converted to double here).  Returns dict."""
    ns, nray = len(m.r_out), len(m.ray_p)
    sel = np.arange(sp.ntrans, dtype=np.int32) if sel is None else np.ascontiguousarray(sel, np.int32)
    nsel = len(sel)
    r, tk, sg, vr = _f64(m.r_out), _f64(m.tkin), _f64(m.sigma), _f64(m.vrad)
    p, w = _f64(m.ray_p), _f64(m.ray_w)
    pops = _f64(pops)
    ABS, P, LAM = np.zeros((nsel, ns)), np.zeros((nsel, ns)), np.zeros((nsel, ns))
    visits = np.zeros(ns, np.int64)
    ledger = np.zeros(len(LEDGER))
    nout = np.zeros((nray, nsel, m.nchannel)) if want_nout else None
    lib().orc_sim_1d(sp.ref(), C.c_int(ns), _p(r), _p(tk), _p(sg), _p(vr), C.c_int(nray), _p(p), _p(w), _p(pops),
                     C.c_int(m.nchannel), C.c_double(m.band_half), C.c_double(m.t_bg), C.c_int(nsel), _p(sel),
                     C.c_int(int(ali)), _p(ABS), _p(P), _p(LAM), _p(visits), _p(ledger),
                     _p(nout) if want_nout else None)
    return dict(ABS=ABS, P=P, LAM=LAM, visits=visits, ledger=dict(zip(LEDGER, ledger)), nout=nout,
                veff=veff_1d(r, p, w))


def spectra_1d(sp: OSpecies, m, pops, t, b):
    r, tk, sg, vr = _f64(m.r_out), _f64(m.tkin), _f64(m.sigma), _f64(m.vrad)
    b = _f64(b)
    pops = _f64(pops)
    TA = np.zeros((len(b), m.nchannel))
    lib().orc_spectra_1d(sp.ref(), C.c_int(len(r)), _p(r), _p(tk), _p(sg), _p(vr), _p(pops), C.c_int(m.nchannel),
                         C.c_double(m.band_half), C.c_double(m.t_bg), C.c_int(t), C.c_int(len(b)), _p(b), _p(TA))
    return TA


def line_area(TA, dv_cm_s):
    """Line-area map (Fig. 5c): W = sum over channels of T_A dv, K km/s; the definition written out in
    float64.  TA [..., nchannel] in K, dv in cm/s."""
    return np.asarray(TA, np.float64).sum(axis=-1) * (float(dv_cm_s) * 1e-5)


def sim_3d(sp: OSpecies, m, pops, sel=None, ali=True, geom_only=False, dirs=None, off64=(25, 41), root_stride=1):
    """m: loc_workloads.OctreeModel.  pops [ncell][NL] float64.  Returns dict of counters.
    root_stride > 1: a bounded TIMING sample for bench.py (every root_stride-th line of the root lattice only); its
    counters are incomplete and must not be compared with anything."""
    G = OGrid(m)
    n = G.ncell
    sel = np.arange(sp.ntrans, dtype=np.int32) if sel is None else np.ascontiguousarray(sel, np.int32)
    nsel = len(sel)
    dirs = _f64(m.dirs if dirs is None else dirs).reshape(-1, 3)
    tk, sg, vx, vy, vz = _f64(m.tkin), _f64(m.sigma), _f64(m.vx), _f64(m.vy), _f64(m.vz)
    pops = _f64(pops) if pops is not None else np.zeros((n, sp.nlevel))
    ABS, P, LAM = np.zeros((nsel, n)), np.zeros((nsel, n)), np.zeros((nsel, n))
    visits, pathz = np.zeros(n, np.int64), np.zeros(n, np.int64)
    ledger = np.zeros(len(LEDGER))
    off = np.array(off64, np.int32)
    lib().orc_sim_3d(sp.ref(), G.ref(), _p(tk), _p(sg), _p(vx), _p(vy), _p(vz), _p(pops), C.c_int(m.nchannel),
                     C.c_double(m.band_half), C.c_double(m.t_bg), C.c_int(len(dirs)), _p(dirs), C.c_int(nsel), _p(sel),
                     C.c_int(int(ali)), C.c_int(int(geom_only)), _p(off), _p(ABS), _p(P), _p(LAM), _p(visits), _p(pathz),
                     _p(ledger), C.c_int(int(root_stride)))
    lev = np.asarray(m.level, np.int64)
    veff = (m.root_cm / 2.0 ** lev) ** 3
    return dict(ABS=ABS, P=P, LAM=LAM, visits=visits, pathz=pathz, ledger=dict(zip(LEDGER, ledger)), veff=veff)


def leaf_visits(m, d, leaf_org_model, level):
    G = OGrid(m)
    d = _f64(d)
    org = np.ascontiguousarray(leaf_org_model, np.int64)
    nv, pz = C.c_int64(0), C.c_int64(0)
    lib().orc_leaf_visits(G.ref(), _p(d), _p(org), C.c_int(int(level)), C.byref(nv), C.byref(pz))
    return nv.value, pz.value


def line_position(d, nx, ny, nz, bp, bq, zeta):
    d = _f64(d)
    xp, xq = C.c_int64(0), C.c_int64(0)
    lib().orc_line_position(_p(d), C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int64(bp), C.c_int64(bq), C.c_int64(zeta),
                            C.byref(xp), C.byref(xq))
    return xp.value, xq.value


def spectra_3d(sp: OSpecies, m, pops, t, d, npx, npy, aff):
    G = OGrid(m)
    d = _f64(d)
    aff = np.ascontiguousarray(aff, np.int64)
    tk, sg, vx, vy, vz = _f64(m.tkin), _f64(m.sigma), _f64(m.vx), _f64(m.vy), _f64(m.vz)
    pops = _f64(pops)
    TA = np.zeros((npy, npx, m.nchannel))
    lib().orc_spectra_3d(sp.ref(), G.ref(), _p(tk), _p(sg), _p(vx), _p(vy), _p(vz), _p(pops), C.c_int(m.nchannel),
                         C.c_double(m.band_half), C.c_double(m.t_bg), C.c_int(t), _p(d), C.c_int(npx), C.c_int(npy),
                         _p(aff), _p(TA))
    return TA


def slab(sp: OSpecies, t, nch, band_half, tbg, a, veff_each, s, sigma, v0, n_u, n_l, ali=True, N=None):
    s = _f64(s)
    inject = N is None
    N = np.zeros(nch) if N is None else _f64(N).copy()
    acc = np.zeros(3)
    ledger = np.zeros(len(LEDGER))
    lib().orc_slab(sp.ref(), C.c_int(t), C.c_int(nch), C.c_double(band_half), C.c_double(tbg), C.c_double(a),
                   C.c_double(veff_each), C.c_int(len(s)), _p(s), C.c_double(sigma), C.c_double(v0), C.c_double(n_u),
                   C.c_double(n_l), C.c_int(int(ali)), _p(N), _p(acc), _p(ledger), C.c_int(int(inject)))
    return N, acc, dict(zip(LEDGER, ledger))


def profile(nch, dv, sigma, v0):
    phi = np.zeros(nch)
    lib().orc_profile(C.c_int(nch), C.c_double(dv), C.c_double(sigma), C.c_double(v0), _p(phi))
    return phi


def profile_t(sp: OSpecies, t, nch, dv, sigma, v0):
    """profile of transition t including its hyperfine components"""
    phi = np.zeros(nch)
    lib().orc_profile_t(sp.ref(), C.c_int(t), C.c_int(nch), C.c_double(dv), C.c_double(sigma), C.c_double(v0), _p(phi))
    return phi


def iterate(sp: OSpecies, m, niter, sel=None, ali=True, pops=None, history=False, nsub=1):
    """O10: niter x (simulate all selected transitions from the old populations; solve) from LTE (O3).
    nsub > 1: sub-iterations of the solve between the ray passes (solve_sub; ALI only)."""
    is3d = hasattr(m, "child")
    dens, tk, ab = _f64(m.density), _f64(m.tkin), _f64(m.abundance)
    if pops is None:
        pops = lte(sp, dens, tk, ab)
    sel_arr = np.arange(sp.ntrans, dtype=np.int32) if sel is None else np.ascontiguousarray(sel, np.int32)
    dv = 2.0 * m.band_half / m.nchannel
    changes, last = [], None
    for _ in range(niter):
        r = sim_3d(sp, m, pops, sel_arr, ali) if is3d else sim_1d(sp, m, pops, sel_arr, ali)
        last = r
        if nsub > 1:
            assert ali
            changes.append(solve_sub(sp, dens, tk, ab, r["veff"], sel_arr, r["P"], r["LAM"], dv, m.t_bg, pops, nsub))
        else:
            changes.append(solve(sp, dens, tk, ab, r["veff"], sel_arr, r["P"], r["LAM"], dv, m.t_bg, pops, ali))
    return (pops, changes, last) if history else (pops, changes[-1] if changes else 0.0)
