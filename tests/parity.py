"""Helpers shared by the GPU parity tests: unit conversions between the oracle's photon counters and the
library's normalised counters (include/loc.h, loc_get_counters), and the comparison rules of DESIGN.md section 7."""
import numpy as np

import oracle as O

_C = 2.99792458e10
_H = 6.62607015e-27
_K = 1.380649e-16


def f32_pops_from_oracle_lte(sp, m):
    """LTE populations by the ORACLE, rounded to float32 by numpy: the common input of both sides.
    returns (pops64 [ncell][NL] holding the float32-rounded values, pops32 level-major [NL][ncell])"""
    p = O.lte(sp, m.density, m.tkin, m.abundance)
    p32 = np.ascontiguousarray(p.T.astype(np.float32))
    return np.ascontiguousarray(p32.T.astype(np.float64)), p32


def oracle_SJ_ESC(sp, m, res, sel):
    """oracle counters P, LAM -> the library's SJ, ESC ([ncell][nsel])
       SJ  = c^3 P / (8 pi nu^3 dv V_eff)   (so that S_lu = (g_u/g_l) A SJ, oracle O9)
       ESC = 1 - LAM                        (sum of ray weights per cell is exactly 1, pin P7)"""
    dv = 2.0 * m.band_half / m.nchannel
    out_sj = np.zeros((res["P"].shape[1], len(sel)))
    for k, t in enumerate(sel):
        nu = sp.freq(int(t))
        out_sj[:, k] = _C ** 3 * res["P"][k] / (8.0 * np.pi * nu ** 3 * dv * res["veff"])
    return out_sj, 1.0 - res["LAM"].T


def rel_err(a, ref, floor=0.0):
    a, ref = np.asarray(a, np.float64), np.asarray(ref, np.float64)
    return np.abs(a - ref) / np.maximum(np.abs(ref), floor if floor > 0 else 1e-300)


def tex_all(sp, pops, species):
    """T_ex [ncell][ntrans] from populations [ncell][NL] (oracle's definition O9, evaluated with numpy)"""
    e, g = np.asarray(species.energy_K), np.asarray(species.g)
    out = np.zeros((pops.shape[0], len(species.upper)))
    for t, (u, l) in enumerate(zip(species.upper, species.lower)):
        r = pops[:, u] * g[l] / (pops[:, l] * g[u])
        out[:, t] = -(e[u] - e[l]) / np.log(r)
    return out


def check_pops(gpu_pops_lm, ora_pops, tol=1e-3, floor=1e-10):
    """R20: relative tolerance on levels holding >= floor of the molecules, absolute 1e-13 of the total below."""
    g = np.asarray(gpu_pops_lm, np.float64).T
    tot = ora_pops.sum(axis=1, keepdims=True)
    ok_cells = tot[:, 0] > 0
    g, o, tot = g[ok_cells], ora_pops[ok_cells], tot[ok_cells]
    big = o >= floor * tot
    rel = np.abs(g - o) / np.maximum(o, 1e-300)
    worst = rel[big].max() if big.any() else 0.0
    small_abs = (np.abs(g - o) / tot)[~big].max() if (~big).any() else 0.0
    return worst, small_abs
