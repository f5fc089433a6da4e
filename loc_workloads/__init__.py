"""Seeded synthetic inputs for the LOC hot path (shared by the oracle tests, the CUDA tests and bench.py).

This module holds NONE of the method's arithmetic (no profiles, optical depths, transfer, rate
equations): it only manufactures inputs -- model clouds, an artificial linear rotor, ray
directions, octree hierarchies -- with the shapes and value ranges of the paper's workloads
("Input recipe").  The paper's own inputs (van Zadelhoff et al. 2002 benchmark
models, Padoan et al. 2016 MHD snapshots, LAMDA files) are not available
and are not reproduced.

All arrays handed to the oracle and to the CUDA library are the SAME float32 arrays.
Units: CGS (cm, cm/s, K, cm^-3).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

BASE_SEED = 200912609
PC = 3.0856775814913673e18  # cm
KMS = 1.0e5  # cm/s
# unit conversions needed to express the rotor in the interface's units (not method arithmetic)
_H = 6.62607015e-27
_K = 1.380649e-16
_C = 2.99792458e10
_DEBYE = 1.0e-18


def rng(config: int, stream: int) -> np.random.Generator:
    return np.random.default_rng([BASE_SEED, config, stream])


# ----------------------------------------------------------------------------------------------
# species
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Species:
    energy_K: np.ndarray  # [nlevel] float64
    g: np.ndarray  # [nlevel]
    upper: np.ndarray  # [ntrans] int32
    lower: np.ndarray  # [ntrans] int32
    einstein_A: np.ndarray  # [ntrans] float64
    mass_amu: float
    cu: np.ndarray  # [ncoll] int32
    cl: np.ndarray  # [ncoll] int32
    temps_K: np.ndarray  # [ntemp]
    rate_down: np.ndarray  # [ntemp][ncoll] cm^3/s
    # hyperfine structure with LTE between the components: {transition: (velocity offsets cm/s, weights summing to 1)}
    hfs: dict = dataclasses.field(default_factory=dict)

    @property
    def nlevel(self) -> int:
        return len(self.energy_K)

    @property
    def ntrans(self) -> int:
        return len(self.upper)


def rotor_species(nlevel: int, config: int = 0, B_GHz: float = 57.6, dipole_D: float = 0.11,
                  mass_amu: float = 28.0, rate_lo: float = 1e-11, rate_hi: float = 1e-10) -> Species:
    """Synthetic linear rotor of BASELINE.json: E_J = h B J(J+1), g = 2J+1, A from a 0.11 D dipole,
    downward collision rates log-uniform in [1e-11, 1e-10] cm^3/s for every pair u>l, T independent."""
    J = np.arange(nlevel, dtype=np.float64)
    B = B_GHz * 1e9
    energy_K = _H * B * J * (J + 1.0) / _K
    g = 2.0 * J + 1.0
    up = np.arange(1, nlevel, dtype=np.int32)
    lo = up - 1
    nu = 2.0 * B * up
    mu = dipole_D * _DEBYE
    A = 64.0 * math.pi ** 4 * nu ** 3 * mu ** 2 / (3.0 * _H * _C ** 3) * up / (2.0 * up + 1.0)
    cu, cl = [], []
    for u in range(1, nlevel):
        for l in range(u):
            cu.append(u)
            cl.append(l)
    r = rng(config, 1)
    rates = 10.0 ** r.uniform(math.log10(rate_lo), math.log10(rate_hi), size=len(cu))
    return Species(energy_K, g, up, lo, A, mass_amu, np.array(cu, np.int32), np.array(cl, np.int32),
                   np.array([10.0]), rates[None, :].copy())


# ----------------------------------------------------------------------------------------------
# directions (HEALPix ring-scheme pixel centres, Gorski et al. 2005)
# ----------------------------------------------------------------------------------------------
def healpix_dirs(nside: int) -> np.ndarray:
    npix = 12 * nside * nside
    out = np.zeros((npix, 3))
    ncap = 2 * nside * (nside - 1)
    for p in range(npix):
        if p < ncap:
            ph = (p + 1) / 2.0
            i = int(math.floor(math.sqrt(ph - math.sqrt(math.floor(ph))))) + 1
            j = p + 1 - 2 * i * (i - 1)
            z = 1.0 - i * i / (3.0 * nside * nside)
            phi = (j - 0.5) * math.pi / (2.0 * i)
        elif p < npix - ncap:
            pp = p - ncap
            i = pp // (4 * nside) + nside
            j = pp % (4 * nside) + 1
            z = 4.0 / 3.0 - 2.0 * i / (3.0 * nside)
            s = (i - nside + 1) % 2
            phi = (j - s / 2.0) * math.pi / (2.0 * nside)
        else:
            ps = npix - p
            ph = ps / 2.0
            i = int(math.floor(math.sqrt(ph - math.sqrt(math.floor(ph))))) + 1
            j = 4 * i + 1 - (ps - 2 * i * (i - 1))
            z = -1.0 + i * i / (3.0 * nside * nside)
            phi = (j - 0.5) * math.pi / (2.0 * i)
        st = math.sqrt(max(0.0, 1.0 - z * z))
        out[p] = (st * math.cos(phi), st * math.sin(phi), z)
    return out


# ----------------------------------------------------------------------------------------------
# 1D shell models (configs C1, C2)
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class ShellModel:
    r_out: np.ndarray  # [ns] float64 outer radii, cm
    density: np.ndarray  # float32 [ns]
    tkin: np.ndarray
    sigma: np.ndarray  # turbulent 1-D std dev, cm/s
    vrad: np.ndarray
    abundance: np.ndarray
    ray_p: np.ndarray  # [nray] float64 impact parameters
    ray_w: np.ndarray  # [nray] float64 annulus areas
    nchannel: int
    band_half: float  # cm/s
    t_bg: float
    species: Species
    niter: int
    name: str = ""


def shell_rays(r_out: np.ndarray, nsub: int):
    """Each shell's annulus split into nsub equal-width sub-annuli (R15)."""
    r_in = np.concatenate([[0.0], r_out[:-1]])
    p, w = [], []
    for a, b in zip(r_in, r_out):
        edges = np.linspace(a, b, nsub + 1)
        for lo, hi in zip(edges[:-1], edges[1:]):
            p.append(math.sqrt(0.5 * (lo * lo + hi * hi)))
            w.append(math.pi * (hi * hi - lo * lo))
    return np.array(p), np.array(w)


def shell_config(which: int, ns: int | None = None, nchannel: int | None = None, nsub: int | None = None,
                 nlevel: int | None = None) -> ShellModel:
    """C1 / C2 of BASELINE.json (optionally shrunk for tests via ns/nchannel/nsub/nlevel)."""
    if which == 1:
        ns = ns or 64
        r0, R = 1e-3 * PC, 0.1 * PC
        r = r0 * (R / r0) ** (np.arange(ns) / (ns - 1.0))
        rin = np.concatenate([[0.0], r[:-1]])
        rm = 0.5 * (rin + r)
        dens = 1e4 / (1.0 + (rm / (0.02 * PC)) ** 2)
        tk = np.full(ns, 10.0)
        sig = np.full(ns, 0.2 * KMS)
        v = -0.1 * KMS * rm / R
        sp = rotor_species(nlevel or 5, 1)
        nch, nsub_, niter = nchannel or 64, nsub or 1, 20
    elif which == 2:
        ns = ns or 1000
        r0, R = 1e-4 * PC, 0.1 * PC
        r = r0 * (R / r0) ** (np.arange(ns) / (ns - 1.0))
        rin = np.concatenate([[0.0], r[:-1]])
        rm = 0.5 * (rin + r)
        dens = 1e6 / (1.0 + (rm / (0.005 * PC)) ** 2)
        tk = 8.0 + 7.0 * rm / R
        sig = np.full(ns, 0.15 * KMS)
        v = -0.3 * KMS * np.sqrt(0.005 * PC / np.maximum(rm, 0.005 * PC))
        sp = rotor_species(nlevel or 10, 2)
        nch, nsub_, niter = nchannel or 256, nsub or 4, 50
    else:
        raise ValueError(which)
    p, w = shell_rays(r, nsub_)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return ShellModel(r, f32(dens), f32(tk), f32(sig), f32(v), f32(np.full(ns, 1e-4)), p, w, nch, 2.0 * KMS, 2.73, sp,
                      niter, f"C{which}")


# ----------------------------------------------------------------------------------------------
# 3D octree models (configs C3, C4, C5)
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class OctreeModel:
    nx: int
    ny: int
    nz: int
    nlev: int
    noff: np.ndarray  # int64 [nlev+1]
    child: np.ndarray  # int32 [ncell]; first child within next level or -1 (level-major, R17)
    root_cm: float
    density: np.ndarray  # float32 [ncell] (all cells, leaves and refined)
    tkin: np.ndarray
    sigma: np.ndarray
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray
    abundance: np.ndarray
    coords: np.ndarray  # int32 [ncell][3] cell index (x,y,z) at the cell's own level (harness use only)
    level: np.ndarray  # int8 [ncell]
    dirs: np.ndarray  # [ndir][3]
    nchannel: int
    band_half: float
    t_bg: float
    species: Species
    niter: int
    sel: np.ndarray | None = None  # transitions that are ray traced (None = all)
    name: str = ""

    @property
    def ncell(self) -> int:
        return int(self.noff[-1])

    @property
    def nleaf(self) -> int:
        return int((self.child < 0).sum())


def gaussian_field(n: int, slope: float, gen: np.random.Generator, dtype=np.float32) -> np.ndarray:
    """Zero-mean unit-variance periodic Gaussian random field on n^3 with power spectrum P(k) ~ k^slope."""
    white = gen.standard_normal((n, n, n), dtype=np.float32)
    fk = np.fft.rfftn(white)
    del white
    kx = np.fft.fftfreq(n) * n
    kz = np.fft.rfftfreq(n) * n
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    fk *= k2 ** (slope / 4.0)
    fk[0, 0, 0] = 0.0
    f = np.fft.irfftn(fk, s=(n, n, n), axes=(0, 1, 2)).astype(dtype)
    f -= f.mean()
    f /= f.std()
    return f


def _coarsen(a: np.ndarray, w: np.ndarray | None = None) -> np.ndarray:
    n = a.shape[0] // 2
    if w is None:
        return a.reshape(n, 2, n, 2, n, 2).mean(axis=(1, 3, 5))
    return (a * w).reshape(n, 2, n, 2, n, 2).sum(axis=(1, 3, 5)) / w.reshape(n, 2, n, 2, n, 2).sum(axis=(1, 3, 5))


def build_octree(fields: dict, nroot: int, nlev: int, refine_frac) -> dict:
    """Level-major octree (R17) from fields given at the finest resolution (nroot * 2^(nlev-1))^3, arrays [z][y][x].

    Density is averaged upward (mean of 8 children), velocities density-weighted; at every
    level the densest `refine_frac[l]` of the existing cells are refined (R16).
    """
    if np.isscalar(refine_frac):
        refine_frac = [refine_frac] * (nlev - 1)
    pyr = [None] * nlev
    cur = {k: v for k, v in fields.items()}
    for l in range(nlev - 1, -1, -1):
        pyr[l] = cur
        if l > 0:
            d = cur["density"].astype(np.float64)
            nxt = {"density": _coarsen(d)}
            for k in cur:
                if k == "density":
                    continue
                nxt[k] = _coarsen(cur[k].astype(np.float64), d if k in ("vx", "vy", "vz") else None)
            cur = nxt
    # level 0: raster, x fastest
    n0 = nroot
    iz, iy, ix = np.meshgrid(np.arange(n0), np.arange(n0), np.arange(n0), indexing="ij")
    coords = [np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.int32)]
    childs = []
    for l in range(nlev):
        c = coords[l]
        dens = pyr[l]["density"][c[:, 2], c[:, 1], c[:, 0]]
        ch = np.full(len(c), -1, np.int32)
        if l < nlev - 1 and refine_frac[l] > 0:
            nref = int(round(refine_frac[l] * len(c)))
            if nref > 0:
                thr = np.partition(dens, len(c) - nref)[len(c) - nref]
                refined = np.flatnonzero(dens >= thr)[:]
                if len(refined) > nref:  # ties: keep the first nref in cell order
                    refined = refined[:nref]
                ch[refined] = 8 * np.arange(len(refined), dtype=np.int32)
                par = c[refined]
                oct_ = np.array([[cx, cy, cz] for cz in (0, 1) for cy in (0, 1) for cx in (0, 1)], np.int32)
                coords.append((2 * par[:, None, :] + oct_[None, :, :]).reshape(-1, 3))
            else:
                coords.append(np.zeros((0, 3), np.int32))
        elif l < nlev - 1:
            coords.append(np.zeros((0, 3), np.int32))
        childs.append(ch)
    # drop empty trailing levels
    while len(coords) > 1 and len(coords[-1]) == 0:
        coords.pop()
    nlev_eff = len(coords)
    childs = childs[:nlev_eff]
    noff = np.zeros(nlev_eff + 1, np.int64)
    for l in range(nlev_eff):
        noff[l + 1] = noff[l] + len(coords[l])
    out = {"nlev": nlev_eff, "noff": noff, "child": np.concatenate(childs),
           "coords": np.concatenate(coords), "level": np.concatenate(
               [np.full(len(coords[l]), l, np.int8) for l in range(nlev_eff)])}
    for k in fields:
        out[k] = np.concatenate([pyr[l][k][coords[l][:, 2], coords[l][:, 1], coords[l][:, 0]] for l in range(nlev_eff)]
                                ).astype(np.float32)
    return out


# ---- the same recipe on torch (CUDA when there is one): full-size C4 / C5 only ---------------------------------
# numpy needs minutes for the 512^3 / 1024^3 fields (complex128 FFTs, fancy indexing over 2e8 cells); the white noise still
# comes from the seeded numpy generator, so the realisation does not depend on the machine beyond the rounding of the FFT.
TORCH_FROM_NFINE = 512


def _torch_device():
    import torch
    return torch.device("cuda", torch.cuda.current_device()) if torch.cuda.is_available() else torch.device("cpu")


def gaussian_field_t(n: int, slope: float, gen: np.random.Generator, device):
    """gaussian_field() with the FFTs and the filter on `device` in float32 / complex64; returns a torch tensor [z][y][x]"""
    import torch
    white = torch.from_numpy(gen.standard_normal((n, n, n), dtype=np.float32)).to(device)
    fk = torch.fft.rfftn(white)
    del white
    kx = torch.fft.fftfreq(n, device=device) * n
    kz = torch.fft.rfftfreq(n, device=device) * n
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    fk *= k2 ** (slope / 4.0)
    del k2
    fk[0, 0, 0] = 0.0
    f = torch.fft.irfftn(fk, s=(n, n, n))
    del fk
    f -= f.mean()
    f /= f.std(unbiased=False)
    return f


def build_octree_t(fields: dict, nroot: int, nlev: int, refine_frac, device) -> dict:
    """build_octree() on torch tensors (same rules, same array layout); returns numpy arrays"""
    import torch
    if np.isscalar(refine_frac):
        refine_frac = [refine_frac] * (nlev - 1)

    def coarsen(a, w=None):
        n = a.shape[0] // 2
        if w is None:
            return a.reshape(n, 2, n, 2, n, 2).mean(dim=(1, 3, 5))
        return (a * w).reshape(n, 2, n, 2, n, 2).sum(dim=(1, 3, 5)) / w.reshape(n, 2, n, 2, n, 2).sum(dim=(1, 3, 5))

    pyr = [None] * nlev
    cur = dict(fields)
    for l in range(nlev - 1, -1, -1):
        pyr[l] = cur
        if l > 0:
            d = cur["density"].double()
            nxt = {"density": coarsen(d)}
            for k in cur:
                if k != "density":
                    nxt[k] = coarsen(cur[k].double(), d if k in ("vx", "vy", "vz") else None)
            del d
            cur = nxt
    r = torch.arange(nroot, device=device, dtype=torch.int32)
    iz, iy, ix = torch.meshgrid(r, r, r, indexing="ij")
    coords = [torch.stack([ix.reshape(-1), iy.reshape(-1), iz.reshape(-1)], dim=1)]
    oct_ = torch.tensor([[cx, cy, cz] for cz in (0, 1) for cy in (0, 1) for cx in (0, 1)], dtype=torch.int32, device=device)
    childs = []
    for l in range(nlev):
        c = coords[l]
        nc = c.shape[0]
        ch = torch.full((nc,), -1, dtype=torch.int32, device=device)
        if l < nlev - 1:
            nref = int(round(refine_frac[l] * nc)) if refine_frac[l] > 0 else 0
            if nref > 0:
                dens = pyr[l]["density"][c[:, 2].long(), c[:, 1].long(), c[:, 0].long()]
                thr = torch.kthvalue(dens, nc - nref + 1).values
                refined = torch.nonzero(dens >= thr).reshape(-1)[:nref]  # ties: the first nref in cell order
                del dens
                ch[refined] = 8 * torch.arange(refined.shape[0], dtype=torch.int32, device=device)
                coords.append((2 * c[refined][:, None, :] + oct_[None, :, :]).reshape(-1, 3))
            else:
                coords.append(torch.zeros((0, 3), dtype=torch.int32, device=device))
        childs.append(ch)
    while len(coords) > 1 and coords[-1].shape[0] == 0:
        coords.pop()
    nlev_eff = len(coords)
    childs = childs[:nlev_eff]
    noff = np.zeros(nlev_eff + 1, np.int64)
    for l in range(nlev_eff):
        noff[l + 1] = noff[l] + coords[l].shape[0]
    out = {"nlev": nlev_eff, "noff": noff, "child": torch.cat(childs).cpu().numpy(),
           "level": np.concatenate([np.full(coords[l].shape[0], l, np.int8) for l in range(nlev_eff)])}
    idx = [(coords[l][:, 2].long(), coords[l][:, 1].long(), coords[l][:, 0].long()) for l in range(nlev_eff)]
    for k in fields:
        out[k] = torch.cat([pyr[l][k][idx[l]].float() for l in range(nlev_eff)]).cpu().numpy()
    del idx
    out["coords"] = torch.cat(coords).cpu().numpy()
    return out


def cloud_config(which: int, nroot: int | None = None, nlev: int | None = None, nchannel: int | None = None,
                 nside: int | None = None, refine_frac=None, nlevel_species: int | None = None,
                 seed_config: int | None = None) -> OctreeModel:
    """C3 / C4 / C5 of BASELINE.json, optionally shrunk (nroot, nlev, nchannel, nside) for tests.

    C3: 128^3 root only.  C4: root 64^3 + 3 levels.  C5: root 256^3 + 2 levels, 3 transitions traced.
    Readings R14 (bandwidths, sigma_turb, 3-D rms) and R16 (refined fraction instead of a 4x threshold).
    """
    cfg = {3: dict(nroot=128, nlev=1, nch=128, band=4.0, nside=2, sln=1.5, vrms=1.0, cell_pc=0.02, frac=0.0, niter=10),
           4: dict(nroot=64, nlev=4, nch=128, band=4.0, nside=2, sln=1.5, vrms=1.0, cell_pc=0.04, frac=0.60, niter=10),
           5: dict(nroot=256, nlev=3, nch=256, band=8.0, nside=1, sln=2.0, vrms=2.0, cell_pc=0.04, frac=0.38, niter=5)}[which]
    nroot = nroot or cfg["nroot"]
    nlev = nlev or cfg["nlev"]
    nch = nchannel or cfg["nch"]
    nside = nside or cfg["nside"]
    frac = cfg["frac"] if refine_frac is None else refine_frac
    sc = seed_config if seed_config is not None else which
    nfine = nroot * 2 ** (nlev - 1)
    sln = cfg["sln"]
    s1 = cfg["vrms"] * KMS / math.sqrt(3.0)
    if nfine >= TORCH_FROM_NFINE:
        import torch
        dev = _torch_device()
        g = gaussian_field_t(nfine, -11.0 / 3.0, rng(sc, 2), dev)
        fields = {"density": 1e3 * torch.exp(sln * g - 0.5 * sln * sln)}
        del g
        for k, st in (("vx", 3), ("vy", 4), ("vz", 5)):
            fields[k] = torch.clamp(gaussian_field_t(nfine, -11.0 / 3.0, rng(sc, st), dev) * s1, -5 * s1, 5 * s1)
        if which == 4:
            fields["tkin"] = torch.from_numpy(rng(sc, 6).uniform(10.0, 20.0, size=(nfine,) * 3).astype(np.float32)).to(dev)
        else:
            fields["tkin"] = torch.full((nfine,) * 3, 10.0, dtype=torch.float32, device=dev)
        tree = build_octree_t(fields, nroot, nlev, frac, dev)
        del fields
        if dev.type == "cuda":
            torch.cuda.empty_cache()
    else:
        g = gaussian_field(nfine, -11.0 / 3.0, rng(sc, 2))
        dens = (1e3 * np.exp(sln * g - 0.5 * sln * sln)).astype(np.float32)
        del g
        fields = {"density": dens}
        for k, st in (("vx", 3), ("vy", 4), ("vz", 5)):
            fields[k] = np.clip(gaussian_field(nfine, -11.0 / 3.0, rng(sc, st)) * s1, -5 * s1, 5 * s1).astype(np.float32)
        if which == 4:
            fields["tkin"] = rng(sc, 6).uniform(10.0, 20.0, size=(nfine,) * 3).astype(np.float32)
        else:
            fields["tkin"] = np.full((nfine,) * 3, 10.0, np.float32)
        tree = build_octree(fields, nroot, nlev, frac)
    ncell = int(tree["noff"][-1])
    sp = rotor_species(nlevel_species or 10, sc)
    sel = np.array([0, 1, 2], np.int32) if which == 5 else None
    return OctreeModel(nroot, nroot, nroot, tree["nlev"], tree["noff"], tree["child"], cfg["cell_pc"] * PC,
                       tree["density"], tree["tkin"], np.full(ncell, 0.2 * KMS, np.float32), tree["vx"], tree["vy"],
                       tree["vz"], np.full(ncell, 1e-4, np.float32), tree["coords"], tree["level"],
                       healpix_dirs(nside), nch, cfg["band"] * KMS, 2.73, sp, cfg["niter"], sel, f"C{which}")


def uniform_octree(nroot, nlev_full: int, root_cm: float, density, tkin, sigma, v, abundance, species, dirs, nchannel,
                   band_half, t_bg) -> OctreeModel:
    """Grid with every cell refined (nlev_full-1) times and constant values (test helper for pins P4, P10)."""
    nfine = nroot * 2 ** (nlev_full - 1)
    fields = {"density": np.full((nfine,) * 3, density, np.float32), "tkin": np.full((nfine,) * 3, tkin, np.float32),
              "vx": np.full((nfine,) * 3, v[0], np.float32), "vy": np.full((nfine,) * 3, v[1], np.float32),
              "vz": np.full((nfine,) * 3, v[2], np.float32)}
    tree = build_octree(fields, nroot, nlev_full, 1.0)
    ncell = int(tree["noff"][-1])
    return OctreeModel(nroot, nroot, nroot, tree["nlev"], tree["noff"], tree["child"], root_cm, tree["density"],
                       tree["tkin"], np.full(ncell, sigma, np.float32), tree["vx"], tree["vy"], tree["vz"],
                       np.full(ncell, abundance, np.float32), tree["coords"], tree["level"], np.asarray(dirs, float),
                       nchannel, band_half, t_bg, species, 1, None, "uniform")
