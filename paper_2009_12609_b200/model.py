"""LocModel: owns the device buffers (PyTorch tensors) of one model and forwards to the C-ABI binding.

No arithmetic of the method lives here: tensors are allocated / copied with PyTorch and handed to the library as raw
pointers; results come back as views of the library's workspace.
"""
from __future__ import annotations

import contextlib
import ctypes as C

import numpy as np
import torch

from . import binding as B


def _as_tensor_view(ptr: int, nbytes: int, owner: torch.Tensor, dtype):
    """view [ptr, ptr+nbytes) of the uint8 workspace tensor `owner` as dtype"""
    off = ptr - owner.data_ptr()
    assert 0 <= off and off + nbytes <= owner.numel(), "pointer outside the workspace"
    return owner[off:off + nbytes].view(dtype)


class LocModel:
    """device-resident model.  `m` is a duck-typed description:
       shells : r_out, ray_p, ray_w, density, tkin, sigma, vrad, abundance, nchannel, band_half, t_bg, species
       octree : nx, ny, nz, root_cm, noff, child, density, tkin, sigma, vx, vy, vz, abundance, dirs, nchannel, ...
    Host arrays may be numpy arrays or (pinned) torch CPU tensors; they are copied to `device` on `stream`.
    stream: the torch.cuda.Stream the library enqueues on (None: torch's current stream at construction).  Every tensor
    operation of this class (uploads, allocations, copies) runs inside `torch.cuda.stream(self.stream)`, so the copies are
    ordered with the library's kernels and the caching allocator ties the buffers to that stream."""

    def __init__(self, m, device="cuda:0", ntrans_sim=None, ndir_max=None, stream=None):
        if not torch.cuda.is_available():
            raise B.LocError(B.LOC_ECUDA, "no CUDA device: the LOC library has no CPU path")
        self.dev = torch.device(device)
        torch.cuda.set_device(self.dev)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.dev)
        with self._on_stream():
            self._init(m, ntrans_sim, ndir_max)

    def _on_stream(self):
        return torch.cuda.stream(self.stream)

    def _init(self, m, ntrans_sim, ndir_max):
        self.is3d = hasattr(m, "child")
        sp = m.species
        self.nlevel, self.ntrans = len(sp.energy_K), len(sp.upper)
        self.nch = int(m.nchannel)
        up = lambda a, dt=torch.float32: self._to_dev(a, dt)
        self.density, self.tkin, self.sigma, self.abundance = up(m.density), up(m.tkin), up(m.sigma), up(m.abundance)
        if self.is3d:
            self.vx, self.vy, self.vz = up(m.vx), up(m.vy), up(m.vz)
            self.child = up(m.child, torch.int32)
            self.grid, self._keep = B.make_octree_grid(m.nx, m.ny, m.nz, m.root_cm, m.noff, self.child)
            self.ncell = int(np.asarray(m.noff)[-1])
            ndir_max = ndir_max or len(m.dirs)
        else:
            self.vx, self.vy, self.vz = up(m.vrad), None, None
            self.grid, self._keep = B.make_shell_grid(m.r_out, m.ray_p, m.ray_w)
            self.ncell = len(m.r_out)
            ndir_max = 1
        self.cells = B.loc_cells(B._dp(self.density), B._dp(self.tkin), B._dp(self.sigma), B._dp(self.vx), B._dp(self.vy),
                                 B._dp(self.vz), B._dp(self.abundance))
        nts = ntrans_sim or self.ntrans
        nbytes = B.loc_workspace_bytes(self.grid, self.nch, self.nlevel, nts, ndir_max)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.dev)
        sptr = self.stream.cuda_stream
        self.h = B.loc_create_model(self.grid, self.cells, self.nch, m.band_half, m.t_bg, self.nlevel, nts, ndir_max,
                                    self.workspace, sptr)
        B.loc_set_species(self.h, sp)
        for t, (dvk, wk) in sorted((getattr(sp, "hfs", None) or {}).items()):
            B.loc_set_hyperfine(self.h, t, dvk, wk)
        if self.is3d:
            B.loc_set_directions(self.h, m.dirs)
        self.pops = torch.empty((self.nlevel, self.ncell), dtype=torch.float32, device=self.dev)
        B.loc_set_populations(self.h, self.pops)

    def _to_dev(self, a, dt):
        t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
        return t.to(device=self.dev, dtype=dt, non_blocking=True).contiguous()

    # ---- forwarding -------------------------------------------------------------------------------------
    def set_directions(self, dirs):
        B.loc_set_directions(self.h, dirs)

    def update_cells(self, **arrays):
        """overwrite per-cell input arrays (density, tkin, sigma, vx, vy, vz, abundance) from host or device data"""
        with self._on_stream():
            for k, a in arrays.items():
                getattr(self, k).copy_(a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a)),
                                       non_blocking=True)
        B.loc_refresh_cells(self.h)

    def init_lte(self):
        B.loc_init_lte(self.h)

    def set_populations(self, pops_level_major):
        """pops_level_major: [nlevel][ncell] host or device array; copied into the registered buffer"""
        with self._on_stream():
            self.pops.copy_(self._to_dev(pops_level_major, torch.float32))
        B.loc_set_populations(self.h, self.pops)

    def simulate(self, sel=None, geometry_counters=False):
        B.loc_simulate(self.h, sel, geometry_counters)

    def solve(self) -> float:
        return B.loc_solve(self.h)

    def iterate(self, niter) -> float:
        return B.loc_iterate(self.h, niter)

    def set_ali(self, ali: bool) -> None:
        B.loc_set_ali(self.h, ali)

    def iterate_until(self, max_iter, tol):
        """(iterations run, last max relative change)"""
        return B.loc_iterate_until(self.h, max_iter, tol)

    def stats(self) -> dict:
        return B.loc_get_stats(self.h)

    def counters(self):
        """(SJ, ESC) as float32 device tensors [ncell][nsel] (views into the workspace, valid until next simulate)"""
        cptr, nsp, _, _ = B.loc_get_counters(self.h)
        nsel = self.stats()["ntrans_sim"]
        v = _as_tensor_view(cptr, self.ncell * nsp * 8, self.workspace, torch.float32).view(self.ncell, nsp, 2)
        return v[:, :nsel, 0], v[:, :nsel, 1]

    def geometry_counters(self):
        _, _, vptr, pptr = B.loc_get_counters(self.h)
        vis = _as_tensor_view(vptr, self.ncell * 4, self.workspace, torch.int32)
        pz = _as_tensor_view(pptr, self.ncell * 4, self.workspace, torch.int32)
        return vis, pz

    def set_option(self, key: int, value: float) -> None:
        B.loc_set_option(self.h, key, value)

    def spectra(self, trans, nx, ny=1, dir=None, aff=None, offsets_cm=None):
        with self._on_stream():
            out = torch.empty((ny, nx, self.nch), dtype=torch.float32, device=self.dev)
        B.loc_spectra(self.h, trans, out, nx, ny, dir, aff, offsets_cm)
        return out

    def spectra_map(self, trans, nx, ny, dir, pixel_cm, centre_cm):
        """map in the caller's frame (include/loc.h, loc_spectra_map): [ny][nx][nchannel] K"""
        with self._on_stream():
            out = torch.empty((ny, nx, self.nch), dtype=torch.float32, device=self.dev)
        B.loc_spectra_map(self.h, trans, out, nx, ny, dir, pixel_cm, centre_cm)
        return out

    def tex(self, trans):
        """T_ex [ncell] (K) of a transition from the current populations; 0 in non-leaf cells / cells without molecules"""
        with self._on_stream():
            out = torch.empty(self.ncell, dtype=torch.float32, device=self.dev)
        B.loc_tex(self.h, trans, out)
        return out

    def line_area(self, cube):
        """W = sum_c T_A dv in K km/s for a cube [..., nchannel] of loc_spectra (float32 CUDA tensor)"""
        with self._on_stream():
            cube = cube.contiguous()
            out = torch.empty(cube.shape[:-1], dtype=torch.float32, device=self.dev)
        npix = cube.numel() // self.nch
        B.loc_line_area(self.h, cube, npix, out)
        return out

    def close(self):
        if getattr(self, "h", None) is not None:
            B.loc_destroy_model(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
