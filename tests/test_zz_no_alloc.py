"""loc_spectra_shells_static: the one entry point for callers that cannot allocate device memory (include/loc.h).

Who that is: code that is handed its device buffers by somebody else and has no allocator of its own -- a plug-in or
callback inside a host application that owns all device memory, a display / monitoring step running beside a solver
whose workspace fills the GPU, a latency-critical loop that must not hit the device-wide synchronisation of cudaMalloc.
Every other call of the library needs a loc_model, hence a workspace; this one keeps its scratch (shell radii and the
packed velocity / line-width record) in a fixed array inside the library, for at most LOC_STATIC_MAX_SHELLS shells.

The test checks the new entry point against the existing path (LocModel -> loc_create_model + loc_spectra, whose
scratch sits in the caller's workspace) at the tolerance of tests/test_gpu_spectra.py, on two calls in a row that are
enqueued on one stream without a synchronisation between them: first a model of 64 shells, then one of 12 shells with
other velocities and another transition, so that the second call runs over what the first left in the shared array.
It also checks that the entry point allocates nothing (torch's allocator statistics and the free device memory stay
where they were) and that too large a model is refused with a message naming the limit.

The file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call then performs the per-device look-up of the array's address) and after
the other tests.
"""
import numpy as np
import pytest

import loc_workloads as W

pytestmark = pytest.mark.gpu

_H, _K = 6.62607015e-27, 1.380649e-16


def _close(ta, ref):
    """tolerance of tests/test_gpu_spectra.py: 1e-3 relative + 2e-5 of the peak, per channel"""
    ta, ref = np.asarray(ta, np.float64), np.asarray(ref, np.float64)
    tol = 1e-3 * np.abs(ref) + 2e-5 * np.max(np.abs(ref))
    assert np.all(np.abs(ta - ref) <= tol), f"worst {np.max(np.abs(ta - ref) / tol):.2f} x tolerance"


def _case(ns, nch, trans, niter):
    """a shell model brought to `niter` ALI iterations through the existing path; returns what both paths need"""
    from paper_2009_12609_b200 import LocModel
    m = W.shell_config(1, ns=ns, nchannel=nch)
    g = LocModel(m)
    g.init_lte()
    if niter:
        g.iterate(niter)
    # 300 lines of sight (two launches of the kernel): centre, ragged offsets, the edge, outside, negative side
    b = np.concatenate([[0.0], np.linspace(0.0, 1.05, 297), [0.9999999, -0.4]]) * m.r_out[-1]
    ref = g.spectra(trans, len(b), offsets_cm=b)[0].clone()
    return m, g, b, ref


def _static_call(m, g, b, trans, out):
    from paper_2009_12609_b200 import binding as B
    sp = m.species
    u, l = int(sp.upper[trans]), int(sp.lower[trans])
    freq = (sp.energy_K[u] - sp.energy_K[l]) * _K / _H  # as loc_set_species derives it from the level energies
    B.loc_spectra_shells_static(m.r_out, g.vx, g.sigma, g.tkin, sp.mass_amu, g.pops[u], g.pops[l], freq, sp.einstein_A[trans],
                                sp.g[u], sp.g[l], m.nchannel, m.band_half, m.t_bg, b, out, g.stream.cuda_stream)


def test_static_scratch_matches_workspace_path_twice_in_a_row():
    import torch
    m1, g1, b1, ref1 = _case(64, 67, 0, 3)
    m2, g2, b2, ref2 = _case(12, 64, 1, 0)
    m2_vr = (np.linspace(-1.0, 1.0, 12) * 0.3e5).astype(np.float32)  # another velocity law: the packed records must be rewritten
    g2.update_cells(vx=m2_vr)
    ref2 = g2.spectra(1, len(b2), offsets_cm=b2)[0].clone()
    assert g1.stream.cuda_stream == g2.stream.cuda_stream
    out1 = torch.full((len(b1), m1.nchannel), float("nan"), device=g1.dev)
    out2 = torch.full((len(b2), m2.nchannel), float("nan"), device=g2.dev)
    torch.cuda.synchronize()
    stats0 = torch.cuda.memory_stats(g1.dev)["allocation.all.allocated"]
    free0 = torch.cuda.mem_get_info(g1.dev)[0]
    _static_call(m1, g1, b1, 0, out1)  # no synchronisation between the two calls: same stream, shared scratch
    _static_call(m2, g2, b2, 1, out2)
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats(g1.dev)["allocation.all.allocated"] == stats0, "the binding created a tensor"
    # free device memory may only drop by what the driver itself takes on a first launch (module loading); never by a buffer
    assert free0 - torch.cuda.mem_get_info(g1.dev)[0] < (32 << 20)
    for out, ref, b, m in ((out1, ref1, b1, m1), (out2, ref2, b2, m2)):
        ta, rf = out.cpu().numpy(), ref.cpu().numpy()
        assert np.all(np.isfinite(ta)) and np.max(np.abs(rf)) > 0
        _close(ta, rf)
        assert np.all(ta[np.abs(b) >= m.r_out[-1]] == 0.0)
    # and once more in the other order (large after small)
    out1.fill_(float("nan"))
    _static_call(m1, g1, b1, 0, out1)
    torch.cuda.synchronize()
    _close(out1.cpu().numpy(), ref1.cpu().numpy())
    g1.close()
    g2.close()


def test_static_scratch_rejects_what_does_not_fit():
    import torch
    from paper_2009_12609_b200 import binding as B
    n = B.LOC_STATIC_MAX_SHELLS + 1
    z = torch.ones(n, device="cuda:0")
    out = torch.zeros((1, 8), device="cuda:0")
    r = np.arange(1, n + 1, dtype=np.float64)
    with pytest.raises(B.LocError) as e:
        B.loc_spectra_shells_static(r, z, z, z, 28.0, z, z, 1e11, 1e-7, 3.0, 1.0, 8, 1e5, 2.73, [0.0], out)
    assert e.value.code == B.LOC_EINVAL and str(B.LOC_STATIC_MAX_SHELLS) in str(e.value)
    with pytest.raises(B.LocError):  # radii must ascend
        B.loc_spectra_shells_static([2.0, 1.0], z[:2], z[:2], z[:2], 28.0, z[:2], z[:2], 1e11, 1e-7, 3.0, 1.0, 8, 1e5, 2.73, [0.0], out)
    assert torch.all(out == 0)
