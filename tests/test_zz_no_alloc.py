"""trimeg_gather_noalloc (the gather for callers that must not call cudaMalloc: its scratch is a static device array of
TRIMEG_GATHER_NOALLOC_MAX points inside the library) against the existing trimeg_gather paths, same inputs.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.  It must pass alone in a
fresh process and after the other tests; it depends on nothing they leave behind (own context, own mesh).

Tolerance: GATHER_TOL (1e-12 per gathered quantity, tests/test_gpu_parity.py); the new entry point runs the same staged
kernels as trimeg_gather in mode 2, so against that mode the results must be identical bit for bit.
"""
import dataclasses

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_24327_b200 import synth  # noqa: E402
from test_gpu_parity import GATHER_TOL, _make, _rel  # noqa: E402


def _points(cfg, m, n, shift):
    """n points of the marker set, some moved outside the mesh and into the hole, phi far outside [0, period)"""
    R, Z, phi = m["R"][shift:shift + n].copy(), m["Z"][shift:shift + n].copy(), m["phi"][shift:shift + n].copy()
    R[::97] = cfg.R0 + 2.0 * cfg.a
    R[5::101] = cfg.R0 + 0.01 * cfg.a
    Z[5::101] = 0.0
    phi[::7] += 5 * cfg.phi_period
    phi[3::11] -= 3 * cfg.phi_period
    return R, Z, phi


def test_gather_noalloc_matches_existing_paths_two_calls_in_a_row():
    import torch
    from paper_2606_24327_b200.binding import Trimeg, TrimegError
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=Trimeg.GATHER_NOALLOC_MAX + 1000)
    RZ, tri, o, g, m = _make(cfg)
    nmax = Trimeg.GATHER_NOALLOC_MAX
    # two calls in a row on the same stream, different points and sizes: the full limit first, then a ragged smaller count,
    # so that the second call runs over the first call's leftovers in the static array
    calls = [(nmax, 0), (70_001, 937)]
    outs = []
    w = [torch.from_numpy(m[k][:33].copy()).cuda() for k in ("R", "Z", "phi")]
    g.gather_noalloc(*w, torch.empty((8, 33), dtype=torch.float64, device="cuda"))   # first launch of each kernel loads its code
    g.sync()
    for n, shift in calls:
        R, Z, phi = _points(cfg, m, n, shift)
        d = [torch.from_numpy(a).cuda() for a in (R, Z, phi)]
        out = torch.full((8, n), float("nan"), dtype=torch.float64, device="cuda")
        tout = torch.full((n,), -7, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        g.gather_noalloc(*d, out, tout)                    # no synchronisation in between: the next call follows on the stream
        assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory: something allocated"
        outs.append((d, out, tout))
    g.sync()
    for (n, shift), (d, out, tout) in zip(calls, outs):
        g.set_gather_mode(2)
        ref2, tref2 = g.gather(*d)                         # existing staged path: same kernels, library-owned workspace
        assert torch.equal(out, ref2) and torch.equal(tout, tref2)
        g.set_gather_mode(1)
        ref1, tref1 = g.gather(*d)                         # existing direct kernel
        a, b = out.cpu().numpy(), ref1.cpu().numpy()
        lost = tref1.cpu().numpy() < 0
        assert lost.sum() > 100 and ((tout.cpu().numpy() < 0) == lost).all() and np.abs(a[:, lost]).max() == 0.0
        for q in range(8):
            assert _rel(a[q], b[q]) < GATHER_TOL, (n, q, _rel(a[q], b[q]))
        assert (tout == tref1).float().mean() > 0.995      # points on an edge may be given to either triangle
    # and against the oracle, on a sample of the second call
    (d, out, tout) = outs[1]
    idx = np.arange(0, calls[1][0], 7)
    ref, tref = o.gather(*[a.cpu().numpy()[idx] for a in d])
    for q in range(8):
        assert _rel(out.cpu().numpy()[q][idx], ref[q]) < GATHER_TOL
    # beyond the limit: refused with a message that names it, nothing written
    n = nmax + 1
    R, Z, phi = (torch.from_numpy(m[k][:n].copy()).cuda() for k in ("R", "Z", "phi"))
    out = torch.zeros((8, n), dtype=torch.float64, device="cuda")
    with pytest.raises(TrimegError, match="TRIMEG_GATHER_NOALLOC_MAX"):
        g.gather_noalloc(R, Z, phi, out)
    g.sync()
    assert float(out.abs().max()) == 0.0
    # a second context on the same device shares the array: used one after the other (synchronised) it gives the same result
    RZ2, tri2, o2, g2, m2 = _make(cfg)
    (d, out, tout) = outs[1]
    out2 = torch.empty_like(out)
    g2.gather_noalloc(*d, out2)
    g2.sync()
    assert torch.equal(out2, out)
    g.close(); g2.close()
