"""tridsk_dock_static: the docking run for callers that may not allocate (include/tridsk.h) against the existing
tridsk_dock path, on two calls in a row that share the library's static scratch array.  Collected last on purpose
(the suite runs with pytest -x); needs nothing from the other test modules.  Run on the B200 box: pytest -m gpu.
"""
import numpy as np
import pytest

from workloads import synth

pytestmark = pytest.mark.gpu

RTOL, ATOL = 1e-4, 1e-3          # the energy tolerance of tests/test_gpu_parity.py (BASELINE.json north_star)


def _close(got, want):
    got, want = np.asarray(got, np.float64), np.asarray(want, np.float64)
    return np.all(np.abs(got - want) <= ATOL + RTOL * np.abs(want))


@pytest.fixture(scope="module")
def setup():
    import torch
    from paper_2510_24186_b200 import Engine, default_params
    rec = synth.receptor(300, 20.0, 16, seed=1001, grid_n=54)
    radius, role = synth.type_table(16)
    batch = synth.ligands([12, 30, 50, 80], [2, 6, 10, 20], 16, seed=4242)   # both instances of the CTA kernel (<= 64 atoms, above)
    eng = Engine(0)
    gp = default_params()
    grid = eng.build_grid(rec.xyz, rec.type, radius, role, gp, rec.origin, rec.dims, rec.spacing)
    ligs = eng.load_ligands(batch, radius, role)
    yield dict(torch=torch, eng=eng, gp=gp, rec=rec, grid=grid, ligs=ligs, radius=radius, role=role)
    ligs.free(); grid.free(); eng.close()


def _outs(torch, dev, L, k, stride):
    return (torch.full((L, k, 2), float("nan"), device=dev), torch.full((L, k, stride), float("nan"), device=dev),
            torch.full((L, k), -7, dtype=torch.int32, device=dev))


def test_dock_static_matches_dock_on_two_calls_in_a_row(setup):
    S = setup
    torch, eng, rec, ligs = S["torch"], S["eng"], S["rec"], S["ligs"]
    L, stride = ligs.n_lig, 7 + ligs.max_tor
    box = (rec.box_min, rec.box_max, rec.pocket_center, rec.pocket_radius)
    # two different shapes back to back: the second call finds the first call's chain state in the shared array
    calls = [dict(n_chains=48, n_steps=25, top_k=5, seed=11), dict(n_chains=20, n_steps=40, top_k=3, seed=12)]
    # the existing path first (CTA per chain, the mapping tridsk_dock_static runs), into its own buffers
    eng.set_kernel(3)
    want = []
    for c in calls:
        r = eng.dock(S["grid"], ligs, S["gp"], *box, c["n_chains"], c["n_steps"], c["top_k"], seed=c["seed"], pose_stride=stride)
        assert eng.last_kernel() == 3
        want.append(r)
    eng.set_kernel(0)
    outs = [_outs(torch, eng.device, L, c["top_k"], stride) for c in calls]
    torch.cuda.synchronize()
    n0 = eng.launch_count() if hasattr(eng, "launch_count") else None
    for c, o in zip(calls, outs):                                              # two calls in a row, nothing in between
        eng.dock_static(S["grid"], ligs, S["gp"], *box, c["n_chains"], c["n_steps"], c["top_k"], o, seed=c["seed"], pose_stride=stride)
    torch.cuda.synchronize()
    if n0 is not None:
        assert eng.launch_count() - n0 == 2 * 3                                # per call: two MC kernel instances + top-k
    for c, o, w in zip(calls, outs, want):
        e, p, ch = (t.cpu().numpy() for t in o)
        assert np.array_equal(ch, w["chain"]), c                               # index work: exact
        assert np.all(np.isfinite(e)) and np.all(np.isfinite(p))
        assert _close(e, w["energy"]), (c, np.abs(e - w["energy"]).max())
        assert _close(p, w["pose"]), c
        assert np.array_equal(e, w["energy"]) and np.array_equal(p, w["pose"]), c   # same kernels, same arguments: bit-identical
    # the first call once more, after the second: the stale contents of the array do not matter
    o = _outs(torch, eng.device, L, calls[0]["top_k"], stride)
    free0 = torch.cuda.mem_get_info()[0]
    c = calls[0]
    eng.dock_static(S["grid"], ligs, S["gp"], *box, c["n_chains"], c["n_steps"], c["top_k"], o, seed=c["seed"], pose_stride=stride)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                               # no device memory was taken by the call
    assert np.array_equal(o[2].cpu().numpy(), want[0]["chain"]) and np.array_equal(o[0].cpu().numpy(), want[0]["energy"])


def test_dock_static_rejects_what_it_cannot_hold(setup):
    from paper_2510_24186_b200 import TridskError
    S = setup
    torch, eng, rec, ligs = S["torch"], S["eng"], S["rec"], S["ligs"]
    L, stride = ligs.n_lig, 7 + ligs.max_tor
    box = (rec.box_min, rec.box_max, rec.pocket_center, rec.pocket_radius)
    # chain state beyond the 4 MiB array: 4 ligands x 6,000 chains x (2 x 27 + 2) floats = 5.4 MB
    o = _outs(torch, eng.device, L, 1, stride)
    with pytest.raises(TridskError, match="static scratch array holds 4194304"):
        eng.dock_static(S["grid"], ligs, S["gp"], *box, 6000, 1, 1, o, pose_stride=stride)
    assert int(o[2][0, 0]) == -7                                               # nothing was launched
    # host outputs would need a staging allocation
    h = (np.empty((L, 1, 2), np.float32), np.empty((L, 1, stride), np.float32), np.empty((L, 1), np.int32))
    with pytest.raises(TridskError, match="device memory only"):
        eng.dock_static(S["grid"], ligs, S["gp"], *box, 8, 1, 1, h, pose_stride=stride)
    # and the call still works afterwards
    eng.dock_static(S["grid"], ligs, S["gp"], *box, 8, 2, 1, o, pose_stride=stride)
    torch.cuda.synchronize()
    assert int(o[2].min()) >= 0 and bool(torch.isfinite(o[0]).all())
