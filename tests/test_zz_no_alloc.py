"""sp_tensor_filter_noalloc (include/spshell.h): the Yn filter for callers that cannot call cudaMalloc or pass a workspace -- its
scratch is a 32 MiB file-scope static device array inside the library.  Checked against the existing path (sp_tensor_filter with a
caller workspace) on two calls in a row that share the array.  Collected LAST on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _rel(a, b):
    a = a.reshape(a.shape[0], -1); b = b.reshape(a.shape)
    den = np.max(np.abs(b), axis=1)
    den[den == 0] = 1.0
    return float(np.max(np.max(np.abs(a - b), axis=1) / den))


def _shell(cfg):
    from paper_1104_3408_b200 import Shell
    return Shell(cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"], cfg["L"])


def test_noalloc_filter_matches_the_workspace_path_on_two_calls_in_a_row():
    """Call 1: config 2 (50-field GHG layout: rank 2 fused kernels + rank 3 five-stage path, 20.9 MB of the 32 MiB) on white noise.
    Call 2, straight after on the same stream, reuses the array with the previous call's contents in it: the seeded band-limited
    state of the same config, then a third call with a DIFFERENT layout (every field a scalar) so that the regions mean something
    else.  Each result equals sp_tensor_filter's within the tests' tolerance, and the second and third call change the device's
    free memory by nothing (no allocation)."""
    import torch
    cfg = synth.config(2)
    sh = _shell(cfg)
    scal = [{"rank": 0, "dims": (), "sym": (-1, -1), "fields": [f]} for f in range(cfg["nfields"])]
    cases = [(synth.white_state(cfg), cfg["tensors"]), (synth.make_state(cfg), cfg["tensors"]), (synth.white_state(cfg), scal)]
    want = [sh.tensor_filter(torch.from_numpy(u).cuda(), t).cpu().numpy() for u, t in cases]      # existing path, own workspace
    ud = [torch.from_numpy(u).cuda() for u, _ in cases]
    out = [torch.empty_like(x) for x in ud]
    descs = [sh.make_descs(t) for _, t in cases]
    sh.tensor_filter_noalloc(ud[0], cases[0][1], out[0], descs=descs[0])                          # first call: resolves the symbol
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    sh.tensor_filter_noalloc(ud[1], cases[1][1], out[1], descs=descs[1])                          # in a row, same stream
    sh.tensor_filter_noalloc(ud[2], cases[2][1], out[2], descs=descs[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    for q in range(3):
        got = out[q].cpu().numpy()
        assert np.all(np.isfinite(got))
        assert _rel(got, want[q]) < TOL, q
    # in place (out == u), as sp_tensor_filter allows
    v = ud[1].clone()
    sh.tensor_filter_noalloc(v, cases[1][1], v, descs=descs[1])
    assert _rel(v.cpu().numpy(), want[1]) < TOL


def test_noalloc_filter_rejects_sizes_beyond_the_static_array():
    """Config 3's GHG state needs 172 MB of scratch: SP_ERR_SCRATCH_LIMIT, nothing launched, output untouched; a part of the state
    that fits (g_ab alone: 34 MB does not, a 4-vector does) goes through."""
    import torch
    from paper_1104_3408_b200 import launch_count
    from paper_1104_3408_b200.binding import SpError
    cfg = synth.config(3)
    sh = _shell(cfg)
    assert sh.workspace_bytes(50)[1] > sh.NOALLOC_SCRATCH_BYTES
    u = torch.from_numpy(synth.make_state(cfg)).cuda()
    out = torch.full_like(u, 7.0)
    n0 = launch_count()
    with pytest.raises(SpError, match="SCRATCH_LIMIT"):
        sh.tensor_filter_noalloc(u, cfg["tensors"], out)
    torch.cuda.synchronize()
    assert launch_count() == n0 and bool((out == 7.0).all())
    vec = [{"rank": 1, "dims": (4,), "sym": (-1, -1), "fields": [0, 1, 2, 3]}]
    assert sh.workspace_bytes(4)[1] <= sh.NOALLOC_SCRATCH_BYTES
    got = sh.tensor_filter_noalloc(u, vec, out).cpu().numpy()
    want = sh.tensor_filter(u, vec).cpu().numpy()
    assert _rel(got, want) < TOL
