"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Tolerance: 1e-12 relative, max-norm over each field (north_star)."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _torch():
    import torch
    return torch


def _shell(cfg):
    from paper_1104_3408_b200 import Shell
    return Shell(cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"], cfg["L"])


def _rel(a, b):
    """worst field of max|a-b| / max|b| (fields = leading axes, last three axes are the grid)."""
    a = a.reshape(-1, a.shape[-3] * a.shape[-2] * a.shape[-1])
    b = b.reshape(a.shape)
    den = np.max(np.abs(b), axis=1)
    den[den == 0] = 1.0
    return float(np.max(np.max(np.abs(a - b), axis=1) / den))


def _grad_gpu(sh, u):
    torch = _torch()
    return sh.cartesian_gradient(torch.from_numpy(u).cuda()).cpu().numpy()


def _filt_gpu(sh, u, tensors):
    torch = _torch()
    return sh.tensor_filter(torch.from_numpy(u).cuda(), tensors).cpu().numpy()


@pytest.mark.parametrize("cid,white", [(1, False), (2, False), (2, True), (3, False)])
def test_gradient_full(cid, white):
    cfg = synth.config(cid)
    u = synth.white_state(cfg) if white else synth.make_state(cfg)
    nf = u.shape[0] if cid < 3 else 10                      # config 3: 10 of the 50 fields in full
    u = np.ascontiguousarray(u[:nf])
    got = _grad_gpu(_shell(cfg), u)
    want = oracle.gradient(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"])
    assert _rel(got, want) < TOL


def _stratified_gradient_samples(cfg, rng, nplanes_full=3):
    """(k, i, j, mu) samples that leave no work item of the gradient kernels unchecked: one seeded (k, i) in EVERY (field, longitude)
    plane (the persistent (r,theta) kernel walks (field, antipodal plane pair) items, the d/dphi kernels (field, column tile) items),
    both radial boundary shells and both polar rows in every field, and `nplanes_full` whole (field, j) planes (every
    (latitude tile, radial tile group) warp task, every lane of its epilogue) -- among them the very last item of the launch."""
    Nr, Nt, Np, nf = cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["nfields"]
    mu, j = np.meshgrid(np.arange(nf), np.arange(Np), indexing="ij")
    mu, j = mu.ravel(), j.ravel()
    k, i = rng.integers(Nr, size=mu.size), rng.integers(Nt, size=mu.size)
    k[0::7], k[3::7] = 0, Nr - 1
    i[1::5], i[2::5] = 0, Nt - 1
    rows = [np.stack([k, i, j, mu], axis=1)]
    planes = [(nf - 1, Np - 1)] + [(int(rng.integers(nf)), int(rng.integers(Np))) for _ in range(nplanes_full - 1)]
    kk, ii = np.meshgrid(np.arange(Nr), np.arange(Nt), indexing="ij")
    for f, jj in planes:
        rows.append(np.stack([kk.ravel(), ii.ravel(), np.full(kk.size, jj), np.full(kk.size, f)], axis=1))
    return np.concatenate(rows).astype(np.int32)


@pytest.mark.parametrize("cid", [3, 4, 5])
def test_gradient_sampled_full_size(cid):
    """Full-size launch (the bench configuration) against the oracle on a STRATIFIED sample (see above; 30 000 outputs x 3 at
    config 4) with the tolerance relative to each output field's max-norm."""
    cfg = synth.config(cid)
    u = synth.make_state(cfg)
    got = _grad_gpu(_shell(cfg), u)
    samp = _stratified_gradient_samples(cfg, np.random.default_rng(cid))
    want = oracle.gradient_at(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"], samp)      # [ns, 3]
    fmax = np.max(np.abs(got.reshape(3, cfg["nfields"], -1)), axis=2)        # [3, nf]
    k, i, j, mu = samp.T
    g = got[:, mu, j, i, k].T                                                # [ns, 3]
    err = np.abs(g - want) / fmax[:, mu].T
    worst = np.unravel_index(np.argmax(err), err.shape)
    assert err.max() <= TOL, (samp[worst[0]], g[worst[0]], want[worst[0]], err.max())
    assert len(set(zip(mu.tolist(), j.tolist()))) == cfg["nfields"] * cfg["Np"]      # every (field, j) plane was sampled


@pytest.mark.parametrize("cid,white", [(1, False), (2, False), (2, True)])
def test_filter_full(cid, white):
    cfg = synth.config(cid)
    u = synth.white_state(cfg) if white else synth.make_state(cfg)
    got = _filt_gpu(_shell(cfg), u, cfg["tensors"])
    want = oracle.tensor_filter(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"], cfg["tensors"])
    assert _rel(got, want) < TOL
    if cid == 1:      # config 1's data lies inside the kept band: the filter must preserve it
        assert _rel(got, u) < TOL


@pytest.mark.parametrize("cid,radii,white", [(3, (0, 17), False), (3, (32,), True), (4, (0, 20, 40, 64), True), (4, (7, 51), False), (5, (0, 16, 32), False),
                                             (5, (5,), True)])
def test_filter_sampled_radii_full_size(cid, radii, white):
    """Full-size launch; the oracle filters whole spheres at sampled radii (F is independent of r).  The radii cover both
    boundary shells and every radial block / column-tile tail of the theta and phi kernels (config 4: 65 radii = blocks 0-35 and
    36-64)."""
    cfg = synth.config(cid)
    if white:
        u = synth.white_state(cfg)
    else:
        u = synth.make_state(cfg)
    got = _filt_gpu(_shell(cfg), u, cfg["tensors"])
    for k in radii:
        want = oracle.tensor_filter(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"], cfg["tensors"], ksel=k)
        a, b = got[..., k:k + 1], want[..., k:k + 1]
        assert _rel(a, b) < TOL, (cid, k)


TYPES = [
    {"rank": 0, "dims": (), "sym": (-1, -1)},
    {"rank": 1, "dims": (3,), "sym": (-1, -1)},
    {"rank": 1, "dims": (4,), "sym": (-1, -1)},
    {"rank": 2, "dims": (3, 3), "sym": (0, 1)},
    {"rank": 2, "dims": (4, 4), "sym": (0, 1)},
    {"rank": 3, "dims": (3, 3, 3), "sym": (1, 2)},
    {"rank": 3, "dims": (3, 4, 4), "sym": (1, 2)},
    {"rank": 3, "dims": (4, 3, 3), "sym": (1, 2)},
    {"rank": 3, "dims": (4, 4, 4), "sym": (1, 2)},
]


@pytest.mark.parametrize("shape", [(5, 7, 14, 4), (9, 8, 16, 6), (6, 10, 20, 9), (12, 9, 18, 0)])
def test_every_tensor_type_ragged_grids(shape):
    """All supported index structures on grids that are not multiples of the 8x8x4 tile (odd Ntheta,
    even Nr, L = 0 and L = Ntheta-1), white-noise data, scattered field order, pass-through fields."""
    from paper_1104_3408_b200 import Shell
    Nr, Nt, Np, L = shape
    rng = np.random.default_rng(Nr * 100 + Nt)
    tensors, nf = [], 0
    for t in TYPES:
        nc = synth.tensor_ncomp(t)
        tensors.append(dict(t, fields=list(range(nf, nf + nc))))
        nf += nc + 1                                           # leave a gap field that no tensor owns
    perm = rng.permutation(nf)
    for t in tensors:
        t["fields"] = [int(perm[f]) for f in t["fields"]]
    u = rng.standard_normal((nf, Np, Nt, Nr))
    sh = Shell(Nr, Nt, Np, 1.3, 4.1, L)
    got = _filt_gpu(sh, u, tensors)
    want = oracle.tensor_filter(u, Nr, Nt, Np, L, tensors)
    assert _rel(got, want) < TOL
    owned = {f for t in tensors for f in t["fields"]}
    for f in range(nf):
        if f not in owned:
            assert np.array_equal(got[f], u[f])
    g = _grad_gpu(sh, u)
    assert _rel(g, oracle.gradient(u, Nr, Nt, Np, 1.3, 4.1)) < TOL


def test_filter_invariants_and_edge_cases():
    torch = _torch()
    from paper_1104_3408_b200 import Shell, SpError
    cfg = synth.config(2)
    sh = _shell(cfg)
    u = torch.from_numpy(synth.white_state(cfg)).cuda()
    f1 = sh.tensor_filter(u, cfg["tensors"])
    f2 = sh.tensor_filter(f1, cfg["tensors"])
    assert _rel(f2.cpu().numpy(), f1.cpu().numpy()) < TOL          # idempotent
    f1b = sh.tensor_filter(u, cfg["tensors"])
    assert torch.equal(f1, f1b)                                    # deterministic, bit for bit
    v = u.clone()
    sh.tensor_filter(v, cfg["tensors"], out=v)                     # in place
    assert torch.equal(v, f1)
    g1 = sh.cartesian_gradient(u); g2 = sh.cartesian_gradient(u)
    assert torch.equal(g1, g2)
    # empty inputs
    e = torch.empty((0, cfg["Np"], cfg["Nt"], cfg["Nr"]), dtype=torch.float64, device="cuda")
    assert sh.cartesian_gradient(e).numel() == 0
    assert torch.equal(sh.tensor_filter(u, []), u)                 # no tensors: copy through
    # errors: a field in two tensors; unsupported structure; short workspace
    bad = [dict(cfg["tensors"][0]), dict(cfg["tensors"][0])]
    with pytest.raises(SpError):
        sh.tensor_filter(u, bad)
    with pytest.raises(SpError):
        sh.tensor_filter(u, [{"rank": 2, "dims": (3, 3), "sym": (-1, -1), "fields": list(range(9))}])
    with pytest.raises(SpError):
        sh.cartesian_gradient(u, workspace=torch.empty(8, dtype=torch.float64, device="cuda"))


def test_gradient_exact_polynomial_on_gpu():
    """Invariant that needs no oracle: exact Cartesian gradient of a polynomial in x, y, z."""
    cfg = synth.config(2)
    r, th, ph = oracle.grid(cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"])
    P, T, R = np.meshgrid(ph, th, r, indexing="ij")
    x, y, z = R * np.sin(T) * np.cos(P), R * np.sin(T) * np.sin(P), R * np.cos(T)
    f = (x ** 3 * y - 2 * z ** 2 * x + y * z) / 100.0
    g = _grad_gpu(_shell(cfg), f[None])
    want = np.stack([(3 * x ** 2 * y - 2 * z ** 2) / 100, (x ** 3 + z) / 100, (-4 * z * x + y) / 100])[:, None]
    assert _rel(g, want) < 1e-11


def test_scalar_Y_filter_is_the_all_scalars_layout():
    """The paper's scalar Y-filter (the n = 0 matrices applied to every Cartesian component, ignoring the
    tensor character) is the same call with every field declared rank 0; the graded Yg-filter (eq. 59) is that call
    on shells created with L - d(u^mu).  Parity on config 2 data, and it must differ from the Yn result."""
    cfg = synth.config(2)
    u = synth.white_state(cfg, nfields=20)
    scal = [{"rank": 0, "dims": (), "sym": (-1, -1), "fields": [f]} for f in range(20)]
    sh = _shell(cfg)
    got = _filt_gpu(sh, u, scal)
    want = oracle.tensor_filter(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"], scal)
    assert _rel(got, want) < TOL
    yn = _filt_gpu(sh, u, cfg["tensors"][:2])
    assert _rel(got, yn) > 1e-3


def test_misaligned_buffers_take_the_general_path():
    """Buffers that start at an odd element (8-byte but not 16-byte aligned) cannot use the 16-byte cp.async fast paths:
    the library must fall back to its general kernels (d/dphi into the workspace, unfolded plane kernel, global-memory
    GEMMs) and still match the oracle.  Config 2 sizes, white noise."""
    torch = _torch()
    cfg = synth.config(2)
    sh = _shell(cfg)
    u = synth.white_state(cfg, nfields=20)
    n = u.size
    flat = torch.empty(n + 1, dtype=torch.float64, device="cuda")
    ud = flat[1:].view(u.shape)
    ud.copy_(torch.from_numpy(u))
    assert ud.data_ptr() % 16 == 8
    oflat = torch.empty(3 * n + 1, dtype=torch.float64, device="cuda")
    out = oflat[1:].view((3,) + u.shape)
    wflat = torch.empty(sh.workspace_bytes(20)[1] // 8 + 1, dtype=torch.float64, device="cuda")
    got = sh.cartesian_gradient(ud, out=out, workspace=wflat[1:]).cpu().numpy()
    want = oracle.gradient(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"])
    assert _rel(got, want) < TOL
    tens = cfg["tensors"][:2]
    fo = torch.empty(n + 1, dtype=torch.float64, device="cuda")[1:].view(u.shape)
    gotf = sh.tensor_filter(ud, tens, out=fo, workspace=wflat[1:]).cpu().numpy()
    wantf = oracle.tensor_filter(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"], tens)
    assert _rel(gotf, wantf) < TOL
    # and the aligned fast path gives the same numbers to rounding
    fast = sh.cartesian_gradient(torch.from_numpy(u).cuda()).cpu().numpy()
    assert _rel(fast, got) < TOL


def test_bench_launch_configuration_two_streams():
    """The step exactly as bench.py times it (config 3, pre-allocated outputs and workspaces, gradient and filter of
    one state issued on two CUDA streams, several steps in flight): bit-identical to the same calls on one stream, and
    sampled against the oracle."""
    import bench
    torch = _torch()
    cfg = synth.config(3)
    wl = bench.GpuWorkload(cfg, nsets=2)
    wl.step()
    torch.cuda.synchronize()
    du1, fu1 = wl.du.clone(), wl.fu.clone()                  # serial, input set 0
    wl.it = 0
    sg, sf = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(4):                                       # sets 0, 1, 0, 1 back to back: the pipeline is full
        wl.step(sg, sf)
    wl.it = 0
    wl.step(sg, sf)                                          # ends on set 0
    torch.cuda.synchronize()
    assert torch.equal(wl.du, du1) and torch.equal(wl.fu, fu1)
    wl.capture()                                             # the same step as replayed CUDA graphs (bench.py's default)
    wl.du.zero_(); wl.fu.zero_()
    for n in (0, 1, 0, 1, 0):
        wl.graphs[n].replay()
    torch.cuda.synchronize()
    assert torch.equal(wl.du, du1) and torch.equal(wl.fu, fu1)
    wl.du.zero_(); wl.fu.zero_()
    wl.round_graph.replay()                                  # sets 0, 1 in one graph without an inner join ...
    wl.graphs[0].replay()                                    # ... then set 0 again
    torch.cuda.synchronize()
    assert torch.equal(wl.du, du1) and torch.equal(wl.fu, fu1)
    u = wl.u_host
    got = wl.du.cpu().numpy()
    rng = np.random.default_rng(33)
    ns = 500
    samp = np.stack([rng.integers(cfg["Nr"], size=ns), rng.integers(cfg["Nt"], size=ns), rng.integers(cfg["Np"], size=ns),
                     rng.integers(cfg["nfields"], size=ns)], axis=1).astype(np.int32)
    want = oracle.gradient_at(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"], samp)
    fmax = np.max(np.abs(got.reshape(3, cfg["nfields"], -1)), axis=2)
    for s, (k, i, j, mu) in enumerate(samp):
        assert np.all(np.abs(got[:, mu, j, i, k] - want[s]) <= TOL * fmax[:, mu])
    k = 11
    wantf = oracle.tensor_filter(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"], cfg["tensors"], ksel=k)
    assert _rel(wl.fu.cpu().numpy()[..., k:k + 1], wantf[..., k:k + 1]) < TOL


def test_gradient_is_deterministic():
    torch = _torch()
    cfg = synth.config(2)
    sh = _shell(cfg)
    u = torch.from_numpy(synth.white_state(cfg)).cuda()
    a = sh.cartesian_gradient(u).clone()
    for _ in range(3):
        assert torch.equal(sh.cartesian_gradient(u), a)


def test_shell_too_large_for_the_plane_kernels_is_refused_and_extreme_small_shells_work():
    """Maximum size: an antipodal (r, theta) plane pair must fit one SM's shared memory (spshell.h, SIZE LIMIT); the build
    refuses larger shells with SP_ERR_UNSUPPORTED instead of launching anything.  Minimum size: Nr = Ntheta = 2."""
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.binding import SpError
    torch = _torch()
    with pytest.raises(SpError, match="UNSUPPORTED"):
        Shell(129, 128, 256, 1.5, 9.0, 100)
    Nr, Nt, Np, L = 2, 2, 4, 1
    sh = Shell(Nr, Nt, Np, 1.5, 9.0, L)
    u = np.random.default_rng(2).standard_normal((2, Np, Nt, Nr))
    got = sh.cartesian_gradient(torch.from_numpy(u).cuda()).cpu().numpy()
    assert _rel(got, oracle.gradient(u, Nr, Nt, Np, 1.5, 9.0)) < TOL
    tens = [{"name": "s", "rank": 0, "dims": (), "sym": (-1, -1), "fields": [0]}]
    gotf = sh.tensor_filter(torch.from_numpy(u).cuda(), tens).cpu().numpy()
    assert _rel(gotf, oracle.tensor_filter(u, Nr, Nt, Np, L, tens)) < TOL


@pytest.mark.parametrize("env", [
    {"SP_THETA_NT": "1", "SP_GRAD_NWARPS": "2", "SP_GRAD_CTAS": "1", "SP_DPHI_FOLD_MIN": "16", "SP_PHI_NC": "32"},
    {"SP_THETA_NT": "3", "SP_GRAD_KT": "3", "SP_GRAD_NWARPS": "4", "SP_PHI_NC": "64", "SP_PHI_MSPLIT": "1"},
    {"SP_THETA_NT": "23", "SP_THETA_FOLD": "0"},
    {"SP_THETA_NT": "21", "SP_PHI_MSPLIT": "2"},
    {"SP_FUSE": "2", "SP_FUSE_NBUF": "2", "SP_GRAD_CHUNK": "3"},
    {"SP_FUSE": "1", "SP_FAN_NC4": "1", "SP_FAN_THREADS": "256", "SP_FSYN_NW": "8", "SP_THETA_TUNE": "1"},
])
def test_tuning_overrides_keep_parity(env):
    """Every kernel variant the environment overrides can select (README, "tuning overrides") computes the same numbers: the
    oracle comparisons of this file are rerun in a child process with the overrides set (they are read once per process)."""
    import os
    import subprocess
    import sys
    child = dict(os.environ, **env)
    sel = ("test_gradient_full or test_filter_full or test_every_tensor_type_ragged_grids or test_gradient_sampled_full_size "
           "or test_filter_sampled_radii_full_size")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.abspath(__file__), "-x", "-q", "-k", sel], env=child,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert " passed" in r.stdout and "failed" not in r.stdout


def test_a_shell_built_later_does_not_break_an_earlier_larger_one():
    """The dynamic shared-memory opt-in is a per-function, process-wide attribute: building a small shell after a large one must
    not lower the cap the large shell's kernels launch with (multi-resolution runs, nested shells).  Config-3 shell A, then a
    9 x 8 x 16 shell B, then gradient and filter on A against the oracle; and B works too."""
    torch = _torch()
    from paper_1104_3408_b200 import Shell
    cfg = synth.config(3)
    A = _shell(cfg)
    B = Shell(9, 8, 16, 1.0, 3.0, 6)
    u = synth.make_state(cfg)
    got = _grad_gpu(A, u)
    samp = _stratified_gradient_samples(cfg, np.random.default_rng(7), nplanes_full=1)
    want = oracle.gradient_at(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"], samp)
    fmax = np.max(np.abs(got.reshape(3, cfg["nfields"], -1)), axis=2)
    k, i, j, mu = samp.T
    assert (np.abs(got[:, mu, j, i, k].T - want) / fmax[:, mu].T).max() <= TOL
    gf = _filt_gpu(A, u, cfg["tensors"])
    wantf = oracle.tensor_filter(u, cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"], cfg["tensors"], ksel=9)
    assert _rel(gf[..., 9:10], wantf[..., 9:10]) < TOL
    c1 = synth.config(1)
    u1 = synth.make_state(c1)
    assert _rel(_grad_gpu(B, u1), oracle.gradient(u1, 9, 8, 16, 1.0, 3.0)) < TOL
    assert _rel(_filt_gpu(B, u1, c1["tensors"]), oracle.tensor_filter(u1, 9, 8, 16, 6, c1["tensors"])) < TOL


@pytest.mark.parametrize("mode", ["0", "1", "2"])
def test_fused_and_five_stage_filter_paths_agree_with_the_oracle(mode):
    """SP_FUSE selects which tensors take the fused kernels (k_fan: projection + analysis, k_fsyn: synthesis + recombination) and
    which the five-stage path; every mode must match the oracle.  Child process (the variable is read once per process): all
    index structures on ragged grids, config 2 in full, sampled radii of configs 3 and 5."""
    import os
    import subprocess
    import sys
    child = dict(os.environ, SP_FUSE=mode)
    sel = "test_filter_full or test_every_tensor_type_ragged_grids or (test_filter_sampled_radii_full_size and not 4-)"
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.abspath(__file__), "-x", "-q", "-k", sel], env=child,
                       capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert " passed" in r.stdout and "failed" not in r.stdout
