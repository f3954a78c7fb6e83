"""Writes tests/golden/wave200_<variant>.npz: config 5's own workload computed by the ORACLE ONLY.

BASELINE.json config 5: 33 x 64 x 128, shell [2, 12], 200 RK4 steps of the first-order scalar wave system with the
characteristic boundary condition and the Yn filter after each substep (DESIGN.md readings
W1-W6), "compared to oracle and to the exact solution".  The oracle needs ~25 min on 8 cores for the 200 steps, so its
result is stored: per-field max-norms and a stratified sample (every radius of every field, seeded latitudes and
longitudes) of the state after 100 and 200 steps.  tests/test_gpu_wave.py compares the GPU run with these values at
1e-12 and checks `key` (hash of the oracle sources with comments stripped, the input generator and the parameters)
so that a changed oracle cannot be compared against stale values.

This script imports oracle/ and synth/ only (never the CUDA library).

    python tests/golden/make_wave200.py clean      # the config's data: outgoing l <= 4 pulses
    python tests/golden/make_wave200.py noise      # + 1e-6 white noise: the filter's truncation acts inside the loop
"""
import hashlib
import os
import re
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CHECKPOINTS = (100, 200)
NSAMP_PER_RADIUS = 60
NOISE = {"clean": 0.0, "noise": 1e-6}
NOISE_SEED = 3


def _strip_c(src):
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    src = re.sub(r"//[^\n]*", "", src)
    return "\n".join(l.strip() for l in src.splitlines() if l.strip())


def golden_key(variant):
    """Hash of everything the stored values depend on."""
    h = hashlib.sha256()
    with open(os.path.join(ROOT, "oracle", "sp_oracle.c")) as f:
        h.update(_strip_c(f.read()).encode())
    import inspect
    import oracle
    import synth.wave
    for fn in (oracle.wave_rk4, oracle.wave_rhs, oracle.tensor_filter, oracle.wave_dt):
        h.update(inspect.getsource(fn).encode())
    h.update(inspect.getsource(synth.wave).encode())
    h.update(repr((variant, NOISE[variant], NOISE_SEED, CHECKPOINTS, NSAMP_PER_RADIUS)).encode())
    return h.hexdigest()


def initial_data(variant):
    import synth
    c = synth.config(5)
    u0 = synth.wave_exact(c, 0.0)
    if NOISE[variant]:
        u0 = u0 + NOISE[variant] * np.random.default_rng(NOISE_SEED).standard_normal(u0.shape)
    return c, u0


def sample_indices(c):
    """[ns, 4] = (field, j, i, k): every radius of every field, NSAMP_PER_RADIUS seeded (i, j) each, plus both poles' rows."""
    rng = np.random.default_rng(5200)
    rows = []
    for f in range(5):
        for k in range(c["Nr"]):
            i = rng.integers(0, c["Nt"], NSAMP_PER_RADIUS)
            j = rng.integers(0, c["Np"], NSAMP_PER_RADIUS)
            i[0], i[1] = 0, c["Nt"] - 1
            rows.append(np.stack([np.full_like(i, f), j, i, np.full_like(i, k)], axis=1))
    return np.concatenate(rows).astype(np.int32)


def main(variant):
    import oracle
    oracle.set_threads(int(os.environ.get("ORACLE_THREADS", os.cpu_count() or 1)))
    c, u = initial_data(variant)
    Nr, Nt, Np = c["Nr"], c["Nt"], c["Np"]
    dt = oracle.wave_dt(Nr, Nt, Np, c["rmin"], c["rmax"])
    idx = sample_indices(c)
    out = {"key": np.array(golden_key(variant)), "idx": idx, "dt": np.array(dt)}
    t0 = time.time()

    def snapshot(step, v):
        if step in CHECKPOINTS:
            out[f"maxabs_{step}"] = np.max(np.abs(v.reshape(5, -1)), axis=1)
            out[f"val_{step}"] = v[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]].copy()
        if step % 10 == 0:
            print(f"step {step}  {time.time() - t0:.0f} s", flush=True)

    oracle.wave_rk4(u, Nr, Nt, Np, c["rmin"], c["rmax"], c["L"], c["tensors"], dt, max(CHECKPOINTS), on_step=snapshot)
    np.savez_compressed(os.path.join(HERE, f"wave200_{variant}.npz"), **out)


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "clean")
