"""Grid sizes, shells and tensor layouts of the five configurations (BASELINE.json)."""

_SYM10 = 10  # symmetric 4x4: tt,tx,ty,tz,xx,xy,xz,yy,yz,zz (row-major upper triangle)


def tensor_ncomp(t):
    """Number of stored components: row-major over indices, symmetric pair as its upper triangle."""
    dims = list(t["dims"])
    s0, s1 = t.get("sym", (-1, -1))
    n = 0
    idx = [0] * len(dims)

    def rec(q):
        nonlocal n
        if q == len(dims):
            if s0 < 0 or idx[s0] <= idx[s1]:
                n += 1
            return
        for a in range(dims[q]):
            idx[q] = a
            rec(q + 1)

    rec(0)
    return n


def ghg_tensors(extra_gauge=False):
    """GHG state: g_ab (10), Pi_ab (10), Phi_iab (30) [+ H_a, d_t H_a]."""
    t = [
        {"name": "g_ab", "rank": 2, "dims": (4, 4), "sym": (0, 1), "fields": list(range(0, 10))},
        {"name": "Pi_ab", "rank": 2, "dims": (4, 4), "sym": (0, 1), "fields": list(range(10, 20))},
        {"name": "Phi_iab", "rank": 3, "dims": (3, 4, 4), "sym": (1, 2), "fields": list(range(20, 50))},
    ]
    if extra_gauge:
        t.append({"name": "H_a", "rank": 1, "dims": (4,), "sym": (-1, -1), "fields": list(range(50, 54))})
        t.append({"name": "dtH_a", "rank": 1, "dims": (4,), "sym": (-1, -1), "fields": list(range(54, 58))})
    return t


def wave_tensors():
    """First-order scalar wave: psi, Pi scalars; Phi_i a spatial vector."""
    return [
        {"name": "psi", "rank": 0, "dims": (), "sym": (-1, -1), "fields": [0]},
        {"name": "Pi", "rank": 0, "dims": (), "sym": (-1, -1), "fields": [1]},
        {"name": "Phi_i", "rank": 1, "dims": (3,), "sym": (-1, -1), "fields": [2, 3, 4]},
    ]


# L for configs 2-5 is the paper's default n_f = 4: L = Ntheta - 5 (reading Q6);
# config 4 reuses config 3's shell (reading Q6b).  lmax = highest degree put into the synthetic data.
CONFIGS = {
    1: dict(Nr=9, Nt=8, Np=16, rmin=1.0, rmax=3.0, L=6, nfields=1, lmax=6,
            tensors=[{"name": "u", "rank": 0, "dims": (), "sym": (-1, -1), "fields": [0]}]),
    2: dict(Nr=17, Nt=24, Np=48, rmin=1.8, rmax=10.0, L=19, nfields=50, lmax=23, tensors=ghg_tensors()),
    3: dict(Nr=33, Nt=48, Np=96, rmin=1.8, rmax=20.0, L=43, nfields=50, lmax=47, tensors=ghg_tensors()),
    4: dict(Nr=65, Nt=96, Np=192, rmin=1.8, rmax=20.0, L=91, nfields=58, lmax=95, tensors=ghg_tensors(True)),
    5: dict(Nr=33, Nt=64, Np=128, rmin=2.0, rmax=12.0, L=59, nfields=5, lmax=4, tensors=wave_tensors()),
}


def config(n):
    c = dict(CONFIGS[n])
    c["id"] = n
    c["seed"] = 11043408 + n
    c["npts"] = c["Nr"] * c["Nt"] * c["Np"]
    return c
