"""RK4 driver of the GHG single-black-hole evolution (Sec. 4.1, Appendix A).

Host-side sequencing only: every arithmetic step is a kernel behind the C ABI (sp_rhs_ghg incl. the boundary condition
as part of each substep, sp_rk4_stage, sp_tensor_filter).  "After one complete RK4 step, we apply the filter"
(PAPER.md:176): one Yn filter per step, on g_ab, k_ab (rank 2, symmetric, 4-dimensional indices) and d_iab (rank 3).
"""


def ghg_tensors():
    """Tensor layout of the 50-field GHG state for sp_tensor_filter."""
    return [
        {"name": "g_ab", "rank": 2, "dims": (4, 4), "sym": (0, 1), "fields": list(range(0, 10))},
        {"name": "k_ab", "rank": 2, "dims": (4, 4), "sym": (0, 1), "fields": list(range(10, 20))},
        {"name": "d_iab", "rank": 3, "dims": (3, 4, 4), "sym": (1, 2), "fields": list(range(20, 50))},
    ]


def scalar_tensors(fields):
    return [{"name": f"u{q}", "rank": 0, "dims": (), "sym": (-1, -1), "fields": [q]} for q in fields]


class GhgRK4:
    """filter: "Yn" (spin-weighted tensor filter, the method of the paper), "Y" (every component filtered as a scalar with
    the same L), "Yg" (graded scalar filter, eq. 59: component mu keeps l <= L + d(u^mu); the same kernels with the matrix
    tables of four shells of kept degree L .. L+3) -- the three filters compared in PAPER.md Sec. 3.5 / 4.1 (Fig. 5-6)."""

    def __init__(self, shell, H, dH, bc_outer=True, filter="Yn"):
        import torch
        from .binding import Shell
        self.sh, self.H, self.dH, self.bc = shell, H, dH, bc_outer
        self.filter_mode = filter
        if filter == "Yn":
            self.passes = [(shell, ghg_tensors())]
        elif filter == "Y":
            self.passes = [(shell, scalar_tensors(range(50)))]
        elif filter == "Yg":
            kept = [shell.ghg_graded_degree(q) for q in range(50)]      # eq. 59, evaluated behind the ABI
            self.passes = []
            for L in sorted(set(kept)):
                shd = shell if L == shell.L else Shell(shell.Nr, shell.Nt, shell.Np, shell.r_in, shell.r_out, L)
                self.passes.append((shd, scalar_tensors([q for q in range(50) if kept[q] == L])))
        else:
            raise ValueError("filter must be 'Yn', 'Y' or 'Yg'")
        self.passes = [(shd, t, shd.make_descs(t)) for shd, t in self.passes]
        dev = torch.device("cuda")
        shape = (50, shell.Np, shell.Nt, shell.Nr)
        self.k = torch.empty(shape, dtype=torch.float64, device=dev)
        self.acc = torch.empty(shape, dtype=torch.float64, device=dev)
        self.stage = torch.empty(shape, dtype=torch.float64, device=dev)
        f = max(shd.workspace_bytes(50)[1] for shd, _, _ in self.passes)
        self.ws_r = torch.empty(shell.ghg_workspace_bytes() // 8, dtype=torch.float64, device=dev)
        self.ws_f = torch.empty(f // 8, dtype=torch.float64, device=dev)
        self._graph, self._graph_key = None, None

    def rhs(self, v, out=None):
        return self.sh.rhs_ghg(v, self.H, self.dH, out=self.k if out is None else out, bc_outer=self.bc, workspace=self.ws_r)

    def filter(self, v):
        for shd, tensors, descs in self.passes:      # fields outside a pass are left as they are
            shd.tensor_filter(v, tensors, out=v, workspace=self.ws_f, descs=descs)

    def _step(self, u, dt):
        st = self.sh.rk4_stage
        self.rhs(u)                                                       # k1
        st(u, self.k, u, self.acc, self.stage, dt / 6.0, 0.5 * dt)
        self.rhs(self.stage)                                              # k2
        st(u, self.k, self.acc, self.acc, self.stage, dt / 3.0, 0.5 * dt)
        self.rhs(self.stage)                                              # k3
        st(u, self.k, self.acc, self.acc, self.stage, dt / 3.0, dt)
        self.rhs(self.stage)                                              # k4
        st(u, self.k, self.acc, u, None, dt / 6.0, 0.0)                   # new state over u
        self.filter(u)

    def evolve(self, u, dt, nsteps, graph=False):
        """u: CUDA tensor [50, Np, Nt, Nr], advanced in place by nsteps RK4 steps; returns u.  graph=True replays one
        captured RK4 step (4 RHS with gradient and boundary kernels, 4 combinations, 1 filter)."""
        import torch
        if graph and nsteps > 0:
            key = (u.data_ptr(), float(dt))
            if self._graph_key != key:
                side = torch.cuda.Stream()
                side.wait_stream(torch.cuda.current_stream())
                with torch.cuda.stream(side):
                    keep = u.clone()
                    self._step(u, dt)                                     # warm-up outside capture
                    u.copy_(keep)
                torch.cuda.current_stream().wait_stream(side)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    self._step(u, dt)
                self._graph, self._graph_key = g, key
            for _ in range(nsteps):
                self._graph.replay()
            return u
        for _ in range(nsteps):
            self._step(u, dt)
        return u
