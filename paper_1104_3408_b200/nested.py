"""RK4 driver of the first-order scalar wave system on NESTED shells.

Host-side sequencing only: every arithmetic step is a kernel behind the C ABI (sp_rhs_wave_shell, sp_wave_interface, sp_rk4_stage,
sp_tensor_filter).  Shells [R_a, R_a+1] share their interface spheres and the angular grid; between two exchanges the shells are
independent units (each has its own sp_shell, state, workspaces), which is also where a multi-GPU layout would cut.
"""


class NestedWaveRK4:
    def __init__(self, shells, tensors):
        """shells: list of binding.Shell ordered from the innermost outwards, shells[a].r_out == shells[a+1].r_in."""
        import torch
        self.shells, self.tensors = list(shells), tensors
        dev = torch.device("cuda")
        self.descs = [sh.make_descs(tensors) for sh in self.shells]
        mk = lambda sh: torch.empty((5, sh.Np, sh.Nt, sh.Nr), dtype=torch.float64, device=dev)
        self.k = [mk(sh) for sh in self.shells]
        self.acc = [mk(sh) for sh in self.shells]
        self.stage = [mk(sh) for sh in self.shells]
        self.ws_w, self.ws_f = [], []
        for sh in self.shells:
            _, f, w = sh.workspace_bytes(5)
            self.ws_w.append(torch.empty(w // 8, dtype=torch.float64, device=dev))
            self.ws_f.append(torch.empty(f // 8, dtype=torch.float64, device=dev))
        self._graph, self._graph_key = None, None

    def dt(self, lam=4.0):
        """lambda * min(dx) over all shells (eq. 63)."""
        return min(sh.wave_dt(lam) for sh in self.shells)

    def rhs(self, vs, out=None):
        """Coupled right-hand side of all shells: raw RHS per shell (freezing condition on the two physical boundary spheres only),
        then the characteristic exchange on every interface."""
        out = self.k if out is None else out
        n = len(self.shells)
        for a, sh in enumerate(self.shells):
            sh.rhs_wave_shell(vs[a], bc_inner=(a == 0), bc_outer=(a == n - 1), out=out[a], workspace=self.ws_w[a])
        for a in range(n - 1):
            self.shells[a].wave_interface(self.shells[a], out[a], self.shells[a + 1], out[a + 1])
        return out

    def _filter(self, vs):
        for a, sh in enumerate(self.shells):
            sh.tensor_filter(vs[a], self.tensors, out=vs[a], workspace=self.ws_f[a], descs=self.descs[a])

    def _combine(self, us, c_acc, c_stage, first=False, last=False):
        for a, sh in enumerate(self.shells):
            acc_in = us[a] if first else self.acc[a]
            if last:
                sh.rk4_stage(us[a], self.k[a], acc_in, us[a], None, c_acc, 0.0)
            else:
                sh.rk4_stage(us[a], self.k[a], acc_in, self.acc[a], self.stage[a], c_acc, c_stage)

    def _step(self, us, dt):
        self.rhs(us)                                                      # k1
        self._combine(us, dt / 6.0, 0.5 * dt, first=True); self._filter(self.stage)
        self.rhs(self.stage)                                              # k2
        self._combine(us, dt / 3.0, 0.5 * dt); self._filter(self.stage)
        self.rhs(self.stage)                                              # k3
        self._combine(us, dt / 3.0, dt); self._filter(self.stage)
        self.rhs(self.stage)                                              # k4
        self._combine(us, dt / 6.0, 0.0, last=True)                       # new states written over us
        self._filter(us)

    def evolve(self, us, dt, nsteps, graph=False):
        """us: list of CUDA tensors [5, Np, Nt, Nr_a], advanced in place by nsteps RK4 steps (filter placement as WaveRK4)."""
        import torch
        self._filter(us)
        if graph and nsteps > 0:
            key = (tuple(u.data_ptr() for u in us), float(dt))
            if self._graph_key != key:
                side = torch.cuda.Stream()
                side.wait_stream(torch.cuda.current_stream())
                with torch.cuda.stream(side):
                    keep = [u.clone() for u in us]
                    self._step(us, dt)                                    # warm-up outside capture
                    for u, k in zip(us, keep):
                        u.copy_(k)
                torch.cuda.current_stream().wait_stream(side)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    self._step(us, dt)
                for u, k in zip(us, keep):
                    u.copy_(k)
                self._graph, self._graph_key = g, key
            for _ in range(nsteps):
                self._graph.replay()
            return us
        for _ in range(nsteps):
            self._step(us, dt)
        return us
