"""RK4 driver of the first-order scalar wave system (BASELINE.json config 5; eq. 63).

Host-side sequencing only: every arithmetic step is a kernel behind the C ABI
(sp_rhs_first_order_wave, sp_axpby, sp_tensor_filter).  Filter placement (reading W5):
the initial data, every stage state before its RHS, and the final combination -- 4 filters per step.
"""


def wave_dt(Nr, Nt, Np, r_in, r_out, lam=4.0):
    """dt = lambda * min(dx), eq. 63 (reading W4): computed behind the C ABI (sp_wave_dt); this is marshalling only."""
    from .binding import Shell
    return Shell(Nr, Nt, Np, r_in, r_out, 0, build=False).wave_dt(lam)


class WaveRK4:
    def __init__(self, shell, tensors):
        import torch
        self.sh, self.tensors = shell, tensors
        self.descs = shell.make_descs(tensors)
        dev = torch.device("cuda")
        shape = (5, shell.Np, shell.Nt, shell.Nr)
        self.k = torch.empty(shape, dtype=torch.float64, device=dev)
        self.acc = torch.empty(shape, dtype=torch.float64, device=dev)
        self.stage = torch.empty(shape, dtype=torch.float64, device=dev)
        _, f, w = shell.workspace_bytes(5)
        self.ws_w = torch.empty(w // 8, dtype=torch.float64, device=dev)
        self.ws_f = torch.empty(f // 8, dtype=torch.float64, device=dev)
        self._graph, self._graph_key = None, None

    def _filter(self, v):
        self.sh.tensor_filter(v, self.tensors, out=v, workspace=self.ws_f, descs=self.descs)

    def _rhs(self, v):
        self.sh.rhs_first_order_wave(v, out=self.k, workspace=self.ws_w)

    def _step(self, u, dt):
        st = self.sh.rk4_stage
        self._rhs(u)                                                      # k1
        st(u, self.k, u, self.acc, self.stage, dt / 6.0, 0.5 * dt); self._filter(self.stage)
        self._rhs(self.stage)                                             # k2
        st(u, self.k, self.acc, self.acc, self.stage, dt / 3.0, 0.5 * dt); self._filter(self.stage)
        self._rhs(self.stage)                                             # k3
        st(u, self.k, self.acc, self.acc, self.stage, dt / 3.0, dt); self._filter(self.stage)
        self._rhs(self.stage)                                             # k4
        st(u, self.k, self.acc, u, None, dt / 6.0, 0.0)                   # new state written over u
        self._filter(u)

    def evolve(self, u, dt, nsteps, graph=False):
        """u: CUDA tensor [5, Np, Nt, Nr], advanced in place by nsteps RK4 steps; returns u.
        graph=True captures one RK4 step (4 RHS, 4 filters, 4 combinations: every pointer is fixed) in a CUDA graph and
        replays it nsteps times: the step is ~50 short launches, so the replay removes their launch gaps."""
        import torch
        self._filter(u)
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
                u.copy_(keep)                                             # capture does not execute, but keep the state explicit
                self._graph, self._graph_key = g, key
            for _ in range(nsteps):
                self._graph.replay()
            return u
        for _ in range(nsteps):
            self._step(u, dt)
        return u
