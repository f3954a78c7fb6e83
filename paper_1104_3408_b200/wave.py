"""RK4 driver of the first-order scalar wave system (BASELINE.json config 5; eq. 63).

Host-side sequencing only: every arithmetic step is a kernel behind the C ABI
(sp_rhs_first_order_wave, sp_axpby, sp_tensor_filter).  Filter placement (reading W5):
the initial data, every stage state before its RHS, and the final combination -- 4 filters per step.
"""
import math


def wave_dt(Nr, Nt, Np, r_in, r_out, lam=4.0):
    """dt = lambda * min(dx), eq. 63 (reading W4)."""
    r0 = 0.5 * (r_out + r_in) - 0.5 * (r_out - r_in)
    r1 = 0.5 * (r_out + r_in) - 0.5 * (r_out - r_in) * math.cos(math.pi / (Nr - 1))
    th0 = math.pi * 0.5 / Nt
    return lam * min(r1 - r0, 2.0 * r0 * math.sin(th0) * math.sin(math.pi / Np))


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

    def _filter(self, v):
        self.sh.tensor_filter(v, self.tensors, out=v, workspace=self.ws_f, descs=self.descs)

    def _rhs(self, v):
        self.sh.rhs_first_order_wave(v, out=self.k, workspace=self.ws_w)

    def evolve(self, u, dt, nsteps):
        """u: CUDA tensor [5, Np, Nt, Nr], advanced in place by nsteps RK4 steps; returns u."""
        ax = self.sh.axpby
        self._filter(u)
        for _ in range(nsteps):
            self._rhs(u)                                   # k1
            self.acc.copy_(u); ax(dt / 6.0, self.k, 1.0, self.acc)
            self.stage.copy_(u); ax(0.5 * dt, self.k, 1.0, self.stage); self._filter(self.stage)
            self._rhs(self.stage)                          # k2
            ax(dt / 3.0, self.k, 1.0, self.acc)
            self.stage.copy_(u); ax(0.5 * dt, self.k, 1.0, self.stage); self._filter(self.stage)
            self._rhs(self.stage)                          # k3
            ax(dt / 3.0, self.k, 1.0, self.acc)
            self.stage.copy_(u); ax(dt, self.k, 1.0, self.stage); self._filter(self.stage)
            self._rhs(self.stage)                          # k4
            ax(dt / 6.0, self.k, 1.0, self.acc)
            u.copy_(self.acc)
            self._filter(u)
        return u
