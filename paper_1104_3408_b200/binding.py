import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libspshell.so")
_lib = None

# every symbol include/spshell.h declares
EXPORTED_SYMBOLS = [
    "sp_shell_create", "sp_shell_destroy", "sp_build_matrices", "sp_workspace_bytes", "sp_cartesian_gradient",
    "sp_tensor_filter", "sp_tensor_filter_noalloc", "sp_rhs_first_order_wave", "sp_rhs_wave_shell", "sp_wave_interface", "sp_wave_dt", "sp_axpby", "sp_rk4_stage", "sp_ghg_graded_degree", "sp_ghg_workspace_bytes", "sp_rhs_ghg", "sp_ghg_init", "sp_get_tuning", "sp_get_matrix", "sp_probe_fp64_peak",
    "sp_status_string", "sp_profile_enable", "sp_profile_read", "sp_launch_count",
]


class SpError(RuntimeError):
    pass


class _TensorDesc(C.Structure):
    _fields_ = [("rank", C.c_int), ("index_dim", C.c_int * 3), ("sym_first", C.c_int), ("sym_second", C.c_int),
                ("field", C.POINTER(C.c_int))]


def library_path():
    return _LIB_PATH


def lib():
    """Load libspshell.so (built in-tree by paper_1104_3408_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise SpError(f"{_LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.sp_status_string.restype = C.c_char_p
        L.sp_status_string.argtypes = [C.c_int]
        L.sp_shell_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.POINTER(C.c_void_p)]
        L.sp_shell_destroy.argtypes = [C.c_void_p]
        L.sp_build_matrices.argtypes = [C.c_void_p]
        L.sp_workspace_bytes.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.sp_cartesian_gradient.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sp_tensor_filter.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(_TensorDesc), C.c_int,
                                       C.c_void_p, C.c_size_t, C.c_void_p]
        L.sp_tensor_filter_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(_TensorDesc), C.c_int, C.c_void_p]
        L.sp_rhs_first_order_wave.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sp_rhs_wave_shell.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sp_wave_interface.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sp_wave_dt.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.sp_axpby.argtypes = [C.c_double, C.c_void_p, C.c_double, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sp_rk4_stage.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_size_t,
                                   C.c_void_p]
        L.sp_ghg_graded_degree.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int)]
        L.sp_ghg_workspace_bytes.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.sp_rhs_ghg.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
        L.sp_ghg_init.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sp_get_tuning.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
        L.sp_get_matrix.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.sp_probe_fp64_peak.argtypes = [C.c_int, C.POINTER(C.c_double)]
        L.sp_profile_enable.argtypes = [C.c_void_p, C.c_int]
        L.sp_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.sp_launch_count.restype = C.c_ulonglong
        L.sp_launch_count.argtypes = []
        _lib = L
    return _lib


def status_string(code):
    return lib().sp_status_string(code).decode()


def _check(code, what):
    if code != 0:
        raise SpError(f"{what}: {status_string(code)}")


def probe_fp64_peak(mode=0):
    """TFLOP/s of a register-only DMMA (mode 0) or DFMA (mode 1) loop on the current device."""
    v = C.c_double()
    _check(lib().sp_probe_fp64_peak(mode, C.byref(v)), "sp_probe_fp64_peak")
    return v.value


def launch_count():
    return int(lib().sp_launch_count())


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev_f64(t, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise SpError(f"{name} must be a contiguous CUDA float64 tensor")
    return t


class Shell:
    """sp_shell_create + sp_build_matrices.  Arrays are torch CUDA float64 tensors shaped
    [nfields, Nphi, Ntheta, Nr] (C order == the ABI's p = k + Nr(i + Nt(j + Np mu)))."""

    def __init__(self, Nr, Ntheta, Nphi, r_in, r_out, L, build=True, host_only=False):
        self._h = C.c_void_p()
        _check(lib().sp_shell_create(Nr, Ntheta, Nphi, float(r_in), float(r_out), L, C.byref(self._h)), "sp_shell_create")
        self.Nr, self.Nt, self.Np, self.L = Nr, Ntheta, Nphi, L
        self.r_in, self.r_out = float(r_in), float(r_out)
        self.npts = Nr * Ntheta * Nphi
        self._ws = None
        if build:
            self.build_matrices(host_only=host_only)

    def __del__(self):
        try:
            if getattr(self, "_h", None) is not None and self._h.value:
                lib().sp_shell_destroy(self._h)
                self._h = C.c_void_p()
        except Exception:
            pass

    def build_matrices(self, host_only=False):
        code = lib().sp_build_matrices(self._h)
        if host_only and code == 4:      # SP_ERR_CUDA: no device; host matrices are available via get_matrix
            return
        _check(code, "sp_build_matrices")

    def workspace_bytes(self, nfields):
        g, f, w = C.c_size_t(), C.c_size_t(), C.c_size_t()
        _check(lib().sp_workspace_bytes(self._h, nfields, C.byref(g), C.byref(f), C.byref(w)), "sp_workspace_bytes")
        return g.value, f.value, w.value

    def _workspace(self, nbytes, device):
        import torch
        if self._ws is None or self._ws.numel() * 8 < nbytes or self._ws.device != device:
            self._ws = torch.empty((nbytes + 7) // 8, dtype=torch.float64, device=device)
        return self._ws

    def get_matrix(self, which, n=0, m=0):
        import numpy as np
        r, c = C.c_int(), C.c_int()
        _check(lib().sp_get_matrix(self._h, which, n, m, None, C.byref(r), C.byref(c)), "sp_get_matrix")
        out = np.zeros((r.value, c.value))
        _check(lib().sp_get_matrix(self._h, which, n, m, out.ctypes.data_as(C.c_void_p), C.byref(r), C.byref(c)), "sp_get_matrix")
        return out

    STAGES = ("grad_dphi", "grad_rtheta", "filt_project", "filt_analysis", "filt_theta", "filt_synthesis", "filt_recombine")

    def tuning(self):
        """Kernel variants chosen at build time (sp_get_tuning)."""
        out = (C.c_int * 4)()
        _check(lib().sp_get_tuning(self._h, out), "sp_get_tuning")
        return {"theta_NT": out[0], "grad_KT": out[1], "dphi_folded": bool(out[2]), "grad_plane_buffers": out[3]}

    def profile(self, on=True):
        _check(lib().sp_profile_enable(self._h, 1 if on else 0), "sp_profile_enable")

    def profile_read(self):
        """dict stage -> milliseconds of the last profiled call(s)."""
        ms = (C.c_double * 7)()
        _check(lib().sp_profile_read(self._h, ms), "sp_profile_read")
        return {k: ms[q] for q, k in enumerate(self.STAGES)}

    # ---- hot calls (marshalling only) ---------------------------------------------------------
    def cartesian_gradient(self, u, out=None, workspace=None, stream=None):
        import torch
        u = _dev_f64(u, "u")
        nf = u.numel() // self.npts
        if nf * self.npts != u.numel():
            raise SpError("u has the wrong size")
        if out is None:
            out = torch.empty((3, nf, self.Np, self.Nt, self.Nr), dtype=torch.float64, device=u.device)
        _dev_f64(out, "out")
        need = self.workspace_bytes(nf)[0]
        ws = self._workspace(need, u.device) if workspace is None else _dev_f64(workspace, "workspace")
        _check(lib().sp_cartesian_gradient(self._h, u.data_ptr(), nf, out.data_ptr(), ws.data_ptr(), ws.numel() * 8,
                                           _stream_ptr(stream)), "sp_cartesian_gradient")
        return out

    def make_descs(self, tensors):
        """tensors: list of dicts {rank, dims, sym, fields} (synth.configs layout) -> ctypes array (+ keepalive)."""
        arr = (_TensorDesc * max(len(tensors), 1))()
        keep = []
        for q, t in enumerate(tensors):
            arr[q].rank = t["rank"]
            for a in range(3):
                arr[q].index_dim[a] = t["dims"][a] if a < len(t["dims"]) else 0
            s = t.get("sym", (-1, -1))
            arr[q].sym_first, arr[q].sym_second = s[0], s[1]
            f = (C.c_int * max(len(t["fields"]), 1))(*t["fields"])
            keep.append(f)
            arr[q].field = C.cast(f, C.POINTER(C.c_int))
        return arr, keep, len(tensors)

    def tensor_filter(self, u, tensors, out=None, workspace=None, stream=None, descs=None):
        import torch
        u = _dev_f64(u, "u")
        nf = u.numel() // self.npts
        if out is None:
            out = torch.empty_like(u)
        _dev_f64(out, "out")
        arr, keep, nt = descs if descs is not None else self.make_descs(tensors)
        ndof = sum(len(t["fields"]) for t in tensors)
        need = self.workspace_bytes(ndof)[1]
        ws = self._workspace(need, u.device) if workspace is None else _dev_f64(workspace, "workspace")
        _check(lib().sp_tensor_filter(self._h, u.data_ptr(), out.data_ptr(), nf, arr, nt, ws.data_ptr(), ws.numel() * 8,
                                      _stream_ptr(stream)), "sp_tensor_filter")
        return out

    NOALLOC_SCRATCH_BYTES = 32 * 1024 * 1024

    def tensor_filter_noalloc(self, u, tensors, out, stream=None, descs=None):
        """sp_tensor_filter_noalloc: the Yn filter with its scratch in the library's static 32 MiB device array -- no workspace
        argument, no device allocation (the caller passes input and output).  Raises SpError (SP_ERR_SCRATCH_LIMIT) beyond the limit."""
        u = _dev_f64(u, "u")
        _dev_f64(out, "out")
        nf = u.numel() // self.npts
        arr, keep, nt = descs if descs is not None else self.make_descs(tensors)
        _check(lib().sp_tensor_filter_noalloc(self._h, u.data_ptr(), out.data_ptr(), nf, arr, nt, _stream_ptr(stream)),
               "sp_tensor_filter_noalloc")
        return out

    def rhs_first_order_wave(self, u, out=None, workspace=None, stream=None):
        import torch
        u = _dev_f64(u, "u")
        if u.numel() != 5 * self.npts:
            raise SpError("u must hold the 5 fields psi, Pi, Phi_x, Phi_y, Phi_z")
        if out is None:
            out = torch.empty_like(u)
        need = self.workspace_bytes(5)[2]
        ws = self._workspace(need, u.device) if workspace is None else _dev_f64(workspace, "workspace")
        _check(lib().sp_rhs_first_order_wave(self._h, u.data_ptr(), out.data_ptr(), ws.data_ptr(), ws.numel() * 8,
                                             _stream_ptr(stream)), "sp_rhs_first_order_wave")
        return out

    def rhs_wave_shell(self, u, bc_inner=True, bc_outer=True, out=None, workspace=None, stream=None):
        """sp_rhs_wave_shell: the scalar-wave RHS with the freezing condition only on the physical boundary spheres."""
        import torch
        u = _dev_f64(u, "u")
        if u.numel() != 5 * self.npts:
            raise SpError("u must hold the 5 fields psi, Pi, Phi_x, Phi_y, Phi_z")
        if out is None:
            out = torch.empty_like(u)
        need = self.workspace_bytes(5)[2]
        ws = self._workspace(need, u.device) if workspace is None else _dev_f64(workspace, "workspace")
        _check(lib().sp_rhs_wave_shell(self._h, u.data_ptr(), out.data_ptr(), 1 if bc_inner else 0, 1 if bc_outer else 0,
                                       ws.data_ptr(), ws.numel() * 8, _stream_ptr(stream)), "sp_rhs_wave_shell")
        return out

    @staticmethod
    def wave_interface(inner, dudt_inner, outer, dudt_outer, stream=None):
        """sp_wave_interface: characteristic coupling of two shells on their shared sphere (both RHS arrays updated in place)."""
        _dev_f64(dudt_inner, "dudt_inner"); _dev_f64(dudt_outer, "dudt_outer")
        _check(lib().sp_wave_interface(inner._h, dudt_inner.data_ptr(), outer._h, dudt_outer.data_ptr(), _stream_ptr(stream)),
               "sp_wave_interface")

    def wave_dt(self, lam=4.0):
        """dt = lambda * min(dx), eq. 63 (sp_wave_dt)."""
        v = C.c_double()
        _check(lib().sp_wave_dt(self._h, float(lam), C.byref(v)), "sp_wave_dt")
        return v.value

    def ghg_graded_degree(self, field):
        """Kept degree of component `field` under the graded Yg filter, eq. 59 (sp_ghg_graded_degree)."""
        v = C.c_int()
        _check(lib().sp_ghg_graded_degree(self._h, int(field), C.byref(v)), "sp_ghg_graded_degree")
        return v.value

    def ghg_workspace_bytes(self):
        n = C.c_size_t()
        _check(lib().sp_ghg_workspace_bytes(self._h, C.byref(n)), "sp_ghg_workspace_bytes")
        return n.value

    def rhs_ghg(self, u, H, dH, out=None, bc_outer=True, workspace=None, stream=None):
        """GHG right-hand side (A.8)-(A.10) of the 50-field state u [50, Np, Nt, Nr]; H [4, ...], dH [3, 4, ...]."""
        import torch
        for t, nm in ((u, "u"), (H, "H"), (dH, "dH")):
            _dev_f64(t, nm)
        if u.numel() != 50 * self.Np * self.Nt * self.Nr or H.numel() * 3 != dH.numel() or H.numel() * 50 != 4 * u.numel():
            raise ValueError("rhs_ghg: u must hold 50 fields, H 4, dH 12")
        if out is None:
            out = torch.empty_like(u)
        _dev_f64(out, "out")
        nbytes = self.ghg_workspace_bytes()
        ws = workspace if workspace is not None else self._workspace(nbytes, u.device)
        _check(lib().sp_rhs_ghg(self._h, u.data_ptr(), H.data_ptr(), dH.data_ptr(), out.data_ptr(), 1 if bc_outer else 0,
                                ws.data_ptr(), ws.numel() * ws.element_size(), _stream_ptr(stream)), "sp_rhs_ghg")
        return out

    def ghg_init(self, g, stream=None):
        """Initial data of PAPER.md:732-737 from a static metric g [10, Np, Nt, Nr]: d = gradient of g, k by (A.6),
        H = -Gamma (A.18), dH = gradient of H.  Returns (u [50], H [4], dH [3, 4])."""
        import torch
        _dev_f64(g, "g")
        shape = (self.Np, self.Nt, self.Nr)
        u = torch.zeros((50,) + shape, dtype=torch.float64, device=g.device)
        u[:10].copy_(g.reshape((10,) + shape))
        u[20:].copy_(self.cartesian_gradient(u[:10], stream=stream).reshape((30,) + shape))
        H = torch.empty((4,) + shape, dtype=torch.float64, device=g.device)
        _check(lib().sp_ghg_init(self._h, u.data_ptr(), H.data_ptr(), _stream_ptr(stream)), "sp_ghg_init")
        dH = self.cartesian_gradient(H, stream=stream).reshape((3, 4) + shape)
        return u, H, dH

    @staticmethod
    def axpby(a, x, b, y, stream=None):
        """y <- a x + b y (device)."""
        _dev_f64(x, "x"); _dev_f64(y, "y")
        _check(lib().sp_axpby(float(a), x.data_ptr(), float(b), y.data_ptr(), y.numel(), _stream_ptr(stream)), "sp_axpby")
        return y

    @staticmethod
    def rk4_stage(u, k, acc_in, acc_out, stage_out, c_acc, c_stage, stream=None):
        """acc_out <- acc_in + c_acc k;  stage_out <- u + c_stage k (skipped if stage_out is None)."""
        for t, nm in ((u, "u"), (k, "k"), (acc_in, "acc_in"), (acc_out, "acc_out")):
            _dev_f64(t, nm)
        if stage_out is not None:
            _dev_f64(stage_out, "stage_out")
        _check(lib().sp_rk4_stage(u.data_ptr(), k.data_ptr(), acc_in.data_ptr(), acc_out.data_ptr(),
                                  stage_out.data_ptr() if stage_out is not None else None, float(c_acc), float(c_stage),
                                  u.numel(), _stream_ptr(stream)), "sp_rk4_stage")
