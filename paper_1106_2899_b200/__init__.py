"""paper_1106_2899_b200 -- Python binding of libssm.so (include/ssm.h).

Argument marshalling only: every step of the method runs in the CUDA kernels behind the
C ABI.  PyTorch is used for device memory (the workspace, state buffers) and streams.
There is no CPU fallback: importing works without a GPU (so that the library can be built
and its symbols checked), but creating an Ensemble without CUDA raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

SSM_OK, SSM_EINVAL, SSM_ENOMEM, SSM_ECUDA, SSM_ESTATE, SSM_ERANGE = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_GROUPS = 4096          # SSM_NOALLOC_MAX_GROUPS of include/ssm.h

EXPORTS = ["ssm_workspace_bytes", "ssm_init", "ssm_step", "ssm_stress_count", "ssm_stress", "ssm_stress_sums",
           "ssm_stress_sums_device", "ssm_chain_stress", "ssm_gt", "ssm_gt_sums", "ssm_get_state", "ssm_set_state",
           "ssm_reset_accumulators", "ssm_launch_count", "ssm_set_fusion", "ssm_set_grid", "ssm_destroy", "ssm_last_error",
           "ssm_moduli", "ssm_eta0", "ssm_tau_d", "ssm_issue_rates8",
           "ssm_gt_virtual", "ssm_gt_sums_virtual", "ssm_step_kappa", "ssm_group_stress",
           "ssm_step_kappa_device", "ssm_group_stress_device", "ssm_recenter",
           "ssm_eta_star", "ssm_stress_from_sums", "ssm_stream_wait_ctx", "ssm_ctx_wait_stream", "ssm_step_from_host",
           "ssm_group_stress_noalloc", "ssm_noise_calibration", "ssm_state_status"]


class Params(C.Structure):
    """ssm_params of include/ssm.h."""
    _fields_ = [("n_beads", C.c_int32), ("n_chains", C.c_int64), ("n_s", C.c_double), ("n_0", C.c_double),
                ("zeta_s", C.c_double), ("dt", C.c_double), ("seed", C.c_uint64), ("chain_offset", C.c_uint64),
                ("stress_every", C.c_int32), ("stress_capacity", C.c_int64), ("sample_every", C.c_int32),
                ("corr_levels", C.c_int32), ("corr_bins", C.c_int32), ("corr_groups", C.c_int32),
                ("k_attempts", C.c_int32), ("corr_components", C.c_int32), ("stage_chains", C.c_int64)]


class SsmError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("libssm error %d: %s" % (code, text))
        self.code = code


_lib = None


def lib():
    """Load libssm.so (building it with nvcc if missing or stale) and declare prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    # SSM_LIB=check in the environment loads libssm_check.so: the same library with device-side assertions
    path = _build.build(check=os.environ.get("SSM_LIB") == "check")
    L = C.CDLL(path)
    PP, vp, dp, fp = C.POINTER(Params), C.c_void_p, C.POINTER(C.c_double), C.c_void_p
    L.ssm_workspace_bytes.argtypes = [PP]; L.ssm_workspace_bytes.restype = C.c_size_t
    L.ssm_init.argtypes = [C.POINTER(vp), PP, vp, C.c_size_t, vp]; L.ssm_init.restype = C.c_int
    L.ssm_step.argtypes = [vp, C.c_int64, C.c_double]; L.ssm_step.restype = C.c_int
    L.ssm_stress_count.argtypes = [vp]; L.ssm_stress_count.restype = C.c_int64
    L.ssm_stress.argtypes = [vp, C.c_int64, C.c_int64, dp]; L.ssm_stress.restype = C.c_int
    L.ssm_stress_sums.argtypes = [vp, C.c_int64, C.c_int64, C.POINTER(C.c_int64)]; L.ssm_stress_sums.restype = C.c_int
    L.ssm_stress_sums_device.argtypes = [vp, C.c_int64, C.c_int64, C.POINTER(vp)]; L.ssm_stress_sums_device.restype = C.c_int
    L.ssm_chain_stress.argtypes = [vp, fp, C.c_int]; L.ssm_chain_stress.restype = C.c_int
    L.ssm_gt.argtypes = [vp, C.POINTER(C.c_int32), dp, dp, dp]; L.ssm_gt.restype = C.c_int
    L.ssm_gt_sums.argtypes = [vp, dp, C.POINTER(C.c_int64)]; L.ssm_gt_sums.restype = C.c_int
    L.ssm_get_state.argtypes = [vp, fp, fp, vp, C.POINTER(C.c_int64), C.c_int]; L.ssm_get_state.restype = C.c_int
    L.ssm_set_state.argtypes = [vp, fp, fp, vp, C.c_int64, C.c_int]; L.ssm_set_state.restype = C.c_int
    L.ssm_reset_accumulators.argtypes = [vp]; L.ssm_reset_accumulators.restype = C.c_int
    L.ssm_launch_count.argtypes = [vp]; L.ssm_launch_count.restype = C.c_int64
    L.ssm_set_fusion.argtypes = [vp, C.c_int32]; L.ssm_set_fusion.restype = C.c_int
    L.ssm_set_grid.argtypes = [vp, C.c_int32]; L.ssm_set_grid.restype = C.c_int
    L.ssm_destroy.argtypes = [vp]; L.ssm_destroy.restype = None
    L.ssm_last_error.argtypes = [vp]; L.ssm_last_error.restype = C.c_char_p
    L.ssm_issue_rates8.argtypes = [vp, dp]; L.ssm_issue_rates8.restype = C.c_int
    L.ssm_state_status.argtypes = [vp]; L.ssm_state_status.restype = C.c_int
    L.ssm_gt_virtual.argtypes = [vp, C.POINTER(C.c_int32), dp, dp, dp]; L.ssm_gt_virtual.restype = C.c_int
    L.ssm_gt_sums_virtual.argtypes = [vp, dp]; L.ssm_gt_sums_virtual.restype = C.c_int
    L.ssm_step_kappa.argtypes = [vp, C.c_int64, C.c_int64, dp]; L.ssm_step_kappa.restype = C.c_int
    L.ssm_group_stress.argtypes = [vp, C.c_int64, dp]; L.ssm_group_stress.restype = C.c_int
    L.ssm_step_kappa_device.argtypes = [vp, C.c_int64, C.c_int64, vp]; L.ssm_step_kappa_device.restype = C.c_int
    L.ssm_group_stress_device.argtypes = [vp, C.c_int64, vp]; L.ssm_group_stress_device.restype = C.c_int
    L.ssm_group_stress_noalloc.argtypes = [vp, C.c_int64, vp]; L.ssm_group_stress_noalloc.restype = C.c_int
    L.ssm_recenter.argtypes = [vp]; L.ssm_recenter.restype = C.c_int
    L.ssm_noise_calibration.argtypes = [vp, dp]; L.ssm_noise_calibration.restype = C.c_int
    L.ssm_moduli.argtypes = [C.c_int32, dp, dp, C.c_int32, dp, dp, dp]; L.ssm_moduli.restype = C.c_int
    L.ssm_eta0.argtypes = [C.c_int32, dp, dp, dp]; L.ssm_eta0.restype = C.c_int
    L.ssm_eta_star.argtypes = [C.c_int32, dp, dp, C.c_int32, dp, dp]; L.ssm_eta_star.restype = C.c_int
    L.ssm_stress_from_sums.argtypes = [C.POINTER(C.c_int64), C.c_int64, C.c_int64, dp]; L.ssm_stress_from_sums.restype = C.c_int
    L.ssm_step_from_host.argtypes = [vp, fp, fp, vp, C.c_int64, C.c_int64, C.c_double]; L.ssm_step_from_host.restype = C.c_int
    L.ssm_stream_wait_ctx.argtypes = [vp, vp]; L.ssm_stream_wait_ctx.restype = C.c_int
    L.ssm_ctx_wait_stream.argtypes = [vp, vp]; L.ssm_ctx_wait_stream.restype = C.c_int
    L.ssm_tau_d.argtypes = [C.c_int32, dp, dp, C.c_double, C.c_double, dp]; L.ssm_tau_d.restype = C.c_int
    _lib = L
    return L


def library_path():
    return _build.LIB


def workspace_bytes(params):
    return lib().ssm_workspace_bytes(C.byref(params))


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _ck0(rc, what):
    if rc != SSM_OK:
        raise SsmError(rc, what)


def moduli(t, G, omega):
    """ssm_moduli: (G'(omega), G''(omega)) of a tabulated G(t), eqs 55-56."""
    t, tp = _d(t); G, Gp = _d(G); w, wp = _d(omega)
    g1 = np.zeros(len(w)); g2 = np.zeros(len(w))
    _ck0(lib().ssm_moduli(len(t), tp, Gp, len(w), wp, _d(g1)[1], _d(g2)[1]), "ssm_moduli: bad arguments")
    return g1, g2


def eta_star(t, G, omega):
    """ssm_eta_star: dynamic viscosity sqrt(G'^2 + G''^2) / omega, eq 64 (for the Cox-Merz rule, eq 63)."""
    t, tp = _d(t); G, Gp = _d(G); w, wp = _d(omega)
    out = np.zeros(len(w))
    _ck0(lib().ssm_eta_star(len(t), tp, Gp, len(w), wp, _d(out)[1]), "ssm_eta_star: bad arguments")
    return out


def stress_from_sums(sums, n_chains_total):
    """ssm_stress_from_sums: ensemble means [n][12] from (all-reduced) fixed-point sums [n][12] int64."""
    a = np.ascontiguousarray(sums, dtype=np.int64).reshape(-1, 12)
    out = np.zeros((max(len(a), 1), 12))
    _ck0(lib().ssm_stress_from_sums(a.ctypes.data_as(C.POINTER(C.c_int64)), len(a), int(n_chains_total),
                                    out.ctypes.data_as(C.POINTER(C.c_double))), "ssm_stress_from_sums: bad arguments")
    return out[:len(a)]


def eta0(t, G):
    """ssm_eta0: zero-shear viscosity, eq 59."""
    t, tp = _d(t); G, Gp = _d(G)
    out = C.c_double()
    _ck0(lib().ssm_eta0(len(t), tp, Gp, C.byref(out)), "ssm_eta0: bad arguments")
    return out.value


def tau_d(t, G, t_lo, t_hi):
    """ssm_tau_d: longest relaxation time from the tail slope of ln G(t), eq 58."""
    t, tp = _d(t); G, Gp = _d(G)
    out = C.c_double()
    _ck0(lib().ssm_tau_d(len(t), tp, Gp, float(t_lo), float(t_hi), C.byref(out)), "ssm_tau_d: bad arguments or no decaying tail in the window")
    return out.value


class Ensemble:
    """M chains on one GPU.  Thin wrapper: each method is one C-ABI call of the same name."""

    def __init__(self, n_beads, n_chains, n_s=0.5, n_0=4.0, zeta_s=0.1, dt=0.01, seed=1, chain_offset=0,
                 stress_every=0, stress_capacity=0, sample_every=0, corr_levels=16, corr_bins=16,
                 corr_groups=32, k_attempts=0, corr_components=1, stage_chains=0, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise SsmError(SSM_ECUDA, "no CUDA device: libssm has no CPU fallback")
        self._torch = torch
        self.device = torch.device(device)
        self.p = Params(n_beads, n_chains, n_s, n_0, zeta_s, dt, seed, chain_offset, stress_every,
                        stress_capacity, sample_every, corr_levels, corr_bins, corr_groups, k_attempts, corr_components,
                        stage_chains)
        self.N, self.M = n_beads, n_chains
        L = lib()
        nbytes = L.ssm_workspace_bytes(C.byref(self.p))
        if nbytes == 0:
            raise SsmError(SSM_EINVAL, L.ssm_last_error(None).decode())
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = L.ssm_init(C.byref(h), C.byref(self.p), C.c_void_p(base), nbytes, C.c_void_p(self.stream.cuda_stream))
        if rc != SSM_OK:
            raise SsmError(rc, L.ssm_last_error(None).decode())
        self.h = h

    def _ck(self, rc):
        if rc != SSM_OK:
            raise SsmError(rc, lib().ssm_last_error(self.h).decode())

    def _dev(self):
        """Every call of the C ABI runs with the context's device current (its kernels and copies go there)."""
        return self._torch.cuda.device(self.device)

    def step(self, n_steps, shear_rate=0.0):
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_step(self.h, n_steps, shear_rate))

    def step_kappa(self, n_steps, kappa, chains_per_group=None):
        """ssm_step_kappa: kappa [groups][3][3] (or one [3][3]); group of local chain k = k // chains_per_group."""
        cpg = self.M if chains_per_group is None else int(chains_per_group)
        kap = np.ascontiguousarray(np.asarray(kappa, dtype=np.float64).reshape(-1, 9))
        if kap.shape[0] != -(-self.M // min(cpg, self.M)):
            raise SsmError(SSM_EINVAL, "kappa must hold one tensor per group")
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_step_kappa(self.h, n_steps, cpg, kap.ctypes.data_as(C.POINTER(C.c_double))))

    def step_kappa_device(self, n_steps, kappa, chains_per_group=None):
        """ssm_step_kappa_device: kappa = CUDA float64 tensor [groups][3][3]; asynchronous."""
        cpg = self.M if chains_per_group is None else int(chains_per_group)
        assert kappa.is_cuda and kappa.dtype == self._torch.float64 and kappa.is_contiguous()
        assert kappa.numel() == 9 * -(-self.M // min(cpg, self.M))
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_step_kappa_device(self.h, n_steps, cpg, C.c_void_p(kappa.data_ptr())))

    def group_stress_device(self, chains_per_group=None, out=None):
        """ssm_group_stress_device: fills / returns a CUDA float64 tensor [groups][13]; asynchronous."""
        cpg = self.M if chains_per_group is None else min(int(chains_per_group), self.M)
        ng = -(-self.M // cpg)
        if out is None:
            out = self._torch.empty((ng, 13), dtype=self._torch.float64, device=self.device)
        assert out.is_cuda and out.dtype == self._torch.float64 and out.is_contiguous() and out.numel() == ng * 13
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_group_stress_device(self.h, cpg, C.c_void_p(out.data_ptr())))
        return out

    def group_stress_noalloc(self, chains_per_group=None, out=None):
        """ssm_group_stress_noalloc: group_stress_device for callers that may not allocate device memory and have no
        scratch to lend (a plug-in inside an application whose memory pool owns the GPU, a loop that cannot afford
        cudaMalloc's device-wide stall).  The intermediate sums sit in a fixed array inside libssm.so, so at most
        NOALLOC_MAX_GROUPS (4096) groups (SsmError SSM_ERANGE beyond), and calls whose GPU work overlaps race on it:
        keep them on one stream.  Fills `out`, a CUDA float64 tensor [groups][13] that the CALLER passes (unlike
        group_stress_device, this method does not create one: that would be an allocation); asynchronous."""
        cpg = self.M if chains_per_group is None else min(int(chains_per_group), self.M)
        ng = -(-self.M // cpg)
        if out is None:
            raise SsmError(SSM_EINVAL, "group_stress_noalloc: pass the output tensor (this call allocates nothing)")
        assert out.is_cuda and out.dtype == self._torch.float64 and out.is_contiguous() and out.numel() == ng * 13
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_group_stress_noalloc(self.h, cpg, C.c_void_p(out.data_ptr())))
        return out

    def recenter(self):
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_recenter(self.h))

    def group_stress(self, chains_per_group=None):
        """ssm_group_stress: [groups][13] = means of sigma[6], sigma_v[6] and Z over each group, current state."""
        cpg = self.M if chains_per_group is None else min(int(chains_per_group), self.M)
        out = np.zeros((-(-self.M // cpg), 13))
        with self._torch.cuda.device(self.device):
            self._ck(lib().ssm_group_stress(self.h, cpg, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def stress_count(self):
        return lib().ssm_stress_count(self.h)

    def stress(self, first=0, n=None):
        with self._dev():
            n = self.stress_count() - first if n is None else n
            out = np.zeros((max(n, 1), 12))
            self._ck(lib().ssm_stress(self.h, first, n, out.ctypes.data_as(C.POINTER(C.c_double))))
            return out[:n]

    def stress_sums(self, first=0, n=None):
        with self._dev():
            n = self.stress_count() - first if n is None else n
            out = np.zeros((max(n, 1), 12), dtype=np.int64)
            self._ck(lib().ssm_stress_sums(self.h, first, n, out.ctypes.data_as(C.POINTER(C.c_int64))))
            return out[:n]

    def stress_sums_device(self, first=0, n=None):
        """int64 CUDA tensor [n][12] aliasing the fixed-point sums inside the workspace."""
        n = self.stress_count() - first if n is None else n
        p = C.c_void_p()
        self._ck(lib().ssm_stress_sums_device(self.h, first, n, C.byref(p)))
        off = (p.value or 0) - self.workspace.data_ptr()
        return self.workspace[off:off + n * 96].view(self._torch.int64).view(n, 12)

    def chain_stress(self, out=None):
        """[12][M] float32: numpy (host) by default, or fill a given CUDA tensor."""
        with self._dev():
            if out is None:
                a = np.zeros((12, self.M), dtype=np.float32)
                self._ck(lib().ssm_chain_stress(self.h, C.c_void_p(a.ctypes.data), 0))
                return a
            self._ck(lib().ssm_chain_stress(self.h, C.c_void_p(out.data_ptr()), 1))
            return out

    def gt_virtual(self):
        """ssm_gt_virtual: (lag times, dGv(t) of eq 66, standard error)."""
        with self._dev():
            cap = self.p.corr_levels * self.p.corr_bins
            n = C.c_int32(cap)
            t = np.zeros(cap); d = np.zeros(cap); se = np.zeros(cap)
            dd = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
            self._ck(lib().ssm_gt_virtual(self.h, C.byref(n), dd(t), dd(d), dd(se)))
            return t[:n.value].copy(), d[:n.value].copy(), se[:n.value].copy()

    def gt(self):
        with self._dev():
            cap = self.p.corr_levels * self.p.corr_bins
            n = C.c_int32(cap)
            t = np.zeros(cap); G = np.zeros(cap); se = np.zeros(cap)
            d = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
            self._ck(lib().ssm_gt(self.h, C.byref(n), d(t), d(G), d(se)))
            return t[:n.value].copy(), G[:n.value].copy(), se[:n.value].copy()

    def gt_sums(self):
        with self._dev():
            shape = (self.p.corr_groups, self.p.corr_levels, self.p.corr_bins)
            s = np.zeros(shape); c = np.zeros(shape, dtype=np.int64)
            self._ck(lib().ssm_gt_sums(self.h, s.ctypes.data_as(C.POINTER(C.c_double)),
                                       c.ctypes.data_as(C.POINTER(C.c_int64))))
            return s, c

    def get_state(self, R=None, A=None, S=None):
        """External SoA layout: R[3][N][M], A[4][N][M] float32 (x, y, z, low part of x), S[N][M] uint8.  Host numpy
        arrays by default; pass CUDA tensors (all three) to stay on the device."""
        with self._dev():
            step = C.c_int64()
            if R is None:
                R = np.zeros((3, self.N, self.M), dtype=np.float32); A = np.zeros((4, self.N, self.M), dtype=np.float32)
                S = np.zeros((self.N, self.M), dtype=np.uint8)
                self._ck(lib().ssm_get_state(self.h, C.c_void_p(R.ctypes.data), C.c_void_p(A.ctypes.data),
                                             C.c_void_p(S.ctypes.data), C.byref(step), 0))
            elif isinstance(R, np.ndarray):
                self._ck(lib().ssm_get_state(self.h, C.c_void_p(R.ctypes.data), C.c_void_p(A.ctypes.data),
                                             C.c_void_p(S.ctypes.data), C.byref(step), 0))
            else:
                dev = 1 if R.is_cuda else 0
                self._ck(lib().ssm_get_state(self.h, C.c_void_p(R.data_ptr()), C.c_void_p(A.data_ptr()),
                                             C.c_void_p(S.data_ptr()), C.byref(step), dev))
            return R, A, S, step.value

    def set_state(self, R, A, S, global_step):
        with self._dev():
            if isinstance(R, np.ndarray):
                assert R.dtype == np.float32 and A.dtype == np.float32 and S.dtype == np.uint8
                assert R.flags.c_contiguous and A.flags.c_contiguous and S.flags.c_contiguous
                assert R.shape == (3, self.N, self.M) and A.shape == (4, self.N, self.M) and S.shape == (self.N, self.M)
                self._ck(lib().ssm_set_state(self.h, C.c_void_p(R.ctypes.data), C.c_void_p(A.ctypes.data),
                                             C.c_void_p(S.ctypes.data), global_step, 0))
            else:
                dev = 1 if R.is_cuda else 0
                self._ck(lib().ssm_set_state(self.h, C.c_void_p(R.data_ptr()), C.c_void_p(A.data_ptr()),
                                             C.c_void_p(S.data_ptr()), global_step, dev))

    def state_status(self):
        """ssm_state_status: synchronises; raises SsmError(SSM_EINVAL) if a state imported from device pointers since the
        last check had a malformed S."""
        with self._dev():
            self._ck(lib().ssm_state_status(self.h))

    def step_from_host(self, R, A, S, global_step, n_steps, shear_rate=0.0):
        """ssm_step_from_host: upload the state from host numpy arrays (pinned for overlap) and advance n_steps, pipelined."""
        assert R.dtype == np.float32 and A.dtype == np.float32 and S.dtype == np.uint8
        assert R.flags.c_contiguous and A.flags.c_contiguous and S.flags.c_contiguous
        assert R.shape == (3, self.N, self.M) and A.shape == (4, self.N, self.M) and S.shape == (self.N, self.M)
        with self._dev():
            self._ck(lib().ssm_step_from_host(self.h, C.c_void_p(R.ctypes.data), C.c_void_p(A.ctypes.data),
                                              C.c_void_p(S.ctypes.data), global_step, n_steps, shear_rate))

    def reset_accumulators(self):
        with self._dev():
            self._ck(lib().ssm_reset_accumulators(self.h))

    def launch_count(self):
        return lib().ssm_launch_count(self.h)

    def set_fusion(self, steps_per_launch):
        self._ck(lib().ssm_set_fusion(self.h, steps_per_launch))

    def issue_rates(self):
        """ssm_issue_rates8 (diagnostic): cycles per instruction group per scheduler; imad_wide = the issue cycles one
        32 x 32 -> 64-bit multiply occupies inside a Philox round (the round's cycles minus one slot for each of its
        two LOP3, halved)."""
        out = np.zeros(8)
        with self._dev():
            self._ck(lib().ssm_issue_rates8(self.h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return {"ffma": out[0], "alu": out[1], "imad": out[2], "imad_wide": 0.5 * (out[7] - 2.0), "wide_lop3": out[3],
                "wide_lop3_4ffma": out[4], "mufu": out[5], "i2f_f2i": out[6], "philox_round": out[7]}

    def noise_calibration(self):
        """ssm_noise_calibration (diagnostic): what ssm_init's Box-Muller calibration found for the thermal noise."""
        out = np.zeros(8)
        self._ck(lib().ssm_noise_calibration(self.h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return {"bm_plain": out[0], "bm_used": out[1], "variance_error_plain": out[2], "variance_error_used": out[3],
                "cos2_bias": out[4], "sin2_bias": out[5], "ulps_moved": int(out[6])}

    def stream_wait_ctx(self, stream):
        """ssm_stream_wait_ctx: later work on `stream` (a torch.cuda.Stream) waits for this context's queued work."""
        with self._dev():
            self._ck(lib().ssm_stream_wait_ctx(self.h, C.c_void_p(stream.cuda_stream)))

    def ctx_wait_stream(self, stream):
        """ssm_ctx_wait_stream: this context's later work waits for what is queued on `stream` so far."""
        with self._dev():
            self._ck(lib().ssm_ctx_wait_stream(self.h, C.c_void_p(stream.cuda_stream)))

    def set_grid(self, blocks):
        self._ck(lib().ssm_set_grid(self.h, blocks))

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "h", None):
            lib().ssm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
