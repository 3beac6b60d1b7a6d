"""ctypes binding of the fp64 CPU oracle (oracle/ssm_oracle.c).

TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It shares nothing with
the CUDA path under paper_1106_2899_b200/ and never imports it.

All arithmetic of the method lives in ssm_oracle.c; this file only marshals arguments.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ssm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_ssm.so")

DOM_NOISE, DOM_SLOT, DOM_ATTEMPT, DOM_ANCHOR = 0, 1, 2, 3
DOM_INIT_BOND, DOM_INIT_Z, DOM_INIT_SLOT, DOM_INIT_ANCHOR = 4, 5, 6, 7
K_EMPTY, K_ONE = 0, 1


def build(force=False):
    """Compile the oracle with gcc (no fast-math, no FMA contraction).  ORACLE_SANITIZE=1 in the environment builds
    it with -fsanitize=address,undefined into a library of its own (run the tests with libasan preloaded:
    LD_PRELOAD=$(gcc -print-file-name=libasan.so) ORACLE_SANITIZE=1 python -m pytest tests -m "not gpu" -k oracle)."""
    global _LIB
    san = os.environ.get("ORACLE_SANITIZE") == "1"
    if san:
        _LIB = os.path.join(_HERE, "liboracle_ssm_san.so")
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC),
                                              os.path.getmtime(os.path.join(_HERE, "ssm_oracle.h")))):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared", "-pthread"] \
        + (["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if san else []) \
        + ["-o", _LIB, _SRC, "-lm"]
    subprocess.check_call(cmd)
    return _LIB


class Params(C.Structure):
    _fields_ = [("n_beads", C.c_int32), ("n_chains", C.c_int64), ("z_max", C.c_int32),
                ("n_s", C.c_double), ("n_0", C.c_double), ("zeta_s", C.c_double), ("dt", C.c_double),
                ("seed", C.c_uint64), ("k_mode", C.c_int32), ("chain_offset", C.c_uint64),
                ("noise_bits", C.c_int32)]


class State(C.Structure):
    _fields_ = [("R", C.POINTER(C.c_double)), ("A", C.POINTER(C.c_double)),
                ("S", C.POINTER(C.c_int32)), ("Z", C.POINTER(C.c_int32)), ("step", C.c_int64),
                ("first_fragile_step", C.POINTER(C.c_int64)), ("min_margin", C.POINTER(C.c_double))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, dp, i32p, i64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_double),
                                C.POINTER(C.c_int32), C.POINTER(C.c_int64))
        PP = C.POINTER(Params)
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_stream.argtypes = [C.c_uint64, C.c_int, C.c_uint64, C.c_uint64, C.c_uint32, u32p]
        L.oracle_code23.argtypes = [C.c_uint32]; L.oracle_code23.restype = C.c_uint32
        L.oracle_u23.argtypes = [C.c_uint32]; L.oracle_u23.restype = C.c_double
        L.oracle_threshold23.argtypes = [C.c_double]; L.oracle_threshold23.restype = C.c_int64
        L.oracle_box_muller.argtypes = [C.c_uint32, dp]
        L.oracle_box_muller23.argtypes = [C.c_uint32, C.c_uint32, dp]
        L.oracle_stream_normal.argtypes = [C.c_uint64, C.c_int, C.c_uint64, C.c_uint64, C.c_uint32]
        L.oracle_stream_normal.restype = C.c_double
        L.oracle_zmax.argtypes = [PP]; L.oracle_zmax.restype = C.c_int
        L.oracle_hop_probabilities.argtypes = [PP, dp, dp, C.c_int, dp, dp]
        L.oracle_chain_stress.argtypes = [PP, dp, dp, i32p, C.c_int, dp, dp]
        L.oracle_poisson_thresholds.argtypes = [PP, i64p]
        L.oracle_init_chain.argtypes = [PP, C.c_uint64, dp, dp, i32p, i32p]
        L.oracle_step_chain.argtypes = [PP, C.c_uint64, C.c_uint64, C.c_double, dp, dp, i32p, i32p, dp]
        L.oracle_corr_create.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int]
        L.oracle_corr_create.restype = C.c_void_p
        L.oracle_corr_create_iso.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int]
        L.oracle_corr_create_iso.restype = C.c_void_p
        L.oracle_corr_destroy.argtypes = [C.c_void_p]
        L.oracle_corr_push.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_double, C.c_double]
        L.oracle_corr_sums.argtypes = [C.c_void_p, dp, dp, i64p]
        L.oracle_corr_result.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int, dp, dp, dp]
        L.oracle_corr_result.restype = C.c_int
        L.oracle_corr_result_virtual.argtypes = [C.c_void_p, C.c_double, C.c_int, dp, dp, dp]
        L.oracle_corr_result_virtual.restype = C.c_int
        L.oracle_run.argtypes = [PP, C.POINTER(State), C.c_int64, C.c_double, C.c_int, dp, C.c_int,
                                 C.c_void_p, C.c_double, C.c_int]
        L.oracle_run.restype = C.c_int64
        L.oracle_step_chain_kappa.argtypes = [PP, C.c_uint64, C.c_uint64, dp, dp, dp, i32p, i32p, dp]
        L.oracle_run_kappa.argtypes = [PP, C.POINTER(State), C.c_int64, C.c_int64, dp, C.c_int, dp, C.c_int,
                                       C.c_void_p, C.c_double, C.c_int]
        L.oracle_run_kappa.restype = C.c_int64
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def stream(seed, domain, step, chain, item):
    o = (C.c_uint32 * 4)()
    lib().oracle_stream(seed, domain, step, chain, item, o)
    return [int(x) for x in o]


def u23(w):
    return lib().oracle_u23(w)


def threshold23(p):
    return lib().oracle_threshold23(p)


def box_muller(w):
    """Two normals from one Philox word (16-bit codes in its low and high half)."""
    z = (C.c_double * 2)()
    lib().oracle_box_muller(w, z)
    return z[0], z[1]


def box_muller23(wa, wb):
    """Two normals from two Philox words at 23-bit resolution (the oracle's noise_bits = 23 law)."""
    z = (C.c_double * 2)()
    lib().oracle_box_muller23(wa, wb, z)
    return z[0], z[1]


def stream_normal(seed, domain, step, chain, m):
    return lib().oracle_stream_normal(seed, domain, step, chain, m)


class Correlator:
    """Per-chain multi-tau correlator."""

    def __init__(self, n_chains, levels=16, bins=16, groups=32, components=1):
        self.h = lib().oracle_corr_create_iso(n_chains, levels, bins, groups, components)
        self.levels, self.bins, self.groups = levels, bins, groups

    def push(self, chain_local, group, f, g):
        lib().oracle_corr_push(self.h, chain_local, group, f, g)

    def sums(self):
        """Raw accumulators [groups][levels][bins]: (sum f_new g_old, sum g_new g_old, product counts)."""
        shape = (self.groups, self.levels, self.bins)
        s = np.zeros(shape); gg = np.zeros(shape); c = np.zeros(shape, dtype=np.int64)
        lib().oracle_corr_sums(self.h, _dp(s), _dp(gg), c.ctypes.data_as(C.POINTER(C.c_int64)))
        return s, gg, c

    def result(self, n_beads, base_dt):
        cap = self.levels * self.bins
        t = np.zeros(cap); G = np.zeros(cap); se = np.zeros(cap)
        n = lib().oracle_corr_result(self.h, n_beads, base_dt, cap, _dp(t), _dp(G), _dp(se))
        assert n >= 0
        return t[:n].copy(), G[:n].copy(), se[:n].copy()

    def result_virtual(self, base_dt):
        """eq 66: relative contribution of the virtual stress to G(t), with its standard error."""
        cap = self.levels * self.bins
        t = np.zeros(cap); d = np.zeros(cap); se = np.zeros(cap)
        n = lib().oracle_corr_result_virtual(self.h, base_dt, cap, _dp(t), _dp(d), _dp(se))
        assert n >= 0
        return t[:n].copy(), d[:n].copy(), se[:n].copy()

    def __del__(self):
        if getattr(self, "h", None):
            lib().oracle_corr_destroy(self.h); self.h = None


class Ensemble:
    """M chains held as numpy fp64 arrays R[M][N][3], A[M][zmax][3], S[M][zmax], Z[M]."""

    def __init__(self, n_beads, n_chains, n_s=0.5, n_0=4.0, zeta_s=0.1, dt=0.01, seed=1,
                 z_max=0, k_mode=K_EMPTY, chain_offset=0, init=True, noise_bits=16):
        # noise_bits = 23: the full-resolution noise law (no GPU counterpart; the A/B pin of DESIGN.md reading R24)
        assert noise_bits in (16, 23)
        self.p = Params(n_beads, n_chains, z_max, n_s, n_0, zeta_s, dt, seed, k_mode, chain_offset, noise_bits)
        self.N, self.M = n_beads, n_chains
        self.zmax = lib().oracle_zmax(C.byref(self.p))
        self.R = np.zeros((n_chains, n_beads, 3)); self.A = np.zeros((n_chains, self.zmax, 3))
        self.S = np.zeros((n_chains, self.zmax), dtype=np.int32); self.Z = np.zeros(n_chains, dtype=np.int32)
        self.first_fragile = np.full(n_chains, -1, dtype=np.int64)
        self.min_margin = np.full(n_chains, np.inf)
        self.step = 0
        if init:
            self.init_equilibrium()

    def init_equilibrium(self):
        L = lib()
        z = C.c_int32()
        for k in range(self.M):
            L.oracle_init_chain(C.byref(self.p), self.p.chain_offset + k, _dp(self.R[k]), _dp(self.A[k]),
                                _ip(self.S[k]), C.byref(z))
            self.Z[k] = z.value

    def round_to_fp32(self):
        """Reading R19: parity runs start from the fp32-rounded state on both sides."""
        self.R[:] = self.R.astype(np.float32).astype(np.float64)
        self.A[:] = self.A.astype(np.float32).astype(np.float64)

    def _state(self):
        return State(_dp(self.R), _dp(self.A), _ip(self.S), _ip(self.Z), self.step,
                     self.first_fragile.ctypes.data_as(C.POINTER(C.c_int64)), _dp(self.min_margin))

    def run(self, n_steps, shear_rate=0.0, stress_every=0, sample_every=0, corr=None, guard=1e-5,
            n_threads=1):
        """Advance n_steps; returns stress means [n_samples][12] (sigma[6], sigma_v[6])."""
        ns = 0
        if stress_every > 0:
            ns = (self.step + n_steps) // stress_every - self.step // stress_every
        out = np.zeros((max(ns, 1), 12))
        st = self._state()
        got = lib().oracle_run(C.byref(self.p), C.byref(st), n_steps, shear_rate, stress_every, _dp(out),
                               sample_every, corr.h if corr is not None else None, guard, n_threads)
        assert got == ns
        self.step = st.step
        return out[:ns]

    def run_kappa(self, n_steps, kappa, chains_per_group=None, stress_every=0, sample_every=0, corr=None,
                  guard=1e-5, n_threads=1):
        """As run(), under a general velocity gradient (eqs 18, 21): kappa [groups][3][3] (or one [3][3]),
        group of local chain k = k // chains_per_group (default: one group)."""
        cpg = self.M if chains_per_group is None else int(chains_per_group)
        kap = np.ascontiguousarray(np.asarray(kappa, dtype=np.float64).reshape(-1, 9))
        assert kap.shape[0] == -(-self.M // cpg)
        ns = 0
        if stress_every > 0:
            ns = (self.step + n_steps) // stress_every - self.step // stress_every
        out = np.zeros((max(ns, 1), 12))
        st = self._state()
        got = lib().oracle_run_kappa(C.byref(self.p), C.byref(st), n_steps, cpg, _dp(kap), stress_every, _dp(out),
                                     sample_every, corr.h if corr is not None else None, guard, n_threads)
        assert got == ns
        self.step = st.step
        return out[:ns]

    def chain_stress(self, k):
        sig = np.zeros(6); sv = np.zeros(6)
        lib().oracle_chain_stress(C.byref(self.p), _dp(self.R[k]), _dp(self.A[k]), _ip(self.S[k]),
                                  int(self.Z[k]), _dp(sig), _dp(sv))
        return sig, sv

    def hop_probabilities(self, k, j):
        pp = C.c_double(); pm = C.c_double()
        a = np.ascontiguousarray(self.A[k, j])
        lib().oracle_hop_probabilities(C.byref(self.p), _dp(self.R[k]), _dp(a), int(self.S[k, j]),
                                       C.byref(pp), C.byref(pm))
        return pp.value, pm.value
