"""The C-ABI boundary without a GPU: libssm.so builds, loads, and exports every symbol
include/ssm.h declares; parameter checking and the workspace size are host logic."""
import ctypes as C
import os
import re

import pytest

import paper_1106_2899_b200 as m

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "ssm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ssm_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound():
    names = _declared_symbols()
    assert "ssm_init" in names and "ssm_step" in names and "ssm_stress" in names and "ssm_gt" in names
    L = m.lib()
    for n in names:
        assert hasattr(L, n), "libssm.so does not export %s" % n
    assert sorted(m.EXPORTS) == names, "python binding and header disagree"


def test_params_struct_matches_header_layout():
    # field order and types as in include/ssm.h; natural alignment on x86-64
    p = m.Params
    assert [f[0] for f in p._fields_] == ["n_beads", "n_chains", "n_s", "n_0", "zeta_s", "dt", "seed",
                                          "chain_offset", "stress_every", "stress_capacity", "sample_every",
                                          "corr_levels", "corr_bins", "corr_groups", "k_attempts",
                                          "corr_components", "stage_chains"]
    # ask the C compiler what the header says
    import subprocess
    import tempfile
    names = [f[0] for f in p._fields_]
    src = '#include <stdio.h>\n#include <stddef.h>\n#include "ssm.h"\nint main(void){printf("%zu", sizeof(ssm_params));' \
        + "".join('printf(" %%zu", offsetof(ssm_params, %s));' % n for n in names) + "return 0;}\n"
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "t.c"), "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(d, "t"), os.path.join(d, "t.c")])
        out = [int(x) for x in subprocess.check_output([os.path.join(d, "t")]).split()]
    assert C.sizeof(p) == out[0]
    assert [getattr(p, n).offset for n in names] == out[1:]


def _params(**kw):
    d = dict(n_beads=32, n_chains=1000, n_s=0.5, n_0=4.0, zeta_s=0.1, dt=0.01, seed=1, chain_offset=0,
             stress_every=1, stress_capacity=10, sample_every=0, corr_levels=16, corr_bins=16, corr_groups=32,
             k_attempts=0, corr_components=1, stage_chains=0)
    d.update(kw)
    return m.Params(**d)


def test_workspace_bytes_and_parameter_checks():
    n = m.workspace_bytes(_params())
    # 1000 chains of N=32: 125 warp tiles (8 chains each) of 7552 B, plus stress and staging
    assert n >= 125 * 7552 + 10 * 96
    assert m.workspace_bytes(_params(n_chains=2000)) > n
    assert m.workspace_bytes(_params(sample_every=10)) > n + 1000 * 16 * 16 * 4
    # any bead number 2..128 is accepted: N = 20 takes the 32 bead places per chain of N = 32
    assert m.workspace_bytes(_params(n_beads=20)) == n
    for bad in (dict(n_beads=1), dict(n_beads=129), dict(n_beads=256), dict(n_chains=0), dict(dt=0.0), dict(dt=0.2), dict(n_s=0.0),
                dict(zeta_s=-1.0), dict(stress_capacity=0), dict(sample_every=10, corr_bins=15),
                dict(sample_every=10, corr_levels=0), dict(chain_offset=2**32), dict(k_attempts=-1),
                dict(sample_every=10, corr_components=2), dict(stage_chains=-1)):
        assert m.workspace_bytes(_params(**bad)) == 0, bad
        assert len(m.lib().ssm_last_error(None)) > 0


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(m.SsmError):
        m.Ensemble(32, 16)
    # the C ABI itself refuses too
    h = C.c_void_p()
    p = _params(n_chains=16)
    need = m.lib().ssm_workspace_bytes(C.byref(p))
    buf = C.create_string_buffer(need + 256)
    base = (C.addressof(buf) + 255) // 256 * 256
    rc = m.lib().ssm_init(C.byref(h), C.byref(p), C.c_void_p(base), need, None)
    assert rc == m.SSM_ECUDA
    assert b"no CUDA device" in m.lib().ssm_last_error(None)


def test_null_ctx_calls_fail_cleanly():
    L = m.lib()
    assert L.ssm_step(None, 1, 0.0) == m.SSM_EINVAL
    assert L.ssm_stress_count(None) == 0
    assert L.ssm_reset_accumulators(None) == m.SSM_EINVAL
    L.ssm_destroy(None)


def test_round3_entry_points_check_their_arguments_without_a_gpu():
    """NULL contexts and outputs are refused before any CUDA call (no device needed): the no-allocation group stress,
    the deferred state verdict and the calibration record."""
    L = m.lib()
    assert L.ssm_group_stress_noalloc(None, 1, None) == m.SSM_EINVAL
    assert L.ssm_state_status(None) == m.SSM_EINVAL
    assert L.ssm_noise_calibration(None, None) == m.SSM_EINVAL
    assert m.NOALLOC_MAX_GROUPS == 4096
    text = open(os.path.join(ROOT, "include", "ssm.h")).read()
    assert re.search(r"#define\s+SSM_NOALLOC_MAX_GROUPS\s+4096\b", text)      # header and binding state the same limit
