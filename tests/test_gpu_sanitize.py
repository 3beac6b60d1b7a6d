"""Smoke-sized pass over every kernel of libssm -- the step kernel at G = 1, 4, 16 with no flow, simple shear and
a velocity-gradient tensor, a ragged bead number, the sampler, the state import / export, the correlator, the
per-chain / per-group stress, recentring -- small enough to run under compute-sanitizer:

    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitize.py -m gpu -q      (memcheck, initcheck alike)

("race detection / sanitizers"; the shared-memory scatter of P:L376's fixed-point atomics and the
warp-private shared memory synchronised by __syncwarp are what racecheck is asked about.)  Summaries of those runs:
profiles/r2_sanitizers.md.  As an ordinary test it checks that everything stays finite and the bookkeeping adds up."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,M", [(8, 70), (20, 37), (32, 50), (128, 5)])
def test_every_kernel_once(N, M):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1106_2899_b200 as ssm
    g = ssm.Ensemble(N, M, seed=3, stress_every=1, stress_capacity=200, sample_every=5, corr_levels=3, corr_bins=8,
                     corr_groups=4, corr_components=3 if N == 8 else 1, stage_chains=16)
    g.step(33)                                                   # FLOW 0, two launches (32 + 1)
    g.step(9, shear_rate=0.2)                                    # FLOW 1
    kap = np.array([[0.0, 0.3, 0.0], [0.0, 0.0, 0.1], [0.05, 0.0, 0.0]])
    g.step_kappa(9, kap)                                         # FLOW 2 (the low words change encoding: clear kernel)
    g.step(5, shear_rate=0.2)
    dk = torch.tensor(kap, dtype=torch.float64, device="cuda").reshape(1, 3, 3).contiguous()
    g.step_kappa_device(4, dk)
    assert g.stress_count() == 60
    s = g.stress()
    assert np.all(np.isfinite(s)) and np.all(np.isfinite(g.stress_sums().astype(np.float64)))
    t, G, se = g.gt()
    assert len(t) > 0 and np.all(np.isfinite(G))
    assert np.all(np.isfinite(g.gt_virtual()[1][:1]))
    R, A, S, step = g.get_state()                                # export through the staging area, chunks of 16 chains
    assert step == 60 and np.all(np.isfinite(R)) and np.all(np.isfinite(A)) and S.max() <= N
    Z = (S > 0).sum(0)
    assert np.array_equal(S > 0, np.arange(N)[:, None] < Z[None, :])
    cs = g.chain_stress()
    gs = g.group_stress()
    assert np.allclose(cs.mean(1), gs[0, :12], rtol=0, atol=1e-3) and abs(gs[0, 12] - Z.mean()) < 1e-9
    assert np.all(np.isfinite(g.group_stress_device().cpu().numpy()))
    g.recenter()
    R2 = g.get_state()[0]
    assert np.all(R2[:, 0, :] == 0.0)
    g.reset_accumulators()
    g.set_state(R, A, S, step)                                   # import (host pointers, chunks)
    dR, dA, dS = [torch.from_numpy(x).cuda() for x in (R, A, S)]
    g.set_state(dR, dA, dS, step)                                # import (device pointers)
    R3, A3, S3, _ = g.get_state(torch.empty_like(dR), torch.empty_like(dA), torch.empty_like(dS))
    assert torch.equal(R3, dR) and torch.equal(S3, dS)
    g.step(3)
    assert g.stress_count() == 3 and g.launch_count() > 10


def test_every_kernel_once_with_device_assertions():
    """The same pass with libssm_check.so (-DSSM_CHECK): every shared-memory and tile index the kernels form is
    tested against its bounds on the device and a violation traps.  The library is chosen when it is first loaded,
    so this runs in a process of its own."""
    import os
    import subprocess
    import sys
    env = dict(os.environ, SSM_LIB="check")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.abspath(__file__), "-m", "gpu", "-q", "-k", "test_every_kernel_once and not assertions",
                        "-p", "no:cacheprovider"], cwd=root, env=env, capture_output=True, text=True)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-2000:]
    assert "4 passed" in r.stdout


def _digest():
    """Hashes of everything a set of small runs leaves behind (state, stress sums, correlator sums), over every G,
    the three kinds of flow, a ragged bead number and the host / device state paths."""
    import hashlib
    import paper_1106_2899_b200 as ssm
    out = []
    kap = np.array([[0.0, 0.3, 0.0], [0.0, 0.0, 0.1], [0.05, 0.0, 0.0]])
    for N, M, kw in ((8, 333, dict(sample_every=5, corr_levels=3, corr_components=3)), (16, 250, dict(k_attempts=1)),
                     (20, 99, dict()), (32, 500, dict(sample_every=10, corr_levels=3)), (64, 60, dict()),
                     (128, 40, dict(dt=0.005))):
        g = ssm.Ensemble(N, M, seed=17, stress_every=1, stress_capacity=400, stage_chains=48, **kw)
        g.step(70)
        g.step(20, shear_rate=0.3)
        g.step_kappa(20, kap)
        R, A, S, step = g.get_state()
        g.set_state(R, A, S, step)                               # through the import kernel and back into the run
        g.step(40)
        R, A, S, _ = g.get_state()
        m = hashlib.sha1()
        for x in (R, A, S, g.stress_sums()) + ((g.gt_sums()[0],) if "sample_every" in kw else ()):
            m.update(np.ascontiguousarray(x).tobytes())
        out.append(m.hexdigest()[:16])
    return out


def test_checked_build_from_poisoned_shared_memory_gives_the_same_bits():
    """libssm_check.so fills the shared memory of the step and the import / export kernels with all-ones words before
    they start (NaN as a float, -1 as an index): if any path read a word nothing had written, its results would
    differ from the product build's.  They are compared bit for bit.  (Stands in for compute-sanitizer's initcheck,
    which the B200 pool this was developed on does not run; profiles/r2_sanitizers.md.)"""
    import json
    import os
    import subprocess
    import sys
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    mine = _digest()
    env = dict(os.environ, SSM_LIB="check")
    code = ("import json, sys, importlib.util; sys.path.insert(0, %r); "
            "sp = importlib.util.spec_from_file_location('sanitize_digest', %r); t = importlib.util.module_from_spec(sp); "
            "sp.loader.exec_module(t); import paper_1106_2899_b200 as ssm; "
            "assert ssm.lib()._name.endswith('libssm_check.so'), ssm.lib()._name; "
            "print('DIGEST ' + json.dumps(t._digest()))" % (root, os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-3000:]
    theirs = json.loads([l for l in r.stdout.split("\n") if l.startswith("DIGEST ")][-1][7:])
    assert mine == theirs
