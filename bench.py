#!/usr/bin/env python
"""bench.py -- throughput of the slip-spring ensemble hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

Workload (BASELINE.json configs[3], "Throughput scaling", the configuration north_star's
target is quoted on): 1,048,576 chains per GPU, N = 32 beads, N_s = 0.5, N_0 = 4,
zeta_s = 0.1, dt = 0.01, no flow, ensemble stress reduced after every time step.
One bench "step" = one pass of the whole hot path (rows a1..a8, a10 of DESIGN.md section 2)
over the ensemble for --inner time steps (default 128) = one ssm_step(inner) call.

Prints ONE JSON line (rank 0).  metric = bead-updates/s summed over all GPUs.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# Frozen algorithmic thread-instruction count per bead-update of the N = 32, <Z> = 8 step
# (DESIGN.md section 9.2).  The roofline numerator is I_ALG x bead-updates/s, NOT the number
# of instructions the kernel happens to execute, so padding cannot raise the fraction.
I_ALG = 95.0
# of which 32 x 32 -> 64-bit multiplies (IMAD.WIDE) of Philox: 0.594 calls x 20.  On B200 each of them holds the issue
# port for about three cycles beyond its own slot (other instructions do not overlap it: profiles/r2_issue_model.md);
# ssm_issue_rates8() measures that cost live for the rate-weighted fraction.
I_ALG_WIDE = 0.59375 * 20.0
N_SM, SMSP_PER_SM, LANES = 148, 4, 32


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--chains", type=int, default=1 << 20, help="chains per GPU")
    ap.add_argument("--beads", type=int, default=32)
    ap.add_argument("--inner", type=int, default=128, help="time steps per bench step")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-contexts", type=int, default=2, help="contexts (streams, host threads) of the e2e leg")
    ap.add_argument("--e2e-steps", type=int, default=0, help="e2e steps per context (0: min(steps, 10), at least 2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=20.0)
    ap.add_argument("--table1", action="store_true",
                    help="context only: the paper's Table 1 shapes (65,536 beads, 1e4 steps) timed on this GPU")
    ap.add_argument("--configs", action="store_true",
                    help="context only: the other BASELINE.json configs (C2, C3, C5 shapes) timed on this GPU, device-resident")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


TRAFFIC_CSV = os.path.join("profiles", "r3_step_kernel_metrics.csv")


def ncu_traffic(n_beads, n_chains):
    """DRAM bytes per launch of the step kernel (dram__bytes_read.sum + dram__bytes_write.sum)
    from the committed `ncu --set full` capture of this workload (NOT measured by this run: a profiler cannot
    run inside a timed bench; the line says where the number comes from); None for other workloads."""
    if (n_beads, n_chains) != (32, 1 << 20):
        return None
    path = os.path.join(ROOT, TRAFFIC_CSV)
    try:
        import csv
        tot = 0.0
        for name, unit, value in csv.reader(open(path)):
            if name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                tot += float(value) * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[unit]
        return tot or None
    except (OSError, ValueError, KeyError):
        return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(float(r[2]) for r in rows)}


def cpu_baseline(n_beads, seconds, threads=None):
    """The fp64 oracle, as it stands, on the host cores: a bounded sample of the same
    workload (same parameters and initial-state law; the rate is intensive in M)."""
    import oracle
    threads = threads or (os.cpu_count() or 1)
    M = 4096
    e = oracle.Ensemble(n_beads, M, seed=4)
    t0 = time.perf_counter(); e.run(4, stress_every=1, n_threads=threads); probe = (time.perf_counter() - t0) / 4
    n = int(max(8, min(20000, seconds / max(probe, 1e-6))))
    t0 = time.perf_counter(); e.run(n, stress_every=1, n_threads=threads); dt = time.perf_counter() - t0
    # once more on ONE thread (the paper's own CPU column is a single thread)
    M1 = 256
    e1 = oracle.Ensemble(n_beads, M1, seed=4)
    n1 = int(max(8, min(20000, 0.25 * seconds / max(probe * threads * M1 / M, 1e-6))))
    t0 = time.perf_counter(); e1.run(n1, stress_every=1, n_threads=1); dt1 = time.perf_counter() - t0
    return {"value": M * n_beads * n / dt, "unit": "bead-updates/s", "cores": threads, "kind": "oracle",
            "sample": "%d chains x N=%d x %d steps, stress every step, %d threads, %.1f s" % (M, n_beads, n, threads, dt),
            "one_thread": {"value": M1 * n_beads * n1 / dt1, "unit": "bead-updates/s", "cores": 1,
                           "sample": "%d chains x N=%d x %d steps, 1 thread, %.1f s" % (M1, n_beads, n1, dt1)}}


def run_reference(a):
    """--impl reference: the oracle on the host cores, same config / metric / unit; each step
    is a bounded sample (4096 chains x inner_ref time steps) of the workload."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    threads = os.cpu_count() or 1
    M = 4096
    e = oracle.Ensemble(a.beads, M, seed=4)
    t0 = time.perf_counter(); e.run(2, stress_every=1, n_threads=threads); probe = (time.perf_counter() - t0) / 2
    budget = 120.0 / max(1, a.steps + a.warmup)                # whole run within a few minutes
    inner = int(max(1, min(a.inner, budget / max(probe, 1e-6))))
    for _ in range(a.warmup):
        e.run(inner, stress_every=1, n_threads=threads)
    t0 = time.perf_counter()
    for _ in range(a.steps):
        e.run(inner, stress_every=1, n_threads=threads)
    dt = time.perf_counter() - t0
    v = M * a.beads * inner * a.steps / dt
    sample = "%d chains x N=%d x %d time steps per step, %d threads" % (M, a.beads, inner, threads)
    print(json.dumps({
        "impl": "reference", "metric": "bead-updates/s", "value": v, "unit": "bead-updates/s", "n_gpus": a.gpus,
        "steps": a.steps, "warmup": a.warmup, "ms_per_step": 1e3 * dt / a.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(a, M, inner, 1),
        "cpu_baseline": {"value": v, "unit": "bead-updates/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "bead-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "chain_steps_per_s": v / a.beads}))


def workload_config(a, chains_per_gpu, inner, world):
    return {"workload": "BASELINE.json configs[3] 'Throughput scaling': %d chains/GPU x N=%d, N_s=0.5, N_0=4, "
                        "zeta_s=0.1, dt=0.01, no flow, stress reduced every step" % (chains_per_gpu, a.beads),
            "chains_per_gpu": chains_per_gpu, "n_beads": a.beads, "time_steps_per_step": inner,
            "global_chains": chains_per_gpu * world, "parallelism": "ensemble-dp%d" % world,
            "l2": ("state (%.0f MB/GPU) is larger than the 126 MB L2; no flush needed" % (chains_per_gpu * 25 * a.beads * 1.04 / 1e6)
                   if a.impl == "ours" else "CPU arm: bounded sample of the workload on the host cores")}


def run_table1():
    """PAPER.md Table 1 (lines 706-719): N x M = 16x4096 .. 128x512 (65,536 beads), dt = 0.01, 1e4 steps
    from the equilibrium start, shear rate 0 and 0.05, K = N - Z.  Context beside the paper's
    own times (Tesla C1060); 65,536 beads are 256 warp tiles and cannot fill a B200."""
    import torch
    import paper_1106_2899_b200 as ssm
    paper = {(16, 0.0): 8.97e-1, (16, 0.05): 8.95e-1, (32, 0.0): 9.02e-1, (32, 0.05): 8.95e-1,
             (64, 0.0): 8.70e-1, (64, 0.05): 8.63e-1, (128, 0.0): 8.45e-1, (128, 0.05): 8.40e-1}
    rows = []
    for N in (16, 32, 64, 128):
        for rate in (0.0, 0.05):
            g = ssm.Ensemble(N, 65536 // N, seed=1)
            g.step(64, rate)                                  # warm-up (and the kernel variant's first launch)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); g.step(10000, rate); e1.record(); torch.cuda.synchronize()
            t = e0.elapsed_time(e1) * 1e-3
            rows.append({"n_beads": N, "n_chains": 65536 // N, "shear_rate": rate, "steps": 10000, "seconds": t,
                         "bead_updates_per_s": 65536 * 1e4 / t, "paper_gpu_seconds": paper[(N, rate)]})
    print(json.dumps({"workload": "PAPER.md Table 1 (context)", "rows": rows}))


# The other BASELINE.json shapes (C2, C3, C5 of SURVEY 8d): (name, Ensemble keywords, shear rate, timed steps)
OTHER_CONFIGS = [
    ("C2 equilibrium G(t)", dict(n_beads=16, n_chains=65536, stress_every=10, sample_every=10), 0.0, 6400),
    ("C2 without the correlator", dict(n_beads=16, n_chains=65536, stress_every=10), 0.0, 6400),
    ("C3 start-up shear", dict(n_beads=32, n_chains=262144, stress_every=10), 0.1, 2560),
    ("C5 long chains, G(t)", dict(n_beads=128, n_chains=131072, dt=0.005, stress_every=10, sample_every=10), 0.0, 1280),
    ("C5 long chains, steady shear", dict(n_beads=128, n_chains=131072, dt=0.005, stress_every=10), 1e-3, 1280)]


def i_alg_config(stress_every, sample_every):
    """Frozen algorithmic thread-instructions per bead-update of a configuration: the table behind
    I_ALG = 95 is per bead and does not depend on N (noise, bead update, slot work and attempts scale with the beads at
    <Z> = N/4, K = N - Z); what depends on the configuration is the stress work, done on recorded steps only -- bond
    virial 6.0, ensemble reduction 4.5, slip-spring virial 7 x 1/4 = 1.75 per bead-update -- and the correlator's feed
    (per-chain sigma_xy, sigma^(v)_xy and the level-0 products of ssm_corr_kernel: about 3 per bead-update of a sampled step)."""
    rec = 6.0 + 4.5 + 1.75
    v = I_ALG - rec + (rec / stress_every if stress_every > 0 else 0.0)
    if sample_every > 0:
        v += 3.0 / sample_every
    return v


def time_configs(ssm, torch, peak_alu=None):
    """The C2 / C3 / C5 shapes as they are run in production: same kernels as the bench line, their own shapes, sampling
    and flow, device-resident; CUDA events around a few thousand steps after a warm-up.  Context beside the bench line
    (which is configs[3]); parity of these shapes is tests/test_gpu_configs.py.  With peak_alu (T thread-instr/s) every
    row carries its own roofline fraction: i_alg_config() x bead-updates/s / peak (time = everything on the stream,
    correlator launches included)."""
    rows = []
    for name, kw, rate, steps in OTHER_CONFIGS:
        g = ssm.Ensemble(seed=2, stress_capacity=steps // 5, **kw)
        g.step(steps // 5, rate)
        torch.cuda.synchronize()
        l0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); g.step(steps, rate); e1.record(); torch.cuda.synchronize()
        t = e0.elapsed_time(e1) * 1e-3
        rate_bu = kw["n_beads"] * kw["n_chains"] * steps / t
        row = {"config": name, "n_beads": kw["n_beads"], "n_chains": kw["n_chains"], "shear_rate": rate, "steps": steps,
               "seconds": t, "bead_updates_per_s": rate_bu, "ms_per_32_steps": 1e3 * t / steps * 32,
               "launches": int(g.launch_count() - l0)}
        if peak_alu:
            ia = i_alg_config(kw.get("stress_every", 0), kw.get("sample_every", 0))
            row["roofline"] = {"bound": "alu", "i_alg_per_bead_update": ia, "achieved": ia * rate_bu / 1e12, "peak": peak_alu,
                               "unit": "T thread-instr/s", "frac": ia * rate_bu / 1e12 / peak_alu}
        rows.append(row)
        del g
    return rows


def run_configs():
    import torch
    import paper_1106_2899_b200 as ssm
    peaks = measured_peaks()
    peak_alu = N_SM * SMSP_PER_SM * LANES * peaks["sm_max_mhz"] * 1e6 / 1e12
    print(json.dumps({"workload": "BASELINE.json configs[1], [2], [4] (context)", "rows": time_configs(ssm, torch, peak_alu)}))


def spawn_command(n_gpus, port, argv):
    """The launcher line of `python bench.py --gpus N` run without one: the driver's own torchrun line."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n_gpus),
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def main():
    a = parse()
    if a.impl == "reference":
        return run_reference(a)
    if a.table1:
        return run_table1()
    if a.configs:
        return run_configs()

    # `python bench.py --gpus N` without a launcher: start the N ranks ourselves, exactly as the driver's
    # torchrun line does (one process per GPU, NCCL), and let rank 0's JSON line through.  A run whose world size
    # differs from --gpus never reports: one rank must not stand in for an N-GPU measurement.
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        import socket
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0)); port = so.getsockname()[1]
        raise SystemExit(subprocess.call(spawn_command(a.gpus, port, sys.argv[1:])))

    import torch
    import torch.distributed as dist
    from paper_1106_2899_b200 import shard
    import paper_1106_2899_b200 as ssm

    rank, local_rank, world = shard.world()
    if world != a.gpus:
        raise SystemExit("bench.py: --gpus %d but the launcher started %d rank(s)" % (a.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit("bench.py: rank %d has no GPU (%d visible)" % (local_rank, torch.cuda.device_count()))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    M, N, inner, K, W = a.chains, a.beads, a.inner, a.steps, a.warmup
    k0, _ = shard.weak_range(M, rank)
    total_steps = (K + W + 2) * inner
    g = ssm.Ensemble(N, M, seed=4, chain_offset=k0, stress_every=1, stress_capacity=total_steps + 2 * inner,
                     device="cuda:%d" % local_rank)
    g.step(200)                                   # leave the sampled state's first transient behind
    g.reset_accumulators()
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: K bench steps, inputs already in HBM
    def one_step():
        first = g.stress_count()
        g.step(inner)
        if world > 1:                              # the path's only exchange: exact int64 sums (eq 54)
            shard.allreduce_sums(g.stress_sums_device(first, inner), ctx=g)

    for _ in range(W):
        one_step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = g.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    t_wall0 = time.time()
    ev[0].record()
    for i in range(K):
        one_step()
        ev[i + 1].record()
    barrier()
    t_wall1 = time.time()
    launches = g.launch_count() - l0
    ms = ev[0].elapsed_time(ev[K])
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    bead_updates = float(M) * N * inner * K * world
    value = bead_updates / (ms_max * 1e-3)
    launch_ms = ms / max(launches, 1)             # only the step kernel launches inside the region at N = 1

    # ---- end to end through the public API with HOST buffers (pinned): every step uploads its input
    # state (ssm_set_state, host pointers), steps, and reads the stress samples back (ssm_stress, host
    # pointers).  --e2e-contexts (2) contexts on as many streams, one host thread each (ctypes releases the GIL),
    # so that the upload of one batch overlaps the stepping of the other; every batch still pays its own copies.
    e2e = None
    if not a.no_e2e:
        import threading
        R, A, S, step = g.get_state()
        pin = [torch.from_numpy(x).pin_memory() for x in (R, A, S)]
        Rp, Ap, Sp = [p.numpy() for p in pin]
        h2d = Rp.nbytes + Ap.nbytes + Sp.nbytes
        ke = a.e2e_steps if a.e2e_steps > 0 else max(2, min(K, 10))
        nctx = max(1, a.e2e_contexts)
        pair = [ssm.Ensemble(N, M, seed=4, chain_offset=k0, stress_every=1, stress_capacity=inner, stage_chains=M,
                             device="cuda:%d" % local_rank, stream=torch.cuda.Stream(dev)) for _ in range(nctx)]
        # one context alone, through the pipelined call: upload in chunks on a copy stream, chunks stepped as they land
        solo = ssm.Ensemble(N, M, seed=4, chain_offset=k0, stress_every=1, stress_capacity=inner, stage_chains=max(64, M // 8),
                            device="cuda:%d" % local_rank, stream=torch.cuda.Stream(dev))
        outs = [None] * nctx
        errs = []

        # context i starts when context i-1 has uploaded its first batch (inside the timed region), so that the
        # contexts do not begin in phase (all uploading, then all stepping) but as a pipeline
        def e2e_steps(i, n, uploaded=None):
            torch.cuda.set_device(local_rank)
            if uploaded is not None and i > 0:
                uploaded[i - 1].wait()
            try:
                for k in range(n):
                    pair[i].reset_accumulators()
                    pair[i].set_state(Rp, Ap, Sp, step)
                    if uploaded is not None and k == 0:
                        uploaded[i].set()
                    pair[i].step(inner)
                    outs[i] = pair[i].stress()
            except BaseException as exc:                       # re-raised by e2e_run: a failed leg must not pass
                errs.append(exc)
            finally:
                if uploaded is not None:
                    uploaded[i].set()                          # never leave the next context waiting

        def e2e_run(n):
            uploaded = [threading.Event() for _ in range(nctx)]
            th = [threading.Thread(target=e2e_steps, args=(i, n, uploaded)) for i in range(nctx)]
            for x in th:
                x.start()
            for x in th:
                x.join()
            if errs:
                raise errs[0]

        e2e_run(1)
        barrier()
        t0 = time.perf_counter()
        e2e_run(ke)
        barrier()
        dt = time.perf_counter() - t0
        barrier()
        t1 = time.perf_counter()
        e2e_steps(0, 2)                                         # one context alone: copies and stepping in series
        if errs:
            raise errs[0]
        barrier()
        dt_serial = (time.perf_counter() - t1) / 2
        assert all(np.array_equal(outs[0], o) for o in outs[1:])    # same input, same seed: same samples

        def solo_steps(n, bring_back=None):
            out = None
            for _ in range(n):
                solo.reset_accumulators()
                solo.step_from_host(Rp, Ap, Sp, step, inner)
                out = solo.stress()
                if bring_back is not None:                          # the checkpointing user's step: the state comes home too
                    solo.get_state(*bring_back)
            return out
        solo_steps(1)
        barrier()
        t2 = time.perf_counter()
        out_solo = solo_steps(ke)
        barrier()
        dt_solo = (time.perf_counter() - t2) / ke
        assert np.array_equal(out_solo, outs[0])                    # the pipelined call gives the same samples
        # round trip: as above, and ssm_get_state brings the advanced state back into pinned host buffers every step
        back_pin = [torch.empty_like(p_).pin_memory() for p_ in pin]
        back = [p_.numpy() for p_ in back_pin]
        solo_steps(1, back)
        barrier()
        t3 = time.perf_counter()
        solo_steps(3, back)
        barrier()
        dt_round = (time.perf_counter() - t3) / 3
        d2h_state = sum(x.nbytes for x in back)
        t = torch.tensor([dt_solo, dt / (nctx * ke), dt_round], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        per = float(M) * N * inner * world
        e2e = {"value": per / float(t[0].item()), "unit": "bead-updates/s",
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(outs[0].nbytes),
               "steps": ke, "contexts": 1, "pipelined_value": per / float(t[0].item()),
               "two_context_value": per / float(t[1].item()),
               "serial_value": float(M) * N * inner / dt_serial,
               "round_trip": {"value": per / float(t[2].item()), "unit": "bead-updates/s", "h2d_bytes_per_step": int(h2d),
                              "d2h_bytes_per_step": int(outs[0].nbytes + d2h_state), "steps": 3,
                              "what": "as value, and ssm_get_state(host pinned) brings the advanced state back every step"},
               "what": "value = pipelined_value: ONE context, one host thread, per step ssm_step_from_host(host pinned, %d time "
                       "steps: the upload in chunks on a copy stream, chunks stepped as they land) + ssm_stress(host).  "
                       "two_context_value: ssm_set_state(host pinned) + ssm_step + ssm_stress per step on %d contexts "
                       "(streams, host threads, twice the device memory) started one upload apart; every context pays its "
                       "own copies but they all upload the SAME input, so this is pipelining, not more distinct work.  "
                       "serial_value: one context, ssm_set_state then ssm_step then ssm_stress, nothing overlapped "
                       "(its meaning in BENCH_r01)." % (inner, nctx)}
        # the state import / export kernel alone, full size, device pointers: CUDA events on the
        # context's stream, median of 5; algorithmic bytes = the rows read / written + the tiles written / read
        if rank == 0:
            dRAS = [torch.from_numpy(x).to(dev) for x in (Rp, Ap, Sp)]
            cpw = 256 // max(8, 1 << (N - 1).bit_length())          # chains per warp tile of 7552 bytes
            tile_bytes = 7552 * ((M + cpw - 1) // cpw)
            io_bytes = float(h2d + tile_bytes)
            io = {}
            for name, fn in (("import", lambda: pair[0].set_state(dRAS[0], dRAS[1], dRAS[2], step)),
                             ("export", lambda: pair[0].get_state(dRAS[0], dRAS[1], dRAS[2]))):
                fn()
                ts = []
                for _ in range(5):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    with torch.cuda.stream(pair[0].stream):
                        e0.record()
                        fn()
                        e1.record()
                    pair[0].stream.synchronize()
                    ts.append(e0.elapsed_time(e1))
                io[name + "_ms"] = sorted(ts)[2]
                io[name + "_GBps"] = io_bytes / (sorted(ts)[2] * 1e-3) / 1e9
            io["bytes"] = io_bytes
            io["what"] = "ssm_set_state / ssm_get_state with device pointers, %d chains (asynchronous calls, CUDA events on the ctx's stream)" % M
            e2e["state_io"] = io
            del dRAS
        del solo
        del pair

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    if e2e is not None and "state_io" in e2e:
        for name in ("import", "export"):
            e2e["state_io"][name + "_frac_of_copy_peak"] = e2e["state_io"][name + "_GBps"] / peaks["hbm_gbs"]
    peak_alu = N_SM * SMSP_PER_SM * LANES * peaks["sm_max_mhz"] * 1e6 / 1e12      # T thread-instr/s
    per_launch_updates = float(M) * N * inner * K / max(launches, 1)
    achieved = I_ALG * per_launch_updates / (launch_ms * 1e-3) / 1e12
    # algorithmic state bytes per launch: read + write of the dense-slot
    # state, 25 N bytes per chain (R 12N, A 12N, S N); the tiles the kernel really moves are larger
    # (7552 B per 256 beads = 29.5 N per chain: anchors are float4 with the low part of x, plus Z)
    alg_bytes = 2.0 * 25.0 * N * M
    hbm_achieved = alg_bytes / (launch_ms * 1e-3) / 1e9
    traffic = ncu_traffic(N, M)
    rates = g.issue_rates()
    i_alg_cycles = (I_ALG - I_ALG_WIDE) + I_ALG_WIDE * max(1.0, rates["imad_wide"])
    weighted = i_alg_cycles * per_launch_updates / (launch_ms * 1e-3) / 1e12
    line = {
        "metric": "bead-updates/s", "value": value, "unit": "bead-updates/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": workload_config(a, M, inner, world),
        "chain_steps_per_s": value / N,
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": e2e,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_alu, "unit": "T thread-instr/s",
                     "frac": achieved / peak_alu, "traffic": traffic,
                     "traffic_source": (TRAFFIC_CSV + " (committed ncu --set full capture of this workload, not this run)") if traffic else None,
                     "kernel": "ssm_step_kernel<G=%d>" % (N // 8), "launch_ms": launch_ms,
                     "i_alg_per_bead_update": I_ALG,
                     "rate_weighted": {"frac": weighted / peak_alu, "i_alg_issue_cycles_per_bead_update": i_alg_cycles,
                                       "measured_cycles_per_warp_instruction": rates,
                                       "how": "as frac, but the %.1f IMAD.WIDE of the algorithmic count are charged the "
                                              "issue cycles ssm_issue_rates8() measures for them on this GPU instead of 1"
                                              % I_ALG_WIDE},
                     "peak_how": "148 SM x 4 SMSP x 32 lanes x %.0f MHz (sm_max_mhz, %s)" % (peaks["sm_max_mhz"], peaks["source"]),
                     "hbm": {"achieved": hbm_achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": hbm_achieved / peaks["hbm_gbs"], "bytes_per_launch": alg_bytes,
                             "peak_source": peaks["source"]}},
        "paper_context": {"gpu_bead_updates_per_s": 7.3e8, "cpu_bead_updates_per_s": 2.5e6,
                          "hardware": "Tesla C1060 / Core 2 Duo E8500 1 thread (PAPER.md Table 1)"},
    }
    if world == 1 and not a.no_e2e:
        # context, not the metric: the other BASELINE.json shapes with the same kernels in the same run (clock record above)
        del g
        line["other_configs"] = time_configs(ssm, torch, peak_alu)
    if not a.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(N, a.cpu_seconds)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
