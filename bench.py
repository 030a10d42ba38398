#!/usr/bin/env python
"""bench.py -- Liouville applies/s of the CUDA path on the 215-atom NV- shaped configuration (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--mode 0|1|2] [--impl reference]

A step = one tddft_apply_liouville call (all of SURVEY S1-S8) on a block of nvec seeded synthetic trial
vectors.  One JSON line is printed by rank 0.  N > 1 (torchrun) shards independent trial-vector blocks
across ranks (the paper's "images" level): no data-path collective, weak scaling.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# dram__bytes_read.sum + dram__bytes_write.sum of the three S4 kernels per batch of 180 pairs at NV215, from the ncu --set full
# capture summarised in profiles/r01i_summary.md (361.2 + 623.9 + 822.7 MB), per pair
NCU_TRAFFIC_PER_PAIR = 1807.8e6 / 180
METRIC = "liouville_vector_applies_per_s"
UNIT = "vector-applies/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        try:
            with open(self.path) as f:
                for line in f:
                    p = [x.strip() for x in line.split(",")]
                    if len(p) < 9:
                        continue
                    try:
                        sm.append(float(p[1])); mx.append(float(p[2]))
                    except ValueError:
                        continue
                    for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                        if val.lower().startswith("active"):
                            reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out["sm_mhz"] = float(np.median(sm)); out["sm_max_mhz"] = float(max(mx)); out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def oracle_sample(cfg, sample_nocc=6):
    """Time the oracle, as it stands, on a bounded sample of the workload and extrapolate to one vector apply.

    Sample: the full oracle apply (prepare + every column) of ONE trial vector on the configuration's lattice,
    grid and cutoff, but with `sample_nocc` occupied orbitals per spin.  The oracle's cost per vector apply is
    dominated by its sum_s nocc_s^2 pair potentials (it uses no symmetry and no reuse across trial vectors), so
    the time is scaled by (sum_s nocc_s^2) / (sum_s sample_nocc^2)."""
    from oracle import lattice as olat
    from oracle import liouville as olv
    import synthetic_inputs as inputs
    miller, g2 = olat.enumerate_half_sphere(cfg["lattice"], cfg["ecut"])
    rng = np.random.Generator(np.random.PCG64(cfg["seed"]))
    nsp = cfg["nspin"]
    psi = [inputs.orbitals(rng, sample_nocc, g2, cfg["ecut"], cfg["envelope"], cfg["ortho"]) for _ in range(nsp)]
    eig = [inputs.eigenvalues(rng, sample_nocc) for _ in range(nsp)]
    P = olv.Problem(cfg["lattice"], cfg["grid"], cfg["ecut"], nsp, psi, eig, cfg["alpha"])
    X = inputs.trial_vectors(rng, [(sample_nocc, p) for p in psi], 1)
    t0 = time.perf_counter()
    P.apply(X, 0)
    dt = time.perf_counter() - t0
    pairs_sample = nsp * sample_nocc ** 2
    pairs_full = sum(n * n for n in cfg["nocc"])
    t_vec = dt * pairs_full / pairs_sample
    try:
        import threadpoolctl
        cores = max([p["num_threads"] for p in threadpoolctl.threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    return {
        "value": 1.0 / t_vec, "unit": UNIT, "cores": int(cores), "kind": "oracle",
        "sample": "oracle.apply of 1 trial vector on the %s lattice/grid/cutoff with %d occupied orbitals per spin "
                  "(%d pair potentials, %.1f s); scaled by the oracle's pair-potential count %d/%d per vector apply"
                  % (cfg["name"], sample_nocc, pairs_sample, dt, pairs_full, pairs_sample),
        "sample_seconds": dt,
    }


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    base = None
    for i in range(args.warmup + args.steps):
        base = oracle_sample(cfg, args.sample_nocc)
        if i >= args.warmup:
            vals.append(base["value"])
    v = float(np.mean(vals))
    base["value"] = v
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * cfg["nvec"] / v, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": list(cfg["grid"]), "nocc": list(cfg["nocc"]), "nvec": cfg["nvec"],
                   "mode": "spin_conserving", "alpha": cfg["alpha"]},
        "cpu_baseline": base,
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--mode", type=int, default=0)
    ap.add_argument("--impl", default="cuda")
    ap.add_argument("--nocc", type=int, nargs="*", default=None, help="override occupied counts (debugging only)")
    ap.add_argument("--nvec", type=int, default=None)
    ap.add_argument("--sample-nocc", type=int, default=6)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--pair-tile", type=int, default=0)
    ap.add_argument("--fft-batch", type=int, default=0)
    ap.add_argument("--davidson", type=int, default=0, help="also run tddft_davidson for this many roots (not timed into `value`)")
    ap.add_argument("--max-iter", type=int, default=0)
    args = ap.parse_args()

    import synthetic_inputs as inputs
    cfg = inputs.config(args.config)
    if args.nocc:
        cfg["nocc"] = tuple(args.nocc)
    if args.nvec:
        cfg["nvec"] = args.nvec
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2309_03513_b200 import binding as b

    # ---- inputs: same orbitals on every rank, rank-specific trial-vector block (weak scaling over images) ----
    miller, g2 = b.tddft_enumerate_gvectors(cfg["lattice"], cfg["ecut"])
    inp = inputs.make_problem_inputs(cfg, g2, scale_nocc=cfg["nocc"])
    rng = np.random.Generator(np.random.PCG64(cfg["seed"] + 1000 * (rank + 1)))
    inp["rng"] = rng
    nvec, mode = cfg["nvec"], args.mode
    Xh = inputs.make_trial_block(cfg, inp, nvec, mode)
    d_psi = [torch.from_numpy(p).cuda() for p in inp["psi"]]
    opts = {}
    if args.pair_tile:
        opts["pair_tile"] = args.pair_tile
    if args.fft_batch:
        opts["fft_batch"] = args.fft_batch
    if args.max_iter:
        opts["max_iter"] = args.max_iter
    ctx = b.tddft_init(cfg["lattice"], cfg["grid"], cfg["ecut"], cfg["nspin"], cfg["nocc"], d_psi[0],
                       d_psi[1] if cfg["nspin"] == 2 else None, inp["eig"][0],
                       inp["eig"][1] if cfg["nspin"] == 2 else None, cfg["alpha"], **opts)
    dX = torch.from_numpy(Xh).cuda()
    dAX = torch.empty_like(dX)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ------------------------------------------------------------------------
    for _ in range(args.warmup):
        b.tddft_apply_liouville(ctx, dX, dAX, nvec, mode)
    barrier()
    b.tddft_set_timing(ctx, True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    stage_ms = {}
    launches = 0
    pair_ffts = 0
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        b.tddft_apply_liouville(ctx, dX, dAX, nvec, mode)
        st = b.tddft_get_stats(ctx)
        launches += st["kernel_launches"]; pair_ffts += st["pair_ffts"]
        for k, v in st.items():
            if k.startswith("ms_"):
                stage_ms[k] = stage_ms.get(k, 0.0) + v
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1)
    b.tddft_set_timing(ctx, False)
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    value = world * nvec * args.steps / (ms * 1e-3)

    # ---- end to end through the C ABI with pinned host buffers ------------------------------------------
    e2e = None
    if not args.no_e2e:
        Xp = torch.from_numpy(Xh).pin_memory()
        AXp = torch.empty_like(Xp).pin_memory()
        b.tddft_apply_liouville_host(ctx, Xp, AXp, nvec, mode)
        barrier()
        e0.record(stream)
        for _ in range(args.steps):
            b.tddft_apply_liouville_host(ctx, Xp, AXp, nvec, mode)
        e1.record(stream)
        barrier()
        t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        nbytes = Xp.numel() * 16
        e2e = {"value": world * nvec * args.steps / (float(t.item()) * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes}
        # sanity: host path equals device path
        assert torch.equal(AXp, dAX.cpu()), "host and device entry points disagree"

    davidson = None
    if args.davidson > 0 and rank == 0:      # SURVEY S9 on the same context: block Davidson for the lowest roots (reading A11)
        del dX, dAX
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ev, iters, res = b.tddft_davidson(ctx, args.davidson, mode, allow_unconverged=True)
        torch.cuda.synchronize()
        davidson = {"nroots": args.davidson, "seconds": time.perf_counter() - t0, "iterations": int(iters),
                    "eigenvalues_ha": [float(x) for x in ev], "residual_norms": [float(x) for x in res]}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    nr = int(np.prod(cfg["grid"]))
    peak, peak_src = measured_peaks()
    s4_ms = stage_ms.get("ms_s4_pair_fft", 0.0)
    pairs_per_step = pair_ffts / max(args.steps, 1)
    pb = st["pair_batch"]
    roofline = None
    if s4_ms > 0 and pair_ffts > 0:
        bytes_per_pair = 32.0 * nr                      # one HBM round trip per direction per pair density
        achieved = pair_ffts * bytes_per_pair / (s4_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": NCU_TRAFFIC_PER_PAIR * pb if st["fft_path"] == 0 and args.config == 3 else None,
                    "algorithmic_bytes": bytes_per_pair * pb, "units_per_launch": "%d pairs (one launch of each of the three kernels)" % pb,
                    "kernel": "S4 pair-FFT pipeline (%s, batches of %d pairs)" % ("plane_kernel fwd + xpass_kernel conv + plane_kernel inv" if st["fft_path"] == 0 else "5 general pass kernels", pb),
                    "algorithmic_bytes_per_pair": bytes_per_pair, "peak_source": peak_src,
                    "share_of_step": s4_ms / max(stage_ms.get("ms_total", 1e-9), 1e-9)}
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        cpu_baseline = oracle_sample(cfg, args.sample_nocc)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": list(cfg["grid"]), "nocc": list(cfg["nocc"]), "nvec": nvec,
                   "mode": ["spin_conserving", "spin_flip_up_down", "spin_flip_down_up"][mode], "alpha": cfg["alpha"],
                   "pair_tile": st["pair_tile"], "l2": "inputs_exceed_l2 (X, Phi(r), a(r), out(r), tau tiles >> 126 MB)", "parallelism": "images x%d" % world},
        "block_applies_per_s": value / nvec,
        "pair_ffts_per_s": (world * pair_ffts / (s4_ms * 1e-3)) if s4_ms > 0 else None,
        "pair_ffts_per_step": pairs_per_step,
        "stage_ms_per_step": {k: v / args.steps for k, v in stage_ms.items()},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "e2e": e2e,
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "workspace_gb": b.tddft_workspace_bytes(ctx) / 2 ** 30,
    }
    if davidson:
        line["davidson"] = davidson
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
