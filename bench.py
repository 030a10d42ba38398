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


def ncu_traffic(pair_batch, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of the S4 kernels per launch triple, from the tracked ncu summary
    profiles/s4_traffic.csv (written from an `ncu --set full` capture, command in profiles/r02_summary.md).  None when the
    capture was taken with another pair batch or workload than the one running now."""
    path = os.path.join(ROOT, "profiles", "s4_traffic.csv")
    if not os.path.exists(path):
        return None
    total, ok = 0.0, False
    with open(path) as f:
        header = f.readline().strip().split(",")
        for line in f:
            row = dict(zip(header, line.strip().split(",")))
            if not row.get("kernel"):
                continue
            if row["workload"] != workload or int(row["pair_batch"]) != int(pair_batch):
                return None
            total += float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
            ok = True
    return total if ok else None


def _threads_used():
    try:
        import threadpoolctl
        return max([p["num_threads"] for p in threadpoolctl.threadpool_info()] + [1])
    except Exception:
        return 1


def oracle_problem(cfg):
    """The oracle on the full configuration (numpy.fft as its transform step, pinned equal to its radix FFT in
    tests/test_oracle_dft.py) and one seeded trial vector.  Set-up, not timed (the counterpart of tddft_init)."""
    from oracle import lattice as olat
    from oracle import liouville as olv
    import synthetic_inputs as inputs
    miller, g2 = olat.enumerate_half_sphere(cfg["lattice"], cfg["ecut"])
    inp = inputs.make_problem_inputs(cfg, g2)
    P = olv.Problem(cfg["lattice"], cfg["grid"], cfg["ecut"], cfg["nspin"], inp["psi"], inp["eig"], cfg["alpha"], fft_backend="numpy")
    X = inputs.make_trial_block(cfg, inp, 1, 0)
    return P, X


def oracle_column_sample(P, ctx, s, v, n_pp, rng):
    """Seconds for `n_pp` of the N_occ pair potentials of one output column (spin s, orbital v) of A x, exactly as
    oracle.column computes them (oracle.coulomb on phi_v phi_v', multiply by a_v', accumulate), plus the column's fixed part
    (to_sphere + D + projector).  Returns (t_pair_potentials, t_fixed)."""
    vps = rng.choice(P.nocc[s], size=min(n_pp, P.nocc[s]), replace=False)
    y = np.zeros(P.grid)
    t0 = time.perf_counter()
    for vp in vps:
        y -= P.alpha * ctx["a"][s][vp] * P.coulomb(P.phi[s][v] * P.phi[s][vp])
    t1 = time.perf_counter()
    yg = P.to_sphere(y) + (0.5 * P.g2 - P.eig[s][v]) * ctx["x"][s][v]
    P.project_c(yg, s)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1, len(vps)


def oracle_sample(cfg, P=None, X=None, n_pp=None):
    """SURVEY 8(d) protocol: time the oracle, as it stands, on sampled columns of the real configuration and scale to one
    vector apply:  t_vec = t_prepare + sum_s N_occ,s * t_column,s.  With n_pp = None a full column (all N_occ pair potentials)
    of each spin is computed through oracle.column; with n_pp set only n_pp seeded pair potentials of one column are computed
    and the column time is scaled by N_occ / n_pp (used by --impl reference to bound a step)."""
    if P is None:
        P, X = oracle_problem(cfg)
    rng = np.random.Generator(np.random.PCG64(cfg["seed"] + 77))
    t0 = time.perf_counter()
    ctx = P.prepare(X[0], 0)
    t_prep = time.perf_counter() - t0
    t_cols, desc = 0.0, []
    work = t_prep
    for s in range(P.nspin):
        v = int(rng.integers(P.nocc[s]))
        if n_pp is None:
            if s > 0:      # one full column is enough for the estimate; the other spin's columns cost the same per pair potential
                t_cols += P.nocc[s] * (t_col * P.nocc[s] / P.nocc[0])
                continue
            t1 = time.perf_counter()
            P.column(ctx, s, v)
            t_col = time.perf_counter() - t1
            work += t_col
            t_cols += P.nocc[s] * t_col
            desc.append("column (spin %d, v %d): %d pair potentials, %.1f s" % (s, v, P.nocc[s], t_col))
        else:
            if s > 0:
                t_cols += P.nocc[s] * (tpp / npp * P.nocc[s] + tfix)
                continue
            tpp, tfix, npp = oracle_column_sample(P, ctx, s, v, n_pp, rng)
            work += tpp + tfix
            t_cols += P.nocc[s] * (tpp / npp * P.nocc[s] + tfix)
            desc.append("%d of the %d pair potentials of column (spin %d, v %d): %.1f s" % (npp, P.nocc[s], s, v, tpp))
    t_vec = t_prep + t_cols
    return {
        # the oracle's time is in its FFTs (numpy pocketfft, one thread); BLAS threads only touch the small projector dot products
        "value": 1.0 / t_vec, "unit": UNIT, "cores": 1, "blas_threads_available": int(_threads_used()), "kind": "oracle",
        "sample": "oracle on the full %s configuration (numpy.fft backend): prepare of one trial vector (%.1f s) + %s; "
                  "scaled to one vector apply = prepare + (N_up + N_dn) columns (an extrapolation: %.0f s per vector apply)"
                  % (cfg["name"], t_prep, "; ".join(desc), t_vec),
        "sample_seconds": work,
    }


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    P, X = oracle_problem(cfg)
    # size a step so that warmup + steps samples end within a few minutes: calibrate on 4 pair potentials
    ctx = P.prepare(X[0], 0)
    tpp, _, npp = oracle_column_sample(P, ctx, 0, 0, 4, np.random.Generator(np.random.PCG64(1)))
    budget = 150.0 / max(args.warmup + args.steps, 1)
    del ctx
    t_prep_est = None
    vals = []
    base = None
    t_begin = time.perf_counter()
    for i in range(args.warmup + args.steps):
        # the prepare step (N_occ transforms per spin) is part of every sample; bound the pair potentials by what is left of the step budget
        t0 = time.perf_counter()
        if t_prep_est is None:
            n_pp = 4
        else:
            n_pp = int(max(4, min(P.nocc[0], (budget - t_prep_est) / max(tpp / npp, 1e-6))))
        base = oracle_sample(cfg, P, X, n_pp=n_pp)
        if t_prep_est is None:
            t_prep_est = time.perf_counter() - t0
        if i >= args.warmup:
            vals.append(base["value"])
    v = float(np.mean(vals))
    base["value"] = v
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * (time.perf_counter() - t_begin) / max(args.warmup + args.steps, 1),
        "higher_is_better": True, "scaling": "weak",
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-coupling", action="store_true", help="skip the (phi, a, phi) pair-FFT figure (tddft_apply_coupling, 1 vector)")
    ap.add_argument("--pair-tile", type=int, default=0)
    ap.add_argument("--fft-batch", type=int, default=0)
    ap.add_argument("--fft-path", type=int, default=0)
    ap.add_argument("--workspace-gb", type=float, default=0.0)
    ap.add_argument("--work-l2-mb", type=float, default=0.0)
    ap.add_argument("--tile-width", type=int, default=0)
    ap.add_argument("--plan", type=int, default=0, help="0 auto, 1 resident, 2 streamed")
    ap.add_argument("--emulate-shard", type=int, nargs=2, default=None, metavar=("RANK", "COUNT"), help="N = 1 only: time ONE shard of a sharded apply (partial result; a timing probe for the scaling estimate in DESIGN.md, not a bench value)")
    ap.add_argument("--shard-apply", action="store_true", help="N > 1: shard ONE block apply over the ranks (tiles dealt to the ranks, one all-reduce of AX; strong scaling) instead of one block per rank")
    ap.add_argument("--davidson", type=int, default=0, help="also run tddft_davidson for this many roots (not timed into `value`)")
    ap.add_argument("--max-iter", type=int, default=0)
    ap.add_argument("--precond", type=int, default=0)
    ap.add_argument("--verbose", type=int, default=0)
    ap.add_argument("--probes", action="store_true", help="also run the read-bandwidth probe (fp64_peaks.read_gbs_by_piece_bytes)")
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
    shard = args.shard_apply and world > 1
    rng = np.random.Generator(np.random.PCG64(cfg["seed"] + 1000 * ((0 if shard else rank) + 1)))      # sharded: the same block on every rank
    inp["rng"] = rng
    nvec, mode = cfg["nvec"], args.mode
    Xh = inputs.make_trial_block(cfg, inp, nvec, mode)
    d_psi = [torch.from_numpy(p).cuda() for p in inp["psi"]]
    opts = {}
    if shard:
        opts["shard_rank"] = rank; opts["shard_count"] = world
    elif args.emulate_shard and world == 1:
        opts["shard_rank"], opts["shard_count"] = args.emulate_shard
    for k, v in (("pair_tile", args.pair_tile), ("fft_batch", args.fft_batch), ("max_iter", args.max_iter), ("fft_path", args.fft_path),
                 ("workspace_gb", args.workspace_gb), ("work_l2_mb", args.work_l2_mb), ("tile_width", args.tile_width), ("plan", args.plan), ("precond", args.precond), ("verbose", args.verbose)):
        if v:
            opts[k] = v
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

    def max_over_ranks(ms):
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ---- device-resident timing: K applies back to back, stage timing OFF (no host synchronisation inside) ----------
    apply = (lambda: b.tddft_apply_liouville_sharded(ctx, dX, dAX, nvec, mode)) if shard else (lambda: b.tddft_apply_liouville(ctx, dX, dAX, nvec, mode))
    for _ in range(args.warmup):
        apply()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    launches = 0
    pair_ffts = 0
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        apply()
        st = b.tddft_get_stats(ctx)            # host counters only
        launches += st["kernel_launches"]; pair_ffts += st["pair_ffts"]
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(e0.elapsed_time(e1))
    value = (1 if shard else world) * nvec * args.steps / (ms * 1e-3)

    # ---- stage breakdown: a separate pass with CUDA events around every stage (adds a synchronisation per apply) -------
    b.tddft_set_timing(ctx, True)
    stage_ms = {}
    nstage = max(1, min(args.steps, 3))
    for _ in range(nstage):
        b.tddft_apply_liouville(ctx, dX, dAX, nvec, mode)
        st = b.tddft_get_stats(ctx)
        for k, v in st.items():
            if k.startswith("ms_"):
                stage_ms[k] = stage_ms.get(k, 0.0) + v / nstage
    b.tddft_set_timing(ctx, False)
    pairs_per_step = pair_ffts / max(args.steps, 1)

    # ---- end to end through the C ABI with pinned host buffers ------------------------------------------
    e2e = None
    if not args.no_e2e and not shard:
        Xp = torch.from_numpy(Xh).pin_memory()
        AXp = torch.empty_like(Xp).pin_memory()
        b.tddft_apply_liouville_host(ctx, Xp, AXp, nvec, mode)
        barrier()
        e0.record(stream)
        for _ in range(args.steps):
            b.tddft_apply_liouville_host(ctx, Xp, AXp, nvec, mode)
        e1.record(stream)
        barrier()
        t = max_over_ranks(e0.elapsed_time(e1))
        nbytes = Xp.numel() * 16
        e2e = {"value": world * nvec * args.steps / (t * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes}
        # sanity: host path equals device path
        assert torch.equal(AXp, dAX.cpu()), "host and device entry points disagree"
        del Xp, AXp

    # ---- FP64 peaks measured in this run and the (phi, a, phi) operand pattern -------------
    fp64 = None
    coupling = None
    if rank == 0:
        dfma, dmma = b.tddft_fp64_peak(ctx)
        fp64 = {"dfma_tflops": dfma, "dmma_tflops": dmma}
        if args.probes:      # read bandwidth of the contraction's access pattern (32-byte pieces) against whole 256-byte runs
            fp64["read_gbs_by_piece_bytes"] = {str(pb_): b.tddft_stream_probe(ctx, pb_) for pb_ in (32, 64, 128, 256)}
        if not args.no_coupling and mode == 0 and not shard:
            b.tddft_apply_coupling(ctx, dX[:1], dAX[:1], 1, 0)      # warm-up
            torch.cuda.synchronize()
            e0.record(stream)
            b.tddft_apply_coupling(ctx, dX[:1], dAX[:1], 1, 0)
            e1.record(stream)
            torch.cuda.synchronize()
            stc = b.tddft_get_stats(ctx)
            tms = e0.elapsed_time(e1)
            coupling = {"what": "tddft_apply_coupling (K2e - K2d, Eqs. 5 and 7), 1 trial vector: pair densities phi_v * a_v'",
                        "pair_ffts": int(stc["pair_ffts"]), "ms": tms, "pair_ffts_per_s_whole_call": stc["pair_ffts"] / (tms * 1e-3)}

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
    pb = st["pair_batch"]
    roofline = None
    if s4_ms > 0 and pairs_per_step > 0:
        bytes_per_pair = 32.0 * nr                      # one HBM round trip per direction per pair density
        achieved = pairs_per_step * bytes_per_pair / (s4_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": ncu_traffic(pb, cfg["name"]) if st["fft_path"] == 0 else None,
                    "algorithmic_bytes": bytes_per_pair * pb, "units_per_launch": "%d pairs (one launch of each of the three kernels)" % pb,
                    "kernel": "S4 pair-FFT pipeline (%s, batches of %d pairs)" % ("plane_kernel fwd + xpass_kernel conv + plane_kernel inv" if st["fft_path"] == 0 else "5 general pass kernels", pb),
                    "algorithmic_bytes_per_pair": bytes_per_pair, "peak_source": peak_src,
                    "share_of_step": s4_ms / max(stage_ms.get("ms_total", 1e-9), 1e-9)}
    # FP64 tensor-core rooflines of the dense contractions (BASELINE.json metric: "FP64 TC %"): S5 and S8
    fp64_rooflines = None
    if fp64:
        tc_peak = max(fp64["dmma_tflops"], 1e-9)
        npwh = len(g2)
        blocks = list(range(cfg["nspin"])) if mode == 0 else [0 if mode == 1 else 1]
        f_s5 = sum(2.0 * cfg["nocc"][s] ** 2 * nvec * nr for s in blocks) if cfg["alpha"] != 0 else 0.0
        tgt = (lambda s: s) if mode == 0 else (lambda s: 1 - s)
        f_s8 = sum(2 * 2.0 * cfg["nocc"][tgt(s)] * cfg["nocc"][s] * nvec * (2 * npwh) for s in blocks)
        fp64_rooflines = {}
        for name, fl, key in (("s5_contraction", f_s5, "ms_s5_contract"), ("s8_projector", f_s8, "ms_s8_project")):
            t = stage_ms.get(key, 0.0)
            if t > 0 and fl > 0:
                ach = fl / (t * 1e-3) / 1e12
                fp64_rooflines[name] = {"bound": "fp64_tc", "achieved": ach, "peak": tc_peak, "unit": "TFLOP/s", "frac": ach / tc_peak,
                                        "flops": fl, "ms": t, "peak_source": "tddft_fp64_peak (register-resident mma.sync.m8n8k4.f64 loop, this run)"}
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1 and mode == 0:
        cpu_baseline = oracle_sample(cfg)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": list(cfg["grid"]), "nocc": list(cfg["nocc"]), "nvec": nvec,
                   "mode": ["spin_conserving", "spin_flip_up_down", "spin_flip_down_up"][mode], "alpha": cfg["alpha"],
                   "pair_tile": st["pair_tile"], "tile_width": st["tile_width"], "k_chunk": st["k_chunk"], "blocks_resident": st["blocks_resident"],
                   "l2": "inputs_exceed_l2 (X, Phi(r), a(r), out(r), tau tiles >> 126 MB)", "parallelism": ("one apply sharded over %d ranks (tiles dealt to the ranks, one all-reduce of AX)" if shard else "images x%d") % world,
                   **({"emulated_shard": list(args.emulate_shard)} if args.emulate_shard else {})},
        "block_applies_per_s": value / nvec,
        "pair_ffts_per_s": (world * pairs_per_step / (s4_ms * 1e-3)) if s4_ms > 0 else None,
        "pair_ffts_per_step": pairs_per_step,
        "stage_ms_per_step": stage_ms,
        "exchange_only_ms": stage_ms.get("ms_s4_pair_fft", 0.0) + stage_ms.get("ms_s5_contract", 0.0),
        "projector_ms": stage_ms.get("ms_s8_project", 0.0),
        "gpu_launches": int(launches),
        "clocks": clocks,
        "e2e": e2e,
        "roofline": roofline,
        "fp64_peaks": fp64,
        "fp64_rooflines": fp64_rooflines,
        "phi_a_phi_pattern": coupling,
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
