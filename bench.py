#!/usr/bin/env python
"""bench.py -- RT-TDA hot path at the 1280-AO molecule (BASELINE.json metric: sigma-vectors/s and RT-TDA
steps/s at 1280 AO; FP64 pipe % of peak).

    python bench.py --gpus N --steps K --warmup W [--config 4] [--ntraj 3] [--impl reference]

One *step* = one RK4 step of `rttda_propagate` on config 4: every row a1-a7 of
the hot path -- 4 ERI passes, each serving the 2*ntraj real vectors of the batch, the MO<->AO GEMMs, the
field coupling and the RK4 combine.  value = sigma-vectors/s = 8*ntraj*N_gpus / t_step (one sigma-vector =
A x for one real x).  Inputs are seeded synthetic (workloads/), resident in HBM before the timed
region; the `e2e` number goes through `rttda_propagate_host` (host buffers, copies inside the timed region).
Multi-GPU (N > 1): replicas only -- every rank runs the same batch of trajectories on
its own GPU, no data-path collective, "weak" scaling; time = max over ranks.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores for the same metric.
"""
from __future__ import annotations

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

UNIT = "sigma-vectors/s"


def metric_name(nao: int) -> str:
    """BASELINE.json's metric is quoted at 1280 AO (config 4, the default); other --config values name their own size."""
    return "sigma_vectors_per_s_%dao" % nao
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SMs x 64 DFMA/clk/SM x 2 x max SM clock


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4, help="workload (4 = the 1280-AO molecule; 2, 3 smaller)")
    ap.add_argument("--ntraj", type=int, default=0, help="trajectories per call (0 = all of the config's fields)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="CPU budget of the cpu_baseline sample")
    ap.add_argument("--propagator", default="rk4", choices=["rk4", "sso"],
                    help="rk4 (BASELINE.json configs; 8 sigma-vectors per trajectory and step) or the paper's SSO "
                         "(NEXT-1; 2 per trajectory and step)")
    ap.add_argument("--tau", type=float, default=0.0, help="Schwarz threshold (0 = the config's: 1e-12, reading R15)")
    ap.add_argument("--exchange", default="1,0,0", metavar="CX,CX_LR,OMEGA",
                    help="exchange kernel of A: -cx (ij|ab) - cx_lr (ij|erf(omega r)/r|ab); default 1,0,0 = the exchange-only "
                         "headline (BASELINE.json); 0.19,0.46,0.33 = the exchange part of the paper's CAM-B3LYP (second ERI pass)")
    ap.add_argument("--parity-tau", type=float, default=1e-14,
                    help="second, tighter threshold at which config 4 is also timed: the largest tau of the sweep at which "
                         "sigma meets the 1e-10 oracle tolerance at 1280 AO (tests/test_gpu_parity.py, DESIGN.md section 11); 0 = skip")
    ap.add_argument("--omega", type=float, default=0.0, help="carrier frequency in Ha (0 = from rttda_eigs, see run_b200)")
    ap.add_argument("--sweep-point", nargs=2, metavar=("NVEC", "TAU"), default=None,
                    help="config 5, ONE point: 2 warm rttda_sigma calls, then one call between cudaProfilerStart/Stop "
                         "(for `ncu --profile-from-start off`: FP64 pipe utilisation per point, profiles/README.md)")
    ap.add_argument("--sweep", action="store_true", help="run the config-5 sigma sweep (nvec x tau) instead of the step bench -> gpurun_out/sweep.json")
    return ap.parse_args()


def reduce_max(x: float, world: int, device) -> float:
    """Time of the slowest replica: the one collective of the N > 1 path (replicas only)."""
    if world <= 1:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(ntraj: int, world: int, ms_per_step: float, per_traj: float = 8.0) -> float:
    """Whole-job sigma-vectors/s: every replica builds per_traj*ntraj sigma-vectors per step (RK4: 8, SSO: 2)."""
    return per_traj * ntraj * world / (ms_per_step * 1e-3)


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


# ------------------------------------------------------------------------------------------ workload
def build_inputs(k: int, overlap_fn):
    """Seeded synthetic molecule of config k.  overlap_fn(basis) -> S comes from the side being timed."""
    from workloads import get_config, make_basis, make_mos
    cfg = get_config(k)
    bump = 0
    while True:
        basis = make_basis(cfg, bump)
        S = overlap_fn(basis)
        C_o, C_v, eps, cond = make_mos(cfg, S, bump)
        if cond <= 1e5:
            break
        bump += 1
    return cfg, basis, C_o, C_v, eps, cond, bump


def fields_for(cfg, ntraj, omega):
    fs = [dict(f) for f in cfg.fields]
    if ntraj:
        fs = [dict(fs[i % len(fs)]) for i in range(ntraj)]
    for f in fs:
        if f.get("omega", 0.0) is None:
            f["omega"] = omega
    return fs


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[1])); smax.append(float(p[2])); pw.append(float(p[3]))
            except ValueError:
                continue
            for nm, v in zip(names, p[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ CPU oracle legs
def count_unique_quartets(Q: np.ndarray, sh_nprim: np.ndarray, tau: float):
    """Unique shell quartets (a>=b, c>=d, ab>=cd) with Q_ab Q_cd >= tau (R14) and the primitive quartets in
    them, from the Schwarz matrix alone (pure counting; used to scale the CPU sample to one full pass)."""
    ns = Q.shape[0]
    ia, ib = np.tril_indices(ns)
    q = Q[ia, ib]
    w = (sh_nprim[ia].astype(np.float64) * sh_nprim[ib])
    order = np.argsort(-q, kind="stable")
    qs, ws = q[order], w[order]
    cw = np.concatenate([[0.0], np.cumsum(ws)])
    with np.errstate(divide="ignore"):
        thr = np.where(qs > 0, tau / qs, np.inf)
    n = np.searchsorted(-qs, -thr, side="right")          # kets with Q_cd >= tau / Q_ab
    ordered, ordered_p = float(np.sum(n)), float(np.sum(ws * cw[n]))
    dmask = qs * qs >= tau
    return 0.5 * (ordered + float(np.sum(dmask))), 0.5 * (ordered_p + float(np.sum(ws[dmask] ** 2)))


def oracle_sample(cfg_k: int, nvec: int, cpu_seconds: float):
    """Time the oracle's matrix-free J/K (oracle/, as it stands, all host cores) on a bounded sample of the
    bra shell pairs of config cfg_k and scale by the primitive-quartet fraction of the sample.
    Returns (sigma_vectors_per_s, cores, description, seconds per full ERI pass)."""
    from oracle.integrals import OracleBasis, num_threads
    from oracle import tda
    from workloads import make_vectors
    cfg, basis, C_o, C_v, eps, _, _ = build_inputs(cfg_k, lambda b: OracleBasis(b).overlap())
    ob = OracleBasis(basis)
    Q = ob.schwarz()
    nq_total, nprim_total = count_unique_quartets(Q, np.asarray(basis.sh_nprim), cfg.tau)
    X = make_vectors(cfg, nvec)
    T = np.stack([tda.transition_density(x.reshape(cfg.nocc, cfg.nvirt), C_o, C_v) for x in X])
    npair = ob.nshells * (ob.nshells + 1) // 2
    # pilot: a thin sample to learn the rate, then one sample sized for the CPU budget
    stride = max(1, npair // 256)
    t0 = time.perf_counter()
    _, _, nq, npq = ob.jk_strided(T, cfg.tau, Q, stride, stride // 2)
    dt = time.perf_counter() - t0
    rate = max(npq, 1) / max(dt, 1e-6)
    stride2 = int(max(1, min(stride, round(nprim_total / max(rate * cpu_seconds, 1.0)))))
    t0 = time.perf_counter()
    _, _, nq2, npq2 = ob.jk_strided(T, cfg.tau, Q, stride2, stride2 // 2)
    dt2 = time.perf_counter() - t0
    frac = npq2 / nprim_total
    t_pass = dt2 / frac
    desc = ("oracle_jk over bra shell pairs ab %% %d == %d of config %d: %d of %.4g unique shell quartets, %.4g of "
            "%.4g primitive quartets (fraction %.5f of one ERI pass, tau=%g, nvec=%d) in %.1f s, scaled to one "
            "pass; MO<->AO transforms (<1%% of the flops) not included"
            % (stride2, stride2 // 2, cfg_k, nq2, nq_total, npq2, nprim_total, frac, cfg.tau, nvec, dt2))
    return nvec / t_pass, num_threads(), desc, t_pass


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    k = args.config
    from workloads import get_config
    cfg = get_config(k)
    ntraj = args.ntraj or len(cfg.fields)
    nvec = 2 * ntraj
    vals, desc, cores = [], "", 0
    per = max(5.0, min(30.0, 120.0 / max(args.steps + args.warmup, 1)))
    for i in range(args.warmup + args.steps):
        v, cores, desc, t_pass = oracle_sample(k, nvec, per)
        if i >= args.warmup:
            vals.append((v, t_pass))
    v = float(np.mean([x[0] for x in vals]))
    t_step = 4.0 * float(np.mean([x[1] for x in vals]))
    out = {"impl": "reference", "metric": metric_name(cfg.nocc + cfg.nvirt), "value": v, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "config %d (%s): %d AO, nocc %d, nvirt %d, ntraj %d (nvec %d), tau %g; one step = "
                                  "one RK4 step = 4 ERI passes" % (k, cfg.name, cfg.nocc + cfg.nvirt, cfg.nocc,
                                                                  cfg.nvirt, ntraj, nvec, cfg.tau)},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                            "extrapolated": True, "scatter": "values of repeated samples differ by up to 2x (dynamic OpenMP "
                            "schedule over bra pairs of very different cost); read as an order of magnitude"},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ------------------------------------------------------------------------------------------ B200 arm
def run_b200(args):
    import torch
    import paper_2601_16949_b200 as R
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    k = args.config
    t0 = time.perf_counter()
    cfg, basis, C_o, C_v, eps, cond, bump = build_inputs(k, R.rttda_overlap)
    st = torch.cuda.current_stream()
    tau = args.tau if args.tau > 0 else cfg.tau
    Co_d, Cv_d = torch.from_numpy(C_o).to(dev), torch.from_numpy(C_v).to(dev)
    cx, cx_lr, rs_omega = (float(x) for x in args.exchange.split(","))
    h = R.Rttda(basis, Co_d, Cv_d, eps, cx, tau, st)
    if cx_lr != 0.0 and rs_omega > 0.0:
        h.rttda_set_option(R.OPT_CX_LR, cx_lr)
        h.rttda_set_option(R.OPT_RS_OMEGA, rs_omega)
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    info = h.info()
    ncsf, n1 = h.ncsf, h.ncsf + 1

    # carrier frequency (R9/R10): configs 3 and 4 name an eigenvalue of A.  rttda_eigs (block Davidson on multi-vector
    # sigma builds) gives the lowest states; config 3 takes the lowest one, config 4 half the excitation energy of the
    # BRIGHT state, i.e. the one with the largest z-dipole weight |d_z . x_I|^2 among them.  Loose tolerance: any
    # recorded omega serves the timing, and the value is printed.
    D = R.rttda_dipole_ao(basis)
    dz = (C_o.T @ D[2] @ C_v).reshape(-1)
    nst = 1 if k == 3 else 6
    if args.omega > 0:
        nst = 0
    Xe = torch.zeros((max(nst, 1), ncsf), dtype=torch.float64, device=dev)
    t_e = time.perf_counter()
    if nst:
        om_e, res_e, it_e, nsig_e = h.rttda_eigs(nst, Xe, max(nst, 6), tol=1e-4, maxiter=40 if k != 4 else 12, stream=st,
                                                 allow_nonconverged=True)
        torch.cuda.synchronize()
        eigs_s = time.perf_counter() - t_e
        wts = (Xe.cpu().numpy() @ dz) ** 2
        bright = int(np.argmax(wts))
        omega = float(om_e[0]) if k != 4 else 0.5 * float(om_e[bright])
        eigs_info = {"omega_states": [float(x) for x in om_e], "residuals": [float(x) for x in res_e], "iterations": it_e,
                     "sigma_vectors": nsig_e, "seconds": eigs_s, "bright_state": bright,
                     "dipole_weights": [float(x) for x in wts]}
    else:
        omega, eigs_info = args.omega, "--omega given"
    fields = fields_for(cfg, args.ntraj, omega)
    ntraj = len(fields)
    nvec = 2 * ntraj

    y0 = np.zeros((ntraj, 2, n1))
    y0[:, 0, 0] = 1.0
    y = torch.from_numpy(y0).to(dev)
    log = torch.zeros((1, ntraj, 3), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    dt = cfg.dt if cfg.dt > 0 else 0.1

    sso = args.propagator == "sso"
    per_traj = 2.0 if sso else 8.0
    if sso:
        nvec = ntraj                      # one real plane per sigma build
    prop = h.rttda_propagate_sso if sso else h.rttda_propagate

    def step(i):
        prop(y, fields if i == 0 else cont, i * dt, dt, 1, log, st)

    cont = [dict(f, **{"continue": True}) for f in fields]      # RTTDA_FIELD_CONTINUE: no second kick, R(t) reference kept
    for i in range(args.warmup):
        step(i)
        flush.zero_()
    barrier()
    h.rttda_jk_time()
    l0 = h.rttda_get_info("kernel_launches")
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for i in range(args.steps):
        ev[i][0].record(st)
        step(args.warmup + i)
        ev[i][1].record(st)
        flush.zero_()
    barrier()
    clocks = sampler.stop()
    ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(ms))
    jk_ms, jk_n = h.rttda_jk_time()
    info["flops_eval"] = h.rttda_get_info("flops_eval")      # counted by the kernels of the last timed ERI pass
    info["nprim_eval"] = h.rttda_get_info("nprim_eval")
    launches = int(h.rttda_get_info("kernel_launches") - l0)
    total_ms = reduce_max(total_ms, world, dev)
    ms_per_step = total_ms / args.steps
    value = aggregate_value(ntraj, world, ms_per_step, per_traj)

    # end to end: host buffers through rttda_propagate_host (H2D of the state, D2H of state + log inside)
    yh = torch.from_numpy(y0.copy()).pin_memory()
    lh = torch.zeros((1, ntraj, 3), dtype=torch.float64).pin_memory()
    h.rttda_propagate_host(yh.numpy(), fields, 0.0, dt, 1, lh.numpy(), st)
    barrier()
    e0 = time.perf_counter()
    for i in range(args.steps):
        h.rttda_propagate_host(yh.numpy(), cont, (i + 1) * dt, dt, 1, lh.numpy(), st)
    barrier()
    e2e_s = time.perf_counter() - e0
    e2e_s = reduce_max(e2e_s, world, dev)
    e2e_val = aggregate_value(ntraj, world, e2e_s * 1e3 / args.steps, 8.0)
    h2d = yh.numel() * 8
    d2h = yh.numel() * 8 + lh.numel() * 8

    # optional in-core mode (NOT the headline: the evaluation is skipped after the first pass; include/rttda.h)
    incore = None
    if world == 1 and not sso:
        try:
            h.rttda_set_option(R.OPT_INCORE, 1)
            yi = torch.from_numpy(y0).to(dev)
            h.rttda_propagate(yi, fields, 0.0, dt, 1, log, st)                   # fills the store
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            for i in range(args.steps):
                h.rttda_propagate(yi, cont, (i + 1) * dt, dt, 1, log, st)
            b.record(st)
            torch.cuda.synchronize()
            ms_i = a.elapsed_time(b) / args.steps
            incore = {"sigma_vectors_per_s": 8.0 * ntraj / (ms_i * 1e-3), "ms_per_step": ms_i,
                      "store_bytes": info["eri_all_bytes"],
                      "note": "RTTDA_OPT_INCORE: integrals resident in HBM, evaluation skipped after the first pass; "
                              "not the paper's direct method and not the headline value"}
        except R.RttdaError as e:
            incore = {"unavailable": str(e)}
        finally:
            h.rttda_set_option(R.OPT_INCORE, 0)
    # roofline of the dominant kernel group (the J/K ERI pass): algorithmic flops / measured device time.  The evaluation
    # part is counted by the kernels themselves (primitive quartets actually evaluated in the last ERI pass).
    flops_pass = info["flops_eval"] + nvec * info["flops_digest_per_vec"]
    jk_src = "CUDA events around every ERI pass of the timed steps (rttda_jk_time)"
    if jk_n == 0:
        # graph-replayed steps (RTTDA_OPT_GRAPH, small molecules) carry no per-pass events: time the ERI pass of one
        # rttda_sigma call on the same number of vectors instead
        from workloads import make_vectors
        Xs = torch.from_numpy(make_vectors(cfg, nvec)).to(dev)
        Ss = torch.empty_like(Xs)
        for _ in range(3):
            h.rttda_sigma(Xs, Ss, st)
        torch.cuda.synchronize()
        jk_ms, jk_n = h.rttda_last_timings()["jk_ms"], 1
        jk_src = "ERI pass of one rttda_sigma call on nvec vectors (the timed steps were CUDA-graph replays without per-pass events)"
    jk_avg_ms = jk_ms / max(jk_n, 1)
    achieved = flops_pass / (jk_avg_ms * 1e-3) / 1e12
    peak = R.rttda_fp64_peak(1.0, st)
    # DRAM bytes of one ERI pass from the committed ncu launch list of this same command (profiles/README.md)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "r2_traffic_per_pass.txt")
    if k == 4 and nvec == 6 and os.path.exists(tpath):
        with open(tpath) as f:
            tj = json.load(f)
        traffic = tj["dram_read_bytes"] + tj["dram_write_bytes"]
    out = None
    if rank == 0:
        out = {"metric": metric_name(h.nao), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
               "vs_baseline": None, "dtype": "f64", "data": "synthetic",
               "config": {"workload": "config %d (%s): %d AO, nocc %d, nvirt %d, %d singles, ntraj %d (nvec %d per ERI "
                                      "pass), tau %g, dt %g; one step = one RK4 step of rttda_propagate = 4 ERI passes "
                                      "+ 16 GEMM launches + field + combine" % (k, cfg.name, h.nao, h.nocc, h.nvirt,
                                                                               ncsf, ntraj, nvec, tau, dt),
                          "l2": "256 MiB buffer written between timed steps (L2 flush)",
                          "exchange": {"cx": cx, "cx_lr": cx_lr, "rs_omega": rs_omega,
                                       "eri_passes_per_sigma": 2 if (cx_lr != 0.0 and rs_omega > 0.0) else 1},
                          "parallelism": "replicas" if world > 1 else "1 GPU", "omega": omega,
                          "propagator": args.propagator + (" (one call per step: H(t0) q is recomputed, 3 sigma builds "
                                                           "of ntraj vectors per timed step)" if sso else ""),
                          "cond_S": cond, "seed_bump": bump, "omega_from": eigs_info},
               "rt_tda_steps_per_s": world * 1e3 / ms_per_step,
               "eri_quartets_per_s": info["nquartets"] / (jk_avg_ms * 1e-3),
               "counts": {"shell_pairs_kept": info["npairs_kept"], "unique_shell_quartets": info["nquartets"],
                          "primitive_quartets": info["nprim_quartets"], "quartets_evaluated": info["nquartets_eval"],
                          "primitive_evaluated": info["nprim_eval"], "flops_eval_per_pass": info["flops_eval"],
                          "flops_digest_per_vec": info["flops_digest_per_vec"],
                          "eri_staging_buffer_bytes": info["eri_buf_bytes"]},
               "setup_s": setup_s, "create_ms": info["create_ms"],
               "jk_ms_per_pass": jk_avg_ms, "jk_ms_source": jk_src,
               "jk_share_of_step": 4.0 * jk_avg_ms / ms_per_step if not sso else None,
               "roofline": {"bound": "alu", "kernel": "eval_kernel<*> + digest_j_kernel<*> + digest_k/b_kernel<*> (all launches of one ERI pass)",
                            "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                            "flop_model": "evaluation: per-class minimal McMurchie-Davidson count x primitive quartets the kernels "
                                          "EVALUATED (device counters, after primitive screening); digestion: 20 flops per "
                                          "integral value per density.  Round 1 counted every primitive quartet of the R14 "
                                          "quartets; on that count this pass reads %.3f" % (
                                              (info["nprim_quartets"] / max(info["nprim_eval"], 1.0) * info["flops_eval"]
                                               + nvec * info["flops_digest_per_vec"]) / (jk_avg_ms * 1e-3) / 1e12 / peak),
                            "traffic": traffic, "traffic_source": "NOT measured in this run: profiles/r2_traffic_per_pass.txt (ncu "
                            "dram__bytes_read+write summed over the launches of one ERI pass of this same command, config 4, "
                            "nvec 6)" if traffic else None,
                            "peak_source": "measured live: rttda_fp64_peak DFMA chain, 1 s "
                            "(MEASURED_PEAKS.json has no FP64 entry; nominal %.1f)" % FP64_NOMINAL_TFLOPS,
                            "flops_per_launch_group": flops_pass},
               "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
               "incore_mode": incore, "gpu_launches": launches, "clocks": clocks}
    # the same step at the tighter threshold at which sigma meets the oracle tolerance at this size (config 4 only)
    at_parity = None
    if k == 4 and world == 1 and not sso and args.parity_tau > 0 and args.parity_tau != tau:
        h.close()
        h = R.Rttda(basis, Co_d, Cv_d, eps, 1.0, args.parity_tau, st)
        yp = torch.from_numpy(y0).to(dev)
        h.rttda_propagate(yp, fields, 0.0, dt, 1, log, st)
        torch.cuda.synchronize()
        h.rttda_jk_time()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(st)
        for i in range(args.steps):
            h.rttda_propagate(yp, cont, (i + 1) * dt, dt, 1, log, st)
        b.record(st)
        torch.cuda.synchronize()
        ms_p = a.elapsed_time(b) / args.steps
        jk_p, jk_pn = h.rttda_jk_time()
        ip = h.info()                                    # after the timed passes: device-counted evaluation work
        fl_p = ip["flops_eval"] + nvec * ip["flops_digest_per_vec"]
        at_parity = {"tau": args.parity_tau, "sigma_vectors_per_s": 8.0 * ntraj / (ms_p * 1e-3), "ms_per_step": ms_p,
                     "jk_ms_per_pass": jk_p / max(jk_pn, 1), "unique_shell_quartets": ip["nquartets"],
                     "roofline_frac": fl_p / (jk_p / max(jk_pn, 1) * 1e-3) / 1e12 / peak,
                     "note": "sigma parity with the long-double oracle samples at 1280 AO is asserted at this tau "
                             "(tests/test_gpu_parity.py::test_sigma_config4_vs_stored_oracle_samples); tau = 1e-12 (R15) is "
                             "the headline configuration and its sigma error is a reported number (DESIGN.md section 11)"}
        out and out.update({"at_parity_tau": at_parity})
    h.close()
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            v, cores, desc, _ = oracle_sample(k, nvec, args.cpu_seconds)
            out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                   "extrapolated": True,
                                   "scatter": "a %.0f s sample scaled to one pass by its primitive-quartet share; repeated samples "
                                              "differ by up to 2x (bra pairs of very different cost under a dynamic OpenMP "
                                              "schedule): an order of magnitude, not a measurement of a full pass" % args.cpu_seconds}
        else:
            out["cpu_baseline"] = None
        print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()


# ------------------------------------------------------------------------------------------ config 5, one point under ncu
def run_sweep_point(args):
    import torch
    import paper_2601_16949_b200 as R
    from workloads import make_vectors
    nvec, tau = int(args.sweep_point[0]), float(args.sweep_point[1])
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    cfg, basis, C_o, C_v, eps, cond, bump = build_inputs(4, R.rttda_overlap)
    st = torch.cuda.current_stream()
    h = R.Rttda(basis, torch.from_numpy(C_o).to(dev), torch.from_numpy(C_v).to(dev), eps, 1.0, tau, st)
    X = torch.from_numpy(make_vectors(cfg, nvec)).to(dev)
    out = torch.empty_like(X)
    for _ in range(2):
        h.rttda_sigma(X, out, st)
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStart()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(st); h.rttda_sigma(X, out, st); b.record(st)
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStop()
    info = h.info()
    print(json.dumps({"nvec": nvec, "tau": tau, "ms": a.elapsed_time(b), "unique_shell_quartets": info["nquartets"],
                      "primitive_quartets": info["nprim_quartets"]}))
    h.close()


# ------------------------------------------------------------------------------------------ config 5 sweep
def run_sweep(args):
    """BJ:configs[4]: batched sigma microbenchmark at the 1280-AO molecule, nvec x tau; 3 warm-ups + 10 timed
    rttda_sigma calls per point (CUDA events on the call's stream), median and min.  The error column compares
    against the GPU result at tau = 1e-14 (convergence under screening; oracle parity at full size is the sampled
    test in tests/test_gpu_parity.py)."""
    import torch
    import paper_2601_16949_b200 as R
    from workloads import make_vectors
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    cfg, basis, C_o, C_v, eps, cond, bump = build_inputs(4, R.rttda_overlap)
    st = torch.cuda.current_stream()
    peak = R.rttda_fp64_peak(1.0, st)
    Co, Cv = torch.from_numpy(C_o).to(dev), torch.from_numpy(C_v).to(dev)
    points, ref = [], {}
    for tau in (1e-14, 1e-12, 1e-10):
        h = R.Rttda(basis, Co, Cv, eps, 1.0, tau, st)
        info = h.info()
        for nvec in (2, 8, 16, 32):
            X = torch.from_numpy(make_vectors(cfg, nvec)).to(dev)
            out = torch.empty_like(X)
            for _ in range(3):
                h.rttda_sigma(X, out, st)
            torch.cuda.synchronize()
            h.rttda_jk_time()
            ms = []
            for _ in range(10):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(st); h.rttda_sigma(X, out, st); b.record(st)
                torch.cuda.synchronize()
                ms.append(a.elapsed_time(b))
            jk_ms, jk_n = h.rttda_jk_time()
            jk = jk_ms / max(jk_n, 1)
            res = out.cpu().numpy()
            if tau == 1e-14:
                ref[nvec] = res
            err = float(np.max(np.abs(res - ref[nvec])) / np.max(np.abs(ref[nvec])))
            flops = h.rttda_get_info("flops_eval") + nvec * info["flops_digest_per_vec"]     # counted by the last pass
            points.append({"tau": tau, "nvec": nvec, "primitive_quartets_evaluated": h.rttda_get_info("nprim_eval"), "ms_median": float(np.median(ms)), "ms_min": float(min(ms)),
                           "sigma_vectors_per_s": nvec / (float(np.median(ms)) * 1e-3),
                           "eri_quartets_per_s": info["nquartets"] / (jk * 1e-3), "jk_ms": jk,
                           "unique_shell_quartets": info["nquartets"], "primitive_quartets": info["nprim_quartets"],
                           "fp64_roofline_frac": flops / (jk * 1e-3) / 1e12 / peak,
                           "rel_inf_err_vs_tau1e-14": err})
            print(json.dumps(points[-1]), file=sys.stderr)
        h.close()
    out = {"metric": "sigma_sweep_1280ao", "unit": UNIT, "fp64_peak_tflops": peak, "cond_S": cond, "points": points}
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    with open(os.path.join(ROOT, "gpurun_out", "sweep.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out))


if __name__ == "__main__":
    a = parse()
    if a.sweep_point:
        run_sweep_point(a)
    elif a.sweep:
        run_sweep(a)
    elif a.impl == "reference":
        run_reference(a)
    else:
        run_b200(a)
