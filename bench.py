#!/usr/bin/env python
"""bench.py — throughput of the whole hot path on BASELINE.json configs[1] (class sweep).

One "step" = one pass of lx_eri3_batch over all 45 (Lx|LaLb) classes of config 2 (Lx 0..4; La,Lb 0..2; primary K=3,
aux K=1 → K_total = 9; 1024 shell pairs x 256 aux shells per class = 262 144 shell-sets per class), i.e. Boys → VRR1 →
VRR2 → contraction → HRR → store for 11.8 M shell-sets / 0.92 G integrals (7.3 GB of output), inputs resident in HBM.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Prints ONE JSON line (contract in the task statement).  `--impl reference` times the CPU oracle (as it stands) on the
host cores for the same metric on a bounded sample of the same workload.
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

import lx_inputs as gen  # noqa: E402

METRIC = "3-center integrals/sec (class sweep, config 2)"
UNIT = "integrals/s"
WORKLOAD = "configs[1]: 45 classes (Lx 0..4 | La,Lb 0..2), K_total=9, 1024 pairs x 256 aux per class"
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 FMA/clk/SM x 2 x sm_max_mhz
HBM_PEAK_GBS = 6555.5                                   # BASELINE.md §2 (MEASURED_PEAKS.json of round 1; overridden below if the file is there)
# dram__bytes_read.sum + dram__bytes_write.sum per launch, copied from the tracked ncu --set full summaries under
# profiles/ (never measured by this run: ncu is not available inside a timed bench); class -> (bytes, source file)
NCU_422_WRITE, NCU_422_READ = 1.072212e9, 1.057e6
NCU_DRAM_BYTES_PER_LAUNCH = {(4, 2, 2): (NCU_422_WRITE + NCU_422_READ, "profiles/r02_ncu_chain_4_2_2.md (ncu --set full capture, end of round 2)")}
# SURVEY.md §8(d) table, flops per shell-set for the classes it lists (K = 9 for config 2; config 3 as stated there)
SURVEY_FLOPS_PER_SET = {(0, 0, 0): 414, (1, 1, 1): 2286, (2, 1, 1): 6156, (2, 2, 2): 24816, (3, 2, 2): 52970,
                        (4, 1, 1): 29322, (4, 2, 2): 111054}
SURVEY_FLOPS_CONFIG3 = {(6, 2, 2, 1): 43792, (5, 3, 3, 1): 70320, (6, 3, 3, 1): 116448, (4, 4, 4, 1): 93910,
                        (5, 2, 2, 5): 566418}


def _measured_hbm():
    """HBM peak of this pool's B200s as the driver measured it (MEASURED_PEAKS.json), else the BASELINE.md figure."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json"
    except Exception:
        return HBM_PEAK_GBS, "BASELINE.md section 2 (MEASURED_PEAKS.json absent)"


def ncart(l):
    return (l + 1) * (l + 2) // 2


def nint_set(c):
    return ncart(c[0]) * ncart(c[1]) * ncart(c[2])


class ClockSampler:
    """Samples nvidia-smi SM clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(classes, npair_s, nx_s, seed):
    """Oracle (double instantiation, OpenMP over pairs) on the first npair_s pairs x nx_s aux shells of every class."""
    import oracle
    oracle.build()
    total_int, total_t = 0, 0.0
    for c in classes:
        cfg = gen.config2(*c, seed=seed)
        t0 = time.perf_counter()
        o = oracle.eri3_batch(c[0], c[1], c[2], cfg["aux"], cfg["prim"], cfg["x_idx"][:nx_s], cfg["pair_idx"][:npair_s], real="d")
        total_t += time.perf_counter() - t0
        total_int += o.size
    return total_int, total_t, oracle.max_threads()


def run_reference(args, rank, world):
    if rank != 0:
        return
    classes = gen.CONFIG2_CLASSES
    npair_s, nx_s = 32, 256
    times = []
    nint = 0
    for it in range(args.warmup + args.steps):
        n, t, cores = oracle_sample(classes, npair_s, nx_s, seed=2)
        nint = n
        if it >= args.warmup:
            times.append(t)
    tot = sum(times)
    val = nint * len(times) / tot
    sample = f"first {npair_s} pairs x {nx_s} aux shells of each of the 45 classes per step ({nint} integrals)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def _time_calls(fn, reps, flush=None):
    """CUDA-event times (ms) of `reps` calls of fn() on the current stream, each bracketed by a synchronize; the L2 is
    flushed before every call when `flush` is given."""
    import torch
    out = []
    for _ in range(reps):
        if flush is not None:
            flush.fill_(1)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a0.record()
        fn()
        a1.record()
        torch.cuda.synchronize()
        out.append(a0.elapsed_time(a1))
    return out


def bench_config1(lx, dev):
    """configs[0]: (d|pp), 64 pairs x 32 aux shells, K = 1 — launch-latency-sized: the time
    of ONE lx_eri3_batch call (pre-pass + class kernel), median of 200 calls, and the back-to-back rate."""
    import torch
    cfg = gen.config1()
    da, dp = lx.DeviceShells(cfg["aux"], dev), lx.DeviceShells(cfg["prim"], dev)
    dx, dpr = torch.from_numpy(cfg["x_idx"]).to(dev), torch.from_numpy(cfg["pair_idx"]).to(dev)
    out = torch.empty((64, 32, 6, 3, 3), dtype=torch.float64, device=dev)
    ws = torch.empty(lx.lx_eri3_workspace_bytes(2, 1, 1, 32, 64, 1), dtype=torch.uint8, device=dev)

    def call():
        lx.lx_eri3_batch(2, 1, 1, da, dp, dx, dpr, out=out, workspace=ws, kmax=1)
    for _ in range(10):
        call()
    ms = _time_calls(call, 200)
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a0.record()
    for _ in range(200):
        call()
    a1.record()
    torch.cuda.synchronize()
    b2b = a0.elapsed_time(a1) / 200
    nint = out.numel()
    return {"workload": "configs[0]: class (2|11), 64 pairs x 32 aux shells, K=1, 110 592 integrals, 0.885 MB",
            "us_per_call_median": 1e3 * float(np.median(ms)), "us_per_call_min": 1e3 * float(np.min(ms)),
            "us_per_call_back_to_back": 1e3 * b2b, "integrals_per_s_back_to_back": nint / (b2b * 1e-3),
            "launches_per_call": 2, "note": "device time between CUDA events around one C-ABI call; launch-latency-bound"}


def bench_config3(lx, dev, costmodel):
    """configs[2]: the five high-angular-momentum classes at 4096 pairs x 128 aux shells, one at a time (3.2-14.2 GB of
    output each, far beyond the L2).  Per class: ms (median of 5 after 2 warm-ups), integrals/s, and the fraction of the
    class's own floor max(8*nint / HBM peak, SURVEY.md §8(d) flops / FP64 peak)."""
    import torch
    res = {}
    buf = None
    hbm, hbm_src = _measured_hbm()
    for cls in gen.CONFIG3_CLASSES:
        lxa, la, lb, k = cls
        cfg = gen.config3(lxa, la, lb, kprim=k)
        da, dp = lx.DeviceShells(cfg["aux"], dev), lx.DeviceShells(cfg["prim"], dev)
        dx, dpr = torch.from_numpy(cfg["x_idx"]).to(dev), torch.from_numpy(cfg["pair_idx"]).to(dev)
        nset = 4096 * 128
        nint = nset * ncart(lxa) * ncart(la) * ncart(lb)
        if buf is None or buf.numel() < nint:
            buf = None
            buf = torch.empty(nint, dtype=torch.float64, device=dev)
        ws = torch.empty(lx.lx_eri3_workspace_bytes(lxa, la, lb, 128, 4096, k * k), dtype=torch.uint8, device=dev)

        def call():
            lx.lx_eri3_batch(lxa, la, lb, da, dp, dx, dpr, out=buf[:nint], workspace=ws, kmax=k * k)
        call()
        call()
        ms = float(np.median(_time_calls(call, 5)))
        t_hbm = 8.0 * nint / (hbm * 1e9) * 1e3
        fl_s, fl_m = SURVEY_FLOPS_CONFIG3[cls], costmodel.flops_per_set(lxa, la, lb, k * k)
        t_f64 = fl_s * nset / (FP64_NOMINAL_TFLOPS * 1e12) * 1e3
        floor = max(t_hbm, t_f64)
        res[f"({lxa}|{la}{lb}) K={k * k}"] = {
            "kernel": lx.lx_kernel_family_k(lxa, la, lb, k * k), "ms": ms, "integrals_per_s": nint / (ms * 1e-3),
            "shell_sets_per_s": nset / (ms * 1e-3), "hbm_write_gbs": 8.0 * nint / (ms * 1e-3) / 1e9,
            "floor_ms_hbm": t_hbm, "floor_ms_fp64_survey_flops": t_f64, "bound": "hbm" if t_hbm >= t_f64 else "alu",
            "frac_of_floor": floor / ms, "tflops_survey_count": fl_s * nset / (ms * 1e-3) / 1e12,
            "tflops_costmodel_count": fl_m * nset / (ms * 1e-3) / 1e12}
    return {"workload": "configs[2]: 4096 pairs x 128 aux shells per class, 256 atoms >= 1.5 bohr apart in a 15-bohr cube",
            "peaks": {"hbm_gbs": hbm, "hbm_source": hbm_src, "fp64_tflops": FP64_NOMINAL_TFLOPS}, "classes": res}


def _df_model_flops(costmodel, aux, prim, pairs, qx, qp, tau):
    """Cost-model flops of one DF pass: sum over (aux L,K) x (pair La,Lb,KaKb) buckets of surviving sets x flops/set."""
    La, Lb = prim.L[pairs[:, 0]], prim.L[pairs[:, 1]]
    la, lb = np.maximum(La, Lb), np.minimum(La, Lb)
    kab = prim.K[pairs[:, 0]] * prim.K[pairs[:, 1]]
    key = (la.astype(np.int64) * 8 + lb) * 4096 + kab
    total = 0.0
    for lxa in np.unique(aux.L):
        for kx in np.unique(aux.K[aux.L == lxa]):
            sel = (aux.L == lxa) & (aux.K == kx)
            if qx is None:
                cnt = np.full(len(pairs), int(sel.sum()), dtype=np.int64)
            else:
                qs = np.sort(qx[sel])
                # survivors: qx >= tau / qp  (the schedule takes the decision as qx*qp >= tau; the model only needs counts)
                with np.errstate(divide="ignore"):
                    cnt = len(qs) - np.searchsorted(qs, tau / np.maximum(qp, 1e-300), side="left")
            for kk in np.unique(key):
                m = key == kk
                n = int(cnt[m].sum())
                if n:
                    c = int(kk // 4096)
                    total += n * costmodel.flops_per_set(int(lxa), c // 8, c % 8, int(kk % 4096) * int(kx))
    return total


def bench_df(lx, dev, costmodel, cfg, name, reps, unscreened=False):
    """BASELINE.json metric "DF-J time": integral-direct gamma and J through lx_df_gamma / lx_df_J with Schwarz screening at
    the config's tau.  The Schwarz factors are made on the GPU (lx_schwarz_*_host), the schedule on the host; both are
    once-per-basis steps, timed and reported beside the per-iteration DF-J time, not inside it."""
    import torch
    aux, prim, pairs, tau = cfg["aux"], cfg["prim"], cfg["pair_idx"], cfg["tau"]
    ha, hp = lx.HostShells(aux), lx.HostShells(prim)
    t0 = time.perf_counter()
    qx = lx.lx_schwarz_aux_host(ha)
    qp = lx.lx_schwarz_pair_host(hp, pairs)
    t_q = time.perf_counter() - t0
    t0 = time.perf_counter()
    sched = lx.Schedule(ha, hp, qx, qp, pairs, tau)
    t_s = time.perf_counter() - t0
    da, dp = lx.DeviceShells(ha, dev), lx.DeviceShells(hp, dev)
    D, d = torch.from_numpy(cfg["D"]).to(dev), torch.from_numpy(cfg["d"]).to(dev)
    ws = torch.empty(sched.workspace_bytes, dtype=torch.uint8, device=dev)
    gam = torch.empty(aux.nbf, dtype=torch.float64, device=dev)
    J = torch.empty((prim.nbf, prim.nbf), dtype=torch.float64, device=dev)

    def run(sc):
        lx.lx_df_gamma(sc, da, dp, D, gamma=gam, workspace=ws)
        torch.cuda.synchronize()
        mg = min(_time_calls(lambda: lx.lx_df_gamma(sc, da, dp, D, gamma=gam, workspace=ws), reps))
        lx.lx_df_J(sc, da, dp, d, J=J, workspace=ws)
        torch.cuda.synchronize()
        mj = min(_time_calls(lambda: lx.lx_df_J(sc, da, dp, d, J=J, workspace=ws), reps))
        return mg, mj
    mg, mj = run(sched)
    lhs, rhs = float(gam @ d), float((J * D).sum())
    # end to end for the digestion path: D and d come from pinned host memory, gamma and J go back to pinned host memory, all
    # inside the timed interval (wall clock around copies + both passes + synchronisation); tables and schedule are resident
    D_h, d_h = torch.from_numpy(cfg["D"]).pin_memory(), torch.from_numpy(cfg["d"]).pin_memory()
    g_h = torch.empty(aux.nbf, dtype=torch.float64).pin_memory()
    J_h = torch.empty((prim.nbf, prim.nbf), dtype=torch.float64).pin_memory()

    def e2e_once():
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        D.copy_(D_h, non_blocking=True)
        d.copy_(d_h, non_blocking=True)
        lx.lx_df_gamma(sched, da, dp, D, gamma=gam, workspace=ws)
        lx.lx_df_J(sched, da, dp, d, J=J, workspace=ws)
        g_h.copy_(gam, non_blocking=True)
        J_h.copy_(J, non_blocking=True)
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) * 1e3
    e2e_once()
    e2e_ms = min(e2e_once() for _ in range(max(1, reps)))
    e2e = {"df_j_ms": e2e_ms, "integrals_per_s": 2 * sched.num_integrals / (e2e_ms * 1e-3),
           "h2d_bytes": int(D_h.numel() * 8 + d_h.numel() * 8), "d2h_bytes": int(g_h.numel() * 8 + J_h.numel() * 8),
           "note": "wall clock: H2D of D and d from pinned memory, lx_df_gamma, lx_df_J, D2H of gamma and J, synchronise"}
    # the steps between the two passes: metric V = (X|Y) and its Cholesky factor once per basis,
    # d = V^-1 gamma once per iteration (here: on the gamma of pass 1; the timed J pass above uses the synthetic d)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    V = lx.lx_metric_2c(ha)
    t_met1 = time.perf_counter() - t0                 # first call: the driver also sizes the kernels' local-memory stacks
    t0 = time.perf_counter()
    lx.lx_metric_2c(ha, V)
    t_met = time.perf_counter() - t0
    fit = {"naux": aux.nbf, "metric_s": t_met, "metric_first_call_s": t_met1, "metric_integrals_per_s": aux.nbf * (aux.nbf + 1) / 2 / t_met,
           "note": "lx_metric_2c (own kernel, one thread per aux shell pair) on the whole aux basis; lx_fit_solve (cuSOLVER "
                   "potrf / potrs) on the conditioned subset lx_inputs.fit_subset (the synthetic basis with its zeta = 0.1 "
                   "shells is numerically singular, DESIGN.md); wall clock; once-per-basis steps except solve_ms"}
    sub, keep = gen.fit_subset(aux)
    keep = torch.as_tensor(keep, device=dev)
    Vs = V[keep][:, keep].contiguous()
    del V
    gs = gam[keep].contiguous()
    try:
        t0 = time.perf_counter()
        lx.lx_fit_solve(Vs, None)
        fit["cholesky_s"] = time.perf_counter() - t0
        dfit = gs.clone()
        lx.lx_fit_solve(Vs, dfit, factored=True)
        t_sol = []
        for _ in range(max(1, reps)):
            dfit.copy_(gs)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            lx.lx_fit_solve(Vs, dfit, factored=True)
            t_sol.append((time.perf_counter() - t0) * 1e3)
        fit.update({"naux_fit": sub.nbf, "solve_ms": min(t_sol)})
    except lx.LxError as e:
        fit["fit_error"] = str(e)
    del Vs
    fl = _df_model_flops(costmodel, aux, prim, pairs, qx, qp, tau)
    floor_ms = fl / (FP64_NOMINAL_TFLOPS * 1e12) * 1e3
    res = {"workload": name, "screening": f"Schwarz, tau = {tau:g}, factors made on the GPU (lx_schwarz_aux_host / lx_schwarz_pair_host)",
           "nbf": prim.nbf, "naux": aux.nbf, "shell_pairs": len(pairs), "aux_shells": aux.nshell,
           "shell_sets": sched.num_sets, "integrals": sched.num_integrals,
           "surviving_fraction": sched.num_sets / (len(pairs) * aux.nshell),
           "gamma_ms": mg, "J_ms": mj, "df_j_ms": mg + mj,
           "integrals_per_s": 2 * sched.num_integrals / ((mg + mj) * 1e-3),
           "fp64_floor_ms_per_pass_costmodel": floor_ms, "frac_of_fp64_floor": 2 * floor_ms / (mg + mj),
           "check_gamma_dot_d": lhs, "check_J_dot_D": rhs, "check_rel_diff": abs(lhs - rhs) / max(abs(lhs), 1e-300),
           "schwarz_s": t_q, "schedule_s": t_s, "e2e": e2e, "fit": fit}
    if unscreened:
        s0 = lx.Schedule(ha, hp, None, None, pairs, 0.0)
        ug, uj = run(s0)
        res["unscreened"] = {"shell_sets": s0.num_sets, "integrals": s0.num_integrals, "gamma_ms": ug, "J_ms": uj,
                             "integrals_per_s": 2 * s0.num_integrals / ((ug + uj) * 1e-3)}
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--npair", type=int, default=1024, help="pairs per class (default = config 2)")
    ap.add_argument("--nx", type=int, default=256, help="aux shells per class (default = config 2)")
    ap.add_argument("--classes", default="", help="profiling aid: restrict the sweep to e.g. '4,2,1;4,0,0' (default: all 45)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--streams", type=int, default=2, help="CUDA streams the classes of a step are spread over")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-df", action="store_true", help="skip the DF-J (configs 4, 5) and solid-harmonic side measurements")
    ap.add_argument("--no-side", action="store_true", help="skip the config 1 / config 3 side measurements")
    ap.add_argument("--df-once", default="", choices=["", "4", "5"],
                    help="profiling aid: ONE lx_df_gamma + ONE lx_df_J call on configs[3] (4) or configs[4] (5) with GPU-made Schwarz "
                         "factors, print the two times and exit")
    ap.add_argument("--c3", default="", help="profiling aid: run ONLY the given config-3 class, e.g. '6,3,3,1' (lx,la,lb,kprim), "
                                             "three calls at full size (4096 pairs x 128 aux shells), print its time and exit")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        raise SystemExit(f"bench.py --gpus {args.gpus} but WORLD_SIZE={world}: launch N ranks with "
                         f"`python -m torch.distributed.run --nnodes=1 --nproc-per-node {args.gpus} --master-addr 127.0.0.1 "
                         f"bench.py --gpus {args.gpus} ...` (one process per GPU)")
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2210_03192_b200 import lx, costmodel
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    lx.lx_init(local)

    if args.df_once:
        cfg = gen.config4() if args.df_once == "4" else gen.config5()
        ha, hp = lx.HostShells(cfg["aux"]), lx.HostShells(cfg["prim"])
        qx, qp = lx.lx_schwarz_aux_host(ha), lx.lx_schwarz_pair_host(hp, cfg["pair_idx"])
        sched = lx.Schedule(ha, hp, qx, qp, cfg["pair_idx"], cfg["tau"])
        da, dp = lx.DeviceShells(ha, dev), lx.DeviceShells(hp, dev)
        D, d = torch.from_numpy(cfg["D"]).to(dev), torch.from_numpy(cfg["d"]).to(dev)
        ws = torch.empty(sched.workspace_bytes, dtype=torch.uint8, device=dev)
        gam = torch.empty(cfg["aux"].nbf, dtype=torch.float64, device=dev)
        J = torch.empty((cfg["prim"].nbf, cfg["prim"].nbf), dtype=torch.float64, device=dev)
        mg = _time_calls(lambda: lx.lx_df_gamma(sched, da, dp, D, gamma=gam, workspace=ws), 1)[0]
        mj = _time_calls(lambda: lx.lx_df_J(sched, da, dp, d, J=J, workspace=ws), 1)[0]
        print(json.dumps({"df_once": args.df_once, "shell_sets": sched.num_sets, "gamma_ms": mg, "J_ms": mj,
                          "check_gamma_dot_d": float(gam @ d), "check_J_dot_D": float((J * D).sum())}))
        return
    if args.c3:
        lxa, la, lb, k = (int(v) for v in args.c3.split(","))
        cfg = gen.config3(lxa, la, lb, kprim=k)
        da, dp = lx.DeviceShells(cfg["aux"], dev), lx.DeviceShells(cfg["prim"], dev)
        dx, dpr = torch.from_numpy(cfg["x_idx"]).to(dev), torch.from_numpy(cfg["pair_idx"]).to(dev)
        out = torch.empty(4096 * 128 * ncart(lxa) * ncart(la) * ncart(lb), dtype=torch.float64, device=dev)
        ws = torch.empty(lx.lx_eri3_workspace_bytes(lxa, la, lb, 128, 4096, k * k), dtype=torch.uint8, device=dev)
        ms = _time_calls(lambda: lx.lx_eri3_batch(lxa, la, lb, da, dp, dx, dpr, out=out, workspace=ws, kmax=k * k), 3)
        print(json.dumps({"config3_class": args.c3, "kernel": lx.lx_kernel_family_k(lxa, la, lb, k * k), "ms": ms}))
        return

    # ---- inputs: one full config-2 batch per rank (weak scaling: independent shell-sets, no collective) --------
    classes = gen.CONFIG2_CLASSES
    if args.classes:
        classes = [tuple(int(v) for v in c.split(",")) for c in args.classes.split(";")]
    seed = 2 + 1000 * rank                    # config index; other ranks draw their own batch
    host, devs = {}, {}
    for c in classes:
        cfg = gen.config2(*c, npair=args.npair, nx=args.nx, seed=seed)
        ha, hp = lx.HostShells(cfg["aux"]), lx.HostShells(cfg["prim"])
        host[c] = (ha, hp, cfg["x_idx"], cfg["pair_idx"])
        devs[c] = (lx.DeviceShells(ha, dev), lx.DeviceShells(hp, dev),
                   torch.from_numpy(cfg["x_idx"]).to(dev), torch.from_numpy(cfg["pair_idx"]).to(dev))
    nsets = args.npair * args.nx
    max_int = max(nint_set(c) for c in classes) * nsets
    # every class has its own output region and workspace, so that classes may run concurrently on several streams
    ints_cls = [nint_set(c) * nsets for c in classes]
    offs = np.concatenate([[0], np.cumsum(ints_cls)])
    out_all = torch.empty(int(offs[-1]), dtype=torch.float64, device=dev)
    outs = [out_all[int(offs[i]):int(offs[i + 1])] for i in range(len(classes))]
    ws_bytes = lx.lx_eri3_workspace_bytes(0, 0, 0, args.nx, args.npair, 9)
    wss = [torch.empty(ws_bytes, dtype=torch.uint8, device=dev) for _ in classes]
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    ints_per_step = sum(nint_set(c) for c in classes) * nsets
    probe = lx.lx_fp64_probe(20000)

    def launch(i, stream=None):
        c = classes[i]
        da, dp, dx, dpr = devs[c]
        lx.lx_eri3_batch(c[0], c[1], c[2], da, dp, dx, dpr, out=outs[i], workspace=wss[i], kmax=9, stream=stream)

    def serial_step(evs):
        """One pass on the current stream with an event pair per class (per-class times for the roofline)."""
        for i in range(len(classes)):
            evs[i][0].record()
            launch(i)
            evs[i][1].record()

    # The timed step: the independent classes are spread over `--streams` CUDA streams (longest first, each to the least
    # loaded stream by the cost model), so that the latency-bound small classes run in the shadow of the large ones.
    main = torch.cuda.current_stream()
    side = [torch.cuda.Stream(device=dev) for _ in range(max(args.streams, 1) - 1)]
    cost = [costmodel.flops_per_set(*c, 9) + 8.0 * nint_set(c) + 2000.0 for c in classes]
    load = [0.0] * (1 + len(side))
    plan = []
    for i in sorted(range(len(classes)), key=lambda i: -cost[i]):
        k = int(np.argmin(load))
        load[k] += cost[i]
        plan.append((i, k))

    def one_step():
        if not side:
            for i, _ in plan:
                launch(i)
            return
        fork = torch.cuda.Event()
        fork.record(main)
        for st in side:
            st.wait_event(fork)
        for i, k in plan:
            if k == 0:
                launch(i, main)
            else:
                with torch.cuda.stream(side[k - 1]):
                    launch(i, side[k - 1])
        for st in side:
            join = torch.cuda.Event()
            join.record(st)
            main.wait_event(join)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = lx.lx_launch_count()
    step_ms = []
    for _ in range(args.steps):
        flush.fill_(1)                      # L2 flush between timed iterations (outside the timed interval)
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        s0.record()
        one_step()
        s1.record()
        barrier()
        step_ms.append(s0.elapsed_time(s1))
    launches = lx.lx_launch_count() - launches0
    clocks = sampler.stop()
    # per-class kernel times (roofline of the dominant kernel): three serial passes outside the timed region
    class_ms = np.zeros(len(classes))
    for _ in range(3):
        flush.fill_(1)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in classes]
        barrier()
        serial_step(evs)
        barrier()
        class_ms += np.array([a.elapsed_time(b) for a, b in evs]) / 3
    serial_ms = float(class_ms.sum())
    t_total = torch.tensor([sum(step_ms) * 1e-3], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t_total, op=dist.ReduceOp.MAX)
    t_total = float(t_total.item())
    value = world * ints_per_step * args.steps / t_total

    # ---- end to end: host buffers through the C ABI, H2D of inputs and D2H of the result inside the timed region ----
    e2e = None
    if not args.no_e2e:
        pin = torch.empty(max_int, dtype=torch.float64).pin_memory()
        pin_np = pin.numpy()
        h2d = sum(h[0].nbytes() + h[1].nbytes() + h[2].nbytes + h[3].nbytes for h in host.values())
        d2h = ints_per_step * 8

        def e2e_step():
            for c in classes:
                ha, hp, xi, pi = host[c]
                n = nint_set(c) * nsets
                lx.lx_eri3_batch_host(c[0], c[1], c[2], ha, hp, xi, pi,
                                      out=pin_np[:n].reshape(args.npair, args.nx, ncart(c[0]), ncart(c[1]), ncart(c[2])))
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        nrep = max(1, min(args.steps, 3))
        for _ in range(nrep):
            e2e_step()
        barrier()
        te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": world * ints_per_step * nrep / float(te.item()), "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": nrep}

    if rank == 0:
        # ---- roofline of the dominant kernel (the class with the largest share of the step) -----------------------
        i_top = int(np.argmax(class_ms))
        c_top = classes[i_top]
        canon = (c_top[0], max(c_top[1:]), min(c_top[1:]))
        # algorithmic flops per shell-set: SURVEY.md section 8(d)'s per-unit figure where it lists the class (the primary count,
        # as the round-1 review asked), the component-level DAG count of costmodel.py beside it (it lowers along the axis with
        # the smallest positive power: fewer four-term nodes); ncu's executed count is in
        # profiles/r02_flops_per_class.md
        fl_model = costmodel.flops_per_set(*c_top, 9)
        fl_survey = SURVEY_FLOPS_PER_SET.get(canon)
        fl_set = fl_survey if fl_survey else fl_model
        t_top = class_ms[i_top] * 1e-3
        achieved = fl_set * nsets / t_top / 1e12
        roofline = {"bound": "alu", "kernel": f"{lx.lx_kernel_family_k(*canon, 9)}_kernel<{canon[0]},{canon[1]},{canon[2]},0> class ({c_top[0]}|{c_top[1]}{c_top[2]})",
                    "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_NOMINAL_TFLOPS,
                    "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(canon, (None, None))[0],
                    "traffic_source": NCU_DRAM_BYTES_PER_LAUNCH.get(canon, (None, "no ncu capture of this class under profiles/"))[1],
                    "peak_kind": "nominal FP64 DFMA pipe (148 SM x 64 FMA/clk x 1.965 GHz), DESIGN.md",
                    "peak_measured_dfma_probe": probe, "flops_per_set": fl_set,
                    "flops_source": "SURVEY.md section 8(d)" if fl_survey else "costmodel.py (class not in SURVEY.md section 8(d)'s table)",
                    "flops_per_set_costmodel": fl_model,
                    "frac_with_costmodel_flops": fl_model * nsets / t_top / 1e12 / FP64_NOMINAL_TFLOPS,
                    "kernel_ms": class_ms[i_top],
                    "share_of_step": float(class_ms[i_top] / class_ms.sum()),
                    "hbm_write_gbs": nint_set(c_top) * 8 * nsets / t_top / 1e9}
        cpu = None
        if world == 1 and not args.no_cpu:
            # bounded sample: calibrate on 16 pairs per class, then size the sample for ~15 s of CPU work
            _, t_cal, _ = oracle_sample(classes, 16, 256, seed=2)
            npair_s, nx_s = int(min(args.npair, max(16, 16 * 15.0 / max(t_cal, 1e-3)))), min(256, args.nx)
            n, t, cores = oracle_sample(classes, npair_s, nx_s, seed=2)
            cpu = {"value": n / t, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"first {npair_s} pairs x {nx_s} aux shells of each of the 45 classes ({n} integrals, {t:.1f} s)"}
        # ---- side measurements: BASELINE.json metric "DF-J time" on configs[3] and configs[4] at their stated (Schwarz-
        # screened) configuration, configs[2] per class and configs[0] per call; none of them is part of `value`
        df = df5 = c1 = c3 = None
        if world == 1 and not args.no_df and not args.classes:
            df = bench_df(lx, dev, costmodel, gen.config4(), "configs[3]: 64-atom cluster, 960 AO x 6 784 Cartesian DFAO", 3, unscreened=True)
            df5 = bench_df(lx, dev, costmodel, gen.config5(), "configs[4]: 256-atom cluster, 8 960 AO x 54 016 Cartesian DFAO, integral-direct", 1)
        if world == 1 and not args.no_side and not args.classes:
            c1 = bench_config1(lx, dev)
            c3 = bench_config3(lx, dev, costmodel)
        # ---- side measurement: the same sweep with SOLID-HARMONIC aux functions through
        # lx_eri3_batch_pure (fused for Lx >= 2, Cartesian + transform for Lx <= 1); serial on one stream; not part of `value`
        pure = None
        if world == 1 and not args.no_df and not args.classes:
            wsp = torch.empty(max(int(lx._lib.lx_eri3_pure_workspace_bytes(c[0], c[1], c[2], args.nx, args.npair, 9)) for c in classes),
                              dtype=torch.uint8, device=dev)
            n_pure = sum((2 * c[0] + 1) * ncart(c[1]) * ncart(c[2]) for c in classes) * nsets

            def pure_step():
                for i, c in enumerate(classes):
                    da, dp, dx, dpr = devs[c]
                    n = (2 * c[0] + 1) * ncart(c[1]) * ncart(c[2]) * nsets
                    lx.lx_eri3_batch_pure(c[0], c[1], c[2], da, dp, dx, dpr, out=outs[i][:n], workspace=wsp, kmax=9)
            pure_step()
            torch.cuda.synchronize()
            best = 1e30
            for _ in range(3):
                flush.fill_(1)
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                a0.record()
                pure_step()
                a1.record()
                torch.cuda.synchronize()
                best = min(best, a0.elapsed_time(a1))
            pure = {"workload": "configs[1] with solid-harmonic aux functions (2Lx+1 components), one stream",
                    "ms_per_step": best, "integrals_per_step": n_pure, "integrals_per_s": n_pure / (best * 1e-3),
                    "shell_sets_per_s": nsets * len(classes) / (best * 1e-3)}
        per_class = {f"({c[0]}|{c[1]}{c[2]})": round(float(nint_set(c) * nsets / (m * 1e-3)), 1) for c, m in zip(classes, class_ms)}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * t_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOAD if (args.npair, args.nx, args.classes) == (1024, 256, "") else f"reduced config 2: {args.npair} pairs x {args.nx} aux, classes {args.classes or 'all'}",
                           "shell_sets_per_step": nsets * len(classes) * world, "integrals_per_step": ints_per_step * world,
                           "l2": "flushed between timed steps (256 MiB fill, outside the timed interval); each step also writes "
                                 f"{ints_per_step * 8 / 1e9:.1f} GB of output",
                           "parallelism": f"{world} x independent batch (no collective)",
                           "streams": f"{1 + len(side)} CUDA streams per step (independent classes overlap); the same classes launched "
                                      f"back to back on one stream take {serial_ms:.2f} ms (sum of per-class event times)"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
                "shell_sets_per_s": value / ints_per_step * nsets * len(classes), "df_config4": df, "df_config5": df5,
                "config1": c1, "config3": c3, "pure_sweep": pure,
                "integrals_per_s_per_class": per_class}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
