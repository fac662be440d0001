#!/usr/bin/env python
"""bench.py -- throughput of the semi-coherent statistic hot path on B200 (BASELINE.json metric).

One "step" = one swarm iteration of the whole hot path: sc_eval_stat for the whole
population (node evaluation, dense waveform x response x segment reduction, stitch) followed by sc_pso_step,
device-resident, no host round trip.  Workload at N = 1: BASELINE.json configs[2] ("c3": T = 4 yr, band
0.017-0.030 Hz, 1 640 996 bins, 10^4 particles, N_seg = 5000, PSO 0.7/1.5/1.5) -- the configuration the metric's
target is quoted on.  For N > 1 every rank searches its own independent tile (own noise realisation and population,
replicated nothing, no data-path collective): weak scaling.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample.
Inputs are synthetic (sc_synth); injections in the GPU arm come from the library's own
sc_gen_template, never from the oracle.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
import sc_synth as sy  # noqa: E402

METRIC = "particle_x_freq_bin_evals_per_s"
UNIT = "particle-bin/s"
C_DP = 24          # FP64 instructions per (particle, bin) of the fixed op model, SURVEY.md 8(d)
NOMINAL_DFMA = 148 * 64 * 1.965e9   # 148 SMs x 64 FP64 lanes x max SM clock (B200_PROFILING.md unit counts / clocks)
# The kernel's own mix: FP32-pipe lane slots per evaluated (particle, bin) in the k_dense2 loop,
# 26 packed FFMA2/FMUL2/FADD2 (2 slots each) + 3 scalar per bin PAIR; peak = 148 SMs x 128 FP32 lanes x max SM clock.
# The QUAD flavour (quadratic amplitudes over runs, sc_get_launch_info) executes 22 packed instead of 26.
FP32_SLOTS_PER_BIN = (26 * 2 + 3) / 2.0
FP32_SLOTS_PER_BIN_QUAD = (22 * 2 + 3) / 2.0
NOMINAL_FP32_SLOTS = 148 * 128 * 1.965e9
NOMINAL_FP32_TFLOPS = 2.0 * NOMINAL_FP32_SLOTS / 1e12   # 74.5 TFLOP/s: unit counts x clock of B200_PROFILING.md (no measured FP32 peak)
DENSE_PROFILE = os.path.join(ROOT, "profiles", "r02_k_dense2_full.md")   # ncu --set full of the c3 launch (static figure, see roofline.traffic_source)


def dram_traffic_from_profile():
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_dense2 launch, from the committed ncu --set full summary."""
    import re
    try:
        txt = open(DENSE_PROFILE).read()
    except OSError:
        return None
    tot, mult = 0.0, {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(r"\|\s*" + re.escape(name) + r"\s*\|\s*(\w+)\s*\|\s*([0-9.eE+-]+)\s*\|", txt)
        if not m or m.group(1) not in mult:
            return None
        tot += float(m.group(2)) * mult[m.group(1)]
    return tot


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--particles", type=int, default=None, help="override the population size (debug)")
    ap.add_argument("--adaptive-nseg", type=int, default=0, metavar="N",
                    help="time the step with per-particle equal-SNR^2 segments (sc_eval_stat_adaptive, PAPER.md:120) and N "
                         "segments instead of the config's shared edges")
    ap.add_argument("--search", type=float, default=0.0, metavar="RHO",
                    help="extras: also run ONE complete hierarchical search (Fig. 2; sc_search_run) at the paper's scale on "
                         "this config's tile -- 6 swarms x 10^4 particles (PAPER.md:167, 506), ladder N = 100/50/10/1, Table "
                         "IV hyper-parameters, per-particle segments -- with the injection rescaled to SNR RHO; takes minutes")
    ap.add_argument("--fap", type=int, default=0, metavar="SEEDS",
                    help="extras: run the c4 workload (BASELINE configs[3]: noise only, 10^4 particles x 200 PSO iterations at "
                         "N = 50000/5000/500) over SEEDS noise realisations and report the maximum statistic per seed and level")
    ap.add_argument("--search-channels", type=int, default=2, choices=[2, 3],
                    help="with --search: 3 = the search runs on an (A, E, T) handle -- with the per-particle segments of the ladder "
                         "this is the paper's own configuration (PAPER.md:36, 59, 120); the injection is made in all three channels")
    ap.add_argument("--search-ranking", action="store_true",
                    help="with --search: sc_search_config.ranking_precision = 1 (all rungs on the FP32 path, bests re-evaluated in FP64)")
    ap.add_argument("--no-extras", action="store_true", help="skip the extra (untimed-region) measurements")
    ap.add_argument("--dist-selftest", action="store_true",
                    help="CPU-only check of the multi-rank launch and reductions (gloo); used by tests/test_multi_rank.py")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-window-hint", action="store_true",
                    help="do not state the measured window fraction (SC_OPT_WINDOW_FRACTION_PPM): node spacing for N' = 8")
    ap.add_argument("--opt", action="append", default=[], metavar="ID=VALUE",
                    help="extra sc_set_option(ID, VALUE) calls on the handle (experiments)")
    return ap.parse_args()


def workload_name(cid, spec, cfg, P, N):
    return (f"c{cid}: T={spec['T_obs_yr']}yr band {spec['band'][0]}-{spec['band'][1]}Hz n_bins={cfg['n_bins']} "
            f"P={P} N_seg={N}")


def pso_params(spec, N):
    if "pso" in spec:
        return spec["pso"]
    key = min(sy.TABLE_IV, key=lambda k: abs(np.log(k) - np.log(max(N, 1))))
    return sy.TABLE_IV[key]


# ---------------------------------------------------------------------------------------------- reference arm
def oracle_sample_run(inp, N, n_particles, steps, warmup):
    """Times the CPU oracle, as it stands, on the first n_particles of the population: statistic + PSO step."""
    from oracle import sc_oracle as orc
    cfg = orc.make_config(inp["cfg"])
    e = inp["edges"][N]
    pos = inp["particles"][:n_particles].copy()
    vel = inp["velocities"][:n_particles].copy()
    pbp, pbv = pos.copy(), np.full(n_particles, -np.inf)
    gp, gv = np.zeros((1, 8)), np.zeros(1)
    hp = pso_params(inp["spec"], N)
    dA, dE = inp["noise_A"], inp["noise_E"]          # noise-only stream: the oracle's cost does not depend on the data
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        st = orc.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], pos, e)
        orc.pso_step(pos, vel, pbp, pbv, st, gp, gv, inp["lo"], inp["hi"], np.array(hp["eps"], dtype=np.float64),
                     hp["omega"], hp["phi_p"], hp["phi_g"], inp["pso_seed"], it, 1)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    return float(np.mean(times)), orc.num_threads()


def run_reference(args, rank, world):
    if rank != 0:
        return
    cid = args.config
    spec = sy.CONFIGS[cid]
    inp = sy.config_inputs(cid, P=64)
    N = spec["n_segs"][0]
    from oracle import sc_oracle as orc
    cores = orc.num_threads()
    n_p = max(1, min(64, cores))
    steps, warmup = max(1, min(args.steps, 5)), min(args.warmup, 1)
    sec, cores = oracle_sample_run(inp, N, n_p, steps, warmup)
    nb = inp["cfg"]["n_bins"]
    val = n_p * nb / sec
    sample = f"{n_p} particles x all {nb} bins per step ({steps} timed steps, {warmup} warm-up), noise-only stream"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cid, spec, inp["cfg"], n_p, N)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- GPU arm
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 8:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(np.max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def run_search(sc, torch, dev, inp, cid, rho, S_A, S_E, nA, nE, max_iters=1000, ranking=0, channels=2):
    """One complete search of one tile (Fig. 2): init from the prior, the ladder with Table IV
    hyper-parameters, convergence rule of App. B, k-means regrouping between rungs, threshold Upsilon_1 >= 100.
    c5 (BASELINE configs[4]): its own 4 swarms x 10^4 particles, ladder 50000/5000/500/50/1 on shared equal-width edges, both
    injections at their configured SNRs.  Any other config: the paper's set-up -- 6 swarms x 10^4 particles (PAPER.md:167,
    506), ladder 100/50/10/1 with per-particle equal-SNR^2 segments, the injection rescaled to SNR rho."""
    spec = sy.CONFIGS[cid]
    if cid == 5:
        n_swarms, per_swarm, ladder, adaptive = spec["n_swarms"], spec["P"] // spec["n_swarms"], list(spec["n_segs"]), False
    else:
        n_swarms, per_swarm, ladder, adaptive = 6, 10000, [100, 50, 10, 1], True
    big = sy.config_inputs(cid, P=n_swarms * per_swarm)
    cfg, nb = inp["cfg"], inp["cfg"]["n_bins"]
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    ri = lambda z: torch.view_as_real(z).contiguous()
    if channels == 3:
        cfg = dict(cfg, n_channels=3)
        S_T = t(sy.psd_T(sy.freqs(cfg)))
        nT = t(sy.draw_noise(sy.MASTER_SEED + 7 + 100 * cid, sy.psd_T(sy.freqs(cfg)), inp["df"]))
        H0 = sc.Handle(cfg, ri(nA), ri(nE), S_A, S_E, dT=ri(nT), S_T=S_T)
    else:
        H0 = sc.Handle(cfg, ri(nA), ri(nE), S_A, S_E)
    dA, dE, snrs = nA.clone(), nE.clone(), []
    dT = nT.clone() if channels == 3 else None
    for inj in inp["injections"]:
        if channels == 3:
            hA, hE, hT = H0.gen_template3(t(inj["theta"][None, :]))
        else:
            hA, hE = H0.gen_template(t(inj["theta"][None, :]))
        rho2 = 4.0 * inp["df"] * ((hA[0].abs() ** 2 / S_A).sum() + (hE[0].abs() ** 2 / S_E).sum())
        if channels == 3:
            rho2 = rho2 + 4.0 * inp["df"] * (hT[0].abs() ** 2 / S_T).sum()
        snrs.append(float(inj["rho"] if cid == 5 else rho))
        dA += snrs[-1] / torch.sqrt(rho2) * hA[0]
        dE += snrs[-1] / torch.sqrt(rho2) * hE[0]
        if channels == 3:
            dT += snrs[-1] / torch.sqrt(rho2) * hT[0]
    H0.close()
    H = sc.Handle(cfg, ri(dA), ri(dE), S_A, S_E, dT=ri(dT), S_T=S_T) if channels == 3 else sc.Handle(cfg, ri(dA), ri(dE), S_A, S_E)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(big["hi"][2])))
    hyper = [dict(sy.TABLE_IV[min(sy.TABLE_IV, key=lambda k: abs(np.log(k) - np.log(N)))]) for N in ladder]
    scfg = sc.ScSearchConfig.make(ladder, hyper, adaptive_edges=adaptive, max_iters_per_rung=max_iters, seed=2408, threshold=100.0,
                                  ranking_precision=ranking)
    pos, vel = t(big["particles"]), t(big["velocities"])
    label = torch.from_numpy(np.repeat(np.arange(n_swarms, dtype=np.int32), per_swarm)).to(dev)
    ths = np.stack([inj["theta"] for inj in inp["injections"]])
    ups1_inj = H.eval_stat(t(ths), sy.edges(nb, ladder[-1]).astype(np.int32)).cpu().numpy()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = H.search_run(scfg, pos, vel, label, n_swarms, t(big["lo"]), t(big["hi"]))
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    H.close()
    b = int(np.argmax(res["best_val"]))
    near = int(np.argmin(np.abs(ths[:, 0] - res["best_pos"][b, 0])))          # the injection the best swarm sits on
    iters = [int(x) for x in res["iters_per_rung"]]
    return {"what": f"sc_search_run on the c{cid} tile ({'A, E, T' if channels == 3 else 'A, E'}): {n_swarms} swarms x {per_swarm} particles, ladder {ladder}, "
                    + ("per-particle equal-SNR^2 segments" if adaptive else "shared equal-width segments")
                    + f", Table IV hyper-parameters, injection SNRs {snrs}, ranking_precision = {ranking}",
            "wall_s": wall, "iters_per_rung": iters, "particle_bin_evals": float(sum(iters)) * n_swarms * per_swarm * nb,
            "best_val_per_swarm": [float(v) if np.isfinite(v) else None for v in res["best_val"]],
            "best_upsilon": float(res["best_val"][b]), "upsilon_at_injections": [float(v) for v in ups1_inj],
            "swarms_above_threshold": int(np.sum(res["passed"])),
            "best_minus_injected": {"Mc_msun": float(res["best_pos"][b, 0] - ths[near, 0]),
                                    "eta": float(res["best_pos"][b, 1] - ths[near, 1]),
                                    "tc_s": float(res["best_pos"][b, 2] - ths[near, 2])},
            "paper_context": "PAPER.md:365-367: ~1-2 days per search on 1 A100 + 10 CPU processes (other hardware, the authors' "
                             "waveform/response code): context, not a like-for-like baseline"}


def run_fap(sc, torch, dev, cid, n_seeds):
    """The workload of BASELINE configs[3] (c4): noise-only data, 10^4 particles x 200 PSO iterations at every level, repeated
    over noise seeds -> the background of the maximum statistic (the shape of PAPER.md:323, 333-349 at reduced size)."""
    spec = sy.CONFIGS[cid]
    hp, iters, out = spec["pso"], spec["pso"]["iters"], {N: [] for N in spec["n_segs"]}
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    ms, n_eval, frac = 0.0, 0, None
    for r in range(n_seeds):
        inp = sy.config_inputs(cid, replica=r)
        P, nb = inp["particles"].shape[0], inp["cfg"]["n_bins"]
        H = sc.Handle(inp["cfg"], torch.view_as_real(t(inp["noise_A"])).contiguous(),
                      torch.view_as_real(t(inp["noise_E"])).contiguous(), t(inp["S_A"]), t(inp["S_E"]))
        H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
        lo, hi, eps = t(inp["lo"]), t(inp["hi"]), t(np.array(hp["eps"], dtype=np.float64))
        stat = torch.empty(P, dtype=torch.float64, device=dev)
        for N in spec["n_segs"]:
            e = inp["edges"][N].astype(np.int32)
            st = dict(pos=t(inp["particles"]), vel=t(inp["velocities"]), pbest_pos=t(inp["particles"]),
                      pbest_val=torch.full((P,), -np.inf, dtype=torch.float64, device=dev),
                      gbest_pos=torch.zeros((1, 8), dtype=torch.float64, device=dev),
                      gbest_val=torch.zeros(1, dtype=torch.float64, device=dev))
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for it in range(iters):
                H.eval_stat(st["pos"], e, out=stat)
                H.pso_step(st, stat, lo, hi, eps, hp["omega"], hp["phi_p"], hp["phi_g"], inp["pso_seed"], it, 1)
            b.record()
            torch.cuda.synchronize()
            ms += a.elapsed_time(b); n_eval += iters
            out[N].append(float(st["gbest_val"].item()))
            if frac is None:
                frac = H.counters()[0] / (float(P) * nb)
        H.close()
    return {"what": f"c{cid}: noise only, {spec['P']} particles x {iters} PSO iterations per level, {n_seeds} noise seeds; "
                    "max statistic found per seed and level",
            "max_upsilon_per_seed": {str(N): v for N, v in out.items()},
            "noise_mean_2N_eff": {str(N): 2.0 * N * frac for N in out}, "noise_sd_2sqrtN_eff": {str(N): 2.0 * (N * frac) ** 0.5 for N in out},
            "ms_per_iteration": ms / max(n_eval, 1), "iterations": n_eval}


def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    import paper_2408_13170_b200 as sc

    if not torch.cuda.is_available() or local_rank >= torch.cuda.device_count():
        sys.exit(f"bench.py: rank {rank} needs CUDA device {local_rank}; {torch.cuda.device_count() if torch.cuda.is_available() else 0} "
                 f"visible (--gpus {args.gpus} needs that many GPUs on this node; there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cid = args.config
    spec = sy.CONFIGS[cid]
    inp = sy.config_inputs(cid, P=args.particles, replica=rank)
    cfg = inp["cfg"]
    N = spec["n_segs"][0]
    e = inp["edges"][N].astype(np.int32)
    nb = cfg["n_bins"]
    P = inp["particles"].shape[0]
    n_swarms = spec["n_swarms"]
    hp = pso_params(spec, N)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    S_A, S_E = t(inp["S_A"]), t(inp["S_E"])
    nA, nE = t(inp["noise_A"]), t(inp["noise_E"])

    # data = noise + kappa * h(theta_inj), the injection generated by the library itself (sc_gen_template)
    H0 = sc.Handle(cfg, torch.view_as_real(nA).contiguous(), torch.view_as_real(nE).contiguous(), S_A, S_E)
    dA, dE = nA.clone(), nE.clone()
    for inj in inp["injections"]:
        hA, hE = H0.gen_template(t(inj["theta"][None, :]))
        rho2 = 4.0 * inp["df"] * ((hA[0].abs() ** 2 / S_A).sum() + (hE[0].abs() ** 2 / S_E).sum())
        kappa = inj["rho"] / torch.sqrt(rho2)
        dA += kappa * hA[0]
        dE += kappa * hE[0]
    H0.close()
    H = sc.Handle(cfg, torch.view_as_real(dA).contiguous(), torch.view_as_real(dE).contiguous(), S_A, S_E)
    # the caller knows its tile: t_c upper bound of the prior box sets the coarse node spacing (SC_OPT_TC_MAX_S)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    H.set_option(sc.SC_OPT_PROFILE, 1)
    for kv in args.opt:
        k_, v_ = kv.split("=")
        H.set_option(int(k_), int(v_))

    lo, hi, eps = t(inp["lo"]), t(inp["hi"]), t(np.array(hp["eps"], dtype=np.float64))
    state = dict(pos=t(inp["particles"]), vel=t(inp["velocities"]), pbest_pos=t(inp["particles"]),
                 pbest_val=torch.full((P,), -np.inf, dtype=torch.float64, device=dev),
                 gbest_pos=torch.zeros((n_swarms, 8), dtype=torch.float64, device=dev),
                 gbest_val=torch.zeros(n_swarms, dtype=torch.float64, device=dev))
    stat = torch.empty(P, dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    ad_N = args.adaptive_nseg
    if ad_N:
        N = ad_N

    def step(it):
        if ad_N:
            sc.sc_eval_stat_adaptive(H.h, state["pos"], P, ad_N, stat)
        else:
            H.eval_stat(state["pos"], e, out=stat)
        H.pso_step(state, stat, lo, hi, eps, hp["omega"], hp["phi_p"], hp["phi_g"], inp["pso_seed"], it, n_swarms)

    # ... and how much of the band its particles' time windows cover, measured with one evaluation before anything is timed
    # (what sc_search_run does for itself): the node spacing is then set for N' = n_seg x fraction segments per particle
    win_frac = None
    if not ad_N and not args.no_window_hint:
        H.eval_stat(state["pos"], e, out=stat)
        win_frac = H.counters()[0] / (float(P) * nb)
        H.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, int(round(win_frac * 1e6)))

    for it in range(args.warmup):
        step(it)
    torch.cuda.synchronize()
    H.timing()                               # reset the per-class accumulators
    _, launches0 = H.counters()
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ
                           else int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    eval_bins = 0
    barrier()
    t_wall0 = time.perf_counter()
    for i, (a, b) in enumerate(evs):
        flush.fill_(i & 0xFF)                # L2 flush between timed iterations (outside the events)
        a.record()
        step(args.warmup + i)
        b.record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    ms_steps = [a.elapsed_time(b) for a, b in evs]
    ms_total = float(np.sum(ms_steps))
    timing = H.timing()
    eval_bins, launches1 = H.counters()      # evaluated bins of the LAST eval (the swarm moves; representative)
    gpu_launches = launches1 - launches0

    # ---- extras (outside the timed region): the paper's own segment definition at the first rung of its ladder
    extras = {}
    if not args.no_extras and not ad_N and rank == 0:
        H.timing()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(4):
            if i == 1:
                torch.cuda.synchronize(); H.timing(); a.record()
            sc.sc_eval_stat_adaptive(H.h, state["pos"], P, 100, stat)
        b.record()
        torch.cuda.synchronize()
        tma = H.timing()
        extras["adaptive_segments_N100"] = {
            "what": "sc_eval_stat_adaptive (per-particle equal-SNR^2 segments, PAPER.md:120), N = 100, same population",
            "ms_per_eval": a.elapsed_time(b) / 3, "particle_bin_per_s": float(P) * nb / (a.elapsed_time(b) / 3 * 1e-3),
            "kernel_ms_per_eval": {k: v[0] / 3 for k, v in tma.items() if v[1]}}

    # ---- extras: the all-FP64 kernel (every rung with N < 8: the paper's final N = 1 rung), the
    # tensor-core flavour of the FP32-amplitude kernel, and the three-channel statistic (A, E, T)
    def timed_evals(fn, reps=3):
        fn(); torch.cuda.synchronize(); H.timing()
        a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a_.record()
        for _ in range(reps):
            fn()
        b_.record(); torch.cuda.synchronize()
        return a_.elapsed_time(b_) / reps, {k: v[0] / reps for k, v in H.timing().items() if v[1]}

    if not args.no_extras and not ad_N and rank == 0:
        e1 = np.array([0, nb], dtype=np.int32)
        ms1, k1 = timed_evals(lambda: H.eval_stat(state["pos"], e1, out=stat))
        ev1 = H.counters()[0]
        extras["coherent_N1"] = {"what": "sc_eval_stat at N = 1 (all-FP64 path, k_dense<false>), same population",
                                 "ms_per_eval": ms1, "kernel_ms_per_eval": k1, "evaluated_particle_bin_per_s": ev1 / (ms1 * 1e-3),
                                 "fp64_model_frac": (2.0 * C_DP * ev1 / (k1.get("dense", ms1) * 1e-3) / (2.0 * NOMINAL_DFMA))}
        try:
            H.set_option(sc.SC_OPT_TENSOR_CORES, 1)
            mst, kt = timed_evals(lambda: H.eval_stat(state["pos"], e, out=stat))
            extras["tensor_core_flavour"] = {
                "what": "SC_OPT_TENSOR_CORES = 1: k_dense2_tc (amplitude x data factor as a split-TF32 contraction on tcgen05, "
                        "TMEM accumulators), same evaluation; not the default (slower than k_dense2, DESIGN.md 6)",
                "ms_per_eval": mst, "kernel_ms_per_eval": kt}
        except sc.SCError as ex:
            extras["tensor_core_flavour"] = {"skipped": str(ex)[:200]}
        H.set_option(sc.SC_OPT_TENSOR_CORES, 0)
        try:
            cfg3 = dict(cfg, n_channels=3)
            S_T = t(sy.psd_T(sy.freqs(cfg3)))
            nT = t(sy.draw_noise(sy.MASTER_SEED + 7 + 100 * cid if hasattr(sy, "MASTER_SEED") else 240813177 + 100 * cid,
                                 sy.psd_T(sy.freqs(cfg3)), inp["df"]))
            H3 = sc.Handle(cfg3, torch.view_as_real(dA).contiguous(), torch.view_as_real(dE).contiguous(), S_A, S_E,
                           dT=torch.view_as_real(nT).contiguous(), S_T=S_T)
            H3.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
            if win_frac is not None:
                H3.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, int(round(win_frac * 1e6)))
            H3.eval_stat(state["pos"], e, out=stat); torch.cuda.synchronize()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record()
            for _ in range(2):
                H3.eval_stat(state["pos"], e, out=stat)
            b_.record(); torch.cuda.synchronize()
            extras["three_channels"] = {"what": "sc_eval_stat on an (A, E, T) handle (T noise only), same population and edges: "
                                                "one pass through the fused kernel k_dense3 (SC_OPT_FUSED_AET = 1)", "ms_per_eval": a_.elapsed_time(b_) / 2}
            sc.sc_eval_stat_adaptive(H3.h, state["pos"], P, 100, stat); torch.cuda.synchronize()
            a_.record(); sc.sc_eval_stat_adaptive(H3.h, state["pos"], P, 100, stat); b_.record(); torch.cuda.synchronize()
            extras["three_channels"]["ms_per_eval_adaptive_N100"] = a_.elapsed_time(b_)   # the paper's own configuration
            H3.set_option(sc.SC_OPT_FUSED_AET, 0)
            H3.eval_stat(state["pos"], e, out=stat); torch.cuda.synchronize()
            a_.record(); H3.eval_stat(state["pos"], e, out=stat); b_.record(); torch.cuda.synchronize()
            extras["three_channels"]["ms_per_eval_two_passes"] = a_.elapsed_time(b_)
            H3.close()
            del H3, nT, S_T
        except (RuntimeError, sc.SCError, KeyError, AttributeError) as ex:
            extras["three_channels"] = {"skipped": str(ex)[:200]}

    # ---- extras: the second workload (Fig. 3): many data streams x one template, HBM-bound
    if not args.no_extras and not ad_N and rank == 0:
        D = 256
        try:
            Ws = torch.randn((D, nb, 4), dtype=torch.float32, device=dev)       # whitened noise-only streams, 16 B per bin
            th = state["gbest_pos"][0].contiguous()
            e100 = sy.edges(nb, 100).astype(np.int32)
            outs = torch.empty(D, dtype=torch.float64, device=dev)
            H.eval_stat_streams(th, Ws, e100, out=outs)
            torch.cuda.synchronize(); H.timing()
            reps = 5
            for _ in range(reps):
                flush.fill_(1)
                H.eval_stat_streams(th, Ws, e100, out=outs)
            torch.cuda.synchronize()
            tms = H.timing()
            z_ms = tms["dense"][0] / reps
            peaks = {}
            try:
                peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            except (OSError, ValueError):
                pass
            peak = float(peaks.get("hbm_gbs", 6650.0))
            gbs = D * nb * 16.0 / (z_ms * 1e-3) / 1e9
            extras["streams_x_one_template"] = {
                "what": f"sc_eval_stat_streams: {D} FP32 streams x {nb} bins (c{cid} grid), N = 100, one template",
                "kernel": "k_streams_z<float4,float>", "kernel_ms_per_launch": z_ms,
                "ms_per_eval_all_kernels": sum(v[0] for v in tms.values()) / reps,
                "stream_bin_per_s": D * nb / (z_ms * 1e-3),
                "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                             "traffic": None, "algorithmic_bytes_per_stream_bin": 16,
                             "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "fallback 6650 GB/s (of fallback)"}}
            del Ws
        except (RuntimeError, sc.SCError) as ex:                                # e.g. not enough memory for the streams
            extras["streams_x_one_template"] = {"skipped": str(ex)[:200]}

    # ---- extras (opt-in): one complete hierarchical search at the paper's scale (context for PAPER.md:365-367)
    if args.search > 0 and rank == 0 and inp["injections"]:
        extras["hierarchical_search"] = run_search(sc, torch, dev, inp, cid, args.search, S_A, S_E, nA, nE, ranking=int(args.search_ranking),
                                                  channels=args.search_channels)
    if args.fap > 0 and rank == 0:
        extras["false_alarm_background"] = run_fap(sc, torch, dev, 4, args.fap)

    # ---- e2e: the same step through the HOST-buffer entry point, copies inside the timed region
    e2e = None
    if not args.no_e2e and not ad_N:
        k2 = max(1, min(args.steps, 5))
        pos_h = torch.empty((P, 8), dtype=torch.float64).pin_memory()
        stat_h = torch.empty(P, dtype=torch.float64).pin_memory()
        pos_h.copy_(state["pos"])
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        a.record()
        for i in range(k2):
            H.eval_stat_host(pos_h.numpy(), e, out=stat_h.numpy())               # H2D params, D2H Upsilon (inside the C call)
            stat.copy_(stat_h, non_blocking=True)                                 # H2D Upsilon for the device-side PSO
            H.pso_step(state, stat, lo, hi, eps, hp["omega"], hp["phi_p"], hp["phi_g"], inp["pso_seed"],
                       args.warmup + args.steps + i, n_swarms)
            pos_h.copy_(state["pos"], non_blocking=True)                          # D2H new positions
            torch.cuda.synchronize()
        b.record()
        barrier()
        ms_e2e = a.elapsed_time(b) / k2
        e2e = dict(ms=ms_e2e, h2d=P * 64 + P * 8, d2h=P * 8 + P * 64)
        H.timing()

    # ---- reduce over ranks: max time, summed work
    # work = EVALUATED (particle, bin) pairs: bins inside the particle's time window and [e_0, e_N) (the count of the last
    # evaluation; the swarm moves a little from step to step).  The nominal P x n_bins rate is reported beside it.
    ms_max, units, units_nominal = ms_total, float(eval_bins) * args.steps, float(P) * nb * args.steps
    e2e_ms_max = e2e["ms"] if e2e else 0.0
    if world > 1:
        v = torch.tensor([ms_total, e2e_ms_max], dtype=torch.float64, device=dev)
        dist.all_reduce(v, op=dist.ReduceOp.MAX)
        ms_max, e2e_ms_max = v[0].item(), v[1].item()
        u = torch.tensor([units, units_nominal], dtype=torch.float64, device=dev)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
        units, units_nominal = u[0].item(), u[1].item()

    if rank == 0:
        value = units / (ms_max * 1e-3)
        ms_per_step = ms_max / args.steps
        dense_ms, dense_n = timing["dense"]
        dense_avg = dense_ms / max(dense_n, 1)
        try:
            dfma = sc.sc_measure_fp64_peak()
        except sc.SCError:
            dfma = None
        # roofline of the dominant kernel (k_dense), fixed FP64 op model of SURVEY.md 8(d): 24 FP64 instr = 48 flop per
        # EVALUATED (particle, bin); peak = measured DFMA rate x 2 flop
        # populations beyond the scratch cap run in several batches: one evaluation = dense_per_eval launches of k_dense
        dense_per_eval = max(1, int(round(dense_n / max(args.steps, 1))))
        eval_bins_launch = eval_bins / dense_per_eval
        ach = 2.0 * C_DP * eval_bins_launch / (dense_avg * 1e-3) / 1e12 if dense_avg > 0 else None
        peak = 2.0 * (dfma or NOMINAL_DFMA) / 1e12
        pbs = eval_bins_launch / (dense_avg * 1e-3) if dense_avg > 0 else None
        # Two fractions (both kept): (1) frac = frac_pipe_fma -- the pipe the kernel as built runs on: FP32 lane slots it
        # executes per evaluated bin (SASS of the pair loop: 26 packed x 2 + 3 scalar per bin pair; 22 packed in the QUAD flavour,
        # so a faster kernel can show a LOWER fraction: it does less work) x evaluated bins/s
        # against 148 SM x 128 lanes x max clock; ncu's sm__pipe_fma_cycles_active of the same launch is in profiles/.
        # (2) frac_model -- the contract's fixed op model (24 FP64 instructions per evaluated bin)
        # against the FP64 rate measured in this run; the kernel does NOT execute that FP64 work (3 DADD per bin), so
        # this one is a speed-up over the model, not a utilisation, and may exceed 1.
        lg_nodes, flavour = H.launch_info()
        quad = bool(flavour & sc.SC_FLAVOUR_QUAD) and not ad_N
        slots_per_bin = FP32_SLOTS_PER_BIN_QUAD if quad else FP32_SLOTS_PER_BIN
        slots = (pbs * slots_per_bin) if pbs else None
        is_c3_shared = (cid == 3 and not ad_N and not args.particles)
        roof = {"bound": "alu", "achieved": (2.0 * slots / 1e12) if slots else None, "peak": NOMINAL_FP32_TFLOPS, "unit": "TFLOP/s",
                "frac": (slots / NOMINAL_FP32_SLOTS) if slots else None,
                "frac_pipe_fma": (slots / NOMINAL_FP32_SLOTS) if slots else None,
                "frac_model": (ach / peak) if ach else None,
                "traffic": dram_traffic_from_profile() if is_c3_shared else None,
                "traffic_source": ("static: profiles/r02_k_dense2_full.md (ncu --set full of one k_dense2 launch of this c3 command), "
                                   "not measured in this run") if is_c3_shared else None,
                "kernel": "k_dense2_ad<2,MERGE>" if ad_N else ("k_dense2<false," + ("2" if flavour & sc.SC_FLAVOUR_MUFU else "0")
                                                                + (",MERGE" if flavour & sc.SC_FLAVOUR_MERGE else "") + (",QUAD" if quad else "") + ">"),
                "kernel_ms_per_launch": dense_avg, "node_stride_log2": lg_nodes, "flavour_bits": flavour,
                "peak_source": "FP32 pipe: 148 SM x 128 lanes x 1.965 GHz x 2 flop (unit counts and clocks of B200_PROFILING.md; "
                               "MEASURED_PEAKS.json has no FP32 figure)",
                "pipe_fma": {"fp32_lane_slots_per_evaluated_bin": slots_per_bin,
                             "packed_fp32_instructions_per_bin_pair": 22 if quad else 26, "lane_slots_per_s": slots,
                             "peak_lane_slots_per_s": NOMINAL_FP32_SLOTS},
                "model": {"what": f"{C_DP} FP64 instr (= {2 * C_DP} flop) per evaluated particle-bin, SURVEY.md 8(d)",
                          "achieved_tflops": ach, "peak_tflops": peak,
                          "peak_source": ("measured in this run by sc_measure_fp64_peak (DFMA/s x 2)" if dfma else
                                          "nominal 148 SM x 64 lanes x 1.965 GHz x 2"),
                          "peak_nominal_max_clock": 2.0 * NOMINAL_DFMA / 1e12,
                          "frac_vs_nominal_max_clock": (ach / (2.0 * NOMINAL_DFMA / 1e12)) if ach else None},
                "evaluated_particle_bins_per_launch": eval_bins_launch, "launches_per_evaluation": dense_per_eval,
                "evaluated_pb_per_s_dense_kernel": pbs}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64 phase + f32 amplitude/accumulate-flush-to-f64", "data": "synthetic",
                "config": {"workload": workload_name(cid, spec, cfg, P, N), "l2": "flushed between timed steps "
                           "(256 MiB write); per-step node tables + fragments (~1 GB) exceed L2 anyway",
                           "pso": {k: hp[k] for k in ("omega", "phi_p", "phi_g")}, "n_swarms": n_swarms,
                           "window_fraction_stated": win_frac,
                           "parallelism": f"independent tiles x{world}" if world > 1 else "1 GPU"},
                "value_counts": "evaluated (particle, bin) pairs (inside the time windows and [e_0, e_N))",
                "nominal_particle_bin_per_s": units_nominal / (ms_max * 1e-3),
                "evaluated_fraction": units / units_nominal if units_nominal else None,
                "swarm_iters_per_s": world * 1e3 / ms_per_step,
                "kernel_ms_per_step": {k: v[0] / args.steps for k, v in timing.items() if v[1]},
                "wall_s_timed_region": t_wall,
                "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"],
                           "samples": clocks["samples"]},
                "roofline": roof, "gpu_launches": int(gpu_launches)}
        if ad_N:
            line["config"]["segments"] = f"per-particle equal-SNR^2 (PAPER.md:120), N = {ad_N}"
        if extras:
            line["extras"] = extras
        if e2e:
            line["e2e"] = {"value": units / args.steps / (e2e_ms_max * 1e-3), "unit": UNIT,
                           "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                           "ms_per_step": e2e_ms_max}
        if not args.no_cpu_baseline and world == 1:
            from oracle import sc_oracle as orc
            cores = orc.num_threads()
            n_p, k_cpu = 4 * max(8, min(32, cores)), 3          # ~10-20 s of CPU work on the box's cores
            sec, cores = oracle_sample_run(sy.config_inputs(cid, P=n_p), N, n_p, k_cpu, 0)
            # (the oracle evaluates every bin of the band and masks those outside the window: its rate counts all of them)
            line["cpu_baseline"] = {"value": n_p * nb / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{n_p} particles x all {nb} bins per step, {k_cpu} steps (statistic + PSO), "
                                              f"{sec * k_cpu:.1f} s wall"}
        print(json.dumps(line), flush=True)
    H.close()
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: re-execute this script under torch.distributed.run with N ranks on
    this node (one process per GPU, rendezvous on 127.0.0.1), exactly as the driver launches it; returns its exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_dist_selftest(args, rank, world):
    """CPU check of the multi-rank plumbing (tests/test_multi_rank.py): gloo process group, the partition rule, and the
    reduction bench.py applies to its timings (max over ranks) and work (sum over ranks).  No GPU, no kernels."""
    import torch.distributed as dist
    from paper_2408_13170_b200 import dist as scd
    dist.init_process_group("gloo")
    a, b, need = scd.shard_swarms(40000, 4, rank, world) if world <= 4 else scd.shard_swarms(40000, 4, rank, world)
    ms = scd.max_over_ranks(10.0 + rank)
    units = scd.sum_over_ranks(float(b - a))
    if rank == 0:
        print(json.dumps({"selftest": "dist", "n_gpus": world, "ms_max": ms, "units": units, "shard0": [a, b, need]}), flush=True)
    dist.destroy_process_group()


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and (args.impl == "ours" or args.dist_selftest):
        sys.exit(spawn_ranks(args))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.dist_selftest:
        run_dist_selftest(args, rank, world)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        if world != args.gpus:
            sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE = {world}")
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
