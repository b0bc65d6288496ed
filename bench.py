#!/usr/bin/env python
"""bench.py -- throughput of the Wannier-to-Bloch e-ph interpolation path on B200.

Metric (BASELINE.json): interpolated |g(k,q)|^2 elements/s in FP64, elements = Nk * Nq * Nb^2 * Nm.
Workload at N = 1: BASELINE.json configs[1] ("Si-like production": Nb=8, Nm=6, Ne=Np=343, 40^3 k grid, random q).
A step = one interpolate call over ALL 64,000 k and a batch of `--nq-step` q-points: every stage of the path (S0 phase
tables, S1 Rp->q, D(q)/H(k)/H(k+q) + eigensolves, S4a, S2 Re->k, S4b + |g|^2).  `--k-mode grid` (default) hands the k-points
over as the uniform grid they are (epw_interp_interpolate_grid: factorised S2); `--k-mode list` as a plain list (dense FP64
tensor-path S2); in grid mode the list form is timed as well and reported as `klist_path`.
With N > 1 the q-points are sharded over ranks (the paper's image level: no communication inside
the loop) -> weak scaling, no data-path collective; `--rp-shard` splits g(Re,Rp) by Rp instead (one reduce-scatter per step).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--nq-step Q] [--k-mode grid|list] [--impl reference]
    python bench.py --eq6 [--config I]                 Eq. 6 (Bloch -> Wannier), own JSON line
    python bench.py --energy-window EMIN EMAX          with pair pre-screening, own metric name

`--impl reference` times the CPU oracle (oracle/, plain C) on the host cores on a bounded sample of the same
workload; it is a deliberately slow baseline, not a target.
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
sys.path.insert(0, ROOT)

METRIC = "interpolated |g(k,q)|^2 elements/s (FP64)"
UNIT = "elements/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1 = Si-like production)")
    ap.add_argument("--configs", default="2,3,4",
                    help="with the default --config 1: the other configs run for a few steps after the headline and reported "
                         "under `configs` in the same JSON line (comma list; `none` to skip)")
    ap.add_argument("--nq-step", type=int, default=0,
                    help="q-points per step (per GPU); 0 = the config's default (96 / 32 / 13 / 2 for configs 1-4), reduced so "
                         "that the |g|^2 buffer of a step stays below 40 GB")
    ap.add_argument("--q-batch", type=int, default=0, help="library q_batch for S1 (0 = default)")
    ap.add_argument("--energy-window", type=float, nargs=2, metavar=("EMIN", "EMAX"), default=None,
                    help="NEXT-3 (PAPER.md:L241): pre-screen the pairs with this energy window (eV); the line then reports "
                         "KEPT elements/s under its own metric name (not comparable with the unscreened headline)")
    ap.add_argument("--consumer", action="store_true",
                    help="NEXT-4: reduce |g|^2 on the device into the Im Sigma_nk accumulator (g2 = NULL: the Nk x Nq output "
                         "never exists); own metric name")
    ap.add_argument("--rp-shard", action="store_true",
                    help="NEXT-1 (PAPER.md:L186-188): g(Re,Rp) split by Rp over the ranks; per step every rank contracts "
                         "its slabs for the q-points of ALL ranks, one NCCL reduce-scatter of g(Re,q) hands each rank the "
                         "summed g(Re,q) of its own q-points, and the rest of the path runs unchanged")
    ap.add_argument("--rp-fused", action="store_true",
                    help="with --rp-shard: the exchange step fused into the S1 kernel (epw_interp_rp_to_q_scatter_add): every "
                         "rank adds its partial g(Re,q) straight into the owner's buffer over NVLink peer mappings "
                         "(torch symmetric memory) instead of a reduce-scatter after the pass.  On one GPU the owner is "
                         "this GPU; the multi-GPU branch has never run (one GPU per call here)")
    ap.add_argument("--grid-unfused", action="store_true", help="EPW_FLAG_GRID_UNFUSED: keep g~ in HBM between S2 and S4b")
    ap.add_argument("--grid-fused", action="store_true", help="EPW_FLAG_GRID_FUSED: force the fused last-pass + rotation kernel")
    ap.add_argument("--k-mode", default="grid", choices=["grid", "list"],
                    help="grid: epw_interp_interpolate_grid (the configs' k-points ARE uniform grids; factorised S2); "
                         "list: epw_interp_interpolate on the same k-points as a plain list (dense DMMA S2)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-klist-arm", action="store_true", help="skip the extra list-mode measurement of --k-mode grid")
    ap.add_argument("--stages", action="store_true", help="also print per-stage device times to stderr")
    ap.add_argument("--eq6", action="store_true",
                    help="time Eq. 6 (Bloch -> Wannier, epw_wannier_from_bloch) on coarse grids that match the config's "
                         "R sets instead of the interpolation path; prints its own JSON line")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------------------
# clocks: sample nvidia-smi during the timed region (B200_PROFILING.md "clocks DURING the timed region")
# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.samples = []
        self.proc = None
        self.gpu_index = gpu_index
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu_index), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            f = [x.strip() for x in s.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------------------------
def oracle_sample(w, n_q: int, n_k: int, seed: int = 1234, q_pool=None):
    """Time the oracle, as it stands, on n_q sampled q x n_k sampled k of workload w.  g(Re,Rp) is taken whole when it
    fits the host, else Eq. 9 is accumulated one Rp slab at a time (it is a sum over Rp; slab generation is not timed).
    q_pool: draw the q-points from these indices of w.q_list only (the q block of one bench step).
    Returns (elements/s amortising Eq. 9 over the full Nk, seconds spent, threads, description, raw results)."""
    import oracle

    rng = np.random.default_rng(seed)
    pool = np.arange(w.nq) if q_pool is None else np.asarray(q_pool)
    iq = np.sort(rng.choice(pool, size=min(n_q, len(pool)), replace=False))
    ik = np.sort(rng.choice(w.nk, size=min(n_k, w.nk), replace=False))
    ks = np.ascontiguousarray(w.k_list[ik])
    qs = np.ascontiguousarray(w.q_list[iq])
    E = w.elements_per_pair
    threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    pairs = len(iq) * len(ik)
    if w.g_bytes <= (8 << 30):
        g = w.g_full()
        t0 = time.perf_counter()
        g1 = oracle.rp_to_q(g, w.Rp, w.w_p, qs[0])  # Eq. 9 for one q (single thread, as written)
        t_eq9 = time.perf_counter() - t0
        del g1
        t0 = time.perf_counter()
        res = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, ks, qs)
        t_all = time.perf_counter() - t0
        t_pair = max(t_all - len(iq) * t_eq9, 1e-9) / pairs
    else:
        t_eq9, t_pairs, res = 0.0, 0.0, []
        for q in qs:
            g1 = np.zeros((w.nmodes, w.ne, w.nbnd, w.nbnd), dtype=np.complex128)
            for ip in range(w.np_):
                slab = w.g_slabs(ip, 1)
                t0 = time.perf_counter()
                g1 += oracle.rp_to_q(slab, w.Rp[ip:ip + 1], w.w_p[ip:ip + 1], q)
                t_eq9 += time.perf_counter() - t0
                del slab
            t0 = time.perf_counter()
            e_cm, om = oracle.phonon(w.D_R, w.Rp, w.w_p, q)
            for k in ks:
                res.append(oracle.pair(g1, w.H_R, w.Re, w.w_e, e_cm, om, k, q) + (om,))
            t_pairs += time.perf_counter() - t0
        t_eq9 /= len(qs)
        t_all = t_pairs + len(qs) * t_eq9
        t_pair = t_pairs / pairs
    per_elem = (t_pair + t_eq9 / w.nk) / E
    desc = (f"{len(iq)} random q x {len(ik)} random k of config {w.index} ({pairs} pairs); Eq. 9 per q "
            f"({t_eq9:.3f} s, 1 thread) amortised over the full Nk={w.nk}")
    return 1.0 / per_elem, t_all + t_eq9, threads, desc, (iq, ik, res)


def parity_of_last_step(w, q_blk, eps_k, eps_kq, omega, g2):
    """The oracle on a small sample of the (q, k) pairs of ONE bench step (q_blk = indices of its q-points), compared with
    that step's device outputs at the parity tolerances of tests/parity.py (north_star: eigenvalues 1e-10, |g|^2 1e-9
    relative over degenerate subspaces).  Returns a JSON-able record; never raises on a mismatch (it is reported)."""
    import torch

    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity import eig_close, g2_pair_close

    big = w.elements_per_pair > 1_000_000
    n_q, n_k = (1, 2) if big else (2, 48)   # configs[4]: a pair costs the oracle ~45 s; Eq. 9 (20 s) is shared by the two
    _, secs, threads, desc, (iq, ik, res) = oracle_sample(w, n_q, n_k, seed=77, q_pool=q_blk)
    pos = [int(np.nonzero(np.asarray(q_blk) == q)[0][0]) for q in iq]
    kt = torch.as_tensor(ik, device=eps_k.device)
    g_eps_k = eps_k[kt].cpu().numpy()
    ok_all, worst_g2, worst_eig = True, 0.0, 0.0
    for a, p in enumerate(pos):
        g_om = omega[p].cpu().numpy()
        g_ekq = eps_kq[p][kt].cpu().numpy()
        g_g2 = g2[p][kt].cpu().numpy()
        for b in range(len(ik)):
            if isinstance(res, list):
                r_g2, r_ek, r_ekq, r_om = res[a * len(ik) + b]
            else:
                r_ek, r_ekq, r_om, r_g2 = res[0][b], res[1][a, b], res[2][a], res[3][a, b]
            for got, ref in ((g_eps_k[b], r_ek), (g_ekq[b], r_ekq), (g_om, r_om)):
                e, ok = eig_close(got, ref)
                worst_eig, ok_all = max(worst_eig, float(e)), ok_all and ok
            e, ok = g2_pair_close(g_g2[b], r_g2, r_ekq, r_ek, r_om)
            worst_g2, ok_all = max(worst_g2, float(e)), ok_all and ok
    return {"ok": bool(ok_all), "pairs": len(pos) * len(ik), "worst_g2_over_tolerance": worst_g2,
            "worst_eig_scaled_error": worst_eig, "tolerances": "eig 1e-10, |g|^2 1e-9 rel + 1e-11 max (tests/parity.py)",
            "sample": desc, "oracle_seconds": secs}


def sample_size(w):
    """(n_q, n_k) of the bounded oracle sample: about 10-30 s of CPU work."""
    E = w.elements_per_pair
    if E > 1_000_000:
        return 1, 2     # configs[4]: ~50 s per pair in the oracle's plain loops
    return (8, 8192) if E < 2000 else (4, 512)


def run_reference(args):
    """`--impl reference`: the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import synth

    w = synth.make_config(args.config)
    n_q, n_k = sample_size(w)
    n_q, n_k = max(1, n_q // 2), max(1, n_k // 4)
    vals, secs = [], []
    threads, desc = 1, ""
    for step in range(args.warmup + args.steps):
        v, s, threads, desc, _ = oracle_sample(w, n_q, n_k, seed=100 + step)
        if step >= args.warmup:
            vals.append(v); secs.append(s)
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{w.index}] {w.name}", "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------------------
# B200 arm
# ------------------------------------------------------------------------------------------------------------
def run_eq6(args):
    """Eq. 6 at the size of the config's operator: coarse k', q' grids with one lattice vector per residue class
    (so that the transform is the exact inverse of the interpolation), random coarse-grid data on the device."""
    import torch

    import paper_2603_10295_b200 as epw
    import synth

    torch.cuda.set_device(0)
    w = synth.make_config(args.config)
    Nc = [int(w.Re[:, d].max() - w.Re[:, d].min() + 1) for d in range(3)]
    ax = [np.arange(n) / n for n in Nc]
    kc = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)
    nkc = nqc = len(kc)
    nb, nm = w.nbnd, w.nmodes
    G = torch.randn((nqc, nkc, nm, nb, nb, 2), dtype=torch.float64, device="cuda")
    out = torch.empty((w.np_, nm, w.ne, nb, nb, 2), dtype=torch.float64, device="cuda")
    kd, Red, Rpd = torch.from_numpy(kc).cuda(), torch.from_numpy(w.Re).cuda(), torch.from_numpy(w.Rp).cuda()

    def call():
        epw.epw_wannier_from_bloch(G, kd, nkc, kd, nqc, Red, w.ne, Rpd, w.np_, nb, nm, out)

    for _ in range(args.warmup):
        call()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        call()
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    E = nb * nb * nm
    flops = 8.0 * E * (float(w.ne) * nkc * nqc + float(w.ne) * w.np_ * nqc)
    peaks = epw.epw_probe_peaks(0)
    print(json.dumps({
        "metric": "Eq. 6 Bloch->Wannier: g(Re,Rp) elements/s (FP64)", "value": E * w.ne * w.np_ / (ms * 1e-3),
        "unit": "elements/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"Eq. 6 for the operator of configs[{w.index}]: {nkc} k' x {nqc} q' coarse points "
                               f"({'x'.join(map(str, Nc))} grids), Nb={nb} Nm={nm} Ne={w.ne} Np={w.np_}; includes the "
                               "call's own workspace allocation and phase tables"},
        "roofline": {"bound": "tensor", "kernel": "zgemm_strided_kernel (2 launches)", "achieved": flops / (ms * 1e-3) / 1e12,
                     "peak": peaks["fp64_dmma_tflops"], "unit": "TFLOP/s",
                     "frac": flops / (ms * 1e-3) / 1e12 / peaks["fp64_dmma_tflops"], "traffic": None},
    }))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.eq6:
        run_eq6(args)
        return

    import torch
    import torch.distributed as dist

    import paper_2603_10295_b200 as epw

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the interpolation path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    epw.load_library()
    ctx = {"world": world, "rank": rank, "local_rank": local_rank, "dist": dist if world > 1 else None}

    special = bool(args.energy_window or args.consumer or args.rp_shard or args.k_mode == "list")
    legs = set()
    if not args.no_e2e:
        legs.add("e2e")
    if not args.no_klist_arm:
        legs.add("klist")
    if not args.no_cpu_baseline:
        legs.add("cpu")
    line = run_config(args, ctx, args.config, args.steps, args.warmup, legs)

    # ---- the other production shapes (north_star: "reported on ... silicon, MoS2 and stanene-nanoribbon cases"): a few
    #      steps of configs[2], [3], [4] after the headline, each with its own stage rooflines, clocks and a sampled
    #      parity check of that very run against the oracle ----
    extra = [] if args.configs == "none" else [int(x) for x in args.configs.split(",") if x]
    if world == 1 and args.config == 1 and not special and extra:
        line_cfgs = {}
        for idx in extra:
            if idx == args.config:
                continue
            t0 = time.perf_counter()
            sub = run_config(args, ctx, idx, EXTRA_STEPS[idx][0], EXTRA_STEPS[idx][1], {"klist", "parity"})
            line_cfgs[str(idx)] = summarise_config(sub, time.perf_counter() - t0)
        # the on-device consumer end to end (host API, Im Sigma_nk instead of |g|^2 comes back): a few steps of the headline config
        e2e_consumer = None
        if "e2e" in legs:
            import copy

            args_c = copy.copy(args)
            args_c.consumer = True
            sub = run_config(args_c, ctx, args.config, 5, 3, {"e2e"})
            if rank == 0 and sub.get("e2e"):
                e2e_consumer = {"value": sub["e2e"]["value"], "ms": round(sub["e2e"]["ms_per_step"], 3),
                                "d2h_bytes_per_step": sub["e2e"]["d2h_bytes_per_step"], "device_ms": round(sub["ms_per_step"], 3)}
        if rank == 0:
            # the verbose per-config records first, the compact summary LAST: a record that keeps only the tail of this line
            # (it is > 10 KB) still shows value, dominant stage, fractions, clocks and parity of configs[2..4]
            line["configs"] = line_cfgs
            line["configs_brief"] = brief_of(line_cfgs, e2e_consumer)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# default q-points per step (per GPU) of each config: a caller batches as many q as its |g|^2 buffer allows.  On a uniform
# grid the k side (phases, H(k), U_k, eps_k) is computed by the FIRST call on that grid and kept in the handle, so the timed
# steps (which follow the warm-up steps on the same handle and grid) do not contain it: every record says so ("k_side") and
# carries the time of one step with the cache emptied ("cold_call_ms").  configs[1]: 96 q = 18.9 GB of output per step and a 50 ms step, so that
# the driver's 20 timed steps last a second; configs[3]: 13 q = 40 GB; configs[4]: 2 q = 34 GB.
NQ_STEP = {0: 64, 1: 96, 2: 32, 3: 13, 4: 2}
# (timed steps, warm-up steps) of the extra configs of the default run
EXTRA_STEPS = {0: (5, 3), 1: (5, 3), 2: (5, 3), 3: (3, 3), 4: (2, 1)}


def _r(x, n=4):
    return None if x is None else float(f"{x:.{n}g}")


def brief_of(line_cfgs: dict, e2e_consumer) -> dict:
    """<= 1,200 characters: per extra config the value, step time, dominant stage (kernel, fraction of its roofline, share of
    the step), the fractions of S4b / S2 / S1 / the H(k+q) eigensolves, the sampled parity verdict and the clocks."""
    out = {}
    for idx, c in line_cfgs.items():
        d, st, par, clk = c["dominant"], c["stages"], c.get("parity") or {}, c.get("clocks") or {}
        fr = lambda n: _r((st.get(n) or {}).get("frac"), 3)
        out[idx] = {"value": _r(c["value"]), "ms": _r(c["ms_per_step"]), "cold_ms": _r(c.get("cold_call_ms")),
                    "dom": d.get("stage"), "kernel": (d.get("kernel") or "").split(" ")[0], "frac": _r(d.get("frac"), 3),
                    "share": _r(d.get("share_of_step"), 3), "s4b": fr("S4b_rotate_g2"), "s2": fr("S2_re_to_k"),
                    "s1": fr("S1_rp_to_q"), "eig": fr("Hkq_eig"), "parity_ok": par.get("ok"),
                    "worst": _r(par.get("worst_g2_over_tolerance"), 3), "pairs": par.get("pairs"),
                    "sm_mhz": clk.get("sm_mhz"), "reasons": clk.get("reasons")}
    if e2e_consumer:
        out["e2e_consumer"] = {k: (_r(v) if isinstance(v, float) else v) for k, v in e2e_consumer.items()}
    return out


def summarise_config(sub: dict, wall_s: float) -> dict:
    """What the headline line keeps of an extra config's run."""
    r = sub["roofline"] or {}
    stages = r.get("stages", {})
    kl = sub.get("klist_path") or {}
    return {
        "workload": sub["config"]["workload"], "value": sub["value"], "unit": sub["unit"], "ms_per_step": sub["ms_per_step"],
        "steps": sub["steps"], "warmup": sub["warmup"], "gpu_launches": sub["gpu_launches"], "clocks": sub["clocks"],
        "dominant": {k: r.get(k) for k in ("stage", "kernel", "bound", "achieved", "peak", "unit", "frac", "share_of_step",
                                           "traffic")},
        "stages": {n: {k: st.get(k) for k in ("kernel", "bound", "frac", "share_of_step", "hbm_frac") if k in st}
                   for n, st in stages.items()},
        "klist_path": None if not kl else {"value": kl.get("value"), "ms_per_step": kl.get("ms_per_step"),
                                           "S2_re_to_k": {k: (kl.get("S2_re_to_k") or {}).get(k)
                                                          for k in ("kernel", "bound", "frac", "share_of_step")}},
        "parity": sub.get("parity"), "wall_s": wall_s, "k_side": (sub["config"].get("k_side") or "").split(":")[0],
        "cold_call_ms": sub["config"].get("cold_call_ms"),
    }


def run_config(args, ctx, cfg_index: int, steps: int, warmup: int, legs: set) -> dict:
    """Time `steps` steps (after `warmup`) of BASELINE.json configs[cfg_index] and return the JSON line of that run.
    legs: "e2e" (host-buffer entry point), "klist" (the same k as a plain list), "cpu" (oracle timed on the host cores),
    "parity" (sampled pairs of the last timed step against the oracle)."""
    import torch

    import paper_2603_10295_b200 as epw
    import synth
    from paper_2603_10295_b200 import shard

    world, rank, local_rank, dist = ctx["world"], ctx["rank"], ctx["local_rank"], ctx["dist"]
    want_e2e = "e2e" in legs
    w = synth.make_config(cfg_index)
    nk, E = w.nk, w.elements_per_pair
    # q-points per interpolate call: as many q as the |g|^2 buffer allows, at most 40 GB of output per step.  (k-list calls
    # compute the k side -- phases, H(k), U_k -- once per call; grid calls only on the first call on a grid, see "k_side")
    nq_step = (args.nq_step if cfg_index == args.config else 0) or NQ_STEP.get(cfg_index, 32)
    nq_step = max(1, min(nq_step, int((40 << 30) // (8 * nk * E))))
    nq_step = min(nq_step, w.nq)
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, device=local_rank, q_batch=args.q_batch,
                      flags=epw.EPW_FLAG_GRID_UNFUSED if args.grid_unfused else (epw.EPW_FLAG_GRID_FUSED if args.grid_fused else 0))
    t0 = time.perf_counter()
    # upload once; resident for the whole run; with --rp-shard only this rank's Rp slabs
    h.set_operators_from_host(w, rp_range=shard.rp_ranges(w.np_, world)[rank] if args.rp_shard else None)
    torch.cuda.synchronize()
    t_upload = time.perf_counter() - t0

    k_dev = torch.from_numpy(w.k_list).cuda()
    kq_map = w.kq_map
    total_steps = warmup + steps

    def q_block(step):
        """q-points of this rank for this step (ranks own disjoint q: the image level of the paper)."""
        return shard.q_block(step, world, rank, nq_step, w.nq)

    q_blocks = [q_block(s) for s in range(total_steps)]
    q_dev = [torch.from_numpy(np.ascontiguousarray(w.q_list[i])).cuda() for i in q_blocks]
    map_dev = None
    if kq_map is not None:
        map_dev = [torch.from_numpy(np.ascontiguousarray(kq_map[i])).cuda() for i in q_blocks]
    eps_k = torch.empty((nk, w.nbnd), dtype=torch.float64, device="cuda")
    eps_kq = torch.empty((nq_step, nk, w.nbnd), dtype=torch.float64, device="cuda")
    omega = torch.empty((nq_step, w.nmodes), dtype=torch.float64, device="cuda")
    g2 = torch.empty((nq_step, nk, w.nmodes, w.nbnd, w.nbnd), dtype=torch.float64, device="cuda")  # reused every step

    use_grid = args.k_mode == "grid"
    mask_dev = None
    if args.energy_window:
        mask_dev = torch.zeros((nq_step, nk), dtype=torch.uint8, device="cuda")
        epw.epw_interp_set_energy_window(h.h, True, args.energy_window[0], args.energy_window[1], mask_dev)
        want_e2e = False
    acc_dev = None
    if args.consumer:
        acc_dev = torch.zeros((nk, w.nbnd), dtype=torch.float64, device="cuda")
        # chemical potential in the middle of the bands of the first k-point, room temperature, 20 meV broadening
        epw.epw_interp_set_selfenergy_consumer(h.h, True, 0.0, 0.025, 0.02, None, acc_dev)
    if args.rp_shard:
        want_e2e = False   # the host-buffer entry point has no Rp-sharded form
    rows = w.slab_elems
    q_all_dev = None
    if args.rp_shard:
        # the q-points of every rank for each step (rank r owns block r of the step's world*nq_step points)
        q_all_dev = [torch.from_numpy(np.ascontiguousarray(
            w.q_list[np.concatenate([shard.q_block(s, world, r, nq_step, w.nq) for r in range(world)])])).cuda()
            for s in range(total_steps)]
        g1_part = None if args.rp_fused else torch.empty((world * nq_step, rows, 2), dtype=torch.float64, device="cuda")
        symm = None
        if args.rp_fused and world > 1:
            # The owners' buffers as symmetric memory, so that every rank holds a peer mapping of every other rank's buffer.
            # The pointer-table logic below (own pointers + mapped foreign pointers, zero / barrier / add / barrier) is what
            # tests/test_gpu_ipc.py runs across two processes with CUDA-IPC mappings on one GPU; the symmetric-memory
            # rendezvous itself needs a multi-GPU node and has not been executed in this project's runs (one GPU per call).
            import torch.distributed._symmetric_memory as symm_mem

            g1_mine = symm_mem.empty((nq_step, rows, 2), dtype=torch.float64, device="cuda")
            symm = symm_mem.rendezvous(g1_mine, dist.group.WORLD)
            bases = [int(p_) for p_ in symm.buffer_ptrs]
        else:
            g1_mine = torch.empty((nq_step, rows, 2), dtype=torch.float64, device="cuda")
            bases = [g1_mine.data_ptr()]
        # q-point j of rank r's block lives in rank r's buffer, row block j
        dst_ptrs = [bases[r] + j * rows * 16 for r in range(world) for j in range(nq_step)]

    def step(s, grid=None):
        if args.rp_shard and args.rp_fused:
            g1_mine.zero_()
            if symm is not None:
                symm.barrier()    # every owner has zeroed its buffer
            epw.epw_interp_rp_to_q_scatter_add(h.h, q_all_dev[s], world * nq_step, dst_ptrs)
            if symm is not None:
                symm.barrier()    # every rank's additions have landed
            epw.epw_interp_set_gq(h.h, g1_mine)
        elif args.rp_shard:
            epw.epw_interp_rp_to_q_partial(h.h, q_all_dev[s], world * nq_step, g1_part)
            if world > 1:
                dist.reduce_scatter_tensor(g1_mine, g1_part, op=dist.ReduceOp.SUM)   # the one exchange step, on the stream
                epw.epw_interp_set_gq(h.h, g1_mine)
            else:
                epw.epw_interp_set_gq(h.h, g1_part)
        g2_arg, ekq_arg = (None, None) if args.consumer else (g2, eps_kq)
        if use_grid if grid is None else grid:
            epw.epw_interp_interpolate_grid(h.h, w.k_grid, None, q_dev[s], nq_step,
                                            None if map_dev is None else map_dev[s], eps_k, ekq_arg, omega, g2_arg)
        else:
            epw.epw_interp_interpolate(h.h, k_dev, nk, q_dev[s], nq_step, None if map_dev is None else map_dev[s],
                                       eps_k, ekq_arg, omega, g2_arg)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def measure(grid, with_clocks):
        """W warm-up steps, then K timed steps (CUDA events on the launching stream, barrier + synchronize on both
        sides, max over ranks).  Returns everything the JSON line needs about this arm."""
        for s in range(warmup):
            step(s, grid)
        epw.epw_interp_sync(h.h)
        epw.epw_interp_enable_stage_timing(h.h, True)
        sampler = ClockSampler(local_rank)
        if rank == 0 and with_clocks:
            sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        launches = 0
        barrier()
        ev0.record()
        for s in range(warmup, total_steps):
            step(s, grid)
            launches += epw.epw_interp_last_launch_count(h.h)
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1)
        clocks = sampler.stop() if (rank == 0 and with_clocks) else None
        epw.epw_interp_sync(h.h)  # raises if an eigensolve did not converge
        out = {"stage_ms": epw.epw_interp_get_stage_times(h.h), "stage_launches": epw.epw_interp_get_stage_launches(h.h),
               "rotations": epw.epw_interp_get_eigh_rotations(h.h), "plan": epw.epw_interp_last_plan(h.h),
               "launches": launches, "clocks": clocks}
        epw.epw_interp_enable_stage_timing(h.h, False)
        out["ms"] = shard.max_over_ranks_ms(ms, dist, device="cuda")
        return out

    m = measure(use_grid, True)
    ms, clocks, launches = m["ms"], m["clocks"], m["launches"]
    # The timed steps above ran with the k side of the grid cached in the handle (computed by the first warm-up step).  One
    # more step with the cache emptied -- a call on the same grid with another shift evicts it -- gives the cold figure.
    cold_ms = None
    if use_grid and not args.rp_shard:
        ekq_c = None if args.consumer else eps_kq
        g2_c = None if args.consumer else g2
        # (its outputs are overwritten by the step that follows; with a kq_map they are not even meaningful on the shifted grid)
        epw.epw_interp_interpolate_grid(h.h, w.k_grid, np.array([0.5, 0.0, 0.0]), q_dev[-1], nq_step,
                                        None if map_dev is None else map_dev[-1], eps_k, ekq_c, omega, g2_c)
        barrier()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        step(total_steps - 1, True)
        c1.record()
        barrier()
        cold_ms = shard.max_over_ranks_ms(c0.elapsed_time(c1), dist, device="cuda")
        epw.epw_interp_sync(h.h)
    parity = None
    if "parity" in legs and rank == 0 and not (args.consumer or args.energy_window):
        # the outputs of the LAST timed step are still in the device buffers: compare a sample of them with the oracle
        parity = parity_of_last_step(w, q_blocks[-1], eps_k, eps_kq, omega, g2)
    elements_per_step = nk * nq_step * E
    value = world * elements_per_step * steps / (ms * 1e-3)
    window = None
    if mask_dev is not None:
        kept = float(mask_dev.float().mean().item())   # of the last step's pairs
        window = {"emin": args.energy_window[0], "emax": args.energy_window[1], "kept_fraction_last_step": kept,
                  "nominal_elements_per_s": value}
        value *= kept
    # the same k-points handed over as a plain list (dense FP64 tensor-path S2), reported beside the grid arm
    # (the large-Nb kernel family expands a grid to a list itself: one arm)
    m_list = measure(False, False) if (use_grid and "klist" in legs and w.nbnd <= 16) else None

    # ---- rooflines: every stage with a stated bound, the dominant one (largest share of the step) at top level ----
    roofline = None
    klist_path = None
    if rank == 0:
        peaks = epw.epw_probe_peaks(local_rank)
        mp = {}
        if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")):
            mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        traffic = {}
        tpath = os.path.join(ROOT, "profiles", "roofline_traffic.txt")
        if os.path.exists(tpath):
            traffic = json.load(open(tpath))
        nb, nm, ne = w.nbnd, w.nmodes, w.ne
        dmma, dfma, hbm = peaks["fp64_dmma_tflops"], peaks["fp64_dfma_tflops"], mp.get("hbm_gbs")
        Lbox = [int(w.Re[:, d].max() - w.Re[:, d].min() + 1) for d in range(3)]

        def stage_table(mm):
            """Algorithmic work of the algorithm actually executed / CUDA-event time of the stage."""
            plan, stage_ms, stage_launches, rot = mm["plan"], mm["stage_ms"], mm["stage_launches"], mm["rotations"]
            large, grid, fused = plan["path"] == "large", plan["k_mode"].startswith("grid"), plan["k_mode"] == "grid-fused"
            nsteps = steps
            pairs = float(nk) * nq_step * nsteps
            nq_tot = float(nq_step) * nsteps
            # H(k+q) rides on S2 as Nb^2 extra columns in the small path when k+q is not folded onto the grid
            ncols = E + (0 if (kq_map is not None or large) else nb * nb)
            n_eig = "eigh_thread_kernel" if nb <= 8 else ("eigh_cols_kernel" if nb <= 16 else "eigh_cluster_kernel")
            # FP64 flops of one plane rotation: thread kernel 20(2n-2)+25, column-pair kernel 36n+25
            rot_flops = (20.0 * (2 * nb - 2) + 25.0) if nb <= 8 else (36.0 * nb + 25.0)
            spec = {}
            if grid:
                N1, N2, N3 = w.k_grid
                L1, L2, L3 = Lbox
                # the last axis pass runs on all columns, or (fused form) only on the Nb^2 H(k+q) columns
                nc_last = (ncols - E) if fused else ncols
                mults = ncols * (L1 * L2 * N3 * L3 + L1 * N2 * N3 * L2) + nc_last * float(nk) * L1     # per q
                byts = 16.0 * (ncols * ((L1 * L2 * L3 + L1 * L2 * N3) + (L1 * L2 * N3 + L1 * N2 * N3))
                               + nc_last * (L1 * N2 * N3 + nk))
                # (two-kernel form: the last of the three passes is the pass-only variant of grid_fused_kernel; one-kernel
                #  form: it is inside grid_fused_kernel and counted with S4b)
                spec["S2_re_to_k"] = ("hbm", "axis_pass_kernel (axis passes)" if fused else
                                      "axis_pass_kernel (axes 3, 2) + grid_fused_kernel pass-only variant (axis 1)",
                                      byts * nq_tot, hbm, "GB/s",
                                      {"flops": 8.0 * mults * nq_tot})
            else:
                s2_kernel = "zgemm_dmma_kernel"
                if large:   # short lattice-vector lists go through the DMMA last-axis pass (interp.cu: s2_pass)
                    s2_kernel = "grid_fused_kernel (pass-only variant)" if (ne <= 18 and E % 64 == 0) else "zgemm_strided_kernel"
                spec["S2_re_to_k"] = ("tensor", s2_kernel,
                                      8.0 * ncols * ne * pairs, dmma, "TFLOP/s", {})
            if fused:
                # last axis pass of S2 (8 L1 E flops per pair, plain DFMA) + both rotation products (DMMA): one FP64 pipe
                spec["S4b_rotate_g2"] = ("tensor", "grid_fused_kernel", (8.0 * Lbox[0] * E + 16.0 * nb ** 3 * nm) * pairs,
                                         dmma, "TFLOP/s",
                                         {"hbm_bytes": (32.0 * nb * nb + 8.0 * E) * pairs
                                                       + 16.0 * E * Lbox[0] * w.k_grid[1] * w.k_grid[2] * nq_tot})
            else:
                # rotate_g2.cu: bulk-TMA staged kernel when g~, the two U and T of a pair fit 56 KB (four CTAs per SM)
                mt_rows = -(-(nm * nb) // 8) * 8
                rot_tma = 16 * ((nm + 2) * nb * nb + mt_rows * (nb + ((6 - (nb & 3)) & 3))) + 144 <= 56 * 1024 and nk >= 1024
                spec["S4b_rotate_g2"] = ("tensor", "zgemm_strided_kernel" if large else
                                         ("rotate_g2_tma_kernel" if rot_tma else "rotate_g2_dmma_kernel"),
                                         16.0 * nb ** 3 * nm * pairs, dmma, "TFLOP/s",
                                         {"hbm_bytes": (16.0 * (E + 2 * nb * nb) + 8.0 * E) * pairs})
            spec["S4a_mode_rotation"] = ("tensor" if large else "alu",
                                         "zgemm_strided_kernel" if large else ("box_scatter_kernel" if grid else "pack_b_kernel"),
                                         8.0 * nb * nb * nm * nm * ne * nq_tot, dmma if large else dfma, "TFLOP/s", {})
            if rot["Hkq"]:
                spec["Hkq_eig"] = ("alu", n_eig, rot_flops * rot["Hkq"], dfma, "TFLOP/s",
                                   {"rotations": rot["Hkq"], "solves": pairs, "rotations_per_solve": rot["Hkq"] / pairs})
            if rot["Hk"]:
                spec["Hk_eig"] = ("alu", n_eig + " (+ H(k) interpolation)", rot_flops * rot["Hk"], dfma, "TFLOP/s",
                                  {"rotations": rot["Hk"]})
            names = {"S2_re_to_k": "S2_re_to_k_dmma"}
            stages = {}
            for name, (bound, kernel, work, peak, unit, extra) in spec.items():
                key = names.get(name, name)
                t_ms, nl = stage_ms[key], max(1, stage_launches[key])
                if t_ms <= 0 or not peak:
                    continue
                ach = work / (t_ms * 1e-3) / (1e9 if unit == "GB/s" else 1e12)
                st = {"bound": bound, "kernel": kernel, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
                      ("bytes_per_launch" if unit == "GB/s" else "flops_per_launch"): work / nl, "launches": nl,
                      "avg_launch_ms": t_ms / nl, "share_of_step": t_ms / stage_ms["total"]}
                if "hbm_bytes" in extra and hbm:
                    st["hbm_frac"] = extra["hbm_bytes"] / (t_ms * 1e-3) / 1e9 / hbm
                st.update({k: v for k, v in extra.items() if k != "hbm_bytes"})
                stages[name] = st
            if use_grid and mm is m and warmup > 0 and not rot["Hk"]:
                # no H(k) solve ran inside the timed steps: the k side came from the handle's cache (config.k_side)
                stages["Hk_eig"] = {"cached": True, "kernel": n_eig, "share_of_step": 0.0,
                                    "note": "H(k), U_k, eps_k reused from the first call on this grid; see config.cold_call_ms"}
            n_s1 = -(-nq_step // plan["q_batch"])
            s1_bytes = (16.0 * w.slab_elems * w.np_ * n_s1 + 16.0 * w.slab_elems * nq_step) * nsteps
            s1 = {"bound": "hbm", "kernel": "rp_to_q_kernel", "achieved": s1_bytes / (stage_ms["S1_rp_to_q"] * 1e-3) / 1e9,
                  "peak": hbm, "unit": "GB/s", "bytes_per_launch": s1_bytes / (n_s1 * nsteps),
                  "launches": n_s1 * nsteps, "avg_launch_ms": stage_ms["S1_rp_to_q"] / (n_s1 * nsteps),
                  "share_of_step": stage_ms["S1_rp_to_q"] / stage_ms["total"]}
            if hbm:
                s1["frac"] = s1["achieved"] / hbm
            stages["S1_rp_to_q"] = s1
            return stages

        stages = stage_table(m)
        dom = max(stages, key=lambda n: stages[n]["share_of_step"])
        roofline = dict(stages[dom])
        roofline["stage"] = dom
        roofline["traffic"] = traffic.get(f"{stages[dom]['kernel'].split(' ')[0]}:{dom}:config{w.index}:{m['plan']['k_mode']}")
        roofline["peak_source"] = ("tensor: FP64 DMMA m8n8k4 issue-loop probe, alu: dependent-free DFMA loop probe, both run live on "
                                   "this GPU by epw_probe_peaks (MEASURED_PEAKS.json has no FP64 entry); hbm: MEASURED_PEAKS.json hbm_gbs")
        roofline["peak_from_measured_bf16_x_nominal_ratio"] = (mp.get("bf16_tflops_sustained", 0.0) * 45.0 / 2250.0) or None
        roofline["hbm_read_gbs_probe"] = peaks["hbm_read_gbs"]
        roofline["fp64_dfma_tflops_probe"] = dfma
        roofline["fp64_dmma_tflops_probe"] = dmma
        roofline["plan"] = m["plan"]
        roofline["stages"] = stages
        roofline["stage_ms_per_step"] = {k: v / steps for k, v in m["stage_ms"].items()}
        if m_list is not None:
            st_l = stage_table(m_list)
            klist_path = {"what": "the same k-points passed as a plain list to epw_interp_interpolate: dense S2 on the FP64 "
                                  "tensor path (zgemm_dmma_kernel), everything else identical",
                          "value": world * elements_per_step * steps / (m_list["ms"] * 1e-3), "unit": UNIT,
                          "ms_per_step": m_list["ms"] / steps, "S2_re_to_k": st_l.get("S2_re_to_k"),
                          "traffic": traffic.get(f"zgemm_dmma_kernel:S2_re_to_k_dmma:config{w.index}"),
                          "stage_ms_per_step": {k: v / steps for k, v in m_list["stage_ms"].items()}}
    if args.stages and rank == 0:
        print(json.dumps({k: round(v / steps, 4) for k, v in m["stage_ms"].items()}), file=sys.stderr)

    # ---- e2e: the same steps through the host-buffer entry point (H2D of k/q lists, D2H of all outputs) ----
    e2e = None
    if want_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        k_host = pin(w.k_list)
        q_host = [pin(w.q_list[i]) for i in q_blocks]
        map_host = None if kq_map is None else [pin(kq_map[i]) for i in q_blocks]
        o_eps_k = torch.empty((nk, w.nbnd), dtype=torch.float64).pin_memory()
        o_eps_kq = torch.empty((nq_step, nk, w.nbnd), dtype=torch.float64).pin_memory()
        o_omega = torch.empty((nq_step, w.nmodes), dtype=torch.float64).pin_memory()
        # with the consumer on nothing of size nk x nq leaves the device: the step returns eps_k, omega_q and Im Sigma_nk
        o_g2 = None if args.consumer else torch.empty((nq_step, nk, w.nmodes, w.nbnd, w.nbnd), dtype=torch.float64).pin_memory()
        o_acc = torch.empty((nk, w.nbnd), dtype=torch.float64).pin_memory() if args.consumer else None
        if args.consumer:
            o_eps_kq = None
        g2 = None   # the host-buffer entry point stages |g|^2 in the library's own device buffer
        torch.cuda.empty_cache()

        def step_host(s):
            if use_grid:
                epw.epw_interp_interpolate_grid_host(h.h, w.k_grid, None, q_host[s], nq_step,
                                                     None if map_host is None else map_host[s], o_eps_k, o_eps_kq,
                                                     o_omega, o_g2)
            else:
                epw.epw_interp_interpolate_host(h.h, k_host, nk, q_host[s], nq_step,
                                                None if map_host is None else map_host[s], o_eps_k, o_eps_kq, o_omega,
                                                o_g2)
            if o_acc is not None:
                o_acc.copy_(acc_dev, non_blocking=True)   # the step's result: the accumulator, device -> pinned host

        n_e2e_warm = min(warmup, 2)
        n_e2e = min(steps, 8)   # PCIe-bound (a third of a second per step on configs[1]): a bounded number of steps
        for s in range(n_e2e_warm):
            step_host(s)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for s in range(warmup, warmup + n_e2e):
            step_host(s)
        e1.record()
        barrier()
        ms_e2e = e0.elapsed_time(e1)
        ms_e2e = shard.max_over_ranks_ms(ms_e2e, dist, device="cuda")
        h2d = (0 if use_grid else k_host.numel() * 8) + q_host[0].numel() * 8 + (0 if map_host is None else map_host[0].numel() * 4)
        d2h = sum(t.numel() for t in (o_eps_k, o_eps_kq, o_omega, o_g2, o_acc) if t is not None) * 8
        e2e = {"value": world * elements_per_step * n_e2e / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e2e / n_e2e, "steps": n_e2e,
               "api": ("epw_interp_interpolate_grid_host" if use_grid else "epw_interp_interpolate_host")
                      + " (pinned host buffers in and out)"}

    # ---- CPU oracle beside it (rank 0, N = 1 only) ----
    cpu_baseline = None
    if rank == 0 and world == 1 and "cpu" in legs:
        n_q, n_k = sample_size(w)
        v, secs, threads, desc, _ = oracle_sample(w, n_q, n_k)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                        "seconds": secs}

    line = None
    if rank == 0:
        line = {
            "metric": (METRIC + " -- reduced on the device into Im Sigma_nk (no |g|^2 output)" if args.consumer else
                       METRIC if window is None else METRIC + " -- KEPT pairs only, energy-window pre-screening on"),
            "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {
                "workload": f"BASELINE.json configs[{w.index}] {w.name}: Nb={w.nbnd} Nm={w.nmodes} Ne={w.ne} Np={w.np_} "
                            f"Nk={nk} ({'x'.join(map(str, w.k_grid))}), {nq_step} q per step per GPU ({w.q_desc})",
                "global_batch_pairs": world * nk * nq_step, "parallelism": ((f"g(Re,Rp) Rp-sharded x{world}, partial g(Re,q) added into the owners' buffers inside the S1 kernel (peer memory)"
                                                                       if args.rp_fused else
                                                                       f"g(Re,Rp) Rp-sharded x{world} + reduce-scatter of g(Re,q) over q") if args.rp_shard
                                                                      else f"q-sharded x{world}"),
                "k_mode": ("uniform grid -> epw_interp_interpolate_grid" if use_grid else "k-list -> epw_interp_interpolate"),
                "l2": "inputs larger than L2: g(Re,Rp) %.0f MB streamed per q-batch, phase table %.0f MB, |g|^2 output %.0f MB "
                      "per step" % (w.g_bytes / 1e6, 16.0 * nk * w.ne / 1e6, 8.0 * elements_per_step / 1e6),
                "operator_upload_s": t_upload,
                "k_side": ("cached after warm-up: H(k), U_k, eps_k of the grid are computed by the first call on the handle and "
                           "reused; the timed steps exclude them, cold_call_ms is one step that recomputes them"
                           + (" (not measured with --rp-shard)" if args.rp_shard else "")
                           if use_grid else "computed inside every timed step (k-list calls keep no k side)"),
                "cold_call_ms": cold_ms,
            },
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "klist_path": klist_path, "energy_window": window, "cpu_baseline": cpu_baseline, "parity": parity,
        }
    h.close()
    h = eps_k = eps_kq = omega = g2 = q_dev = map_dev = k_dev = mask_dev = acc_dev = None
    torch.cuda.empty_cache()
    return line


if __name__ == "__main__":
    main()
