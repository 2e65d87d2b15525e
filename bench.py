#!/usr/bin/env python
"""bench.py -- throughput of the CFNEB hot path (BASELINE.json `metric`) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (K0-K6 of DESIGN.md: cell map, neighbour-list upkeep, batched
force / energy / virial, one-pass reductions, tangent + climbing image + FIRE scalars, fused update) over all
images of the band.  metric = atom x image x NEB-steps per second, counted over the MOVABLE images
(N (P-2) per step, reading A23); the N P figure is printed alongside in `config`.

  value      K graph-launched steps (cfneb_step), state resident in HBM, CUDA events on the library's stream,
             barrier + synchronize on both sides, max over ranks.
  roofline   the projection + FIRE kernels (K4 reduce + K6 update) the metric names: algorithmic bytes
             (192 B per atom-image-step) / their CUDA-event time per step, measured live by
             cfneb_step_timed over min(K, 200) further steps of the same band; against MEASURED_PEAKS.json hbm_gbs.
             `kernels` carries every class's time share and the force kernel's fp64 "alu" fraction.
  steady_state  the same measurement over max(K, 100) FURTHER steps, so that a short window cannot fall into a gap
             between neighbour-list rebuilds (an image rebuilds its list only when it left its skin: ~0.8 image
             rebuilds per step at configs[4]); `value` stays the K-step figure the contract asks for.
  e2e        the same metric through the C ABI with HOST (pinned) buffers, as a true continuation of the band:
             every step is one cfneb_step_hosted call: X, v and the FIRE scalars host -> device (image blocks on a
             second stream, evaluated while later blocks arrive), one iteration, X, v and the scalars back.
  cpu_baseline  the oracle as it stands, on this box's host cores, on a bounded sample of the same workload.

N > 1: the path does not shard (BASELINE.json: one GPU, no collectives) -- "replicas only": every rank runs the
same band on its own GPU; value = all ranks' units / max-over-ranks time.
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

METRIC = "atom_image_neb_steps_per_s"
UNIT = "atom*image*steps/s"
POTENTIAL_NAMES = ("lj_shifted_force", "finnis_sinclair_morse", "stillinger_weber", "descriptor_network", "nep_shaped_network")
ALGO_BYTES_PER_UNIT = 192.0  # K4 reads X, F, v (72 B); K6 reads X, F, v (72 B), writes X_new, v (48 B)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default 4: 101306 x 100); 5-8: the extra workloads of cfneb_workloads")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-steady", action="store_true", help="skip the steady-state window (profiling runs)")
    ap.add_argument("--no-preroll", action="store_true", help="time right after the warm-up, on fresh neighbour lists (the round-2 window)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.2] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full
    capture (profiles/dram_traffic.csv: workload,kernel,read_bytes,write_bytes,source), or None."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return None
    with open(path) as fh:
        for line in fh:
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and f[0] == workload and f[1] == kernel:
                return float(f[2]) + float(f[3])
    return None


def ncu_pipe(workload, kernel):
    """fp64-pipe and issue-slot utilisation of `kernel` from the committed ncu capture (profiles/pipe_utilisation.csv:
    workload,kernel,fp64 pipe %,issue active %,source), or None.  Context for the ALU roofline: the pair kernels are
    bound by instruction issue (an fp64 instruction holds its scheduler for two cycles), not by the flop count."""
    path = os.path.join(ROOT, "profiles", "pipe_utilisation.csv")
    if not os.path.exists(path):
        return None
    with open(path) as fh:
        for line in fh:
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and f[0] == workload and f[1] == kernel:
                return {"fp64_pipe_frac": float(f[2]) / 100.0, "issue_active_frac": float(f[3]) / 100.0}
    return None


# fp64 operations per in-range pair as the formulas of kernels_force.cu are written (FMA = 2, everything else = 1;
# DESIGN.md section 5): density pass plain / taper, force pass plain / taper (beta = 2 alpha: one exponential).
FLOPS_DENSITY = (40.0, 70.0)
FLOPS_FORCE = (71.0, 131.0)


def bain_pair_counts(cells, dims, r_on, r_cut):
    """In-range pairs per atom (plain, taper-zone) of every image of a perfect bcc supercell (dims conventional
    cells per axis) under the image's cell: lattice vectors v = (n + basis) a with |v| <= r_on, r_on < |v| < r_cut."""
    rng = np.arange(-5, 6)
    g = np.stack(np.meshgrid(rng, rng, rng, indexing="ij"), -1).reshape(-1, 3).astype(np.float64)
    frac = np.concatenate([g, g + 0.5])
    frac = frac[np.any(frac != 0.0, axis=1)]
    out = []
    for h in cells:
        r = np.linalg.norm(frac @ (np.asarray(h) / np.asarray(dims, dtype=np.float64)[:, None]), axis=1)
        out.append((int(np.sum(r <= r_on)), int(np.sum((r > r_on) & (r < r_cut)))))
    return out


def nep_flops_per_atom(pot, n_r_pairs, n_a_pairs):
    """fp64 operations per atom of K2 for the NEP-shaped potential, as the formulas of kernels_nep.cu / pass 2 are
    written (FMA = 2, everything else = 1; reciprocal-square-root seed and integer work not counted), for an atom with
    n_r_pairs neighbours inside rc_r and n_a_pairs inside rc_a.  Terms, with K_r, K_a the basis sizes, T the atom types,
    n_r / n_a the radial descriptors / angular channels, D descriptors, H neurons (DESIGN.md section 10 item 6):
      pair vector 8, own rsqrt 8, cos(pi t) 23 (with sin(pi t): 45), cut-off and Chebyshev argument 7-11;
      radial descriptors, per pair:      50 + 2 T K_r + 2 (K_r - 1)      (T multiply-adds and one recurrence step per k)
      radial forces pair by pair:        99 + 2 K_r + 10 (K_r - 1)       (T_k, T_k' recurrences, two sums, F and virial)
      quad kernel walk 1, per pair:      50 + 14 K_a + 101 n_a           (basis, g_n of 4 channels; per channel 31 monomial
                                                                          products + 35 multiply-adds into the moments)
      quad kernel walk 2, per pair:      76 + 32 K_a + 205 n_a           (basis with derivative, g_n and g_n'; per channel
                                                                          16 monomial products, 60 multiply-adds of the
                                                                          gradient polynomial, Euler sums, the 3 components)
      pass 2 over the angular pairs:     35
      per atom: network 4 D H + 35 H, moments -> descriptors and back 225 n_a, radial coefficients 3 T K_r n_r + 2 T K_r n_r."""
    n_r, n_a, k_r, k_a, L, H, T = (int(pot[i]) for i in (2, 3, 4, 5, 6, 7, 8))
    D = n_r + n_a * L
    radial = (50 + 2 * T * k_r + 2 * (k_r - 1)) + (99 + 2 * k_r + 10 * (k_r - 1))
    angular = (50 + 14 * k_a + 101 * n_a) + (76 + 32 * k_a + 205 * n_a) + 35
    per_atom = 4 * D * H + 35 * H + 225 * n_a + 5 * T * k_r * n_r
    return n_r_pairs * radial + n_a_pairs * angular + per_atom


def nep_pair_counts(band, images, rc_r, rc_a):
    """Mean number of neighbours inside rc_r and inside rc_a per atom, counted on the host from the band's own Verlet
    lists (parity hook) and current positions, for the given images."""
    pos, cells, _ = band.get_path()
    out = []
    for p in images:
        count, lst, shift = band.get_neighbors(p)
        mask = np.arange(lst.shape[1])[None, :] < count[:, None]
        j = np.where(mask, lst, 0)
        d = pos[p][j] + shift.astype(np.float64) @ cells[p] - pos[p][:, None, :]
        r = np.sqrt(np.sum(d * d, axis=2))
        out.append((float(np.sum((r < rc_r) & mask) / len(count)), float(np.sum((r < rc_a) & mask) / len(count))))
    return out


# ------------------------------------------------------------------------------------------------------------
def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


ORACLE_RATE = 1.5e4  # atom-images per second per thread, order of magnitude only (sizes the bounded sample)


def oracle_sample_plan(k, total_steps, budget_s):
    """Choose a bounded sample of configs[k] for the oracle: (n_images, dims or None, threads, description)."""
    from cfneb_workloads import CONFIGS
    spec = CONFIGS[k]
    cores = host_cores()
    movable = spec.n_images - 2
    threads = max(1, min(cores, movable, 16))
    if spec.lattice == "fcc_vacancy":
        return spec.n_images, None, threads, "full config (%d atoms x %d images)" % (spec.n_atoms, spec.n_images)
    m = threads  # one image per thread: the only parallelism the oracle has is over images
    per_step = budget_s / max(total_steps + 2.0, 1.0)  # + 2: the two endpoint evaluations at construction
    atoms = int(min(spec.n_atoms, max(432, per_step * ORACLE_RATE)))
    if atoms >= 0.5 * spec.n_atoms:
        return m + 2, None, threads, "%d consecutive movable images (mid-path) of the %d, all %d atoms" % (m, movable, spec.n_atoms)
    per_cell = spec.n_atoms / float(np.prod(spec.dims))  # atoms per conventional cell (2 bcc, 8 diamond)
    n = max(4, int(round((atoms / per_cell) ** (1.0 / 3.0))))
    return (m + 2, (n, n, n), threads,
            "%d movable images of a %dx%dx%d conventional-cell supercell (%d atoms) built by the same recipe as the %d-atom config"
            % (m, n, n, n, int(round(per_cell * n ** 3)), spec.n_atoms))


def run_oracle(k, steps, warmup, budget_s):
    """Time `steps` oracle iterations (after `warmup`) on a bounded sample.  Returns a dict."""
    from cfneb_workloads import build_workload
    from oracle import cfneb as oc
    n_images, dims, threads, what = oracle_sample_plan(k, steps + warmup, budget_s)
    spec, pos, cells = build_workload(k, dims=dims)
    P = pos.shape[0]
    if n_images < P:  # consecutive images around the middle of the path, between the two true endpoints
        lo = max(1, (P - (n_images - 2)) // 2)
        idx = [0] + list(range(lo, lo + n_images - 2)) + [P - 1]
        pos, cells = pos[idx], cells[idx]
    types = None
    if spec.types is not None:  # NEP-shaped potential: the generators' two-species ordering at the sample's atom count
        from cfneb_workloads import two_sublattice_types
        types = two_sublattice_types(pos.shape[1], int(spec.pot[8]))
    band = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb,
                    cell_factor=0.0, fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors, threads=threads,
                    types=types)
    for _ in range(warmup):
        band.step(1)
    t0 = time.perf_counter()
    for _ in range(steps):
        band.step(1)
    dt = time.perf_counter() - t0
    units = pos.shape[1] * (pos.shape[0] - 2) * steps
    return {"value": units / dt, "unit": UNIT, "cores": threads, "kind": "oracle", "host_cores": host_cores(),
            "sample": "%s; %d timed step(s) after %d warm-up" % (what, steps, warmup), "seconds": dt,
            "ms_per_step": 1e3 * dt / max(steps, 1), "n_atoms": int(pos.shape[1]), "n_images": int(pos.shape[0])}


def build_cfg(k):
    from cfneb_workloads import CONFIGS
    return CONFIGS[k]


def workload_name(k):
    spec = build_cfg(k)
    return "configs[%d] %s: %d atoms x %d images, fp64" % (k, spec.name, spec.n_atoms, spec.n_images)


def main_reference(args):
    """--impl reference: the oracle as it stands on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    r = run_oracle(args.config, args.steps, args.warmup, budget_s=150.0)
    spec = build_cfg(args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config), "potential": POTENTIAL_NAMES[int(spec.potential)],
                   "sample": r["sample"], "runs_on": "host CPU (oracle/, plain fp64 C + numpy)"},
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------------------
def main_ours(args):
    import torch
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import build_workload

    from paper_2510_16721_b200.replicas import Ranks
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CFNEB path has no CPU fallback")
    cf.lib()  # fail loudly if libcfneb.so is missing
    torch.cuda.set_device(local)
    ranks = Ranks("nccl", torch.device("cuda", local))
    rank, world = ranks.rank, ranks.world

    def barrier():
        ranks.barrier()
        torch.cuda.synchronize()

    max_over_ranks = ranks.max_over_ranks

    k = args.config
    spec, pos, cells = build_workload(k)
    P, N = pos.shape[0], pos.shape[1]
    prm = cf.params_for(spec, cell_factor=0.0)
    band = cf.CFNEB(pos, cells, prm, device="cuda:%d" % local)
    stream = band.stream
    units_per_step = N * (P - 2)

    # ---- device-resident throughput: W warm-up + K timed graph-launched steps ----
    band.step(args.warmup)
    band.synchronize()
    # ---- untimed pre-roll to the steady state of the list upkeep ----
    # Right after cfneb_create every list is fresh: no rebuild falls into a short window and K2 walks the shortest
    # columns it ever will (no dead tail rows yet), which flattered a 20-step window by ~15 % in round 2.  Step until
    # the band has rebuilt as many lists as it has movable images (every list has aged and been renewed about once),
    # at most 150 iterations; the timed region, the steady-state window and the per-class breakdown then all see the
    # same regime.
    preroll = 0
    if not args.no_preroll:
        r_start = band.get_status().rebuilds
        while preroll < 150 and band.get_status().rebuilds - r_start < P - 2:
            band.step(10)
            preroll += 10
        band.synchronize()
    st0 = band.get_status()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_wall0 = time.time()
    e0.record(stream)
    band.step(args.steps)
    e1.record(stream)
    stream.synchronize()
    barrier()
    t_wall1 = time.time()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    st1 = band.get_status()
    if st1.error != 0:
        raise RuntimeError("device error %d during the timed region" % st1.error)
    ms_per_step = ms_total / args.steps
    value = world * units_per_step * args.steps / (ms_total * 1e-3)

    # ---- steady state: max(K, 100) further graph-launched steps (list rebuilds amortised) ----
    n_ss = 0 if args.no_steady else max(args.steps, 100)
    barrier()
    e0.record(stream)
    band.step(n_ss)
    e1.record(stream)
    stream.synchronize()
    barrier()
    ms_ss = max_over_ranks(e0.elapsed_time(e1))
    st2 = band.get_status()
    steady = None if n_ss == 0 else {"value": world * units_per_step * n_ss / (ms_ss * 1e-3), "unit": UNIT, "steps": n_ss, "ms_per_step": ms_ss / n_ss,
              "neighbor_rebuilds": int(st2.rebuilds - st1.rebuilds),
              "what": "the next max(K, 100) steps of the same band, same timing; includes the amortised list rebuilds"}

    # ---- per-kernel-class CUDA-event times over K further steps of the same band (roofline) ----
    n_bd = min(args.steps, 200)  # breakdown window: bounded, so that a long --steps run does not double its time
    kms = band.step_timed(n_bd) / n_bd  # ms per step per class
    clocks = sampler.stop(t_wall0, time.time())
    peak, peak_src = measured_peaks()
    t_proj = (kms[cf.binding.K_REDUCE] + kms[cf.binding.K_UPDATE]) * 1e-3
    algo_bytes = ALGO_BYTES_PER_UNIT * units_per_step
    achieved = algo_bytes / t_proj / 1e9
    wl = "c%d" % k
    tr_reduce, tr_update = ncu_traffic(wl, "reduce_kernel"), ncu_traffic(wl, "update_kernel")
    roofline = {"kernel": "K4 reduce_kernel + K6 update_kernel (projection + FIRE)", "bound": "hbm", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": (tr_reduce + tr_update) if (tr_reduce and tr_update) else None,
                "traffic_source": "committed ncu --set full capture (profiles/dram_traffic.csv), not measured by this run",
                "algorithmic_bytes": algo_bytes, "ms": t_proj * 1e3,
                "share_of_step": float((kms[cf.binding.K_REDUCE] + kms[cf.binding.K_UPDATE]) / kms.sum())}
    kernels = {name: {"ms_per_step": float(kms[i]), "share": float(kms[i] / kms.sum())}
               for i, name in enumerate(cf.KERNEL_CLASSES)}
    kernels["sum_ms_per_step"] = float(kms.sum())
    kernels["update_only_GBps"] = 120.0 * units_per_step / (kms[cf.binding.K_UPDATE] * 1e-3) / 1e9
    kernels["reduce_only_GBps"] = 72.0 * units_per_step / (kms[cf.binding.K_REDUCE] * 1e-3) / 1e9
    # the dominant kernel class (K2 density + force) against the fp64 ALU: algorithmic fp64 operations of the
    # in-range pairs of this band (counted on the perfect lattice of every movable image) / its live time
    roofline_force = None
    if spec.lattice == "bcc_bain":  # (for the disordered variant: the pair counts of the underlying perfect lattice)
        pc = bain_pair_counts(cells[1:P - 1], spec.dims, spec.pot[6], spec.pot[7])
        flop = N * sum(npl * (FLOPS_DENSITY[0] + FLOPS_FORCE[0]) + ntp * (FLOPS_DENSITY[1] + FLOPS_FORCE[1]) for npl, ntp in pc)
        t_force = kms[cf.binding.K_FORCE] * 1e-3
        roofline_force = {"kernel": "K2 density_kernel + force_kernel", "bound": "alu", "achieved": flop / t_force / 1e12,
                          "peak": None, "unit": "TFLOP/s", "frac": None, "algorithmic_flop": flop, "ms": t_force * 1e3,
                          "in_range_pairs_per_atom_mean": float(np.mean([a + b for a, b in pc])),
                          "taper_zone_pairs_per_atom_mean": float(np.mean([b for _, b in pc])),
                          "peak_source": "measured DFMA chain, cfneb_util_fp64_peak (no fp64 figure in MEASURED_PEAKS.json)",
                          "share_of_step": float(kms[cf.binding.K_FORCE] / kms.sum()),
                          "ncu": {"force_kernel": ncu_pipe("c4", "force_kernel"), "density_kernel": ncu_pipe("c4", "density_kernel"),
                                  "note": "committed ncu capture of configs[4] (profiles/r2_ncu_full_c4.txt): share of the fp64 pipe's and "
                                          "of the issue slots' peak; 2 x fp64 + other instructions = 91 % of the scheduler cycles"}}

    if spec.potential == cf.POT_NEP:
        sample = sorted({1, P // 2, P - 2})
        pcs = nep_pair_counts(band, sample, spec.pot[0], spec.pot[1])
        n_rp, n_ap = float(np.mean([a for a, _ in pcs])), float(np.mean([b for _, b in pcs]))
        flop = units_per_step * nep_flops_per_atom(spec.pot, n_rp, n_ap)
        t_force = kms[cf.binding.K_FORCE] * 1e-3
        roofline_force = {"kernel": "K2 nep_radial_desc_kernel + nep_partial_kernel + nep_radial_pair_kernel + pair_force_batched_kernel",
                          "bound": "alu", "achieved": flop / t_force / 1e12, "peak": None, "unit": "TFLOP/s", "frac": None,
                          "algorithmic_flop": flop, "ms": t_force * 1e3,
                          "pairs_inside_rc_r_per_atom_mean": n_rp, "pairs_inside_rc_a_per_atom_mean": n_ap,
                          "pair_count_sample": "images %s, from the band's own lists" % sample,
                          "peak_source": "measured DFMA chain, cfneb_util_fp64_peak (no fp64 figure in MEASURED_PEAKS.json)",
                          "share_of_step": float(kms[cf.binding.K_FORCE] / kms.sum()),
                          "ncu": {kn: ncu_pipe(wl, kn) for kn in ("nep_partial_kernel", "nep_radial_pair_kernel",
                                                                   "nep_radial_desc_kernel", "pair_force_batched_kernel")}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_name(k), "n_atoms": N, "n_images": P, "movable_images": P - 2,
                   "potential": POTENTIAL_NAMES[int(spec.potential)],
                   "cell_filter": "rotation-free B = D D^T (Eq. 17), cell_factor auto", "climb": bool(spec.climb),
                   "value_counts": "N x (P-2) per step", "value_counting_all_images": value * P / (P - 2),
                   "parallelism": "replicas only (x%d)" % world if world > 1 else "single GPU",
                   "l2": "state streamed per step (X, v, F: %.0f MB) exceeds the 126 MB L2; no explicit flush"
                         % (72.0 * N * P / 1e6),
                   "disorder_sigma": float(spec.disorder_sigma),
                   "preroll_steps": preroll,
                   "preroll": "untimed iterations after the warm-up, until the band has rebuilt P - 2 lists (bounded by 150): "
                              "list staleness in steady state before the timed region",
                   "workspace_GB": band.workspace_bytes / 1e9, "neighbor_rebuilds_in_timed_region": int(st1.rebuilds - st0.rebuilds),
                   "window_note": ("no list rebuild fell into the timed region: see steady_state" if st1.rebuilds == st0.rebuilds
                                   else "list rebuilds included"),
                   "max_neighbors_seen": int(st1.max_neighbors_seen)},
        "steady_state": steady,
        "clocks": clocks, "roofline": roofline, "roofline_force": roofline_force, "kernels": kernels,
        "gpu_launches": int(st1.graph_kernel_nodes) * args.steps,
        "status": {"fmax": st1.fmax, "barrier": st1.barrier, "steps": int(st1.steps)},
    }
    return band, line, (pos, cells, spec, barrier, max_over_ranks, world, rank, units_per_step, ranks)


def measure_e2e(band, n_steps, barrier, max_over_ranks, world, units_per_step):
    """Host-buffer loop through the C ABI, a true continuation of the band whose state lives in pinned host memory:
    every step is one cfneb_step_hosted call -- X, v and the FIRE scalars go host -> device (in image blocks on a
    second stream, each block evaluated while the next ones are on their way), the iteration runs, and X, v and
    the scalars come back.  The sequence of states is bit-identical to the device-resident run (GPU test)."""
    import torch
    ck = band.get_checkpoint()

    def pinned(a):
        t = torch.empty(a.shape, dtype=torch.float64, pin_memory=True)
        t.numpy()[...] = a
        return t

    keep = [pinned(ck[k]) for k in ("X", "v")]
    X, v = (t.numpy() for t in keep)
    fire = ck["fire"]

    band.step_hosted(X, v, fire)  # warm-up
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_steps):
        band.step_hosted(X, v, fire)
    barrier()
    dt = max_over_ranks(time.perf_counter() - t0)
    nbytes = 2 * X.size * 8 + 32
    out = {"value": world * units_per_step * n_steps / dt, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
           "steps": n_steps, "ms_per_step": 1e3 * dt / n_steps,
           "what": "per step: cfneb_step_hosted(pinned host X, v, FIRE scalars in; the same out); wall clock; a continuation, "
                   "bit-identical to the resident run; uploads in 10 image blocks overlapped with the force evaluation"}
    # the same loop with the optimizer's state (v, FIRE scalars) resident in the handle: coordinates only, half the bytes
    band.step_hosted(X, None, None)
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_steps):
        band.step_hosted(X, None, None)
    barrier()
    dt = max_over_ranks(time.perf_counter() - t0)
    out["positions_only"] = {"value": world * units_per_step * n_steps / dt, "ms_per_step": 1e3 * dt / n_steps,
                             "h2d_bytes_per_step": X.size * 8, "d2h_bytes_per_step": X.size * 8,
                             "what": "cfneb_step_hosted(X, NULL, NULL): v and the FIRE scalars stay in the handle; same states bit for bit"}
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        return main_reference(args)
    band, line, ctx = main_ours(args)
    pos, cells, spec, barrier, max_over_ranks, world, rank, units_per_step, ranks = ctx
    if not args.no_e2e:
        line["e2e"] = measure_e2e(band, max(1, args.e2e_steps), barrier, max_over_ranks, world, units_per_step)
    try:
        import paper_2510_16721_b200 as cf
        tf = cf.fp64_peak_tflops()
        line["kernels"]["fp64_dfma_peak_tflops_measured"] = tf
        if line.get("roofline_force"):
            line["roofline_force"]["peak"] = tf
            line["roofline_force"]["frac"] = line["roofline_force"]["achieved"] / tf
    except Exception as exc:  # measurement utility only
        line["kernels"]["fp64_dfma_peak_tflops_measured"] = "failed: %s" % exc
    band.close()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r = run_oracle(args.config, steps=2, warmup=0, budget_s=25.0)
        line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                "sample": r["sample"], "host_cores": r["host_cores"], "seconds": r["seconds"]}
    if rank == 0:
        print(json.dumps(line))
    ranks.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
