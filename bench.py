#!/usr/bin/env python
"""bench.py -- TPC tracking throughput on B200 (BASELINE.json metric: clusters/s and Time Frames/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

One "step" = one pass of the whole hot path (tpc_grid_build -> tpc_find_tracks -> tpc_fit_tracks, SURVEY.md
§8(a) rows a1..a6) over one synthetic event.  The default workload is BASELINE.json configs[4]: one 128-orbit
50 kHz min-bias Pb-Pb Time Frame (~1.4e8 clusters, seeded synthetic).

 value        clusters/s with the clusters resident in HBM (CUDA events around K steps, no per-kernel events inside;
              max over ranks)
 e2e          same metric through tpc_track_host_async / tpc_track_host_fetch: pinned host buffers, H2D of the inputs
              and D2H of EVERY output inside the timed region, four Time Frames in flight
 kernels      per-kernel CUDA-event times from a second, separately profiled loop (tpc_profile_*)
 roofline     the dominant kernel of that table; the FP32 roof is measured by the library (tpc_fp32_peak, FFMA chains),
              the HBM roof is MEASURED_PEAKS.json; `traffic` comes from profiles/*_ncu_traffic.csv and is null when
              csrc/ has changed since that capture
 cpu_baseline the CPU oracle, as it stands: the whole Time Frame with its sectors dealt to all host cores, and one
              thread on a slab of one sector beside it (rank 0, N = 1 only)
 --impl reference : times the oracle alone on the host cores (this tier's reference arm)
 --ncu-traffic RAW.csv --out profiles/NAME.csv : turn `ncu -i REP --page raw --csv` output into the stamped
              per-kernel DRAM traffic table `roofline.traffic` reads (no GPU needed)

N > 1 (torchrun): every rank tracks its OWN Time Frame (TF-level replicas: GPUs process
independent TFs); no data-path collective; "scaling": "weak".
"""
from __future__ import annotations

import argparse
import csv
import glob
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "tpc_clusters_tracked_per_s"
UNIT = "clusters/s"
L2_BYTES = 126e6

# Algorithmic HBM bytes per unit and fp32 operations per unit of every kernel (DESIGN.md "Kernels and
# rooflines").  unit: "cluster" = per input cluster, "bin" = per grid bin,
# "step" = per follower row step (propagate + search + update), "hit" = per refitted hit.
KERNEL_MODEL = {
    # name: (bound, {unit: algorithmic HBM bytes per unit}, unit the alu-bound kernels are counted in)
    # units: cluster = input cluster, bin = grid bin, tracklet = followed start hit, claim = (tracklet,row) hit
    # recorded by the follower, hit = hit of an accepted track
    "k_bucket_hist": ("hbm", {"cluster": 12}, None),                # y, z, sector_row in
    "k_scan_*": ("hbm", {"cluster": 12, "tracklet": 24}, None),     # all scans of a step: 2 reads + 1 write per element
    "k_part_scatter": ("hbm", {"cluster": 12 + 16}, None),          # inputs in, 16 B record out (part order)
    "k_bucket_scatter": ("hbm", {"cluster": 16 + 16}, None),        # record in, record out (bucket order)
    "k_bucket_sort": ("hbm", {"cluster": 16 + 16, "bin": 4}, None), # records in (second read from L2), records + bin_first out
    "k_neighbours": ("hbm", {"cluster": 16 + 8}, None),           # own record in, two links out (neighbours from L2)
    "k_clean": ("hbm", {"cluster": 8 + 8}, None),
    "k_compact_starts": ("hbm", {"cluster": 4, "tracklet": 32}, None),
    "k_follow": ("alu", {}, "step"),                              # two waves of phase A + phase B (three launches per step)
    "k_survivor_*": ("hbm", {"tracklet": 32 + 4 + 3 * (32 + 1 + 4 + 12 + 4)}, None),   # wave test + three list builds
    "k_push_keys": ("hbm", {"claim": 4 + 8 + 8, "tracklet": 12}, None),   # row_hit in, 8-byte atomicMax RMW
    "k_count_kept": ("hbm", {"claim": 4 + 8, "tracklet": 12 + 20 + 8}, None),   # row_hit, owner in; mask, value out
    "k_write_tracks": ("hbm", {"hit": 4 + 16 + 4 + 16 + 8, "tracklet": 16 + 20}, None),  # row_hit, rec in; trk_hits, hit_rec, (orig, track) pair out
    "k_assign": ("hbm", {"hit": 8 + 4}, None),                    # pair in, cluster_track out
    "k_fit": ("alu", {}, "hit"),
}


# ------------------------------------------------------------------------------------------------
# roofline.traffic: ncu DRAM bytes per kernel, from a tracked capture stamped with the csrc/ it was taken on
# ------------------------------------------------------------------------------------------------
CSRC = os.path.join(ROOT, "paper_2106_03636_b200", "csrc")


def csrc_digest() -> str:
    """sha256 over the CUDA sources (names and contents): identifies the build a capture belongs to."""
    h = hashlib.sha256()
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            with open(os.path.join(CSRC, f), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()


KERNEL_GROUPS = (("k_follow", "k_follow"), ("k_fit_seed", "k_fit"), ("k_fit_gather", "k_fit"), ("k_scan", "k_scan_*"), ("k_wave_test", "k_survivor_*"),
                 ("k_list_", "k_survivor_*"), ("k_chunk_counts", "k_compact_starts"), ("k_clear_start_bits", "k_compact_starts"),
                 ("k_fit_physics", "k_fit_physics+k_tag_*"), ("k_tag_", "k_fit_physics+k_tag_*"), ("k_merge_", "k_merge_*"),
                 ("k_digit_", "k_digit_*"), ("k_cluster_count", "k_digit_*"))


def bench_kernel_name(ncu_name: str) -> str:
    """Name of the bench table row a kernel of the ncu launch list belongs to."""
    base = ncu_name.split("(")[0].split("::")[-1].split("<")[0].strip().split(" ")[-1]     # drops "void", namespaces, template arguments
    if base == "k_fit":
        return "k_fit"
    for prefix, row in KERNEL_GROUPS:
        if base.startswith(prefix):
            return row
    return base


def write_ncu_traffic(raw_csv: str, out_csv: str, config: int, steps_captured: int):
    """profiles/*_ncu_traffic.csv from `ncu -i REP --page raw --csv`: DRAM read + write bytes per bench kernel row,
    summed over its launches and divided by the number of steps captured."""
    with open(raw_csv) as f:
        rows = list(csv.reader(f))
    hdr, units = rows[0], rows[1]
    ik, ir, iw = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    tot = {}
    for r in rows[2:]:
        if len(r) <= max(ik, ir, iw):
            continue
        name = bench_kernel_name(r[ik])
        by = float(r[ir].replace(",", "")) * scale[units[ir]] + float(r[iw].replace(",", "")) * scale[units[iw]]
        a = tot.setdefault(name, [0.0, 0])
        a[0] += by
        a[1] += 1
    with open(out_csv, "w") as f:
        f.write(f"# csrc_sha256: {csrc_digest()}\n# config: {config}\n# steps_captured: {steps_captured}\n")
        f.write("kernel,dram_bytes_per_step,launches_per_step\n")
        for k in sorted(tot):
            f.write(f"{k},{tot[k][0] / steps_captured:.0f},{tot[k][1] / steps_captured:g}\n")
    print(f"wrote {out_csv}: {len(tot)} kernels, csrc {csrc_digest()[:12]}")


def load_ncu_traffic(config: int):
    """({kernel: DRAM bytes per step}, source) of the newest tracked capture taken on exactly these csrc/ sources and
    this config; ({}, reason) otherwise -- a capture of another build says nothing about this one."""
    want = csrc_digest()
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_ncu_traffic.csv")), reverse=True):
        meta, table = {}, {}
        with open(path) as f:
            for ln in f:
                if ln.startswith("#"):
                    k, _, v = ln[1:].partition(":")
                    meta[k.strip()] = v.strip()
                elif ln.strip() and not ln.startswith("kernel,"):
                    k, by, _ = ln.strip().split(",")
                    table[k] = float(by)
        if meta.get("csrc_sha256") == want and int(meta.get("config", -1)) == config:
            return table, os.path.relpath(path, ROOT) + " (ncu dram__bytes_read.sum + dram__bytes_write.sum)"
    return {}, "no ncu capture of this build and config under profiles/ (csrc/ changed since the last one)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (default 4: one Time Frame)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--ncu-traffic", default=None, help="raw csv of `ncu -i REP --page raw --csv` to convert (no GPU needed)")
    ap.add_argument("--out", default=None, help="with --ncu-traffic: the profiles/*_ncu_traffic.csv to write")
    ap.add_argument("--steps-captured", type=int, default=1, help="with --ncu-traffic: steps the capture covers")
    return ap.parse_args()


def make_event(cfg: int, rank: int, world: int):
    from paper_2106_03636_b200.synth import make_config
    kw = {}
    if cfg >= 2:
        kw["workers"] = max(1, min(32, (os.cpu_count() or 1) // max(world, 1)))
    seed = cfg + 1 + 100 * rank            # A7: seed = config index + 1; other ranks get their own Time Frame
    return make_config(cfg, seed=seed, **kw)


def workload_name(cfg: int) -> str:
    return {0: "configs[0]: tiny single sector, 200 helices",
            1: "configs[1]: one central Pb-Pb collision, full TPC",
            2: "configs[2]: pp-like continuous slice, 200 collisions over 1 ms",
            3: "configs[3]: pileup stress, 5 central Pb-Pb + loopers + 20% noise",
            4: "configs[4]: one 128-orbit 50 kHz min-bias Pb-Pb Time Frame"}[cfg]


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks DURING the timed region")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._pump, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for r in self.rows if t0 <= r[0] <= t1] or self.rows[-3:]
        for _, line in rows:
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1])
                for nm, v in zip(names, f[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
                power.append(float(f[6]))
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power) if power else None}


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference): bounded sample of the same workload
# ------------------------------------------------------------------------------------------------
def oracle_sample(ev, max_clusters: int):
    """Clusters of sector 0 (sectors are independent through the whole hot path), cut to the lowest-zeta slab
    holding <= max_clusters clusters.  Returns (y, z, sector_row, description)."""
    nrows = int(ev.params.n_rows)
    sel = np.nonzero(ev.sector_row < nrows)[0]
    desc = f"sector 0 of {ev.params.n_sectors}"
    if sel.size > max_clusters:
        zs = ev.z[sel]
        cut = np.partition(zs, max_clusters)[max_clusters]
        sel = sel[zs < cut]
        desc += f", z < {float(cut):.1f} cm slab"
    return ev.y[sel].copy(), ev.z[sel].copy(), ev.sector_row[sel].copy(), f"{desc}: {sel.size} clusters"


def time_oracle(ev, y, z, sr, steps: int, warmup: int):
    from oracle import tpc_oracle as orc
    orc.build()
    p1 = ev.params.with_(n_sectors=1) if int(ev.params.n_sectors) > 1 else ev.params
    times, ntr = [], 0
    for i in range(warmup + steps):
        tm = {}
        t0 = time.perf_counter()
        o = orc.run(p1, y, z, sr, "f32", True, timings=tm)
        dt = time.perf_counter() - t0
        ntr = int(o["trk_seed"].size)
        if i >= warmup:
            times.append(dt)
    return float(np.mean(times)), ntr


_POOL_EV = None


def _oracle_sector(sector: int):
    """Worker of time_oracle_all_cores: the whole hot path of one sector, single-threaded (the oracle as it stands)."""
    from oracle import tpc_oracle as orc
    ev = _POOL_EV
    nrows = int(ev.params.n_rows)
    sel = np.nonzero(ev.sector_row // nrows == sector)[0]
    p1 = ev.params
    t0 = time.perf_counter()
    o = orc.run(p1, ev.y[sel], ev.z[sel], ev.sector_row[sel], "f32", True)
    return sector, int(sel.size), int(o["trk_seed"].size), int((o["cluster_track"] >= 0).sum()), time.perf_counter() - t0


def time_oracle_all_cores(ev, cores: int | None = None):
    """BASELINE.md §2 leg (ii): the whole event with its sectors dealt to all host cores (sectors are independent
    through the whole hot path; the oracle stays single-threaded per sector).  Returns a dict for cpu_baseline."""
    import multiprocessing as mp
    global _POOL_EV
    from oracle import tpc_oracle as orc
    orc.build()
    nsec = int(ev.params.n_sectors)
    cores = max(1, min(cores or (os.cpu_count() or 1), nsec))
    nrows = int(ev.params.n_rows)
    sizes = np.bincount(ev.sector_row // nrows, minlength=nsec)
    order = [int(s) for s in np.argsort(-sizes)]          # largest first: the pool deals them as workers free up
    _POOL_EV = ev
    t0 = time.perf_counter()
    with mp.get_context("fork").Pool(cores) as pool:      # fork: the workers see the event without a copy
        res = pool.map(_oracle_sector, order, chunksize=1)
    wall = time.perf_counter() - t0
    _POOL_EV = None
    return {"value": ev.n / wall, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"whole event: {ev.n} clusters, {nsec} sectors dealt to {cores} processes (one oracle thread each)",
            "seconds": wall, "cpu_seconds": float(sum(r[4] for r in res)), "tracks_found": int(sum(r[2] for r in res)),
            "clusters_assigned": int(sum(r[3] for r in res)), "host_cores_available": os.cpu_count()}


def run_reference(args, rank: int):
    """This tier's reference arm: the CPU oracle, as it stands, on a bounded sample per step."""
    if rank != 0:
        return
    ev = make_event(args.config, 0, 1)
    per_step_s = min(12.0, 200.0 / max(args.steps + args.warmup, 1))
    y, z, sr, desc = oracle_sample(ev, int(per_step_s * 1.2e5))
    dt, ntr = time_oracle(ev, y, z, sr, args.steps, args.warmup)
    val = y.size / dt
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": workload_name(args.config), "n_clusters": int(y.size), "sample": desc},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "tracks_found": ntr}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def reduce_over_ranks(ms_step: float, t_e2e: float, n_clusters: int, world: int, device):
    """TF-level replicas: the job's step time is the MAX over ranks, its work the SUM of the ranks'
    clusters.  The only collectives of a multi-GPU run; `device` is the tensor device of the process group's
    backend (cuda for nccl, cpu for the gloo test in tests/test_multirank_gloo.py)."""
    if world <= 1:
        return ms_step, t_e2e, float(n_clusters)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_step, t_e2e], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([float(n_clusters)], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(c[0])


def run_ours(args, rank: int, local_rank: int, world: int):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU implementation")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=dev)
    from paper_2106_03636_b200 import binding

    t_gen = time.perf_counter()
    ev = make_event(args.config, rank, world)
    t_gen = time.perf_counter() - t_gen
    n = ev.n
    hy, hz, hs = (torch.from_numpy(a).pin_memory() for a in (ev.y, ev.z, ev.sector_row))
    y, z, sr = (a.to(dev, non_blocking=True) for a in (hy, hz, hs))
    trk = binding.Tracker(ev.params, n, device=dev)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()

    for _ in range(max(args.warmup, 3)):
        trk.step(y, z, sr)
    torch.cuda.synchronize()
    cnt = trk.counters.cpu().numpy()
    if int(cnt[binding.CNT_STATUS]) & (binding.ST_TRACKLET_OVERFLOW | binding.ST_TRACK_OVERFLOW):
        raise RuntimeError(f"capacity overflow, status bits {int(cnt[binding.CNT_STATUS])}: the run would skip work")

    # ---- timed region: K steps, inputs resident in HBM, CUDA events on the launching stream, no per-kernel events ----
    binding.profile_enable(False)
    binding.profile_collect(reset=True)
    sampler = ClockSampler(local_rank)
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    w0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        trk.step(y, z, sr)
    e1.record()
    torch.cuda.synchronize(); barrier()
    w1 = time.perf_counter()
    clocks = sampler.stop(w0, w1)
    ms_total = e0.elapsed_time(e1)
    launches = int(sum(v[1] for v in binding.profile_collect(reset=True).values()))   # counted always, timed only below
    res = trk.results()
    K_tracks = int(res["trk_seed"].size)
    n_tracklets = int(res["counters"][binding.CNT_TRACKLETS])
    n_hits = int(res["counters"][binding.CNT_HITS])

    # ---- per-kernel table: a second loop with an event pair around every launch ---------------------
    binding.profile_enable(True)
    prof_steps = min(args.steps, 150)          # the library keeps at most 8192 timed launches between collects
    for _ in range(prof_steps):
        trk.step(y, z, sr)
    torch.cuda.synchronize()
    prof = binding.profile_collect(reset=True)
    binding.profile_enable(False)
    fp32_peak = binding.fp32_peak(dev)

    # ---- after the hot path (not part of `value`): tpc_merge_tracks (R26) on the tracks of the last step ----------
    merge = None
    if int(ev.params.n_sectors) > 1:
        trk.merge_enqueue()
        torch.cuda.synchronize()
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        m0.record()
        for _ in range(3):
            trk.merge_enqueue()
        m1.record()
        torch.cuda.synchronize()
        ng = trk._merge["out"]["n_global"].cpu().numpy()
        if int(ng[3]) != 0:
            raise RuntimeError(f"tpc_merge_tracks left {int(ng[3])} candidate pairs untested (pair list full): the merge figure is void")
        merge = {"ms": m0.elapsed_time(m1) / 3, "global_tracks": int(ng[0]), "links": int(ng[1]), "pairs": int(ng[2]), "pairs_dropped": int(ng[3]),
                 "what": "tpc_merge_tracks: sector-local tracks linked across sector edges / the central electrode / long "
                         "holes, merged hit lists refitted (DESIGN.md R26); not included in `value`"}
        binding.profile_collect(reset=True)

    # ---- after the hot path: the refit with every R28 option on + the cluster tags a compression step would use --------
    physics = None
    if int(ev.params.n_sectors) > 1:
        from paper_2106_03636_b200.synth import V_DRIFT
        trk.track_time(V_DRIFT)                              # R24: the time offsets the drift lengths of R28e come from
        popt = dict(x0inv=2e-4, outlier_cut=12.0, dedx=2e-6, eloss_sigma=0.3, err_ang_y=1.5, err_ang_z=0.8, err_drift_y=2e-4,
                    err_drift_z=3e-4, v_drift=V_DRIFT, z_len=250.0)

        def physics_step():
            trk.fit_tracks_physics(trk_t0=trk.trk_t0, want_numpy=False, **popt)
            return trk.tag_clusters(qpt_max=4.0, use_physics_fit=True, want_numpy=False)

        physics_step()
        torch.cuda.synchronize()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record()
        for _ in range(3):
            tag = physics_step()
        p1.record()
        torch.cuda.synchronize()
        physics = {"ms": p0.elapsed_time(p1) / 3, "options": popt,
                   "hits_rejected": int(trk._physics["hit_flag"][:n_hits].sum().item()),
                   "clusters_tagged_for_removal": int(((tag[:n] & 2) != 0).sum().item()),
                   "what": "tpc_fit_tracks_physics (scattering noise, energy loss, angle- and drift-dependent cluster errors, "
                           "outlier rejection; DESIGN.md R28a-e) + tpc_tag_clusters; not included in `value`"}
        del tag
        binding.profile_collect(reset=True)

    # ---- in front of the hot path (not part of `value`): tpc_clusterize (R27) on the digits of a slab of the event ---
    cluster = None
    if world == 1 and not args.no_cpu_baseline:
        from types import SimpleNamespace
        from paper_2106_03636_b200.synth import digitize
        ys, zs, ss, desc = oracle_sample(ev, 1_000_000)
        qs = np.full(ys.size, 50.0, np.float32)
        d = digitize(SimpleNamespace(params=ev.params, y=ys, z=zs, q=qs, sector_row=ss))
        dd = [torch.from_numpy(a).to(dev) for a in (d.sector_row, d.pad, d.time, d.adc)]
        binding.clusterize(ev.params, *dd, d.pad_width, d.time_width)                   # warm-up
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(3):
            r = binding.clusterize(ev.params, *dd, d.pad_width, d.time_width, want_numpy=False)
        c1.record()
        torch.cuda.synchronize()
        ms = c0.elapsed_time(c1) / 3
        cluster = {"ms": ms, "digits": d.n, "clusters": int(r["n_clusters"][0].item()), "digits_per_s": d.n / (ms * 1e-3),
                   "sample": desc, "what": "tpc_clusterize on synthetic digits of that slab (DESIGN.md R27; hash-table build + "
                                           "peak finding + centre of gravity; includes the table memsets); not included in `value`"}
        del dd, r
        binding.profile_collect(reset=True)

    # ---- end to end through the host-buffer entry points -----------------------------------------
    # Two Time Frames in flight (two Tracker contexts, own workspace / staging / pinned outputs, one stream each):
    # the H2D copy of one TF overlaps the tracking of the previous one and the D2H of the one before -- the
    # steady state of a continuous TF stream.  Every step copies its inputs from pinned host
    # memory and reads EVERY output back (counters and cluster_track with the step; the per-track arrays and the hit
    # lists, whose sizes the host only knows from the counters, by tpc_track_host_fetch once those have arrived).
    t_e2e, h2d, d2h = 0.0, 0, 0
    NC = 4     # Time Frames in flight: a stream's H2D + tracking + D2H chain is ~2.5x the step time (measured: 46 / 36 /
               # 34.7 ms per Time Frame with 2 / 3 / 4 in flight)
    if not args.no_e2e:
        ctx = [trk] + [binding.Tracker(ev.params, n, device=dev) for _ in range(NC - 1)]
        streams = [torch.cuda.Stream(device=dev) for _ in range(NC)]
        events = [torch.cuda.Event() for _ in range(NC)]
        for c, st in zip(ctx, streams):
            c.make_host_staging()
            with torch.cuda.stream(st):
                h2d, d2h = c.track_host(hy, hz, hs)      # warm-up (first touch of the staging buffers), synchronous
        barrier(); torch.cuda.synchronize()

        def fetch(j):                                    # TF j: wait for its counters, then enqueue the exact-size copies
            events[j % NC].synchronize()
            with torch.cuda.stream(streams[j % NC]):
                ctx[j % NC].track_host_fetch()

        def enqueue(i):
            with torch.cuda.stream(streams[i % NC]):
                ctx[i % NC].track_host_async(hy, hz, hs)
                events[i % NC].record()

        # steady state of a continuous stream of Time Frames: the pipeline is primed with NC - 1 Time Frames and run for NC
        # untimed iterations, then the clock covers K iterations, each enqueueing one new Time Frame and delivering (fetching) one; it stops when the
        # K-th result has arrived on the host; the NC - 1 Time Frames still in flight drain untimed
        for i in range(NC - 1):
            enqueue(i)
        W = NC                                           # untimed iterations until the pipeline is in steady state
        for i in range(NC - 1, NC - 1 + W):
            enqueue(i)
            fetch(i - (NC - 1))
        t0 = time.perf_counter()
        for i in range(NC - 1 + W, NC - 1 + W + args.steps):
            enqueue(i)
            fetch(i - (NC - 1))
        last = W + args.steps - 1                        # the K-th Time Frame delivered inside the timed region
        streams[last % NC].synchronize()                 # nothing later was enqueued on that stream
        t_e2e = (time.perf_counter() - t0) / args.steps
        for j in range(last + 1, last + NC):
            fetch(j)
        for st in streams:
            st.synchronize()
        for c in ctx:
            hr = c.host_results()
            assert hr["trk_seed"].size == K_tracks and int(hr["trk_nhits"].sum()) == n_hits
            assert np.array_equal(hr["par"], res["par"]) and np.array_equal(hr["trk_hits"], res["trk_hits"])
        del ctx

    # ---- max over ranks ----------------------------------------------------------------------------
    ms_step, t_e2e, tot_clusters = reduce_over_ranks(ms_total / args.steps, t_e2e, n, world, dev)
    if rank != 0:
        return

    hbm_peak, sm_max_mhz, peak_src = load_peaks()
    value = tot_clusters / (ms_step * 1e-3)
    # ---- per-kernel table and roofline of the dominant kernel -----------------------------------
    # A row sums all launches of that kernel in a step (k_follow: two waves of phase A + phase B; k_fit: seeds + fit;
    # scans, list builds); its algorithmic bytes / flops (KERNEL_MODEL) cover the same launches.
    kern = {k: {"ms_per_step": v[0] / prof_steps, "launches_per_step": v[1] / prof_steps}
            for k, v in prof.items() if v[1] > 0}
    top = max(kern, key=lambda k: kern[k]["ms_per_step"])
    nb = binding.grid_bins(ev.params)
    work = binding.work_counts(res["counters"])
    units = {"cluster": n, "bin": nb, "tracklet": int(res["counters"][binding.CNT_TRACKLETS]), "claim": work["claims"],
             "hit": n_hits}
    peaks = {"hbm": hbm_peak, "hbm_source": peak_src, "fp32": fp32_peak, "sm_max_mhz": sm_max_mhz}
    traffic, traffic_src = load_ncu_traffic(args.config)
    roofline = kernel_roofline(top, kern[top]["ms_per_step"], units, work, int(ev.params.n_fit_passes), peaks)
    roofline["launches_per_step"] = kern[top]["launches_per_step"]
    roofline["traffic"] = traffic.get(top)
    roofline["traffic_source"] = traffic_src
    for k in kern:       # every kernel's own fraction of its roof, so that the table can be read without DESIGN.md
        r = kernel_roofline(k, kern[k]["ms_per_step"], units, work, int(ev.params.n_fit_passes), peaks)
        kern[k]["bound"], kern[k]["frac"] = r["bound"], round(r["frac"], 4)
        if k in traffic:
            kern[k]["ncu_dram_gb"] = round(traffic[k] / 1e9, 3)
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
           "data": "synthetic",
           "config": {"workload": workload_name(args.config), "n_clusters": n, "n_bins": nb,
                      "time_frames_per_step_per_gpu": 1 if args.config == 4 else None,
                      "l2": f"inputs ({12 * n / 1e6:.0f} MB/step) and workspace exceed the 126 MB L2; no explicit flush",
                      "parallelism": f"tf-replicas x{world}", "gen_seconds": round(t_gen, 1)},
           "time_frames_per_s": (world / (ms_step * 1e-3)) if args.config == 4 else None,
           "tracks_found": K_tracks, "tracklets_followed": n_tracklets,
           "tracklets_followed_down": int(res["counters"][binding.CNT_FOLLOWED_DOWN]), "clusters_assigned": n_hits,
           "follower_work": work,
           "clocks": clocks, "gpu_launches": launches, "gpu_launches_per_step": launches / args.steps, "kernels": kern,
           "kernels_ms_sum": round(sum(v["ms_per_step"] for v in kern.values()), 3), "roofline": roofline,
           "after_hot_path": {"merge": merge, "physics_refit_and_tags": physics}, "before_hot_path": {"clusterizer": cluster}}
    if not args.no_e2e:
        out["e2e"] = {"value": tot_clusters / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d) * world,
                      "d2h_bytes_per_step": int(d2h) * world, "ms_per_step": t_e2e * 1e3,
                      "bound": "pcie" if t_e2e * 1e3 > 1.1 * ms_step else "gpu (the tracking itself: copies hidden behind it)",
                      "h2d_gb_per_s": int(h2d) / t_e2e / 1e9, "d2h_gb_per_s": int(d2h) / t_e2e / 1e9,
                      "returns": "every output of tpc_find_tracks + tpc_fit_tracks: counters, cluster_track, trk_seed / sector / "
                                 "nhits / first_hit, trk_hits, par, cov, xref, zref, chi2, ndf (exactly K tracks and H hits)",
                      "pipeline": f"tpc_track_host_async + tpc_track_host_fetch, {NC} Time Frames in flight on {NC} streams (own "
                                  "workspace, staging and pinned outputs each), primed; wall clock over K iterations (one Time Frame enqueued, one "
                                  "delivered to the host each) until the K-th result has arrived"}
    if world == 1 and not args.no_cpu_baseline:
        ys, zs, ss, desc = oracle_sample(ev, 1_500_000)
        dt, ntr = time_oracle(ev, ys, zs, ss, 1, 0)
        one = {"value": ys.size / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": dt}
        if int(ev.params.n_sectors) > 1:
            out["cpu_baseline"] = time_oracle_all_cores(ev)
            out["cpu_baseline"]["one_core"] = one
            out["cpu_baseline"]["same_tracks_as_gpu"] = bool(out["cpu_baseline"]["tracks_found"] == K_tracks and
                                                            out["cpu_baseline"]["clusters_assigned"] == n_hits)
        else:
            out["cpu_baseline"] = dict(one, host_cores_available=os.cpu_count())
    print(json.dumps(out), flush=True)


def kernel_roofline(name, ms, units, work, n_passes, peaks):
    """Roofline entry of one row of the kernel table.  ms = summed time of the row's launches in one step;
    units: {"cluster": N, "bin": B, "tracklet": S, "claim": follower updates, "hit": hits of accepted tracks};
    peaks: {"hbm": GB/s (MEASURED_PEAKS.json), "fp32": TFLOP/s measured by tpc_fp32_peak, ...}."""
    bound, per_unit, unit = KERNEL_MODEL.get(name, ("hbm", {}, None))
    if bound == "hbm":
        by = sum(b * units[u] for u, b in per_unit.items())
        ach = by / (ms * 1e-3) / 1e9
        return {"kernel": name, "bound": "hbm", "achieved": ach, "peak": peaks["hbm"], "unit": "GB/s", "frac": ach / peaks["hbm"],
                "traffic": None, "algorithmic_bytes_per_step": by, "ms_per_step": ms, "peak_source": peaks["hbm_source"]}
    # alu-bound kernels: fp32 operations the method requires per unit (a fused multiply-add counts 2)
    from paper_2106_03636_b200 import flops
    if name == "k_follow":
        n_units, fl = work["propagations"], flops.follow_flop(work)
    else:
        n_units, fl = units["hit"] * n_passes, flops.fit_flop(units["hit"], n_passes)
    nominal = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    ach = fl / (ms * 1e-3) / 1e12
    # SURVEY.md 8(d) asks for both views of the per-track kernels: the follower gathers ~100 bytes of 32-byte sectors
    # per transport when nothing hits L2 (two bin-offset sectors, one or two cluster records, its row_hit entry); the
    # refit streams 16 bytes per hit and pass
    gather = (work["propagations"] * 100) if name == "k_follow" else (units["hit"] * n_passes * 16)
    hbm_view = {"bound": "hbm", "algorithmic_bytes_per_step": gather, "achieved": gather / (ms * 1e-3) / 1e9,
                "peak": peaks["hbm"], "unit": "GB/s", "frac": gather / (ms * 1e-3) / 1e9 / peaks["hbm"]}
    return {"kernel": name, "bound": "alu", "achieved": ach, "peak": peaks["fp32"], "unit": "TFLOP/s", "frac": ach / peaks["fp32"],
            "traffic": None, "algorithmic_flop_per_step": fl, "units": n_units, "unit_kind": unit, "ms_per_step": ms,
            "peak_nominal": nominal, "frac_of_nominal": ach / nominal, "hbm_view": hbm_view,
            "peak_source": "measured in this run by tpc_fp32_peak (FFMA chains, 8 per thread); peak_nominal = 148 SMs x 128 "
                           f"lanes x 2 x {peaks['sm_max_mhz']:.0f} MHz"}


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.ncu_traffic:
        write_ncu_traffic(args.ncu_traffic, args.out or os.path.join(ROOT, "profiles", "ncu_traffic.csv"), args.config,
                          args.steps_captured)
        return
    if args.impl == "reference":
        run_reference(args, rank)
        return
    run_ours(args, rank, local_rank, world)
    if world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
