#!/usr/bin/env python
"""bench.py — HEALPix forward+backward rasterisation throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

One "step" = one pass of the whole hot path (preprocess -> tile query -> sort -> ranges -> blend forward -> blend
backward -> preprocess backward) over one seeded synthetic scene.  Default workload: BASELINE.json config 4
("large_sphere": Nside 1024, 12.58 M px, 2 M Gaussians, SH degree 3), the configuration the metric is quoted on.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_29794_b200 import scenes  # noqa: E402  (input generator: no method arithmetic)

METRIC = "healpix_px_per_s_fwd_bwd"
UNIT = "px/s"
# default: Alg.1 l.9-16 through uts_tile_lists (one call); --lists staged times uts_tile_query / uts_sort / uts_tile_ranges one by one
STAGES_FUSED = ["preprocess", "depth_order", "tile_lists", "render_fwd", "render_bwd", "preprocess_bwd"]
STAGES_STAGED = ["preprocess", "depth_order", "tile_query", "sort", "tile_ranges", "render_fwd", "render_bwd", "preprocess_bwd"]
# FP32 operations of the blend kernels per (Gaussian, pixel) pair (counted from the arithmetic of Eq.6 +
# SphericalOffset as implemented, FMA = 2): an EVALUATED pair costs 41 (forward) / 46 (backward: the same evaluation + the reach
# test and exp kept for the gradient), a CONTRIBUTING pair another 9 (forward: blend) / 72 (backward: gradient chain + its share
# of the warp reduction).
FLOP_FWD_EVAL, FLOP_FWD_CONTRIB, FLOP_BWD_EVAL, FLOP_BWD_CONTRIB = 41, 9, 46, 72
# the ONE bounded oracle sample both arms time (--impl reference, and the cpu_baseline leg of the default arm)
ORACLE_SAMPLE = dict(n_pre=500_000, n_query=60_000, n_tiles_sample=192)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set(); self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=reasons, samples=len(sm))


# ----------------------------------------------------------------------------------------------- reference arm
class OracleSample:
    """The oracle, as it stands, on a BOUNDED sample of the workload.  Set-up (scene, full preprocess, choice of the sampled
    tiles and their candidate Gaussians) happens once, untimed; step() times the oracle stages and extrapolates per stage:

    per-Gaussian stages (preprocess, preprocess backward) : first n_pre Gaussians, scaled by P/n_pre
    tile query + sort + ranges                           : first n_query Gaussians on every tile, scaled by P/n_query
    blend forward + backward                             : n_tiles_sample random tiles with their COMPLETE lists (all P
                                                           Gaussians pre-filtered by a conservative angular test, the oracle's
                                                           own query decides), scaled by active tiles / sampled tiles
    """

    def __init__(self, cfg_id, seed=0, n_pre=100_000, n_query=10_000, n_tiles_sample=24):
        import oracle as orc
        self.orc, self.cfg_id = orc, cfg_id
        sc = self.sc = scenes.make_scene(cfg_id, seed=seed)
        P, V = sc["n_gauss"], sc["n_views"]
        oc = self.oc = orc.Config(order=sc["order"], n_gauss=P, n_views=V, sh_degree=sc["sh_degree"])
        self.bits = self.act = self.slot = None
        if sc["mask"] is not None:
            self.bits = orc.mask_bits(oc.order, sc["mask"]["kind"], sc["mask"]["params"]); self.act, self.slot = orc.mask_tiles(oc, self.bits)
        self.n_active = oc.n_tiles if self.act is None else int(self.act.shape[0])
        self.n_pre, self.n_query = min(n_pre, P), min(n_query, P)
        self.n_pix = V * self.n_active * oc.ppt
        pr = self.pr = orc.preprocess(oc, sc["means"], sc["scales"], sc["quats"], sc["opac"], sc["sh"], sc["W"], sc["b"])
        rng = np.random.default_rng(seed + 17)
        pool = np.arange(oc.n_tiles) if self.act is None else self.act.astype(np.int64)
        pick = self.pick = np.sort(rng.choice(pool, min(n_tiles_sample, pool.shape[0]), replace=False))
        self.sact = pick.astype(np.uint32)
        self.sslot = np.full(oc.n_tiles, -1, np.int32); self.sslot[pick] = np.arange(pick.shape[0], dtype=np.int32)
        _, _, tc = orc.centers(oc.tile_order, which=2)
        reach = pr.rs.astype(np.float64) + orc.rho_max_closed(oc.tile_order + oc.query_refine_log2) + orc.rho_max_closed(oc.tile_order) + 1e-6
        cand = np.zeros(P, bool)
        for v in range(V):
            for g0 in range(0, P, 262144):                 # chunked: the (Gaussian x sampled tile) table stays small
                g1 = min(P, g0 + 262144)
                d = pr.dir[v][g0:g1].astype(np.float64) @ tc[pick].T
                cand[g0:g1] |= (np.arccos(np.clip(d, -1, 1)) <= reach[v][g0:g1, None]).any(axis=1)
        self.cand_ids = np.flatnonzero(cand).astype(np.int32)
        self.gcol = scenes.upstream_grad(V, pick.shape[0] * oc.ppt, seed=seed)
        _, keys, vals, _ = orc.tile_query(oc, pr, self.sslot, gauss_subset=self.cand_ids)          # complete lists of the sampled tiles
        self.sk, self.sv = orc.sort_pairs(keys, vals)
        self.rg = orc.tile_ranges(oc, self.sk)

    def _sub(self, n):
        sc = self.sc
        return {k: (sc[k][:n] if k in ("means", "scales", "quats", "opac", "sh") else sc[k]) for k in sc}

    def step(self):
        orc, oc, sc = self.orc, self.oc, self.sc
        P, V = oc.n_gauss, oc.n_views
        s1 = self._sub(self.n_pre); c1 = orc.Config(order=oc.order, n_gauss=self.n_pre, n_views=V, sh_degree=oc.sh_degree)
        z3 = np.ones((V, self.n_pre, 3)); z2 = np.ones((V, self.n_pre, 2))
        t = time.perf_counter()
        orc.preprocess(c1, s1["means"], s1["scales"], s1["quats"], s1["opac"], s1["sh"], s1["W"], s1["b"])
        orc.preprocess_bwd(c1, s1["means"], s1["scales"], s1["quats"], s1["sh"], s1["W"], s1["b"], z3, z3, z2)
        t_pre = (time.perf_counter() - t) * (P / self.n_pre)

        s2 = self._sub(self.n_query); c2 = orc.Config(order=oc.order, n_gauss=self.n_query, n_views=V, sh_degree=oc.sh_degree)
        pr2 = orc.preprocess(c2, s2["means"], s2["scales"], s2["quats"], s2["opac"], s2["sh"], s2["W"], s2["b"])
        t = time.perf_counter()
        _, keys, vals, _ = orc.tile_query(c2, pr2, self.slot)
        sk, sv = orc.sort_pairs(keys, vals)
        orc.tile_ranges(c2, sk)
        t_qs = (time.perf_counter() - t) * (P / self.n_query)
        pairs_est = keys.shape[0] * (P / self.n_query)

        sk, sv, rg = self.sk, self.sv, self.rg
        t = time.perf_counter()
        col, al, nl, _, ctr = orc.render_fwd(oc, self.pr, rg, sv, self.sact, self.bits)
        orc.render_bwd(oc, self.pr, rg, sv, nl, self.gcol, None, self.sact, self.bits)
        t_blend = time.perf_counter() - t
        scale = self.n_active / self.pick.shape[0]
        total = t_pre + t_qs + t_blend * scale
        desc = (f"oracle (single thread, fp64) on a bounded sample of config {self.cfg_id}: preprocess+preprocess_bwd on {self.n_pre} of {P} "
                f"Gaussians (x{P / self.n_pre:.0f}), query+sort+ranges on {self.n_query} Gaussians (x{P / self.n_query:.0f}, ~{pairs_est:.3g} pairs), "
                f"blend fwd+bwd on {self.pick.shape[0]} of {self.n_active} tiles with complete lists ({sk.shape[0]} pairs, {ctr['evaluated']} "
                f"evaluations; x{scale:.0f}); extrapolated whole-frame time {total:.1f} s = pre {t_pre:.1f} + query/sort {t_qs:.1f} + "
                f"blend {t_blend * scale:.1f}; measured CPU time of the sample {t_pre * self.n_pre / P + t_qs * self.n_query / P + t_blend:.1f} s")
        return total, desc


def workload_config(cfg_id, n_gpus, n_pix):
    """The `config` object of the JSON line: the same keys and values in both arms (--impl ours / reference)."""
    m = scenes.CONFIGS[cfg_id]
    return dict(workload=f"config{cfg_id}:{m['name']}", order=m["order"], nside=1 << m["order"], n_pix=int(n_pix), n_gauss=m["n_gauss"],
                sh_degree=m["sh_degree"], n_views=m["n_views"], parallelism=f"replicas{n_gpus}",
                l2="inputs larger than L2 (Gaussians + pair buffers: GBs at config 4); no flush needed")


def oracle_timing(cfg_id, repeats, warmup=0):
    """The oracle as it stands on ORACLE_SAMPLE of the workload, `repeats` timed steps.  Returns (sample object, step times, description)."""
    smp = OracleSample(cfg_id, seed=0, **ORACLE_SAMPLE)
    times, desc = [], ""
    for i in range(warmup + repeats):
        t, desc = smp.step()
        if i >= warmup:
            times.append(t)
    return smp, times, desc


def cpu_baseline_object(smp, times, desc):
    t = float(np.mean(times))
    return dict(value=smp.n_pix / t, unit=UNIT, cores=1, kind="oracle", sample=desc, repeats=len(times),
                spread=dict(min_s=float(np.min(times)), max_s=float(np.max(times)), mean_s=t,
                            note="extrapolated whole-frame seconds of each timed repeat of the same sample"))


def run_reference(args):
    """The reference arm for this tier is the oracle (there is no reference code): rank 0 alone times it, the other ranks exit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    smp, times, desc = oracle_timing(args.config, args.steps, args.warmup)
    t = float(np.mean(times))
    val = smp.n_pix / t
    line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup, ms_per_step=t * 1e3,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic", impl="reference",
                config=workload_config(args.config, args.gpus, smp.n_pix),
                note=("ms_per_step is the EXTRAPOLATED whole-frame time of the single-thread fp64 oracle from a bounded sample (cpu_baseline.sample); "
                      "the CPU time actually spent per step is about 1/100 of it"),
                cpu_baseline=cpu_baseline_object(smp, times, desc),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------------------- our arm
def stage_bytes(stage, P, V, M, n_tiles, n_pairs):
    """Algorithmic HBM bytes of one call of an HBM-bound stage."""
    tile_bytes = (max(1, (V * n_tiles - 1)).bit_length() + 7) // 8
    return {"preprocess": P * V * (44 + 12 * M + 57),
            "preprocess_bwd": P * (44 + 12 * M + V * 33 + 40 + 12 * M),
            "depth_order": P * V * (4 + 5 * 32 + 16),
            "tile_query": P * V * 2 * 29 + 8 * P * V + 12 * n_pairs,
            "tile_lists": P * V * 2 * 29 + 12 * n_pairs + 16 * V * n_tiles,      # floor: every sorted pair written once
            "sort": 32.0 * n_pairs * tile_bytes,
            "tile_ranges": 8.0 * n_pairs + 16 * V * n_tiles}[stage]


def measure_config(args, cfg_id, steps, warmup, rank, world, dist, local, sample_clocks=False):
    """Times `steps` whole steps of config cfg_id on this rank (CUDA events on the launching stream, per stage and whole).
    Returns a dict with the rasteriser still alive under "r" (the caller deletes it)."""
    import torch
    from paper_2606_29794_b200 import binding as B, rasterizer as R, replicas
    scene = scenes.make_scene(cfg_id, seed=replicas.rank_seed(rank))
    cfg = R.config_of(scene)
    mask = B.Mask.full() if scene["mask"] is None else B.uts_build_mask(cfg, scene["mask"]["kind"], scene["mask"]["params"])
    g, views = R.scene_to_device(scene)
    fused = args.lists == "fused"
    STAGES = STAGES_FUSED if fused else STAGES_STAGED
    NS = len(STAGES)
    r = R.Rasterizer(cfg, mask, fused_lists=fused, marks=(args.marks == "on"))
    V, S = cfg.n_views, r.S
    npx = S * cfg.ppt
    gcol = torch.from_numpy(scenes.upstream_grad(V, npx, seed=rank)).cuda()
    if scene["mask"] is None:
        n_pix_active = int(V * cfg.n_pix)
    else:
        w = mask.pixel_mask_bits.to(torch.int64) & 0xffffffff
        w = w - ((w >> 1) & 0x55555555); w = (w & 0x33333333) + ((w >> 2) & 0x33333333); w = (w + (w >> 4)) & 0x0f0f0f0f
        n_pix_active = int(V * int((((w * 0x01010101) & 0xffffffff) >> 24).sum().item()))
    stream = torch.cuda.current_stream()

    def step(events=None):
        def mark(i):
            if events is not None:
                events[i].record(stream)
        mark(0); r.preprocess(g, views)
        mark(1); r.depth_order()
        if fused:
            mark(2); r.tile_lists()
            i = 3
        else:
            mark(2); r.tile_query()
            mark(3); r.sort()
            mark(4); r.tile_ranges()
            i = 5
        mark(i); r.render_fwd()
        mark(i + 1); r.render_bwd(gcol)
        mark(i + 2); r.preprocess_bwd(g, views)
        mark(i + 3)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = None
    if sample_clocks:
        sampler = ClockSampler(local); sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(NS + 1)] for _ in range(steps)]
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    launches0 = B.uts_launch_count()
    t0.record(stream)
    for k in range(steps):
        step(ev[k])
    t1.record(stream)
    torch.cuda.synchronize()
    launches = B.uts_launch_count() - launches0          # counted by the library itself, one tick per kernel launch
    clocks = sampler.stop() if sampler else None
    ms_step = t0.elapsed_time(t1) / steps
    stage_ms = {STAGES[i]: float(np.mean([ev[k][i].elapsed_time(ev[k][i + 1]) for k in range(steps)])) for i in range(NS)}
    ms_fwd = sum(stage_ms[s] for s in STAGES[:NS - 2])

    # ---- work counters (measurement plumbing, after the timed region)
    # evaluated / contributing pairs of Alg.1's loop, counted on the device by uts_render_fwd_counted (same decisions as the timed kernels)
    work = torch.zeros(4, dtype=torch.int64, device="cuda")
    scratch_img = [torch.empty_like(t) for t in (r.color, r.alpha, r.trans, r.n_last)]
    B.uts_render_fwd_counted(cfg, r.proj, mask, r.ranges, r.vals, *scratch_img, work)
    ev_f, contrib, ev_cull, ev_full = (int(x) for x in work.cpu().tolist())
    del scratch_img
    ev_b = int(r.n_last.long().sum().item())              # SURVEY 8(d)'s E_bwd: every entry before n_last, for every pixel
    # with marks the backward evaluates only the (patch, entry) pairs the forward marked: 32 pixel evaluations each (a population
    # count of the mark words; the buffer starts zeroed and every step writes the same words)
    ev_b_visited = None
    if r.use_marks:
        tot = 0
        mk = r.marks
        for c0 in range(0, mk.numel(), 1 << 24):
            t = mk[c0:c0 + (1 << 24)].to(torch.int64) & 0xffffffff
            t = t - ((t >> 1) & 0x55555555); t = (t & 0x33333333) + ((t >> 2) & 0x33333333); t = (t + (t >> 4)) & 0x0f0f0f0f
            tot += int((((t * 0x01010101) & 0xffffffff) >> 24).sum().item())
        ev_b_visited = 32 * tot
    return dict(scene=scene, cfg=cfg, mask=mask, g=g, views=views, r=r, gcol=gcol, STAGES=STAGES, ms_step=ms_step, ms_fwd=ms_fwd, stage_ms=stage_ms,
                launches=int(launches), clocks=clocks, n_pix_active=n_pix_active, n_pairs=int(r.n_pairs), ev_f=ev_f, ev_b=ev_b, contrib=contrib, ev_cull=ev_cull, ev_full=ev_full,
                ev_b_visited=ev_b_visited, npx=npx)


def per_kernel_table(m, peaks, fp32_peak):
    """Per stage: ms and the achieved fraction of the roofline that bounds it (HBM stages: algorithmic bytes / time against the measured
    copy bandwidth; blend stages: FP32 operations of the work the kernel EXECUTES / time against the derived FP32 peak)."""
    cfg = m["cfg"]
    P, V, M = cfg.n_gauss, cfg.n_views, cfg.n_sh
    out = {}
    for s_, ms in m["stage_ms"].items():
        sec = ms * 1e-3
        if s_ == "render_fwd":
            # executed work: evaluations that pass the patch cull 41, contributing pairs + 9
            flop = m["ev_cull"] * FLOP_FWD_EVAL + m["contrib"] * FLOP_FWD_CONTRIB
            flop_alg = m["ev_f"] * FLOP_FWD_EVAL + m["contrib"] * FLOP_FWD_CONTRIB
            out[s_] = dict(ms=ms, bound="alu", tflops=flop / sec / 1e12, frac_fp32_peak=flop / sec / 1e12 / fp32_peak,
                           frac_fp32_peak_alg1_units=flop_alg / sec / 1e12 / fp32_peak)
        elif s_ == "render_bwd":
            ev_exec = m["ev_b_visited"] if m["ev_b_visited"] is not None else m["ev_b"]
            flop = ev_exec * FLOP_BWD_EVAL + m["contrib"] * FLOP_BWD_CONTRIB
            flop_alg = m["ev_b"] * FLOP_BWD_EVAL + m["contrib"] * FLOP_BWD_CONTRIB
            out[s_] = dict(ms=ms, bound="alu", tflops=flop / sec / 1e12, frac_fp32_peak=flop / sec / 1e12 / fp32_peak,
                           frac_fp32_peak_alg1_units=flop_alg / sec / 1e12 / fp32_peak)
        else:
            byts = stage_bytes(s_, P, V, M, cfg.n_tiles, m["n_pairs"])
            out[s_] = dict(ms=ms, bound="hbm", gbs=byts / sec / 1e9, frac_hbm_peak=byts / sec / 1e9 / peaks["hbm_gbs"])
            if s_ == "tile_lists":        # secondary: SURVEY 8(d)'s separate floors of F2 + F3 + F4 (12 + 24 + 8 B per pair) instead of write-once
                out[s_]["frac_hbm_peak_survey8d_units"] = 44.0 * m["n_pairs"] / sec / 1e9 / peaks["hbm_gbs"]
    return out


def roofline_of_dominant(m, pk, peaks, fp32_peak, traffic):
    """`roofline` = the stage with the largest time, whichever it is (uts_tile_lists is one ABI call of about 25 kernels; its line is
    the call's algorithmic bytes against the HBM peak, and profiles/ holds its kernels one by one)."""
    dom = max(m["stage_ms"], key=m["stage_ms"].get)
    e = pk[dom]
    if e["bound"] == "alu":
        roof = dict(kernel=dom, bound="alu", achieved=e["tflops"], peak=fp32_peak, unit="TFLOP/s", frac=e["frac_fp32_peak"], traffic=traffic.get(dom),
                    peak_source="derived: 148 SM x 128 FP32 lanes x 2 x sm_max_mhz",
                    note="flops of the evaluations the kernel executes (41/46 per evaluated pair + 9/72 per contributing pair, counted on the device)")
    else:
        roof = dict(kernel=dom, bound="hbm", achieved=e["gbs"], peak=peaks["hbm_gbs"], unit="GB/s", frac=e["frac_hbm_peak"], traffic=traffic.get(dom),
                    peak_source=peaks["source"] + " (MEASURED_PEAKS.json hbm_gbs: copy bandwidth)" if peaks["source"] == "measured" else "fallback 6650 GB/s")
        if dom == "tile_lists":
            roof["note"] = ("one ABI call = Alg.1 l.9-16 (tile query + depth sort + ranges): algorithmic bytes = every sorted pair written once (12 B) + "
                            "58 B per (view, Gaussian) + 16 B per (view, tile); the call is issue-bound geometry + a merge, see profiles/")
    return roof


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_29794_b200 import binding as B, rasterizer as R, replicas

    world, rank, local = replicas.world()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = _peaks()
    fp32_peak = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12       # TFLOP/s at the maximum SM clock

    # replicas only: every rank renders its own scene of the same recipe; no data-path collective
    m = measure_config(args, args.config, args.steps, args.warmup, rank, world, dist, local, sample_clocks=True)
    scene, cfg, mask, g, views, r, gcol = m["scene"], m["cfg"], m["mask"], m["g"], m["views"], m["r"], m["gcol"]
    V, npx, n_pix_active = cfg.n_views, m["npx"], m["n_pix_active"]
    fused = args.lists == "fused"
    ms_step = m["ms_step"]

    extras = {}
    run_extras = not args.no_extras
    r._color_full = r.color.clone()          # the full lists' image, for the bit-identity check of the depth-prefix leg below
    # next step after the hot path (not part of the step): Interp_H of Eq.7 to the camera image and its adjoint,
    # timed on view 0's HEALPix image.  Camera: the paper's case for this grid where there is no mask (6080 x 3040 panorama ->
    # Nside 1024, Table 5), else a 1920 x 1080 pinhole of 60 x 45 degrees (config 5's frustum).
    try:
        if not run_extras:
            raise RuntimeError("skipped (--no-extras)")
        cam = B.Camera("equirect", 6080, 3040) if mask.active_tiles is None else B.Camera("pinhole", 1920, 1080, np.radians(60.0), np.radians(45.0))
        img = r.color[0].contiguous()
        o_img = torch.empty(cam.height, cam.width, 3, dtype=torch.float32, device="cuda")
        g_img = torch.randn(cam.height, cam.width, 3, device="cuda")
        gi = torch.empty_like(img)
        tms = []
        for fn in (lambda: B.uts_resample_fwd(cfg, cam, mask, img, o_img, None), lambda: B.uts_resample_bwd(cfg, cam, mask, g_img, gi)):
            for _ in range(3):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                fn()
            e1.record(); torch.cuda.synchronize()
            tms.append(e0.elapsed_time(e1) / 5)
        byts = cam.width * cam.height * 12 + img.numel() * 4
        extras["resample"] = dict(camera=f"{cam.model} {cam.width}x{cam.height}", fwd_ms=tms[0], bwd_ms=tms[1], fwd_gbs=byts / (tms[0] * 1e-3) / 1e9,
                                  bwd_gbs=(byts + img.numel() * 4) / (tms[1] * 1e-3) / 1e9, bytes_model="12 B per image pixel + 12 B per HEALPix pixel (+ its zero-fill in the adjoint)")
        del o_img, g_img, gi, img
    except Exception as e:      # measurement plumbing only; never hides a failure of the step itself
        extras["resample"] = dict(error=str(e))

    # the step before the backward hot path (not part of the step): L1 + HEALPix-SSIM loss and dL/dI on view 0's
    # image against a seeded target (the image plus N(0, 0.05) noise, clipped)
    try:
        if not run_extras:
            raise RuntimeError("skipped (--no-extras)")
        img = r.color[0].contiguous()
        tgt = (img + 0.05 * torch.randn(img.shape, device="cuda", generator=torch.Generator(device="cuda").manual_seed(7))).clamp_(0, 1)
        loss3 = torch.empty(3, dtype=torch.float64, device="cuda")
        g_l = torch.empty_like(img)
        sc_l = torch.empty(B.uts_hssim_scratch_bytes(cfg), dtype=torch.uint8, device="cuda")
        tms = []
        for fn in (lambda: B.uts_hssim_loss(cfg, mask, img, tgt, loss3, sc_l, dL_dX=g_l), lambda: B.uts_hssim_loss(cfg, mask, img, tgt, loss3, sc_l)):
            for _ in range(3):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                fn()
            e1.record(); torch.cuda.synchronize()
            tms.append(e0.elapsed_time(e1) / 5)
        npx_l = img.shape[0]
        extras["hssim_loss"] = dict(loss=float(loss3[0]), l1=float(loss3[1]), hssim=float(loss3[2]), fwd_bwd_ms=tms[0], fwd_ms=tms[1],
                                    gtap_per_s=npx_l * 121 * 3 / (tms[0] * 1e-3) / 1e9,
                                    work_model="121 taps x 3 channels per pixel, forward sums + gradient scatter; 36 B compulsory traffic per pixel")
        del img, tgt, g_l
    except Exception as e:      # measurement plumbing only
        extras["hssim_loss"] = dict(error=str(e))

    # inverse radial depth as a fourth channel of the blend (not part of the step): the marked pair with and without it
    try:
        if not run_extras:
            raise RuntimeError("skipped (--no-extras)")
        depth = torch.empty_like(r.alpha)
        g_d = torch.randn(r.alpha.shape, device="cuda")
        G_ = r._alloc_grads()
        invr = torch.empty(cfg.n_views, cfg.n_gauss, dtype=torch.float32, device="cuda")
        legs = dict(fwd=lambda: r.render_fwd(), fwd_depth=lambda: B.uts_render_fwd_depth(cfg, r.proj, mask, r.ranges, r.vals, r.capacity, r.color, r.alpha, r.trans, r.n_last, depth, r.marks),
                    bwd=lambda: r.render_bwd(gcol), bwd_depth=lambda: B.uts_render_bwd_depth(cfg, r.proj, mask, r.ranges, r.vals, r.capacity, r.trans, r.n_last, r.marks, gcol, None, g_d,
                                                                                          G_["rgb"], G_["conic"], G_["mu2"], G_["opac"], invr))
        tms = {}
        for name, fn in legs.items():
            for _ in range(2):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                fn()
            e1.record(); torch.cuda.synchronize()
            tms[name + "_ms"] = e0.elapsed_time(e1) / 5
        tms["overhead_fwd"] = tms["fwd_depth_ms"] / tms["fwd_ms"] - 1.0
        tms["overhead_bwd"] = tms["bwd_depth_ms"] / tms["bwd_ms"] - 1.0
        extras["depth_channel"] = tms
        del depth, g_d, invr
    except Exception as e:      # measurement plumbing only
        extras["depth_channel"] = dict(error=str(e))

    # occlusion-bounded lists (not the step: Alg.1 builds the full lists): lists from the nearest `keep`
    # Gaussians, verified every time by uts_count_unsaturated — when no visible pixel is left open, image and gradients are exactly
    # the full lists' ones.  keep is found by doubling from P/256; the timed steps include the check.
    try:
        if not run_extras:
            raise RuntimeError("skipped (--no-extras)")
        if fused:
            Pn = cfg.n_gauss
            keep, n_open = max(Pn // 256, 1), 1
            while True:
                _, _, n_open = r.forward_depth_prefix(g, views, keep)
                if n_open == 0 or keep >= Pn:
                    break
                keep = min(Pn, keep * 2)
            if n_open == 0:
                same = bool(torch.equal(r.color, color_full)) if (color_full := getattr(r, "_color_full", None)) is not None else None
                for _ in range(2):
                    r.forward_depth_prefix(g, views, keep); r.backward(g, views, gcol)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for _ in range(5):
                    r.forward_depth_prefix(g, views, keep); r.backward(g, views, gcol)
                e1.record(); torch.cuda.synchronize()
                extras["depth_prefix"] = dict(keep=keep, n_gauss=Pn, n_pairs=int(r.n_pairs), ms_per_step=e0.elapsed_time(e1) / 5,
                                              image_bit_identical_to_full_lists=same,
                                              note="lists from the nearest `keep` Gaussians per view; every step checks that no visible pixel is left open")
            else:
                extras["depth_prefix"] = dict(keep=keep, open_pixels=int(n_open), note="not every pixel saturates on this workload: the full lists are needed")
            r.forward(g, views)          # leave the rasteriser in the state of the full path for what follows
    except Exception as e:      # measurement plumbing only
        extras["depth_prefix"] = dict(error=str(e))

    # end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region)
    h = {k: torch.from_numpy(scene[k]).contiguous().pin_memory() for k in ("means", "scales", "quats", "opac", "sh", "W", "b")}
    hg = gcol.cpu().pin_memory()
    P, M = cfg.n_gauss, cfg.n_sh
    pin = lambda *s: torch.empty(*s, dtype=torch.float32).pin_memory()
    out = dict(color=pin(V, npx, 3), alpha=pin(V, npx), dL_dmeans=pin(P, 3), dL_dscales=pin(P, 3), dL_dquats=pin(P, 4), dL_dopac=pin(P),
               dL_dsh=pin(P, M, 3))
    cap = m["n_pairs"] + 1024
    ws_bytes = B.uts_host_workspace_bytes(cfg, mask.n_active, cap)
    del r
    m["r"] = None
    torch.cuda.empty_cache()
    ws = torch.empty(ws_bytes // 8 + 64, dtype=torch.int64, device="cuda")
    h2d = sum(t.numel() * 4 for t in h.values()) + hg.numel() * 4
    d2h = sum(t.numel() * 4 for t in out.values())
    e2e_steps = max(10, min(args.steps, 20)) if args.steps >= 3 else args.steps      # at least 10 timed end-to-end steps in a normal run
    for _ in range(2):
        B.uts_host_forward_backward(cfg, h, mask, hg, out, cap, ws)       # warm-up
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    tt = time.perf_counter()
    for _ in range(e2e_steps):
        B.uts_host_forward_backward(cfg, h, mask, hg, out, cap, ws)       # synchronises the stream itself
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - tt) * 1e3 / e2e_steps
    del ws, h, hg, out
    torch.cuda.empty_cache()

    ms_step_max, e2e_ms_max = replicas.max_over_ranks([ms_step, e2e_ms], device="cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = replicas.aggregate_throughput(n_pix_active, ms_step_max, world)
    # DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed ncu --set full capture of this workload
    # (profiles/), or None
    traffic = {}
    for name in ("r02_traffic.csv", "r01_traffic.csv"):
        tp = os.path.join(ROOT, "profiles", name)
        if os.path.exists(tp):
            with open(tp) as f:
                for ln in f.read().splitlines()[1:]:
                    w_, st_, by_ = ln.split(",")
                    if w_ == f"config{args.config}":
                        traffic[st_] = int(by_)
            break
    pk = per_kernel_table(m, peaks, fp32_peak)
    roof = roofline_of_dominant(m, pk, peaks, fp32_peak, traffic)

    # the other BASELINE.json configs, a few steps each (headline stays args.config): ms forward / forward+backward, px/s and the
    # dominant stage's roofline fraction, so that the driver-run record covers all five configs
    if run_extras and world == 1:
        others = {}
        for cid in (1, 2, 3, 5):
            if cid == args.config:
                continue
            try:
                mo = measure_config(args, cid, 5, 3, rank, world, dist, local)
                pko = per_kernel_table(mo, peaks, fp32_peak)
                domo = max(mo["stage_ms"], key=mo["stage_ms"].get)
                fr = pko[domo].get("frac_hbm_peak", pko[domo].get("frac_fp32_peak"))
                others[f"config{cid}"] = dict(workload=f"config{cid}:{mo['scene']['name']}", n_pix=mo["n_pix_active"], n_pairs=mo["n_pairs"], steps=5, warmup=3,
                                              ms_forward=mo["ms_fwd"], ms_forward_backward=mo["ms_step"], px_per_s=mo["n_pix_active"] / (mo["ms_step"] * 1e-3),
                                              stage_ms=mo["stage_ms"], dominant=dict(stage=domo, bound=pko[domo]["bound"], frac=fr), gpu_launches_per_step=mo["launches"] / 5)
                for k_ in ("r", "g", "views", "gcol", "mask"):
                    mo[k_] = None
                del mo
                torch.cuda.empty_cache()
            except Exception as e:      # measurement plumbing only
                others[f"config{cid}"] = dict(error=str(e))
        extras["configs"] = others

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=ms_step_max,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=workload_config(args.config, world, n_pix_active),
                path=dict(lists=args.lists, marks=args.marks, n_pairs=m["n_pairs"]),
                ms_forward=m["ms_fwd"], ms_forward_backward=ms_step, stage_ms=m["stage_ms"], per_kernel=pk,
                evaluated_pairs=dict(forward=m["ev_f"], forward_after_patch_cull=m["ev_cull"], forward_q_above_cut=m["ev_full"], contributing=m["contrib"], backward_alg1=m["ev_b"], backward_executed=m["ev_b_visited"],
                                     listed=int(m["n_pairs"]) * cfg.ppt,
                                     note="forward (Alg.1's loop) / after the per-patch cull (a lower bound of what the forward executes: a warp owns two patches and walks an entry for both when it reaches either) / of those, patches where q alone cannot rule the entry out (informational) / contributing: counted on the device by uts_render_fwd_counted; backward_alg1: sum of n_last; "
                                          "backward_executed: 32 x marked (patch, entry) pairs; listed: pairs x 256 pixels"),
                roofline=roof, clocks=m["clocks"], extras=extras,
                e2e=dict(value=replicas.aggregate_throughput(n_pix_active, e2e_ms_max, world), unit=UNIT, ms_per_step=e2e_ms_max, steps=e2e_steps,
                         h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h),
                gpu_launches=m["launches"])                # uts_launch_count() over the timed region
    if not args.no_cpu_baseline:
        smp, times, desc = oracle_timing(args.config, 3)
        line["cpu_baseline"] = cpu_baseline_object(smp, times, desc)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_selftest(args):
    """CPU-only check of the multi-rank plumbing (tests/test_replicas_gloo.py): every rank joins a gloo group, the ranks agree on
    max-over-ranks times, rank 0 prints a line with n_gpus = world size.  Runs no kernel and reports no measurement."""
    import torch.distributed as dist
    from paper_2606_29794_b200 import replicas
    world, rank, _ = replicas.world()
    if world > 1:
        dist.init_process_group("gloo")
    mx = replicas.max_over_ranks([10.0 + rank, 5.0 - rank])
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(dict(selftest=True, n_gpus=world, max_over_ranks=mx)))


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start the N ranks here, the way the driver does
    (python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py ...),
    and pass their output through.  NCCL's own log stays on (NCCL_DEBUG=INFO unless the caller set it) and goes to stderr."""
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config id 1..5 (default 4 = the metric's workload)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "selftest"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--lists", default="fused", choices=["fused", "staged"],
                    help="Alg.1 l.9-16 as one uts_tile_lists call (default) or as uts_tile_query + uts_sort + uts_tile_ranges")
    ap.add_argument("--no-extras", action="store_true", help="skip the legs that are not part of the step (resample, loss, depth prefix, other configs): used for the launch list")
    ap.add_argument("--marks", default="on", choices=["on", "off"],
                    help="blend through uts_render_fwd_marked / uts_render_bwd_marked (default) or the plain pair")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    if args.impl == "reference":
        run_reference(args)
    elif args.impl == "selftest":
        run_selftest(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
