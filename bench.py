#!/usr/bin/env python
"""bench.py -- headline benchmark of the CAS hot path on B200.

One "step" = one pass of the whole hot path over one batch of BASELINE.json configs[1]
(c2, bf16 3B-like layer): slot-table build (host) -> prefix-attention forward -> backward (dK/dV
scatter-accumulated into the cartridge gradient slots) -> fused Adam over the resident cartridges.
(c2 has no rotation; c3 adds the plan + swap-out/in overlapped on the side streams.)

metric  = prefix-attn fwd+bwd TFLOP/s: algorithmic FLOPs 14*D*Hq*pairs (visible pairs only,
          DESIGN.md "Algorithmic work") divided by the time of the WHOLE step (Adam included).
roofline= the dominant kernel (attention backward) against the measured bf16 peak: the BURST figure when the
          timed region is shorter than a second, the sustained one otherwise (decode configs: HBM).
e2e     = the same metric through cas_train_step_host_async(): pinned HOST buffers, H2D of Q/K_self/V_self/dO
          and D2H of O/LSE/dQ/dK_self/dV_self of every step inside the timed region, steps pipelined over two
          device buffer sets, cas_train_step_host_wait before the clock stops; the per-call-complete variant
          (cas_train_step_host) is reported beside it.
cpu_baseline = the oracle (numpy fp64, as it stands) timed on a bounded sample of the same workload.

The default run (`python bench.py`, about two minutes) prints ONE JSON line: c2 is the headline; `sustained` is a
>= 3 s loop of the same steps with its own clock samples; `extra` carries one compact record each for c3 (with and
without rotation, swap alone against the host-link peak measured in the same run), c4, c5 "all loaded", c5 top-8
and c_pages.  `--no-extra` gives the headline config only; `--config X` benches another config as the headline.

`--impl reference` times the oracle alone (this tier has no reference implementation to install).
Multi-GPU: replicas only -- every rank runs its own batch on its own pool,
no data-path collective; value = total FLOPs of all ranks / max-over-ranks time ("scaling": "weak").
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

METRIC = "prefix_attn_fwd_bwd_tflops"
UNIT = "TFLOP/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sust=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sust=1400.0, src="fallback")


def load_traffic():
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the dominant kernels, taken
    from the committed `ncu --set full` capture (profiles/traffic.json names the capture)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p))
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs
    (an nvidia-smi subprocess per sample is too slow for a region of tens of milliseconds; it is
    the fallback when NVML cannot be loaded)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag = index, False
        self.sm, self.reasons, self.sm_max = [], set(), None
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        self.sm.append(float(n.nvmlDeviceGetClockInfo(self.h, n.NVML_CLOCK_SM)))
        r = n.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        for name, bit in (("sw_power_cap", 0x4), ("hw_slowdown", 0x8), ("sw_thermal_slowdown", 0x20),
                          ("hw_thermal_slowdown", 0x40)):
            if r & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                              "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
        r = [x.strip() for x in out.strip().split(",")]
        if len(r) >= 7 and r[0].replace(".", "").isdigit():
            self.sm.append(float(r[0]))
            self.sm_max = float(r[1])
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    self.reasons.add(name)

    def run(self):
        while not self.stop_flag:
            try:
                if self.nvml:
                    self._sample_nvml()
                else:
                    self._sample_smi()
            except Exception:
                pass
            time.sleep(0.002 if self.nvml else 0.1)

    def summary(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.sm),
                "source": "nvml" if self.nvml else "nvidia-smi"}


def attn_flops(wl):
    cfg = wl.cfg
    pairs = wl.pairs_per_head()
    fwd = 4 * cfg.D * cfg.Hq * pairs
    return fwd, (2.5 * fwd if cfg.backward else 0.0)


def oracle_sample(wl, budget_s=12.0, max_units=64):
    """Times the oracle (as it stands) on (sequence, KV-head) units of the workload until about
    `budget_s` seconds of CPU work are done.  Returns (TFLOP/s, description, seconds, threads)."""
    from oracle import cas_oracle as orc

    cfg = wl.cfg
    bK = [wl.cart_kv(c)[0] for c in range(cfg.n_carts)]
    bV = [wl.cart_kv(c)[1] for c in range(cfg.n_carts)]
    scale = 1.0 / float(np.sqrt(cfg.D))
    G = cfg.Hq // cfg.Hkv
    units = [(b, g) for b in range(cfg.B) for g in range(cfg.Hkv)]
    done_flops, t_used, n = 0.0, 0.0, 0
    for (b, g) in units[:max_units]:
        t0, t1 = int(wl.seq_off[b]), int(wl.seq_off[b + 1])
        sel = [wl.sel_cart[wl.sel_off[b]:wl.sel_off[b + 1]].tolist()]
        so = np.array([0, t1 - t0])
        a = time.perf_counter()
        orc.attn_fwd(wl.Q[t0:t1], bK, bV, sel, so, wl.K_self[t0:t1], wl.V_self[t0:t1], scale, cfg.Hkv, kv_heads=[g])
        if cfg.backward:
            orc.attn_bwd(wl.Q[t0:t1], bK, bV, sel, so, wl.K_self[t0:t1], wl.V_self[t0:t1], wl.dO[t0:t1], scale,
                         cfg.Hkv, kv_heads=[g])
        t_used += time.perf_counter() - a
        lq = t1 - t0
        pb = int(wl.cart_len[sel[0]].sum()) if sel[0] else 0
        pairs = lq * pb + lq * (lq + 1) // 2
        done_flops += (14 if cfg.backward else 4) * cfg.D * G * pairs
        n += 1
        if t_used >= budget_s:
            break
    try:
        from threadpoolctl import threadpool_info

        threads = max([i.get("num_threads", 1) for i in threadpool_info()] or [1])
    except Exception:
        threads = os.cpu_count() or 1
    desc = (f"{n} of {len(units)} (sequence, KV-head) units of {cfg.name}: complete fwd"
            f"{'+bwd' if cfg.backward else ''} of those units, numpy float64")
    return done_flops / t_used / 1e12, desc, t_used, threads


def reduce_over_ranks(ms_step, e2e_ms, flops, world, device):
    """Replica aggregation: every rank ran its own batch on its own pool, so the job's
    time is the MAX over ranks and its work the SUM over ranks.  No data-path collective: these two
    all-reduces only combine the measurements.  Returns (ms_step_max, e2e_ms_max, total_flops)."""
    import torch

    times = torch.tensor([ms_step, e2e_ms], dtype=torch.float64, device=device)
    work = torch.tensor([flops], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist

        dist.all_reduce(times, op=dist.ReduceOp.MAX)
        dist.all_reduce(work, op=dist.ReduceOp.SUM)
    return float(times[0]), float(times[1]), float(work[0])


def run_reference(args, wl):
    """The reference arm of this tier = the oracle, timed on the host cores."""
    tf, desc, secs, threads = 0.0, "", 0.0, 1
    vals = []
    for i in range(args.warmup + args.steps):
        tf, desc, secs, threads = oracle_sample(wl, budget_s=args.ref_budget, max_units=args.ref_units)
        if i >= args.warmup:
            vals.append((tf, secs))
    tf = float(np.mean([v[0] for v in vals]))
    ms = float(np.mean([v[1] for v in vals])) * 1e3
    line = {"metric": METRIC, "value": tf, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": wl.cfg.name, "note": "each step = a bounded sample of the workload"},
            "cpu_baseline": {"value": tf, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": tf, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def measure_host_link(torch, dev):
    """Pinned-copy peak of the host link (not in MEASURED_PEAKS.json, so measured in the same run):
    256 MiB copies, each direction alone and both at once, best of 4."""
    hbuf = torch.empty(256 << 20, dtype=torch.uint8).pin_memory()
    hbuf2 = torch.empty(256 << 20, dtype=torch.uint8).pin_memory()
    dbuf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    dbuf2 = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    s2 = torch.cuda.Stream()
    best = {}
    for name in ("h2d", "d2h", "both"):
        ts = []
        for _ in range(4):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if name in ("h2d", "both"):
                dbuf.copy_(hbuf, non_blocking=True)
            if name in ("d2h", "both"):
                with torch.cuda.stream(s2):
                    hbuf2.copy_(dbuf2, non_blocking=True)
            torch.cuda.synchronize()
            ts.append(time.perf_counter() - t0)
        best[name] = (256 << 20) / min(ts) / 1e9
    return best


def run_config(args, cfg_name, steps, warmup, rank, world, local_rank, do_e2e, do_cpu, no_swap=False, sustain_s=0.0):
    """One workload: W warm-up steps, K timed steps (CUDA events on the launching stream, barrier + synchronize on
    both sides, clocks sampled through NVML during the timed region).  Returns (line, ms_step_max) on every rank;
    `line` is the JSON record on rank 0, None elsewhere."""
    import torch

    from paper_2606_04557_b200 import cas
    from paper_2606_04557_b200.harness import Session
    from workloads import BASE_SEED, CONFIGS, make_workload

    cfg = CONFIGS[cfg_name]
    dev = f"cuda:{local_rank}"
    if world > 1:
        import torch.distributed as dist
    wl = make_workload(cfg, BASE_SEED + rank)          # every rank: its own batch, its own pool
    sess = Session(wl, device=dev)
    stream = torch.cuda.current_stream()
    fwd_fl, bwd_fl = attn_flops(wl)
    # resident K+V elements the Adam call updates (with rotation: slots in transit this step are skipped, K4)
    # algorithmic bytes: 30 B per element of a slot that holds gradients this step (read g,p,m,v,
    # write p,m,v + bf16 copy), 26 B per element of a clean slot (g = 0 is not read).  Counted per step in prepare().
    adam_acc = {"bytes": 0, "steps": 0}

    rotate = cfg.rotate_in > 0 and not no_swap
    rot = {"step": 0, "rng": np.random.Generator(np.random.PCG64(BASE_SEED + 1000 + rank)), "bytes": 0}
    if cfg.rotate_in > 0:
        from workloads.generate import draw_batch_selection, draw_batch_selection_uniform

    def prepare():
        tau = rot["step"]
        rot["step"] += 1
        sel_off, sel_cart = wl.sel_off, wl.sel_cart
        stable = None
        if cfg.rotate_in > 0:
            # K4 step protocol: draw among resident+stable cartridges, protect them, plan, swap on
            # the side stream while fwd/bwd/Adam run on the main stream, commit.
            c = cas.cas_pool_counters(sess.pool)
            stable = np.nonzero((c["slot_of"] >= 0) & (c["in_transit"] == 0))[0]
            if cfg.selection == "uniform" and cfg.n_dist != -2:
                # the same recipe drawn for the whole batch at once: per-sequence Generator.choice calls cost more
                # host time than a c_pages step costs on the GPU
                sel_off, sel_cart = draw_batch_selection_uniform(cfg, rot["rng"], stable)
            else:
                sel_off, sel_cart = draw_batch_selection(cfg, rot["rng"], stable.tolist(), wl.cart_len)
        rot["sel"] = (sel_off, sel_cart)
        if cfg.backward or tau == 0:
            # training: a new batch and a new slot table every step.  Decode (c5): the selection is fixed while
            # a request generates, so the table (and its split-KV work list) is built once and reused per token.
            sess.tab.close()
            sess.tab = cas.cas_slot_table_build(sess.pool, wl.seq_off, sel_off, sel_cart, tau)
        if rotate:
            prot = np.unique(sel_cart).tolist()
            man, n = cas.cas_plan_rotation(sess.pool, tau, cfg.rotate_in, cfg.rotate_out, prot, 260604)
            cas.cas_swap_out(sess.pool, man, n, tau, after_stream=stream)
            cas.cas_swap_in(sess.pool, man, n, tau)
            rot["bytes"] += sum(int(man[i].nbytes) for i in range(n))
            leaving = set(int(man[i].cart) for i in range(n) if man[i].dir == cas.CAS_DIR_OUT)
        else:
            leaving = set()
        if cfg.backward:
            # Adam updates every resident cartridge that is not in transit this step (K4); algorithmic bytes: 30 B per
            # element of a slot that holds gradients, 26 B per element of a clean one
            upd = np.asarray(stable if cfg.rotate_in > 0 else np.arange(cfg.n_slots), dtype=np.int64)
            if leaving:
                upd = upd[~np.isin(upd, np.fromiter(leaving, dtype=np.int64))]
            per_el = np.where(np.isin(upd, sel_cart), 30, 26)
            adam_acc["bytes"] += int((per_el * 2 * wl.cart_len[upd].astype(np.int64) * cfg.Hkv * cfg.D).sum())
            adam_acc["steps"] += 1

    def finish():
        if rotate:
            cas.cas_swap_commit(sess.pool, stream)

    def step(record=None):
        prepare()
        if record:
            record[0].record(stream)
        sess.fwd()
        if record:
            record[1].record(stream)
        if cfg.backward:
            sess.bwd()
        if record:
            record[2].record(stream)
        if cfg.backward:
            sess.adam()
        if record:
            record[3].record(stream)
        finish()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(n_steps):
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(n_steps)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(local_rank)
        barrier()
        sampler.start()
        e0.record(stream)
        for i in range(n_steps):
            step(evs[i])
        e1.record(stream)
        barrier()
        sampler.stop_flag = True
        sampler.join(timeout=1.0)
        return e0.elapsed_time(e1), evs, sampler.summary()

    for _ in range(max(warmup, 3)):
        step()
    total_ms, evs, clocks = timed(steps)
    adam_bytes = adam_acc["bytes"] / max(adam_acc["steps"], 1)
    t_fwd = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    t_bwd = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    t_adam = float(np.mean([e[2].elapsed_time(e[3]) for e in evs]))
    ms_step = total_ms / steps

    # ---- the same steps back to back for >= sustain_s seconds: the clocks settle under the power cap
    sustained = None
    if sustain_s > 0:
        n_sus = max(steps, int(sustain_s * 1e3 / ms_step) + 1)
        s_ms, s_evs, s_clk = timed(n_sus)
        sustained = {"seconds": s_ms * 1e-3, "steps": n_sus, "ms_per_step": s_ms / n_sus,
                     "fwd_ms": float(np.mean([e[0].elapsed_time(e[1]) for e in s_evs])),
                     "bwd_ms": float(np.mean([e[1].elapsed_time(e[2]) for e in s_evs])),
                     "adam_ms": float(np.mean([e[2].elapsed_time(e[3]) for e in s_evs])), "clocks": s_clk}

    # ---- host time of one slot-table build on an IDLE blob ring (nothing in flight): median of 9
    table_ms = None
    if rank == 0:
        torch.cuda.synchronize()
        ts = []
        for i in range(9):
            t0 = time.perf_counter()
            tab = cas.cas_slot_table_build(sess.pool, wl.seq_off, rot["sel"][0], rot["sel"][1], rot["step"] - 1)
            ts.append((time.perf_counter() - t0) * 1e3)
            tab.close()
            torch.cuda.synchronize()
        table_ms = float(np.median(ts))

    # ---- c3: the swap alone (no compute on the main stream) and the host link's own pinned-copy peak
    swap_only = None
    if rotate:
        for _ in range(2):
            prepare(); finish()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b0 = rot["bytes"]
        a.record(stream)
        for _ in range(4):
            prepare(); finish()
        b.record(stream)
        barrier()
        swap_ms = a.elapsed_time(b) / 4
        per_dir = (rot["bytes"] - b0) / 4 / 2
        best = measure_host_link(torch, dev)
        swap_only = {"ms": swap_ms, "gbs_per_direction": per_dir / (swap_ms * 1e-3) / 1e9,
                     "host_link_h2d_gbs": best["h2d"], "host_link_d2h_gbs": best["d2h"],
                     "host_link_bidir_gbs_per_direction": best["both"],
                     "frac_of_host_link": per_dir / (swap_ms * 1e-3) / 1e9 / best["both"]}

    # ---- e2e: host buffers through cas_train_step_host
    e2e = None
    if cfg.backward and do_e2e:
        tdt = sess.tdt
        pin = lambda a: torch.from_numpy(a).to(tdt).pin_memory()
        hQ, hKs, hVs, hdO = pin(wl.Q), pin(wl.K_self), pin(wl.V_self), pin(wl.dO)
        hO = torch.empty_like(hQ).pin_memory()
        hdQ = torch.empty_like(hQ).pin_memory()
        hdKs, hdVs = torch.empty_like(hKs).pin_memory(), torch.empty_like(hKs).pin_memory()
        hLSE = torch.empty((sess.tab.T, cfg.Hq), dtype=torch.float32).pin_memory()
        nb = cas.cas_train_step_host_scratch_bytes(sess.pool, sess.tab, cfg.Hq)
        scratch = torch.empty(nb, dtype=torch.uint8, device=dev)
        acfg = sess.adam_cfg()

        def e2e_loop(step_fn, n):
            for _ in range(3):
                prepare()
                step_fn(sess.pool, sess.tab, cfg.Hq, hQ, hKs, hVs, hdO, sess.scale, acfg, hO, hLSE, hdQ, hdKs, hdVs,
                        scratch)
                finish()
            cas.cas_train_step_host_wait(sess.pool)
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(n):
                prepare()
                step_fn(sess.pool, sess.tab, cfg.Hq, hQ, hKs, hVs, hdO, sess.scale, acfg, hO, hLSE, hdQ, hdKs, hdVs,
                        scratch)
                finish()
            cas.cas_train_step_host_wait(sess.pool)      # the last results are in host memory when the clock stops
            b.record(stream)
            barrier()
            return a.elapsed_time(b) / n

        # the pipelined call (results of step i cross the link while step i+1 computes) is the e2e figure; the
        # per-call-complete variant (the stream waits for each call's read-back) is reported beside it
        e2e_ms = e2e_loop(cas.cas_train_step_host_async, steps)
        e2e_sync_ms = e2e_loop(cas.cas_train_step_host, steps)
        h2d = sum(t.numel() * t.element_size() for t in (hQ, hKs, hVs, hdO))
        d2h = sum(t.numel() * t.element_size() for t in (hO, hdQ, hLSE, hdKs, hdVs))
        e2e = (e2e_ms, h2d, d2h, e2e_sync_ms)

    ms_step_max, e2e_ms_max, total_flops = reduce_over_ranks(ms_step, e2e[0] if e2e else 0.0, fwd_fl + bwd_fl,
                                                             world, dev)
    line = None
    if rank == 0:
        peaks = load_peaks()
        tc = bool(cfg.dtype == "bf16" and cfg.D == 128 and args.kernels != "simt")
        dom_fl, dom_ms, dom_name = (bwd_fl, t_bwd, "attn_bwd") if cfg.backward else (fwd_fl, t_fwd, "attn_fwd")
        achieved = dom_fl / (dom_ms * 1e-3) / 1e12
        traffic = load_traffic().get(cfg_name, {}).get(dom_name)
        # denominator: the BURST bf16 peak when the timed region is short (the clocks have not settled under the power
        # cap -- what MEASURED_PEAKS' burst figure was taken at), the sustained one for a seconds-long region
        burst = total_ms < 1000.0
        pk = peaks["bf16"] if burst else peaks["bf16_sust"]
        roof = {"kernel": dom_name, "bound": "tensor", "achieved": achieved, "peak": pk,
                "unit": "TFLOP/s", "frac": achieved / pk, "traffic": traffic,
                "peak_source": peaks["src"] + (" bf16_tflops (burst: timed region %.0f ms)" % total_ms if burst else
                                               " bf16_tflops_sustained (timed region %.1f s)" % (total_ms * 1e-3)),
                "frac_of_burst_peak": achieved / peaks["bf16"], "frac_of_sustained_peak": achieved / peaks["bf16_sust"]}
        if not cfg.backward:
            # decode (c5): HBM-bound; algorithmic bytes = unique selected K+V bytes + Q + O
            uniq = sorted(set(int(x) for x in wl.sel_cart))
            kv_bytes = 2 * sum(int(wl.cart_len[c]) for c in uniq) * cfg.Hkv * cfg.D * 2
            io_bytes = 2 * int(wl.T) * cfg.Hq * cfg.D * 2
            gbs = (kv_bytes + io_bytes) / (t_fwd * 1e-3) / 1e9
            roof = {"kernel": "attn_fwd", "bound": "hbm", "achieved": gbs, "peak": peaks["hbm"], "unit": "GB/s",
                    "frac": gbs / peaks["hbm"], "traffic": traffic, "peak_source": peaks["src"] + " hbm_gbs",
                    "algorithmic_bytes": kv_bytes + io_bytes, "tflops": achieved,
                    # c5 "all loaded" (256 rows x 256 k keys per KV head) needs as long on the tensor pipe at its
                    # peak as on HBM at its peak: both fractions are reported
                    "frac_of_bf16_burst_peak": achieved / peaks["bf16"]}
        # fwd (+ fwd_combine when the tail is split), bwd_prep, bwd, dq_convert, adam  /  decode (+ decode_combine)
        fwd_split = tc and cas.cas_slot_table_fwd_split(sess.tab)[0] > 0
        n_launch = (5 + int(fwd_split)) if cfg.backward else (1 if sess.tab.B * cfg.Hq <= 256 else 2)
        adam_dram = load_traffic().get(cfg_name, {}).get("adam") if cfg.backward else None
        line = {
            "metric": METRIC, "value": total_flops / (ms_step_max * 1e-3) / 1e12, "unit": UNIT,
            "n_gpus": world, "steps": steps, "warmup": max(warmup, 3), "ms_per_step": ms_step_max,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if cfg.dtype == "bf16" else "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "Hq": cfg.Hq, "Hkv": cfg.Hkv, "D": cfg.D, "n_carts": cfg.n_carts,
                       "n_slots": cfg.n_slots, "B": cfg.B, "T": int(wl.T), "pairs_per_head": int(wl.pairs_per_head()),
                       "kernels": "tcgen05" if tc else "simt",
                       "l2": "inputs larger than L2 (pool + optimizer state > 1 GB per step)",
                       "slot_table": ("rebuilt every step (inside the timed region)" if cfg.backward else
                                      "built once before the timed region (selection fixed during generation)"),
                       "slot_table_build_host_ms": table_ms,
                       "slot_table_build_note": "median of 9 builds on an idle blob ring (host time only)",
                       "parallelism": "replicas" if world > 1 else "single"},
            "breakdown": {"fwd_ms": t_fwd, "bwd_ms": t_bwd, "adam_ms": t_adam,
                          "fwd_tflops": fwd_fl / (t_fwd * 1e-3) / 1e12,
                          "bwd_tflops": (bwd_fl / (t_bwd * 1e-3) / 1e12) if cfg.backward else None,
                          "fwd_bwd_tflops": (fwd_fl + bwd_fl) / ((t_fwd + t_bwd) * 1e-3) / 1e12,
                          "fwd_bwd_frac_of_bf16_sustained_peak": (fwd_fl + bwd_fl) / ((t_fwd + t_bwd) * 1e-3) / 1e12 / peaks["bf16_sust"],
                          "fwd_bwd_frac_of_bf16_burst_peak": (fwd_fl + bwd_fl) / ((t_fwd + t_bwd) * 1e-3) / 1e12 / peaks["bf16"],
                          "adam_gbs": (adam_bytes / (t_adam * 1e-3) / 1e9) if cfg.backward else None,
                          "adam_frac_of_hbm_peak": (adam_bytes / (t_adam * 1e-3) / 1e9 / peaks["hbm"]) if cfg.backward else None,
                          # the same launch against its REAL DRAM traffic (ncu dram__bytes_read + write of the committed
                          # capture): the fraction that is a bound -- the algorithmic one above can exceed 1
                          "adam_dram_bytes": adam_dram,
                          "adam_dram_gbs": (adam_dram / (t_adam * 1e-3) / 1e9) if adam_dram else None,
                          "adam_frac_of_hbm_peak_dram": (adam_dram / (t_adam * 1e-3) / 1e9 / peaks["hbm"]) if adam_dram else None,
                          "adam_note": ("algorithmic 30/26 B per element; a fraction above 1 means part of it is served by "
                                        "L2 (gradient rows the backward pass has just written): adam_dram_* use the DRAM "
                                        "bytes of the ncu capture in profiles/") if cfg.backward else None},
            "roofline": roof,
            "gpu_launches": steps * (n_launch + (cfg.rotate_in if rotate else 0)),
            "clocks": clocks,
        }
        if sustained:
            s_fb = (fwd_fl + bwd_fl) / ((sustained["fwd_ms"] + sustained["bwd_ms"]) * 1e-3) / 1e12
            sustained.update({"value": (fwd_fl + bwd_fl) / (sustained["ms_per_step"] * 1e-3) / 1e12,
                              "fwd_bwd_tflops": s_fb, "fwd_bwd_frac_of_bf16_sustained_peak": s_fb / peaks["bf16_sust"],
                              "bwd_tflops": bwd_fl / (sustained["bwd_ms"] * 1e-3) / 1e12 if cfg.backward else None})
            line["sustained"] = sustained
        if cfg.rotate_in > 0:
            per_step = rot["bytes"] / max(rot["step"], 1)
            line["swap"] = {"enabled": rotate, "bytes_per_step_both_directions": per_step,
                            "gbs_over_step_time": per_step / (ms_step_max * 1e-3) / 1e9,
                            "swap_alone": swap_only,
                            "note": "overlap efficiency = ms_per_step of a --no-swap run / this ms_per_step"}
        if e2e:
            line["e2e"] = {"value": total_flops / (e2e_ms_max * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": e2e_ms_max,
                           "h2d_bytes_per_step": e2e[1], "d2h_bytes_per_step": e2e[2],
                           "call": "cas_train_step_host_async (+ cas_train_step_host_wait before the clock stops)",
                           "ms_per_step_call_complete": e2e[3]}
        if do_cpu and world == 1:
            tf, desc, secs, threads = oracle_sample(wl, budget_s=12.0)
            line["cpu_baseline"] = {"value": tf, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                                    "seconds": secs, "note": "numpy float64 oracle as it stands, not tuned"}
    sess.close()
    del sess, wl
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    return line


def compact(line):
    """The part of a config's record that goes into the headline line's `extra` block."""
    b, r = line["breakdown"], line["roofline"]
    out = {"ms_per_step": line["ms_per_step"], "fwd_ms": b["fwd_ms"], "steps": line["steps"], "clocks": line["clocks"],
           "T": line["config"]["T"], "pairs_per_head": line["config"]["pairs_per_head"]}
    if b["bwd_tflops"] is not None:
        out.update({"bwd_ms": b["bwd_ms"], "adam_ms": b["adam_ms"], "fwd_tflops": b["fwd_tflops"],
                    "bwd_tflops": b["bwd_tflops"], "fwd_bwd_tflops": b["fwd_bwd_tflops"],
                    "fwd_bwd_frac_of_bf16_burst_peak": b["fwd_bwd_frac_of_bf16_burst_peak"],
                    "fwd_bwd_frac_of_bf16_sustained_peak": b["fwd_bwd_frac_of_bf16_sustained_peak"],
                    "adam_gbs": b["adam_gbs"], "adam_frac_of_hbm_peak": b["adam_frac_of_hbm_peak"]})
    else:
        out.update({"hbm_gbs_unique_kv": r["achieved"], "frac_of_hbm_peak": r["frac"], "tflops": r["tflops"]})
    if "swap" in line:
        out["swap"] = line["swap"]
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c2")
    ap.add_argument("--kernels", default="auto", choices=["auto", "simt", "tc"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-swap", action="store_true", help="c3: the same steps without rotation (overlap baseline)")
    ap.add_argument("--no-extra", action="store_true", help="headline config only (no c3/c4/c5 records, no sustained loop)")
    ap.add_argument("--ref-budget", type=float, default=8.0)
    ap.add_argument("--ref-units", type=int, default=64)
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from workloads import BASE_SEED, CONFIGS, make_workload

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, make_workload(CONFIGS[args.config], BASE_SEED))
        return

    import torch

    from paper_2606_04557_b200 import _build, cas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    _build.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    cas.cas_set_impl({"auto": 0, "simt": 1, "tc": 2}[args.kernels])
    headline = args.config == "c2" and not args.no_extra and world == 1
    line = run_config(args, args.config, args.steps, args.warmup, rank, world, local_rank, do_e2e=not args.no_e2e,
                      do_cpu=not args.no_cpu_baseline, no_swap=args.no_swap, sustain_s=3.0 if headline else 0.0)
    if headline:
        # BASELINE.json's metric spans five configs: one compact record each for the others (fewer steps; the
        # headline stays c2).  c3 twice: with rotation overlapped, and the same steps without it.
        extra = {}
        for name, kw in (("c3", {}), ("c3_no_swap", {"no_swap": True}), ("c4", {}), ("c5_all", {}), ("c5_top8", {}),
                         ("c_pages", {})):
            cname = "c3" if name.startswith("c3") else name
            st = {"c3": 8, "c4": 4}.get(cname, 30)
            rec = run_config(args, cname, st, 3, rank, world, local_rank, do_e2e=False, do_cpu=False, **kw)
            extra[name] = compact(rec)
        if "c3" in extra and "c3_no_swap" in extra:
            extra["c3"]["overlap_efficiency"] = extra["c3_no_swap"]["ms_per_step"] / extra["c3"]["ms_per_step"]
        line["extra"] = extra
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
