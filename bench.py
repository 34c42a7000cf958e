#!/usr/bin/env python
"""bench.py -- full-config samples/sec (with log q) of the FlashVAN hot path on B200.

One "step" = one pass of the whole hot path over one batch of the workload:
    fv_sample (Alg. 2)  ->  fv_log_prob (Alg. 1)  ->  fv_energy_*  ->  fv_free_energy (Eq. 5)
`value` = samples/s with the uniforms already resident in HBM; `e2e` = the same through the
public binding with HOST buffers (pinned uniforms in, spins/logq/E/F out) inside the timed region.
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
"""
import argparse
import csv
import hashlib
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

from paper_2606_22984_b200 import workloads as W  # noqa: E402

METRIC = "full-config samples/sec (with log q)"
UNIT = "samples/s"


def parse():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=3)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--workload", default="cfg5", choices=list(W.CONFIGS))
    p.add_argument("--batch", type=int, default=0, help="override the workload's batch (debug only)")
    p.add_argument("--cpu-samples", type=int, default=0, help="oracle samples for cpu_baseline (0 = 2 x cores)")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--no-other-configs", action="store_true", help="skip the short cfg1-cfg4 / W_O timings after the headline")
    return p.parse_args()


def sampler_source_hash():
    """sha256 over the sources of the fv_sample kernels: a committed ncu figure is only quoted while they are unchanged."""
    h = hashlib.sha256()
    for f in ("fv_chain.cu", "fv_decode.cu", "fv_decode_tc.cu", "fv_ring.cuh", "fv_device.cuh", "fv_umma.cuh"):
        h.update(open(os.path.join(ROOT, "paper_2606_22984_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload, batch, kind="ring"):
    """DRAM and L2->SM bytes of the fv_sample launch from the committed ncu capture: the row of
    profiles/sampler_traffic.csv for this (workload, batch), quoted only if it was captured on the
    sampler sources as they are now.  Returns (dict or None, note)."""
    path = os.path.join(ROOT, "profiles", "sampler_traffic.csv")
    if not os.path.exists(path):
        return None, "no profiles/sampler_traffic.csv"
    rows = [r for r in csv.DictReader(l for l in open(path) if not l.startswith("#"))
            if r["workload"] == workload and int(r["batch"]) == batch and r["sampler"] == kind]
    if not rows:
        return None, f"no ncu capture of {workload} at batch {batch} in profiles/sampler_traffic.csv"
    r = rows[-1]
    if r["source_sha256_16"] != sampler_source_hash():
        return None, (f"the capture in profiles/sampler_traffic.csv (sources {r['source_sha256_16']}, {r['capture']}) predates "
                      f"the current sampler sources ({sampler_source_hash()})")
    return {"dram_bytes": float(r["dram_bytes"]), "l2_to_sm_bytes": float(r["l2_to_sm_bytes"]), "kernel": r["kernel"],
            "capture": r["capture"]}, "ncu --set full, one launch: " + r["capture"]


def algorithmic_kv_bytes_per_sample(w, rowptr):
    """KV rows named by the mask only: read sum_t nnz(t) rows + write N rows,
    each 2d bf16 = 4d bytes, per layer."""
    row_bytes = 4 * w.d_model
    return int(rowptr[-1]) * w.n_layers * row_bytes, w.n_sites * w.n_layers * row_bytes


def load_peaks():
    """(HBM GB/s, sustained bf16 TFLOP/s, source): MEASURED_PEAKS.json, else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            j = json.load(open(path))
            return float(j["hbm_gbs"]), float(j["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, 1400.0, "fallback (B200_PROFILING.md: 6.65 TB/s, ~1.4 PFLOP/s sustained)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        rows = [l.split(", ") for t, l in self.lines if t0 <= t <= t1] or [l.split(", ") for _, l in self.lines[-3:]]
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.strip().lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_step(w, inp, n):
    """The oracle as it stands on n samples of the workload: sample + log_prob + energy + F_q."""
    from oracle import oracle as O
    u = inp["uniforms"][:n]
    spins, lq, _ = O.sample(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"], u)
    lq2, _ = O.log_prob(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"], spins)
    if w.model == "sk":
        E = O.energy_dense(spins, inp["J"])
    else:
        E = O.energy_csr(spins, inp["bond_rowptr"], inp["bond_col"], inp["bond_val"])
    return O.free_energy(E, lq2, w.betas[0])


def config_of(w, B, n_gpus):
    return {"workload": f"{w.name}: {'SK' if w.model == 'sk' else str(w.dim) + 'D EA L=' + str(w.L)} N={w.n_sites}, "
                        f"{w.n_layers} layers, d={w.d_model}, {w.n_heads} heads, {w.coupling} couplings, "
                        f"mask window {w.window}", "batch_per_gpu": B, "global_batch": B * n_gpus,
            "n_sites": w.n_sites, "parallelism": f"dp{n_gpus} (independent sample shards, no data-path collective)",
            "l2_policy": "inputs_exceed_l2 (KV pool >> 126 MB; uniforms/spins rewritten every step)"}


def run_reference(args):
    """--impl reference: the fp64 oracle on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    w = W.CONFIGS[args.workload]
    cores = O.n_threads()
    n = args.cpu_samples or cores                       # one sample per thread per step
    inp = W.make_all(w, batch=n)
    for _ in range(min(args.warmup, 1)):                # one warm-up pass is enough for a CPU program
        oracle_step(w, inp, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(w, inp, n)
    dt = time.perf_counter() - t0
    v = n * args.steps / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, workloads.py)",
        "config": config_of(w, args.batch or w.batch, args.gpus),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{n} samples of {w.name} per step (sample + log_prob + energy + F_q)"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per GPU, NCCL),
    exactly as the driver's torchrun line would, and pass rank 0's JSON line through."""
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "INFO"))
    raise SystemExit(subprocess.call(cmd, env=env))


def time_other_config(fv, torch, name, w, B, steps=3, seed_u=None, mask=None):
    """Short timing of fv_sample / fv_log_prob on another BASELINE config (the headline's model is closed by
    then): CUDA events, one warm-up pass, `steps` timed passes."""
    inp = W.make_all(w, batch=B) if seed_u is None else W.make_all(w, batch=B, u_seed=seed_u)
    if mask is not None:
        inp["mask_rowptr"], inp["mask_col"] = mask
    model = fv.create_model(w, inp["weights"], inp["mask_rowptr"], inp["mask_col"], inp["posemb"], B)
    u = torch.from_numpy(np.ascontiguousarray(inp["uniforms"])).cuda()
    spins = torch.empty((B, w.n_sites), dtype=torch.int8, device="cuda")
    logq = torch.empty(B, dtype=torch.float32, device="cuda")
    lq2 = torch.empty(B, dtype=torch.float32, device="cuda")
    model.sample(u, out=(spins, logq)); model.log_prob(spins, out=lq2)
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps + 1)]
    for k in range(steps):
        ev[2 * k].record(); model.sample(u, out=(spins, logq))
        ev[2 * k + 1].record(); model.log_prob(spins, out=lq2)
    ev[2 * steps].record()
    torch.cuda.synchronize()
    ts = sum(ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(steps)) / steps
    tl = sum(ev[2 * k + 1].elapsed_time(ev[2 * k + 2]) for k in range(steps)) / steps
    chain_gap = float((logq - lq2).abs().max().item())
    kv_window, kv_pool = model.kv_window, model.kv_bytes
    model.close()
    rd, wr = algorithmic_kv_bytes_per_sample(w, inp["mask_rowptr"])
    peak, _, _ = load_peaks()
    kv_us = 1e6 * (rd + wr) * B / w.n_sites / (peak * 1e9)           # KV bytes of one site step at the HBM peak
    out = {"workload": name, "batch": B, "fv_sample_ms": ts, "fv_log_prob_ms": tl, "samples_per_s": B / ((ts + tl) * 1e-3),
           "us_per_site_step": 1e3 * ts / w.n_sites, "algorithmic_kv_frac_of_hbm_peak": (rd + wr) * B / (ts * 1e-3) / 1e9 / peak,
           "max_abs_logq_sample_vs_log_prob": chain_gap}
    if kv_window:
        out["kv_window_rows"], out["kv_pool_bytes"] = kv_window, kv_pool
    out["bound"] = "latency (KV traffic of a site step is %.1f us at the HBM peak)" % kv_us if kv_us < 10.0 else "hbm"
    return out


def run_ours(args):
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    import torch
    import torch.distributed as dist
    from paper_2606_22984_b200 import binding as fv
    from paper_2606_22984_b200 import build as fvbuild
    from paper_2606_22984_b200 import shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not os.path.exists(fv._LIB_PATH):
        if local == 0:
            fvbuild.build()
        if world > 1:
            dist.barrier()

    w = W.CONFIGS[args.workload]
    B = args.batch or w.batch
    inp = W.make_all(w, batch=B, u_seed=W.SEED_U + 1000 * rank)       # each rank: its own sample shard
    model = fv.create_model(w, inp["weights"], inp["mask_rowptr"], inp["mask_col"], inp["posemb"], B)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    u = d(inp["uniforms"])
    if w.model == "sk":
        J = d(inp["J"])
    else:
        brp, bcol, bval = d(inp["bond_rowptr"]), d(inp["bond_col"]), d(inp["bond_val"])
    N = w.n_sites
    spins = torch.empty((B, N), dtype=torch.int8, device="cuda")
    logq = torch.empty(B, dtype=torch.float32, device="cuda")
    logq_tf = torch.empty(B, dtype=torch.float32, device="cuda")
    E = torch.empty(B, dtype=torch.float32, device="cuda")
    F = torch.empty(4, dtype=torch.float64, device="cuda")
    T = 1.0 / w.betas[0]

    def step(evs=None):
        if evs: evs[0].record()
        model.sample(u, out=(spins, logq))
        if evs: evs[1].record()
        model.log_prob(spins, out=logq_tf)
        if evs: evs[2].record()
        if w.model == "sk":
            fv.energy_dense(spins, J, out=E)
        else:
            fv.energy_csr(spins, brp, bcol, bval, w.coupling == "pm1", out=E)
        fv.free_energy(E, logq_tf, T, out=F)
        if evs: evs[3].record()

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sync_all()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = fv.launch_count()
    fv.profile(True)                                  # per-kernel events (library side) during the timed region
    t0 = time.perf_counter()
    for k in range(args.steps):
        step(evs[k])
    sync_all()
    t1 = time.perf_counter()
    kernel_ms = fv.profile(False)
    launches = fv.launch_count() - launches0
    clocks = sampler.stop(t0, t1) if sampler else None
    total_ms = evs[0][0].elapsed_time(evs[-1][3])
    t_sample = sum(e[0].elapsed_time(e[1]) for e in evs) / args.steps
    t_logp = sum(e[1].elapsed_time(e[2]) for e in evs) / args.steps
    t_rest = sum(e[2].elapsed_time(e[3]) for e in evs) / args.steps
    total_ms = shard.max_over_ranks(total_ms, device="cuda")          # multi-GPU time = max over ranks
    Fq_mean, Fq_std = shard.merge_free_energy(F)                      # the one data exchange: fv_free_energy's outputs
    ms_per_step = total_ms / args.steps
    value = world * B / (ms_per_step * 1e-3)

    # ---- end to end through the public binding with HOST buffers -----------------------------
    u_host = torch.from_numpy(inp["uniforms"]).pin_memory()
    spins_host = torch.empty((B, N), dtype=torch.int8).pin_memory()
    lq_host = torch.empty(B, dtype=torch.float32).pin_memory()
    E_host = torch.empty(B, dtype=torch.float32).pin_memory()
    F_host = torch.empty(4, dtype=torch.float64).pin_memory()

    def e2e_step():
        u.copy_(u_host, non_blocking=True)
        step()
        spins_host.copy_(spins, non_blocking=True)
        lq_host.copy_(logq_tf, non_blocking=True)
        E_host.copy_(E, non_blocking=True)
        F_host.copy_(F, non_blocking=True)

    e2e_step()
    sync_all()
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ea.record()
    for _ in range(args.steps):
        e2e_step()
    eb.record()
    sync_all()
    e2e_ms = ea.elapsed_time(eb)
    e2e_ms = shard.max_over_ranks(e2e_ms, device="cuda")
    e2e_value = world * B / (e2e_ms / args.steps * 1e-3)
    h2d = u_host.numel() * 4
    d2h = spins_host.numel() + 4 * B + 4 * B + 32
    F_val = F_host.clone().numpy()
    spins_np = spins_host.numpy().copy()
    sampler_kind = model.sampler_kind(B)
    model.close()

    if rank == 0:
        rd, wr = algorithmic_kv_bytes_per_sample(w, inp["mask_rowptr"])
        peak, tf_peak, peak_src = load_peaks()
        k_sample_ms = kernel_ms["sample"][0] / max(1, kernel_ms["sample"][1])      # library-side events, kernel only
        achieved = (rd + wr) * B / (k_sample_ms * 1e-3) / 1e9
        traffic, traffic_note = ncu_traffic(w.name, B, sampler_kind)
        ffn_ms = kernel_ms["lp_ffn"][0] / max(1, kernel_ms["lp_ffn"][1])
        ffn_flop = 2.0 * B * N * (w.d_model * 4 * w.d_model) * 2
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16 GEMM operands + bf16 KV cache, fp32 accumulate/softmax/LN",
            "data": "synthetic (seeded couplings, random-init N(0,0.02) weights; workloads.py)",
            "config": config_of(w, B, world),
            "phases_ms": {"fv_sample": t_sample, "fv_log_prob": t_logp, "energy+free_energy": t_rest},
            "kernel_ms_per_launch": {k: (v[0] / v[1] if v[1] else None) for k, v in kernel_ms.items()},
            "us_per_site_step": 1e3 * t_sample / N,
            "F_q": {"mean": Fq_mean, "std": Fq_std, "per_spin": Fq_mean / N,
                    "rank0_kernel": [float(F_val[0]), float(F_val[1])]},
            "roofline": {"kernel": {"chain": "fv_chain_kernel (fv_sample: layer-pipelined clusters, weights resident in TMEM / shared memory)",
                                    "ring-tc": "fv_decode_tc_kernel (fv_sample: persistent KV-ring sampler, projections on tcgen05)",
                                    "ring": "fv_decode_kernel (fv_sample: persistent KV-ring sampler, projections on mma.sync)"}[sampler_kind],
                         "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "achieved_is": "ALGORITHMIC KV bytes (rows the mask names: read + append) / kernel duration; L2 hits "
                                        "between consecutive steps make the DRAM bytes smaller, see dram_*",
                         "duration_ms": k_sample_ms, "frac_of_nominal_8TBs": achieved / 8000.0, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": (rd + wr) * B,
                         "traffic": traffic["dram_bytes"] if traffic else None,
                         "l2_to_sm_bytes": traffic["l2_to_sm_bytes"] if traffic else None,
                         "dram_gbs": traffic["dram_bytes"] / (k_sample_ms * 1e-3) / 1e9 if traffic else None,
                         "dram_frac": traffic["dram_bytes"] / (k_sample_ms * 1e-3) / 1e9 / peak if traffic else None,
                         "traffic_source": traffic_note},
            "roofline_gemm": {"kernel": "lp_ffn_kernel (fv_log_prob: fused LN2 -> W1 -> GELU -> W2 -> residual, tcgen05/TMEM)",
                              "bound": "tensor", "achieved": ffn_flop / (ffn_ms * 1e-3) / 1e12 if ffn_ms else None,
                              "peak": tf_peak, "unit": "TFLOP/s",
                              "frac": ffn_flop / (ffn_ms * 1e-3) / 1e12 / tf_peak if ffn_ms else None,
                              "flop_per_launch": ffn_flop, "duration_ms": ffn_ms, "launches_timed": kernel_ms["lp_ffn"][1],
                              "peak_source": peak_src + " bf16_tflops_sustained (the launches sit inside a long step)"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(launches), "clocks": clocks,
        }
        if world == 1 and not args.no_other_configs:
            others = []
            for name in ("cfg1", "cfg2", "cfg3", "cfg4"):
                wo = W.CONFIGS[name]
                others.append(time_other_config(fv, torch, name, wo, wo.batch))
                if name == "cfg3":                              # second temperature: its own uniforms (reading A18)
                    others.append(time_other_config(fv, torch, "cfg3 (beta = 1.5 seed)", wo, wo.batch, seed_u=W.SEED_U + 1))
            import dataclasses
            others.append(time_other_config(fv, torch, "cfg5 with W_O (has_wo = 1, reading A8)",
                                            dataclasses.replace(w, has_wo=1), B))
            # the same model at four times BASELINE's batch (28 instead of 7 samples per SM share one weight stream), and
            # the band-only fast path: the open-boundary 64 x 64 lattice's exact mask, previous L spins
            # (PAPER.md:549), whose KV lives in a ring-buffer window of W + 1 rows -- which is what lets the batch grow
            others.append(time_other_config(fv, torch, "cfg5 at B = 4096 (28 samples per SM)", w, 4 * B))
            band = W.band_mask_csr(w.n_sites, w.L)
            others.append(time_other_config(fv, torch, "cfg5 model, pure band W = 64 (Eq. S1), B = 1024", w, B, mask=band))
            others.append(time_other_config(fv, torch, "cfg5 model, pure band W = 64 (Eq. S1), B = 4096", w, 4 * B, mask=band))
            out["other_configs"] = others
        if world == 1 and not args.no_cpu_baseline:
            from oracle import oracle as O
            cores = O.n_threads()
            n = args.cpu_samples or 2 * cores
            t0 = time.perf_counter()
            oracle_step(w, W.make_all(w, batch=n), n)
            dt = time.perf_counter() - t0
            out["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"{n} samples of {w.name} (sample + log_prob + energy + F_q), {dt:.1f} s"}
            # the north star's counters on the GPU's own samples of the last timed step: spins against
            # (u < p_oracle) re-synchronised on the GPU's spins, near ties counted
            idx = np.unique(np.linspace(0, B - 1, n).astype(np.int64))
            _, cp_o = O.log_prob(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"], spins_np[idx])
            uu = inp["uniforms"][idx].astype(np.float64)
            mism = spins_np[idx] != np.where(uu < cp_o, 1, -1)
            tie = np.abs(uu - cp_o) < 2e-3
            out["parity_counters"] = {"samples_checked": int(len(idx)), "sites_checked": int(tie.size),
                                      "near_tie_sites": int(tie.sum()), "flips_in_tie_band": int((mism & tie).sum()),
                                      "flips_outside_tie_band": int((mism & ~tie).sum())}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
