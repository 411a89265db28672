#!/usr/bin/env python
"""bench.py — Evoformer trunk throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2|cfg3|cfg4|tiny]

Workload at N=1 (default): BASELINE.json configs[1] ("cfg2"): 64 proteins, lengths U[50,128] padded to the 128
bucket, N_seq=128 with 0-30 % of MSA rows masked per protein, 4 Evoformer blocks, bf16 operands / fp32
accumulation / fp32 residual streams.  A *step* is one pf_evoformer_forward over that whole batch
(all nine sub-steps x 4 blocks).  value = real proteins per second over all ranks (padding does not count).

N>1 (torchrun): replicas only: every rank runs its own seeded batch, no data-path collective;
time = max over ranks, value = N * 64 * K / time ("weak").

--impl reference: the fp64 numpy oracle (oracle/) timed on the host cores on a bounded sample of the same
workload (one protein, cropped to its true length because the CPU code needs no padding, one block per step;
scaled to the workload's 4 blocks).  Rank 0 only.

The oracle is imported only by the cpu_baseline leg and --impl reference.  The CUDA path never falls back.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "evoformer_proteins_per_s"
UNIT = "proteins/s"

WORKLOADS = {
    # name: (B, S, N, n_blocks, lengths law, msa mask frac)
    "tiny": dict(B=2, S=16, N=40, n_blocks=1, lengths="cfg2small", mask=0.3,
                 desc="smoke-size batch (not a BASELINE config)"),
    "cfg2": dict(B=64, S=128, N=128, n_blocks=4, lengths="cfg2", mask=0.3,
                 desc="BASELINE.json configs[1]: 64 proteins U[50,128] -> bucket 128, N_seq=128, 4 blocks"),
    "cfg3": dict(B=1, S=512, N=384, n_blocks=48, lengths="full", mask=0.0,
                 desc="BASELINE.json configs[2]: 1 protein N_res=384 N_seq=512, 48 blocks"),
    "cfg4": dict(B=1, S=512, N=768, n_blocks=48, lengths="full", mask=0.0,
                 desc="BASELINE.json configs[3]: 1 protein N_res=768 N_seq=512, 48 blocks"),
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    source="measured (MEASURED_PEAKS.json)")
    # fallback stated in the B200 profiling guide
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback (profiling guide)")


def make_batch(ps, wl, seed):
    import numpy as np
    B, S, N = wl["B"], wl["S"], wl["N"]
    if wl["lengths"] == "cfg2":
        lengths = ps.cfg2_lengths(seed, B)
    elif wl["lengths"] == "cfg2small":
        lengths = ps.cfg2_lengths(seed, B, lo=N // 2, hi=N)
    else:
        lengths = np.full(B, N)
    msa, pair, sm, mm = ps.make_inputs(seed, B, S, N, lengths=lengths, msa_mask_frac_max=wl["mask"])
    return msa, pair, sm, mm, lengths


# ------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region (B200_PROFILING.md)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.gpu = gpu_index
        self.f = None
        self.p = None

    def start(self):
        try:
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        try:
            self.p.terminate()
            self.p.wait(timeout=5)
        except Exception:
            pass
        try:
            self.f.flush()
            self.f.seek(0)
            sm, mx, reasons = [], [], set()
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for line in self.f.read().splitlines():
                c = [x.strip() for x in line.split(",")]
                if len(c) < 8:
                    continue
                try:
                    sm.append(float(c[1]))
                    mx.append(float(c[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, c[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            if sm:
                sm.sort()
                out = {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                       "samples": len(sm)}
            self.f.close()
            os.unlink(self.f.name)
        except Exception:
            pass
        return out


# ------------------------------------------------------------------------------------------------
# the oracle timed on host cores (cpu_baseline leg and --impl reference; the only users of oracle/ here)
# ------------------------------------------------------------------------------------------------
def host_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [int(i.get("num_threads", 0)) for i in threadpool_info() if i.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count() or 1


def oracle_step(oracle, ps, wl, seed, step, blocks):
    """One bounded sample: one protein of the batch law, cropped to its true length, ONE block in fp64.
    Returns (seconds, true length)."""
    import numpy as np
    S, N = wl["S"], wl["N"]
    if wl["lengths"] in ("cfg2", "cfg2small"):
        lo = 50 if wl["lengths"] == "cfg2" else N // 2
        L = int(ps.cfg2_lengths(seed, max(wl["B"], step + 1), lo=lo, hi=N)[step % max(wl["B"], 1)])
    else:
        L = N
    msa, pair, sm, mm = ps.make_inputs(seed + 1000 + step, 1, S, L, msa_mask_frac_max=wl["mask"])
    t0 = time.perf_counter()
    m, z = oracle.evoformer_block(msa[0], pair[0], sm[0], mm[0], blocks[0])
    dt = time.perf_counter() - t0
    assert np.isfinite(m).all() and np.isfinite(z).all()
    return dt, L


def run_reference(args, wl, wl_name):
    """--impl reference: the fp64 oracle on the host cores; K timed samples after W warm-up samples."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    import pf_synth as ps
    blocks = ps.make_weights(7, 1, bf16_weights=True)
    for s in range(args.warmup):
        oracle_step(oracle, ps, wl, 11, s, blocks)
    t = 0.0
    for s in range(args.steps):
        dt, _ = oracle_step(oracle, ps, wl, 11, args.warmup + s, blocks)
        t += dt
    per_protein = t / args.steps * wl["n_blocks"]           # one block timed per sample; the workload has n_blocks
    value = 1.0 / per_protein
    cores = host_threads()
    sample = (f"{args.steps} samples, each 1 protein of the {wl_name} length law cropped to its true length, "
              f"N_seq={wl['S']}, 1 of {wl['n_blocks']} blocks in fp64 numpy; seconds scaled x{wl['n_blocks']}")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl_name, "desc": wl["desc"], "B": wl["B"], "N_seq": wl["S"], "N_res": wl["N"],
                   "n_blocks": wl["n_blocks"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def cpu_baseline(wl, wl_name, budget_s=25.0):
    import oracle
    import pf_synth as ps
    blocks = ps.make_weights(7, 1, bf16_weights=True)
    t, n, lens = 0.0, 0, []
    while t < budget_s and n < 8:
        dt, L = oracle_step(oracle, ps, wl, 11, n, blocks)
        t += dt
        n += 1
        lens.append(L)
        if dt > budget_s / 2:
            break
    per_protein = t / n * wl["n_blocks"]
    return {"value": 1.0 / per_protein, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
            "sample": (f"{n} protein(s) of the {wl_name} length law (true lengths {lens}, unpadded), N_seq={wl['S']}, "
                       f"1 of {wl['n_blocks']} blocks each in fp64 numpy, {t:.1f} s total; scaled x{wl['n_blocks']} blocks"),
            "seconds_per_protein_block": t / n}


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
KIND_BOUND = {"gemm": "tensor", "attn_core": "tensor", "tri_einsum": "tensor", "opm_core": "tensor",
              "ln_rows": "hbm", "ln_channels": "hbm", "ln_gemm": "hbm", "transition": "tensor"}


def roofline_from_profile(prof, peaks, n_steps, wl_name):
    """Dominant kernel kind (largest share of device time) -> roofline object; plus the per-kind table."""
    total_ms = sum(v["ms"] for v in prof.values()) or 1e-9
    table = {}
    for k, v in prof.items():
        if v["launches"] == 0:
            continue
        sec = v["ms"] * 1e-3
        table[k] = {"launches_per_step": v["launches"] / n_steps, "ms_per_step": v["ms"] / n_steps,
                    "share": v["ms"] / total_ms, "tflops": v["flops"] / sec / 1e12 if sec > 0 else 0.0,
                    "gbs": v["bytes"] / sec / 1e9 if sec > 0 else 0.0}
    top = max(table, key=lambda k: table[k]["share"])
    bound = KIND_BOUND.get(top, "hbm")
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")       # dram bytes per launch from the committed ncu capture
    if os.path.exists(tp):
        try:
            with open(tp) as f:
                traffic = json.load(f).get(wl_name, {}).get(top)   # captured per workload (launch sizes differ)
        except Exception:
            traffic = None
    if bound == "tensor":
        peak, unit, ach = peaks["bf16_tflops_sustained"], "TFLOP/s", table[top]["tflops"]
        peak_name = "bf16_tflops_sustained"
    else:
        peak, unit, ach = peaks["hbm_gbs"], "GB/s", table[top]["gbs"]
        peak_name = "hbm_gbs"
    roof = {"kernel": top, "bound": bound, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
            "traffic": traffic, "peak_source": f"{peak_name}, {peaks['source']}", "share_of_step": table[top]["share"]}
    return roof, table


def per_bucket_sweep(h, pf, ps, torch, dev, nb, peaks, n_proteins=2000, S=512, cap=48):
    """BASELINE.json metric: proteins/s and TFLOP/s per length bucket (configs[4]: lengths R10, buckets {64..320}, N_seq=512,
    random msa_mask R11, 48 blocks).  The length-bucketing scheduler (pf_sched_*) cuts the protein list into batches; ONE
    batch per bucket is timed on the GPU (nb blocks, CUDA events) and the 48-block, whole-list figures are derived from it."""
    import numpy as np
    lengths = ps.cfg5_lengths(5, n_proteins)
    sched = pf.Scheduler(list(ps.CFG5_BUCKETS), 16 << 30, S)
    for i, L in enumerate(lengths):
        sched.add(i, int(L))
    per_bucket, order = {}, []
    for ids, lens, bucket in sched.batches(cap):
        e = per_bucket.setdefault(bucket, {"proteins": 0, "batches": 0, "first": None})
        e["proteins"] += len(ids)
        e["batches"] += 1
        if e["first"] is None or len(ids) > len(e["first"][1]):
            e["first"] = (ids, lens)
        if bucket not in order:
            order.append(bucket)
    sched.close()
    out, total_s = [], 0.0
    g = torch.Generator(device=dev).manual_seed(55)
    for bucket in order:
        e = per_bucket[bucket]
        ids, lens = e["first"]
        B, N = len(ids), bucket
        sm = np.zeros((B, N), np.float32)
        for b, L in enumerate(lens):
            sm[b, :L] = 1.0
        mm = np.ones((B, S), np.float32)
        r = ps.rng(77, bucket)
        for b in range(B):                                           # R11: 0-30 % of the MSA rows masked, never row 0
            k = int(r.uniform(0.0, 0.3) * S)
            mm[b, 1 + r.choice(S - 1, size=k, replace=False)] = 0.0
        m = torch.randn(B, S, N, 256, device=dev, generator=g)
        z = torch.randn(B, N, N, 128, device=dev, generator=g)
        smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
        h.forward(m, z, smd, mmd, nb)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 2
        e0.record()
        for _ in range(reps):
            h.forward(m, z, smd, mmd, nb)
        e1.record()
        torch.cuda.synchronize()
        ms_block = e0.elapsed_time(e1) / reps / nb
        ok = bool(torch.isfinite(m).all().item() and torch.isfinite(z).all().item())
        del m, z
        flops_block = ps.gemm_flops_per_block(S, N) * B
        s48 = ms_block * 48e-3                                       # seconds for this batch through 48 blocks
        total_s += s48 / B * e["proteins"]
        out.append({"bucket": bucket, "B": B, "proteins_in_list": e["proteins"], "batches_in_list": e["batches"],
                    "mean_len": float(np.mean(lens)), "ms_per_block": ms_block,
                    "tflops_padded": flops_block / (ms_block * 1e-3) / 1e12,
                    "frac_bf16_sustained": flops_block / (ms_block * 1e-3) / 1e12 / peaks["bf16_tflops_sustained"],
                    "proteins_per_s_48_blocks": B / s48, "outputs_finite": ok})
    return {"workload": f"cfg5-style: {n_proteins} proteins, lengths R10, buckets {list(ps.CFG5_BUCKETS)}, N_seq={S}, "
                        f"msa_mask R11; batches by pf_sched (16 GB budget, cap {cap}); one batch per bucket timed over "
                        f"{nb} blocks, 48-block figures derived",
            "buckets": out, "sweep_seconds_48_blocks_derived": total_s,
            "proteins_per_hour_derived": n_proteins / total_s * 3600.0}


def run_ours(args, wl, wl_name):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_2111_06340_b200 as pf
    import pf_synth as ps

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    pf.lib()                                                     # fail loudly if the extension is not built

    dtype = pf.PF_F32 if args.dtype == "f32" else pf.PF_BF16
    B, S, N, nb = wl["B"], wl["S"], wl["N"], wl["n_blocks"]
    # the weights of nb distinct blocks (R8/R15); for 48-block workloads the same seeded recipe
    blocks = ps.make_weights(7, nb, bf16_weights=(dtype != pf.PF_F32))
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, dtype))
    del blocks
    msa, pair, sm, mm, lengths = make_batch(ps, wl, 100 + rank)
    n_prot, n_res = B, int(np.sum(lengths))
    m0 = torch.from_numpy(msa).pin_memory()
    z0 = torch.from_numpy(pair).pin_memory()
    smh, mmh = torch.from_numpy(sm).pin_memory(), torch.from_numpy(mm).pin_memory()
    m, z = m0.to(dev), z0.to(dev)
    smd, mmd = smh.to(dev), mmh.to(dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # first call (workspace growth, module load) vs steady state — the analogue of the paper's per-model compile
    barrier()
    t0 = time.perf_counter()
    h.forward(m, z, smd, mmd, nb)
    torch.cuda.synchronize()
    first_call_ms = (time.perf_counter() - t0) * 1e3
    launches_per_step = h.last_launch_count()
    for _ in range(max(args.warmup - 1, 0)):
        h.forward(m, z, smd, mmd, nb)

    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        h.forward(m, z, smd, mmd, nb)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    # per-kernel pass: the same steps with every launch bracketed by events on the launch stream
    n_prof = max(1, min(args.steps, 3))
    h.set_profiling(True)
    for _ in range(n_prof):
        h.forward(m, z, smd, mmd, nb)
    torch.cuda.synchronize()
    prof = h.get_profile()
    h.set_profiling(False)
    clocks = sampler.stop() if rank == 0 else None
    finite = bool(torch.isfinite(m).all().item() and torch.isfinite(z).all().item())

    # end to end through the public host-buffer call: pinned host -> device, forward, device -> pinned host
    n_e2e = max(1, min(args.steps, 3))
    mh, zh = m0.clone().pin_memory(), z0.clone().pin_memory()
    h.forward_host(mh, zh, smh, mmh, nb)                          # warm-up (staging buffers)
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        h.forward_host(mh, zh, smh, mmh, nb)                      # synchronises the stream before returning
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    h2d = m0.numel() * 4 + z0.numel() * 4 + smh.numel() * 4 + mmh.numel() * 4
    d2h = m0.numel() * 4 + z0.numel() * 4

    t = torch.tensor([ms, e2e_s * 1e3], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, e2e_ms = float(t[0]), float(t[1])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks = load_peaks()
    ms_per_step = ms / args.steps
    value = world * n_prot * args.steps / (ms * 1e-3)
    flops_step = ps.gemm_flops_per_block(S, N) * nb * B          # padded FLOPs: what the GPU executes
    roof, table = roofline_from_profile(prof, peaks, n_prof, wl_name)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": wl_name, "desc": wl["desc"], "B": B, "N_seq": S, "N_res": N, "n_blocks": nb,
                   "parallelism": f"replicas x{world}", "l2": "inputs larger than L2 (msa+pair residual streams "
                   f"{(m0.numel() + z0.numel()) * 4 / 1e6:.0f} MB per step)", "path": args.dtype,
                   "masked_work": "128-row tiles, attention rows and key tiles that are entirely masked are skipped; "
                                  "roofline / kernels count executed work only, tflops_padded counts the padded bucket"},
        "residues_per_s": world * n_res * args.steps / (ms * 1e-3),
        "tflops_padded": world * flops_step / (ms_per_step * 1e-3) / 1e12,
        "tflops_frac_of_bf16_sustained": world * flops_step / (ms_per_step * 1e-3) / 1e12 / peaks["bf16_tflops_sustained"] / world,
        # GEMM FLOPs actually executed (fully masked tiles / rows / key tiles are skipped) per GPU
        "tflops_executed": sum(v["flops"] for v in prof.values()) / n_prof / (ms_per_step * 1e-3) / 1e12,
        "first_call_ms": first_call_ms, "steady_ms": ms_per_step, "outputs_finite": finite,
        "e2e": {"value": world * n_prot * n_e2e / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": n_e2e, "api": "pf_evoformer_forward_host (pinned host buffers)"},
        "gpu_launches": int(launches_per_step * args.steps),
        "clocks": clocks, "roofline": roof, "kernels": table,
        "paper_context": "ParaFold: ~20,000 50-res proteins / 5.4 h on 16 V100 (whole model), 13.8x from compile reuse; "
                         "no Evoformer-only number (BASELINE.md)",
    }
    if world == 1 and not args.no_buckets:
        del m, z, mh, zh
        torch.cuda.empty_cache()
        line["per_bucket"] = per_bucket_sweep(h, pf, ps, torch, dev, nb, peaks)
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(wl, wl_name)
    print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(WORKLOADS))
    ap.add_argument("--dtype", default="bf16", choices=["bf16", "f32"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-buckets", action="store_true", help="skip the per-length-bucket sweep (cfg5-style)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    wl = WORKLOADS[args.workload]
    if args.impl == "reference":
        return run_reference(args, wl, args.workload)
    return run_ours(args, wl, args.workload)


if __name__ == "__main__":
    sys.exit(main())
