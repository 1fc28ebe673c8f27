#!/usr/bin/env python
"""bench.py -- UniFrac all-pairs hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload emp|large|medium|small|tiny]
                    [--impl ours|reference] [--no-cpu-baseline] [--no-e2e] [--no-emp] [--replicas]

A "step" is one pass of the whole hot path (plan, embedding, stripe accumulation, finalize) for
every variant the workload lists (unweighted and weighted-normalized), inputs resident in HBM.
metric = dense-equivalent sample-pair x branch updates per second  (BASELINE.json "metric"):
         sum over the step's calls of P * B_emb, divided by the step time.
Prints ONE JSON line (rank 0).  The default workload is Large (N = 50,000); before it the EMP-shaped workload
(N = 25,000) runs for max(1, steps/4) steps and is reported under "wall_emp" (BASELINE.json's metric names both sizes).
N > 1: one process per GPU computing disjoint SHARDS of one matrix (unifrac_dm_shard) followed, inside the timed
region, by the NCCL merge of the shard buffers (strong scaling); --replicas gives independent replicas instead (weak).
Barrier + max-over-ranks timing either way.
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

from paper_2107_05397_b200 import synth  # noqa: E402

METRIC = "unifrac_dense_equivalent_pair_branch_updates_per_s"
UNIT = "updates/s"
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965        # B200_PROFILING.md / MEASURED_PEAKS.json
ALU_PEAK_TFLOPS = SM_COUNT * FP32_LANES * SM_MAX_GHZ / 1e3    # FADD/FMNMX-class lane-ops (not FMA-doubled)
# fallbacks when unifrac_measure_rates is not run (values it measured on this pool's B200: 8.84 shared-memory atomic
# lane-ops/clk/SM, independent of bank conflicts; 1.94e11 L2-resident scattered fp32 REDs/s)
SMEM_ATOMIC_PER_S, L2_RED_PER_S = 8.84 * SM_COUNT * SM_MAX_GHZ * 1e9, 1.94e11

# dram__bytes_read.sum + dram__bytes_write.sum per launch, copied from the ncu --set full captures summarised in the file
# TRAFFIC_SOURCE names (default flags, seed 0; k_midg / k_mid: mean of the unweighted and the weighted launch; k_mid and k_zone:
# the earlier captures of section 2, for runs with UNIFRAC_B200_MID_GROUPS=0 / --flags 512); not measured by this
# run -- other workloads and kernels that changed since the capture report null
TRAFFIC_SOURCE = "profiles/r02_summary.md section 0 (ncu --set full captures of the final kernels of the round, Large, seed 0)"
NCU_TRAFFIC_BYTES = {"large": {"k_dense16": 80.5e9, "k_gram": 260.8e9, "k_midg": 187.3e9, "k_mid": 240.1e9, "k_zone": 307.1e9}}

WORKLOADS = {   # name -> (variants, precision)    BASELINE.json:7-11
    "tiny": ((0, 1), 1), "small": ((0, 1), 1), "medium": ((0,), 0), "emp": ((0, 1), 0), "large": ((0, 1), 0),
}


def clocks_sampler(stop, out, gpu_index):
    q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    try:
        pr = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={q}", "--format=csv,noheader,nounits",
                               "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
    except Exception:
        return
    def rd():
        for line in pr.stdout:
            out.append(line.strip())
    th = threading.Thread(target=rd, daemon=True)
    th.start()
    stop.wait()
    pr.terminate()
    th.join(timeout=2)


def summarize_clocks(lines):
    sm, mx, reasons = [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for ln in lines:
        f = [x.strip() for x in ln.split(",")]
        if len(f) < 7:
            continue
        try:
            sm.append(float(f[0])); mx.append(float(f[1]))
        except ValueError:
            continue
        for k, nm in enumerate(names):
            if f[3 + k].lower().startswith("active"):
                reasons.add(nm)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
    busy = sorted(sm)[len(sm) // 2:]           # upper half = under load
    return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def reduce_over_ranks(ms_local: float, updates_local: float, world: int, device=None):
    """Max of the per-rank step time and sum of the per-rank updates (replicas: no data-path collective)."""
    if world <= 1:
        return ms_local, updates_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([updates_local], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def rank_seed(seed: int, rank: int) -> int:
    """Replica r works on its own seeded problem."""
    return seed + rank


def oracle_leg(p, variants, budget_s, seed=0):
    """Times the oracle's pair-list driver, as it stands, on a bounded seeded sample of pairs."""
    from oracle import oracle
    def run(npairs, variant):
        pairs = synth.sample_pairs(p.n_samples, npairs, seed=seed)
        t = time.perf_counter()
        oracle.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, pairs)
        return time.perf_counter() - t
    probe = max(200, min(2000, p.n_pairs))
    t_probe = run(probe, variants[0])
    per_pair = t_probe / probe
    npairs = int(max(probe, min(p.n_pairs, budget_s / max(per_pair, 1e-9) / len(variants))))
    npairs = min(npairs, 2_000_000)
    total_t, total_pairs = 0.0, 0
    for v in variants:
        total_t += run(npairs, v)
        total_pairs += npairs
    return dict(pairs=total_pairs, seconds=total_t, cores=oracle.num_threads(),
                sample=f"{npairs} seeded pairs per variant x {len(variants)} variant(s), pair-list driver "
                       f"(includes building the per-sample branch lists)")


def cpu_model_name():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def variant_name(v):
    return "unweighted" if v == 0 else "weighted_normalized"


def wall_of(all_stats, variants, n_nodes, nnz):
    """Per-variant wall time split and derived figures."""
    per_variant = {}
    for k, v in enumerate(variants):
        ss = [st[k] for st in all_stats]
        mean = lambda key: float(np.mean([s[key] for s in ss]))
        s0 = ss[0]
        t_a5 = (mean("ms_tail") + mean("ms_mid") + mean("ms_stripe")) * 1e-3
        n_words = (s0["n_samples"] + 31) // 32 if "n_samples" in s0 else 0
        # algorithmic bytes of a-1 .. a-4 (estimate from the list sizes): CSR read, presence bits written + read once,
        # sparse (sample, value) entries written (+ integer counts written and read for the weighted variant)
        embed_bytes = nnz * 8.0 + 2.0 * n_nodes * n_words * 4 + s0["tail_entries"] * (8.0 if v == 0 else 16.0)
        per_variant[variant_name(v)] = dict(
            ms_total=mean("ms_total"), ms_plan=mean("ms_plan"), ms_embed=mean("ms_embed"), ms_tail=mean("ms_tail"),
            ms_mid=mean("ms_mid"), ms_stripe=mean("ms_stripe"),
            algorithmic_frac=(2.0 * s0["updates_inter"] / (ALU_PEAK_TFLOPS * 1e12) / t_a5) if t_a5 > 0 else None,
            updates_executed_per_s=(s0["updates_executed"] / t_a5) if t_a5 > 0 else None,
            embed_gbs=(embed_bytes / (mean("ms_embed") * 1e-3) / 1e9) if mean("ms_embed") > 0 else None,
            mid_rows=s0["mid_rows"], mid_updates=s0["mid_updates"], mid_F=s0["mid_F"],
            mid_groups=s0["mid_groups"], mid_group_rows=s0["mid_group_rows"], mid_atomics=s0["mid_atomics"],
            head_rows=s0["head_rows"], tail_rows=s0["tail_rows"], tail_updates=s0["tail_updates"],
            gram=s0["gram"], gram_k=s0["gram_k"], gram_q=s0["gram_q"], guard_pairs=s0["guard_pairs"],
            skip=s0["skip"], skip_rows=s0["skip_rows"], list_rows=s0["list_rows"], skip_row_pair_visits=s0["skip_row_pair_visits"],
            skip_updates_executed=s0["skip_updates_executed"],
            tail_entries=s0["tail_entries"], tail_launches=s0["tail_launches"],
            updates_executed_head=s0["updates_executed_head"], updates_dense=s0["updates_dense"],
            updates_executed=s0["updates_executed"], updates_union=s0["updates_union"], updates_inter=s0["updates_inter"],
            branches_embedded=s0["branches_embedded"], workspace_gb=s0["workspace_bytes"] / 2**30)
    return per_variant


def parity_check(p, variants, outs, n_pairs=2000, seed=3):
    """max / p99.99 relative error of resident outputs against the oracle on a seeded pair sample."""
    import torch
    from oracle import oracle
    pairs = synth.sample_pairs(p.n_samples, n_pairs, seed=seed)
    idx = torch.from_numpy(synth.condensed_index(p.n_samples, pairs[:, 0], pairs[:, 1])).to(next(iter(outs.values())).device)
    rels = []
    for v in variants:
        want = oracle.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, v, pairs)
        got = outs[v][idx].double().cpu().numpy()
        rels.append(np.abs(got - want) / np.maximum(np.abs(want), 1e-30))
    rel = np.concatenate(rels)
    return dict(max_rel=float(rel.max()), p9999_rel=float(np.quantile(rel, 0.9999)), pairs=int(rel.shape[0]),
                sample=f"{n_pairs} seeded pairs per variant vs the oracle's pair-list driver, after the timed region")


def run_workload(binding, torch, dist, p, variants, precision, dev, steps, warmup, flags, shard, world, sampler_gpu=None):
    """warm-up, then `steps` timed steps (one unifrac_dm[_shard] call per variant [+ the NCCL merge of the shard buffers]),
    CUDA events on the launch stream, barrier + synchronize on both sides.  Returns (ms, all_stats, outs, clock lines)."""
    from paper_2107_05397_b200 import multigpu
    args = binding.to_device(p, dev)
    outs = {v: torch.empty(p.n_pairs, dtype=torch.float32 if precision == 0 else torch.float64, device=dev) for v in variants}

    def step():
        stats = []
        for v in variants:
            binding.unifrac_dm(*args, p.n_samples, v, precision, out=outs[v], flags=flags, shard=shard)
            st = binding.unifrac_last_stats()               # waits for the call's stripe kernel (stats event)
            st["n_samples"] = p.n_samples
            stats.append(st)
            if shard:
                multigpu.merge_shards(outs[v])              # all-reduce(SUM) over NCCL: every pair has one owner
        return stats

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    for _ in range(warmup):
        step()
    barrier()
    stop, lines = threading.Event(), []
    th = None
    if sampler_gpu is not None:
        th = threading.Thread(target=clocks_sampler, args=(stop, lines, sampler_gpu), daemon=True)
        th.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    all_stats = []
    e0.record()
    for _ in range(steps):
        all_stats.append(step())
    e1.record()
    barrier()
    stop.set()
    if th is not None:
        th.join(timeout=3)
    return e0.elapsed_time(e1), all_stats, outs, lines, args, barrier


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=os.environ.get("UNIFRAC_BENCH_WORKLOAD", "large"))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--cpu-budget-s", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-emp", action="store_true", help="skip the EMP-shaped (N = 25,000) leg that precedes the Large workload")
    ap.add_argument("--no-next", action="store_true", help="skip the Mantel / PCoA legs that follow the timed region")
    ap.add_argument("--mantel-perms", type=int, default=9,
                    help="after the timed region: Mantel test (Pearson, then Spearman) between the unweighted and the weighted "
                         "matrix with this many permutations (0 = skip); reported under \"mantel\", not part of the step")
    ap.add_argument("--shard", action="store_true", help="accepted for compatibility: shards are the default for N > 1")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: independent replicas (weak scaling, no merge) instead of shards of one matrix + NCCL merge")
    a = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    variants, precision = WORKLOADS[a.workload]
    dtype = "f32" if precision == 0 else "f64"

    # ---------------------------------------------------------------- reference arm = the oracle on host cores
    if a.impl == "reference":
        if rank != 0:
            return 0
        p = synth.make_config(a.workload, seed=a.seed)
        legs = [oracle_leg(p, variants, a.cpu_budget_s / max(1, a.steps + a.warmup), seed=k) for k in range(a.warmup + a.steps)]
        timed = legs[a.warmup:]
        b_emb = int(((p.parent >= 0) & (p.branch_len > 0)).sum())      # upper bound of B_emb (all branches with len > 0)
        upd = sum(l["pairs"] for l in timed) * b_emb
        secs = sum(l["seconds"] for l in timed)
        val = upd / secs
        line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=a.gpus, steps=a.steps, warmup=a.warmup,
                    ms_per_step=1e3 * secs / a.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="f64", data="synthetic", impl="reference",
                    config=dict(workload=a.workload, n_samples=p.n_samples, n_nodes=p.n_nodes, nnz=p.nnz, seed=a.seed,
                                variants=list(variants), step="bounded pair sample of the workload"),
                    cpu_baseline=dict(value=val, unit=UNIT, cores=timed[0]["cores"], kind="oracle", sample=timed[0]["sample"],
                                      cpu_model=cpu_model_name()),
                    e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
        print(json.dumps(line))
        return 0

    # ---------------------------------------------------------------- our arm
    shard = (rank, world) if (world > 1 and not a.replicas) else None
    seed = a.seed if (shard or world == 1) else rank_seed(a.seed, rank)
    run_emp = a.workload == "large" and not a.no_emp
    p_emp = synth.make_config("emp", seed=seed) if run_emp else None     # generated before CUDA is touched (fork pool)
    p = synth.make_config(a.workload, seed=seed)
    os.environ["UNIFRAC_B200_TIMING"] = "1"
    import torch
    from paper_2107_05397_b200 import binding
    binding.load()
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    wall_emp = None
    launches_emp = 0
    if run_emp:
        steps_emp = max(1, a.steps // 4)
        ms_e, st_e, outs_e, _, args_e, _ = run_workload(binding, torch, dist, p_emp, (0, 1), 0, dev, steps_emp, a.warmup, a.flags,
                                                         shard, world)
        ms_e, _ = reduce_over_ranks(ms_e, 0.0, world, dev)
        wall_emp = dict(n_samples=p_emp.n_samples, n_nodes=p_emp.n_nodes, steps=steps_emp, ms_per_step=ms_e / steps_emp,
                        **wall_of(st_e, (0, 1), p_emp.n_nodes, p_emp.nnz))
        if rank == 0:
            wall_emp["parity"] = parity_check(p_emp, (0, 1), outs_e)
        launches_emp = int(sum(s["kernel_launches"] for st in st_e for s in st))
        del outs_e, args_e
        torch.cuda.empty_cache()

    ms, all_stats, outs, lines, args, barrier = run_workload(binding, torch, dist, p, variants, precision, dev, a.steps, a.warmup,
                                                             a.flags, shard, world, sampler_gpu=local_rank)
    flat = [s for st in all_stats for s in st]
    upd_local = float(sum(s["updates_dense"] for s in flat))
    if shard:
        upd_local /= world               # the ranks share one matrix: its updates are counted once
    ms, upd_all = reduce_over_ranks(ms, upd_local, world, dev)
    value = upd_all / (ms * 1e-3)
    parity = parity_check(p, variants, outs) if rank == 0 else None      # on the merged matrix when sharded

    # ---------------- next rows on the two matrices still resident in HBM; not part of the step
    mantel = pcoa = None
    single = world == 1
    if single and not a.no_next and len(variants) == 2 and a.mantel_perms > 0:
        g = torch.Generator(device=dev).manual_seed(a.seed)
        perms = torch.stack([torch.randperm(p.n_samples, device=dev, generator=g) for _ in range(a.mantel_perms)]).to(torch.int32).contiguous()
        def timed(fn):
            fn()                                                       # warm-up
            barrier()
            m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            m0.record()
            r = fn()
            m1.record()
            barrier()
            return m0.elapsed_time(m1), r
        x, y = outs[variants[0]], outs[variants[1]]
        esz = x.element_size()
        m_ms, mo = timed(lambda: binding.unifrac_mantel_pearson(x, y, p.n_samples, perms))
        alg = (a.mantel_perms + 1) * 2.0 * p.n_pairs * esz          # both condensed matrices once per (permuted) statistic
        mantel = dict(n_samples=p.n_samples, permutations=a.mantel_perms,
                      pearson=dict(ms=m_ms, ms_per_permutation=m_ms / (a.mantel_perms + 1), r=float(mo[0]), p_two_sided=float(mo[1]),
                                   algorithmic_gbs=alg / m_ms / 1e6))
        try:
            s_ms, so = timed(lambda: binding.unifrac_mantel_spearman(x, y, p.n_samples, perms))
            # the rank transform: 2 vectors x 4 radix passes x (4 + 8 + 8) bytes per element, then the fp64 rank vectors
            mantel["spearman"] = dict(ms=s_ms, rho=float(so[0]), p_two_sided=float(so[1]),
                                      ms_rank_transform_and_fp64_statistics=s_ms,
                                      note="device radix-sort rank transform of both matrices + the same permutation kernel on the 32-bit 2 x rank vectors (fp64 sums)")
        except binding.UnifracError as e:                              # e.g. workspace
            mantel["spearman"] = dict(error=str(e))
        del perms, mo
        torch.cuda.empty_cache()
    if single and not a.no_next:
        try:
            x = outs[variants[-1]]
            def run_pcoa(iters):
                torch.cuda.synchronize(dev)
                t0 = time.perf_counter()
                lam, prop, _, its = binding.unifrac_pcoa(x, p.n_samples, 5, max_iter=iters, tol=0.0)
                torch.cuda.synchronize(dev)
                return time.perf_counter() - t0, lam, prop, its
            run_pcoa(4)
            t8, _, _, _ = run_pcoa(8)
            t24, lam, prop, its = run_pcoa(24)
            per_product = (t24 - t8) / 16.0
            n_pad = (p.n_samples + 127) // 128 * 128
            gbs = 8.0 * n_pad * n_pad / per_product / 1e9
            pcoa = dict(matrix=variant_name(variants[-1]), axes=5, products=its, seconds=t24, ms_per_product=1e3 * per_product,
                        setup_seconds=t8 - 8 * per_product, eigenvalues=[float(v) for v in lam], proportion_explained=[float(v) for v in prop],
                        bound="hbm", product_gbs=gbs, note="Y = B Q streams B_hi and B_lo (8 N^2 bytes) per product; tcgen05 kind::tf32, 3-term split; "
                        "fixed 24 products here (convergence is checked in tests/test_gpu_pcoa.py)")
        except binding.UnifracError as e:
            pcoa = dict(error=str(e))
        torch.cuda.empty_cache()

    # ---------------- end to end through the host-buffer C-ABI call (H2D + D2H inside the timed region)
    e2e = None
    if not a.no_e2e and not shard:      # the host-buffer entry point computes whole matrices
        pin = lambda arr: torch.from_numpy(np.ascontiguousarray(arr)).pin_memory().numpy()
        hp = [pin(x) for x in (p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts)]
        houts = [torch.empty(p.n_pairs, dtype=torch.float32 if precision == 0 else torch.float64).pin_memory().numpy() for _ in variants]
        del outs
        torch.cuda.empty_cache()
        os.environ["UNIFRAC_B200_TIMING"] = "0"      # the per-stage event timing synchronises every call: off for the end-to-end leg
        def e2e_step():                              # one call for the step's variants: inputs uploaded once, D2H overlaps compute
            binding.unifrac_dm_host_multi(*hp, p.n_samples, list(variants), precision, outs=houts)
        e2e_step()                                   # one untimed warm-up step (device memory pool, page mappings)
        barrier()
        t0 = time.perf_counter()
        for _ in range(a.steps):
            e2e_step()
        barrier()
        t_e2e = (time.perf_counter() - t0) / a.steps
        t_e2e, _ = reduce_over_ranks(t_e2e, 0.0, world, dev)
        h2d = sum(x.nbytes for x in hp)
        d2h = sum(h.nbytes for h in houts)
        binding.unifrac_release_host_pool()
        e2e = dict(value=(upd_all / a.steps) / t_e2e, unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                   seconds_per_step=t_e2e)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    # ---------------- device rates of the atomic units (peaks of the k_mid / k_tail_scatter rooflines), measured live
    rates = dict(smem_atomic_random_per_s=SMEM_ATOMIC_PER_S, l2_red_random_per_s=L2_RED_PER_S)
    rates_src = "fallback constants (bench.py)"
    try:
        rates = binding.unifrac_measure_rates()
        rates_src = "measured live by unifrac_measure_rates on this GPU"
    except Exception as e:                                   # noqa: BLE001 - the probe is not on the data path
        rates_src += f" [probe failed: {e}]"

    # ---------------- rooflines of the a-5 kernels; the one with the most time in the step is "roofline"
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    src = "measured" if peaks else "fallback"
    step_s = ms * 1e-3
    rl = []
    # (1) k_dense (default) / k_stripe (debug forms): CUDA-core register-tile kernel (head branches; weighted, fp64, or NO_TENSOR)
    ss = [s for s in flat if not s["gram"]]
    if ss:
        kname = "k_zone" if all(s["skip"] for s in ss) else \
                ("k_dense16" if precision == 0 else "k_dense") if all(s["dense"] for s in ss) else "k_stripe"
        t = sum(s["ms_stripe"] for s in ss) * 1e-3
        w_exec = sum(s["updates_executed_head"] for s in ss)
        nl = sum(s["stripe_launches"] for s in ss)
        ach = 2.0 * w_exec / t / 1e12 if t > 0 else 0.0
        rl.append(dict(bound="alu", achieved=ach, peak=ALU_PEAK_TFLOPS, unit="TFLOP/s", frac=ach / ALU_PEAK_TFLOPS, traffic=None,
                       kernel=kname, launches=nl, ms_per_launch=1e3 * t / max(1, nl),
                       executed_updates_per_launch=w_exec / max(1, nl), seconds=t, share_of_step=t / step_s,
                       peak_source=f"{SM_COUNT} SMs x {FP32_LANES} FP32 lanes x {SM_MAX_GHZ} GHz (sm_max_mhz of MEASURED_PEAKS.json, {src}); "
                                   "2 FP32-pipe lane-ops (FMNMX+FADD) per (pair, branch) update",
                       measured_fmnmx_fadd_tflops=rates.get("fmnmx_fadd_per_s", 0.0) / 1e12 or None))
    # (2) k_gram: tcgen05 kind::i8 Gram kernel (head branches, unweighted fp32): 3 u8 digit MACs per update
    gs = [s for s in flat if s["gram"]]
    if gs:
        t = sum(s["ms_stripe"] for s in gs) * 1e-3
        macs = sum(float(s["gram_k"]) * s["n_tile_pairs"] * 128 * 128 * 3 for s in gs)
        nl = sum(s["stripe_launches"] for s in gs)
        bf16 = peaks.get("bf16_tflops", 1590.0)
        peak = 2.0 * bf16                       # int8 : bf16 nominal ratio 2 (4.5 vs 2.25 PFLOP/s dense, B200_PROFILING.md)
        ach = 2.0 * macs / t / 1e12 if t > 0 else 0.0
        rl.append(dict(bound="tensor", achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak, traffic=None, kernel="k_gram",
                       launches=nl, ms_per_launch=1e3 * t / max(1, nl), macs_per_launch=macs / max(1, nl), seconds=t,
                       share_of_step=t / step_s,
                       peak_source=f"2 x bf16_tflops ({bf16}, {src} burst) = int8 dense peak by the guide's nominal 2:1 ratio; "
                                   "algorithmic ops = 2 x 3 digit-MACs x 128 x 128 x K per tile pair",
                       operand_gbs=sum(float(s["gram_k"]) * s["n_tile_pairs"] * 512 for s in gs) / t / 1e9 if t > 0 else 0.0))
    # (3) k_tail_scatter: RED.ADD of min(u_a, u_b) into the L2-resident super tile
    t = sum(s["ms_tail"] for s in flat) * 1e-3
    reds = sum(s["tail_updates"] for s in flat)
    nl = sum(s["tail_launches"] for s in flat)
    if nl:
        RED_PEAK = rates["l2_red_random_per_s"]
        rl.append(dict(bound="l2_atomic", achieved=reds / t / 1e9 if t > 0 else 0.0, peak=RED_PEAK / 1e9, unit="GRED/s",
                       frac=reds / t / RED_PEAK if t > 0 else 0.0, traffic=None, kernel="k_tail_scatter", launches=nl,
                       ms_per_launch=1e3 * t / max(1, nl), seconds=t, share_of_step=t / step_s,
                       peak_source=f"scattered RED.ADD.F32 into a 48 MB L2-resident footprint, {rates_src}"))
    # (4) the mid stage: tile-pair join with native shared-memory integer atomics (ATOMS.ADD).  k_mid: one atomic per
    # (pair, branch) update; k_midg (grouped join, default): one atomic per pair of a group ROOT serves the update of every
    # member, so the algorithmic update rate may pass the rate of the atomic unit
    t = sum(s["ms_mid"] for s in flat) * 1e-3
    mu = sum(s["mid_updates"] for s in flat)
    ma = sum(s["mid_atomics"] for s in flat)
    nl = sum(s["mid_launches"] for s in flat)
    grouped = any(s["mid_groups"] for s in flat)
    if nl:
        ATOMS_PEAK = rates["smem_atomic_random_per_s"]
        rl.append(dict(bound="smem_atomic", achieved=mu / t / 1e9 if t > 0 else 0.0, peak=ATOMS_PEAK / 1e9, unit="GATOM/s",
                       frac=mu / t / ATOMS_PEAK if t > 0 else 0.0, traffic=None, kernel="k_midg" if grouped else "k_mid", launches=nl,
                       ms_per_launch=1e3 * t / max(1, nl), seconds=t, share_of_step=t / step_s,
                       updates_per_launch=mu / max(1, nl), atomics_executed_per_launch=ma / max(1, nl),
                       frac_atomics_executed=(ma / t / ATOMS_PEAK) if t > 0 else 0.0,
                       frac_of_fp32_lane_roofline=(2.0 * mu / t / (ALU_PEAK_TFLOPS * 1e12)) if t > 0 else 0.0,
                       note="achieved = algorithmic (pair, mid branch) updates per second against the rate of the shared-memory atomic unit "
                            "(one atomic per update is what the ungrouped join k_mid needs); the grouped join executes atomics_executed "
                            "atomics for them (frac_atomics_executed of the unit's rate).  ms_mid also covers the list preparation "
                            "kernels (grouping, k_mid_seg/off/pack, k_midg_pack_*).  frac_of_fp32_lane_roofline = 2 lane-ops per update "
                            "against the FP32-lane peak of SURVEY 8(d)",
                       peak_source=f"shared-memory u32 atomic adds on random cells of a 128 x 128 tile, 3 CTAs/SM x 512 threads "
                                   f"(= {ATOMS_PEAK / SM_COUNT / SM_MAX_GHZ / 1e9:.2f} lane-ops/clk/SM; same rate conflict-free), {rates_src}"))
    for r in rl:
        if a.flags == 0 and a.seed == 0:
            r["traffic"] = NCU_TRAFFIC_BYTES.get(a.workload, {}).get(r["kernel"])
    rl.sort(key=lambda r: -r["seconds"])
    roofline = dict(rl[0])
    roofline["others"] = rl[1:]
    w_inter = sum(s["updates_inter"] for s in flat)
    w_exec_all = sum(s["updates_executed"] for s in flat)
    roofline["step_updates"] = dict(dense=upd_all / max(1, world), executed=w_exec_all, inter=w_inter,
                                    embed_seconds=sum(s["ms_embed"] for s in flat) * 1e-3)

    roofline["traffic_source"] = TRAFFIC_SOURCE + "; null = no capture of the current kernel"

    cpu = None
    if not a.no_cpu_baseline:
        leg = oracle_leg(p, variants, a.cpu_budget_s)
        b_emb = flat[0]["branches_embedded"]
        per_pair = leg["seconds"] / leg["pairs"]
        cpu = dict(value=leg["pairs"] * b_emb / leg["seconds"], unit=UNIT, cores=leg["cores"], kind="oracle",
                   sample=leg["sample"], seconds=leg["seconds"], cpu_model=cpu_model_name(),
                   extrapolated_all_pairs_s=per_pair * p.n_pairs * len(variants),
                   extrapolated_note="EXTRAPOLATED: sampled seconds per pair x N(N-1)/2 x variants; the oracle is a plain "
                                     "definition (long double, Neumaier sums), not an optimised CPU implementation")

    per_variant = wall_of(all_stats, variants, p.n_nodes, p.nnz)
    if shard:
        par = f"shards x{world}: disjoint tile-pair blocks per rank, then NCCL all-reduce(SUM) merge inside the timed region"
    else:
        par = f"replicas x{world}"
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=a.steps, warmup=a.warmup, ms_per_step=ms / a.steps,
                higher_is_better=True, scaling="strong" if shard else "weak", vs_baseline=None, dtype=dtype, data="synthetic",
                config=dict(workload=a.workload, n_samples=p.n_samples, n_nodes=p.n_nodes, nnz=p.nnz, seed=a.seed,
                            variants=list(variants), precision=dtype, flags=a.flags, parallelism=par,
                            l2="inputs larger than L2 (compact embedding >> 126 MB)"),
                clocks=summarize_clocks(lines), e2e=e2e,
                gpu_launches=int(sum(s["kernel_launches"] for s in flat)),
                roofline=roofline, cpu_baseline=cpu, wall=per_variant, parity=parity)
    if wall_emp is not None:
        line["wall_emp"] = wall_emp
        line["gpu_launches_emp_leg"] = launches_emp
    if mantel:
        hbm = peaks.get("hbm_gbs", 6550.0)
        mantel["pearson"].update(bound="hbm", peak_gbs=hbm, frac=mantel["pearson"]["algorithmic_gbs"] / hbm,
                                 note="algorithmic bytes = both condensed matrices once per statistic; the kernel moves ~1.5x that "
                                      "(full rows of the square copy)")
        line["mantel"] = mantel
    if pcoa:
        if "product_gbs" in pcoa:
            hbm = peaks.get("hbm_gbs", 6550.0)
            pcoa.update(peak_gbs=hbm, frac=pcoa["product_gbs"] / hbm)
        line["pcoa"] = pcoa
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
