#!/usr/bin/env python
"""bench.py — candidates/s of the lgx hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (the persistent kernel
pair lgx_decode_walk + lgx_finish per chunk, over the shared-memory images built by a1) over
one batch of candidates:
`lgx_search` over the Medium config's full budget (2^28 ids, 100 fields / 8 BPs / 5 tours;
the config the north_star target of >= 1e9 cand/s is quoted on).  Synthetic, seeded
instance (paper_1909_10286_b200/workloads.py); nothing is read from /root/reference.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload medium]

Prints ONE JSON line (rank 0).  `value` is device-timed (CUDA events on the launching
stream, max over ranks) with the instance image resident in HBM; `e2e` re-creates the
instance from HOST arrays (H2D of the image) and reads the result back to the host inside
the timed region, through the C ABI.  `--impl reference` times the CPU oracle instead.
"""
from __future__ import annotations
import argparse, json, os, subprocess, sys, threading, time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "candidate plans evaluated/sec"
UNIT = "candidates/s"
# Algorithmic thread-instructions per candidate: what the method itself needs,
# split into the part every candidate pays (decode + pass 1: kernel lgx_decode_walk) and the part
# only feasible candidates pay (tour statistics, Algorithm 2, pass 2, cost: kernel lgx_finish).
ALG2_ITERS = {"toy": 2.3, "small": 5.6, "medium": 9.9, "large": 12.7, "sweep": 19.5}   # oracle-measured means


def w_alg(inst, workload):
    nf, nb, nt, nhu, nsu = inst.n_fields, inst.n_bps, inst.n_tours, inst.n_hu, inst.n_su
    cd = lambda a, b: -(-a // b)
    part_blocks = lambda n: cd(n, 4) + cd(n - nt, 4)            # Philox blocks of one ordered partition
    # every candidate: BP partition, field permutation + extras, pass 1  (kernel lgx_decode_walk)
    blocks_a = cd(nf, 4) + part_blocks(nb) + cd((nb - 1) * 4 // 3 + 8, 4)
    decode_walk = 40 * blocks_a + 7 * (nf + nb) + 2 * (nb - nt) + 6 * nb + 14 * nf + 10 * (nb + nt)
    # feasible candidates only: HU / SU partitions, tour statistics, Algorithm 2, pass 2, cost  (lgx_finish)
    blocks_c = part_blocks(nhu) + part_blocks(nsu)
    finish = (40 * blocks_c + 7 * (nhu + nsu) + 2 * (nhu + nsu - 2 * nt) + 6 * nhu + 10 * nsu
              + 6 * nb + 92 * nt + 110 * ALG2_ITERS.get(workload, 10.0) + 18 * nf + 10 * (nb + nt) + 9 * nt + 5)
    return decode_walk, finish


SM_MAX_MHZ_FALLBACK = 1965.0
# dram__bytes_read.sum + dram__bytes_write.sum of ONE lgx_decode_walk launch (757 760 Medium candidates) from the
# `ncu --set full` capture summarised in profiles/r01_v7_medium_ncu_full.md: 0.12 MB read + 4.08 MB written (the
# queue records of the feasible candidates that do not stay in L2).  Per launch, like `achieved`.
TRAFFIC_BYTES_DECODE_WALK_MEDIUM = 4.20e6


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return json.load(open(p)), "measured"
    except Exception:      # noqa: BLE001
        return {"sm_max_mhz": SM_MAX_MHZ_FALLBACK, "hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True); self.t.start()
        except Exception:  # noqa: BLE001
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try: self.proc.wait(2)
        except Exception: self.proc.kill()  # noqa: BLE001,E701
        sm = sorted(float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit())
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) >= 7 and r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def oracle_rate(name, n_ids, procs):
    """The oracle as it stands (single-threaded by design), run as `procs` independent
    processes over disjoint contiguous id ranges on the host cores."""
    import multiprocessing as mp
    ctx = mp.get_context("fork")
    per = max(1, n_ids // procs)
    with ctx.Pool(procs) as pool:
        t0 = time.perf_counter()
        res = pool.starmap(_oracle_chunk, [(name, r * per, per) for r in range(procs)])
        dt = time.perf_counter() - t0
    best = min(res, key=lambda p: (p[0], p[1]))
    return per * procs / dt, dt, best


def _oracle_chunk(name, first, n):
    from oracle import lgo
    from paper_1909_10286_b200 import workloads as wl
    inst = wl.make(name)
    o = lgo.Oracle(inst)
    return o.search(inst.seed, n, first_id=first)


def _oracle_moves_chunk(name, first, n):
    from oracle import lgo
    from paper_1909_10286_b200 import workloads as wl
    o = lgo.Oracle(wl.make(name))
    p0 = o.init_plan()
    return float(o.move_eval_batch(p0, 1, first, n)[3].mean())


def bench_alg1(args, torch, binding, wl):
    """The paper's own loop (Algorithm 1) on its own problem shape: nearest-neighbour start,
    one batch of remove/reinsert workers, and N_iters iterations inside the persistent kernel."""
    import multiprocessing as mp
    inst = wl.make(args.alg1_workload)
    g = binding.Instance(inst)
    sm, tmv = g.query(6), g.query(15)
    stream = torch.cuda.current_stream()
    g.init_plan()
    t0 = time.perf_counter(); p0 = g.init_plan(); t_init = time.perf_counter() - t0
    n = sm * tmv * 16
    out = g.move_eval_batch(p0, 1, 0, n); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(3):
        g.move_eval_batch(p0, 1, 0, n, out=out)
    b.record(stream); torch.cuda.synchronize()
    ms_batch = a.elapsed_time(b) / 3
    n_workers, eps = sm * tmv * 8, 0.4        # 8 rounds per block and iteration: the warps balance them dynamically
    c0 = g.local_search(p0, inst.seed, 0, 1, 0, history=False)[1]
    g.local_search(p0, inst.seed, 10, n_workers, int(eps * 2**32), history=False)          # warm-up
    t0 = time.perf_counter()
    _, c_star, hc, _ = g.local_search(p0, inst.seed, args.alg1_iters, n_workers, int(eps * 2**32))
    t_ls = time.perf_counter() - t0
    res = {"workload": f"{args.alg1_workload}: N_T={inst.n_tours} N_B={inst.n_bps} N_F={inst.n_fields} N_HU={inst.n_hu} N_SU={inst.n_su}",
           "threads_per_block": tmv, "grid": sm, "smem_bytes": g.query(16),
           "init_plan_ms": 1e3 * t_init,
           "move_eval_batch": {"value": n / ms_batch * 1e3, "unit": "workers/s", "workers": n,
                               "feasible_fraction": float(out[3].float().mean().item())},
           "local_search": {"iterations": args.alg1_iters, "workers_per_iteration": n_workers, "eps": eps,
                            "wall_s": t_ls, "iterations_per_s": args.alg1_iters / t_ls,
                            "worker_evals_per_s": args.alg1_iters * n_workers / t_ls,
                            "cost_init": c0, "cost_best": c_star, "delta_pct": 100.0 * (c_star - c0) / c0,
                            "what": "lgx_local_search through the C ABI, host plan in / x* out, wall clock",
                            "paper_context": "T_solve 81.89 s for 5000 iterations on a Titan V, workers per iteration "
                                             "not stated (PAPER.md Table 3, L355): another machine, not a target"}}
    # N2: the same loop with the embedded HU assignment (LGX_FLAG_HU_BALANCE) on an instance that has spare HUs
    from dataclasses import replace
    inst_h = replace(wl.make("large"), flags=2)
    gh = binding.Instance(inst_h)
    ph = gh.init_plan()
    nwh = sm * gh.query(15) * 8
    ch0 = gh.local_search(ph, inst_h.seed, 0, 1, 0, history=False)[1]
    gh.local_search(ph, inst_h.seed, 10, nwh, int(eps * 2**32), history=False)
    t0 = time.perf_counter()
    _, ch, _, _ = gh.local_search(ph, inst_h.seed, args.alg1_iters, nwh, int(eps * 2**32))
    t_h = time.perf_counter() - t0
    res["local_search_hu_balance"] = {"workload": f"large: N_T={inst_h.n_tours} N_B={inst_h.n_bps} N_F={inst_h.n_fields} N_HU={inst_h.n_hu} N_SU={inst_h.n_su}",
                                      "iterations": args.alg1_iters, "workers_per_iteration": nwh, "wall_s": t_h,
                                      "iterations_per_s": args.alg1_iters / t_h, "worker_evals_per_s": args.alg1_iters * nwh / t_h,
                                      "cost_init": ch0, "cost_best": ch, "delta_pct": 100.0 * (ch - ch0) / ch0}
    gh.close()
    if not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        per = 2048
        with mp.get_context("fork").Pool(cores) as pool:
            t0 = time.perf_counter()
            pool.starmap(_oracle_moves_chunk, [(args.alg1_workload, r * per, per) for r in range(cores)])
            dt = time.perf_counter() - t0
        res["cpu_baseline"] = {"value": per * cores / dt, "unit": "workers/s", "cores": cores, "kind": "oracle",
                               "sample": f"{per * cores} workers of the same batch, {cores} processes, {dt:.1f} s wall"}
    g.close()
    return res


def run_reference(args):
    """--impl reference: the oracle (the only reference implementation of this tier)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    sample = 1 << 21          # ids per step; ~1 s per step on 16 cores for Medium
    for _ in range(args.warmup):
        oracle_rate(args.workload, sample // 4, cores)
    tot_t, tot_n = 0.0, 0
    for _ in range(args.steps):
        r, dt, _ = oracle_rate(args.workload, sample, cores)
        tot_t += dt; tot_n += (sample // cores) * cores
    v = tot_n / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": args.workload, "ids_per_step": sample},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{sample} ids/step of the {args.workload} budget, {cores} processes"},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="lgx", choices=["lgx", "reference"])
    ap.add_argument("--workload", default="medium")
    ap.add_argument("--batch-log2", type=int, default=None, help="candidates per GPU per step (default: config budget, capped 2^28)")
    ap.add_argument("--chunk-log2", type=int, default=None, help="candidates per kernel pair (LGX_OPT_CHUNK_LOG2; profiling)")
    ap.add_argument("--threads-a", type=int, default=None, help="LGX_OPT_THREADS_A (tuning)")
    ap.add_argument("--threads-b", type=int, default=None, help="LGX_OPT_THREADS_B (tuning)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--alg1-workload", default="paper_scale", help="instance of the Algorithm 1 leg (SURVEY §8(f) N1/N3)")
    ap.add_argument("--alg1-iters", type=int, default=500)
    ap.add_argument("--no-alg1", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "lgx" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    from paper_1909_10286_b200 import binding, workloads as wl, sharding

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    inst = wl.make(args.workload)
    per_gpu = 1 << (args.batch_log2 if args.batch_log2 is not None else min(28, inst.budget.bit_length() - 1))
    total = per_gpu * world                      # weak scaling: fixed ids per GPU
    g = binding.Instance(inst)
    for key, val in ((4, args.chunk_log2), (1, args.threads_a), (2, args.threads_b)):
        if val is not None:
            g.set_option(key, val)
    info = g.info()
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step(first_total=0):
        # this rank's contiguous share of [0, total); one 16-byte exchange when world > 1
        if world == 1:
            return g.search(inst.seed, per_gpu, first_id=first_total)
        return sharding.search_sharded(lambda s, n, f: g.search(s, n, first_id=f), inst.seed, total, rank, world, first_total)

    for _ in range(args.warmup):
        step()
    # ---- timed: EXACTLY K steps, device time from CUDA events on the launching stream
    sampler = ClockSampler(local); sampler.start()
    g.set_timing(True)                           # CUDA events around every kernel launch, on the launching stream
    launches0 = g.query(7)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_wall0 = time.perf_counter()
    best = None
    for k in range(args.steps):
        flush.fill_(k & 0xFF)                    # L2 flush between timed iterations (untimed)
        ev[k][0].record(stream)
        best = step()
        ev[k][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = g.query(7) - launches0
    ns_a, ns_c, n_pairs = g.kernel_times()
    g.set_timing(False)
    clocks = sampler.stop()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    if dist is not None:
        t = torch.tensor([dev_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX); dev_ms = float(t.item())
    value = total * args.steps / (dev_ms * 1e-3)

    # ---- e2e: host arrays -> lgx_instance_create (H2D image) -> lgx_search -> host result
    e2e_steps = max(2, min(args.steps, 3))

    def e2e_step():
        g2 = binding.Instance(inst)
        for key, val in ((4, args.chunk_log2), (1, args.threads_a), (2, args.threads_b)):
            if val is not None:
                g2.set_option(key, val)
        if world == 1:
            r = g2.search(inst.seed, per_gpu)
        else:
            r = sharding.search_sharded(lambda s, n, f: g2.search(s, n, first_id=f), inst.seed, total, rank, world)
        g2.close()
        return r

    e2e_step()                                   # untimed warm-up of the create/destroy path
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        r2 = e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX); e2e_s = float(t.item())
    e2e_value = total * e2e_steps / e2e_s
    assert r2 == best, "e2e result differs from the device-timed result"

    # ---- eval_batch (per-candidate outputs) timed separately, device and host buffers
    extra = {}
    if rank == 0:
        n_ev = 1 << 24
        out = g.eval_batch(inst.seed, first_id=0, n=n_ev)
        torch.cuda.synchronize()
        ev_list = []
        for _ in range(3):                       # median of 3 device-timed calls
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); g.eval_batch(inst.seed, first_id=0, n=n_ev, out=out); b.record(stream)
            torch.cuda.synchronize()
            ev_list.append(a.elapsed_time(b))
        ev_ms = sorted(ev_list)[1]
        n_h = 1 << 22
        host_out = (np.empty(n_h), np.empty(n_h), np.empty(n_h), np.empty(n_h, np.uint8))
        g.eval_batch_host(inst.seed, first_id=0, n=n_h, out=host_out)
        t0 = time.perf_counter(); g.eval_batch_host(inst.seed, first_id=0, n=n_h, out=host_out); th = time.perf_counter() - t0
        extra["eval_batch"] = {"value": n_ev / ev_ms * 1e3, "unit": UNIT, "ids": n_ev,
                               "feasible_fraction": float(out[3].float().mean().item()),
                               "e2e_host_buffers": {"value": n_h / th, "unit": UNIT, "ids": n_h,
                                                    "d2h_bytes": 25 * n_h, "h2d_bytes": 0}}

    if rank == 0 and world == 1 and not args.no_alg1:
        extra["alg1"] = bench_alg1(args, torch, binding, wl)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    pk, pk_src = peaks()
    sm_max = float(pk.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK))
    n_sm = info["sm_count"]
    peak_ginst = n_sm * 4 * 32 * sm_max * 1e6 / 1e9          # thread-instructions/s at max clock
    feas = extra.get("eval_batch", {}).get("feasible_fraction", 1.0)
    w_dw, w_fin = w_alg(inst, args.workload)
    cand_timed = per_gpu * args.steps                         # this rank's candidates in the timed region
    per_launch = cand_timed / max(n_pairs, 1)                 # candidates per launch of each kernel
    ms_a = ns_a * 1e-6 / max(n_pairs, 1); ms_c = ns_c * 1e-6 / max(n_pairs, 1)
    ach_a = per_launch * w_dw / (ms_a * 1e-3) / 1e9 if ms_a > 0 else None
    ach_c = per_launch * feas * w_fin / (ms_c * 1e-3) / 1e9 if ms_c > 0 else None
    ach_all = (w_dw + feas * w_fin) * value / world / 1e9
    obs = clocks.get("sm_mhz") or sm_max
    roofline = {"bound": "alu", "kernel": "lgx_decode_walk (dominant: %.0f %% of the kernel time of a step)" % (100.0 * ns_a / max(ns_a + ns_c, 1)),
                "achieved": ach_a, "peak": peak_ginst, "unit": "G thread-inst/s", "frac": ach_a / peak_ginst if ach_a else None,
                "traffic": TRAFFIC_BYTES_DECODE_WALK_MEDIUM if args.workload == "medium" else None, "launch_ms": ms_a, "launches_timed": n_pairs, "candidates_per_launch": per_launch,
                "w_alg_thread_inst_per_candidate": w_dw,
                "peak_source": f"{n_sm} SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz ({pk_src} sm_max_mhz; DESIGN.md s8)",
                "frac_at_observed_clock": ach_a / (peak_ginst * obs / sm_max) if ach_a else None,
                "other_kernels": [{"kernel": "lgx_finish", "launch_ms": ms_c, "achieved": ach_c,
                                   "frac": ach_c / peak_ginst if ach_c else None,
                                   "w_alg_thread_inst_per_feasible_candidate": w_fin, "feasible_fraction": feas}],
                "whole_step": {"w_alg_thread_inst_per_candidate": w_dw + feas * w_fin, "achieved": ach_all,
                               "frac": ach_all / peak_ginst},
                "hbm_note": "queue traffic ~%.0f B per candidate; dram bytes per launch in profiles/ (negligible)" % (feas * info["record_bytes"])}

    cpu = None
    if not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_cpu = 1 << 21 if args.workload in ("toy", "small", "medium") else 1 << 18
        rate, dt, cbest = oracle_rate(args.workload, n_cpu, cores)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"ids [0, {n_cpu // cores * cores}) of the {args.workload} budget, {cores} processes, {dt:.1f} s wall"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: N_T={inst.n_tours} N_B={inst.n_bps} N_F={inst.n_fields} "
                                   f"N_HU={inst.n_hu} N_SU={inst.n_su}",
                       "candidates_per_gpu_per_step": per_gpu, "seed": inst.seed,
                       "l2": "flushed between timed iterations (256 MiB write)",
                       "parallelism": f"id-range shards x{world}", "threads_per_block": info["threads"],
                       "grid": info["grid"], "smem_bytes": info["smem_bytes"]},
            "best": {"cost": best[0], "id": best[1]},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": info["image_bytes"],
                    "d2h_bytes_per_step": 16, "steps": e2e_steps,
                    "what": "lgx_instance_create(host arrays) + lgx_search + lgx_instance_destroy, wall clock"},
            "wall_s_timed_region": t_wall, "roofline": roofline, "cpu_baseline": cpu}
    line.update(extra)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
