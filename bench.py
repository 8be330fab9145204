#!/usr/bin/env python
"""bench.py — candidates/s of the lgx hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (the persistent kernel
pair lgx_decode_cut + lgx_walk_finish per chunk, over the shared-memory images built by a1) over
one batch of candidates:
`lgx_search` over the Medium config's full budget (2^28 ids, 100 fields / 8 BPs / 5 tours;
the config the north_star target of >= 1e9 cand/s is quoted on).  Synthetic, seeded
instance (paper_1909_10286_b200/workloads.py); nothing is read from /root/reference.
Beside the headline the line carries `configs` (lgx_search and lgx_eval_batch timed separately on toy, small,
medium, large, sweep and paper_scale, each with its roofline fractions) and `best_vs_oracle` (the GPU's (cost, id)
over an id prefix against the oracle's, bit for bit: the second half of BASELINE.json's metric).

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
ALL_CONFIGS = ("toy", "small", "medium", "large", "sweep", "paper_scale")
# log2 of the ids per lgx_search step / per lgx_eval_batch call of the `configs` leg (about 0.3-1 s of GPU time each),
# and of the id prefix [0, 2^k) the oracle scans for `best_vs_oracle` (about 1 s on the host cores each)
CONFIG_SEARCH_LOG2 = {"toy": 30, "small": 30, "medium": 29, "large": 28, "sweep": 26, "paper_scale": 25}
CONFIG_EVAL_LOG2   = {"toy": 24, "small": 24, "medium": 24, "large": 24, "sweep": 23, "paper_scale": 22}
ORACLE_PREFIX_LOG2 = {"toy": 21, "small": 21, "medium": 21, "large": 19, "sweep": 18, "paper_scale": 17}


def w_alg(inst, a2_iters):
    """MODEL, not a measurement: thread-instructions the method itself needs per candidate.
    Returns (round-1 model: decode + pass 1 for every candidate, the rest for feasible ones;
             strict model of the round-2 kernel split: (every candidate, feasible candidate))."""
    nf, nb, nt, nhu, nsu = inst.n_fields, inst.n_bps, inst.n_tours, inst.n_hu, inst.n_su
    cd = lambda a, b: -(-a // b)
    part_blocks = lambda n: cd(n, 4) + cd(n - nt, 4)            # Philox blocks of one ordered partition
    blocks_a = cd(nf, 4) + part_blocks(nb) + cd((nb - 1) * 4 // 3 + 8, 4)
    decode = 40 * blocks_a + 7 * (nf + nb) + 2 * (nb - nt) + 6 * nb
    pass1 = 14 * nf + 10 * (nb + nt)
    blocks_c = part_blocks(nhu) + part_blocks(nsu)
    finish = (40 * blocks_c + 7 * (nhu + nsu) + 2 * (nhu + nsu - 2 * nt) + 6 * nhu + 10 * nsu
              + 6 * nb + 92 * nt + 110 * a2_iters + 18 * nf + 10 * (nb + nt) + 9 * nt + 5)
    # round 2: lgx_decode_cut decides the cuts and eq. (2) on quanta alone (s_q look-up, add, compare, extras bit:
    # 6 per field, 4 per BP); the geometry of pass 1 (8 per field + the flushes) is paid by feasible candidates only
    cut = 6 * nf + 4 * nb
    geo1 = 8 * nf + 10 * (nb + nt)
    return (decode + pass1, finish), (decode + cut, geo1 + finish)


def w_alg_coords(inst, a2_iters, mode):
    """The same MODEL with the distances computed from coordinates (a leg = 2 sub, 2 mul, 1 add and an
    FP64 square root ~ 20 thread-instructions instead of one table look-up ~ 3).  Distance mode 1 (coordinates only):
    the field->BP leg of pass 1, the route leg and the field->BP leg of pass 2 = 3 legs per field; mode 2 (field x BP
    table + coordinates): the route leg only.  Returns the walk/finish kernel's work per feasible candidate."""
    (_, _), (_, w_b) = w_alg(inst, a2_iters)
    legs = {0: 0, 1: 3, 2: 1}[mode]
    return w_b + 17 * legs * inst.n_fields


# PROFILE CONSTANTS (not measured in this run): each pipe's utilisation (sm__inst_executed_pipe_*.avg.pct_of_peak_sustained_active)
# in ONE captured launch of each kernel, with that launch's duration and candidates, from the `ncu --set full` capture named
# per entry.  pipes_of() scales them to this run's time per candidate; the binding pipe is the busiest one.  The pipe peaks
# measured IN this run (lgx_selftest 1..5, `pipe_peaks`) say what those pipes sustain on this GPU: ALU 2, FP64 2, IMAD.WIDE 1,
# shared-memory byte accesses 1, MUFU.RSQ64H 0.5 warp-instructions/clk/SM against the schedulers' 4.
PIPE_MIX = {
    "medium": {"file": "profiles/r03_medium_ncu_full.md",
               "lgx_decode_cut":  {"ms": 3.862624, "candidates": 16777216, "pct": {"alu": 57.93, "fma": 26.90, "lsu": 43.59, "fp64": 0.0, "xu": 0.66}},
               "lgx_walk_finish": {"ms": 3.505408, "candidates": 16777216 * 0.23804, "pct": {"alu": 44.18, "fma": 19.13, "lsu": 29.90, "fp64": 12.75, "xu": 11.33}}},
}


PIPE_OF = {"alu": "alu_lop3", "fma": "imad_wide_u32", "lsu": "lds_sts_u8", "fp64": "fp64_dfma", "xu": "mufu_rsq64h"}


def pipe_peaks(binding, n_sm):
    """Sustained warp-instructions per clock per SM of five pipes, measured by lgx_selftest what = 1..5."""
    names = {1: "imad_wide_u32", 2: "alu_lop3", 3: "lds_sts_u8", 4: "fp64_dfma", 5: "mufu_rsq64h"}
    out = {}
    for what, nm in names.items():
        binding.selftest(what, 1 << 10)
        n_inst, cyc = binding.selftest(what, 1 << 14)
        out[nm] = n_inst / max(cyc, 1) / n_sm
    out["unit"] = "warp-instructions / clk / SM (scheduler limit: 4)"
    out["how"] = "lgx_selftest what=1..5: 8 independent chains per thread, 2 x 1024 threads per SM, cycles by clock64 in the kernel"
    return out


SM_MAX_MHZ_FALLBACK = 1965.0
# PROFILE CONSTANTS (not measured in this run): dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the
# config's dominant kernel from the `ncu --set full` captures summarised under profiles/ (file named per entry),
# with the candidates that launch covered.  The path's algorithmic HBM bytes are 0 per candidate in lgx_search
# (everything lives in shared memory and the L2-resident queue); these numbers show the real traffic is negligible.
TRAFFIC = {
    # name: (capture, candidates the captured kernel pair covered, bytes of lgx_decode_cut, bytes of lgx_walk_finish)
    "medium":      ("profiles/r03_medium_ncu_full.md", 16777216, 4.412e+08, 5.019e+08),
    "large":       ("profiles/r03_large_ncu_full.md", 932068, 1.765e+08, 2.399e+08),
    "sweep":       ("profiles/r03_sweep_ncu_full.md", 123362, 3.452e+07, 9.736e+07),
    "paper_scale": ("profiles/r03_paper_scale_ncu_full.md", 188206, 3.838e+08, 8.302e+08),
}


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
    processes over disjoint contiguous id ranges on the host cores.  Returns (ids/s, seconds, (cost, id) of the
    ordered minimum over ids [0, n_ids // procs * procs))."""
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


def _oracle_a2_chunk(name, first, n):
    """Accepted Algorithm-2 moves (scalars[7] of lgo_score) of the feasible candidates among ids [first, first+n)."""
    import numpy as np
    from oracle import lgo
    from paper_1909_10286_b200 import workloads as wl
    inst = wl.make(name)
    o = lgo.Oracle(inst)
    sc = np.zeros(8)
    moves = feas = 0
    for i in range(first, first + n):
        pl = o.decode(inst.seed, i)
        o.score_fast(pl["bp_tour"], pl["bp_pos"], pl["field_bp"], pl["field_pos"], pl["hu_tour"], pl["su_tour"], sc)
        if sc[0] != 0.0:
            feas += 1; moves += int(sc[7])
    return moves, feas


def oracle_alg2_iters(name, n_ids, procs):
    """Mean number of accepted Algorithm-2 moves per feasible candidate, measured with the oracle on ids [0, n_ids):
    the `A2` of the work model."""
    import multiprocessing as mp
    per = max(1, n_ids // procs)
    with mp.get_context("fork").Pool(procs) as pool:
        res = pool.starmap(_oracle_a2_chunk, [(name, r * per, per) for r in range(procs)])
    moves = sum(r[0] for r in res); feas = sum(r[1] for r in res)
    return (moves / feas if feas else 0.0), feas, per * procs


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
    ap.add_argument("--walk-lockstep", type=int, default=None, help="LGX_OPT_WALK_LOCKSTEP (tuning)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--alg1-workload", default="paper_scale", help="instance of the Algorithm 1 leg (SURVEY §8(f) N1/N3)")
    ap.add_argument("--alg1-iters", type=int, default=500)
    ap.add_argument("--no-alg1", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config leg (toy .. paper_scale)")
    ap.add_argument("--torchrun", action="store_true",
                    help="start the ranks through torch.distributed.run even for --gpus 1 (always done for --gpus N > 1 when no launcher did)")
    args = ap.parse_args()
    if args.impl == "lgx" and "WORLD_SIZE" not in os.environ and (args.gpus > 1 or args.torchrun):
        # `python bench.py --gpus N` run plainly: become N ranks, one per GPU, the way the driver launches them
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")             # the communicator's rank lines reach stderr
        env["LGX_BENCH_LAUNCHER"] = "bench.py -> torch.distributed.run"
        argv = [a for a in sys.argv[1:] if a != "--torchrun"]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + argv
        os.execvpe(sys.executable, cmd, env)
    args.warmup = max(args.warmup, 3) if args.impl == "lgx" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    from paper_1909_10286_b200 import binding, workloads as wl, sharding

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s) (WORLD_SIZE); they must agree")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    if local >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} wants cuda:{local}, the node has {torch.cuda.device_count()} GPU(s)")
    torch.cuda.set_device(local)
    dist = None
    if "WORLD_SIZE" in os.environ:                       # under a launcher: NCCL even for one rank, so the exchange path runs
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    inst = wl.make(args.workload)
    per_gpu = 1 << (args.batch_log2 if args.batch_log2 is not None else min(28, inst.budget.bit_length() - 1))
    total = per_gpu * world                      # weak scaling: fixed ids per GPU
    opts = ((4, args.chunk_log2), (1, args.threads_a), (2, args.threads_b), (7, args.walk_lockstep))

    def new_instance(ins):
        gi = binding.Instance(ins)
        for key, val in opts:
            if val is not None:
                gi.set_option(key, val)
        return gi

    g = new_instance(inst)
    info = g.info()
    binding_mode = {args.workload: info["coords"]}           # distance mode per config (lgx_instance_query 4)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step(first_total=0):
        # this rank's contiguous share of [0, total); one 24-byte exchange when world > 1
        if dist is None:
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
    rank_ms = [dev_ms / args.steps]
    if dist is not None:
        t = torch.tensor([dev_ms], dtype=torch.float64, device="cuda")
        allt = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(allt, t)
        rank_ms = [float(x.item()) / args.steps for x in allt]      # device ms per step of every rank
        dev_ms = max(float(x.item()) for x in allt)                  # the job's time: max over ranks
    value = total * args.steps / (dev_ms * 1e-3)

    # ---- e2e: host arrays -> lgx_instance_create (H2D image) -> lgx_search -> host result
    e2e_steps = max(2, min(args.steps, 3))

    def e2e_step():
        g2 = new_instance(inst)
        if dist is None:
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
    # the same step with the library's workspace pool emptied first: what the FIRST call of a process pays
    # (the driver maps the queue of feasible candidates again, ~150 ms per 2 GiB)
    e2e_cold = None
    if world == 1:
        binding.workspace_trim()
        torch.cuda.synchronize()
        t0 = time.perf_counter(); r3 = e2e_step(); torch.cuda.synchronize(); cold_s = time.perf_counter() - t0
        assert r3 == best
        e2e_cold = {"value": total / cold_s, "unit": UNIT, "seconds": cold_s,
                    "what": "one e2e step right after lgx_workspace_trim(): the queue's memory is mapped again inside the step"}

    def time_eval_batch(gi, ins, n_ev, n_h):
        """lgx_eval_batch (per-candidate outputs): median of 3 device-timed calls, plus one call with host buffers."""
        out = gi.eval_batch(ins.seed, first_id=0, n=n_ev)
        torch.cuda.synchronize()
        ev_list = []
        for _ in range(3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); gi.eval_batch(ins.seed, first_id=0, n=n_ev, out=out); b.record(stream)
            torch.cuda.synchronize()
            ev_list.append(a.elapsed_time(b))
        ev_ms = sorted(ev_list)[1]
        res = {"value": n_ev / ev_ms * 1e3, "unit": UNIT, "ids": n_ev,
               "feasible_fraction": float(out[3].float().mean().item())}
        if n_h:
            # page-locked host buffers (the caller's choice; pageable ones work too, without the overlap of copies and kernels)
            host_out = tuple(torch.empty(n_h, dtype=dt, pin_memory=True).numpy() for dt in (torch.float64, torch.float64, torch.float64, torch.uint8))
            gi.eval_batch_host(ins.seed, first_id=0, n=n_h, out=host_out)
            t0 = time.perf_counter(); gi.eval_batch_host(ins.seed, first_id=0, n=n_h, out=host_out); th = time.perf_counter() - t0
            res["e2e_host_buffers"] = {"value": n_h / th, "unit": UNIT, "ids": n_h, "d2h_bytes": 25 * n_h, "h2d_bytes": 0}
        return res

    extra = {}
    if rank == 0:
        extra["eval_batch"] = time_eval_batch(g, inst, 1 << 24, 1 << 22)

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
    cores = os.cpu_count() or 1
    ppeaks = pipe_peaks(binding, n_sm)                       # measured in this run (five short kernels)

    def pipes_of(name, kernel, ms_per_cand):
        """Utilisation of each pipe by `kernel` in this run: the captured launch's utilisation (profile constant, PIPE_MIX)
        scaled by captured / current time per candidate.  The binding pipe is the busiest."""
        mix = PIPE_MIX.get(name, {}).get(kernel)
        if not mix or ms_per_cand <= 0:
            return None
        scale = (mix["ms"] / mix["candidates"]) / ms_per_cand
        util = {pipe: pct / 100.0 * scale for pipe, pct in mix["pct"].items()}
        bind = max(util, key=util.get)
        return {"binding_pipe": bind, "frac_of_binding_pipe": util[bind], "pipe_utilisation": util,
                "binding_pipe_peak_warp_inst_per_clk_per_sm": ppeaks.get(PIPE_OF[bind]),
                "source": "pipe utilisation of the captured launch in %s (profile constant) scaled to this run's time per candidate; "
                          "pipe peaks measured in this run" % PIPE_MIX[name]["file"]}

    def roofline_of(ins, name, feas, a2, rate_per_gpu, ns_a_, ns_b_, pairs, cand_timed, rec_bytes):
        """Issue roofline of one config from the work MODEL w_alg (a model) and the measured kernel times."""
        (w_dw, w_fin), (w_a, w_b) = w_alg(ins, a2)
        per_launch = cand_timed / max(pairs, 1)
        ms_a_ = ns_a_ * 1e-6 / max(pairs, 1); ms_b_ = ns_b_ * 1e-6 / max(pairs, 1)
        ach_a = per_launch * w_a / (ms_a_ * 1e-3) / 1e9 if ms_a_ > 0 else None
        ach_b = per_launch * feas * w_b / (ms_b_ * 1e-3) / 1e9 if ms_b_ > 0 else None
        a_dominant = ns_a_ >= ns_b_
        ach_d, ms_d = (ach_a, ms_a_) if a_dominant else (ach_b, ms_b_)
        ach_r1 = (w_dw + feas * w_fin) * rate_per_gpu / 1e9
        ach_strict = (w_a + feas * w_b) * rate_per_gpu / 1e9
        mode = {"toy": 0, "small": 0, "medium": 0}.get(name)
        w_b_coords = None
        if ms_b_ > 0:
            try:
                mode = binding_mode[name]
            except KeyError:
                pass
            if mode:
                w_b_coords = w_alg_coords(ins, a2, mode)
        ach_b_coords = per_launch * feas * w_b_coords / (ms_b_ * 1e-3) / 1e9 if w_b_coords and ms_b_ > 0 else None
        # each kernel's share of the step's candidates/s: the kernel alone would run at per_launch / its launch time
        pa = pipes_of(name, "lgx_decode_cut", ms_a_ / per_launch) if ms_a_ > 0 else None
        pb = pipes_of(name, "lgx_walk_finish", ms_b_ / max(per_launch * feas, 1e-9)) if ms_b_ > 0 else None
        pd = pa if a_dominant else pb
        tr = TRAFFIC.get(name)
        if tr:      # the dominant kernel's bytes, scaled from the captured launch to this run's candidates per launch
            tr = {"file": tr[0], "candidates_per_launch": tr[1], "bytes_per_launch": (tr[2] if a_dominant else tr[3]) * per_launch / tr[1]}
        return {"bound": "alu",
                "kernel": "%s (dominant: %.0f %% of the kernel time of a step)" % ("lgx_decode_cut" if a_dominant else "lgx_walk_finish", 100.0 * max(ns_a_, ns_b_) / max(ns_a_ + ns_b_, 1)),
                "achieved": ach_d, "peak": peak_ginst, "unit": "G thread-inst/s", "frac": ach_d / peak_ginst if ach_d else None,
                "traffic": tr["bytes_per_launch"] if tr else None,
                "traffic_source": ("profile constant, not measured in this run: dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel in %s "
                                   "(%d candidates in the captured launch), scaled to this run's candidates per launch; it is the queue of "
                                   "feasible candidates, the path's algorithmic HBM bytes are 0" % (tr["file"], tr["candidates_per_launch"])) if tr else None,
                "pipe_peaks": ppeaks,
                "binding_pipe": pd["binding_pipe"] if pd else None, "frac_of_binding_pipe": pd["frac_of_binding_pipe"] if pd else None,
                "launch_ms": ms_d, "launches_timed": pairs, "candidates_per_launch": per_launch,
                "work_model": "w_alg (bench.py; DESIGN.md s8): a hand model of the thread-instructions the method needs, not a measured count; "
                              "A2 = mean accepted Algorithm-2 moves, oracle-measured in this run",
                "alg2_moves_mean": a2,
                "peak_source": f"{n_sm} SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz ({pk_src} sm_max_mhz; DESIGN.md s8)",
                "kernels": [{"kernel": "lgx_decode_cut", "launch_ms": ms_a_, "achieved": ach_a, "frac": ach_a / peak_ginst if ach_a else None,
                             "w_alg_thread_inst_per_candidate": w_a, "pipes": pa},
                            {"kernel": "lgx_walk_finish", "launch_ms": ms_b_, "achieved": ach_b, "frac": ach_b / peak_ginst if ach_b else None,
                             "w_alg_thread_inst_per_feasible_candidate": w_b, "feasible_fraction": feas, "pipes": pb,
                             "coordinate_model": ({"distance_mode": mode, "w_alg_thread_inst_per_feasible_candidate": w_b_coords,
                                                   "achieved": ach_b_coords, "frac": ach_b_coords / peak_ginst,
                                                   "model": "w_alg + 17 thread-inst per leg computed from coordinates (SURVEY.md s8(d)): "
                                                            "3 legs per field in mode 1, 1 in mode 2"} if ach_b_coords else None)}],
                "whole_step": {"w_alg_thread_inst_per_candidate": w_dw + feas * w_fin, "achieved": ach_r1, "frac": ach_r1 / peak_ginst,
                               "model": "round-1 model (unchanged): decode + pass 1 charged to every candidate"},
                "whole_step_strict": {"w_alg_thread_inst_per_candidate": w_a + feas * w_b, "achieved": ach_strict, "frac": ach_strict / peak_ginst,
                                      "model": "round-2 kernel split: pass-1 geometry charged to feasible candidates only (PAPER.md L186)"},
                "kernel_time_share_of_step": (ns_a_ + ns_b_) * 1e-6 / max(cand_timed / rate_per_gpu * 1e3, 1e-9),
                "hbm_note": "queue traffic ~%.0f B per candidate, L2-resident in practice; algorithmic HBM bytes of lgx_search: 0" % (feas * rec_bytes)}

    def best_vs_oracle(gi, ins, name):
        """The second half of the metric: the GPU's (cost, id) over an id prefix must equal the oracle's, bit for bit."""
        n_pre = 1 << ORACLE_PREFIX_LOG2.get(name, 18)
        rate, dt, cbest = oracle_rate(name, n_pre, cores)
        n_scanned = n_pre // cores * cores
        gbest = gi.search(ins.seed, n_scanned)
        return {"ids": n_scanned, "oracle": {"cost": cbest[0], "id": cbest[1]}, "lgx": {"cost": gbest[0], "id": gbest[1]},
                "match": bool(gbest[0] == cbest[0] and gbest[1] == cbest[1])}, rate, dt

    feas = extra.get("eval_batch", {}).get("feasible_fraction", 1.0)
    a2_main = 0.0
    cpu = None
    bvo = None
    if not args.no_cpu_baseline:
        a2_main, _, _ = oracle_alg2_iters(args.workload, 2048 if inst.n_fields <= 250 else 512, cores)
        bvo, rate, dt = best_vs_oracle(g, inst, args.workload)
        n_cpu = 1 << 23 if args.workload in ("toy", "small", "medium") else 1 << 19
        rate, dt, _ = oracle_rate(args.workload, n_cpu, cores)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"ids [0, {n_cpu // cores * cores}) of the {args.workload} budget, {cores} processes, {dt:.1f} s wall"}
    else:
        a2_main = {"toy": 2.3, "small": 5.5, "medium": 9.8, "large": 12.9, "sweep": 18.5, "paper_scale": 8.4}.get(args.workload, 10.0)
    roofline = roofline_of(inst, args.workload, feas, a2_main, value / world, ns_a, ns_c, n_pairs, per_gpu * args.steps, info["record_bytes"])

    # ---- every config (BASELINE.json: "on all five configs", config 5: lgx_eval_batch and lgx_search timed separately)
    configs = {}
    if world == 1 and not args.no_configs:
        for name in ALL_CONFIGS:
            ins = wl.make(name)
            gi = g if name == args.workload and not any(v is not None for _, v in opts) else binding.Instance(ins)
            binding_mode[name] = gi.query(4)
            n_s = 1 << CONFIG_SEARCH_LOG2[name]
            gi.search(ins.seed, n_s // 4); gi.search(ins.seed, n_s // 4); gi.search(ins.seed, n_s // 4)      # W = 3 warm-up calls
            # the reported rate comes from a call WITHOUT the per-kernel timing hook (which creates and records three events
            # per kernel pair inside the call); a second call with the hook gives the kernel split only
            l0 = gi.query(7)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            flush.fill_(1); a.record(stream)
            cbest = gi.search(ins.seed, n_s)
            b.record(stream); torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            n_launch = gi.query(7) - l0
            gi.set_timing(True)
            flush.fill_(2)
            assert gi.search(ins.seed, n_s) == cbest
            ka, kb, kp = gi.kernel_times(); gi.set_timing(False)
            evb = time_eval_batch(gi, ins, 1 << CONFIG_EVAL_LOG2[name], 0)
            c = {"workload": f"N_T={ins.n_tours} N_B={ins.n_bps} N_F={ins.n_fields} N_HU={ins.n_hu} N_SU={ins.n_su}",
                 "lgx_search": {"value": n_s / ms * 1e3, "unit": UNIT, "ids": n_s, "ms": ms, "gpu_launches": n_launch,
                                "best": {"cost": cbest[0], "id": cbest[1]}},
                 "lgx_eval_batch": evb, "threads_per_block": [gi.query(1), gi.query(8)], "distance_mode": gi.query(4)}
            if not args.no_cpu_baseline:
                a2, _, _ = oracle_alg2_iters(name, 1024 if ins.n_fields <= 250 else 256, cores)
                c["best_vs_oracle"], orate, odt = best_vs_oracle(gi, ins, name)
                c["cpu_baseline"] = {"value": orate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                     "sample": f"ids [0, {c['best_vs_oracle']['ids']}), {odt:.1f} s wall"}
            else:
                a2 = {"toy": 2.3, "small": 5.5, "medium": 9.8, "large": 12.9, "sweep": 18.5, "paper_scale": 8.4}[name]
            r = roofline_of(ins, name, evb["feasible_fraction"], a2, n_s / ms * 1e3, ka, kb, kp, n_s, gi.query(11))
            c["roofline"] = {k: r[k] for k in ("kernel", "frac", "binding_pipe", "frac_of_binding_pipe", "launch_ms", "candidates_per_launch", "alg2_moves_mean", "kernels",
                                               "whole_step", "whole_step_strict", "kernel_time_share_of_step", "traffic", "traffic_source")}
            configs[name] = c
            if gi is not g:
                gi.close()

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: N_T={inst.n_tours} N_B={inst.n_bps} N_F={inst.n_fields} "
                                   f"N_HU={inst.n_hu} N_SU={inst.n_su}",
                       "candidates_per_gpu_per_step": per_gpu, "seed": inst.seed,
                       "l2": "flushed between timed iterations (256 MiB write)",
                       "parallelism": f"id-range shards x{world}", "threads_per_block": [info["threads"], info["threads_finish"]],
                       "grid": info["grid"], "smem_bytes": [info["smem_bytes"], info["smem_bytes_finish"]]},
            "rank_ms_per_step": rank_ms,
            "launcher": os.environ.get("LGX_BENCH_LAUNCHER", "external (torchrun)" if dist is not None else "none (single process)"),
            "best": {"cost": best[0], "id": best[1]}, "best_vs_oracle": bvo,
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": info["image_bytes"],
                    "d2h_bytes_per_step": 16, "steps": e2e_steps,
                    "what": "lgx_instance_create(host arrays) + lgx_search + lgx_instance_destroy, wall clock, with the library's "
                            "per-device workspace pool WARM (an earlier call in this process mapped the queue; the pool keeps it)",
                    "cold_first_call": e2e_cold},
            "wall_s_timed_region": t_wall, "roofline": roofline, "cpu_baseline": cpu}
    line.update(extra)
    if configs:
        line["configs"] = configs
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
