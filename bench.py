"""bench.py — plan latency (µs/layer) of the UltraEP post-gating balance step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload NAME]

A "step" is one pass of the whole hot path (uep_balance = histogram -> plan -> remap || pack)
over one (layer, microbatch) instance of the DeepSeek-V3-like prefill workload
(BASELINE.json configs[2]: E=256, k=8, R=64, 2 redundant slots, 262144 tokens, fp32 gates,
bf16 expert state 3x[7168x2048] per expert).  Inputs are seeded synthetic Zipf routing
 resident in HBM before the timed region; the step rotates over 32 distinct
instances (0.5 GB of ids+gates, > the 126 MB L2) and each pack moves several GB, so every
timed pass is L2-cold.

One JSON line on stdout (rank 0).  `value` = plan latency: device µs per layer of
histogram+plan+remap (graph-captured, CUDA events); `ms_per_step` = the whole step incl. the
pack; `stages_us` breaks it down; `roofline` is the dominant kernel (pack) and `rooflines`
lists the three HBM-bound kernels.  See DESIGN.md §7 for the arithmetic.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "plan latency us/layer (histogram+plan+remap, device time)"
UNIT = "us/layer"
N_INSTANCES = 32          # distinct (layer, microbatch) inputs the step rotates over
BASE_SEED = 20260604


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=64)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="uep", choices=["uep", "reference"])
    ap.add_argument("--workload", default="dsv3_prefill",
                    choices=["tiny", "glm_air", "dsv3_prefill", "dsv3_train"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--size-sweep", action="store_true",
                    help="instead of the bench line: stage times and roofline fractions at E=256, k=8, "
                         "R=64 over S = 256 Ki .. 16 Mi slots, one JSON line per size (DESIGN.md §7)")
    ap.add_argument("--pack-grid-sweep", action="store_true",
                    help="instead of the bench line: uep_pack and uep_grad_reduce throughput over the number of "
                         "streaming CTAs (developer override UEP_PACK_CTAS), one JSON line per grid size")
    ap.add_argument("--state-scale", type=float, default=1.0,
                    help="shrink bytes per expert (debug only; the line then says so)")
    return ap.parse_args()


def measured_peaks():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written), else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thr = threading.Thread(target=self._read, daemon=True)
        self.thr.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(name: str, state_scale: float = 1.0):
    from paper_2606_04101_b200 import synth
    c = dict(synth.CONFIGS[name])
    state = []
    for nm, elems, dt in c["state"]:
        elems = max(8, int(elems * state_scale) // 8 * 8)
        state.append((nm, elems, dt))
    c["state"] = state
    return c


def instance_inputs(c, idx: int, device):
    """ids/gates of instance idx (fresh permutation per instance; Zipf s per the config)."""
    from paper_2606_04101_b200 import synth
    seed = synth.instance_seed(BASE_SEED, idx // 4, idx % 4)
    s = c["zipf_s"] if c["zipf_s"] is not None else synth.train_sweep_s(BASE_SEED, idx // 4, idx % 4)
    ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], s, seed, device=device)
    if c["gate"] == "bf16":
        gate = synth.gates_softmax_bf16(c["T"], c["k"], seed, device=device)
    else:
        gate = synth.gates_uniform_renorm(c["T"], c["k"], seed, device=device)
    return ids, gate, s


# ------------------------------------------------------------------------------------------
# uep arm
# ------------------------------------------------------------------------------------------
_DT = {"bf16": ("bfloat16", 2), "f32": ("float32", 4)}


class Rig:
    """All device buffers of one rank: N_INSTANCES input sets, one output/plan set each
    (so that graph-captured chains over different instances do not alias), resident state."""

    def __init__(self, c, device, n_inst, inst_base=0):
        import torch
        from paper_2606_04101_b200 import binding, synth
        self.c, self.device, self.n_inst = c, device, n_inst
        gd = binding.GATE_BF16 if c["gate"] == "bf16" else binding.GATE_F32
        self.ctx = binding.Context(c["T"], c["k"], c["E"], c["R"], c["n_slot"], c["u_min"],
                                   gate_dtype=gd, device=device)
        self.ids, self.gates, self.zipf = [], [], []
        for i in range(n_inst):
            ids, gate, s = instance_inputs(c, inst_base + i, device)
            self.ids.append(ids); self.gates.append(gate); self.zipf.append(s)
        self.ws = [self.ctx.new_workspace() for _ in range(n_inst)]
        self.plans = [self.ctx.new_plan() for _ in range(n_inst)]
        self.counts = [torch.zeros(c["E"], dtype=torch.int32, device=device) for _ in range(n_inst)]
        self.outs = [self.ctx.new_outputs(self.gates[i]) for i in range(n_inst)]
        self.src, self.dst = [], []
        for j, (nm, elems, dt) in enumerate(c["state"]):
            tdt = getattr(torch, _DT[dt][0])
            self.src.append(synth.expert_state(c["E"], elems, 7 + j, dtype=tdt, device=device))
            self.dst.append(torch.zeros((c["R"], c["n_slot"], elems), dtype=tdt, device=device))
        self.state_bytes_per_expert = sum(e * _DT[dt][1] for _, e, dt in c["state"])
        torch.cuda.synchronize(device)

    # one step = uep_balance on instance i
    def balance(self, i, with_pack=True):
        o = self.outs[i]
        self.ctx.uep_balance(self.ids[i], self.gates[i], self.counts[i], self.plans[i], o[0], o[1],
                             o[2], o[3], self.src if with_pack else [], self.dst if with_pack else [],
                             self.ws[i])

    def hist(self, i):
        self.ctx.uep_histogram(self.ids[i], self.counts[i], self.ws[i])

    def plan(self, i):
        self.ctx.uep_plan(self.counts[i], self.plans[i], self.ws[i])

    def remap(self, i):
        o = self.outs[i]
        self.ctx.uep_remap(self.ids[i], self.gates[i], self.plans[i], o[0], o[1], o[2], o[3],
                           self.ws[i])

    def rank(self, i):
        self.ctx.uep_remap_rank(self.ids[i], self.ws[i])

    def lookup(self, i):
        o = self.outs[i]
        self.ctx.uep_remap_lookup(self.gates[i], self.plans[i], o[0], o[1], o[2], o[3], self.ws[i])

    def pack(self, i):
        self.ctx.uep_pack(self.plans[i], self.src, self.dst)


def capture(fn_list, stream):
    """Capture a list of callables (each launching on the current stream) into one CUDA graph."""
    import torch
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(stream):
        with torch.cuda.graph(g, stream=stream):
            for fn in fn_list:
                fn()
    return g


def time_graph(g, stream, reps, warm=2):
    """Median and min device ms of `reps` replays (CUDA events on the replay stream)."""
    import torch
    with torch.cuda.stream(stream):
        for _ in range(warm):
            g.replay()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(reps)]
        for a, b in evs:
            a.record(stream)
            g.replay()
            b.record(stream)
    stream.synchronize()
    ts = [a.elapsed_time(b) for a, b in evs]
    return statistics.median(ts), min(ts)


def dist_setup(args):
    """One process per GPU under torchrun; plain single process otherwise."""
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 or (os.environ.get("UEP_BENCH_FORCE_PG") == "1" and "RANK" in os.environ):
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if torch.cuda.is_available():
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return world, rank, local


def barrier_and_max(world, value_ms, device):
    """max over ranks of a device-measured time (the contract's multi-GPU timing rule)."""
    if world == 1:
        return value_ms
    from paper_2606_04101_b200 import shard
    return shard.reduce_max_time(value_ms)


def run_token_sharded(c, rig, world, rank, device, stream, reps):
    """ONE layer's tokens sharded over the `world` GPUs (the paper's deployment,
    PAPER.md:162): uep_shard_count -> in-place all-gather of the count rows -> uep_shard_finish
    (identical plan on every GPU, lookup of the local slots).  world == 1 is the whole problem on
    one GPU.  All ranks take their slice of the SAME seeded instances."""
    import torch
    import torch.distributed as dist
    from paper_2606_04101_b200 import binding, shard
    n = min(4, rig.n_inst)
    S = c["T"] * c["k"]
    Sl = S // world
    ids_l, gate_l = [], []
    for i in range(n):
        if world == 1:
            ids, gate = rig.ids[i], rig.gates[i]
        else:                               # same instance on every rank, then this rank's slots
            ids, gate, _ = instance_inputs(c, 100000 + i, device)
        ids_l.append(ids.reshape(-1)[rank * Sl:(rank + 1) * Sl].clone())
        gate_l.append(gate.reshape(-1)[rank * Sl:(rank + 1) * Sl].clone())
        del ids, gate
    layers = [shard.TokenShardedLayer(rig.ctx, rank, world) for _ in range(n)]
    with torch.cuda.stream(stream):
        for _ in range(3):
            for i in range(n):
                layers[i].step(ids_l[i], gate_l[i])
    stream.synchronize()
    use_graph = not (dist.is_available() and dist.is_initialized())
    if use_graph:
        g = capture([lambda i=i: layers[i].step(ids_l[i], gate_l[i]) for i in range(n)], stream)
        ms, _ = time_graph(g, stream, reps)
        ms /= n
    else:                                   # the collective is enqueued by torch.distributed: timed as launched
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        dist.barrier()
        torch.cuda.synchronize(device)
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(reps):
                for i in range(n):
                    layers[i].step(ids_l[i], gate_l[i])
            e1.record(stream)
        stream.synchronize()
        ms = shard.reduce_max_time(e0.elapsed_time(e1) / (reps * n))
    # every rank must hold the identical plan: compare a digest of (lambda, plan arrays) over ranks
    L0 = layers[0]
    dig = torch.stack([L0.expert_count.sum(dtype=torch.int64), L0.plan.inst_cum.sum(dtype=torch.int64),
                       L0.plan.inst_rank.sum(dtype=torch.int64), L0.plan.scalars[binding.SC_TAU].to(torch.int64)])
    same = True
    if not use_graph:
        lo, hi = dig.clone(), dig.clone()
        dist.all_reduce(lo, op=dist.ReduceOp.MIN)
        dist.all_reduce(hi, op=dist.ReduceOp.MAX)
        same = bool((lo == hi).all())
    rps = c["R"] // world
    fly = int(L0.n_inflight[rank * rps:(rank + 1) * rps].sum())
    return {"us_per_layer": round(ms * 1e3, 2), "n_shards": world, "slots_per_gpu": Sl,
            "allgather_bytes_per_gpu": layers[0].n_bytes, "cuda_graph": use_graph,
            "plans_identical_over_ranks": same, "lambda_sum": int(dig[0]),
            "inflight_ratio_this_shard": round(fly / max(Sl, 1), 4),
            "note": "uep_shard_count -> all-gather of count rows (torch.distributed, in place in the workspace) -> "
                    "uep_shard_finish; one layer of T tokens split over the GPUs (strong scaling of the plan "
                    "latency), max over ranks; `value` above is the weak-scaling instance-sharded number"}


def run_uep(args):
    import torch
    from paper_2606_04101_b200 import binding, shard
    world, rank, local = dist_setup(args)
    assert torch.cuda.is_available(), "bench.py (uep arm) needs a CUDA device; no CPU fallback"
    device = torch.device("cuda", local if world > 1 else torch.cuda.current_device())
    torch.cuda.set_device(device)
    c = workload(args.workload, args.state_scale)
    K, W = args.steps, max(args.warmup, 3)
    n_inst = min(N_INSTANCES, max(K, 1)) if args.workload != "tiny" else min(8, max(K, 1))
    rig = Rig(c, device, n_inst, shard.global_instance(rank, 0, n_inst))
    peak_gbs, peak_src = measured_peaks()
    stream = torch.cuda.Stream(device)
    # which instances this rank's K steps process (weak scaling: every rank does K steps of its
    # own instances; no data-path collective — DESIGN.md §8)
    sched = shard.step_schedule(K, n_inst, rank, world)

    def sync_all():
        torch.cuda.synchronize(device)
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
            torch.cuda.synchronize(device)

    # ---- warm-up (also builds every plan, needed by the stage graphs below) -----------------
    with torch.cuda.stream(stream):
        for w in range(max(W, n_inst)):
            rig.balance(w % n_inst)
    sync_all()

    # ---- timed region: exactly K whole steps -------------------------------------------------
    sampler = ClockSampler(device.index or 0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for i in sched:
            rig.balance(i)
        e1.record(stream)
    sync_all()
    step_ms_local = e0.elapsed_time(e1)
    step_ms = barrier_and_max(world, step_ms_local, device)

    # ---- stage timing: graph-captured chains over all instances (L2-cold by rotation) --------
    reps = 5
    # the chain is uep_balance without state tensors: histogram -> plan -> lookup on the stream,
    # the rank half of the remap forked beside histogram + plan (as the library schedules it)
    chain = capture([lambda i=i: rig.balance(i, with_pack=False) for i in range(n_inst)], stream)
    g_rank = capture([lambda i=i: rig.rank(i) for i in range(n_inst)], stream)
    g_lookup = capture([lambda i=i: rig.lookup(i) for i in range(n_inst)], stream)
    g_hist = capture([lambda i=i: rig.hist(i) for i in range(n_inst)], stream)
    g_plan = capture([lambda i=i: rig.plan(i) for i in range(n_inst)], stream)
    g_remap = capture([lambda i=i: rig.remap(i) for i in range(n_inst)], stream)
    chain_ms, chain_min = time_graph(chain, stream, reps)
    hist_ms, _ = time_graph(g_hist, stream, reps)
    plan_ms, _ = time_graph(g_plan, stream, reps)
    remap_ms, _ = time_graph(g_remap, stream, reps)
    rank_ms, _ = time_graph(g_rank, stream, reps)
    lookup_ms, _ = time_graph(g_lookup, stream, reps)
    n_pack = min(n_inst, 8)
    g_pack = capture([lambda i=i: rig.pack(i) for i in range(n_pack)], stream)
    pack_ms, _ = time_graph(g_pack, stream, 3, warm=1)
    # NEXT-4: all instances' planners in ONE launch, one cluster per instance
    import torch as _t
    counts_all = _t.stack(rig.counts).contiguous()
    bplan = rig.ctx.new_plan(batch=n_inst)
    _t.cuda.synchronize(device)
    g_bplan = capture([lambda: rig.ctx.uep_plan_batched(n_inst, counts_all, bplan)], stream)
    bplan_ms, _ = time_graph(g_bplan, stream, reps)
    # NEXT-2: backward gradient reduction (fp32, one [7168 x 2048]-like matrix per
    # expert for the DSV3 shapes) and the inverse remap, on the plans of this run
    g_elems = 7168 * 2048 if c["E"] >= 256 else (4096 * 1408 if c["E"] >= 128 else 256 * 512)
    g_elems = max(8, int(g_elems * args.state_scale) // 8 * 8)
    main_grad = _t.ones((c["E"], g_elems), dtype=_t.float32, device=device)
    slot_grad = _t.ones((c["R"], max(c["n_slot"], 1), g_elems), dtype=_t.float32, device=device)
    out_src = _t.empty(S_slots := c["T"] * c["k"], dtype=_t.int32, device=device)
    n_red = min(n_inst, 4)
    _t.cuda.synchronize(device)
    g_red = capture([lambda i=i: rig.ctx.uep_grad_reduce(rig.plans[i], [main_grad], [slot_grad])
                     for i in range(n_red)], stream)
    red_ms, _ = time_graph(g_red, stream, 3, warm=1)
    g_inv = capture([lambda i=i: rig.ctx.uep_remap_inverse(rig.outs[i][1], rig.outs[i][2], rig.plans[i], out_src)
                     for i in range(n_inst)], stream)
    inv_ms, _ = time_graph(g_inv, stream, reps)
    # NEXT-1: source-aware reroute; in-flight token ratio against the global remap
    local = None
    if c["T"] % c["R"] == 0:
        infl = [_t.zeros(c["R"], dtype=_t.int32, device=device) for _ in range(n_inst)]
        src_rank = (_t.arange(c["T"], device=device, dtype=_t.int64) * c["R"] // c["T"]).to(_t.int32)
        glob_fly = []
        for i in range(min(n_inst, 4)):      # the global remap's outputs are still in rig.outs
            glob_fly.append(int((rig.outs[i][1] != src_rank[:, None]).sum()))
        g_loc = capture([lambda i=i: rig.ctx.uep_remap_local(rig.ids[i], rig.gates[i], rig.plans[i], rig.outs[i][0],
                                                            rig.outs[i][1], rig.outs[i][2], rig.outs[i][3],
                                                            infl[i], rig.ws[i]) for i in range(n_inst)], stream)
        loc_ms, _ = time_graph(g_loc, stream, reps)
        loc_fly = [int(infl[i].sum()) for i in range(min(n_inst, 4))]
        S_all = c["T"] * c["k"]
        local = {"remap_local_us": round(loc_ms * 1e3 / n_inst, 2),
                 "inflight_ratio_global": round(statistics.mean(glob_fly) / S_all, 4),
                 "inflight_ratio_local": round(statistics.mean(loc_fly) / S_all, 4),
                 "note": "uep_remap_local = rank + prefix + reroute + lookup on one stream; in-flight = slots whose "
                         "destination rank differs from their source rank floor(i*R/T) (paper: 96.0 % vs 98.4 %, "
                         "PAPER.md:440, its own traces)"}
        with _t.cuda.stream(stream):         # leave the global remap's outputs in place again
            for i in range(n_inst):
                rig.remap(i)
        stream.synchronize()
    tok = None
    if c["T"] % c["R"] == 0 and c["R"] % world == 0 and (c["T"] * c["k"]) % world == 0:
        try:
            tok = run_token_sharded(c, rig, world, rank, device, stream, reps)
        except Exception as ex:              # an extra line must never take the bench line down
            tok = {"error": repr(ex)[:300]}
    clocks = sampler.stop()
    chain_ms = barrier_and_max(world, chain_ms, device)
    # whole-job aggregate: `world` ranks each planned n_inst layers in chain_ms (max over ranks)
    plan_latency_us = chain_ms * 1e3 / (n_inst * world)

    # ---- quality + algorithmic bytes (from the plans on the device) --------------------------
    S = c["T"] * c["k"]
    sc = [rig.plans[i].scalars.cpu().numpy() for i in range(n_inst)]
    n_rep = [int(s[binding.SC_N_REPLICAS]) for s in sc]
    n_grp = [int(s[binding.SC_N_GROUPS]) for s in sc]
    imb_after = [float(s[binding.SC_MAX_LOAD]) / (S / c["R"]) for s in sc]
    imb_before = [float(s[binding.SC_TAU_HI0]) / (S / c["R"]) for s in sc]
    B = rig.state_bytes_per_expert
    gbytes = 2 if c["gate"] == "bf16" else 4
    bytes_hist = 4 * S
    bytes_remap = (4 + gbytes + 12 + gbytes) * S
    # pack: every replicated expert is read ONCE and written once per replica
    bytes_pack = [(n_grp[i] + n_rep[i]) * B for i in range(n_pack)]
    us = lambda ms, n: ms * 1e3 / n

    # DRAM traffic per launch from the committed ncu --set full capture (dsv3_prefill only; that
    # capture is not re-taken here: a number printed under a profiler is never a bench value)
    traffic = {}
    tpath = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "r01c_traffic.csv")
    if args.workload == "dsv3_prefill" and args.state_scale == 1.0 and os.path.exists(tpath):
        with open(tpath) as f:
            for line in f.read().splitlines()[1:]:
                k_, v_ = line.rsplit(",", 1)
                traffic[k_] = int(v_)

    def roof(name, nbytes, dur_us, tkey=None):
        a = nbytes / (dur_us * 1e-6) / 1e9 if dur_us > 0 else 0.0
        return {"kernel": name, "bound": "hbm", "achieved": round(a, 1), "peak": peak_gbs,
                "unit": "GB/s", "frac": round(a / peak_gbs, 4), "frac_of_nominal_8TBs": round(a / 8000.0, 4),
                "traffic": traffic.get(tkey or name), "bytes_per_launch": int(nbytes),
                "us_per_launch": round(dur_us, 2), "peak_source": peak_src}

    pack_us = us(pack_ms, n_pack)
    r_pack = roof("pack_kernel", sum(bytes_pack) / n_pack, pack_us)
    # remap = rank_kernel + lookup_kernel: 24 B/slot algorithmic (fp32 gates) over both; each half
    # also against its own traffic (rank: 4 B id in + 4 B packed out; lookup: 4 B packed + g in,
    # 12 B + g out)
    rooflines = [r_pack, roof("rank_kernel+prefix_kernel+lookup_kernel (uep_remap)", bytes_remap, us(remap_ms, n_inst), "lookup_kernel"),
                 roof("lookup_kernel", bytes_remap, us(lookup_ms, n_inst)),
                 roof("rank_kernel+prefix_kernel (uep_remap_rank)", 8 * S, us(rank_ms, n_inst), "rank_kernel"),
                 roof("hist_kernel", bytes_hist, us(hist_ms, n_inst))]
    result = {
        "metric": METRIC, "value": round(plan_latency_us, 3), "unit": UNIT, "n_gpus": world,
        "steps": K, "warmup": W, "ms_per_step": round(step_ms / K, 4), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": args.workload, "T": c["T"], "k": c["k"], "E": c["E"], "R": c["R"],
                   "n_slot": c["n_slot"], "u_min": c["u_min"], "beta": "101/100",
                   "floor_mode": "tolerant", "gate": c["gate"],
                   "state_bytes_per_expert": B, "zipf_s": c["zipf_s"], "instances": n_inst,
                   "l2": "cold: rotates over %d distinct instances (%.0f MB of ids+gates) and "
                         "each pack streams GBs" % (n_inst, n_inst * S * (4 + gbytes) / 1e6),
                   "parallelism": "instances sharded over ranks, no collective",
                   "state_scale": args.state_scale},
        "stages_us": {"histogram": round(us(hist_ms, n_inst), 2), "plan": round(us(plan_ms, n_inst), 2),
                      "remap": round(us(remap_ms, n_inst), 2),
                      "remap_rank": round(us(rank_ms, n_inst), 2),
                      "remap_lookup": round(us(lookup_ms, n_inst), 2), "pack": round(pack_us, 2),
                      "hist_plan_remap_chain": round(plan_latency_us, 2),
                      "hist_plan_remap_chain_min": round(chain_min * 1e3 / n_inst, 2),
                      "whole_step": round(step_ms * 1e3 / K, 2)},
        "quality": {"imbalance_before": [round(min(imb_before), 3), round(statistics.mean(imb_before), 3), round(max(imb_before), 3)],
                    "imbalance_after": [round(min(imb_after), 4), round(statistics.mean(imb_after), 4), round(max(imb_after), 4)],
                    "n_replicas_mean": round(statistics.mean(n_rep), 1),
                    "max_fanout_max": max(int(s[binding.SC_MAX_FANOUT]) for s in sc),
                    "n_probes_mean": round(statistics.mean(int(s[binding.SC_N_PROBES]) for s in sc), 1)},
        "batched_plan": {"instances": n_inst, "us_total": round(bplan_ms * 1e3, 2),
                         "us_per_layer": round(bplan_ms * 1e3 / n_inst, 3),
                         "note": "uep_plan_batched: one launch, one 8-CTA cluster per instance"},
        "backward": {"grad_reduce_us": round(red_ms * 1e3 / n_red, 2),
                     "grad_reduce_bytes": int(statistics.mean(2 * (n_grp[i] + n_rep[i]) for i in range(n_red)) * g_elems * 4),
                     "grad_reduce_frac_of_peak": round(statistics.mean(2 * (n_grp[i] + n_rep[i]) for i in range(n_red))
                                                       * g_elems * 4 / (red_ms * 1e-3 / n_red) / 1e9 / peak_gbs, 4),
                     "grad_reduce_traffic": traffic.get("grad_reduce_kernel"),
                     "inverse_remap_us": round(inv_ms * 1e3 / n_inst, 2),
                     "note": "uep_grad_reduce: fp32 [E, %d] main + [R, n_slot, %d] slot grads, bytes = 2 x (groups + replicas) x B; "
                             "uep_remap_inverse: 8 B/slot read, 4 B/slot scattered write" % (g_elems, g_elems)},
        "source_aware_remap": local,
        "token_sharded": tok,
        "roofline": {k: r_pack[k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic")},
        "rooflines": rooflines,
        "gpu_launches": 6 * K,
        "clocks": clocks,
        "launch_info": rig.ctx.launch_info,
    }
    return result, rig, (world, rank, device, stream)


def run_e2e(rig, ctxinfo, steps):
    """Same step through the C ABI with HOST buffers: pinned ids+gates H2D, uep_balance
    (expert state stays resident: it is model state, not a step input), remap outputs + plan
    scalars D2H, stream sync — all inside the timed region (wall clock around the calls)."""
    import torch
    world, rank, device, stream = ctxinfo
    c = rig.c
    S = c["T"] * c["k"]
    n = min(rig.n_inst, 4)
    h_ids = [rig.ids[i].cpu().pin_memory() for i in range(n)]
    h_gate = [rig.gates[i].cpu().pin_memory() for i in range(n)]
    pin = lambda t: torch.empty(t.shape, dtype=t.dtype).pin_memory()
    o = rig.outs[0]
    h_out = [pin(o[0]), pin(o[1]), pin(o[2]), pin(o[3])]
    h_sc = torch.zeros(16, dtype=torch.int32).pin_memory()
    d_ids, d_gate = torch.empty_like(rig.ids[0]), torch.empty_like(rig.gates[0])

    def one(i, with_pack):
        rig.ctx.uep_balance_host(h_ids[i % n], h_gate[i % n], d_ids, d_gate, rig.counts[0],
                                 rig.plans[0], o[0], o[1], o[2], o[3], h_out[0], h_out[1],
                                 h_out[2], h_out[3], h_sc, rig.src if with_pack else [],
                                 rig.dst if with_pack else [], rig.ws[0], stream)

    res = {}
    for with_pack, key in ((False, "value"), (True, "whole_step_value")):
        for i in range(3):
            one(i, with_pack)
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        for i in range(steps):
            one(i, with_pack)
        torch.cuda.synchronize(device)
        res[key] = round((time.perf_counter() - t0) * 1e6 / steps, 2)
    gb = 2 if c["gate"] == "bf16" else 4
    res.update({"unit": "us/layer (wall clock around uep_balance_host: pinned ids+gates H2D, histogram+plan+remap, "
                        "remap outputs+scalars D2H, sync; whole_step_value = same call with the state tensors, i.e. "
                        "incl. pack, whose time the D2H copies overlap)",
                "h2d_bytes_per_step": S * (4 + gb), "d2h_bytes_per_step": S * (12 + gb) + 64,
                "steps": steps})
    return res


def oracle_step(c, ids_np, gate_np, pack_frac, src_np=None):
    """One bounded oracle pass: histogram + plan + remap, and the pack on 1/pack_frac of every
    expert's bytes.  Returns per-stage seconds."""
    import numpy as np
    import oracle
    t = {}
    t0 = time.perf_counter()
    lam, _ = oracle.histogram(ids_np, c["E"])
    t["histogram"] = time.perf_counter() - t0
    t0 = time.perf_counter()
    p = oracle.plan(lam, c["R"], c["n_slot"], c["u_min"], S_total=ids_np.size)
    t["plan"] = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.remap(ids_np, gate_np, p)
    t["remap"] = time.perf_counter() - t0
    if src_np is not None:
        dst = np.zeros((c["R"], c["n_slot"], src_np.shape[1]), dtype=src_np.dtype)
        t0 = time.perf_counter()
        oracle.pack(p.slot_expert, src_np, dst)
        t["pack"] = (time.perf_counter() - t0) * pack_frac
    return t, p


def cpu_inputs(c, idx):
    import numpy as np
    import torch
    ids, gate, _ = instance_inputs(c, idx, "cpu")
    g = gate.view(torch.int16).numpy().view(np.uint16) if gate.element_size() == 2 \
        else gate.view(torch.int32).numpy().view(np.uint32)
    return ids.numpy(), g


def cpu_baseline(c, n_samples=12, pack_frac=16, reps=32):
    """The oracle as it stands, single-threaded, on this box's host cores, on a bounded sample
    (about 10 s of CPU work at the DeepSeek-V3 shape: n_samples instances x reps passes of
    histogram+plan+remap, and the pack of 1/pack_frac of every expert's bytes)."""
    import numpy as np
    B = sum(e * _DT[dt][1] for _, e, dt in c["state"])
    src = np.zeros((c["E"], max(16, B // pack_frac // 16 * 16)), dtype=np.uint8)
    src[:] = np.arange(src.shape[1], dtype=np.uint8)[None, :]
    acc = {}
    for i in range(n_samples):
        ids, g = cpu_inputs(c, i)
        for r in range(reps):
            t, _ = oracle_step(c, ids, g, pack_frac, src if (i < 4 and r == 0) else None)
            for k, v in t.items():
                acc.setdefault(k, []).append(v)
    st = {k: round(statistics.mean(v) * 1e6, 1) for k, v in acc.items()}
    try:
        model = [l.split(":")[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")][0]
    except Exception:
        model = "unknown"
    return {"value": round(st["histogram"] + st["plan"] + st["remap"], 1), "unit": UNIT, "cores": 1,
            "kind": "oracle", "host_cores": os.cpu_count(), "cpu_model": model,
            "stages_us": st,
            "sample": "%d instances of the workload x %d passes of histogram+plan+remap (single thread, g++ -O2); "
                      "pack timed on 4 instances over 1/%d of each expert's bytes and scaled x%d"
                      % (n_samples, reps, pack_frac, pack_frac)}


def run_reference(args):
    """--impl reference: the oracle as it stands, timed on the host cores. Rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return None
    import oracle
    oracle.build()
    c = workload(args.workload, args.state_scale)
    K, W = args.steps, max(args.warmup, 0)
    n_in = min(4, max(1, K))
    inputs = [cpu_inputs(c, i) for i in range(n_in)]
    for w in range(min(W, 2)):
        oracle_step(c, *inputs[w % n_in], 1)
    t0 = time.perf_counter()
    for k in range(K):
        oracle_step(c, *inputs[k % n_in], 1)
    dt = time.perf_counter() - t0
    v = round(dt * 1e6 / max(K, 1), 1)
    sample = ("each step = histogram+plan+remap of one full-size instance (%d cached inputs), "
              "single thread; the pack (a memcpy of GBs) is left out of the reference step"
              % n_in)
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": K, "warmup": W,
            "ms_per_step": round(dt * 1e3 / max(K, 1), 4), "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": args.workload, "T": c["T"], "k": c["k"], "E": c["E"],
                       "R": c["R"], "n_slot": c["n_slot"], "u_min": c["u_min"]},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "host_cores": os.cpu_count(), "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def run_size_sweep(args):
    """Stage times vs problem size (same kernels, same launch rules as the library picks): shows
    which part of a stage time is fixed (launch ramp, one memory round trip, tails) and which part
    scales with bytes.  Each stage is graph-captured over 4-8 distinct instances, CUDA events."""
    import torch
    from paper_2606_04101_b200 import binding, synth
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; no CPU fallback"
    dev = torch.device("cuda", torch.cuda.current_device())
    peak_gbs, peak_src = measured_peaks()
    k, E, R, ns = 8, 256, 64, 2
    for T in (1 << 15, 1 << 16, 1 << 17, 1 << 18, 1 << 19, 1 << 20, (1 << 21) - 8):
        S = T * k
        um = synth.stress_u_min(S, R)
        n_inst = 8 if S <= (1 << 22) else 4
        ctx = binding.Context(T, k, E, R, ns, um, device=dev)
        ids = [synth.zipf_topk_ids(T, k, E, 1.0, 100 + i, device=dev) for i in range(n_inst)]
        gates = [synth.gates_uniform_renorm(T, k, i, device=dev) for i in range(n_inst)]
        ws = [ctx.new_workspace() for _ in range(n_inst)]
        plans = [ctx.new_plan() for _ in range(n_inst)]
        cnt = [torch.zeros(E, dtype=torch.int32, device=dev) for _ in range(n_inst)]
        outs = [ctx.new_outputs(gates[i]) for i in range(n_inst)]
        stream = torch.cuda.Stream(dev)
        torch.cuda.synchronize(dev)                 # workspace init ran on the default stream
        stages = {
            "histogram": lambda i: ctx.uep_histogram(ids[i], cnt[i], ws[i]),
            "plan": lambda i: ctx.uep_plan(cnt[i], plans[i], ws[i]),
            "remap_rank": lambda i: ctx.uep_remap_rank(ids[i], ws[i]),
            "remap_lookup": lambda i: ctx.uep_remap_lookup(gates[i], plans[i], *outs[i], ws[i]),
            "chain": lambda i: ctx.uep_balance(ids[i], gates[i], cnt[i], plans[i], *outs[i], [], [], ws[i]),
        }
        with torch.cuda.stream(stream):
            for i in range(n_inst):
                stages["chain"](i)
        stream.synchronize()
        us = {}
        for name, fn in stages.items():
            g = capture([lambda i=i, fn=fn: fn(i) for i in range(n_inst)], stream)
            ms, _ = time_graph(g, stream, 5)
            us[name] = ms * 1e3 / n_inst
        frac = lambda nbytes, t: round(nbytes / (t * 1e-6) / 1e9 / peak_gbs, 3)
        print(json.dumps({"slots": S, "instances": n_inst, "stages_us": {n: round(v, 2) for n, v in us.items()},
                          "frac_of_peak": {"hist_kernel (4 B/slot)": frac(4 * S, us["histogram"]),
                                           "rank+prefix (8 B/slot)": frac(8 * S, us["remap_rank"]),
                                           "lookup_kernel (24 B/slot)": frac(24 * S, us["remap_lookup"])},
                          "peak_gbs": peak_gbs, "peak_source": peak_src}), flush=True)
        del ctx, ids, gates, ws, plans, cnt, outs
        torch.cuda.synchronize(dev)


def run_pack_grid_sweep(args):
    """uep_pack / uep_grad_reduce throughput against the number of persistent CTAs (the library's
    own choice is printed first).  Same workload, plans and buffers for every grid size; every
    launch event-timed alone, median of 16; bytes = the algorithmic bytes of DESIGN.md §6."""
    import torch
    from paper_2606_04101_b200 import binding, synth
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; no CPU fallback"
    dev = torch.device("cuda", torch.cuda.current_device())
    peak_gbs, peak_src = measured_peaks()
    c = workload(args.workload, args.state_scale)
    n_inst = 4
    inputs = [instance_inputs(c, i, dev) for i in range(n_inst)]
    elems = c["state"][0][1]
    src = [synth.expert_state(c["E"], elems, 7, dtype=torch.bfloat16, device=dev)]
    dst = [torch.zeros((c["R"], c["n_slot"], elems), dtype=torch.bfloat16, device=dev)]
    g_elems = elems // 2                       # fp32 gradients of the same byte size
    mg = [torch.zeros((c["E"], g_elems), dtype=torch.float32, device=dev)]
    sg = [torch.ones((c["R"], c["n_slot"], g_elems), dtype=torch.float32, device=dev)]
    st = torch.cuda.Stream(dev)
    for n_ctas in [None, 64, 96, 112, 120, 124, 126, 128, 130, 131, 132, 133, 134, 136, 140, 144, 148]:
        if n_ctas is None:
            os.environ.pop("UEP_PACK_CTAS", None)
        else:
            os.environ["UEP_PACK_CTAS"] = str(n_ctas)
        ctx = binding.Context(c["T"], c["k"], c["E"], c["R"], c["n_slot"], c["u_min"], device=dev)
        ws = ctx.new_workspace()
        plans = [ctx.new_plan() for _ in range(n_inst)]
        cnt = torch.zeros(c["E"], dtype=torch.int32, device=dev)
        tp, tr = [], []
        with torch.cuda.stream(st):
            for i in range(n_inst):
                ctx.uep_histogram(inputs[i][0], cnt, ws)
                ctx.uep_plan(cnt, plans[i], ws)
            st.synchronize()
            moved = []
            for i in range(n_inst):
                sc = plans[i].scalars.cpu().numpy()
                moved.append(int(sc[binding.SC_N_GROUPS]) + int(sc[binding.SC_N_REPLICAS]))
            for rep in range(5):               # first pass = warm-up
                for i in range(n_inst):
                    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
                    e[0].record(st)
                    ctx.uep_pack(plans[i], src, dst)
                    e[1].record(st)
                    ctx.uep_grad_reduce(plans[i], mg, sg)
                    e[2].record(st)
                    st.synchronize()
                    if rep:
                        tp.append(moved[i] * elems * 2 / (e[0].elapsed_time(e[1]) * 1e-3) / 1e9)
                        tr.append(2 * moved[i] * g_elems * 4 / (e[1].elapsed_time(e[2]) * 1e-3) / 1e9)
        print(json.dumps({"workload": args.workload, "pack_ctas": ctx.launch_info["pack_ctas"],
                          "library_default": n_ctas is None,
                          "pack_gbs": round(statistics.median(tp), 1), "pack_frac": round(statistics.median(tp) / peak_gbs, 4),
                          "grad_reduce_gbs": round(statistics.median(tr), 1),
                          "grad_reduce_frac": round(statistics.median(tr) / peak_gbs, 4),
                          "peak_gbs": peak_gbs, "peak_source": peak_src}), flush=True)
        del ctx, ws, plans
    os.environ.pop("UEP_PACK_CTAS", None)


def main():
    args = parse_args()
    if args.size_sweep:
        run_size_sweep(args)
        return
    if args.pack_grid_sweep:
        run_pack_grid_sweep(args)
        return
    if args.impl == "reference":
        out = run_reference(args)
        if out is not None:
            print(json.dumps(out), flush=True)
        return
    result, rig, info = run_uep(args)
    world, rank = info[0], info[1]
    result["e2e"] = run_e2e(rig, info, max(4, min(args.steps, 16)))
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        result["cpu_baseline"] = cpu_baseline(rig.c)
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(result), flush=True)


if __name__ == "__main__":
    main()
