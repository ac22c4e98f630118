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
pack; `stages_us` breaks it down; `roofline` is the dominant kernel of the step (pack) and
`rooflines` lists every HBM-bound kernel of the path.  DESIGN.md §7 has the arithmetic.

`--gpus N` with no torchrun environment starts N ranks itself (re-executes under
`python -m torch.distributed.run`); it fails if fewer than N CUDA devices are visible.
`--workload all` prints one JSON line per configuration instead (the Table-3 mirror of
DESIGN.md §7: BASELINE configs, the 160-expert shape of the paper's Table 2, stress and size points).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
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
WORKLOADS = ["tiny", "glm_air", "dsv3_prefill", "dsv3_train"]


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=64)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="uep", choices=["uep", "reference"])
    ap.add_argument("--workload", default="dsv3_prefill", choices=WORKLOADS + ["all"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--state-scale", type=float, default=1.0,
                    help="shrink bytes per expert (debug only; the line then says so)")
    return ap.parse_args(argv)


# ------------------------------------------------------------------------------------------
# N ranks
# ------------------------------------------------------------------------------------------
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def ensure_ranks(args, argv):
    """`--gpus N` outside torchrun: start N ranks (one process per GPU) by re-executing this
    command under torch.distributed.run.  Never falls back to fewer ranks."""
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is not None:
        if int(world_env) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}")
        return
    if args.gpus == 1:
        return
    if args.impl == "uep":
        import torch
        n = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if n < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} requested but only {n} CUDA device(s) are "
                             "visible; refusing to run on fewer GPUs")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
           f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.abspath(__file__)] + list(argv)
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


def dist_setup(use_cuda: bool):
    """One process per GPU under torchrun (NCCL; gloo for the CPU reference arm); plain single
    process otherwise.  Returns (world, rank, local_rank)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if use_cuda:
            # keep the communicator's own log (rings/trees, NVLS) with the run, off stdout
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT,GRAPH")
            os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
            if torch.cuda.device_count() < world:
                raise SystemExit(f"bench.py: {world} ranks but {torch.cuda.device_count()} CUDA devices")
            torch.cuda.set_device(local)
        dist.init_process_group(backend="nccl" if use_cuda else "gloo", rank=rank, world_size=world)
    return world, rank, local


def measured_peaks():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written), else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json: torch copy_, burst)"
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


_DT = {"bf16": ("bfloat16", 2), "f32": ("float32", 4)}


def workload(name: str, state_scale: float = 1.0):
    from paper_2606_04101_b200 import synth
    c = dict(synth.CONFIGS[name])
    state = []
    for nm, elems, dt in c["state"]:
        elems = max(8, int(elems * state_scale) // 8 * 8)
        state.append((nm, elems, dt))
    c["state"] = state
    c["name"] = name
    return c


def n_instances(name: str, steps: int) -> int:
    return min(N_INSTANCES, max(steps, 1)) if name != "tiny" else min(8, max(steps, 1))


def config_of(args, c):
    """The `config` object: identical keys and values in both arms for the same arguments."""
    S = c["T"] * c["k"]
    gb = 2 if c["gate"] == "bf16" else 4
    n_inst = n_instances(args.workload, args.steps)
    return {"workload": args.workload, "T": c["T"], "k": c["k"], "E": c["E"], "R": c["R"],
            "n_slot": c["n_slot"], "u_min": c["u_min"], "beta": "101/100", "floor_mode": "tolerant",
            "gate": c["gate"],
            "state_bytes_per_expert": sum(e * _DT[dt][1] for _, e, dt in c["state"]),
            "zipf_s": c["zipf_s"], "instances": n_inst,
            "l2": "cold: rotates over %d distinct instances (%.0f MB of ids+gates) and each pack "
                  "streams GBs" % (n_inst, n_inst * S * (4 + gb) / 1e6),
            "parallelism": "instances sharded over ranks, no collective",
            "state_scale": args.state_scale}


def instance_inputs(c, idx: int, device):
    """ids/gates of instance idx (fresh permutation per instance; Zipf s per the config)."""
    from paper_2606_04101_b200 import synth
    seed = synth.instance_seed(BASE_SEED, idx // 4, idx % 4)
    s = c["zipf_s"] if c["zipf_s"] is not None else synth.train_sweep_s(BASE_SEED, idx // 4, idx % 4)
    if c.get("dist") == "one":
        ids = synth.one_expert_ids(c["T"], c["k"], c["E"] // 3, device=device)
    else:
        ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], s, seed, device=device)
    if c["gate"] == "bf16":
        gate = synth.gates_softmax_bf16(c["T"], c["k"], seed, device=device)
    else:
        gate = synth.gates_uniform_renorm(c["T"], c["k"], seed, device=device)
    return ids, gate, s


# ------------------------------------------------------------------------------------------
# uep arm
# ------------------------------------------------------------------------------------------
class Rig:
    """All device buffers of one rank: n_inst input sets, one output/plan set each (so that
    graph-captured chains over different instances do not alias), resident state."""

    def __init__(self, c, device, n_inst, inst_base=0, with_state=True):
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
        if with_state:
            for j, (nm, elems, dt) in enumerate(c["state"]):
                tdt = getattr(torch, _DT[dt][0])
                self.src.append(synth.expert_state(c["E"], elems, 7 + j, dtype=tdt, device=device))
                self.dst.append(torch.zeros((c["R"], max(c["n_slot"], 1), elems), dtype=tdt, device=device))
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


def barrier_and_max(world, value_ms):
    """max over ranks of a device-measured time (the contract's multi-GPU timing rule)."""
    if world == 1:
        return value_ms
    from paper_2606_04101_b200 import shard
    return shard.reduce_max_time(value_ms)


def csrc_digest():
    """sha256 over the CUDA sources: ties a committed ncu capture to the kernels it measured."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_04101_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def load_traffic(args):
    """DRAM bytes per launch from the committed `ncu --set full` capture (profiles/r02_traffic.json:
    one capture, one provenance).  A number printed under a profiler is never a bench value, so it
    is not re-taken here; it is DROPPED when the sources have changed since the capture."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.json")
    if args.workload != "dsv3_prefill" or args.state_scale != 1.0 or not os.path.exists(path):
        return {}, None
    try:
        d = json.load(open(path))
    except Exception:
        return {}, None
    src = {"file": "profiles/r02_traffic.json", "commit": d.get("commit"), "csrc_sha": d.get("csrc_sha")}
    if d.get("csrc_sha") != csrc_digest():
        src["stale"] = "csrc changed since the capture: traffic dropped"
        return {}, src
    return d.get("dram_bytes_per_launch", {}), src


def run_token_sharded(c, rig, world, rank, device, stream, reps):
    """ONE layer's tokens sharded over the `world` GPUs (the paper's deployment,
    PAPER.md:162): uep_shard_count -> all-gather of the R x E count rows -> uep_shard_finish
    (identical plan on every GPU, lookup of the local slots).  world == 1 is the whole problem on
    one GPU.  All ranks take their slice of the SAME seeded instances."""
    import torch
    import torch.distributed as dist
    from paper_2606_04101_b200 import binding, shard
    n = min(8, rig.n_inst)
    rounds = max(1, -(-32 // n))            # at least 32 steps per timed graph, as for the other stages
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
    use_graph, ms = True, None
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
    try:                                    # count -> exchange -> finish is one capturable sequence
        g = capture([lambda i=i: layers[i].step(ids_l[i], gate_l[i]) for _ in range(rounds) for i in range(n)], stream)
        ms, _ = time_graph(g, stream, reps)
        ms /= n * rounds
    except Exception:                       # a process group that cannot be captured: time as launched
        use_graph = False
        torch.cuda.synchronize(device)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(reps):
                for i in range(n):
                    layers[i].step(ids_l[i], gate_l[i])
            e1.record(stream)
        stream.synchronize()
        ms = e0.elapsed_time(e1) / (reps * n)
    ms = shard.reduce_max_time(ms)
    # every rank must hold the identical plan: compare a digest of (lambda, plan arrays) over ranks
    L0 = layers[0]
    dig = torch.stack([L0.expert_count.sum(dtype=torch.int64), L0.plan.inst_cum.sum(dtype=torch.int64),
                       L0.plan.inst_rank.sum(dtype=torch.int64), L0.plan.scalars[binding.SC_TAU].to(torch.int64)])
    same = True
    if dist.is_available() and dist.is_initialized():
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
            "note": "uep_shard_count -> all-gather of the R x E count rows (torch.distributed, in place in the "
                    "workspace) -> uep_shard_finish; one layer of T tokens split over the GPUs (strong scaling "
                    "of the plan latency), max over ranks; `value` is the weak-scaling instance-sharded number"}


def roof(name, nbytes, dur_us, peak_gbs, peak_src, traffic, what, parts=None):
    a = nbytes / (dur_us * 1e-6) / 1e9 if dur_us > 0 else 0.0
    parts = parts or [name]
    tr = sum(traffic[k] for k in parts) if all(k in traffic for k in parts) else None
    return {"kernel": name, "bound": "hbm", "achieved": round(a, 1), "peak": peak_gbs, "unit": "GB/s",
            "frac": round(a / peak_gbs, 4), "frac_of_nominal_8TBs": round(a / 8000.0, 4),
            "traffic": tr, "bytes_per_launch": int(nbytes), "us_per_launch": round(dur_us, 2),
            "peak_source": peak_src, "achieved_is": what}


ALGO = "algorithmic bytes per second (not DRAM traffic: at this size outputs partly stay in L2)"


def run_uep(args):
    import torch
    from paper_2606_04101_b200 import binding, shard
    world, rank, local = dist_setup(use_cuda=True)
    assert torch.cuda.is_available(), "bench.py (uep arm) needs a CUDA device; no CPU fallback"
    device = torch.device("cuda", local if world > 1 else torch.cuda.current_device())
    torch.cuda.set_device(device)
    c = workload(args.workload, args.state_scale)
    K, W = args.steps, max(args.warmup, 3)
    n_inst = n_instances(args.workload, K)
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
    launches0 = rig.ctx.uep_launch_count()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for i in sched:
            rig.balance(i)
        e1.record(stream)
    sync_all()
    gpu_launches = rig.ctx.uep_launch_count() - launches0      # counted by the library, per launch
    step_ms = barrier_and_max(world, e0.elapsed_time(e1))

    # ---- stage timing: graph-captured chains over all instances (L2-cold by rotation) --------
    reps = 5
    # Every timed graph holds at least 32 calls (the instances in order, as many rounds as that takes),
    # so that the gap between two graph launches — harness, not layer — weighs the same whatever
    # --steps is (with 20 instances in a graph of 20 calls it added 0.5 us per call to the chain).
    g_rounds = max(1, -(-32 // n_inst))
    order = [i for _ in range(g_rounds) for i in range(n_inst)]

    def timed(fn):
        ms, mn = time_graph(capture([lambda i=i: fn(i) for i in order], stream), stream, reps)
        return ms / g_rounds, mn / g_rounds       # per round over the n_inst instances

    # the chain is uep_balance without state tensors: histogram -> plan -> lookup on the stream,
    # the rank half of the remap forked beside histogram + plan (as the library schedules it)
    chain_ms, chain_min = timed(lambda i: rig.balance(i, with_pack=False))
    hist_ms, _ = timed(rig.hist)
    plan_ms, _ = timed(rig.plan)
    remap_ms, _ = timed(rig.remap)
    rank_ms, _ = timed(rig.rank)
    lookup_ms, _ = timed(rig.lookup)
    n_pack = min(n_inst, 8)
    g_pack = capture([lambda i=i: rig.pack(i) for i in range(n_pack)], stream)
    pack_ms, _ = time_graph(g_pack, stream, 3, warm=1)
    # NEXT-4: all instances' planners in ONE launch, one cluster per instance
    counts_all = torch.stack(rig.counts).contiguous()
    bplan = rig.ctx.new_plan(batch=n_inst)
    torch.cuda.synchronize(device)
    g_bplan = capture([lambda: rig.ctx.uep_plan_batched(n_inst, counts_all, bplan)], stream)
    bplan_ms, _ = time_graph(g_bplan, stream, reps)
    # NEXT-2: backward gradient reduction (fp32, one [7168 x 2048]-like matrix per
    # expert for the DSV3 shapes) and the inverse remap, on the plans of this run
    g_elems = 7168 * 2048 if c["E"] >= 256 else (4096 * 1408 if c["E"] >= 128 else 256 * 512)
    g_elems = max(8, int(g_elems * args.state_scale) // 8 * 8)
    main_grad = torch.ones((c["E"], g_elems), dtype=torch.float32, device=device)
    slot_grad = torch.ones((c["R"], max(c["n_slot"], 1), g_elems), dtype=torch.float32, device=device)
    out_src = torch.empty(c["T"] * c["k"], dtype=torch.int32, device=device)
    n_red = min(n_inst, 4)
    torch.cuda.synchronize(device)
    g_red = capture([lambda i=i: rig.ctx.uep_grad_reduce(rig.plans[i], [main_grad], [slot_grad])
                     for i in range(n_red)], stream)
    red_ms, _ = time_graph(g_red, stream, 3, warm=1)
    g_inv = capture([lambda i=i: rig.ctx.uep_remap_inverse(rig.outs[i][1], rig.outs[i][2], rig.plans[i], out_src)
                     for i in range(n_inst)], stream)
    inv_ms, _ = time_graph(g_inv, stream, reps)
    del main_grad, slot_grad
    # NEXT-1: source-aware reroute; in-flight token ratio against the global remap
    local_res = None
    if c["T"] % c["R"] == 0:
        local_res = source_aware(rig, stream, reps)
    tok = None
    if c["T"] % c["R"] == 0 and c["R"] % world == 0 and (c["T"] * c["k"]) % world == 0:
        try:
            tok = run_token_sharded(c, rig, world, rank, device, stream, reps)
        except Exception as ex:              # an extra key must never take the bench line down
            tok = {"error": repr(ex)[:300]}
    clocks = sampler.stop()
    chain_ms = barrier_and_max(world, chain_ms)
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
    traffic, traffic_src = load_traffic(args)
    rf = lambda name, nb, t, what, parts=None: roof(name, nb, t, peak_gbs, peak_src, traffic, what, parts)

    pack_us = us(pack_ms, n_pack)
    r_pack = rf("pack_kernel", sum(bytes_pack) / max(n_pack, 1), pack_us,
                "algorithmic bytes per second; the peak is a torch copy_ measurement, so a streaming kernel can "
                "read slightly above 1.0 (also given against the nominal 8 TB/s)")
    rooflines = [r_pack,
                 rf("uep_remap (rank_kernel+prefix_kernel+lookup_kernel)", bytes_remap, us(remap_ms, n_inst), ALGO,
                    ["rank_kernel", "prefix_kernel", "lookup_kernel"]),
                 rf("lookup_kernel", bytes_remap, us(lookup_ms, n_inst), ALGO),
                 rf("rank_kernel+prefix_kernel", 8 * S, us(rank_ms, n_inst), ALGO, ["rank_kernel", "prefix_kernel"]),
                 rf("hist_kernel", bytes_hist, us(hist_ms, n_inst), ALGO)]
    red_bytes = statistics.mean(2 * (n_grp[i] + n_rep[i]) for i in range(n_red)) * g_elems * 4
    result = {
        "metric": METRIC, "value": round(plan_latency_us, 3), "unit": UNIT, "n_gpus": world,
        "steps": K, "warmup": W, "ms_per_step": round(step_ms / K, 4), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": config_of(args, c),
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
        "calls_per_timed_graph": n_inst * g_rounds,
        "batched_plan": {"instances": n_inst, "us_total": round(bplan_ms * 1e3, 2),
                         "us_per_layer": round(bplan_ms * 1e3 / n_inst, 3),
                         "note": "uep_plan_batched: one launch, one 8-CTA cluster per instance"},
        "backward": {"grad_reduce_us": round(red_ms * 1e3 / n_red, 2), "grad_reduce_bytes": int(red_bytes),
                     "grad_reduce_frac_of_peak": round(red_bytes / (red_ms * 1e-3 / n_red) / 1e9 / peak_gbs, 4),
                     "grad_reduce_traffic": traffic.get("grad_reduce_kernel"),
                     "inverse_remap_us": round(inv_ms * 1e3 / n_inst, 2),
                     "note": "uep_grad_reduce: fp32 [E, %d] main + [R, n_slot, %d] slot grads, bytes = 2 x (groups + replicas) x B; "
                             "uep_remap_inverse: 8 B/slot read, 4 B/slot scattered write" % (g_elems, g_elems)},
        "source_aware_remap": local_res,
        "token_sharded": tok,
        "roofline": {k: r_pack[k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic")},
        "roofline_note": "`roofline` is the dominant kernel of the STEP (pack: %.0f of %.0f us); `value` is the "
                         "planning chain WITHOUT the pack — its own kernels (hist, rank+prefix, lookup) are in "
                         "`rooflines`, and the planner is latency-bound (no byte roofline)" % (pack_us, step_ms * 1e3 / K),
        "traffic_source": traffic_src,
        "rooflines": rooflines,
        "gpu_launches": int(gpu_launches),
        "gpu_launches_note": "kernels launched by libuep inside the timed region of K steps, counted by the library "
                             "at every launch (uep_launch_count)",
        "clocks": clocks,
        "launch_info": rig.ctx.launch_info,
    }
    return result, rig, (world, rank, device, stream)


def source_aware(rig, stream, reps):
    """uep_remap_local against the global remap: time and in-flight token ratio."""
    import torch
    c, n_inst, device = rig.c, rig.n_inst, rig.device
    infl = [torch.zeros(c["R"], dtype=torch.int32, device=device) for _ in range(n_inst)]
    src_rank = (torch.arange(c["T"], device=device, dtype=torch.int64) * c["R"] // c["T"]).to(torch.int32)
    with torch.cuda.stream(stream):          # the global remap's outputs for the comparison
        for i in range(min(n_inst, 4)):
            rig.remap(i)
    stream.synchronize()
    glob_fly = [int(((rig.outs[i][1] != src_rank[:, None]) & (rig.outs[i][1] >= 0)).sum()) for i in range(min(n_inst, 4))]
    g_loc = capture([lambda i=i: rig.ctx.uep_remap_local(rig.ids[i], rig.gates[i], rig.plans[i], rig.outs[i][0],
                                                        rig.outs[i][1], rig.outs[i][2], rig.outs[i][3],
                                                        infl[i], rig.ws[i]) for i in range(n_inst)], stream)
    loc_ms, _ = time_graph(g_loc, stream, reps)
    loc_fly = [int(infl[i].sum()) for i in range(min(n_inst, 4))]
    S_all = c["T"] * c["k"]
    with torch.cuda.stream(stream):          # leave the global remap's outputs in place again
        for i in range(n_inst):
            rig.remap(i)
    stream.synchronize()
    return {"remap_local_us": round(loc_ms * 1e3 / n_inst, 2),
            "inflight_ratio_global": round(statistics.mean(glob_fly) / S_all, 4),
            "inflight_ratio_local": round(statistics.mean(loc_fly) / S_all, 4),
            "note": "uep_remap_local = rank + prefix + reroute + lookup on one stream; in-flight = slots whose "
                    "destination rank differs from their source rank floor(i*R/T) (paper: 96.0 % vs 98.4 %, "
                    "PAPER.md:440, its own traces)"}


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
    res.update({"unit": UNIT,
                "h2d_bytes_per_step": S * (4 + gb), "d2h_bytes_per_step": S * (12 + gb) + 64,
                "steps": steps,
                "note": "wall clock around uep_balance_host: pinned ids+gates H2D, histogram+plan+remap, remap "
                        "outputs+scalars D2H, sync (PCIe-bound); whole_step_value = the same call with the state "
                        "tensors, i.e. incl. the pack, whose time the D2H copies overlap"})
    return res


# ------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline, --impl reference): the only places that execute oracle/
# ------------------------------------------------------------------------------------------
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


def cpu_model():
    try:
        return [l.split(":")[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")][0]
    except Exception:
        return "unknown"


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
    return {"value": round(st["histogram"] + st["plan"] + st["remap"], 1), "unit": UNIT, "cores": 1,
            "kind": "oracle", "host_cores": os.cpu_count(), "cpu_model": cpu_model(),
            "stages_us": st,
            "sample": "%d instances of the workload x %d passes of histogram+plan+remap (single thread, g++ -O2); "
                      "pack timed on 4 instances over 1/%d of each expert's bytes and scaled x%d"
                      % (n_samples, reps, pack_frac, pack_frac)}


def run_reference(args):
    """--impl reference: the oracle as it stands, timed on the host cores.  Under N ranks rank 0
    alone runs and prints; the others exit 0 without work (after the rendezvous, on gloo)."""
    world, rank, _ = dist_setup(use_cuda=False)
    ranks_started = world
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.ones(1, dtype=torch.int64)
        dist.all_reduce(t)                       # every rank showed up
        ranks_started = int(t.item())
        dist.barrier()
        dist.destroy_process_group()
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
            "n_gpus": world, "ranks_started": ranks_started, "steps": K, "warmup": W,
            "ms_per_step": round(dt * 1e3 / max(K, 1), 4), "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": config_of(args, c),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "host_cores": os.cpu_count(), "cpu_model": cpu_model(), "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# ------------------------------------------------------------------------------------------
# --workload all: one line per configuration (the Table-3 mirror)
# ------------------------------------------------------------------------------------------
def table_configs():
    from paper_2606_04101_b200 import synth
    base = {n: dict(synth.CONFIGS[n]) for n in WORKLOADS}
    rows = [("tiny", dict(base["tiny"]), 8)]
    for s in (0.6, 1.0, 1.4):
        rows.append((f"glm_air s={s}", dict(base["glm_air"], zipf_s=s), 8))
    rows.append(("dsv3_prefill", dict(base["dsv3_prefill"]), 8))
    rows.append(("dsv3_train (8 of 232 instances: layers 0-1 x 4 microbatches; bf16 W + fp32 grad, m, v = "
                 "205.5 MB/expert)", dict(base["dsv3_train"]), 8))
    rows.append(("table2_160 (PAPER.md:372: 160 experts top-8, EP40, N_slot=4; 40 x 4096 tokens; the paper gives "
                 "no expert dimensions for this model: expert state as glm_air)",
                 dict(T=40 * 4096, k=8, E=160, R=40, n_slot=4, u_min=1024, zipf_s=1.0, gate="bf16",
                      state=list(base["glm_air"]["state"])), 8))
    st = [("w", 2048 * 1024, "bf16")]
    def stress(S, k, E, R, ns, dist, s):
        return dict(T=S // k, k=k, E=E, R=R, n_slot=ns, u_min=synth.stress_u_min(S, R), zipf_s=s,
                    gate="f32", state=st, dist=dist)
    rows += [("stress 1Ki slots E=64 R=8 uniform", stress(1024, 1, 64, 8, 1, "zipf", 0.0), 4),
             ("stress 256Ki slots E=64 R=256 N_slot=3 Zipf 2.0", stress(262144, 8, 64, 256, 3, "zipf", 2.0), 4),
             ("stress 1Mi slots E=512 R=64 uniform", stress(1 << 20, 8, 512, 64, 2, "zipf", 0.0), 4),
             ("stress 4Mi slots E=256 R=64 N_slot=4 Zipf 2.0", stress(1 << 22, 8, 256, 64, 4, "zipf", 2.0), 4),
             ("stress 4Mi slots E=512 R=256 N_slot=4 Zipf 2.0", stress(1 << 22, 4, 512, 256, 4, "zipf", 2.0), 4),
             ("stress 4Mi slots E=512 R=256 N_slot=4 all-to-one", stress(1 << 22, 8, 512, 256, 4, "one", 0.0), 4),
             ("stress 4Mi slots E=64 R=8 k=1 uniform", stress(1 << 22, 1, 64, 8, 1, "zipf", 0.0), 4)]
    # size points of the DeepSeek-V3 shape (marginal rates of the slot-streaming kernels)
    for T in (1 << 19, 1 << 20, (1 << 21) - 64):
        rows.append((f"size E=256 k=8 R=64 S={T * 8}", stress(T * 8, 8, 256, 64, 2, "zipf", 1.0), 4))
    return rows


def run_table(args):
    import torch
    from paper_2606_04101_b200 import binding
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; no CPU fallback"
    device = torch.device("cuda", torch.cuda.current_device())
    peak_gbs, peak_src = measured_peaks()
    for name, c, n_inst in table_configs():
        c = dict(c)
        c["state"] = [(nm, max(8, int(e * args.state_scale) // 8 * 8), dt) for nm, e, dt in c["state"]]
        rig = Rig(c, device, n_inst)
        stream = torch.cuda.Stream(device)
        with torch.cuda.stream(stream):
            for i in range(n_inst):
                rig.balance(i, with_pack=False)
        stream.synchronize()
        stages = {"chain": lambda i: rig.balance(i, with_pack=False), "histogram": rig.hist, "plan": rig.plan,
                  "remap": rig.remap, "remap_rank": rig.rank, "remap_lookup": rig.lookup}
        us = {}
        for nm, fn in stages.items():
            g = capture([lambda i=i, fn=fn: fn(i) for i in range(n_inst)], stream)
            ms, _ = time_graph(g, stream, 5)
            us[nm] = ms * 1e3 / n_inst
        S = c["T"] * c["k"]
        sc = [rig.plans[i].scalars.cpu().numpy() for i in range(n_inst)]
        n_rep = [int(s[binding.SC_N_REPLICAS]) for s in sc]
        n_grp = [int(s[binding.SC_N_GROUPS]) for s in sc]
        pack_us, pack_frac = None, None
        if c["n_slot"] > 0 and sum(n_rep) > 0:
            n_pack = min(n_inst, 4)
            g = capture([lambda i=i: rig.pack(i) for i in range(n_pack)], stream)
            ms, _ = time_graph(g, stream, 3, warm=1)
            pack_us = ms * 1e3 / n_pack
            nb = statistics.mean((n_grp[i] + n_rep[i]) for i in range(n_pack)) * rig.state_bytes_per_expert
            pack_frac = nb / (pack_us * 1e-6) / 1e9 / peak_gbs
        gb = 2 if c["gate"] == "bf16" else 4
        frac = lambda nbytes, t: round(nbytes / (t * 1e-6) / 1e9 / peak_gbs, 3) if t > 0 else None
        mean_load = S / c["R"]
        # relay trees (NEXT-3): the busiest sender's fan-out with direct sends and with relays
        parent = torch.empty(c["E"] + c["R"] * c["n_slot"], dtype=torch.int32, device=device)
        vol = torch.empty(max(c["R"], 4), dtype=torch.int32, device=device)
        direct, relayed = [], []
        for i in range(n_inst):
            hp = rig.plans[i].host()
            fan = (hp.inst_off[1:] - hp.inst_off[:-1] - 1)
            home = hp.inst_rank[hp.inst_off[:-1]]
            d = torch.zeros(c["R"], dtype=torch.int64).index_add_(0, torch.from_numpy(home).long(),
                                                                  torch.from_numpy(fan).long())
            direct.append(int(d.max()))
            rig.ctx.uep_relay_plan(rig.plans[i], parent, vol)
            torch.cuda.synchronize(device)
            relayed.append(int(vol[:c["R"]].max()))
        loc = source_aware(rig, stream, 3) if (c["T"] % c["R"] == 0 and c["T"] > 0) else None
        row = {"table3_row": name, "T": c["T"], "k": c["k"], "E": c["E"], "R": c["R"], "n_slot": c["n_slot"],
               "slots": S, "u_min": c["u_min"], "zipf_s": c["zipf_s"], "dist": c.get("dist", "zipf"),
               "gate": c["gate"], "instances": n_inst, "state_bytes_per_expert": rig.state_bytes_per_expert,
               "chain_us": round(us["chain"], 2),
               "stages_us": {k_: round(v, 2) for k_, v in us.items() if k_ != "chain"},
               "pack_us": None if pack_us is None else round(pack_us, 1),
               "frac_of_peak": {"hist_kernel (4 B/slot)": frac(4 * S, us["histogram"]),
                                "uep_remap (%d B/slot)" % (16 + 2 * gb): frac((16 + 2 * gb) * S, us["remap"]),
                                "rank+prefix (8 B/slot)": frac(8 * S, us["remap_rank"]),
                                "lookup_kernel": frac((16 + 2 * gb) * S, us["remap_lookup"]),
                                "pack_kernel": None if pack_frac is None else round(pack_frac, 3)},
               "imbalance_before": round(statistics.mean(float(s[binding.SC_TAU_HI0]) for s in sc) / mean_load, 3),
               "imbalance_after": round(statistics.mean(float(s[binding.SC_MAX_LOAD]) for s in sc) / mean_load, 4),
               "slots_used": round(statistics.mean(n_rep), 1), "slots_available": c["R"] * c["n_slot"],
               "max_fanout": round(statistics.mean(int(s[binding.SC_MAX_FANOUT]) for s in sc), 1),
               "n_probes": round(statistics.mean(int(s[binding.SC_N_PROBES]) for s in sc), 1),
               "solving_time_us": round(us["plan"], 2),
               "inflight_ratio": None if loc is None else {"without_locality": loc["inflight_ratio_global"],
                                                           "with_locality": loc["inflight_ratio_local"],
                                                           "remap_local_us": loc["remap_local_us"]},
               "max_send_fanout": {"direct": round(statistics.mean(direct), 1),
                                   "with_relay_trees": round(statistics.mean(relayed), 1)},
               "peak_gbs": peak_gbs, "peak_source": peak_src}
        print(json.dumps(row), flush=True)
        del rig, parent, vol
        torch.cuda.synchronize(device)
        torch.cuda.empty_cache()


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    args = parse_args(argv)
    ensure_ranks(args, argv)
    if args.impl == "reference":
        if args.workload == "all":
            raise SystemExit("bench.py: --workload all has no reference arm")
        out = run_reference(args)
        if out is not None:
            print(json.dumps(out), flush=True)
        return
    if args.workload == "all":
        run_table(args)
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
