#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole cloaked-layout hot path over one LLaMA-8B-shaped decoder
layer (BASELINE.json configs[1]): S1 keygen -> S3 arena plan -> S5 neuron/head permutation -> S4 block
shuffle into the 2 MiB page pool (the 7 tensors in one cloak_shuffle_many call) -> S8 re-layout key A -> key B ->
S6 cloaked GEMV of the 7 projections at batch 1, 4, 16 (one cloak_gemv_chain call per batch) -> S4 unshuffle.
(S2, the VMM mapper, is load-time setup: timed separately, `pool_map_ms`.)

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cloak|reference]

Prints ONE JSON line (rank 0).  `value` = algorithmic GB moved by the step / step time, whole job (N replicas:
the path does not shard -- SURVEY.md 8(e) "replicas only" -- so N GPUs run N independent copies, weak scaling).
Per-stage GB/s, fractions of the measured HBM peak and the cloaked-vs-native GEMV overhead ride along.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import importlib
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

METRIC = "shuffle GB/s and cloaked decode GEMV GB/s (frac of HBM peak); cloaked-vs-native overhead %"
BATCHES = (1, 4, 16)
KEY_A, KEY_B = 0x1234, 0x5678          # G11
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of one gemv_chain_kernel launch (the 7 projections at one
# batch; algorithmic bytes are 436 207 616), read from the kept summary of the `ncu --set full` capture of this command.
NCU_TRAFFIC_FILE = "profiles/r2_ncu_gemv_chain_traffic.json"
FALLBACK_HBM_GBS = 6650.0              # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


def ncu_traffic():
    """(bytes per launch, source) from the committed ncu summary, or (None, why)."""
    try:
        with open(os.path.join(ROOT, NCU_TRAFFIC_FILE)) as f:
            d = json.load(f)
        return float(d["dram_bytes_per_launch_mean"]), NCU_TRAFFIC_FILE
    except Exception as e:          # noqa: BLE001
        return None, f"{NCU_TRAFFIC_FILE} unreadable: {type(e).__name__}"


def layer_tensors():
    from synth import gen
    c = gen.CONFIGS[1]
    shapes = gen.layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"])
    return c, shapes


def step_bytes(shapes, names=None):
    """Algorithmic bytes one step moves: 2 B/B for permute, shuffle, relayout, unshuffle;
    weight bytes once per GEMV batch."""
    B = sum(2 * n * k for nm, (n, k) in shapes if names is None or nm in names)
    return dict(B=B, permute=2 * B, shuffle=2 * B, relayout=2 * B, unshuffle=2 * B, gemv=len(BATCHES) * B,
                total=(8 + len(BATCHES)) * B)


# ------------------------------------------------------------------------------------------ clocks
ClockSampler = importlib.import_module("paper_2606_18400_b200.clocks").ClockSampler   # (loads no CUDA library)


# ------------------------------------------------------------------------------------------ CPU oracle arm
ORACLE_ATTN = ("q", "k", "v", "o")                               # the attention projections: 84 MB of the 436 MB
ORACLE_LAYER = ("q", "k", "v", "o", "gate", "up", "down")        # the whole cfg1 layer


def oracle_setup(names=ORACLE_LAYER):
    """Inputs of the oracle arm (not timed).  They come from the shared generator: its CUDA twin when a GPU is there (the
    numpy twin makes ~10 M elements/s, the layer has 218 M; tests/ check that the twins agree byte for byte), else numpy."""
    from synth import gen
    c, shapes = layer_tensors()
    fill = None
    try:
        import torch
        if torch.cuda.is_available():
            from synth import cuda as synth_cuda

            def fill(seed, tid, shp, kind=gen.KIND_WEIGHT):
                t = synth_cuda.fill(torch.empty(shp, dtype=torch.bfloat16, device="cuda"), seed, tid, kind=kind)
                return t.view(torch.int16).cpu().numpy().view(np.uint16)
    except ImportError:
        pass
    if fill is None:
        def fill(seed, tid, shp, kind=gen.KIND_WEIGHT):
            return gen.synth(seed, tid, shp, "bf16", kind=kind)
    W = {nm: fill(c["seed"], i, shp) for i, (nm, shp) in enumerate(shapes) if nm in names}
    X = {b: {k: fill(c["seed"] + 100, b * 2 + (k != c["hidden"]), (b, k), gen.KIND_NORMAL) for k in (c["hidden"], c["inter"])}
         for b in BATCHES}
    return c, shapes, W, X


def oracle_step(c, shapes, W, X, names=ORACLE_LAYER):
    """The same stages as the GPU step over the tensors in `names`, run by oracle/ as it stands (never tuned for this)."""
    import oracle as O
    block, page = c["block"], c["page"]
    sizes = [2 * n * k for nm, (n, k) in shapes]
    offs, total, _ = O.arena_plan(KEY_A, sizes, block)                              # S3 (+ S1 for the order)
    g = O.pool_geometry(total, block, page)
    ta, tb = O.pool_tables(KEY_A, g), O.pool_tables(KEY_B, g)                       # S1
    kappa, eta = O.head_maps(KEY_A, 0, c["n_q"], c["n_kv"])
    q2, k2, v2, o2 = O.permute_heads(W["q"], W["k"], W["v"], W["o"], kappa, eta, c["head_dim"])   # S5
    P = dict(q=q2, k=k2, v=v2, o=o2)
    if "gate" in names:
        pi = O.mlp_perm(KEY_A, 0, c["inter"])
        P["gate"], P["up"], P["down"] = O.permute_mlp(W["gate"], W["up"], W["down"], pi)
    off = {nm: o for (nm, _), o in zip(shapes, offs)}
    pool_a = np.zeros(g.nslots * block, np.uint8)
    for nm in names:                                                                # S4
        O.shuffle_into(pool_a, ta.T_vmm, P[nm].view(np.uint8).ravel(), off[nm], block)
    pool_b = np.zeros(g.nslots * block, np.uint8)                                   # S8 (the blocks of `names`)
    for nm in names:
        L = O.unshuffle(pool_a, ta.T_vmm, total, block, off[nm], P[nm].size * 2)
        O.shuffle_into(pool_b, tb.T_vmm, L, off[nm], block)
    ys = []
    for b in BATCHES:                                                               # S6
        for nm in names:
            ys.append(O.linear_f64(X[b][P[nm].shape[1]], P[nm]))
    for nm in names:                                                                # S4 unshuffle
        O.unshuffle(pool_a, ta.T_vmm, total, block, off[nm], P[nm].size * 2)
    return ys


def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
        return int(n)
    except Exception:
        return os.cpu_count() or 1


def oracle_time(names, reps_max, budget_s, threads=None):
    """Seconds per oracle step over `names`, at most reps_max repetitions / budget_s seconds; threads=1 limits numpy's BLAS
    to one thread (the rest of the oracle is single-threaded Python + numpy anyway)."""
    import contextlib
    c, shapes, W, X = oracle_setup(names)
    ctx = contextlib.nullcontext()
    if threads is not None:
        from threadpoolctl import threadpool_limits
        ctx = threadpool_limits(limits=threads)
    with ctx:
        used = oracle_threads() if threads is None else threads
        t0 = time.perf_counter()
        reps = 0
        while reps < 1 or (time.perf_counter() - t0 < budget_s and reps < reps_max):
            oracle_step(c, shapes, W, X, names)
            reps += 1
        dt = (time.perf_counter() - t0) / reps
    return dt, reps, used, step_bytes(shapes, names)


def oracle_cfg3_layer(batch=32):
    """SURVEY.md 8(d) "oracle beside it", cfg3: the fp64 contraction of ONE Qwen-32B-shaped layer's 7 projections at batch 32 on
    the host cores (numpy BLAS, all threads), multiplied by 64 and stated as extrapolated.  The 62 GB model is never on the host."""
    import oracle as O
    from synth import gen
    c = gen.CONFIGS[3]
    shapes = gen.layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"])
    import torch
    from synth import cuda as synth_cuda
    t_total, nbytes = 0.0, 0
    for i, (nm, (n, k)) in enumerate(shapes):               # tensor by tensor: a layer in fp64 would be 3.9 GB
        W = synth_cuda.fill(torch.empty(n, k, dtype=torch.bfloat16, device="cuda"), c["seed"], i).view(torch.int16).cpu().numpy().view(np.uint16)
        X = synth_cuda.fill(torch.empty(batch, k, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, i,
                            kind=gen.KIND_NORMAL).view(torch.int16).cpu().numpy().view(np.uint16)
        t0 = time.perf_counter()
        O.linear_f64(X, W)
        t_total += time.perf_counter() - t0
        nbytes += 2 * n * k
    return {"kind": "oracle", "what": f"linear_f64 of one layer's 7 projections at batch {batch} (bf16 -> fp64 conversion included)",
            "cores": oracle_threads(), "one_layer_ms": t_total * 1e3, "one_layer_gbs": nbytes / t_total / 1e9,
            "oracle_extrapolated": True, "t_ms_64_layers_extrapolated": t_total * 1e3 * c["layers"]}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    # each step is a bounded sample of the cfg1 workload: the whole layer when the run is short enough for that to end
    # within a few minutes (~4 s per step on 16 cores), the attention projections (19 % of the bytes) otherwise
    names = ORACLE_LAYER if args.steps + args.warmup <= 30 else ORACLE_ATTN
    c, shapes, W, X = oracle_setup(names)
    sb = step_bytes(shapes, names)
    for _ in range(args.warmup):
        oracle_step(c, shapes, W, X, names)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(c, shapes, W, X, names)
    dt = time.perf_counter() - t0
    val = sb["total"] * args.steps / dt / 1e9
    sample = (f"cfg1 {'whole layer' if names == ORACLE_LAYER else 'attention projections ' + '/'.join(names)} "
              f"({sb['B']/1e6:.1f} MB of 436.2 MB), all stages")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": "cfg1: one LLaMA-8B-shaped decoder layer (oracle on the host cores)", "sample": sample},
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": oracle_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "note": "the numpy oracle as it stands, a deliberately plain program: a ratio against it is not a headline"}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ replicas (N > 1)
def sm_weights_summary(C):
    """The per-SM streaming weights the library measured on this device (calibrate.cu), summarised."""
    w = np.array(C.cloak_sm_weights(0))
    if w.size == 0:
        return {"measured": False}
    return {"measured": True, "n_sm": int(w.size), "min": float(w.min()), "max": float(w.max()),
            "tiers": {f"{v:.3f}": int(c) for v, c in zip(*np.unique(np.round(w * 8) / 8, return_counts=True))}}


def max_over_ranks(ms, dist, device):
    """The path does not shard (replicas only): every rank times its own replica of the step and the
    job's time is the slowest rank's.  One scalar all_reduce(MAX); `dist` is None on a single rank."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gbs(bytes_per_replica_step, ms_per_step, world):
    """`value`: bytes all replicas moved per step / the slowest replica's step time (weak scaling)."""
    return world * bytes_per_replica_step / ms_per_step / 1e6


# ------------------------------------------------------------------------------------------ GPU arm
def run_cloak(args):
    import torch
    import paper_2606_18400_b200 as C          # raises if libcloak.so is missing: no fallback
    from synth import cuda as synth_cuda
    from synth import gen

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the cloak path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    c, shapes = layer_tensors()
    block, page, seed = c["block"], c["page"], c["seed"]
    sb = step_bytes(shapes)
    sizes = [2 * n * k for _, (n, k) in shapes]
    stream = torch.cuda.current_stream()

    # ---- setup (not timed): raw logical weights, pools, activations
    raw = {nm: synth_cuda.fill(torch.empty(shp, dtype=torch.bfloat16, device="cuda"), seed, i)
           for i, (nm, shp) in enumerate(shapes)}
    perm = {nm: torch.empty_like(t) for nm, t in raw.items()}
    back = {nm: torch.empty_like(t) for nm, t in raw.items()}
    offs, total = C.cloak_arena_plan(KEY_A, sizes, block)
    t0 = time.perf_counter()
    pool_a = C.cloak_pool_create(local, total, block, page, KEY_A)
    pool_create_s = time.perf_counter() - t0
    pool_b = C.cloak_pool_create(local, total, block, page, KEY_B)
    pool_n = C.cloak_pool_create(local, total, block, page, KEY_A, C.CLOAK_POOL_IDENTITY)   # the "native" layout
    # the same identity layout in ONE plain allocation: exposes any cost of the 2 MiB-fragmented VMM mapping
    pool_p = C.cloak_pool_create(local, total, block, page, KEY_A, C.CLOAK_POOL_IDENTITY | C.CLOAK_POOL_PLAIN_ALLOC)
    info = C.cloak_pool_info(pool_a)
    scratch = torch.empty(2 * info["nslots"] + 2 * info["npages"], dtype=torch.int32, device="cuda")
    X = {b: {k: synth_cuda.fill(torch.empty(b, k, dtype=torch.bfloat16, device="cuda"), seed + 100, b * 2 + (k != c["hidden"]),
                                kind=gen.KIND_NORMAL) for k in (c["hidden"], c["inter"])} for b in BATCHES}
    Y = {b: {nm: torch.empty(b, shp[0], dtype=torch.bfloat16, device="cuda") for nm, shp in shapes} for b in BATCHES}
    sh = C.cloak_block_shape(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, 0)
    tens = {nm: C.cloak_tensor(o, shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for (nm, shp), o in zip(shapes, offs)}
    STAGES = ["keygen", "permute", "shuffle", "relayout"] + [f"gemv_b{b}" for b in BATCHES] + ["unshuffle"]

    # S6: the layer's 7 projections at one batch = ONE cloak_gemv_chain launch (the inputs are fixed synthetic
    # vectors, so no op depends on another); `per_call` issues the same 7 GEMVs as 7 cloak_gemv calls.
    chain_ops = {b: C.cloak_gemv_ops([(tens[nm], X[b][k], Y[b][nm], 0) for nm, (n, k) in shapes]) for b in BATCHES}

    def gemv_chain(pool, b, per_call=False):
        if per_call:
            for nm, (n, k) in shapes:
                C.cloak_gemv(pool, tens[nm], X[b][k], Y[b][nm], b)
        else:
            C.cloak_gemv_chain(pool, chain_ops[b], b)

    # The stages of one step.  Every call is asynchronous on torch's current stream (stream=None in the binding), so
    # the same functions serve plain stream launches and CUDA-graph capture.
    ns, npg = info["nslots"], info["npages"]

    def st_keygen():                                                                                       # S1
        C.cloak_keygen(KEY_A, 1 << 32, ns, scratch[:ns], scratch[ns:2 * ns])
        C.cloak_keygen(KEY_A, 2 << 32, npg, scratch[2 * ns:2 * ns + npg], scratch[2 * ns + npg:])

    def st_permute():                                                                                      # S5
        C.cloak_permute_mlp_heads(KEY_A, sh, **raw, **{k + "_o": v for k, v in perm.items()})

    lay_t = [perm[nm] for nm, _ in shapes]
    lay_back = [back[nm] for nm, _ in shapes]
    lay_b = [perm[nm].numel() * 2 for nm, _ in shapes]

    def st_shuffle():                                                                                      # S4, the layer's 7 tensors in one call
        C.cloak_shuffle_many(pool_a, lay_t, offs, lay_b)

    def st_relayout():                                                                                     # S8
        C.cloak_relayout(pool_a, pool_b)

    def st_unshuffle():                                                                                    # S4^-1
        C.cloak_unshuffle_many(pool_a, lay_back, offs, lay_b)

    stage_fns = ([st_keygen, st_permute, st_shuffle, st_relayout]
                 + [(lambda b=b: gemv_chain(pool_a, b)) for b in BATCHES] + [st_unshuffle])

    def capture(fn):
        """One CUDA graph of the kernels fn() launches through the C ABI; returns (replay, kernels in the graph)."""
        if args.launch == "stream":
            n0 = C.cloak_launch_count()
            fn()
            return fn, C.cloak_launch_count() - n0
        g = torch.cuda.CUDAGraph()
        n0 = C.cloak_launch_count()
        with torch.cuda.graph(g):
            fn()
        return g.replay, C.cloak_launch_count() - n0

    # first pass on the stream (allocates the library's scratch, loads kernels), then one graph per stage
    for fn in stage_fns:
        fn()
    torch.cuda.synchronize()
    staged = [capture(fn) for fn in stage_fns]
    launches_per_step = sum(n for _, n in staged)

    def step(ev=None):
        def mark(i):
            if ev is not None:
                ev[i].record(stream)
        mark(0)
        C.cloak_arena_plan(KEY_A, sizes, block)                                                            # S3 (host)
        for i, (replay, _) in enumerate(staged):
            replay()
            mark(i + 1)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # The clock sampler starts here, ahead of the warm-up: nvidia-smi's start-up (NVML initialisation) contends
    # with kernel launches for the driver, so it must be over before the timed region begins.
    clocks = ClockSampler(local) if rank == 0 else None
    if clocks is not None:
        clocks.wait_first_sample()

    # ---- native layout gets the same permuted weights once (needs one permute first)
    step()
    for (nm, _), o in zip(shapes, offs):
        C.cloak_shuffle(pool_n, perm[nm], o, perm[nm].numel() * 2, stream)
        C.cloak_shuffle(pool_p, perm[nm], o, perm[nm].numel() * 2, stream)
    for _ in range(max(args.warmup - 1, 0)):
        step()
    barrier()

    # ---- timed region: exactly K steps, CUDA events on the launching stream
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(STAGES) + 1)] for _ in range(args.steps)]
    wall0 = time.time()
    for k in range(args.steps):
        step(evs[k])
    barrier()
    wall1 = time.time()
    launches = launches_per_step * args.steps
    clk = clocks.window(wall0, wall1) if clocks else None
    total_ms = evs[0][0].elapsed_time(evs[-1][-1])
    stage_ms = {s: float(np.mean([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(args.steps)]))
                for i, s in enumerate(STAGES)}
    total_ms = max_over_ranks(total_ms, dist, "cuda")

    # ---- the same GEMV chains on the identity-table ("native") pool: the overhead denominator.  Same launch mode,
    # cloaked and native interleaved rep by rep so that drift hits both alike.
    native_ms, cloaked_iso_ms, per_call_ms, plain_ms, matmul_ms = {}, {}, {}, {}, {}
    for b in (() if args.no_ab else BATCHES):
        gemv_chain(pool_n, b)
        gemv_chain(pool_p, b)
        gemv_chain(pool_n, b, per_call=True)

        def torch_matmul():                       # context only: cuBLAS on the plain permuted tensors, same shapes
            for nm, (n, k) in shapes:
                torch.matmul(X[b][k], perm[nm].t(), out=Y[b][nm])
        torch_matmul()
        torch.cuda.synchronize()
        variants = [(capture(lambda: gemv_chain(pool_n, b))[0], []), (capture(lambda: gemv_chain(pool_a, b))[0], []),
                    (capture(lambda: gemv_chain(pool_a, b, per_call=True))[0], []), (capture(lambda: gemv_chain(pool_p, b))[0], []),
                    (capture(torch_matmul)[0], [])]
        reps = max(args.steps, 5)
        for r_, _ in variants:
            for _ in range(3):
                r_()
        torch.cuda.synchronize()
        for _ in range(reps):
            for r_, acc_ in variants:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                r_()
                e1.record(stream)
                acc_.append((e0, e1))
        torch.cuda.synchronize()
        med = [float(np.median([e0.elapsed_time(e1) for e0, e1 in acc_])) for _, acc_ in variants]
        native_ms[b], cloaked_iso_ms[b], per_call_ms[b], plain_ms[b], matmul_ms[b] = med

    # ---- correctness inside the bench: the round trip restores the permuted weights bit for bit
    ok = all(torch.equal(back[nm], perm[nm]) for nm in perm)

    # ---- e2e: the same stages through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if (rank == 0 or world > 1) and not args.no_ab:
        hW = {nm: perm[nm].cpu().pin_memory() for nm in perm}            # permuted weights, for the staged variant
        hR = {nm: raw[nm].cpu().pin_memory() for nm in raw}              # the checkpoint as it is: raw weights in pinned host memory
        load_items = C.cloak_load_items([(hR[nm], o, 0, nm) for (nm, _), o in zip(shapes, offs)])
        hX = {nm: X[1][shp[1]].cpu().pin_memory() for nm, shp in shapes}
        hY = {nm: torch.empty(1, shp[0], dtype=torch.bfloat16).pin_memory() for nm, shp in shapes}
        h2d = sum(t.numel() * 2 for t in hW.values()) + sum(t.numel() * 2 for t in hX.values())
        d2h = sum(t.numel() * 2 for t in hY.values())

        def e2e_step(variant="load"):
            if variant == "shuffle_host":   # pre-permuted weights through one device staging buffer, one tensor at a time
                for (nm, _), o in zip(shapes, offs):
                    C.cloak_shuffle_host(pool_a, hW[nm], o, hW[nm].numel() * 2, stream)
            else:           # the fused load of the RAW weights: permutation + block scatter in one pass, keyed tensor order
                C.cloak_load_tensors(KEY_A, sh, pool_a, load_items, C.CLOAK_ROWMAJOR, stream)
            C.cloak_gemv_chain_host(pool_a, host_ops, 1, stream)     # X up, the 7 projections, Y back: one synchronisation
        host_ops = C.cloak_gemv_ops([(tens[nm], hX[nm], hY[nm], 0) for nm, _ in shapes])
        n_e2e = max(1, min(args.steps, 5))
        times = {}
        for variant in ("shuffle_host", "load"):
            for _ in range(2):                  # warm-up: the library's stream-ordered pool settles on its buffers
                e2e_step(variant)
            barrier()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                e2e_step(variant)
            barrier()
            times[variant] = (time.perf_counter() - t0) / n_e2e
        dt = times["load"]
        e2e_bytes = 2 * sb["B"] + sb["B"]           # shuffle (2 B/B) + one batch-1 GEMV pass over the layer
        # context: what the link itself delivers for the same bytes (one pinned -> device copy per tensor, nothing else)
        dst = {nm: torch.empty_like(perm[nm]) for nm in perm}
        for nm in perm:
            dst[nm].copy_(hW[nm], non_blocking=True)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            for nm in perm:
                dst[nm].copy_(hW[nm], non_blocking=True)
        barrier()
        h2d_peak = sb["B"] * n_e2e / (time.perf_counter() - t0) / 1e9
        del dst
        e2e = {"value": world * e2e_bytes / dt / 1e9, "unit": "GB/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3,
               "h2d_gbs": h2d / dt / 1e9, "h2d_peak_gbs_measured": h2d_peak, "frac_of_h2d_peak": h2d / dt / 1e9 / h2d_peak,
               "variants_ms_per_step": {"cloak_shuffle_host_of_pre_permuted_weights": times["shuffle_host"] * 1e3},
               "what": "cloak_load_tensors of the layer's RAW weights from pinned host memory (the gather kernels read across PCIe, "
                       "permute and scatter through the table in one pass; keyed tensor order) + cloak_gemv_chain_host of the 7 projections (batch 1); PCIe-bound: frac_of_h2d_peak = achieved "
                       "host->device rate / a plain pinned copy of the same tensors"}

    map_ms = C.cloak_pool_map_ms(pool_a)
    adjacency = C.cloak_pool_adjacency(pool_a)          # layout quality (G8): neighbours that stayed neighbours
    layout_report = {"cloaked": C.cloak_pool_layout_report(pool_a), "identity_pool": C.cloak_pool_layout_report(pool_n),
                     "paper_context": "PAPER.md:226-227 (L40S, vLLM): VA ranges backed by contiguous physical pages, default -> CloakLM: "
                                      "91.41 % -> 2.38 % (Llama 3.1 8B), 95.57 % -> 1.57 % (Qwen3 14B); unit undefined (G12): "
                                      "`pages.adjacent_fraction` is the closest analogue here"}
    torch.cuda.synchronize()
    for p in (pool_a, pool_b, pool_n, pool_p):
        C.cloak_pool_destroy(p)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peak, peak_kind = hbm_peak()
    ms_per_step = total_ms / args.steps
    gbs = lambda nbytes, ms: nbytes / ms / 1e6          # noqa: E731
    stages = {}
    for s in STAGES:
        nbytes = {"keygen": 0, "permute": sb["permute"], "shuffle": sb["shuffle"], "relayout": sb["relayout"],
                  "unshuffle": sb["unshuffle"]}.get(s, sb["B"])
        stages[s] = {"ms": stage_ms[s], "gbs": gbs(nbytes, stage_ms[s]) if nbytes else None,
                     "frac_hbm": gbs(nbytes, stage_ms[s]) / peak if nbytes else None}
    if args.no_ab:
        native_ms = cloaked_iso_ms = per_call_ms = plain_ms = matmul_ms = {b: float("nan") for b in BATCHES}
    overhead = {f"b{b}": (cloaked_iso_ms[b] - native_ms[b]) / native_ms[b] * 100.0 for b in BATCHES}
    gemv_ms = sum(stage_ms[f"gemv_b{b}"] for b in BATCHES)
    gemv_launches = len(BATCHES)                        # one chain launch (7 projections) per batch
    achieved = gbs(sb["gemv"], gemv_ms)
    line = {
        "metric": METRIC, "value": whole_job_gbs(sb["total"], ms_per_step, world), "unit": "GB/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "cfg1: one LLaMA-8B-shaped decoder layer, bf16, 436.2 MB, 64 KiB blocks, 2 MiB VMM pages",
                   "stages": STAGES, "batches": list(BATCHES), "key_a": hex(KEY_A), "key_b": hex(KEY_B),
                   "launch": ("one CUDA graph per stage, captured from the C-ABI calls" if args.launch == "graph"
                              else "stream launches from Python"),
                   "l2": "inputs larger than L2 (436 MB layer vs 126 MB L2); no flush",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "stages": stages,
        "shuffle_gbs": stages["shuffle"]["gbs"], "shuffle_frac_hbm": stages["shuffle"]["frac_hbm"],
        "gemv_gbs": {f"b{b}": stages[f"gemv_b{b}"]["gbs"] for b in BATCHES},
        "gemv_frac_hbm": {f"b{b}": stages[f"gemv_b{b}"]["frac_hbm"] for b in BATCHES},
        "gemv_isolated_ms": {"cloaked": cloaked_iso_ms, "native": native_ms, "cloaked_7_separate_calls": per_call_ms,
                             "native_one_plain_allocation": plain_ms, "torch_matmul_context": matmul_ms},
        "cloaked_vs_native_overhead_pct": overhead,
        "cloaked_vs_cublas_pct": {f"b{b}": (cloaked_iso_ms[b] - matmul_ms[b]) / matmul_ms[b] * 100.0 for b in BATCHES},
        "overhead_note": "north_star's target is cloaked vs THE SAME KERNEL on the unshuffled (identity-table) layout: "
                         "cloaked_vs_native_overhead_pct.  cloaked_vs_cublas_pct puts it next to torch.matmul (cuBLAS) on the plain "
                         "permuted tensors with plain pointers, 7 calls per batch in one CUDA graph: negative = faster than cuBLAS.",
        "hbm_peak_gbs": peak, "hbm_peak_kind": peak_kind, "hbm_nominal_gbs": 8000.0,
        "sm_weights": sm_weights_summary(C), "pool_map_ms": map_ms, "layout_adjacency": adjacency, "layout_report": layout_report, "pool_create_s": pool_create_s, "roundtrip_bit_exact": bool(ok),
        "roofline": {"bound": "hbm", "kernel": "gemv_chain_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": ncu_traffic()[0], "traffic_source": ncu_traffic()[1],
                     "launches_per_step": gemv_launches,
                     "bytes_per_launch": sb["gemv"] / gemv_launches, "avg_launch_us": gemv_ms / gemv_launches * 1e3,
                     "peak_kind": peak_kind},
        "clocks": clk, "e2e": e2e, "gpu_launches": int(launches), "runtime_info": C.cloak_runtime_info(),
    }
    if args.configs != "cfg1" and world == 1:
        # ---- the other configs of BASELINE.json, in the same process and under the same clock sampler
        from paper_2606_18400_b200 import workloads
        torch.cuda.empty_cache()
        want = args.configs.split(",")
        if "cfg2" in want:
            line["cfg2"] = workloads.bench_cfg2(clocks, args.min_seconds)
            torch.cuda.empty_cache()
        if "cfg3" in want:
            line["cfg3"] = workloads.bench_cfg3(clocks, args.min_seconds)
            torch.cuda.empty_cache()
        if "cfg4" in want:
            line["cfg4"] = workloads.bench_cfg4(clocks, args.min_seconds / 2)
            torch.cuda.empty_cache()
        if "moe" in want:
            line["moe"] = workloads.bench_moe(clocks, args.min_seconds / 2)
            torch.cuda.empty_cache()
        line["gpu_launches_other_configs"] = int(sum(line[k]["gpu_launches"] for k in ("cfg2", "cfg3", "cfg4", "moe") if k in line))
    if clocks is not None:
        clocks.stop()
    if not args.no_cpu_baseline and world == 1:      # (the oracle is timed on rank 0 at N = 1 only)
        # the oracle beside it: the WHOLE cfg1 layer through the same stages, bounded by repetitions, once with
        # numpy's BLAS on all cores and once limited to one thread
        dt, reps, used, sbo = oracle_time(ORACLE_LAYER, 3, 12.0)
        dt1, reps1, _, _ = oracle_time(ORACLE_LAYER, 1, 1.0, threads=1)
        line["cpu_baseline"] = {"value": sbo["total"] / dt / 1e9, "unit": "GB/s", "cores": used, "kind": "oracle",
                                "host_cpus": os.cpu_count(), "ms_per_step": dt * 1e3,
                                "single_thread": {"value": sbo["total"] / dt1 / 1e9, "unit": "GB/s", "ms_per_step": dt1 * 1e3, "reps": reps1},
                                "sample": f"cfg1 whole layer ({sbo['B']/1e6:.1f} MB), all stages of the step, {reps} rep(s); only the "
                                          "fp64 contraction (numpy BLAS) is threaded, the byte loops are single-threaded Python + numpy"}
        if "cfg3" in line:
            line["cfg3"]["oracle"] = oracle_cfg3_layer()
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cloak", choices=["cloak", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--launch", default="graph", choices=["graph", "stream"],
                    help="graph (default): each stage's C-ABI launches are captured once into a CUDA graph and replayed; "
                         "stream: plain launches from Python every step")
    ap.add_argument("--workload", default="cfg1", choices=["cfg1", "cfg2", "cfg3", "cfg4"],
                    help="cfg1 (default) is the headline step; cfg2-4 are the other BASELINE.json configs "
                         "(paper_2606_18400_b200/workloads.py), each printing its own JSON line")
    ap.add_argument("--reps", type=int, default=10, help="repetitions per measurement for --workload cfg2-4")
    ap.add_argument("--configs", default="cfg1,cfg2,cfg3,cfg4,moe",
                    help="what the line carries besides the cfg1 step (`value`): cfg2, cfg3, cfg4 blocks (BASELINE.json configs[2..4]) and the MoE decode chain (NEXT-4); "
                         "`--configs cfg1` for the step alone.  N > 1 replicas run the step alone.")
    ap.add_argument("--min-seconds", type=float, default=1.0, help="minimum length of each timed loop of the cfg2-4 blocks")
    ap.add_argument("--no-ab", action="store_true", help="skip the isolated native / per-call / cuBLAS A/B runs and the e2e leg (for ncu launch lists of the step alone)")
    ap.add_argument("--copy-hint", type=int, default=-1, help="A/B: cloak_set_copy_cache_hint (bit 0 stores, bit 1 loads evict_first)")
    ap.add_argument("--gemv-engine", type=int, default=0,
                    help="A/B: cloak_set_gemv_engine (0 auto, 1 one-shot kernel, 2 no PDL, 3 exclusive mode)")
    args = ap.parse_args()
    if args.workload != "cfg1":
        from paper_2606_18400_b200 import workloads
        return workloads.main([args.workload, "--reps", str(args.reps), "--gemv-engine", str(args.gemv_engine)])
    if args.impl == "cloak":
        import paper_2606_18400_b200 as C
        if args.gemv_engine:
            C.cloak_set_gemv_engine(args.gemv_engine)
        if args.copy_hint >= 0:
            C.cloak_set_copy_cache_hint(args.copy_hint)
    args.warmup = max(args.warmup, 3) if args.impl == "cloak" else args.warmup
    return run_reference(args) if args.impl == "reference" else run_cloak(args)


if __name__ == "__main__":
    sys.exit(main())
