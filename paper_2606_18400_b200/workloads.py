"""Measurement drivers for BASELINE.json configs[2..4]; configs[1] is bench.py's own step.

    python -m paper_2606_18400_b200.workloads cfg2|cfg3|cfg4|moe|rekey [--reps R] [--out file.json]
    python bench.py --workload cfg2|cfg3|cfg4            (same thing)

Each prints ONE JSON line.  Everything on the timed path is a C-ABI call of libcloak.so (through the ctypes
binding); torch supplies device buffers, streams, events and CUDA-graph capture.  Inputs are seeded and
synthetic (synth/, the shared generator: shapes of the paper's Llama-3.1-8B / Qwen3-32B checkpoints, values
~N(0, 0.02)).  Parity of these sizes against the CPU oracle is the job of tests/test_gpu_fullsize.py; here the
only checks are self-consistency ones (round trip restores the bytes, cloaked == identity-table output).
"""
import argparse
import json
import os
import sys
import time

import numpy as np

from .clocks import ClockSampler

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


def _imports():
    import torch
    import paper_2606_18400_b200 as C
    from synth import cuda as synth_cuda
    from synth import gen
    if not torch.cuda.is_available():
        raise SystemExit("workloads: no CUDA device; the cloak path has no CPU fallback")
    return torch, C, synth_cuda, gen


def time_gpu(torch, fn, reps, warmup=3, stream=None):
    """Median and min milliseconds of fn() over `reps` runs, CUDA events on the launching stream."""
    stream = stream or torch.cuda.current_stream()
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
    ev[0].record(stream)
    for i in range(reps):
        fn()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    ts = [ev[i].elapsed_time(ev[i + 1]) for i in range(reps)]
    return float(np.median(ts)), float(np.min(ts))


def graphed(torch, fn):
    """Capture fn() (asynchronous C-ABI launches on torch's current stream) into a CUDA graph; returns the replay
    callable.  Capture runs on a side stream, which is the current stream inside the `with`."""
    fn()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    torch.cuda.synchronize()
    return g.replay


def rate(nbytes, ms, peak):
    gbs = nbytes / ms / 1e6
    return {"ms": ms, "gbs": gbs, "frac_measured": gbs / peak, "frac_nominal": gbs / NOMINAL_HBM_GBS}


# ------------------------------------------------------------------------------------------ cfg4
def run_cfg4(args):
    """Granularity sweep (BASELINE.json configs[4]): shuffle, unshuffle, re-layout A->B of a 4 GiB buffer at block
    sizes 4 KiB .. 2 MiB, beside a device-to-device cudaMemcpy and the same kernel on an identity table."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[4]
    nbytes = int(args.bytes or c["bytes"])
    peak, peak_kind = hbm_peak()
    L = synth_cuda.fill(torch.empty(nbytes // 2, dtype=torch.bfloat16, device="cuda"), c["seed"], 0)
    back = torch.empty_like(L)
    memcpy_ms, _ = time_gpu(torch, lambda: back.copy_(L), args.reps)
    rows, ok = [], True
    launches0 = C.cloak_launch_count()
    for b in c["blocks"]:
        pa = C.cloak_pool_create(0, nbytes, b, c["page"], c["key"])
        pb = C.cloak_pool_create(0, nbytes, b, c["page"], c["key_b"])
        pn = C.cloak_pool_create(0, nbytes, b, c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
        try:
            r = {"block_bytes": b, "nblocks": nbytes // b, "pool_map_ms": C.cloak_pool_map_ms(pa)}
            for name, fn in (("shuffle", lambda: C.cloak_shuffle(pa, L, 0, nbytes)),
                             ("unshuffle", lambda: C.cloak_unshuffle(pa, back, 0, nbytes)),
                             ("relayout", lambda: C.cloak_relayout(pa, pb)),
                             ("identity_table", lambda: C.cloak_shuffle(pn, L, 0, nbytes))):
                med, mn = time_gpu(torch, fn, args.reps)
                r[name] = rate(2 * nbytes, med, peak)
                r[name]["ms_min"] = mn
            # self-consistency: the round trip and the re-laid-out pool both give the buffer back
            back.zero_()
            C.cloak_unshuffle(pa, back, 0, nbytes)
            r["roundtrip_bit_exact"] = bool(torch.equal(back, L))
            # NEXT-1: the same re-key in place (A -> B -> A -> ...), spare buffer 1/64 of the pool; host work included
            keys = (c["key_b"], c["key"])
            ts = []
            for i in range(4):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                C.cloak_rekey_inplace(pa, keys[i % 2], nbytes // 64)
                torch.cuda.synchronize()
                ts.append((time.perf_counter() - t0) * 1e3)
            r["rekey_inplace"] = dict(rate(2 * nbytes, float(np.median(ts)), peak), spare_bytes=nbytes // 64,
                                      note="wall clock: host cycle decomposition + upload + the two move passes")
            back.zero_()
            C.cloak_unshuffle(pa, back, 0, nbytes)
            r["rekey_inplace_bit_exact"] = bool(torch.equal(back, L))
            ok = ok and r["rekey_inplace_bit_exact"]
            back.zero_()
            C.cloak_unshuffle(pb, back, 0, nbytes)
            r["relayout_bit_exact"] = bool(torch.equal(back, L))
            ok = ok and r["roundtrip_bit_exact"] and r["relayout_bit_exact"]
            rows.append(r)
        finally:
            torch.cuda.synchronize()
            for p in (pa, pb, pn):
                C.cloak_pool_destroy(p)
    return {"workload": "cfg4: granularity sweep, %.2f GiB bf16 buffer, 2 MiB VMM pages" % (nbytes / 2**30),
            "bytes": nbytes, "reps": args.reps, "hbm_peak_gbs": peak, "hbm_peak_kind": peak_kind,
            "hbm_nominal_gbs": NOMINAL_HBM_GBS, "memcpy_d2d": rate(2 * nbytes, memcpy_ms, peak),
            "sweep": rows, "all_bit_exact": ok, "gpu_launches": C.cloak_launch_count() - launches0,
            "convention": "GB/s = 2 x payload bytes / time (one read + one write), as MEASURED_PEAKS.json's hbm_gbs"}


# ------------------------------------------------------------------------------------------ cfg2
def _load_model(torch, C, synth_cuda, gen, cfg, pools, offs, tile128, keep=None, layers=None):
    """Generates every tensor of a model config on the GPU (tensor id = position in gen.model_tensors), applies the
    S5 neuron/head permutation per layer (and the TILE128 conversion when asked), and shuffles it into each pool.
    keep: optional dict name -> tensor that receives the permuted logical bytes (cfg2's shuffle timing needs them
    resident).  Returns seconds spent."""
    c = gen.CONFIGS[cfg]
    tensors = gen.model_tensors(cfg)
    off = {nm: o for (nm, _), o in zip(tensors, offs)}
    tid = {nm: i for i, (nm, _) in enumerate(tensors)}
    t0 = time.perf_counter()
    lshapes = gen.layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"])
    raw = {nm: torch.empty(shp, dtype=torch.bfloat16, device="cuda") for nm, shp in lshapes}
    prm = {nm: torch.empty(shp, dtype=torch.bfloat16, device="cuda") for nm, shp in lshapes}
    til = {nm: torch.empty(shp, dtype=torch.bfloat16, device="cuda") for nm, shp in lshapes} if tile128 else None

    def put(name, t):
        for p in pools:
            C.cloak_shuffle(p, t, off[name], t.numel() * 2)

    for l in range(c.get("layers", 1) if layers is None else layers):
        for nm, _ in lshapes:
            synth_cuda.fill(raw[nm], c["seed"], tid[f"l{l}.{nm}"])
        sh = C.cloak_block_shape(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, l)
        dst = {nm: (keep[f"l{l}.{nm}"] if keep is not None else prm[nm]) for nm, _ in lshapes}
        C.cloak_permute_mlp_heads(c["key"], sh, **raw, **{k + "_o": v for k, v in dst.items()})
        for nm, (n, k) in lshapes:
            src = dst[nm]
            if tile128:
                C.cloak_to_tile128(src, til[nm], n, k, C.CLOAK_BF16)
                src = til[nm]
            put(f"l{l}.{nm}", src)
    for nm in ("embed", "lm_head"):
        if nm in tid:
            t = keep[nm] if keep is not None else torch.empty(tensors[tid[nm]][1], dtype=torch.bfloat16, device="cuda")
            synth_cuda.fill(t, c["seed"], tid[nm])
            put(nm, t)
    torch.cuda.synchronize()
    return time.perf_counter() - t0


def run_cfg2(args):
    """Full 32-layer LLaMA-8B-shaped model (BASELINE.json configs[2]): VMM mapper ms, whole-model shuffle GB/s,
    and the batch-1 decode chain of all projection GEMVs + lm_head, cloaked vs identity table."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[2]
    peak, peak_kind = hbm_peak()
    tensors = gen.model_tensors(2)
    sizes = [2 * n * k for _, (n, k) in tensors]
    offs, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    off = {nm: o for (nm, _), o in zip(tensors, offs)}
    payload = sum(sizes)
    t0 = time.perf_counter()
    pc = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
    create_s = time.perf_counter() - t0
    pn = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
    info = C.cloak_pool_info(pc)
    adjacency = C.cloak_pool_adjacency(pc)
    launches0 = C.cloak_launch_count()
    try:
        # ---- load path, two ways, on one layer's worth of source tensors reused for all 32 layers (timing only; the
        # real contents are loaded right after): S5 then S4 (permute into a scratch tensor, shuffle it) against the
        # fused cloak_load_mlp_heads (permuted rows/columns written straight through the block table)
        lshapes = gen.layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"])
        raw = {nm: synth_cuda.fill(torch.empty(shp, dtype=torch.bfloat16, device="cuda"), c["seed"], i)
               for i, (nm, shp) in enumerate(lshapes)}
        tmp = {nm: torch.empty_like(t) for nm, t in raw.items()}
        shs = [C.cloak_block_shape(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, l)
               for l in range(c["layers"])]
        loffs = [{nm: off[f"l{l}.{nm}"] for nm, _ in lshapes} for l in range(c["layers"])]

        def load_two_pass():
            for l in range(c["layers"]):
                C.cloak_permute_mlp_heads(c["key"], shs[l], **raw, **{k + "_o": v for k, v in tmp.items()})
                for nm, t in tmp.items():
                    C.cloak_shuffle(pc, t, loffs[l][nm], t.numel() * 2)

        def load_fused():
            for l in range(c["layers"]):
                C.cloak_load_mlp_heads(c["key"], shs[l], pc, loffs[l], **raw)

        layer_bytes = sum(t.numel() * 2 for t in raw.values()) * c["layers"]
        two_med, _ = time_gpu(torch, load_two_pass, max(3, args.reps // 2), warmup=1)
        fus_med, _ = time_gpu(torch, load_fused, max(3, args.reps // 2), warmup=1)
        load_paths = {"layers_bytes": layer_bytes,
                      "permute_then_shuffle": dict(rate(2 * layer_bytes, two_med, peak), passes=2),
                      "fused_load": dict(rate(2 * layer_bytes, fus_med, peak), passes=1),
                      "note": "GB/s = 2 x payload / time for both, so the fused path's advantage shows as a higher rate"}
        del raw, tmp

        # ---- NEXT-2 at model scale: the whole RAW checkpoint in pinned host memory, loaded by ONE cloak_load_tensors call (the
        # kernels read across PCIe, permute and scatter in the same pass, keyed tensor order); beside it the plain pinned copy
        host_load = None
        if not getattr(args, "no_host_load", False):
            tid = {nm: i for i, (nm, _) in enumerate(tensors)}
            t0 = time.perf_counter()
            hraw = {}
            tmp_d = {}
            for nm, shp in tensors:
                key_ = shp
                if key_ not in tmp_d:
                    tmp_d[key_] = torch.empty(shp, dtype=torch.bfloat16, device="cuda")
                synth_cuda.fill(tmp_d[key_], c["seed"], tid[nm])
                hraw[nm] = torch.empty(shp, dtype=torch.bfloat16).pin_memory()
                hraw[nm].copy_(tmp_d[key_])
            torch.cuda.synchronize()
            prep_s = time.perf_counter() - t0
            items = []
            for nm, shp in tensors:
                if "." in nm:
                    l, role = nm[1:].split(".")
                    items.append((hraw[nm], off[nm], int(l), role))
                else:
                    items.append((hraw[nm], off[nm], 0, "plain", shp[0], shp[1]))
            items = C.cloak_load_items(items)
            sh0 = C.cloak_block_shape(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, 0)
            ts = []
            for _ in range(3):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                C.cloak_load_tensors(c["key"], sh0, pc, items, C.CLOAK_ROWMAJOR)
                torch.cuda.synchronize()
                ts.append((time.perf_counter() - t0) * 1e3)
            dst = torch.empty(max(sizes) // 2, dtype=torch.bfloat16, device="cuda")
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for nm, shp in tensors:
                dst[:hraw[nm].numel()].view(shp).copy_(hraw[nm], non_blocking=True)
            torch.cuda.synchronize()
            plain_ms = (time.perf_counter() - t0) * 1e3
            ms = float(np.median(ts))
            host_load = {"bytes": payload, "load_tensors_ms": ms, "gbs": payload / ms / 1e6, "plain_pinned_copy_ms": plain_ms,
                         "plain_pinned_copy_gbs": payload / plain_ms / 1e6, "frac_of_plain_copy": plain_ms / ms,
                         "mapper_plus_load_s": (C.cloak_pool_map_ms(pc) + ms) / 1e3, "pinned_alloc_and_fill_s": prep_s,
                         "paper_context": "PAPER.md:226 (L40S): physical shuffle latency of Llama 3.1 8B 1.58 s"}
            del hraw, tmp_d, dst, items

        keep = {nm: torch.empty(shp, dtype=torch.bfloat16, device="cuda") for nm, shp in tensors}
        load_s = _load_model(torch, C, synth_cuda, gen, 2, (pc, pn), offs, False, keep=keep)

        # ---- S4 at model scale: all 226 tensors, one call each
        def shuffle_all():
            for nm, _ in tensors:
                C.cloak_shuffle(pc, keep[nm], off[nm], keep[nm].numel() * 2)
        sh_med, sh_min = time_gpu(torch, shuffle_all, args.reps)
        m_t, m_o, m_b = [keep[nm] for nm, _ in tensors], [off[nm] for nm, _ in tensors], [keep[nm].numel() * 2 for nm, _ in tensors]
        shm_med, shm_min = time_gpu(torch, lambda: C.cloak_shuffle_many(pc, m_t, m_o, m_b), args.reps)
        back = torch.empty(payload // 2, dtype=torch.bfloat16, device="cuda")
        views, at = {}, 0
        for nm, (n, k) in tensors:
            views[nm] = back[at:at + n * k].view(n, k)
            at += n * k

        def unshuffle_all():
            for nm, _ in tensors:
                C.cloak_unshuffle(pc, views[nm], off[nm], views[nm].numel() * 2)
        un_med, un_min = time_gpu(torch, unshuffle_all, args.reps)
        m_v = [views[nm] for nm, _ in tensors]
        unm_med, unm_min = time_gpu(torch, lambda: C.cloak_unshuffle_many(pc, m_v, m_o, m_b), args.reps)
        roundtrip = all(torch.equal(views[nm], keep[nm]) for nm, _ in tensors)
        del back, views

        # ---- S6 decode chain at batch 1: q,k,v <- xh; o <- xa; gate,up <- xh; down <- silu(gate)*up; lm_head <- xh
        H, I, Q = c["hidden"], c["inter"], c["n_q"] * c["head_dim"]
        xh = synth_cuda.fill(torch.empty(1, H, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 0, kind=gen.KIND_NORMAL)
        xa = synth_cuda.fill(torch.empty(1, Q, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 1, kind=gen.KIND_NORMAL)
        T = {nm: C.cloak_tensor(off[nm], shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for nm, shp in tensors}
        Y = {pool_name: {nm: torch.zeros(1, shp[0], dtype=torch.bfloat16, device="cuda") for nm, shp in tensors if nm != "embed"}
             for pool_name in ("cloaked", "native")}
        act = torch.empty(1, I, dtype=torch.bfloat16, device="cuda")

        def chain(pool, y):
            """Call by call: 7 cloak_gemv + 1 cloak_silu_mul per layer, lm_head last (257 launches)."""
            for l in range(c["layers"]):
                p = f"l{l}."
                for nm in ("q", "k", "v"):
                    C.cloak_gemv(pool, T[p + nm], xh, y[p + nm], 1)
                C.cloak_gemv(pool, T[p + "o"], xa, y[p + "o"], 1)
                C.cloak_gemv(pool, T[p + "gate"], xh, y[p + "gate"], 1)
                C.cloak_gemv(pool, T[p + "up"], xh, y[p + "up"], 1)
                C.cloak_silu_mul(y[p + "gate"], y[p + "up"], act, I, C.CLOAK_BF16)
                C.cloak_gemv(pool, T[p + "down"], act, y[p + "down"], 1)
            C.cloak_gemv(pool, T["lm_head"], xh, y["lm_head"], 1)

        def chain_ops(y):
            """The same 225 GEMVs as ONE cloak_gemv_chain: up also emits silu(gate_y) * up_y in its epilogue, down reads
            that and is the only op that waits for earlier ones (the library splits the list into launches of <= 48 ops)."""
            ops = []
            for l in range(c["layers"]):
                p = f"l{l}."
                ops += [(T[p + nm], xh, y[p + nm], 0) for nm in ("q", "k", "v")]
                ops += [(T[p + "o"], xa, y[p + "o"], 0), (T[p + "gate"], xh, y[p + "gate"], 0),
                        (T[p + "up"], xh, y[p + "up"], 0, y[p + "gate"], act), (T[p + "down"], act, y[p + "down"], 1)]
            ops.append((T["lm_head"], xh, y["lm_head"], 0))
            return C.cloak_gemv_ops(ops)

        read_bytes = payload - sizes[0]                     # every tensor but the embedding table
        res = {}
        for pool_name, pool in (("cloaked", pc), ("native", pn)):
            y = Y[pool_name]
            ops = chain_ops(y)
            r = {}
            for mode, fn in (("per_call", lambda: chain(pool, y)), ("chain", lambda: C.cloak_gemv_chain(pool, ops, 1))):
                med, mn = time_gpu(torch, fn, args.reps)
                gmed, gmn = time_gpu(torch, graphed(torch, fn), args.reps)
                r[mode] = {"stream": dict(rate(read_bytes, med, peak), ms_min=mn, tokens_per_s=1e3 / med),
                           "graph": dict(rate(read_bytes, gmed, peak), ms_min=gmn, tokens_per_s=1e3 / gmed)}
                if mode == "per_call":
                    snap = {nm: t.clone() for nm, t in y.items()}
            r["chain_identical_to_per_call"] = bool(all(torch.equal(snap[nm], y[nm]) for nm in y))
            res[pool_name] = r
        identical = all(torch.equal(Y["cloaked"][nm], Y["native"][nm]) for nm in Y["cloaked"])

        # ---- NEXT-1: periodic in-place re-key under decode.  Wall clock of one re-key (host cycle decomposition included)
        # for three spare-buffer sizes; the decode chain afterwards must give the same outputs through the new table.
        ops_c = chain_ops(Y["cloaked"])
        t_dec = res["cloaked"]["chain"]["graph"]["ms"]
        rekey = {}
        for label, spare, newkey in (("one_page", 0, 0x5678), ("64MiB", 64 << 20, 0x9abc), ("256MiB", 256 << 20, c["key"])):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            C.cloak_rekey_inplace(pc, newkey, spare)
            torch.cuda.synchronize()
            ms = (time.perf_counter() - t0) * 1e3
            snap = {nm: t.clone() for nm, t in Y["cloaked"].items()}
            for t in Y["cloaked"].values():
                t.zero_()
            C.cloak_gemv_chain(pc, ops_c, 1)
            torch.cuda.synchronize()
            rekey[label] = {"spare_bytes": spare or c["page"], "ms": ms, "gbs": 2 * total / ms / 1e6,
                            "decode_identical_after": bool(all(torch.equal(snap[nm], Y["cloaked"][nm]) for nm in snap)),
                            "amortised_overhead_pct": {f"every_{n}": ms / (n * t_dec) * 100 for n in (1000, 1500)}}
        ov = {f"{mode}_{k}": (res["cloaked"][mode][k]["ms"] - res["native"][mode][k]["ms"]) / res["native"][mode][k]["ms"] * 100
              for mode in ("per_call", "chain") for k in ("stream", "graph")}
    finally:
        torch.cuda.synchronize()
        map_ms = C.cloak_pool_map_ms(pc)
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
    return {"workload": "cfg2: 32-layer LLaMA-8B-shaped model, bf16, 226 tensors, 64 KiB blocks, 2 MiB VMM pages",
            "payload_bytes": payload, "arena_bytes": total, "npages": info["npages"], "nblocks": info["nb"],
            "reps": args.reps, "hbm_peak_gbs": peak, "hbm_peak_kind": peak_kind, "hbm_nominal_gbs": NOMINAL_HBM_GBS,
            "pool_map_ms": map_ms, "pool_create_s": create_s, "generate_permute_load_s": load_s,
            "layout_adjacency": adjacency,
            "shuffle": dict(rate(2 * payload, sh_med, peak), ms_min=sh_min),
            "unshuffle": dict(rate(2 * payload, un_med, peak), ms_min=un_min), "roundtrip_bit_exact": bool(roundtrip),
            "shuffle_many": dict(rate(2 * payload, shm_med, peak), ms_min=shm_min, launches=2),
            "unshuffle_many": dict(rate(2 * payload, unm_med, peak), ms_min=unm_min, launches=2),
            "load_paths": load_paths, "load_from_pinned_host": host_load,
            "decode_chain": res, "decode_read_bytes": read_bytes,
            "ideal_tokens_per_s_at_measured_peak": peak * 1e9 / read_bytes,
            "cloaked_vs_native_overhead_pct": ov, "cloaked_identical_to_native": bool(identical),
            "rekey_inplace": rekey,
            "gpu_launches": C.cloak_launch_count() - launches0}


# ------------------------------------------------------------------------------------------ cfg3
def run_cfg3(args):
    """Qwen-32B-shaped model, 64 layers, TILE128 storage (BASELINE.json configs[3]): cloaked decode GEMM of every
    projection at batch 32 and 128 on the tcgen05 path, cloaked vs identity table.  Layers are generated on the GPU
    one at a time; the host never holds the model."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[3]
    layers = int(args.layers or c["layers"])
    peak, peak_kind = hbm_peak()
    tensors = gen.model_tensors(3)[:7 * layers]
    sizes = [2 * n * k for _, (n, k) in tensors]
    offs, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    off = {nm: o for (nm, _), o in zip(tensors, offs)}
    payload = sum(sizes)
    t0 = time.perf_counter()
    pc = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
    create_s = time.perf_counter() - t0
    pn = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
    info = C.cloak_pool_info(pc)
    launches0 = C.cloak_launch_count()
    try:
        load_s = _load_model(torch, C, synth_cuda, gen, 3, (pc, pn), offs, True, layers=layers)
        H, I, Q = c["hidden"], c["inter"], c["n_q"] * c["head_dim"]
        T = {nm: C.cloak_tensor(off[nm], shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_TILE128) for nm, shp in tensors}
        lnames = [nm for nm, _ in gen.layer_shapes(H, I, c["n_q"], c["n_kv"], c["head_dim"])]
        out = {}
        for batch in ([int(v) for v in args.batches.split(",")] if getattr(args, "batches", "") else (32, 128)):
            X = {k: synth_cuda.fill(torch.empty(batch, k, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100,
                                    2 * batch + i, kind=gen.KIND_NORMAL) for i, k in enumerate(sorted({H, I, Q}))}
            Y = {pn_: {nm: torch.zeros(batch, dict(tensors)[f"l0.{nm}"][0], dtype=torch.bfloat16, device="cuda") for nm in lnames}
                 for pn_ in ("cloaked", "native")}

            def sweep(pool, y):
                """Call by call: 7 cloak_gemm per layer."""
                for l in range(layers):
                    for nm in lnames:
                        t = T[f"l{l}.{nm}"]
                        C.cloak_gemm(pool, t, X[t.K], y[nm], batch)

            def sweep_ops(yl):
                """The same 7 x layers GEMMs as one cloak_gemm_chain (the library launches 16 ops at a time).  The
                inputs are fixed synthetic matrices, so no op depends on another; every op has its own output."""
                return C.cloak_gemm_ops([(T[f"l{l}.{nm}"], X[T[f"l{l}.{nm}"].K], yl[l][nm]) for l in range(layers) for nm in lnames])

            res = {}
            sampler = ClockSampler(0)                   # SM clock, power, throttle reasons while this batch is measured
            sampler.wait_first_sample()
            t_start = time.time()
            for pool_name, pool in (("cloaked", pc), ("native", pn)):
                y = Y[pool_name]
                yl = [{nm: torch.zeros_like(y[nm]) for nm in lnames} for _ in range(layers)]
                ops = sweep_ops(yl)
                flops = 2.0 * batch * (payload / 2)
                r = {}
                modes = [m for m in ("per_call", "chain") if m in getattr(args, "modes", "per_call,chain").split(",")]
                for mode, fn in (("per_call", lambda: sweep(pool, y)), ("chain", lambda: C.cloak_gemm_chain(pool, ops, batch))):
                    if mode not in modes:
                        continue
                    med, mn = time_gpu(torch, fn, args.reps, warmup=2)
                    gmed, gmn = time_gpu(torch, graphed(torch, fn), args.reps, warmup=2)
                    r[mode] = {"stream": dict(rate(payload, med, peak), ms_min=mn, tflops=flops / med / 1e9),
                               "graph": dict(rate(payload, gmed, peak), ms_min=gmn, tflops=flops / gmed / 1e9)}
                # the call-by-call sweep reuses one output set, so what it leaves behind is the last layer's; a chain cuts K
                # where its ranges fall, so the two agree up to the fp32 summation order
                if len(modes) == 2:
                    r["chain_vs_per_call_max_rel"] = max(float((yl[layers - 1][nm].float() - y[nm].float()).norm() / y[nm].float().norm())
                                                     for nm in lnames)
                res[pool_name] = r
                Y[pool_name + "_chain"] = yl
            torch.cuda.synchronize()
            res["clocks"] = sampler.stop(t_start, time.time())
            res["identical"] = bool(all(torch.equal(Y["cloaked"][nm], Y["native"][nm]) for nm in lnames)
                                    and all(torch.equal(a[nm], b[nm]) for a, b in zip(Y["cloaked_chain"], Y["native_chain"]) for nm in lnames))
            del Y
            res["overhead_pct"] = {f"{mode}_{k}": (res["cloaked"][mode][k]["ms"] - res["native"][mode][k]["ms"])
                                   / res["native"][mode][k]["ms"] * 100 for mode in modes for k in ("stream", "graph")}
            out[f"b{batch}"] = res
    finally:
        torch.cuda.synchronize()
        map_ms = C.cloak_pool_map_ms(pc)
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
    return {"workload": "cfg3: Qwen-32B-shaped model, %d layers, bf16 TILE128, 64 KiB blocks, 2 MiB VMM pages" % layers,
            "payload_bytes": payload, "npages": info["npages"], "nblocks": info["nb"], "reps": args.reps,
            "hbm_peak_gbs": peak, "hbm_peak_kind": peak_kind, "hbm_nominal_gbs": NOMINAL_HBM_GBS,
            "pool_map_ms": map_ms, "pool_create_s": create_s, "generate_permute_tile_load_s": load_s,
            "gemm": out, "gemm_engine": int(getattr(args, "gemm_engine", 0)), "modes": getattr(args, "modes", "per_call,chain"), "launches_per_sweep": 7 * layers, "gpu_launches": C.cloak_launch_count() - launches0}


# ------------------------------------------------------------------------------------------ MoE (NEXT-4)
def _moe_model(torch, C, synth_cuda, gen, L):
    """Pools (cloaked, identity) holding L Qwen3-30B-A3B-shaped sparse layers, loaded generator -> S5 (heads; experts) ->
    shuffle_many layer by layer; the tensors and what the load cost."""
    c = gen.CONFIGS[5]
    H, I, E = c["hidden"], c["inter"], c["n_experts"]
    Q, KV = c["n_q"] * c["head_dim"], c["n_kv"] * c["head_dim"]
    names = []
    for l in range(L):
        for nm, n, k in (("q", Q, H), ("k", KV, H), ("v", KV, H), ("o", H, Q), ("router", E, H)):
            names.append((l, nm, n, k))
        for e in range(E):
            names += [(l, f"gate{e}", I, H), (l, f"up{e}", I, H), (l, f"down{e}", H, I)]
    sizes = [2 * n * k for _, _, n, k in names]
    offs, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    off = {(l, nm): o for (l, nm, _, _), o in zip(names, offs)}
    T = {(l, nm): C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for (l, nm, n, k), o in zip(names, offs)}
    pc = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
    pn = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
    m = {"c": c, "L": L, "pc": pc, "pn": pn, "T": T, "total": total, "perm_ms": 0.0}
    try:
        t0 = time.perf_counter()
        att = {nm: torch.empty(n, k, dtype=torch.bfloat16, device="cuda") for nm, n, k in (("q", Q, H), ("k", KV, H), ("v", KV, H), ("o", H, Q))}
        att_p = {nm: torch.empty_like(t) for nm, t in att.items()}
        raw = [torch.empty(s_, dtype=torch.bfloat16, device="cuda") for s_ in ((E, H), (E, I, H), (E, I, H), (E, H, I))]
        prm = [torch.empty_like(t) for t in raw]
        for l in range(L):
            for i, nm in enumerate(att):
                synth_cuda.fill(att[nm], c["seed"], l * 8 + i)
            for i, t in enumerate(raw):
                synth_cuda.fill(t, c["seed"], l * 8 + 4 + i, kind=gen.KIND_NORMAL if i == 0 else gen.KIND_WEIGHT)
            sh = C.cloak_block_shape(H, I, c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, l)
            C.cloak_permute_mlp_heads(c["key"], sh, **att, **{k + "_o": v for k, v in att_p.items()})
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            C.cloak_permute_experts(c["key"], C.cloak_moe_shape(H, I, E, C.CLOAK_BF16, l), *raw, *prm)
            e1.record()
            ts = [att_p[nm] for nm in att] + [prm[0]]
            os_ = [off[l, nm] for nm in att] + [off[l, "router"]]
            for e in range(E):
                ts += [prm[1][e], prm[2][e], prm[3][e]]
                os_ += [off[l, f"gate{e}"], off[l, f"up{e}"], off[l, f"down{e}"]]
            for p in (pc, pn):
                C.cloak_shuffle_many(p, ts, os_, [t.numel() * 2 for t in ts])
            torch.cuda.synchronize()
            m["perm_ms"] += e0.elapsed_time(e1)
        m["load_s"] = time.perf_counter() - t0
    except BaseException:
        torch.cuda.synchronize()
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
        raise
    return m


def _moe_chain(torch, C, synth_cuda, gen, m, batch=1):
    """The decode chain of every layer of _moe_model -- q, k, v, o, router, and gate | up (silu epilogue) | down of 8 seeded
    experts -- on fixed synthetic inputs: (marshalled ops, output tensors, weight bytes read)."""
    c, L, T = m["c"], m["L"], m["T"]
    H, I, E, K = c["hidden"], c["inter"], c["n_experts"], c["top_k"]
    Q, KV = c["n_q"] * c["head_dim"], c["n_kv"] * c["head_dim"]
    xh = synth_cuda.fill(torch.empty(batch, H, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 0, kind=gen.KIND_NORMAL)
    xa = synth_cuda.fill(torch.empty(batch, Q, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 1, kind=gen.KIND_NORMAL)
    rng = np.random.default_rng(c["seed"])
    sel = [sorted(int(e) for e in rng.choice(E, K, replace=False)) for _ in range(L)]
    ops, outs, rb = [], [xh, xa], 0
    z = lambda n: torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda")       # noqa: E731
    for l in range(L):
        y = {nm: z(n) for nm, n in (("q", Q), ("k", KV), ("v", KV), ("o", H), ("router", E))}
        ops += [(T[l, nm], xa if nm == "o" else xh, y[nm], 0) for nm in y]
        rb += 2 * (2 * Q * H + 2 * KV * H + E * H)
        downs = []
        for i, e in enumerate(sel[l]):
            yg, yu, act, yd = z(I), z(I), z(I), z(H)
            ops += [(T[l, f"gate{e}"], xh, yg, 0), (T[l, f"up{e}"], xh, yu, 0, yg, act)]
            downs.append((T[l, f"down{e}"], act, yd, 1 if i == 0 else 2))
            outs += [yg, yu, act, yd]
            rb += 2 * 3 * I * H
        ops += downs
        outs += list(y.values())
    return C.cloak_gemv_ops(ops), outs, rb


def run_moe(args):
    """Qwen3-30B-A3B-shaped sparse layers (hidden 2048, 128 experts of 768, top-8; attention 32 q / 4 kv heads): expert
    permutation + shuffle at load, then the batch-1 decode chain of every layer -- q, k, v, o, router, and gate | up | down
    of 8 (seeded) selected experts -- as one cloak_gemv_chain, cloaked vs identity table.  --layers picks the depth
    (default 12 of the model's 48: 15 GB per pool)."""
    torch, C, synth_cuda, gen = _imports()
    L = int(args.layers or 12)
    peak, peak_kind = hbm_peak()
    launches0 = C.cloak_launch_count()
    m = _moe_model(torch, C, synth_cuda, gen, L)
    c, pc, pn = m["c"], m["pc"], m["pn"]
    H, I, E = c["hidden"], c["inter"], c["n_experts"]
    try:
        res, outs = {}, {}
        for pool_name, pool in (("cloaked", pc), ("native", pn)):
            ops, outs[pool_name], read_bytes = _moe_chain(torch, C, synth_cuda, gen, m)
            fn = lambda: C.cloak_gemv_chain(pool, ops, 1)        # noqa: E731
            med, mn = time_gpu(torch, fn, args.reps)
            gmed, gmn = time_gpu(torch, graphed(torch, fn), args.reps)
            res[pool_name] = {"stream": dict(rate(read_bytes, med, peak), ms_min=mn), "graph": dict(rate(read_bytes, gmed, peak), ms_min=gmn),
                              "ops": len(ops)}
        identical = all(torch.equal(a_, b_) for a_, b_ in zip(outs["cloaked"], outs["native"]))
        ov = {k: (res["cloaked"][k]["ms"] - res["native"][k]["ms"]) / res["native"][k]["ms"] * 100 for k in ("stream", "graph")}
    finally:
        torch.cuda.synchronize()
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
    return {"workload": "moe: Qwen3-30B-A3B-shaped sparse layers, %d of 48 layers, 128 experts, top-8, bf16, 64 KiB blocks" % L,
            "arena_bytes": m["total"], "layers": L, "reps": args.reps, "hbm_peak_gbs": peak, "hbm_peak_kind": peak_kind,
            "load_s": m["load_s"], "permute_experts_ms_per_layer": m["perm_ms"] / L,
            "permute_experts_gbs": 2 * 2 * (E * H + 3 * E * I * H) / (m["perm_ms"] / L) / 1e6,
            "gemv_engine": int(getattr(args, "gemv_engine", 0)),
            "decode_chain": res, "decode_read_bytes": read_bytes, "decode_read_bytes_full_model": read_bytes // L * 48,
            "tokens_per_s_extrapolated_48_layers": 1e3 / (res["cloaked"]["graph"]["ms"] / L * 48),
            "cloaked_vs_native_overhead_pct": ov, "cloaked_identical_to_native": bool(identical),
            "gpu_launches": C.cloak_launch_count() - launches0}


# ------------------------------------------------------------------------------------------ brief blocks for bench.py
# bench.py's default run carries cfg2, cfg3 and cfg4 next to the cfg1 step: one sub-object per measurement
# with the report schema's fields, every timed loop at least `min_s` seconds long so that the clock record means something.
def time_loop(torch, fn, min_s=1.0, min_reps=10, max_reps=50000, warmup=3):
    """fn() repeated for at least min_s seconds of device time, one CUDA event per repetition on the launching stream."""
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(3):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    est = max(e0.elapsed_time(e1) / 3, 1e-3)
    reps = int(min(max(min_reps, np.ceil(min_s * 1e3 / est)), max_reps))
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
    w0 = time.time()
    ev[0].record(stream)
    for i in range(reps):
        fn()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    w1 = time.time()
    ts = np.array([ev[i].elapsed_time(ev[i + 1]) for i in range(reps)])
    return {"t_ms_median": float(np.median(ts)), "t_ms_min": float(ts.min()), "t_ms_mean": float(ev[0].elapsed_time(ev[-1]) / reps),
            "reps": reps, "wall": (w0, w1)}


def ab_loop(torch, fn_a, fn_b, reps):
    """fn_a and fn_b alternated rep by rep (drift hits both alike); medians in ms."""
    stream = torch.cuda.current_stream()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * reps + 1)]
    ev[0].record(stream)
    for i in range(reps):
        fn_a()
        ev[2 * i + 1].record(stream)
        fn_b()
        ev[2 * i + 2].record(stream)
    torch.cuda.synchronize()
    ta = [ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(reps)]
    tb = [ev[2 * i + 1].elapsed_time(ev[2 * i + 2]) for i in range(reps)]
    return float(np.median(ta)), float(np.median(tb))


def measure(torch, sampler, peak, nbytes, fn, fn_identity=None, min_s=1.0, flops=None, extra=None):
    """One report-schema entry: the cloaked call timed for >= min_s seconds, then (if given) alternated with the same call
    on the identity-table pool for the overhead figure."""
    r = time_loop(torch, fn, min_s)
    w0, w1 = r.pop("wall")
    gbs = nbytes / r["t_ms_median"] / 1e6
    out = {"bytes_algorithmic": int(nbytes), **r, "gbs": gbs, "frac_measured": gbs / peak, "frac_nominal": gbs / NOMINAL_HBM_GBS}
    if flops:
        out["flops"] = float(flops)
        out["tflops"] = flops / r["t_ms_median"] / 1e9
    out["clocks"] = sampler.window(w0, w1) if sampler is not None else None
    if fn_identity is not None:
        for _ in range(3):
            fn_identity()
        pairs = int(min(max(20, np.ceil(0.5 * min_s * 1e3 / r["t_ms_median"])), 5000))
        tc, ti = ab_loop(torch, fn, fn_identity, pairs)
        out.update({"t_identity_ms": ti, "t_cloaked_ms_alternated": tc, "overhead_pct": (tc - ti) / ti * 100.0})
    if extra:
        out.update(extra)
    return out


def _graph(torch, fn):
    """fn() (C-ABI launches on torch's current stream) run once, then captured into a CUDA graph."""
    fn()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        fn()
    torch.cuda.synchronize()
    return g


def bench_cfg2(sampler, min_s=1.0):
    """cfg2 for the bench line: mapper ms, whole-model cloak_shuffle_many / cloak_unshuffle_many, the 225-op decode chain
    (graph replay) cloaked vs identity table."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[2]
    peak, _ = hbm_peak()
    tensors = gen.model_tensors(2)
    sizes = [2 * n * k for _, (n, k) in tensors]
    offs, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    off = {nm: o for (nm, _), o in zip(tensors, offs)}
    payload = sum(sizes)
    pc = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
    pn = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
    launches0 = C.cloak_launch_count()
    out = {"workload": "cfg2: 32-layer LLaMA-8B-shaped model, bf16, 226 tensors, 64 KiB blocks, 2 MiB VMM pages",
           "payload_bytes": payload, "npages": C.cloak_pool_info(pc)["npages"],
           "layout_report": {"cloaked": C.cloak_pool_layout_report(pc), "identity_pool": C.cloak_pool_layout_report(pn)},
           "pool_map_ms": {"cloaked": C.cloak_pool_map_ms(pc), "identity": C.cloak_pool_map_ms(pn)}}
    try:
        keep = {nm: torch.empty(shp, dtype=torch.bfloat16, device="cuda") for nm, shp in tensors}
        t0 = time.perf_counter()
        _load_model(torch, C, synth_cuda, gen, 2, (), offs, False, keep=keep)
        out["generate_permute_s"] = time.perf_counter() - t0
        m_t, m_o, m_b = [keep[nm] for nm, _ in tensors], [off[nm] for nm, _ in tensors], [keep[nm].numel() * 2 for nm, _ in tensors]
        C.cloak_shuffle_many(pn, m_t, m_o, m_b)
        out["shuffle"] = measure(torch, sampler, peak, 2 * payload, lambda: C.cloak_shuffle_many(pc, m_t, m_o, m_b),
                                 lambda: C.cloak_shuffle_many(pn, m_t, m_o, m_b), min_s, extra={"call": "cloak_shuffle_many, 226 ranges, 2 launches"})
        back = torch.empty(payload // 2, dtype=torch.bfloat16, device="cuda")
        views, at = [], 0
        for nm, (n, k) in tensors:
            views.append(back[at:at + n * k].view(n, k))
            at += n * k
        out["unshuffle"] = measure(torch, sampler, peak, 2 * payload, lambda: C.cloak_unshuffle_many(pc, views, m_o, m_b), None, min_s,
                                   extra={"call": "cloak_unshuffle_many, 226 ranges, 2 launches"})
        out["roundtrip_bit_exact"] = bool(all(torch.equal(v, keep[nm]) for v, (nm, _) in zip(views, tensors)))
        del back, views, keep, m_t
        torch.cuda.empty_cache()
        # ---- decode chain at batch 1 (same op list as run_cfg2)
        H, I, Q = c["hidden"], c["inter"], c["n_q"] * c["head_dim"]
        xh = synth_cuda.fill(torch.empty(1, H, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 0, kind=gen.KIND_NORMAL)
        xa = synth_cuda.fill(torch.empty(1, Q, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 1, kind=gen.KIND_NORMAL)
        T = {nm: C.cloak_tensor(off[nm], shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for nm, shp in tensors}
        read_bytes = payload - sizes[0]
        graphs, Y = {}, {}
        for name, pool in (("cloaked", pc), ("native", pn)):
            y = {nm: torch.zeros(1, shp[0], dtype=torch.bfloat16, device="cuda") for nm, shp in tensors if nm != "embed"}
            act = torch.empty(1, I, dtype=torch.bfloat16, device="cuda")
            ops = []
            for l in range(c["layers"]):
                p = f"l{l}."
                ops += [(T[p + nm], xh, y[p + nm], 0) for nm in ("q", "k", "v")]
                ops += [(T[p + "o"], xa, y[p + "o"], 0), (T[p + "gate"], xh, y[p + "gate"], 0),
                        (T[p + "up"], xh, y[p + "up"], 0, y[p + "gate"], act), (T[p + "down"], act, y[p + "down"], 1)]
            ops.append((T["lm_head"], xh, y["lm_head"], 0))
            ops = C.cloak_gemv_ops(ops)
            graphs[name] = (_graph(torch, lambda: C.cloak_gemv_chain(pool, ops, 1)), ops, act)
            Y[name] = y
        d = measure(torch, sampler, peak, read_bytes, graphs["cloaked"][0].replay, graphs["native"][0].replay, min_s,
                    extra={"call": "cloak_gemv_chain, 225 ops, batch 1, CUDA-graph replay"})
        d["tokens_per_s"] = 1e3 / d["t_ms_median"]
        d["ideal_tokens_per_s_at_measured_peak"] = peak * 1e9 / read_bytes
        d["cloaked_identical_to_native"] = bool(all(torch.equal(Y["cloaked"][nm], Y["native"][nm]) for nm in Y["cloaked"]))
        out["decode_chain"] = d
    finally:
        torch.cuda.synchronize()
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
    out["gpu_launches"] = C.cloak_launch_count() - launches0
    return out


def bench_cfg3(sampler, min_s=1.0, layers=None, batches=(32, 128), depths=(8, 64)):
    """cfg3 for the bench line: the tcgen05 GEMM chain over the first 8 layers and over all 64 layers of the 62 GB TILE128 pool
    at batch 32 and 128 (graph replay), cloaked vs identity table."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[3]
    layers = int(layers or c["layers"])
    peak, _ = hbm_peak()
    tensors = gen.model_tensors(3)[:7 * layers]
    sizes = [2 * n * k for _, (n, k) in tensors]
    offs, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    off = {nm: o for (nm, _), o in zip(tensors, offs)}
    pc = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
    pn = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
    launches0 = C.cloak_launch_count()
    out = {"workload": "cfg3: Qwen-32B-shaped model, %d layers, bf16 TILE128, 64 KiB blocks, 2 MiB VMM pages" % layers,
           "payload_bytes": sum(sizes), "npages": C.cloak_pool_info(pc)["npages"],
           "pool_map_ms": {"cloaked": C.cloak_pool_map_ms(pc), "identity": C.cloak_pool_map_ms(pn)}, "gemm": {}}
    try:
        t0 = time.perf_counter()
        _load_model(torch, C, synth_cuda, gen, 3, (pc, pn), offs, True, layers=layers)
        out["generate_permute_tile_load_s"] = time.perf_counter() - t0
        torch.cuda.empty_cache()
        H, I, Q = c["hidden"], c["inter"], c["n_q"] * c["head_dim"]
        T = {nm: C.cloak_tensor(off[nm], shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_TILE128) for nm, shp in tensors}
        lnames = [nm for nm, _ in gen.layer_shapes(H, I, c["n_q"], c["n_kv"], c["head_dim"])]
        for batch in batches:
            X = {k: synth_cuda.fill(torch.empty(batch, k, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 2 * batch + i,
                                    kind=gen.KIND_NORMAL) for i, k in enumerate(sorted({H, I, Q}))}
            for depth in [d for d in depths if d <= layers]:
                nbytes = sum(sizes[:7 * depth])
                g, ys = {}, {}
                for name, pool in (("cloaked", pc), ("native", pn)):
                    yl = [{nm: torch.zeros(batch, dict(tensors)[f"l0.{nm}"][0], dtype=torch.bfloat16, device="cuda") for nm in lnames}
                          for _ in range(depth)]
                    ops = C.cloak_gemm_ops([(T[f"l{l}.{nm}"], X[T[f"l{l}.{nm}"].K], yl[l][nm]) for l in range(depth) for nm in lnames])
                    C.cloak_pool_reserve_workspace(pool, C.cloak_gemm_chain_scratch_bytes(pool, ops, batch))
                    g[name] = (_graph(torch, lambda: C.cloak_gemm_chain(pool, ops, batch)), ops)
                    ys[name] = yl
                # the same chain captured with single tile rows (cloak_set_gemm_engine(1)), alternated replay by replay with the
                # default grouping: what sharing the X tile between two rows is worth on THIS board under THIS power state
                C.cloak_set_gemm_engine(1)
                try:
                    ops_c = g["cloaked"][1]
                    C.cloak_pool_reserve_workspace(pc, C.cloak_gemm_chain_scratch_bytes(pc, ops_c, batch))
                    g1 = _graph(torch, lambda: C.cloak_gemm_chain(pc, ops_c, batch))
                finally:
                    C.cloak_set_gemm_engine(0)
                for _ in range(3):
                    g1.replay()
                t_once = time_loop(torch, g1.replay, 0.05)["t_ms_median"]
                tp, ts1 = ab_loop(torch, g["cloaked"][0].replay, g1.replay, int(min(max(10, np.ceil(0.5 * min_s * 1e3 / t_once)), 2000)))
                del g1
                d = measure(torch, sampler, peak, nbytes, g["cloaked"][0].replay, g["native"][0].replay, min_s,
                            flops=2.0 * batch * (nbytes / 2),
                            extra={"call": "cloak_gemm_chain, %d ops, batch %d, CUDA-graph replay" % (7 * depth, batch)})
                d["cloaked_identical_to_native"] = bool(all(torch.equal(a[nm], b[nm]) for a, b in zip(ys["cloaked"], ys["native"]) for nm in lnames))
                d.update({"t_row_pairs_ms_alternated": tp, "t_single_rows_ms": ts1, "row_pairs_gain_pct": (ts1 - tp) / ts1 * 100.0,
                          "single_rows_frac_measured": nbytes / ts1 / 1e6 / peak})
                out["gemm"][f"b{batch}_{depth}layers"] = d
                del g, ys
            del X
            torch.cuda.empty_cache()
    finally:
        torch.cuda.synchronize()
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
    out["gpu_launches"] = C.cloak_launch_count() - launches0
    return out


def bench_moe(sampler, min_s=0.5, layers=12):
    """The MoE decode chain for the bench line: `layers` Qwen3-30B-A3B-shaped sparse layers, batch 1, graph
    replay, cloaked vs identity table, and alternated with the same chain captured without the fusion of the experts' ops."""
    torch, C, synth_cuda, gen = _imports()
    peak, _ = hbm_peak()
    launches0 = C.cloak_launch_count()
    m = _moe_model(torch, C, synth_cuda, gen, layers)
    c, pc, pn = m["c"], m["pc"], m["pn"]
    H, I, E = c["hidden"], c["inter"], c["n_experts"]
    out = {"workload": "moe: Qwen3-30B-A3B-shaped sparse layers, %d of 48 layers, 128 experts, top-8, bf16, 64 KiB blocks" % layers,
           "arena_bytes": m["total"], "pool_map_ms": {"cloaked": C.cloak_pool_map_ms(pc), "identity": C.cloak_pool_map_ms(pn)},
           "generate_permute_load_s": m["load_s"], "permute_experts_ms_per_layer": m["perm_ms"] / layers,
           "permute_experts_gbs": 2 * 2 * (E * H + 3 * E * I * H) / (m["perm_ms"] / layers) / 1e6}
    try:
        g, outs = {}, {}
        for name, pool in (("cloaked", pc), ("native", pn)):
            ops, outs[name], read_bytes = _moe_chain(torch, C, synth_cuda, gen, m)
            g[name] = (_graph(torch, lambda: C.cloak_gemv_chain(pool, ops, 1)), ops)
        C.cloak_set_gemv_engine(4)                     # the same chain, every expert projection an op of its own
        try:
            ops_u, outs["unfused"], _ = _moe_chain(torch, C, synth_cuda, gen, m)
            gu = _graph(torch, lambda: C.cloak_gemv_chain(pc, ops_u, 1))
        finally:
            C.cloak_set_gemv_engine(0)
        d = measure(torch, sampler, peak, read_bytes, g["cloaked"][0].replay, g["native"][0].replay, min_s,
                    extra={"call": "cloak_gemv_chain, %d ops, batch 1, CUDA-graph replay" % len(g["cloaked"][1])})
        tf, tu = ab_loop(torch, g["cloaked"][0].replay, gu.replay, int(min(max(20, np.ceil(0.5 * min_s * 1e3 / d["t_ms_median"])), 5000)))
        d.update({"t_fused_ms_alternated": tf, "t_unfused_ms": tu, "fusion_gain_pct": (tu - tf) / tu * 100.0,
                  "unfused_frac_measured": read_bytes / tu / 1e6 / peak,
                  "tokens_per_s_extrapolated_48_layers": 1e3 / (d["t_ms_median"] / layers * 48),
                  "cloaked_identical_to_native": bool(all(torch.equal(a_, b_) for a_, b_ in zip(outs["cloaked"], outs["native"]))),
                  "fused_identical_to_unfused": bool(all(torch.equal(a_, b_) for a_, b_ in zip(outs["cloaked"], outs["unfused"])))})
        out["decode_chain"] = d
    finally:
        torch.cuda.synchronize()
        C.cloak_pool_destroy(pc)
        C.cloak_pool_destroy(pn)
    out["gpu_launches"] = C.cloak_launch_count() - launches0
    return out


def bench_cfg4(sampler, min_s=0.5):
    """cfg4 for the bench line: shuffle (vs identity table), unshuffle and re-layout A -> B of the 4 GiB buffer at the five
    block sizes, beside a device-to-device copy."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[4]
    nbytes = int(c["bytes"])
    peak, _ = hbm_peak()
    L = synth_cuda.fill(torch.empty(nbytes // 2, dtype=torch.bfloat16, device="cuda"), c["seed"], 0)
    back = torch.empty_like(L)
    launches0 = C.cloak_launch_count()
    out = {"workload": "cfg4: granularity sweep, 4 GiB bf16 buffer, 2 MiB VMM pages, keys 0x1234 -> 0x5678", "bytes": nbytes,
           "memcpy_d2d": measure(torch, sampler, peak, 2 * nbytes, lambda: back.copy_(L), None, min_s, extra={"call": "torch copy_ (context)"}),
           "sweep": {}}
    ok = True
    for b in c["blocks"]:
        pa = C.cloak_pool_create(0, nbytes, b, c["page"], c["key"])
        pb = C.cloak_pool_create(0, nbytes, b, c["page"], c["key_b"])
        pn = C.cloak_pool_create(0, nbytes, b, c["page"], c["key"], C.CLOAK_POOL_IDENTITY)
        try:
            r = {"block_bytes": b, "nblocks": nbytes // b, "pool_map_ms": C.cloak_pool_map_ms(pa)}
            r["shuffle"] = measure(torch, sampler, peak, 2 * nbytes, lambda: C.cloak_shuffle(pa, L, 0, nbytes),
                                   lambda: C.cloak_shuffle(pn, L, 0, nbytes), min_s)
            r["unshuffle"] = measure(torch, sampler, peak, 2 * nbytes, lambda: C.cloak_unshuffle(pa, back, 0, nbytes), None, min_s)
            r["roundtrip_bit_exact"] = bool(torch.equal(back, L))
            r["relayout"] = measure(torch, sampler, peak, 2 * nbytes, lambda: C.cloak_relayout(pa, pb), None, min_s)
            back.zero_()
            C.cloak_unshuffle(pb, back, 0, nbytes)
            r["relayout_bit_exact"] = bool(torch.equal(back, L))
            ok = ok and r["roundtrip_bit_exact"] and r["relayout_bit_exact"]
            out["sweep"][f"{b // 1024}KiB"] = r
        finally:
            torch.cuda.synchronize()
            for p in (pa, pb, pn):
                C.cloak_pool_destroy(p)
    out["all_bit_exact"] = ok
    out["gpu_launches"] = C.cloak_launch_count() - launches0
    return out


# ------------------------------------------------------------------------------------------ NEXT-1: page re-key under live decode
def run_rekey(args):
    """The cfg2 decode chain (225 GEMVs, batch 1, CUDA-graph replay) run continuously while the pool's PHYSICAL PAGE MAP is
    re-randomised (cloak_rekey_pages_begin / _step): per-step latency (CUDA event to CUDA event) p50 / p99 / max against the
    cadence of the re-key -- one full re-randomisation of the 7 658 pages every 1 000 / 1 500 decode steps
    and at one page per step.  The serving loop keeps one step in flight: launch step i, then do the re-key's driver calls
    for it while the GPU runs, then wait for step i-1."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[2]
    layers = int(args.layers or c["layers"])
    peak, peak_kind = hbm_peak()
    tensors = [t for t in gen.model_tensors(2) if "." not in t[0] or int(t[0][1:].split(".")[0]) < layers]
    sizes = [2 * n * k for _, (n, k) in tensors]
    offs, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    off = {nm: o for (nm, _), o in zip(tensors, offs)}
    pc = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
    npages = C.cloak_pool_info(pc)["npages"]
    out = {"workload": "rekey: cfg2 decode chain (%d layers + lm_head, batch 1) under periodic page-map re-randomisation" % layers,
           "npages": npages, "arena_bytes": total, "hbm_peak_gbs": peak, "cadences": {}}
    try:
        lshapes = gen.layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"])
        raw = {nm: torch.empty(shp, dtype=torch.bfloat16, device="cuda") for nm, shp in lshapes}
        tid = {nm: i for i, (nm, _) in enumerate(gen.model_tensors(2))}
        for l in range(layers):
            for nm, _ in lshapes:
                synth_cuda.fill(raw[nm], c["seed"], tid[f"l{l}.{nm}"])
            sh = C.cloak_block_shape(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, l)
            C.cloak_load_mlp_heads(c["key"], sh, pc, {nm: off[f"l{l}.{nm}"] for nm, _ in lshapes}, **raw)
        for nm in ("embed", "lm_head"):
            t = synth_cuda.fill(torch.empty(dict(tensors)[nm], dtype=torch.bfloat16, device="cuda"), c["seed"], tid[nm])
            C.cloak_shuffle(pc, t, off[nm], t.numel() * 2)
            del t
        H, I, Q = c["hidden"], c["inter"], c["n_q"] * c["head_dim"]
        xh = synth_cuda.fill(torch.empty(1, H, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 0, kind=gen.KIND_NORMAL)
        xa = synth_cuda.fill(torch.empty(1, Q, dtype=torch.bfloat16, device="cuda"), c["seed"] + 100, 1, kind=gen.KIND_NORMAL)
        T = {nm: C.cloak_tensor(off[nm], shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for nm, shp in tensors}
        y = {nm: torch.zeros(1, shp[0], dtype=torch.bfloat16, device="cuda") for nm, shp in tensors if nm != "embed"}
        act = torch.empty(1, I, dtype=torch.bfloat16, device="cuda")
        ops = []
        for l in range(layers):
            p = f"l{l}."
            ops += [(T[p + nm], xh, y[p + nm], 0) for nm in ("q", "k", "v")]
            ops += [(T[p + "o"], xa, y[p + "o"], 0), (T[p + "gate"], xh, y[p + "gate"], 0),
                    (T[p + "up"], xh, y[p + "up"], 0, y[p + "gate"], act), (T[p + "down"], act, y[p + "down"], 1)]
        ops.append((T["lm_head"], xh, y["lm_head"], 0))
        ops = C.cloak_gemv_ops(ops)
        g = _graph(torch, lambda: C.cloak_gemv_chain(pc, ops, 1))
        g.replay()
        torch.cuda.synchronize()
        ref = {nm: t.clone() for nm, t in y.items()}
        stream = torch.cuda.current_stream()

        def serve(nsteps, moves_per_step, spares, new_key):
            """nsteps decode steps (or until the re-key is complete when moves_per_step > 0); per-step GPU latency in ms."""
            if moves_per_step:
                C.cloak_rekey_pages_begin(pc, new_key, spares)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(nsteps + 1)]
            host = []
            ev[0].record(stream)
            done_at, i = None, 0
            t_wall = time.perf_counter()
            while i < nsteps:
                g.replay()
                ev[i + 1].record(stream)
                if moves_per_step and done_at is None:
                    t0 = time.perf_counter()
                    if C.cloak_rekey_pages_step(pc, moves_per_step) == 0:
                        done_at = i + 1
                    host.append((time.perf_counter() - t0) * 1e3)
                if i >= 1:
                    ev[i].synchronize()                       # the loop keeps one step in flight
                i += 1
                if moves_per_step and done_at is not None and i >= done_at + 50:
                    break
            torch.cuda.synchronize()
            wall = time.perf_counter() - t_wall
            lat = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(i)])
            same = bool(all(torch.equal(y[nm], ref[nm]) for nm in y))
            r = {"steps": int(i), "p50_ms": float(np.percentile(lat, 50)), "p99_ms": float(np.percentile(lat, 99)),
                 "max_ms": float(lat.max()), "mean_ms": float(lat.mean()), "tokens_per_s": i / wall,
                 "outputs_identical_to_before": same,
                 "latency_histogram_ms": {f"<={b}": int(np.count_nonzero(lat <= b)) for b in (3, 4, 6, 10, 20, 50, 100, 1000, 10000)},
                 "slowest_steps": [(int(k), round(float(lat[k]), 2)) for k in np.argsort(lat)[::-1][:12]]}
            if moves_per_step:
                r.update({"moves_per_step": moves_per_step, "spare_pages": spares, "rekey_complete_after_steps": done_at,
                          "host_ms_per_step_call_median": float(np.median(host)) if host else None,
                          "host_ms_per_page": float(np.median(host)) / moves_per_step if host else None})
            return r

        sampler = ClockSampler(0)
        sampler.wait_first_sample()
        w0 = time.time()
        out["baseline_no_rekey"] = serve(2000, 0, 0, 0)
        keys = [0x5678, 0x9abc, 0xdef0, 0x1357]
        for (label, cadence), key in zip((("every_1000_steps", 1000), ("every_1500_steps", 1500), ("one_page_per_step", npages),
                                          ("stop_the_world", 0)), keys):
            if cadence:
                k = int(np.ceil(npages / cadence))
                # a move retires two steps after it was issued (one step in flight + its own), so 3 k spare pages keep k cycles ready
                r = serve(4 * cadence + 400, k, max(1, min(3 * k, 64)), key)
                base = out["baseline_no_rekey"]
                r["p50_overhead_pct"] = (r["p50_ms"] - base["p50_ms"]) / base["p50_ms"] * 100
                r["mean_overhead_pct"] = (r["mean_ms"] - base["mean_ms"]) / base["mean_ms"] * 100
            else:
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                C.cloak_rekey_pages_begin(pc, key, 16)
                C.cloak_rekey_pages_finish(pc)
                ms = (time.perf_counter() - t0) * 1e3
                g.replay()
                torch.cuda.synchronize()
                r = {"ms": ms, "ms_per_page": ms / npages, "spare_pages": 16,
                     "outputs_identical_to_before": bool(all(torch.equal(y[nm], ref[nm]) for nm in y)),
                     "amortised_pct_of_decode": {f"every_{n}_steps": ms / (n * out["baseline_no_rekey"]["p50_ms"]) * 100 for n in (1000, 1500)}}
            if pc is not None and r.get("rekey_complete_after_steps") is None and cadence:
                C.cloak_rekey_pages_finish(pc)               # (did not complete inside the step budget: finish it off)
            out["cadences"][label] = r
        out["clocks"] = sampler.stop(w0, time.time())
    finally:
        torch.cuda.synchronize()
        C.cloak_pool_destroy(pc)
    out["paper_context"] = "PAPER.md:207 / :271 / :283 (L40S, vLLM): re-shuffle every 1000-1500 iterations, < 2 % end-to-end; 1.5 s per shuffle (:265)"
    return out


# ------------------------------------------------------------------------------------------ S2: the VMM mapper
def run_mapper(args):
    """S2 alone: cloak_pool_create / cloak_pool_destroy of a cfg2-sized pool (7 658 pages of 2 MiB), `--reps` times: median and
    spread of the mapper and of its phases (cuMemCreate, cuMemMap, cuMemSetAccess), and of the teardown."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[2]
    sizes = [2 * n * k for _, (n, k) in gen.model_tensors(2)]
    _, total = C.cloak_arena_plan(c["key"], sizes, c["block"])
    rows = []
    for _ in range(max(3, args.reps if args.reps != 10 else 5)):
        t0 = time.perf_counter()
        p = C.cloak_pool_create(0, total, c["block"], c["page"], c["key"])
        t1 = time.perf_counter()
        r = dict(C.cloak_pool_map_phases(p), mapper_ms=C.cloak_pool_map_ms(p), pool_create_ms=(t1 - t0) * 1e3, npages=C.cloak_pool_info(p)["npages"])
        t0 = time.perf_counter()
        C.cloak_pool_destroy(p)
        r["pool_destroy_ms"] = (time.perf_counter() - t0) * 1e3
        rows.append(r)
    med = {k: float(np.median([r[k] for r in rows])) for k in rows[0]}
    return {"workload": "mapper: cfg2-sized pool, %d pages of 2 MiB" % rows[0]["npages"], "runs": rows, "median": med,
            "min": {k: float(np.min([r[k] for r in rows])) for k in rows[0]}, "max": {k: float(np.max([r[k] for r in rows])) for k in rows[0]},
            "us_per_page": {k: med[k] * 1e3 / rows[0]["npages"] for k in ("create_ms", "map_ms", "set_access_ms", "mapper_ms")},
            "paper_context": "PAPER.md:226 / :265 (L40S): physical page shuffle of Llama 3.1 8B 1.58 s, ~1.5 s per GPU"}


# ------------------------------------------------------------------------------------------ S5 A/B: the column gather
def run_permute_ab(args):
    """cloak_permute_mlp_heads of the cfg1 layer, and of `down` alone, under both column-gather engines (cloak_set_gather_engine:
    1 = element gather, 0 = pair-interleaved gather); the outputs must be identical."""
    torch, C, synth_cuda, gen = _imports()
    c = gen.CONFIGS[1]
    shapes = gen.layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"])
    raw = {nm: synth_cuda.fill(torch.empty(shp, dtype=torch.bfloat16, device="cuda"), c["seed"], i) for i, (nm, shp) in enumerate(shapes)}
    out = {nm: torch.empty_like(t) for nm, t in raw.items()}
    sh = C.cloak_block_shape(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"], C.CLOAK_BF16, 0)
    peak, _ = hbm_peak()
    B = sum(t.numel() * 2 for t in raw.values())
    res, keep = {}, {}
    try:
        for eng, name in ((1, "element_gather"), (0, "pair_interleaved_gather")):
            C.cloak_set_gather_engine(eng)
            full, _ = time_gpu(torch, lambda: C.cloak_permute_mlp_heads(c["key"], sh, **raw, **{k + "_o": v for k, v in out.items()}), 30)
            down, _ = time_gpu(torch, lambda: C.cloak_permute_mlp_heads(c["key"], sh, down=raw["down"], down_o=out["down"]), 30)
            keep[eng] = {nm: t.clone() for nm, t in out.items()}
            res[name] = {"layer_permute": rate(2 * B, full, peak), "down_alone_incl_keygen": rate(4 * raw["down"].numel(), down, peak)}
    finally:
        C.cloak_set_gather_engine(0)
    res["identical"] = bool(all(torch.equal(keep[0][nm], keep[1][nm]) for nm in out))
    return {"workload": "permute_ab: cfg1 layer, S5 under both column-gather engines", **res}


RUNNERS = {"cfg2": run_cfg2, "cfg3": run_cfg3, "cfg4": run_cfg4, "moe": run_moe, "rekey": run_rekey, "mapper": run_mapper, "permute_ab": run_permute_ab}


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("workload", choices=sorted(RUNNERS))
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--bytes", type=int, default=0, help="cfg4: buffer bytes (default 4 GiB)")
    ap.add_argument("--layers", type=int, default=0, help="cfg3: number of layers (default 64); moe: default 12 of 48")
    ap.add_argument("--batches", default="", help="cfg3: batch sizes, e.g. 16,64,256 (default 32,128)")
    ap.add_argument("--gemm-schedule", default="", help="cfg3: static_pct,dyn_chunk_tiles (cloak_set_gemm_schedule), e.g. 100,0")
    ap.add_argument("--gemm-engine", type=int, default=0, help="cloak_set_gemm_engine: 0 auto (row pairs in long launches), 1 single rows, 2 fours, 3 pairs always")
    ap.add_argument("--modes", default="per_call,chain", help="cfg3: which call patterns to time (per_call, chain)")
    ap.add_argument("--gemv-engine", type=int, default=0, help="cloak_set_gemv_engine: 0 auto, 1 one-shot, 2 no PDL, 3 exclusive mode (no cooperative launches), 4 no fusion of small ops")
    ap.add_argument("--out", default="")
    args = ap.parse_args(argv)
    if args.gemv_engine:
        _imports()[1].cloak_set_gemv_engine(args.gemv_engine)
    if args.gemm_engine:
        _imports()[1].cloak_set_gemm_engine(args.gemm_engine)
    if args.gemm_schedule:
        _imports()[1].cloak_set_gemm_schedule(*[int(v) for v in args.gemm_schedule.split(",")])
    line = json.dumps(RUNNERS[args.workload](args))
    print(line)
    if args.out:
        with open(args.out, "w") as f:
            f.write(line + "\n")
    return 0


if __name__ == "__main__":
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    sys.exit(main())
