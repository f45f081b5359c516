"""Thin ctypes binding of libcloak.so: same names as include/cloak.h, argument marshalling only.

Every step of the hot path runs in the CUDA library; this module adds no arithmetic.  PyTorch is used
by callers for device memory and streams; here a "pointer" argument is a torch tensor (its data_ptr()
is taken), a numpy array (host pointer) or a plain int address.  `stream` is a torch.cuda.Stream, an int
cudaStream_t, or None (= torch's current stream when torch.cuda is initialised, else the default stream).

The library must exist: importing this module raises if libcloak.so is missing (no CPU fallback).
"""
import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_int, c_uint32, c_uint64, c_void_p)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcloak.so")

CLOAK_OK, CLOAK_ERR_INVALID, CLOAK_ERR_ALIGN, CLOAK_ERR_UNSUPPORTED, CLOAK_ERR_OOM, CLOAK_ERR_CUDA = 0, -1, -2, -3, -4, -5
CLOAK_F32, CLOAK_BF16 = 0, 1
CLOAK_ROWMAJOR, CLOAK_TILE128 = 0, 1
CLOAK_POOL_IDENTITY, CLOAK_POOL_PLAIN_ALLOC = 1, 2
STATUS_NAMES = {0: "CLOAK_OK", -1: "CLOAK_ERR_INVALID", -2: "CLOAK_ERR_ALIGN", -3: "CLOAK_ERR_UNSUPPORTED",
                -4: "CLOAK_ERR_OOM", -5: "CLOAK_ERR_CUDA"}

# every symbol include/cloak.h declares
SYMBOLS = ["cloak_last_error", "cloak_version", "cloak_runtime_info", "cloak_launch_count", "cloak_keygen", "cloak_pool_create", "cloak_pool_destroy",
           "cloak_pool_info", "cloak_pool_tables", "cloak_pool_dump", "cloak_pool_map_ms", "cloak_pool_map_phases", "cloak_pool_adjacency", "cloak_pool_layout_report", "cloak_shuffle",
           "cloak_unshuffle", "cloak_shuffle_many", "cloak_unshuffle_many", "cloak_relayout", "cloak_rekey_inplace", "cloak_rekey_pages_begin", "cloak_rekey_pages_step", "cloak_rekey_pages_finish", "cloak_shuffle_host", "cloak_unshuffle_host",
           "cloak_set_copy_engine", "cloak_set_copy_cache_hint", "cloak_set_gather_engine", "cloak_arena_plan", "cloak_permute_mlp_heads", "cloak_permute_experts", "cloak_load_mlp_heads", "cloak_load_tensors", "cloak_to_tile128",
           "cloak_gemv", "cloak_gemv_chain", "cloak_gemm", "cloak_gemm_chain", "cloak_gemv_chain_scratch_bytes",
           "cloak_gemm_chain_scratch_bytes", "cloak_pool_reserve_workspace", "cloak_set_gemv_engine", "cloak_sm_weights", "cloak_set_trace", "cloak_set_gemm_schedule", "cloak_set_gemm_engine", "cloak_gemm_plan", "cloak_gemv_static", "cloak_gemv_host", "cloak_gemv_chain_host", "cloak_silu_mul"]


class CloakError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {text}")
        self.status = status


class cloak_block_shape(Structure):
    _fields_ = [("hidden", c_uint32), ("inter", c_uint32), ("n_q", c_uint32), ("n_kv", c_uint32),
                ("head_dim", c_uint32), ("dt", c_int), ("layer", c_uint32)]


class cloak_moe_shape(Structure):
    _fields_ = [("hidden", c_uint32), ("inter", c_uint32), ("n_experts", c_uint32), ("dt", c_int), ("layer", c_uint32)]


class cloak_load_item(Structure):
    _fields_ = [("src", c_void_p), ("arena_offset", c_uint64), ("layer", c_uint32), ("role", c_uint32), ("N", c_uint32), ("K", c_uint32)]


CLOAK_ROLE = {"gate": 0, "up": 1, "down": 2, "q": 3, "k": 4, "v": 5, "o": 6, "plain": 7}


class cloak_run_stats(Structure):
    _fields_ = [("items", c_uint64), ("runs", c_uint64), ("longest_run", c_uint64), ("items_in_runs_of_2_or_more", c_uint64),
                ("adjacent_fraction", c_double), ("histogram", c_uint64 * 32)]


class cloak_layout_report(Structure):
    _fields_ = [("va_blocks", cloak_run_stats), ("physical_blocks", cloak_run_stats), ("pages", cloak_run_stats)]


class cloak_tensor(Structure):
    _fields_ = [("w_offset", c_uint64), ("N", c_uint32), ("K", c_uint32), ("dt", c_int), ("layout", c_int)]


class cloak_gemv_op(Structure):
    _fields_ = [("w", cloak_tensor), ("d_x", c_void_p), ("d_y", c_void_p), ("d_gate", c_void_p), ("d_act", c_void_p),
                ("after", c_uint32)]


class cloak_gemm_op(Structure):
    _fields_ = [("w", cloak_tensor), ("d_x", c_void_p), ("d_y", c_void_p)]


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_18400_b200.build` "
                      "(there is no CPU fallback)")
lib = ctypes.CDLL(LIB_PATH)

_P = c_void_p
lib.cloak_last_error.restype = c_char_p
lib.cloak_version.restype = c_char_p
lib.cloak_runtime_info.restype = c_char_p
lib.cloak_keygen.argtypes = [c_uint64, c_uint64, c_uint32, _P, _P, _P]
lib.cloak_pool_create.argtypes = [c_int, c_uint64, c_uint32, c_uint64, c_uint64, c_uint32, POINTER(_P)]
lib.cloak_pool_destroy.argtypes = [_P]
lib.cloak_pool_info.argtypes = [_P, POINTER(_P), POINTER(_P), POINTER(c_uint32), POINTER(c_uint32),
                                POINTER(c_uint32), POINTER(c_int)]
lib.cloak_pool_tables.argtypes = [_P, _P, _P, _P, _P]
lib.cloak_pool_dump.argtypes = [_P, _P, _P]
lib.cloak_pool_map_ms.argtypes = [_P, POINTER(c_double)]
lib.cloak_pool_map_phases.argtypes = [_P, POINTER(c_double), POINTER(c_double), POINTER(c_double)]
lib.cloak_pool_adjacency.argtypes = [_P, POINTER(c_double), POINTER(c_double), POINTER(c_double), _P]
lib.cloak_pool_reserve_workspace.argtypes = [_P, c_uint64]
lib.cloak_pool_layout_report.argtypes = [_P, POINTER(cloak_layout_report), _P]
lib.cloak_shuffle.argtypes = [_P, _P, c_uint64, c_uint64, _P]
lib.cloak_unshuffle.argtypes = [_P, _P, c_uint64, c_uint64, _P]
lib.cloak_shuffle_many.argtypes = [_P, c_uint32, POINTER(c_void_p), POINTER(c_uint64), POINTER(c_uint64), _P]
lib.cloak_unshuffle_many.argtypes = [_P, c_uint32, POINTER(c_void_p), POINTER(c_uint64), POINTER(c_uint64), _P]
lib.cloak_relayout.argtypes = [_P, _P, _P]
lib.cloak_rekey_inplace.argtypes = [_P, c_uint64, c_uint64, _P]
lib.cloak_rekey_pages_begin.argtypes = [_P, c_uint64, c_uint32, _P]
lib.cloak_rekey_pages_step.argtypes = [_P, c_uint32, _P, POINTER(c_uint32)]
lib.cloak_rekey_pages_finish.argtypes = [_P, _P]
lib.cloak_shuffle_host.argtypes = [_P, _P, c_uint64, c_uint64, _P]
lib.cloak_unshuffle_host.argtypes = [_P, _P, c_uint64, c_uint64, _P]
lib.cloak_set_copy_engine.argtypes = [c_int]
lib.cloak_set_copy_cache_hint.argtypes = [c_int]
lib.cloak_set_gather_engine.argtypes = [c_int]
lib.cloak_set_gemv_engine.argtypes = [c_int]
lib.cloak_sm_weights.argtypes = [c_int, c_uint32, _P, POINTER(c_uint32)]
lib.cloak_set_trace.argtypes = [_P]
lib.cloak_set_gemm_schedule.argtypes = [c_int, c_int]
lib.cloak_set_gemm_engine.argtypes = [c_int]
lib.cloak_gemm_plan.argtypes = [c_uint32, POINTER(c_uint32), POINTER(c_uint32), c_uint32, c_uint32, c_uint32,
                                POINTER(c_uint32), POINTER(c_uint32), POINTER(c_uint32), POINTER(c_uint32), POINTER(c_uint32)]
lib.cloak_arena_plan.argtypes = [c_uint64, c_uint32, POINTER(c_uint64), c_uint32, POINTER(c_uint64), POINTER(c_uint64)]
lib.cloak_permute_mlp_heads.argtypes = [c_uint64, POINTER(cloak_block_shape)] + [_P] * 15
lib.cloak_permute_experts.argtypes = [c_uint64, POINTER(cloak_moe_shape)] + [_P] * 9
lib.cloak_load_mlp_heads.argtypes = [c_uint64, POINTER(cloak_block_shape), _P] + [_P] * 7 + [POINTER(c_uint64), _P]
lib.cloak_to_tile128.argtypes = [_P, _P, c_uint32, c_uint32, c_int, _P]
lib.cloak_load_tensors.argtypes = [c_uint64, POINTER(cloak_block_shape), _P, POINTER(cloak_load_item), c_uint32, c_int, _P]
lib.cloak_gemv.argtypes = [_P, POINTER(cloak_tensor), _P, _P, c_uint32, _P]
lib.cloak_gemv_static.argtypes = [_P, POINTER(cloak_tensor), _P, _P, c_uint32, _P]
lib.cloak_gemv_chain.argtypes = [_P, POINTER(cloak_gemv_op), c_uint32, c_uint32, _P]
lib.cloak_gemm_chain.argtypes = [_P, POINTER(cloak_gemm_op), c_uint32, c_uint32, _P]
lib.cloak_gemv_chain_scratch_bytes.argtypes = [_P, POINTER(cloak_gemv_op), c_uint32, c_uint32, POINTER(c_uint64)]
lib.cloak_gemm_chain_scratch_bytes.argtypes = [_P, POINTER(cloak_gemm_op), c_uint32, c_uint32, POINTER(c_uint64)]
lib.cloak_gemm.argtypes = [_P, POINTER(cloak_tensor), _P, _P, c_uint32, _P]
lib.cloak_gemv_host.argtypes = [_P, POINTER(cloak_tensor), _P, _P, c_uint32, _P]
lib.cloak_gemv_chain_host.argtypes = [_P, POINTER(cloak_gemv_op), c_uint32, c_uint32, _P]
lib.cloak_silu_mul.argtypes = [_P, _P, _P, c_uint64, c_int, _P]
lib.cloak_launch_count.restype = c_uint64
for _n in SYMBOLS[4:]:
    getattr(lib, _n).restype = c_int


def _ptr(x):
    """Address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream(s):
    if s is None:
        try:
            import torch
            if torch.cuda.is_available() and torch.cuda.is_initialized():
                return torch.cuda.current_stream().cuda_stream
        except ImportError:
            pass
        return None
    if isinstance(s, int):
        return s
    return s.cuda_stream


def _check(status):
    if status != CLOAK_OK:
        raise CloakError(status, lib.cloak_last_error().decode())


def cloak_last_error():
    return lib.cloak_last_error().decode()


def cloak_version():
    return lib.cloak_version().decode()


def cloak_runtime_info():
    return lib.cloak_runtime_info().decode()


def cloak_launch_count():
    return int(lib.cloak_launch_count())


def cloak_keygen(key, stream_id, n, d_perm, d_inv, stream=None):
    _check(lib.cloak_keygen(key, stream_id, n, _ptr(d_perm), _ptr(d_inv), _stream(stream)))


def cloak_pool_create(device, payload_bytes, block_bytes, page_bytes, key, flags=0):
    out = _P()
    _check(lib.cloak_pool_create(device, payload_bytes, block_bytes, page_bytes, key, flags, byref(out)))
    return out


def cloak_pool_destroy(pool):
    _check(lib.cloak_pool_destroy(pool))


def cloak_pool_info(pool):
    base, tab = _P(), _P()
    nb, nslots, npages, vmm = c_uint32(), c_uint32(), c_uint32(), c_int()
    _check(lib.cloak_pool_info(pool, byref(base), byref(tab), byref(nb), byref(nslots), byref(npages), byref(vmm)))
    return dict(d_base=base.value, d_table=tab.value, nb=nb.value, nslots=nslots.value, npages=npages.value,
                is_vmm=bool(vmm.value))


def cloak_pool_tables(pool, h_blockperm=None, h_blockinv=None, h_pageperm=None, h_pageinv=None):
    _check(lib.cloak_pool_tables(pool, _ptr(h_blockperm), _ptr(h_blockinv), _ptr(h_pageperm), _ptr(h_pageinv)))


def cloak_pool_dump(pool, d_out, stream=None):
    _check(lib.cloak_pool_dump(pool, _ptr(d_out), _stream(stream)))


def cloak_pool_map_ms(pool):
    ms = c_double()
    _check(lib.cloak_pool_map_ms(pool, byref(ms)))
    return ms.value


def cloak_pool_map_phases(pool):
    a, b, c = c_double(), c_double(), c_double()
    _check(lib.cloak_pool_map_phases(pool, byref(a), byref(b), byref(c)))
    return dict(create_ms=a.value, map_ms=b.value, set_access_ms=c.value)


def cloak_pool_adjacency(pool, stream=None):
    va, ph, pg = c_double(), c_double(), c_double()
    _check(lib.cloak_pool_adjacency(pool, byref(va), byref(ph), byref(pg), _stream(stream)))
    return dict(va_blocks=va.value, physical_blocks=ph.value, pages=pg.value)


def cloak_pool_layout_report(pool, stream=None):
    """{view: {items, runs, longest_run, items_in_runs_of_2_or_more, adjacent_fraction, histogram: {"2^k": count}}}"""
    rep = cloak_layout_report()
    _check(lib.cloak_pool_layout_report(pool, byref(rep), _stream(stream)))
    out = {}
    for name in ("va_blocks", "physical_blocks", "pages"):
        r = getattr(rep, name)
        out[name] = dict(items=r.items, runs=r.runs, longest_run=r.longest_run, items_in_runs_of_2_or_more=r.items_in_runs_of_2_or_more,
                         adjacent_fraction=r.adjacent_fraction, histogram={f"2^{k}": r.histogram[k] for k in range(32) if r.histogram[k]})
    return out


def cloak_pool_reserve_workspace(pool, nbytes):
    _check(lib.cloak_pool_reserve_workspace(pool, nbytes))


def cloak_shuffle(pool, d_logical, logical_offset, nbytes, stream=None):
    _check(lib.cloak_shuffle(pool, _ptr(d_logical), logical_offset, nbytes, _stream(stream)))


def cloak_unshuffle(pool, d_logical, logical_offset, nbytes, stream=None):
    _check(lib.cloak_unshuffle(pool, _ptr(d_logical), logical_offset, nbytes, _stream(stream)))


def _many(tensors, offsets, nbytes):
    n = len(tensors)
    ptrs = (c_void_p * n)(*[_ptr(t) for t in tensors])
    return n, ptrs, (c_uint64 * n)(*offsets), (c_uint64 * n)(*nbytes)


def cloak_shuffle_many(pool, tensors, offsets, nbytes, stream=None):
    _check(lib.cloak_shuffle_many(pool, *_many(tensors, offsets, nbytes), _stream(stream)))


def cloak_unshuffle_many(pool, tensors, offsets, nbytes, stream=None):
    _check(lib.cloak_unshuffle_many(pool, *_many(tensors, offsets, nbytes), _stream(stream)))


def cloak_relayout(from_a, to_b, stream=None):
    _check(lib.cloak_relayout(from_a, to_b, _stream(stream)))


def cloak_rekey_inplace(pool, new_key, spare_bytes=0, stream=None):
    _check(lib.cloak_rekey_inplace(pool, new_key, spare_bytes, _stream(stream)))


def cloak_rekey_pages_begin(pool, new_key, spare_pages=1, stream=None):
    _check(lib.cloak_rekey_pages_begin(pool, new_key, spare_pages, _stream(stream)))


def cloak_rekey_pages_step(pool, max_moves, stream=None):
    """Returns the number of pages not yet home (0 = the re-key is complete)."""
    left = c_uint32()
    _check(lib.cloak_rekey_pages_step(pool, max_moves, _stream(stream), byref(left)))
    return left.value


def cloak_rekey_pages_finish(pool, stream=None):
    _check(lib.cloak_rekey_pages_finish(pool, _stream(stream)))


def cloak_shuffle_host(pool, h_logical, logical_offset, nbytes, stream=None):
    _check(lib.cloak_shuffle_host(pool, _ptr(h_logical), logical_offset, nbytes, _stream(stream)))


def cloak_unshuffle_host(pool, h_logical, logical_offset, nbytes, stream=None):
    _check(lib.cloak_unshuffle_host(pool, _ptr(h_logical), logical_offset, nbytes, _stream(stream)))


def cloak_set_copy_engine(engine):
    _check(lib.cloak_set_copy_engine(engine))


def cloak_set_copy_cache_hint(hint):
    _check(lib.cloak_set_copy_cache_hint(hint))


def cloak_set_gather_engine(engine):
    _check(lib.cloak_set_gather_engine(engine))


def cloak_set_gemv_engine(engine):
    _check(lib.cloak_set_gemv_engine(engine))


def cloak_sm_weights(device=0):
    """Relative streaming speeds of the device's SMs (mean 1), indexed by SM id; [] if they could not be measured."""
    n = c_uint32()
    _check(lib.cloak_sm_weights(device, 0, None, byref(n)))
    if n.value == 0:
        return []
    w = (ctypes.c_float * n.value)()
    _check(lib.cloak_sm_weights(device, n.value, w, byref(n)))
    return list(w)


def cloak_set_trace(d_trace):
    _check(lib.cloak_set_trace(_ptr(d_trace)))


def cloak_set_gemm_schedule(static_pct, dyn_chunk_tiles=0):
    _check(lib.cloak_set_gemm_schedule(static_pct, dyn_chunk_tiles))


def cloak_set_gemm_engine(engine):
    _check(lib.cloak_set_gemm_engine(engine))


def cloak_gemm_plan(shapes, batch, sms=148):
    """Host only: (chunks, n_static, group) -- chunks[c] = (begin, end) in the launch's unit sequence, a unit spanning `group`
    tile rows -- for ops of shapes [(N, K)]."""
    n = len(shapes)
    Ns = (c_uint32 * n)(*[s[0] for s in shapes])
    Ks = (c_uint32 * n)(*[s[1] for s in shapes])
    nch, nst, grp = c_uint32(0), c_uint32(0), c_uint32(0)
    _check(lib.cloak_gemm_plan(n, Ns, Ks, batch, sms, 0, None, None, ctypes.byref(nch), ctypes.byref(nst), ctypes.byref(grp)))
    b, e = (c_uint32 * max(nch.value, 1))(), (c_uint32 * max(nch.value, 1))()
    _check(lib.cloak_gemm_plan(n, Ns, Ks, batch, sms, nch.value, b, e, ctypes.byref(nch), ctypes.byref(nst), ctypes.byref(grp)))
    return [(b[i], e[i]) for i in range(nch.value)], nst.value, grp.value


def cloak_arena_plan(key, sizes, block_bytes):
    T = len(sizes)
    arr = (c_uint64 * max(T, 1))(*sizes)
    offs = (c_uint64 * max(T, 1))()
    total = c_uint64()
    _check(lib.cloak_arena_plan(key, T, arr, block_bytes, offs, byref(total)))
    return list(offs)[:T], total.value


def cloak_permute_mlp_heads(key, shape, gate=None, up=None, down=None, q=None, k=None, v=None, o=None,
                            gate_o=None, up_o=None, down_o=None, q_o=None, k_o=None, v_o=None, o_o=None,
                            stream=None):
    ptrs = [_ptr(t) for t in (gate, up, down, q, k, v, o, gate_o, up_o, down_o, q_o, k_o, v_o, o_o)]
    _check(lib.cloak_permute_mlp_heads(key, byref(shape), *ptrs, _stream(stream)))


def cloak_permute_experts(key, shape, router, gate, up, down, router_o, gate_o, up_o, down_o, stream=None):
    ptrs = [_ptr(t) for t in (router, gate, up, down, router_o, gate_o, up_o, down_o)]
    _check(lib.cloak_permute_experts(key, byref(shape), *ptrs, _stream(stream)))


def cloak_load_mlp_heads(key, shape, pool, offsets, gate=None, up=None, down=None, q=None, k=None, v=None, o=None,
                         stream=None):
    """offsets: dict name -> arena offset, or a sequence of 7 in the order gate, up, down, q, k, v, o."""
    names = ("gate", "up", "down", "q", "k", "v", "o")
    if isinstance(offsets, dict):
        offsets = [offsets.get(n, 0) for n in names]
    arr = (c_uint64 * 7)(*offsets)
    ptrs = [_ptr(t) for t in (gate, up, down, q, k, v, o)]
    _check(lib.cloak_load_mlp_heads(key, byref(shape), pool, *ptrs, arr, _stream(stream)))


def cloak_load_items(items):
    """Marshals [(src, arena_offset, layer, role name or number[, N, K]), ...] into a ctypes array for cloak_load_tensors."""
    arr = (cloak_load_item * len(items))()
    for o, it in zip(arr, items):
        src, off, layer, role = it[:4]
        N, K = it[4:] if len(it) == 6 else (0, 0)
        o.src, o.arena_offset, o.layer, o.role, o.N, o.K = _ptr(src), off, layer, CLOAK_ROLE.get(role, role), N, K
    return arr


def cloak_load_tensors(key, shape, pool, items, layout=CLOAK_ROWMAJOR, stream=None):
    arr = items if isinstance(items, ctypes.Array) else cloak_load_items(items)
    _check(lib.cloak_load_tensors(key, byref(shape), pool, arr, len(arr), layout, _stream(stream)))


def cloak_to_tile128(d_src, d_dst, N, K, dt, stream=None):
    _check(lib.cloak_to_tile128(_ptr(d_src), _ptr(d_dst), N, K, dt, _stream(stream)))


def cloak_gemv(pool, tensor, d_x, d_y, batch, stream=None):
    _check(lib.cloak_gemv(pool, byref(tensor), _ptr(d_x), _ptr(d_y), batch, _stream(stream)))


def cloak_gemv_static(pool, tensor, d_x, d_y, batch, stream=None):
    """cloak_gemv with its scratch in the library's fixed device array: allocates nothing (see cloak.h for the limits)."""
    _check(lib.cloak_gemv_static(pool, byref(tensor), _ptr(d_x), _ptr(d_y), batch, _stream(stream)))


def cloak_gemv_ops(ops):
    """Marshals [(tensor, d_x, d_y, after) or (tensor, d_x, d_y, after, d_gate, d_act), ...] into a ctypes array
    for cloak_gemv_chain (reusable across calls)."""
    arr = (cloak_gemv_op * len(ops))()
    for o, op in zip(arr, ops):
        t, x, y, after = op[:4]
        gate, act = op[4:] if len(op) == 6 else (None, None)
        o.w, o.d_x, o.d_y, o.d_gate, o.d_act, o.after = t, _ptr(x), _ptr(y), _ptr(gate), _ptr(act), int(after)
    return arr


def cloak_gemv_chain(pool, ops, batch, stream=None):
    arr = ops if isinstance(ops, ctypes.Array) else cloak_gemv_ops(ops)
    _check(lib.cloak_gemv_chain(pool, arr, len(arr), batch, _stream(stream)))


def cloak_gemv_chain_scratch_bytes(pool, ops, batch):
    arr = ops if isinstance(ops, ctypes.Array) else cloak_gemv_ops(ops)
    n = c_uint64()
    _check(lib.cloak_gemv_chain_scratch_bytes(pool, arr, len(arr), batch, byref(n)))
    return n.value


def cloak_gemm_chain_scratch_bytes(pool, ops, batch):
    arr = ops if isinstance(ops, ctypes.Array) else cloak_gemm_ops(ops)
    n = c_uint64()
    _check(lib.cloak_gemm_chain_scratch_bytes(pool, arr, len(arr), batch, byref(n)))
    return n.value


def cloak_gemm(pool, tensor, d_x, d_y, batch, stream=None):
    _check(lib.cloak_gemm(pool, byref(tensor), _ptr(d_x), _ptr(d_y), batch, _stream(stream)))


def cloak_gemm_ops(ops):
    """Marshals [(tensor, d_x, d_y), ...] into a ctypes array for cloak_gemm_chain (reusable across calls)."""
    arr = (cloak_gemm_op * len(ops))()
    for o, (t, x, y) in zip(arr, ops):
        o.w, o.d_x, o.d_y = t, _ptr(x), _ptr(y)
    return arr


def cloak_gemm_chain(pool, ops, batch, stream=None):
    arr = ops if isinstance(ops, ctypes.Array) else cloak_gemm_ops(ops)
    _check(lib.cloak_gemm_chain(pool, arr, len(arr), batch, _stream(stream)))


def cloak_gemv_host(pool, tensor, h_x, h_y, batch, stream=None):
    _check(lib.cloak_gemv_host(pool, byref(tensor), _ptr(h_x), _ptr(h_y), batch, _stream(stream)))


def cloak_gemv_chain_host(pool, ops, batch, stream=None):
    """ops as for cloak_gemv_chain, with HOST x / y buffers (numpy arrays or pinned torch tensors)."""
    arr = ops if isinstance(ops, ctypes.Array) else cloak_gemv_ops(ops)
    _check(lib.cloak_gemv_chain_host(pool, arr, len(arr), batch, _stream(stream)))


def cloak_silu_mul(d_g, d_u, d_out, n, dt, stream=None):
    _check(lib.cloak_silu_mul(_ptr(d_g), _ptr(d_u), _ptr(d_out), n, dt, _stream(stream)))
