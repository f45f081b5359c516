"""ctypes binding of synth/libcloaksynth.so (the CUDA twin of synth/gen.py).  Harness, not method."""
import ctypes
import os

_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libcloaksynth.so")
if not os.path.exists(_PATH):
    raise ImportError(f"{_PATH} is missing: build it with `python -m paper_2606_18400_b200.build`")
_lib = ctypes.CDLL(_PATH)
_lib.synth_fill.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64,
                            ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
_lib.synth_fill.restype = ctypes.c_int


def fill(tensor_out, seed, tensor_id, kind=0, start=0, stream=None):
    """Fill a contiguous torch CUDA tensor (float32 or bfloat16) with elements [start, start+numel)."""
    import torch
    assert tensor_out.is_cuda and tensor_out.is_contiguous()
    bf16 = {torch.float32: 0, torch.bfloat16: 1}[tensor_out.dtype]
    s = torch.cuda.current_stream().cuda_stream if stream is None else stream
    err = _lib.synth_fill(tensor_out.data_ptr(), seed, tensor_id, start, tensor_out.numel(), kind, bf16, s)
    if err:
        raise RuntimeError(f"synth_fill: cudaError {err}")
    return tensor_out
