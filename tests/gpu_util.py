"""Helpers for the GPU parity tests: torch <-> numpy plumbing, pool wrappers.  No method arithmetic."""
import numpy as np
import torch

import paper_2606_18400_b200 as C


def dev_bytes(n):
    return torch.zeros(n, dtype=torch.uint8, device="cuda")


def to_dev_bytes(a):
    """numpy array of any dtype -> uint8 CUDA tensor with the same bytes."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1).copy()).cuda()


def to_host_bytes(t):
    return t.detach().contiguous().view(torch.uint8).reshape(-1).cpu().numpy()


def bf16_dev_from_bits(bits):
    """uint16 numpy array of bf16 bit patterns -> torch.bfloat16 CUDA tensor of the same shape."""
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16).copy()).cuda().view(torch.bfloat16)


def bits_from_bf16_dev(t):
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


class Pool:
    """RAII wrapper around cloak_pool_* for tests."""

    def __init__(self, payload, block, page, key, flags=0, device=0):
        self.h = C.cloak_pool_create(device, payload, block, page, key, flags)
        self.payload, self.block, self.page = payload, block, page
        self.info = C.cloak_pool_info(self.h)

    def tables(self):
        i = self.info
        bp, bi = np.empty(i["nslots"], np.uint32), np.empty(i["nslots"], np.uint32)
        pp, pi = np.empty(i["npages"], np.uint32), np.empty(i["npages"], np.uint32)
        C.cloak_pool_tables(self.h, bp, bi, pp, pi)
        return bp, bi, pp, pi

    def table_T(self):
        """The authorised table T[0..nb) read back from the device."""
        out = torch.empty(self.info["nb"], dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        ctypes_cudart_copy(out.data_ptr(), self.info["d_table"], 4 * self.info["nb"])
        return out.cpu().numpy().view(np.uint32)

    def raw(self):
        """The pool's memory as seen through its base pointer (V for vmm, D for emulated)."""
        n = self.info["nslots"] * self.block
        out = dev_bytes(n)
        torch.cuda.synchronize()
        ctypes_cudart_copy(out.data_ptr(), self.info["d_base"], n)
        return out.cpu().numpy()

    def dump(self):
        out = dev_bytes(self.info["nslots"] * self.block)
        C.cloak_pool_dump(self.h, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def close(self):
        if self.h is not None:
            torch.cuda.synchronize()
            C.cloak_pool_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


_cudart = None


def ctypes_cudart_copy(dst, src, n):
    """cudaMemcpy(dst, src, n, cudaMemcpyDefault) through torch's own libcudart."""
    import ctypes
    global _cudart
    if _cudart is None:
        import glob
        import os
        cands = glob.glob(os.path.join(os.path.dirname(torch.__file__), "lib", "libcudart*.so*"))
        cands += glob.glob("/usr/local/cuda/lib64/libcudart.so*")
        try:
            import nvidia.cuda_runtime
            cands = glob.glob(os.path.join(os.path.dirname(nvidia.cuda_runtime.__file__), "lib", "libcudart.so*")) + cands
        except ImportError:
            pass
        _cudart = ctypes.CDLL(cands[0])
        _cudart.cudaMemcpy.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int]
    rc = _cudart.cudaMemcpy(dst, src, n, 4)
    assert rc == 0, f"cudaMemcpy failed: {rc}"
