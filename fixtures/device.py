"""Device-side input generator (fixture): ctypes wrapper over fixtures/gen_device.cu.

Same values as fixtures/generator.py, produced directly in HBM.  Build: python -m fixtures.device
"""
import ctypes
import os
import subprocess
import sys

from . import generator as gen

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gen_device.cu")
SRC_MEMBENCH = os.path.join(HERE, "membench.cu")
LIB = os.path.join(HERE, "libhadpsgd_fixture.so")
_lib = None


def build(force=False):
    newest = max(os.path.getmtime(SRC), os.path.getmtime(SRC_MEMBENCH))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--ftz=false",
                    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-o", LIB, SRC, SRC_MEMBENCH], check=True)
    return LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.hadpsgd_fixture_fill.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_uint64,
                                           ctypes.c_float, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
        L.hadpsgd_fixture_membench.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_int,
                                               ctypes.c_void_p, ctypes.c_void_p]
        _lib = L
    return _lib


def membench(total_bytes=8 << 30, n_streams=12, write=False, reps=5):
    """This device's streaming rate in GB/s (best of `reps`), read or write, n_streams buffers walked in
    lock step with the step kernel's access shape (fixtures/membench.cu)."""
    import torch
    stream_bytes = total_bytes // n_streams // 8192 * 8192
    buf = torch.empty(stream_bytes * n_streams + 256, dtype=torch.uint8, device="cuda")
    if not write:
        buf.random_(0, 255)
    sink = buf[stream_bytes * n_streams:]
    st = torch.cuda.current_stream().cuda_stream
    best = 0.0
    for i in range(reps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        rc = lib().hadpsgd_fixture_membench(buf.data_ptr(), stream_bytes, n_streams, 1 if write else 0, sink.data_ptr(), st)
        if rc != 0:
            raise RuntimeError(f"membench launch failed: cudaError {rc}")
        e1.record()
        torch.cuda.synchronize()
        if i:                                   # the first pass is a warm-up
            best = max(best, stream_bytes * n_streams / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    del buf
    return best


def fill(tensor, key, dist="normal", scale=1e-3, elem_offset=0, n=None, stream=None):
    """Fill a contiguous CUDA tensor (float32 or bfloat16) with value(elem_offset + i)."""
    import torch
    assert tensor.is_cuda and tensor.is_contiguous()
    bf16 = tensor.dtype == torch.bfloat16
    assert bf16 or tensor.dtype == torch.float32
    n = tensor.numel() if n is None else n
    sc = gen.normal_scale(scale) if dist == "normal" else gen.uniform_scale(scale)
    st = (stream or torch.cuda.current_stream(tensor.device)).cuda_stream
    rc = lib().hadpsgd_fixture_fill(tensor.data_ptr(), n, elem_offset, key, float(sc), 1 if dist == "normal" else 0,
                                    1 if bf16 else 0, st)
    if rc != 0:
        raise RuntimeError(f"fixture fill launch failed: cudaError {rc}")


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
