"""Thin ctypes binding over libhadpsgd.so -- same names as include/hadpsgd.h.

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the
C ABI.  There is no CPU fallback: if the shared library is missing or the device is not an
sm_100a GPU, calls raise.
"""
import ctypes
import os

import numpy as np

F32, BF16 = 0, 1
OK, INVALID_ARG, OUT_OF_MEMORY, CUDA_ERROR, UNSUPPORTED_DEVICE, DIAG_TIMEOUT = 0, -1, -2, -3, -4, -5
DETERMINISTIC, NO_MIX, NO_DIAG, EQ7_LITERAL, SHARE_PAIR_WEIGHTS, PEER = 1, 2, 4, 8, 16, 32
SEG_ALIGN_ELEMS = 64
MAX_S = 512

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhadpsgd.so")


class hadpsgd_dtypes(ctypes.Structure):
    _fields_ = [("grad_dtype", ctypes.c_int32), ("master_dtype", ctypes.c_int32), ("working_dtype", ctypes.c_int32),
                ("peer_stage", ctypes.c_int32)]


class hadpsgd_opts(ctypes.Structure):
    _fields_ = [("arena", ctypes.c_void_p), ("arena_bytes", ctypes.c_size_t), ("stream", ctypes.c_void_p),
                ("flags", ctypes.c_uint32), ("device", ctypes.c_int32)]


class hadpsgd_diag(ctypes.Structure):
    _fields_ = [("S", ctypes.c_int32), ("n_pairs", ctypes.c_int32), ("step_k", ctypes.c_uint64),
                ("gsq", ctypes.c_double * MAX_S), ("wsq", ctypes.c_double * MAX_S), ("gap", ctypes.c_double * MAX_S),
                ("pend_wsq", ctypes.c_double * MAX_S), ("pend_gap", ctypes.c_double * MAX_S),
                ("pending", ctypes.c_int32 * MAX_S)]


class HadpsgdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"hadpsgd status {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libhadpsgd.so (built in-tree by paper_1907_05701_b200.build).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1907_05701_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        i32, i64p, vp, sz_p = ctypes.c_int, ctypes.POINTER(ctypes.c_int64), ctypes.c_void_p, ctypes.POINTER(ctypes.c_size_t)
        f32, u64 = ctypes.c_float, ctypes.c_uint64
        L.hadpsgd_required_bytes.argtypes = [i32, i32, i64p, i32, hadpsgd_dtypes, sz_p]
        L.hadpsgd_layout.argtypes = [i32, i32, i64p, i32, hadpsgd_dtypes, i64p, i64p, sz_p, sz_p, sz_p, sz_p]
        L.hadpsgd_pairing.argtypes = [i32, u64, ctypes.POINTER(ctypes.c_int32)]
        L.hadpsgd_shard_range.argtypes = [ctypes.c_int64, i32, i32, i64p, i64p]
        L.hadpsgd_lr_schedule.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_double, i32, i32,
                                          ctypes.POINTER(ctypes.c_double)]
        L.hadpsgd_create.argtypes = [i32, i32, i64p, i32, hadpsgd_dtypes, ctypes.POINTER(hadpsgd_opts), ctypes.POINTER(vp)]
        L.hadpsgd_destroy.argtypes = [vp]
        L.hadpsgd_step.argtypes = [vp, f32, f32, u64]
        L.hadpsgd_step_matching.argtypes = [vp, f32, f32, u64, ctypes.POINTER(ctypes.c_int32)]
        L.hadpsgd_step_host.argtypes = [vp, ctypes.POINTER(vp), f32, f32, u64, ctypes.POINTER(hadpsgd_diag)]
        L.hadpsgd_weights.argtypes = [vp, i32, ctypes.POINTER(vp)]
        L.hadpsgd_momentum.argtypes = [vp, i32, ctypes.POINTER(vp)]
        L.hadpsgd_grads.argtypes = [vp, i32, i32, ctypes.POINTER(vp)]
        L.hadpsgd_weights_bf16.argtypes = [vp, i32, ctypes.POINTER(vp)]
        L.hadpsgd_segment.argtypes = [vp, i32, i64p, i64p]
        L.hadpsgd_padded_len.argtypes = [vp, i64p]
        L.hadpsgd_diagnostics.argtypes = [vp, ctypes.POINTER(hadpsgd_diag)]
        i32p = ctypes.POINTER(ctypes.c_int32)
        L.hadpsgd_unshare.argtypes = [vp]
        L.hadpsgd_plan_slots.argtypes = [i32, i32p, i32, i32p, i32p, i32p, i32p, i32p, i32p]
        L.hadpsgd_consensus.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
        L.hadpsgd_consensus_noalloc.argtypes = [ctypes.POINTER(vp), i32, ctypes.c_int64, vp, vp]
        L.hadpsgd_consensus_noalloc_error.argtypes = []
        L.hadpsgd_consensus_noalloc_error.restype = ctypes.c_char_p
        L.hadpsgd_peer_init.argtypes = [vp, i32, i32, i32p]
        L.hadpsgd_peer_stage.argtypes = [vp, ctypes.POINTER(vp)]
        L.hadpsgd_peer_attach.argtypes = [vp, i32, vp]
        L.hadpsgd_peer_ipc_export.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_uint64)]
        L.hadpsgd_peer_ipc_attach.argtypes = [vp, i32, vp, ctypes.c_uint64]
        L.hadpsgd_peer_flush.argtypes = [vp]
        L.hadpsgd_plan_peer.argtypes = [i32, i32, i32p, i32p, u64, i32p, i32p, i32p, i32p, i32p, i32p]
        L.hadpsgd_set_launch.argtypes = [vp, i32]
        L.hadpsgd_set_diagnostics.argtypes = [vp, i32]
        L.hadpsgd_launch_count.argtypes = [vp, ctypes.POINTER(u64)]
        L.hadpsgd_error_string.argtypes = [i32]
        L.hadpsgd_error_string.restype = ctypes.c_char_p
        L.hadpsgd_last_error.argtypes = [vp]
        L.hadpsgd_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _seg(seg_len):
    arr = (ctypes.c_int64 * len(seg_len))(*[int(x) for x in seg_len])
    return arr, len(seg_len)


def _check(rc, h=None):
    if rc != OK:
        L = lib()
        detail = L.hadpsgd_last_error(h).decode() if True else ""
        raise HadpsgdError(rc, f"{L.hadpsgd_error_string(rc).decode()}: {detail}")


def hadpsgd_required_bytes(S, G, seg_len, grad_dtype=F32, working_dtype=F32, peer_stage=0):
    arr, n = _seg(seg_len)
    out = ctypes.c_size_t(0)
    _check(lib().hadpsgd_required_bytes(S, G, arr, n, hadpsgd_dtypes(grad_dtype, F32, working_dtype, peer_stage),
                                        ctypes.byref(out)))
    return out.value


def hadpsgd_layout(S, G, seg_len, grad_dtype=F32, working_dtype=F32, peer_stage=0):
    arr, n = _seg(seg_len)
    seg_off = (ctypes.c_int64 * n)()
    P = ctypes.c_int64(0)
    w, v, g, wb = ctypes.c_size_t(0), ctypes.c_size_t(0), ctypes.c_size_t(0), ctypes.c_size_t(0)
    _check(lib().hadpsgd_layout(S, G, arr, n, hadpsgd_dtypes(grad_dtype, F32, working_dtype, peer_stage), seg_off, ctypes.byref(P),
                                ctypes.byref(w), ctypes.byref(v), ctypes.byref(g), ctypes.byref(wb)))
    return dict(seg_offset=list(seg_off), P_padded=P.value, w_off=w.value, v_off=v.value, g_off=g.value,
                wb_off=wb.value)


def hadpsgd_pairing(S, step_k):
    out = (ctypes.c_int32 * max(S, 1))()
    _check(lib().hadpsgd_pairing(S, step_k, out))
    return list(out)[:S]


def hadpsgd_shard_range(P_padded, world, rank):
    lo, hi = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(lib().hadpsgd_shard_range(P_padded, world, rank, ctypes.byref(lo), ctypes.byref(hi)))
    return lo.value, hi.value


def hadpsgd_lr_schedule(base_lr, base_batch, total_batch, warmup_epochs, epoch):
    out = ctypes.c_double(0.0)
    _check(lib().hadpsgd_lr_schedule(base_lr, base_batch, total_batch, warmup_epochs, epoch, ctypes.byref(out)))
    return out.value


def hadpsgd_plan_slots(partner, w_slot, share=True):
    """Pure host function: (w_slot_after, read_slot, write_slot, copies[(src, dst)...]) of one step."""
    S = len(partner)
    arr = lambda v: (ctypes.c_int32 * S)(*[int(x) for x in v])
    pt, ws, rd, wr, cs, cd = arr(partner), arr(w_slot), arr([0] * S), arr([0] * S), arr([0] * S), arr([0] * S)
    n = ctypes.c_int32(0)
    _check(lib().hadpsgd_plan_slots(S, pt, 1 if share else 0, ws, rd, wr, cs, cd, ctypes.byref(n)))
    return list(ws), list(rd), list(wr), [(cs[i], cd[i]) for i in range(n.value)]


def hadpsgd_plan_peer(world, rank, rank_begin, partner, epoch, pending):
    """Pure host function: the peer plan of one step for `rank` (see include/hadpsgd.h).  Returns a dict
    of lists indexed by the LOCAL member: pending (after the step), kind, mate, read_buf, write_buf,
    read_peer."""
    ok = 0 <= rank < world and len(rank_begin) == world + 1
    S_l = max(rank_begin[rank + 1] - rank_begin[rank], 1) if ok else 1      # the library rejects bad ranks
    if len(rank_begin) != world + 1:
        raise HadpsgdError(INVALID_ARG, "rank_begin must have world + 1 entries")
    i32a = lambda v: (ctypes.c_int32 * len(v))(*[int(x) for x in v])
    rb, pt, pend = i32a(rank_begin), i32a(partner), i32a(pending)
    outs = [i32a([0] * S_l) for _ in range(5)]
    _check(lib().hadpsgd_plan_peer(world, rank, rb, pt, epoch, pend, *outs))
    names = ("kind", "mate", "read_buf", "write_buf", "read_peer")
    d = {n: list(o) for n, o in zip(names, outs)}
    d["pending"] = list(pend)
    return d


def hadpsgd_consensus_noalloc(weight_ptrs, n, out_ptr, stream_ptr=0):
    """Consensus distance of S borrowed weight buffers, for callers that cannot let the library allocate
    (a framework allocator that already holds the GPU, a monitor that must not stall the device with
    cudaMalloc, a hook without an arena): see include/hadpsgd.h.  weight_ptrs: S device addresses of n
    floats each; out_ptr: device address of one double, written in stream order; stream_ptr: a
    cudaStream_t as int.  Marshalling only -- nothing is allocated here either.  Calls that may overlap
    on the GPU share one scratch array and race; the first call on a device must be outside capture."""
    S = len(weight_ptrs)
    arr = (ctypes.c_void_p * max(S, 1))(*[int(p) for p in weight_ptrs])
    L = lib()
    rc = L.hadpsgd_consensus_noalloc(arr, S, int(n), ctypes.c_void_p(int(out_ptr)), ctypes.c_void_p(int(stream_ptr)))
    if rc != OK:
        raise HadpsgdError(rc, f"{L.hadpsgd_error_string(rc).decode()}: {L.hadpsgd_consensus_noalloc_error().decode()}")


class Hadpsgd:
    """Handle wrapper.  Device memory is a torch uint8 tensor (the arena) so that torch owns
    allocation and stream plumbing; everything else happens behind the C ABI."""

    def __init__(self, S, G, seg_len, grad_dtype=F32, flags=0, device=0, stream=None, own_arena=False,
                 working_dtype=F32):
        peer_stage = 1 if flags & PEER else 0
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("hadpsgd needs a CUDA device (sm_100a); there is no CPU fallback")
        self.S, self.G, self.seg_len = int(S), int(G), [int(x) for x in seg_len]
        self.grad_dtype, self.flags, self.working_dtype = grad_dtype, flags, working_dtype
        self.torch = torch
        self.device = torch.device("cuda", device)
        arr, n = _seg(self.seg_len)
        nbytes = hadpsgd_required_bytes(S, G, self.seg_len, grad_dtype, working_dtype, peer_stage)
        self.layout = hadpsgd_layout(S, G, self.seg_len, grad_dtype, working_dtype, peer_stage)
        self.P_padded = self.layout["P_padded"]
        opts = hadpsgd_opts()
        opts.flags, opts.device = flags, device
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        opts.stream = self.stream.cuda_stream
        if own_arena:
            self.arena = None
            opts.arena, opts.arena_bytes = None, 0
        else:
            self.arena = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            opts.arena, opts.arena_bytes = self.arena.data_ptr(), nbytes
        self.arena_bytes = nbytes
        h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib().hadpsgd_create(S, G, arr, n, hadpsgd_dtypes(grad_dtype, F32, working_dtype, peer_stage), ctypes.byref(opts),
                                        ctypes.byref(h)))
        self.h = h

    # -- the three core calls ------------------------------------------------------------
    def hadpsgd_step(self, lr, momentum, step_k):
        _check(lib().hadpsgd_step(self.h, lr, momentum, step_k), self.h)

    def hadpsgd_step_matching(self, lr, momentum, step_k, partner):
        arr = (ctypes.c_int32 * len(partner))(*[int(p) for p in partner])   # S entries (S_global in peer mode)
        _check(lib().hadpsgd_step_matching(self.h, lr, momentum, step_k, arr), self.h)

    def hadpsgd_step_host(self, host_grad_ptrs, lr, momentum, step_k, want_diag=True):
        """host_grad_ptrs: S*G host addresses (ints), each P_padded grad elements (pinned)."""
        arr = (ctypes.c_void_p * (self.S * self.G))(*host_grad_ptrs)
        d = hadpsgd_diag() if want_diag else None
        _check(lib().hadpsgd_step_host(self.h, arr, lr, momentum, step_k, ctypes.byref(d) if want_diag else None), self.h)
        return self._diag_dict(d) if want_diag else None

    def _view(self, ptr, n, dtype):
        # borrowed view into the arena (or library-owned memory) as a torch tensor
        torch = self.torch
        esz = torch.empty(0, dtype=dtype).element_size()
        if self.arena is not None:
            off = ptr - self.arena.data_ptr()
            return self.arena[off:off + n * esz].view(dtype)

        class _Borrowed:      # library-owned memory: wrap the device pointer, no copy, no ownership
            __cuda_array_interface__ = {"shape": (n * esz,), "typestr": "|u1", "data": (ptr, False), "version": 2}
        with torch.cuda.device(self.device):
            return torch.as_tensor(_Borrowed(), device=self.device).view(dtype)

    def hadpsgd_weights(self, s):
        p = ctypes.c_void_p()
        _check(lib().hadpsgd_weights(self.h, s, ctypes.byref(p)), self.h)
        return self._view(p.value, self.P_padded, self.torch.float32)

    def hadpsgd_momentum(self, s):
        p = ctypes.c_void_p()
        _check(lib().hadpsgd_momentum(self.h, s, ctypes.byref(p)), self.h)
        return self._view(p.value, self.P_padded, self.torch.float32)

    def hadpsgd_grads(self, s, g):
        p = ctypes.c_void_p()
        _check(lib().hadpsgd_grads(self.h, s, g, ctypes.byref(p)), self.h)
        dt = self.torch.bfloat16 if self.grad_dtype == BF16 else self.torch.float32
        return self._view(p.value, self.P_padded, dt)

    def hadpsgd_weights_bf16(self, s):
        p = ctypes.c_void_p()
        _check(lib().hadpsgd_weights_bf16(self.h, s, ctypes.byref(p)), self.h)
        return self._view(p.value, self.P_padded, self.torch.bfloat16)

    def hadpsgd_grads_ptr(self, s, g):
        p = ctypes.c_void_p()
        _check(lib().hadpsgd_grads(self.h, s, g, ctypes.byref(p)), self.h)
        return p.value

    def hadpsgd_segment(self, seg):
        off, ln = ctypes.c_int64(0), ctypes.c_int64(0)
        _check(lib().hadpsgd_segment(self.h, seg, ctypes.byref(off), ctypes.byref(ln)), self.h)
        return off.value, ln.value

    def _diag_dict(self, d):
        S = d.S
        return dict(step_k=d.step_k, n_pairs=d.n_pairs, gsq=np.array(d.gsq[:S]), wsq=np.array(d.wsq[:S]),
                    gap=np.array(d.gap[:S]), pend_wsq=np.array(d.pend_wsq[:S]), pend_gap=np.array(d.pend_gap[:S]),
                    pending=np.array(d.pending[:S]))

    def hadpsgd_diagnostics(self):
        d = hadpsgd_diag()
        _check(lib().hadpsgd_diagnostics(self.h, ctypes.byref(d)), self.h)
        return self._diag_dict(d)

    def hadpsgd_unshare(self):
        _check(lib().hadpsgd_unshare(self.h), self.h)

    def hadpsgd_consensus(self):
        out = ctypes.c_double(0.0)
        _check(lib().hadpsgd_consensus(self.h, ctypes.byref(out)), self.h)
        return out.value

    # -- super-learner partition (HADPSGD_PEER) ------------------------------------------
    def hadpsgd_peer_init(self, rank, world, rank_begin):
        arr = (ctypes.c_int32 * (world + 1))(*[int(x) for x in rank_begin])
        _check(lib().hadpsgd_peer_init(self.h, rank, world, arr), self.h)

    def hadpsgd_peer_stage(self):
        p = ctypes.c_void_p()
        _check(lib().hadpsgd_peer_stage(self.h, ctypes.byref(p)), self.h)
        return p.value

    def hadpsgd_peer_attach(self, r, stage_ptr):
        _check(lib().hadpsgd_peer_attach(self.h, r, ctypes.c_void_p(stage_ptr)), self.h)

    def hadpsgd_peer_ipc_export(self):
        buf = ctypes.create_string_buffer(64)
        off = ctypes.c_uint64(0)
        _check(lib().hadpsgd_peer_ipc_export(self.h, buf, ctypes.byref(off)), self.h)
        return bytes(buf.raw), off.value

    def hadpsgd_peer_ipc_attach(self, r, ipc_bytes, stage_offset):
        buf = ctypes.create_string_buffer(ipc_bytes, 64)
        _check(lib().hadpsgd_peer_ipc_attach(self.h, r, buf, stage_offset), self.h)

    def hadpsgd_peer_flush(self):
        _check(lib().hadpsgd_peer_flush(self.h), self.h)

    def hadpsgd_set_diagnostics(self, enable):
        _check(lib().hadpsgd_set_diagnostics(self.h, 1 if enable else 0), self.h)

    def hadpsgd_set_launch(self, blocks_per_sm=0):
        _check(lib().hadpsgd_set_launch(self.h, blocks_per_sm), self.h)

    def hadpsgd_launch_count(self):
        out = ctypes.c_uint64(0)
        _check(lib().hadpsgd_launch_count(self.h, ctypes.byref(out)), self.h)
        return out.value

    def natural_index(self):
        """Indices of the real (non-padding) elements inside a padded buffer, in model order."""
        idx = [np.arange(o, o + n, dtype=np.int64) for o, n in zip(self.layout["seg_offset"], self.seg_len)]
        return np.concatenate(idx)

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            lib().hadpsgd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
