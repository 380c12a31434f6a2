"""TEST INFRASTRUCTURE: run the scripts the driver runs on a B200 (bench.py, __graft_entry__.smoke, tests/preflight.py)
on a machine WITHOUT a GPU, so that a Python-level mistake in them (a wrong key, a renamed binding call, a bad format
string) is found here and not in the one device run a round gets.

How: inside `with shim_as_cuda():` the ctypes binding talks to tests/cpu_shim's build of the kernel sources instead of
libcbct_b200.so, and the handful of torch.cuda calls the scripts make are answered by CPU stand-ins (`.cuda()` returns
the CPU tensor, whose address the shim accepts as a "device" pointer; events are wall-clock stamps).  Nothing outside
tests/ imports this module; the package itself still refuses to run without the CUDA library and a device, and no
parity or performance claim is made from a dry run -- the numbers it prints are meaningless, only "the script runs to
its last line and prints what the contract asks for" is checked.
"""
from __future__ import annotations

import contextlib
import time

import torch

from cpu_shim import shimlib as sl
from paper_1008_2042_b200 import binding as cb


class _Event:
    def __init__(self, enable_timing=False):
        self.t = None

    def record(self, stream=None):
        self.t = time.perf_counter()

    def synchronize(self):
        pass

    def elapsed_time(self, other):
        return max((other.t - self.t) * 1e3, 1e-6)


class _Stream:
    cuda_stream = 0


def _dptr(t, n=None):
    if not (isinstance(t, torch.Tensor) and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 tensor")
    if n is not None and t.numel() != n:
        raise ValueError(f"expected {n} elements, got {t.numel()}")
    return t.data_ptr()


@contextlib.contextmanager
def shim_as_cuda():
    saved = []

    def patch(obj, name, value):
        saved.append((obj, name, getattr(obj, name)))
        setattr(obj, name, value)

    def no_device(fn):
        def wrapped(*a, **k):
            if str(k.get("device", "")).startswith("cuda"):
                k = dict(k, device="cpu")
            return fn(*a, **k)
        return wrapped

    try:
        patch(cb, "_lib", sl.lib())
        patch(cb, "_dptr", _dptr)
        patch(cb, "_stream", lambda stream=None: 0)
        real_microbench = cb.microbench                            # default loop length (2000) would take hours on the host
        patch(cb, "microbench", lambda stream=None, iters=0: real_microbench(stream, iters if iters > 0 else 1))
        from paper_1008_2042_b200 import replicas
        real_init = replicas.init                                  # N > 1 dry runs rendezvous over gloo
        patch(replicas, "init", lambda backend="nccl", device=None: real_init("gloo", None))
        patch(torch.cuda, "is_available", lambda: True)
        patch(torch.cuda, "set_device", lambda *a, **k: None)
        patch(torch.cuda, "synchronize", lambda *a, **k: None)
        patch(torch.cuda, "current_stream", lambda *a, **k: _Stream())
        patch(torch.cuda, "Event", _Event)
        patch(torch.Tensor, "cuda", lambda self, *a, **k: self)
        patch(torch.Tensor, "pin_memory", lambda self, *a, **k: self)
        for name in ("empty", "zeros", "ones", "tensor", "empty_like", "zeros_like"):
            patch(torch, name, no_device(getattr(torch, name)))
        yield
    finally:
        for obj, name, value in reversed(saved):
            setattr(obj, name, value)
        sl.check(0, "dry run")
