"""Helpers for the -m gpu parity tests: device buffers come from torch (plumbing only), results are compared
with the CPU oracle element by element."""
from __future__ import annotations

import numpy as np

from paper_1410_6685_b200 import sg

NP2SG = {np.dtype(np.float32): sg.SG_F32, np.dtype(np.float64): sg.SG_F64, np.dtype(np.int32): sg.SG_I32,
         np.dtype(np.int64): sg.SG_I64, np.dtype(np.uint8): sg.SG_BOOL}
SG2NP = {v: k for k, v in NP2SG.items()}


def dev(a: np.ndarray):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def empty_dev(n: int, dtype):
    import torch
    return torch.empty(n, dtype=getattr(torch, np.dtype(dtype).name), device="cuda")


class Ctx:
    """A context on cuda:0 using torch's current stream."""

    def __init__(self, flags: int = 0):
        import torch
        self.torch = torch
        self.ctx = sg.sg_ctx_create(0, torch.cuda.current_stream().cuda_stream)
        if flags:
            sg.sg_ctx_set_flags(self.ctx, flags)
        self.keep = []

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        sg.sg_ctx_destroy(self.ctx)
        self.keep.clear()

    def vec(self, a: np.ndarray) -> int:
        t = dev(a)
        self.keep.append(t)
        return sg.sg_vec_create(self.ctx, NP2SG[a.dtype], a.size, t.data_ptr())

    def vec_t(self, t) -> int:
        self.keep.append(t)
        return sg.sg_vec_create(self.ctx, NP2SG[np.dtype(str(t.dtype).replace("torch.", ""))], t.numel(), t.data_ptr())

    def read_vec(self, h: int, dtype, n: int | None = None) -> np.ndarray:
        """Device -> host copy of a collection's storage (the caller-side half of to_array)."""
        cnt = sg.sg_vec_count(self.ctx, h) if n is None else n
        out = np.empty(cnt, dtype=dtype)
        sg.sg_vec_read(self.ctx, h, out.ctypes.data, out.nbytes)
        return out

    def get(self, h: int):
        return sg.sg_scalar_get(self.ctx, h)


def rel_err(got: float, want: float, sum_abs: float) -> float:
    if want == 0.0:
        return abs(got) / max(sum_abs, 1e-300)
    return abs(got - want) / abs(want)
