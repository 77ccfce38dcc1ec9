"""sg_vec_sum_noalloc (include/sg.h): the allocation-free sum against the existing path, sg_reduce(SG_SUM) through a context, on
the same device data — two calls in a row (the static scratch array keeps the first call's contents), within the sum tolerances
of the parity tests (fp64 1e-12, fp32 1e-5 relative).  Named test_zz_* so that pytest collects it last."""
from __future__ import annotations

import numpy as np
import pytest

import oracle as orc
from paper_1410_6685_b200 import inputs, sg
from gpu_util import NP2SG, Ctx, dev, rel_err

pytestmark = pytest.mark.gpu

TOL = {np.dtype(np.float64): 1e-12, np.dtype(np.float32): 1e-5}


def existing_path_sum(t) -> float:
    """The same device buffer summed by the library's deferred path: create, reduce, flush, hand-back."""
    with Ctx() as c:
        h = c.vec_t(t)
        return c.get(sg.sg_reduce(c.ctx, h, sg.SG_SUM))


def noalloc_sum(torch, t, out) -> None:
    sg.sg_vec_sum_noalloc(0, torch.cuda.current_stream().cuda_stream, NP2SG[np.dtype(str(t.dtype).replace("torch.", ""))], t.data_ptr(), t.numel(),
                          out.data_ptr())


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_two_calls_in_a_row_match_the_existing_path(dtype):
    import torch
    tol = TOL[np.dtype(dtype)]
    # first call: many tiles and a ragged tail; second call: SHORTER (stale partials of the first call lie behind its own) and
    # starting one element off 16-byte alignment (the scalar path)
    n1, n2 = 148 * 8 * 8192 * 3 + 4099, 8192 * 37 + 5
    a = inputs.normal_f32(11, 0, n1).astype(dtype) * dtype(3.0) + dtype(0.25)
    b = (inputs.normal_f32(12, 0, n2 + 1).astype(dtype) - dtype(0.5))
    ta, tb = dev(a), dev(b)[1:]
    assert tb.data_ptr() % 16 != 0
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    noalloc_sum(torch, ta, out[0:1])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    noalloc_sum(torch, tb, out[1:2])                 # back to back on the same stream: ordered, no race on the scratch array
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before          # the call took no device memory
    got = out.cpu().numpy()
    for g, t, host in ((got[0], ta, a), (got[1], tb, b[1:])):
        want = existing_path_sum(t)
        sum_abs = float(np.abs(host.astype(np.float64)).sum())
        assert rel_err(float(g), want, sum_abs) <= tol, (g, want)
        assert rel_err(float(g), orc.sum(host), sum_abs) <= tol, (g, orc.sum(host))
    # the same input again gives the same bits (partials are combined in tile order, whatever the last call left behind)
    again = torch.zeros(1, dtype=torch.float64, device="cuda")
    noalloc_sum(torch, ta, again)
    assert again.cpu().numpy().tobytes() == got[0:1].tobytes()


def test_largest_size_empty_input_and_rejections():
    import torch
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    # the maximum size the scratch array supports
    n = sg.SG_NOALLOC_MAX_N
    t = torch.from_numpy(inputs.normal_f32(13, 0, n)).cuda()
    noalloc_sum(torch, t, out)
    got = float(out.item())
    want = existing_path_sum(t)
    assert rel_err(got, want, float(t.abs().sum(dtype=torch.float64).item())) <= 1e-5, (got, want)
    # empty input: +0.0, and the output is written
    sg.sg_vec_sum_noalloc(0, stream, sg.SG_F64, 0, 0, out.data_ptr())
    assert out.cpu().numpy().tobytes() == np.zeros(1).tobytes()
    # one element beyond the maximum: a clear error, nothing launched (the pointer is never touched)
    out.fill_(7.0)
    with pytest.raises(sg.SgError) as e:
        sg.sg_vec_sum_noalloc(0, stream, sg.SG_F32, t.data_ptr(), n + 1, out.data_ptr())
    assert e.value.status == sg.SG_ERR_CAPACITY and "SG_NOALLOC_MAX_N" in str(e.value)
    for args, status in (((0, stream, sg.SG_I32, t.data_ptr(), 16, out.data_ptr()), sg.SG_ERR_DTYPE),
                         ((0, stream, sg.SG_F32, t.data_ptr(), -1, out.data_ptr()), sg.SG_ERR_ARG),
                         ((0, stream, sg.SG_F32, 0, 16, out.data_ptr()), sg.SG_ERR_ARG),
                         ((0, stream, sg.SG_F32, t.data_ptr(), 16, 0), sg.SG_ERR_ARG),
                         ((64, stream, sg.SG_F32, t.data_ptr(), 16, out.data_ptr()), sg.SG_ERR_ARG)):
        with pytest.raises(sg.SgError) as e:
            sg.sg_vec_sum_noalloc(*args)
        assert e.value.status == status
    torch.cuda.synchronize()
    assert float(out.item()) == 7.0
