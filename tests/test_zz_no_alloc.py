"""ikv_decode_attn_static: paged decode with its split partials in the library's static device array (no allocation in
the call).  Collected last on purpose (the run uses pytest -x).  Checked against the existing ikv_decode_attn
on the same inputs, within the decode tolerance of the other GPU tests, on two calls in a row (the second call finds the
first call's contents in the shared array), and against the oracle."""
import math

import numpy as np
import pytest
import torch

from paper_2606_09916_b200 import workloads as wl
from tests import gpu_common as gc

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ikv():
    from paper_2606_09916_b200 import ikv as m
    return m


def _case(ikv, oracle, shape, n_tokens, seed):
    w = wl.small(seed=seed, shape=shape, n_tokens=n_tokens, budget=n_tokens // 3, decode_tokens=4, kv_dtype=shape.kv_dtype)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    S = s.slot_map[:s.N].clone()
    rng = np.random.default_rng(seed)
    S[torch.from_numpy(rng.choice(s.N, size=s.N // 3, replace=False))] = w.dead_slot   # a pruned map: dead entries
    return w, kp, vp, ctx, s, S


@pytest.mark.parametrize("name,shape,n_tokens", [("bf16 d128 g4", wl.ModelShape(2, 8, 2, 128, "bf16"), 5000),
                                                  ("f32 d64 g2", wl.ModelShape(2, 4, 2, 64, "f32"), 700)])
def test_static_scratch_decode_matches_existing_path(ikv, oracle, name, shape, n_tokens):
    w, kp, vp, ctx, s, S = _case(ikv, oracle, shape, n_tokens, 91)
    S_dev = S.cuda()
    g = gc.oracle_geom(oracle, w)
    is_bf16 = shape.kv_dtype == "bf16"
    dt = torch.bfloat16 if is_bf16 else torch.float32
    scale = 1.0 / math.sqrt(shape.D)
    req = gc.request(ikv, s, S_dev)
    req.flags = ikv.REQ_RESCAN
    # two calls in a row: different layer, different query, different length (the second finds the first's partials)
    for call, (layer, n) in enumerate(((0, s.N), (shape.L - 1, s.N - 37))):
        q = torch.randn((1, shape.Hq, shape.D), generator=torch.Generator().manual_seed(100 + call)).to(dt)
        q_dev = q.cuda()
        req.seq_len = n
        ref = torch.empty((1, shape.Hq, shape.D), dtype=dt, device="cuda")
        ctx.decode_attn(layer, [req], q_dev, ref, scale)
        got = torch.full((1, shape.Hq, shape.D), float("nan"), dtype=dt, device="cuda")
        ctx.decode_attn_static(layer, req, q_dev, got, scale)
        torch.cuda.synchronize()
        err = gc.assert_decode_close(got[0].float().cpu().numpy(), ref[0].float().cpu().numpy(), is_bf16,
                                     f"{name} call {call} vs ikv_decode_attn")
        want = oracle.decode(g, kp, vp, layer, S[:n].numpy(), q[0].float().numpy(), scale)
        err_o = gc.assert_decode_close(got[0].float().cpu().numpy(), want, is_bf16, f"{name} call {call} vs oracle")
        print(f"[{name}] call {call}: max abs diff to ikv_decode_attn {err:.3e}, to the oracle {err_o:.3e}")


def test_static_scratch_decode_rejects_what_does_not_fit(ikv, oracle):
    """64 query heads at head_dim 128: 116 splits would need 3.9 MB of partials, the array holds 3 MiB."""
    shape = wl.ModelShape(1, 64, 8, 128, "bf16")
    w, kp, vp, ctx, s, S = _case(ikv, oracle, shape, 3000, 92)
    S_dev = S.cuda()
    q = torch.randn((1, shape.Hq, shape.D), generator=torch.Generator().manual_seed(5)).to(torch.bfloat16).cuda()
    out = torch.zeros_like(q)
    req = gc.request(ikv, s, S_dev)
    with pytest.raises(ikv.IkvError) as ei:
        ctx.decode_attn_static(0, req, q, out, 0.1)
    assert ei.value.status == ikv.ERR_CAPACITY and "static" in str(ei.value)
    torch.cuda.synchronize()
    assert float(out.float().abs().sum()) == 0.0          # nothing was enqueued
    req.seq_len = 1000                                    # 63 splits: fits
    ctx.decode_attn_static(0, req, q, out, 0.1)
    torch.cuda.synchronize()
    want = oracle.decode(gc.oracle_geom(oracle, w), kp, vp, 0, S[:1000].numpy(), q[0].float().cpu().numpy(), 0.1)
    gc.assert_decode_close(out[0].float().cpu().numpy(), want, True, "64 heads, 1000 positions")
