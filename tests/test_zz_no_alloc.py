"""tq_decode_attn_noalloc: decode attention for callers that cannot allocate device memory.

tq_decode_attn wants a workspace that somebody has to cudaMalloc.  A plug-in inside an application whose memory pool owns
the whole device, code on a path where cudaMalloc's device-wide synchronisation is not acceptable, or a process whose
HBM is already handed to others cannot do that; for them libtq.so carries a 24 MiB workspace array of its own and
tq_decode_attn_noalloc uses it (include/tq.h has the full contract: the limit, the one-time address look-up on the
first call per device, the sharing rule).

What is checked here: the new entry point gives what tq_decode_attn gives with a caller-owned workspace, within the
output tolerance of the parity tests (tests/tq_testlib.py: max-abs 2e-3, cosine 0.9999), on calls made one after the
other — same shape twice, then a second shape whose split-K arrival counters lie where the first shape left query
operands (the array keeps the last call's contents; the entry point must clear what has to start at zero), then the
first shape again.  The reference path is the existing one and is itself compared with the CPU oracle in
test_gpu_parity.py.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It builds everything it needs itself, so it passes alone in a fresh process as well as after the others.
"""
import numpy as np
import pytest

from paper_2603_26110_b200 import workloads as W
import tq_testlib as TL


@pytest.fixture(scope="module")
def tq():
    from paper_2603_26110_b200 import build

    build.build()
    from paper_2603_26110_b200 import binding

    binding.lib()
    return binding


class _Case:
    """A cache filled by the library's own tq_quantize_pack, its queries, and the existing path's answer."""

    def __init__(self, tq, w: W.Workload, v_qjl=0):
        import torch

        self.tq, self.w = tq, w
        self.shape = tq.make_shape(w.n_layers, w.batch, w.n_heads, w.head_dim, w.seq, w.rope_base, 0, v_qjl=v_qjl)
        self.params = tq.Params(tq.tq_calibrate_host(self.shape, 1, seed=5))
        self.cache = tq.Cache(self.shape)
        qs = []
        for layer in range(w.n_layers):
            k, v = W.layer_activations(w, layer)
            tq.tq_quantize_pack(self.shape, self.params, self.cache, layer, torch.from_numpy(k).cuda(), torch.from_numpy(v).cuda())
            qs.append(W.queries(w, layer))
        self.q = torch.from_numpy(np.stack(qs)).cuda()
        ws = tq.Workspace(self.shape, w.n_layers)
        ref = torch.full_like(self.q, float("nan"))
        tq.tq_decode_attn(self.shape, self.params, self.cache, 0, w.n_layers, self.q, ref, ws)
        torch.cuda.synchronize()
        self.ref = ref.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(self.ref)) and np.abs(self.ref).max() > 0
        self.torch = torch

    def check_noalloc(self, what):
        out = self.torch.full_like(self.q, float("nan"))
        self.tq.tq_decode_attn_noalloc(self.shape, self.params, self.cache, 0, self.w.n_layers, self.q, out)
        self.torch.cuda.synchronize()
        rep = TL.compare_outputs(out.cpu().numpy(), self.ref, what)
        print(what, rep)
        return rep


@pytest.mark.gpu
def test_noalloc_decode_matches_the_workspace_path_on_consecutive_calls(tq):
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    # A: two units, 130 tiles -> many split-K CTAs per unit; its query operands start 256 bytes into the array
    a = _Case(tq, W.CONFIGS["cfg3_long_splitk"].scaled(batch=1, n_heads=2, seq=4096 + 37))
    # B: 72 units (288 bytes of arrival counters: they reach into what A left behind), 32 tiles, split in two
    b = _Case(tq, W.CONFIGS["cfg2_650m_batch32"].scaled(batch=9, n_heads=8, seq=1024))
    # C: d = 128 with the V-side sketch and three layers in one call (another record size, another table region)
    c = _Case(tq, W.CONFIGS["cfg4_15b_heads"].scaled(n_layers=3, batch=2, n_heads=3, seq=330), v_qjl=1)
    for need in (tq.tq_decode_workspace_bytes(x.shape, x.w.n_layers) for x in (a, b, c)):
        assert 0 < need <= tq.tq_noalloc_scratch_bytes()
    a.check_noalloc("A, first call on this device")
    a.check_noalloc("A, second call in a row")
    b.check_noalloc("B after A (counters over A's leftovers)")
    b.check_noalloc("B again")
    c.check_noalloc("C after B")
    a.check_noalloc("A after C")
    # the existing path is untouched by all this: same answer as before from a fresh caller-owned workspace
    ws = tq.Workspace(b.shape, 1)
    again = torch.full_like(b.q, float("nan"))
    tq.tq_decode_attn(b.shape, b.params, b.cache, 0, 1, b.q, again, ws)
    torch.cuda.synchronize()
    assert np.array_equal(again.cpu().numpy().astype(np.float64), b.ref)


def test_noalloc_refuses_a_shape_beyond_the_built_in_array(tq):
    """Host-side check (no GPU needed): the size test comes before anything touches the device, and an invalid shape
    is reported as by tq_decode_attn."""
    import ctypes as C

    limit = tq.tq_noalloc_scratch_bytes()
    assert limit == 24 << 20
    big = tq.make_shape(1, 64, 40, 64, 32)  # 2560 units x 64 partial records each: about 43 MB
    assert tq.tq_decode_workspace_bytes(big, 1) > limit
    dummy = C.c_void_p(256)
    args = (C.byref(tq.TqParams()), C.byref(tq.TqCache(dummy)), C.c_int32(0), C.c_int32(1), dummy, None, C.c_int(tq.TQ_F16),
            dummy, C.c_int32(0), None)
    assert tq.lib().tq_decode_attn_noalloc(C.byref(big), *args) == tq.TQ_ERR_CAPACITY
    bad = tq.make_shape(1, 2, 2, 96, 32)  # head_dim 96
    assert tq.lib().tq_decode_attn_noalloc(C.byref(bad), *args) == tq.TQ_ERR_UNSUPPORTED
    ok_shape = tq.make_shape(2, 2, 2, 64, 32)
    args3 = args[:3] + (C.c_int32(3),) + args[4:]  # more layers than the shape has
    assert tq.lib().tq_decode_attn_noalloc(C.byref(ok_shape), *args3) == tq.TQ_ERR_INVALID_ARG
    # every BASELINE.json configuration fits, the V-side sketch and all 33 layers of configs[1] in one call included
    for w in W.CONFIGS.values():
        for vq in (0, 1):
            s = tq.make_shape(w.n_layers, w.batch, w.n_heads, w.head_dim, w.seq, v_qjl=vq)
            assert 0 < tq.tq_decode_workspace_bytes(s, w.n_layers) <= limit, (w.name, vq)
