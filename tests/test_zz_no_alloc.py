"""rotattn_fwd_int4_static - the INT4 attention forward for callers that cannot allocate device memory.

A serving process that gave all of HBM to its own arena at start-up, or an operator wired into another runtime through
an "inputs, outputs" signature, has no workspace to pass to rotattn_fwd_int4 and is not allowed to cudaMalloc one (the
allocation would synchronise the device in the middle of a denoising step, and may fail because the arena owns the
memory).  For them the library carries an 8 MiB workspace of its own (ROTATTN_STATIC_WS_BYTES) and this entry point
takes inputs and outputs only.

The test drives it twice in a row, on two different shapes, and compares each O with the one the ordinary path
(prologue-written workspace -> rotattn_fwd_int4) produced from the same packed inputs.  Both paths run the same
attention kernel on the same operand bytes, so the repository's bound for that comparison is equality bit for bit
(tests/test_gpu_bounds.py does the same for a caller-allocated fresh workspace).  The second shape is smaller and
ragged, so the shared array still holds the first call's bytes where the second call pads - they must not leak into O.

Collected last on purpose (file name): under `pytest -x` a failure here hides nothing that comes after it.
"""
import pytest
import torch

from synth import video_qkv as syn

pytestmark = pytest.mark.gpu


def _ordinary_path(api, w, H, **modes):
    """prepare_qk -> quant_v -> fwd_int4 on a caller-allocated workspace; returns (params, buffers)."""
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=api.ROT_HALF, **modes)
    torch.cuda.synchronize()
    return res['p'], res['buffers']


def _static_path(api, p, b, head_sel=None):
    O = torch.full_like(b.O, 7.0)                 # a value attention never produces here: untouched rows stay visible
    api.rotattn_fwd_int4_static(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, O, head_sel=head_sel)
    torch.cuda.synchronize()
    return O


def test_static_workspace_matches_ordinary_path_twice_in_a_row():
    from paper_2607_02584_b200 import api
    # call 1: three heads, N = 3*9*13 + 17 text tokens = 368 (two full key blocks and a ragged third)
    w1 = syn.small_variant(syn.HUNYUAN, (3, 9, 13), n_text=17, H=3)
    p1, b1 = _ordinary_path(api, w1, 3)
    assert api.rotattn_workspace_bytes(p1, 1) <= api._b.STATIC_WS_BYTES
    assert torch.equal(_static_path(api, p1, b1), b1.O), 'first call differs from the ordinary path'
    # call 2, straight after: one head, N = 2*7*11 = 154, per-block Q/K scales - the array still holds call 1's bytes
    w2 = syn.small_variant(syn.WAN_1_3B, (2, 7, 11), H=1)
    p2, b2 = _ordinary_path(api, w2, 1, qk_group=128)
    assert torch.equal(_static_path(api, p2, b2), b2.O), 'second call differs from the ordinary path'
    # and shape 1 again, now on a head subset: the other head's rows must stay untouched
    sel = torch.tensor([2, 0], dtype=torch.int32, device='cuda')
    O = _static_path(api, p1, b1, head_sel=sel)
    assert torch.equal(O[0, 0], b1.O[0, 0]) and torch.equal(O[0, 2], b1.O[0, 2])
    assert bool(torch.all(O[0, 1] == 7.0))


def test_static_workspace_rejects_what_it_cannot_hold():
    from paper_2607_02584_b200 import api
    w = syn.small_variant(syn.WAN_1_3B, (2, 7, 11), H=1)
    p, b = _ordinary_path(api, w, 1)
    # too large: all 12 heads of the 480p shape need ~150 MB of operand copies, the built-in array holds 8 MiB
    big = api.params_for(syn.WAN_1_3B)
    assert api.rotattn_workspace_bytes(big, 1) > api._b.STATIC_WS_BYTES
    st = api.lib.rotattn_fwd_int4_static(*_raw_args(api, big, b))
    assert st == -4, st                                               # ROTATTN_ERR_WORKSPACE_TOO_SMALL
    assert b'built-in' in api.lib.rotattn_last_cuda_error()
    # smoothing keeps its state in the prologue's workspace: not available here
    sm = api.params_for(w, H=1, smooth=1)
    assert api.lib.rotattn_fwd_int4_static(*_raw_args(api, sm, b)) == -2   # ROTATTN_ERR_UNSUPPORTED
    # a rejected call must leave the entry point usable
    assert torch.equal(_static_path(api, p, b), b.O)


def _raw_args(api, p, b):
    """ctypes argument list of rotattn_fwd_int4_static for buffers b (the calls above are rejected before any launch,
    so the buffers need not match the parameter block)."""
    import ctypes as C
    ptr = lambda t: C.c_void_p(t.data_ptr())
    return (C.byref(p), ptr(b.Q4), ptr(b.Qs), ptr(b.K4), ptr(b.Ks), ptr(b.V4), ptr(b.Vs), ptr(b.O), None, 0,
            C.c_void_p(torch.cuda.current_stream().cuda_stream))
