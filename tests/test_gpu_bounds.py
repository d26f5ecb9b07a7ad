"""Memory-safety check of every kernel of the hot path without a sanitizer (compute-sanitizer is closed on the GPU pool):
all output and workspace buffers of one problem are carved out of a single arena filled with a canary byte, with guard
gaps before, between and after them; after the whole path has run (prologue with and without smoothing, V quantiser,
INT4 attention from the prologue's workspace and from the packed buffers alone, FP16 attention) every guard byte must be
intact.  Shapes are ragged in N (last tile of 95 / 2 valid rows), with text tokens, D = 128 and D = 64."""
import numpy as np
import pytest

torch = pytest.importorskip('torch')
pytestmark = pytest.mark.gpu

import __graft_entry__ as entry  # noqa: E402

entry.build()
from paper_2607_02584_b200 import api  # noqa: E402
from synth import video_qkv as syn  # noqa: E402

CANARY = 0xA5
GAP = 4096


class Arena:
    def __init__(self, sizes):
        self.offsets, off = {}, GAP
        for name, nbytes in sizes.items():
            self.offsets[name] = (off, nbytes)
            off += (nbytes + 255) // 256 * 256 + GAP
        self.buf = torch.full((off,), CANARY, dtype=torch.uint8, device='cuda')
        self.total = off

    def view(self, name, dtype, shape):
        off, nbytes = self.offsets[name]
        t = self.buf[off:off + nbytes].view(dtype)
        return t.view(shape)

    def guards_intact(self):
        mask = torch.ones(self.total, dtype=torch.bool, device='cuda')
        for off, nbytes in self.offsets.values():
            mask[off:off + nbytes] = False
        return bool((self.buf[mask] == CANARY).all())


def _arena_buffers(p, b):
    """Re-home every tensor of an api.Buffers object in one guarded arena."""
    names = ['Q4', 'K4', 'V4', 'Qs', 'Ks', 'Vs', 'O', 'ws', 'Q16', 'K16', 'O16', 'ws16']
    sizes = {n: getattr(b, n).numel() * getattr(b, n).element_size() for n in names}
    ar = Arena(sizes)
    for n in names:
        t = getattr(b, n)
        setattr(b, n, ar.view(n, t.dtype, t.shape))
    return ar


CASES = [  # grid, n_text, base workload, qk_group, v_scale, smooth, p_norm
    ((3, 9, 13), 0, 'wan', 1, 0, 0, 0),
    ((3, 9, 13), 21, 'hunyuan', 1, 0, 0, 0),
    ((1, 10, 13), 0, 'wan', 1, 0, 0, 1),
    ((3, 9, 13), 21, 'hunyuan', 128, 1, 0, 0),
    ((3, 9, 13), 0, 'wan', 1, 0, 1, 0),
    (None, 0, 'tiny', 1, 0, 0, 0),
    (None, 0, 'tiny', 128, 0, 0, 0),
]


@pytest.mark.parametrize('grid,n_text,base,qk_group,v_scale,smooth,p_norm', CASES)
def test_no_kernel_writes_outside_its_buffers(grid, n_text, base, qk_group, v_scale, smooth, p_norm):
    if base == 'tiny':
        w = syn.TINY
    else:
        w = syn.small_variant(syn.WAN_1_3B if base == 'wan' else syn.HUNYUAN, grid, n_text=n_text, H=2)
    q, k, v = syn.gen_all(w)
    p = api.params_for(w, api.ROT_HALF, api.P_ASYM15, p_norm, H=q.shape[1], qk_group=qk_group, v_scale=v_scale, smooth=smooth)
    coef = torch.from_numpy(api.rotattn_build_tables(p)).cuda()
    Q, K, V = (torch.from_numpy(x).cuda() for x in (q, k, v))
    b = api.Buffers(p, want_fp16=True)
    ar = _arena_buffers(p, b)
    assert ar.guards_intact()
    if smooth:
        api.rotattn_smooth_stats(p, coef, None, Q, K, V, b.ws)
    api.rotattn_prepare_qk(p, coef, None, Q, K, b.Q4, b.Qs, b.K4, b.Ks, b.Q16, b.K16, b.ws)
    api.rotattn_quant_v(p, V, b.V4, b.Vs, b.ws)
    api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, api.ws_state_full(p))
    torch.cuda.synchronize()
    assert ar.guards_intact(), 'a kernel of the INT4 path wrote outside its buffers'
    o_first = b.O.clone()
    if not smooth:      # the smoothing state lives only in the prologue's workspace
        api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, 0)     # operand copies rebuilt from the packed buffers
        torch.cuda.synchronize()
        assert ar.guards_intact(), 'the unpack path wrote outside its buffers'
        assert torch.equal(o_first, b.O), 'fresh-workspace launch differs from the prologue-workspace launch'
    api.rotattn_fwd_fp16(p, b.Q16, b.K16, V, b.O16, b.ws16)
    torch.cuda.synchronize()
    assert ar.guards_intact(), 'the FP16 path wrote outside its buffers'
    assert bool(torch.isfinite(b.O.float()).all()) and bool(torch.isfinite(b.O16.float()).all())
