"""Python face of the C-ABI: the same entry-point names taking torch CUDA tensors (PyTorch is used
for device memory and streams only).  No arithmetic of the method happens here."""
from __future__ import annotations

import ctypes as C

import numpy as np
import torch

from . import binding as _b
from .binding import (ROT_NONE, ROT_INTERLEAVED, ROT_HALF, ROT_FULL, P_ASYM15, P_SYM7, NORM_ROWBLOCK, NORM_RUNNING,
                      WS_HAS_QK, WS_HAS_V, WS_HAS_STATS, VSCALE_CHANNEL, VSCALE_GROUP, make_params, check)

lib = _b.lib


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous()
        return C.c_void_p(t.data_ptr())
    if isinstance(t, np.ndarray):
        assert t.flags['C_CONTIGUOUS']
        return C.c_void_p(t.ctypes.data)
    raise TypeError(type(t))


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _need_cuda(*ts):
    for t in ts:
        if t is not None and not t.is_cuda:
            raise ValueError('device tensors required: librotattn has no CPU path')


# ---- host helpers --------------------------------------------------------------------------------
def rotattn_build_tables(p, rot=None) -> np.ndarray:
    n = lib.rotattn_table_floats(C.byref(p))
    if n == 0:
        check(lib.rotattn_validate(C.byref(p)), 'rotattn_validate')
    out = np.empty(n, dtype=np.float32)
    rot_arr = None if rot is None else np.ascontiguousarray(rot, dtype=np.float32).reshape(-1)
    check(lib.rotattn_build_tables(C.byref(p), _ptr(rot_arr), _ptr(out)), 'rotattn_build_tables')
    return out.reshape(-1, 4)


def rotattn_workspace_bytes(p, which: int) -> int:
    return int(lib.rotattn_workspace_bytes(C.byref(p), which))


def _policy_struct(pol: dict):
    mask = pol.get('fp16_head_mask')
    arr = None
    if mask is not None:
        arr = (C.c_uint8 * len(mask))(*[int(x) for x in mask])
    st = _b.RotattnPolicy(pol['n_steps'], pol['n_blocks'], pol['first_steps'], pol['last_steps'],
                          pol['first_blocks'], pol['last_blocks'], 0 if mask is None else len(mask), arr)
    return st, arr          # arr is returned so that it stays alive while the struct points at it


def rotattn_policy_select(pol: dict, step: int, block: int, head: int = 0) -> int:
    st, _keep = _policy_struct(pol)
    return int(lib.rotattn_policy_select(C.byref(st), step, block, head))


def rotattn_policy_split_heads(pol: dict, step: int, block: int, B: int, H: int):
    st, _keep = _policy_struct(pol)
    a = np.zeros(B * H, dtype=np.int32)
    b = np.zeros(B * H, dtype=np.int32)
    na, nb = C.c_int32(0), C.c_int32(0)
    check(lib.rotattn_policy_split_heads(C.byref(st), step, block, B, H, _ptr(a), C.cast(C.byref(na), C.c_void_p),
                                         _ptr(b), C.cast(C.byref(nb), C.c_void_p)), 'rotattn_policy_split_heads')
    return a[:na.value].copy(), b[:nb.value].copy()


def ws_state_full(p) -> int:
    """ws_state of a workspace that went through the whole prologue for p (smooth_stats too when p.smooth)."""
    return WS_HAS_QK | WS_HAS_V | (WS_HAS_STATS if p.smooth else 0)


# ---- device entry points -------------------------------------------------------------------------
def rotattn_prepare_qk(p, coef_dev, rot_dev, Q, K, Q4, Qs, K4, Ks, Qrope16=None, Krope16=None,
                       workspace=None, stream=None):
    _need_cuda(coef_dev, rot_dev, Q, K, Q4, Qs, K4, Ks, Qrope16, Krope16, workspace)
    check(lib.rotattn_prepare_qk(C.byref(p), _ptr(coef_dev), _ptr(rot_dev), _ptr(Q), _ptr(K), _ptr(Q4), _ptr(Qs),
                                 _ptr(K4), _ptr(Ks), _ptr(Qrope16), _ptr(Krope16), _ptr(workspace),
                                 0 if workspace is None else workspace.numel() * workspace.element_size(),
                                 _stream(stream)), 'rotattn_prepare_qk')


def rotattn_quant_v(p, V, V4, Vs, workspace=None, stream=None):
    _need_cuda(V, V4, Vs, workspace)
    check(lib.rotattn_quant_v(C.byref(p), _ptr(V), _ptr(V4), _ptr(Vs), _ptr(workspace),
                              0 if workspace is None else workspace.numel() * workspace.element_size(),
                              _stream(stream)), 'rotattn_quant_v')


def rotattn_fwd_int4(p, Q4, Qs, K4, Ks, V4, Vs, O, workspace, ws_state, head_sel=None, stream=None):
    _need_cuda(Q4, Qs, K4, Ks, V4, Vs, O, workspace, head_sel)
    check(lib.rotattn_fwd_int4(C.byref(p), _ptr(Q4), _ptr(Qs), _ptr(K4), _ptr(Ks), _ptr(V4), _ptr(Vs), _ptr(O),
                               _ptr(head_sel), 0 if head_sel is None else head_sel.numel(), _ptr(workspace),
                               workspace.numel() * workspace.element_size(), ws_state, _stream(stream)),
          'rotattn_fwd_int4')


def rotattn_fwd_int4_static(p, Q4, Qs, K4, Ks, V4, Vs, O, head_sel=None, stream=None):
    """rotattn_fwd_int4 without a workspace argument, for callers that may not allocate device memory (a serving
    process whose arena owns all of HBM, an operator with an inputs/outputs-only signature): the scratch is an 8 MiB
    array inside librotattn.so.  Shapes whose workspace exceeds it raise; calls that overlap on the GPU race on it."""
    _need_cuda(Q4, Qs, K4, Ks, V4, Vs, O, head_sel)
    check(lib.rotattn_fwd_int4_static(C.byref(p), _ptr(Q4), _ptr(Qs), _ptr(K4), _ptr(Ks), _ptr(V4), _ptr(Vs), _ptr(O),
                                      _ptr(head_sel), 0 if head_sel is None else head_sel.numel(), _stream(stream)),
          'rotattn_fwd_int4_static')


def rotattn_smooth_stats(p, coef_dev, rot_dev, Q, K, V, workspace, stream=None):
    _need_cuda(coef_dev, rot_dev, Q, K, V, workspace)
    check(lib.rotattn_smooth_stats(C.byref(p), _ptr(coef_dev), _ptr(rot_dev), _ptr(Q), _ptr(K), _ptr(V), _ptr(workspace),
                                   workspace.numel() * workspace.element_size(), _stream(stream)), 'rotattn_smooth_stats')


def rotattn_smooth_read(p, workspace, means_out=None, kcorr_out=None, stream=None):
    _need_cuda(workspace, means_out, kcorr_out)
    check(lib.rotattn_smooth_read(C.byref(p), _ptr(workspace), workspace.numel() * workspace.element_size(),
                                  _ptr(means_out), _ptr(kcorr_out), _stream(stream)), 'rotattn_smooth_read')


def rotattn_fwd_int4_debug(p, Q4, Qs, K4, Ks, V4, Vs, bh, q_tile, S_dump, P_dump, O_tile, workspace, ws_state,
                           PV_dump=None, stream=None):
    _need_cuda(Q4, Qs, K4, Ks, V4, Vs, S_dump, P_dump, PV_dump, O_tile, workspace)
    check(lib.rotattn_fwd_int4_debug(C.byref(p), _ptr(Q4), _ptr(Qs), _ptr(K4), _ptr(Ks), _ptr(V4), _ptr(Vs),
                                     bh, q_tile, _ptr(S_dump), _ptr(P_dump), _ptr(PV_dump), _ptr(O_tile), _ptr(workspace),
                                     workspace.numel() * workspace.element_size(), ws_state, _stream(stream)),
          'rotattn_fwd_int4_debug')


def rotattn_fwd_fp16(p, Q16, K16, V16, O, workspace=None, head_sel=None, stream=None):
    """workspace is ignored by the library since ABI version 3 (V is read in place); the parameter stays for old callers."""
    _need_cuda(Q16, K16, V16, O, workspace, head_sel)
    check(lib.rotattn_fwd_fp16(C.byref(p), _ptr(Q16), _ptr(K16), _ptr(V16), _ptr(O), _ptr(head_sel),
                               0 if head_sel is None else head_sel.numel(), _ptr(workspace),
                               0 if workspace is None else workspace.numel() * workspace.element_size(), _stream(stream)),
          'rotattn_fwd_fp16')


def rotattn_fwd_fp16_debug_f32(p, Q16, K16, V16, O32, workspace=None, head_sel=None, stream=None):
    """rotattn_debug.h: rotattn_fwd_fp16 with O/l stored as fp32 (test aid)."""
    _need_cuda(Q16, K16, V16, O32, workspace, head_sel)
    assert O32.dtype == torch.float32
    check(lib.rotattn_fwd_fp16_debug_f32(C.byref(p), _ptr(Q16), _ptr(K16), _ptr(V16), _ptr(O32), _ptr(head_sel),
                                         0 if head_sel is None else head_sel.numel(), _ptr(workspace),
                                         0 if workspace is None else workspace.numel() * workspace.element_size(), _stream(stream)),
          'rotattn_fwd_fp16_debug_f32')


def rotattn_probe_gemm8(M, N, K, A, B, Cout, mode=0, stream=None):
    _need_cuda(A, B, Cout)
    check(lib.rotattn_probe_gemm8(M, N, K, _ptr(A), _ptr(B), _ptr(Cout), mode, _stream(stream)), 'rotattn_probe_gemm8')


# ---- convenience for tests / bench: allocate buffers and run the whole path ----------------------
class Buffers:
    """Device buffers of one problem (allocation only)."""

    def __init__(self, p, want_fp16=False, device='cuda'):
        B, H, N, D = p.B, p.H, p.N, p.D
        nG = (N + 127) // 128
        u8, f32, f16 = torch.uint8, torch.float32, torch.float16
        self.Q4 = torch.empty((B, H, N, D // 2), dtype=u8, device=device)
        self.K4 = torch.empty_like(self.Q4)
        self.V4 = torch.empty_like(self.Q4)
        self.Qs = torch.empty((B, H, N if p.qk_group == 1 else nG), dtype=f32, device=device)
        self.Ks = torch.empty_like(self.Qs)
        self.Vs = torch.empty((B, H, nG, D) if p.v_scale == VSCALE_CHANNEL else (B, H, nG), dtype=f32, device=device)
        self.O = torch.zeros((B, H, N, D), dtype=f16, device=device)
        self.ws = torch.empty(rotattn_workspace_bytes(p, 0), dtype=u8, device=device)
        self.Q16 = self.K16 = self.O16 = self.ws16 = None
        if want_fp16:
            self.Q16 = torch.empty((B, H, N, D), dtype=f16, device=device)
            self.K16 = torch.empty_like(self.Q16)
            self.O16 = torch.zeros_like(self.Q16)
            self.ws16 = torch.empty(rotattn_workspace_bytes(p, 2), dtype=u8, device=device)


def params_for(w, rot_mode=ROT_HALF, p_mode=P_ASYM15, p_norm=NORM_ROWBLOCK, H=None, qk_group=1,
               v_scale=VSCALE_CHANNEL, smooth=0):
    return make_params(w.B, w.H if H is None else H, w.N, w.D, w.grid, w.pairs, 10000.0, rot_mode, p_mode, p_norm,
                       qk_group=qk_group, v_scale=v_scale, smooth=smooth)


def run_int4(w, q, k, v, rot_mode=ROT_HALF, p_mode=P_ASYM15, p_norm=NORM_ROWBLOCK, want_fp16=False,
             coef=None, rot=None, use_ws=True, qk_group=1, v_scale=VSCALE_CHANNEL, smooth=0):
    """Whole hot path on numpy fp16 inputs [B,H',N,D]; returns a dict of device tensors."""
    p = params_for(w, rot_mode, p_mode, p_norm, H=q.shape[1], qk_group=qk_group, v_scale=v_scale, smooth=smooth)
    tab = rotattn_build_tables(p, rot) if coef is None else np.ascontiguousarray(coef, dtype=np.float32)
    coef_dev = torch.from_numpy(tab).cuda()
    rot_dev = None if rot is None else torch.from_numpy(np.ascontiguousarray(rot, dtype=np.float32)).cuda()
    Q, K, V = (torch.from_numpy(x).cuda() for x in (q, k, v))
    b = Buffers(p, want_fp16)
    ws = b.ws if use_ws else None
    if smooth:
        rotattn_smooth_stats(p, coef_dev, rot_dev, Q, K, V, b.ws)
    rotattn_prepare_qk(p, coef_dev, rot_dev, Q, K, b.Q4, b.Qs, b.K4, b.Ks, b.Q16, b.K16, ws)
    rotattn_quant_v(p, V, b.V4, b.Vs, ws)
    rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, ws_state_full(p) if use_ws else 0)
    out = dict(p=p, Q4=b.Q4, K4=b.K4, V4=b.V4, Qs=b.Qs, Ks=b.Ks, Vs=b.Vs, O=b.O, buffers=b, coef=tab, V=V)
    if want_fp16:
        rotattn_fwd_fp16(p, b.Q16, b.K16, V, b.O16, b.ws16)
        out.update(Q16=b.Q16, K16=b.K16, O16=b.O16)
    return out
