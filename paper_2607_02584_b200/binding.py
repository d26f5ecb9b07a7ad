"""ctypes binding of librotattn.so — same names as include/rotattn.h, argument marshalling only.
Every step of the path runs in the CUDA kernels; there is no Python/CPU fallback: a missing
library raises ImportError at import time."""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, 'librotattn.so')

ROT_NONE, ROT_INTERLEAVED, ROT_HALF, ROT_FULL = 0, 1, 2, 3
P_ASYM15, P_SYM7 = 0, 1
NORM_ROWBLOCK, NORM_RUNNING = 0, 1
WS_HAS_QK, WS_HAS_V, WS_HAS_STATS = 1, 2, 4
VSCALE_CHANNEL, VSCALE_GROUP = 0, 1
ABI_VERSION = 3                     # ROTATTN_ABI_VERSION this binding's struct layouts were written for
STATIC_WS_BYTES = 8 << 20          # ROTATTN_STATIC_WS_BYTES of include/rotattn.h


class RotattnParams(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ('B', 'H', 'N', 'D', 'grid_t', 'grid_h', 'grid_w',
                                         'pairs_t', 'pairs_h', 'pairs_w')] + \
               [('rope_base', C.c_float)] + \
               [(n, C.c_int32) for n in ('rot_mode', 'p_mode', 'p_norm', 'qk_group', 'v_group', 'kv_block', 'v_scale', 'smooth')]


class RotattnPolicy(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ('n_steps', 'n_blocks', 'first_steps', 'last_steps',
                                         'first_blocks', 'last_blocks', 'n_heads')] + \
               [('fp16_head_mask', C.POINTER(C.c_uint8))]


if not os.path.exists(LIB_PATH):
    raise ImportError(f'{LIB_PATH} is missing: run `python __graft_entry__.py` (nvcc, sm_100a). '
                      'There is no CPU fallback.')
lib = C.CDLL(LIB_PATH)

_P = C.POINTER(RotattnParams)
_vp, _sz, _i32 = C.c_void_p, C.c_size_t, C.c_int32
EXPORTS = {
    'rotattn_abi_version': (C.c_int, []),
    'rotattn_validate': (C.c_int, [_P]),
    'rotattn_table_floats': (_sz, [_P]),
    'rotattn_build_tables': (C.c_int, [_P, _vp, _vp]),
    'rotattn_workspace_bytes': (_sz, [_P, C.c_int]),
    'rotattn_policy_select': (C.c_int, [C.POINTER(RotattnPolicy), _i32, _i32, _i32]),
    'rotattn_policy_split_heads': (C.c_int, [C.POINTER(RotattnPolicy), _i32, _i32, _i32, _i32, _vp, _vp, _vp, _vp]),
    'rotattn_strerror': (C.c_char_p, [C.c_int]),
    'rotattn_last_cuda_error': (C.c_char_p, []),
    'rotattn_prepare_qk': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    'rotattn_quant_v': (C.c_int, [_P, _vp, _vp, _vp, _vp, _sz, _vp]),
    'rotattn_fwd_int4': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _i32, _vp, _sz, _i32, _vp]),
    'rotattn_fwd_int4_static': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _i32, _vp]),
    'rotattn_smooth_stats': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    'rotattn_smooth_read': (C.c_int, [_P, _vp, _sz, _vp, _vp, _vp]),
    'rotattn_fwd_int4_debug': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _vp, _i32, _i32, _vp, _vp, _vp, _vp, _vp, _sz, _i32, _vp]),
    'rotattn_fwd_fp16': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _i32, _vp, _sz, _vp]),
    'rotattn_fwd_fp16_debug_f32': (C.c_int, [_P, _vp, _vp, _vp, _vp, _vp, _i32, _vp, _sz, _vp]),
    'rotattn_probe_gemm8': (C.c_int, [_i32, _i32, _i32, _vp, _vp, _vp, _i32, _vp]),
}
for _name, (_res, _args) in EXPORTS.items():
    _fn = getattr(lib, _name)          # AttributeError here = the library does not export a declared symbol
    _fn.restype = _res
    _fn.argtypes = _args


if lib.rotattn_abi_version() != ABI_VERSION:
    raise ImportError(f'{LIB_PATH} speaks ABI version {lib.rotattn_abi_version()}, this binding was written for {ABI_VERSION}: '
                      'rebuild with `python __graft_entry__.py`')


class RotattnError(RuntimeError):
    pass


def check(status: int, what: str):
    if status != 0:
        msg = lib.rotattn_strerror(status).decode()
        extra = lib.rotattn_last_cuda_error().decode()
        raise RuntimeError(f'{what}: {msg} ({status}) {extra}')


def make_params(B, H, N, D, grid, pairs, rope_base=10000.0, rot_mode=ROT_HALF, p_mode=P_ASYM15,
                p_norm=NORM_ROWBLOCK, qk_group=1, v_group=128, kv_block=128, v_scale=VSCALE_CHANNEL,
                smooth=0) -> RotattnParams:
    return RotattnParams(B, H, N, D, grid[0], grid[1], grid[2], pairs[0], pairs[1], pairs[2], rope_base,
                         rot_mode, p_mode, p_norm, qk_group, v_group, kv_block, v_scale, smooth)
