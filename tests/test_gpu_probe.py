"""GPU check of the tcgen05 8-bit GEMM probe (validates the descriptor / TMEM layouts the attention
kernels rely on) against torch integer matmul on the CPU."""
import numpy as np
import pytest

torch = pytest.importorskip('torch')
pytestmark = pytest.mark.gpu

import __graft_entry__ as entry  # noqa: E402

entry.build()


def _api():
    from paper_2607_02584_b200 import api
    return api


def test_probe_i8_ss_small_and_multi_tile():
    api = _api()
    rng = np.random.default_rng(0)
    for (M, N, K) in [(128, 256, 128), (384, 512, 640)]:
        a = rng.integers(-128, 128, (M, K)).astype(np.int8)
        b = rng.integers(-128, 128, (N, K)).astype(np.int8)
        A, B = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        C = torch.zeros((M, N), dtype=torch.int32, device='cuda')
        api.rotattn_probe_gemm8(M, N, K, A, B, C, 0)
        torch.cuda.synchronize()
        want = a.astype(np.int64) @ b.astype(np.int64).T
        assert np.array_equal(C.cpu().numpy().astype(np.int64), want)


def test_probe_i8_tmem_a_unsigned():
    api = _api()
    rng = np.random.default_rng(1)
    a = rng.integers(0, 256, (128, 128)).astype(np.uint8)     # unsigned A through tensor memory
    b = rng.integers(-128, 128, (128, 128)).astype(np.int8)
    A, B = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    C = torch.zeros((128, 128), dtype=torch.int32, device='cuda')
    api.rotattn_probe_gemm8(128, 128, 128, A, B, C, 2)
    torch.cuda.synchronize()
    want = a.astype(np.int64) @ b.astype(np.int64).T
    assert np.array_equal(C.cpu().numpy().astype(np.int64), want)


def test_probe_e4m3_integer_valued_exact():
    """Integer-valued E4M3 operands (|x| <= 15) through kind::f8f6f4: are the fp32 accumulators integer-exact?
    Reported (xfail-free): the attention kernel uses kind::i8 regardless; this documents the alternative."""
    api = _api()
    rng = np.random.default_rng(2)
    M, N, K = 128, 256, 128
    a = rng.integers(0, 16, (M, K)).astype(np.float32)        # P codes 0..15
    b = rng.integers(-7, 8, (N, K)).astype(np.float32)        # V codes
    a[0, :] = 15.0
    b[0, :] = 7.0                                             # worst case 13440
    A = torch.from_numpy(a).cuda().to(torch.float8_e4m3fn).view(torch.uint8)
    B = torch.from_numpy(b).cuda().to(torch.float8_e4m3fn).view(torch.uint8)
    C = torch.zeros((M, N), dtype=torch.float32, device='cuda')
    api.rotattn_probe_gemm8(M, N, K, A, B, C, 1)
    torch.cuda.synchronize()
    want = a.astype(np.float64) @ b.astype(np.float64).T
    got = C.cpu().numpy().astype(np.float64)
    assert got[0, 0] == 13440.0
    assert np.array_equal(got, want)
