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


def _code_byte(c):
    """Operand byte of an integer code c in [-15, 15]: sign-magnitude = the E4M3 bit pattern of c * 2^-9 (E4M3
    subnormals are m * 2^-9, bytes 8..15 the first normal binade) -- the encoding the attention kernels feed to
    tcgen05 kind::f8f6f4.  Written out here independently of the library."""
    c = np.asarray(c, dtype=np.int32)
    return (np.abs(c) | np.where(c < 0, 0x80, 0)).astype(np.uint8)


def _gemm_codes(a_codes, b_codes):
    """C = A B^T through rotattn_probe_gemm8 mode 1 (kind::f8f6f4, fp32 accumulators) on code bytes; returns the
    accumulators rescaled by 2^18 as float64 (exact if and only if the tensor core kept every integer)."""
    api = _api()
    M, K = a_codes.shape
    N = b_codes.shape[0]
    A = torch.from_numpy(_code_byte(a_codes)).cuda()
    B = torch.from_numpy(_code_byte(b_codes)).cuda()
    C = torch.zeros((M, N), dtype=torch.float32, device='cuda')
    api.rotattn_probe_gemm8(M, N, K, A, B, C, 1)
    torch.cuda.synchronize()
    return C.cpu().numpy().astype(np.float64) * 2.0 ** 18


def _exact(a_codes, b_codes):
    return (a_codes.astype(np.int64) @ b_codes.astype(np.int64).T).astype(np.float64)


def test_e4m3_code_bytes_decode_to_codes():
    """The byte really is the E4M3 pattern of c * 2^-9 (library decode of the bit pattern, no GPU arithmetic)."""
    c = np.arange(-15, 16)
    dec = torch.from_numpy(_code_byte(c)).view(torch.float8_e4m3fn).float().numpy().astype(np.float64)
    assert np.array_equal(dec * 512.0, c.astype(np.float64))


def test_probe_e4m3_code_bytes_worst_case_magnitude():
    """All-maximum rows on the encoding the kernels use: S worst case 49 * 128 = 6272, P~V worst case 15 * 7 * 128 = 13440."""
    K = 128
    a = np.zeros((128, K), dtype=np.int32)
    b = np.zeros((256, K), dtype=np.int32)
    a[0], a[1], a[2], a[3] = 7, -7, 15, 15
    b[0], b[1], b[2] = 7, -7, 7 * (-1) ** np.arange(K)
    got = _gemm_codes(a, b)
    assert got[0, 0] == 6272 and got[0, 1] == -6272 and got[1, 1] == 6272
    assert got[2, 0] == 13440 and got[2, 1] == -13440 and got[2, 2] == 0
    assert np.array_equal(got, _exact(a, b))


@pytest.mark.parametrize('big', [(7, 7), (15, 7), (15, -7), (-7, 7)])
def test_probe_e4m3_unit_product_on_a_saturated_running_sum(big):
    """Maximum DYNAMIC RANGE: 127 products of maximum magnitude and one +-1-unit product, the unit product at every one
    of the 128 K positions (inside a K=32 MMA and across the four chained ones): row i has its unit at position i.
    A limited-width alignment of the addends to the running maximum would lose the unit."""
    K = 128
    pa, pb = big
    for unit in (1, -1):
        a = np.full((128, K), pa, dtype=np.int32)
        b = np.full((256, K), pb, dtype=np.int32)
        a[np.arange(128), np.arange(128)] = 1
        b[:128][np.arange(128), np.arange(128)] = unit          # column j < 128: unit factor at position j
        want = _exact(a, b)
        assert want[5, 5] == pa * pb * 127 + unit
        got = _gemm_codes(a, b)
        assert np.array_equal(got, want), np.abs(got - want).max()


def test_probe_e4m3_alternating_sign_cancellation_and_prefix_patterns():
    """Large running sums that cancel to a few units; big-then-small and small-then-big orderings along K."""
    K = 128
    rng = np.random.default_rng(21)
    a = np.zeros((256, K), dtype=np.int32)
    b = np.zeros((256, K), dtype=np.int32)
    sgn = (-1) ** np.arange(K)
    for i in range(256):
        kind = i % 4
        if kind == 0:                     # +105, -105, ... with a sprinkle of unit codes
            a[i] = 15
            b[i] = 7 * sgn
            idx = rng.choice(K, 9, replace=False)
            b[i, idx] = rng.choice([-1, 1], 9)
        elif kind == 1:                   # first 96 positions saturated, last 32 (one MMA) units
            a[i, :96], b[i, :96] = 15, 7
            a[i, 96:], b[i, 96:] = 1, rng.choice([-1, 1], 32)
        elif kind == 2:                   # units first, saturation last
            a[i, :32], b[i, :32] = 1, rng.choice([-1, 1], 32)
            a[i, 32:], b[i, 32:] = 15, -7
        else:                             # saturated positive half against saturated negative half, units interleaved
            a[i] = np.where(np.arange(K) % 8 == 3, 1, 15)
            b[i] = np.where(np.arange(K) < 64, 7, -7)
    got = _gemm_codes(a, b)               # every row of a against every row of b: 65536 mixed patterns
    assert np.array_equal(got, _exact(a, b))


def test_probe_e4m3_random_code_rows_full_range():
    """>= 10^4 random code rows from the full ranges: P codes [0,15] x V codes [-7,7] and Q codes x K codes [-7,7]^2."""
    rng = np.random.default_rng(22)
    K = 128
    for lo, hi, rows in ((0, 16, 10240), (-7, 8, 10240)):
        a = rng.integers(lo, hi, (rows, K)).astype(np.int32)
        b = rng.integers(-7, 8, (512, K)).astype(np.int32)
        # skewed rows too: mostly saturated codes, so that sums are large while addends vary
        a[::3] = np.where(rng.random((len(a[::3]), K)) < 0.9, hi - 1, a[::3])
        b[::2] = np.where(rng.random((256, K)) < 0.9, 7, b[::2])
        got = _gemm_codes(a, b)
        assert np.array_equal(got, _exact(a, b))


def test_probe_e4m3_integer_valued_exact():
    """Integer-valued normal E4M3 operands (|x| <= 15, torch's own float8 cast) through kind::f8f6f4."""
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
