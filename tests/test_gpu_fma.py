"""GPU parity of the FMA-chain roofline kernel against Oracle A: BIT-EXACT (BASELINE.json north_star;
SURVEY.md §8(c)).  Calls go through the C ABI (roofline_run / roofline_run_k)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_29629_b200 as tri
from synth_inputs import uniform_pm1, uniform_pm1_torch

pytestmark = pytest.mark.gpu


def run_gpu(x: np.ndarray, k: int, a=None, b=None, inplace=False) -> np.ndarray:
    d_in = torch.from_numpy(x).cuda()
    d_out = d_in if inplace else torch.full_like(d_in, float("nan"))
    if a is None:
        tri.roofline_run(k / 4.0, x.size, d_in, d_out)
    else:
        tri.roofline_run_k(k, a, b, x.size, d_in, d_out)
    torch.cuda.synchronize()
    return d_out.cpu().numpy()


def assert_bits_equal(got, want):
    bad, first = oracle.count_bit_mismatches(got, want)
    assert bad == 0, f"{bad} mismatching bit patterns, first at {first}: got {got[first]!r} want {want[first]!r}"


@pytest.mark.parametrize("k", [1, 4, 16, 64])
def test_config1_bit_exact(k):
    # BASELINE.json config 1: N = 2^20, seed 0, k in {1, 4, 16, 64}
    x = uniform_pm1(0, 1 << 20)
    assert_bits_equal(run_gpu(x, k), oracle.fma_chain(x, k))


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 7, 1023, 1024, 4096, 4097, 4099, 256 * 16 * 3 + 2, 100003])
@pytest.mark.parametrize("k", [1, 7, 9, 33, 100])
def test_ragged_sizes_and_odd_k(n, k):
    # tails (n % 4 != 0), partial tiles, k that is neither a power of two nor a multiple of the unroll
    x = uniform_pm1(5, n, stream=3)
    got = run_gpu(x, k)
    assert_bits_equal(got, oracle.fma_chain(x, k))


def test_in_place_and_untouched_neighbours():
    n = 70001
    x = uniform_pm1(6, n)
    assert_bits_equal(run_gpu(x, 12, inplace=True), oracle.fma_chain(x, 12))
    # the kernel writes exactly n elements: a guard band after the output stays intact
    d_in = torch.from_numpy(x).cuda()
    d_out = torch.full((n + 64,), 7.0, device="cuda")
    tri.roofline_run(3.0, n, d_in, d_out)
    torch.cuda.synchronize()
    assert (d_out[n:] == 7.0).all()


def test_empty_input_is_a_no_op():
    d = torch.ones(16, device="cuda")
    tri.roofline_run(1.0, 0, d, d)
    tri.roofline_run(1.0, 0, None, None)
    torch.cuda.synchronize()
    assert (d == 1.0).all()


def test_other_constants_and_special_values():
    # roofline_run_k with a, b that are not the config-1 pair; inputs include 0, -0, the fixed point 1,
    # subnormals and large values: fused single rounding must hold everywhere (no FTZ, no fast-math)
    x = np.concatenate([uniform_pm1(7, 5000),
                        np.array([0.0, -0.0, 1.0, -1.0, 1e-40, -1e-40, 1.17549435e-38, 3e38, -3e38, 65504.0], np.float32)])
    for a, b in [(0.5, 0.25), (-0.75, 1e-3), (1.0000001, -1e-7), (0.33333334, 1e-39)]:
        a32, b32 = np.float32(a), np.float32(b)
        got = run_gpu(x, 11, float(a32), float(b32))
        assert_bits_equal(got, oracle.fma_chain(x, 11, a32, b32))


def test_fixed_point_and_worked_values():
    # pins that do not go through the oracle: y0 = 1 is a fixed point; SURVEY §8(c) worked values
    x = np.array([1.0, -1.0, 0.0, 0.5, -0.5, 0.25] + [1.0] * 10, np.float32)
    got = run_gpu(x, 64).view(np.uint32)
    assert got[0] == 0x3F800000
    assert list(got[1:6]) == [0xBF60F6FF, 0x3D784819, 0x3F07C240, 0xBED17279, 0x3E9746C0]
    got = run_gpu(x, 4096).view(np.uint32)
    assert list(got[:6]) == [0x3F800000, 0x3F76A400, 0x3F7B5204, 0x3F7DA903, 0x3F78FB0E, 0x3F7C7D82]


@pytest.mark.parametrize("k", [1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096, 100, 200, 400, 800])
def test_config2_full_size_sampled_blocks(k):
    """BASELINE.json config 2 at full size (N = 2^28, seed 1) in the launch configuration bench.py times;
    every k of the sweep and of the paper's A.I. set; the oracle checks the first and last 2^16-element blocks and 14
    seeded blocks (6 for k > 512), plus the closed-form
    bound 2^-15 (1 - a^k) on a strided sample of the whole output (SURVEY §8(c) pin 2)."""
    n = 1 << 28
    d_in = uniform_pm1_torch(1, n, device="cuda")
    d_out = torch.empty_like(d_in)
    tri.roofline_run(k / 4.0, n, d_in, d_out)
    torch.cuda.synchronize()
    blk = 1 << 16
    nblk = n // blk
    rng = np.random.default_rng(1234 + k)
    blocks = [0, nblk - 1] + list(rng.integers(1, nblk - 1, 14 if k <= 512 else 6))
    for bi in blocks:
        lo = int(bi) * blk
        x = uniform_pm1(1, blk, start=lo)
        assert (d_in[lo:lo + blk].cpu().numpy().view(np.uint32) == x.view(np.uint32)).all()   # device generator == host generator
        assert_bits_equal(d_out[lo:lo + blk].cpu().numpy(), oracle.fma_chain(x, k))
    y0 = d_in[::4099].double().cpu().numpy()
    y = d_out[::4099].double().cpu().numpy()
    a = 1.0 - 2.0 ** -10
    exact = 1.0 + a ** k * (y0 - 1.0)
    assert np.abs(y - exact).max() <= 2.0 ** -15 * (1.0 - a ** k) + 1e-12
