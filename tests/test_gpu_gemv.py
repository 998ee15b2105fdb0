"""GPU parity of decode_gemv against Oracle B: |gpu - c64| <= 1e-3 * sum_k |a_ik w_kj| per element
(BASELINE.json north_star), exact equality on structured cases.  Through the C ABI."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_29629_b200 as tri
from tests.tolerance import stated_bound, widened_bound
from synth_inputs import bf16_bits_to_f32, f32_to_bf16_bits, normal_bf16

pytestmark = pytest.mark.gpu

TOL = 1e-3   # BASELINE.json north_star: |err| <= 1e-3 * sum |a_ik * b_kj|


def to_dev(bits: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(bits.view(np.int16)).cuda()


def phys_w(w_logical_bits: np.ndarray, layout: int, ld_pad: int = 0) -> np.ndarray:
    """Logical W[k][n] bit patterns -> physical array in the requested layout, optionally row-padded."""
    p = np.ascontiguousarray(w_logical_bits.T if layout == tri.TRI_W_NK else w_logical_bits)
    if ld_pad:
        q = np.full((p.shape[0], p.shape[1] + ld_pad), 0x7FC0, np.uint16)   # NaN padding must never be read
        q[:, :p.shape[1]] = p
        p = q
    return p


def run_gemv(x_bits, w_phys, m, n, k, layout, ldx=None, ldw=None, pad_y=0):
    dx, dw = to_dev(x_bits), to_dev(w_phys)
    ldy = n + pad_y
    dy = torch.full((m, ldy), 0x7FC0, dtype=torch.int16, device="cuda")
    tri.decode_gemv(m, n, k, dx, ldx or x_bits.shape[1], dw, ldw or w_phys.shape[1], layout, dy, ldy)
    torch.cuda.synchronize()
    y = dy.cpu().numpy().view(np.uint16)
    if pad_y:
        assert (y[:, n:] == 0x7FC0).all(), "kernel wrote outside its n columns"
    return y[:, :n]


def check_against_oracle(y_bits, x_bits, w_phys_unpadded, layout, stated=False):
    """stated=True: the north_star bound as written (configured workload); else widened by the bf16 output
    half-ulp where that exceeds it (tests/tolerance.py)."""
    r = oracle.gemm_rows(x_bits, w_phys_unpadded, w_layout=layout)
    g = bf16_bits_to_f32(y_bits).astype(np.float64)
    assert np.isfinite(g).all()
    err = np.abs(g - r["c64"])
    bound = stated_bound(r["s64"]) if stated else widened_bound(r["c64"], r["s64"], x_bits.shape[1])
    worst = np.unravel_index(np.argmax(err - bound), err.shape)
    assert (err <= bound).all(), f"worst at {worst}: err {err[worst]:.3e} bound {bound[worst]:.3e}"
    return float((err / np.maximum(bound, 1e-300)).max())


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
def test_config3_full_output(layout):
    # BASELINE.json config 3: X [8 x 3584] ~ N(0,1), W [3584 x 18944] ~ N(0, 0.02), seed 2; full output
    m, k, n = 8, 3584, 18944
    x = normal_bf16(2, (m, k), 1.0, stream=0)
    w = normal_bf16(2, (k, n), 0.02, stream=1)
    wp = phys_w(w, layout)
    y = run_gemv(x, wp, m, n, k, layout)
    frac = check_against_oracle(y, x, wp, layout, stated=True)
    assert frac < 1.0


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
@pytest.mark.parametrize("m", [1, 2, 4, 5, 16])
def test_config3_shape_other_batch_sizes(layout, m):
    """The config-3 weight matrix at the other decode batch sizes: m = 1, 4 run the FHFMA kernels,
    m = 5 the warp-MMA kernel with zero-filled rows, m = 16 its two-tile form; full output, stated bound."""
    k, n = 3584, 18944
    x = normal_bf16(2, (m, k), 1.0, stream=7)
    w = normal_bf16(2, (k, n), 0.02, stream=1)
    wp = phys_w(w, layout)
    y = run_gemv(x, wp, m, n, k, layout)
    assert check_against_oracle(y, x, wp, layout, stated=True) < 1.0


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
@pytest.mark.parametrize("m", [1, 2, 4, 5, 8, 16])
def test_down_projection_shape_full_output(layout, m):
    """The Thinker MLP down-projection at decode batch sizes (18944 -> 3584): 56 column blocks, so the launch
    is a grid of 4-CTA clusters along K (gemv_impl picks 1, 2 or 4 ranks; 74 stages per rank through the 10-slot ring,
    partial sums through distributed shared memory); every kernel of both paths; full output, stated bound."""
    k, n = 18944, 3584
    x = normal_bf16(2, (m, k), 1.0, stream=8)
    w = normal_bf16(2, (k, n), 0.02, stream=9)
    wp = phys_w(w, layout)
    y = run_gemv(x, wp, m, n, k, layout)
    assert check_against_oracle(y, x, wp, layout, stated=True) < 1.0


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
@pytest.mark.parametrize("m", [1, 3, 4, 8, 11, 16])            # FHFMA kernels (1, 2, 4 rows) and the MMA kernel (1 and 2 batch tiles)
def test_identity_and_permutation_are_exact(layout, m):
    k = n = 256
    x = normal_bf16(21, (m, k))
    eye = f32_to_bf16_bits(np.eye(k, dtype=np.float32))
    assert (run_gemv(x, phys_w(eye, layout), m, n, k, layout) == x).all()
    pi = np.random.default_rng(3).permutation(k)
    wl = np.zeros((k, n), np.float32)
    wl[pi, np.arange(n)] = 1.0                                   # Y[:, j] = X[:, pi(j)]
    y = run_gemv(x, phys_w(f32_to_bf16_bits(wl), layout), m, n, k, layout)
    assert (y == x[:, pi]).all()


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
@pytest.mark.parametrize("m", [2, 8, 13])
@pytest.mark.parametrize("k", [16, 256, 3584])
def test_ones_give_k_exactly(layout, m, k):
    n = 136
    ones_x = np.full((m, k), 0x3F80, np.uint16)
    ones_w = np.full((k, n), 0x3F80, np.uint16)
    y = run_gemv(ones_x, phys_w(ones_w, layout), m, n, k, layout)
    assert (bf16_bits_to_f32(y) == float(k)).all()


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
@pytest.mark.parametrize("m,n,k", [(1, 8, 8), (7, 264, 80), (8, 1000, 136), (9, 129, 264), (16, 520, 4096),
                                   (3, 18944, 128), (8, 127, 3584), (2, 72, 18944), (4, 200, 8200), (5, 64, 64), (12, 65, 72),
                                   (5, 200, 4104), (8, 136, 8200), (6, 72, 18944), (13, 200, 4104), (16, 72, 8200), (10, 3, 24)])
def test_ragged_shapes(layout, m, n, k):
    x = normal_bf16(30 + m, (m, k))
    w = normal_bf16(31 + m, (k, n), 0.05)
    wp = phys_w(w, layout)
    pad = (-n) % 8 if layout == tri.TRI_W_KN else 0          # ldw must be a multiple of 8 elements
    wq = phys_w(w, layout, ld_pad=pad) if pad else wp
    y = run_gemv(x, wq, m, n, k, layout, ldw=wq.shape[1], pad_y=5)
    check_against_oracle(y, x, wp, layout)


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
def test_leading_dimensions(layout):
    m, n, k = 8, 392, 200
    x = normal_bf16(40, (m, k))
    w = normal_bf16(41, (k, n), 0.05)
    xp = np.full((m, k + 24), 0x7FC0, np.uint16)
    xp[:, :k] = x
    wp_unpadded = phys_w(w, layout)
    wp = phys_w(w, layout, ld_pad=16)
    y = run_gemv(xp, wp, m, n, k, layout, ldx=k + 24, ldw=wp.shape[1], pad_y=3)
    check_against_oracle(y, x, wp_unpadded, layout)


def test_bf16_accumulation_would_fail_the_bound():
    """The tolerance has teeth: the same product accumulated in bf16 (not allowed) violates it."""
    m, k, n = 8, 3584, 64
    x = normal_bf16(2, (m, k), 1.0, stream=0)
    w = normal_bf16(2, (k, n), 0.02, stream=1)
    r = oracle.gemm_rows(x, np.ascontiguousarray(w.T), w_layout=tri.TRI_W_NK)
    xt = torch.from_numpy(bf16_bits_to_f32(x)).bfloat16()
    wt = torch.from_numpy(bf16_bits_to_f32(w)).bfloat16()
    acc = torch.zeros(m, n, dtype=torch.bfloat16)
    for kk in range(k):
        acc = acc + xt[:, kk:kk + 1] * wt[kk:kk + 1, :]
    err = np.abs(acc.double().numpy() - r["c64"])
    assert (err > TOL * r["s64"]).any()
