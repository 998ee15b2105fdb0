"""Race / ordering stress of the asynchronous paths, in place of compute-sanitizer (closed on this pool: profiles/r2_sanitizer.md).
What a race in the mbarrier / TMEM / TMA-store / split-K code would show as is run-to-run variation or a stale tile, so every
case here runs a kernel many times back to back with no host synchronisation in between, into NaN-prefilled outputs, and
demands that every repetition is bit-identical to the first and that the first is within the oracle's bound."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_29629_b200 as tri
from synth_inputs import bf16_bits_to_f32, normal_bf16
from tests.tolerance import widened_bound

pytestmark = pytest.mark.gpu
NAN16 = 0x7FC0


def dev(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda()


def within_bound(c_bits, a, wp, layout):
    r = oracle.gemm_rows(a, wp, w_layout=layout)
    g = bf16_bits_to_f32(c_bits).astype(np.float64)
    assert np.isfinite(g).all()
    assert (np.abs(g - r["c64"]) <= widened_bound(r["c64"], r["s64"], a.shape[1])).all()


@pytest.mark.parametrize("m,n,k", [(300, 129, 512),     # pair kernel; column groups 2, 3 of the only tile store nothing (ADVICE: bulk-group count)
                                   (257, 136, 256),     # second row block almost empty: whole warps skip their stores
                                   (520, 1096, 640),    # 3 x 5 tiles, ragged in both directions, two tiles per pair never happens: one round
                                   (1536, 4352, 448),   # 204 tiles: three rounds, both accumulators, ring wrap-arounds
                                   (300, 704, 2048),    # pair kernel, every tile cut 12 ways + reduction kernel under PDL
                                   (64, 3584, 2048),    # one-CTA kernel, 28 tiles cut 5 ways
                                   (100, 1000, 256)])   # one-CTA kernel, whole tiles
def test_gemm_back_to_back_is_bit_stable(m, n, k):
    a, w = normal_bf16(95, (m, k)), normal_bf16(96, (k, n), 0.05)
    wp = np.ascontiguousarray(w.T)
    da, dw = dev(a), dev(wp)
    reps, ldc = 24, (n + 7) // 8 * 8
    outs = [torch.full((m, ldc), NAN16, dtype=torch.int16, device="cuda") for _ in range(reps)]
    for c in outs:                                        # no synchronisation between the calls
        tri.prefill_gemm(m, n, k, da, k, dw, k, tri.TRI_W_NK, c, ldc)
    torch.cuda.synchronize()
    first = outs[0].cpu().numpy().view(np.uint16)
    assert (first[:, n:] == NAN16).all(), "kernel wrote outside its n columns"
    within_bound(first[:, :n], a, wp, tri.TRI_W_NK)
    for i, c in enumerate(outs[1:], 1):
        assert torch.equal(c, outs[0]), f"repetition {i} differs from the first"


@pytest.mark.parametrize("layout", [tri.TRI_W_NK, tri.TRI_W_KN])
@pytest.mark.parametrize("m,n,k", [(8, 1000, 3584), (3, 520, 4104), (16, 264, 8200), (1, 18944, 512)])
def test_gemv_back_to_back_under_pdl_is_bit_stable(layout, m, n, k):
    """decode_gemv launches with programmatic stream serialization: call i + 1 prefetches W while call i drains.  X and Y are
    touched only after the previous grid completed; alternating two weight matrices and 32 outputs checks exactly that."""
    x = normal_bf16(97, (m, k))
    ws = [normal_bf16(98 + j, (k, n), 0.05) for j in range(2)]
    wps = [np.ascontiguousarray(w.T if layout == tri.TRI_W_NK else w) for w in ws]
    ldw = wps[0].shape[1]
    if ldw % 8:                                           # TRI_W_KN with ragged n: pad the rows
        pad = (-ldw) % 8
        wps = [np.concatenate([p, np.full((p.shape[0], pad), NAN16, np.uint16)], axis=1) for p in wps]
        ldw += pad
    dx, dws = dev(x), [dev(p) for p in wps]
    reps = 32
    outs = [torch.full((m, n), NAN16, dtype=torch.int16, device="cuda") for _ in range(reps)]
    for i, y in enumerate(outs):
        tri.decode_gemv(m, n, k, dx, k, dws[i & 1], ldw, layout, y, n)
    torch.cuda.synchronize()
    for j in range(2):
        ref = outs[j].cpu().numpy().view(np.uint16)
        within_bound(ref, x, np.ascontiguousarray(wps[j][:, :(k if layout == tri.TRI_W_NK else n)]), layout)
        for i in range(j + 2, reps, 2):
            assert torch.equal(outs[i], outs[j]), f"call {i} differs from call {j}"


def test_gemv_then_gemm_then_gemv_chain():
    """The bench step's order: PDL-launched GEMVs around a (split) GEMM and its reduction kernel on one stream."""
    m, n, k = 8, 1096, 2048
    x, w = normal_bf16(101, (m, k)), normal_bf16(102, (k, n), 0.05)
    a = normal_bf16(103, (300, k))
    wp = np.ascontiguousarray(w.T)
    dx, dw, da = dev(x), dev(wp), dev(a)
    ys = [torch.full((m, n), NAN16, dtype=torch.int16, device="cuda") for _ in range(12)]
    cs = [torch.full((300, n), NAN16, dtype=torch.int16, device="cuda") for _ in range(6)]
    for i in range(6):
        tri.decode_gemv(m, n, k, dx, k, dw, k, tri.TRI_W_NK, ys[2 * i], n)
        tri.prefill_gemm(300, n, k, da, k, dw, k, tri.TRI_W_NK, cs[i], n)       # 2 x 5 tiles < 74 pairs: split, reduction kernel
        tri.decode_gemv(m, n, k, dx, k, dw, k, tri.TRI_W_NK, ys[2 * i + 1], n)
    torch.cuda.synchronize()
    within_bound(ys[0].cpu().numpy().view(np.uint16), x, wp, tri.TRI_W_NK)
    within_bound(cs[0].cpu().numpy().view(np.uint16), a, wp, tri.TRI_W_NK)
    assert all(torch.equal(y, ys[0]) for y in ys) and all(torch.equal(c, cs[0]) for c in cs)


@pytest.mark.parametrize("m,n", [(16, 1024), (100, 640), (128, 2048), (300, 768), (1000, 512)])
def test_short_gemm_chain_orders_its_data_under_pdl(m, n):
    """prefill_gemm launches with programmatic stream serialization (GEMV kernels for m <= 32, the one-CTA kernel to 128 rows,
    the CTA-pair kernel with its tail split and reduction kernel above): call i + 1 starts (and, for m <= 128, prefetches W) while
    call i drains, but may read A only after call i completed.  Here A of call i + 1 IS the output of call i (k = n, a
    permutation-like W keeps the values bounded): C_{i+1} = C_i . W.  The chain without any host synchronisation must equal,
    bit for bit, the same chain with a synchronisation after every call."""
    k = n
    a0 = normal_bf16(111, (m, k))
    pi = np.random.default_rng(7).permutation(k)
    wl = np.zeros((k, n), np.float32)
    wl[pi, np.arange(n)] = 1.0
    wl[(pi + 1) % k, np.arange(n)] = -0.5                       # two terms per output: not a pure copy
    from synth_inputs import f32_to_bf16_bits
    dw = dev(np.ascontiguousarray(f32_to_bf16_bits(wl).T))
    depth = 12

    def chain(sync):
        bufs = [dev(a0)] + [torch.full((m, n), NAN16, dtype=torch.int16, device="cuda") for _ in range(depth)]
        for i in range(depth):
            tri.prefill_gemm(m, n, k, bufs[i], k, dw, k, tri.TRI_W_NK, bufs[i + 1], n)
            if sync:
                torch.cuda.synchronize()
        torch.cuda.synchronize()
        return bufs

    ref, got = chain(True), chain(False)
    first = ref[1].cpu().numpy().view(np.uint16)
    within_bound(first, a0, np.ascontiguousarray(f32_to_bf16_bits(wl).T), tri.TRI_W_NK)
    assert not torch.equal(ref[depth], ref[1])
    for i in range(1, depth + 1):
        assert torch.equal(got[i], ref[i]), f"link {i} of the unsynchronised chain differs"


def test_shutdown_then_reuse():
    """tri_shutdown() frees what the library allocated (split-K workspaces, the clock-probe scratch, NVML) and the next call
    re-initialises lazily: the same calls give the same bits before and after, and NVML sampling comes back."""
    m, n, k = 64, 392, 2048                                  # one-CTA kernel, 4 tiles cut along K: needs the workspace
    a, w = normal_bf16(121, (m, k)), normal_bf16(122, (k, n), 0.05)
    wp = np.ascontiguousarray(w.T)
    da, dw = dev(a), dev(wp)
    x = normal_bf16(123, (8, k))
    dx = dev(x)

    def once():
        c = torch.full((m, n), NAN16, dtype=torch.int16, device="cuda")
        y = torch.full((8, n), NAN16, dtype=torch.int16, device="cuda")
        tri.prefill_gemm(m, n, k, da, k, dw, k, tri.TRI_W_NK, c, n)
        tri.decode_gemv(8, n, k, dx, k, dw, k, tri.TRI_W_NK, y, n)
        mhz = tri.tri_sm_clock_mhz(200)
        torch.cuda.synchronize()
        return c, y, mhz

    c0, y0, mhz0 = once()
    within_bound(c0.cpu().numpy().view(np.uint16), a, wp, tri.TRI_W_NK)
    tri.tri_shutdown()
    tri.tri_shutdown()                                       # idempotent
    c1, y1, mhz1 = once()
    assert torch.equal(c0, c1) and torch.equal(y0, y1)
    assert 500 < mhz0 < 2200 and 500 < mhz1 < 2200
    assert tri.tri_nvml_sample(0)["sm_mhz"] > 0
    assert tri.sm_count() == 148 or tri.sm_count() > 0


def test_calls_are_capturable_in_a_cuda_graph():
    """Every compute call enqueues kernels only (tensor maps are host-encoded kernel parameters, the split-K workspace of a
    stream is allocated on that stream's first split call), so after one warm-up step on the capture stream a step can be
    captured in a CUDA graph — programmatic dependent launches, the reduction kernel and the K-split clusters included — and
    the replay gives the bits of the eager step."""
    n_f = (1 << 20) + 3
    x = torch.from_numpy(np.random.default_rng(3).uniform(-1, 1, n_f).astype(np.float32)).cuda()
    y = torch.empty_like(x)
    gx, gw = dev(normal_bf16(131, (8, 3584))), dev(np.ascontiguousarray(normal_bf16(132, (3584, 520), 0.05).T))   # K-split cluster launch
    gy = torch.empty((8, 520), dtype=torch.int16, device="cuda")
    pa, pw = dev(normal_bf16(133, (300, 2048))), dev(np.ascontiguousarray(normal_bf16(134, (2048, 704), 0.05).T))  # pair kernel, tail split
    pc = torch.empty((300, 704), dtype=torch.int16, device="cuda")
    sa, sw = dev(normal_bf16(135, (64, 2048))), dev(np.ascontiguousarray(normal_bf16(136, (2048, 392), 0.05).T))   # one-CTA kernel, split, PDL
    sc = torch.empty((64, 392), dtype=torch.int16, device="cuda")

    def step():
        tri.roofline_run(6.0, n_f, x, y)
        tri.prefill_gemm(300, 704, 2048, pa, 2048, pw, 2048, tri.TRI_W_NK, pc, 704)
        tri.prefill_gemm(64, 392, 2048, sa, 2048, sw, 2048, tri.TRI_W_NK, sc, 392)
        for _ in range(3):
            tri.decode_gemv(8, 520, 3584, gx, 3584, gw, 3584, tri.TRI_W_NK, gy, 520)

    outs = (y, pc, sc, gy)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        step()
        s.synchronize()
        ref = [t.clone() for t in outs]
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            step()
        for t in outs:
            t.zero_()
        g.replay()
        g.replay()
        s.synchronize()
    for a, b in zip(ref, outs):
        assert torch.equal(a, b)


_W_PRODUCER_SCRIPT = r"""
import numpy as np, torch
import paper_2606_29629_b200 as tri
from synth_inputs import normal_bf16

def dev(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda()

k, n = 3584, 4608
srcs = [dev(np.ascontiguousarray(normal_bf16(130 + i, (k, n), 0.03).T)) for i in range(2)]     # physical [n][k]
w = torch.zeros_like(srcs[0])
for m, fn in ((8, tri.decode_gemv), (64, tri.prefill_gemm), (300, tri.prefill_gemm)):
    x = dev(normal_bf16(140 + m, (m, k)))
    want = []
    for s in srcs:                                   # the product for each W, computed with everything synchronised
        w.copy_(s); torch.cuda.synchronize()
        y = torch.zeros((m, n), dtype=torch.int16, device="cuda")
        fn(m, n, k, x, k, w, k, tri.TRI_W_NK, y, n); torch.cuda.synchronize()
        want.append(y.clone())
    assert not torch.equal(want[0], want[1])
    outs = []
    for it in range(24):                             # W rewritten by a plain kernel DIRECTLY before each call, no sync anywhere
        y = torch.full((m, n), 0x7FC0, dtype=torch.int16, device="cuda")
        w.copy_(srcs[it & 1])
        fn(m, n, k, x, k, w, k, tri.TRI_W_NK, y, n)
        outs.append(y)
    torch.cuda.synchronize()
    for it, y in enumerate(outs):
        assert torch.equal(y, want[it & 1]), (m, it, int((y != want[it & 1]).sum()))
print("ok")
"""


def test_w_written_by_the_preceding_kernel_with_pdl_off():
    """include/triroof.h, decode_gemv: with the environment's TRI_PDL=0 the kernels are launched without programmatic
    stream serialization, so a W produced by the kernel directly before the call (here a device-to-device copy kernel,
    alternating between two weight matrices, 24 calls with no synchronisation) is the W the call reads.  The variable is
    read once per process, hence the subprocess."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, TRI_PDL="0", PYTHONPATH=root + os.pathsep + os.environ.get("PYTHONPATH", ""))
    r = subprocess.run([sys.executable, "-c", _W_PRODUCER_SCRIPT], cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.strip().endswith("ok"), (r.stdout[-500:], r.stderr[-3000:])
