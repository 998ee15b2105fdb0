"""Compile-time pin of what the kernels ARE (SURVEY.md §4 tier 2): the SASS of the built libtriroof.so, per kernel.
A refactor that silently compiled tcgen05 / TMA out, split the fused multiply-add or pulled a special-function call into
the FMA chain would pass every parity test; it fails here.  No GPU: cuobjdump reads the embedded sm_100a cubin.
profiles/r3_sass_summary.txt is the same histogram, written by `python -m paper_2606_29629_b200.sass_summary`."""
import pytest

from paper_2606_29629_b200.sass_summary import families, histograms


@pytest.fixture(scope="module")
def sass():
    return histograms()


def kernels(sass, prefix):
    out = {n: h for n, h in sass.items() if n.replace("void ", "").startswith("tri::" + prefix)}
    assert out, prefix
    return out


def test_kernel_set(sass):
    short = sorted({n.replace("void ", "").split("(")[0].split("<")[0] for n in sass})
    assert short == ["tri::fma_chain_kernel", "tri::gemm_1sm_kernel", "tri::gemm_2sm_kernel", "tri::gemv_kernel", "tri::gemv_mma_kernel",
                     "tri::sm_clock_probe", "tri::splitk_reduce_kernel"], short


def test_fma_chain_is_packed_fused_and_free_of_special_functions(sass):
    """a1: k dependent fused multiply-adds per element and nothing else that costs issue slots: FFMA2 (two chains
    per instruction) carries the loop; no MUFU; no separate FMUL / FADD (a split multiply-add would also break bit-exactness);
    128-bit global loads and stores."""
    ks = kernels(sass, "fma_chain_kernel")
    assert len(ks) == 4
    for name, h in ks.items():
        assert families(h, "FFMA2") >= 32, (name, h)
        assert families(h, "FFMA") - families(h, "FFMA2") <= 2, name        # the odd-k tail step
        for bad in ("MUFU", "FMUL", "FADD", "FMNMX", "DFMA"):      # (HFMA2 with RZ operands is how ptxas loads constants)
            assert families(h, bad) == 0, (name, bad)
        assert any(op.startswith("LDG") and ("128" in op or "256" in op) for op in h), (name, [op for op in h if op.startswith("LDG")])
        assert any(op.startswith("STG") and ("128" in op or "256" in op) for op in h), (name, [op for op in h if op.startswith("STG")])


def test_pair_gemm_is_tcgen05_with_tma_both_ways(sass):
    """a3: CTA-pair MMA on tensor memory, operands by multicast-aware TMA, accumulators read by tcgen05.ld,
    C stored by TMA."""
    (name, h), = kernels(sass, "gemm_2sm_kernel").items()
    assert h["UTCHMMA.2CTA"] >= 4, h
    assert h["UTMALDG.2D.2CTA"] >= 3
    assert families(h, "LDTM") >= 1 and families(h, "UTMASTG") >= 1
    assert families(h, "UTCBAR.2CTA") >= 1
    assert families(h, "HMMA") == 0 and families(h, "FFMA") == 0         # no warp-level MMA, no CUDA-core contraction


def test_one_cta_gemm_is_tcgen05(sass):
    (name, h), = kernels(sass, "gemm_1sm_kernel").items()
    assert h["UTCHMMA"] >= 4 and families(h, "LDTM") >= 1 and families(h, "UTMALDG.2D") >= 4 and families(h, "UTCBAR") >= 1
    assert families(h, "HMMA") == 0 and families(h, "FFMA") == 0


def test_gemv_kernels_stream_w_by_tma(sass):
    """a2: every GEMV variant takes W through the TMA ring; the 1-4 row kernels multiply on CUDA cores with the
    mixed-precision FMA (bf16 x bf16 + f32), the 5-32 row kernels with warp-level bf16 MMA, fp32 accumulate."""
    cc, mma = kernels(sass, "gemv_kernel"), kernels(sass, "gemv_mma_kernel")
    assert len(cc) == 6 and len(mma) == 6
    for name, h in cc.items():
        assert families(h, "UTMALDG.2D") >= 4 and families(h, "FHFMA.BF16") >= 64 and families(h, "HMMA") == 0, (name, h)
    for name, h in mma.items():
        assert families(h, "UTMALDG.2D") >= 4 and families(h, "HMMA.16816.F32.BF16") >= 4 and families(h, "FHFMA") == 0, (name, h)


def test_splitk_reduction_adds_in_fp32(sass):
    (name, h), = kernels(sass, "splitk_reduce_kernel").items()
    assert families(h, "FADD") >= 16 and families(h, "F2FP.BF16") + families(h, "F2FP") >= 1, h
