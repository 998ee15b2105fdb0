"""The register-file property the GEMV design rests on, measured through tri_probe_fma_issue:
an FHFMA.BF16 issues every cycle when it fetches one register, every ~2 cycles when it fetches two registers of the
same parity, ~1.5 when that happens on every other instruction.  Asserted loosely (ordering and rough size)."""
import pytest

import paper_2606_29629_b200 as tri

pytestmark = pytest.mark.gpu


def test_fhfma_issue_cost_depends_on_register_fetches():
    tri.tri_init(0)
    mhz = tri.tri_sm_clock_mhz(2000)
    c = [tri.tri_probe_fma_issue(p, mhz) for p in (0, 1, 2)]
    print("cycles per FHFMA by pattern:", c, "at", mhz, "MHz")
    assert 0.9 < c[0] < 1.4, c             # 8 FMAs + loop overhead per iteration: ~1.1
    assert 1.6 < c[1] < 2.6, c             # two same-parity registers per FMA: ~2.05
    assert c[0] < c[2] < c[1], c           # every other FMA conflicts: ~1.5


def test_probe_argument_errors():
    with pytest.raises(tri.TriError):
        tri.tri_probe_fma_issue(3, 1965.0)
    with pytest.raises(tri.TriError):
        tri.tri_probe_fma_issue(0, 0.0)
