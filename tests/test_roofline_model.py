"""Host logic of the measurement: the byte model and the paper's own lower bounds."""
import os

import pytest

from paper_2401_09843_b200 import roofline as rf

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_table2.txt")


def golden():
    out = {}
    for line in open(GOLDEN):
        line = line.strip()
        if line and not line.startswith("#"):
            k, *v = line.split()
            out[k] = [float(x) for x in v]
    return out


def test_paper_table2_lower_bounds_reproduced():
    """Reading A16: with s = sizeof(float) = 4, eq. (5.1)-(5.3) and Table 1 give Table 2's t_opt column."""
    g = golden()
    N, p, s = int(g["N"][0]), int(g["p"][0]), int(g["scalar_bytes"][0])
    GB = 1e9
    ms = 1e3
    assert rf.paper_t_pad(N, p, s, g["beta_D"][0] * GB) * ms == pytest.approx(g["pad_topt_ms"][0], abs=5e-4)
    assert rf.paper_t_unpad(N, p, s, g["beta_D"][0] * GB) * ms == pytest.approx(g["unpad_topt_ms"][0], abs=5e-4)
    for key, comps in (("transpose_u_topt_ms", 3), ("transpose_B_topt_ms", 6)):
        t9 = comps * rf.paper_t_transpose(N, p, s, g["beta_D"][0] * GB, g["beta_HD"][0] * GB, g["beta_MPI"][0] * GB) * ms
        t4 = comps * rf.paper_t_transpose(N, p, s, g["beta_D"][0] * GB, g["beta_HD"][0] * GB, g["beta_MPI_alltoall"][0] * GB) * ms
        assert t9 == pytest.approx(g[key][0], abs=2e-3)
        assert t4 == pytest.approx(g[key][1], abs=2e-3)
    # the other reading (s = hyperviscosity order 1) is off by 4x
    assert rf.paper_t_pad(N, p, 1, g["beta_D"][0] * GB) * ms < 0.3 * g["pad_topt_ms"][0]


def test_model_bytes_match_survey_table():
    # 6.61 / 52.8 / 211.6 / 422.3 GB per fp64 step, 211.1 GB fp32 at 512^3
    assert rf.step_bytes(128) / 1e9 == pytest.approx(6.61, abs=0.01)
    assert rf.step_bytes(256) / 1e9 == pytest.approx(52.8, abs=0.05)
    assert rf.step_bytes(128, batch=32) / 1e9 == pytest.approx(211.6, abs=0.1)
    assert rf.step_bytes(512) / 1e9 == pytest.approx(422.3, abs=0.1)
    assert rf.step_bytes(512, complex_bytes=8) / 1e9 == pytest.approx(211.1, abs=0.1)
    # per-RHS totals in units of N^3 bytes: 1032 (stage 1) / 1056 (stages 2, 3), up to the Hs = N/2+1 terms
    N = 512
    assert sum(rf.pass_bytes(N, stage=1).values()) / N ** 3 == pytest.approx(1032, rel=2e-3)
    assert sum(rf.pass_bytes(N, stage=2).values()) / N ** 3 == pytest.approx(1056, rel=2e-3)
    assert rf.grid_point_stages(128, 32, 2.0) == 32 * 128 ** 3 * 6
