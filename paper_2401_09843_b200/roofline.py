"""Bytes-over-bandwidth roofline model of the RHS / RK3 step (host arithmetic only).

The FIXED reference model is the pass structure of SURVEY.md section 8(a): every 1-D axis pass reads its
input once and writes its output once, padded zeros never touch HBM, the six products are fused into the
last inverse pass, one fused spectral/RK pass per stage.  Per sample, with c = bytes per complex,
  S = N^2 (N/2+1) c,  A1 = M N H c,  A2 = M^2 H c,  P = M^3 c / 2,   M = 3N/2, H = N/2:
  a1 3(S+A1)  a2 3(A1+A2)  a3 3 A2 + 6 P  a4 6(P+A2)  a5 6(A2+A1)  a6 6(A1+S)  a7 12 S (stage 1) / 15 S (stages 2,3)
  step = 3 (inverse + forward) + 42 S   ~ 3146 N^3 bytes in fp64.

Also holds the paper's own lower-bound formulas (eq. 5.1-5.3) used by a CPU test to
pin the reading that the symbol `s` in them is sizeof(scalar).
"""
from __future__ import annotations

PASS_NAMES = ["a1_col_inv_x", "a2_col_inv_y", "a3_z_inv_prod", "a4_z_fwd", "a5_col_fwd_y", "a6_col_fwd_x", "a7_spectral"]


def sizes(N: int, complex_bytes: int):
    M, H, Hs = 3 * N // 2, N // 2, N // 2 + 1
    S = N * N * Hs * complex_bytes
    A1 = M * N * H * complex_bytes
    A2 = M * M * H * complex_bytes
    P = M ** 3 * complex_bytes // 2
    return S, A1, A2, P


def pass_bytes(N: int, batch: int = 1, complex_bytes: int = 16, stage: int = 1) -> dict:
    """Algorithmic bytes of each pass of ONE RHS evaluation + stage update (stage 1 reads no u_n)."""
    S, A1, A2, P = sizes(N, complex_bytes)
    b = {
        "a1_col_inv_x": 3 * (S + A1),
        "a2_col_inv_y": 3 * (A1 + A2),
        "a3_z_inv_prod": 3 * A2 + 6 * P,
        "a4_z_fwd": 6 * (P + A2),
        "a5_col_fwd_y": 6 * (A2 + A1),
        "a6_col_fwd_x": 6 * (A1 + S),
        "a7_spectral": (12 if stage == 1 else 15) * S,
    }
    return {k: v * batch for k, v in b.items()}


def pass_bytes_per_step(N: int, batch: int = 1, complex_bytes: int = 16) -> dict:
    """Algorithmic bytes of each pass summed over the three stages of one SSP-RK3 step."""
    out = {k: 0 for k in PASS_NAMES}
    for stage in (1, 2, 3):
        for k, v in pass_bytes(N, batch, complex_bytes, stage).items():
            out[k] += v
    return out


NFLUX = 5  # flux components carried through a4-a7 by the built path (trace-free combinations, csrc/kernels_z.cuh)

BUILT_PASS_NAMES = ["a1_col_inv_x", "a2_col_inv_y", "a3a4_z_fused", "a5_col_fwd_y", "a6_col_fwd_x", "a7_spectral"]


def built_pass_bytes(N: int, batch: int = 1, complex_bytes: int = 16, stage: int = 1) -> dict:
    """Bytes each kernel of the pass structure actually built must move for ONE RHS evaluation + stage update:
    a3 and a4 are one kernel (the M^3 physical arrays never reach HBM) and only
    the NFLUX = 5 trace-free flux components are transformed forward (item 5(iii)).  Spectral rows are stored
    with H = N/2 entries (the zero kz = N/2 column is not stored), which the S term below ignores (< 0.4 %)."""
    S, A1, A2, _ = sizes(N, complex_bytes)
    b = {
        "a1_col_inv_x": 3 * (S + A1),
        "a2_col_inv_y": 3 * (A1 + A2),
        "a3a4_z_fused": (3 + NFLUX) * A2,
        "a5_col_fwd_y": NFLUX * (A2 + A1),
        "a6_col_fwd_x": NFLUX * (A1 + S),
        "a7_spectral": (NFLUX + 3 + 3 + (0 if stage == 1 else 3)) * S,
    }
    return {k: v * batch for k, v in b.items()}


def built_pass_bytes_per_step(N: int, batch: int = 1, complex_bytes: int = 16) -> dict:
    out = {k: 0 for k in BUILT_PASS_NAMES}
    for stage in (1, 2, 3):
        for k, v in built_pass_bytes(N, batch, complex_bytes, stage).items():
            out[k] += v
    return out


def actual_step_bytes(N: int, batch: int = 1, complex_bytes: int = 16) -> int:
    """Bytes per RK3 step of the pass structure actually built."""
    return sum(built_pass_bytes_per_step(N, batch, complex_bytes).values())


def step_bytes(N: int, batch: int = 1, complex_bytes: int = 16) -> int:
    return sum(pass_bytes_per_step(N, batch, complex_bytes).values())


def grid_point_stages(N: int, batch: int, steps: float) -> float:
    return float(batch) * N ** 3 * 3.0 * steps


# ---- two-dimensional solver: same accounting with d = 2.  Per sample, c = bytes per complex,
#   S = N (N/2+1) c,  A1 = M H c,  P = M^2 c / 2.  Built passes: b1 x inverse 2(S+A1), b2 fused y (2 in + 2 trace-free flux out) 4 A1,
#   b3 x forward 2(A1+S), b4 spectral 6 S (stage 1) / 8 S.  Fixed (unfused, three products) model: b2 = 2 A1 + 3 P, 3 (P + A1);
#   b3 = 3 (A1 + S); b4 = 7 S / 9 S.
BUILT_PASS_NAMES_2D = ["b1_x_inv", "b2_y_fused", "b3_x_fwd", "b4_spectral"]


def built_pass_bytes_per_step_2d(N: int, batch: int = 1, complex_bytes: int = 16) -> dict:
    M, H, Hs = 3 * N // 2, N // 2, N // 2 + 1
    S, A1 = N * Hs * complex_bytes, M * H * complex_bytes
    b = {"b1_x_inv": 3 * 2 * (S + A1), "b2_y_fused": 3 * 4 * A1, "b3_x_fwd": 3 * 2 * (A1 + S), "b4_spectral": (6 + 8 + 8) * S}
    return {k: v * batch for k, v in b.items()}


def fixed_step_bytes_2d(N: int, batch: int = 1, complex_bytes: int = 16) -> int:
    M, H, Hs = 3 * N // 2, N // 2, N // 2 + 1
    S, A1, P = N * Hs * complex_bytes, M * H * complex_bytes, M * M * complex_bytes // 2
    per_stage = 2 * (S + A1) + (2 * A1 + 3 * P) + 3 * (P + A1) + 3 * (A1 + S)
    return batch * (3 * per_stage + (7 + 9 + 9) * S)


def grid_point_stages_2d(N: int, batch: int, steps: float) -> float:
    return float(batch) * N ** 2 * 3.0 * steps


# ---- the paper's own lower bounds, eq. (5.1)-(5.3); s = sizeof(scalar), 2s = bytes per complex, p = ranks
def paper_t_pad(N, p, s, beta):
    return 213.0 / 16.0 * N ** 3 / p * 2 * s / beta


def paper_t_unpad(N, p, s, beta):
    return 78.0 / 4.0 * N ** 3 / p * 2 * s / beta


def paper_t_transpose(N, p, s, beta_d, beta_hd, beta_mpi):
    return (9.0 / 2.0 * N ** 3 / p ** 2 * 2 * s / beta_d + 9.0 / 4.0 * N ** 3 / p ** 2 * 2 * s / beta_hd
            + 9.0 / 8.0 * N ** 3 / p * 2 * s / beta_mpi)
