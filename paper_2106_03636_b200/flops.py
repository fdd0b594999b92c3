"""fp32 operation counts of the per-track arithmetic (bench.py `roofline` for the ALU-bound kernels).

Counted from the formulas of R12 / R13 with one operation per add / mul / div / sqrt; a fused
multiply-add of the arithmetic contract is two of them (a multiplication and an addition), so the count does not
depend on which terms are fused and the roof it is compared with is the FFMA rate (2 flop per lane per cycle):

  propagate (R12)    state + Jacobian 53, F C (rows 0-2) 60, (F C) F^T 50              = 163
  innovation (R13)   S, det, inverse                                                    =   9
  search window      2 sqrt + 2 mul + zc + bin range (4 x (add, mul))                   =  13
  candidate test     residuals 3 + chi2 8                                               =  11
  update (R13)       residuals 2, chi2 8, gain 30, covariance 60, state 20              = 120

DESIGN.md "Kernels / follower" restates this table.  The counts are what the METHOD requires per unit; they
are multiplied by the unit counts the kernels report (TPC_CNT_PROP / UPD / CAND) - not by instructions issued.
"""
FLOP_PROPAGATE = 163
FLOP_INNOVATION = 9
FLOP_WINDOW = 13
FLOP_CANDIDATE = 11
FLOP_UPDATE = 120


def follow_flop(work: dict) -> int:
    """Algorithmic fp32 operations of one k_follow launch from its work counters."""
    return (work["propagations"] * (FLOP_PROPAGATE + FLOP_INNOVATION + FLOP_WINDOW)
            + work["candidates"] * FLOP_CANDIDATE + work["updates"] * FLOP_UPDATE)


def fit_flop(n_hits: int, n_passes: int = 2) -> int:
    """k_fit: every hit is transported to and updated once per pass (R22)."""
    return n_hits * n_passes * (FLOP_PROPAGATE + FLOP_INNOVATION + FLOP_UPDATE)
