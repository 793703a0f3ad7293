"""Parity metrics shared by the GPU tests (reading R18)."""
import numpy as np

from paper_1905_05727_b200 import inputs

TOL_ONE_STEP = 1e-11      # BASELINE.json north_star: max relative difference in every conserved variable after one step
TOL_L1_500 = 1e-7         # L1-relative field difference after 500 steps
TOL_RATE = 5e-3           # global-reaction-rate curve and overtake time


def rel_diff(qa, qb, c_field, z_min=inputs.EOS["z_min"], rho1_0=inputs.AMBIENT["rho1_0"], rho2_0=inputs.AMBIENT["rho2_0"]):
    """max over cells of |a-b| / max(|a|, |b|, floor_k) per conserved variable (R18).

    floors: q0, q1 -> z_min * ambient phase density; q2, q3 -> rho*c of the cell (acoustic momentum scale);
    q4 -> none needed (|q4| >> 0); q5 -> 1; q6 -> q1.   c_field: sound speed of the reference state."""
    rho = qb[0] + qb[1]
    floors = [z_min * rho1_0, z_min * rho2_0, rho * c_field, rho * c_field, 0.0, 1.0, np.abs(qb[1])]
    out = []
    for k in range(7):
        den = np.maximum(np.maximum(np.abs(qa[k]), np.abs(qb[k])), floors[k])
        den = np.where(den == 0.0, 1.0, den)
        out.append(float(np.max(np.abs(qa[k] - qb[k]) / den)))
    return out


def l1_rel(qa, qb):
    """sum |a-b| / sum |b| per conserved variable; momentum components share one scale sum(|q2|+|q3|)."""
    out = []
    mom = float(np.sum(np.abs(qb[2])) + np.sum(np.abs(qb[3])))
    for k in range(7):
        den = mom if k in (2, 3) else float(np.sum(np.abs(qb[k])))
        out.append(float(np.sum(np.abs(qa[k] - qb[k])) / (den if den > 0 else 1.0)))
    return out


def rate_curve(t, M2r, M2tot0):
    """Eq. 12-13 on samples (R14): |dM2r/dt| / M2tot0 by backward differences between consecutive samples,
    assigned to the mid time.  Returns (t_mid, rate)."""
    t, M2r = np.asarray(t, dtype=np.float64), np.asarray(M2r, dtype=np.float64)
    return 0.5 * (t[1:] + t[:-1]), np.abs(np.diff(M2r)) / np.diff(t) / M2tot0
