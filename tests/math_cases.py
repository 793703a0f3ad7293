"""Inputs, long-double references and error bounds shared by the host and device checks of the fused kernels' own
elementary functions (paper_1905_05727_b200/csrc/nmsdt_math.cuh).  References are numpy long double (64-bit mantissa
on x86-64), i.e. library routines, not a retyping of the kernels' polynomials."""
import numpy as np

C_EXP, D_EXP = 4.53, 1.42          # Table II


def inputs(seed=7, n=20000):
    r = np.random.default_rng(seed)
    pos = np.concatenate([10.0 ** r.uniform(-12, 12, n), 1.0 + r.uniform(-1e-3, 1e-3, n), [1.0, 2.0, 0.5, 1e-300, 1e300]])
    xrho = np.concatenate([10.0 ** r.uniform(-3, 3, n), 1.0 + r.uniform(-1e-6, 1e-6, n), r.uniform(0.5, 3.0, n), [1.0]])
    yexp = np.concatenate([r.uniform(0, 700, n), 10.0 ** r.uniform(-8, 2.8, n), [0.0, 690.0, 689.999, 691.0, 1e4]])
    clampv = np.concatenate([r.uniform(-2, 3, n), [0.0, -0.0, 1.0, 1.0 - 1e-16, 1.0 + 3e-16, 690.0, 690.0000001, 1e300, -1e300]])
    return pos, xrho, yexp, clampv


def check(probe):
    """probe(fn, x, a, b) -> (y0, y1).  Returns {name: max error} and asserts the documented bounds."""
    L = np.longdouble
    pos, xrho, yexp, clampv = inputs()
    out = {}

    def rel(y, ref):
        return float(np.max(np.abs((y.astype(L) - ref) / ref)))

    y, _ = probe(0, pos, 0, 0)
    out["rcp"] = rel(y, 1 / pos.astype(L));                    assert out["rcp"] <= 4e-16, out
    y, _ = probe(1, pos, 0, 0)
    out["sqrt"] = rel(y, np.sqrt(pos.astype(L)));              assert out["sqrt"] <= 4e-16, out
    y, _ = probe(2, pos, 0, 0)
    ref = np.log(pos.astype(L))
    out["log"] = float(np.max(np.abs(y.astype(L) - ref) / np.maximum(np.abs(ref), 1.0)))
    assert out["log"] <= 4e-16, out
    # x^a = exp(a ln x) with a correctly rounded-ish ln: the error grows with the condition number |a ln x|
    yc, yd = probe(3, xrho, C_EXP, D_EXP)
    lx = np.abs(np.log(xrho))
    eC = np.abs((yc.astype(L) - np.power(xrho.astype(L), L(C_EXP))) / np.power(xrho.astype(L), L(C_EXP))).astype(np.float64)
    eD = np.abs((yd.astype(L) - np.power(xrho.astype(L), L(D_EXP))) / np.power(xrho.astype(L), L(D_EXP))).astype(np.float64)
    out["powC"] = float(np.max(eC / (8e-16 + 3e-16 * C_EXP * lx)))     # in units of the bound
    out["powD"] = float(np.max(eD / (6e-16 + 3e-16 * D_EXP * lx)))
    assert out["powC"] <= 1.0 and out["powD"] <= 1.0, out
    phys = (xrho > 0.5) & (xrho < 3.0)                        # rho2/rho02 of liquid NM from expansion to the von Neumann spike
    out["powC_phys"], out["powD_phys"] = float(eC[phys].max()), float(eD[phys].max())
    assert out["powC_phys"] <= 1.5e-15 and out["powD_phys"] <= 6e-16, out
    # the step kernels' route for Eq. 3-4: binade / mantissa tables of c^C, c^D and a binomial series (library powers outside
    # 2^-8 <= x < 2^8): no condition-number growth
    yc, yd = probe(7, xrho, C_EXP, D_EXP)
    out["tabC"] = rel(yc, np.power(xrho.astype(L), L(C_EXP)))
    out["tabD"] = rel(yd, np.power(xrho.astype(L), L(D_EXP)))
    assert out["tabC"] <= 4e-16 and out["tabD"] <= 4e-16, out
    edge = np.array([2.0 ** -8, np.nextafter(2.0 ** -8, 0), np.nextafter(256.0, 0), 256.0, 1.0, np.nextafter(1.0, 0), 0.5, 2.0, 255.99, 0.00391])
    yc, yd = probe(7, edge, C_EXP, D_EXP)
    out["tab_edge"] = max(rel(yc, np.power(edge.astype(L), L(C_EXP))), rel(yd, np.power(edge.astype(L), L(D_EXP))))
    assert out["tab_edge"] <= 4e-16, out
    # floored sound speed max(sqrt(n/d), 1) by the refined reciprocal square root of n d (n <= 0 -> 1)
    dd = 1134.0 * 0.84
    nn = np.concatenate([pos[(pos > 1e-6) & (pos < 1e12)] * dd, [dd, dd * (1 + 1e-15), dd * (1 - 1e-15), 0.0, -5.0, -1e300]])
    y0, y1 = probe(8, nn, dd, 0)
    ref = np.maximum(np.sqrt(np.maximum(nn, 0).astype(L) / L(dd)), 1)
    out["sqrt_ratio"] = rel(y0, ref)
    assert out["sqrt_ratio"] <= 5e-16, out
    assert np.all(y0 >= 1.0) and np.all(y0[-3:] == 1.0) and np.all(np.isfinite(y1[:-3])) and np.all(y1[-3:] == 1.0)
    # exp(-y) = 2^(-y log2 e): the rounding of log2(e) is amplified by y (y = Ta/T2 is 3..40 on this path, Eq. 6)
    y, _ = probe(4, yexp, 0, 0)
    yc = np.minimum(yexp, 690.0)
    ref = np.exp(-yc.astype(L))
    e = np.abs((y.astype(L) - ref) / ref).astype(np.float64)
    out["exp_neg"] = float(np.max(e / (6e-16 + 2e-17 * yc)))   # in units of the bound
    assert out["exp_neg"] <= 1.0, out
    out["exp_neg_phys"] = float(e[yc <= 40.0].max())
    assert out["exp_neg_phys"] <= 1e-15, out
    f1, c01 = probe(5, clampv, 0, 0)
    assert np.array_equal(f1, np.maximum(clampv, 1.0)) and np.array_equal(c01, np.minimum(np.maximum(clampv, 0.0), 1.0))
    nn, c690 = probe(6, clampv, 0, 0)
    assert np.array_equal(nn, np.maximum(clampv, 0.0)) and np.array_equal(c690, np.minimum(clampv, 690.0))
    return out
