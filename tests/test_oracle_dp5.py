"""Pins for the oracle's Dormand-Prince 5(4) step and Boost-rule controller."""
import math

import numpy as np
from scipy.integrate import RK45
from scipy.integrate._ivp.rk import rk_step


def test_tableau_row_sums_and_order_conditions(oracle):
    c, a, b, e = oracle.dp5_tableau()
    assert np.allclose(a.sum(axis=1), c, atol=1e-15)
    assert abs(b.sum() - 1) < 1e-15 and abs(e.sum()) < 1e-15
    bh = b - e                                    # 4th-order embedded weights
    for w, order in ((b, 5), (bh, 4)):
        assert abs(w @ c - 1 / 2) < 1e-15
        assert abs(w @ c ** 2 - 1 / 3) < 1e-15
        assert abs(w @ (a @ c) - 1 / 6) < 1e-15
        assert abs(w @ c ** 3 - 1 / 4) < 1e-15
        assert abs((w * c) @ (a @ c) - 1 / 8) < 1e-15
        assert abs(w @ (a @ c ** 2) - 1 / 12) < 1e-15
        assert abs(w @ (a @ (a @ c)) - 1 / 24) < 1e-15
    assert abs(b @ c ** 4 - 1 / 5) < 1e-15        # order 5 only for b
    assert abs(bh @ c ** 4 - 1 / 5) > 1e-4
    assert np.allclose(a[6, :6], b[:6]) and b[6] == 0  # first-same-as-last


def test_single_step_equals_scipy_rk45(oracle):
    """Same tableau, independent implementation: new state, stage derivatives and error vector."""
    O = oracle

    def fun(t, y):
        return np.array([y[1] + 0.1 * t, -4.0 * y[0] + 0.3 * math.sin(t), 0.5 * y[2] * y[0], -y[3] ** 2 + y[1]])

    t0, h = 0.3, 0.07
    y0 = np.array([1.0, -0.5, 0.8, 0.25])
    ynew, k7, err, kall = O.dp5_attempt(fun, t0, y0, h)
    sol = RK45(fun, t0, y0, 10.0)
    K = np.empty_like(sol.K)
    y_ref, f_ref = rk_step(fun, t0, y0, fun(t0, y0), h, sol.A, sol.B, sol.C, K)
    assert np.allclose(ynew, y_ref, rtol=1e-14, atol=1e-15)
    assert np.allclose(k7, f_ref, rtol=1e-14, atol=1e-15)
    assert np.allclose(kall, K, rtol=1e-13, atol=1e-15)
    err_ref = (K.T @ sol.E) * h                   # scipy: E = b_hat - b ... sign checked below
    assert np.allclose(np.abs(err), np.abs(err_ref), rtol=1e-10, atol=1e-18)


def test_error_vector_is_fifth_minus_fourth(oracle):
    """err = y5 - y4 with y4 the embedded 4th-order solution built from b_hat (Dormand-Prince)."""
    O = oracle
    bhat = np.array([5179 / 57600, 0, 7571 / 16695, 393 / 640, -92097 / 339200, 187 / 2100, 1 / 40])
    fun = lambda t, y: np.array([y[1], -y[0]])
    y0 = np.array([0.3, 1.1])
    h = 0.2
    ynew, k7, err, kall = O.dp5_attempt(fun, 0.0, y0, h)
    y4 = y0 + h * (bhat @ kall)
    assert np.allclose(err, ynew - y4, rtol=1e-8, atol=1e-17)  # cancellation in y5-y4


def test_fifth_order_convergence(oracle):
    O = oracle
    fun = lambda t, y: np.array([y[1], -y[0]])      # harmonic oscillator, exact solution known
    errs = []
    for nst in (8, 16, 32):
        h = 1.0 / nst
        y = np.array([1.0, 0.0])
        t = 0.0
        for _ in range(nst):
            y, _, _, _ = O.dp5_attempt(fun, t, y, h)
            t += h
        errs.append(np.hypot(y[0] - math.cos(1.0), y[1] + math.sin(1.0)))
    s1 = math.log2(errs[0] / errs[1])
    s2 = math.log2(errs[1] / errs[2])
    assert 4.7 < s1 < 5.6 and 4.7 < s2 < 5.6
    # exponential: one step reproduces the degree-5 Taylor polynomial of exp(h) closely
    y, _, err, _ = O.dp5_attempt(lambda t, y: y, 0.0, np.array([1.0]), 0.1)
    assert abs(y[0] - math.exp(0.1)) < 2e-9


def test_error_ratio_eq4(oracle):
    """PAPER.md:85 Eq. 4 on hand-computed numbers; the vpar component carries c = v_total."""
    O = oracle
    err = np.array([1e-10, -3e-10, 0.0, 2e-3])
    y = np.array([0.5, -0.25, 3.0, 1e7])
    k1 = np.array([1e5, 2e5, 1e6, -1e12])
    h, rtol, atol, c = 1e-7, 1e-9, 1e-12, np.array([1.0, 1.0, 1.0, 1.3e7])
    want = max(1e-10 / (1e-12 + 1e-9 * (0.5 + 1e-7 * 1e5)),
               3e-10 / (1e-12 + 1e-9 * (0.25 + 1e-7 * 2e5)),
               0.0,
               2e-3 / (1e-12 * 1.3e7 + 1e-9 * (1e7 + 1e-7 * 1e12)))
    assert abs(O.error_ratio(err, y, k1, h, rtol, atol, c) / want - 1) < 1e-14
    assert math.isnan(O.error_ratio(np.array([math.nan, 0, 0, 0]), y, k1, h, rtol, atol, c))


def test_controller_table(oracle):
    """Boost odeint default rule for dopri5 (restated in DESIGN.md S2), hand-computed."""
    O = oracle
    h, big = 1e-7, 1.0
    table = {
        0.0: (True, 4.5),                          # growth capped: 0.9 * (5^-5)^(-1/5) = 4.5
        1e-6: (True, 4.5),
        0.4: (True, 0.9 * 0.4 ** (-0.2)),
        0.5: (True, 1.0),                          # not < 0.5: unchanged
        0.75: (True, 1.0),
        1.0: (True, 1.0),
        1.0 + 1e-12: (False, 0.9 * (1.0 + 1e-12) ** (-1 / 3)),
        8.0: (False, 0.45),
        1e6: (False, 0.2),                         # shrink floored at 1/5
        math.nan: (False, 0.2),
    }
    for r, (acc, fac) in table.items():
        dt, a = O.controller(h, r, big)
        assert a == acc, r
        assert abs(dt / h - fac) < 1e-14, (r, dt / h, fac)
    dt, a = O.controller(h, 0.0, 2e-7)             # dtmax cap
    assert a and dt == 2e-7
    # constant RHS => e == 0 => r = 0 => dt grows by exactly 4.5x per step until dtmax
    dt = 1e-9
    seq = []
    for _ in range(5):
        dt, _ = O.controller(dt, 0.0, 1e-7)
        seq.append(dt)
    assert np.allclose(seq[:3], [4.5e-9, 20.25e-9, 91.125e-9], rtol=1e-14) and seq[3] == 1e-7 and seq[4] == 1e-7
