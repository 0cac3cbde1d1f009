"""Pins for the oracle's guiding-centre right-hand sides (Eq. 3; R1-R3).

R1/R2 are checked against the Euler-Lagrange equations of the paper's Lagrangian derived here with
sympy (independent of the oracle's formulas), then against closed forms and invariants.
"""
import math

import numpy as np
import pytest
import sympy as sp

from paper_2604_07617_b200 import workloads as W

M, Q = W.ALPHA_MASS, W.ALPHA_CHARGE


def _boozer_fd(nquant=4):
    return dict(coord=0, ncell=[1, 1, 1], lo=[0, 0, 0], hi=[1, 2 * math.pi, 2 * math.pi / 4], nfp=4,
                nquant=nquant, nodes=None, G0=W.G0, I0=0.0, iota0=W.IOTA0, iota1=W.IOTA1, psi0=W.PSI0)


def _euler_lagrange_solver(saw):
    """Euler-Lagrange equations of L = q(psi + rho_c I) thdot + q(rho_c G - psi_p) zedot - H,
    H = M v^2/2 + M mu B + q Phi, rho_c = M v/(q B) + alpha  (Eq. 3 in Boozer form with
    A = psi grad(theta) - psi_p grad(zeta), B = G grad(zeta), vacuum I = 0)."""
    psi, th, ze, v, t = sp.symbols("psi theta zeta v t", real=True)
    mu = sp.Symbol("mu", positive=True)
    s = psi / W.PSI0
    B = W.B0 * (1 + sp.Rational(1, 10) * sp.sqrt(s) * sp.cos(th) + sp.Rational(1, 20) * sp.sqrt(s) * sp.cos(th - 4 * ze))
    iota = W.IOTA0 + W.IOTA1 * s
    psi_p = W.PSI0 * (W.IOTA0 * s + W.IOTA1 * s ** 2 / 2)
    G = W.G0
    if saw:
        Phi0, s0, w2, om, mm, nn = saw
        Phi = Phi0 * sp.exp(-(s - s0) ** 2 / w2) * sp.sin(mm * th - nn * ze + om * t)
        alpha = -(iota * mm - nn) * Phi / (om * G)
    else:
        Phi, alpha = sp.Integer(0), sp.Integer(0)
    rho_c = M * v / (Q * B) + alpha
    z = [psi, th, ze, v]
    A = [sp.Integer(0), Q * psi, Q * (rho_c * G - psi_p), sp.Integer(0)]
    H = M * v ** 2 / 2 + M * mu * B + Q * Phi
    Om = sp.Matrix(4, 4, lambda i, j: sp.diff(A[i], z[j]) - sp.diff(A[j], z[i]))
    rhs = sp.Matrix([-sp.diff(A[i], t) - sp.diff(H, z[i]) for i in range(4)])
    fOm = sp.lambdify((psi, th, ze, v, t, mu), Om, "numpy")
    frhs = sp.lambdify((psi, th, ze, v, t, mu), rhs, "numpy")
    fB = sp.lambdify((psi, th, ze), [B, sp.diff(B, psi) * W.PSI0, sp.diff(B, th), sp.diff(B, ze)], "numpy")

    def solve(psi_, th_, ze_, v_, t_, mu_):
        zd = np.linalg.solve(np.array(fOm(psi_, th_, ze_, v_, t_, mu_), dtype=float),
                             np.array(frhs(psi_, th_, ze_, v_, t_, mu_), dtype=float).ravel())
        zd[0] /= W.PSI0                           # psidot -> sdot
        return zd

    return solve, fB


@pytest.mark.parametrize("saw", [None, (1.0e3, 0.5, 0.01, 2 * math.pi * 1e5, 1, 1), (5.0e4, 0.4, 0.05, 2 * math.pi * 3e4, 3, -2)])
def test_boozer_rhs_equals_euler_lagrange_of_eq3(oracle, saw):
    O = oracle
    solve, fB = _euler_lagrange_solver(saw)
    pd = W.base_params(1e-4)
    if saw:
        pd.update(saw_on=1, saw_Phi0=saw[0], saw_s0=saw[1], saw_w2=saw[2], saw_omega=saw[3], saw_m=saw[4], saw_n=saw[5])
    p = O.make_params(pd)
    f = O.Field(_boozer_fd())
    rng = np.random.default_rng(23)
    for _ in range(25):
        s = 0.1 + 0.8 * rng.random()
        th, ze = 2 * math.pi * rng.random(), 2 * math.pi * rng.random()
        v = (2 * rng.random() - 1) * W.V_TOTAL
        t = 1e-5 * rng.random()
        fv = np.array(fB(s * W.PSI0, th, ze), dtype=float)
        mu = (W.V_TOTAL ** 2 - v ** 2) / (2 * fv[0])
        got = O.gc_boozer(f, p, mu, t, s, th, ze, v, fv)
        want = solve(s * W.PSI0, th, ze, v, t, mu)
        scale = np.array([1e5, 1e6, 1e6, 1e12])   # typical magnitudes of (sdot, thdot, zedot, vdot)
        assert np.all(np.abs(got - want) <= 1e-9 * np.maximum(np.abs(want), 1e-6 * scale)), (got, want)


def test_saw_amplitude_zero_reduces_to_vacuum(oracle):
    O = oracle
    f = O.Field(_boozer_fd())
    p0 = O.make_params(W.base_params(1e-4))
    pd = W.base_params(1e-4)
    pd.update(saw_on=1, saw_Phi0=0.0, saw_m=1, saw_n=1, saw_omega=2 * math.pi * 1e5)
    p1 = O.make_params(pd)
    fv = np.array([5.5, 0.3, -0.2, 0.4])
    a = O.gc_boozer(f, p0, 3e12, 1e-6, 0.4, 1.0, 2.0, 7e6, fv)
    b = O.gc_boozer(f, p1, 3e12, 1e-6, 0.4, 1.0, 2.0, 7e6, fv)
    assert np.allclose(a, b, rtol=1e-15, atol=0)


def _analytic_boozer(O, fn, saw=None, T=2e-5, rtol=1e-10):
    pd = W.base_params(T, rtol=rtol, atol=1e-13)
    if saw:
        pd.update(saw)
    return O.Field(_boozer_fd(), analytic=fn), O.make_params(pd)


def test_field_depending_on_s_only_closed_form(oracle):
    """B = B(s): sdot = vpardot = 0, theta and zeta linear in t (closed form)."""
    O = oracle
    Bs = lambda s: W.B0 * (1 + 0.2 * s)
    f, p = _analytic_boozer(O, lambda x: [Bs(x[0]), W.B0 * 0.2, 0.0, 0.0], T=3e-6)
    x0 = np.array([[0.3], [0.7], [0.2], [0.6 * W.V_TOTAL]])
    r = O.trace(f, p, x0)
    s, v = 0.3, 0.6 * W.V_TOTAL
    B = Bs(s)
    mu = (W.V_TOTAL ** 2 - v * v) / (2 * B)
    Wd = (M / Q) * (v * v / B + mu)
    thdot = (W.B0 * 0.2 / W.PSI0) * Wd + (W.IOTA0 + W.IOTA1 * s) * v * B / W.G0
    zedot = v * B / W.G0
    T = 3e-6
    assert r["status"][0] == 0 and r["tstop"][0] == T
    # stepped in pseudo-Cartesian variables: the circle is integrated, not exact
    assert abs(r["xf"][0, 0] - s) < 1e-9 and abs(r["xf"][3, 0] / v - 1) < 1e-12
    th = 0.7 + thdot * T
    assert abs(math.remainder(r["xf"][1, 0] - th, 2 * math.pi)) < 1e-9
    assert abs(r["xf"][2, 0] - (0.2 + zedot * T)) < 1e-9


def test_energy_and_pzeta_conserved_in_analytic_fields(oracle):
    """Analytic-field mode: E = vpar^2/2 + mu B conserved to integrator tolerance; in an axisymmetric
    field P_zeta = G M vpar / B - q psi_p is conserved too."""
    O = oracle
    modes = W.boozer_modes_cfg0()
    fn = lambda x: [float(v) for v in W.boozer_field_values(modes, x[0], x[1], x[2])]
    f, p = _analytic_boozer(O, fn)
    axi = lambda x: [float(v) for v in W.boozer_field_values([(1, 0, 0.1), (2, 0, 0.03)], x[0], x[1], x[2])]
    fa, _ = _analytic_boozer(O, axi)
    rng = np.random.default_rng(29)
    for field, fun, check_p in ((f, fn, False), (fa, axi, True)):
        for _ in range(3):
            x0 = np.array([0.2 + 0.5 * rng.random(), 2 * math.pi * rng.random(), 2 * math.pi * rng.random(),
                           (2 * rng.random() - 1) * W.V_TOTAL])
            traj, ts, st = O.trace_record(field, p, x0)
            assert st == 0 and len(traj) > 50
            B = np.array([fun(row[1:4])[0] for row in traj])
            mu = (W.V_TOTAL ** 2 - x0[3] ** 2) / (2 * B[0])
            E = 0.5 * traj[:, 4] ** 2 + mu * B
            assert np.max(np.abs(E / E[0] - 1)) < 1e-8
            if check_p:
                s = traj[:, 1]
                psi_p = W.PSI0 * (W.IOTA0 * s + 0.5 * W.IOTA1 * s * s)
                P = W.G0 * M * traj[:, 4] / B - Q * psi_p
                assert np.max(np.abs(P - P[0])) < 1e-8 * Q * W.PSI0


def test_saw_invariant_nH_minus_omega_Pzeta(oracle):
    """Axisymmetric B + one harmonic (m,n,omega): n H - omega P_zeta is invariant while H and P_zeta move."""
    O = oracle
    axi = lambda x: [float(v) for v in W.boozer_field_values([(1, 0, 0.1)], x[0], x[1], x[2])]
    mm, nn, om, Phi0, s0, w2 = 2, 1, 2 * math.pi * 1e5, 5.0e4, 0.5, 0.05
    saw = dict(saw_on=1, saw_m=mm, saw_n=nn, saw_omega=om, saw_Phi0=Phi0, saw_s0=s0, saw_w2=w2)
    f, p = _analytic_boozer(O, axi, saw=saw, T=4e-5, rtol=1e-11)
    rng = np.random.default_rng(31)
    moved = 0.0
    for _ in range(3):
        x0 = np.array([0.35 + 0.3 * rng.random(), 2 * math.pi * rng.random(), 2 * math.pi * rng.random(),
                       (2 * rng.random() - 1) * W.V_TOTAL])
        traj, ts, st = O.trace_record(f, p, x0)
        t, s, th, ze, v = traj.T
        B = np.array([axi(row[1:4])[0] for row in traj])
        mu = (W.V_TOTAL ** 2 - x0[3] ** 2) / (2 * B[0])
        iota = W.IOTA0 + W.IOTA1 * s
        Phi = Phi0 * np.exp(-(s - s0) ** 2 / w2) * np.sin(mm * th - nn * ze + om * t)
        alpha = -(iota * mm - nn) * Phi / (om * W.G0)
        H = 0.5 * M * v * v + M * mu * B + Q * Phi
        psi_p = W.PSI0 * (W.IOTA0 * s + 0.5 * W.IOTA1 * s * s)
        Pz = Q * ((M * v / (Q * B) + alpha) * W.G0 - psi_p)
        inv = nn * H - om * Pz
        assert np.max(np.abs(inv - inv[0])) < 1e-8 * abs(nn * H[0])
        moved = max(moved, np.max(np.abs(H / H[0] - 1)))
    assert moved > 1e-5                            # the test has teeth: H itself is not conserved


def test_cartesian_energy_identity_and_toroidal_closed_form(oracle):
    O = oracle
    p = O.make_params(W.base_params(1e-5))
    rng = np.random.default_rng(37)
    for _ in range(20):                            # vpar*vpardot + mu*grad|B|.xdot = 0 for ANY (B, grad|B|)
        fv = np.concatenate([rng.normal(size=3) * 3, rng.normal(size=3), [0.0]])
        pos = rng.normal(size=3) + np.array([6.0, 0, 0])
        v = (2 * rng.random() - 1) * W.V_TOTAL
        mu = 1e12 * rng.random()
        d = O.gc_cartesian(p, mu, pos, v, fv)
        R = math.hypot(pos[0], pos[1])
        c, s_ = pos[0] / R, pos[1] / R
        g = np.array([fv[3] * c - fv[4] * s_, fv[3] * s_ + fv[4] * c, fv[5]])
        assert abs(v * d[3] + mu * (g @ d[:3])) < 1e-12 * (abs(v * d[3]) + abs(mu) * np.linalg.norm(g) * np.linalg.norm(d[:3]))
    # pure toroidal field B = B0 R0 / R phi_hat: Rdot = 0, phidot = vpar/R, Zdot = (M/(q B R))(vpar^2 + vperp^2/2)
    R, phi, Z, v = 7.0, 0.9, 0.3, 0.4 * W.V_TOTAL
    B = W.B0 * W.R0 / R
    fv = np.array([0.0, B, 0.0, -B / R, 0.0, 0.0, 0.0])
    mu = (W.V_TOTAL ** 2 - v * v) / (2 * B)
    d = O.gc_cartesian(p, mu, [R * math.cos(phi), R * math.sin(phi), Z], v, fv)
    Rdot = d[0] * math.cos(phi) + d[1] * math.sin(phi)
    phidot = (-d[0] * math.sin(phi) + d[1] * math.cos(phi)) / R
    assert abs(Rdot) < 1e-9 * abs(v)
    assert abs(phidot / (v / R) - 1) < 1e-14
    assert abs(d[2] / ((M / (Q * B * R)) * (v * v + 0.5 * 2 * mu * B)) - 1) < 1e-13
    assert abs(d[3]) < 1e-3                        # b . grad|B| = 0


def test_cartesian_pphi_and_energy_conserved_axisymmetric(oracle):
    """P_phi = M R (B_phi/|B|) vpar + q psi is an exact invariant of the vacuum-form equations when
    R B_phi = const (config 3's field), energy for any field."""
    O = oracle
    fd = dict(coord=1, ncell=[1, 1, 1], lo=[4, -4, 0], hi=[11, 4, 2 * math.pi], nfp=1, nquant=7, nodes=None,
              G0=0.0, I0=0.0, iota0=0.0, iota1=0.0, psi0=W.PSI_EDGE_CYL)
    fn = lambda x: [float(v) for v in W.cyl_field_values(x[0], x[1])]
    f = O.Field(fd, analytic=fn)
    p = O.make_params(W.base_params(3e-5, rtol=1e-10, atol=1e-13))
    x0s = W.cyl_births(np.random.default_rng(41), 3)
    for i in range(3):
        x0 = x0s[:, i]
        traj, ts, st = O.trace_record(f, p, x0)
        assert st == 0 and len(traj) > 50
        R = np.hypot(traj[:, 1], traj[:, 2])
        vals = np.array([fn([r, z, 0.0]) for r, z in zip(R, traj[:, 3])])
        modB = np.sqrt((vals[:, :3] ** 2).sum(axis=1))
        mu = (W.V_TOTAL ** 2 - x0[3] ** 2) / (2 * modB[0])
        E = 0.5 * traj[:, 4] ** 2 + mu * modB
        assert np.max(np.abs(E / E[0] - 1)) < 1e-8
        P = M * R * vals[:, 1] / modB * traj[:, 4] + Q * vals[:, 6]
        assert np.max(np.abs(P - P[0])) < 1e-8 * Q * W.PSI_EDGE_CYL


# ---- R1b: non-vacuum Boozer with tabulated profiles ("vacuum, finite beta, etc.") ----
_NV_G = lambda s: W.G0 * (1.0 + 0.05 * s - 0.02 * s ** 2)            # cubic or lower: reproduced exactly by one cell
_NV_I = lambda s: W.G0 * (0.02 * s + 0.01 * s ** 3)
_NV_IOTA = lambda s: 0.42 + 0.1 * s + 0.05 * s ** 2


def _nonvacuum_fd(ncell0=1):
    fd = _boozer_fd()
    fd["ncell"] = [ncell0, 1, 1]
    sn = np.linspace(0.0, 1.0, 3 * ncell0 + 1)
    fd.update(G_nodes=_NV_G(sn), I_nodes=_NV_I(sn), iota_nodes=_NV_IOTA(sn))
    return fd


def test_profiles_reproduce_cubics_and_their_derivatives(oracle):
    """A profile on the unique s-nodes is interpolated by the tables' piecewise cubic: cubics and their derivatives
    are reproduced to round-off, in the end cells also outside [0, 1] (extrapolation)."""
    O = oracle
    for k0 in (1, 3):
        f = O.Field(_nonvacuum_fd(k0))
        sn = np.linspace(0.0, 1.0, 3 * k0 + 1)
        for s in (-0.05, 0.0, 0.2, 1.0 / 3.0, 0.77, 1.0, 1.03):
            v, d = O.profile(f, _NV_I(sn), s)
            assert abs(v - _NV_I(s)) <= 1e-13 * W.G0
            assert abs(d - W.G0 * (0.02 + 0.03 * s ** 2)) <= 1e-12 * W.G0


def test_nonvacuum_rhs_equals_euler_lagrange_of_eq3(oracle):
    """R1b against the Euler-Lagrange equations of Eq. 3 with B = G(psi) grad(zeta) + I(psi) grad(theta),
    derived here with sympy: L = q (psi + rho I) thdot + q (rho G - psi_p) zedot - H, rho = M v / (q B)."""
    O = oracle
    psi, th, ze, v = sp.symbols("psi theta zeta v", real=True)
    mu = sp.Symbol("mu", positive=True)
    s = psi / W.PSI0
    B = W.B0 * (1 + sp.Rational(1, 10) * sp.sqrt(s) * sp.cos(th) + sp.Rational(1, 20) * sp.sqrt(s) * sp.cos(th - 4 * ze))
    G = W.G0 * (1 + sp.Rational(1, 20) * s - sp.Rational(1, 50) * s ** 2)
    I = W.G0 * (sp.Rational(1, 50) * s + sp.Rational(1, 100) * s ** 3)
    iota = sp.Rational(42, 100) + sp.Rational(1, 10) * s + sp.Rational(1, 20) * s ** 2
    psi_p = W.PSI0 * sp.integrate(iota.subs(psi, sp.Symbol("x") * W.PSI0), (sp.Symbol("x"), 0, s))
    rho = M * v / (Q * B)
    z = [psi, th, ze, v]
    A = [sp.Integer(0), Q * (psi + rho * I), Q * (rho * G - psi_p), sp.Integer(0)]
    H = M * v ** 2 / 2 + M * mu * B
    Om = sp.Matrix(4, 4, lambda i, j: sp.diff(A[i], z[j]) - sp.diff(A[j], z[i]))
    rhs = sp.Matrix([-sp.diff(H, z[i]) for i in range(4)])
    fOm = sp.lambdify((psi, th, ze, v, mu), Om, "numpy")
    frhs = sp.lambdify((psi, th, ze, v, mu), rhs, "numpy")
    fB = sp.lambdify((psi, th, ze), [B, sp.diff(B, psi) * W.PSI0, sp.diff(B, th), sp.diff(B, ze)], "numpy")
    f = O.Field(_nonvacuum_fd())
    p = O.make_params(W.base_params(1e-4))
    rng = np.random.default_rng(29)
    for _ in range(25):
        s_ = 0.1 + 0.8 * rng.random()
        th_, ze_ = 2 * math.pi * rng.random(), 2 * math.pi * rng.random()
        v_ = (2 * rng.random() - 1) * W.V_TOTAL
        fv = np.array(fB(s_ * W.PSI0, th_, ze_), dtype=float)
        mu_ = (W.V_TOTAL ** 2 - v_ ** 2) / (2 * fv[0])
        got = O.gc_boozer(f, p, mu_, 0.0, s_, th_, ze_, v_, fv)
        want = np.linalg.solve(np.array(fOm(s_ * W.PSI0, th_, ze_, v_, mu_), dtype=float),
                               np.array(frhs(s_ * W.PSI0, th_, ze_, v_, mu_), dtype=float).ravel())
        want[0] /= W.PSI0
        scale = np.array([1e5, 1e6, 1e6, 1e12])
        assert np.all(np.abs(got - want) <= 1e-9 * np.maximum(np.abs(want), 1e-6 * scale)), (got, want)


def test_nonvacuum_reduces_to_vacuum(oracle):
    """Constant G, I = 0 and the linear iota given as PROFILES give the vacuum right-hand side R1."""
    O = oracle
    fd = _boozer_fd()
    sn = np.linspace(0.0, 1.0, 4)
    fd1 = dict(fd, G_nodes=np.full(4, W.G0), I_nodes=np.zeros(4), iota_nodes=W.IOTA0 + W.IOTA1 * sn)
    p = O.make_params(W.base_params(1e-4))
    fv = np.array([5.5, 0.3, -0.2, 0.4])
    a = O.gc_boozer(O.Field(fd), p, 3e12, 0.0, 0.4, 1.0, 2.0, 7e6, fv)
    b = O.gc_boozer(O.Field(fd1), p, 3e12, 0.0, 0.4, 1.0, 2.0, 7e6, fv)
    assert np.allclose(a, b, rtol=1e-14, atol=0)


def test_nonvacuum_energy_and_pzeta_conserved(oracle):
    """Invariants of R1b in an analytic axisymmetric field B(s, theta): energy v^2/2 + mu B and the canonical toroidal
    momentum P_zeta = rho G - psi_p (per unit charge), along a traced orbit."""
    O = oracle

    def fn(x):
        s, th = max(x[0], 1e-12), x[1]
        r = math.sqrt(s)
        return [W.B0 * (1 + 0.1 * r * math.cos(th)), W.B0 * 0.05 / r * math.cos(th), -W.B0 * 0.1 * r * math.sin(th), 0.0]

    f = O.Field(_nonvacuum_fd(), analytic=fn)
    p = O.make_params(W.base_params(2e-5, rtol=1e-10, atol=1e-13))
    x0 = np.array([[0.3, 0.5], [0.4, 2.0], [0.1, 1.0], [0.6 * W.V_TOTAL, -0.3 * W.V_TOTAL]])
    r = O.trace(f, p, x0)
    assert np.all(r["status"] == 0)

    def invariants(x):
        s, th, v = x[0], x[1], x[3]
        B = np.array([fn([s[i], th[i], 0.0])[0] for i in range(len(s))])
        B0v = np.array([fn([x0[0][i], x0[1][i], 0.0])[0] for i in range(len(s))])
        muv = (W.V_TOTAL ** 2 - x0[3] ** 2) / (2 * B0v)
        E = 0.5 * v ** 2 + muv * B
        psi_p = W.PSI0 * (0.42 * s + 0.05 * s ** 2 + 0.05 * s ** 3 / 3)
        Pz = (M * v / (Q * B)) * _NV_G(s) - psi_p
        return E, Pz

    E0, P0 = invariants(x0)
    E1, P1 = invariants(r["xf"])
    assert np.all(np.abs(E1 / E0 - 1) < 1e-8)
    assert np.all(np.abs(P1 - P0) < 1e-8 * W.PSI0)
