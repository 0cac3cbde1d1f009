"""Pins for the oracle's whole tracer and estimator."""
import math

import numpy as np

from paper_2604_07617_b200 import workloads as W


def _rk4_bruteforce(O, f, p, x0, T, nsteps):
    """Classical fixed-step RK4 on the oracle's RHS: shares only the RHS with the DP5 tracer."""
    y = np.zeros(4)
    y[0], y[1], y[2], y[3] = x0[0] * math.cos(x0[1]), x0[0] * math.sin(x0[1]), x0[2], x0[3]
    mu = O.mu_init(f, p, x0)
    h = T / nsteps
    t = 0.0
    for _ in range(nsteps):
        k1, _ = O.rhs(f, p, mu, t, y)
        k2, _ = O.rhs(f, p, mu, t + h / 2, y + h / 2 * k1)
        k3, _ = O.rhs(f, p, mu, t + h / 2, y + h / 2 * k2)
        k4, _ = O.rhs(f, p, mu, t + h, y + h * k3)
        y = y + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        t += h
    return np.array([math.hypot(y[0], y[1]), math.atan2(y[1], y[0]), y[2], y[3]])


def test_trace_agrees_with_fine_step_rk4(oracle):
    """Brute force: the adaptive DP5 trace converges to a fixed-step RK4 solution of the same RHS.
    Global error of an accepted-step sequence is bounded by ~ n_steps * rtol * scale (Eq. 4)."""
    O = oracle
    cfg = W.config(0, n=4, T=1e-5)
    f = O.Field(cfg["field"])
    p9 = O.make_params(cfg["params"])
    r9 = O.trace(f, p9, cfg["x0"])
    assert np.all(r9["status"] == 0) and np.all(r9["tstop"] == 1e-5)
    r12 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-12, atol=1e-15)), cfg["x0"])
    nst = int(r9["nacc"].max()) * 12
    scale = np.array([1.0, 1.0, 10.0, W.V_TOTAL])
    for i in range(4):
        ref = _rk4_bruteforce(O, f, p9, cfg["x0"][:, i], 1e-5, nst)
        for r, tol in ((r12, 1e-8), (r9, 3 * r9["nacc"][i] * 1e-9)):
            d = r["xf"][:, i] - ref
            d[1] = math.remainder(d[1], 2 * math.pi)
            assert np.all(np.abs(d) < tol * scale), (i, d, tol)


def test_tolerance_refinement_converges(oracle):
    """The end state moves toward a tight-tolerance reference as rtol shrinks."""
    O = oracle
    cfg = W.config(0, n=3, T=1e-5)
    f = O.Field(cfg["field"])
    ends = {}
    for rtol in (1e-6, 1e-8, 1e-11):
        pd = dict(cfg["params"], rtol=rtol, atol=rtol * 1e-3)
        ends[rtol] = O.trace(f, O.make_params(pd), cfg["x0"])["xf"]
    e6 = np.abs(ends[1e-6][0] - ends[1e-11][0]).max()
    e8 = np.abs(ends[1e-8][0] - ends[1e-11][0]).max()
    # bounded by n_steps * rtol (Eq. 4 is a per-step control), and monotone in the tolerance
    assert e8 < e6 and e8 < 200 * 1e-8 and e6 < 200 * 1e-6


def test_stop_logic(oracle):
    O = oracle
    cfg = W.config(0, n=8, T=2e-6)
    f = O.Field(cfg["field"])
    x0 = cfg["x0"].copy()
    x0[0, 0] = 1.2                                  # born outside: status 1, t_stop 0, state returned
    x0[0, 1] = 0.999
    x0[3, 1] = 0.05 * W.V_TOTAL                     # barely trapped near the edge, drifts out or stays
    r = O.trace(f, O.make_params(cfg["params"]), x0)
    assert r["status"][0] == 1 and r["tstop"][0] == 0.0 and np.array_equal(r["xf"][:, 0], x0[:, 0])
    assert r["nacc"][0] == 0
    alive = r["status"] == 0
    assert np.all(r["tstop"][alive] == 2e-6)        # the last step lands exactly on T (reading S4)
    lost = r["status"] == 1
    assert np.all(r["xf"][0][lost] >= 1.0)          # loss = first accepted state with s >= 1 (S5)
    assert np.all(r["xf"][0][alive] < 1.0)
    # max_steps => status 3 ; tiny max_consecutive_rejects with absurd dt0 => status 2
    pd = dict(cfg["params"], max_steps=5)
    r3 = O.trace(f, O.make_params(pd), cfg["x0"])
    assert np.all(r3["status"] == 3) and np.all(r3["nacc"] + r3["nrej"] == 5)
    pd = dict(cfg["params"], dt0=1e-3, dtmax=1e-3, max_consecutive_rejects=2)
    r2 = O.trace(f, O.make_params(pd), cfg["x0"])
    assert np.all(r2["status"] == 2) and np.all(r2["nrej"] == 2)


def test_particle_crossing_the_edge_is_lost_and_extrapolates(oracle):
    """stages beyond s = 1 use the last cell's polynomial; tracing stops at s >= 1."""
    O = oracle
    cfg = W.config(0, n=64, T=1e-4)
    f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
    r = O.trace(f, p, cfg["x0"])
    lost = np.flatnonzero(r["status"] == 1)
    assert len(lost) >= 1
    assert np.all(r["xf"][0][lost] >= 1.0) and np.all(r["xf"][0][lost] < 1.05)
    assert np.all(r["tstop"][lost] < 1e-4) and np.all(r["tstop"][lost] > 0)
    # table energy drift is interpolation-limited (reading Q3): same order as O(h^4)
    keep = np.flatnonzero(r["status"] == 0)
    B0v = O.tricubic_many(f, cfg["x0"][:3])[0]
    Bf = O.tricubic_many(f, r["xf"][:3])[0]
    mu = (W.V_TOTAL ** 2 - cfg["x0"][3] ** 2) / (2 * B0v)
    E = 0.5 * r["xf"][3] ** 2 + mu * Bf
    drift = np.abs(E / (0.5 * W.V_TOTAL ** 2) - 1)
    assert np.median(drift[keep]) < 5e-6


def test_cartesian_trace_on_tables_conserves_pphi(oracle):
    """Config 3 at reduced size: canonical toroidal momentum and energy from tabulated columns."""
    O = oracle
    cfg = W.config(3, n=6, T=2e-5, ncell=[24, 24, 4])
    f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
    r = O.trace(f, p, cfg["x0"])
    assert np.all(r["status"] == 0)

    def inv(x):
        R = np.hypot(x[0], x[1])
        v = O.tricubic_many(f, np.array([R, x[2], np.arctan2(x[1], x[0])]))
        modB = np.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
        return R, v, modB

    R0_, v0, B0_ = inv(cfg["x0"])
    R1_, v1, B1_ = inv(r["xf"])
    mu = (W.V_TOTAL ** 2 - cfg["x0"][3] ** 2) / (2 * B0_)
    E1 = 0.5 * r["xf"][3] ** 2 + mu * B1_
    assert np.max(np.abs(E1 / (0.5 * W.V_TOTAL ** 2) - 1)) < 1e-6
    P0 = W.ALPHA_MASS * R0_ * v0[1] / B0_ * cfg["x0"][3] + W.ALPHA_CHARGE * v0[6]
    P1 = W.ALPHA_MASS * R1_ * v1[1] / B1_ * r["xf"][3] + W.ALPHA_CHARGE * v1[6]
    assert np.max(np.abs(P1 - P0)) < 1e-6 * W.ALPHA_CHARGE * W.PSI_EDGE_CYL


def test_estimator_matches_numpy(oracle):
    O = oracle
    rng = np.random.default_rng(43)
    status = rng.integers(0, 3, size=1000).astype(np.int32)
    tstop = rng.random(1000)
    out = O.estimate(0, status=status, tstop=tstop)
    g = (status == 1).astype(float)
    assert out[2] == g.sum() and abs(out[0] - g.mean()) < 1e-15
    assert abs(out[1] - math.sqrt(g.mean() * (1 - g.mean()) / (len(g) - 1))) < 1e-12
    out = O.estimate(1, status=status, tstop=tstop)
    assert abs(out[0] - tstop.mean()) < 1e-14 and abs(out[1] - tstop.std(ddof=0) / math.sqrt(999)) < 1e-12
    out = O.estimate(2, status=status, tstop=tstop, g_user=tstop ** 2)
    assert abs(out[0] - (tstop ** 2).mean()) < 1e-14


def test_scripted_replay_reproduces_the_adaptive_trace(oracle):
    """orc_trace_scripted walks a given accepted-step sequence with no accept/reject decision.  Pins:
    (i) fed the step sizes the adaptive trace accepted, it lands on the adaptive trace's end state (the
    sizes are differences of recorded times, equal to the attempted h up to one rounding of t);
    (ii) the error ratios it reports are all <= 1 (they were accepted) and equal one-step ratios
    computed independently through step_once from the recorded states;
    (iii) a script of one step equals step_once; an empty script returns the initial state."""
    O = oracle
    for idx, kw in ((0, dict(n=3, T=1e-5)), (3, dict(n=2, T=1e-5, ncell=[12, 11, 5])),
                    (4, dict(n=2, T=1e-5, ncell=[12, 10, 9]))):
        cfg = W.config(idx, **kw)
        f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
        full = O.trace(f, p, cfg["x0"])
        for i in range(cfg["x0"].shape[1]):
            x0 = cfg["x0"][:, i]
            traj, ts, st = O.trace_record(f, p, x0)
            h = np.diff(traj[:, 0])
            assert len(h) == full["nacc"][i]
            xf, t_end, st2, r = O.trace_scripted(f, p, x0, h)
            assert st2 == st == full["status"][i] and len(r) == len(h)
            assert abs(t_end - ts) <= 1e-15 * ts * len(h)
            d = xf - full["xf"][:, i]
            d[1] = math.remainder(d[1], 2 * math.pi)
            sc = np.maximum(np.abs(full["xf"][:, i]), [1.0, 1.0, 1.0, W.V_TOTAL])
            assert np.all(np.abs(d) <= 1e-12 * sc * len(h)), d
            assert np.all(r <= 1.0 + 1e-3)
            for j in (0, len(h) // 2, len(h) - 2):
                # traj row = (t, state in the API's coordinates).  r is a quotient of a difference that
                # cancels to ~1e-9 of its terms: a few per cent of round-off noise is its own precision
                # (DESIGN.md "Tolerances"); the clamped last step can be arbitrarily short and is left out
                _, rj, _ = O.step_once(f, p, traj[j, 1:5], traj[j, 0], h[j])
                assert abs(rj - r[j]) <= 5e-2 * max(r[j], 1e-3), (j, rj, r[j])
            x1, t1, s1, r1 = O.trace_scripted(f, p, x0, h[:1])
            xs, rs, _ = O.step_once(f, p, x0, 0.0, h[0])
            assert np.array_equal(x1, xs) and r1[0] == rs and t1 == h[0]
            xe, te, se, re = O.trace_scripted(f, p, x0, np.zeros(0))
            de = xe - x0
            if idx != 3:
                de[1] = math.remainder(de[1], 2 * math.pi)   # theta is returned in (-pi, pi]
            assert te == 0.0 and len(re) == 0 and np.all(np.abs(de) <= 1e-15 * np.maximum(1.0, np.abs(x0)))


def test_default_steps_hand_values(oracle):
    """Pin of reading S3 (the paper is silent on the initial / maximum step): dtmax = (pi/2) L / v_total,
    dt0 = 1e-3 dtmax, L = |G| / |B|(first node) for a Boozer grid, L = R_max for the cylindrical grid.
    Hand values: 3.5 MeV alphas, v_total = 1.29963e7 m/s; config 0 has |B|(node 0) = B0 exactly,
    so L = R0 = 7.75 m and dtmax = (pi/2) 7.75 / 1.29963e7 = 9.37e-7 s."""
    O = oracle
    v = math.sqrt(2.0 * 3.5e6 * 1.602176634e-19 / 6.64e-27)          # retyped from the constants, not from W
    assert abs(v - 1.29963e7) < 5e2
    cfg = W.config(0, n=1)
    p0 = O.make_params(dict(cfg["params"], dt0=0.0, dtmax=0.0))
    dt0, dtmax = O.default_steps(O.Field(cfg["field"]), p0)
    assert abs(dtmax - 9.37e-7) < 5e-10                               # the survey's printed three digits
    assert abs(dtmax / (0.5 * math.pi * 7.75 / v) - 1) < 1e-14 and abs(dt0 / (1e-3 * dtmax) - 1) < 1e-15
    # a field whose first node is not B0: L follows the node (m = 0 modes shift |B| on the axis)
    cfg2 = W.config(2, n=1, ncell=[4, 4, 4])
    b00 = float(cfg2["field"]["nodes"][0, 0, 0, 0])
    assert abs(b00 / W.B0 - 1) > 1e-3                                 # the case really differs from config 0
    dt0, dtmax = O.default_steps(O.Field(cfg2["field"]), O.make_params(dict(cfg2["params"], dt0=0.0, dtmax=0.0)))
    assert abs(dtmax / (0.5 * math.pi * (W.B0 * W.R0 / abs(b00)) / v) - 1) < 1e-14
    # cylindrical grid: L = R_max = R0 + 1.25 a (reading Q12)
    cfg3 = W.config(3, n=1, ncell=[4, 4, 2])
    dt0, dtmax = O.default_steps(O.Field(cfg3["field"]), O.make_params(dict(cfg3["params"], dt0=0.0, dtmax=0.0)))
    assert abs(dtmax / (0.5 * math.pi * (7.75 + 1.25 * 1.7) / v) - 1) < 1e-14
    # explicit values win; an explicit dt0 above dtmax is clamped
    f0 = O.Field(cfg["field"])
    assert O.default_steps(f0, O.make_params(dict(cfg["params"], dt0=2e-9, dtmax=3e-7))) == (2e-9, 3e-7)
    assert O.default_steps(f0, O.make_params(dict(cfg["params"], dt0=1e-3, dtmax=3e-7))) == (3e-7, 3e-7)
    assert O.default_steps(f0, O.make_params(dict(cfg["params"], dt0=5e-9, dtmax=0.0)))[0] == 5e-9


def test_default_steps_drive_the_trace(oracle):
    """orc_trace with dt0 = dtmax = 0 equals orc_trace with the values orc_default_steps returns, bit for bit."""
    O = oracle
    cfg = W.config(2, n=6, T=2e-6, ncell=[6, 5, 4])
    f = O.Field(cfg["field"])
    pdef = dict(cfg["params"], dt0=0.0, dtmax=0.0)
    dt0, dtmax = O.default_steps(f, O.make_params(pdef))
    a = O.trace(f, O.make_params(pdef), cfg["x0"])
    b = O.trace(f, O.make_params(dict(cfg["params"], dt0=dt0, dtmax=dtmax)), cfg["x0"])
    assert np.array_equal(a["xf"], b["xf"]) and np.array_equal(a["nacc"], b["nacc"])
    c = O.trace(f, O.make_params(cfg["params"]), cfg["x0"])          # L = R0 instead of |G|/|B|(node 0): another run
    assert not np.array_equal(a["nacc"] + a["nrej"], c["nacc"] + c["nrej"]) or not np.array_equal(a["xf"], c["xf"])


def test_step_sequences_are_not_reproducible_across_arithmetics(oracle):
    """Reading Q13, measured with the oracle alone: on the tabulated Boozer fields the sequence of
    accepted / rejected attempts is chaotic -- the tricubic interpolant's derivative jumps at cell faces make
    Eq. 4's error ratio a rough function of the step length -- so a relative change of 1e-12 in rtol (less than
    any two correct arithmetics differ by) changes the step counts of most particles within a 1e-5 s window,
    while the end states still agree within the method's global error.  In the smooth axisymmetric field of
    config 3 the counts are reproducible.  This is why the GPU parity of whole trajectories is taken on a scripted
    step sequence, and the adaptive run is compared per particle only on config 3."""
    O = oracle
    out = {}
    for idx, kw in ((0, dict(n=64, T=1e-5)), (3, dict(n=50, T=1e-5, ncell=[12, 11, 5]))):
        cfg = W.config(idx, **kw)
        f = O.Field(cfg["field"])
        a = O.trace(f, O.make_params(cfg["params"]), cfg["x0"])
        b = O.trace(f, O.make_params(dict(cfg["params"], rtol=cfg["params"]["rtol"] * (1 + 1e-12))), cfg["x0"])
        same = (a["nacc"] == b["nacc"]) & (a["nrej"] == b["nrej"])
        out[idx] = same.mean()
        # both runs are correct: end states within the global error nacc * rtol of each other
        ya = np.array([a["xf"][0] * np.cos(a["xf"][1]), a["xf"][0] * np.sin(a["xf"][1]), a["xf"][2], a["xf"][3]]) \
            if idx == 0 else a["xf"]
        yb = np.array([b["xf"][0] * np.cos(b["xf"][1]), b["xf"][0] * np.sin(b["xf"][1]), b["xf"][2], b["xf"][3]]) \
            if idx == 0 else b["xf"]
        scale = np.maximum(np.array([1.0, 1.0, 1.0, W.V_TOTAL])[:, None], np.abs(ya))
        assert np.all(np.abs(ya - yb) <= 8 * a["nacc"][None, :] * 1e-9 * scale)
    assert out[0] < 0.5, out      # measured: 5 of 64 particles keep their counts
    assert out[3] == 1.0, out     # measured: 50 of 50


def test_hermite_interpolant_reproduces_cubic_motion(oracle):
    """Reading S5b: the interpolant of a step's end states and end derivatives is exact for motion that is cubic
    in time (closed form, retyped here), and hits both ends."""
    O = oracle
    rng = np.random.default_rng(11)
    c = rng.normal(size=(4, 4))                    # y_i(t) = c0 + c1 t + c2 t^2 + c3 t^3
    yt = lambda t: c[:, 0] + c[:, 1] * t + c[:, 2] * t ** 2 + c[:, 3] * t ** 3
    dyt = lambda t: c[:, 1] + 2 * c[:, 2] * t + 3 * c[:, 3] * t ** 2
    t0, h = 0.3, 0.7
    for th in (0.0, 0.125, 0.5, 0.9, 1.0):
        y = O.hermite_state(yt(t0), dyt(t0), yt(t0 + h), dyt(t0 + h), h, th)
        assert np.allclose(y, yt(t0 + th * h), rtol=0, atol=1e-14)


def test_loss_refine_finds_the_crossing_of_a_known_orbit(oracle):
    """Reading S5b on an outward spiral in the pseudo-Cartesian plane whose radius s(t) is known in closed form:
    y = (s cos w t, s sin w t) with s(t) = s0 + v t crosses s = 1 at t* = (1 - s0)/v.  The cubic interpolant of a
    short step finds t* to O(h^4); the bracket is as tight as 48 bisections make it."""
    O = oracle
    cfg = W.config(0, n=1, T=1e-6)
    f = O.Field(cfg["field"])
    s0, v, w = 0.98, 40.0, 300.0
    y = lambda t: np.array([(s0 + v * t) * math.cos(w * t), (s0 + v * t) * math.sin(w * t), 0.1 + t, 1e5])
    dy = lambda t: np.array([v * math.cos(w * t) - (s0 + v * t) * w * math.sin(w * t),
                             v * math.sin(w * t) + (s0 + v * t) * w * math.cos(w * t), 1.0, 0.0])
    tstar = (1.0 - s0) / v
    errs = []
    for h in (8e-4, 4e-4):
        t0 = tstar - 0.37 * h
        th, yl = O.loss_refine(f, y(t0), dy(t0), y(t0 + h), dy(t0 + h), h)
        assert 0.0 < th <= 1.0
        assert math.hypot(yl[0], yl[1]) >= 1.0                      # the returned state is beyond the boundary ...
        ybelow = O.hermite_state(y(t0), dy(t0), y(t0 + h), dy(t0 + h), h, th - 2.0 ** -40)
        assert math.hypot(ybelow[0], ybelow[1]) < 1.0               # ... and a hair earlier it is not
        errs.append(abs(t0 + th * h - tstar))
    assert errs[0] < 1e-3 * 8e-4                                    # far inside the step
    assert errs[1] < errs[0] / 8.0                                  # fourth order in h (16x; 8x asserted)


def test_loss_time_mode_sharpens_the_loss_time(oracle):
    """Reading S5 puts the loss time at the END of the crossing step (an error of up to one step length); reading
    S5b inside it.  Against a run at a 100x tighter tolerance (steps ~2.5x shorter, orbit converged to 1e-9) the
    refined loss times of a loose run are much closer than the unrefined ones; states that reached T are
    untouched by the mode; the step counts are identical."""
    O = oracle
    cfg = W.config(0, n=64, T=1e-4)
    f = O.Field(cfg["field"])
    loose0 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-7)), cfg["x0"])
    loose1 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-7, loss_time_mode=1)), cfg["x0"])
    tight1 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-11, loss_time_mode=1)), cfg["x0"])
    assert np.array_equal(loose0["status"], loose1["status"]) and np.array_equal(loose0["nacc"], loose1["nacc"])
    kept = loose0["status"] == 0
    assert np.array_equal(loose0["xf"][:, kept], loose1["xf"][:, kept])
    lost = np.flatnonzero((loose0["status"] == 1) & (tight1["status"] == 1))
    assert len(lost) >= 3
    assert np.all(loose1["tstop"][lost] <= loose0["tstop"][lost])
    assert np.all(loose1["xf"][0][lost] >= 1.0) and np.all(loose1["xf"][0][lost] < 1.0 + 1e-9)
    e0 = np.abs(loose0["tstop"][lost] - tight1["tstop"][lost])
    e1 = np.abs(loose1["tstop"][lost] - tight1["tstop"][lost])
    assert np.median(e1) < 0.05 * np.median(e0)


def test_derivative_of_interpolant_mode(oracle):
    """Reading R1c: only |B| tabulated, its derivatives taken from the interpolant.  (1) On a field that is one
    tricubic polynomial per variable (one cell) the four-table mode holds the exact derivatives in its columns, so both
    modes give the same right-hand side.  (2) On the config-0 tables the right-hand side now jumps at cell faces:
    the controller takes more and rejects more steps (SURVEY Q2's probe), and the energy drift stays at the level of
    the four-table mode (no better, no more than ~3x worse)."""
    O = oracle
    rng = np.random.default_rng(9)
    c = 0.02 * rng.normal(size=(4, 3, 3))
    k = [1, 1, 1]
    lo, hi = [0.0, 0.0, 0.0], [1.0, 2 * math.pi, 2 * math.pi / 4]
    ax = [np.linspace(lo[d], hi[d], 4) for d in range(3)]
    P = lambda s, th, ze: W.B0 * (1 + sum(c[i, j, l] * s ** i * th ** j * ze ** l for i in range(4) for j in range(3) for l in range(3)))
    Ps = lambda s, th, ze: W.B0 * sum(i * c[i, j, l] * s ** (i - 1) * th ** j * ze ** l for i in range(1, 4) for j in range(3) for l in range(3))
    Pt = lambda s, th, ze: W.B0 * sum(j * c[i, j, l] * s ** i * th ** (j - 1) * ze ** l for i in range(4) for j in range(1, 3) for l in range(3))
    Pz = lambda s, th, ze: W.B0 * sum(l * c[i, j, l] * s ** i * th ** j * ze ** (l - 1) for i in range(4) for j in range(3) for l in range(1, 3))
    S, T, Z = np.meshgrid(*ax, indexing="ij")
    fd4 = dict(coord=0, ncell=k, lo=lo, hi=hi, nfp=4, nquant=4, nodes=np.stack([P(S, T, Z), Ps(S, T, Z), Pt(S, T, Z), Pz(S, T, Z)]),
               G0=W.G0, I0=0.0, iota0=W.IOTA0, iota1=W.IOTA1, psi0=W.PSI0)
    fd1 = dict(fd4, nquant=1, nodes=fd4["nodes"][:1])
    p = O.make_params(W.base_params(1e-5))
    for _ in range(10):
        s, th, ze = 0.1 + 0.8 * rng.random(), 0.2 + 5.8 * rng.random(), 0.1 + 1.3 * rng.random()
        y = [s * math.cos(th), s * math.sin(th), ze, 0.4 * W.V_TOTAL]
        d4, fv4 = O.rhs(O.Field(fd4), p, 3e12, 0.0, y)
        d1, fv1 = O.rhs(O.Field(fd1), p, 3e12, 0.0, y)
        assert np.allclose(fv1, fv4, rtol=1e-11, atol=1e-11 * W.B0)
        assert np.allclose(d1, d4, rtol=1e-9, atol=0)
    cfg = W.config(0, n=24, T=2e-5)
    f4 = O.Field(cfg["field"])
    f1 = O.Field(dict(cfg["field"], nquant=1, nodes=cfg["field"]["nodes"][:1]))
    p = O.make_params(cfg["params"])
    r4, r1 = O.trace(f4, p, cfg["x0"]), O.trace(f1, p, cfg["x0"])

    def drift(f, r):
        keep = r["status"] == 0
        B0v = O.tricubic_many(f, cfg["x0"][:3])[0]
        Bf = O.tricubic_many(f, r["xf"][:3])[0]
        mu = (W.V_TOTAL ** 2 - cfg["x0"][3] ** 2) / (2 * B0v)
        E = 0.5 * r["xf"][3] ** 2 + mu * Bf
        return np.abs(E / (0.5 * W.V_TOTAL ** 2) - 1)[keep]

    d4, d1 = drift(f4, r4), drift(f1, r1)
    assert np.median(d1) < 3 * np.median(d4) + 1e-7
    assert r1["nacc"].sum() > 1.2 * r4["nacc"].sum()          # more steps ...
    rej = lambda r: r["nrej"].sum() / (r["nacc"].sum() + r["nrej"].sum())
    assert rej(r1) > rej(r4)                                  # ... and more of the attempts rejected


def _psi_closed_form(x):
    """Config 3's level function in closed form (workloads.cyl_field_values): psi = B0/(2 q0) [(R-R0)^2 + (Z/kappa)^2].
    It is a quadratic in (R, Z), so its local tricubic reproduces it to rounding: the interpolated level the tracer
    tests and this expression agree to ~1e-15 psi_edge, and the loss surface is the ellipse
    (R-R0)^2 + (Z/kappa)^2 = a^2."""
    R = np.hypot(x[0], x[1])
    return (W.B0 / (2.0 * W.Q0_CYL)) * ((R - W.R0) ** 2 + (x[2] / W.KAPPA_CYL) ** 2)


def test_cartesian_loss_is_the_first_accepted_state_beyond_the_closed_form_surface(oracle):
    """"in Cartesian coordinates we detect a sign change in the interpolation of a signed distance
    function" -- here the level function psi - psi_edge in column 6 (R3).  Pins of orc_is_lost's
    cylindrical branch against the closed-form surface, none of which uses the oracle's own interpolation:
    born outside => status 1, t_stop 0, state unchanged, no step; born just inside => steps are taken; along every
    recorded trajectory the status flips exactly at the first accepted end state with psi >= psi_edge (all earlier
    states are inside, the last one of a lost particle is outside, particles that reach T never were outside)."""
    O = oracle
    cfg = W.config(3, n=4, T=2e-5, ncell=[12, 11, 5])
    f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
    edge = W.PSI_EDGE_CYL
    # interpolated level == closed form on and around the surface (cubic exactness), so the pin below has teeth
    rng = np.random.default_rng(11)
    xs = W.cyl_births(rng, 32, psi_frac=1.0)
    R, phi = np.hypot(xs[0], xs[1]), np.mod(np.arctan2(xs[1], xs[0]), 2 * np.pi)
    lev = O.tricubic_many(f, np.array([R, xs[2], phi]))[6]
    assert np.max(np.abs(lev - _psi_closed_form(xs))) < 1e-13 * edge
    # born outside / just inside
    out = W.cyl_births(np.random.default_rng(12), 8, psi_frac=1.1)
    r = O.trace(f, p, out)
    assert np.all(r["status"] == 1) and np.all(r["tstop"] == 0.0) and np.array_equal(r["xf"], out)
    assert np.all(r["nacc"] == 0) and np.all(r["nrej"] == 0)
    inside = W.cyl_births(np.random.default_rng(12), 8, psi_frac=1.0 - 1e-6)
    r = O.trace(f, p, inside)
    assert np.all(r["tstop"] > 0.0) and np.all(r["nacc"] >= 1)
    # crossing: births on 0.97 psi_edge, many leave within the window
    x0 = W.cyl_births(np.random.default_rng(13), 64, psi_frac=0.97)
    r = O.trace(f, p, x0)
    nlost = int(np.sum(r["status"] == 1))
    assert 10 <= nlost <= 60, nlost                      # both outcomes are present
    margin = 1e-12 * edge
    for i in range(x0.shape[1]):
        traj, ts, st = O.trace_record(f, p, x0[:, i])
        assert st == r["status"][i] and ts == r["tstop"][i]
        psi = _psi_closed_form(traj[:, 1:5].T)
        assert np.all(np.abs(psi - edge) > margin)       # no state so close that rounding decides
        assert np.all(psi[:-1] < edge), i                # every state before the last is inside ...
        if st == 1:
            assert psi[-1] >= edge and traj[-1, 0] == ts and ts < 2e-5, i    # ... and a lost one ends outside
            assert np.array_equal(traj[-1, 1:5], r["xf"][:, i])
        else:
            assert st == 0 and psi[-1] < edge and ts == 2e-5, i
    # a wrong level column, or the Boozer flux psi0 in place of psi_edge, changes the verdicts: the closed form on the
    # final states alone separates the two classes
    pf = _psi_closed_form(r["xf"])
    assert np.array_equal(pf >= edge, r["status"] == 1)


def test_cartesian_loss_time_inside_the_step_ends_on_the_closed_form_surface(oracle):
    """Reading S5b for the cylindrical model (sign change of the interpolated level function; the root
    is looked for along the step's cubic Hermite interpolant, one table evaluation per bisection step).  Config 3's
    level function is a quadratic, so the surface is known in closed form and the oracle's interpolation is not
    needed to check it: with loss_time_mode 1 every lost particle ends ON the ellipse psi = psi_edge (from outside,
    within the bisection's resolution), at a time inside the crossing step; statuses, step counts and the particles
    that reach T are untouched; against a run at a 100x tighter tolerance the refined loss times of a loose run are
    much closer than the unrefined ones."""
    O = oracle
    cfg = W.config(3, n=4, T=2e-5, ncell=[12, 11, 5])
    f = O.Field(cfg["field"])
    x0 = W.cyl_births(np.random.default_rng(13), 64, psi_frac=0.97)
    edge = W.PSI_EDGE_CYL
    loose0 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-6)), x0)
    loose1 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-6, loss_time_mode=1)), x0)
    tight1 = O.trace(f, O.make_params(dict(cfg["params"], rtol=1e-11, atol=1e-14, loss_time_mode=1)), x0)
    assert np.array_equal(loose0["status"], loose1["status"]) and np.array_equal(loose0["nacc"], loose1["nacc"])
    kept = loose0["status"] == 0
    assert np.array_equal(loose0["xf"][:, kept], loose1["xf"][:, kept])
    lost = np.flatnonzero((loose0["status"] == 1) & (tight1["status"] == 1))
    assert len(lost) >= 10
    psi0_, psi1_ = _psi_closed_form(loose0["xf"][:, lost]), _psi_closed_form(loose1["xf"][:, lost])
    assert np.all(psi0_ >= edge) and np.median(psi0_ / edge - 1) > 1e-6      # mode 0 ends well beyond the surface
    assert np.all(psi1_ >= edge * (1 - 1e-13)) and np.all(psi1_ < edge * (1 + 1e-9))   # mode 1 ends on it
    assert np.all(loose1["tstop"][lost] <= loose0["tstop"][lost]) and np.all(loose1["tstop"][lost] > 0)
    e0 = np.abs(loose0["tstop"][lost] - tight1["tstop"][lost])
    e1 = np.abs(loose1["tstop"][lost] - tight1["tstop"][lost])
    assert np.median(e1) < 0.05 * np.median(e0), (np.median(e1), np.median(e0))
    # the crossing step brackets the refined time (trajectory record of mode 0: its last two rows are the step's ends)
    for i in lost[:16]:
        traj, ts, st = O.trace_record(f, O.make_params(dict(cfg["params"], rtol=1e-6)), x0[:, i])
        assert traj[-2, 0] < loose1["tstop"][i] <= traj[-1, 0]


def test_lost_energy_measurement(oracle):
    """Reading G2 ("energy loss"): g = 1[lost] (vpar^2/2 + mu |B|(x_f)) / (v_total^2/2).
    (1) Hand value: a "lost" particle placed ON a grid node, where the interpolant returns the nodal value, which
    is the closed-form |B| of the workload (workloads.boozer_field_values) -- the oracle's interpolation does not
    enter the expected number.  (2) A particle that is not lost contributes 0 whatever its state.  (3) In a static
    field the guiding-centre energy is an invariant: every particle the tracer loses left with the energy it was
    born with, g = 1 to the interpolation-limited drift (a few 1e-6 on config 0's grid, reading Q3).  A dropped
    mu |B| term, a missing factor 1/2 or |B| taken at the wrong point fails (1) or (3)."""
    O = oracle
    cfg = W.config(0, n=64, T=1e-4)
    f, p = O.Field(cfg["field"]), O.make_params(cfg["params"])
    k = cfg["field"]["ncell"]
    node = (37, 20, 11)                                           # unique-node indices (s, theta, zeta)
    s, th, ze = node[0] / (3.0 * k[0]), 2 * math.pi * node[1] / (3.0 * k[1]), (2 * math.pi / W.NFP) * node[2] / (3.0 * k[2])
    B = float(W.boozer_field_values(cfg["field"]["modes"], s, th, ze)[0])
    assert B == cfg["field"]["nodes"][0][node]
    vpar, mu = 0.3 * W.V_TOTAL, 0.41 * W.V_TOTAL ** 2 / B
    xf = np.array([[s, 0.5], [th, 1.0], [ze, 0.2], [vpar, vpar]])
    g = O.lost_energy(f, p, xf, np.array([mu, mu]), np.array([1, 0], dtype=np.int32))
    assert abs(g[0] - (0.5 * 0.09 + 0.41) / 0.5) < 1e-13 and g[1] == 0.0
    r = O.trace(f, p, cfg["x0"])
    mu0 = np.array([O.mu_init(f, p, cfg["x0"][:, i]) for i in range(64)])
    g = O.lost_energy(f, p, r["xf"], mu0, r["status"])
    lost = r["status"] == 1
    assert lost.sum() >= 1 and np.all(g[~lost] == 0.0)
    assert np.all(np.abs(g[lost] - 1.0) < 2e-5)
    est = O.estimate(2, g_user=g)
    assert abs(est[0] - lost.mean()) < 2e-5 * max(lost.mean(), 1e-3)      # lost power fraction ~ loss fraction here


def test_exit_histogram_matches_numpy(oracle):
    """Reading G3 ("wall-loads"): lost particles per bin of the exit point.  Against numpy.histogram2d on
    angles reduced with np.mod (a library routine and an independent reduction), on both coordinate systems; hand-placed
    particles land in the bins worked out by hand; particles that are not lost are not counted; values outside a
    non-periodic range fall into the end bins."""
    O = oracle
    rng = np.random.default_rng(21)
    n = 5000
    status = (rng.random(n) < 0.6).astype(np.int32)
    # Boozer: theta in (-pi, pi], zeta unreduced (as catapult_trace returns them)
    cfg = W.config(0, n=1, T=1e-6)
    f = O.Field(cfg["field"])
    xf = np.array([1.0 + 0.01 * rng.random(n), rng.uniform(-math.pi, math.pi, n), rng.uniform(-40.0, 40.0, n), rng.normal(size=n)])
    per = 2 * math.pi / W.NFP
    h = O.exit_histogram(f, xf, status, 12, 7)
    lost = status == 1
    want, _, _ = np.histogram2d(np.mod(xf[1][lost], 2 * math.pi), np.mod(xf[2][lost], per), bins=[12, 7],
                                range=[[0, 2 * math.pi], [0, per]])
    assert h.sum() == lost.sum() and np.array_equal(h, want.astype(np.int64))
    hand = np.array([[1.0, 1.0, 1.0], [0.1, -0.1, math.pi - 1e-9], [0.5 * per / 7, per + 2.5 * per / 7, -0.5 * per / 7], [0, 0, 0]])
    hh = O.exit_histogram(f, hand, np.array([1, 1, 1], dtype=np.int32), 12, 7)
    assert hh[0, 0] == 1 and hh[11, 2] == 1 and hh[5, 6] == 1 and hh.sum() == 3
    # cylindrical: phi from (x, y), Z clamped into the grid's range
    c3 = W.config(3, n=1, T=1e-6, ncell=[4, 4, 2])
    f3 = O.Field(c3["field"])
    R, phi = rng.uniform(6.0, 9.5, n), rng.uniform(-math.pi, math.pi, n)
    zlo, zhi = c3["field"]["lo"][1], c3["field"]["hi"][1]
    Z = rng.uniform(1.2 * zlo, 1.2 * zhi, n)
    x3 = np.array([R * np.cos(phi), R * np.sin(phi), Z, rng.normal(size=n)])
    h3 = O.exit_histogram(f3, x3, status, 16, 9)
    want3, _, _ = np.histogram2d(np.mod(phi[lost], 2 * math.pi), np.clip(Z[lost], zlo, np.nextafter(zhi, zlo)), bins=[16, 9],
                                 range=[[0, 2 * math.pi], [zlo, zhi]])
    assert h3.sum() == lost.sum()
    # numpy's bin edges are lo + k (hi - lo) / nb, the oracle's rule is floor((a - lo) / span * nb): equal except for
    # a point within a rounding of an edge; none of the 3000 seeded points is
    assert np.array_equal(h3, want3.astype(np.int64))
