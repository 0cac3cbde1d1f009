"""Seeded synthetic inputs shared by the CUDA path and the oracle (numpy only).

Holds none of the method's arithmetic: it samples closed-form fields on the interpolant grid and
draws birth ensembles.  The five configurations are BASELINE.json `configs[0..4]`; they stand in
for the equilibria of the paper's refs [13],[14], which are not available.
Recipe and readings (Q1, Q4, Q10, Q12): DESIGN.md "Inputs".

A field dict has: coord (0 Boozer (s,theta,zeta) / 1 cylindrical (R,Z,phi)), ncell[3] (cells per
dimension, nodes per dimension = 3*ncell+1), lo[3], hi[3], nfp, nquant,
nodes [nquant][n0][n1][n2] float64, G0, I0, iota0, iota1, psi0.
A params dict mirrors catapult_trace_params (include/catapult.h).
x0 is [4][n]: (s,theta,zeta,vpar) or (x,y,z,vpar).
"""
from __future__ import annotations

import math

import numpy as np

# shared constants (BASELINE.json configs)
ALPHA_MASS = 6.64e-27
E_CHARGE = 1.602176634e-19
ALPHA_CHARGE = 2.0 * E_CHARGE
ALPHA_ENERGY = 3.5e6 * E_CHARGE
B0 = 5.7
R0 = 7.75
A_MINOR = 1.7
NFP = 4
G0 = B0 * R0
PSI0 = B0 * A_MINOR * A_MINOR / 2.0
IOTA0, IOTA1 = 0.42, 0.1
Q0_CYL, KAPPA_CYL = 1.5, 1.6
PSI_EDGE_CYL = B0 * A_MINOR * A_MINOR / (2.0 * Q0_CYL)

V_TOTAL = math.sqrt(2.0 * ALPHA_ENERGY / ALPHA_MASS)


def base_params(T: float, rtol: float = 1e-9, atol: float = 1e-12, L: float = R0) -> dict:
    dtmax = 0.5 * math.pi * L / V_TOTAL
    return dict(mass=ALPHA_MASS, charge=ALPHA_CHARGE, energy=ALPHA_ENERGY, T=T, rtol=rtol,
                atol=atol, dt0=1e-3 * dtmax, dtmax=dtmax, max_steps=0,
                max_consecutive_rejects=500, saw_on=0, saw_m=0, saw_n=0, saw_Phi0=0.0,
                saw_s0=0.5, saw_w2=0.01, saw_omega=0.0)


# ---------------------------------------------------------------------------------------------
# Boozer fields:  |B| = B0 [1 + sum_{m,n} b_mn s^{m/2} cos(m theta - nfp n zeta)]
# ---------------------------------------------------------------------------------------------
def boozer_modes_cfg0():
    """(m, n, b_mn) of |B|=B0[1+0.1 sqrt(s) cos(theta)+0.05 sqrt(s) cos(theta-4 zeta)]."""
    return [(1, 0, 0.1), (1, 1, 0.05)]


def boozer_modes_random(seed: int = 2, mmax: int = 8, nmax: int = 8, rng=None):
    """b_mn ~ N(0,(0.08/(1+m+|n|))^2), m=0..mmax, n=-nmax..nmax, drawn m-major."""
    rng = np.random.default_rng(seed) if rng is None else rng
    modes = []
    for m in range(mmax + 1):
        for n in range(-nmax, nmax + 1):
            modes.append((m, n, float(rng.normal(0.0, 0.08 / (1 + m + abs(n))))))
    return modes


def boozer_field_values(modes, s, theta, zeta, s_floor: float = 0.0):
    """Closed-form (|B|, d/ds, d/dtheta, d/dzeta) at broadcastable points.

    The d/ds value is taken at max(s, s_floor) (reading Q4: s^(-1/2) is singular on the axis)."""
    s = np.asarray(s, dtype=np.float64)
    theta = np.asarray(theta, dtype=np.float64)
    zeta = np.asarray(zeta, dtype=np.float64)
    sf = np.maximum(s, s_floor)
    b = 1.0
    bs = 0.0
    bt = 0.0
    bz = 0.0
    for (m, n, c) in modes:
        ang = m * theta - NFP * n * zeta
        sm = s ** (0.5 * m) if m > 0 else np.ones_like(s)
        b = b + c * sm * np.cos(ang)
        if m > 0:
            bs = bs + c * (0.5 * m) * sf ** (0.5 * m - 1.0) * np.cos(ang)
        bt = bt + c * sm * (-m) * np.sin(ang)
        bz = bz + c * sm * (NFP * n) * np.sin(ang)
    return B0 * b, B0 * bs, B0 * bt, B0 * bz


def boozer_field(modes, ncell) -> dict:
    k0, k1, k2 = (int(v) for v in ncell)
    n0, n1, n2 = 3 * k0 + 1, 3 * k1 + 1, 3 * k2 + 1
    s = np.arange(n0, dtype=np.float64) / (3.0 * k0)
    th = 2.0 * math.pi * np.arange(n1, dtype=np.float64) / (3.0 * k1)
    ze = (2.0 * math.pi / NFP) * np.arange(n2, dtype=np.float64) / (3.0 * k2)
    s_floor = 0.5 / (3.0 * k0)
    sf = np.maximum(s, s_floor)
    nodes = np.zeros((4, n0, n1, n2))
    nodes[0] += 1.0
    # group by m: s^{m/2} (outer) C_m(theta,zeta)
    by_m = {}
    for (m, n, c) in modes:
        by_m.setdefault(m, []).append((n, c))
    TH, ZE = np.meshgrid(th, ze, indexing="ij")
    for m, lst in by_m.items():
        Cc = np.zeros_like(TH)
        Ct = np.zeros_like(TH)
        Cz = np.zeros_like(TH)
        for (n, c) in lst:
            ang = m * TH - NFP * n * ZE
            cs, sn = np.cos(ang), np.sin(ang)
            Cc += c * cs
            Ct += c * (-m) * sn
            Cz += c * (NFP * n) * sn
        sm = s ** (0.5 * m) if m > 0 else np.ones_like(s)
        nodes[0] += sm[:, None, None] * Cc[None]
        if m > 0:
            dsm = (0.5 * m) * sf ** (0.5 * m - 1.0)
            nodes[1] += dsm[:, None, None] * Cc[None]
        nodes[2] += sm[:, None, None] * Ct[None]
        nodes[3] += sm[:, None, None] * Cz[None]
    nodes *= B0
    return dict(coord=0, ncell=[k0, k1, k2], lo=[0.0, 0.0, 0.0],
                hi=[1.0, 2.0 * math.pi, 2.0 * math.pi / NFP], nfp=NFP, nquant=4, nodes=nodes,
                G0=G0, I0=0.0, iota0=IOTA0, iota1=IOTA1, psi0=PSI0, modes=list(modes))


def boozer_births(rng, n: int, s_range=None, s_fixed=None) -> np.ndarray:
    """Draw order: [s,] theta, zeta, xi=vpar/v (reading Q10: zeta on [0,2pi))."""
    x0 = np.zeros((4, n))
    if s_fixed is not None:
        x0[0] = s_fixed
    else:
        x0[0] = s_range[0] + (s_range[1] - s_range[0]) * rng.random(n)
    x0[1] = 2.0 * math.pi * rng.random(n)
    x0[2] = 2.0 * math.pi * rng.random(n)
    x0[3] = (2.0 * rng.random(n) - 1.0) * V_TOTAL
    return x0


# ---------------------------------------------------------------------------------------------
# Cylindrical-grid axisymmetric field (config 3)
# ---------------------------------------------------------------------------------------------
def cyl_field_values(R, Z):
    """Closed-form (B_R,B_phi,B_Z,d|B|/dR,(1/R)d|B|/dphi,d|B|/dZ,psi) of
    B_phi=B0 R0/R, psi=(B0/(2 q0))[(R-R0)^2+(Z/kappa)^2], B_R=-psi_Z/R, B_Z=psi_R/R."""
    R = np.asarray(R, dtype=np.float64)
    Z = np.asarray(Z, dtype=np.float64)
    psi_R = (B0 / Q0_CYL) * (R - R0)
    psi_Z = (B0 / Q0_CYL) * Z / KAPPA_CYL ** 2
    psi_RR = B0 / Q0_CYL
    psi_ZZ = B0 / (Q0_CYL * KAPPA_CYL ** 2)
    psi = (B0 / (2.0 * Q0_CYL)) * ((R - R0) ** 2 + (Z / KAPPA_CYL) ** 2)
    BR = -psi_Z / R
    BZ = psi_R / R
    Bp = B0 * R0 / R
    modB = np.sqrt(BR * BR + Bp * Bp + BZ * BZ)
    num = (B0 * R0) ** 2 + psi_R ** 2 + psi_Z ** 2
    dB2_dR = -2.0 * num / R ** 3 + 2.0 * psi_R * psi_RR / R ** 2
    dB2_dZ = 2.0 * psi_Z * psi_ZZ / R ** 2
    return BR, Bp, BZ, dB2_dR / (2.0 * modB), np.zeros_like(modB), dB2_dZ / (2.0 * modB), psi


def cyl_field(ncell) -> dict:
    k0, k1, k2 = (int(v) for v in ncell)
    lo = [R0 - 1.25 * A_MINOR, -1.25 * KAPPA_CYL * A_MINOR, 0.0]
    hi = [R0 + 1.25 * A_MINOR, 1.25 * KAPPA_CYL * A_MINOR, 2.0 * math.pi]
    n0, n1, n2 = 3 * k0 + 1, 3 * k1 + 1, 3 * k2 + 1
    R = lo[0] + (hi[0] - lo[0]) * np.arange(n0, dtype=np.float64) / (3.0 * k0)
    Z = lo[1] + (hi[1] - lo[1]) * np.arange(n1, dtype=np.float64) / (3.0 * k1)
    RR, ZZ = np.meshgrid(R, Z, indexing="ij")
    vals = cyl_field_values(RR, ZZ)
    nodes = np.zeros((7, n0, n1, n2))
    for q in range(7):
        nodes[q] = vals[q][:, :, None]
    return dict(coord=1, ncell=[k0, k1, k2], lo=lo, hi=hi, nfp=1, nquant=7, nodes=nodes,
                G0=0.0, I0=0.0, iota0=0.0, iota1=0.0, psi0=PSI_EDGE_CYL)


def cyl_births(rng, n: int, psi_frac: float = 0.25) -> np.ndarray:
    """Born on psi = psi_frac*psi_edge; draw order: poloidal angle, phi, xi."""
    rho = math.sqrt(psi_frac) * A_MINOR
    chi = 2.0 * math.pi * rng.random(n)
    phi = 2.0 * math.pi * rng.random(n)
    xi = 2.0 * rng.random(n) - 1.0
    R = R0 + rho * np.cos(chi)
    Z = KAPPA_CYL * rho * np.sin(chi)
    x0 = np.zeros((4, n))
    x0[0] = R * np.cos(phi)
    x0[1] = R * np.sin(phi)
    x0[2] = Z
    x0[3] = xi * V_TOTAL
    return x0


# ---------------------------------------------------------------------------------------------
# The five configurations
# ---------------------------------------------------------------------------------------------
CONFIG_NAMES = ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"]
FULL_N = [64, 10_000, 100_000, 100_000, 1_000_000]
FULL_T = [1e-4, 1e-3, 1e-2, 1e-2, 1e-2]
FULL_NCELL = [[16, 16, 16], [16, 16, 16], [64, 64, 64], [48, 48, 32], [64, 64, 64]]


def config(idx: int, n: int | None = None, T: float | None = None, ncell=None,
           with_nodes: bool = True, ensemble: int = 0) -> dict:
    """Returns dict(name, field, params, x0, g_kind).  n/T/ncell override the full sizes (parity
    tests run reduced sizes of the same recipe; the first n particles of the seeded stream).
    ensemble > 0 draws an independent birth ensemble of the same distribution (seed [seed, ensemble]):
    used only to give every rank of a multi-GPU weak-scaling run its own particles."""
    idx = int(idx)

    def _rng(seed):
        return np.random.default_rng(seed if ensemble == 0 else [seed, int(ensemble)])

    nfull = FULL_N[idx]
    n = nfull if n is None else int(n)
    T = FULL_T[idx] if T is None else float(T)
    ncell = FULL_NCELL[idx] if ncell is None else [int(v) for v in ncell]
    if idx in (0, 1):
        modes = boozer_modes_cfg0()
        rng = _rng(idx)
        x0 = boozer_births(rng, max(n, nfull), s_fixed=0.25)[:, :n]
        params = base_params(T)
        field = boozer_field(modes, ncell) if with_nodes else None
    elif idx in (2, 4):
        rng2 = np.random.default_rng(2)
        modes = boozer_modes_random(rng=rng2)
        prng = (rng2 if ensemble == 0 else _rng(2)) if idx == 2 else _rng(4)
        x0 = boozer_births(prng, max(n, nfull), s_range=(0.1, 0.9))[:, :n]
        params = base_params(T)
        if idx == 4:
            params.update(saw_on=1, saw_m=1, saw_n=1, saw_Phi0=1.0e3, saw_s0=0.5, saw_w2=0.01,
                          saw_omega=2.0 * math.pi * 1.0e5)
        field = boozer_field(modes, ncell) if with_nodes else None
    elif idx == 3:
        rng = _rng(3)
        x0 = cyl_births(rng, max(n, nfull))[:, :n]
        field = cyl_field(ncell) if with_nodes else None
        params = base_params(T, L=R0 + 1.25 * A_MINOR)
    else:
        raise ValueError(f"no config {idx}")
    return dict(name=CONFIG_NAMES[idx], field=field, params=params,
                x0=np.ascontiguousarray(x0), g_kind=0)


def nonvacuum_profiles(ncell0: int) -> dict:
    """Profiles of a non-vacuum Boozer equilibrium on the 3*ncell0+1 unique s-nodes (a NEXT-row input,
    not one of BASELINE.json's configs): G(s) = G0 (1 + 0.05 s - 0.02 s^2), I(s) = G0 (0.02 s + 0.01 s^3),
    iota(s) = 0.42 + 0.1 s + 0.05 s^2.  Merge into a Boozer field dict."""
    s = np.linspace(0.0, 1.0, 3 * ncell0 + 1)
    return dict(G_nodes=G0 * (1.0 + 0.05 * s - 0.02 * s ** 2), I_nodes=G0 * (0.02 * s + 0.01 * s ** 3),
                iota_nodes=0.42 + 0.1 * s + 0.05 * s ** 2)
