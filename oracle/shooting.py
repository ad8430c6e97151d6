"""Oracle of the shooting map of the overdetermined shooting method -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle/__init__.py
for who may import it).  Plain restatement of PAPER.md section 3.1 / 3.3 on the uniform mesh (xi(alpha) = alpha, E = 1, M = N);
shoot_segments below is the same map with the mesh-refinement strategy of section 2.2:

  (3.15) PAPER.md:197-200   eta^_k(0) = c_|k| for even k, phi^_k(0) = c_|k| for odd k, 1 <= |k| <= n, all other modes zero:
                            eta(x, 0) = sum_{k even} 2 c_k cos kx,  phi(x, 0) = sum_{k odd} 2 c_k cos kx  (eta about the mean level)
  (3.16) PAPER.md:204       T = c_0
  (3.17) PAPER.md:208       r_i = phi(alpha_i, T/4) sqrt(1/N),  f = r.r / 2
  (3.31) PAPER.md:296       J_ik = d r_i / d c_k:  k >= 1: phidot_k(alpha_i, T/4) sqrt(1/N) with qdot_k(0) = d q_0 / d c_k, advanced
                            together with q by (3.32);  k = 0: d/dT of phi at the time T/4, i.e. phi_t(., T/4) / 4 times the
                            weight (the paper prints the k = 0 row without the 1/4 of the chain rule: reading R13 of DESIGN.md;
                            tests/test_oracle_pins.py checks the row against finite differences (3.33))
The time integration is Oracle.rk_advance with nsteps steps of size T / (4 nsteps); phi_t at T/4 is Oracle.rhs of the final state.
shoot_quad is the same map with the initial state and the final scaling carried to ~40 digits (mpmath) as (hi, lo) fp64 pairs, for the
__float128 build of the oracle (the double-double instance of the path); pinned against shoot in tests/test_oracle_pins.py.
"""
from __future__ import annotations

import numpy as np

LD = np.longdouble
LD_PI = LD("3.14159265358979323846264338327950288")   # pi to the precision of long double (np.pi is its fp64 rounding)


def _split(x):
    hi = np.asarray(x, dtype=np.float64)
    return hi, np.asarray(x - hi.astype(LD), dtype=np.float64)


def initial_state(c, N: int):
    """(3.15): -> eta0, phi0 (long double, N) and the columns d q0 / d c_k, k = 1..n, as (deta, dphi) of shape (n, N)"""
    c = np.asarray(c, dtype=np.float64)
    n = c.shape[0] - 1
    j = np.arange(N, dtype=np.int64)
    eta, phi = np.zeros(N, dtype=LD), np.zeros(N, dtype=LD)
    deta, dphi = np.zeros((n, N), dtype=LD), np.zeros((n, N), dtype=LD)
    for k in range(1, n + 1):
        col = 2 * np.cos(2 * LD_PI * ((k * j) % N).astype(LD) / N)   # 2 cos(k alpha_j), phase reduced exactly
        if k % 2 == 0:
            eta += LD(c[k]) * col
            deta[k - 1] = col
        else:
            phi += LD(c[k]) * col
            dphi[k - 1] = col
    return eta, phi, deta, dphi


def shoot(orc, c, N: int, h: float, g: float, nsteps: int, filter: bool = True, sigma: float = 0.0, method: str = "rk8"):
    """-> dict r (N), J (N x (n+1)), eta, phi (the state at T/4), all long double"""
    c = np.asarray(c, dtype=np.float64)
    n = c.shape[0] - 1
    T = float(c[0])
    eta0, phi0, deta0, dphi0 = initial_state(c, N)
    dt = T / (4 * nsteps)
    nthr = orc.num_threads()
    if N * n <= 4096:
        orc.set_num_threads(1)   # hundreds of tiny right-hand sides: the OpenMP barriers would dominate
    try:
        out = orc.rk_advance(_split(eta0), _split(phi0), h, g, dt, nsteps, deta=_split(deta0), dphi=_split(dphi0), filter=filter, sigma=sigma, method=method)
    finally:
        orc.set_num_threads(nthr)
    ld = lambda p: p[0].astype(LD) + p[1].astype(LD)
    eta, phi, dphi = ld(out["eta"]), ld(out["phi"]), ld(out["dphi"])
    phi_t = ld(orc.rhs(out["eta"], out["phi"], h, g, filter=filter, sigma=sigma)["phi_t"])
    w = 1 / np.sqrt(LD(N))
    J = np.empty((N, n + 1), dtype=LD)
    J[:, 0] = phi_t * w / 4
    J[:, 1:] = dphi.T * w
    return {"r": phi * w, "J": J, "eta": eta, "phi": phi}


def shoot_segments(orc, c, segments, h: float, g: float, filter: bool = True, sigma: float = 0.0, method: str = "rk8"):
    """The shooting map with the mesh-refinement strategy of section 2.2: segments = [(M_l, theta_l, rho_l, where_l,
    N_l), ...], theta_1 + ... + theta_nu = 1, rho_1 = 1 (the initial state (3.15) lives on the uniform mesh).  Segment l advances N_l
    steps of size theta_l (T/4) / N_l on M_l points x = xi_l(alpha); the state and the columns are respaced from l to l + 1 (Oracle.respace).
      (3.17) PAPER.md:208-212   r_i = phi(xi_nu(alpha_i), T/4) sqrt(E_nu(alpha_i) / M_nu)   (trapezoidal weight of dx = E_nu dalpha)
      (3.31)                    J_ik likewise from the columns on the last mesh; k = 0: phi_t(., T/4) / 4 times the weight (R13)
    -> dict r (M_nu), J (M_nu x (n+1)), eta, phi (the state at T/4 on the last mesh), long double.  Leaves the oracle on the uniform mesh."""
    c = np.asarray(c, dtype=np.float64)
    n = c.shape[0] - 1
    T = float(c[0])
    ld = lambda p: p[0].astype(LD) + p[1].astype(LD)
    M1, th1, rho1, where1, _ = segments[0]
    assert rho1 == 1.0 and abs(sum(sg[1] for sg in segments) - 1.0) < 1e-12
    eta0, phi0, deta0, dphi0 = initial_state(c, M1)
    st = {"eta": _split(eta0), "phi": _split(phi0), "deta": _split(deta0), "dphi": _split(dphi0)}
    prev = None
    try:
        for (M, theta, rho, where, nst) in segments:
            if prev is not None:
                st = {k: orc.respace(st[k], prev, (M, rho, where)) for k in ("eta", "phi", "deta", "dphi")}
            orc.set_mesh(rho, where)
            st = orc.rk_advance(st["eta"], st["phi"], h, g, theta * T / (4 * nst), nst, deta=st["deta"], dphi=st["dphi"], filter=filter,
                                sigma=sigma, method=method)
            prev = (M, rho, where)
        phi_t = ld(orc.rhs(st["eta"], st["phi"], h, g, filter=filter, sigma=sigma)["phi_t"])
        E = ld(orc.mesh_tables(prev[0])[1])
    finally:
        orc.set_mesh()
    M = prev[0]
    w = np.sqrt(E / LD(M))
    eta, phi, dphi = ld(st["eta"]), ld(st["phi"]), ld(st["dphi"])
    J = np.empty((M, n + 1), dtype=LD)
    J[:, 0] = phi_t * w / 4
    J[:, 1:] = dphi.T * w[:, None]
    return {"r": phi * w, "J": J, "eta": eta, "phi": phi}


def _mp_split(x):
    hi = float(x)
    return hi, float(x - hi)


def initial_state_quad(c, N: int):
    """(3.15) to ~40 digits: -> (eta, phi, deta, dphi), each a pair (hi, lo) of float64 arrays"""
    import mpmath as mp
    c = np.asarray(c, dtype=np.float64)
    n = c.shape[0] - 1
    with mp.workprec(160):
        col = [[2 * mp.cos(2 * mp.pi * ((k * j) % N) / N) for j in range(N)] for k in range(n + 1)]
        eta = [sum((mp.mpf(float(c[k])) * col[k][j] for k in range(2, n + 1, 2)), mp.mpf(0)) for j in range(N)]
        phi = [sum((mp.mpf(float(c[k])) * col[k][j] for k in range(1, n + 1, 2)), mp.mpf(0)) for j in range(N)]
        pair = lambda v: tuple(np.array(t, dtype=np.float64) for t in zip(*[_mp_split(x) for x in v]))
        zero = [mp.mpf(0)] * N
        deta = [pair(col[k] if k % 2 == 0 else zero) for k in range(1, n + 1)]
        dphi = [pair(col[k] if k % 2 == 1 else zero) for k in range(1, n + 1)]
        stack = lambda ps: (np.stack([p[0] for p in ps]), np.stack([p[1] for p in ps]))
        return pair(eta), pair(phi), stack(deta), stack(dphi)


def shoot_quad(orc, c, N: int, h: float, g: float, nsteps: int, filter: bool = True, sigma: float = 0.0, method: str = "rk8"):
    """shoot() for the __float128 oracle: -> dict r (hi, lo), J (hi, lo) with J[.] of shape (N, n + 1)"""
    import mpmath as mp
    c = np.asarray(c, dtype=np.float64)
    n = c.shape[0] - 1
    T = float(c[0])
    eta0, phi0, deta0, dphi0 = initial_state_quad(c, N)
    out = orc.rk_advance(eta0, phi0, h, g, T / (4 * nsteps), nsteps, deta=deta0, dphi=dphi0, filter=filter, sigma=sigma, method=method)
    phi_t = orc.rhs(out["eta"], out["phi"], h, g, filter=filter, sigma=sigma)["phi_t"]
    with mp.workprec(160):
        w = 1 / mp.sqrt(mp.mpf(N))
        val = lambda p, i: mp.mpf(float(p[0][i])) + mp.mpf(float(p[1][i]))
        r = [val(out["phi"], i) * w for i in range(N)]
        Jc = [[val(phi_t, i) * w / 4 for i in range(N)]]
        for k in range(n):
            Jc.append([(mp.mpf(float(out["dphi"][0][k][i])) + mp.mpf(float(out["dphi"][1][k][i]))) * w for i in range(N)])
        sp = lambda v: tuple(np.array(t, dtype=np.float64) for t in zip(*[_mp_split(x) for x in v]))
        rr = sp(r)
        Js = [sp(col) for col in Jc]
        return {"r": rr, "J": (np.stack([j[0] for j in Js], axis=1), np.stack([j[1] for j in Js], axis=1))}


def shoot_segments_quad(orc, c, segments, h: float, g: float, filter: bool = True, sigma: float = 0.0, method: str = "rk8"):
    """shoot_segments for the __float128 oracle (initial state and the weights sqrt(E/M) to ~40 digits): -> dict r (hi, lo),
    J (hi, lo) with J[.] of shape (M_nu, n + 1)"""
    import mpmath as mp
    c = np.asarray(c, dtype=np.float64)
    n = c.shape[0] - 1
    T = float(c[0])
    M1, _, rho1, _, _ = segments[0]
    assert rho1 == 1.0 and abs(sum(sg[1] for sg in segments) - 1.0) < 1e-12
    eta0, phi0, deta0, dphi0 = initial_state_quad(c, M1)
    st = {"eta": eta0, "phi": phi0, "deta": deta0, "dphi": dphi0}
    prev = None
    try:
        for (M, theta, rho, where, nst) in segments:
            if prev is not None:
                st = {k: orc.respace(st[k], prev, (M, rho, where)) for k in ("eta", "phi", "deta", "dphi")}
            orc.set_mesh(rho, where)
            st = orc.rk_advance(st["eta"], st["phi"], h, g, theta * T / (4 * nst), nst, deta=st["deta"], dphi=st["dphi"], filter=filter,
                                sigma=sigma, method=method)
            prev = (M, rho, where)
        phi_t = orc.rhs(st["eta"], st["phi"], h, g, filter=filter, sigma=sigma)["phi_t"]
        E = orc.mesh_tables(prev[0])[1]
    finally:
        orc.set_mesh()
    M = prev[0]
    with mp.workprec(160):
        val = lambda p, i: mp.mpf(float(p[0][i])) + mp.mpf(float(p[1][i]))
        w = [mp.sqrt(val(E, i) / M) for i in range(M)]
        r = [val(st["phi"], i) * w[i] for i in range(M)]
        Jc = [[val(phi_t, i) * w[i] / 4 for i in range(M)]]
        for k in range(n):
            Jc.append([(mp.mpf(float(st["dphi"][0][k][i])) + mp.mpf(float(st["dphi"][1][k][i]))) * w[i] for i in range(M)])
        sp = lambda v: tuple(np.array(t, dtype=np.float64) for t in zip(*[_mp_split(x) for x in v]))
        Js = [sp(col) for col in Jc]
        return {"r": sp(r), "J": (np.stack([j[0] for j in Js], axis=1), np.stack([j[1] for j in Js], axis=1))}
