"""Pins of the oracle's pointwise pieces (limiter O3, HLLD O6, 2D EMF solver O7) against
what the paper and the mathematics fix -- never against the oracle itself.

HLLD (Miyoshi & Kusano 2005) is pinned through properties any correct
six-region solver must have:
  * consistency with Eq. 6;
  * Rankine-Hugoniot conditions at EVERY wave of the fan, checked from the outside
    through Galilean boosts: G_f(V) = F_f(xi=V) - V U_f(xi=V) must be a continuous
    function of the frame velocity V (a jump at a wave = a wrong star/double-star
    formula).  This is the "fan integral" identity in differential form;
  * exact resolution of isolated contact, tangential and rotational discontinuities;
  * the B -> 0 limit equals the textbook HLLC flux; mirror symmetry.
"""
import numpy as np
import pytest

import oracle

G = 5.0 / 3.0


# ------------------------------------------------------------------- helpers ------
def phys_flux(q, bn, gamma):
    """Eq. 6 typed from the paper: q = (rho,u,v,w,p,By,Bz)."""
    rho, u, v, w, p, by, bz = q
    B2 = bn * bn + by * by + bz * bz
    P = p + 0.5 * B2
    E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * B2
    ub = u * bn + v * by + w * bz
    return np.array([rho * u, rho * u * u + P - bn * bn, rho * v * u - by * bn, rho * w * u - bz * bn,
                     u * (E + P) - bn * ub, by * u - bn * v, bz * u - bn * w])


def cons(q, bn, gamma):
    rho, u, v, w, p, by, bz = q
    E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * (bn * bn + by * by + bz * bz)
    return np.array([rho, rho * u, rho * v, rho * w, E, by, bz])


def rand_state(rng, mach=1.0, bscale=1.0):
    return np.array([np.exp(rng.normal(0, 0.5)), mach * rng.normal(), mach * rng.normal(), mach * rng.normal(),
                     np.exp(rng.normal(0, 0.5)), bscale * rng.normal(), bscale * rng.normal()])


def boosted_G(L, R, bn, V, gamma):
    """G_f(V) for f = rho, mu, mv, mw, E, By, Bz from the flux in the frame moving at V."""
    Lb, Rb = L.copy(), R.copy()
    Lb[1] -= V
    Rb[1] -= V
    Fp = oracle.hlld(gamma, Lb, Rb, bn)
    Gv = Fp.copy()
    Gv[1] = Fp[1] + V * Fp[0]
    Gv[4] = Fp[4] + V * Fp[1] + 0.5 * V * V * Fp[0]
    return Gv


# ------------------------------------------------------------------- limiter ------
@pytest.mark.parametrize("kind", [1, 2])
def test_limiter_properties(kind):
    rng = np.random.default_rng(1)
    for _ in range(2000):
        a, b = rng.normal(size=2)
        s = oracle.limiter(kind, a, b)
        if a * b <= 0:
            assert s == 0.0                      # local extremum -> flat
        else:
            assert np.sign(s) == np.sign(a)
            assert abs(s) <= 2 * min(abs(a), abs(b)) * (1 + 1e-15)
            if kind == 1:
                assert abs(s) == min(abs(a), abs(b))
        assert oracle.limiter(kind, b, a) == s   # symmetric
        assert oracle.limiter(kind, -a, -b) == -s
    for a in (0.3, -2.0, 1e-9):                  # linear data -> exact slope
        assert oracle.limiter(kind, a, a) == a
    # monotonised central picks the central difference when it is the smallest
    assert oracle.limiter(2, 1.0, 1.5) == 1.25
    assert oracle.limiter(2, 1.0, 10.0) == 2.0
    assert oracle.limiter(1, 1.0, 10.0) == 1.0


# ---------------------------------------------------------------------- HLLD ------
def test_hlld_consistency_with_eq6():
    rng = np.random.default_rng(2)
    for _ in range(500):
        q = rand_state(rng)
        bn = rng.normal()
        F = oracle.hlld(G, q, q, bn)
        ref = phys_flux(q, bn, G)
        assert np.allclose(F, ref, rtol=0, atol=2e-13 * (1 + np.abs(ref).max()))


def test_hlld_supersonic_upwinding():
    rng = np.random.default_rng(3)
    for _ in range(200):
        L, R = rand_state(rng), rand_state(rng)
        bn = rng.normal()
        for shift, side in ((+30.0, L), (-30.0, R)):
            Ls, Rs, s = L.copy(), R.copy(), side.copy()
            Ls[1] += shift; Rs[1] += shift; s[1] += shift
            assert np.array_equal(oracle.hlld(G, Ls, Rs, bn), phys_flux(s, bn, G)) or \
                np.allclose(oracle.hlld(G, Ls, Rs, bn), phys_flux(s, bn, G), rtol=1e-14)


@pytest.mark.parametrize("bnzero", [False, True])
def test_hlld_rankine_hugoniot_at_every_wave(bnzero):
    """G(V) continuous in the boost V: refine the steepest intervals by bisection; a jump
    survives refinement, a kink of a continuous piecewise-linear function does not."""
    rng = np.random.default_rng(4)
    for trial in range(40):
        L, R = rand_state(rng), rand_state(rng)
        bn = 0.0 if bnzero else rng.normal()
        scale = max(np.abs(cons(L, bn, G)).max(), np.abs(cons(R, bn, G)).max(), 1.0)
        Vs = np.linspace(min(L[1], R[1]) - 6.0, max(L[1], R[1]) + 6.0, 600)
        Gs = np.array([boosted_G(L, R, bn, V, G) for V in Vs])
        # ends: outside the fan G = F_K - V U_K exactly
        for V, q in ((Vs[0], L), (Vs[-1], R)):
            ref = phys_flux(q, bn, G) - V * cons(q, bn, G)
            assert np.allclose(boosted_G(L, R, bn, V, G), ref, rtol=1e-12, atol=1e-12 * scale)
        dG = np.abs(np.diff(Gs, axis=0)).max(axis=1)
        for idx in np.argsort(dG)[-8:]:
            a, b = Vs[idx], Vs[idx + 1]
            Ga, Gb = Gs[idx], Gs[idx + 1]
            for _ in range(36):
                m = 0.5 * (a + b)
                Gm = boosted_G(L, R, bn, m, G)
                if np.abs(Gm - Ga).max() > np.abs(Gb - Gm).max():
                    b, Gb = m, Gm
                else:
                    a, Ga = m, Gm
            assert np.abs(Gb - Ga).max() <= 1e-9 * scale * 50, (trial, a, np.abs(Gb - Ga))


def test_hlld_fan_slopes_are_the_outer_states():
    """dG/dV = -U(xi): just inside... outside the fan the slope is -U_L / -U_R, and the
    mass slope stays negative (positive density) everywhere in between."""
    rng = np.random.default_rng(5)
    for _ in range(40):
        L, R = rand_state(rng), rand_state(rng)
        bn = rng.normal()
        Vs = np.linspace(min(L[1], R[1]) - 8.0, max(L[1], R[1]) + 8.0, 801)
        Grho = np.array([boosted_G(L, R, bn, V, G)[0] for V in Vs])
        slope = np.diff(Grho) / np.diff(Vs)
        assert np.isclose(slope[0], -L[0], rtol=1e-9) and np.isclose(slope[-1], -R[0], rtol=1e-9)
        assert (slope < 0).all()


def test_hlld_isolated_contact_exact():
    rng = np.random.default_rng(6)
    for _ in range(200):
        L = rand_state(rng)
        R = L.copy()
        R[0] = L[0] * np.exp(rng.normal())        # density jump only; u, pT, v, w, B continuous
        bn = rng.normal()
        u = L[1]
        F = oracle.hlld(G, L, R, bn)
        ref = phys_flux(L if u > 0 else R, bn, G)
        assert np.allclose(F, ref, rtol=0, atol=1e-12 * (1 + np.abs(ref).max())), (F - ref)


def test_hlld_isolated_tangential_discontinuity_exact():
    """Bn = 0: density, tangential velocity and tangential field jump at constant total
    pressure and normal velocity."""
    rng = np.random.default_rng(7)
    for _ in range(200):
        L, R = rand_state(rng), rand_state(rng)
        R[1] = L[1]
        pT = L[4] + 0.5 * (L[5] ** 2 + L[6] ** 2)
        R[4] = pT * rng.uniform(0.2, 0.9)
        b2 = 2 * (pT - R[4])
        th = rng.uniform(0, 2 * np.pi)
        R[5], R[6] = np.sqrt(b2) * np.cos(th), np.sqrt(b2) * np.sin(th)
        F = oracle.hlld(G, L, R, 0.0)
        ref = phys_flux(L if L[1] > 0 else R, 0.0, G)
        assert np.allclose(F, ref, rtol=0, atol=1e-12 * (1 + np.abs(ref).max()))


def test_hlld_isolated_rotational_discontinuity_exact():
    """A single Alfven wave: rho, p, u, |Bt| continuous, Bt rotates, [vt] = -+[Bt]/sqrt(rho)."""
    rng = np.random.default_rng(8)
    for _ in range(300):
        L = rand_state(rng)
        bn = rng.normal()
        bt = np.hypot(L[5], L[6])
        th = rng.uniform(0, 2 * np.pi)
        R = L.copy()
        R[5], R[6] = bt * np.cos(th), bt * np.sin(th)
        sgn = rng.choice([-1.0, 1.0])              # +1: wave moving right relative to the gas
        fac = -sgn * np.sign(bn) / np.sqrt(L[0])
        R[2] = L[2] + fac * (R[5] - L[5])
        R[3] = L[3] + fac * (R[6] - L[6])
        speed = L[1] + sgn * abs(bn) / np.sqrt(L[0])
        F = oracle.hlld(G, L, R, bn)
        ref = phys_flux(L if speed > 0 else R, bn, G)
        assert np.allclose(F, ref, rtol=0, atol=2e-12 * (1 + np.abs(ref).max())), (F - ref, speed)


def hllc_euler(L, R, gamma):
    """Textbook HLLC for the Euler equations (Toro 2009 ch. 10) with the same
    outer-speed estimate as O6: S = min/max u -+ max c."""
    def prim(q):
        rho, u, v, w, p = q[:5]
        E = p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w)
        U = np.array([rho, rho * u, rho * v, rho * w, E])
        F = np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, u * (E + p)])
        return U, F, np.sqrt(gamma * p / rho)
    UL, FL, cL = prim(L)
    UR, FR, cR = prim(R)
    c = max(cL, cR)
    SL, SR = min(L[1], R[1]) - c, max(L[1], R[1]) + c
    SM = (R[4] - L[4] + L[0] * L[1] * (SL - L[1]) - R[0] * R[1] * (SR - R[1])) / (L[0] * (SL - L[1]) - R[0] * (SR - R[1]))
    def starU(q, U, S):
        rho, u, v, w, p = q[:5]
        f = rho * (S - u) / (S - SM)
        return f * np.array([1, SM, v, w, U[4] / rho + (SM - u) * (SM + p / (rho * (S - u)))])
    if SL > 0:
        return FL
    if SM >= 0:
        return FL + SL * (starU(L, UL, SL) - UL)
    if SR >= 0:
        return FR + SR * (starU(R, UR, SR) - UR)
    return FR


def test_hlld_reduces_to_hllc_without_field():
    rng = np.random.default_rng(9)
    for _ in range(300):
        L, R = rand_state(rng, bscale=0.0), rand_state(rng, bscale=0.0)
        F = oracle.hlld(G, L, R, 0.0)
        ref = hllc_euler(L, R, G)
        assert np.allclose(F[:5], ref, rtol=0, atol=1e-12 * (1 + np.abs(ref).max()))
        assert F[5] == 0 and F[6] == 0


def test_hlld_small_normal_field_is_continuous_limit():
    rng = np.random.default_rng(10)
    for _ in range(100):
        L, R = rand_state(rng), rand_state(rng)
        F0 = oracle.hlld(G, L, R, 0.0)
        F1 = oracle.hlld(G, L, R, 1e-9)
        assert np.allclose(F0, F1, rtol=0, atol=1e-6 * (1 + np.abs(F0).max()))


def test_hlld_mirror_symmetry():
    rng = np.random.default_rng(11)
    flip = np.array([-1, 1, -1, -1, -1, -1, -1.0])
    for _ in range(300):
        L, R = rand_state(rng), rand_state(rng)
        bn = rng.normal()
        Lm, Rm = R.copy(), L.copy()
        Lm[1] *= -1; Rm[1] *= -1
        F = oracle.hlld(G, L, R, bn)
        Fm = oracle.hlld(G, Lm, Rm, -bn)
        assert np.allclose(Fm, flip * F, rtol=0, atol=1e-12 * (1 + np.abs(F).max()))


def test_hlld_transverse_rotation_covariance():
    """Rotating (v,w) and (By,Bz) together by an angle about the normal rotates the
    transverse fluxes and leaves the others unchanged (catches a v<->w / By<->Bz mix-up)."""
    rng = np.random.default_rng(12)
    for _ in range(200):
        L, R = rand_state(rng), rand_state(rng)
        bn = rng.normal()
        th = rng.uniform(0, 2 * np.pi)
        c, s = np.cos(th), np.sin(th)
        def rot(q):
            o = q.copy()
            o[2], o[3] = c * q[2] - s * q[3], s * q[2] + c * q[3]
            o[5], o[6] = c * q[5] - s * q[6], s * q[5] + c * q[6]
            return o
        F, Fr = oracle.hlld(G, L, R, bn), oracle.hlld(G, rot(L), rot(R), bn)
        ref = F.copy()
        ref[2], ref[3] = c * F[2] - s * F[3], s * F[2] + c * F[3]
        ref[5], ref[6] = c * F[5] - s * F[6], s * F[5] + c * F[6]
        assert np.allclose(Fr, ref, rtol=0, atol=1e-12 * (1 + np.abs(F).max()))


def test_fast_speed_closed_forms():
    # no field: sound speed; field along the normal only: max(sound, Alfven); perpendicular: magnetosonic
    assert np.isclose(oracle.fast_speed(1.4, 2.0, 3.0, 0, 0, 0), np.sqrt(1.4 * 3 / 2), rtol=1e-15)
    assert np.isclose(oracle.fast_speed(1.4, 2.0, 3.0, 5.0, 0, 0), max(np.sqrt(1.4 * 3 / 2), 5 / np.sqrt(2)), rtol=1e-15)
    assert np.isclose(oracle.fast_speed(1.4, 2.0, 3.0, 0, 1.0, 2.0), np.sqrt((1.4 * 3 + 5) / 2), rtol=1e-15)


# ------------------------------------------------------------ 2D EMF solver -------
def rand_corners(rng):
    c = np.zeros((4, 6))
    for q in range(4):
        c[q] = [np.exp(rng.normal(0, 0.4)), rng.normal(), rng.normal(), rng.normal(), np.exp(rng.normal(0, 0.4)), rng.normal()]
    return c


@pytest.mark.parametrize("solver", [0, 1])
def test_emf2d_uniform_state(solver):
    rng = np.random.default_rng(20)
    for _ in range(300):
        c = np.tile(rand_corners(rng)[0], (4, 1))
        A, B = rng.normal(size=2)
        e = oracle.emf2d(G, solver, c, A, A, B, B)
        ref = c[0, 1] * B - c[0, 2] * A           # Eq. 7: u By - v Bx
        assert abs(e - ref) <= 1e-13 * (1 + abs(ref))


def test_emf2d_planar_reduction_to_hlld_x():
    """Data independent of b (south == north): the edge EMF is O6's flux of B_b along a,
    for every wave pattern (sweep the frame velocity) and for zero normal field."""
    rng = np.random.default_rng(21)
    worst = 0.0
    for trial in range(400):
        W, E = rand_corners(rng)[0], rand_corners(rng)[1]
        A = 0.0 if trial % 5 == 0 else rng.normal()
        BW, BE = rng.normal(size=2)
        shift = rng.uniform(-3, 3)
        W[1] += shift; E[1] += shift
        c = np.array([W, E, W, E])
        e = oracle.emf2d(G, 0, c, A, A, BW, BE)
        # 1D problem along a: (rho, un=ua, ut1=ub, ut2=ue, p, Bt1=B_b, Bt2=B_e), bn = A
        L = [W[0], W[1], W[2], W[3], W[4], BW, W[5]]
        R = [E[0], E[1], E[2], E[3], E[4], BE, E[5]]
        F = oracle.hlld(G, L, R, A)
        worst = max(worst, abs(e - F[5]) / (1 + abs(F[5])))
    assert worst <= 5e-13, worst


def test_emf2d_planar_reduction_to_hlld_y():
    """Data independent of a (west == east): EMF = minus O6's flux of B_a along b."""
    rng = np.random.default_rng(22)
    worst = 0.0
    for trial in range(400):
        S, N = rand_corners(rng)[0], rand_corners(rng)[1]
        B = 0.0 if trial % 5 == 0 else rng.normal()
        AS, AN = rng.normal(size=2)
        shift = rng.uniform(-3, 3)
        S[2] += shift; N[2] += shift
        c = np.array([S, S, N, N])
        e = oracle.emf2d(G, 0, c, AS, AN, B, B)
        # 1D problem along b: un = ub, ut1 = ue, ut2 = ua, Bt1 = B_e, Bt2 = B_a, bn = B
        L = [S[0], S[2], S[3], S[1], S[4], S[5], AS]
        R = [N[0], N[2], N[3], N[1], N[4], N[5], AN]
        F = oracle.hlld(G, L, R, B)
        worst = max(worst, abs(e + F[6]) / (1 + abs(F[6])))
    assert worst <= 5e-13, worst


@pytest.mark.parametrize("solver", [0, 1])
def test_emf2d_antisymmetry_under_axis_swap(solver):
    """Swap a<->b: ua<->ub, A<->B, SE<->NW, and the out-of-plane axis flips  =>  E -> -E."""
    rng = np.random.default_rng(23)
    for _ in range(400):
        c = rand_corners(rng)
        AS, AN, BW, BE = rng.normal(size=4)
        e = oracle.emf2d(G, solver, c, AS, AN, BW, BE)
        cs = c[[0, 2, 1, 3]].copy()
        cs[:, [1, 2]] = cs[:, [2, 1]]
        es = oracle.emf2d(G, solver, cs, BW, BE, AS, AN)
        assert abs(e + es) <= 1e-13 * (1 + abs(e))


@pytest.mark.parametrize("solver", [0, 1])
def test_emf2d_doubly_supersonic_is_upwind_corner(solver):
    rng = np.random.default_rng(24)
    for _ in range(200):
        c = rand_corners(rng)
        AS, AN, BW, BE = rng.normal(size=4)
        for sa, sb, corner in ((+1, +1, 0), (-1, +1, 1), (+1, -1, 2), (-1, -1, 3)):
            cc = c.copy()
            cc[:, 1] += 40.0 * sa
            cc[:, 2] += 40.0 * sb
            A = (AS, AS, AN, AN)[corner]
            B = (BW, BE, BW, BE)[corner]
            ref = cc[corner, 1] * B - cc[corner, 2] * A
            assert oracle.emf2d(G, solver, cc, AS, AN, BW, BE) == ref


def test_emf2d_supersonic_in_one_direction_ignores_downwind_column():
    """Flow supersonic towards +a: the east corners' own EMFs and fields carry zero weight.
    They still enter through the shared outer-speed estimate, so the check perturbs them
    in a way that leaves min/max u_a and max c_f unchanged (the out-of-plane velocity)."""
    rng = np.random.default_rng(25)
    for _ in range(100):
        c = rand_corners(rng)
        AS, AN, BW, BE = rng.normal(size=4)
        c[:, 1] += 40.0
        e0 = oracle.emf2d(G, 0, c, AS, AN, BW, BE)
        c2 = c.copy()
        c2[1, 3] += 1.0; c2[3, 3] -= 2.0          # ue of SE and NE
        assert oracle.emf2d(G, 0, c2, AS, AN, BW, BE) == e0


def _one_way_case(rng, sign):
    """Corner set with flow supersonic towards sign*b and (mostly) subsonic along a, built so that
    the DOWNWIND row can change nothing but the quantities under test:
      * every corner of a column has the column's u_a, so min/max u_a come from the upwind row;
      * the downwind row is denser (rho x kappa >= 1), colder, carries no A field and a weaker
        out-of-plane field, so its fast speeds lie below the upwind row's (c_f grows with p, with
        every field component and with 1/rho), i.e. the outer speeds are the upwind row's;
      * total pressure is equal along each row, so both rows' contact speeds are the same |m|-weighted
        mean of u_W and u_E; with A = 0 the downwind row's Alfven bounds collapse onto that contact
        speed, strictly inside the upwind row's bounds: the inner speeds are the upwind row's too.
    Returns (corners, AS, AN, BW, BE, L, R, bn): L, R, bn = the 1D problem of the upwind row."""
    c = rand_corners(rng)
    up, dn = ((0, 1), (2, 3)) if sign > 0 else ((2, 3), (0, 1))
    A_up = rng.choice([-1.0, 1.0]) * rng.uniform(0.4, 1.5)
    BW, BE = rng.normal(size=2)
    c[:, 2] += 40.0 * sign
    # equal total pressure along the upwind row: adjust the pressure of its east corner
    w, e = up
    pT = c[w, 4] + 0.5 * (A_up ** 2 + BW ** 2 + c[w, 5] ** 2)
    c[e, 4] = pT - 0.5 * (A_up ** 2 + BE ** 2 + c[e, 5] ** 2)
    if c[e, 4] <= 0.05:
        return None
    kappa = rng.uniform(1.0, 3.0)
    for k in (0, 1):
        c[dn[k], 0] = kappa * c[up[k], 0]
        c[dn[k], 1] = c[up[k], 1]
        c[dn[k], 3] = rng.normal()
        c[dn[k], 5] = rng.uniform(-1, 1) * abs(c[up[k], 5])
    pTd = rng.uniform(0.3, 0.9) * min(c[up[0], 4], c[up[1], 4]) + 0.5 * max(BW ** 2 + c[dn[0], 5] ** 2, BE ** 2 + c[dn[1], 5] ** 2)
    c[dn[0], 4] = pTd - 0.5 * (BW ** 2 + c[dn[0], 5] ** 2)
    c[dn[1], 4] = pTd - 0.5 * (BE ** 2 + c[dn[1], 5] ** 2)
    if min(c[dn[0], 4], c[dn[1], 4]) <= 0 or max(c[dn[0], 4], c[dn[1], 4]) > min(c[up[0], 4], c[up[1], 4]):
        return None
    AS, AN = (A_up, 0.0) if sign > 0 else (0.0, A_up)
    # precondition, checked with the (separately pinned) fast speed: the maxima are upwind
    A = [AS, AS, AN, AN]; B = [BW, BE, BW, BE]
    cfa = [oracle.fast_speed(G, c[q, 0], c[q, 4], A[q], B[q], c[q, 5]) for q in range(4)]
    cfb = [oracle.fast_speed(G, c[q, 0], c[q, 4], B[q], A[q], c[q, 5]) for q in range(4)]
    assert max(cfa[dn[0]], cfa[dn[1]]) < max(cfa[up[0]], cfa[up[1]])
    assert max(cfb[dn[0]], cfb[dn[1]]) < max(cfb[up[0]], cfb[up[1]])
    L = [c[w, 0], c[w, 1], c[w, 2], c[w, 3], c[w, 4], BW, c[w, 5]]
    R = [c[e, 0], c[e, 1], c[e, 2], c[e, 3], c[e, 4], BE, c[e, 5]]
    return c, AS, AN, BW, BE, L, R, A_up


@pytest.mark.parametrize("sign", [+1, -1])
def test_emf2d_supersonic_along_b_takes_the_upwind_rows_star_fields(sign):
    """O7 step 5.  Flow supersonic towards +b: S_S = 0, so the weights of the composition are 1 on
    the south row and 0 on the north row -- for the corner EMFs AND for the edge-side star fields
    B*_W, B*_E that feed the x-dissipation term.  The 2D problem then IS the 1D problem of the south
    row along a: the edge EMF must equal O6's induction flux of that row (a separately pinned
    function) while the flow is subsonic along a, so that the dissipation weight is not zero.  A
    solver that weighted the star fields the other way round would pick the north row's values."""
    rng = np.random.default_rng(31 + sign)
    done = subsonic = 0
    while done < 300:
        case = _one_way_case(rng, sign)
        if case is None:
            continue
        c, AS, AN, BW, BE, L, R, bn = case
        F = oracle.hlld(G, L, R, bn)
        e = oracle.emf2d(G, 0, c, AS, AN, BW, BE)
        assert abs(e - F[5]) <= 5e-13 * (1 + abs(F[5])), (e, F[5])
        # ... bit for bit whatever the downwind row holds (inside the precondition)
        dn = (2, 3) if sign > 0 else (0, 1)
        c2 = c.copy()
        c2[dn[0], 3] += 0.7; c2[dn[1], 3] -= 0.3                       # out-of-plane velocity
        c2[dn[0], 0] *= 1.25; c2[dn[1], 0] *= 1.25                     # density (same factor: same contact speed)
        assert oracle.emf2d(G, 0, c2, AS, AN, BW, BE) == e
        done += 1
        cf = max(oracle.fast_speed(G, L[0], L[4], bn, L[5], L[6]), oracle.fast_speed(G, R[0], R[4], bn, R[5], R[6]))
        subsonic += (min(L[1], R[1]) - cf < 0 < max(L[1], R[1]) + cf)
    assert subsonic > 200          # the x-dissipation term was exercised


@pytest.mark.parametrize("sign", [+1, -1])
def test_emf2d_supersonic_along_a_takes_the_upwind_columns_star_fields(sign):
    """The same statement with the roles of a and b exchanged (weights a_E, a_W of A*_S, A*_N):
    the case above mapped by a <-> b (u_a <-> u_b, A <-> B, SE <-> NW), under which the EMF changes
    sign; expected value = minus O6's flux of the upwind COLUMN's 1D problem along b."""
    rng = np.random.default_rng(41 + sign)
    done = 0
    while done < 300:
        case = _one_way_case(rng, sign)
        if case is None:
            continue
        c, AS, AN, BW, BE, L, R, bn = case
        F = oracle.hlld(G, L, R, bn)
        cs = c[[0, 2, 1, 3]].copy()
        cs[:, [1, 2]] = cs[:, [2, 1]]
        e = oracle.emf2d(G, 0, cs, BW, BE, AS, AN)
        assert abs(e + F[5]) <= 5e-13 * (1 + abs(F[5])), (e, F[5])
        done += 1


def _hlld2d_typed(c, AS, AN, BW, BE):
    """DESIGN.md reading O7 typed from its text; the Miyoshi-Kusano star
    relations of a 1D sub-problem with prescribed outer speeds are typed from O6."""
    SW_, SE_, NW_, NE_ = 0, 1, 2, 3
    A = [AS, AS, AN, AN]; B = [BW, BE, BW, BE]
    rho, ua, ub, p, be = c[:, 0], c[:, 1], c[:, 2], c[:, 4], c[:, 5]
    emf = [ua[q] * B[q] - ub[q] * A[q] for q in range(4)]
    pT = [p[q] + 0.5 * (A[q] ** 2 + B[q] ** 2 + be[q] ** 2) for q in range(4)]
    ca = max(oracle.fast_speed(G, rho[q], p[q], A[q], B[q], be[q]) for q in range(4))
    cb = max(oracle.fast_speed(G, rho[q], p[q], B[q], A[q], be[q]) for q in range(4))
    tW, tE, tS, tN = ua.min() - ca, ua.max() + ca, ub.min() - cb, ub.max() + cb       # step 1

    def sub(l, r, un, bt_l, bt_r, bn, SL, SR):                                          # step 2
        mL, mR = rho[l] * (SL - un[l]), rho[r] * (SR - un[r])
        SM = (mR * un[r] - mL * un[l] - pT[r] + pT[l]) / (mR - mL)
        rsL, rsR = mL / (SL - SM), mR / (SR - SM)
        star = []
        for m, S, u, bt in ((mL, SL, un[l], bt_l), (mR, SR, un[r], bt_r)):
            D = m * (S - SM) - bn ** 2
            star.append(bt if abs(D) <= 16 * np.finfo(float).eps * m * (S - u) else bt * (m * (S - u) - bn ** 2) / D)
        return star[0], star[1], SM - abs(bn) / np.sqrt(rsL), SM + abs(bn) / np.sqrt(rsR)

    xS = sub(SW_, SE_, ua, BW, BE, AS, tW, tE)
    xN = sub(NW_, NE_, ua, BW, BE, AN, tW, tE)
    yW = sub(SW_, NW_, ub, AS, AN, BW, tS, tN)
    yE = sub(SE_, NE_, ub, AS, AN, BE, tS, tN)
    S_W = 0.0 if tW >= 0 else min(0.0, xS[2], xN[2])                                   # step 3
    S_E = 0.0 if tE <= 0 else max(0.0, xS[3], xN[3])
    S_S = 0.0 if tS >= 0 else min(0.0, yW[2], yE[2])
    S_N = 0.0 if tN <= 0 else max(0.0, yW[3], yE[3])
    Bs = {SW_: xS[0], SE_: xS[1], NW_: xN[0], NE_: xN[1]}
    As = {SW_: yW[0], NW_: yW[1], SE_: yE[0], NE_: yE[1]}
    Sx = {SW_: min(tW, 0.0), NW_: min(tW, 0.0), SE_: max(tE, 0.0), NE_: max(tE, 0.0)}   # step 4
    Sy = {SW_: min(tS, 0.0), SE_: min(tS, 0.0), NW_: max(tN, 0.0), NE_: max(tN, 0.0)}
    es = {q: emf[q] + Sx[q] * (Bs[q] - B[q]) - Sy[q] * (As[q] - A[q]) for q in range(4)}
    BsW = (S_N * Bs[SW_] - S_S * Bs[NW_]) / (S_N - S_S)                                 # step 5
    BsE = (S_N * Bs[SE_] - S_S * Bs[NE_]) / (S_N - S_S)
    AsS = (S_E * As[SW_] - S_W * As[SE_]) / (S_E - S_W)
    AsN = (S_E * As[NW_] - S_W * As[NE_]) / (S_E - S_W)
    return (S_E * S_N * es[SW_] - S_W * S_N * es[SE_] - S_E * S_S * es[NW_] + S_W * S_S * es[NE_]) \
        / ((S_E - S_W) * (S_N - S_S)) + S_W * S_E / (S_E - S_W) * (BsE - BsW) - S_S * S_N / (S_N - S_S) * (AsN - AsS)   # step 6


def test_emf2d_hlld_matches_typed_reading():
    """HLLD-2D against DESIGN.md's reading O7 typed a second time (numpy, in the printed form of
    the formulas, weights of step 5 included), on non-planar subsonic corner sets where both
    dissipation terms are active and the star fields of the two rows / columns differ."""
    rng = np.random.default_rng(28)
    n = 0
    while n < 400:
        c = rand_corners(rng)
        c[:, 1:3] *= 0.5                                    # subsonic in both directions
        AS, AN, BW, BE = rng.normal(size=4)
        ref = _hlld2d_typed(c, AS, AN, BW, BE)
        if not np.isfinite(ref):
            continue
        e = oracle.emf2d(G, 0, c, AS, AN, BW, BE)
        assert abs(e - ref) <= 1e-11 * (1 + abs(ref)), (e, ref)
        n += 1


def test_emf2d_hll_matches_typed_formula():
    """HLL-2D is the composition (dagger) of DESIGN.md O7 with the corner values and the
    fast speeds clipped at zero -- typed here from that formula in its printed form."""
    rng = np.random.default_rng(26)
    for _ in range(300):
        c = rand_corners(rng)
        AS, AN, BW, BE = rng.normal(size=4)
        A = [AS, AS, AN, AN]; B = [BW, BE, BW, BE]
        e = [c[q, 1] * B[q] - c[q, 2] * A[q] for q in range(4)]
        cfa = max(oracle.fast_speed(G, c[q, 0], c[q, 4], A[q], B[q], c[q, 5]) for q in range(4))
        cfb = max(oracle.fast_speed(G, c[q, 0], c[q, 4], B[q], A[q], c[q, 5]) for q in range(4))
        SW, SE = min(0, c[:, 1].min() - cfa), max(0, c[:, 1].max() + cfa)
        SS, SN = min(0, c[:, 2].min() - cfb), max(0, c[:, 2].max() + cfb)
        ref = (SE * SN * e[0] - SW * SN * e[1] - SE * SS * e[2] + SW * SS * e[3]) / ((SE - SW) * (SN - SS)) \
            + SW * SE / (SE - SW) * (BE - BW) - SS * SN / (SN - SS) * (AN - AS)
        assert abs(oracle.emf2d(G, 1, c, AS, AN, BW, BE) - ref) <= 1e-13 * (1 + abs(ref))


def test_emf2d_hlld_and_hll_agree_for_weak_field_smooth_data():
    """With nearly uniform data the two solvers differ only at second order in the jumps."""
    rng = np.random.default_rng(27)
    for _ in range(100):
        base = rand_corners(rng)[0]
        c = np.tile(base, (4, 1)) + 1e-4 * rng.normal(size=(4, 6))
        A, B = rng.normal(size=2)
        d = 1e-4 * rng.normal(size=4)
        e0 = oracle.emf2d(G, 0, c, A + d[0], A + d[1], B + d[2], B + d[3])
        e1 = oracle.emf2d(G, 1, c, A + d[0], A + d[1], B + d[2], B + d[3])
        assert abs(e0 - e1) <= 5e-3 * (1 + abs(e0)) * 1e-1


# ----------------------------------------------------------------------- HLL ------
# PAPER.md section 2.1.1 (L70-72): three regions; the star state is the integral average of
# the solution between the two outer waves.  Pinned through what that sentence fixes.
def _outer_speeds(L, R, bn):
    c = max(oracle.fast_speed(G, L[0], L[4], bn, L[5], L[6]), oracle.fast_speed(G, R[0], R[4], bn, R[5], R[6]))
    return min(L[1], R[1]) - c, max(L[1], R[1]) + c


def test_hll_consistency_and_supersonic_upwinding():
    rng = np.random.default_rng(21)
    for _ in range(300):
        q, L, R = rand_state(rng), rand_state(rng), rand_state(rng)
        bn = rng.normal()
        ref = phys_flux(q, bn, G)
        assert np.allclose(oracle.hll(G, q, q, bn), ref, rtol=0, atol=2e-13 * (1 + np.abs(ref).max()))
        for shift, side in ((+30.0, L), (-30.0, R)):
            Ls, Rs, s = L.copy(), R.copy(), side.copy()
            Ls[1] += shift; Rs[1] += shift; s[1] += shift
            assert np.allclose(oracle.hll(G, Ls, Rs, bn), phys_flux(s, bn, G), rtol=1e-14, atol=0)


def test_hll_star_state_is_the_integral_average_and_both_jumps_hold():
    """Integrating the conservation law over [SL*t, SR*t] x [0, t] gives the average state
    U* = (SR UR - SL UL - (FR - FL)) / (SR - SL); the flux at x = 0 inside the fan must then
    satisfy the jump condition across BOTH outer waves with that one state."""
    rng = np.random.default_rng(22)
    n_sub = 0
    for _ in range(400):
        L, R = rand_state(rng, mach=0.7), rand_state(rng, mach=0.7)
        bn = rng.normal()
        SL, SR = _outer_speeds(L, R, bn)
        if not (SL < 0 < SR):
            continue
        n_sub += 1
        UL, UR, FL, FR = cons(L, bn, G), cons(R, bn, G), phys_flux(L, bn, G), phys_flux(R, bn, G)
        Us = (SR * UR - SL * UL - (FR - FL)) / (SR - SL)
        F = oracle.hll(G, L, R, bn)
        scale = 1 + max(np.abs(FL).max(), np.abs(FR).max())
        assert np.allclose(F - FL, SL * (Us - UL), rtol=0, atol=1e-12 * scale)
        assert np.allclose(F - FR, SR * (Us - UR), rtol=0, atol=1e-12 * scale)
        assert Us[0] > 0                                   # the average density is positive
    assert n_sub > 200


def test_hll_galilean_fan_is_one_linear_piece():
    """G(V) = F(V) - V U(V) of the boosted problem is linear in V inside the fan with slope
    -U* (one star state), and equals F_K - V U_K outside: three regions, no more."""
    rng = np.random.default_rng(23)
    for _ in range(40):
        L, R = rand_state(rng), rand_state(rng)
        bn = rng.normal()
        SL, SR = _outer_speeds(L, R, bn)

        def Gv(V):
            Lb, Rb = L.copy(), R.copy()
            Lb[1] -= V; Rb[1] -= V
            Fp = oracle.hll(G, Lb, Rb, bn)
            g = Fp.copy()
            g[1] = Fp[1] + V * Fp[0]
            g[4] = Fp[4] + V * Fp[1] + 0.5 * V * V * Fp[0]
            return g
        UL, UR = cons(L, bn, G), cons(R, bn, G)
        Us = (SR * UR - SL * UL - (phys_flux(R, bn, G) - phys_flux(L, bn, G))) / (SR - SL)
        Vs = np.linspace(SL + 1e-3 * (SR - SL), SR - 1e-3 * (SR - SL), 9)
        g = np.array([Gv(V) for V in Vs])
        slope = (g[-1] - g[0]) / (Vs[-1] - Vs[0])
        scale = 1 + np.abs(g).max()
        assert np.allclose(slope, -Us, rtol=0, atol=1e-10 * scale)
        assert np.allclose(g, g[0] + np.outer(Vs - Vs[0], slope), rtol=0, atol=1e-10 * scale)
        for V, q in ((SL - 0.5, L), (SR + 0.5, R)):
            assert np.allclose(Gv(V), phys_flux(q, bn, G) - V * cons(q, bn, G), rtol=1e-12, atol=1e-12 * scale)


def test_hll_mirror_symmetry_and_diffusive_contact():
    rng = np.random.default_rng(24)
    flip = np.array([-1, 1, -1, -1, -1, -1, -1.0])     # same parity as test_hlld_mirror_symmetry
    for _ in range(300):
        L, R = rand_state(rng), rand_state(rng)
        bn = rng.normal()
        Lm, Rm = R.copy(), L.copy()
        Lm[1] *= -1; Rm[1] *= -1
        F = oracle.hll(G, L, R, bn)
        Fm = oracle.hll(G, Lm, Rm, -bn)
        assert np.allclose(Fm, flip * F, rtol=0, atol=1e-12 * (1 + np.abs(F).max()))
    # a stationary contact: HLLD keeps it exactly (zero mass flux), HLL smears it (the paper: "quite diffusive")
    L = np.array([1.0, 0, 0, 0, 1.0, 0.3, -0.2]); R = np.array([0.25, 0, 0, 0, 1.0, 0.3, -0.2])
    assert oracle.hlld(G, L, R, 0.5)[0] == 0.0
    assert oracle.hll(G, L, R, 0.5)[0] > 1e-2
