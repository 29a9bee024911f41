"""Mutation harness for the oracle's pins.

Every entry of MUTANTS is a plausible mistake -- a swapped weight, a dropped term, a wrong sign,
index or metric factor -- applied as an exact text substitution to a COPY of oracle/mhd_oracle.c in
a temporary directory.  The copy is compiled and the pin suites (tests/test_oracle_pointwise.py,
test_oracle_stages.py, test_oracle_scheme.py, test_oracle_local.py) are run against it in a subprocess
(MHD_ORACLE_LIBDIR, see oracle/__init__.py).  A mutant that passes every pin is a hole in the
pins, and this test fails.  The unmutated copy must pass (the harness itself is sound) and every
substitution must match exactly once (the list follows the source).
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "mhd_oracle.c")
PINS = ["tests/test_oracle_pointwise.py", "tests/test_oracle_stages.py", "tests/test_oracle_scheme.py",
        "tests/test_oracle_local.py"]

# name: (old text, new text, pin files to try first)
MUTANTS = {
    # ---- O7, the 2D Riemann problem -------------------------------------------------------
    "emf2d step 5: B* weights swapped (north/south)": (
        "BsW = bN * Bs[SW] + bS * Bs[NW];\n    BsE = bN * Bs[SE] + bS * Bs[NE];",
        "BsW = bS * Bs[SW] + bN * Bs[NW];\n    BsE = bS * Bs[SE] + bN * Bs[NE];", PINS[:1]),
    "emf2d step 5: A* weights swapped (east/west)": (
        "AsS = aE * As[SW] + aW * As[SE];\n    AsN = aE * As[NW] + aW * As[NE];",
        "AsS = aW * As[SW] + aE * As[SE];\n    AsN = aW * As[NW] + aE * As[NE];", PINS[:1]),
    "emf2d step 5: all four star-field weights swapped": (
        "BsW = bN * Bs[SW] + bS * Bs[NW];\n    BsE = bN * Bs[SE] + bS * Bs[NE];\n"
        "    AsS = aE * As[SW] + aW * As[SE];\n    AsN = aE * As[NW] + aW * As[NE];",
        "BsW = bS * Bs[SW] + bN * Bs[NW];\n    BsE = bS * Bs[SE] + bN * Bs[NE];\n"
        "    AsS = aW * As[SW] + aE * As[SE];\n    AsN = aW * As[NW] + aE * As[NE];", PINS[:1]),
    "emf2d step 5: star fields replaced by plain means": (
        "BsW = bN * Bs[SW] + bS * Bs[NW];", "BsW = HALF * (Bs[SW] + Bs[NW]);", PINS[:1]),
    "emf2d step 3: inner speed max <-> min": (
        "SEs = tE <= ZERO ? ZERO : rmax(ZERO, rmax(xS.hi, xN.hi));",
        "SEs = tE <= ZERO ? ZERO : rmax(ZERO, rmin(xS.hi, xN.hi));", PINS[:1]),
    "emf2d step 4: star EMF, sign of the y jump term": (
        "es[q] = e[q] + Sx[q] * (Bs[q] - B[q]) - Sy[q] * (As[q] - A[q]);",
        "es[q] = e[q] + Sx[q] * (Bs[q] - B[q]) + Sy[q] * (As[q] - A[q]);", PINS[:1]),
    "emf2d step 4: star EMF, y jump term dropped": (
        "es[q] = e[q] + Sx[q] * (Bs[q] - B[q]) - Sy[q] * (As[q] - A[q]);",
        "es[q] = e[q] + Sx[q] * (Bs[q] - B[q]);", PINS[:1]),
    "emf2d step 6: sign of the y dissipation": (
        "+ dissx * (BsE - BsW) - dissy * (AsN - AsS);", "+ dissx * (BsE - BsW) + dissy * (AsN - AsS);", PINS[:1]),
    "emf2d step 6: x dissipation dropped": (
        "+ dissx * (BsE - BsW) - dissy * (AsN - AsS);", "- dissy * (AsN - AsS);", PINS[:1]),
    "emf2d: corner EMF sign (u B - v A)": (
        "e[q] = ua * B[q] - ub * A[q];", "e[q] = ub * A[q] - ua * B[q];", PINS[:1]),
    "emf2d: sub-problem star field, wrong numerator": (
        "s.btsL = (R_FABS(DL) <= (real)16 * R_EPS * refL) ? btL : btL * (refL - bn * bn) / DL;",
        "s.btsL = (R_FABS(DL) <= (real)16 * R_EPS * refL) ? btL : btL * (refL + bn * bn) / DL;", PINS[:1]),
    # ---- O6, HLLD -------------------------------------------------------------------------
    "hlld: v** sign of the field term": (
        "real vss = (rL * vsL + rR * vsR + (bysR - bysL) * sg) / rsum;",
        "real vss = (rL * vsL + rR * vsR - (bysR - bysL) * sg) / rsum;", PINS[:1]),
    "hlld: E** sign": (
        "UssL[4] = UsL[4] - rL * (ubsL - ubss) * sg;", "UssL[4] = UsL[4] + rL * (ubsL - ubss) * sg;", PINS[:1]),
    "hlld: E* drops the u.B term": (
        "real EsL = (sdL * UL[4] - pTL * uL + pTs * SM + bn * (ubL - ubs)) / (SL - SM);",
        "real EsL = (sdL * UL[4] - pTL * uL + pTs * SM) / (SL - SM);", PINS[:1]),
    "hlld: B* numerator": (
        "bysL = byL * (ref - bn * bn) / D;", "bysL = byL * (ref + bn * bn) / D;", PINS[:1]),
    "hlld: By** weights transposed": (
        "real byss = (rL * bysR + rR * bysL + rL * rR * (vsR - vsL) * sg) / rsum;",
        "real byss = (rL * bysL + rR * bysR + rL * rR * (vsR - vsL) * sg) / rsum;", PINS[:1]),
    # ---- stages ---------------------------------------------------------------------------
    "O3: face-field slopes zeroed": (
        "S->dbf[dbf_index(a, t)][c] = orc_limiter(G->limiter, b[c] - b[c - s[t]], b[c + s[t]] - b[c]);",
        "S->dbf[dbf_index(a, t)][c] = ZERO;", PINS[1:]),
    "O4a: averaging stencil of the edge EMF (one cell dropped)": (
        "real ub = QUART * (u[c] + u[c - sy] + u[c - sx] + u[c - sx - sy]);   /* Eq. 8  */",
        "real ub = QUART * (u[c] + u[c - sy] + u[c - sx] + u[c - sx]);   /* Eq. 8  */", PINS[1:]),
    "O4b: metric factors of the half-step bx swapped": (
        "S->bh[0][c] = Up[5][c] + hdt * ((ez[c + sy] - ez[c]) / G->dx[1] - (ey[c + sz] - ey[c]) / G->dx[2]);",
        "S->bh[0][c] = Up[5][c] + hdt * ((ez[c + sy] - ez[c]) / G->dx[2] - (ey[c + sz] - ey[c]) / G->dx[1]);", PINS[1:]),
    "O4c: gamma missing in the pressure predictor": (
        "p_h -= lam[d] * (vel[d] * S->dq[d][4][c] + G->gamma * p * du_d);",
        "p_h -= lam[d] * (vel[d] * S->dq[d][4][c] + p * du_d);", PINS[1:]),
    "O4c: sign of the magnetic tension": (
        "vel_h[a] += (lam[b] * bc[b] * S->dq[b][5 + a][c] + lam[e] * bc[e] * S->dq[e][5 + a][c]) / rho;",
        "vel_h[a] -= (lam[b] * bc[b] * S->dq[b][5 + a][c] + lam[e] * bc[e] * S->dq[e][5 + a][c]) / rho;", PINS[1:]),
    "O5: corner signs flipped along b": (
        "real sga[4] = {1, -1, 1, -1}, sgb[4] = {1, 1, -1, -1};",
        "real sga[4] = {1, -1, 1, -1}, sgb[4] = {-1, -1, 1, 1};", PINS[1:]),
    "O5: corner cells (SE and NW exchanged)": (
        "long cc[4] = {c - s[a] - s[b], c - s[b], c - s[a], c};",
        "long cc[4] = {c - s[a] - s[b], c - s[a], c - s[b], c};", PINS[1:]),
    "O5: sign of the A_S face-field slope": (
        "real AS = S->bh[a][c - s[b]] + HALF * dba[c - s[b]];",
        "real AS = S->bh[a][c - s[b]] - HALF * dba[c - s[b]];", PINS[1:]),
    "O6 call: flux rotation (transverse momenta exchanged)": (
        "S->flux[d][1 + t1][c] = F[2];\n      S->flux[d][1 + t2][c] = F[3];",
        "S->flux[d][1 + t2][c] = F[2];\n      S->flux[d][1 + t1][c] = F[3];", PINS[1:]),
    "O8: EMF metric factors swapped (PAPER.md L154)": (
        "Un[5 + a][c] = Up[5 + a][c] + dt * ((S->emf[e][c + s[b]] - S->emf[e][c]) / G->dx[b]\n"
        "                                        - (S->emf[b][c + s[e]] - S->emf[b][c]) / G->dx[e]);",
        "Un[5 + a][c] = Up[5 + a][c] + dt * ((S->emf[e][c + s[b]] - S->emf[e][c]) / G->dx[e]\n"
        "                                        - (S->emf[b][c + s[e]] - S->emf[b][c]) / G->dx[b]);", PINS[1:]),
    # ---- O10, local time steps -------------------------------------------------------------
    "O10: interpolation weight measured from the wrong slice": (
        "real w = (real)((t_new[p] - t_old[q]) / (t_new[q] - t_old[q]));",
        "real w = (real)((t_new[q] - t_new[p]) / (t_new[q] - t_old[q]));", PINS[3:]),
    "O10: interpolation to the patch's OLD time": (
        "real w = (real)((t_new[p] - t_old[q]) / (t_new[q] - t_old[q]));",
        "real w = (real)((t_old[p] - t_old[q]) / (t_new[q] - t_old[q]));", PINS[3:]),
    "O10: no interpolation (newer slice always)": (
        "v = vold + w * (vnew - vold);", "v = vnew;", PINS[3:]),
    "O10: readiness accepts a patch that is ahead of a neighbour": (
        "int hi_ok = t_new[p] <= t_new[q] || times_equal(t_new[p], t_new[q]);", "int hi_ok = 1;", PINS[3:]),
    "O10: the step writes the newer slice instead of the older": (
        "Un[f] = S[1 - cur[p]] + ((long)f * G.np + p) * G.M;", "Un[f] = S[cur[p]] + ((long)f * G.np + p) * G.M;", PINS[3:]),
    "O9: CFL sum over directions replaced by the last term": (
        "rate += (R_FABS(vel[a]) + cf) / G.dx[a];", "rate = (R_FABS(vel[a]) + cf) / G.dx[a];", PINS[1:2]),
}


def _run_pins(libdir, files):
    env = dict(os.environ, MHD_ORACLE_LIBDIR=libdir)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-m", "not gpu", *files],
                       cwd=ROOT, env=env, capture_output=True, text=True)
    return r.returncode, r.stdout[-1500:]


def _mutant_survives(args):
    name, tmp = args
    from oracle import build as obuild
    old, new, first = MUTANTS[name]
    src = open(SRC).read()
    if src.count(old) != 1:
        return name, "substitution does not match the source exactly once"
    d = os.path.join(tmp, "m%03d" % (sorted(MUTANTS).index(name)))
    os.makedirs(d)
    path = os.path.join(d, "mhd_oracle.c")
    with open(path, "w") as fh:
        fh.write(src.replace(old, new))
    obuild.compile_to(path, d)
    rest = [f for f in PINS if f not in first]
    for files in (first, rest):
        if files and _run_pins(d, files)[0] != 0:
            return name, None          # killed
    return name, "SURVIVED every pin"


def test_unmutated_copy_passes_through_the_harness(tmp_path):
    from oracle import build as obuild
    obuild.compile_to(SRC, str(tmp_path))
    rc, out = _run_pins(str(tmp_path), PINS[:1])
    assert rc == 0, out


def test_every_mutant_of_the_oracle_fails_a_pin(tmp_path):
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(_mutant_survives, [(name, str(tmp_path)) for name in MUTANTS]))
    bad = {name: why for name, why in results if why}
    assert not bad, bad
