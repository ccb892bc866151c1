"""Pins of the CPU oracle (oracle/dgo.c) to things OTHER than itself (-m "not gpu").

Each test names the passage of the paper (PAPER.md = the extracted text of arXiv 2509.25347) or the piece of
mathematics that fixes the expected value.  None of the expected values comes from the oracle or the CUDA path.
"""
import os

import mpmath as mpm
import numpy as np
import pytest
from mpmath import mp, mpf

LD = np.longdouble
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "table1_collisions.txt")


def read_table1():
    tab = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, b, c = line.split()
            tab[k] = (float(b), float(c))
    return tab


def E_of(oracle, rho_g, rho_d, t_s, dt):
    """exp(dt*Omega) of ONE cell from the oracle's whole-path entry point, as an n x n longdouble matrix."""
    rho_d = np.asarray(rho_d, dtype=np.float64).reshape(-1, 1)
    t_s = np.asarray(t_s, dtype=np.float64).reshape(-1, 1)
    N = rho_d.shape[0]
    p = np.zeros((3, N + 1, 1))
    _, E, s = oracle.drag_update(np.array([rho_g], dtype=np.float64), rho_d, t_s, dt, p, want_E=True)
    return E[:, 0].reshape(N + 1, N + 1)


def omega_mp(rho_g, rho_d, t_s, dt):
    """dt*Omega of Eq. 17 in 50-digit arithmetic, retyped from the paper for the tests."""
    N = len(rho_d)
    A = mpm.zeros(N + 1, N + 1)
    for i in range(N):
        alpha = 1 / mpf(float(t_s[i]))
        eps = mpf(float(rho_d[i])) / mpf(float(rho_g))
        A[0, 0] -= eps * alpha * mpf(dt)
        A[0, i + 1] = alpha * mpf(dt)
        A[i + 1, 0] = eps * alpha * mpf(dt)
        A[i + 1, i + 1] = -alpha * mpf(dt)
    return A


def to_float_err(E_ld, E_mp):
    n = E_ld.shape[0]
    worst = mpf(0)
    for r in range(n):
        for c in range(n):
            # longdouble -> exact mpf via two doubles
            hi = float(E_ld[r, c]); lo = float(E_ld[r, c] - LD(hi))
            worst = max(worst, abs(mpf(hi) + mpf(lo) - E_mp[r, c]))
    return float(worst)


# ---------------------------------------------------------------- P1: N = 1 closed form (Dustybox)
@pytest.mark.parametrize("eps,ts,dt", [(0.5, 0.3, 0.1), (1e-3, 1e-6, 1e-2), (10.0, 1e2, 1e-2), (1.0, 1e-3, 5.0),
                                       (0.01, 1.0, 0.1), (3.0, 2e-5, 1e-2), (1e-4, 50.0, 1e-2)])
def test_p1_closed_form_one_dust_species(oracle, eps, ts, dt):
    """For N = 1, Omega^2 = -kappa*Omega with kappa = (1+eps)*alpha, hence exp(t*Omega) = I + phi*Omega with
    phi = (1 - exp(-kappa*t))/kappa: the classical Dustybox relaxation (Eq. 27-29 with N = 1, PAPER.md:212-220;
    Eq. 17)."""
    mp.dps = 50
    rho_g = 1.7
    rho_d = eps * rho_g
    E = E_of(oracle, rho_g, [rho_d], [ts], dt)
    e = mpf(float(rho_d)) / mpf(rho_g)
    alpha = 1 / mpf(ts)
    kappa = (1 + e) * alpha
    phi = -mpm.expm1(-kappa * mpf(dt)) / kappa
    Om = mpm.matrix([[-e * alpha, alpha], [e * alpha, -alpha]])
    Eref = mpm.eye(2) + phi * Om
    # the plain recurrence doubles its rounding error at every squaring: budget 2^s * 2^-62 (s from ||A||_1 <= 2^s)
    norm1 = 2 * dt / ts * max(1.0, eps)
    s = max(0, int(np.ceil(np.log2(norm1))))
    assert to_float_err(E, Eref) < max(4e-18, 2.0 ** (s - 62))


# ---------------------------------------------------------------- P2: Table 1 of the paper
@pytest.mark.parametrize("col", [0, 1])
def test_p2_table1_collision_tests(oracle, col):
    """PAPER.md:226-239 (Table 1) with Eq. 27-28: V(t) = V_CM + sum_i c_i exp(lambda_i t), in
    velocities, for tests B (col 0) and C (col 1).  The oracle acts on MOMENTA (Eq. 13, 16-18); velocities are
    momenta / densities.  The printed values carry 5 decimals, so |error| <= ~3e-5."""
    T = read_table1()
    g = lambda k: T[k][col]
    rho = np.array([g("rho_g"), g("rho_d1"), g("rho_d2")])
    v0 = np.array([g("v_g"), g("v_d1"), g("v_d2")])
    # Eq. 28 with the sum restored (R2)
    vcm = (rho * v0).sum() / rho.sum()
    assert abs(vcm - g("V_CM")) < 6e-6
    lam = np.array([g("lambda_1"), g("lambda_2")])
    coef = np.array([[g("c_g_1"), g("c_g_2")], [g("c_d1_1"), g("c_d1_2")], [g("c_d2_1"), g("c_d2_2")]])
    dt0 = g("dt_fig1")
    for mult in (0.0, 0.2, 1.0, 2.0, 5.0, 20.0, 200.0):
        t = dt0 * mult
        p_in = np.zeros((3, 3, 1))
        p_in[0, :, 0] = rho * v0            # x momenta
        p_in[1, :, 0] = -2.0 * rho * v0     # linearity in the other components
        out = oracle.drag_update(np.array([rho[0]]), rho[1:].reshape(2, 1), np.array([[g("T_s1")], [g("T_s2")]]), t, p_in)
        v = (out[0, :, 0] / rho).astype(np.float64)
        v_paper = g("V_CM") + (coef * np.exp(lam * t)[None, :]).sum(axis=1)
        assert np.max(np.abs(v - v_paper)) < 3e-5, (mult, v, v_paper)
        assert np.max(np.abs(out[1, :, 0] + 2 * out[0, :, 0])) < 1e-17


@pytest.mark.parametrize("col", [0, 1])
def test_p6_table1_eigenvalues_solve_secular_equation(col):
    """The non-zero eigenvalues of Eq. 17 solve 1 + sum_i eps_i alpha_i/(alpha_i + lambda) = 0 (expand det(Omega -
    lambda I) along the arrowhead; PAPER.md:218 says lambda_i < 0).  Checks the reading of the golden file itself."""
    T = read_table1()
    g = lambda k: T[k][col]
    eps = np.array([g("rho_d1"), g("rho_d2")]) / g("rho_g")
    alpha = 1.0 / np.array([g("T_s1"), g("T_s2")])
    for lam in (g("lambda_1"), g("lambda_2")):
        f = 1.0 + (eps * alpha / (alpha + lam)).sum()
        fp = -(eps * alpha / (alpha + lam) ** 2).sum()
        assert abs(f / fp) < 6e-6 * max(1.0, abs(lam) * 1e-3)  # Newton correction below the printed precision


# ---------------------------------------------------------------- P3, P4, P7: invariants of Eq. 17
def random_cell(rng, N, stiff):
    rho_g = 10 ** rng.uniform(-2, 2)
    if stiff:
        eps = 10 ** rng.uniform(-4, 1, N); ts = 10 ** rng.uniform(-6, 2, N)
    else:
        eps = 10 ** rng.uniform(-3, 0, N); ts = 10 ** rng.uniform(-3, 1, N)
    return rho_g, eps * rho_g, ts


@pytest.mark.parametrize("N", [1, 2, 3, 4, 7, 8, 12, 16])
@pytest.mark.parametrize("stiff", [False, True])
def test_p3_p4_p7_conservation_fixed_point_bounds(oracle, N, stiff):
    """Columns of Eq. 17 sum to zero (total momentum) => columns of exp sum to one.  Omega*rho = 0 =>
    equal velocities are a fixed point (long-time limit).  Omega is Metzler with zero column sums =>
    0 <= exp(t Omega)_ij <= 1."""
    rng = np.random.default_rng(100 + N)
    for _ in range(6):
        rho_g, rho_d, ts = random_cell(rng, N, stiff)
        E = E_of(oracle, rho_g, rho_d, ts, 1e-2)
        assert np.max(np.abs(E.sum(axis=0) - 1)) < 2e-14
        rho = np.concatenate(([rho_g], rho_d)).astype(LD)
        assert np.max(np.abs(E @ rho - rho) / rho.max()) < 2e-14
        assert E.min() > -1e-15 and E.max() < 1 + 1e-15


# ---------------------------------------------------------------- P5 / P10: independent algorithms in 50 digits
@pytest.mark.parametrize("N", [1, 2, 3, 4])
def test_p5_symmetric_eigendecomposition(oracle, N):
    """S = D^-1/2 (dt Omega) D^1/2 with D = diag(1, eps_i) is a symmetric arrowhead (S_00 = -sum eps_i a_i,
    S_0i = a_i sqrt(eps_i), S_ii = -a_i), so exp(dt Omega) = D^1/2 Q exp(Lambda) Q^T D^-1/2 (Eq. 29).
    mpmath's symmetric eigen-solver at 50 digits is an algorithm unrelated to scaling and squaring."""
    mp.dps = 50
    rng = np.random.default_rng(7 + N)
    for stiff in (False, True):
        rho_g, rho_d, ts = random_cell(rng, N, stiff)
        dt = 1e-2
        E = E_of(oracle, rho_g, rho_d, ts, dt)
        eps = [mpf(float(x)) / mpf(float(rho_g)) for x in rho_d]
        a = [mpf(dt) / mpf(float(x)) for x in ts]
        n = N + 1
        S = mpm.zeros(n, n)
        for i in range(N):
            S[0, 0] -= eps[i] * a[i]
            S[0, i + 1] = S[i + 1, 0] = a[i] * mpm.sqrt(eps[i])
            S[i + 1, i + 1] = -a[i]
        lam, Q = mpm.eigsy(S)
        d = [mpf(1)] + [mpm.sqrt(e) for e in eps]
        Eref = mpm.zeros(n, n)
        for r in range(n):
            for c in range(n):
                Eref[r, c] = d[r] / d[c] * sum(Q[r, k] * mpm.exp(lam[k]) * Q[c, k] for k in range(n))
        assert max(abs(l) for l in lam) > 0 and min(abs(l) for l in lam) < mpf(10) ** -40  # one zero eigenvalue
        assert all(l < mpf(10) ** -40 for l in lam)                                       # the rest negative
        assert to_float_err(E, Eref) < 2e-16


@pytest.mark.parametrize("N", [2, 4, 8, 16])
def test_p10_self_error_against_mpmath_expm(oracle, N):
    """Oracle self-error on the stiff regime of BASELINE.json config 4 (t_s log-uniform [1e-6,1e2], eps log-uniform
    [1e-4,10], dt = 1e-2) against mpmath.expm in 50 digits applied to Eq. 17 retyped above.  The plain long-double
    recurrence loses ~2^s * 2^-64; DESIGN.md budgets 3e-14 of the 1e-12 parity tolerance for it."""
    mp.dps = 50
    rng = np.random.default_rng(2024 + N)
    worst = 0.0
    for _ in range(4 if N == 16 else 8):
        rho_g = 1.0
        eps = 10 ** rng.uniform(-4, 1, N); ts = 10 ** rng.uniform(-6, 2, N)
        E = E_of(oracle, rho_g, eps * rho_g, ts, 1e-2)
        Eref = mpm.expm(omega_mp(rho_g, eps * rho_g, ts, 1e-2), method="taylor")
        worst = max(worst, to_float_err(E, Eref))
    assert worst < 3e-14, worst


# ---------------------------------------------------------------- P8, P9 and edge cases
def test_p8_semigroup_identity_and_long_time_limit(oracle):
    """Eq. 18: E(t)E(t) = E(2t); E(0) = I; t -> infinity: every column -> rho / sum(rho)
    (all fluids reach V_CM)."""
    rng = np.random.default_rng(5)
    rho_g, rho_d, ts = random_cell(rng, 5, False)
    E1 = E_of(oracle, rho_g, rho_d, ts, 0.037)
    E2 = E_of(oracle, rho_g, rho_d, ts, 0.074)
    assert np.max(np.abs(E1 @ E1 - E2)) < 1e-17
    E0 = E_of(oracle, rho_g, rho_d, ts, 0.0)
    assert np.array_equal(E0, np.eye(6, dtype=LD))
    Einf = E_of(oracle, rho_g, rho_d, ts, 2e3)     # slowest mode ~ exp(-2e3/max(t_s)) <= exp(-200)
    rho = np.concatenate(([rho_g], rho_d))
    # ||A||_1 ~ 4e6 here, so the plain recurrence carries ~2^22 * 2^-64 per entry; the limit itself is exact
    assert np.max(np.abs(Einf - (rho / rho.sum())[:, None])) < 1e-11


def test_p9_equivariance(oracle):
    """Eq. 14, 17: permuting the dust species permutes the result; scaling all densities changes nothing;
    the update is linear in the momenta."""
    rng = np.random.default_rng(9)
    N, nc = 6, 5
    rho_g = 10 ** rng.uniform(-1, 1, nc); rho_d = 10 ** rng.uniform(-3, 1, (N, nc)); ts = 10 ** rng.uniform(-4, 1, (N, nc))
    p = rng.standard_normal((3, N + 1, nc))
    base = oracle.drag_update(rho_g, rho_d, ts, 1e-2, p)
    perm = rng.permutation(N)
    pp = p.copy(); pp[:, 1:, :] = p[:, 1 + perm, :]
    out = oracle.drag_update(rho_g, rho_d[perm], ts[perm], 1e-2, pp)
    assert np.max(np.abs(out[:, 1:, :] - base[:, 1 + perm, :])) < 2e-16   # summation order changes
    assert np.max(np.abs(out[:, 0, :] - base[:, 0, :])) < 2e-16
    out = oracle.drag_update(4.0 * rho_g, 4.0 * rho_d, ts, 1e-2, p)   # exact scaling by a power of two
    assert np.array_equal(out, base)
    out = oracle.drag_update(rho_g, rho_d, ts, 1e-2, 8.0 * p)
    assert np.array_equal(out, 8.0 * base)


def test_zero_dust_density_species(oracle):
    """DESIGN.md R12: rho_d = 0 zeroes the column-0 entry of that species.  For N = 1 and eps = 0 the matrix is
    [[0, a],[0, -a]], whose exponential is [[1, 1-exp(-a)],[0, exp(-a)]] (upper triangular, by direct summation)."""
    mp.dps = 50
    E = E_of(oracle, 2.0, [0.0], [0.25], 0.1)
    a = mpf(0.1) / mpf(0.25)          # the fp64 input values, exactly
    Eref = mpm.matrix([[1, -mpm.expm1(-a)], [0, mpm.exp(-a)]])
    assert to_float_err(E, Eref) < 1e-19


def test_orientation_is_not_transposed(oracle):
    """Eq. 12: d M_g/dt = -sum alpha_i (eps_i M_g - M_d,i).  With all momentum initially in one
    dust species of a dust-poor cell (eps = 1e-3) and t >> T_s, the species keeps the fraction rho_d/(rho_g+rho_d)
    ~ 1e-3 of the momentum; a transposed matrix would keep ~1."""
    p = np.zeros((3, 2, 1)); p[0, 1, 0] = 1.0
    out = oracle.drag_update(np.array([1.0]), np.array([[1e-3]]), np.array([[1e-3]]), 1.0, p)
    assert abs(float(out[0, 1, 0]) - 1e-3 / 1.001) < 1e-15
    assert abs(float(out[0, 0, 0]) - 1.0 / 1.001) < 1e-15


def test_stage_functions_compose_to_whole_path(oracle):
    """The stage-level oracle entry points (a1, a2-a4, a5) are the same definitions as the whole path."""
    rng = np.random.default_rng(3)
    N, nc = 4, 7
    rho_g = 10 ** rng.uniform(-1, 1, nc); rho_d = 10 ** rng.uniform(-3, 1, (N, nc)); ts = 10 ** rng.uniform(-3, 1, (N, nc))
    p = rng.standard_normal((3, N + 1, nc))
    ref, Eref, sref = oracle.drag_update(rho_g, rho_d, ts, 1e-2, p, want_E=True)
    A = oracle.drag_matrix_build(rho_g, rho_d, ts, 1e-2)
    # Eq. 17 entry by entry
    n = N + 1
    for c in range(nc):
        M = A[:, c].reshape(n, n)
        for i in range(N):
            assert M[0, i + 1] == LD(1e-2) * (LD(1) / LD(ts[i, c]))
            assert M[i + 1, 0] == LD(1e-2) * ((LD(rho_d[i, c]) / LD(rho_g[c])) * (LD(1) / LD(ts[i, c])))
            assert M[i + 1, i + 1] == -M[0, i + 1]
        assert abs(M[0, 0] + M[1:, 0].sum()) < 1e-18 * abs(M[0, 0])
        assert np.count_nonzero(M) == 3 * N + 1
    E, s = oracle.expm_batch(A.astype(np.float64), N, rebuild_diag=True)
    assert np.array_equal(s, sref)
    assert np.max(np.abs(E - Eref)) < 1e-15   # A rounded to fp64 here, so not bitwise
    out = oracle.drag_apply(Eref.astype(np.float64), p, N)
    assert np.max(np.abs(out - ref)) < 1e-15
