"""First-order implicit RK1 drag step (App. A.1-A.2): U^(n+1) = (I - dt Omega)^-1 U^(n).

  -m "not gpu": pins of the ORACLE (oracle/dgo.c::dgo_rk1_update, a dense pivoted solve of Eq. A.6), none of whose
                expected values come from the oracle or the CUDA path;
  -m gpu:       the CUDA kernel behind dg_drag_rk1 (the O(N) closed form, Eq. A.8-A.9) against the oracle, element
                by element, and the EXP / RK1 accuracy comparison of Fig. 2 (RK1 first order, EXP flat).

Tolerance: the closed form is a handful of sums of non-negative terms and one division per species,
so per cell max|q_gpu - q_oracle| <= 1e-13 * max|p_in| with a wide margin (measured ~3e-16).
"""
import numpy as np
import pytest

from test_dustybox import table1_case, exact_velocities, fields, momenta

RK1_TOL = 1e-13


def random_cells(N, ncells, seed, stiff=True):
    g = np.random.default_rng(seed)
    rho_g = 10.0 ** g.uniform(-2, 2, ncells)
    eps = 10.0 ** g.uniform(-4, 1, (N, ncells))
    t_s = 10.0 ** (g.uniform(-6, 2, (N, ncells)) if stiff else g.uniform(-1, 1, (N, ncells)))
    p_in = g.normal(size=(3, N + 1, ncells))
    return rho_g, eps * rho_g[None, :], t_s, p_in


# ------------------------------------------------------------------------------------------------ oracle pins (CPU)
@pytest.mark.parametrize("N", [1, 2, 5, 16, 20])
def test_rk1_oracle_residual_in_50_digits(oracle, N):
    """(I - dt Omega) q = b (Eq. A.6) with Omega of Eq. 17 retyped here in mpmath."""
    import mpmath as mpm
    from mpmath import mp, mpf
    mp.dps = 50
    dt = 1e-2
    rho_g, rho_d, t_s, p_in = random_cells(N, 6, seed=N)
    q = oracle.rk1_update(rho_g, rho_d, t_s, dt, p_in)
    n = N + 1
    for c in range(6):
        M = mpm.eye(n)
        for i in range(1, n):
            a = mpf(dt) / mpf(float(t_s[i - 1, c]))
            e = mpf(float(rho_d[i - 1, c])) / mpf(float(rho_g[c]))
            M[0, 0] += e * a; M[0, i] -= a; M[i, 0] -= e * a; M[i, i] += a
        for comp in range(3):
            qv = mpm.matrix([mpf(float(np.float64(q[comp, k, c]))) + mpf(float(q[comp, k, c] - np.float64(q[comp, k, c])))
                             for k in range(n)])
            res = M * qv - mpm.matrix([mpf(float(x)) for x in p_in[comp, :, c]])
            scale = max(abs(float(x)) for x in p_in[comp, :, c]) * float(max(abs(M[r, r]) for r in range(n)))
            assert max(abs(res[k]) for k in range(n)) < 1e-17 * scale


def test_rk1_oracle_n1_closed_form(oracle):
    """N = 1: eliminating q_1 from Eq. A.7 by hand gives q_0 = (b_0 + c b_1) / (1 + eps c), c = a / (1 + a)."""
    rho_g = np.array([2.0]); rho_d = np.array([[0.6]]); t_s = np.array([[0.03]]); dt = 0.1
    b = np.array([[[1.5], [-0.25]], [[0.0], [1.0]], [[2.0], [0.6]]])
    q = oracle.rk1_update(rho_g, rho_d, t_s, dt, b)
    a = dt / 0.03; eps = 0.3; c = a / (1 + a)
    for comp in range(3):
        q0 = (b[comp, 0, 0] + c * b[comp, 1, 0]) / (1 + eps * c)
        q1 = (b[comp, 1, 0] + eps * a * q0) / (1 + a)
        assert abs(float(q[comp, 0, 0]) - q0) < 1e-15 and abs(float(q[comp, 1, 0]) - q1) < 1e-15


@pytest.mark.parametrize("N", [1, 4, 16])
def test_rk1_oracle_invariants(oracle, N):
    """Columns of Eq. 17 sum to zero, so 1^T (I - dt Omega) = 1^T: total momentum is conserved;
    Omega rho = 0, so equal velocities are a fixed point; dt -> infinity drives every fluid to V_CM (Eq. 28)."""
    # the dense solve's own rounding is ~cond(I - dt Omega) * 2^-64: ~1e-18 for the mild cells, ~1e-15 for the stiff
    for stiff, tol in ((False, 2e-17), (True, 1e-14)):
        rho_g, rho_d, t_s, p_in = random_cells(N, 50, seed=10 + N, stiff=stiff)
        q = oracle.rk1_update(rho_g, rho_d, t_s, 1e-2, p_in)
        assert float(oracle.conservation_error(q, p_in).max()) < tol
        rho = np.concatenate([rho_g[None], rho_d], axis=0)
        p_eq = np.stack([0.7 * rho, -1.3 * rho, 2.0 * rho])
        q = oracle.rk1_update(rho_g, rho_d, t_s, 1e-2, p_eq)
        assert float((np.abs(q - p_eq).max(axis=(0, 1)) / np.abs(p_eq).max(axis=(0, 1))).max()) < tol
    # backward Euler with dt >> T_s: every fluid lands on V_CM up to O(T_s / dt) (mild cells: I - dt Omega stays solvable)
    rho_g, rho_d, t_s, p_in = random_cells(N, 50, seed=10 + N, stiff=False)
    rho = np.concatenate([rho_g[None], rho_d], axis=0)
    q = oracle.rk1_update(rho_g, rho_d, t_s, 1e8, p_in)
    vcm = p_in.sum(axis=1) / rho.sum(axis=0)[None, :]
    assert float(np.abs(q / rho[None] - vcm[:, None, :]).max()) < 1e-5 * float(np.abs(p_in / rho[None]).max())


@pytest.mark.parametrize("col,t_final", [(0, 0.01), (1, 2.0)])
def test_rk1_oracle_is_first_order(oracle, col, t_final):
    """Fig. 2: RK1 is first order — halving dt halves the error against exp(t Omega) p(0)."""
    rho, v0, ts = table1_case(col)
    rho_g, rho_d, t_s = fields(rho, ts)
    v_ex = np.array([float(x) for x in exact_velocities(rho, ts, v0, [t_final])[0]])
    errs = []
    for M in (64, 128, 256):
        p = momenta(rho, v0)
        for _ in range(M):
            p = np.asarray(oracle.rk1_update(rho_g, rho_d, t_s, t_final / M, p), dtype=np.float64)
        errs.append(np.max(np.abs(p[0, :, 0] / rho - v_ex)))
    assert 1.8 < errs[0] / errs[1] < 2.2 and 1.8 < errs[1] / errs[2] < 2.2, errs


# ------------------------------------------------------------------------------------------------ CUDA path (GPU)
@pytest.mark.gpu
@pytest.mark.parametrize("N", list(range(1, 17)))
def test_gpu_rk1_parity_every_species_count(dg, oracle, cuda, N):
    import torch
    from paper_2509_25347_b200 import workloads as W
    wl = W.make_workload(5, ncells=2000 + 13 * N, N=N, device=cuda)
    out = dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in)
    torch.cuda.synchronize()
    rho_g, rho_d, t_s, p_in = wl.cells(torch.arange(wl.ncells))
    ref = oracle.rk1_update(rho_g, rho_d, t_s, wl.dt, p_in)
    got = out.cpu().numpy()
    assert np.isfinite(got).all()
    assert float(oracle.parity_error(got, ref, p_in).max()) <= RK1_TOL
    assert float(oracle.conservation_error(got, p_in).max()) <= 1e-13
    # in place, and dt = 0 is the identity bit for bit
    p = wl.p_in.clone()
    dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, p, p_out=p)
    assert torch.equal(p, out)
    assert torch.equal(dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, 0.0, wl.p_in), wl.p_in)


@pytest.mark.gpu
@pytest.mark.parametrize("config", [2, 3, 4])
def test_gpu_rk1_full_size_sampled(dg, oracle, cuda, config):
    import torch
    from paper_2509_25347_b200 import workloads as W
    wl = W.make_workload(config, device=cuda)
    out = dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in)
    idx = W.sample_cells(wl.ncells, 2048)
    rho_g, rho_d, t_s, p_in = wl.cells(idx)
    ref = oracle.rk1_update(rho_g, rho_d, t_s, wl.dt, p_in)
    got = out[:, :, idx.to(cuda)].cpu().numpy()
    assert float(oracle.parity_error(got, ref, p_in).max()) <= RK1_TOL
    drift = (out.sum(dim=1) - wl.p_in.sum(dim=1)).abs() / wl.p_in.abs().sum(dim=1)
    assert torch.isfinite(out).all() and float(drift.max()) <= 1e-13


@pytest.mark.gpu
@pytest.mark.parametrize("N,ncells", [(1, 1), (3, 31), (8, 129), (16, 257)])
def test_gpu_rk1_ragged_and_empty(dg, oracle, cuda, N, ncells):
    import torch
    from paper_2509_25347_b200 import workloads as W
    wl = W.make_workload(5, ncells=ncells, N=N, device=cuda)
    out = dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in)
    rho_g, rho_d, t_s, p_in = wl.cells(torch.arange(ncells))
    ref = oracle.rk1_update(rho_g, rho_d, t_s, wl.dt, p_in)
    assert float(oracle.parity_error(out.cpu().numpy(), ref, p_in).max()) <= RK1_TOL
    z = lambda *s: torch.empty(s, dtype=torch.float64, device=cuda)
    assert dg.dg_drag_rk1(z(0), z(N, 0), z(N, 0), 0.1, z(3, N + 1, 0)).shape == (3, N + 1, 0)


@pytest.mark.gpu
def test_gpu_exp_beats_rk1_by_orders_of_magnitude(dg, cuda):
    """Collision test B stepped to t = 0.01: RK1's error falls linearly with dt, EXP's is at
    rounding level for every dt."""
    import torch
    rho, v0, ts = table1_case(0)
    rho_g, rho_d, t_s = fields(rho, ts)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(cuda)
    t_final = 0.01
    v_ex = np.array([float(x) for x in exact_velocities(rho, ts, v0, [t_final])[0]])
    e_rk1, e_exp = [], []
    for M in (25, 50, 100):
        p = dev(momenta(rho, v0)); q = p.clone()
        for _ in range(M):
            p = dg.dg_drag_rk1(dev(rho_g), dev(rho_d), dev(t_s), t_final / M, p)
        q = dg.dg_drag_update_steps(dev(rho_g), dev(rho_d), dev(t_s), t_final / M, q, M)
        e_rk1.append(np.max(np.abs(p[0, :, 0].cpu().numpy() / rho - v_ex)))
        e_exp.append(np.max(np.abs(q[0, :, 0].cpu().numpy() / rho - v_ex)))
    assert 1.7 < e_rk1[0] / e_rk1[1] < 2.3 and 1.7 < e_rk1[1] / e_rk1[2] < 2.3
    assert max(e_exp) < 1e-13 and min(e_rk1) > 1e-4
