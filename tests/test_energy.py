"""Frictional heating over one exact drag step (Eq. 4 and Eq. 11; R20).

The paper gives no discrete formula for the gas energy in the EXP step.  The reading: integrate Eq. 4's drag terms
exactly along the exact momenta p(t) = exp(t Omega) p(0).  CPU pins of the oracle (not gpu): the heating integral
against a high-order quadrature of Eq. 4's w-term retyped here (mpmath), and the N = 1 closed form.  GPU test: the
CUDA entry point dg_drag_update_energy against the oracle.
"""
import numpy as np
import pytest
import torch

LD = np.longdouble


def _cell(N, seed, stiff=1.0):
    rng = np.random.default_rng(seed)
    rho_g = np.array([10 ** rng.uniform(-1, 1)])
    rho_d = (10 ** rng.uniform(-3, 0.5, size=(N, 1))) * rho_g
    t_s = 10 ** rng.uniform(-2, 1, size=(N, 1)) / stiff
    p = rng.normal(size=(3, N + 1, 1))
    E = np.array([5.0 + rng.uniform()])
    return rho_g, rho_d, t_s, p, E


@pytest.mark.parametrize("N,seed,dt,stiff", [(1, 1, 0.3, 1.0), (2, 2, 0.05, 1.0), (3, 3, 1.0, 1.0), (4, 4, 0.2, 30.0), (8, 5, 0.1, 3.0)])
def test_heating_equals_the_quadrature_of_eq_4(oracle, N, seed, dt, stiff):
    """int_0^dt  sum_i rho_d,i |v_d,i - v_g|^2 / T_s,i  dt'  along p(t') = exp(t' Omega) p(0), Omega of Eq. 17
     and the integrand of Eq. 4 both retyped here, by Gauss-Legendre quadrature in
    30-digit arithmetic; and the work term  int v_g . dM_g  = change of the gas kinetic energy."""
    import mpmath as mpm
    from mpmath import mp, mpf
    mp.dps = 30
    rho_g, rho_d, t_s, p, E = _cell(N, seed, stiff)
    n = N + 1
    Om = mpm.zeros(n, n)
    for i in range(N):
        al = 1 / mpf(float(t_s[i, 0])); e = mpf(float(rho_d[i, 0])) / mpf(float(rho_g[0]))
        Om[0, 0] -= e * al; Om[0, i + 1] = al; Om[i + 1, 0] = e * al; Om[i + 1, i + 1] = -al
    rho = [mpf(float(rho_g[0]))] + [mpf(float(x)) for x in rho_d[:, 0]]
    p0 = [mpm.matrix([mpf(float(x)) for x in p[c, :, 0]]) for c in range(3)]

    def state(t):
        Et = mpm.expm(Om * t)
        return [Et * v for v in p0]

    def dissipation(t):
        pt = state(t)
        tot = mpf(0)
        for i in range(1, n):
            dv2 = sum((pt[c][i] / rho[i] - pt[c][0] / rho[0]) ** 2 for c in range(3))
            tot += rho[i] * dv2 / mpf(float(t_s[i - 1, 0]))
        return tot

    heat = mpm.quad(dissipation, mpm.linspace(0, dt, 9))
    pe = state(mpf(dt))
    keg = lambda q: sum(q[c][0] ** 2 for c in range(3)) / (2 * rho[0])
    work = keg(pe) - keg(p0)
    for w in (0.0, 1.0, 0.37):
        E_out, _ = oracle.energy_update(rho_g, rho_d, t_s, dt, p, E, w)
        expect = mpf(float(E[0])) + work + mpf(w) * heat
        scale = float(sum(sum(p0[c][k] ** 2 / (2 * rho[k]) for k in range(n)) for c in range(3)))
        assert abs(mpf(float(E_out[0])) - expect) <= 1e-15 * max(scale, abs(float(E[0])))


def test_heating_n1_closed_form(oracle):
    """N = 1: the relative velocity decays as exp(-kappa t), kappa = (1 + eps)/T_s (Eq. 27-29), so
    the dissipated energy is  mu |dv_0|^2 (1 - exp(-2 kappa dt)) / 2  with the reduced density mu = rho_g rho_d /
    (rho_g + rho_d); the total momentum, hence the centre-of-mass kinetic energy, does not change."""
    rng = np.random.default_rng(7)
    for _ in range(20):
        rho_g = np.array([10 ** rng.uniform(-2, 2)]); rho_d = np.array([[10 ** rng.uniform(-3, 2)]])
        t_s = np.array([[10 ** rng.uniform(-3, 2)]]); dt = 10 ** rng.uniform(-3, 1)
        p = rng.normal(size=(3, 2, 1)); E = np.array([rng.uniform(1, 10)])
        mu = rho_g[0] * rho_d[0, 0] / (rho_g[0] + rho_d[0, 0])
        dv2 = sum((p[c, 1, 0] / rho_d[0, 0] - p[c, 0, 0] / rho_g[0]) ** 2 for c in range(3))
        kappa = (1 + rho_d[0, 0] / rho_g[0]) / t_s[0, 0]
        heat = 0.5 * mu * dv2 * -np.expm1(-2 * kappa * dt)
        E1, p_out = oracle.energy_update(rho_g, rho_d, t_s, dt, p, E, 1.0)
        E0, _ = oracle.energy_update(rho_g, rho_d, t_s, dt, p, E, 0.0)
        assert abs(float(E1[0] - E0[0]) - heat) <= 2e-15 * max(heat, 1e-300) + 1e-16 * float(E[0])
        # w = 1: gas energy + dust kinetic energy is conserved over the step
        kd = lambda q: sum(float(q[c, 1, 0]) ** 2 for c in range(3)) / (2 * rho_d[0, 0])
        assert abs((float(E1[0]) + kd(p_out)) - (float(E[0]) + kd(p))) <= 1e-15 * (float(E[0]) + kd(p))


@pytest.mark.gpu
@pytest.mark.parametrize("ncells", [1501, 2048, 2570])
@pytest.mark.parametrize("N", [1, 2, 4, 7, 8, 12, 13, 14, 15, 16])
def test_gpu_energy_update_matches_the_oracle(dg, oracle, cuda, N, ncells):
    """dg_drag_update_energy through the C ABI against the oracle: momenta at BASELINE.json's tolerance, gas energy to
    1e-13 of the cell's energy scale (E_g and the kinetic energies: a handful of fp64 products and one difference).
    One launch for every N: the sorted-tile kernel for N <= 12 (whole tiles by bulk copies for the even cell counts,
    per-thread copies for the odd one and the ragged tails), the pair-per-cell kernel for N >= 13 (each lane sums over the
    rows it applies; the ragged last chunk has lanes without a cell)."""
    from paper_2509_25347_b200 import workloads as W
    wl = W.make_workload(5, ncells=ncells, N=N, device=cuda)
    wl.rho_d[0, ::5] = 0.0
    g = torch.Generator(device="cpu"); g.manual_seed(N)
    E_in = (1.0 + 10 * torch.rand(wl.ncells, generator=g, dtype=torch.float64)).to(cuda)
    rho_g, rho_d, t_s, p_in = wl.cells(torch.arange(wl.ncells))
    for w in (0.0, 1.0, 0.5):
        p_out, E_out = dg.dg_drag_update_energy(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, E_in, w)
        torch.cuda.synchronize()
        E_ref, p_ref = oracle.energy_update(rho_g, rho_d, t_s, wl.dt, p_in, E_in.cpu().numpy(), w)
        assert float(oracle.parity_error(p_out.cpu().numpy(), p_ref, p_in).max()) <= 1e-12
        kin = (p_in[:, 0] ** 2).sum(axis=0) / (2 * rho_g)
        rd = np.where(rho_d > 0, rho_d, 1.0)
        kin = kin + np.where(rho_d > 0, (p_in[:, 1:] ** 2).sum(axis=0) / (2 * rd), 0.0).sum(axis=0)
        scale = np.abs(E_in.cpu().numpy()) + kin
        assert float((np.abs(E_out.cpu().numpy().astype(LD) - E_ref) / scale).max()) <= 1e-13
    # the momenta are those of the plain update, bit for bit
    assert torch.equal(p_out, dg.dg_drag_update(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in))
    # E arrays that are 8 but not 16 bytes aligned (no bulk copies): same bits
    big = torch.empty(wl.ncells + 3, dtype=torch.float64, device=cuda)
    E_sh = big[1:1 + wl.ncells]; E_sh.copy_(E_in)
    big2 = torch.empty(wl.ncells + 3, dtype=torch.float64, device=cuda)
    E_sh_out = big2[1:1 + wl.ncells]
    p3, _ = dg.dg_drag_update_energy(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, E_sh, 0.5, E_out=E_sh_out)
    assert torch.equal(p3, p_out) and torch.equal(E_sh_out, E_out)
    # in place (p_out aliases p_in, E_out aliases E_in) gives the same bits
    p2 = wl.p_in.clone(); E2 = E_in.clone()
    dg.dg_drag_update_energy(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, p2, E2, 0.5, p_out=p2, E_out=E2)
    assert torch.equal(p2, p_out) and torch.equal(E2, E_out)
