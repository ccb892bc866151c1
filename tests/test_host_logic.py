"""CPU-side checks (-m "not gpu"): the C-ABI library builds, loads and exports what include/dg.h declares; argument
validation that returns before any CUDA call; the Table B.1 constants compiled into the kernels; the seeded workload
generators; the bench's cross-rank aggregation over gloo (world_size 2)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "dg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dg_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(dg):
    names = declared_functions()
    assert {"dg_drag_matrix_build", "dg_expm_scale_square", "dg_drag_apply", "dg_drag_update"} <= set(names)
    lib = C.CDLL(dg.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), name
    assert set(names) == set(dg.EXPORTS)
    assert dg.dg_version() == 100
    for N in range(1, 17):
        assert dg.dg_variant_name(N)
        assert dg.dg_launches_per_update(N, 1000) >= 1
    assert dg.dg_launches_per_update(4, 0) == 0


def test_argument_validation_without_a_gpu(dg):
    """These calls return before any CUDA call is made (include/dg.h, 'Errors')."""
    lib = dg.raw()
    buf = (C.c_double * 64)()
    p = C.addressof(buf)
    assert lib.dg_drag_update(p, p, p, 0.1, p, 0, 4, p, None) == dg.DG_ERANGE
    assert lib.dg_drag_update(p, p, p, 0.1, p, 17, 4, p, None) == dg.DG_ERANGE
    assert lib.dg_drag_update(p, p, p, 0.1, p, 4, -1, p, None) == dg.DG_ERANGE
    assert lib.dg_drag_update(p, p, p, float("nan"), p, 4, 4, p, None) == dg.DG_EINVAL
    assert lib.dg_drag_update(p, p, p, float("inf"), p, 4, 4, p, None) == dg.DG_EINVAL
    assert lib.dg_drag_update(p, p, p, -1.0, p, 4, 4, p, None) == dg.DG_EINVAL
    assert lib.dg_drag_update(None, p, p, 0.1, p, 4, 4, p, None) == dg.DG_ENULL
    assert lib.dg_drag_update(p, p, p, 0.1, p, 4, 4, p + 1, None) == dg.DG_EALIGN
    assert lib.dg_drag_update(None, None, None, 0.1, None, 4, 0, None, None) == dg.DG_OK     # ncells = 0: no-op
    assert lib.dg_drag_matrix_build(p, p, p, 0.1, 4, 0, None, None) == dg.DG_OK
    assert lib.dg_drag_matrix_build(p, p, None, 0.1, 4, 8, p, None) == dg.DG_ENULL
    assert lib.dg_expm_scale_square(None, 4, 8, p, None, None) == dg.DG_ENULL
    assert lib.dg_expm_scale_square(p, 4, 8, p, p + 2, None) == dg.DG_EALIGN
    assert lib.dg_drag_apply(p, p, 99, 8, p, None) == dg.DG_ERANGE
    assert lib.dg_drag_update_host(p, p, p, 0.1, p, 4, 0, p, 0, -1) == dg.DG_OK
    assert lib.dg_drag_update_host(p, p, p, 0.1, p, 4, 8, None, 0, -1) == dg.DG_ENULL
    assert lib.dg_drag_update_host(p, p, p, 0.1, p, 4, 8, p, -5, -1) == dg.DG_EINVAL
    # dg_drag_update_variant: unknown variants, and the sorted-tile kernel beyond the species counts it is built for
    v = lib.dg_drag_update_variant
    assert v(p, p, p, 0.1, p, 4, 4, p, None, None, 8, None) == dg.DG_EINVAL
    assert v(p, p, p, 0.1, p, 4, 4, p, None, None, -1, None) == dg.DG_EINVAL
    assert v(p, p, p, 0.1, p, 13, 4, p, None, None, dg.DG_VARIANT_TPS, None) == dg.DG_EINVAL
    assert v(p, p, p, 0.1, p, 12, 0, p, None, None, dg.DG_VARIANT_TPS, None) == dg.DG_OK          # ncells = 0: no-op
    for N in range(1, 17):   # the default mapping named for every N: sorted tiles up to 12, pair per cell above
        name = dg.dg_variant_name(N)
        assert ("thread-per-cell" in name) == (N <= 12) and ("pair-per-cell" in name) == (N >= 13), (N, name)
    for st in range(7):
        assert dg.raw().dg_status_string(st).decode().startswith("DG_")
    # the test hook that replaced the DG_HOST_MAX_PITCH environment variable
    assert lib.dg_host_set_max_pitch(-1) == dg.DG_EINVAL
    assert lib.dg_host_set_max_pitch(4096) == dg.DG_OK and lib.dg_host_set_max_pitch(0) == dg.DG_OK
    with pytest.raises(TypeError):
        dg.dg_drag_update(torch.zeros(4), torch.zeros(1, 4), torch.zeros(1, 4), 0.1, torch.zeros(3, 2, 4))


def test_table_b1_constants_in_the_kernels():
    """theta_m of Eq. B.4-B.8 recomputed here from the definition with mpmath at 60 digits:
    f_m(theta) = sum_{j>m} |c_j| theta^j with c_j the series coefficients of e^{-x} T_m(x) - 1, and theta_m the largest
    theta with -log(1 - f_m(theta))/theta <= 2^-53.  The constants compiled into the kernels must lie just BELOW these
    (rounded down) and agree with Table B.1 where it is legible."""
    from mpmath import mp, mpf, factorial, log
    mp.dps = 60
    src = open(os.path.join(ROOT, "paper_2509_25347_b200", "csrc", "dg_params.cuh")).read()
    ms = [int(x) for x in re.search(r"c_m\[kRows\]\s*=\s*\{([^}]*)\}", src).group(1).split(",")]
    th = [float(x) for x in re.search(r"c_theta\[kRows\]\s*=\s*\{([^}]*)\}", src, flags=re.S).group(1).split(",")]
    assert ms == [2, 4, 6, 9, 12, 16, 20, 25, 30]                      # m_k column of Table B.1
    printed = {2: 2.5810e-8, 4: 3.3972e-4, 6: 9.0657e-3, 9: 8.9578e-2, 20: 1.4383, 25: 2.4286, 30: 3.5397}
    u = mpf(2) ** -53
    for m, theta_c in zip(ms, th):
        c = {}
        for tot in range(m + 1, m + 120):
            c[tot] = -sum((mpf(-1) ** (tot - j) / factorial(tot - j)) / factorial(j) for j in range(m + 1, tot + 1))
        f = lambda t: sum(abs(v) * t ** k for k, v in c.items())
        bound = lambda t: -log(1 - f(t)) / t
        t = mpf(theta_c)
        assert bound(t) <= u                      # the compiled constant satisfies Theorem 1's premise
        assert bound(t * (1 + mpf(10) ** -8)) > u   # and is tight to 1e-8
        if m in printed:
            assert abs(theta_c / printed[m] - 1) < 6e-5
    # q_k * r_k = m_k and Pi = q + r - 2 (Eq. B.9 as repaired in DESIGN.md R7) reproduce the Pi column 1..9
    qr = [(1, 2), (2, 2), (2, 3), (3, 3), (3, 4), (4, 4), (4, 5), (5, 5), (5, 6)]
    assert [q * r for q, r in qr] == ms and [q + r - 2 for q, r in qr] == list(range(1, 10))


def test_single_precision_thresholds_of_eq_b8():
    """Eq. B.8 names u = 2^-24 as an alternative unit round-off.  The single-precision thresholds compiled
    into the kernels (dg_params.cuh c_theta32) are recomputed here from Eq. B.4-B.8 with the same 60-digit routine as
    the u = 2^-53 column above: each constant must satisfy the bound and be tight to 1e-6 (they are floats)."""
    from mpmath import mp, mpf, factorial, log
    mp.dps = 60
    src = open(os.path.join(ROOT, "paper_2509_25347_b200", "csrc", "dg_params.cuh")).read()
    th = [float(np.float32(x.strip().rstrip("f"))) for x in
          re.search(r"c_theta32\[kRows\]\s*=\s*\{([^}]*)\}", src, flags=re.S).group(1).split(",")]
    ms = [2, 4, 6, 9, 12, 16, 20, 25, 30]
    assert len(th) == 9
    u = mpf(2) ** -24
    for m, theta_c in zip(ms, th):
        c = {}
        for tot in range(m + 1, m + 140):
            c[tot] = -sum((mpf(-1) ** (tot - j) / factorial(tot - j)) / factorial(j) for j in range(m + 1, tot + 1))
        f = lambda t: sum(abs(v) * t ** k for k, v in c.items())
        bound = lambda t: -log(1 - f(t)) / t
        t = mpf(theta_c)
        assert f(t) < 1 and bound(t) <= u
        assert bound(t * (1 + mpf(10) ** -6)) > u
    assert all(a < b for a, b in zip(th, th[1:]))
    # every single-precision threshold is larger than its double-precision twin: fewer squarings for the same norm
    th64 = [float(x) for x in re.search(r"c_theta\[kRows\]\s*=\s*\{([^}]*)\}", src, flags=re.S).group(1).split(",")]
    assert all(a > b for a, b in zip(th, th64))


def test_workload_generators_are_seeded_and_shaped():
    from paper_2509_25347_b200 import workloads as W
    for cfg, N in [(1, 1), (2, 4), (3, 8), (4, 16), (5, 12)]:
        a = W.make_workload(cfg, ncells=512, N=N if cfg == 5 else None)
        b = W.make_workload(cfg, ncells=512, N=N if cfg == 5 else None)
        assert a.N == N and a.rho_g.shape == (512,) and a.rho_d.shape == (N, 512) and a.t_s.shape == (N, 512)
        assert a.p_in.shape == (3, N + 1, 512) and a.p_in.dtype == torch.float64
        for x, y in zip((a.rho_g, a.rho_d, a.t_s, a.p_in), (b.rho_g, b.rho_d, b.t_s, b.p_in)):
            assert torch.equal(x, y) and torch.isfinite(x).all()
        assert (a.rho_g > 0).all() and (a.rho_d > 0).all() and (a.t_s > 0).all()
    w3 = W.make_workload(3, ncells=4096)
    eps = w3.rho_d / w3.rho_g
    assert abs(float(eps.sum(dim=0)[0]) - 0.01) < 1e-15                      # dust-to-gas ratios sum to 0.01
    assert float(w3.t_s[0].min()) >= 0.9e-4 and float(w3.t_s[-1].max()) <= 1.1  # geometric grid with +-10 % jitter
    w4 = W.make_workload(4, ncells=4096)
    assert float(w4.t_s.min()) >= 1e-6 and float(w4.t_s.max()) <= 1e2
    idx = W.sample_cells(10 ** 6, 1000)
    assert idx[0] == 0 and idx[-1] == 10 ** 6 - 1 and len(torch.unique(idx)) == len(idx)
    assert W.CONFIG_CELLS == {1: 32 ** 3, 2: 128 ** 3, 3: 256 ** 3, 4: 256 ** 3, 5: 2 ** 22}


def test_bench_rank_aggregation_over_gloo_world_size_2(tmp_path):
    """bench.py --gpus N runs replicas (the path does not shard; no data-path collective).  The only
    cross-rank step is the max-over-ranks of the timed region and the sum of the cells processed; cover it with two
    gloo ranks on the CPU."""
    script = tmp_path / "agg.py"
    script.write_text(
        "import sys, json\n"
        f"sys.path.insert(0, {ROOT!r})\n"
        "import torch.distributed as dist\n"
        "import bench\n"
        "dist.init_process_group('gloo')\n"
        "r = dist.get_rank()\n"
        "ms, cells = bench.aggregate_over_ranks(10.0 + 5.0 * r, 1000 * (r + 1))\n"
        "if r == 0: print(json.dumps({'ms': ms, 'cells': cells}))\n"
        "dist.destroy_process_group()\n")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29517", str(script)],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    import json
    res = json.loads(line)
    assert res == {"ms": 15.0, "cells": 3000}
