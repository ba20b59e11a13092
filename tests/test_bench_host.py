"""Host-side pieces of bench.py that run without a GPU."""
import importlib.util
import os

import numpy as np

from oracle import nf_oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_sweep_residual_operator_equals_oracle():
    """bench.py --sweep evaluates ||b - A p|| in fp64 with its own plain NumPy operator: same as the oracle's."""
    b = _bench()
    rng = np.random.default_rng(0)
    p = rng.standard_normal((5, 6, 7))
    au, av, aw = rng.uniform(0, 1, (5, 6, 8)), rng.uniform(0, 1, (5, 7, 7)), rng.uniform(0, 1, (6, 6, 7))
    assert np.max(np.abs(b._apply_A_fp64(p, au, av, aw, 3.0) - orc.apply_A(p, [au, av, aw], 3.0))) <= 1e-13


def test_reference_arm_line_has_contract_keys(capsys):
    """--impl reference (the oracle, timed) prints one JSON line with the contract's keys."""
    import json
    import types
    b = _bench()
    b._oracle_case = lambda n: _small_case()  # (a 12^3 sample keeps the CPU suite fast)
    args = types.SimpleNamespace(steps=1, warmup=0, cpu_n=0, cpu_n_forced=False)
    b.run_reference(args)
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
              "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in line
    assert line["impl"] == "reference" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle"


def _small_case():
    from paper_2405_14903_b200 import workloads as wl
    P = wl.config4_params(12)
    U = wl.config4_initial_velocity(P)
    phi, us = wl.config4_solid(P, 1)
    rng = np.random.default_rng(77)
    gin = [rng.standard_normal(a.shape).astype(np.float32) for a in U]
    bc = orc.BC(P["bc_types"], P["bc_values"])
    return P, U, orc.face_weights(phi, bc), us, gin, bc


def test_coarse_kernel_bytes_follow_the_sweep_counts():
    """bench.coarse_bytes_per_fine_cell: the V(1,1) figure is the 41/7 B per fine cell of DESIGN.md 8.1 (41 B per cell of
    a level, levels of 1/8 + 1/64 + ... of the fine cells); every further sweep adds four half sweeps of 13 B per cell
    and, once, the 4 B of the right-hand side that the general residual reads."""
    import bench
    assert abs(bench.coarse_bytes_per_fine_cell(1, 1) - 41.0 / 7.0) < 1e-12
    assert abs(bench.coarse_bytes_per_fine_cell(2, 1) - (97.0 / 8.0 + 41.0 / 56.0)) < 1e-12
    assert abs(bench.coarse_bytes_per_fine_cell(2, 3) - (97.0 / 8.0 + 149.0 / 56.0)) < 1e-12
    assert abs(bench.coarse_bytes_per_fine_cell(1, 2) - (41.0 / 8.0 + 97.0 / 56.0)) < 1e-12
