"""Host-side logic that needs no GPU: the Nystrom-collapsed tableau constants the kernels carry
(re-derived here in exact rational arithmetic from the Dormand-Prince tableau of ref [22],
PAPER.md:106), the input recipes of BASELINE.json's configs, index sharding, and the multi-process
summary reduction (gloo, world_size 2)."""
import os
import re
import socket
from fractions import Fraction as F

import numpy as np
import pytest

import ia_inputs as I
from paper_2509_15117_b200 import dist as D

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# Dormand & Prince 1980, RK5(4)7M -- typed here from the published tableau (independent of oracle/ and csrc/)
C_ = [F(0), F(1, 5), F(3, 10), F(4, 5), F(8, 9), F(1), F(1)]
A_ = [[], [F(1, 5)], [F(3, 40), F(9, 40)], [F(44, 45), F(-56, 15), F(32, 9)],
      [F(19372, 6561), F(-25360, 2187), F(64448, 6561), F(-212, 729)],
      [F(9017, 3168), F(-355, 33), F(46732, 5247), F(49, 176), F(-5103, 18656)],
      [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84)]]
BH_ = [F(5179, 57600), F(0), F(7571, 16695), F(393, 640), F(-92097, 339200), F(187, 2100), F(1, 40)]


def amat():
    a = [[F(0)] * 7 for _ in range(7)]
    for s, row in enumerate(A_):
        for l, v in enumerate(row):
            a[s][l] = v
    return a


def device_macros():
    """IA_* rational constants of csrc/ia_dev.cuh as exact Fractions."""
    text = open(os.path.join(ROOT, "paper_2509_15117_b200", "csrc", "ia_dev.cuh")).read()
    out = {}
    for name, num, den in re.findall(r"#define\s+(IA_[A-Z]+\d+)\s+\((-?\d+)\.0\s*/\s*(\d+)\.0\)", text):
        out[name] = F(int(num), int(den))
    return out


def test_collapsed_tableau_constants_are_the_exact_products():
    """abar = a.a, ebar = (b - bhat).a, E = b - bhat: the second-order form the kernels integrate is
    algebraically the first-order DP5(4) step for dx/dt = v, dv/dt = A(t, x)."""
    a = amat()
    b = a[6]
    m = device_macros()
    assert len(m) == 34
    abar = [[sum(a[s][j] * a[j][l] for j in range(7)) for l in range(7)] for s in range(7)]
    E = [b[l] - BH_[l] for l in range(7)]
    ebar = [sum(E[j] * a[j][l] for j in range(7)) for l in range(7)]
    seen = set()
    for s in range(2, 7):
        for l in range(7):
            key = f"IA_AB{s + 1}{l + 1}"
            if abar[s][l] != 0:
                assert m[key] == abar[s][l], key
                seen.add(key)
            else:
                assert key not in m
        assert sum(abar[s]) == C_[s] ** 2 / 2                  # row sums of a.a (order-2 condition per stage)
    for l in range(7):
        for pre, vec in (("IA_B", b), ("IA_E", E), ("IA_EB", ebar)):
            key = f"{pre}{l + 1}"
            if vec[l] != 0:
                assert m[key] == vec[l], key
                seen.add(key)
            else:
                assert key not in m, key
    for s in range(1, 5):
        assert m[f"IA_C{s + 1}"] == C_[s]
    assert sum(E) == 0 and sum(ebar) == sum(E[j] * C_[j] for j in range(7))
    assert seen | {f"IA_C{k}" for k in (2, 3, 4, 5)} == set(m)   # no stray constant


def test_device_cosine_polynomial_is_accurate_to_half_an_ulp():
    """The degree-8 polynomial in z = r^2 that csrc/ia_dev.cuh evaluates for cos(r), |r| <= pi/2: its double
    literals, evaluated exactly (rationals), stay within 6e-17 of a 50-digit cosine over the whole range
    and beyond the rounding slack of the argument reduction (1.0001 pi/2)."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 50
    text = open(os.path.join(ROOT, "paper_2509_15117_b200", "csrc", "ia_dev.cuh")).read()
    lit = dict(re.findall(r"#define\s+IA_COS_C(\d)\s+\(([-+0-9.e]+)\)", text))
    assert sorted(lit) == [str(k) for k in range(9)]
    c = [F(float(lit[str(k)])) for k in range(9)]            # the doubles the compiler sees, exactly
    worst = 0.0
    for i in range(0, 4001):
        r = mp.mpf("1.0001") * mp.pi / 2 * i / 4000
        z = F(float(r)) ** 2                                   # a double r, squared exactly
        p = sum(ck * z ** k for k, ck in enumerate(c))
        err = abs(mp.mpf(p.numerator) / mp.mpf(p.denominator) - mp.cos(mp.mpf(float(r))))
        worst = max(worst, float(err))
    assert worst < 6e-17, worst
    assert c[0] == 1


def test_observables_formatting_on_constructed_records():
    """observables.py is array arithmetic on records: back-scattering gives chi = pi and q = 2 m v, a 90 degree
    deflection chi = pi/2 and q = sqrt(2) m v, forward flight zero; the survival curve of a known histogram and the
    slope of an exact power law come back."""
    import paper_2509_15117_b200 as P
    from paper_2509_15117_b200 import observables as Ob
    v, m = 1.0e-8, 158425.415
    ic = np.zeros((4, 14)); ic[:, 9] = -v
    rec = np.zeros(4, dtype=P.RECORD_DTYPE)
    rec["va_f"] = [[v, 0, 0], [0, v, 0], [-v, 0, 0], [0, 0, -2 * v]]
    rec["n_coll"] = [1, 100, 1, 3]
    chi, q = Ob.scattering(rec, ic, m)
    assert np.allclose(chi, [np.pi, np.pi / 2, 0.0, np.pi / 2], atol=1e-15)
    assert np.allclose(q, [2 * m * v, np.sqrt(2) * m * v, 0.0, np.sqrt(5) * m * v], rtol=1e-15)
    mp = Ob.maps(rec, ic, m, 2, 2)
    assert mp["log10_bounces"].tolist() == [[0.0, 2.0], [0.0, np.log10(3.0)]]
    assert mp["complex"].tolist() == [[False, True], [False, True]]
    assert mp["momentum_transfer_clipped"].max() <= Ob.Q_CLIP_AU
    T = 2.0e10
    summ = np.zeros(1, dtype=P.SUMMARY_DTYPE)[0]
    h = np.zeros(P.IA_LIFE_BINS, dtype=np.uint64); h[8] = 2; h[12] = 1; h[16] = 1      # q in [1,2^.25), [2,..), [4,..)
    summ["hist_tlife"] = h
    t, S = Ob.survival_curve(summ, T)
    assert len(t) == P.IA_LIFE_BINS - 1 and t[7] == T and t[11] == 2 * T
    assert S[6] == 1.0 and S[7] == 1.0 and S[8] == 0.5 and S[11] == 0.5 and S[12] == 0.25 and S[16] == 0.0
    tt = T * 2.0 ** np.arange(0, 10)
    assert abs(Ob.power_law_exponent(tt, 3.0 * tt ** -1.5, t_min=2 * T) + 1.5) < 1e-12


def test_config_recipes_match_baseline_json():
    import json
    cfg = json.load(open(os.path.join(ROOT, "BASELINE.json")))["configs"]
    c0, c1 = I.config0(), I.config1()
    assert "32" in cfg[0] and c0.launch.n == 1024 and c0.params.t_max_rf == 2000 and c0.launch.E_min_uK == 10.0
    assert c0.params.m_atom_u == 7.016 and c0.params.alpha_au == 164.1 and c0.params.m_ion_u == 173.94
    assert c0.params.q == (0.1, -0.1, 0.0) and c0.params.a == (-0.0005, -0.0005, 0.001)
    assert c0.params.rtol == 1e-10 and c0.params.atol == 1e-12 and c0.params.r0_a0 == 5000.0
    assert abs(c0.params.omega_rf_au - 3.0396596921148e-10) < 1e-22
    assert c1.launch.n == 262144 and c1.params.m_atom_u == 86.909 and c1.params.alpha_au == 319.2
    assert c1.launch.E_min_uK == 1.5 and c1.params.t_max_rf == 1e4 and c1.launch.phase_mode == 0
    c2 = I.config2()
    assert len(c2) == 25 and all(c.launch.n == 2 ** 20 and c.launch.domain == 0 and c.launch.phase_mode == 1 for c in c2)
    assert len({c.launch.cell for c in c2}) == 25 and len({c.launch.seed for c in c2}) == 1
    assert sorted({c.params.alpha_au for c in c2}) == [162.7, 164.1, 290.0, 319.2, 401.0]
    c3 = I.config3()
    assert len(c3) == 20 and all(c.launch.n == 2 ** 22 and c.launch.E_min_uK == 3.0 for c in c3)
    assert sorted({c.params.De_K for c in c3}) == [0.1, 1.0, 10.0, 100.0]
    assert all(c.params.q[0] == -c.params.q[1] and c.params.q[2] == 0.0 for c in c3)
    c4 = I.config4()
    assert len(c4) == 18 and sum(c.launch.n for c in c4) == 300_000_000 and c4[-1].launch.n == 14_787_328
    assert all(c.launch.domain == 1 and (c.launch.E_min_uK, c.launch.E_max_uK) == (1.0, 100.0) for c in c4)
    firsts = [c.launch.first_index for c in c4]
    assert firsts == [k * 2 ** 24 for k in range(18)]                        # one Philox stream, advancing


def test_thermal_cells_and_sweep_lists():
    """The thermal bars: ion at 10 uK, full sphere, uniform phase, one Philox cell per bar,
    none shared with configs 2-4; sweep.cells_of lists every config with its own sizes and --scale shrinks them."""
    from paper_2509_15117_b200 import sweep
    bars = [I.thermal(sp, T, De) for De in (1.0, 100.0) for sp in I.SPECIES_ORDER for T in I.THERMAL_T_UK]
    assert len({b.launch.cell for b in bars}) == 50
    used = {c.launch.cell for c in I.config2(8) + I.config3(8) + I.config4(64, 64)}
    assert not used & {b.launch.cell for b in bars}
    for b in bars:
        L = b.launch
        assert L.mode == I.MODE_THERMAL and L.domain == 1 and L.phase_mode == 1 and L.T_ion_uK == 10.0
        assert b.params.q[0] != 0.0 and b.params.r0_a0 == 5000.0
    assert [len(sweep.cells_of(k, 1.0)) for k in ("0", "2", "3", "4", "thermal")] == [1, 25, 20, 18, 50]
    assert sum(c.launch.n for c in sweep.cells_of("4", 1.0)) == 300_000_000
    assert {c.launch.n for c in sweep.cells_of("2", 1.0 / 1024)} == {1024}
    assert sweep.cells_of("1", 1.0)[0].launch.n == 512 * 512


def test_subgrid_and_shards_tile_the_index_range():
    idx = I.subgrid_indices(512, 8)
    assert len(idx) == 4096 and len(set(idx.tolist())) == 4096 and idx.max() < 512 * 512
    for n, world in ((262144, 8), (1000, 7), (5, 8), (0, 3)):
        spans = [D.shard_range(n, r, world) for r in range(world)]
        assert spans[0][0] == 0 and sum(c for _, c in spans) == n
        for (f0, c0), (f1, _) in zip(spans, spans[1:]):
            assert f0 + c0 == f1
        assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
    l = I.config4(n_total=1000, batch=1000)[0].launch
    parts = [D.shard_launch(l, r, 3) for r in range(3)]
    assert [p.first_index for p in parts] == [0, 334, 667] and [p.n for p in parts] == [334, 333, 333]
    with pytest.raises(ValueError):
        D.shard_range(10, 3, 3)


def _summary(seed):
    import paper_2509_15117_b200 as P
    rng = np.random.default_rng(seed)
    s = np.zeros(1, dtype=P.SUMMARY_DTYPE)[0]
    s["n_done"] = rng.integers(1, 1 << 40)
    s["n_status"] = rng.integers(0, 1 << 30, 5)
    s["n_complex"] = rng.integers(0, 1 << 30)
    s["steps_acc"], s["steps_rej"], s["steps_loc"] = rng.integers(0, 1 << 50, 3)
    s["sum_ke"], s["sum_ke2"] = rng.random(2)
    s["hist_ncoll"] = rng.integers(0, 1 << 30, 32)
    return s


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    tot = D.all_reduce_summary(_summary(100 + rank))
    tmax = D.all_reduce_max(1.5 + rank)
    first, count = D.shard_range(1001, rank, world)
    dist.destroy_process_group()
    q.put((rank, tot, tmax, first, count))


def test_summary_reduction_over_two_gloo_ranks():
    """N > 1 path (no data-path collective): index-range shards + one sum of the summaries + max of times."""
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in procs], key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    a, b = _summary(100), _summary(101)
    for rank, tot, tmax, first, count in res:
        assert tmax == 2.5
        assert tot["n_done"] == int(a["n_done"]) + int(b["n_done"])
        assert tot["n_status"] == [int(x) + int(y) for x, y in zip(a["n_status"], b["n_status"])]
        assert tot["hist_ncoll"] == [int(x) + int(y) for x, y in zip(a["hist_ncoll"], b["hist_ncoll"])]
        assert tot["steps_acc"] == int(a["steps_acc"]) + int(b["steps_acc"])
        assert abs(tot["sum_ke"] - (a["sum_ke"] + b["sum_ke"])) < 1e-15
    assert (res[0][3], res[0][4], res[1][3], res[1][4]) == (0, 501, 501, 500)


def test_fig4_cells_and_summary_sums():
    """ia_inputs.fig4: r0 = 20 000 a0, D_e = 1 K, octant directions, random or fixed phase, a Philox cell of
    its own; sweep lists the six cells of profiles/r02_summary.md section 8; dist.sum_summaries adds field by field."""
    import paper_2509_15117_b200 as P
    from paper_2509_15117_b200 import sweep
    c = I.fig4("Rb87", 10.0, n=100)
    assert c.params.r0_a0 == 20000.0 and c.params.De_K == 1.0 and c.params.m_atom_u == I.ATOMS["Rb87"]["m_u"]
    assert c.launch.mode == I.MODE_PHILOX and c.launch.domain == 0 and c.launch.phase_mode == 1
    assert c.launch.E_min_uK == c.launch.E_max_uK == 10.0
    f = I.fig4("Rb87", 10.0, n=100, phase_mode=0, phase0=1.25)
    assert f.launch.phase_mode == 0 and f.launch.phase0 == 1.25 and f.launch.cell == c.launch.cell and f.name != c.name
    used = {x.launch.cell for x in I.config2(8) + I.config3(8) + I.config4(64, 64)} | \
           {I.thermal(sp, T, De).launch.cell for De in (1.0, 100.0) for sp in I.SPECIES_ORDER for T in I.THERMAL_T_UK}
    assert not used & {I.fig4(sp).launch.cell for sp in I.SPECIES_ORDER}
    cells = sweep.cells_of("fig4", 1.0)
    assert len(cells) == 6 and sum(x.launch.phase_mode == 0 for x in cells) == 2
    arr = np.zeros(3, dtype=P.SUMMARY_DTYPE)
    arr["n_done"] = [1, 2, 3]
    arr["hist_ncoll"][:, 1] = [5, 6, 7]
    arr["steps_kernel"] = [10, 20, 30]
    arr["sum_ke"] = [0.5, 0.25, 0.125]
    tot = D.sum_summaries(arr)
    assert int(tot["n_done"]) == 6 and int(tot["hist_ncoll"][1]) == 18 and int(tot["steps_kernel"]) == 60
    assert float(tot["sum_ke"]) == 0.875
    assert "steps_kernel" in D._SUM_FIELDS


def test_persistent_kernels_use_no_local_memory():
    """BASELINE.json north_star: register spills must be zero.  Checked on the built library itself: the SASS of the
    two persistent kernels holds no LDL / STL at all (no stack frame, no spill), and the step loop is where the
    histogram tool says it is (an FP64-dominated loop with seven reciprocals)."""
    import shutil
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not on PATH")
    import paper_2509_15117_b200 as P
    import sass_histogram as H          # tests/sass_histogram.py
    P.load()
    for kernel, fp64_min in (("bulk", 550), ("coop", 280)):
        ins = H.instructions(kernel)
        assert len(ins) > 1000
        ops = [t.split()[0].split(".")[0] for _, t in ins]
        assert "LDL" not in ops and "STL" not in ops
        lo, hi, body = H.step_loop(ins)
        n64 = sum(t.split()[0].split(".")[0] in ("DFMA", "DMUL", "DADD", "DSETP") for t in body)
        assert n64 >= fp64_min and n64 > 0.4 * len(body)
        assert sum(t.startswith("MUFU.RCP64H") for t in body) >= 7
