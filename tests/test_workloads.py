"""Pins for the input side (workloads/): tables, thresholds, unit conversions.  CPU only."""
import os

import numpy as np
import pytest

from workloads import configs, model

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            yield line.split()


def test_thresholds_worked_values():
    for p, thr in _rows("thresholds.txt"):
        assert model.prob_to_thr(float(p)) == int(thr)


def test_gauss_table_worked_values_and_invariants():
    for D, dt, lo, hi, ssq in _rows("gauss_table_values.txt"):
        sigma = model.sigma_units(float(D), float(dt))
        t = model.gaussian_table(sigma, 12).astype(np.int64)
        assert t[0] == int(lo) and t[-1] == int(hi)
        if int(ssq) >= 0:
            assert int((t * t).sum()) == int(ssq)
        assert (t == -t[::-1]).all()            # antisymmetric
        assert (np.diff(t) >= 0).all()          # monotone
        assert t.sum() == 0
        assert abs((t * t).mean() / float(sigma) ** 2 - 1.0) < 2e-3
    t = model.gaussian_table(model.sigma_units(10.0, 1.0), 12)
    assert t[1] == -151 and t[1023] == -30 and t[2047] == 0 and t[2048] == 0


def test_sigma_units():
    # sigma = sqrt(2 D dt): D = 10 um^2/s, dt = 1 us -> 4.4721 nm = 44.721 units
    assert abs(model.sigma_units(10.0, 1.0) - 44.7214) < 1e-3
    assert abs(model.sigma_units(4.0, 10.0) - 89.4427) < 1e-3
    assert abs(model.sigma_units(50.0, 1.0) - 100.0) < 1e-9


def test_paper_table1_counts_closed_form():
    """PAPER.md:84-97 + :109 — count = c * N_A * V; cube edges match the printed ~14.4 / ~6.7 um."""
    conc = {}
    vols = []
    for row in _rows("paper_table1.txt"):
        if row[0] == "volume":
            vols.append((float(row[1]), float(row[2])))
        else:
            conc[row[0]] = float(row[1])
    for v_l, edge_um in vols:
        edge = (v_l * 1e15) ** (1.0 / 3.0)
        assert abs(edge - edge_um) < 0.05
    counts = {k: int(round(c * model.N_AVOGADRO * 3e-12)) for k, c in conc.items()}
    assert counts["BRAF"] == 5420 and counts["MEK"] == 2167971
    assert sum(counts.values()) == 4556124
    # and the inverse used for the derived float curves (rel. tol 1e-6, north_star)
    back = model.concentration_molar(np.array([counts["MEK"]]), 3e-12 * 1e15)[0]
    assert abs(back / 1.2e-6 - 1.0) < 1e-6


def test_config_sizes():
    assert configs.w0().n_agents0 == 10_000
    assert configs.w1().n_agents0 == 1_050_000
    assert configs.w2().n_agents0 == 8_854_860
    m3 = configs.w3()
    assert 300_000 <= m3.n_agents0 <= 500_000
    for n, L in configs.W4_EDGES.items():
        dens = n / (L / 10_000.0) ** 3
        assert abs(dens - 30_000.0) < 1.0               # reading S21
    # sphere volume 523.6 um^3; 315,000 molecules ~ 999 nM [CFG 2]
    v = configs.w1().volume_um3
    assert abs(v - 523.6) < 0.01
    nM = model.concentration_molar(np.array([315_000]), v)[0] * 1e9
    assert abs(nM - 999.0) < 1.0


@pytest.mark.parametrize("f", [configs.w0, configs.w1, configs.w2, configs.w3, configs.w4])
def test_table_bounds(f):
    m = f()
    assert m.tables.dtype == np.int16 and m.tables.shape[1] == 1 << m.table_bits
    assert (m.tables[0] == 0).all()
    rmax = max(int(np.sqrt(r.r2)) for r in m.reactions)
    assert m.cell_size >= rmax
