"""GPU parity for the two read-outs next to the step: the CUDA
monitor and picture, through the C ABI, against oracle/monitor_view.py — bit-exact (integers, bytes)."""
import numpy as np
import pytest

from oracle.monitor_view import monitor_eval, render
from workloads import configs
from workloads.model import SeedRecord

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_14603_b200 as pkg

    pkg.load_library()
    return pkg


def check_monitors(sim, counts, monitors):
    got = sim.monitor_eval(monitors)
    for m, g in zip(monitors, got):
        want = monitor_eval(counts, m["replica"], m["species"], m["threshold"], m["first_row"], m["n_rows"])
        for k in ("first_above", "n_above", "last_state", "max_value", "max_row", "n_switches"):
            assert g[k] == want[k], (m, k, g[k], want[k])
        assert (g["states"] == want["states"]).all(), m


def test_monitor_parity_on_w0_counts_log(gpu):
    """[CFG 0]: 1,000 steps; windows that span several 256-row strides and a ragged tail, thresholds that are
    crossed once (C grows), never, always, and many times (a noisy plateau)."""
    m = configs.w0()
    sim = gpu.Sim(m); sim.seed_population(); sim.step(1000)
    counts = sim.read_counts()
    A, B, Cx = 0, 1, 2
    plateau = int(counts[600:, 0, Cx].mean())
    mons = [dict(replica=0, species=[Cx], threshold=1000, first_row=0, n_rows=1001),
            dict(replica=0, species=[Cx], threshold=plateau, first_row=300, n_rows=701),
            dict(replica=0, species=[A, Cx], threshold=4999, first_row=0, n_rows=1001),      # A + C is conserved = 5000
            dict(replica=0, species=[A, Cx], threshold=5000, first_row=5, n_rows=777),
            dict(replica=0, species=[A, B, Cx, Cx], threshold=9000, first_row=1000, n_rows=1),
            dict(replica=0, species=[B], threshold=4000, first_row=1, n_rows=255)]
    check_monitors(sim, counts, mons)
    got = sim.monitor_eval(mons[:1], with_states=False)[0]
    assert got["n_above"] > 0 and got["n_switches"] == 1 and got["last_state"] == 1      # C passes 1000 once
    assert sim.monitor_eval(mons[2:4])[0]["n_above"] == 1001 and sim.monitor_eval(mons[2:4])[1]["n_above"] == 0


def test_monitor_treatment_mid_run_per_replica(gpu):
    """[CFG 2]-shaped: the inhibitor is added mid-run by a second sim_seed_population call (PAPER.md:7, 64
    'real-time modification of treatment strategies'); per-replica pERK monitors before / after, GPU = oracle."""
    from oracle.binding import Oracle

    m = configs.w2(scale=0.002, n_steps=160)
    names = [s.name for s in m.species]
    inh, perk = names.index("INH"), names.index("pERK")
    recs0 = [r for r in m.seed_records if r.species != inh]
    treat = [SeedRecord(inh, 400, replica=r) for r in (1, 3, 6)]
    sim, orc = gpu.Sim(m), Oracle(m)
    for s in (sim, orc):
        s.seed_population(recs0); s.step(80); s.seed_population(treat, place_seed=77); s.step(80)
    cg, co = sim.read_counts(), orc.read_counts()
    assert (cg == co).all()
    mons = [dict(replica=r, species=[perk], threshold=int(co[80, r, perk]), first_row=f, n_rows=n)
            for r in range(m.n_replicas) for f, n in ((0, 81), (80, 81))]
    check_monitors(sim, co, mons)


def test_monitor_errors(gpu):
    m = configs.w0(n_steps=10)
    sim = gpu.Sim(m); sim.seed_population(); sim.step(10)
    ok = dict(replica=0, species=[2], threshold=1, first_row=0, n_rows=11)
    assert len(sim.monitor_eval([ok])) == 1
    for bad in (dict(ok, n_rows=12), dict(ok, first_row=11, n_rows=1), dict(ok, replica=1), dict(ok, species=[3]),
                dict(ok, n_rows=0), dict(ok, species=[])):
        with pytest.raises(gpu.SimError):
            sim.monitor_eval([bad])


def picture_case(gpu, m, steps, views):
    sim = gpu.Sim(m); sim.seed_population(); sim.step(steps)
    a = sim.read_agents()
    comp = [s.compartment for s in m.species]
    for v in views:
        got = sim.render(**v)
        pal = v.get("palette") or [(255, 165, 0), (255, 255, 0)]
        pal = list(pal) + [(0, 0, 0)] * (len(m.compartments) - len(pal))
        ext = [e for k, e in enumerate(m.extent) if k != v.get("axis", 2)]
        if v.get("axis", 2) != 0 and m.n_replicas > 1:
            ext[0] = min(ext[0], 1 << m.stride_shift)       # one replica tile (the binding's default window)
        want = render(a["x"], a["y"], a["z"], a["species"], comp, m.stride_shift, v.get("replica", 0),
                      v.get("axis", 2), v.get("u0", 0), v.get("v0", 0), v.get("eu", ext[0]), v.get("ev", ext[1]),
                      v.get("width", 256), v.get("height", 256), v.get("gain", 255), pal[:len(m.compartments)])
        assert got.shape == want.shape
        bad = np.nonzero((got != want).any(axis=2))
        assert len(bad[0]) == 0, f"{v}: {len(bad[0])} pixels differ, first {bad[0][0], bad[1][0]}"
        assert (got[:, :, 3] == 255).any()
    return sim


def test_picture_parity_nucleus_and_cytoplasm(gpu):
    """[CFG 3] scaled: shell + nucleus, so both palette entries are used; all three projection axes, a
    zoomed window with a ragged size, a low gain that does not saturate."""
    m = configs.w3(scale=0.004, n_steps=20)
    R = m.extent[1]
    picture_case(gpu, m, 20, [
        dict(axis=2, width=64, height=64, gain=255),
        dict(axis=0, width=33, height=17, gain=40),
        dict(axis=1, u0=R // 4, v0=R // 3, eu=R // 2 + 3, ev=R // 3 + 1, width=50, height=21, gain=9),
        dict(axis=2, width=8, height=8, gain=1, palette=[(255, 0, 0), (0, 0, 255)])])


def test_picture_parity_replicas_and_dense_cube(gpu):
    """[CFG 2] scaled: one replica tile is drawn, the others are ignored; [CFG 0]: 10 k agents in few pixels,
    so the per-pixel counts saturate and many agents share a (pixel, compartment) counter."""
    m = configs.w2(scale=0.002, n_steps=5)
    picture_case(gpu, m, 5, [dict(replica=7, axis=2, width=40, height=40, gain=128),
                             dict(replica=0, axis=1, width=24, height=31, gain=255)])
    sim = picture_case(gpu, configs.w0(n_steps=30), 30, [dict(axis=2, width=4, height=4, gain=1),
                                                          dict(axis=0, width=120, height=75, gain=200)])
    with pytest.raises(gpu.SimError):
        sim.render(width=4096, height=4096)            # more pixels than the scratch of a 10 k-agent handle
    with pytest.raises(gpu.SimError):
        sim.render(axis=3)


def test_compiled_physical_model_parity(gpu):
    """N2: a model given in physical units (molecular weights, concentrations, k_cat, volume) is compiled to
    integer tables by workloads/compiler.py and stepped on both sides: bit-exact state and counts."""
    from oracle.binding import Oracle
    from test_model_compiler import toy
    from workloads import compiler

    m = compiler.compile_model(toy(), cell_size=64)
    sim, orc = gpu.Sim(m), Oracle(m)
    for s in (sim, orc):
        s.seed_population(); s.step(50)
    a, b = sim.read_agents(), orc.read_agents()
    for k in ("id", "species", "x", "y", "z"):
        assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(sim.read_counts(), orc.read_counts())


def test_compiled_compartmentalised_model_parity(gpu):
    """N2 with the paper's localisation / translocation / expressor / degradation fields: a
    [CFG 3]-shaped model written in physical units, compiled, and stepped on both sides: bit-exact state and counts,
    membrane crossings, expression and degradation included."""
    from oracle.binding import Oracle
    from test_model_compiler import nuclear_spec
    from workloads import compiler

    m = compiler.compile_model(nuclear_spec(n_steps=400), cell_size=512)
    sim, orc = gpu.Sim(m), Oracle(m)
    for s in (sim, orc):
        s.seed_population()
    for chunk in range(4):
        sim.step(100); orc.step(100)
        a, b = sim.read_agents(), orc.read_agents()
        for k in ("id", "species", "x", "y", "z"):
            assert np.array_equal(a[k], b[k]), (chunk, k)
    c = orc.read_counts()
    assert np.array_equal(sim.read_counts(), c) and sim.read_checksum() == orc.read_checksum()
    ix = {s.name: i for i, s in enumerate(m.species)}
    assert c[:, 0, ix["mRNA_n"]].max() > 0 and c[:, 0, ix["pS"]].max() > 0        # expression and the cascade happened


def test_derived_concentration_curves_and_perk_fraction(gpu):
    """SURVEY 8(a) a11 / [NS]: the only floating-point outputs are derived on the host in double from the integer
    counts — concentration curves c(t) = n(t) / (N_A V) and [CFG 2]'s steady-state pERK fraction (reading S19) — and
    are held to a relative tolerance of 1e-6 against the same derivation from the oracle's counts."""
    from oracle.binding import Oracle
    from workloads import model as wm

    m = configs.w2(scale=0.002, n_steps=120)
    sim, orc = gpu.Sim(m), Oracle(m)
    for s in (sim, orc):
        s.seed_population(); s.step(120)
    cg, co = sim.read_counts(), orc.read_counts()
    curves_g = wm.concentration_molar(cg, m.volume_um3)          # the product-side derivation, on the CUDA path's counts
    assert curves_g.dtype == np.float64 and curves_g.shape == cg.shape
    # expected curve: the definition c = n / (N_A V) written out here (CODATA N_A; volume of the 5 um sphere scaled by
    # the model's count scale, in litres), applied to the ORACLE's counts -- not the function under test
    R_um = m.compartments[0].r_out / 10_000.0
    litres = 4.0 / 3.0 * np.pi * R_um ** 3 * 1e-15
    curves_o = co.astype(np.float64) / (6.02214076e23 * litres)
    nz = curves_o != 0
    assert nz.any()
    assert np.all(np.abs(curves_g[nz] - curves_o[nz]) <= 1e-6 * np.abs(curves_o[nz])) and np.all(curves_g[~nz] == 0)
    names = [s.name for s in m.species]
    perk, erk_like = names.index("pERK"), [names.index(n) for n in ("ERK", "pERK", "pMEK:ERK", "P:pERK")]
    frac_g = cg[-50:, :, perk].mean(axis=0) / cg[0][:, erk_like].sum(axis=1)
    frac_o = co[-50:, :, perk].mean(axis=0) / co[0][:, erk_like].sum(axis=1)
    assert np.allclose(frac_g, frac_o, rtol=1e-6, atol=0.0)
    # closed form: one molecule in the replica volume
    one = wm.concentration_molar(np.array([1]), m.volume_um3)[0]
    assert abs(one * wm.N_AVOGADRO * m.volume_um3 * 1e-15 - 1.0) < 1e-12
