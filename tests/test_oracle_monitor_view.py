"""CPU pins for oracle/monitor_view.py (N3 monitor, N4 headless picture)."""
import os

import numpy as np

from oracle.monitor_view import NONE, monitor_eval, render

GOLD = os.path.join(os.path.dirname(__file__), "golden", "monitor_worked_example.txt")
ORANGE, YELLOW = (255, 165, 0), (255, 255, 0)      # PAPER.md:68 (Fig. 1): cytoplasm orange, nucleus yellow


def _gold():
    d = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if ":" in line:
            k, v = line.split(":")
            d[k.strip()] = [int(w) for w in v.split()]
    return d


def test_monitor_hand_worked_example():
    g = _gold()
    counts = np.zeros((7, 1, 3), dtype=np.uint32)
    counts[:, 0, 0] = g["a"]; counts[:, 0, 2] = g["b"]; counts[:, 0, 1] = 1000   # species 1 is not monitored
    r = monitor_eval(counts, 0, [0, 2], g["threshold"][0], g["first_row"][0], g["n_rows"][0])
    for k in ("first_above", "n_above", "last_state", "max_value", "max_row", "n_switches"):
        assert r[k] == g[k][0], k
    assert r["states"].tolist() == [0, 1, 1, 0, 1, 0]


def test_monitor_closed_forms_on_a_ramp_and_never_above():
    T = 50
    counts = np.zeros((T, 2, 1), dtype=np.uint32)
    counts[:, 1, 0] = np.arange(T)                          # value(t) = t in replica 1, 0 in replica 0
    r = monitor_eval(counts, 1, [0], 20, 5, 40)             # rows 5..44, above iff t > 20
    assert (r["first_above"], r["n_above"], r["last_state"], r["n_switches"]) == (21, 24, 1, 1)
    assert (r["max_value"], r["max_row"]) == (44, 44)
    r = monitor_eval(counts, 0, [0], 0, 0, T)               # strict inequality: 0 > 0 is false
    assert (r["first_above"], r["n_above"], r["last_state"], r["n_switches"], r["max_value"], r["max_row"]) == \
        (NONE, 0, 0, 0, 0, 0)


def test_monitor_against_vectorised_recomputation():
    rng = np.random.default_rng(3)
    counts = rng.integers(0, 50, size=(300, 3, 5), dtype=np.uint32)
    for rep, sp, thr, f, n in [(0, [1], 25, 0, 300), (2, [0, 3, 4], 70, 17, 200), (1, [2, 2], 40, 299, 1)]:
        r = monitor_eval(counts, rep, sp, thr, f, n)
        v = counts[f:f + n, rep][:, sp].astype(np.int64).sum(axis=1)
        a = v > thr
        assert r["n_above"] == int(a.sum())
        assert r["first_above"] == (f + int(np.argmax(a)) if a.any() else NONE)
        assert r["last_state"] == int(a[-1])
        assert (r["max_value"], r["max_row"]) == (int(v.max()), f + int(np.argmax(v)))   # argmax = first maximum
        assert r["n_switches"] == int((a[1:] != a[:-1]).sum())
        assert (r["states"] == a).all()


def _view(**kw):
    d = dict(comp_of_species=[0, 1], stride_shift=17, replica=0, axis=2, u0=0, v0=0, eu=100, ev=100, width=10,
             height=10, gain=255, palette=[ORANGE, YELLOW])
    d.update(kw)
    return d


def test_render_single_agents_land_in_the_right_pixel_with_the_compartment_colour():
    x = np.array([5, 95, 50]); y = np.array([5, 15, 99]); z = np.array([7, 7, 7]); s = np.array([0, 1, 0])
    img = render(x, y, z, s, **_view())
    assert img[0][0].tolist() == [255, 165, 0, 255]          # cytoplasm species, pixel (u 0, v 0)
    assert img[1][9].tolist() == [255, 255, 0, 255]          # nucleus species, pixel (u 9, v 1)
    assert img[9][5].tolist() == [255, 165, 0, 255]
    assert int((img[:, :, 3] == 255).sum()) == 3 and int(img[:, :, :3][img[:, :, 3] == 0].sum()) == 0
    # projecting along x instead: (u, v) = (y, z)
    img = render(x, y, z, s, **_view(axis=0))
    assert img[0][0].tolist() == [255, 165, 0, 255] and img[0][1].tolist() == [255, 255, 0, 255]
    assert img[0][9].tolist() == [255, 165, 0, 255]


def test_render_gain_saturation_and_mixing():
    x = np.array([1, 2, 3, 4]); y = np.array([1, 1, 1, 1]); z = np.zeros(4, dtype=int)
    img = render(x, y, z, np.array([0, 0, 0xFFFF, 0]), **_view(gain=64))       # DEAD agents are not drawn
    assert img[0][0].tolist() == [255 * 192 // 255, 165 * 192 // 255, 0, 255]  # three live agents: intensity 192
    img = render(x, y, z, np.array([0, 0, 1, 1]), **_view(gain=255))
    assert img[0][0].tolist() == [255, 255, 0, 255]          # orange + yellow, saturating per channel
    img = render(x, y, z, np.array([0, 0, 1, 1]), **_view(gain=64, palette=[(200, 0, 0), (0, 0, 90)]))
    assert img[0][0].tolist() == [200 * 128 // 255, 0, 90 * 128 // 255, 255]


def test_render_window_replica_and_count_conservation():
    rng = np.random.default_rng(5)
    n = 4000
    rep = rng.integers(0, 2, n)
    x = rng.integers(0, 300, n) + (rep << 17); y = rng.integers(0, 300, n); z = rng.integers(0, 300, n)
    s = rng.integers(0, 2, n)
    v = _view(replica=1, axis=1, u0=50, v0=20, eu=200, ev=240, width=16, height=12, gain=1,
              palette=[(255, 0, 0), (0, 255, 0)])
    img = render(x, y, z, s, **v)
    lx = x - (rep << 17)
    inside = (rep == 1) & (lx >= 50) & (lx < 250) & (z >= 20) & (z < 260)
    # gain 1 and fewer than 255 agents per pixel: red = cytoplasm count, green = nucleus count
    assert int(img[:, :, 0].sum()) == int((inside & (s == 0)).sum())
    assert int(img[:, :, 1].sum()) == int((inside & (s == 1)).sum())
    h, _, _ = np.histogram2d(z[inside & (s == 0)], lx[inside & (s == 0)], bins=[12, 16], range=[[20, 260], [50, 250]])
    assert (img[:, :, 0] == h.astype(np.int64)).all()       # 240/12 and 200/16: bin edges fall on integers
