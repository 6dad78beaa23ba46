"""Oracle for the two read-out operations next to the step.  TEST INFRASTRUCTURE:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this; it shares nothing
with the CUDA path.  Plain Python / numpy, integers only, written from DESIGN.md §10 (readings S24, S25).

* monitor_eval — threshold monitor over a window of the per-step counts log.  PAPER.md:58 ("designate specific
  molecular species for continuous monitoring ... concentration thresholds within specified time windows"),
  PAPER.md:72 (Fig. 2: the status switches between *Cancerous* and *Normal* as the monitored species crosses
  the preset threshold).
* render — headless stand-in for the 3-D viewer, PAPER.md:64, 68 (Fig. 1: "highlighting molecules by
  compartment (orange for cytoplasm, yellow for nucleus)"): an orthographic point splat of the agents into an
  RGBA image, coloured by the compartment of their species.

Pins: tests/test_oracle_monitor_view.py (hand-worked fixtures under tests/golden/, closed forms, brute force).
"""
import numpy as np

NONE = 0xFFFFFFFF


def monitor_eval(counts, replica, species, threshold, first_row, n_rows):
    """counts[T][R][S] (uint32).  value(t) = sum over `species` of counts[t][replica][s];
    above(t) = value(t) > threshold.  Returns the S24 summary over rows first_row .. first_row+n_rows-1
    and the per-row states."""
    states = []
    first_above, n_above, max_value, max_row, n_switches = NONE, 0, 0, NONE, 0
    for t in range(first_row, first_row + n_rows):
        value = 0
        for s in species:
            value += int(counts[t][replica][s])
        above = 1 if value > threshold else 0
        if above:
            n_above += 1
            if first_above == NONE:
                first_above = t
        if max_row == NONE or value > max_value:
            max_value, max_row = value, t
        if states and states[-1] != above:
            n_switches += 1
        states.append(above)
    return {"first_above": first_above, "n_above": n_above, "last_state": states[-1] if states else 0,
            "max_value": max_value, "max_row": max_row, "n_switches": n_switches,
            "states": np.array(states, dtype=np.uint8)}


def render(x, y, z, species, comp_of_species, stride_shift, replica, axis, u0, v0, eu, ev, width, height,
           gain, palette):
    """S25.  The image plane holds the two axes other than `axis`, in increasing order (u, v); an agent of
    `replica` at local coordinates (x minus the replica tile base) with u0 <= u < u0+eu and v0 <= v < v0+ev
    falls into pixel (pu, pv) = ((u-u0)*width // eu, (v-v0)*height // ev).  Per pixel and compartment c the
    agents are counted (n_c); colour channel k = min(255, sum_c palette[c][k] * min(n_c*gain, 255) // 255),
    alpha = 255 where any agent fell, else 0.  Returns uint8[height][width][4], row 0 = smallest v."""
    n_comp = len(palette)
    cnt = np.zeros((height, width, n_comp), dtype=np.int64)
    for i in range(len(x)):
        s = int(species[i])
        if s == 0xFFFF:
            continue
        xi = int(x[i])
        if (xi >> stride_shift) != replica:
            continue
        p = (xi - (replica << stride_shift), int(y[i]), int(z[i]))
        uv = [p[a] for a in range(3) if a != axis]
        du, dv = uv[0] - u0, uv[1] - v0
        if du < 0 or du >= eu or dv < 0 or dv >= ev:
            continue
        cnt[(dv * height) // ev][(du * width) // eu][comp_of_species[s]] += 1
    img = np.zeros((height, width, 4), dtype=np.uint8)
    for r in range(height):
        for c in range(width):
            if cnt[r][c].sum() == 0:
                continue
            for k in range(3):
                acc = 0
                for q in range(n_comp):
                    acc += int(palette[q][k]) * min(int(cnt[r][c][q]) * gain, 255) // 255
                img[r][c][k] = min(255, acc)
            img[r][c][3] = 255
    return img
