"""Exact pins of the oracle's decision rules and Philox stream layouts (CPU only).

Each test recomputes, with nothing but numpy and PyTorch's own CPU Philox engine (tests/helpers/), what
DESIGN.md §1 / reading S2 says a phase must produce, and compares it with the oracle element by element:
the proposal argmin and its tie-break (S9), cube and sphere seeding (S15), the UNI word of channel k and
the BIRTH offsets (S2, S11, S13, S14), the crossing draw (S7), DEGRADE with BIRTH emissions (§1 phase 3),
the sphere fallback of a newborn (S11) and the homodimer anchor (S10).  None of them calls into oracle code
to get an expected value, and none touches the CUDA path.
"""
import numpy as np

from oracle.binding import MODE_BRUTE, MODE_GRID, NOPROP, Oracle
from workloads.model import (CH_BIRTH, CH_DEGRADE, CH_RELEASE, NONE16, SHAPE_CUBE, SHAPE_SPHERE, Channel,
                             Compartment, Model, Reaction, SeedRecord, Species, prob_to_thr, stack_tables)

TAG_MOVE, TAG_PAIR, TAG_UNI, TAG_BIRTH, TAG_PLACE = 1, 2, 3, 4, 5


def key_of(seed):
    return [seed & 0xFFFFFFFF, seed >> 32]


def ctr(c0, c1, c2, tag):
    c0 = np.asarray(c0, dtype=np.uint32)
    n = len(c0)
    f = lambda v: np.broadcast_to(np.asarray(v, dtype=np.uint32), (n,))
    return np.stack([c0, f(c1), f(c2), f(tag)], axis=1)


def fire(u, thr):
    return (u.astype(np.uint64) < thr) | (thr == 0xFFFFFFFF)


def mirror(q, L):
    q = np.where(q < 0, -1 - q, q)
    return np.where(q >= L, 2 * L - 1 - q, q)


def ab_model(L, n_a, n_b, p_bind, seed, r2=2500, cell=64, same=False):
    A, B, Cx = 0, 1, 2
    rx = [Reaction(A, A, Cx, r2, prob_to_thr(p_bind))] if same else [Reaction(A, B, Cx, r2, prob_to_thr(p_bind))]
    m = Model(name="pin", species=[Species("A", 1), Species("B", 1), Species("C", 2)], reactions=rx,
              compartments=[Compartment(SHAPE_CUBE, L=L)], table_bits=12, tables=stack_tables([44.7214, 31.6228], 12),
              extent=(L, L, L), seed=seed, place_seed=seed + 1,
              seed_records=[SeedRecord(A, n_a), SeedRecord(B, n_b)], n_steps=8, cell_size=cell)
    return m.finalize()


# --------------------------------------------------------------------------- proposal rule (S9, north_star (4))
def expected_proposals(a, species_ok, r2, thr, t, seed, torch_philox):
    """prop(i) = partner with the smallest (d2, id_j) among eligible partners within r2 that pass the symmetric pair
    draw philox(min id, max id, t, 2).r0; evaluated densely over all pairs."""
    n = len(a["id"])
    pos = np.stack([a["x"], a["y"], a["z"]], axis=1).astype(np.int64)
    d2 = ((pos[:, None, :] - pos[None, :, :]) ** 2).sum(axis=2)
    ids = a["id"].astype(np.int64)
    ii, jj = np.nonzero((d2 <= r2) & species_ok & ~np.eye(n, dtype=bool))
    lo, hi = np.minimum(ids[ii], ids[jj]), np.maximum(ids[ii], ids[jj])
    r = torch_philox(ctr(lo, hi, t, TAG_PAIR), key_of(seed))
    ok = fire(r[:, 0], thr)
    ii, jj = ii[ok], jj[ok]
    out = np.full(n, NOPROP, dtype=np.uint32)
    # lexicographic order: first by agent, then d2, then partner id; the first row of every agent is its proposal
    order = np.lexsort((ids[jj], d2[ii, jj], ii))
    ii, jj = ii[order], jj[order]
    first = np.ones(len(ii), dtype=bool)
    first[1:] = ii[1:] != ii[:-1]
    out[ii[first]] = a["id"][jj[first]]
    return out, len(ii)


def test_proposal_is_argmin_of_d2_then_id_among_pair_draw_passers(torch_philox):
    m = ab_model(L=260, n_a=500, n_b=500, p_bind=0.5, seed=0x5EED0001)
    o = Oracle(m); o.seed_population()
    o.debug_move_only()
    a = o.read_agents()                              # id-sorted, as debug_proposals reports
    sp = a["species"]
    ok = (sp[:, None] == 0) & (sp[None, :] == 1) | (sp[:, None] == 1) & (sp[None, :] == 0)
    want, n_pass = expected_proposals(a, ok, 2500, prob_to_thr(0.5), 0, m.seed, torch_philox)
    assert n_pass > 400                              # dense enough: many agents choose among several passers
    multi = 0
    for mode in (MODE_BRUTE, MODE_GRID):
        got = o.debug_proposals(mode)
        assert (got == want).all(), (mode, np.nonzero(got != want)[0][:5])
    # the choice really is a choice: some agent has >= 2 passing partners at different distances
    pos = np.stack([a["x"], a["y"], a["z"]], axis=1).astype(np.int64)
    d2 = ((pos[:, None, :] - pos[None, :, :]) ** 2).sum(axis=2)
    multi = int((((d2 <= 2500) & ok).sum(axis=1) >= 2).sum())
    assert multi > 50


def test_proposal_tie_on_d2_goes_to_the_smaller_partner_id():
    # p_bind = 1 (thr 2^32-1: certain), immobile lattice input: an A with two / three B at the same d2
    m = ab_model(L=400, n_a=1, n_b=1, p_bind=1.0, seed=3)
    o = Oracle(m)
    #            A0              B (d2 = 900)      B (d2 = 900)     B (d2 = 900)      A, one partner   its B
    x = np.array([100, 130, 100, 100, 300, 300], dtype=np.int32)
    y = np.array([100, 100, 130, 100, 300, 320], dtype=np.int32)
    z = np.array([100, 100, 100, 70, 300, 300], dtype=np.int32)
    s = np.array([0, 1, 1, 1, 0, 1], dtype=np.uint16)
    for ids in ([10, 7, 5, 9, 1, 2], [10, 5, 7, 9, 1, 2], [3, 40, 41, 6, 50, 8]):
        ids = np.array(ids, dtype=np.uint32)
        o.load_agents(x, y, z, s, ids, step=0, next_id=64)
        order = np.argsort(ids)
        rank = {int(i): k for k, i in enumerate(ids[order])}
        for mode in (MODE_BRUTE, MODE_GRID):
            got = o.debug_proposals(mode)
            assert got[rank[int(ids[0])]] == min(ids[1:4]), (ids, mode)     # tie -> smallest partner id
            for k in (1, 2, 3):
                assert got[rank[int(ids[k])]] == ids[0]                      # each B's only partner
            assert got[rank[int(ids[4])]] == ids[5] and got[rank[int(ids[5])]] == ids[4]
    # a nearer partner beats a smaller id: B at d2 = 400 with a LARGER id than the three at 900
    x2 = np.append(x, 100).astype(np.int32); y2 = np.append(y, 100).astype(np.int32); z2 = np.append(z, 120).astype(np.int32)
    ids = np.array([10, 7, 5, 9, 1, 2, 60], dtype=np.uint32)
    o.load_agents(x2, y2, z2, np.append(s, 1).astype(np.uint16), ids, step=0, next_id=64)
    got = o.debug_proposals(MODE_BRUTE)
    assert got[list(np.sort(ids)).index(10)] == 60


# --------------------------------------------------------------------------- seeding layouts (S15)
def test_cube_seeding_is_philox_place_words_times_L(torch_philox):
    m = ab_model(L=777, n_a=300, n_b=200, p_bind=0.5, seed=0xABCDEF0123)
    o = Oracle(m); o.seed_population()
    a = o.read_agents()
    r = torch_philox(ctr(a["id"], 0, 0, TAG_PLACE), key_of(m.place_seed)).astype(np.uint64)
    for axis, k in enumerate("xyz"):
        assert (a[k] == ((r[:, axis] * 777) >> 32).astype(np.int32)).all(), k
    assert (a["id"] == np.arange(500)).all() and (a["species"] == np.repeat([0, 1], [300, 200])).all()


def sphere_model(R, r_in, seed, species, reactions=(), n_rules=0, recs=()):
    comps = [Compartment(SHAPE_SPHERE, R, R, R, r_out=R, r_in=r_in)]
    if r_in >= 0:
        comps.append(Compartment(SHAPE_SPHERE, R, R, R, r_out=r_in))
    m = Model(name="sph", species=species, reactions=list(reactions), compartments=comps, table_bits=12,
              tables=stack_tables([60.0, 30.0], 12), extent=(2 * R + 1,) * 3, seed=seed, place_seed=seed ^ 0x77,
              seed_records=list(recs), n_steps=8, cell_size=128, n_rules=n_rules)
    return m.finalize()


def test_sphere_and_shell_seeding_is_first_valid_attempt(torch_philox):
    R, Rn = 900, 450
    m = sphere_model(R, Rn, 0x1234, [Species("cyt", 1, 0), Species("nuc", 1, 1)],
                     recs=[SeedRecord(0, 700), SeedRecord(1, 500)])
    o = Oracle(m); o.seed_population()
    a = o.read_agents()
    side = 2 * R + 1
    n_retry = 0
    for rec_sp, lo, hi, rout in ((0, Rn, R, R), (1, -1, Rn, Rn)):
        sel = a["species"] == rec_sp
        ids = a["id"][sel]
        want = np.zeros((len(ids), 3), dtype=np.int64)
        done = np.zeros(len(ids), dtype=bool)
        side = 2 * rout + 1
        for attempt in range(64):
            r = torch_philox(ctr(ids, attempt, 0, TAG_PLACE), key_of(m.place_seed)).astype(np.uint64)
            q = R - rout + ((r[:, :3] * side) >> 32).astype(np.int64)       # bounding cube of the outer sphere
            r2 = ((q - R) ** 2).sum(axis=1)
            valid = (r2 <= hi * hi) & ((lo < 0) | (r2 > lo * lo))
            take = valid & ~done
            want[take] = q[take]; done |= take
            if attempt == 0:
                n_retry += int((~valid).sum())
        assert done.all()
        for axis, k in enumerate("xyz"):
            assert (a[k][sel] == want[:, axis]).all(), (rec_sp, k)
    assert n_retry > 300          # the attempt loop was exercised


# --------------------------------------------------------------------------- UNI word k, BIRTH offsets, id order
def test_release_uses_word_k_of_uni_and_birth_stream_offsets(torch_philox):
    L, n = 300, 1500
    A, B, Cx = 0, 1, 2
    p = 0.35
    m = Model(name="rel", species=[Species("A", 1), Species("B", 1),
                                   Species("C", 2, channels=[Channel(CH_DEGRADE, 0),          # thr 0: never fires
                                                             Channel(CH_RELEASE, prob_to_thr(p), A, B)])],
              reactions=[Reaction(A, B, Cx, 2500, prob_to_thr(0.5))], compartments=[Compartment(SHAPE_CUBE, L=L)],
              table_bits=12, tables=stack_tables([44.7214, 31.6228], 12), extent=(L, L, L), seed=0xC0FFEE12345,
              place_seed=5, seed_records=[SeedRecord(Cx, n)], n_steps=8, cell_size=64).finalize()
    o = Oracle(m); o.seed_population()
    before = o.read_agents()
    t = 0
    ids = before["id"]
    key = key_of(m.seed)
    # phase 1: C moves with sigma class 2
    r = torch_philox(ctr(ids, 0, t, TAG_MOVE), key)
    tab = m.tables[2].astype(np.int64)
    pos = np.stack([mirror(before[k].astype(np.int64) + tab[r[:, ax] >> 20], L) for ax, k in enumerate("xyz")], axis=1)
    # phase 3: channel k = 1 reads word r1 of the UNI call
    u = torch_philox(ctr(ids, 0, t, TAG_UNI), key)
    fired = fire(u[:, 1], prob_to_thr(p))
    assert 0.25 * n < fired.sum() < 0.45 * n and (fire(u[:, 0], prob_to_thr(p)) != fired).any()
    # phase 4: newborns in parent-id order get ids n, n+1, ...; offsets from the BIRTH stream (parent id, k = 1, t, 4)
    par = ids[fired]
    b = torch_philox(ctr(par, 1, t, TAG_BIRTH), key).astype(np.uint64)
    off = ((b[:, :3] * 21) >> 32).astype(np.int64) - 10
    assert off.min() == -10 and off.max() == 10
    born = mirror(pos[fired] + off, L)
    o.step(1)
    a = o.read_agents()
    assert len(a["id"]) == n + fired.sum() and (a["id"] == np.arange(n + fired.sum())).all()
    assert (a["species"][:n] == np.where(fired, A, Cx)).all() and (a["species"][n:] == B).all()
    for ax, k in enumerate("xyz"):
        assert (a[k][:n] == pos[:, ax]).all(), k
        assert (a[k][n:] == born[:, ax]).all(), k
    assert o.info()["next_id"] == n + fired.sum()


# --------------------------------------------------------------------------- crossing draw = word r3 (S7)
def test_membrane_crossing_uses_word_r3(torch_philox):
    R, Rn = 900, 450
    px = prob_to_thr(0.4)
    sp = [Species("c", 1, 0, cross_to=1, cross_thr=px), Species("n", 1, 1, cross_to=0, cross_thr=px)]
    m = sphere_model(R, Rn, 0xFACE, sp)
    o = Oracle(m)
    # agents on a thin layer on both sides of the membrane, so that many proposed moves end in the other compartment
    rng = np.random.default_rng(5)
    n = 3000
    v = rng.normal(size=(n, 3)); v /= np.linalg.norm(v, axis=1)[:, None]
    rad = Rn + rng.integers(-40, 41, size=n)
    q = np.rint(R + v * rad[:, None]).astype(np.int64)
    r2 = ((q - R) ** 2).sum(axis=1)
    s = np.where(r2 <= Rn * Rn, 1, 0).astype(np.uint16)
    ids = np.arange(n, dtype=np.uint32)
    o.load_agents(q[:, 0], q[:, 1], q[:, 2], s, ids, step=3, next_id=n)
    o.debug_move_only()
    a = o.read_agents()
    r = torch_philox(ctr(ids, 0, 3, TAG_MOVE), key_of(m.seed))
    tab = m.tables[1].astype(np.int64)
    qq = q + np.stack([tab[r[:, ax] >> 20] for ax in range(3)], axis=1)
    rr2 = ((qq - R) ** 2).sum(axis=1)
    in_nuc, in_cyt = rr2 <= Rn * Rn, (rr2 > Rn * Rn) & (rr2 <= R * R)
    stays = np.where(s == 1, in_nuc, in_cyt)
    other = np.where(s == 1, in_cyt, in_nuc)
    cross = ~stays & other & fire(r[:, 3], px)
    assert cross.sum() > 200 and (~stays & other & ~cross).sum() > 200
    assert (fire(r[:, 2], px) != fire(r[:, 3], px)).any()
    want_s = np.where(cross, 1 - s, s)
    moved = stays | cross
    assert (a["species"] == want_s).all()
    for ax, k in enumerate("xyz"):
        assert (a[k] == np.where(moved, qq[:, ax], q[:, ax])).all(), k


# --------------------------------------------------------------------------- DEGRADE with BIRTH (phase 3), S13
def test_degrade_still_emits_its_births_and_lowest_consuming_channel_wins():
    from workloads.model import CH_CONVERT
    L = 300
    X, Y, Z, W, V = 0, 1, 2, 3, 4
    always = 0xFFFFFFFF
    m = Model(name="deg", species=[
        Species("X", 0, channels=[Channel(CH_BIRTH, always, prod1=Y), Channel(CH_DEGRADE, always),
                                  Channel(CH_RELEASE, always, Z, Y), Channel(CH_BIRTH, always, prod1=Z)]),
        Species("Y", 0), Species("Z", 0),
        Species("W", 0, channels=[Channel(CH_CONVERT, always, prod0=Y), Channel(CH_DEGRADE, always),
                                  Channel(CH_RELEASE, always, Z, Y)]),
        Species("V", 0, channels=[Channel(CH_RELEASE, always, Z, Y), Channel(CH_CONVERT, always, prod0=X),
                                  Channel(CH_DEGRADE, always)])],
        reactions=[], compartments=[Compartment(SHAPE_CUBE, L=L)], table_bits=12, tables=stack_tables([10.0], 12),
        extent=(L, L, L), seed=1, place_seed=2, seed_records=[SeedRecord(X, 40), SeedRecord(W, 30), SeedRecord(V, 20)],
        n_steps=4, cell_size=64).finalize()
    o = Oracle(m); o.seed_population()
    par = o.read_agents()
    o.step(1)
    a = o.read_agents()
    # every X dies (DEGRADE, channel 1, is the lowest consuming channel that fires: the RELEASE of channel 2 does not
    # apply and emits nothing), its two BIRTH channels (0 and 3) still emit;
    # every W is converted to Y by channel 0: its DEGRADE and RELEASE fire too but do not apply;
    # every V releases (becomes Z, emits one Y): its CONVERT and DEGRADE do not apply.
    # Newborn ids follow (parent id, channel): X parents 0..39 (two each), then V parents 70..89 (one each).
    assert (a["id"] == np.concatenate([40 + np.arange(50), 90 + np.arange(100)])).all()
    assert (a["species"] == np.concatenate([np.full(30, Y), np.full(20, Z), np.tile([Y, Z], 40), np.full(20, Y)])).all()
    parents = np.concatenate([np.repeat(np.arange(40), 2), 70 + np.arange(20)])
    for k in "xyz":                                        # a newborn sits within +-10 units of its (immobile) parent
        assert (a[k][:50] == par[k][40:90]).all()
        assert (np.abs(a[k][50:].astype(np.int64) - par[k][parents].astype(np.int64)) <= 10).all()
    assert list(o.read_counts()[1, 0]) == [0, 30 + 40 + 20, 40 + 20, 0, 0]


# --------------------------------------------------------------------------- sphere newborn fallback (S11)
def test_newborn_outside_the_sphere_takes_the_parent_position(torch_philox):
    R = 300
    sp = [Species("E", 0, 0, channels=[Channel(CH_BIRTH, 0xFFFFFFFF, prod1=1)]), Species("Y", 0, 0)]
    m = sphere_model(R, -1, 0xBEEF, sp)
    o = Oracle(m)
    rng = np.random.default_rng(11)
    n = 400
    v = rng.normal(size=(n, 3)); v /= np.linalg.norm(v, axis=1)[:, None]
    q = np.trunc(v * (R - rng.integers(0, 4, size=n))[:, None]).astype(np.int64) + R      # on / just inside the surface
    assert (((q - R) ** 2).sum(axis=1) <= R * R).all()
    ids = np.arange(n, dtype=np.uint32)
    o.load_agents(q[:, 0], q[:, 1], q[:, 2], np.zeros(n, np.uint16), ids, step=5, next_id=n)
    o.step(1)
    a = o.read_agents()
    b = torch_philox(ctr(ids, 0, 5, TAG_BIRTH), key_of(m.seed)).astype(np.uint64)
    cand = q + ((b[:, :3] * 21) >> 32).astype(np.int64) - 10
    inside = ((cand - R) ** 2).sum(axis=1) <= R * R
    assert inside.sum() > 50 and (~inside).sum() > 50
    want = np.where(inside[:, None], cand, q)
    assert (a["id"] == np.arange(2 * n)).all() and (a["species"][n:] == 1).all()
    for ax, k in enumerate("xyz"):
        assert (a[k][:n] == q[:, ax]).all() and (a[k][n:] == want[:, ax]).all(), k


# --------------------------------------------------------------------------- homodimer anchor (S10)
def test_homodimer_anchor_is_the_smaller_id(torch_philox):
    m = ab_model(L=400, n_a=2, n_b=0, p_bind=1.0, seed=9, same=True)
    m.species[0].sigma_class = 0                   # immobile: positions stay where they are loaded
    o = Oracle(m)
    x = np.array([100, 110, 300, 320], dtype=np.int32)
    s = np.zeros(4, dtype=np.uint16)
    for ids in ([4, 9, 30, 2], [9, 4, 2, 30]):
        ids = np.array(ids, dtype=np.uint32)
        o.load_agents(x, x, x, s, ids, step=0, next_id=64)
        o.step(1)
        a = o.read_agents()
        assert list(a["id"]) == [2, 4] and list(a["species"]) == [2, 2]         # the smaller id of each pair survives
        xs = dict(zip(ids.tolist(), x.tolist()))
        assert [int(v) for v in a["x"]] == [xs[2], xs[4]]                       # ... at its own position
    # a dense random A-only population: grid == brute, and every bound pair leaves exactly the smaller id behind
    m2 = ab_model(L=220, n_a=700, n_b=0, p_bind=0.6, seed=0x77AA, same=True)
    o1, o2 = Oracle(m2), Oracle(m2, mode=MODE_BRUTE)
    for o in (o1, o2):
        o.seed_population()
    o1.debug_move_only()
    a = o1.read_agents()
    sp_ok = np.ones((700, 700), dtype=bool)
    want, _ = expected_proposals(a, sp_ok, 2500, prob_to_thr(0.6), 0, m2.seed, torch_philox)
    assert (o1.debug_proposals(MODE_GRID) == want).all()
    idx = {int(i): k for k, i in enumerate(a["id"])}
    mutual = [(int(i), int(j)) for i, j in zip(a["id"], want) if j != NOPROP and want[idx[int(j)]] == i and i < j]
    assert len(mutual) > 30
    o2.step(1); o3 = Oracle(m2); o3.seed_population(); o3.step(1)
    b2, b3 = o2.read_agents(), o3.read_agents()
    assert all((b2[k] == b3[k]).all() for k in b2)
    alive = dict(zip(b3["id"].tolist(), b3["species"].tolist()))
    for i, j in mutual:
        assert alive.get(i) == 2 and j not in alive


# --------------------------------------------------------------------------- replicas: local coordinates (S16)
def test_replica_move_uses_local_coordinates_and_keeps_the_tile(torch_philox):
    R, shift, n_rep = 1500, 12, 4
    c = 1600
    m = Model(name="rep", species=[Species("a", 1, 0)], reactions=[], table_bits=12, tables=stack_tables([60.0], 12),
              compartments=[Compartment(SHAPE_SPHERE, c, c, c, r_out=R, r_in=-1)], extent=(n_rep << shift, 2 * c + 1, 2 * c + 1),
              n_replicas=n_rep, stride_shift=shift, seed=0xD1CE, place_seed=1, seed_records=[], n_steps=16, cell_size=128).finalize()
    o = Oracle(m)
    rng = np.random.default_rng(3)
    n = 2000
    v = rng.normal(size=(n, 3)); v /= np.linalg.norm(v, axis=1)[:, None]
    q = np.rint(c + v * (R - rng.integers(0, 60, size=n))[:, None]).astype(np.int64)          # near the surface
    q = q[((q - c) ** 2).sum(axis=1) <= R * R]
    n = len(q)
    rep = rng.integers(0, n_rep, size=n)
    ids = rng.permutation(n).astype(np.uint32)
    o.load_agents(q[:, 0] + (rep << shift), q[:, 1], q[:, 2], np.zeros(n, np.uint16), ids, step=7, next_id=n)
    o.debug_move_only()
    a = o.read_agents()
    order = np.argsort(ids)
    q, rep, ids = q[order], rep[order], ids[order]
    r = torch_philox(ctr(ids, 0, 7, TAG_MOVE), key_of(m.seed))
    tab = m.tables[1].astype(np.int64)
    qq = q + np.stack([tab[r[:, ax] >> 20] for ax in range(3)], axis=1)                     # in LOCAL coordinates
    ok = ((qq - c) ** 2).sum(axis=1) <= R * R
    assert ok.sum() > 300 and (~ok).sum() > 300
    want = np.where(ok[:, None], qq, q)
    assert (a["x"] == want[:, 0] + (rep << shift)).all() and (a["y"] == want[:, 1]).all() and (a["z"] == want[:, 2]).all()
    assert ((a["x"] >> shift) == rep).all()                                                  # nobody changes replica
    cnt = o.read_counts()[-1, :, 0]
    assert (cnt == np.bincount(rep, minlength=n_rep)).all()                                  # counts are per replica


# --------------------------------------------------------------------------- delayed births (S17) and expressors
def test_delayed_birth_fires_exactly_delay_steps_after_the_first_marked_birth(torch_philox):
    from workloads.model import CH_DELAYED_BIRTH

    L, delay, p0 = 400, 4, 0.04
    G, Mx, F = 0, 1, 2
    thr = prob_to_thr(p0)
    m = Model(name="delay", species=[
        Species("G", 0, channels=[Channel(CH_BIRTH, thr, prod1=Mx, rule=0, marks_first=True),
                                  Channel(CH_DELAYED_BIRTH, delay, prod1=F, rule=0)]),
        Species("M", 0), Species("F", 0)], reactions=[], compartments=[Compartment(SHAPE_CUBE, L=L)], table_bits=12,
        tables=stack_tables([10.0], 12), extent=(L, L, L), seed=0xC0DE00, place_seed=4, n_rules=1,
        seed_records=[SeedRecord(G, 6)], n_steps=40, cell_size=64).finalize()
    o = Oracle(m); o.seed_population()
    g = o.read_agents()
    gid = g["id"]
    gpos = np.stack([g["x"], g["y"], g["z"]], axis=1).astype(np.int64)
    key = key_of(m.seed)
    T = 30
    rows, t_first, next_id = [], None, 6
    born_ids, born_sp, born_pos = [], [], []
    for t in range(T):
        u = torch_philox(ctr(gid, 0, t, TAG_UNI), key)
        fired0 = fire(u[:, 0], thr)                                    # channel 0 reads word r0
        delayed = t_first is not None and t == t_first + delay          # t_first as of the start of the step
        for k_parent in range(6):                                       # (parent id, channel) order: ids ascend with k_parent
            for ch, on, spc in ((0, fired0[k_parent], Mx), (1, delayed, F)):
                if not on:
                    continue
                b = torch_philox(ctr([gid[k_parent]], ch, t, TAG_BIRTH), key).astype(np.uint64)[0]
                off = ((b[:3] * 21) >> 32).astype(np.int64) - 10
                born_ids.append(next_id); next_id += 1
                born_sp.append(spc); born_pos.append(mirror(gpos[k_parent] + off, L))
        if fired0.any() and t_first is None:
            t_first = t
        rows.append((6, born_sp.count(Mx), born_sp.count(F)))
    assert t_first is not None and t_first + delay < T - 2 and t_first > 0
    o.step(T)
    a, c = o.read_agents(), o.read_counts()[:, 0, :]
    assert o.info()["t_first0"] == t_first and o.info()["next_id"] == next_id
    assert (c[1:] == np.array(rows)).all()
    assert c[t_first + delay, F] == 0 and c[t_first + delay + 1, F] == 6      # every locus emits one, exactly then, once
    assert (a["id"][6:] == np.array(born_ids)).all() and (a["species"][6:] == np.array(born_sp)).all()
    bp = np.array(born_pos)
    for ax, k in enumerate("xyz"):
        assert (a[k][6:] == bp[:, ax]).all(), k


# --------------------------------------------------------------------------- mid-run seeding (run-time treatment)
def test_mid_run_seeding_continues_ids_and_uses_its_own_place_seed(torch_philox):
    m = ab_model(L=900, n_a=100, n_b=0, p_bind=0.5, seed=11)
    o = Oracle(m); o.seed_population()
    o.step(2)
    before, n0 = o.read_agents(), o.info()["next_id"]
    o.seed_population([SeedRecord(1, 50), SeedRecord(0, 7)], place_seed=0xFEED)
    a = o.read_agents()
    new = a["id"] >= n0
    assert new.sum() == 57 and (a["id"][new] == n0 + np.arange(57)).all()
    assert (a["species"][new] == np.repeat([1, 0], [50, 7])).all()
    r = torch_philox(ctr(a["id"][new], 0, 0, TAG_PLACE), key_of(0xFEED)).astype(np.uint64)
    for ax, k in enumerate("xyz"):
        assert (a[k][new] == ((r[:, ax] * 900) >> 32).astype(np.int32)).all(), k
        assert (a[k][~new] == before[k]).all()                          # the old agents are untouched
    c = o.read_counts()
    assert c.shape[0] == 3 and list(c[2, 0]) == [int((a["species"] == s).sum()) for s in range(3)]   # row t rewritten
    assert o.info()["step"] == 2 and o.info()["next_id"] == n0 + 57
