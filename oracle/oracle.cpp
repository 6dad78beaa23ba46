// oracle.cpp — CPU ORACLE of the molecule-agent time step.  TEST INFRASTRUCTURE.
//
// Plain single-threaded C++17, written from DESIGN.md "Step specification" (which
// freezes BASELINE.json north_star (1)-(5) + SURVEY.md Appendix A).  Every function
// cites the passage it follows.  No blocking, fusion or reordering beyond the spec:
// phases run one after another over a std::vector of agents.  Shares nothing with
// paper_2606_14603_b200/csrc.  See oracle.h for the "parity unpinned" list.
#include "oracle.h"

#include <algorithm>
#include <cstring>
#include <vector>

namespace {

struct Agent { int32_t x, y, z; uint16_t s; uint32_t id; };
struct Birth { uint32_t parent_id; uint32_t k; uint16_t species; uint32_t parent_index; };

constexpr uint16_t DEAD = 0xFFFF;
constexpr uint32_t NEVER = 0xFFFFFFFFu;
constexpr uint32_t NOPROP = 0xFFFFFFFFu;
enum { TAG_MOVE = 1, TAG_PAIR = 2, TAG_UNI = 3, TAG_BIRTH = 4, TAG_PLACE = 5 };

// Philox4x32-10 (Salmon et al., SC'11; S2).  ctr = (c0,c1,c2,c3), key = (k0,k1).
// One round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
// the key is bumped by (W0,W1) between rounds: 10 rounds, 9 bumps.
void philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    uint64_t p0 = M0 * c0, p1 = M1 * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// DESIGN.md S4: fire(u, thr) = (thr == 2^32-1) || (u < thr)
inline bool fire(uint32_t u, uint32_t thr) { return thr == 0xFFFFFFFFu || u < thr; }

}  // namespace

struct oracle {
  orc_config_t cfg;
  std::vector<orc_species_t> sp;
  std::vector<orc_reaction_t> rx;
  std::vector<orc_compartment_t> comp;
  std::vector<int16_t> tables;
  std::vector<int> rxmap;        // [n_species*n_species] -> reaction index or -1 (symmetric)
  std::vector<uint8_t> binds;    // species takes part in some reaction
  std::vector<Agent> ag;
  std::vector<uint32_t> counts;  // [counts_rows][n_replicas][n_species]
  std::vector<uint32_t> t_first;
  uint32_t key[2];
  uint32_t t = 0, next_id = 0;
  int mode = ORC_MODE_GRID;
  int err = ORC_OK;

  void rng(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t tag, uint32_t out[4]) const {
    uint32_t c[4] = {c0, c1, c2, tag};
    philox(c, key, out);
  }

  // DESIGN.md S1: compartment membership in LOCAL coordinates (replica offset removed).
  bool valid(const orc_compartment_t& c, int64_t x, int64_t y, int64_t z) const {
    if (c.shape == ORC_SHAPE_CUBE)
      return x >= 0 && x < c.L && y >= 0 && y < c.L && z >= 0 && z < c.L;
    int64_t dx = x - c.cx, dy = y - c.cy, dz = z - c.cz;
    int64_t r2 = dx * dx + dy * dy + dz * dz;
    if (r2 > (int64_t)c.r_out * c.r_out) return false;
    if (c.r_in >= 0 && r2 <= (int64_t)c.r_in * c.r_in) return false;
    return true;
  }

  // DESIGN.md S5: mirror about planes at -1/2 and L-1/2.
  static int32_t mirror(int32_t q, int32_t L) {
    if (q < 0) return -1 - q;
    if (q >= L) return 2 * L - 1 - q;
    return q;
  }

  uint32_t replica_of(int32_t x) const { return (uint32_t)x >> cfg.stride_shift; }

  // ---- Phase 1: Brownian move + boundary / compartment rule (spec phase 1; S2,S3,S5,S6,S7)
  void phase_move() {
    const uint32_t B = cfg.table_bits;
    for (Agent& a : ag) {
      const orc_species_t& s = sp[a.s];
      if (s.sigma_class == 0) continue;
      uint32_t r[4];
      rng(a.id, 0, t, TAG_MOVE, r);
      const int16_t* tab = &tables[(size_t)s.sigma_class << B];
      int32_t base = (int32_t)(replica_of(a.x) << cfg.stride_shift);
      int32_t qx = a.x - base + tab[r[0] >> (32 - B)];
      int32_t qy = a.y + tab[r[1] >> (32 - B)];
      int32_t qz = a.z + tab[r[2] >> (32 - B)];
      const orc_compartment_t& c = comp[s.compartment];
      if (c.shape == ORC_SHAPE_CUBE) {
        a.x = mirror(qx, c.L) + base; a.y = mirror(qy, c.L); a.z = mirror(qz, c.L);
      } else if (valid(c, qx, qy, qz)) {
        a.x = qx + base; a.y = qy; a.z = qz;
      } else if (s.cross_to != ORC_NONE16 && valid(comp[sp[s.cross_to].compartment], qx, qy, qz) &&
                 fire(r[3], s.cross_thr)) {
        a.x = qx + base; a.y = qy; a.z = qz; a.s = s.cross_to;
      }  // else: move rejected, agent stays (S6)
    }
  }

  // ---- Phase 2 candidate predicate (spec phase 2; S8, S9), without the pair draw
  int in_range_reaction(const Agent& a, const Agent& b) const {
    int e = rxmap[(size_t)a.s * cfg.n_species + b.s];
    if (e < 0) return -1;
    int64_t dx = (int64_t)a.x - b.x, dy = (int64_t)a.y - b.y, dz = (int64_t)a.z - b.z;
    int64_t d2 = dx * dx + dy * dy + dz * dz;
    return d2 <= (int64_t)rx[e].r2 ? e : -1;
  }
  bool pair_draw(const Agent& a, const Agent& b, int e) const {
    uint32_t r[4];
    rng(std::min(a.id, b.id), std::max(a.id, b.id), t, TAG_PAIR, r);
    return fire(r[0], rx[e].thr);
  }
  static int64_t dist2(const Agent& a, const Agent& b) {
    int64_t dx = (int64_t)a.x - b.x, dy = (int64_t)a.y - b.y, dz = (int64_t)a.z - b.z;
    return dx * dx + dy * dy + dz * dz;
  }

  // Visit candidate indices j for agent i.  BRUTE: every j (the definition).
  // GRID: agents in the 27 cells around i's cell (valid because cell_size >= max R).
  struct Grid {
    int32_t cs; int64_t nx, ny, nz;
    std::vector<uint32_t> start, order;
  } grid;
  void build_grid() {
    Grid& g = grid;
    g.cs = (int32_t)cfg.cell_size;
    g.nx = (cfg.extent[0] + g.cs - 1) / g.cs; g.ny = (cfg.extent[1] + g.cs - 1) / g.cs;
    g.nz = (cfg.extent[2] + g.cs - 1) / g.cs;
    size_t nc = (size_t)(g.nx * g.ny * g.nz);
    g.start.assign(nc + 1, 0);
    g.order.resize(ag.size());
    auto cell = [&](const Agent& a) {
      return (size_t)(((int64_t)(a.z / g.cs) * g.ny + a.y / g.cs) * g.nx + a.x / g.cs);
    };
    for (const Agent& a : ag) g.start[cell(a) + 1]++;
    for (size_t c = 0; c < nc; ++c) g.start[c + 1] += g.start[c];
    std::vector<uint32_t> cur(g.start.begin(), g.start.end() - 1);
    for (size_t i = 0; i < ag.size(); ++i) g.order[cur[cell(ag[i])]++] = (uint32_t)i;
  }
  template <class F> void for_candidates(size_t i, int use_mode, F&& f) const {
    if (use_mode == ORC_MODE_BRUTE) {
      for (size_t j = 0; j < ag.size(); ++j) if (j != i) f(j);
      return;
    }
    const Grid& g = grid;
    int64_t cx = ag[i].x / g.cs, cy = ag[i].y / g.cs, cz = ag[i].z / g.cs;
    for (int64_t z = cz - 1; z <= cz + 1; ++z) {
      if (z < 0 || z >= g.nz) continue;
      for (int64_t y = cy - 1; y <= cy + 1; ++y) {
        if (y < 0 || y >= g.ny) continue;
        for (int64_t x = cx - 1; x <= cx + 1; ++x) {
          if (x < 0 || x >= g.nx) continue;
          size_t c = (size_t)((z * g.ny + y) * g.nx + x);
          for (uint32_t p = g.start[c]; p < g.start[c + 1]; ++p)
            if (g.order[p] != i) f((size_t)g.order[p]);
        }
      }
    }
  }

  // prop(i) = argmin over cand(i) of (d2, id_j)   (spec phase 2; S9)
  void compute_proposals(int use_mode, std::vector<uint32_t>& prop) {
    if (use_mode == ORC_MODE_GRID) build_grid();
    prop.assign(ag.size(), NOPROP);
    for (size_t i = 0; i < ag.size(); ++i) {
      if (ag[i].s == DEAD || !binds[ag[i].s]) continue;
      bool have = false; int64_t best_d2 = 0; uint32_t best_id = 0, best_j = NOPROP;
      for_candidates(i, use_mode, [&](size_t j) {
        if (ag[j].s == DEAD) return;
        int e = in_range_reaction(ag[i], ag[j]);
        if (e < 0 || !pair_draw(ag[i], ag[j], e)) return;
        int64_t d2 = dist2(ag[i], ag[j]);
        if (!have || d2 < best_d2 || (d2 == best_d2 && ag[j].id < best_id)) {
          have = true; best_d2 = d2; best_id = ag[j].id; best_j = (uint32_t)j;
        }
      });
      prop[i] = best_j;
    }
  }

  // ---- Phase 2: mutual proposals bind (spec phase 2; S10)
  void phase_bind() {
    std::vector<uint32_t> prop;
    compute_proposals(mode, prop);
    for (size_t i = 0; i < ag.size(); ++i) {
      uint32_t j = prop[i];
      if (j == NOPROP || j <= i || prop[j] != (uint32_t)i) continue;  // each mutual pair once (i < j)
      const orc_reaction_t& e = rx[rxmap[(size_t)ag[i].s * cfg.n_species + ag[j].s]];
      size_t anchor, other;
      if (ag[i].s == ag[j].s) { anchor = ag[i].id < ag[j].id ? i : j; }
      else                    { anchor = ag[i].s == e.a ? i : j; }
      other = anchor == i ? j : i;
      ag[anchor].s = e.cplx;
      ag[other].s = DEAD;
    }
  }

  // ---- Phase 3: unimolecular channels (spec phase 3; S13, S17)
  void phase_unimolecular(std::vector<Birth>& births) {
    std::vector<uint32_t> tf0 = t_first;  // t_first as of the start of the step
    for (size_t i = 0; i < ag.size(); ++i) {
      Agent& a = ag[i];
      if (a.s == DEAD) continue;
      const orc_species_t s = sp[a.s];
      if (s.n_channels == 0) continue;
      uint32_t r[4];
      rng(a.id, 0, t, TAG_UNI, r);
      bool consumed = false;
      for (uint32_t k = 0; k < s.n_channels; ++k) {
        const orc_channel_t& ch = s.ch[k];
        bool fired;
        if (ch.kind == ORC_CH_NONE) continue;
        if (ch.kind == ORC_CH_DELAYED_BIRTH)
          fired = tf0[ch.rule] != NEVER && t == tf0[ch.rule] + ch.thr;
        else
          fired = fire(r[k], ch.thr);
        if (!fired) continue;
        switch (ch.kind) {
          case ORC_CH_BIRTH:
            births.push_back({a.id, k, ch.prod1, (uint32_t)i});
            if (ch.marks_first) t_first[ch.rule] = std::min(t_first[ch.rule], t);
            break;
          case ORC_CH_DELAYED_BIRTH:
            births.push_back({a.id, k, ch.prod1, (uint32_t)i});
            break;
          case ORC_CH_RELEASE:
            if (!consumed) { consumed = true; a.s = ch.prod0; births.push_back({a.id, k, ch.prod1, (uint32_t)i}); }
            break;
          case ORC_CH_CONVERT:
            if (!consumed) { consumed = true; a.s = ch.prod0; }
            break;
          case ORC_CH_DEGRADE:
            if (!consumed) { consumed = true; a.s = DEAD; }
            break;
        }
      }
    }
  }

  // ---- Phase 4: births in (parent id, channel) order (spec phase 4; S11, S14)
  void phase_births(std::vector<Birth>& births) {
    std::sort(births.begin(), births.end(), [](const Birth& p, const Birth& q) {
      return p.parent_id != q.parent_id ? p.parent_id < q.parent_id : p.k < q.k;
    });
    if ((uint64_t)next_id + births.size() > (uint64_t)cfg.id_capacity) { err = ORC_E_IDSPACE; return; }
    for (size_t g = 0; g < births.size(); ++g) {
      const Birth& b = births[g];
      const Agent par = ag[b.parent_index];   // position = parent's phase-1 position
      uint32_t r[4];
      rng(b.parent_id, b.k, t, TAG_BIRTH, r);
      int32_t o[3];
      for (int a = 0; a < 3; ++a) o[a] = (int32_t)(((uint64_t)r[a] * 21u) >> 32) - 10;
      int32_t base = (int32_t)(replica_of(par.x) << cfg.stride_shift);
      int32_t lx = par.x - base;
      int32_t qx = lx + o[0], qy = par.y + o[1], qz = par.z + o[2];
      const orc_compartment_t& c = comp[sp[b.species].compartment];
      Agent nb;
      if (c.shape == ORC_SHAPE_CUBE) { qx = mirror(qx, c.L); qy = mirror(qy, c.L); qz = mirror(qz, c.L); }
      else if (!valid(c, qx, qy, qz)) { qx = lx; qy = par.y; qz = par.z; }
      nb.x = qx + base; nb.y = qy; nb.z = qz; nb.s = b.species; nb.id = next_id + (uint32_t)g;
      ag.push_back(nb);
    }
    next_id += (uint32_t)births.size();
  }

  // ---- Phase 5: compaction   ---- Phase 6: counts row
  void phase_compact() {
    ag.erase(std::remove_if(ag.begin(), ag.end(), [](const Agent& a) { return a.s == DEAD; }), ag.end());
  }
  void write_counts_row(uint32_t row) {
    size_t w = (size_t)cfg.n_replicas * cfg.n_species;
    uint32_t* c = &counts[(size_t)row * w];
    std::fill(c, c + w, 0u);
    for (const Agent& a : ag) c[(size_t)replica_of(a.x) * cfg.n_species + a.s]++;
  }

  int step_once() {
    if (t + 1 >= cfg.counts_rows) return ORC_E_CAPACITY;
    phase_move();
    phase_bind();
    std::vector<Birth> births;
    phase_unimolecular(births);
    phase_births(births);
    if (err) return err;
    phase_compact();
    if (ag.size() > cfg.capacity) return ORC_E_CAPACITY;
    write_counts_row(t + 1);
    t += 1;
    return ORC_OK;
  }
};

// ------------------------------------------------------------------ validation
static int validate(const orc_config_t* c) {
  if (!c || !c->species || !c->compartments || !c->tables) return ORC_E_INVAL;
  if (c->n_reactions && !c->reactions) return ORC_E_INVAL;
  if (c->n_species == 0 || c->n_species >= 0xFFFF || c->n_compartments == 0) return ORC_E_INVAL;
  if (c->table_bits < 1 || c->table_bits > 16 || c->n_sigma_classes < 1) return ORC_E_INVAL;
  if (c->n_replicas < 1 || c->stride_shift > 31 || c->cell_size == 0) return ORC_E_INVAL;
  if (c->capacity == 0 || c->counts_rows == 0) return ORC_E_INVAL;
  for (int a = 0; a < 3; ++a) if (c->extent[a] <= 0) return ORC_E_INVAL;
  if (c->n_replicas > 1 && ((uint64_t)c->n_replicas << c->stride_shift) > 0x80000000ull) return ORC_E_INVAL;
  if ((uint64_t)c->extent[0] > ((uint64_t)c->n_replicas << c->stride_shift)) return ORC_E_INVAL;
  int32_t max_tab = 0;
  for (size_t i = (size_t)1 << c->table_bits; i < ((size_t)c->n_sigma_classes << c->table_bits); ++i)
    max_tab = std::max<int32_t>(max_tab, std::abs((int32_t)c->tables[i]));
  // DESIGN.md S16: replicas are independent populations, so with several of them a compartment must end at least the
  // largest interaction radius (ceil sqrt max r2) before the next tile begins
  int64_t max_r = 0;
  if (c->reactions)
    for (uint32_t e = 0; e < c->n_reactions; ++e)
      while (max_r * max_r < (int64_t)c->reactions[e].r2) ++max_r;
  for (uint32_t i = 0; i < c->n_compartments; ++i) {
    const orc_compartment_t& k = c->compartments[i];
    int64_t hi;
    if (k.shape == ORC_SHAPE_CUBE) { if (k.L <= 0 || max_tab >= k.L) return ORC_E_INVAL; hi = k.L; }
    else if (k.shape == ORC_SHAPE_SPHERE) {
      if (k.r_out <= 0 || k.r_in >= k.r_out) return ORC_E_INVAL;
      if (k.cx - k.r_out < 0 || k.cy - k.r_out < 0 || k.cz - k.r_out < 0) return ORC_E_INVAL;
      hi = (int64_t)k.cx + k.r_out + 1;
      if ((int64_t)k.cy + k.r_out >= c->extent[1] || (int64_t)k.cz + k.r_out >= c->extent[2]) return ORC_E_INVAL;
    } else return ORC_E_INVAL;
    if (k.shape == ORC_SHAPE_CUBE && (k.L > c->extent[1] || k.L > c->extent[2])) return ORC_E_INVAL;
    if (c->n_replicas == 1 && hi > c->extent[0]) return ORC_E_INVAL;
    if (c->n_replicas > 1 && hi + max_r > ((int64_t)1 << c->stride_shift)) return ORC_E_INVAL;
  }
  for (uint32_t i = 0; i < c->n_species; ++i) {
    const orc_species_t& s = c->species[i];
    if (s.sigma_class >= c->n_sigma_classes || s.compartment >= c->n_compartments) return ORC_E_INVAL;
    if (s.n_channels > ORC_MAX_CHANNELS) return ORC_E_INVAL;
    if (s.cross_to != ORC_NONE16) {
      if (s.cross_to >= c->n_species) return ORC_E_INVAL;
      uint32_t oc = c->species[s.cross_to].compartment;
      if (oc == s.compartment) return ORC_E_INVAL;
      if (c->compartments[oc].shape == ORC_SHAPE_CUBE || c->compartments[s.compartment].shape == ORC_SHAPE_CUBE)
        return ORC_E_INVAL;
    }
    for (uint32_t k = 0; k < s.n_channels; ++k) {
      const orc_channel_t& ch = s.ch[k];
      bool needs0 = ch.kind == ORC_CH_RELEASE || ch.kind == ORC_CH_CONVERT;
      bool needs1 = ch.kind == ORC_CH_RELEASE || ch.kind == ORC_CH_BIRTH || ch.kind == ORC_CH_DELAYED_BIRTH;
      if (ch.kind > ORC_CH_DELAYED_BIRTH) return ORC_E_INVAL;
      if (needs0 && (ch.prod0 >= c->n_species || c->species[ch.prod0].compartment != s.compartment)) return ORC_E_INVAL;
      if (needs1 && (ch.prod1 >= c->n_species || c->species[ch.prod1].compartment != s.compartment)) return ORC_E_INVAL;
      if ((ch.kind == ORC_CH_DELAYED_BIRTH || ch.marks_first) && ch.rule >= c->n_rules) return ORC_E_INVAL;
      if (ch.kind == ORC_CH_DELAYED_BIRTH && ch.thr < 1) return ORC_E_INVAL;
    }
  }
  for (uint32_t e = 0; e < c->n_reactions; ++e) {
    const orc_reaction_t& r = c->reactions[e];
    if (r.a >= c->n_species || r.b >= c->n_species || r.cplx >= c->n_species) return ORC_E_INVAL;
    uint32_t ca = c->species[r.a].compartment;
    if (c->species[r.b].compartment != ca || c->species[r.cplx].compartment != ca) return ORC_E_INVAL;
    if ((uint64_t)r.r2 > (uint64_t)c->cell_size * c->cell_size) return ORC_E_INVAL;
    for (uint32_t f = 0; f < e; ++f) {
      const orc_reaction_t& q = c->reactions[f];
      if ((q.a == r.a && q.b == r.b) || (q.a == r.b && q.b == r.a)) return ORC_E_INVAL;
    }
  }
  return ORC_OK;
}

// ------------------------------------------------------------------ C ABI
extern "C" {

int oracle_create(const orc_config_t* cfg, oracle_t** out) {
  if (!out) return ORC_E_INVAL;
  *out = nullptr;
  int v = validate(cfg);
  if (v) return v;
  oracle* o = new oracle();
  o->cfg = *cfg;
  o->sp.assign(cfg->species, cfg->species + cfg->n_species);
  if (cfg->n_reactions) o->rx.assign(cfg->reactions, cfg->reactions + cfg->n_reactions);
  o->comp.assign(cfg->compartments, cfg->compartments + cfg->n_compartments);
  o->tables.assign(cfg->tables, cfg->tables + ((size_t)cfg->n_sigma_classes << cfg->table_bits));
  o->cfg.species = nullptr; o->cfg.reactions = nullptr; o->cfg.compartments = nullptr; o->cfg.tables = nullptr;
  o->rxmap.assign((size_t)cfg->n_species * cfg->n_species, -1);
  o->binds.assign(cfg->n_species, 0);
  for (uint32_t e = 0; e < cfg->n_reactions; ++e) {
    const orc_reaction_t& r = o->rx[e];
    o->rxmap[(size_t)r.a * cfg->n_species + r.b] = (int)e;
    o->rxmap[(size_t)r.b * cfg->n_species + r.a] = (int)e;
    o->binds[r.a] = o->binds[r.b] = 1;
  }
  o->counts.assign((size_t)cfg->counts_rows * cfg->n_replicas * cfg->n_species, 0);
  o->t_first.assign(std::max<uint32_t>(cfg->n_rules, 1), NEVER);
  o->key[0] = (uint32_t)cfg->seed; o->key[1] = (uint32_t)(cfg->seed >> 32);
  *out = o;
  return ORC_OK;
}

void oracle_destroy(oracle_t* o) { delete o; }

int oracle_set_mode(oracle_t* o, int mode) {
  if (!o || (mode != ORC_MODE_GRID && mode != ORC_MODE_BRUTE)) return ORC_E_INVAL;
  o->mode = mode;
  return ORC_OK;
}

// Seeding (S15): ids in record order; position from the PLACE stream keyed by the
// placement seed: counter (id, attempt, 0, 5).
int oracle_seed_population(oracle_t* o, const orc_seed_rec_t* recs, uint32_t n_recs, uint64_t place_seed) {
  if (!o || (!recs && n_recs)) return ORC_E_INVAL;
  uint64_t total = 0;
  for (uint32_t i = 0; i < n_recs; ++i) {
    if (recs[i].species >= o->cfg.n_species || recs[i].replica >= o->cfg.n_replicas) return ORC_E_INVAL;
    total += recs[i].count;
  }
  if (o->ag.size() + total > o->cfg.capacity) return ORC_E_CAPACITY;
  if ((uint64_t)o->next_id + total > o->cfg.id_capacity) return ORC_E_IDSPACE;
  const uint32_t pkey[2] = {(uint32_t)place_seed, (uint32_t)(place_seed >> 32)};
  for (uint32_t i = 0; i < n_recs; ++i) {
    const orc_compartment_t& c = o->comp[o->sp[recs[i].species].compartment];
    int32_t base = (int32_t)((uint32_t)recs[i].replica << o->cfg.stride_shift);
    for (uint32_t n = 0; n < recs[i].count; ++n) {
      Agent a; a.id = o->next_id++; a.s = recs[i].species;
      if (c.shape == ORC_SHAPE_CUBE) {
        uint32_t ctr[4] = {a.id, 0, 0, TAG_PLACE}, r[4];
        philox(ctr, pkey, r);
        a.x = (int32_t)(((uint64_t)r[0] * (uint32_t)c.L) >> 32);
        a.y = (int32_t)(((uint64_t)r[1] * (uint32_t)c.L) >> 32);
        a.z = (int32_t)(((uint64_t)r[2] * (uint32_t)c.L) >> 32);
      } else {
        uint32_t side = 2u * (uint32_t)c.r_out + 1u;
        a.x = c.cx + c.r_out; a.y = c.cy; a.z = c.cz;   // fixed valid fallback point
        for (uint32_t attempt = 0; attempt < 64; ++attempt) {
          uint32_t ctr[4] = {a.id, attempt, 0, TAG_PLACE}, r[4];
          philox(ctr, pkey, r);
          int32_t qx = c.cx - c.r_out + (int32_t)(((uint64_t)r[0] * side) >> 32);
          int32_t qy = c.cy - c.r_out + (int32_t)(((uint64_t)r[1] * side) >> 32);
          int32_t qz = c.cz - c.r_out + (int32_t)(((uint64_t)r[2] * side) >> 32);
          if (o->valid(c, qx, qy, qz)) { a.x = qx; a.y = qy; a.z = qz; break; }
        }
      }
      a.x += base;
      o->ag.push_back(a);
    }
  }
  o->write_counts_row(o->t);   // S22: row t = state after t steps
  return ORC_OK;
}

int oracle_step(oracle_t* o, uint32_t n_steps) {
  if (!o) return ORC_E_INVAL;
  if (o->err) return o->err;
  for (uint32_t i = 0; i < n_steps; ++i) {
    int e = o->step_once();
    if (e) { o->err = e; return e; }
  }
  return ORC_OK;
}

int oracle_read_counts(oracle_t* o, uint32_t first_row, uint32_t n_rows, uint32_t* out) {
  if (!o || !out || (uint64_t)first_row + n_rows > (uint64_t)o->t + 1) return ORC_E_INVAL;
  size_t w = (size_t)o->cfg.n_replicas * o->cfg.n_species;
  std::memcpy(out, &o->counts[first_row * w], (size_t)n_rows * w * sizeof(uint32_t));
  return ORC_OK;
}

int oracle_read_agents(oracle_t* o, uint32_t cap, int32_t* x, int32_t* y, int32_t* z,
                       uint16_t* species, uint32_t* id, uint32_t* n_out) {
  if (!o || !n_out) return ORC_E_INVAL;
  *n_out = (uint32_t)o->ag.size();
  if (cap < o->ag.size()) return ORC_E_CAPACITY;
  std::vector<Agent> s(o->ag);
  std::sort(s.begin(), s.end(), [](const Agent& a, const Agent& b) { return a.id < b.id; });
  for (size_t i = 0; i < s.size(); ++i) {
    if (x) x[i] = s[i].x; if (y) y[i] = s[i].y; if (z) z[i] = s[i].z;
    if (species) species[i] = s[i].s; if (id) id[i] = s[i].id;
  }
  return ORC_OK;
}

int oracle_load_agents(oracle_t* o, uint32_t n, const int32_t* x, const int32_t* y, const int32_t* z,
                       const uint16_t* species, const uint32_t* id, uint32_t step, uint32_t next_id) {
  if (!o || n > o->cfg.capacity || step >= o->cfg.counts_rows || next_id > o->cfg.id_capacity) return ORC_E_INVAL;
  o->ag.resize(n);
  for (uint32_t i = 0; i < n; ++i) {
    if (species[i] >= o->cfg.n_species || id[i] >= next_id) return ORC_E_INVAL;
    o->ag[i] = Agent{x[i], y[i], z[i], species[i], id[i]};
  }
  o->t = step; o->next_id = next_id; o->err = ORC_OK;
  o->write_counts_row(step);
  return ORC_OK;
}

int oracle_info(oracle_t* o, uint32_t* n_live, uint32_t* step, uint32_t* next_id, uint32_t* t_first0) {
  if (!o) return ORC_E_INVAL;
  if (n_live) *n_live = (uint32_t)o->ag.size();
  if (step) *step = o->t;
  if (next_id) *next_id = o->next_id;
  if (t_first0) *t_first0 = o->t_first[0];
  return ORC_OK;
}

// Order-independent 64-bit checksum of the live state (DESIGN.md §1 "Checksum"):
// sum over live agents, modulo 2^64, of h = mix(mix(mix(x | y << 32) ^ (z | id << 32)) ^ species) with the
// coordinates taken as 32-bit patterns and mix = the splitmix64 finaliser written out below.
static uint64_t mix64(uint64_t v) {
  v ^= v >> 30; v *= 0xBF58476D1CE4E5B9ull;
  v ^= v >> 27; v *= 0x94D049BB133111EBull;
  v ^= v >> 31;
  return v;
}
int oracle_read_checksum(oracle_t* o, uint64_t* out) {
  if (!o || !out) return ORC_E_INVAL;
  uint64_t sum = 0;
  for (const Agent& a : o->ag) {
    uint64_t lo = (uint64_t)(uint32_t)a.x | ((uint64_t)(uint32_t)a.y << 32);
    uint64_t hi = (uint64_t)(uint32_t)a.z | ((uint64_t)a.id << 32);
    sum += mix64(mix64(mix64(lo) ^ hi) ^ (uint64_t)a.s);
  }
  *out = sum;
  return ORC_OK;
}

// Checkpoint state beyond the agents (state = agents, t, next_id, t_first[]): the first-firing
// steps of the delayed rules (S17).  n must equal the model's n_rules.
int oracle_read_t_first(oracle_t* o, uint32_t n, uint32_t* out) {
  if (!o || !out || n != o->cfg.n_rules) return ORC_E_INVAL;
  for (uint32_t r = 0; r < n; ++r) out[r] = o->t_first[r];
  return ORC_OK;
}
int oracle_load_t_first(oracle_t* o, uint32_t n, const uint32_t* in) {
  if (!o || !in || n != o->cfg.n_rules) return ORC_E_INVAL;
  for (uint32_t r = 0; r < n; ++r) o->t_first[r] = in[r];
  return ORC_OK;
}

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox(ctr, key, out); }

int oracle_debug_move_only(oracle_t* o) { if (!o) return ORC_E_INVAL; o->phase_move(); return ORC_OK; }

static std::vector<uint32_t> id_order(const oracle* o) {
  std::vector<uint32_t> ord(o->ag.size());
  for (size_t i = 0; i < ord.size(); ++i) ord[i] = (uint32_t)i;
  std::sort(ord.begin(), ord.end(), [&](uint32_t a, uint32_t b) { return o->ag[a].id < o->ag[b].id; });
  return ord;
}

int oracle_debug_proposals(oracle_t* o, int mode, uint32_t* out) {
  if (!o || !out) return ORC_E_INVAL;
  std::vector<uint32_t> prop;
  o->compute_proposals(mode, prop);
  std::vector<uint32_t> ord = id_order(o);
  for (size_t r = 0; r < ord.size(); ++r) {
    uint32_t j = prop[ord[r]];
    out[r] = j == NOPROP ? NOPROP : o->ag[j].id;
  }
  return ORC_OK;
}

int oracle_debug_pairs(oracle_t* o, int mode, uint32_t cap_pairs, uint32_t* pairs_out, uint32_t* n_pairs) {
  if (!o || !n_pairs) return ORC_E_INVAL;
  if (mode == ORC_MODE_GRID) o->build_grid();
  std::vector<std::pair<uint32_t, uint32_t>> pr;
  for (size_t i = 0; i < o->ag.size(); ++i)
    o->for_candidates(i, mode, [&](size_t j) {
      if (o->ag[i].id < o->ag[j].id && o->in_range_reaction(o->ag[i], o->ag[j]) >= 0)
        pr.push_back({o->ag[i].id, o->ag[j].id});
    });
  std::sort(pr.begin(), pr.end());
  *n_pairs = (uint32_t)pr.size();
  if (pr.size() > cap_pairs) return ORC_E_CAPACITY;
  for (size_t k = 0; k < pr.size(); ++k) { pairs_out[2 * k] = pr[k].first; pairs_out[2 * k + 1] = pr[k].second; }
  return ORC_OK;
}

}  // extern "C"
