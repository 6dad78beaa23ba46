// molsim.cu — host side of the C ABI declared in include/molsim.h.
// Product code (CUDA path): validation, workspace carving, launch sequencing.  Every step of the
// hot path runs in the kernels of kernels.cuh; there is no CPU fallback.
#include "../../include/molsim.h"
#include "kernels.cuh"
#include "readout.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

using namespace molsim;

namespace {

constexpr uint32_t kMaxScanBlocks = 592;  // 148 SMs x 4; small problems get proportionally smaller grids (launch-bound)
constexpr uint32_t kMaxTailBlocks = 148;

enum KernelId { KI_HIST = 0, KI_CELL_ZERO, KI_CELL_REDUCE, KI_CELL_SCAN, KI_SCATTER, KI_PAIRS,
                KI_RESOLVE, KI_UNI_HIST, KI_BIRTHS, KI_OTHER };
const char* kKernelNames[SIM_N_KERNELS] = {
    "k_hist_prologue", "memset_cells", "k_cell_reduce", "k_cell_scan", "k_scatter", "k_pairs",
    "k_resolve", "k_uni_hist", "k_births", "other"};

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
  size_t soa[2][2], prop, best, hasprop, cell[2], partial, bits, birth_mid, birth_top, birth_list, counts,
      scal, tab, gauss, total;
  uint32_t n_cells, nx, ny, nz;
};

bool make_layout(const sim_config_t* c, Layout& L) {
  const uint64_t cs = c->cell_size;
  const uint64_t nx = (c->extent[0] + cs - 1) / cs, ny = (c->extent[1] + cs - 1) / cs, nz = (c->extent[2] + cs - 1) / cs;
  const uint64_t nc = nx * ny * nz;
  if (nc == 0 || nc >= (1ull << 30) - 8 || nx >= (1ull << 30)) return false;   // K4 packs a cell index into 30 bits
  L.nx = (uint32_t)nx; L.ny = (uint32_t)ny; L.nz = (uint32_t)nz; L.n_cells = (uint32_t)nc;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  const size_t cap = c->capacity;
  // records, species; the slack covers the tile (+ halo) that K4's bulk copies read past the last slot
  for (int b = 0; b < 2; ++b) { L.soa[b][0] = take(cap * 16 + (kPairThreads + kPairHalo) * 16); L.soa[b][1] = take(cap * 2 + kPairThreads * 2); }
  L.prop = take(cap * 4);
  L.best = take(cap * 8);
  L.hasprop = take((cap / 32 + 16) * 4);
  // two cell arrays (this step's and the next step's histogram); 4 words of lead so that the counts, which start one
  // word behind the leading zero, are 16-byte aligned; slack for the look-ups K4 makes past the last row
  for (int b = 0; b < 2; ++b) L.cell[b] = take(((size_t)nc + 8 + 1024) * 4);
  L.partial = take(4096 * 4);
  const size_t n_chunks = ((size_t)c->id_capacity + 63) / 64 + 1;
  L.bits = take(n_chunks * 8 * 4);
  L.birth_mid = take((((size_t)c->id_capacity >> kMidShift) + 2) * 4);
  L.birth_top = take((size_t)kMaxTop * 4);
  L.birth_list = take(cap * 8);
  L.counts = take(((size_t)c->counts_rows + 2) * c->n_replicas * c->n_species * 4);
  L.scal = take(sizeof(Scalars));
  L.tab = take(sizeof(DevTables));
  L.gauss = take(((size_t)c->n_sigma_classes << c->table_bits) * 2);
  L.total = o;
  return true;
}

// Table validation: the in-scope part of the paper's consistency checker ("missing reciprocal
// reactions, references to undefined species ... inconsistencies between specified volume and concentration") plus
// the bounds the kernels rely on.  Written from the rule list in include/molsim.h ("Table validation", V1-V7), rule
// by rule; returns the name of the first rule that fails, or nullptr.  tests/test_validation_rules.py states every
// rule and checks that this checker and the oracle's (written from DESIGN.md, separately) both enforce it.
struct ConfigCheck {
  const sim_config_t& c;
  explicit ConfigCheck(const sim_config_t& cfg) : c(cfg) {}

  // largest displacement of any mobile class, and the largest interaction radius (ceil sqrt of the largest r2)
  int64_t max_step() const {
    int64_t m = 0;
    const size_t n = (size_t)1 << c.table_bits;
    for (uint32_t cls = 1; cls < c.n_sigma_classes; ++cls)
      for (size_t k = 0; k < n; ++k) m = std::max<int64_t>(m, std::llabs((long long)c.tables[cls * n + k]));
    return m;
  }
  int64_t max_radius() const {
    uint64_t r2 = 0;
    for (uint32_t e = 0; e < c.n_reactions; ++e) r2 = std::max<uint64_t>(r2, c.reactions[e].r2);
    int64_t r = (int64_t)std::sqrt((double)r2);
    while ((uint64_t)r * (uint64_t)r < r2) ++r;
    while (r > 0 && (uint64_t)(r - 1) * (uint64_t)(r - 1) >= r2) --r;
    return r;
  }
  int64_t tile_width() const { return c.n_replicas > 1 ? ((int64_t)1 << c.stride_shift) : (int64_t)c.extent[0]; }
  bool species_ok(uint32_t s) const { return s < c.n_species; }
  bool same_compartment(uint32_t s, uint32_t other) const {
    return species_ok(other) && c.species[other].compartment == c.species[s].compartment;
  }

  const char* limits() const {                                                    // V1, V2
    if (!c.species || !c.compartments || !c.tables || (c.n_reactions && !c.reactions)) return "V1 table pointer missing";
    if (c.n_species < 1 || c.n_species > SIM_MAX_SPECIES) return "V2 n_species outside 1..SIM_MAX_SPECIES";
    if (c.n_reactions > SIM_MAX_REACTIONS) return "V2 n_reactions above SIM_MAX_REACTIONS";
    if (c.n_compartments < 1 || c.n_compartments > SIM_MAX_COMPARTMENTS) return "V2 n_compartments outside 1..SIM_MAX_COMPARTMENTS";
    if (c.n_rules > SIM_MAX_RULES) return "V2 n_rules above SIM_MAX_RULES";
    if (c.table_bits < 1 || c.table_bits > 16) return "V2 table_bits outside 1..16";
    if (c.n_sigma_classes < 1 || c.n_sigma_classes > 255) return "V2 n_sigma_classes outside 1..255";
    if (c.n_replicas < 1 || c.n_replicas > SIM_MAX_REPLICAS || c.stride_shift > 31) return "V2 replica tiling outside its limits";
    if (c.cell_size < 2 || c.cell_size > 16384) return "V2 cell_size outside 2..16384";
    if (c.capacity < 1 || c.capacity > 0x7FFFFFFFu || c.id_capacity < 1 || c.counts_rows < 1) return "V2 capacity / id_capacity / counts_rows";
    for (int a = 0; a < 3; ++a) if (c.extent[a] <= 0) return "V2 extent not positive";
    return nullptr;
  }
  const char* tiling() const {                                                    // V3
    const uint64_t span = (uint64_t)c.n_replicas << c.stride_shift;
    if (c.n_replicas > 1 && span > 0x80000000ull) return "V3 replica tiles do not fit int32";
    if ((uint64_t)c.extent[0] > span) return "V3 extent[0] wider than the replica tiles";
    return nullptr;
  }
  const char* geometry() const {                                                  // V4
    const int64_t step = max_step(), reach = max_radius(), tile = tile_width();
    for (uint32_t k = 0; k < c.n_compartments; ++k) {
      const sim_compartment_t& g = c.compartments[k];
      int64_t lo[3], hi[3];                       // bounding box in local coordinates, hi exclusive
      if (g.shape == SIM_SHAPE_CUBE) {
        if (g.L <= 0) return "V4 cube edge not positive";
        if (step >= g.L) return "V4 a displacement table entry reaches across the cube (one mirror reflection must suffice)";
        for (int a = 0; a < 3; ++a) { lo[a] = 0; hi[a] = g.L; }
      } else if (g.shape == SIM_SHAPE_SPHERE) {
        if (g.r_out <= 0 || g.r_in >= g.r_out) return "V4 sphere radii (need 0 < r_out and r_in < r_out)";
        const int64_t ctr[3] = {g.cx, g.cy, g.cz};
        for (int a = 0; a < 3; ++a) { lo[a] = ctr[a] - g.r_out; hi[a] = ctr[a] + g.r_out + 1; }
      } else {
        return "V4 unknown compartment shape";
      }
      if (lo[0] < 0 || lo[1] < 0 || lo[2] < 0) return "V4 compartment reaches below 0";
      if (hi[1] > c.extent[1] || hi[2] > c.extent[2]) return "V4 compartment reaches beyond extent (y / z)";
      if (hi[0] > tile) return "V4 compartment reaches beyond its tile / extent (x)";
      if (c.n_replicas > 1 && hi[0] + reach > tile) return "V4 replicas closer than the largest interaction radius";
    }
    return nullptr;
  }
  const char* species() const {                                                   // V5, V6
    for (uint32_t s = 0; s < c.n_species; ++s) {
      const sim_species_t& sp = c.species[s];
      if (sp.sigma_class >= c.n_sigma_classes) return "V5 sigma_class out of range";
      if (sp.compartment >= c.n_compartments) return "V5 compartment out of range";
      if (sp.n_channels > SIM_MAX_CHANNELS) return "V5 more than SIM_MAX_CHANNELS channels";
      if (sp.cross_to != SIM_NONE16) {
        if (!species_ok(sp.cross_to)) return "V5 cross_to is not a species";
        const uint32_t there = c.species[sp.cross_to].compartment;
        if (there >= c.n_compartments || there == sp.compartment) return "V5 cross_to lives in the same compartment";
        if (c.compartments[there].shape != SIM_SHAPE_SPHERE || c.compartments[sp.compartment].shape != SIM_SHAPE_SPHERE)
          return "V5 membrane crossing needs spherical compartments";
      }
      for (uint32_t k = 0; k < sp.n_channels; ++k) {
        const sim_channel_t& ch = sp.ch[k];
        switch (ch.kind) {
          case SIM_CH_NONE: case SIM_CH_DEGRADE: break;
          case SIM_CH_CONVERT:
            if (!same_compartment(s, ch.prod0)) return "V6 product 0 missing or in another compartment";
            break;
          case SIM_CH_RELEASE:
            if (!same_compartment(s, ch.prod0)) return "V6 product 0 missing or in another compartment";
            if (!same_compartment(s, ch.prod1)) return "V6 product 1 missing or in another compartment";
            break;
          case SIM_CH_BIRTH: case SIM_CH_DELAYED_BIRTH:
            if (!same_compartment(s, ch.prod1)) return "V6 product 1 missing or in another compartment";
            break;
          default: return "V6 unknown channel kind";
        }
        if ((ch.kind == SIM_CH_DELAYED_BIRTH || ch.marks_first) && ch.rule >= c.n_rules) return "V6 rule slot out of range";
        if (ch.kind == SIM_CH_DELAYED_BIRTH && ch.thr < 1) return "V6 delay of a delayed birth below one step";
      }
    }
    return nullptr;
  }
  const char* reactions() const {                                                 // V7
    const uint64_t cell2 = (uint64_t)c.cell_size * c.cell_size;
    std::vector<uint8_t> seen((size_t)c.n_species * c.n_species, 0);
    for (uint32_t e = 0; e < c.n_reactions; ++e) {
      const sim_reaction_t& r = c.reactions[e];
      if (!species_ok(r.a) || !species_ok(r.b) || !species_ok(r.cplx)) return "V7 reaction names an undefined species";
      if (!same_compartment(r.a, r.b) || !same_compartment(r.a, r.cplx)) return "V7 reactants and complex in different compartments";
      if ((uint64_t)r.r2 > cell2) return "V7 interaction radius above the cell size";
      uint8_t& ab = seen[(size_t)std::min(r.a, r.b) * c.n_species + std::max(r.a, r.b)];
      if (ab) return "V7 two reactions for the same pair of species";
      ab = 1;
    }
    return nullptr;
  }
  const char* run() const {
    const char* why = limits();
    if (!why) why = tiling();
    if (!why) why = species();
    if (!why) why = reactions();
    if (!why) why = geometry();
    return why;
  }
};

const char* check_config(const sim_config_t* c) { return c ? ConfigCheck(*c).run() : "V1 no configuration"; }
int validate(const sim_config_t* c) { return check_config(c) ? SIM_E_INVAL : SIM_OK; }

}  // namespace

struct sim {
  sim_config_t cfg;
  Layout lay;
  Params prm;         // prm.cur / prm.oth always describe the CURRENT parity
  char* ws = nullptr;
  cudaStream_t stream = nullptr;   // the caller's stream: everything executes here
  cudaStream_t run = nullptr;      // where enqueue_step puts its launches: `stream`, or `cap` while a graph is captured
  cudaStream_t cap = nullptr;      // private stream used only to CAPTURE the step graphs (never executes work)
  cudaGraphExec_t g1[2] = {nullptr, nullptr}, g8[2] = {nullptr, nullptr};   // 1 / 8 steps, by starting parity
  bool graphs_tried = false, graphs_ok = false;
  uint32_t kernels_per_step = 0;
  uint32_t t_host = 0;           // steps enqueued so far (the host knows t exactly)
  uint64_t launches = 0;
  int gauss_in_smem = 0;
  void (*k_scat)(Params) = nullptr;   // K3 / K5 / prologue instantiations picked at create time (Gaussian tables in
  void (*k_unih)(Params) = nullptr;   // shared memory or not; small- or large-population launch shape)
  void (*k_hist)(Params) = nullptr;
  uint32_t k3_unroll = 0;
  size_t gauss_bytes = 0, unih_smem = 0;
  uint32_t grid_scatter = 0, grid_pairs = 0, grid_unih = 0, grid_resolve = 0;
  bool hist_valid = false;            // prm.cell holds the histogram of the current state for the current step
  cudaStream_t side = nullptr;        // zeroes the next cell array beside K3 / K4 (a parallel branch of the step graph)
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  uint32_t cell_seg = 0, scan_blocks = 1, tail_blocks = 1;
  bool profile = false;
  float prof_ms[SIM_N_KERNELS] = {};
  uint32_t prof_n[SIM_N_KERNELS] = {};
  std::vector<std::pair<int, std::pair<cudaEvent_t, cudaEvent_t>>> prof_pending;
  std::string cuda_err;
  int sticky = SIM_OK;

  int cuda_fail(cudaError_t e, const char* where) {
    cuda_err = std::string(where) + ": " + cudaGetErrorString(e);
    return SIM_E_CUDA;
  }
};

#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return s->cuda_fail(e_, #call); } while (0)

namespace {

struct ProfScope {
  sim* s; int k; bool is_kernel; cudaEvent_t a = nullptr, b = nullptr;
  ProfScope(sim* s_, int k_, bool is_kernel_ = true) : s(s_), k(k_), is_kernel(is_kernel_) {
    if (s->profile) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, s->run); }
  }
  ~ProfScope() {
    if (is_kernel) s->launches++;   // memsets are not kernels of ours
    if (s->profile) { cudaEventRecord(b, s->run); s->prof_pending.push_back({k, {a, b}}); }
  }
};

void prof_collect(sim* s) {
  for (auto& pe : s->prof_pending) {
    float ms = 0.f;
    cudaEventSynchronize(pe.second.second);
    cudaEventElapsedTime(&ms, pe.second.first, pe.second.second);
    s->prof_ms[pe.first] += ms; s->prof_n[pe.first]++;
    cudaEventDestroy(pe.second.first); cudaEventDestroy(pe.second.second);
  }
  s->prof_pending.clear();
}

int read_scalars(sim* s, Scalars* out) {
  CK(cudaMemcpyAsync(out, s->prm.scal, sizeof(Scalars), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

int err_from_bits(uint32_t bits) {
  if (bits & 8u) return SIM_E_INTERNAL;
  if (bits & 4u) return SIM_E_INVAL;
  if (bits & 1u) return SIM_E_CAPACITY;
  if (bits & 2u) return SIM_E_IDSPACE;
  return SIM_OK;
}

// counts row r <- histogram of the current state; row r+1 <- copy (base of the next step's deltas)
int recount_row(sim* s, uint32_t r, uint32_t n_slots, bool check = false) {
  CK(cudaMemsetAsync(s->prm.counts + (size_t)r * s->prm.row_width, 0, (size_t)s->prm.row_width * 4, s->stream));
  if (n_slots) {
    ProfScope ps(s, KI_OTHER);
    k_count_row<<<std::min<uint32_t>((n_slots + 255) / 256, 148 * 8), 256, 0, s->stream>>>(s->prm, r, n_slots, check);
    if (check) k_clear_ids<<<std::min<uint32_t>((n_slots + 255) / 256, 148 * 8), 256, 0, s->stream>>>(s->prm, n_slots);
  }
  { ProfScope ps(s, KI_OTHER); k_copy_row<<<1, 256, 0, s->stream>>>(s->prm, r); }
  CK(cudaGetLastError());
  return SIM_OK;
}

// Histogram of the CURRENT arrays for the current step (after seeding / loading; a step leaves the next one's behind).
int enqueue_prologue(sim* s) {
  Params& p = s->prm;
  CK(cudaMemsetAsync(p.cell - 3, 0, ((size_t)p.n_cells + 8) * 4, s->stream));
  { ProfScope ps(s, KI_HIST);
    s->k_hist<<<s->grid_unih, kUniThreads, s->gauss_in_smem ? s->gauss_bytes : 0, s->stream>>>(p); }
  CK(cudaGetLastError());
  s->hist_valid = true;
  return SIM_OK;
}

int enqueue_step(sim* s) {
  Params& p = s->prm;
  // the next step's cell array is zeroed on the side stream while K2 .. K4b run (its last readers were the previous step's)
  CK(cudaEventRecord(s->ev_fork, s->run));
  CK(cudaStreamWaitEvent(s->side, s->ev_fork, 0));
  CK(cudaMemsetAsync(p.cell_next - 3, 0, ((size_t)p.n_cells + 8) * 4, s->side));
  CK(cudaEventRecord(s->ev_join, s->side));
  { ProfScope ps(s, KI_CELL_REDUCE);
    k_cell_reduce<<<s->scan_blocks, kScanThreads, 0, s->run>>>(p.cell + 1, p.n_cells, s->cell_seg, p.partial); }
  { ProfScope ps(s, KI_CELL_SCAN);
    k_cell_scan<<<s->scan_blocks, kScanThreads, 0, s->run>>>(p.cell + 1, p.n_cells, s->cell_seg, p.partial); }
  { ProfScope ps(s, KI_SCATTER);
    s->k_scat<<<s->grid_scatter, kMoveThreads, s->gauss_in_smem ? s->gauss_bytes : 0, s->run>>>(p); }
  { ProfScope ps(s, KI_PAIRS); k_pairs<<<s->grid_pairs, kPairBlock, 0, s->run>>>(p); }
  { ProfScope ps(s, KI_RESOLVE); k_resolve<<<s->grid_resolve, 256, 0, s->run>>>(p); }
  CK(cudaStreamWaitEvent(s->run, s->ev_join, 0));
  { ProfScope ps(s, KI_UNI_HIST); s->k_unih<<<s->grid_unih, kUniThreads, s->unih_smem, s->run>>>(p); }
  { ProfScope ps(s, KI_BIRTHS); k_births<<<s->tail_blocks, kScanThreads, 0, s->run>>>(p); }
  CK(cudaGetLastError());
  std::swap(p.cur, p.oth);   // the sorted copy (+ newborns) is the next step's current state,
  std::swap(p.cell, p.cell_next);   // and its histogram has been taken
  s->t_host++;
  return SIM_OK;
}

}  // namespace

namespace {

constexpr uint32_t kGraphSteps = 8;   // even, so the parity after the graph equals the parity before

void flip(sim* s) { std::swap(s->prm.cur, s->prm.oth); std::swap(s->prm.cell, s->prm.cell_next); }
int parity_of(const sim* s) { return s->prm.cur.r == (const int4*)(s->ws + s->lay.soa[0][0]) ? 0 : 1; }

// Captures `steps` steps starting at the current parity into an executable graph; the handle's
// host-side state is restored afterwards (capturing executes nothing).
bool capture_steps(sim* s, uint32_t steps, cudaGraphExec_t* out) {
  const Params saved = s->prm;
  const uint64_t launches = s->launches;
  const uint32_t t_host = s->t_host;
  cudaGraph_t graph = nullptr;
  bool ok = cudaStreamBeginCapture(s->cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    s->run = s->cap;
    for (uint32_t k = 0; k < steps && ok; ++k) ok = enqueue_step(s) == SIM_OK;
    s->run = s->stream;
    ok = (cudaStreamEndCapture(s->cap, &graph) == cudaSuccess) && ok && graph;
  }
  if (ok) ok = cudaGraphInstantiate(out, graph, 0) == cudaSuccess;
  if (graph) cudaGraphDestroy(graph);
  if (ok) s->kernels_per_step = (uint32_t)((s->launches - launches) / steps);
  s->prm = saved; s->launches = launches; s->t_host = t_host;
  if (!ok) cudaGetLastError();
  return ok;
}

// The 7 launches (+ the memset branch) of a step are replayed as CUDA graphs (one step, or 8 steps, per starting parity of
// the cur/oth ping-pong): the path is launch-bound below ~1 M agents.
void build_graphs(sim* s) {
  s->graphs_tried = true;
  if (cudaStreamCreateWithFlags(&s->cap, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return; }
  const Params saved = s->prm;
  bool ok = true;
  for (int k = 0; k < 2 && ok; ++k) {
    const int par = parity_of(s);
    ok = capture_steps(s, 1, &s->g1[par]) && capture_steps(s, kGraphSteps, &s->g8[par]);
    flip(s);   // the other parity (flipped back by the second round)
  }
  s->prm = saved;   // a capture that fails in the first round must not leave the ping-pong flipped for the direct launches
  s->graphs_ok = ok;
}

}  // namespace

namespace {
// Launch shapes of the two passes that evaluate the move: agents in flight per thread x resident blocks per SM
// (K3), resident blocks per SM (K5 / prologue); small populations like many thin blocks.
template <bool kGauss> void pick_move_kernels(sim* s, bool large) {
  s->k_scat = k_scatter<kGauss, 2, 5>; (void)large;
  s->k3_unroll = 2;
  s->k_unih = k_uni_hist<kGauss, true, 5>;
  s->k_hist = k_uni_hist<kGauss, false, 5>;
}
}  // namespace

extern "C" {

size_t sim_workspace_bytes(const sim_config_t* cfg) {
  Layout L;
  if (validate(cfg) != SIM_OK || !make_layout(cfg, L)) return 0;
  return L.total;
}

int sim_create(const sim_config_t* cfg, void* d_workspace, size_t workspace_bytes, void* cuda_stream, sim_t** out) {
  if (!out) return SIM_E_INVAL;
  *out = nullptr;
  int v = validate(cfg);
  if (v) return v;
  Layout L;
  if (!make_layout(cfg, L)) return SIM_E_INVAL;
  if (!d_workspace || workspace_bytes < L.total || ((uintptr_t)d_workspace & 255u)) return SIM_E_INVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return SIM_E_CUDA;

  sim* s = new sim();
  s->cfg = *cfg;
  s->cfg.species = nullptr; s->cfg.reactions = nullptr; s->cfg.compartments = nullptr; s->cfg.tables = nullptr;
  s->lay = L;
  s->ws = (char*)d_workspace;
  s->stream = (cudaStream_t)cuda_stream;
  s->run = s->stream;
  if (cudaStreamCreateWithFlags(&s->side, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming) != cudaSuccess) { sim_destroy(s); return SIM_E_CUDA; }

  // host image of the device tables
  std::vector<DevTables> tabv(1);
  DevTables& T = tabv[0];
  std::memset(&T, 0, sizeof(T));
  std::memset(T.rxmap, 0xFF, sizeof(T.rxmap));
  uint32_t max_r2 = 0;
  for (uint32_t e = 0; e < cfg->n_reactions; ++e) {
    const sim_reaction_t& r = cfg->reactions[e];
    T.rx[e] = DevRx{r.a, r.b, r.cplx, 0, r.r2, r.thr};
    T.rxmap[r.a * kMaxSpecies + r.b] = (uint8_t)e;
    T.rxmap[r.b * kMaxSpecies + r.a] = (uint8_t)e;
    max_r2 = std::max(max_r2, r.r2);
  }
  for (uint32_t i = 0; i < cfg->n_species; ++i) {
    const sim_species_t& a = cfg->species[i];
    DevSpecies& d = T.sp[i];
    d.sigma_class = (uint8_t)a.sigma_class; d.compartment = (uint8_t)a.compartment;
    d.n_channels = (uint8_t)a.n_channels; d.cross_to = a.cross_to; d.cross_thr = a.cross_thr;
    d.binds = 0;
    for (uint32_t e = 0; e < cfg->n_reactions; ++e)
      if (cfg->reactions[e].a == i || cfg->reactions[e].b == i) d.binds = 1;
    for (uint32_t k = 0; k < a.n_channels; ++k) {
      const sim_channel_t& c = a.ch[k];
      d.ch[k] = DevChannel{(uint8_t)c.kind, (uint8_t)c.rule, (uint8_t)(c.marks_first ? 1 : 0), 0, c.prod0, c.prod1, c.thr};
    }
  }
  for (uint32_t i = 0; i < cfg->n_compartments; ++i) {
    const sim_compartment_t& a = cfg->compartments[i];
    DevComp& d = T.comp[i];
    d.shape = (int32_t)a.shape; d.cx = a.cx; d.cy = a.cy; d.cz = a.cz; d.L = a.L; d.r_out = a.r_out; d.r_in = a.r_in;
    d.r_out2 = (long long)a.r_out * a.r_out;
    d.r_in2 = a.r_in < 0 ? -1ll : (long long)a.r_in * a.r_in;
  }

  Params& p = s->prm;
  std::memset(&p, 0, sizeof(p));
  char* w = s->ws;
  auto soa = [&](int b) { return Soa{(int4*)(w + L.soa[b][0]), (uint16_t*)(w + L.soa[b][1])}; };
  p.cur = soa(0); p.oth = soa(1);
  p.prop = (uint32_t*)(w + L.prop); p.hasprop = (uint32_t*)(w + L.hasprop);
  p.best = (unsigned long long*)(w + L.best);
  p.cell = (uint32_t*)(w + L.cell[0]) + 3; p.cell_next = (uint32_t*)(w + L.cell[1]) + 3;   // cell[1] is 16-byte aligned
  p.partial = (uint32_t*)(w + L.partial);
  p.bits = (uint32_t*)(w + L.bits); p.birth_mid = (uint32_t*)(w + L.birth_mid); p.birth_top = (uint32_t*)(w + L.birth_top);
  p.birth_list = (uint2*)(w + L.birth_list); p.counts = (uint32_t*)(w + L.counts);
  p.scal = (Scalars*)(w + L.scal); p.tab = (const DevTables*)(w + L.tab); p.gauss = (const int16_t*)(w + L.gauss);
  p.key0 = (uint32_t)cfg->seed; p.key1 = (uint32_t)(cfg->seed >> 32);
  for (uint32_t r = 0; r < 10; ++r) { p.rk0[r] = p.key0 + r * 0x9E3779B9u; p.rk1[r] = p.key1 + r * 0xBB67AE85u; }
  p.capacity = cfg->capacity; p.id_capacity = cfg->id_capacity;
  p.n_species = cfg->n_species; p.n_replicas = cfg->n_replicas; p.stride_shift = cfg->stride_shift;
  p.table_bits = cfg->table_bits; p.n_classes = cfg->n_sigma_classes;
  p.cell_size = (int32_t)cfg->cell_size;
  {
    uint32_t l = 0;
    while ((1ull << l) < cfg->cell_size) ++l;                       // l = ceil(log2 cell_size)
    p.cell_mshift = l - 1u;                                          // cell_size >= 2 (validated), so l >= 1
    p.cell_magic = (uint32_t)((1ull << (31u + l)) / cfg->cell_size + 1ull);
  }
  for (uint32_t i = 0; i < cfg->n_species; ++i) {
    if (T.sp[i].binds) p.binds_mask |= 1ull << i;
    if (T.sp[i].n_channels) p.chan_mask |= 1ull << i;
  }
  p.nx = (int32_t)L.nx; p.ny = (int32_t)L.ny; p.nz = (int32_t)L.nz; p.n_cells = L.n_cells;
  p.fwd_row[0] = p.nx; p.fwd_row[1] = (p.ny - 1) * p.nx; p.fwd_row[2] = p.ny * p.nx; p.fwd_row[3] = (p.ny + 1) * p.nx;
  p.max_r2 = max_r2;
  p.max_r = (int32_t)std::ceil(std::sqrt((double)max_r2));
  while ((uint64_t)p.max_r * p.max_r < max_r2) p.max_r++;
  p.row_width = cfg->n_replicas * cfg->n_species;
  {
    // packed window test of K4 (kernels.cuh, pack_key): T = ceil(R / 2^shift) <= 15 coarse units per axis
    uint32_t sh = 0;
    while ((((uint32_t)p.max_r + (1u << sh) - 1u) >> sh) > 15u) ++sh;
    const uint32_t T = ((uint32_t)p.max_r + (1u << sh) - 1u) >> sh;
    p.pack_shift = sh;
    p.pack_k1 = (T + (1u << 10)) | ((T + (1u << 8)) << 12) | ((T + (1u << 8)) << 22);
    p.pack_u = ((1u << 10) - 1u - 2u * T) | (((1u << 8) - 1u - 2u * T) << 12) | (((1u << 8) - 1u - 2u * T) << 22);
    // a slot in the x interval [xlo, xlo + span) has a coarse x at most ((span - 1) >> shift) + 1 above xlo's
    p.pack_span1 = std::min<uint32_t>(((cfg->cell_size - 1u) >> sh) + 1u, 1023u);
    p.pack_span2 = std::min<uint32_t>(((2u * cfg->cell_size - 1u) >> sh) + 1u, 1023u);
  }
  p.top_shift = 16;                                                   // birth_top: at most kMaxTop entries
  while ((((uint64_t)cfg->id_capacity - 1) >> p.top_shift) + 1 > kMaxTop) p.top_shift++;

  s->gauss_bytes = ((size_t)cfg->n_sigma_classes << cfg->table_bits) * 2;
  s->gauss_in_smem = s->gauss_bytes <= 160 * 1024;
  // persistent grids: resident blocks per SM (occupancy API) x SM count, capped by the work there is
  {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    auto sized = [&](int per_sm, uint64_t tile) {
      const uint64_t need = ((uint64_t)cfg->capacity + tile - 1) / tile;
      return (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(need, (uint64_t)sms * (uint64_t)std::max(per_sm, 1)));
    };
    int occ = 0;
    const size_t gsm = s->gauss_in_smem ? s->gauss_bytes : 0;
    const bool large = cfg->capacity >= kLargeFrom;
    if (gsm) pick_move_kernels<true>(s, large); else pick_move_kernels<false>(s, large);
    s->unih_smem = align_up(gsm, 16) + (size_t)p.row_width * 4;      // K5: Gaussian tables, then the counts deltas
    if (s->unih_smem > 48 * 1024) {
      cudaFuncSetAttribute(s->k_scat, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsm);
      cudaFuncSetAttribute(s->k_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsm);
      cudaFuncSetAttribute(s->k_unih, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s->unih_smem);
      cudaFuncSetAttribute(k_move_only<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsm);
    }
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, s->k_scat, kMoveThreads, gsm);
    s->grid_scatter = sized(occ, (uint64_t)kMoveThreads * s->k3_unroll);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, s->k_unih, kUniThreads, s->unih_smem);
    s->grid_unih = sized(occ, kUniTile);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_pairs, kPairBlock, 0);
    s->grid_pairs = sized(occ, kPairThreads);                  // persistent: tiles are dealt round-robin
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_resolve, 256, 0);
    s->grid_resolve = sized(occ, 256 * 32);
    if (cudaGetLastError() != cudaSuccess) { delete s; return SIM_E_CUDA; }
  }
  auto clampu = [](uint64_t v, uint64_t lo, uint64_t hi) { return (uint32_t)std::min(std::max(v, lo), hi); };
  s->scan_blocks = clampu(((uint64_t)L.n_cells + 4095) / 4096, 1, kMaxScanBlocks);          // >= 4 K cells per block
  s->cell_seg = (uint32_t)align_up(((size_t)L.n_cells + s->scan_blocks - 1) / s->scan_blocks, 1024);
  s->tail_blocks = clampu(((uint64_t)cfg->capacity + 65535) / 65536, 2, kMaxTailBlocks);

  Scalars sc;
  std::memset(&sc, 0, sizeof(sc));
  for (int r = 0; r < kMaxRules; ++r) sc.t_first[r] = kNever;
  bool ok = true;
  ok = ok && cudaMemsetAsync(p.bits, 0, L.birth_list - L.bits, s->stream) == cudaSuccess;
  ok = ok && cudaMemsetAsync(p.best, 0xFF, L.hasprop - L.best, s->stream) == cudaSuccess;
  ok = ok && cudaMemsetAsync(p.hasprop, 0, L.partial - L.hasprop, s->stream) == cudaSuccess;   // proposal bits, both cell arrays
  ok = ok && cudaMemsetAsync(p.counts, 0, L.scal - L.counts, s->stream) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(p.scal, &sc, sizeof(sc), cudaMemcpyHostToDevice, s->stream) == cudaSuccess;
  ok = ok && cudaMemcpyAsync((void*)p.tab, &T, sizeof(T), cudaMemcpyHostToDevice, s->stream) == cudaSuccess;
  ok = ok && cudaMemcpyAsync((void*)p.gauss, cfg->tables, s->gauss_bytes, cudaMemcpyHostToDevice, s->stream) == cudaSuccess;
  ok = ok && cudaStreamSynchronize(s->stream) == cudaSuccess;
  if (!ok) { delete s; return SIM_E_CUDA; }
  *out = s;
  return SIM_OK;
}

void sim_destroy(sim_t* s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  prof_collect(s);
  for (int k = 0; k < 2; ++k) {
    if (s->g1[k]) cudaGraphExecDestroy(s->g1[k]);
    if (s->g8[k]) cudaGraphExecDestroy(s->g8[k]);
  }
  if (s->cap) cudaStreamDestroy(s->cap);
  if (s->side) cudaStreamDestroy(s->side);
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  if (s->ev_join) cudaEventDestroy(s->ev_join);
  delete s;
}

int sim_seed_population(sim_t* s, const sim_seed_rec_t* recs, uint32_t n_recs, uint64_t place_seed) {
  if (!s || (!recs && n_recs)) return SIM_E_INVAL;
  uint64_t total = 0;
  for (uint32_t i = 0; i < n_recs; ++i) {
    if (recs[i].species >= s->cfg.n_species || recs[i].replica >= s->cfg.n_replicas) return SIM_E_INVAL;
    total += recs[i].count;
  }
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  if (sc.err) return err_from_bits(sc.err);
  if ((uint64_t)sc.n_slots + total > s->cfg.capacity) return SIM_E_CAPACITY;
  if ((uint64_t)sc.next_id + total > s->cfg.id_capacity) return SIM_E_IDSPACE;
  uint32_t dst = sc.n_slots, id = sc.next_id;
  for (uint32_t i = 0; i < n_recs; ++i) {
    if (!recs[i].count) continue;
    ProfScope ps(s, KI_OTHER);
    k_seed<<<std::min<uint32_t>((recs[i].count + 255) / 256, 148 * 8), 256, 0, s->stream>>>(
        s->prm, recs[i].species, recs[i].replica, recs[i].count, id, dst, (uint32_t)place_seed, (uint32_t)(place_seed >> 32));
    dst += recs[i].count; id += recs[i].count;
  }
  CK(cudaGetLastError());
  sc.n_slots = dst; sc.next_id = id;
  s->hist_valid = false;          // the population changed: the next step starts with the histogram prologue
  CK(cudaMemcpyAsync(s->prm.scal, &sc, sizeof(sc), cudaMemcpyHostToDevice, s->stream));
  r = recount_row(s, sc.t, sc.n_slots);
  if (r) return r;
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

int sim_step_async(sim_t* s, uint32_t n_steps) {
  if (!s) return SIM_E_INVAL;
  if (s->sticky) return s->sticky;
  if ((uint64_t)s->t_host + n_steps >= s->cfg.counts_rows) return SIM_E_CAPACITY;
  if (n_steps && !s->hist_valid) { int r = enqueue_prologue(s); if (r) return r; }
  if (!s->profile && !s->graphs_tried) build_graphs(s);
  uint32_t left = n_steps;
  if (!s->profile && s->graphs_ok) {
    while (left >= kGraphSteps) {
      CK(cudaGraphLaunch(s->g8[parity_of(s)], s->stream));
      s->t_host += kGraphSteps; s->launches += (uint64_t)s->kernels_per_step * kGraphSteps; left -= kGraphSteps;
    }
    while (left) {
      CK(cudaGraphLaunch(s->g1[parity_of(s)], s->stream));
      flip(s);
      s->t_host++; s->launches += s->kernels_per_step; --left;
    }
    return SIM_OK;
  }
  for (uint32_t i = 0; i < left; ++i) {   // per-kernel profiling (events between launches), or no graph support
    int r = enqueue_step(s);
    if (r) return r;
  }
  return SIM_OK;
}

int sim_step(sim_t* s, uint32_t n_steps) {
  int r = sim_step_async(s, n_steps);
  if (r) return r;
  uint32_t err = 0;
  CK(cudaMemcpyAsync(&err, &s->prm.scal->err, 4, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  if (s->profile) prof_collect(s);
  if (err) { s->sticky = err_from_bits(err); return s->sticky; }
  return SIM_OK;
}

int sim_read_counts(sim_t* s, uint32_t first_row, uint32_t n_rows, uint32_t* out) {
  if (!s || !out || (uint64_t)first_row + n_rows > (uint64_t)s->t_host + 1) return SIM_E_INVAL;
  CK(cudaMemcpyAsync(out, s->prm.counts + (size_t)first_row * s->prm.row_width,
                     (size_t)n_rows * s->prm.row_width * 4, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

int sim_info(sim_t* s, uint32_t* n_live, uint32_t* step, uint32_t* next_id, uint32_t* t_first0) {
  if (!s) return SIM_E_INVAL;
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  if (n_live) {
    std::vector<uint32_t> row(s->prm.row_width);
    CK(cudaMemcpy(row.data(), s->prm.counts + (size_t)sc.t * s->prm.row_width, row.size() * 4, cudaMemcpyDeviceToHost));
    uint64_t tot = 0;
    for (uint32_t v : row) tot += v;
    *n_live = (uint32_t)tot;
  }
  if (step) *step = sc.t;
  if (next_id) *next_id = sc.next_id;
  if (t_first0) *t_first0 = sc.t_first[0];
  return SIM_OK;
}

int sim_read_agents(sim_t* s, uint32_t cap, int32_t* x, int32_t* y, int32_t* z, uint16_t* species, uint32_t* id,
                    uint32_t* n_out) {
  if (!s || !n_out) return SIM_E_INVAL;
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  CK(cudaMemsetAsync(&s->prm.scal->n_read, 0, 4, s->stream));
  if (sc.n_slots) {
    ProfScope ps(s, KI_OTHER);
    k_gather_live<<<std::min<uint32_t>((sc.n_slots + 255) / 256, 148 * 8), 256, 0, s->stream>>>(s->prm, sc.n_slots);
  }
  CK(cudaGetLastError());
  uint32_t n = 0;
  CK(cudaMemcpyAsync(&n, &s->prm.scal->n_read, 4, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  *n_out = n;
  if (n > cap) return SIM_E_CAPACITY;
  if (n == 0) return SIM_OK;
  std::vector<uint32_t> hid(n);
  const int32_t* plane = reinterpret_cast<const int32_t*>(s->prm.oth.r);   // k_gather_live wrote four planes
  const size_t pstride = s->cfg.capacity;
  CK(cudaMemcpy(hid.data(), plane + 3 * pstride, (size_t)n * 4, cudaMemcpyDeviceToHost));
  // id-sorted order: ids are unique and < next_id, so one pass over the id space sorts them
  std::vector<uint32_t> where((size_t)sc.next_id, 0xFFFFFFFFu), order;
  order.reserve(n);
  for (uint32_t i = 0; i < n; ++i) where[hid[i]] = i;
  for (uint32_t v = 0; v < sc.next_id; ++v) if (where[v] != 0xFFFFFFFFu) order.push_back(where[v]);
  if (order.size() != n) return SIM_E_INVAL;   // duplicate ids: internal error
  std::vector<int32_t> tmp(n);
  const int32_t* srcs[3] = {plane, plane + pstride, plane + 2 * pstride};
  int32_t* dsts[3] = {x, y, z};
  for (int a = 0; a < 3; ++a) {
    if (!dsts[a]) continue;
    CK(cudaMemcpy(tmp.data(), srcs[a], (size_t)n * 4, cudaMemcpyDeviceToHost));
    for (uint32_t i = 0; i < n; ++i) dsts[a][i] = tmp[order[i]];
  }
  if (species) {
    std::vector<uint16_t> ts(n);
    CK(cudaMemcpy(ts.data(), s->prm.oth.sp, (size_t)n * 2, cudaMemcpyDeviceToHost));
    for (uint32_t i = 0; i < n; ++i) species[i] = ts[order[i]];
  }
  if (id) for (uint32_t i = 0; i < n; ++i) id[i] = hid[order[i]];
  return SIM_OK;
}

int sim_load_agents(sim_t* s, uint32_t n, const int32_t* x, const int32_t* y, const int32_t* z,
                    const uint16_t* species, const uint32_t* id, uint32_t step, uint32_t next_id) {
  if (!s || n > s->cfg.capacity || (uint64_t)step + 1 > s->cfg.counts_rows || next_id > s->cfg.id_capacity)
    return SIM_E_INVAL;
  if (n && (!x || !y || !z || !species || !id)) return SIM_E_INVAL;
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  {
    int32_t* plane = reinterpret_cast<int32_t*>(s->prm.oth.r);   // scratch: four planes, then k_pack_records
    const size_t pstride = s->cfg.capacity;
    CK(cudaMemcpyAsync(plane, x, (size_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(plane + pstride, y, (size_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(plane + 2 * pstride, z, (size_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(plane + 3 * pstride, id, (size_t)n * 4, cudaMemcpyHostToDevice, s->stream));
    if (n) {
      ProfScope ps(s, KI_OTHER);
      k_pack_records<<<std::min<uint32_t>((n + 255) / 256, 148 * 8), 256, 0, s->stream>>>(s->prm, n);
    }
  }
  CK(cudaMemcpyAsync(s->prm.cur.sp, species, (size_t)n * 2, cudaMemcpyHostToDevice, s->stream));
  sc.n_slots = n; sc.next_id = next_id; sc.t = step; sc.err = 0;
  sc.birth_count = sc.total_births = sc.ticket = 0;
  CK(cudaMemcpyAsync(s->prm.scal, &sc, sizeof(sc), cudaMemcpyHostToDevice, s->stream));
  s->t_host = step; s->sticky = SIM_OK; s->hist_valid = false;
  r = recount_row(s, step, n, true);   // also validates every agent on the device (k_count_row)
  if (r) return r;
  uint32_t err = 0;
  CK(cudaMemcpyAsync(&err, &s->prm.scal->err, 4, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  if (err & 4u) {                 // invalid agent data: leave an empty, usable population behind
    sc.n_slots = 0; sc.err = 0;
    CK(cudaMemcpyAsync(s->prm.scal, &sc, sizeof(sc), cudaMemcpyHostToDevice, s->stream));
    r = recount_row(s, step, 0);
    if (r) return r;
    CK(cudaStreamSynchronize(s->stream));
    return SIM_E_INVAL;
  }
  return SIM_OK;
}

int sim_read_checksum(sim_t* s, uint64_t* out) {
  if (!s || !out) return SIM_E_INVAL;
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  unsigned long long* d_sum = (unsigned long long*)s->prm.birth_list;     // scratch that is free between steps
  CK(cudaMemsetAsync(d_sum, 0, 8, s->stream));
  if (sc.n_slots) {
    ProfScope ps(s, KI_OTHER);
    k_checksum<<<std::min<uint32_t>((sc.n_slots + 255) / 256, 148 * 8), 256, 0, s->stream>>>(s->prm, sc.n_slots, d_sum);
  }
  CK(cudaGetLastError());
  unsigned long long h = 0;
  CK(cudaMemcpyAsync(&h, d_sum, 8, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  *out = h;
  return SIM_OK;
}

int sim_read_t_first(sim_t* s, uint32_t n, uint32_t* out) {
  if (!s || !out || n != s->cfg.n_rules) return SIM_E_INVAL;
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  for (uint32_t k = 0; k < n; ++k) out[k] = sc.t_first[k];
  return SIM_OK;
}

int sim_load_t_first(sim_t* s, uint32_t n, const uint32_t* in) {
  if (!s || !in || n != s->cfg.n_rules) return SIM_E_INVAL;
  if (n) CK(cudaMemcpyAsync(s->prm.scal->t_first, in, (size_t)n * 4, cudaMemcpyHostToDevice, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

int sim_debug_move_only(sim_t* s) {
  if (!s) return SIM_E_INVAL;
  { ProfScope ps(s, KI_OTHER);
    if (s->gauss_in_smem) k_move_only<true><<<s->grid_scatter, kMoveThreads, s->gauss_bytes, s->stream>>>(s->prm);
    else k_move_only<false><<<s->grid_scatter, kMoveThreads, 0, s->stream>>>(s->prm); }
  s->hist_valid = false;
  CK(cudaGetLastError());
  // crossing deltas went to row t+1: fold them back so that row t describes the moved state
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  r = recount_row(s, sc.t, sc.n_slots);
  if (r) return r;
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

uint64_t sim_launch_count(const sim_t* s) { return s ? s->launches : 0; }

int sim_profile_enable(sim_t* s, int on) {
  if (!s) return SIM_E_INVAL;
  cudaStreamSynchronize(s->stream);
  prof_collect(s);
  s->profile = on != 0;
  std::memset(s->prof_ms, 0, sizeof(s->prof_ms));
  std::memset(s->prof_n, 0, sizeof(s->prof_n));
  return SIM_OK;
}

int sim_kernel_times(sim_t* s, float ms[SIM_N_KERNELS], uint32_t launches[SIM_N_KERNELS]) {
  if (!s) return SIM_E_INVAL;
  cudaStreamSynchronize(s->stream);
  prof_collect(s);
  for (int k = 0; k < SIM_N_KERNELS; ++k) { if (ms) ms[k] = s->prof_ms[k]; if (launches) launches[k] = s->prof_n[k]; }
  return SIM_OK;
}

const char* sim_kernel_name(int k) { return (k >= 0 && k < SIM_N_KERNELS) ? kKernelNames[k] : ""; }

const char* sim_strerror(int code) {
  switch (code) {
    case SIM_OK: return "ok";
    case SIM_E_INVAL: return "invalid argument or table validation failed";
    case SIM_E_CAPACITY: return "capacity exceeded (agent slots, counts rows or output buffer)";
    case SIM_E_IDSPACE: return "id space exhausted";
    case SIM_E_CUDA: return "CUDA error";
    case SIM_E_INTERNAL: return "internal bound check failed (checked build)";
    default: return "unknown error";
  }
}

const char* sim_last_cuda_error(const sim_t* s) { return s ? s->cuda_err.c_str() : ""; }

const char* sim_check_config(const sim_config_t* cfg) { return check_config(cfg); }

int sim_monitor_eval(sim_t* s, const sim_monitor_t* mons, uint32_t n_mons, sim_monitor_result_t* out,
                     uint8_t* states, uint32_t states_stride) {
  if (!s || !mons || !out || n_mons == 0 || n_mons > 64) return SIM_E_INVAL;
  if (s->sticky) return s->sticky;
  std::vector<DevMonitor> dm(n_mons);
  for (uint32_t m = 0; m < n_mons; ++m) {
    const sim_monitor_t& a = mons[m];
    if (a.replica >= s->cfg.n_replicas || a.n_species == 0 || a.n_species > 4 || a.n_rows == 0) return SIM_E_INVAL;
    if ((uint64_t)a.first_row + a.n_rows > (uint64_t)s->t_host + 1) return SIM_E_INVAL;   // rows not simulated yet
    if (states && a.n_rows > states_stride) return SIM_E_INVAL;
    DevMonitor& d = dm[m];
    d.replica = a.replica; d.n_species = a.n_species; d.threshold = a.threshold;
    d.first_row = a.first_row; d.n_rows = a.n_rows; d.states_off = m * states_stride;
    for (uint32_t k = 0; k < 4; ++k) {
      if (k < a.n_species && a.species[k] >= s->cfg.n_species) return SIM_E_INVAL;
      d.species[k] = k < a.n_species ? a.species[k] : 0;
    }
  }
  // scratch: the birth list is free between steps
  const size_t state_bytes = states ? (size_t)n_mons * states_stride : 0;
  if (8192 + state_bytes > (size_t)s->cfg.capacity * 8) return SIM_E_INVAL;
  char* scratch = (char*)s->prm.birth_list;
  DevMonitor* d_mon = (DevMonitor*)scratch;
  DevMonitorResult* d_res = (DevMonitorResult*)(scratch + 4096);
  uint8_t* d_states = states ? (uint8_t*)(scratch + 8192) : nullptr;
  CK(cudaMemcpyAsync(d_mon, dm.data(), n_mons * sizeof(DevMonitor), cudaMemcpyHostToDevice, s->stream));
  if (d_states) CK(cudaMemsetAsync(d_states, 0, state_bytes, s->stream));
  { ProfScope ps(s, KI_OTHER);
    k_monitor<<<n_mons, kMonThreads, 0, s->stream>>>(s->prm.counts, s->prm.row_width, s->prm.n_species, d_mon, d_res, d_states); }
  CK(cudaGetLastError());
  static_assert(sizeof(DevMonitorResult) == sizeof(sim_monitor_result_t), "result layout");
  CK(cudaMemcpyAsync(out, d_res, n_mons * sizeof(DevMonitorResult), cudaMemcpyDeviceToHost, s->stream));
  if (d_states) CK(cudaMemcpyAsync(states, d_states, state_bytes, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

int sim_render(sim_t* s, const sim_view_t* view, uint8_t* rgba) {
  if (!s || !view || !rgba) return SIM_E_INVAL;
  if (s->sticky) return s->sticky;
  const sim_view_t& a = *view;
  if (a.replica >= s->cfg.n_replicas || a.axis > 2 || a.eu == 0 || a.ev == 0 || a.width == 0 || a.height == 0 ||
      a.gain == 0 || a.gain > 255 || a.eu > 0x7FFFFFFFu || a.ev > 0x7FFFFFFFu)
    return SIM_E_INVAL;
  const uint64_t n_pix = (uint64_t)a.width * a.height, n_comp = s->cfg.n_compartments;
  if (n_pix > s->cfg.capacity || n_pix * n_comp > 2ull * s->cfg.capacity) return SIM_E_INVAL;
  DevView v;
  v.replica = a.replica; v.axis = a.axis; v.u0 = a.u0; v.v0 = a.v0; v.eu = a.eu; v.ev = a.ev;
  v.width = a.width; v.height = a.height; v.gain = a.gain; v.n_comp = (uint32_t)n_comp;
  std::memcpy(v.palette, a.palette, sizeof(v.palette));
  Scalars sc;
  int r = read_scalars(s, &sc);
  if (r) return r;
  uint32_t* d_cnt = (uint32_t*)s->prm.birth_list;      // scratch that is free between steps
  uchar4* d_img = (uchar4*)s->prm.prop;
  CK(cudaMemsetAsync(d_cnt, 0, n_pix * n_comp * 4, s->stream));
  if (sc.n_slots) {
    ProfScope ps(s, KI_OTHER);
    k_splat_count<<<std::min<uint32_t>((sc.n_slots + 255) / 256, 148 * 8), 256, 0, s->stream>>>(s->prm, v, sc.n_slots, d_cnt);
  }
  { ProfScope ps(s, KI_OTHER);
    k_splat_colour<<<(uint32_t)std::min<uint64_t>((n_pix + 255) / 256, 148 * 8), 256, 0, s->stream>>>(v, d_cnt, d_img); }
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(rgba, d_img, n_pix * 4, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return SIM_OK;
}

int sim_debug_philox(const uint32_t* d_ctr, const uint32_t* d_key, uint32_t* d_out, uint32_t n, void* cuda_stream) {
  if (!d_ctr || !d_key || !d_out) return SIM_E_INVAL;
  if (n) k_debug_philox<<<(n + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(d_ctr, d_key, d_out, n);
  return cudaGetLastError() == cudaSuccess ? SIM_OK : SIM_E_CUDA;
}

}  // extern "C"
