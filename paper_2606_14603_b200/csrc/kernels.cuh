// kernels.cuh — the hand-written sm_100a kernels of the molecule-agent step.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// One step = K2 cell scan (2 launches) -> K3 move+scatter -> K4 pair search/proposal -> K4b resolve ->
// K5 unimolecular + cell histogram of the NEXT step -> K6 births + epilogue: 7 launches.
// Every decision is keyed by agent id (never by slot), so the nondeterministic slot order the
// histogram atomics produce inside a cell cannot change any result.
#pragma once
#include "device_types.cuh"
#include "ptx_sm100.cuh"

namespace molsim {

// ----------------------------------------------------------------------------- Philox4x32-10
// north_star (2), S2.  counter (c0,c1,c2,c3), key (k0,k1); 10 rounds, 9 key bumps.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;   // one IMAD.WIDE gives hi and lo
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;   // the bump after the last round is dead code
  }
  return make_uint4(c0, c1, c2, c3);
}

// The simulation streams all use the key (seed lo, seed hi): their ten round keys are precomputed on
// the host into the kernel parameters, so a round is two IMAD.WIDE and two three-input XORs whose
// key operand comes straight from the constant bank.
__device__ __forceinline__ uint4 philox_sim(const Params& p, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ p.rk0[round], n2 = (uint32_t)(p0 >> 32) ^ c3 ^ p.rk1[round];
    c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
  }
  return make_uint4(c0, c1, c2, c3);
}

__global__ void k_debug_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint32_t n) {
  uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

// ----------------------------------------------------------------------------- block scan helper
// Exclusive scan of one value per thread over a 256-thread block (warp-shuffle scan, north_star (3)).
constexpr int kScanThreads = 256;
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t& total, uint32_t* s_warp /*[9]*/) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= d) incl += o;
  }
  __syncthreads();   // protects s_warp reuse across calls
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < kScanThreads / 32 ? s_warp[lane] : 0u;
    uint32_t wi = w;
#pragma unroll
    for (int d = 1; d < 8; d <<= 1) {
      uint32_t o = __shfl_up_sync(0xFFFFFFFFu, wi, d);
      if (lane >= d) wi += o;
    }
    if (lane < kScanThreads / 32) s_warp[lane] = wi - w;
    if (lane == kScanThreads / 32 - 1) s_warp[8] = wi;
  }
  __syncthreads();
  total = s_warp[8];
  return incl - v + s_warp[warp];
}

__device__ __forceinline__ uint32_t block_sum(uint32_t v, uint32_t* s_warp /*[9]*/) {
  uint32_t total;
  block_excl_scan(v, total, s_warp);
  return total;
}

// ----------------------------------------------------------------------------- phase 1: move
// Phase 1 (Brownian move, boundary and compartment rule) is a pure function of
// (species, position, id, t): move_agent() below.  It is evaluated twice per agent and step: by the histogram
// pass, which only needs the cell key of the moved position (and runs at the END of the previous step, fused
// with the unimolecular pass that streams the same agents: k_uni_hist), and by K3 while it scatters, so the
// moved positions are written once, at their sorted slot, and the 12 B/agent write + re-read of an in-place
// move never happens (a second Philox is cheaper).
struct Moved { int32_t x, y, z; uint16_t s; };

// What phase 1 needs of the tables, staged in shared memory next to the Gaussian tables so that
// the move never waits on a chain of dependent global loads.
struct SpLite { uint8_t cls, comp; uint16_t cross_to; uint32_t cross_thr; };
struct MoveTables {
  SpLite sp[kMaxSpecies];
  DevComp comp[kMaxCompartments];
};

__device__ __forceinline__ Moved move_agent(const Params& p, const MoveTables& M, const int16_t* g,
                                            uint16_t s, int32_t x, int32_t y, int32_t z, uint32_t id, uint32_t t) {
  Moved m{x, y, z, s};
  const SpLite S = M.sp[s];
  const uint32_t cls = S.cls;
  if (!cls) return m;
  const uint32_t sh = 32u - p.table_bits;
  const uint4 r = philox_sim(p, id, 0u, t, kTagMove);
  const int16_t* tb = g + (cls << p.table_bits);
  const int32_t rbase = (int32_t)(((uint32_t)x >> p.stride_shift) << p.stride_shift);
  int32_t qx = x - rbase + tb[r.x >> sh], qy = y + tb[r.y >> sh], qz = z + tb[r.z >> sh];
  const DevComp& c = M.comp[S.comp];
  if (c.shape == 0) {
    qx = mirror(qx, c.L); qy = mirror(qy, c.L); qz = mirror(qz, c.L);
  } else if (!comp_valid(c, qx, qy, qz)) {
    const uint16_t ct = S.cross_to;
    if (ct != kDead && comp_valid(M.comp[M.sp[ct].comp], qx, qy, qz) && fire(r.w, S.cross_thr)) m.s = ct;
    else return m;                       // no-flux wall: the agent keeps its position (S6)
  }
  m.x = qx + rbase; m.y = qy; m.z = qz;
  return m;
}

// Gaussian inverse-CDF tables (north_star (2)) and the species / compartment fields are staged in
// shared memory once per (persistent) block.
template <bool kGaussSmem>
__device__ __forceinline__ const int16_t* stage_tables(const Params& p, MoveTables& M, int16_t* s_gauss) {
  const DevTables* __restrict__ T = p.tab;
  for (uint32_t k = threadIdx.x; k < (uint32_t)kMaxSpecies; k += blockDim.x) {
    const DevSpecies& S = T->sp[k];
    M.sp[k] = SpLite{S.sigma_class, S.compartment, S.cross_to, S.cross_thr};
  }
  for (uint32_t k = threadIdx.x; k < (uint32_t)kMaxCompartments; k += blockDim.x) M.comp[k] = T->comp[k];
  const int16_t* g = p.gauss;
  if (kGaussSmem) {
    const uint32_t n_words = (p.n_classes << p.table_bits) >> 1;      // table_bits >= 1: an even number of int16
    const uint32_t n_quads = n_words >> 2;                            // 128-bit copies, then the tail
    const uint4* src4 = reinterpret_cast<const uint4*>(p.gauss);
    uint4* dst4 = reinterpret_cast<uint4*>(s_gauss);
    for (uint32_t k = threadIdx.x; k < n_quads; k += blockDim.x) dst4[k] = src4[k];
    const uint32_t* src = reinterpret_cast<const uint32_t*>(p.gauss);
    uint32_t* dst = reinterpret_cast<uint32_t*>(s_gauss);
    for (uint32_t k = (n_quads << 2) + threadIdx.x; k < n_words; k += blockDim.x) dst[k] = src[k];
    g = s_gauss;
  }
  __syncthreads();
  return g;
}

// Warp aggregation of the counting sort's atomics.  Agents arrive nearly cell-sorted from the previous
// step, so lanes with equal keys are almost always neighbours: a run of equal keys (one shuffle, one
// ballot) is aggregated into one atomic by its first lane.  Equal keys that are not adjacent simply
// issue separate atomics.  (__match_any_sync finds them all but runs on the slow ADU pipe: it was
// the top stall of the histogram kernel when tried.)
__device__ __forceinline__ void run_of_key(uint32_t key, uint32_t lane, int& leader, uint32_t& rank, uint32_t& count) {
  const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, key, 1);
  const uint32_t heads = __ballot_sync(0xFFFFFFFFu, lane == 0u || key != prev);
  const uint32_t upto = (2u << lane) - 1u;                        // lanes 0..lane (lane 31: all ones)
  leader = 31 - __clz(heads & upto);
  const uint32_t above = heads & ~upto;
  const int end = above ? __ffs(above) - 1 : 32;
  rank = lane - (uint32_t)leader;
  count = (uint32_t)(end - leader);
}

// Agents in flight per thread and resident blocks per SM of the two passes that evaluate the move are
// template parameters; the host picks per problem size (swept on B200: profiles/).
constexpr uint32_t kLargeFrom = 2000000;   // capacity (agents) from which the large-population shapes are used
constexpr int kMoveThreads = 256;

// Test hook (sim_debug_move_only): phase 1 in place on the current arrays.
template <bool kGaussSmem>
__global__ void __launch_bounds__(kMoveThreads) k_move_only(Params p) {
  extern __shared__ __align__(16) int16_t s_gauss[];
  __shared__ MoveTables M;
  const int16_t* g = stage_tables<kGaussSmem>(p, M, s_gauss);
  const uint32_t n = p.scal->n_slots, t = p.scal->t;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const uint16_t s = p.cur.sp[i];
    if (s == kDead) continue;
    const int4 q = p.cur.r[i];
    const Moved m = move_agent(p, M, g, s, q.x, q.y, q.z, (uint32_t)q.w, t);
    p.cur.r[i] = make_int4(m.x, m.y, m.z, q.w); p.cur.sp[i] = m.s;
  }
}

// ----------------------------------------------------------------------------- K2 cell scan
// Exclusive scan of the per-cell counts, in place (a4).  Two launches with a fixed block count:
// (a) per-segment sums, (b) every block adds up the partials before it (a few hundred values) and
// rescans its own segment.  No inter-block waiting, deterministic.
__global__ void __launch_bounds__(kScanThreads) k_cell_reduce(const uint32_t* __restrict__ cell, uint32_t n,
                                                              uint32_t seg, uint32_t* __restrict__ partial) {
  __shared__ uint32_t s_warp[9];
  const uint32_t lo = blockIdx.x * seg, hi = min(lo + seg, n);
  uint32_t sum = 0;
  for (uint32_t b = lo + threadIdx.x * 4u; b < hi; b += kScanThreads * 4u) {
    if (b + 4u <= hi) {
      const uint4 v = *reinterpret_cast<const uint4*>(cell + b);
      sum += v.x + v.y + v.z + v.w;
    } else {
      for (uint32_t k = b; k < hi; ++k) sum += cell[k];
    }
  }
  const uint32_t tot = block_sum(sum, s_warp);
  if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kScanThreads) k_cell_scan(uint32_t* __restrict__ cell, uint32_t n, uint32_t seg,
                                                            const uint32_t* __restrict__ partial) {
  __shared__ uint32_t s_warp[9];
  uint32_t mine = 0;
  for (uint32_t b = threadIdx.x; b < blockIdx.x; b += kScanThreads) mine += partial[b];
  uint32_t running = block_sum(mine, s_warp);
  const uint32_t lo = blockIdx.x * seg, hi = min(lo + seg, n);
  for (uint32_t tile = lo; tile < hi; tile += kScanThreads * 4u) {
    const uint32_t b = tile + threadIdx.x * 4u;
    uint32_t v[4] = {0u, 0u, 0u, 0u};
    const bool full = b + 4u <= hi;
    if (full) {
      const uint4 q = *reinterpret_cast<const uint4*>(cell + b);
      v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    } else {
      for (uint32_t k = 0; k < 4u; ++k) if (b + k < hi) v[k] = cell[b + k];
    }
    const uint32_t s = v[0] + v[1] + v[2] + v[3];
    uint32_t total;
    uint32_t e = running + block_excl_scan(s, total, s_warp);
    if (full) {
      uint4 q; q.x = e; q.y = e + v[0]; q.z = q.y + v[1]; q.w = q.z + v[2];
      *reinterpret_cast<uint4*>(cell + b) = q;
    } else {
      for (uint32_t k = 0; k < 4u; ++k) { if (b + k < hi) cell[b + k] = e; e += v[k]; }
    }
    running += total;
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) cell[n] = running;   // = number of live agents
}

// ----------------------------------------------------------------------------- K3 move + scatter / reorder
// Counting-sort scatter that reorders the whole structure of arrays into cell order (a5), applying
// phase 1 on the way (move_agent again: same result as in the histogram pass, so the same cell), and drops
// DEAD slots, which is the compaction of the previous step's deaths (fused, a9).  The cell array holds, after
// the scan, the first slot of every cell one word ahead (cursor[k] = cell[k + 1]); a run of equal keys in a
// warp takes its slots with one atomicAdd on that cursor, so when the kernel ends cursor[k] is the END of
// cell k = the start of cell k + 1, i.e. cell[k] = start of cell k and cell[n_cells] = live agents, which is
// what every later kernel reads.  No per-agent rank array is written or read.  kK3Unroll agents in flight per
// thread.  Membrane crossings change the species here; their counts deltas go straight to counts row t+1
// (rare events).
template <bool kGaussSmem, int kK3Unroll, int kMinBlk>
__global__ void __launch_bounds__(kMoveThreads, kMinBlk) k_scatter(Params p) {
  extern __shared__ __align__(16) int16_t s_gauss[];
  __shared__ MoveTables M;
  const int16_t* g = stage_tables<kGaussSmem>(p, M, s_gauss);
  const uint32_t n = p.scal->n_slots, t = p.scal->t;
  const uint32_t lane = threadIdx.x & 31u;
  uint32_t* __restrict__ cursor = p.cell + 1;
  uint32_t* __restrict__ row = p.counts + (size_t)(t + 1) * p.row_width;
  constexpr uint32_t kTile = kMoveThreads * kK3Unroll;
  for (uint32_t base = blockIdx.x * kTile; base < n; base += gridDim.x * kTile) {   // block-uniform trip count
    uint16_t s[kK3Unroll];
    int32_t x[kK3Unroll], y[kK3Unroll], z[kK3Unroll];
    uint32_t id[kK3Unroll], key[kK3Unroll];
#pragma unroll
    for (int a = 0; a < kK3Unroll; ++a) {
      const uint32_t i = base + a * kMoveThreads + threadIdx.x;
      s[a] = i < n ? p.cur.sp[i] : kDead;
    }
#pragma unroll
    for (int a = 0; a < kK3Unroll; ++a) {
      const uint32_t i = base + a * kMoveThreads + threadIdx.x;
      if (i < n) { const int4 q = p.cur.r[i]; x[a] = q.x; y[a] = q.y; z[a] = q.z; id[a] = (uint32_t)q.w; }   // not gated on the species: one round trip
    }
#pragma unroll
    for (int a = 0; a < kK3Unroll; ++a) {
      key[a] = 0xFFFFFFFFu;
      if (s[a] == kDead) continue;
      const Moved m = move_agent(p, M, g, s[a], x[a], y[a], z[a], id[a], t);
      if (m.s != s[a]) {
        const uint32_t rep = (uint32_t)x[a] >> p.stride_shift;
        atomicSub(&row[rep * p.n_species + s[a]], 1u);
        atomicAdd(&row[rep * p.n_species + m.s], 1u);
      }
      x[a] = m.x; y[a] = m.y; z[a] = m.z; s[a] = m.s;
      key[a] = cell_key(m.x, m.y, m.z, p);
    }
    uint32_t first[kK3Unroll], rank[kK3Unroll];
    int leader[kK3Unroll];
#pragma unroll
    for (int a = 0; a < kK3Unroll; ++a) {
      uint32_t count;
      run_of_key(key[a], lane, leader[a], rank[a], count);
      first[a] = 0;
      if (s[a] != kDead && (int)lane == leader[a]) first[a] = atomicAdd(&cursor[key[a]], count);
    }
#pragma unroll
    for (int a = 0; a < kK3Unroll; ++a) {
      const uint32_t dst = __shfl_sync(0xFFFFFFFFu, first[a], leader[a]) + rank[a];
      if (s[a] == kDead) continue;
      MOLSIM_CHECK(p, key[a] < p.n_cells && dst < p.capacity);
      p.oth.r[dst] = make_int4(x[a], y[a], z[a], (int32_t)id[a]);     // ONE scattered 128-bit store per agent
      p.oth.sp[dst] = s[a];
    }
  }
}

// ----------------------------------------------------------------------------- counts aggregation
// Per-step species counts (a10) are kept as deltas on a running row.  Events are aggregated in a
// per-block shared-memory delta table and flushed once per block, so that thousands of bindings
// per step do not serialise on a handful of global counters.
constexpr int kMaxRowWidth = 64 * kMaxSpecies;   // SIM_MAX_REPLICAS x SIM_MAX_SPECIES
__device__ __forceinline__ void delta_zero(int32_t* s_delta, uint32_t row_width) {
  for (uint32_t k = threadIdx.x; k < row_width; k += blockDim.x) s_delta[k] = 0;
  __syncthreads();
}
__device__ __forceinline__ void delta_flush(const int32_t* s_delta, uint32_t* __restrict__ row, uint32_t row_width) {
  __syncthreads();
  for (uint32_t k = threadIdx.x; k < row_width; k += blockDim.x) {
    const int32_t d = s_delta[k];
    if (d) atomicAdd(&row[k], (uint32_t)d);
  }
}

// ----------------------------------------------------------------------------- K4 pair search + proposal
// Phase 2a: each agent whose species can bind proposes its eligible partner with the smallest
// (dist^2, id) among those that pass the symmetric pair draw (a6).  The predicate and the draw are
// symmetric in the pair, so every unordered pair is examined ONCE, from its lower sorted slot i < j,
// and a qualifying pair is merged into both ends: best[i] <- min(., (d2, id_j)), best[j] <- min(.,
// (d2, id_i)) with 64-bit global atomic min.  Only cells the R-ball overlaps are visited (exact: a
// cell it does not overlap cannot hold an in-range partner), and of those only the "forward" ones:
// the rest of the agent's own cell, the +x cell, and the overlapped cells of the rows (y+1, z) and
// (y-1..y+1, z+1).  With x-fastest cell keys the cells of one (y,z) row are one contiguous slot range.
//
// Work layout (round 2; profiles/r2_pairs.md has the per-phase instruction split and the two discarded
// cuts that led here: set-up, divergent row visits and one-lane hit qualification were 70 % of the
// instructions of the round-1 kernel, and block-wide queues drained behind block barriers were latency-bound).
// The kernel is persistent and its warps run on their own.  A block walks tiles of 256 consecutive sorted
// slots; tile records (plus kPairHalo slots behind them) and species arrive in a four-stage shared-memory
// ring by bulk copies (cp.async.bulk + mbarrier: the TMA engine) issued by a ninth, producer warp up to three
// tiles ahead of the tile being worked on, so no warp waits on the streaming loads; a stage is handed back by one mbarrier arrival per warp, so
// there is no block-wide barrier in the loop.  Per tile a warp owns 32 slots and does dense work only:
//  A  own row.  Every agent tests the kPairWin slots behind its own straight from shared memory: no
//     range look-up, no loop, every lane busy.  A slot that passes the window test (|d| <= R on every
//     axis) is a genuine close pair whatever cell it lies in, so nothing has to bound the window; the
//     own-row range (rest of the own cell, plus the +x cell if the R-ball reaches it) is longer than
//     the window only if the slot right behind the window still lies in that x interval: then the
//     remainder is row code 4 of the agent's entry.
//  B  agents with rows to visit (a +y / +z cell face within R, or a remainder: about a fifth) append one
//     entry (slot, row mask) to the WARP's queue: one ballot, no atomics.  Window hits go to the warp's
//     hit queue as (i, j, id_j, d2).
// The rare work is deferred until a warp's worth has piled up, so that it too runs with every lane busy,
// and while one warp waits on its look-ups the others carry on with their tiles:
//  C  32 entries: one lane per entry re-derives the agent's place in the grid and walks its rows (two
//     cell-range look-ups, then records in groups of four).
//  D  hits: one lane per hit: reaction look-up, exact radius, symmetric pair draw and, if the pair
//     qualifies, the two atomic mins.  best[] is touched only there (rare), so it costs no bandwidth;
//     hasprop gets one bit per touched agent and prop[] the slot of a partner that qualified.  prop[] is a
//     plain store (no round trip for the old key): with several qualifying partners it may name another than the
//     minimum, so K4b checks id[prop[i]] against the key and searches the neighbourhood again in that
//     (rare) case.  A pair reached twice (window and row) is merged twice, which changes nothing.
// The entry queue cannot overflow (fewer than 32 entries before a tile, at most 32 more); a hit that finds
// its queue full (dense test inputs) is qualified on the spot.
constexpr int kPairThreads = 256;
constexpr int kPairWarps = kPairThreads / 32;
constexpr int kPairStages = 4;
constexpr int kPairBlock = kPairThreads + 32;   // 8 warps that own 32 slots of the tile each + the producer warp
constexpr int kPairWin = 5;             // slots behind its own that every agent tests in phase A
constexpr int kPairHalo = 16;           // slots staged behind the tile: kPairWin + the over-run probe, rounded up
constexpr int kPairHitCap = 16, kPairHitDrain = 8;     // per warp
constexpr uint32_t kPairTileBytes = (kPairThreads + kPairHalo) * 16u + kPairThreads * 2u;
constexpr unsigned long long kNoKey = ~0ull;

// mbarrier + bulk copy + fences: ptx_sm100.cuh (PTX, sm_90+; SASS on sm_100a: SYNCS / UBLKCP)

struct PairSmem {
  int4 rec[kPairStages][kPairThreads + kPairHalo];   // x, y, z, id of the tile's slots and the kPairHalo behind them
  uint16_t sp[kPairStages][kPairThreads];            // species
  int4 ent_pos[kPairWarps][64];                      // per warp, agents with rows left to visit: x, y, z, id
  uint4 ent_geo[kPairWarps][64];                     //   slot, own cell, rows | xm << 9 | xp << 10 | species << 16, -
  uint4 hit_a[kPairWarps][kPairHitCap];              // per warp, window hits: i, j, id_i, id_j
  uint2 hit_b[kPairWarps][kPairHitCap];              //   d2, species of i
  uint32_t key[kPairWarps][48];                      // packed coarse positions of the warp's 32 slots + the window behind
  unsigned long long full[kPairStages], empty[kPairStages];
  uint32_t nhit[kPairWarps];
};

// Reaction look-up, exact radius and symmetric pair draw for the geometric hit (i, j); on success both ends are merged.
__device__ __forceinline__ void pair_merge(const Params& p, uint32_t i, uint32_t j, uint32_t id, uint32_t idj, uint32_t d2,
                                           uint32_t si) {
  const DevTables* __restrict__ T = p.tab;
  MOLSIM_CHECK(p, i < p.capacity && j < p.capacity && si < (uint32_t)kMaxSpecies && p.oth.sp[j] < (uint32_t)kMaxSpecies);
  const uint32_t e = T->rxmap[si * kMaxSpecies + p.oth.sp[j]];
  if (e == 0xFFu) return;
  const DevRx& rx = T->rx[e];
  if (d2 > rx.r2) return;
  const uint4 r = philox_sim(p, min(id, idj), max(id, idj), p.scal->t, kTagPair);
  if (!fire(r.x, rx.thr)) return;
  const unsigned long long hi = (unsigned long long)d2 << 32;
  atomicMin(&p.best[i], hi | idj);
  atomicMin(&p.best[j], hi | id);
  p.prop[i] = j; p.prop[j] = i;
  atomicOr(&p.hasprop[i >> 5], 1u << (i & 31u));
  atomicOr(&p.hasprop[j >> 5], 1u << (j & 31u));
}
__device__ __noinline__ void pair_merge_now(const Params* p, uint32_t i, uint32_t j, uint32_t id, uint32_t idj, uint32_t d2,
                                            uint32_t si) {
  pair_merge(*p, i, j, id, idj, d2, si);
}
// A hit that finds the warp's queue full (dense test inputs) is qualified on the spot.  The partner's species is the
// one thing the drain will have to fetch: ask for its line now.
__device__ __forceinline__ void push_hit(const Params& p, PairSmem& S, uint32_t warp, uint32_t i, uint32_t j, uint32_t id,
                                         uint32_t idj, uint32_t d2, uint32_t si) {
  const uint32_t h = atomicAdd(&S.nhit[warp], 1u);
  if (h < (uint32_t)kPairHitCap) {
    S.hit_a[warp][h] = make_uint4(i, j, id, idj); S.hit_b[warp][h] = make_uint2(d2, si);
    prefetch_l1(p.oth.sp + j);
  } else {
    pair_merge_now(&p, i, j, id, idj, d2, si);
  }
}

// Global slots [j0, j1) against agent i (id, species si) at (x, y, z).
__device__ __forceinline__ void scan_rows(const Params& p, PairSmem& S, uint32_t warp, uint32_t j0, uint32_t j1, uint32_t n,
                                          uint32_t i, uint32_t id, uint32_t si, int32_t x, int32_t y, int32_t z) {
  const int32_t R = p.max_r;
  const uint32_t R2 = 2u * (uint32_t)R;
  const int32_t ox = R - x, oy = R - y, oz = R - z;
  const int4* __restrict__ Rr = p.oth.r;
  // groups of four records in flight, branch-free (one predicate bit each), one branch per group.  A group
  // may run up to three slots past j1: those are later slots of the sorted array (a genuine forward pair if
  // they pass) or past the population (never queued: j < n); the record array has slack for them
  MOLSIM_CHECK(p, j1 <= n && (j0 >= j1 || j1 + 3u < p.capacity + (uint32_t)(kPairThreads + kPairHalo)));
  for (uint32_t j = j0; j < j1; j += 4u) {
    uint32_t hits = 0;
#pragma unroll
    for (uint32_t u = 0; u < 4u; ++u) {
      const int4 q = __ldg(Rr + j + u);
      const uint32_t ux = (uint32_t)(q.x + ox), uy = (uint32_t)(q.y + oy), uz = (uint32_t)(q.z + oz);
      hits |= (max(max(ux, uy), uz) <= R2) ? (1u << u) : 0u;    // |d| <= R on every axis
    }
    for (; hits; hits &= hits - 1u) {                       // rare
      const uint32_t jj = j + (uint32_t)__ffs(hits) - 1u;
      const int4 q = __ldg(Rr + jj);
      const int32_t dx = q.x - x, dy = q.y - y, dz = q.z - z;     // each within +-R
      const uint32_t d2 = (uint32_t)(dx * dx) + (uint32_t)(dy * dy) + (uint32_t)(dz * dz);
      if (jj < n && d2 <= p.max_r2) push_hit(p, S, warp, i, jj, id, (uint32_t)q.w, d2, si);
    }
  }
}

// Packed coarse position for the window test.  The LSU data pipe (shared-memory wavefronts), not instruction
// issue, bounds this kernel (profiles/r2_pairs.md), and a 128-bit record per candidate costs four wavefronts per
// warp; a 32-bit key costs one.  Key = three fields (x: 10 bits, y and z: 8 bits of the coordinate >> pack_shift,
// i.e. modulo a few cells) with two guard bits above each, the lower guard set.  For keys a, b the sum
// b + (K1 - a), K1 = T + 2^w per field, holds (b_f - a_f + T) mod 2^w in the low w bits of every field without
// any carry between fields; adding U = 2^w - 1 - 2T per field to those low bits sets the guard iff the field
// exceeds 2T.  T = ceil(R / 2^pack_shift), so |d| <= R on an axis implies a coarse difference within +-T
// (modulo the field): the test never misses a pair; it passes about a third more candidates than the exact
// window, and everything it passes is checked with the full coordinates afterwards.
constexpr uint32_t kKeyLow = 0x3FFu | (0xFFu << 12) | (0xFFu << 22);
constexpr uint32_t kKeyGuard = (1u << 10) | (1u << 20) | (1u << 30);
__device__ __forceinline__ uint32_t pack_key(const Params& p, int32_t x, int32_t y, int32_t z) {
  const uint32_t sh = p.pack_shift;
  return (((uint32_t)x >> sh) & 0x3FFu) | ((((uint32_t)y >> sh) & 0xFFu) << 12) | ((((uint32_t)z >> sh) & 0xFFu) << 22) | kKeyGuard;
}

// Where an agent sits in the cell grid: its own cell (linear index), whether its R-ball reaches the -x / +x
// neighbour, and the forward rows it faces: bit (dz+1)*3 + (dy+1): (y+1, z) = 5; (y-1, z+1), (y, z+1),
// (y+1, z+1) = 6, 7, 8.  R <= cell_size (validated), so the ball reaches at most one cell further on each side.
struct PairGeo { uint32_t cell, xm, xp, rows; int32_t xlo; };
__device__ __forceinline__ PairGeo pair_geo(const Params& p, int32_t x, int32_t y, int32_t z) {
  const int32_t R = p.max_r, cs = p.cell_size;
  const int32_t cx = cell_coord(x, p), cy = cell_coord(y, p), cz = cell_coord(z, p);
  const int32_t lx = x - cx * cs, ly = y - cy * cs, lz = z - cz * cs;
  PairGeo g;
  g.xlo = x - lx;
  g.xm = lx < R && cx > 0; g.xp = lx >= cs - R && cx < p.nx - 1;
  const uint32_t ym = ly < R && cy > 0, yp = ly >= cs - R && cy < p.ny - 1;
  const uint32_t zp = lz >= cs - R && cz < p.nz - 1;
  g.cell = ((uint32_t)cz * (uint32_t)p.ny + (uint32_t)cy) * (uint32_t)p.nx + (uint32_t)cx;
  g.rows = (yp << 5) | (zp ? ((ym | 2u | (yp << 2)) << 6) : 0u);
  return g;
}

// C / D for one warp.  Takes up to 32 entries off the top of its queue and visits ONE row of each (two cell-range
// look-ups, then records in groups of four); an entry with
// further rows goes back on the queue, so every round is dense and costs one memory round trip.  Then, if there are
// enough of them (or `all`), the warp's hits.  Returns the new queue length.  Out of line: its registers (Philox,
// 64-bit keys) must not be charged to the dense per-tile loop.
__device__ __noinline__ uint32_t pair_drain(const Params* pp, PairSmem* Sp, uint32_t n, uint32_t nent, bool all) {
  const Params& p = *pp;
  PairSmem& S = *Sp;
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  __syncwarp();
  const uint32_t take = min(nent, 32u), e0 = nent - take;
  int4 o = make_int4(0, 0, 0, 0);
  uint4 ge = make_uint4(0, 0, 0, 0);
  uint32_t left = 0;
  if (lane < take) {
    o = S.ent_pos[warp][e0 + lane]; ge = S.ent_geo[warp][e0 + lane];
    const uint32_t rows = ge.z & 0x1F0u, xm = ge.z >> 9 & 1u, xp = ge.z >> 10 & 1u;
    const uint32_t c = (uint32_t)__ffs(rows) - 1u;
    left = rows & (rows - 1u);
    uint32_t j0, j1;
    if (c == 4u) { j0 = ge.x + 1u + (uint32_t)kPairWin; j1 = p.cell[ge.y + xp + 1u]; }       // own-row remainder
    else {
      const uint32_t c0 = ge.y + (uint32_t)p.fwd_row[c - 5u];      // host-precomputed row offsets of codes 5..8
      MOLSIM_CHECK(p, c0 >= xm && c0 + xp + 1u <= p.n_cells);
      j0 = p.cell[c0 - xm]; j1 = p.cell[c0 + xp + 1u];
    }
    MOLSIM_CHECK(p, ge.y + xp + 1u <= p.n_cells && e0 + lane < 64u);
    scan_rows(p, S, warp, j0, j1, n, ge.x, (uint32_t)o.w, ge.z >> 16, o.x, o.y, o.z);
  }
  __syncwarp();            // every lane has read its entry: the slots may be overwritten
  const uint32_t again = __ballot_sync(0xFFFFFFFFu, left != 0u);
  if (left) {
    const uint32_t k = e0 + (uint32_t)__popc(again & ((1u << lane) - 1u));
    MOLSIM_CHECK(p, k < 64u);
    ge.z = (ge.z & ~0x1F0u) | left;
    S.ent_pos[warp][k] = o; S.ent_geo[warp][k] = ge;
  }
  nent = e0 + (uint32_t)__popc(again);
  __syncwarp();
  const uint32_t nh = min(S.nhit[warp], (uint32_t)kPairHitCap);
  if (nh >= (uint32_t)kPairHitDrain || (all && nh)) {
    if (lane < nh) {
      const uint4 a = S.hit_a[warp][lane];
      const uint2 b = S.hit_b[warp][lane];
      pair_merge(p, a.x, a.y, a.z, a.w, b.x, b.y);
    }
    __syncwarp();
    if (lane == 0) S.nhit[warp] = 0;
    __syncwarp();
  }
  return nent;
}

__device__ __forceinline__ void pair_issue_tile(const Params& p, PairSmem& S, uint32_t stage, uint32_t tile) {
  // generic-proxy reads of this stage (by the tile that used it before) are ordered before the async-proxy refill
  fence_proxy_async();
  mbar_expect_tx(&S.full[stage], kPairTileBytes);
  bulk_g2s(S.rec[stage], p.oth.r + (size_t)tile * kPairThreads, (kPairThreads + kPairHalo) * 16u, &S.full[stage]);
  bulk_g2s(S.sp[stage], p.oth.sp + (size_t)tile * kPairThreads, kPairThreads * 2u, &S.full[stage]);
}

__global__ void __launch_bounds__(kPairBlock, 4) k_pairs(const __grid_constant__ Params p) {
  __shared__ __align__(128) PairSmem S;
  const uint32_t n = p.cell[p.n_cells];
  const uint32_t ntiles = (n + kPairThreads - 1u) / kPairThreads;
  if (blockIdx.x >= ntiles) return;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  if (tid == 0) {
    for (int k = 0; k < kPairStages; ++k) { mbar_init(&S.full[k], 1u); mbar_init(&S.empty[k], (uint32_t)kPairWarps); }
    fence_mbar_init();
  }
  if (lane == 0 && warp < (uint32_t)kPairWarps) S.nhit[warp] = 0;
  __syncthreads();                  // the only block-wide barrier
  if (warp == (uint32_t)kPairWarps) {
    // ---- producer: keeps the ring full.  Tile `it` goes to stage it % kPairStages once every warp has handed back
    // the tile that used it before.
    if (lane == 0) {
      uint32_t it = 0;
      for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const uint32_t stage = it % (uint32_t)kPairStages, use = it / (uint32_t)kPairStages;
        if (use) while (!mbar_try_wait(&S.empty[stage], (use - 1u) & 1u)) __nanosleep(256);   // do not spin on issue slots
        pair_issue_tile(p, S, stage, tile);
      }
    }
    return;
  }
  uint32_t nent = 0;                // entries in this warp's queue (warp-uniform)
  uint32_t stage = 0, use = 0;      // tile `it` of this block: stage = it % kPairStages, use = it / kPairStages
  for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    while (!mbar_try_wait(&S.full[stage], use & 1u)) {}
    const uint32_t i = tile * kPairThreads + tid;
    const int4 q = S.rec[stage][tid];
    const uint32_t s = S.sp[stage][tid];
    // packed keys of the warp's 32 slots and of the kPairWin + 1 slots behind them (the first of the next warp's)
    uint32_t* K = S.key[warp];
    const uint32_t kq = pack_key(p, q.x, q.y, q.z);
    K[lane] = kq;
    if (lane <= (uint32_t)kPairWin) {
      const int4 h = S.rec[stage][tid + 32u];
      K[32u + lane] = pack_key(p, h.x, h.y, h.z);
    }
    __syncwarp();
    uint32_t rows = 0, cell = 0;        // rows to visit | xm << 9 | xp << 10, own cell
    if (i < n && s != kDead && ((p.binds_mask >> s) & 1ull)) {
      const PairGeo g = pair_geo(p, q.x, q.y, q.z);
      rows = g.rows; cell = g.cell;
      // ---- A: the kPairWin slots behind its own
      const uint32_t cq = p.pack_k1 - kq;
      uint32_t hits = 0;
#pragma unroll
      for (uint32_t u = 0; u < (uint32_t)kPairWin; ++u) {
        const uint32_t e = K[lane + 1u + u] + cq;
        hits |= ((((e & kKeyLow) + p.pack_u) & kKeyGuard) == 0u) ? (1u << u) : 0u;
      }
      for (; hits; hits &= hits - 1u) {                    // rare: the exact test
        const uint32_t u = (uint32_t)__ffs(hits);
        const int4 c = S.rec[stage][tid + u];
        const long long dx = (long long)c.x - q.x, dy = (long long)c.y - q.y, dz = (long long)c.z - q.z;
        const unsigned long long d2 = (unsigned long long)(dx * dx + dy * dy + dz * dz);
        if (i + u < n && d2 <= p.max_r2)                   // never a slot past the population
          push_hit(p, S, warp, i, i + u, (uint32_t)q.w, (uint32_t)c.w, (uint32_t)d2, s);
      }
      // the own-row range goes on behind the window iff the next slot still lies in its x interval (slots of a row
      // are ordered by x cell).  Tested on the coarse x, modulo the field: a slot that only seems to lie in the
      // interval (another row, or an alias) costs a look-up, nothing else.
      const uint32_t xk = (K[lane + 1u + kPairWin] - ((uint32_t)g.xlo >> p.pack_shift)) & 0x3FFu;
      if (xk <= (g.xp ? p.pack_span2 : p.pack_span1)) rows |= 1u << 4;
      if (rows) rows |= (g.xm << 9) | (g.xp << 10);
    }
    // ---- B: one entry per agent with rows to visit, appended to the warp's queue
    const uint32_t any = __ballot_sync(0xFFFFFFFFu, rows != 0u);
    if (rows) {
      const uint32_t k = nent + (uint32_t)__popc(any & ((1u << lane) - 1u));
      MOLSIM_CHECK(p, k < 64u && cell < p.n_cells);
      S.ent_pos[warp][k] = q;
      S.ent_geo[warp][k] = make_uint4(i, cell, rows | (s << 16), 0u);
    }
    nent += (uint32_t)__popc(any);
    // this warp is done with the stage
    __syncwarp();
    if (lane == 0) mbar_arrive(&S.empty[stage]);
    // ---- C / D once a warp's worth has piled up (hits ride along when there are enough of them)
    while (nent >= 32u) nent = pair_drain(&p, &S, n, nent, false);
    if (++stage == (uint32_t)kPairStages) { stage = 0; ++use; }
  }
  do { nent = pair_drain(&p, &S, n, nent, true); } while (nent);
}

// ----------------------------------------------------------------------------- K4b handshake resolve
// Phase 2b: a binding happens iff the proposal is mutual (a7).  One thread per word of the hasprop
// bitmap; the lower slot of a mutual pair rewrites both species in place (anchor -> complex, the
// other -> DEAD; S10).  No other thread reads or writes the species of a matched agent in this
// kernel: a third agent that proposed to one of them only reads best[] / bslot[].

// Slot of the agent with id `idj` at squared distance d2 from agent i (it exists): the plain
// neighbourhood sweep, used only when prop[i] names another qualifying partner than the minimum (see K4, D).
__device__ __noinline__ uint32_t find_partner(const Params* pp, uint32_t i, uint32_t idj) {
  const Params& p = *pp;
  const int4 qi = p.oth.r[i];
  const int32_t x = qi.x, y = qi.y, z = qi.z, R = p.max_r;
  const int32_t xlo = cell_coord(max(x - R, 0), p), xhi = min(cell_coord(x + R, p), p.nx - 1);
  const int32_t ylo = cell_coord(max(y - R, 0), p), yhi = min(cell_coord(y + R, p), p.ny - 1);
  const int32_t zlo = cell_coord(max(z - R, 0), p), zhi = min(cell_coord(z + R, p), p.nz - 1);
  for (int32_t cz = zlo; cz <= zhi; ++cz)
    for (int32_t cy = ylo; cy <= yhi; ++cy) {
      const uint32_t rowc = ((uint32_t)cz * (uint32_t)p.ny + (uint32_t)cy) * (uint32_t)p.nx;
      for (uint32_t j = p.cell[rowc + xlo]; j < p.cell[rowc + xhi + 1]; ++j)
        if ((uint32_t)p.oth.r[j].w == idj) return j;
    }
  return kNoProp;
}

__global__ void __launch_bounds__(256) k_resolve(const __grid_constant__ Params p) {
  __shared__ int32_t s_delta[kMaxRowWidth];
  delta_zero(s_delta, p.row_width);
  const uint32_t n = p.cell[p.n_cells], t = p.scal->t;
  const uint32_t nw = (n + 31u) >> 5;
  const DevTables* __restrict__ T = p.tab;
  for (uint32_t w = blockIdx.x * blockDim.x + threadIdx.x; w < nw; w += gridDim.x * blockDim.x) {
    uint32_t bits = p.hasprop[w];
    while (bits) {
      const uint32_t b = __ffs(bits) - 1u;
      bits &= bits - 1u;
      const uint32_t i = w * 32u + b;
      const uint32_t idj = (uint32_t)p.best[i];            // low word of (d2, id of the proposed partner)
      uint32_t j = p.prop[i];
      if (j >= n || (uint32_t)p.oth.r[j].w != idj) j = find_partner(&p, i, idj);
      MOLSIM_CHECK(p, j < n);                                 // the partner named by the key exists
      if (j <= i || j >= n) continue;                         // the lower slot handles the pair
      const uint32_t idi = (uint32_t)p.oth.r[i].w;
      if ((uint32_t)p.best[j] != idi) continue;               // not mutual (best[j] = kNoKey if j never proposed)
      const uint16_t si = p.oth.sp[i], sj = p.oth.sp[j];
      const DevRx& rx = T->rx[T->rxmap[(uint32_t)si * kMaxSpecies + sj]];
      const bool anchor_i = (si != sj) ? (si == rx.a) : (idi < idj);
      p.oth.sp[i] = anchor_i ? rx.cplx : kDead;
      p.oth.sp[j] = anchor_i ? kDead : rx.cplx;
      int32_t* d = s_delta + ((uint32_t)p.oth.r[i].x >> p.stride_shift) * p.n_species;
      atomicSub(&d[si], 1); atomicSub(&d[sj], 1); atomicAdd(&d[rx.cplx], 1);
    }
  }
  delta_flush(s_delta, p.counts + (size_t)(t + 1) * p.row_width, p.row_width);
}

// ----------------------------------------------------------------------------- K5 unimolecular + next histogram
// Phase 3 (a8): per agent, per channel, Philox(seed, t, id) word < threshold.  Most agents belong to
// a species without channels: a thread reads the species of 8 agents with one 128-bit load; the
// slots of those that have channels (chan_mask) are compacted into a shared list and only these
// are processed, one per thread, so the Philox work is dense.  Species are rewritten in place only
// where they change.  The same pass clears the proposal state K4 left (hasprop byte -> best[]).  Firing parents
// are appended to the birth list and flagged in the id-indexed birth bitmap (4 bits per id) that K6 ranks.
// Counts deltas are block-aggregated.
//
// With the species of the tile final (nothing after this pass changes a sorted agent), the same kernel takes the
// cell histogram of step t+1 (a3): move_agent() for step t+1 gives the cell every survivor will be sorted into,
// and a run of equal keys in a warp adds its length to that cell's counter (fire-and-forget atomics into the
// OTHER cell array, zeroed meanwhile).  The next step therefore starts at its scan: the separate histogram
// pass of round 1, its rank array and one launch are gone, and the species are streamed once for both jobs.
// Newborns are counted by K6, which places them.  With kUni = false the kernel is only the histogram pass, of
// the CURRENT arrays for the current step: the prologue after seeding / loading.
__device__ __forceinline__ void uni_one(const Params& p, const DevTables* __restrict__ T, uint32_t i, uint16_t s0,
                                        uint32_t t, int32_t* s_delta, uint16_t* s_sp_slot) {
  const DevSpecies& S = T->sp[s0];
  const uint32_t nch = S.n_channels;
  const uint32_t id = (uint32_t)p.oth.r[i].w;
  const uint4 r = philox_sim(p, id, 0u, t, kTagUni);
  const uint32_t rr[4] = {r.x, r.y, r.z, r.w};
  bool consumed = false;
  uint16_t s = s0;
  uint32_t mask = 0;
#pragma unroll
  for (uint32_t k = 0; k < 4u; ++k) {
    if (k >= nch) break;
    const DevChannel ch = S.ch[k];
    if (ch.kind == kChNone) continue;
    bool fired;
    if (ch.kind == kChDelayed) {
      const uint32_t tf = *((volatile uint32_t*)&p.scal->t_first[ch.rule]);
      fired = tf != kNever && t == tf + ch.thr;
    } else {
      fired = fire(rr[k], ch.thr);
    }
    if (!fired) continue;
    switch (ch.kind) {
      case kChBirth:
        mask |= 1u << k;
        if (ch.marks_first) atomicMin(&p.scal->t_first[ch.rule], t);
        break;
      case kChDelayed: mask |= 1u << k; break;
      case kChRelease: if (!consumed) { consumed = true; s = ch.prod0; mask |= 1u << k; } break;
      case kChConvert: if (!consumed) { consumed = true; s = ch.prod0; } break;
      case kChDegrade: if (!consumed) { consumed = true; s = kDead; } break;
    }
  }
  if (s == s0 && !mask) return;
  int32_t* d = s_delta + ((uint32_t)p.oth.r[i].x >> p.stride_shift) * p.n_species;
  if (s != s0) {
    p.oth.sp[i] = s;
    *s_sp_slot = s;                        // the tile copy the histogram part reads
    atomicSub(&d[s0], 1);
    if (s != kDead) atomicAdd(&d[s], 1);
  }
  if (mask) {
    for (uint32_t k = 0; k < 4u; ++k) if (mask >> k & 1u) atomicAdd(&d[S.ch[k].prod1], 1);
    atomicOr(&p.bits[id >> 3], mask << ((id & 7u) * 4u));
    atomicAdd(&p.birth_mid[id >> kMidShift], (uint32_t)__popc(mask));     // newborn counts per 256 ids and per
    atomicAdd(&p.birth_top[id >> p.top_shift], (uint32_t)__popc(mask));   // 2^top_shift ids: K6 ranks from these
    const uint32_t e = atomicAdd(&p.scal->birth_count, 1u);
    MOLSIM_CHECK(p, e < p.capacity && id < p.id_capacity);
    p.birth_list[e] = make_uint2(i, mask | ((uint32_t)s0 << 16));
  }
}

constexpr int kUniThreads = 256;
constexpr int kUniTile = kUniThreads * 8;
// Dynamic shared memory: [Gaussian tables (if kGaussSmem)] [counts deltas, row_width words (if kUni)].
template <bool kGaussSmem, bool kUni, int kMinBlk>
__global__ void __launch_bounds__(kUniThreads, kMinBlk) k_uni_hist(Params p) {
  extern __shared__ __align__(16) int16_t s_dyn[];
  __shared__ MoveTables M;
  __shared__ __align__(16) uint16_t s_sp[kUniTile];   // species of the tile, after the unimolecular reactions
  __shared__ uint16_t s_list[kUni ? kUniTile : 1];     // tile-local slots of the agents that have channels
  __shared__ uint32_t s_n;
  const int16_t* g = stage_tables<kGaussSmem>(p, M, s_dyn);
  int32_t* s_delta = reinterpret_cast<int32_t*>(s_dyn + (kGaussSmem ? (((p.n_classes << p.table_bits) + 7u) & ~7u) : 0u));
  if (kUni) delta_zero(s_delta, p.row_width);
  const Soa src = kUni ? p.oth : p.cur;
  uint32_t* __restrict__ hist = (kUni ? p.cell_next : p.cell) + 1;
  const uint32_t n = kUni ? p.cell[p.n_cells] : p.scal->n_slots;
  const uint32_t t = p.scal->t, t_move = kUni ? t + 1u : t;
  const DevTables* __restrict__ T = p.tab;
  const uint32_t lane = threadIdx.x & 31u;
  for (uint32_t base = blockIdx.x * kUniTile; base < n; base += gridDim.x * kUniTile) {   // block-uniform
    if (kUni) {
      if (threadIdx.x == 0) s_n = 0;
      __syncthreads();                      // also: the previous tile's readers of s_sp / s_list are done
      const uint32_t l0 = threadIdx.x * 8u, i0 = base + l0;
      uint32_t w[4] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu};
      if (i0 + 8u <= n) {
        const uint4 q = *reinterpret_cast<const uint4*>(src.sp + i0);
        w[0] = q.x; w[1] = q.y; w[2] = q.z; w[3] = q.w;
      } else {
        for (uint32_t k = 0; i0 + k < n; ++k) {
          const uint32_t v = src.sp[i0 + k];
          w[k >> 1] = (k & 1u) ? ((w[k >> 1] & 0x0000FFFFu) | (v << 16)) : ((w[k >> 1] & 0xFFFF0000u) | v);
        }
      }
      *reinterpret_cast<uint4*>(s_sp + l0) = make_uint4(w[0], w[1], w[2], w[3]);
      // this step's proposals are resolved: put the touched best[] entries back to "none" for the next K4
      if (i0 < n) {
        uint8_t* hp = reinterpret_cast<uint8_t*>(p.hasprop) + (i0 >> 3);
        uint32_t bits = *hp;
        if (bits) {
          *hp = 0;
          while (bits) { p.best[i0 + __ffs(bits) - 1u] = kNoKey; bits &= bits - 1u; }
        }
      }
      uint32_t mask = 0;
#pragma unroll
      for (uint32_t k = 0; k < 8u; ++k) {
        const uint32_t s = (w[k >> 1] >> ((k & 1u) * 16u)) & 0xFFFFu;
        if (s != kDead && ((p.chan_mask >> s) & 1ull)) mask |= 1u << k;
      }
      // compact: warp-inclusive scan of the counts, one shared atomic per warp
      const uint32_t cnt = __popc(mask);
      uint32_t incl = cnt;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl, d);
        if (lane >= (uint32_t)d) incl += o;
      }
      const uint32_t wtotal = __shfl_sync(0xFFFFFFFFu, incl, 31);
      uint32_t wbase = 0;
      if (lane == 31 && wtotal) wbase = atomicAdd(&s_n, wtotal);
      wbase = __shfl_sync(0xFFFFFFFFu, wbase, 31);
      uint32_t pos = wbase + incl - cnt;
      while (mask) {
        s_list[pos++] = (uint16_t)(l0 + __ffs(mask) - 1u);
        mask &= mask - 1u;
      }
      __syncthreads();
      const uint32_t m = s_n;
      for (uint32_t k = threadIdx.x; k < m; k += kUniThreads) {
        const uint32_t l = s_list[k];
        uni_one(p, T, base + l, s_sp[l], t, s_delta, &s_sp[l]);
      }
      __syncthreads();                      // the tile's species are final
    }
    // ---- cell histogram of the step that moves these agents next: two batches of four agents in flight
#pragma unroll
    for (uint32_t half = 0; half < 2u; ++half) {
      uint16_t s[4];
      int4 q[4];
      uint32_t key[4];
#pragma unroll
      for (uint32_t a = 0; a < 4u; ++a) {
        const uint32_t l = (half * 4u + a) * kUniThreads + threadIdx.x, i = base + l;
        s[a] = kDead;
        if (i < n) { s[a] = kUni ? s_sp[l] : src.sp[i]; q[a] = src.r[i]; }   // the record load is not gated on the species
      }
#pragma unroll
      for (uint32_t a = 0; a < 4u; ++a) {
        key[a] = 0xFFFFFFFFu;
        if (s[a] == kDead) continue;
        const Moved m = move_agent(p, M, g, s[a], q[a].x, q[a].y, q[a].z, (uint32_t)q[a].w, t_move);
        key[a] = cell_key(m.x, m.y, m.z, p);
      }
#pragma unroll
      for (uint32_t a = 0; a < 4u; ++a) {
        int leader; uint32_t rank, count;
        run_of_key(key[a], lane, leader, rank, count);
        MOLSIM_CHECK(p, s[a] == kDead || key[a] < p.n_cells);
        if (s[a] != kDead && rank == 0u) atomicAdd(&hist[key[a]], count);     // result unused: a reduction, no round trip
      }
    }
  }
  if (kUni) delta_flush(s_delta, p.counts + (size_t)(t + 1) * p.row_width, p.row_width);
}

// ----------------------------------------------------------------------------- K6 births + epilogue
// New ids are assigned in (parent id, channel) order (north_star (5), S14).  The birth bitmap (4 bits
// per id) is indexed by parent id, so a newborn's rank is the number of set bits below its own; K5
// also keeps the newborn count of every block of 256 ids (birth_mid) and of every 2^top_shift ids
// (birth_top, at most kMaxTop entries).  One launch: every block scans birth_top into shared memory,
// then one warp per firing parent adds the birth_mid entries and bitmap words between the block
// boundaries and the parent (a few dozen coalesced loads per lane at most) and lanes 0..3 place the
// newborns (phase 4, a9): newborn g of the step gets id next_id + g and slot n_sorted + g, and is counted in the
// next step's cell histogram like every survivor (K5).  The last block to finish then clears the touched
// birth-bitmap words and counters, advances the device scalars and seeds counts row t+2 with row t+1 (the
// next step adds its deltas to it; a10).
__global__ void __launch_bounds__(kScanThreads) k_births(Params p) {
  __shared__ uint32_t s_warp[9];
  __shared__ uint32_t s_top[kMaxTop];
  __shared__ MoveTables M;
  __shared__ uint32_t s_last;
  const uint32_t nb = p.scal->birth_count;
  const uint32_t n_sorted = p.cell[p.n_cells];
  const uint32_t t = p.scal->t;
  uint32_t total = 0;
  bool bad_any = false;
  if (nb) {             // block-uniform
    stage_tables<false>(p, M, nullptr);
    const uint32_t next_id = p.scal->next_id;
    const uint32_t n_top = ((next_id - 1u) >> p.top_shift) + 1u;          // parents have ids < next_id
    constexpr uint32_t kPer = kMaxTop / kScanThreads;
    uint32_t v[kPer], sum = 0;
#pragma unroll
    for (uint32_t k = 0; k < kPer; ++k) {
      const uint32_t j = threadIdx.x * kPer + k;
      v[k] = j < n_top ? p.birth_top[j] : 0u;
      sum += v[k];
    }
    uint32_t e0 = block_excl_scan(sum, total, s_warp);
#pragma unroll
    for (uint32_t k = 0; k < kPer; ++k) { s_top[threadIdx.x * kPer + k] = e0; e0 += v[k]; }
    __syncthreads();
    uint32_t bad = 0;
    if ((unsigned long long)n_sorted + total > p.capacity) bad |= 1u;
    if ((unsigned long long)next_id + total > p.id_capacity) bad |= 2u;
    if (bad && blockIdx.x == 0 && threadIdx.x == 0) atomicOr(&p.scal->err, bad);
    bad_any = bad != 0u;
    if (!bad) {
      const DevTables* __restrict__ T = p.tab;
      uint32_t* __restrict__ hist = p.cell_next + 1;
      const uint32_t lane = threadIdx.x & 31u, wpb = kScanThreads / 32;
      for (uint32_t e = blockIdx.x * wpb + (threadIdx.x >> 5); e < nb; e += gridDim.x * wpb) {
        const uint2 ent = p.birth_list[e];
        const uint32_t slot = ent.x, mask = ent.y & 0xFu, pre = ent.y >> 16;
        const uint32_t pid = (uint32_t)p.oth.r[slot].w;
        uint32_t part = 0;
        for (uint32_t j = ((pid >> p.top_shift) << (p.top_shift - kMidShift)) + lane; j < (pid >> kMidShift); j += 32u)
          part += p.birth_mid[j];
        const uint32_t w0 = (pid >> kMidShift) << (kMidShift - 3u), w1 = pid >> 3;      // bitmap words of this 256-id block
        if (w0 + lane < w1) part += __popc(p.bits[w0 + lane]);
        if (lane == 31u) part += __popc(p.bits[w1] & ((1u << ((pid & 7u) * 4u)) - 1u));
        const uint32_t rank0 = s_top[pid >> p.top_shift] + __reduce_add_sync(0xFFFFFFFFu, part);
        if (lane < 4u && (mask >> lane & 1u)) {
          const uint32_t k = lane, rank = rank0 + __popc(mask & ((1u << k) - 1u));
          const int4 qp = p.oth.r[slot];
          const int32_t px = qp.x, py = qp.y, pz = qp.z;
          const int32_t rbase = (int32_t)(((uint32_t)px >> p.stride_shift) << p.stride_shift);
          const int32_t lx = px - rbase;
          const uint16_t sp_new = T->sp[pre].ch[k].prod1;
          const uint4 r = philox_sim(p, pid, k, t, kTagBirth);
          int32_t qx = lx + (int32_t)__umulhi(r.x, 21u) - 10;
          int32_t qy = py + (int32_t)__umulhi(r.y, 21u) - 10;
          int32_t qz = pz + (int32_t)__umulhi(r.z, 21u) - 10;
          const DevComp& c = T->comp[T->sp[sp_new].compartment];
          if (c.shape == 0) { qx = mirror(qx, c.L); qy = mirror(qy, c.L); qz = mirror(qz, c.L); }
          else if (!comp_valid(c, qx, qy, qz)) { qx = lx; qy = py; qz = pz; }
          const uint32_t dst = n_sorted + rank;
          MOLSIM_CHECK(p, dst < p.capacity && rank < total);
          p.oth.r[dst] = make_int4(qx + rbase, qy, qz, (int32_t)(next_id + rank));
          p.oth.sp[dst] = sp_new;
          // the newborn's cell in the next step's sort
          const Moved m = move_agent(p, M, p.gauss, sp_new, qx + rbase, qy, qz, next_id + rank, t + 1u);
          atomicAdd(&hist[cell_key(m.x, m.y, m.z, p)], 1u);
        }
      }
    }
  }
  // ---- epilogue, by the last block to get here (every block's births are placed and its bitmap reads are done)
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(&p.scal->ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  for (uint32_t e = threadIdx.x; e < nb; e += blockDim.x) {
    const uint32_t pid = (uint32_t)p.oth.r[p.birth_list[e].x].w;
    p.bits[pid >> 3] = 0u; p.birth_mid[pid >> kMidShift] = 0u; p.birth_top[pid >> p.top_shift] = 0u;
  }
  Scalars* sc = p.scal;
  const uint32_t* src = p.counts + (size_t)(t + 1) * p.row_width;
  uint32_t* dst = p.counts + (size_t)(t + 2) * p.row_width;
  for (uint32_t k = threadIdx.x; k < p.row_width; k += blockDim.x) dst[k] = __ldcg(src + k);
  if (threadIdx.x == 0) {
    const uint32_t add = (bad_any || sc->err) ? 0u : total;
    sc->n_slots = n_sorted + add;
    sc->next_id += add;
    sc->t = t + 1;
    sc->birth_count = 0; sc->total_births = 0; sc->ticket = 0;
  }
}

// ----------------------------------------------------------------------------- off the hot path
// Seeding (DESIGN.md §1 "Seeding", S15).
__global__ void k_seed(Params p, uint32_t species, uint32_t replica, uint32_t count, uint32_t first_id,
                       uint32_t dst_base, uint32_t pk0, uint32_t pk1) {
  const DevComp c = p.tab->comp[p.tab->sp[species].compartment];
  const int32_t rbase = (int32_t)(replica << p.stride_shift);
  for (uint32_t n = blockIdx.x * blockDim.x + threadIdx.x; n < count; n += gridDim.x * blockDim.x) {
    const uint32_t id = first_id + n;
    int32_t x, y, z;
    if (c.shape == 0) {
      const uint4 r = philox4x32_10(id, 0u, 0u, kTagPlace, pk0, pk1);
      x = (int32_t)__umulhi(r.x, (uint32_t)c.L); y = (int32_t)__umulhi(r.y, (uint32_t)c.L);
      z = (int32_t)__umulhi(r.z, (uint32_t)c.L);
    } else {
      const uint32_t side = 2u * (uint32_t)c.r_out + 1u;
      x = c.cx + c.r_out; y = c.cy; z = c.cz;
      for (uint32_t attempt = 0; attempt < 64u; ++attempt) {
        const uint4 r = philox4x32_10(id, attempt, 0u, kTagPlace, pk0, pk1);
        const int32_t qx = c.cx - c.r_out + (int32_t)__umulhi(r.x, side);
        const int32_t qy = c.cy - c.r_out + (int32_t)__umulhi(r.y, side);
        const int32_t qz = c.cz - c.r_out + (int32_t)__umulhi(r.z, side);
        if (comp_valid(c, qx, qy, qz)) { x = qx; y = qy; z = qz; break; }
      }
    }
    const uint32_t d = dst_base + n;
    p.cur.r[d] = make_int4(x + rbase, y, z, (int32_t)id);
    p.cur.sp[d] = (uint16_t)species;
  }
}

// Full histogram of the current state into counts row `r` (after seeding / loading), and its copy
// into row r+1 as the base of the next step's deltas.  With `check` (sim_load_agents: caller data) every agent is
// validated as well: species, replica tile, id below next_id and not used twice (the id-indexed birth bitmap, all zero
// between steps, serves as the "seen" set and is cleared again by k_clear_ids), and a position inside the compartment
// of its species, which is what bounds every cell key the step computes.  A violation sets err bit 2.
__global__ void __launch_bounds__(256) k_count_row(Params p, uint32_t r, uint32_t n_slots, bool check) {
  __shared__ int32_t s_delta[kMaxRowWidth];
  delta_zero(s_delta, p.row_width);
  const uint32_t next_id = p.scal->next_id;
  const DevTables* __restrict__ T = p.tab;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += gridDim.x * blockDim.x) {
    const uint16_t s = p.cur.sp[i];
    if (s == kDead) continue;
    const int4 q = p.cur.r[i];
    const uint32_t rep = (uint32_t)q.x >> p.stride_shift, id = (uint32_t)q.w;
    if (check) {
      bool ok = q.x >= 0 && s < p.n_species && rep < p.n_replicas && id < next_id;
      if (ok) ok = comp_valid(T->comp[T->sp[s].compartment], q.x - (int32_t)(rep << p.stride_shift), q.y, q.z);
      if (ok) ok = !(atomicOr(&p.bits[id >> 3], 1u << ((id & 7u) * 4u)) >> ((id & 7u) * 4u) & 1u);
      if (!ok) { atomicOr(&p.scal->err, 4u); continue; }
    }
    atomicAdd(&s_delta[rep * p.n_species + s], 1);
  }
  delta_flush(s_delta, p.counts + (size_t)r * p.row_width, p.row_width);
}
__global__ void __launch_bounds__(256) k_clear_ids(Params p, uint32_t n_slots) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += gridDim.x * blockDim.x) {
    const uint32_t id = (uint32_t)p.cur.r[i].w;
    if (id < p.id_capacity) p.bits[id >> 3] = 0u;
  }
}
__global__ void k_copy_row(Params p, uint32_t r) {
  const uint32_t* src = p.counts + (size_t)r * p.row_width;
  uint32_t* dst = p.counts + (size_t)(r + 1) * p.row_width;
  for (uint32_t k = threadIdx.x; k < p.row_width; k += blockDim.x) dst[k] = src[k];
}

// sim_read_agents: gather live agents into the scratch (oth) buffers (warp-aggregated append).
__global__ void __launch_bounds__(256) k_gather_live(Params p, uint32_t n_slots) {
  const uint32_t lane = threadIdx.x & 31u;
  for (uint32_t base = blockIdx.x * blockDim.x; base < n_slots; base += gridDim.x * blockDim.x) {
    const uint32_t i = base + threadIdx.x;
    const uint16_t s = i < n_slots ? p.cur.sp[i] : kDead;
    const uint32_t live = __ballot_sync(0xFFFFFFFFu, s != kDead);
    uint32_t d = 0;
    if (lane == 0 && live) d = atomicAdd(&p.scal->n_read, (uint32_t)__popc(live));
    d = __shfl_sync(0xFFFFFFFFu, d, 0) + __popc(live & ((1u << lane) - 1u));
    if (s == kDead) continue;
    // the C ABI speaks separate arrays: the scratch record buffer is written as four planes of `capacity` words
    const int4 q = p.cur.r[i];
    int32_t* plane = reinterpret_cast<int32_t*>(p.oth.r);
    plane[d] = q.x; plane[(size_t)p.capacity + d] = q.y; plane[2 * (size_t)p.capacity + d] = q.z;
    plane[3 * (size_t)p.capacity + d] = q.w; p.oth.sp[d] = s;
  }
}

// sim_load_agents: the caller's separate x / y / z / id arrays were copied into the four planes of the scratch
// record buffer; interleave them into the current records.
__global__ void __launch_bounds__(256) k_pack_records(Params p, uint32_t n) {
  const int32_t* plane = reinterpret_cast<const int32_t*>(p.oth.r);
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    p.cur.r[i] = make_int4(plane[i], plane[(size_t)p.capacity + i], plane[2 * (size_t)p.capacity + i],
                           plane[3 * (size_t)p.capacity + i]);
}

}  // namespace molsim
