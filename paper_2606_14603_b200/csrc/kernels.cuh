// kernels.cuh — the hand-written sm_100a kernels of the molecule-agent step.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// One step = K1 move+hist -> K2 cell scan (2 launches) -> K3 scatter -> K4 neighbour/proposal ->
// K5 resolve+unimolecular -> K6 birth scan (2 launches) + birth placement -> K7 epilogue.
// Every decision is keyed by agent id (never by slot), so the nondeterministic slot order the
// histogram atomics produce inside a cell cannot change any result.
#pragma once
#include "device_types.cuh"

namespace molsim {

// ----------------------------------------------------------------------------- Philox4x32-10
// north_star (2), S2.  counter (c0,c1,c2,c3), key (k0,k1); 10 rounds, 9 key bumps.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;   // the bump after the last round is dead code
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

// ----------------------------------------------------------------------------- K1 move + histogram
// Phase 1 (Brownian move, boundary and compartment rule) fused with the cell-key histogram of the
// counting sort.  Gaussian inverse-CDF tables are staged in shared memory.
// The histogram uses warp-aggregated atomics (__match_any_sync on the cell key): agents are
// nearly cell-sorted from the previous step, so a warp touches few distinct cells.
// Counts deltas for membrane crossings go straight to counts row t+1 (rare events).
template <bool kHist>
__global__ void __launch_bounds__(256) k_move_hist(Params p, int gauss_in_smem) {
  extern __shared__ int16_t s_gauss[];
  const int16_t* g = p.gauss;
  if (gauss_in_smem) {
    const uint32_t n_tab = p.n_classes << p.table_bits;
    for (uint32_t k = threadIdx.x; k < n_tab; k += blockDim.x) s_gauss[k] = p.gauss[k];
    __syncthreads();
    g = s_gauss;
  }
  const uint32_t n = p.scal->n_slots, t = p.scal->t;
  const DevTables* __restrict__ T = p.tab;
  const uint32_t sh = 32u - p.table_bits;
  const uint32_t lane = threadIdx.x & 31u;
  uint32_t* __restrict__ row = p.counts + (size_t)(t + 1) * p.row_width;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t base = blockIdx.x * blockDim.x; base < n; base += stride) {   // warp-uniform trip count
    const uint32_t i = base + threadIdx.x;
    uint32_t key = 0xFFFFFFFFu;
    bool live = false;
    if (i < n) {
      uint16_t s = p.sp_cur[i];
      if (s != kDead) {
        live = true;
        int32_t x = p.cur.x[i], y = p.cur.y[i], z = p.cur.z[i];
        const DevSpecies& S = T->sp[s];
        const uint32_t cls = S.sigma_class;
        if (cls) {
          const uint32_t id = p.cur.id[i];
          const uint4 r = philox4x32_10(id, 0u, t, kTagMove, p.key0, p.key1);
          const int16_t* tb = g + (cls << p.table_bits);
          const int32_t rbase = (int32_t)(((uint32_t)x >> p.stride_shift) << p.stride_shift);
          int32_t qx = x - rbase + tb[r.x >> sh], qy = y + tb[r.y >> sh], qz = z + tb[r.z >> sh];
          const DevComp& c = T->comp[S.compartment];
          bool accept = true;
          if (c.shape == 0) {
            qx = mirror(qx, c.L); qy = mirror(qy, c.L); qz = mirror(qz, c.L);
          } else if (!comp_valid(c, qx, qy, qz)) {
            accept = false;
            const uint16_t ct = S.cross_to;
            if (ct != kDead && comp_valid(T->comp[T->sp[ct].compartment], qx, qy, qz) && fire(r.w, S.cross_thr)) {
              accept = true;
              p.sp_cur[i] = ct;
              const uint32_t rep = (uint32_t)x >> p.stride_shift;
              atomicSub(&row[rep * p.n_species + s], 1u);
              atomicAdd(&row[rep * p.n_species + ct], 1u);
            }
          }
          if (accept) {
            x = qx + rbase; y = qy; z = qz;
            p.cur.x[i] = x; p.cur.y[i] = y; p.cur.z[i] = z;
          }
        }
        if (kHist) key = cell_key(x, y, z, p);
      }
    }
    if (kHist) {
      const uint32_t peers = __match_any_sync(0xFFFFFFFFu, key);
      const int leader = __ffs(peers) - 1;
      const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
      uint32_t first = 0;
      if (live && (int)lane == leader) first = atomicAdd(&p.cell[key], (uint32_t)__popc(peers));
      first = __shfl_sync(0xFFFFFFFFu, first, leader);
      if (live) p.off[i] = first + rank;
    }
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

// ----------------------------------------------------------------------------- K3 scatter / reorder
// Counting-sort scatter that reorders the whole structure of arrays into cell order (a5) and drops
// DEAD slots, which is the compaction of the previous step's deaths (fused, a9).
__global__ void __launch_bounds__(256) k_scatter(Params p) {
  const uint32_t n = p.scal->n_slots;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint16_t s = p.sp_cur[i];
    if (s == kDead) continue;
    const int32_t x = p.cur.x[i], y = p.cur.y[i], z = p.cur.z[i];
    const uint32_t dst = p.cell[cell_key(x, y, z, p)] + p.off[i];
    p.oth.x[dst] = x; p.oth.y[dst] = y; p.oth.z[dst] = z;
    p.oth.id[dst] = p.cur.id[i];
    p.sp_sorted[dst] = s;
  }
}

// ----------------------------------------------------------------------------- K4 neighbour + proposal
// Phase 2a: each agent whose species can bind proposes its eligible partner with the smallest
// (dist^2, id) among those that pass the symmetric pair draw (a6).  Only the cells its R-ball
// overlaps are visited (exact: a cell it does not overlap cannot hold an in-range partner); with
// x-fastest cell keys the cells of one (y,z) row are one contiguous slot range.
__global__ void __launch_bounds__(128) k_neighbour(Params p) {
  const uint32_t n = p.cell[p.n_cells], t = p.scal->t;
  const DevTables* __restrict__ T = p.tab;
  const int32_t R = p.max_r;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint16_t s = p.sp_sorted[i];
    uint32_t best_j = kNoProp;
    if (T->sp[s].binds) {
      const int32_t x = p.oth.x[i], y = p.oth.y[i], z = p.oth.z[i];
      const uint32_t id = p.oth.id[i];
      const int32_t xlo = cell_coord(max(x - R, 0), p), xhi = min(cell_coord(x + R, p), p.nx - 1);
      const int32_t ylo = cell_coord(max(y - R, 0), p), yhi = min(cell_coord(y + R, p), p.ny - 1);
      const int32_t zlo = cell_coord(max(z - R, 0), p), zhi = min(cell_coord(z + R, p), p.nz - 1);
      unsigned long long best = ~0ull;
      const uint8_t* __restrict__ rxrow = T->rxmap + (uint32_t)s * kMaxSpecies;
      for (int32_t cz = zlo; cz <= zhi; ++cz) {
        for (int32_t cy = ylo; cy <= yhi; ++cy) {
          const uint32_t rowc = ((uint32_t)cz * (uint32_t)p.ny + (uint32_t)cy) * (uint32_t)p.nx;
          const uint32_t j0 = p.cell[rowc + xlo], j1 = p.cell[rowc + xhi + 1];
          for (uint32_t j = j0; j < j1; ++j) {
            const int32_t dx = p.oth.x[j] - x;
            if (abs(dx) > R) continue;
            const int32_t dy = p.oth.y[j] - y;
            if (abs(dy) > R) continue;
            const int32_t dz = p.oth.z[j] - z;
            if (abs(dz) > R) continue;
            const uint32_t d2 = (uint32_t)(dx * dx) + (uint32_t)(dy * dy) + (uint32_t)(dz * dz);
            if (d2 > p.max_r2 || j == i) continue;
            const uint32_t e = rxrow[p.sp_sorted[j]];
            if (e == 0xFFu) continue;
            const DevRx& rx = T->rx[e];
            if (d2 > rx.r2) continue;
            const uint32_t idj = p.oth.id[j];
            const uint4 r = philox4x32_10(min(id, idj), max(id, idj), t, kTagPair, p.key0, p.key1);
            if (!fire(r.x, rx.thr)) continue;
            const unsigned long long k = ((unsigned long long)d2 << 32) | idj;
            if (k < best) { best = k; best_j = j; }
          }
        }
      }
    }
    p.prop[i] = best_j;
  }
}

// ----------------------------------------------------------------------------- K5 resolve + unimolecular
// Phase 2b (mutual proposals bind, a7) and phase 3 (unimolecular channels, a8).  Species are read
// from the sorted copy and written to sp_cur, so a partner's pre-binding species is never
// overwritten while it is still needed.  Firing parents are appended to the birth list and flagged
// in the id-indexed birth bitmap (4 bits per id) that K6 ranks.  Counts row t+1 receives deltas.
__global__ void __launch_bounds__(256) k_resolve_uni(Params p) {
  const uint32_t n = p.cell[p.n_cells], t = p.scal->t;
  const DevTables* __restrict__ T = p.tab;
  uint32_t* __restrict__ row = p.counts + (size_t)(t + 1) * p.row_width;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint16_t s0 = p.sp_sorted[i];
    uint16_t s = s0;
    const uint32_t pr = p.prop[i];
    uint32_t id = 0;
    bool have_id = false;
    if (pr != kNoProp && p.prop[pr] == i) {
      const uint16_t sj = p.sp_sorted[pr];
      const DevRx& rx = T->rx[T->rxmap[(uint32_t)s * kMaxSpecies + sj]];
      id = p.oth.id[i]; have_id = true;
      const bool anchor = (s != sj) ? (s == rx.a) : (id < p.oth.id[pr]);
      s = anchor ? rx.cplx : kDead;
    }
    uint32_t mask = 0;
    const uint16_t pre = s;
    if (s != kDead) {
      const DevSpecies& S = T->sp[s];
      const uint32_t nch = S.n_channels;
      if (nch) {
        if (!have_id) id = p.oth.id[i];
        const uint4 r = philox4x32_10(id, 0u, t, kTagUni, p.key0, p.key1);
        const uint32_t rr[4] = {r.x, r.y, r.z, r.w};
        bool consumed = false;
        uint16_t news = s;
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
            case kChRelease: if (!consumed) { consumed = true; news = ch.prod0; mask |= 1u << k; } break;
            case kChConvert: if (!consumed) { consumed = true; news = ch.prod0; } break;
            case kChDegrade: if (!consumed) { consumed = true; news = kDead; } break;
          }
        }
        s = news;
      }
    }
    p.sp_cur[i] = s;
    if (s != s0 || mask) {
      const uint32_t rep = (uint32_t)p.oth.x[i] >> p.stride_shift;
      uint32_t* rr = row + rep * p.n_species;
      if (s != s0) {
        atomicSub(&rr[s0], 1u);
        if (s != kDead) atomicAdd(&rr[s], 1u);
      }
      if (mask) {
        const DevSpecies& P = T->sp[pre];
        for (uint32_t k = 0; k < 4u; ++k) if (mask >> k & 1u) atomicAdd(&rr[P.ch[k].prod1], 1u);
        atomicOr(&p.bits[id >> 3], mask << ((id & 7u) * 4u));
        const uint32_t e = atomicAdd(&p.scal->birth_count, 1u);
        p.birth_list[e] = make_uint2(i, mask | ((uint32_t)pre << 16));
      }
    }
  }
}

// ----------------------------------------------------------------------------- K6 birth ranking
// New ids are assigned in (parent id, channel) order (north_star (5), S14): the birth bitmap is
// indexed by parent id, so a newborn's rank is the popcount of all lower bits.  Two launches
// (segment sums, then per-64-id-chunk exclusive prefixes); both return at once on steps without births.
__device__ __forceinline__ uint32_t chunk_popc(const uint32_t* __restrict__ bits, uint32_t c) {
  const uint4 a = *reinterpret_cast<const uint4*>(bits + (size_t)c * 8u);
  const uint4 b = *reinterpret_cast<const uint4*>(bits + (size_t)c * 8u + 4u);
  return __popc(a.x) + __popc(a.y) + __popc(a.z) + __popc(a.w) + __popc(b.x) + __popc(b.y) + __popc(b.z) + __popc(b.w);
}

__global__ void __launch_bounds__(kScanThreads) k_birth_reduce(Params p) {
  __shared__ uint32_t s_warp[9];
  if (p.scal->birth_count == 0) return;
  const uint32_t n_chunks = (p.scal->next_id + 63u) >> 6;
  const uint32_t seg = ((n_chunks + gridDim.x - 1) / gridDim.x + kScanThreads - 1) / kScanThreads * kScanThreads;
  const uint32_t lo = min(blockIdx.x * seg, n_chunks), hi = min(lo + seg, n_chunks);
  uint32_t sum = 0;
  for (uint32_t c = lo + threadIdx.x; c < hi; c += kScanThreads) sum += chunk_popc(p.bits, c);
  const uint32_t tot = block_sum(sum, s_warp);
  if (threadIdx.x == 0) p.partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kScanThreads) k_birth_scan(Params p) {
  __shared__ uint32_t s_warp[9];
  if (p.scal->birth_count == 0) {
    if (blockIdx.x == 0 && threadIdx.x == 0) p.scal->total_births = 0;
    return;
  }
  const uint32_t n_chunks = (p.scal->next_id + 63u) >> 6;
  const uint32_t seg = ((n_chunks + gridDim.x - 1) / gridDim.x + kScanThreads - 1) / kScanThreads * kScanThreads;
  const uint32_t lo = min(blockIdx.x * seg, n_chunks), hi = min(lo + seg, n_chunks);
  uint32_t mine = 0;
  for (uint32_t b = threadIdx.x; b < blockIdx.x; b += kScanThreads) mine += p.partial[b];
  uint32_t running = block_sum(mine, s_warp);
  for (uint32_t tile = lo; tile < hi; tile += kScanThreads) {
    const uint32_t c = tile + threadIdx.x;
    const uint32_t v = c < hi ? chunk_popc(p.bits, c) : 0u;
    uint32_t total;
    const uint32_t e = running + block_excl_scan(v, total, s_warp);
    if (c < hi) p.chunk_prefix[c] = e;
    running += total;
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) p.scal->total_births = running;
}

// Phase 4: newborn placement, id assignment and append (a9).  Newborn g of the step gets
// id next_id + g and slot n_sorted + g.
__global__ void __launch_bounds__(128) k_births(Params p) {
  const uint32_t nb = p.scal->birth_count;
  if (nb == 0) return;
  const uint32_t n_sorted = p.cell[p.n_cells], total = p.scal->total_births;
  const uint32_t next_id = p.scal->next_id, t = p.scal->t;
  uint32_t bad = 0;
  if ((unsigned long long)n_sorted + total > p.capacity) bad |= 1u;
  if ((unsigned long long)next_id + total > p.id_capacity) bad |= 2u;
  if (bad) {
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(&p.scal->err, bad);
    return;
  }
  const DevTables* __restrict__ T = p.tab;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < nb; e += stride) {
    const uint2 ent = p.birth_list[e];
    const uint32_t slot = ent.x, mask = ent.y & 0xFu, pre = ent.y >> 16;
    const uint32_t pid = p.oth.id[slot];
    const int32_t px = p.oth.x[slot], py = p.oth.y[slot], pz = p.oth.z[slot];
    uint32_t rank = p.chunk_prefix[pid >> 6];
    for (uint32_t w = (pid >> 6) * 8u; w < (pid >> 3); ++w) rank += __popc(p.bits[w]);
    rank += __popc(p.bits[pid >> 3] & ((1u << ((pid & 7u) * 4u)) - 1u));
    const int32_t rbase = (int32_t)(((uint32_t)px >> p.stride_shift) << p.stride_shift);
    const int32_t lx = px - rbase;
    for (uint32_t k = 0; k < 4u; ++k) {
      if (!(mask >> k & 1u)) continue;
      const uint16_t sp_new = T->sp[pre].ch[k].prod1;
      const uint4 r = philox4x32_10(pid, k, t, kTagBirth, p.key0, p.key1);
      int32_t qx = lx + (int32_t)__umulhi(r.x, 21u) - 10;
      int32_t qy = py + (int32_t)__umulhi(r.y, 21u) - 10;
      int32_t qz = pz + (int32_t)__umulhi(r.z, 21u) - 10;
      const DevComp& c = T->comp[T->sp[sp_new].compartment];
      if (c.shape == 0) { qx = mirror(qx, c.L); qy = mirror(qy, c.L); qz = mirror(qz, c.L); }
      else if (!comp_valid(c, qx, qy, qz)) { qx = lx; qy = py; qz = pz; }
      const uint32_t dst = n_sorted + rank;
      p.oth.x[dst] = qx + rbase; p.oth.y[dst] = qy; p.oth.z[dst] = qz;
      p.oth.id[dst] = next_id + rank;
      p.sp_cur[dst] = sp_new;
      ++rank;
    }
  }
}

// ----------------------------------------------------------------------------- K7 epilogue
// Clears the touched bitmap words; the last block to finish advances the device scalars and
// seeds counts row t+2 with row t+1 (the next step adds its deltas to it; a10).
__global__ void __launch_bounds__(256) k_epilogue(Params p) {
  __shared__ uint32_t s_last;
  const uint32_t nb = p.scal->birth_count;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < nb; e += stride) {
    const uint32_t pid = p.oth.id[p.birth_list[e].x];
    p.bits[pid >> 3] = 0u;
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(&p.scal->ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
  __syncthreads();
  if (!s_last) return;
  Scalars* sc = p.scal;
  const uint32_t t = sc->t;
  const uint32_t* src = p.counts + (size_t)(t + 1) * p.row_width;
  uint32_t* dst = p.counts + (size_t)(t + 2) * p.row_width;
  for (uint32_t k = threadIdx.x; k < p.row_width; k += blockDim.x) dst[k] = __ldcg(src + k);
  if (threadIdx.x == 0) {
    const uint32_t add = sc->err ? 0u : sc->total_births;
    sc->n_slots = p.cell[p.n_cells] + add;
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
    p.cur.x[d] = x + rbase; p.cur.y[d] = y; p.cur.z[d] = z; p.cur.id[d] = id;
    p.sp_cur[d] = (uint16_t)species;
  }
}

// Full histogram of the current state into counts row `r` (after seeding / loading), and its copy
// into row r+1 as the base of the next step's deltas.
__global__ void k_count_row(Params p, uint32_t r, uint32_t n_slots) {
  uint32_t* row = p.counts + (size_t)r * p.row_width;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += gridDim.x * blockDim.x) {
    const uint16_t s = p.sp_cur[i];
    if (s == kDead) continue;
    atomicAdd(&row[((uint32_t)p.cur.x[i] >> p.stride_shift) * p.n_species + s], 1u);
  }
}
__global__ void k_copy_row(Params p, uint32_t r) {
  const uint32_t* src = p.counts + (size_t)r * p.row_width;
  uint32_t* dst = p.counts + (size_t)(r + 1) * p.row_width;
  for (uint32_t k = threadIdx.x; k < p.row_width; k += blockDim.x) dst[k] = src[k];
}

// sim_read_agents: gather live agents into the scratch (oth / sp_sorted) arrays.
__global__ void k_gather_live(Params p, uint32_t n_slots) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += gridDim.x * blockDim.x) {
    const uint16_t s = p.sp_cur[i];
    if (s == kDead) continue;
    const uint32_t d = atomicAdd(&p.scal->n_read, 1u);
    p.oth.x[d] = p.cur.x[i]; p.oth.y[d] = p.cur.y[i]; p.oth.z[d] = p.cur.z[i];
    p.oth.id[d] = p.cur.id[i]; p.sp_sorted[d] = s;
  }
}

}  // namespace molsim
