// device_types.cuh — device-side tables, launch parameters and small helpers.
// Product code (CUDA path).  Written from DESIGN.md §1; shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace molsim {

constexpr uint16_t kDead = 0xFFFFu;
constexpr uint32_t kNever = 0xFFFFFFFFu;
constexpr uint32_t kNoProp = 0xFFFFFFFFu;
constexpr int kMaxSpecies = 64;
constexpr int kMaxReactions = 64;
constexpr int kMaxCompartments = 8;
constexpr int kMaxRules = 8;
constexpr uint32_t kMidShift = 8;     // birth_mid: newborn counts per 2^8 parent ids
constexpr uint32_t kMaxTop = 2048;     // birth_top: entries (per 2^top_shift parent ids)

enum : uint32_t { kTagMove = 1, kTagPair = 2, kTagUni = 3, kTagBirth = 4, kTagPlace = 5 };
enum : uint8_t { kChNone = 0, kChBirth = 1, kChRelease = 2, kChConvert = 3, kChDegrade = 4, kChDelayed = 5 };

struct DevChannel {
  uint8_t kind, rule, marks_first, pad;
  uint16_t prod0, prod1;
  uint32_t thr;
};
struct DevSpecies {
  uint8_t sigma_class, compartment, n_channels, binds;
  uint16_t cross_to, pad;
  uint32_t cross_thr;
  DevChannel ch[4];
};
struct DevComp {
  int32_t shape, cx, cy, cz, L, r_out, r_in, pad;
  long long r_out2, r_in2;   // r_in2 = -1 when there is no hole
};
struct DevRx { uint16_t a, b, cplx, pad; uint32_t r2, thr; };

struct DevTables {
  DevSpecies sp[kMaxSpecies];
  DevComp comp[kMaxCompartments];
  DevRx rx[kMaxReactions];
  uint8_t rxmap[kMaxSpecies * kMaxSpecies];   // 0xFF = no reaction
};

// Scalars that live on the device so that sim_step(n) never needs the host between steps.
struct Scalars {
  uint32_t n_slots;        // length of the current (unsorted) arrays, DEAD slots included
  uint32_t next_id;
  uint32_t t;              // steps done
  uint32_t err;            // sticky: bit0 capacity, bit1 id space
  uint32_t birth_count;    // entries in the birth-parent list of this step
  uint32_t total_births;   // newborns of this step
  uint32_t ticket;         // last-block-done counter of the epilogue
  uint32_t n_read;         // sim_read_agents compaction counter
  uint32_t t_first[kMaxRules];
};

// One agent array set (north_star (1): int32 fixed-point x, y, z, uint32 id, uint16 species = 18 B/agent, all
// integer).  Two parallel arrays: a 16-byte record {x, y, z, id} and the species.  Round 1 kept five separate
// arrays; K1 and K3 turned out to be bound by the NUMBER of HBM streams they keep open, so
// the four 32-bit fields that always travel together are read with one 128-bit load and written with one
// 128-bit store.  The C ABI still speaks separate arrays.
struct Soa {
  int4* r;          // {x, y, z, (int32) id}
  uint16_t* sp;
};

struct Params {
  Soa cur, oth;             // cur: state at step start (moved in place); oth: cell-sorted copy,
                            // on which bind / unimolecular / births act in place
  unsigned long long* best; // proposal key (dist^2 << 32 | partner id) per sorted slot, ~0 = none
  uint32_t* prop;           // slot of the partner that last lowered best[i] (checked against the key in K4b)
  uint32_t* hasprop;        // 1 bit per sorted slot: best[i] was touched this step (cleared by K5)
  uint32_t* cell;           // this step's cell array: cell[0] = 0, cell[k + 1] = count of cell k (histogram), then its first
                            // slot (scan), then its end (scatter): from K4 on cell[k] = first slot of cell k, cell[n_cells] = n_sorted
  uint32_t* cell_next;      // the next step's cell array (histogram taken by this step's K5 / K6); the two swap every step
  uint32_t* partial;        // scan partials
  uint32_t* bits;           // birth bitmap, 4 bits per id
  uint32_t* birth_mid;      // newborns of this step per block of 256 parent ids
  uint32_t* birth_top;      // newborns of this step per 2^top_shift parent ids (<= 2048 entries)
  uint32_t top_shift;
  uint2* birth_list;        // (parent slot, mask | pre-species << 16)
  uint32_t* counts;         // [counts_rows][n_replicas][n_species]
  Scalars* scal;
  const DevTables* tab;
  const int16_t* gauss;     // [n_classes << B]
  uint32_t key0, key1;
  uint32_t rk0[10], rk1[10];   // Philox round keys of the simulation key: key + round * bump
  uint32_t capacity, id_capacity;
  uint32_t n_species, n_replicas, stride_shift, table_bits, n_classes;
  int32_t cell_size;
  uint32_t cell_magic, cell_mshift;   // v / cell_size == umulhi(v, cell_magic) >> cell_mshift for 0 <= v < 2^31
  int32_t nx, ny, nz;
  int32_t fwd_row[4];       // cell-index offset of the forward rows (y+1, z), (y-1, z+1), (y, z+1), (y+1, z+1)
  uint32_t n_cells;
  int32_t max_r;            // max interaction radius (ceil sqrt of max r2)
  uint32_t max_r2;
  uint32_t pack_shift, pack_k1, pack_u;   // K4's packed window test: coordinate shift, T + 2^w and 2^w - 1 - 2T per field
  uint32_t pack_span1, pack_span2;       // one / two cells in coarse x units (clamped to the field)
  uint32_t row_width;       // n_replicas * n_species
  unsigned long long binds_mask;   // bit s: species s takes part in a bimolecular reaction
  unsigned long long chan_mask;    // bit s: species s has unimolecular channels
};

// Checked build (-DMOLSIM_CHECKS, paper_2606_14603_b200/build.py MOLSIM_CHECKS=1 -> libmolsim_checked.so): every index the
// kernels derive from data (cell keys, destination slots, queue positions, look-up ranges) is tested against its
// bound and a violation sets err bit 3 (SIM_E_INTERNAL).  compute-sanitizer is closed on this GPU pool; the GPU parity
// tests run once against this build instead (profiles/r2_sanitizers.md).  The normal build compiles the checks away.
#ifdef MOLSIM_CHECKS
#define MOLSIM_CHECK(p, cond) do { if (!(cond)) atomicOr(&(p).scal->err, 8u); } while (0)
#else
#define MOLSIM_CHECK(p, cond) do { } while (0)
#endif

__device__ __forceinline__ bool fire(uint32_t u, uint32_t thr) { return thr == 0xFFFFFFFFu || u < thr; }

// Mirror about -1/2 and L - 1/2 (S5), branch-free: -1 - q == ~q, and for 0 <= a < 2L the reflected
// value 2L - 1 - a is the smaller of the two exactly when a >= L (one reflection suffices: validated).
__device__ __forceinline__ int32_t mirror(int32_t q, int32_t L) {
  const int32_t a = q ^ (q >> 31);
  return min(a, 2 * L - 1 - a);
}

__device__ __forceinline__ bool comp_valid(const DevComp& c, int32_t x, int32_t y, int32_t z) {
  if (c.shape == 0) return x >= 0 && x < c.L && y >= 0 && y < c.L && z >= 0 && z < c.L;
  long long dx = (long long)x - c.cx, dy = (long long)y - c.cy, dz = (long long)z - c.cz;
  long long r2 = dx * dx + dy * dy + dz * dz;
  return r2 <= c.r_out2 && r2 > c.r_in2;
}

// Exact floor(v / cell_size) for 0 <= v < 2^31 by multiply-high: with l = ceil(log2 d),
// m = floor(2^(31+l) / d) + 1 satisfies 2^(31+l) < m d <= 2^(31+l) + 2^l (Granlund-Montgomery, N = 31),
// so v / d = (v m) >> (31 + l); d >= 2 gives l >= 1 and m < 2^32, hence umulhi and a shift by l - 1.
__device__ __forceinline__ int32_t cell_coord(int32_t v, const Params& p) {
  return (int32_t)(__umulhi((uint32_t)v, p.cell_magic) >> p.cell_mshift);
}
__device__ __forceinline__ uint32_t cell_key(int32_t x, int32_t y, int32_t z, const Params& p) {
  return ((uint32_t)cell_coord(z, p) * (uint32_t)p.ny + (uint32_t)cell_coord(y, p)) * (uint32_t)p.nx +
         (uint32_t)cell_coord(x, p);
}

}  // namespace molsim
