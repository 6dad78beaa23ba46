// readout.cuh — kernels of the two read-outs next to the step.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include "device_types.cuh"

namespace molsim {

// ----------------------------------------------------------------------------- state checksum
// Order-independent 64-bit checksum of the live state (DESIGN.md §1 "Checksum"): the sum, modulo 2^64, over live
// agents of mix(mix(mix(x | y << 32) ^ (z | id << 32)) ^ species), coordinates as 32-bit patterns, mix = the
// splitmix64 finaliser.  A sum, so the slot order the sort leaves behind does not matter.  This is what lets the
// full-size runs the CPU oracle cannot repeat inside a test be compared step by step (tests/golden/trace_*.txt).
__device__ __forceinline__ unsigned long long mix64(unsigned long long v) {
  v ^= v >> 30; v *= 0xBF58476D1CE4E5B9ull;
  v ^= v >> 27; v *= 0x94D049BB133111EBull;
  v ^= v >> 31;
  return v;
}
__global__ void __launch_bounds__(256) k_checksum(Params p, uint32_t n_slots, unsigned long long* __restrict__ out) {
  unsigned long long sum = 0;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += gridDim.x * blockDim.x) {
    const uint16_t s = p.cur.sp[i];
    if (s == kDead) continue;
    const int4 q = p.cur.r[i];
    const unsigned long long lo = (unsigned long long)(uint32_t)q.x | ((unsigned long long)(uint32_t)q.y << 32);
    const unsigned long long hi = (unsigned long long)(uint32_t)q.z | ((unsigned long long)(uint32_t)q.w << 32);
    sum += mix64(mix64(mix64(lo) ^ hi) ^ (unsigned long long)s);
  }
#pragma unroll
  for (int d = 16; d; d >>= 1) sum += __shfl_xor_sync(0xFFFFFFFFu, sum, d);
  if ((threadIdx.x & 31u) == 0u && sum) atomicAdd(out, sum);
}

// ----------------------------------------------------------------------------- N3 threshold monitor
// One block per monitor; threads stride over the rows of the window, then a block reduction.
// Everything is integer and order-free (min / max / sum), so the result is unique (reading S24).
struct DevMonitor {
  uint32_t replica, n_species, threshold, first_row, n_rows, states_off;
  uint16_t species[4];
};
struct DevMonitorResult { uint32_t first_above, n_above, last_state, max_value, max_row, n_switches; };

constexpr int kMonThreads = 256;
__global__ void __launch_bounds__(kMonThreads) k_monitor(const uint32_t* __restrict__ counts, uint32_t row_width,
                                                         uint32_t n_species, const DevMonitor* __restrict__ mons,
                                                         DevMonitorResult* __restrict__ out, uint8_t* __restrict__ states) {
  const DevMonitor m = mons[blockIdx.x];
  auto value = [&](uint32_t t) {
    const uint32_t* row = counts + (size_t)t * row_width + m.replica * n_species;
    uint32_t v = 0;
    for (uint32_t k = 0; k < m.n_species; ++k) v += row[m.species[k]];
    return v;
  };
  uint32_t first = 0xFFFFFFFFu, n_above = 0, n_sw = 0;
  unsigned long long best = 0;     // (value << 32) | ~row: max picks the largest value, then the smallest row
  for (uint32_t k = threadIdx.x; k < m.n_rows; k += kMonThreads) {
    const uint32_t t = m.first_row + k, v = value(t);
    const uint32_t above = v > m.threshold ? 1u : 0u;
    if (above) { ++n_above; first = min(first, t); }
    best = max(best, ((unsigned long long)v << 32) | (0xFFFFFFFFu - t));
    if (k > 0) n_sw += above != (value(t - 1) > m.threshold ? 1u : 0u);
    if (states) states[m.states_off + k] = (uint8_t)above;
  }
  // block reduction: warp shuffles, then one shared slot per warp
  __shared__ uint32_t s_first[kMonThreads / 32], s_above[kMonThreads / 32], s_sw[kMonThreads / 32];
  __shared__ unsigned long long s_best[kMonThreads / 32];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    first = min(first, __shfl_xor_sync(0xFFFFFFFFu, first, d));
    n_above += __shfl_xor_sync(0xFFFFFFFFu, n_above, d);
    n_sw += __shfl_xor_sync(0xFFFFFFFFu, n_sw, d);
    best = max(best, __shfl_xor_sync(0xFFFFFFFFu, best, d));
  }
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  if (lane == 0) { s_first[warp] = first; s_above[warp] = n_above; s_sw[warp] = n_sw; s_best[warp] = best; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < kMonThreads / 32; ++w) {
      first = min(first, s_first[w]); n_above += s_above[w]; n_sw += s_sw[w]; best = max(best, s_best[w]);
    }
    DevMonitorResult r;
    r.first_above = first; r.n_above = n_above; r.n_switches = n_sw;
    r.last_state = value(m.first_row + m.n_rows - 1u) > m.threshold ? 1u : 0u;
    r.max_value = (uint32_t)(best >> 32); r.max_row = 0xFFFFFFFFu - (uint32_t)best;
    out[blockIdx.x] = r;
  }
}

// ----------------------------------------------------------------------------- N4 headless picture
// Pass 1: every live agent of the replica inside the window adds one to the counter of its
// (pixel, compartment) — a streaming read of the records and species with warp-level runs of equal pixels merged
// before the atomic (agents are cell-sorted, so neighbours in memory are neighbours in space).
// Pass 2: one thread per pixel turns the counters into RGBA (reading S25).
struct DevView {
  uint32_t replica, axis;
  int32_t u0, v0;
  uint32_t eu, ev, width, height, gain, n_comp;
  uint8_t palette[kMaxCompartments][4];
};

__global__ void __launch_bounds__(256) k_splat_count(Params p, DevView v, uint32_t n_slots, uint32_t* __restrict__ cnt) {
  const DevTables* __restrict__ T = p.tab;
  const uint32_t lane = threadIdx.x & 31u;
  for (uint32_t base = blockIdx.x * blockDim.x; base < n_slots; base += gridDim.x * blockDim.x) {   // warp-uniform
    const uint32_t i = base + threadIdx.x;
    uint32_t key = 0xFFFFFFFFu;
    if (i < n_slots) {
      const uint16_t s = p.cur.sp[i];
      const int4 r = p.cur.r[i];
      const int32_t x = r.x;
      if (s != kDead && ((uint32_t)x >> p.stride_shift) == v.replica) {
        const int32_t q[3] = {x - (int32_t)(v.replica << p.stride_shift), r.y, r.z};
        const int32_t u = v.axis == 0 ? q[1] : q[0], w = v.axis == 2 ? q[1] : q[2];
        const long long du = (long long)u - v.u0, dv = (long long)w - v.v0;
        if (du >= 0 && du < (long long)v.eu && dv >= 0 && dv < (long long)v.ev) {
          const uint32_t pu = (uint32_t)((unsigned long long)du * v.width / v.eu);
          const uint32_t pv = (uint32_t)((unsigned long long)dv * v.height / v.ev);
          key = (pv * v.width + pu) * v.n_comp + T->sp[s].compartment;
        }
      }
    }
    // merge runs of equal keys in the warp into one atomic
    const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, key, 1);
    const uint32_t heads = __ballot_sync(0xFFFFFFFFu, lane == 0u || key != prev);
    if (key != 0xFFFFFFFFu && (heads >> lane & 1u)) {
      const uint32_t above = heads & ~((2u << lane) - 1u);
      const uint32_t end = above ? (uint32_t)__ffs(above) - 1u : 32u;
      atomicAdd(&cnt[key], end - lane);
    }
  }
}

__global__ void __launch_bounds__(256) k_splat_colour(DevView v, const uint32_t* __restrict__ cnt, uchar4* __restrict__ img) {
  const uint32_t n_pix = v.width * v.height;
  for (uint32_t px = blockIdx.x * blockDim.x + threadIdx.x; px < n_pix; px += gridDim.x * blockDim.x) {
    uint32_t acc[3] = {0u, 0u, 0u}, any = 0u;
    for (uint32_t c = 0; c < v.n_comp; ++c) {
      const uint32_t n = cnt[px * v.n_comp + c];
      any |= n;
      const uint32_t inten = (uint32_t)min((unsigned long long)n * v.gain, 255ull);
#pragma unroll
      for (int k = 0; k < 3; ++k) acc[k] += (uint32_t)v.palette[c][k] * inten / 255u;
    }
    img[px] = any ? make_uchar4((unsigned char)min(acc[0], 255u), (unsigned char)min(acc[1], 255u),
                                (unsigned char)min(acc[2], 255u), 255)
                  : make_uchar4(0, 0, 0, 0);
  }
}

}  // namespace molsim
