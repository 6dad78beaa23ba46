/* molsim.h — C ABI of the B200-native molecule-agent step engine.
 *
 * One handle = one population of molecule agents advanced by hand-written sm_100a CUDA kernels.
 * The operation is the per-time-step agent update of the simulator of arxiv/paper_2606_14603
 * (molecules as agents that diffuse, bind by spatial proximity, release
 * products, cross compartments and are expressed; the per-step update is the
 * memory-bound hot path that scales linearly with agent count), with the algorithm fixed by
 * BASELINE.json `north_star` subsystems (1)-(5) and frozen in DESIGN.md §1 ("Step specification").
 *
 * Conventions
 *  - All arithmetic is integer.  Positions are int32 in 0.1 nm units, species uint16
 *    (0xFFFF = none/DEAD), ids uint32 (DESIGN.md §1 "State").
 *  - HOST pointers unless a parameter says DEVICE.  The library copies every table it is given;
 *    the caller keeps ownership of all arguments.  The only device memory the library uses is the
 *    workspace the caller hands to sim_create (e.g. a torch uint8 tensor) which must outlive the
 *    handle and must not be touched by the caller meanwhile.
 *  - All kernels are enqueued on the cudaStream_t given to sim_create.
 *  - Every function returns SIM_OK (0) or a negative SIM_E_* code; nothing throws or aborts; no
 *    global state.  A handle is not thread-safe.  There is no CPU fallback: without a CUDA device
 *    sim_create returns SIM_E_CUDA.
 */
#ifndef MOLSIM_H
#define MOLSIM_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { SIM_OK = 0,
       SIM_E_INVAL = -1,     /* table validation failed / bad argument (cf. the paper's consistency checker) */
       SIM_E_CAPACITY = -2,  /* agent slots, counts rows or an output buffer too small */
       SIM_E_IDSPACE = -3,   /* next_id would pass id_capacity */
       SIM_E_CUDA = -4,      /* CUDA runtime error (sim_last_cuda_error has the text) */
       SIM_E_INTERNAL = -5 };/* checked build only (-DMOLSIM_CHECKS): an index a kernel derived from data left its bound */

/* unimolecular channel kinds — DESIGN.md §1 phase 3 */
enum { SIM_CH_NONE = 0, SIM_CH_BIRTH = 1, SIM_CH_RELEASE = 2, SIM_CH_CONVERT = 3,
       SIM_CH_DEGRADE = 4, SIM_CH_DELAYED_BIRTH = 5 };
/* compartment shapes — DESIGN.md §1 phase 1, reading S1 */
enum { SIM_SHAPE_CUBE = 0, SIM_SHAPE_SPHERE = 1 };

#define SIM_NONE16 0xFFFFu
#define SIM_MAX_CHANNELS 4
#define SIM_MAX_SPECIES 64
#define SIM_MAX_REACTIONS 64
#define SIM_MAX_COMPARTMENTS 8
#define SIM_MAX_RULES 8
#define SIM_MAX_REPLICAS 64

typedef struct {
  uint32_t kind;        /* SIM_CH_* */
  uint32_t thr;         /* fires iff draw < thr (thr = 2^32-1: always); DELAYED_BIRTH: delay in steps >= 1 */
  uint16_t prod0;       /* species the parent becomes (RELEASE, CONVERT) */
  uint16_t prod1;       /* species of the newborn (BIRTH, RELEASE, DELAYED_BIRTH) */
  uint16_t rule;        /* t_first slot (marks_first BIRTH, DELAYED_BIRTH) */
  uint16_t marks_first; /* BIRTH: firing records t_first[rule] = min(., t) */
} sim_channel_t;

typedef struct {
  uint16_t sigma_class; /* row of `tables`; 0 = immobile */
  uint16_t compartment;
  uint16_t cross_to;    /* twin species in the adjacent compartment (reading S7) or SIM_NONE16 */
  uint16_t n_channels;  /* <= SIM_MAX_CHANNELS */
  uint32_t cross_thr;   /* crossing threshold per membrane contact */
  sim_channel_t ch[SIM_MAX_CHANNELS];
} sim_species_t;

/* bimolecular reaction a + b -> cplx: `a` is the anchor that keeps id and position (reading S10) */
typedef struct { uint16_t a, b, cplx, pad; uint32_t r2 /* units^2 */, thr; } sim_reaction_t;

/* CUBE: lattice 0..L-1 per axis.  SPHERE: |p-c|^2 <= r_out^2 and (r_in < 0 or |p-c|^2 > r_in^2). */
typedef struct { uint32_t shape; int32_t cx, cy, cz, L, r_out, r_in; } sim_compartment_t;

typedef struct { uint16_t species; uint16_t replica; uint32_t count; } sim_seed_rec_t;

typedef struct {
  uint32_t n_species, n_reactions, n_compartments, n_sigma_classes;
  uint32_t table_bits;     /* B: each displacement table has 2^B int16 entries (reading S3) */
  uint32_t n_rules;        /* t_first slots */
  uint32_t n_replicas;     /* replica = x >> stride_shift (reading S16); 1 replica: stride_shift = 31 */
  uint32_t stride_shift;
  int32_t  extent[3];      /* world bounding box: every valid position has 0 <= p < extent */
  uint32_t cell_size;      /* spatial-hash cell edge in units, >= max interaction radius; tuning only */
  uint64_t seed;           /* Philox key of the simulation streams (reading S2) */
  uint32_t capacity;       /* agent slots (live + dead + newborn of one step) */
  uint32_t id_capacity;    /* ids ever issued must stay below this.  Ids are never reused (reading S14): every RELEASE,
                              BIRTH and DELAYED_BIRTH takes a fresh one, so a run needs about n0 + expected events; the
                              id-indexed birth bitmap costs 0.5 B of workspace per id.  SIM_E_IDSPACE when exhausted. */
  uint32_t counts_rows;    /* rows of the per-step counts log; row t = state after t steps */
  uint32_t pad;
  const sim_species_t*     species;       /* [n_species] */
  const sim_reaction_t*    reactions;     /* [n_reactions] */
  const sim_compartment_t* compartments;  /* [n_compartments] */
  const int16_t*           tables;        /* [n_sigma_classes << table_bits], row 0 ignored */
} sim_config_t;

typedef struct sim sim_t;   /* opaque; owned by the library, freed by sim_destroy */

/* Table validation (the in-scope part of the paper's consistency checker, plus the bounds the kernels rely
 * on).  sim_workspace_bytes / sim_create fail with 0 / SIM_E_INVAL unless ALL of these hold:
 *  V1  species, compartments, tables (and reactions when n_reactions > 0) are given.
 *  V2  1 <= n_species <= SIM_MAX_SPECIES, n_reactions <= SIM_MAX_REACTIONS, 1 <= n_compartments <= SIM_MAX_COMPARTMENTS,
 *      n_rules <= SIM_MAX_RULES, 1 <= table_bits <= 16, 1 <= n_sigma_classes <= 255, 1 <= n_replicas <= SIM_MAX_REPLICAS,
 *      stride_shift <= 31, 2 <= cell_size <= 16384, 1 <= capacity < 2^31, id_capacity >= 1, counts_rows >= 1, extent > 0.
 *  V3  the replica tiles fit int32 (n_replicas << stride_shift <= 2^31 when n_replicas > 1) and cover extent[0].
 *  V4  every compartment is well formed (cube: L > 0 and every displacement table entry of a mobile class is smaller than
 *      L in magnitude, so that one mirror reflection suffices, S5; sphere: 0 < r_out, r_in < r_out), its bounding box lies
 *      inside [0, extent) in y and z and inside [0, tile) in x (tile = extent[0], or 2^stride_shift with replicas), and with
 *      replicas its upper x bound stays at least the largest interaction radius below the tile width, so that agents of
 *      neighbouring replicas can never bind (S16: replicas are independent populations).
 *  V5  every species names an existing sigma class and compartment, has at most SIM_MAX_CHANNELS channels, and its
 *      cross_to, if any, is a species of ANOTHER compartment, both spherical (S7).
 *  V6  every channel has a known kind; the products it needs exist and live in the parent's compartment (prod0: RELEASE,
 *      CONVERT; prod1: RELEASE, BIRTH, DELAYED_BIRTH: "references to undefined species"); a rule slot it
 *      uses is below n_rules; a DELAYED_BIRTH delay is at least one step (S17).
 *  V7  every reaction names existing species that share a compartment with their complex, its radius fits the cell
 *      (r2 <= cell_size^2: the 27-cell search is exact, S8), and no unordered species pair has two reactions (the
 *      paper's "reciprocal reactions" are ONE symmetric entry here).
 * sim_check_config returns NULL when the configuration is valid, else a static string that names the first rule
 * that fails (host only; needs no device). */
const char* sim_check_config(const sim_config_t* cfg);

/* Bytes of DEVICE workspace sim_create needs for this configuration (0 if cfg is invalid). */
size_t sim_workspace_bytes(const sim_config_t* cfg);

/* One handle = one population in one cell volume (the paper's model: species classes, reactions, localisation,
 * PAPER.md:45-54; the tables are the integer form of that model file, DESIGN.md §1 "State", readings S3, S4).
 * Validates the tables (SIM_E_INVAL, rules V1-V7 above), copies them to the device, carves the workspace.
 * d_workspace: DEVICE memory, >= sim_workspace_bytes(cfg), 256-byte aligned, owned by the caller.
 * cuda_stream: a cudaStream_t (0 = default stream). */
int sim_create(const sim_config_t* cfg, void* d_workspace, size_t workspace_bytes,
               void* cuda_stream, sim_t** out);

/* Adds agents: record order gives contiguous fresh ids; positions uniform in the species'
 * compartment from the PLACE stream keyed by place_seed (DESIGN.md §1 "Seeding", reading S15).
 * May be called again mid-run (run-time treatment change).  Rewrites counts row t.
 * Synchronises the stream. */
int sim_seed_population(sim_t*, const sim_seed_rec_t* recs, uint32_t n_recs, uint64_t place_seed);

/* Advances n_steps time steps (DESIGN.md §1 phases 1-6 per step).  All work is enqueued on the
 * stream without host synchronisation between steps (the 7 launches of a step are replayed as
 * CUDA graphs captured once per handle); the call then waits for the stream once and
 * returns the sticky device error state (capacity / id space), if any.  Handles are independent:
 * several may step concurrently on different streams ("many seeds per GPU"). */
int sim_step(sim_t*, uint32_t n_steps);
/* Same, but returns after enqueueing; errors surface at the next synchronising call. */
int sim_step_async(sim_t*, uint32_t n_steps);

/* Per-step species counts (DESIGN.md §1 phase 6, reading S22: row 0 = after seeding, row t+1 = after step t; the
 * paper's concentration time series, is counts / (N_A V)), kept on the device while the run goes
 * on; rows first_row .. first_row+n_rows-1 (row <= steps done):
 * out[n_rows][n_replicas][n_species], HOST. */
int sim_read_counts(sim_t*, uint32_t first_row, uint32_t n_rows, uint32_t* out);

/* The agent store (north_star (1): int32 x, y, z in 0.1 nm units, uint16 species, uint32 id; DESIGN.md §1 "State")
 * read back; it stands in for the paper's 3-D view of the molecules.  Memory order on the device is
 * unspecified (reading S23), so the live agents are returned sorted by id into HOST arrays of `cap` elements each (any array may be NULL);
 * *n_out = number of live agents (also set when cap is too small: SIM_E_CAPACITY). */
int sim_read_agents(sim_t*, uint32_t cap, int32_t* x, int32_t* y, int32_t* z,
                    uint16_t* species, uint32_t* id, uint32_t* n_out);

/* Replaces the population by explicit agents in any order (checkpoint reload / test hook);
 * sets the step counter and next_id; rewrites counts row `step`.  HOST arrays (pinned memory makes
 * the copies asynchronous).  Every agent is validated on the device: species < n_species, replica tile
 * (x >> stride_shift) < n_replicas, id < next_id and used once, and a position inside the compartment of its
 * species (the invariant every step keeps, and what bounds the cell keys); on SIM_E_INVAL the handle holds an
 * EMPTY population.  The delayed rules' t_first[] are left as they are (see sim_load_t_first). */
int sim_load_agents(sim_t*, uint32_t n, const int32_t* x, const int32_t* y, const int32_t* z,
                    const uint16_t* species, const uint32_t* id, uint32_t step, uint32_t next_id);

/* Order-independent 64-bit checksum of the live state: the sum, modulo 2^64, over live agents of
 * mix(mix(mix(x | y << 32) ^ (z | id << 32)) ^ species) with mix = the splitmix64 finaliser (DESIGN.md §1
 * "Checksum").  Computed on the device; *out is HOST.  It stands in for the element-by-element
 * comparison at the sizes where the CPU oracle cannot be re-run inside a test (tests/golden/trace_*.txt).
 * Synchronises the stream. */
int sim_read_checksum(sim_t*, uint64_t* out);

/* The part of a checkpoint that is not in the agents (state = agents, t, next_id, t_first[]): the
 * first-firing step of every delayed rule (reading S17), 0xFFFFFFFF = not fired yet.  n must equal n_rules; HOST
 * arrays.  sim_load_agents does not touch them: a reload that is to continue a run restores them with
 * sim_load_t_first.  Both synchronise the stream. */
int sim_read_t_first(sim_t*, uint32_t n, uint32_t* out);
int sim_load_t_first(sim_t*, uint32_t n, const uint32_t* in);

/* Current scalars (any pointer may be NULL).  Synchronises the stream. */
int sim_info(sim_t*, uint32_t* n_live, uint32_t* step, uint32_t* next_id, uint32_t* t_first0);

/* Test hook: phase 1 only (move + boundary/compartment rule) on the current state; the step
 * counter does not advance. */
int sim_debug_move_only(sim_t*);

/* Number of kernels the handle has launched so far (bench.py's gpu_launches). */
uint64_t sim_launch_count(const sim_t*);

/* Per-kernel device time: when enabled, every kernel of sim_step is bracketed by CUDA events on
 * the stream (slower; for bench.py's roofline leg, not for throughput numbers).
 * sim_kernel_times returns, for each of the SIM_N_KERNELS kernels, accumulated milliseconds and
 * launch counts since the last enable. */
#define SIM_N_KERNELS 10
int sim_profile_enable(sim_t*, int on);
int sim_kernel_times(sim_t*, float ms[SIM_N_KERNELS], uint32_t launches[SIM_N_KERNELS]);
const char* sim_kernel_name(int k);

/* Waits for the stream, releases the handle's graphs, streams and host state (north_star boundary list).  The
 * workspace stays the caller's. */
void sim_destroy(sim_t*);
const char* sim_strerror(int code);
const char* sim_last_cuda_error(const sim_t*);

/* ---- read-outs next to the step ------------------------------- */

/* Threshold monitor over a window of the per-step counts log, evaluated on the device (PAPER.md:58:
 * "designate specific molecular species for continuous monitoring ... concentration thresholds within
 * specified time windows"; Fig. 2: the cell state switches between Cancerous and Normal as
 * the monitored species crosses the threshold).  Reading S24: value(t) = sum over `species` of
 * counts[t][replica][s]; above(t) = value(t) > threshold (a concentration threshold is converted to a
 * count by the caller, n = c N_A V). */
typedef struct {
  uint32_t replica;
  uint32_t n_species;          /* 1..4 */
  uint16_t species[4];
  uint32_t threshold;
  uint32_t first_row, n_rows;  /* window: counts rows first_row .. first_row+n_rows-1, all <= steps done */
} sim_monitor_t;
typedef struct {
  uint32_t first_above;        /* first row of the window with above(t), 0xFFFFFFFF if none */
  uint32_t n_above;            /* rows of the window with above(t) */
  uint32_t last_state;         /* above(last row): 1 = over the threshold ("Cancerous" in Fig. 2), 0 = "Normal" */
  uint32_t max_value, max_row; /* maximum of value(t) over the window and the first row that attains it */
  uint32_t n_switches;         /* rows t > first_row of the window with above(t) != above(t-1) */
} sim_monitor_result_t;
/* mons[n_mons] and out[n_mons] are HOST arrays (n_mons <= 64).  states may be NULL; else HOST bytes,
 * above(t) of monitor m at states[m * states_stride + (t - first_row)], states_stride >= every n_rows.
 * SIM_E_INVAL: bad replica / species / empty window / window beyond the steps done.  Synchronises. */
int sim_monitor_eval(sim_t*, const sim_monitor_t* mons, uint32_t n_mons, sim_monitor_result_t* out,
                     uint8_t* states, uint32_t states_stride);

/* Headless stand-in for the paper's 3-D viewer (Fig. 1: molecules highlighted by
 * compartment, orange for cytoplasm, yellow for nucleus): orthographic point splat of the live agents of
 * one replica into an RGBA8 image, computed on the device and copied to `rgba` (HOST,
 * height*width*4 bytes, row 0 = smallest v).  Reading S25: the image plane holds the two axes other than
 * `axis` in increasing order (u, v); an agent with u0 <= u < u0+eu, v0 <= v < v0+ev (local coordinates)
 * falls into pixel ((u-u0)*width / eu, (v-v0)*height / ev); per pixel and compartment c the agents are
 * counted (n_c); channel k = min(255, sum_c palette[c][k] * min(n_c*gain, 255) / 255); alpha = 255 where
 * any agent fell, else 0.  Uses scratch of the handle that is free between steps.
 * SIM_E_INVAL: bad view, or width*height*n_compartments > 2*capacity / width*height > capacity. */
typedef struct {
  uint32_t replica, axis;      /* axis 0, 1, 2 = projected away */
  int32_t u0, v0;
  uint32_t eu, ev;             /* window extent in units (> 0) */
  uint32_t width, height;      /* pixels (> 0) */
  uint32_t gain;               /* 1..255 */
  uint8_t palette[SIM_MAX_COMPARTMENTS][4];   /* r, g, b, unused, per compartment index */
} sim_view_t;
int sim_render(sim_t*, const sim_view_t* view, uint8_t* rgba);

/* Test hook: Philox4x32-10 on the device for n (counter,key) pairs; DEVICE pointers
 * ctr[4n], key[2n], out[4n]; enqueued on `cuda_stream`. */
int sim_debug_philox(const uint32_t* d_ctr, const uint32_t* d_key, uint32_t* d_out, uint32_t n,
                     void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
