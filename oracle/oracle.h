/* oracle.h — C ABI of the CPU ORACLE.  TEST INFRASTRUCTURE, not product code.
 *
 * Plain, slow, single-threaded C++17 implementation of the molecule-agent time step
 * exactly as frozen in DESIGN.md "Step specification" (from BASELINE.json north_star
 * subsystems (1)-(5) and SURVEY.md Appendix A; behaviours: PAPER.md:7, 35, 45-52,
 * 153-157).  It shares no code, header, table or helper with the CUDA path under
 * paper_2606_14603_b200/; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * Parity unpinned (definitional readings, nothing external can confirm them; see
 * DESIGN.md): S6 (sphere wall = move rejection), S10 (anchor survives), S11 (release
 * placement), S12 (phase order), S13 (channel priority), S17 (delayed repressor).
 */
#ifndef ORACLE_H
#define ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_OK = 0, ORC_E_INVAL = -1, ORC_E_CAPACITY = -2, ORC_E_IDSPACE = -3 };
enum { ORC_CH_NONE = 0, ORC_CH_BIRTH = 1, ORC_CH_RELEASE = 2, ORC_CH_CONVERT = 3,
       ORC_CH_DEGRADE = 4, ORC_CH_DELAYED_BIRTH = 5 };
enum { ORC_SHAPE_CUBE = 0, ORC_SHAPE_SPHERE = 1 };
enum { ORC_MODE_GRID = 0, ORC_MODE_BRUTE = 1 };
#define ORC_NONE16 0xFFFFu
#define ORC_MAX_CHANNELS 4

typedef struct {
  uint32_t kind;        /* ORC_CH_* */
  uint32_t thr;         /* uint32 threshold; DELAYED_BIRTH: delay in steps (>= 1) */
  uint16_t prod0;       /* species the parent becomes (RELEASE, CONVERT) */
  uint16_t prod1;       /* species of the newborn (BIRTH, RELEASE, DELAYED_BIRTH) */
  uint16_t rule;        /* t_first slot */
  uint16_t marks_first; /* BIRTH only: firing records t_first[rule] = min(., t) */
} orc_channel_t;

typedef struct {
  uint16_t sigma_class; /* 0 = immobile */
  uint16_t compartment;
  uint16_t cross_to;    /* twin species across the membrane, ORC_NONE16 = none */
  uint16_t n_channels;
  uint32_t cross_thr;
  orc_channel_t ch[ORC_MAX_CHANNELS];
} orc_species_t;

typedef struct { uint16_t a, b, cplx, pad; uint32_t r2, thr; } orc_reaction_t;
typedef struct { uint32_t shape; int32_t cx, cy, cz, L, r_out, r_in; } orc_compartment_t;
typedef struct { uint16_t species; uint16_t replica; uint32_t count; } orc_seed_rec_t;

typedef struct {
  uint32_t n_species, n_reactions, n_compartments, n_sigma_classes;
  uint32_t table_bits, n_rules, n_replicas, stride_shift;
  int32_t  extent[3];
  uint32_t cell_size;
  uint64_t seed;
  uint32_t capacity, id_capacity, counts_rows, pad;
  const orc_species_t*     species;
  const orc_reaction_t*    reactions;
  const orc_compartment_t* compartments;
  const int16_t*           tables;      /* [n_sigma_classes << table_bits] */
} orc_config_t;

typedef struct oracle oracle_t;

int  oracle_create(const orc_config_t* cfg, oracle_t** out);
void oracle_destroy(oracle_t*);
int  oracle_set_mode(oracle_t*, int mode);      /* phase-2 back end: grid (default) or O(N^2) */
int  oracle_seed_population(oracle_t*, const orc_seed_rec_t* recs, uint32_t n_recs, uint64_t place_seed);
int  oracle_step(oracle_t*, uint32_t n_steps);
int  oracle_read_counts(oracle_t*, uint32_t first_row, uint32_t n_rows, uint32_t* out);
int  oracle_read_agents(oracle_t*, uint32_t cap, int32_t* x, int32_t* y, int32_t* z,
                        uint16_t* species, uint32_t* id, uint32_t* n_out);   /* id-sorted */
int  oracle_load_agents(oracle_t*, uint32_t n, const int32_t* x, const int32_t* y, const int32_t* z,
                        const uint16_t* species, const uint32_t* id, uint32_t step, uint32_t next_id);
int  oracle_info(oracle_t*, uint32_t* n_live, uint32_t* step, uint32_t* next_id, uint32_t* t_first0);
/* order-independent 64-bit checksum of the live (id, species, x, y, z): DESIGN.md §1 "Checksum" */
int  oracle_read_checksum(oracle_t*, uint64_t* out);
/* first-firing steps of the delayed rules (S17), the part of a checkpoint that is not in the agents; n = n_rules */
int  oracle_read_t_first(oracle_t*, uint32_t n, uint32_t* out);
int  oracle_load_t_first(oracle_t*, uint32_t n, const uint32_t* in);

/* test hooks */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* phase-1 only on the current state (advances nothing else) */
int  oracle_debug_move_only(oracle_t*);
/* proposals of phase 2 on the current state, per id-sorted agent: partner id or 0xFFFFFFFF */
int  oracle_debug_proposals(oracle_t*, int mode, uint32_t* prop_id_out);
/* all unordered in-range eligible pairs (ignoring the pair draw), as (id_lo,id_hi) rows, id-sorted */
int  oracle_debug_pairs(oracle_t*, int mode, uint32_t cap_pairs, uint32_t* pairs_out, uint32_t* n_pairs);
#ifdef __cplusplus
}
#endif
#endif
