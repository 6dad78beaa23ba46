"""Table validation, rule by rule (include/molsim.h "Table validation" V1-V7; PAPER.md:56 consistency checker).

Each case STATES a rule, breaks exactly that rule in an otherwise valid model, and checks that
  * the product's checker (sim_check_config: host only, no device needed) names that rule, and
  * the oracle's validator (written separately) refuses the same model,
and that both accept the unbroken model.  CPU only.
"""
import copy

import numpy as np
import pytest

import paper_2606_14603_b200 as pkg
from oracle.binding import E_INVAL, Oracle, OracleError
from workloads import configs
from workloads.model import (CH_BIRTH, CH_CONVERT, CH_DELAYED_BIRTH, CH_RELEASE, NONE16, SHAPE_CUBE, SHAPE_SPHERE,
                             Channel, Compartment, Model, Reaction, SeedRecord, Species, prob_to_thr, stack_tables)


def base_cube():
    A, B, Cx = 0, 1, 2
    return Model(name="v", species=[Species("A", 1), Species("B", 1),
                                    Species("C", 2, channels=[Channel(CH_RELEASE, prob_to_thr(1e-3), A, B)])],
                 reactions=[Reaction(A, B, Cx, 2500, prob_to_thr(0.5))], compartments=[Compartment(SHAPE_CUBE, L=2000)],
                 table_bits=12, tables=stack_tables([44.7214, 31.6228], 12), extent=(2000,) * 3, seed=1, place_seed=1,
                 seed_records=[SeedRecord(A, 10)], n_steps=4, cell_size=64).finalize()


def base_nuclear():
    return configs.w3(scale=0.01, n_steps=4)


def base_replicas():
    return configs.w2(scale=0.001, n_steps=4)


def oracle_refuses(m):
    try:
        Oracle(m)
    except OracleError as e:
        return e.code == E_INVAL
    return False


def both_accept(m):
    assert pkg.check_config(m) is None
    Oracle(m)


@pytest.mark.parametrize("make", [base_cube, base_nuclear, base_replicas])
def test_valid_models_pass_both_validators(make):
    both_accept(make())


# (rule tag, statement of the rule, base model, mutation that breaks only this rule, does the oracle have the rule too)
def _ix(m, name):
    return [s.name for s in m.species].index(name)


CASES = [
    ("V2", "cell_size is at least 2 units", base_cube, lambda m: setattr(m, "cell_size", 1), False),
    ("V2", "at most SIM_MAX_SPECIES = 64 species", base_cube,
     lambda m: m.species.extend(Species(f"x{k}", 1) for k in range(70)), False),
    ("V2", "extent is positive on every axis", base_cube, lambda m: setattr(m, "extent", (2000, 0, 2000)), True),
    ("V3", "extent[0] fits inside the replica tiles", base_replicas,
     lambda m: setattr(m, "extent", ((m.n_replicas << m.stride_shift) + 1, m.extent[1], m.extent[2])), True),
    ("V4", "a cube edge is positive", base_cube, lambda m: setattr(m.compartments[0], "L", 0), True),
    ("V4", "no displacement reaches across a cube (one mirror reflection suffices, S5)", base_cube,
     lambda m: (setattr(m.compartments[0], "L", 150), setattr(m, "extent", (150,) * 3)), True),
    ("V4", "a sphere has r_in < r_out", base_nuclear,
     lambda m: setattr(m.compartments[0], "r_in", m.compartments[0].r_out), True),
    ("V4", "a compartment does not reach below 0", base_nuclear,
     lambda m: setattr(m.compartments[0], "cy", m.compartments[0].r_out - 1), True),
    ("V4", "a compartment stays inside extent in y / z", base_nuclear,
     lambda m: setattr(m, "extent", (m.extent[0], m.extent[1], m.extent[2] - 2)), True),
    ("V4", "a compartment stays inside its replica tile in x", base_replicas,
     lambda m: setattr(m.compartments[0], "cx", (1 << m.stride_shift) - m.compartments[0].r_out), True),
    ("V4", "replicas keep at least the largest interaction radius apart (S16: independent populations)", base_replicas,
     lambda m: setattr(m.compartments[0], "cx", (1 << m.stride_shift) - m.compartments[0].r_out - 1 - 49), True),
    ("V5", "sigma_class names a row of the tables", base_cube, lambda m: setattr(m.species[0], "sigma_class", 3), True),
    ("V5", "compartment exists", base_cube, lambda m: setattr(m.species[1], "compartment", 1), True),
    ("V5", "cross_to is a species", base_nuclear,
     lambda m: setattr(m.species[_ix(m, "pERK_n")], "cross_to", len(m.species)), True),
    ("V5", "cross_to lives in ANOTHER compartment", base_nuclear,
     lambda m: setattr(m.species[_ix(m, "pERK_n")], "cross_to", _ix(m, "pRSK_n")), True),
    ("V6", "channel kind is known", base_cube, lambda m: setattr(m.species[2].channels[0], "kind", 9), True),
    ("V6", "a RELEASE names an existing product 0 (undefined species, PAPER.md:56)", base_cube,
     lambda m: setattr(m.species[2].channels[0], "prod0", 7), True),
    ("V6", "a RELEASE names an existing product 1", base_cube,
     lambda m: setattr(m.species[2].channels[0], "prod1", NONE16), True),
    ("V6", "a product lives in its parent's compartment", base_nuclear,
     lambda m: setattr(m.species[_ix(m, "GENE:pERK")].channels[1], "prod1", _ix(m, "pERK")), True),
    ("V6", "a delayed birth waits at least one step (S17)", base_nuclear,
     lambda m: setattr(m.species[_ix(m, "GENE")].channels[0], "thr", 0), True),
    ("V6", "a rule slot is below n_rules", base_nuclear,
     lambda m: setattr(m.species[_ix(m, "GENE")].channels[0], "rule", 1), True),
    ("V7", "a reaction names existing species", base_cube, lambda m: setattr(m.reactions[0], "cplx", 5), True),
    ("V7", "reactants and complex share a compartment", base_nuclear,
     lambda m: setattr(m.reactions[0], "cplx", _ix(m, "pERK_n")), True),
    ("V7", "the interaction radius fits the cell (r2 <= cell_size^2, S8)", base_cube,
     lambda m: setattr(m.reactions[0], "r2", 64 * 64 + 1), True),
    ("V7", "one reaction per unordered species pair (reciprocal reactions are one symmetric entry)", base_cube,
     lambda m: m.reactions.append(Reaction(1, 0, 2, 2500, prob_to_thr(0.1))), True),
]


@pytest.mark.parametrize("tag,rule,make,breakit,in_oracle", CASES, ids=[f"{c[0]}: {c[1]}" for c in CASES])
def test_each_rule_is_enforced_by_both_validators(tag, rule, make, breakit, in_oracle):
    m = make()
    both_accept(m)
    breakit(m)
    why = pkg.check_config(m)
    assert why is not None and why.startswith(tag), (rule, why)
    if in_oracle:
        assert oracle_refuses(m), rule


def test_the_replica_gap_is_exactly_the_largest_radius():
    # hi_x + R <= tile width: with R = 50 the sphere may end 50 units before the next tile, not 49
    m = base_replicas()
    tile, r_out = 1 << m.stride_shift, m.compartments[0].r_out
    m.compartments[0].cx = tile - r_out - 1 - 50
    both_accept(m)
    m.compartments[0].cx += 1
    assert pkg.check_config(m).startswith("V4") and oracle_refuses(m)


def test_workspace_bytes_is_zero_for_an_invalid_model_and_create_needs_no_device_to_say_so():
    import ctypes as C

    from paper_2606_14603_b200.binding import load_library, marshal_config

    m = base_cube()
    m.reactions[0].r2 = 64 * 64 + 1
    cfg, keep = marshal_config(m)
    assert load_library().sim_workspace_bytes(C.byref(cfg)) == 0
    h = C.c_void_p()
    assert load_library().sim_create(C.byref(cfg), None, 0, None, C.byref(h)) == -1      # SIM_E_INVAL, before any CUDA call
