"""Mutation check of the oracle's pins ("What's weak" 1): each case breaks ONE thing in a scratch copy of
oracle/lsm_oracle.c -- a word index, a counter field, a value map, a neighbour direction, the overlap -- and the named
pin files must then FAIL.  The untouched copy must pass the same files (control).  Keeps later oracle additions honest:
a new function needs a mutant here that its pin catches.  No GPU; every mutant runs its pins in a subprocess with
LSM_ORACLE_SRC pointing at the broken copy (see oracle/lsm_oracle.py)."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "lsm_oracle.c")
REST = "tests/test_oracle_restatement.py"
TILE = "tests/test_oracle_random_tile.py"
WIDE = "tests/test_oracle_wider_models.py"

# (name, text in lsm_oracle.c (first occurrence), replacement, pin files that must notice, -k selection of the pins that
# are run: the cheapest ones that see the fault; a selection that matches nothing fails the case).
MUTANTS = [
    ("overlap_compares_reference_with_itself", "int a = o->s0[i], b = o->s[i];", "int a = o->s0[i], b = o->s0[i];", [REST], "overlap_from_two_snapshots"),
    ("overlap_forgets_sigma_of_NE", "a = 2 * a - 1; b = 2 * b - 1;", "", [REST], "overlap_from_two_snapshots"),
    ("checkerboard_word_index_shifted", "uint32_t w = w4[k & 3];\n        int nn", "uint32_t w = w4[(k + 1) & 3];\n        int nn", [REST], "checkerboard_sweep and 2-4-1-0"),
    ("sweep_high_bits_dropped_from_c3", "ctr[3] = stream | ((uint32_t)(t >> 32) << 4);", "ctr[3] = stream;", [REST], "checkerboard_sweep and 2-4-1-0"),
    ("sweep_high_bits_overlap_the_tag", "ctr[3] = stream | ((uint32_t)(t >> 32) << 4);",
     "ctr[3] = stream | ((uint32_t)(t >> 32) << 2);", [REST], "checkerboard_sweep and 2-4-1-0"),
    ("stream_tag_ignored", "ctr[3] = stream | ((uint32_t)(t >> 32) << 4);", "ctr[3] = ((uint32_t)(t >> 32) << 4);", [REST], "checkerboard_sweep and 2-4-1-0"),
    ("init_spin1_modulo_instead_of_mulhi", "(int)(((uint64_t)w * 3u) >> 32) - 1", "(int)(w % 3u) - 1", [REST], "init_matches"),
    ("init_word_index_shifted", "uint32_t w = w4[i & 3];", "uint32_t w = w4[(i + 1) & 3];", [REST], "init_matches"),
    ("init_spin_half_uses_low_bit", "else if (o->two_S == 1)    v = (w >> 31) ? 1 : -1;", "else if (o->two_S == 1)    v = (w & 1u) ? 1 : -1;", [REST], "init_matches"),
    ("spin1_words_swapped", "uint32_t w0 = w4[2 * (k & 1)], w1 = w4[2 * (k & 1) + 1];\n        int nn = neighbour_sum(o, x, y, z);",
     "uint32_t w1 = w4[2 * (k & 1)], w0 = w4[2 * (k & 1) + 1];\n        int nn = neighbour_sum(o, x, y, z);", [REST], "checkerboard_sweep and 2-4-2-0"),
    ("spin1_group_of_four_sites", "/* two words per site: group k>>1, words 2(k&1) and 2(k&1)+1 */\n        words_of_group(o->seed, (uint64_t)k >> 1, o->t, half, w4);",
     "/* two words per site: group k>>1, words 2(k&1) and 2(k&1)+1 */\n        words_of_group(o->seed, (uint64_t)k >> 2, o->t, half, w4);", [REST], "checkerboard_sweep and 2-4-2-0"),
    ("spin1_proposal_other_direction", "return (a + 1 + kk) % 3;", "return (a + 2 - kk) % 3;", [REST], "checkerboard_sweep and 2-4-2-0"),
    ("ne_west_instead_of_east", "east = value_at(o, x + 1, y, 0);", "east = value_at(o, x - 1, y, 0);", [REST], "checkerboard_sweep and 2-6-1-1"),
    ("ne_south_instead_of_north", "int north = value_at(o, x, y + 1, 0),", "int north = value_at(o, x, y - 1, 0),", [REST], "checkerboard_sweep and 2-6-1-1"),
    ("ne_metropolis_wrong_threshold", "uint64_t thr = (s_old == 0) ? o->thr[1] : o->thr[2];\n                if ((uint64_t)w < thr)",
     "uint64_t thr = (s_old == 0) ? o->thr[0] : o->thr[2];\n                if ((uint64_t)w < thr)", [REST], "checkerboard_sweep and 2-6-1-2"),
    ("heat_bath_inverted", "s_new = ((uint64_t)w < o->thr[0]) ? 1 : 0;       /* reading D7 */",
     "s_new = ((uint64_t)w < o->thr[0]) ? 0 : 1;       /* reading D7 */", [REST], "checkerboard_sweep and 2-6-1-1"),
    ("ising_table_row_of_the_other_spin", "uint64_t thr = o->thr[b * (2 * o->dims + 1) + j];",
     "uint64_t thr = o->thr[(1 - b) * (2 * o->dims + 1) + j];", [REST], "checkerboard_sweep and 2-6-1-0"),
    ("second_colour_first", "for (uint32_t half = 0; half < 2; ++half) {\n            if (!descending) {",
     "for (uint32_t hh = 0; hh < 2; ++hh) {\n            uint32_t half = 1u - hh;\n            if (!descending) {", [REST], "checkerboard_sweep and 2-4-1-0"),
    ("changed_on_every_facilitated_redraw", "if (s_new != s_old) o->changed[i] = 1;                   /* reading D12 */",
     "if (s_new != s_old || (o->model != ORC_ISING && value_at(o, x, y + 1, 0) == 1 && value_at(o, x + 1, y, 0) == 1)) o->changed[i] = 1;",
     [REST], "checkerboard_sweep and 2-8-1-1"),
    ("tile_schedule_high_bits_overlap_the_tag", "ctr[3] = (4u + launch) | ((uint32_t)(o->t >> 32) << 4);",
     "ctr[3] = (4u + launch) | ((uint32_t)(o->t >> 32) << 2);", [REST], "counter_fields"),
    ("balanced_schedule_shares_the_tile_tag", "ctr[3] = (8u + launch) | ((uint32_t)(o->t >> 32) << 4);",
     "ctr[3] = (4u + launch) | ((uint32_t)(o->t >> 32) << 4);", [TILE], "balanced_matches"),
    ("tile_lowest_thread_wins", "for (int j2 = j + 1; j2 < lambda; ++j2) dup |= (site[j2] == site[j]);\n                        if (dup) continue;                     /* a higher",
     "for (int j2 = 0; j2 < j; ++j2) dup |= (site[j2] == site[j]);\n                        if (dup) continue;                     /* a higher", [TILE], "matches_the_dict"),
    # ---- NEXT-4 models (tests/test_oracle_wider_models.py)
    ("ea_backward_bond_read_from_the_wrong_site", "bond_sign(o, 0, x - 1, y, z) * value_at(o, x - 1, y, z)",
     "bond_sign(o, 0, x, y, z) * value_at(o, x - 1, y, z)", [WIDE], "ea_"),
    ("ea_bonds_drawn_from_the_init_stream", "words_of_group(o->seed, (uint64_t)b >> 2, 0, 3u, w4);",
     "words_of_group(o->seed, (uint64_t)b >> 2, 0, 2u, w4);", [WIDE], "bonds_from_seed"),
    ("ea_bond_sign_inverted", "o->tau[b] = (w4[b & 3] >> 31) ? 1 : -1;", "o->tau[b] = (w4[b & 3] >> 31) ? -1 : 1;", [WIDE], "bonds_from_seed"),
    ("ea_bond_energy_ignores_the_signs", "int f = bond_sign(o, 0, x, y, z) * value_at(o, x + 1, y, z) + bond_sign(o, 1, x, y, z) * value_at(o, x, y + 1, z);",
     "int f = value_at(o, x + 1, y, z) + value_at(o, x, y + 1, z);", [WIDE], "ea_"),
    ("ea_init_uses_low_bit", "else if (o->model == ORC_EA) v = (w >> 31) ? 1 : -1;", "else if (o->model == ORC_EA) v = (w & 1u) ? 1 : -1;", [WIDE], "ea_"),
    ("potts_words_swapped", "uint32_t w0 = w4[2 * (k & 1)], w1 = w4[2 * (k & 1) + 1];\n        int r =",
     "uint32_t w1 = w4[2 * (k & 1)], w0 = w4[2 * (k & 1) + 1];\n        int r =", [WIDE], "potts_matches"),
    ("potts_group_of_four_sites", "words_of_group(o->seed, (uint64_t)k >> 1, o->t, half, w4);\n        uint32_t w0 = w4[2 * (k & 1)], w1 = w4[2 * (k & 1) + 1];\n        int r =",
     "words_of_group(o->seed, (uint64_t)k >> 2, o->t, half, w4);\n        uint32_t w0 = w4[2 * (k & 1)], w1 = w4[2 * (k & 1) + 1];\n        int r =", [WIDE], "potts_matches"),
    ("potts_proposal_may_repeat_the_state", "int prop = (s_old + 1 + r) % o->q;", "int prop = (s_old + r) % o->q;", [WIDE], "potts_matches"),
    ("potts_energy_difference_sign", "int dn = neighbours_equal_to(o, x, y, z, prop) - neighbours_equal_to(o, x, y, z, s_old);",
     "int dn = neighbours_equal_to(o, x, y, z, s_old) - neighbours_equal_to(o, x, y, z, prop);", [WIDE], "potts_matches"),
    ("potts_init_modulo", "v = (int)(((uint64_t)w * (uint64_t)o->q) >> 32);", "v = (int)(w % (uint32_t)o->q);", [WIDE], "potts_matches"),
    ("potts_overlap_as_product", "if (o->model == ORC_POTTS) { ov += (a == b); continue; }", "if (o->model == ORC_POTTS) { ov += a * b; continue; }", [WIDE], "potts_matches"),
    ("potts_table_shifted", "if ((uint64_t)w1 < o->thr[dn + 2 * o->dims]) s_new = prop;", "if ((uint64_t)w1 < o->thr[dn + 2 * o->dims + 1]) s_new = prop;", [WIDE], "potts_"),
]


def run_pins(src, files, select=None):
    env = dict(os.environ, LSM_ORACLE_SRC=src, PYTHONDONTWRITEBYTECODE="1")
    files = [f for f in files if os.path.exists(os.path.join(ROOT, f))]
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", *(["-k", select] if select else []), *files], cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=600)
    return r.returncode, r.stdout[-1500:]


def test_control_the_untouched_copy_passes(tmp_path):
    dst = tmp_path / "lsm_oracle.c"
    dst.write_text(open(SRC).read())
    rc, out = run_pins(str(dst), [REST])
    assert rc == 0, out


@pytest.mark.parametrize("name,old,new,files,select", MUTANTS, ids=[m[0] for m in MUTANTS])
def test_mutant_is_caught(tmp_path, name, old, new, files, select):
    text = open(SRC).read()
    assert text.count(old) >= 1, f"mutant {name}: its anchor text is no longer in lsm_oracle.c -- update the list"
    dst = tmp_path / "lsm_oracle.c"
    dst.write_text(text.replace(old, new, 1))
    rc, out = run_pins(str(dst), files, select)
    assert rc == 1, f"mutant {name} survived (pytest rc {rc}):\n{out}"
