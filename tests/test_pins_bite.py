"""Proof that the pins of the oracle's decision logic bite: each case below
breaks oracle/inc_oracle.c in one plausible way (a swapped table, the wrong species' E_F, a dropped E_C, ...),
builds the broken copy beside the real one (INC_ORACLE_SRC / INC_ORACLE_LIB, read by oracle/oracle.py) and runs
the pin that is meant to notice it in a subprocess: the pin must FAIL.  The unbroken oracle passing the same
pins is the ordinary test run.  DESIGN.md section 9 lists the same table.
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "inc_oracle.c")
DEC = "tests/test_oracle_decisions.py::"

# (name, text in inc_oracle.c, replacement, pin that must turn red)
MUTATIONS = [
    ("sigma_tables_swapped_for_proton_tracks",
     "tr.type == 1 ? t->sig_pp : t->sig_np", "tr.type == 1 ? t->sig_np : t->sig_pp",
     DEC + "test_zeroed_sigma_table_fixes_the_partner_species"),
    ("sigma_tables_swapped_for_neutron_tracks",
     "tr.type == 0 ? t->sig_pp : t->sig_np", "tr.type == 0 ? t->sig_np : t->sig_pp",
     DEC + "test_zeroed_sigma_table_fixes_the_partner_species"),
    ("densities_transposed_in_Sigma",
     "double Sp = nu->rho_p[i] * sig_p, Sn = nu->rho_n[i] * sig_n;", "double Sp = nu->rho_n[i] * sig_p, Sn = nu->rho_p[i] * sig_n;",
     DEC + "test_flat_sigma_one_shell_closed_forms"),
    ("partner_draw_against_the_neutron_share",
     "int t2 = (u[0] * Sigma < Sp) ? 1 : 0;", "int t2 = (u[0] * Sigma < Sn) ? 1 : 0;",
     DEC + "test_flat_sigma_one_shell_closed_forms"),
    ("mb_to_fm2_factor_dropped",
     "t->plab_max, plab_p) * 0.1;", "t->plab_max, plab_p) * 1.0;",
     DEC + "test_flat_sigma_one_shell_closed_forms"),
    ("impact_parameter_linear_in_u",
     "double b = nu->R * sqrt(u[0]);", "double b = nu->R * u[0];",
     DEC + "test_entry_points_are_uniform_on_the_disc"),
    ("pauli_projectile_tested_against_other_species_EF",
     "double EF1 = tr.type ? nu->EF_p[i] : nu->EF_n[i];", "double EF1 = tr.type ? nu->EF_n[i] : nu->EF_p[i];",
     DEC + "test_blocked_fraction_of_projectile_collisions_vs_quadrature"),
    ("pauli_recoil_tested_against_other_species_EF",
     "double EF2 = t2 ? nu->EF_p[i] : nu->EF_n[i];", "double EF2 = t2 ? nu->EF_n[i] : nu->EF_p[i];",
     DEC + "test_blocked_fraction_of_projectile_collisions_vs_quadrature"),
    ("pauli_either_product_suffices",
     "if (!(T1 > EF1 && T2 > EF2)) {", "if (!(T1 > EF1 || T2 > EF2)) {",
     DEC + "test_blocked_fraction_of_projectile_collisions_vs_quadrature"),
    ("coulomb_barrier_dropped_from_the_proton_cutoff",
     "double cut = ch[c].type ? nu->EC : 0.0;", "double cut = ch[c].type ? 0.0 : 0.0;",
     DEC + "test_cutoff_thresholds_show_in_the_escape_spectra"),
    ("coulomb_barrier_applied_to_neutrons_too",
     "double cut = ch[c].type ? nu->EC : 0.0;", "double cut = ch[c].type ? nu->EC : nu->EC;",
     DEC + "test_cutoff_thresholds_show_in_the_escape_spectra"),
    ("cutoff_uses_the_other_species_well",
     "double Vc = ch[c].type ? nu->V_p[i] : nu->V_n[i];", "double Vc = ch[c].type ? nu->V_n[i] : nu->V_p[i];",
     DEC + "test_cutoff_thresholds_show_in_the_escape_spectra"),
    ("child_path_codes_swapped",
     "ch[c].pi = 2u * tr.pi + (uint32_t)c;", "ch[c].pi = 2u * tr.pi + (uint32_t)(1 - c);",
     DEC + "test_track_tree_is_consistent"),
    ("child_species_swapped",
     "ch[c].type = c == 0 ? tr.type : t2;", "ch[c].type = c == 0 ? t2 : tr.type;",
     DEC + "test_track_tree_is_consistent"),
    ("slope_tables_swapped",
     "same ? t->B_pp : t->B_np", "same ? t->B_np : t->B_pp",
     DEC + "test_angular_tables_wiring"),
    ("backward_probability_a_instead_of_a_over_1_plus_a",
     "u_back * (1.0 + a_back) < a_back", "u_back < a_back",
     DEC + "test_angular_tables_wiring"),
    ("transparent_attempts_accepted",
     "if (transparent && !(flags & ORC_F_KEEP_TRANSPARENT)) {", "if (0) {",
     DEC + "test_retry_rules_recounted_from_traces"),
    ("invalid_residuals_accepted",
     "if (!orc_valid_nucleus(A_res, Z_res)) { if (stats) stats->retry_invalid++; continue; }", "",
     DEC + "test_retry_rules_recounted_from_traces"),
    ("negative_excitation_tolerated",
     "if (Estar < 0.0 && !(transparent", "if (Estar < -5.0 && !(transparent",
     DEC + "test_retry_rules_recounted_from_traces"),
    ("channel_choice_off_by_one",
     "if (W[q] > 0.0) { cum += W[q]; j = q; if (thr < cum) break; }", "if (W[q] > 0.0) { j = q; if (thr < cum) break; cum += W[q]; }",
     DEC + "test_channel_choice_follows_the_widths"),
    ("dostrovsky_row_search_stuck_on_the_first_interval",
     "while (k < n - 2 && z > zz[k + 1]) ++k;", "",
     DEC + "test_dostrovsky_interpolation_interior"),
    ("gem_pre_exponential_power",
     "- 0.25 * log(ld->a) - 1.25 * log(u);", "- 0.25 * log(ld->a) - 1.5 * log(u);",
     "tests/test_oracle_gem.py::test_level_density_constants_and_matching"),
    ("gem_matching_energy",
     "ld->Ux = 150.0 / (double)A_d + 2.5;", "ld->Ux = 150.0 / (double)A_d + 2.0;",
     "tests/test_oracle_gem.py::test_gem_widths_vs_numerical_integration"),
    ("gem_pairing_not_subtracted_in_the_fermi_gas_branch",
     "double u = U - ld->delta;\n    return 2.0", "double u = U;\n    return 2.0",
     "tests/test_oracle_gem.py::test_gem_widths_vs_numerical_integration"),
    ("gem_envelope_uses_the_constant_temperature_slope_only",
     "if (sfg < m) m = sfg;", "",
     "tests/test_oracle_gem.py::test_gem_sampler_matches_pdf"),
    ("dostrovsky_fraction_over_the_whole_grid",
     "double f = (z - zz[k]) / (zz[k + 1] - zz[k]);", "double f = (z - zz[k]) / (zz[n - 1] - zz[0]);",
     DEC + "test_dostrovsky_interpolation_interior"),
]


@pytest.mark.parametrize("name,old,new,pin", MUTATIONS, ids=[m[0] for m in MUTATIONS])
def test_pin_notices(tmp_path, name, old, new, pin):
    with open(SRC) as f:
        text = f.read()
    assert text.count(old) == 1, f"mutation site of {name} not found exactly once in inc_oracle.c"
    broken = tmp_path / "inc_oracle_broken.c"
    broken.write_text(text.replace(old, new))
    env = dict(os.environ, INC_ORACLE_SRC=str(broken), INC_ORACLE_LIB=str(tmp_path / "libinc_oracle_broken.so"))
    p = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", pin], cwd=ROOT, env=env,
                       stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=600)
    assert os.path.exists(env["INC_ORACLE_LIB"]), f"the broken oracle of '{name}' did not build:\n{p.stdout[-2000:]}"
    last = p.stdout.strip().splitlines()[-1]
    assert p.returncode == 1 and " failed" in last and " error" not in last, \
        f"{pin} did not notice '{name}' (exit {p.returncode}):\n{p.stdout[-2000:]}"
