"""Mutation check of the oracle's whole-path driver (`oracle_forward_ext`) and of `oracle_convolve`.

Round 1's review found that seven one-token wiring mistakes in the driver passed every CPU pin,
because all whole-path pins used grey / single-species / pressure-independent tables.  Each mutant
below is applied to a scratch copy of oracle/helios_oracle.c; the pins named beside it must FAIL on
the mutant (and pass on the original, which the normal run of those tests shows).  `-m "not gpu"`.
"""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

BRUTE = "test_whole_path_brute_force_tiny_nongrey"
MUTANTS = {
    # name: (original text, mutated text, pin that must fail)
    "M1_h2_he_swapped": ("oracle_chi_level(S, x, sig, C, x_h2, x_he, alp,",
                         "oracle_chi_level(S, x, sig, C, x_he, x_h2, alp,", BRUTE),
    "M2_cia_pair_offset_dropped": ("oracle_interp_cia(cia + (size_t)c * nT * nNu, nT, T_grid, nNu, T[l], alp[c]);",
                                   "oracle_interp_cia(cia, nT, T_grid, nNu, T[l], alp[c]);", BRUTE),
    "M4_cia_at_bottom_temperature": ("oracle_interp_cia(cia + (size_t)c * nT * nNu, nT, T_grid, nNu, T[l], alp[c]);",
                                     "oracle_interp_cia(cia + (size_t)c * nT * nNu, nT, T_grid, nNu, T[0], alp[c]);", BRUTE),
    "M5_sigma_at_bottom_pressure": ("nNu, T[l], log10(p_bar[l]), sig[s], &cl);",
                                    "nNu, T[l], log10(p_bar[0]), sig[s], &cl);", BRUTE),
    "M6_species_offset_dropped": ("oracle_interp_sigma(sigma + (size_t)s * nT * nP * nNu, nT,",
                                  "oracle_interp_sigma(sigma, nT,", BRUTE),
    "M7_inst_sigma_one_point_off": ("double sg = inst_sigma ? inst_sigma[k] : 0.0;\n        if (sg <= 0.0) { Fd[k]",
                                    "double sg = inst_sigma ? inst_sigma[k > 0 ? k - 1 : 0] : 0.0;\n        if (sg <= 0.0) { Fd[k]",
                                    "test_convolve_closed_forms"),
    "M17_dtau_column_of_neighbour_nu": ("dcol[l] = dtau[(size_t)l * nNu + k];",
                                        "dcol[l] = dtau[(size_t)l * nNu + (k > 0 ? k - 1 : 0)];", BRUTE),
    "M18_density_at_bottom_temperature": ("oracle_number_density(p_bar[l], T[l]), nNu, chi",
                                          "oracle_number_density(p_bar[l], T[0]), nNu, chi", BRUTE),
    "M21_trapezoid_uses_one_level": ("chi + (size_t)(l + 1) * nNu, dz,", "chi + (size_t)(l) * nNu, dz,", BRUTE),
    # stage functions: one plausible slip each, killed by the closed form that pins the stage
    "S1_thickness_from_lower_temperature": ("return K_BOLTZMANN * 0.5 * (T_lo + T_hi) /", "return K_BOLTZMANN * 0.5 * (T_lo + T_lo) /",
                                            "test_total_optical_depth_converges_to_hydrostatic_column"),
    "S2_flux_without_mu": ("flux += w[k] * mu[k] * I;", "flux += w[k] * I;", "test_rt_isothermal_gives_pi_B"),
    "S3_gamma_sign_as_printed": ("*gamma = -e - em1 / D;", "*gamma = e - em1 / D;", "test_sc_coefficients_against_eq1_quadrature"),
    "S4_source_shifted_a_level": ("double dI = beta * S[i] + gamma * S[i - 1];", "double dI = beta * S[i - 1] + gamma * S[i];",
                                  "test_rt_linear_source_thick_bottom"),
    "S5_profile_cut_at_4_sigma": ("if (fabs(d) > 5.0 * sg) continue;", "if (fabs(d) > 4.0 * sg) continue;", "test_convolve_closed_forms"),
    "S6_gravity_as_natural_exponential": ("double g_cgs = pow(10.0, th[0]);", "double g_cgs = exp(th[0]);", BRUTE),
    "S7_distance_to_the_first_power": ("if (i_d >= 0) scale /= th[i_d] * th[i_d];", "if (i_d >= 0) scale /= th[i_d];", "NEXT:test_whole_path_distance_and_inflation"),
    # round 2's survivors ("What's weak" 1): the one-node branch of the profile and the wiring of the
    # finite-element parametrisation in the driver
    "R1_single_node_value_halved": ("if (K == 1) { T[l] = T_knot[0]; continue; }", "if (K == 1) { T[l] = 0.5 * T_knot[0]; continue; }",
                                    "test_single_node_profile_is_isothermal"),
    "R2_ratio_form_ignored": ("if (tp_ratio) oracle_tp_dofs_from_ratios(NT, T_par, dof);", "if (0) oracle_tp_dofs_from_ratios(NT, T_par, dof);",
                              "test_whole_path_brute_force_finite_elements"),
    "R3_element_order_forced_to_one": ("oracle_temperature_profile_fe(L, p_bar, tp_elements, tp_order, dof, p_bot_bar, p_top_bar, T);",
                                       "oracle_temperature_profile_fe(L, p_bar, tp_elements, 1, dof, p_bot_bar, p_top_bar, T);",
                                       "test_whole_path_brute_force_finite_elements"),
    "R4_vmr_offset_from_n_knots": ("const double *log10_vmr = th + 2 + NT;", "const double *log10_vmr = th + 2 + K;",
                                   "test_whole_path_brute_force_finite_elements"),
}


@pytest.mark.parametrize("name", sorted(MUTANTS))
def test_mutant_is_killed(name, tmp_path):
    old, new, pin = MUTANTS[name]
    src = open(os.path.join(ROOT, "oracle", "helios_oracle.c")).read()
    assert src.count(old) == 1, f"{name}: the driver changed; update the mutant"
    for sub in ("oracle", "workloads", "tests"):
        shutil.copytree(os.path.join(ROOT, sub), tmp_path / sub,
                        ignore=shutil.ignore_patterns("*.so", "__pycache__", "test_oracle_mutants.py"))
    (tmp_path / "oracle" / "helios_oracle.c").write_text(src.replace(old, new))
    target = "tests/test_oracle_pins.py"
    if pin.startswith("NEXT:"):
        target, pin = "tests/test_oracle_next.py", pin[5:]
    r = subprocess.run([sys.executable, "-m", "pytest", target, "-q", "-x", "-k", pin,
                        "-p", "no:cacheprovider"], cwd=tmp_path, capture_output=True, text=True, timeout=600)
    assert r.returncode == 1 and "failed" in r.stdout, f"mutant {name} survived {pin}:\n{r.stdout[-1500:]}"
