"""Mutation check of the oracle's pins (test helper; also runnable: python tests/oracle_mutants.py).

Each entry is a plausible one-line misreading of the paper applied to a COPY of oracle/orc.c (never to the file itself),
built into a temporary liborc.so, with the pin test that must FAIL on it.  `ORC_LIBORC` (oracle/orc.py) points the
test subprocess at the broken build.  A mutant that survives means the corresponding reading is "parity unpinned".
"""
from __future__ import annotations

import os
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
T = "tests/test_oracle_pins_timelevels.py::"

# (name, text in orc.c, replacement, pin that kills it); lists = several sites changed together
MUTANTS = [
    ("boris: gamma of u instead of u^- (reading G3)",
     "double gm = sqrt(1.0 + um[0] * um[0] + um[1] * um[1] + um[2] * um[2]);",
     "double gm = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);",
     T + "test_boris_is_time_reversible_with_E_and_B"),
    ("move: gamma of the OLD momentum (reading G4)",
     ["            if (orc_pusher_kind & 1) orc_vay(u, E, B, qm, dt); else orc_boris(u, E, B, qm, dt);\n",
      "            double gam = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);\n            double X[3], xn[3];\n"],
     ["            double gam = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);\n            if (orc_pusher_kind & 1) orc_vay(u, E, B, qm, dt); else orc_boris(u, E, B, qm, dt);\n",
      "            double X[3], xn[3];\n"],
     T + "test_hyperbolic_motion_converges_at_second_order"),
    ("deposit: J^3 from the old momentum (reading G8)",
     "double ux = pn->u[0][p], uy = pn->u[1][p], uz = pn->u[2][p];",
     "double ux = po->u[0][p], uy = po->u[1][p], uz = po->u[2][p];",
     T + "test_out_of_plane_current_2d_uses_the_new_momentum"),
    ("deposit: phi midpoint replaced by the old phi",
     "double phm = po->phi[p] + 0.5 * dphi;",
     "double phm = po->phi[p];",
     T + "test_out_of_plane_current_axisymmetric_midpoint_and_shorter_arc"),
    ("deposit: shorter-arc wrap removed",
     "dphi -= 2.0 * PI * floor((dphi + PI) / (2.0 * PI));",
     "",
     T + "test_out_of_plane_current_axisymmetric_midpoint_and_shorter_arc"),
    ("deposit: sqrt(h33) at the old position instead of the midpoint",
     "double xm[3] = { c1[0] + 0.5 * (a[0] + b[0]), c1[1] + 0.5 * (a[1] + b[1]), phm }, h[3];",
     "double xm[3] = { c1[0] + a[0], c1[1] + a[1], phm }, h[3];",
     T + "test_out_of_plane_current_axisymmetric_midpoint_and_shorter_arc"),
    ("crossing: AXIS clamp at theta = pi deleted (reading G11)",
     "if (inew >= g->N[a]) { inew = g->N[a] - 1; dnew = nextafter(1.0, 0.0); }",
     "",
     T + "test_landing_on_theta_equals_pi_is_clamped_into_the_last_cell"),
    ("vay: final rotation without the (u'.t) t term",
     "u[0] = sfac * (up[0] + udt * t[0] + (up[1] * t[2] - up[2] * t[1]));",
     "u[0] = sfac * (up[0] + (up[1] * t[2] - up[2] * t[1]));",
     "tests/test_oracle_pins_vay.py::test_vay_keeps_a_drifting_particle_force_free"),
    ("vay: half step with gamma of u' instead of the old velocity",
     "double g0 = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);\n    double v[3]",
     "double g0 = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]) * 1.05;\n    double v[3]",
     "tests/test_oracle_pins_vay.py::test_vay_keeps_a_drifting_particle_force_free"),
    ("filter: weight 1/4 for the centre tap (Eq. 9 garbled)",
     "double f = pow(0.5, g->D + abs(di) + abs(dj) + abs(dk));",
     "double f = pow(0.5, g->D + 1 + abs(di) + abs(dj) + abs(dk)) * (1 + (di == 0));",
     "tests/test_oracle_pins_filter.py::test_fourier_mode_is_damped_by_cos2_of_half_k_per_pass"),
    ("filter: J^2 even instead of odd about the axis (P:386)",
     "{ q[d] = q[d] < 0 ? -1 - q[d] : 2 * n - 1 - q[d]; sign = -sign; }",
     "{ q[d] = q[d] < 0 ? -1 - q[d] : 2 * n - 1 - q[d]; }",
     "tests/test_oracle_pins_filter.py::test_axis_rules_hand_example"),
    ("ampere: current term with the wrong sign (Eq. A2)",
     "E[c][at] += dt * (curl - jc * Jc) / sqrt_h_at(g, c, q);",
     "E[c][at] += dt * (curl + jc * Jc) / sqrt_h_at(g, c, q);",
     "tests/test_oracle_pins_fields.py::test_gauss_law_is_carried_by_the_deposited_current"),
    ("faraday: sign of Eq. A1",
     "B[c][at] -= dt * curl / sqrt_h_at(g, cB, q);",
     "B[c][at] += dt * curl / sqrt_h_at(g, cB, q);",
     "tests/test_oracle_pins_fields.py::test_vacuum_plane_wave_follows_the_yee_dispersion_relation_exactly"),
    ("field solver: contravariant instead of covariant components under the curl (h_ii dropped, P:1066)",
     "return h[comp6 % 3] * A[pidx(g, q[0], q[1], g->D == 3 ? q[2] : 0)];",
     "return A[pidx(g, q[0], q[1], g->D == 3 ? q[2] : 0)];",
     "tests/test_oracle_pins_fields.py::test_vacuum_plane_wave_follows_the_yee_dispersion_relation_exactly"),
    ("ampere, Eq. 13: full 4 pi instead of 2 pi on the axis current",
     "E[c][at] += dt * (sgn * B3 - 0.5 * jc * Jc) / orc_axis_area(g, i + 0.5);",
     "E[c][at] += dt * (sgn * B3 - jc * Jc) / orc_axis_area(g, i + 0.5);",
     "tests/test_oracle_pins_fields.py::test_axis_rules_eq12_and_eq13_hand_values"),
    ("ampere, Eq. 13: south pole without the mirror sign",
     "if (q[ax] != 0) { qb[ax] = g->N[ax] - 1; sgn = -1.0; }",
     "if (q[ax] != 0) { qb[ax] = g->N[ax] - 1; sgn = 1.0; }",
     "tests/test_oracle_pins_fields.py::test_axis_rules_eq12_and_eq13_hand_values"),
    ("Eq. 13: A with the stray factor 2 pi of its defining line (P:370)",
     "return r * r * dr * (1.0 - cos(0.5 * dth));",
     "return 2.0 * PI * r * r * dr * (1.0 - cos(0.5 * dth));",
     "tests/test_oracle_pins_fields.py::test_curvilinear_curl_converges_to_the_textbook_curl_at_second_order"),
    ("gca: gyroradius of the momentum AFTER the push (P:976 'at a given timestep', reading G26)",
     "if (orc_pusher_kind & 2) orc_gca_project(u, u_before, E, B, qm);",
     "if (orc_pusher_kind & 2) orc_gca_project(u, u, E, B, qm);",
     "tests/test_oracle_pins_gca.py::test_switch_on_the_gyroradius_of_the_momentum_before_the_push"),
    ("gca: projection on B without the 1/|B|^2",
     "double up = (u[0] * B[0] + u[1] * B[1] + u[2] * B[2]) / B2;",
     "double up = (u[0] * B[0] + u[1] * B[1] + u[2] * B[2]);",
     "tests/test_oracle_pins_gca.py::test_guiding_centre_regime_kills_u_perp_and_follows_E_par"),
    # mutants the round-1 pins already killed, kept so that the list documents them
    ("deposit: 3D weights without the D_a D_b / 12 term (reading G7)",
     "+ sigma * Dv[a] * Dv[b] / 12.0",
     "",
     "tests/test_oracle_pins_deposit.py::test_continuity_holds_to_roundoff_for_random_moves"),
    ("boris: s = 2 t / (1 + t^2) without the factor 2",
     "s[a] = 2.0 * t[a] / (1.0 + t2);",
     "s[a] = t[a] / (1.0 + t2);",
     "tests/test_oracle_pins_push.py::test_boris_pure_B_conserves_energy_and_rotates_by_the_scheme_angle"),
]


def build_mutant(old, new, outdir: str) -> str:
    """old/new: a string each, or equally long lists of strings (several sites changed together)"""
    mutated = open(os.path.join(ROOT, "oracle", "orc.c")).read()
    olds, news = ([old], [new]) if isinstance(old, str) else (old, new)
    for o, n in zip(olds, news):
        assert mutated.count(o) == 1, f"mutation site not found exactly once: {o!r}"
        mutated = mutated.replace(o, n)
    cfile = os.path.join(outdir, "orc.c")
    open(cfile, "w").write(mutated)
    open(os.path.join(outdir, "orc.h"), "w").write(open(os.path.join(ROOT, "oracle", "orc.h")).read())
    lib = os.path.join(outdir, "liborc.so")
    subprocess.check_call(["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", lib, cfile, "-lm"])
    return lib


def run_pin(lib: str | None, test: str) -> int:
    env = dict(os.environ)
    if lib:
        env["ORC_LIBORC"] = lib
    else:
        env.pop("ORC_LIBORC", None)
    return subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", test], cwd=ROOT, env=env,
                          capture_output=True, text=True).returncode


def check(index: int) -> tuple[str, bool]:
    name, old, new, test = MUTANTS[index]
    with tempfile.TemporaryDirectory() as d:
        lib = build_mutant(old, new, d)
        return name, run_pin(lib, test) != 0


if __name__ == "__main__":
    bad = 0
    for k in range(len(MUTANTS)):
        name, killed = check(k)
        print(("killed   " if killed else "SURVIVED ") + name)
        bad += not killed
    sys.exit(1 if bad else 0)
