"""Mutation check of the oracle's pins (not a pytest module; run by hand: python tests/mutation_check.py).

Each entry replaces one line of a scratch copy of oracle/ref_dg.cpp (under /tmp) by a plausible mistake and runs
the `-m "not gpu"` pin tests against that copy; every mutation must turn at least one test red.  The list is the
one of VERDICT round 1 ("What's weak" 1-6): the parts that had no pin then, plus the two survivors of a wider
round-2 run of 75 further single-line mutations over tables, traces, flux, gravity, RHS scalings, boundaries, damping,
CFL, RK, limiter, torque, HLL/HLLC (one more of them only showed up as a test that never ends: the time update).  tests/golden/README.md names the
test that catches each."""
import os
import shutil
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MUTATIONS = [
    ("bc2 W trace side", "else trace_x(c, c->U0.data(), 0, j, -1, r, UL);", "else trace_x(c, c->U0.data(), 0, j, +1, r, UL);"),
    ("bc2 E trace side", "else trace_x(c, c->U0.data(), nx - 1, j, +1, r, UR);", "else trace_x(c, c->U0.data(), nx - 1, j, -1, r, UR);"),
    ("bc2 S trace side", "else trace_y(c, c->U0.data(), i, 0, -1, q, UL);", "else trace_y(c, c->U0.data(), i, 0, +1, q, UL);"),
    ("bc2 N trace side", "else trace_y(c, c->U0.data(), i, ny - 1, +1, q, UR);", "else trace_y(c, c->U0.data(), i, ny - 1, -1, q, UR);"),
    ("c_s^2 on x-faces at the cell centre", "const double yr = p.y0 + (j + 0.5) * dy + 0.5 * dy * T.xi[r];", "const double yr = p.y0 + (j + 0.5) * dy;"),
    ("c_s^2 on y-faces at the cell centre", "const double xq = p.x0 + (i + 0.5) * dx + 0.5 * dx * T.xi[q];\n          if (f > 0 && f < ny)",
     "const double xq = p.x0 + (i + 0.5) * dx;\n          if (f > 0 && f < ny)"),
    ("limiter without the volume Gauss points", "for (int r = 0; r < T.m; ++r) { pts[n].px = T.B[q]; pts[n].py = T.B[r]; ++n; }",
     "for (int r = 0; r < 0; ++r) { pts[n].px = T.B[q]; pts[n].py = T.B[r]; ++n; }"),
    ("eps_rho = lim_eps", "const double eps_rho = std::fmin(p.lim_eps, ubar[0]);", "const double eps_rho = p.lim_eps;"),
    ("no limiter inside the Butcher sub-steps", "if (post) post(post_user, yi.data());", ";"),
    ("HLL jump term sign", "SR * FL[v] - SL * FR[v] + SL * SR * (UR[v] - UL[v])", "SR * FL[v] - SL * FR[v] - SL * SR * (UR[v] - UL[v])"),
    ("HLLC star energy (S* + v_K)", "(Ss - vK) * (Ss + pK / (U[0] * (S - vK)))", "(Ss + vK) * (Ss + pK / (U[0] * (S - vK)))"),
    ("HLLC star energy (S* - p_K/...)", "(Ss - vK) * (Ss + pK / (U[0] * (S - vK)))", "(Ss - vK) * (Ss - pK / (U[0] * (S - vK)))"),
    ("damp_mode 1: momentum relaxed instead of velocity", "const double vx = f0 * v0x + ft * (m[1] / m[0]);", "const double vx = (f0 * v0x * r0 + ft * m[1]) / rho;"),
    ("limiter: eps_p = lim_eps", "const double eps_p = std::fmin(p.lim_eps, pbar);", "const double eps_p = p.lim_eps;"),
    ("Gamma_0 with r_p^2", "p.omega_planet * p.omega_planet * rp2 * rp2 * p.q_planet", "p.omega_planet * p.omega_planet * rp2 * p.q_planet"),
    ("time not advanced after the step", "  damp(c, dt);\n  c->t += dt;", "  damp(c, dt);"),
    ("damp_mode 1: energy relaxed instead of temperature", "const double T = f0 * T0 + ft * (pr / m[0]);", "const double T = (f0 * T0 * r0 + ft * pr) / rho;"),
]
TESTS = ["tests/test_oracle_pins_r2.py", "tests/test_oracle_next.py", "tests/test_oracle_rhs.py"]


def main():
    src = open(os.path.join(ROOT, "oracle", "ref_dg.cpp")).read()
    bad = 0
    for name, old, new in MUTATIONS:
        if src.count(old) < 1:
            print(f"{name}: PATTERN NOT FOUND")
            bad += 1
            continue
        with tempfile.TemporaryDirectory() as w:
            shutil.copytree(os.path.join(ROOT, "oracle"), os.path.join(w, "oracle"),
                            ignore=shutil.ignore_patterns("*.so", "__pycache__"))
            shutil.copytree(os.path.join(ROOT, "tests"), os.path.join(w, "tests"), ignore=shutil.ignore_patterns("__pycache__"))
            os.makedirs(os.path.join(w, "paper_1805_01443_b200"))
            shutil.copy(os.path.join(ROOT, "paper_1805_01443_b200", "workloads.py"), os.path.join(w, "paper_1805_01443_b200"))
            open(os.path.join(w, "paper_1805_01443_b200", "__init__.py"), "w").write("from . import workloads\n")
            open(os.path.join(w, "oracle", "ref_dg.cpp"), "w").write(src.replace(old, new, 1))
            r = subprocess.run([sys.executable, "-m", "pytest", *TESTS, "-x", "-q", "-m", "not gpu"], cwd=w,
                               capture_output=True, text=True)
            red = [ln for ln in r.stdout.splitlines() if ln.startswith("FAILED")]
            print(f"{name}: {'caught by ' + red[0].split(' ')[1] if red else 'NOT CAUGHT'}")
            bad += 0 if red else 1
    sys.exit(1 if bad else 0)


if __name__ == "__main__":
    main()
