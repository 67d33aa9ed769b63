"""The oracle's own pins once more, against a copy of the oracle built with AddressSanitizer and
UndefinedBehaviorSanitizer ("ASan/UBSan on the oracle").  compute-sanitizer is closed on
this pool, so for the CUDA path memory safety rests on the bit-exact comparisons; for the checker itself this
run is the evidence that no pin passes by reading out of bounds."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SUITE = ["tests/test_oracle_tree.py", "tests/test_oracle_hardtree.py", "tests/test_oracle_let.py",
         "tests/test_oracle_step.py", "tests/test_oracle_formulas.py",
         "tests/test_oracle_mac.py::test_walk_lists_are_the_sets_the_rule_defines",
         "tests/test_oracle_mac.py::test_let_counts_are_what_eq14_eq15_define",
         "tests/test_oracle_cut.py",
         "tests/test_oracle_forces.py::test_two_body_closed_form",
         "tests/test_oracle_forces.py::test_theta0_hard_plus_soft_is_direct",
         "tests/test_oracle_forces.py::test_hard_sum_is_exact_at_any_theta_and_conserves_momentum"]


def test_oracle_pins_under_asan_ubsan():
    from oracle.build import build, sanitizer_env
    build(sanitize=True)
    env = dict(os.environ, **sanitizer_env())
    env["OMP_NUM_THREADS"] = "4"
    suite = [s for s in SUITE if os.path.exists(os.path.join(ROOT, s.split("::")[0]))]
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider"] + suite, cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "ERROR: AddressSanitizer" not in tail and "runtime error" not in tail
