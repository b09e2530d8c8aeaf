"""Mutation run of the oracle's pins (CPU only; calls nothing but oracle/ and the not-gpu oracle tests).

Each mutation below is one plausible single-line mistake in oracle/sw_oracle.cpp (a dropped term, a wrong
sign / index / word, a transposed operand).  For each, a mutated copy is compiled into a temporary
directory, the oracle binding is pointed at it (environment variable SWO_LIB) and the oracle's pin tests
(tests/test_oracle_*.py, -m "not gpu", -x) are run: the suite must FAIL.  A mutation that survives means a
function of the oracle is not pinned.

    python tests/oracle_mutations.py            # prints one line per mutation; exit status 1 if any survives

`tests/test_oracle_mutations.py` runs the same thing under pytest when SW_RUN_MUTATIONS=1 (it takes a few
minutes, so it is not part of the default CPU suite); the last recorded run is tests/golden/oracle_mutations.txt.
"""
import os
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "sw_oracle.cpp")
TESTS = ["tests/test_oracle_draws.py", "tests/test_oracle_labeling.py", "tests/test_oracle_sweep.py", "tests/test_oracle_physics.py"]

# (name, text to find exactly once, replacement)
MUTATIONS = [
    ("philox: 9 rounds", "round < 10", "round < 9"),
    ("philox: multipliers swapped", "uint64_t p0 = M0 * (uint64_t)c0;", "uint64_t p0 = M1 * (uint64_t)c0;"),
    ("bond draw: wrong word", "return w[2 * (site & 1) + (dir ? 1 : 0)];", "return w[(site & 1) + (dir ? 2 : 0)];"),
    ("bond draw: one call per site", "draw4(seed, site >> 1, t, PURPOSE_BOND, w);", "draw4(seed, site, t, PURPOSE_BOND, w);"),
    ("flip draw: sweep key dropped", "draw4(seed, root, t, PURPOSE_FLIP, w);", "draw4(seed, root, 0, PURPOSE_FLIP, w);"),
    ("state: modulo instead of mulhi", "return (uint32_t)(((uint64_t)w * (uint64_t)q) >> 32);", "return w % q;"),
    ("threshold: p = exp(-K)", "double p = -std::expm1(-K);", "double p = std::exp(-K);"),
    ("bond test: <= instead of <", "(uint64_t)swo_draw_bond(c->seed, t, i, 0) < c->T", "(uint64_t)swo_draw_bond(c->seed, t, i, 0) <= c->T"),
    ("bond: down neighbour without wrap", "const uint64_t d = ((y + 1) % L) * L + x;\n        uint8_t b = 0;", "const uint64_t d = (y + 1 < L ? y + 1 : y) * L + x;\n        uint8_t b = 0;"),
    ("bond: down bond owned by the wrong site", "if (c->spins[i] == c->spins[d] && (uint64_t)swo_draw_bond(c->seed, t, i, 1)", "if (c->spins[i] == c->spins[d] && (uint64_t)swo_draw_bond(c->seed, t, d, 1)"),
    ("labeling: left bond read from the site itself", "(bonds[l] & 1) != 0, (bonds[u] & 2) != 0", "(bonds[i] & 1) != 0, (bonds[u] & 2) != 0"),
    ("labeling: largest = last cluster", "if (queue.size() > big) big = queue.size();", "big = queue.size();"),
    ("flip: root state not copied to members", "else        c->spins[i] = c->spins[r];", "else        c->spins[i] = c->spins[i];"),
    ("measure: vertical pairs not counted", "if (c->spins[i] == c->spins[((y + 1) % L) * L + x]) ++e;", ""),
    ("sweep_measure: columns 1 and 2 swapped", "rc = swo_measure(c, &row[0], &row[3], &row[1], &row[2]);", "rc = swo_measure(c, &row[0], &row[3], &row[2], &row[1]);"),
    ("init: sweep counter not reset", "c->t = 0; c->have_spins = true; c->have_labels = false; c->n_clusters = c->largest = 0;\n    return SWO_OK;\n}\n\nint swo_set_state",
     "c->have_spins = true; c->have_labels = false; c->n_clusters = c->largest = 0;\n    return SWO_OK;\n}\n\nint swo_set_state"),
]


def run_one(name, find, repl, workdir):
    text = open(SRC).read()
    assert text.count(find) == 1, f"mutation '{name}': pattern found {text.count(find)} times"
    d = os.path.join(workdir, str(abs(hash(name))))
    os.makedirs(d, exist_ok=True)
    with open(os.path.join(d, "sw_oracle.cpp"), "w") as f:
        f.write(text.replace(find, repl))
    with open(os.path.join(d, "sw_oracle.h"), "w") as f:
        f.write(open(os.path.join(ROOT, "oracle", "sw_oracle.h")).read())
    lib = os.path.join(d, "libsw_oracle_mut.so")
    subprocess.run(["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-o", lib, os.path.join(d, "sw_oracle.cpp")], check=True)
    env = dict(os.environ, SWO_LIB=lib)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"] + TESTS,
                       cwd=ROOT, env=env, capture_output=True, text=True)
    failed = [l for l in r.stdout.splitlines() if l.startswith("FAILED")]
    return r.returncode != 0, (failed[0].split(" - ")[0] if failed else r.stdout.strip().splitlines()[-1])


def main():
    survivors = 0
    with tempfile.TemporaryDirectory() as workdir:
        for name, find, repl in MUTATIONS:
            caught, where = run_one(name, find, repl, workdir)
            survivors += not caught
            print(f"{'caught  ' if caught else 'SURVIVED'}  {name:48s} {where}", flush=True)
    print(f"{len(MUTATIONS) - survivors} of {len(MUTATIONS)} mutations caught")
    return 1 if survivors else 0


if __name__ == "__main__":
    sys.exit(main())
