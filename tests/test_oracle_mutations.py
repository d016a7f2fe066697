"""Mutation audit of the oracle's pins (task prompt, section 3: the pins must be "chosen so that a plausible mistake
anywhere in it -- a dropped term, a wrong sign or index, a transposed operand -- fails one of them").

Each mutation below is one such mistake, applied to a scratch copy of oracle/zmc_oracle.c; the copy is built on its own
(ZMC_ORACLE_SRC / ZMC_ORACLE_LIB, oracle/build.py) and the oracle's pin tests are run against it in a subprocess.  The audit
passes when every mutated oracle turns at least one pin test red.  The first two are the ones the round-1 review found
passing (c5's factor, c4's parameter assignment).  By default the first eight run (the CPU suite stays short);
ZMC_MUTATION_AUDIT=1 runs all 24 (about four minutes).  Nothing here touches the CUDA path.
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PIN_TESTS = ["tests/test_oracle_pins.py", "tests/test_oracle_closed_forms.py", "tests/test_user_integrand_cpu.py",
             "tests/test_shard_gloo.py"]

# (label, text in oracle/zmc_oracle.c, what the mistake turns it into)
MUTATIONS = [
    ("c5: factor (1 - x4 y0 y1 y2) -- wrong sign and wrong parameter", "(1.0 + x[4] * y[0] * y[1] * y[2])", "(1.0 - x[3] * y[0] * y[1] * y[2])"),
    ("c4: x3 and x4 swapped", "(k < 2) ? x[1] : (k < 4) ? x[2] : x[3]", "(k < 2) ? x[1] : (k < 4) ? x[3] : x[2]"),
    ("stream: lanes of a block taken in reverse order", "return r[q & 3];", "return r[3 - (q & 3)];"),
    ("estimator: biased variance (n instead of n - 1)", "ss / (long double)(p->n - 1)", "ss / (long double)(p->n)"),
    # reading S5, the four single-line mistakes the round-2 review found passing (pinned by the S5_BOX cases of test_oracle_pins.py)
    ("sample map: width rounded as float(b) - float(a) instead of float(b - a)",
     "width[k] = mirror(p->bounds[2 * k + 1] - p->bounds[2 * k], p->mode);",
     "width[k] = mirror(p->bounds[2 * k + 1], p->mode) - mirror(p->bounds[2 * k], p->mode);"),
    ("sample map: a_k not rounded in mirror mode", "a[k] = mirror(p->bounds[2 * k], p->mode);", "a[k] = p->bounds[2 * k];"),
    ("family constants not rounded in mirror mode", "cst[c] = mirror(p->consts[c], p->mode);", "cst[c] = p->consts[c];"),
    ("sample map: u * width + a without the fused multiply-add", "y[k] = fma(u, width[k], a[k]);", "y[k] = u * width[k] + a[k];"),
    # ---- the rest run with ZMC_MUTATION_AUDIT=1 ----
    ("c5: phase coefficients permuted", "x[1] * y[0] + x[2] * y[1] + x[3] * y[2]", "x[2] * y[0] + x[1] * y[1] + x[3] * y[2]"),
    ("c5: a y_k dropped from the factor", "(1.0 + x[4] * y[0] * y[1] * y[2])", "(1.0 + x[4] * y[0] * y[1])"),
    ("c4: a not squared", "acc += a * a * d * d;", "acc += a * d * d;"),
    ("c3: coefficient k+2 instead of k+1", "x[k % 3] * (double)(k + 1)", "x[k % 3] * (double)(k + 2)"),
    ("c3: parameter index shifted", "x[k % 3] * (double)(k + 1)", "x[(k + 1) % 3] * (double)(k + 1)"),
    ("c2: parameters transposed", "sin(x[0] * y[0] + x[1] * y[1])", "sin(x[1] * y[0] + x[0] * y[1])"),
    ("p6: last parameter dropped", "for (int l = 0; l < M; ++l) arg += x[l];", "for (int l = 0; l < M - 1; ++l) arg += x[l];"),
    ("Philox: wrong key increment", "k1 += 0xBB67AE85u;", "k1 += 0xBB67AE86u;"),
    ("Philox: high halves crossed", "uint32_t n0 = hi1 ^ c1 ^ k0;", "uint32_t n0 = hi0 ^ c1 ^ k0;"),
    ("stream: counter drops the high word of t", "(uint32_t)t, (uint32_t)(t >> 32) };", "(uint32_t)t, 0 };"),
    ("stream: dimensions take their words in reverse order", "s * (uint64_t)p->N + (uint64_t)k;", "s * (uint64_t)p->N + (uint64_t)(p->N - 1 - k);"),
    ("uniform fp64: the half-step offset dropped", "(2.0 * (double)w + 1.0) * 0x1p-33", "(2.0 * (double)w) * 0x1p-33"),
    ("uniform fp32: bits 8..30 instead of 9..31", "(double)(w >> 9)", "(double)((w >> 8) & 0x7fffff)"),
    ("sample map: width = b instead of b - a", "mirror(p->bounds[2 * k + 1] - p->bounds[2 * k], p->mode)", "mirror(p->bounds[2 * k + 1], p->mode)"),
    ("estimator: stderr without the volume", "(long double)V * sqrtl(var / (long double)p->n)", "sqrtl(var / (long double)p->n)"),
    ("decode: first list fastest", "for (int i = p->M - 1; i >= 0; --i) {\n        uint64_t L", "for (int i = 0; i < p->M; ++i) {\n        uint64_t L"),
]
N_DEFAULT = 8
FULL = os.environ.get("ZMC_MUTATION_AUDIT") == "1"


SELECTED = MUTATIONS if FULL else MUTATIONS[:N_DEFAULT]


@pytest.mark.parametrize("label,old,new", SELECTED, ids=[m[0].split(" --")[0] for m in SELECTED])
def test_a_broken_oracle_fails_its_pins(label, old, new, tmp_path):
    src = open(os.path.join(ROOT, "oracle", "zmc_oracle.c")).read()
    assert src.count(old) >= 1, f"the audit no longer matches the oracle text: {old!r}"
    mutated = tmp_path / "zmc_oracle_mutated.c"
    mutated.write_text(src.replace(old, new))
    env = dict(os.environ, ZMC_ORACLE_SRC=str(mutated), ZMC_ORACLE_LIB=str(tmp_path / "libzmc_oracle_mutated.so"))
    env.pop("ZMC_MUTATION_AUDIT", None)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider", *PIN_TESTS],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 1 and " failed" in r.stdout, f"mutation survived: {label}\n{r.stdout[-2000:]}\n{r.stderr[-2000:]}"


def test_the_unmutated_copy_passes_the_same_command(tmp_path):
    """Control: the same subprocess command on an unmodified copy is green, so a red run above is the mutation's doing."""
    src = open(os.path.join(ROOT, "oracle", "zmc_oracle.c")).read()
    copy = tmp_path / "zmc_oracle_copy.c"
    copy.write_text(src)
    env = dict(os.environ, ZMC_ORACLE_SRC=str(copy), ZMC_ORACLE_LIB=str(tmp_path / "libzmc_oracle_copy.so"))
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider",
                        "tests/test_oracle_pins.py", "tests/test_oracle_closed_forms.py"],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
