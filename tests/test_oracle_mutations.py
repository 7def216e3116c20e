"""The pins of tests/test_oracle_pins.py must be able to FAIL: every single-line mutation of the oracle below
(a sign, a dropped factor, x for y, a count for a weight, a missing clamp, the tie rule, the residual sign, the
decode accumulation) is compiled into a scratch library, swapped in for the real one, and at least one pin has to
reject it.  CPU only; the scratch build lives in pytest's tmp_path.
"""
import ctypes as C
import inspect
import subprocess
from pathlib import Path

import pytest

import test_oracle_pins as pins
from oracle import gsrq_oracle as o

SRC = Path(o.__file__).resolve().parent / "gsrq_oracle.c"

# (name, text in gsrq_oracle.c that occurs exactly once, its replacement)
MUTATIONS = [
    ("eq5_sign_of_bias", "sc = 2.0 * gk * dot - gk * gk;", "sc = 2.0 * gk * dot + gk * gk;"),
    ("eq5_dropped_factor_2", "sc = 2.0 * gk * dot - gk * gk;", "sc = gk * dot - gk * gk;"),
    ("eq7_x_for_y", "B[(int64_t)k * d + j] += wi * yj;", "B[(int64_t)k * d + j] += wi * xj;"),
    ("eq8_count_for_weight", "W[k] += wi;", "W[k] += 1.0;"),
    ("eq8_missing_clamp", "g[k] = (float)(gk > 0.0 ? gk : 0.0);", "g[k] = (float)gk;"),
    ("tie_rule_highest_index", "if (sc > b1) { b2 = b1; b1 = sc; k1 = k; }", "if (sc >= b1) { b2 = b1; b1 = sc; k1 = k; }"),
    ("residual_sign", "volatile float v = r[i * d + j] - c;", "volatile float v = r[i * d + j] + c;"),
    ("decode_overwrites_instead_of_adding", "if (st == 0) acc = c; else acc = acc + c;", "acc = c;"),
    ("eq6_unnormalised_weight", "A[(int64_t)k * d + j] += wi * xj;", "A[(int64_t)k * d + j] += xj;"),
    ("break_rule_off_by_one", "if (t > 1 && nch == 0) break;", "if (nch == 0) break;"),
]


def _pin_calls():
    """Every pin of test_oracle_pins.py as a zero-argument callable (parametrised ones at their parameters)."""
    calls = []
    for name, fn in inspect.getmembers(pins, inspect.isfunction):
        if not name.startswith("test_"):
            continue
        marks = [m for m in getattr(fn, "pytestmark", []) if m.name == "parametrize"]
        if not marks:
            calls.append((name, fn))
            continue
        for vals in marks[0].args[1]:
            vals = vals if isinstance(vals, (tuple, list)) else (vals,)
            calls.append((f"{name}{list(vals)}", (lambda f=fn, v=vals: f(*v))))
    return calls


@pytest.mark.parametrize("name,old,new", MUTATIONS, ids=[m[0] for m in MUTATIONS])
def test_a_pin_rejects_the_mutated_oracle(tmp_path, monkeypatch, name, old, new):
    text = SRC.read_text()
    assert text.count(old) == 1, f"mutation target for {name} must occur exactly once in gsrq_oracle.c"
    src = tmp_path / "gsrq_oracle_mut.c"
    src.write_text(text.replace(old, new))
    so = tmp_path / "libgsrq_oracle_mut.so"
    subprocess.run(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
                    "-o", str(so), str(src), "-lm"], check=True)
    mut = C.CDLL(str(so))
    mut.gsrq_oracle_wdist.restype = C.c_double
    mut.gsrq_oracle_splitmix64_next.restype = C.c_uint64
    o.lib()                                   # make sure the real library is loaded before it is swapped out
    monkeypatch.setattr(o, "_lib", mut)
    rejected_by = None
    for pin_name, call in _pin_calls():
        try:
            call()
        except Exception:                     # an assertion (or a crash of the check) rejects the mutant
            rejected_by = pin_name
            break
    assert rejected_by is not None, f"no pin noticed the mutation {name!r}"


def test_the_unmutated_oracle_passes_the_same_calls():
    """The harness above must not reject everything: the real oracle passes every call it makes."""
    for _, call in _pin_calls():
        call()
