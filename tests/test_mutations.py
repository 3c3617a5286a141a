"""Mutation check of the oracle pins: every one-line mutation of the oracle must fail at least one pin.

Each case copies oracle/, tpcsynth/ and tests/ to a temporary directory, changes ONE line of the copy of
oracle/tpcca_oracle.cpp (a decision, a sign, a constant, a tie-break of S5-S8) and runs tests/test_oracle_pins.py
on the copy: the run must FAIL.  A mutation that survives marks a decision no pin fixes.  The oracle in the
repository is never modified.  Mutations 0-15: the S5 decisions and constants; 16-34: S6 (selector), S7
(residuals), S8 (cross-sector merging).

Slow (a rebuild of the oracle and a run of the pins per mutation, ~10 minutes in all): collected always, run only
with `python -m pytest tests/test_mutations.py --slow` (tests/conftest.py).  Last full run: profiles/r3_mutations.md.
"""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def nth(s, old, new, k):
    """s with the k-th (0-based) occurrence of `old` replaced by `new`."""
    i = -1
    for _ in range(k + 1):
        i = s.index(old, i + 1)
    return s[:i] + new + s[i + len(old):]


MUTATIONS = [
 ("B gap >=", lambda s: nth(s, "if (++gap > max_gap) break;", "if (++gap >= max_gap) break;", 0)),
 ("C gap >=", lambda s: nth(s, "if (++gap > max_gap) break;", "if (++gap >= max_gap) break;", 1)),
 ("A gate from 4th", lambda s: s.replace("if (s.n >= 2 && dist2(s, ym, zm) > gate) break;", "if (s.n >= 3 && dist2(s, ym, zm) > gate) break;")),
 ("A gate removed", lambda s: s.replace("if (s.n >= 2 && dist2(s, ym, zm) > gate) break;", "")),
 ("search tie largest id", lambda s: s.replace("order[c] < order[best]", "order[c] > order[best]")),
 ("search window halved", lambda s: s.replace("std::fabs(ry) <= win_y && std::fabs(rz) <= win_z", "std::fabs(ry) <= win_y * (R)0.5 && std::fabs(rz) <= win_z * (R)0.5")),
 ("B gate halved", lambda s: nth(s, "if (b >= 0 && d2 <= gate) {", "if (b >= 0 && d2 <= gate * (R)0.5) {", 0)),
 ("C gate halved", lambda s: nth(s, "if (b >= 0 && d2 <= gate) {", "if (b >= 0 && d2 <= gate * (R)0.5) {", 1)),
 ("C gap on every row", lambda s: s.replace("if (!took && r < r0) {", "if (!took) {")),
 ("R3 off", lambda s: s.replace("if (s.n >= 2) {   // reading R3", "if (true) {   // reading R3")),
 ("min_hits <=", lambda s: s.replace("if (nh < min_hits || !have_snap)", "if (nh <= min_hits || !have_snap)")),
 ("c12 = 1/6", lambda s: s.replace("c12 = (R)(1.0 / 12.0)", "c12 = (R)(1.0 / 6.0)")),
 ("search one z slice", lambda s: s.replace("for (int bz = bz0; bz <= bz1; ++bz) {\n      int64_t b0 = row_bin_base[r] +", "for (int bz = bz0; bz <= bz0; ++bz) {\n      int64_t b0 = row_bin_base[r] +")),
 ("c640 changed", lambda s: s.replace("c640 = (R)(3.0 / 640.0)", "c640 = (R)(3.0 / 64.0)")),
 ("C starts at last", lambda s: s.replace("for (int r = top; r >= 0; --r) {", "for (int r = last; r >= 0; --r) {")),
 ("R2: top -> n_rows-1 start", lambda s: s.replace("for (int r = top; r >= 0; --r) {", "for (int r = n_rows - 1; r >= 0; --r) {")),
 # ---- S6 / S7 / S8 (round 2)
 ("S6 tie -> larger track", lambda s: s.replace("if (o < 0 || nh > hit_offset[o + 1] - hit_offset[o]) owner[c] = (int32_t)t;", "if (o < 0 || nh >= hit_offset[o + 1] - hit_offset[o]) owner[c] = (int32_t)t;")),
 ("S6 keep <", lambda s: s.replace("if (shared * 1000 <= (int64_t)max_shared_permille * nh)", "if (shared * 1000 < (int64_t)max_shared_permille * nh)")),
 ("S7 residual of every hit", lambda s: s.replace("        if (owner[c] != t) continue;\n        const R ry", "        const R ry")),
 ("S7 z residual ignores z_ref", lambda s: s.replace("const R rz = (sz[c] - T.z_ref) - s.p[1];", "const R rz = sz[c] - s.p[1];")),
 ("S7 quantiser truncates", lambda s: s.replace("R v = std::nearbyint(r * res_inv_q);", "R v = std::trunc(r * res_inv_q);")),
 ("S8 gap from 2", lambda s: s.replace("if (gap < 1 || gap > A.mg_gap) continue;", "if (gap < 2 || gap > A.mg_gap) continue;")),
 ("S8 gap >=", lambda s: s.replace("if (gap < 1 || gap > A.mg_gap) continue;", "if (gap < 1 || gap >= A.mg_gap) continue;")),
 ("S8 rotation sign", lambda s: s.replace("const R sa = dir == 0 ? A.sec_sin : -A.sec_sin;", "const R sa = dir == 0 ? -A.sec_sin : A.sec_sin;")),
 ("S8 no mutual check", lambda s: s.replace("if (back.have && back.sec == s && back.trk == (int)ia) {", "if (back.have) {")),
 ("S8 windows halved", lambda s: s.replace("if (!(std::fabs(dy) <= A.mg_dy && std::fabs(dz) <= A.mg_dz && std::fabs(ds) <= A.mg_ds)) continue;", "if (!(std::fabs(dy) <= A.mg_dy * (R)0.25 && std::fabs(dz) <= A.mg_dz * (R)0.25 && std::fabs(ds) <= A.mg_ds * (R)0.25)) continue;")),
 ("S8 z re-reference sign", lambda s: s.replace("st.p[1] = st.p[1] + (tu.z_ref - tg.z_ref);", "st.p[1] = st.p[1] - (tu.z_ref - tg.z_ref);")),
 ("S8 refit rotation sign", lambda s: s.replace("const R sa = up_is_next ? -G.sec_sin : G.sec_sin;", "const R sa = up_is_next ? G.sec_sin : -G.sec_sin;")),
 ("S8 rotate drops j10", lambda s: s.replace("const R j10 = -((s.p[3] * sa) / cf2);", "const R j10 = (R)0 * ((s.p[3] * sa) / cf2);")),
 ("S8 rotate drops j20", lambda s: s.replace("const R j20 = -((s.p[4] * Bc) * sa);", "const R j20 = (R)0 * ((s.p[4] * Bc) * sa);")),
 ("S8 rotate j22 inverted", lambda s: s.replace("const R j22 = cf2 / cf;", "const R j22 = cf / cf2;")),
 ("S8 z pre-cut dropped", lambda s: s.replace("          if (!(std::fabs(zb - za) <= A.mg_zpre)) continue;\n", "")),
 ("S8 dy window strict", lambda s: s.replace("if (!(std::fabs(dy) <= A.mg_dy && ", "if (!(std::fabs(dy) < A.mg_dy && ")),
 ("S8 tie -> larger sector/track", lambda s: s.replace("    if (sec != b.sec) return sec < b.sec;\n    return trk < b.trk;", "    if (sec != b.sec) return sec > b.sec;\n    return trk > b.trk;")),
]


def run_pins_on_copy(tmp, mutate):
    for sub in ("oracle", "tpcsynth", "tests"):
        shutil.copytree(os.path.join(ROOT, sub), os.path.join(tmp, sub),
                        ignore=shutil.ignore_patterns("*.so", "__pycache__", "test_gpu*", "test_abi*", "test_multirank*",
                                                      "test_zz*", "test_mutations*"))
    path = os.path.join(tmp, "oracle", "tpcca_oracle.cpp")
    src = open(path).read()
    out = mutate(src)
    open(path, "w").write(out)
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_oracle_pins.py", "-q", "-x", "-p", "no:cacheprovider"],
                       cwd=str(tmp), capture_output=True, text=True)
    tail = [l for l in r.stdout.splitlines() if l.startswith("FAILED") or " passed" in l or " failed" in l]
    return src != out, r.returncode, " | ".join(tail)[:300]


@pytest.mark.slow
def test_unmutated_copy_passes(tmp_path):
    """The harness itself: an unchanged copy passes every pin (so a failing mutated copy means the mutation)."""
    changed, rc, tail = run_pins_on_copy(str(tmp_path), lambda s: s)
    assert not changed and rc == 0, tail


@pytest.mark.slow
@pytest.mark.parametrize("k", range(len(MUTATIONS)), ids=[f"{k}-{m[0]}".replace(" ", "_") for k, m in enumerate(MUTATIONS)])
def test_mutation_is_caught(tmp_path, k):
    name, mutate = MUTATIONS[k]
    changed, rc, tail = run_pins_on_copy(str(tmp_path), mutate)
    assert changed, f"mutation '{name}' no longer applies: the oracle line it edits has changed"
    assert rc != 0, f"mutation '{name}' SURVIVES every pin: {tail}"
    print(f"[{k}] {name}: CAUGHT :: {tail}")
