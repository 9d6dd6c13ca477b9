"""Mutation check of the oracle's pins (no GPU): every plausible one-line mistake listed below is applied to a COPY
of oracle/autoddl_ref.cpp, built, and the pin files are run against the broken build (AUTODDL_REF_SO); each must
make at least one pin fail.  The pins that count are the ones whose expected values come from the paper, hand
arithmetic, closed forms or brute force: tests that compare with tests/golden/survey_crosscheck.txt or
extra_config_optima.txt (values not fixed by the paper) are deselected here, so a mutant cannot be "killed" by them.

VERDICT round 1 found five result-changing mutants (M01-M05) and three boundary flips (M06-M08) that passed every
CPU test; tests/test_oracle_ragged_pins.py was written against them.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "autoddl_ref.cpp")
PIN_FILES = ["tests/test_oracle_pins.py", "tests/test_oracle_ragged_pins.py", "tests/test_oracle_mh.py",
             "tests/test_oracle_accum.py", "tests/test_oracle_paper_space.py", "tests/test_oracle_pipeline.py", "tests/test_oracle_folded.py",
             "tests/test_shard_gloo.py::test_oracle_best_of_starts_lowest_index"]
DESELECT = "not survey_crosscheck and not brute_force_config1"

# (name, old text, new text, which occurrence of `old` (0-based; None = it must be unique))
MUTANTS = [
    ("M01 all-to-all phase outermost level first",
     "for (int d = D - 1; d >= 0; --d) {\n    const bool cs", "for (int d = 0; d < D; ++d) {\n    const bool cs", None),
    ("M02 all-to-all message taken before the change",
     "      cur[d] = b[d];\n      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size\n      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)\n      cost += autoddl_ref_collective(3,",
     "      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size\n      cur[d] = b[d];\n      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)\n      cost += autoddl_ref_collective(3,", None),
    ("M03 P->B scatters on axis 0", "(b[d] == REF_B) ? REF_S1 : b[d]", "(b[d] == REF_B) ? REF_S0 : b[d]", None),
    ("M04 backward leg replaced by a second forward leg", "return fwd + bwd;", "return fwd + fwd;", None),
    ("M05 producer's element size prices the edge",
     "cur->in_rows, cur->in_cols, cur->act_bytes, Oi, Ij", "cur->in_rows, cur->in_cols, prev->act_bytes, Oi, Ij", None),
    ("M05b producer's element size prices the backward leg",
     "cur->in_rows, cur->in_cols, cur->act_bytes, db, da", "cur->in_rows, cur->in_cols, prev->act_bytes, db, da", None),
    ("M06 column split limit exclusive", "if (colsplit > cur->max_split_cols)", "if (colsplit >= cur->max_split_cols)", None),
    ("M06b row split limit exclusive", "if (rowsplit > cur->max_split_rows)", "if (rowsplit >= cur->max_split_rows)", None),
    ("M07 memory cap exclusive", "> net->mem_cap_bytes / L", ">= net->mem_cap_bytes / L", None),
    ("M08 Metropolis keeps the last strategy attaining the best cost", "if (cur < best) { best = cur; sbest = s; }",
     "if (cur <= best) { best = cur; sbest = s; }", None),
    ("M09 edge tensor taken from the producer's output", "cur->in_rows, cur->in_cols, cur->act_bytes, Oi, Ij",
     "prev->M, prev->N, cur->act_bytes, Oi, Ij", None),
    ("M10 weight gradient of the full weight", "const int64_t nw = autoddl_ref_local_size(cur->Kd, cur->N, W, mesh);\n  int64_t v = 0;",
     "const int64_t nw = cur->Kd * cur->N;\n  int64_t v = 0;", None),
    ("M11 reduce phase outermost level first",
     "for (int d = D - 1; d >= 0; --d)\n    if (cur[d] == REF_P && b[d] != REF_P) {",
     "for (int d = 0; d < D; ++d)\n    if (cur[d] == REF_P && b[d] != REF_P) {", None),
    ("M12 gather phase innermost level first",
     "for (int d = 0; d < D; ++d)\n    if ((cur[d] == REF_S0 || cur[d] == REF_S1) && b[d] == REF_B) {",
     "for (int d = D - 1; d >= 0; --d)\n    if ((cur[d] == REF_S0 || cur[d] == REF_S1) && b[d] == REF_B) {", None),
    ("M13 gather message taken before the gather",
     "      cur[d] = REF_B;\n      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size",
     "      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size\n      cur[d] = REF_B;", None),
    ("M14 reduce-scatter message taken after the scatter",
     "      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // RS input size (Table 2 caption)\n      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)\n      cost += autoddl_ref_collective(1, n, mesh->size[d], net->alpha_ps[c], net->beta_ps_per_byte[c]);\n      cur[d] = (b[d] == REF_B) ? REF_S1 : b[d];",
     "      cur[d] = (b[d] == REF_B) ? REF_S1 : b[d];\n      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // RS input size (Table 2 caption)\n      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)\n      cost += autoddl_ref_collective(1, n, mesh->size[d], net->alpha_ps[c], net->beta_ps_per_byte[c]);", None),
    ("M15 AllReduce latency 2(p-1) alpha", "return (2 * p - 1) * alpha", "return 2 * (p - 1) * alpha", None),
    ("M16 AlltoAll with the (p-1)/p factor", "return (p - 1) * alpha + n * beta;", "return (p - 1) * alpha + (p - 1) * sh * beta;", None),
    ("M17 floor instead of ceil", "return (a + b - 1) / b;", "return a / b;", None),
    ("M18 local size with the axes swapped", "return ceil_div(R, f0) * ceil_div(C, f1);", "return ceil_div(R, f1) * ceil_div(C, f0);", None),
    ("M19 DP keeps the last minimiser", "if (v < best) { best = v; arg = i; }", "if (v <= best) { best = v; arg = i; }", None),
    ("M20 DP end state keeps the last minimiser", "if (f[j] < f[js]) js = j;", "if (f[j] <= f[js]) js = j;", 0),
    ("M48 segment end state keeps the last minimiser", "if (f[j] < f[js]) js = j;", "if (f[j] <= f[js]) js = j;", 1),
    ("M21 CD keeps the last minimiser", "if (arg < 0 || g < best) { best = g; arg = c; }", "if (arg < 0 || g <= best) { best = g; arg = c; }", None),
    ("M22 CD ignores the right neighbour", "if (l < L - 1) g += Tp[((int64_t)(l + 1) * K + c) * K + s[l + 1]];",
     "if (l < L - 2) g += Tp[((int64_t)(l + 1) * K + c) * K + s[l + 1]];", None),
    ("M23 dual keeps B", "if (s == REF_B) return REF_P;", "if (s == REF_B) return REF_B;", None),
    ("M24 weight gradient priced with the activation element size", "nw * cur->wgrad_bytes", "nw * cur->act_bytes", None),
    ("M25 memory without the output activation",
     "mem += (autoddl_ref_local_size(cur->in_rows, cur->in_cols, I, mesh) +\n          autoddl_ref_local_size(cur->M, cur->N, O, mesh)) * cur->act_bytes;",
     "mem += (autoddl_ref_local_size(cur->in_rows, cur->in_cols, I, mesh)) * cur->act_bytes;", None),
    # (not listed: "row split counts the output only" -- equivalent, I = S0 implies O = S0 in every signature row)
    ("M27 memory cap not divided by L", "> net->mem_cap_bytes / L", "> net->mem_cap_bytes", None),
    ("M28 accumulation multiplies the node cost too", "= m * e + v + (ok ? 0 : REF_PEN);", "= m * (e + v) + (ok ? 0 : REF_PEN);", None),
    ("M29 signature 4 outputs B", "{REF_S0, REF_S1, REF_P,  REF_B, REF_P, REF_P};", "{REF_S0, REF_S1, REF_P,  REF_B, REF_B, REF_P};", None),
    ("M30 link classes swapped in the gather", "cur[d] = REF_B;\n      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size\n      const int c = mesh->link[d] & 1;",
     "cur[d] = REF_B;\n      const int64_t n = autoddl_ref_local_size(rows, cols, cur, mesh) * eb;   // output size\n      const int c = 1 - (mesh->link[d] & 1);", None),
    ("M31 level 0 least significant in the signature index", "for (int t = 0; t < D - 1 - d; ++t) div *= 6;", "for (int t = 0; t < d; ++t) div *= 6;", None),
    ("M32 weight states of signature 2", "{REF_B,  REF_S1, REF_S0, REF_B, REF_B, REF_P};", "{REF_B,  REF_S1, REF_S1, REF_B, REF_B, REF_P};", None),
    ("M33 chain cost starts from the strategy's own first state", "int32_t prev = 0;\n  for (int32_t l = 0; l < L; ++l) {\n    c += T[((int64_t)l * K + prev) * K + s[l]];",
     "int32_t prev = s[0];\n  for (int32_t l = 0; l < L; ++l) {\n    c += T[((int64_t)l * K + prev) * K + s[l]];", None),
    ("M34 MH uphill test flipped to strict", "acc = tau_ps * autoddl_ref_neglog_q16(x) >= (d << 16);", "acc = tau_ps * autoddl_ref_neglog_q16(x) > (d << 17);", None),
    ("M35 attention accepts a partial-sum signature", "{REF_S0, REF_S1, -1, REF_B, -1, -1};", "{REF_S0, REF_S1, -1, REF_B, REF_P, -1};", None),
    ("M36 column split counts the input", "if (O[d] == REF_S1) colsplit", "if (I[d] == REF_S1) colsplit", None),
    ("M37 weight-gradient all-reduce charged on P levels", "    if (W[d] == REF_B) {\n      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)\n      v +=",
     "    if (W[d] == REF_B || W[d] == REF_P) {\n      const int c = mesh->link[d] & 1;                 // bit 0: link class; bits 8..13: allowed rows (R24)\n      v +=", None),
    ("M38 memory counts resident weight with the gradient element size", "W, mesh) * cur->wstate_bytes;", "W, mesh) * cur->wgrad_bytes;", None),
    ("M40 a segment's first layer pays the redistribution from the previous stage",
     "for (int j = 0; j < K; ++j) f[j] = node[(int64_t)a * K + j] + (mask[(int64_t)a * K + j] ? 0 : REF_PEN);\n    for (int32_t b = a + 1; b <= L; ++b) {",
     "for (int j = 0; j < K; ++j) f[j] = T[(int64_t)a * K * K + j];\n    for (int32_t b = a + 1; b <= L; ++b) {", None),
    ("M41 partition forgets the transfer at a stage's right boundary", "+ xfer[a] + (b < L ? xfer[b] : 0); };", "+ xfer[a]; };", None),
    ("M42 bottleneck objective takes the faster stage", "objective == 0 ? prev + cs : (prev > cs ? prev : cs);", "objective == 0 ? prev + cs : (prev < cs ? prev : cs);", None),
    ("M43 partition keeps the last start attaining the minimum", "if (v < g[(size_t)k * (L + 1) + b]) {", "if (v <= g[(size_t)k * (L + 1) + b]) {", None),
    ("M44 stage transfer paid in one direction only", "xfer[b] = 2 * m * (net->alpha_ps[1]", "xfer[b] = m * (net->alpha_ps[1]", None),
    ("M45 stage transfer over the intra-node link", "xfer[b] = 2 * m * (net->alpha_ps[1] + ceil_div(bytes, q) * net->beta_ps_per_byte[1]);",
     "xfer[b] = 2 * m * (net->alpha_ps[0] + ceil_div(bytes, q) * net->beta_ps_per_byte[0]);", None),
    ("M46 segment strategies keep the last minimiser", "if (v < best) { best = v; ar = i; }", "if (v <= best) { best = v; ar = i; }", None),
    ("M50 folded space enumerates p1 upwards", "for (int n1 = n - n0; n1 >= 0; --n1) {", "for (int n1 = 0; n1 <= n - n0; ++n1) {", None),
    ("M51 folded groups ignore the link class", "mesh->size[d] == mesh->size[d - 1] && (mesh->link[d] & 1) == (mesh->link[d - 1] & 1)",
     "mesh->size[d] == mesh->size[d - 1]", None),
    ("M47 best of starts keeps the last start", "if (cost[p * S + s] < cost[p * S + arg]) arg = s;", "if (cost[p * S + s] <= cost[p * S + arg]) arg = s;", None),
]


def _kill(args):
    idx, (name, old, new, occ), tmp = args
    src = open(SRC).read()
    n = src.count(old)
    if occ is None:
        assert n == 1, f"{name}: the text to mutate occurs {n} times in oracle/autoddl_ref.cpp (update MUTANTS)"
        mutated = src.replace(old, new)
    else:
        parts = src.split(old)
        mutated = old.join(parts[:occ + 1]) + new + old.join(parts[occ + 1:])
    cpp = os.path.join(tmp, f"m{idx}.cpp")
    so = os.path.join(tmp, f"m{idx}.so")
    with open(cpp, "w") as f:
        f.write(mutated)
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-I", os.path.join(ROOT, "oracle"), cpp, "-o", so])
    env = dict(os.environ, AUTODDL_REF_SO=so)
    files = [f for f in PIN_FILES if os.path.exists(os.path.join(ROOT, f.split("::")[0]))]
    r = subprocess.run([sys.executable, "-m", "pytest", *files, "-x", "-q", "-k", DESELECT, "-p", "no:cacheprovider"],
                       cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return name, r.returncode, r.stdout[-400:]


def test_unmutated_oracle_passes_the_same_selection(tmp_path):
    """the selection used against the mutants is green on the real oracle (otherwise every mutant dies trivially)"""
    so = os.path.join(str(tmp_path), "clean.so")
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", SRC, "-o", so])
    files = [f for f in PIN_FILES if os.path.exists(os.path.join(ROOT, f.split("::")[0]))]
    r = subprocess.run([sys.executable, "-m", "pytest", *files, "-x", "-q", "-k", DESELECT, "-p", "no:cacheprovider"],
                       cwd=ROOT, env=dict(os.environ, AUTODDL_REF_SO=so), stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert r.returncode == 0, r.stdout[-2000:]


def test_every_mutant_is_killed(tmp_path):
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(_kill, [(i, m, str(tmp_path)) for i, m in enumerate(MUTANTS)]))
    survivors = [name for name, rc, _ in results if rc == 0]
    broken = [(name, out) for name, rc, out in results if rc not in (0, 1)]
    assert not broken, broken                           # 1 = tests failed (wanted); anything else = the run itself broke
    assert not survivors, f"mutants that pass every pin: {survivors}"
