"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: a small driver calls every entry
point of oracle/autoddl_ref.cpp on a tiny chain; any out-of-bounds access, signed overflow or misaligned access aborts."""
import os
import shutil
import subprocess
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r'''
#include <cstdio>
#include <vector>
#include "autoddl_ref.h"
int main() {
  ref_mesh mesh{3, {2, 3, 2}, {1, 1, 0}};
  ref_net net{{5000000, 20000000}, {3, 40}, 3000000, 3};
  const int L = 3, Bp = 2, K = autoddl_ref_num_signatures(&mesh), S = 2;
  std::vector<ref_layer> layers(Bp * L);
  for (int i = 0; i < Bp * L; ++i) {
    ref_layer& r = layers[i];
    r = ref_layer{1001 + i, 777, 513 + 7 * i, 1001 + i, 777, (i % 3 == 1) ? REF_ATTN : REF_GEMM, 2, 4, 18, 5 + i, 9};
  }
  std::vector<int64_t> T((size_t)Bp * L * K * K), node((size_t)Bp * L * K), cost(Bp * S), fc(Bp * S), opt(Bp), trace(Bp * S * 64 * L);
  std::vector<uint8_t> mask((size_t)Bp * L * K);
  std::vector<int32_t> strat(Bp * S * L), fs(Bp * S * L), sweeps(Bp * S), acc(Bp * S), dps(Bp * L), init(Bp * S * L);
  for (size_t i = 0; i < init.size(); ++i) init[i] = (int)((i * 37) % K);
  if (autoddl_ref_build_tables(layers.data(), Bp, L, &mesh, &net, T.data(), node.data(), mask.data())) return 1;
  if (autoddl_ref_chain_dp(T.data(), Bp, L, K, opt.data(), dps.data())) return 2;
  if (autoddl_ref_coord_descent(T.data(), Bp, L, K, init.data(), S, 64, cost.data(), strat.data(), sweeps.data(), trace.data())) return 3;
  if (autoddl_ref_metropolis(T.data(), Bp, L, K, init.data(), S, 500, 1000000, 7, cost.data(), strat.data(), fc.data(), fs.data(), acc.data(), nullptr)) return 4;
  ref_mesh m1{1, {4, 0, 0}, {1, 0, 0}};
  std::vector<int64_t> T1((size_t)4 * 6 * 6);
  std::vector<ref_layer> l1(layers.begin(), layers.begin() + 4);
  for (auto& r : l1) r.kind = REF_GEMM;
  if (autoddl_ref_build_tables(l1.data(), 1, 4, &m1, &net, T1.data(), nullptr, nullptr)) return 5;
  int64_t bc; int32_t bs[4];
  if (autoddl_ref_brute_force(T1.data(), 4, 6, &bc, bs)) return 6;
  int64_t dc; int32_t ds[4];
  if (autoddl_ref_chain_dp(T1.data(), 1, 4, 6, &dc, ds) || dc != bc) return 7;
  for (uint64_t x = 1; x < (1ull << 32); x += 99999989ull) if (autoddl_ref_neglog_q16(x) < 0) return 8;
  std::printf("ok %lld %lld\n", (long long)opt[0], (long long)bc);
  return 0;
}
'''


def test_oracle_under_asan_ubsan():
    gxx = shutil.which("g++")
    if gxx is None:
        pytest.skip("no g++")
    with tempfile.TemporaryDirectory() as d:
        drv = os.path.join(d, "drv.cpp")
        open(drv, "w").write(DRIVER)
        exe = os.path.join(d, "drv")
        cmd = [gxx, "-O1", "-g", "-std=c++17", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
               "-I", os.path.join(ROOT, "oracle"), drv, os.path.join(ROOT, "oracle", "autoddl_ref.cpp"), "-o", exe]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0 and ("asan" in r.stderr.lower() or "sanitize" in r.stderr.lower()):
            pytest.skip("g++ cannot link the sanitizer runtimes here: " + r.stderr[-200:])
        assert r.returncode == 0, r.stderr[-2000:]
        env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1")
        env.pop("LD_PRELOAD", None)
        r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=300)
        assert r.returncode == 0 and r.stdout.startswith("ok "), (r.returncode, r.stdout, r.stderr[-3000:])
