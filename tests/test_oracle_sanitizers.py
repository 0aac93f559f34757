"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md section 5 planned `-fsanitize=address,
undefined` for the oracle): oracle/pp_oracle.cpp is compiled together with a small driver that exercises every entry
point -- heap buffers of exactly the documented sizes, an index list, the optional pot = NULL, several OpenMP threads --
and must run to completion without a sanitizer report.  CPU only; skipped if the toolchain has no sanitizer runtime."""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>
extern "C" {
void oracle_forces(const double*, const double*, int64_t, double, double, const int64_t*, int64_t, double*, double*, int);
void oracle_forces_ld(const double*, const double*, int64_t, double, double, const int64_t*, int64_t, double*, double*, int);
int64_t oracle_kdk_paper(double*, double*, const double*, double*, int64_t, double, int64_t, double, double, int, int);
int64_t oracle_kdk_halfkick(double*, double*, const double*, double*, int64_t, double, int64_t, double, double, int, int);
void oracle_invariants(const double*, const double*, const double*, const double*, int64_t, double, double, double*, int);
int oracle_max_threads(void);
}
int main() {
    const int64_t N = 257;
    // heap blocks of exactly the documented sizes, so that any overrun lands in a red zone
    std::vector<double> pos(3 * N), vel(3 * N), mass(N), acc(3 * N), pot(N), out(16);
    uint64_t s = 88172645463325252ull;
    auto rnd = [&]() { s ^= s << 13; s ^= s >> 7; s ^= s << 17; return (double)(s >> 11) / 9007199254740992.0 - 0.5; };
    for (auto& x : pos) x = rnd();
    for (auto& x : vel) x = 0.1 * rnd();
    for (auto& x : mass) x = (1.0 + rnd()) / N;
    for (int threads : {1, 3}) {
        oracle_forces(pos.data(), mass.data(), N, 1.5, 0.05, nullptr, N, acc.data(), pot.data(), threads);
        oracle_forces(pos.data(), mass.data(), N, 1.5, 0.05, nullptr, N, acc.data(), nullptr, threads);     // pot optional
        std::vector<int64_t> idx = {0, 5, N - 1};
        std::vector<double> a3(9), p3(3);
        oracle_forces(pos.data(), mass.data(), N, 1.5, 0.0, idx.data(), 3, a3.data(), p3.data(), threads);  // delta = 0
        oracle_forces_ld(pos.data(), mass.data(), N, 1.5, 0.05, idx.data(), 3, a3.data(), p3.data(), threads);
        std::vector<double> p = pos, v = vel, a(3 * N);
        if (oracle_kdk_paper(p.data(), v.data(), mass.data(), a.data(), N, 1e-3, 3, 1.0, 0.05, 0, threads) != 4) return 2;
        if (oracle_kdk_halfkick(p.data(), v.data(), mass.data(), a.data(), N, 1e-3, 2, 1.0, 0.05, 1, threads) != 2) return 3;
        oracle_invariants(p.data(), v.data(), mass.data(), nullptr, N, 1.0, 0.05, out.data(), threads);
        oracle_invariants(p.data(), v.data(), mass.data(), pot.data(), N, 1.0, 0.05, out.data(), threads);
    }
    const int64_t one = 1;                                      // N = 1: no pairs at all
    double r1[3] = {0, 0, 0}, m1[1] = {1.0}, a1[3], p1[1];
    oracle_forces(r1, m1, one, 1.0, 0.1, nullptr, one, a1, p1, 1);
    if (a1[0] != 0.0 || p1[0] != 0.0 || oracle_max_threads() < 1) return 4;
    std::puts("sanitized oracle ok");
    return 0;
}
"""


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    main = tmp_path / "driver.cpp"
    main.write_text(DRIVER)
    exe = tmp_path / "oracle_san"
    cmd = ["g++", "-O1", "-g", "-fno-omit-frame-pointer", "-ffp-contract=off", "-fopenmp",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
           os.path.join(ROOT, "oracle", "pp_oracle.cpp"), str(main), "-o", str(exe)]
    built = subprocess.run(cmd, capture_output=True, text=True)
    if built.returncode != 0 and ("asan" in built.stderr.lower() or "ubsan" in built.stderr.lower()):
        pytest.skip("no sanitizer runtime in this toolchain: " + built.stderr.strip().splitlines()[-1])
    assert built.returncode == 0, built.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", OMP_NUM_THREADS="3")
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=300)
    assert run.returncode == 0, run.stdout + run.stderr
    assert "sanitized oracle ok" in run.stdout
    assert "AddressSanitizer" not in run.stderr and "runtime error" not in run.stderr, run.stderr
