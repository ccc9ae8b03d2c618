"""AddressSanitizer / UndefinedBehaviorSanitizer run of the oracle (auxiliary subsystems): the oracle's
source is compiled together with a small C++ driver under -fsanitize=address,undefined and stepped on a ragged grid with
mixed boundaries, viscous, with the 8(f)-3 extension on; any out-of-bounds index, use of an uninitialised vector or signed
overflow aborts the run.  CPU only; skipped when the toolchain has no sanitizer runtime."""
import os
import subprocess
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
#include <cmath>
#include <cstdio>
#include <vector>
extern "C" {
void* oracle_create(int, int, int, double, double, double, const int*, int, double, double, int, int, double, double,
                    const double*, const double*, double, double, double, double, double, double, int);
void oracle_destroy(void*);
int oracle_set_option(void*, int, double);
int oracle_load_ext(void*, const double*, const double*, const double*, const double*);
int oracle_step(void*, int);
int oracle_read(void*, double*, double*, double*);
int oracle_read_ext(void*, double*, double*);
int oracle_diag(void*, double*);
}
int main() {
  const int nx = 13, ny = 7, nz = 5, N = nx * ny * nz;
  const int bc[3] = {0, 1, 0};
  for (int ext = 0; ext < 2; ++ext) {
    void* o = oracle_create(nx, ny, nz, 0.2, 0.2, 0.2, bc, 0, 0.02, 0.6, 0, 0, 0.0, 0.0, nullptr, nullptr,
                            47.5 * M_PI * M_PI / 30.0, 0.12, 1.1, 1e-7, 1.0, 0.999, 0);
    if (!o) return 2;
    if (ext) { if (oracle_set_option(o, 3, 1.0) || oracle_set_option(o, 4, 0.03)) return 3; }
    std::vector<double> T(4 * N, 0.0), Pi(N), nb(N);
    for (int c = 0; c < N; ++c) {
      const int i = c % nx, j = (c / nx) % ny, k = c / (nx * ny);
      T[c] = 1e-6 + 20.0 * std::exp(-0.1 * ((i - 6) * (i - 6) + (j - 3) * (j - 3)) - 0.3 * (k - 2) * (k - 2));
      T[N + c] = 0.3 * T[c] * std::sin(0.7 * i);
      Pi[c] = -0.02 * T[c]; nb[c] = 0.1 * T[c];
    }
    if (oracle_load_ext(o, T.data(), nullptr, ext ? Pi.data() : nullptr, ext ? nb.data() : nullptr)) return 4;
    if (oracle_step(o, 3)) return 5;
    std::vector<double> e(N), u(4 * N), pi(10 * N), d(9);
    oracle_read(o, e.data(), u.data(), pi.data());
    oracle_read_ext(o, Pi.data(), nb.data());
    oracle_diag(o, d.data());
    double s = 0;
    for (int c = 0; c < N; ++c) s += e[c] + u[c] + pi[9 * N + c] + Pi[c] + nb[c];
    if (!(s == s)) return 6;
    std::printf("ext=%d step=%g checksum=%.6e\n", ext, d[1], s);
    oracle_destroy(o);
  }
  return 0;
}
"""


def test_oracle_under_asan_ubsan():
    src = os.path.join(ROOT, "oracle", "clvisc_oracle.cpp")
    with tempfile.TemporaryDirectory() as tmp:
        drv, exe = os.path.join(tmp, "driver.cpp"), os.path.join(tmp, "oracle_san")
        with open(drv, "w") as f:
            f.write(DRIVER)
        cmd = ["g++", "-O1", "-g", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fsanitize=address,undefined",
               "-fno-sanitize-recover=all", "-o", exe, src, drv]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            pytest.skip("no sanitizer runtime in this toolchain: " + res.stderr[-300:])
        env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", OMP_NUM_THREADS="2")
        run = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=300)
        print(run.stdout, run.stderr[-2000:])
        assert run.returncode == 0, run.stderr[-2000:]
        assert "ext=0 step=3" in run.stdout and "ext=1 step=3" in run.stdout
