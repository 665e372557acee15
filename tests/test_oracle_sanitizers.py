"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY section 4's sanitizer row, CPU side): a
stand-alone driver compiled together with oracle/oracle.cpp takes subcycled and uniform steps of a three-level
hierarchy with two sibling boxes and two coupled fields under every option (dissipation of both orders, 8th-order
differences at g = 5, RK3 / RK2, radiative boundary, 9-/10-point interpolation, vertex-centred grids); any
out-of-bounds ghost access, overflow or misaligned read aborts the run. (compute-sanitizer on the CUDA side is closed
on this GPU pool: DESIGN.md section 4.)"""
import os
import shutil
import subprocess

import pytest

DRIVER = r"""
#include "oracle.cpp"
#include <cstdlib>
static int run(int ghost, int fd, int ko, double sigma, int integ, int bc, int interp, int vertex) {
  const int lev[4] = {0, 1, 2, 2};
  const int lo[12] = {0, 0, 0, 16, 16, 16, 48, 48, 48, 56, 48, 48};   // level 2: two abutting boxes
  const int n[12] = {32, 32, 32, 32, 32, 32, 8, 16, 16, 8, 16, 16};
  const int dom[3] = {32, 32, 32};
  const double xlo[3] = {-1.0, -0.8, -0.9}, xhi[3] = {1.0, 0.8, 0.9};
  const double A[4] = {-0.3, 0.1, 0.1, -0.25};
  void* h = oc_create(3, 4, lev, lo, n, ghost, 2, dom, xlo, xhi, A);
  if (!h) { fprintf(stderr, "create: %s\n", oc_last_error()); return 1; }
  if (fd == 8 && oc_set_fd_order(h, 8)) return 2;
  if (oc_set_options(h, integ, bc, ko, interp, vertex)) { fprintf(stderr, "options: %s\n", oc_last_error()); return 3; }
  if (sigma > 0 && oc_set_dissipation(h, sigma)) return 4;
  for (int b = 0; b < 4; ++b) {
    const int level = lev[b], box = b < 2 ? 0 : b - 2;
    std::vector<double> v(size_t(n[3 * b]) * n[3 * b + 1] * n[3 * b + 2]);
    for (int c = 0; c < 4; ++c) {
      for (size_t q = 0; q < v.size(); ++q) v[q] = std::sin(0.001 * double(q) + c) * (c < 2 ? 1.0 : 0.1);
      if (oc_set_state(h, level, box, c, v.data())) return 5;
    }
  }
  if (oc_step(h, 0.01, 1) || oc_step(h, 0.01, 0)) return 6;
  std::vector<int> map(7 * 20000);
  if (oc_ghost_map(h, 2, 1, map.data(), map.size()) <= 0) return 7;
  std::vector<double> out(size_t(n[3] + 2 * ghost) * (n[4] + 2 * ghost) * (n[5] + 2 * ghost));
  if (oc_read(h, 1, 0, 0, 3, 1, out.data())) return 8;
  for (double x : out) if (!(x == x)) return 9;
  oc_destroy(h);
  return 0;
}
int main() {
  int rc = 0;
  rc |= run(3, 4, 5, 0.2, 4, 0, 0, 0);
  rc |= run(5, 8, 9, 0.2, 3, 1, 1, 0);
  rc |= run(4, 8, 5, 0.2, 2, 0, 0, 1);
  rc |= run(2, 4, 0, 0.0, 2, 1, 0, 0);
  printf("sanitizer driver rc=%d\n", rc);
  return rc;
}
"""


@pytest.mark.slow
def test_oracle_clean_under_asan_and_ubsan(tmp_path):
    gxx = shutil.which("g++")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = tmp_path / "driver.cpp"
    src.write_text(DRIVER)
    exe = tmp_path / "driver"
    cmd = [gxx, "-std=c++17", "-O2", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=undefined", "-fopenmp", "-I", os.path.join(root, "oracle"), "-o", str(exe), str(src)]
    b = subprocess.run(cmd, capture_output=True, text=True)
    if b.returncode != 0 and ("asan" in b.stderr or "ubsan" in b.stderr or "sanitize" in b.stderr):
        pytest.skip("sanitizer runtimes not installed: " + b.stderr.strip().splitlines()[-1])
    assert b.returncode == 0, b.stderr[-2000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:halt_on_error=1", OMP_NUM_THREADS="4")
    r = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=900)
    assert r.returncode == 0, (r.stdout[-500:], r.stderr[-3000:])
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-3000:]
    assert "sanitizer driver rc=0" in r.stdout
