"""The oracle's C file under AddressSanitizer + UndefinedBehaviorSanitizer (row (c)): the file is
compiled with -fsanitize=address,undefined into a small driver that runs hand-worked pins (the P2 golden, a partial
tile, the spectrum, the harmonic sum, the interpolation and localisation) on exact inputs; any out-of-bounds access,
leak of the malloc'ed scratch or undefined arithmetic aborts the driver.  CPU only."""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = textwrap.dedent(r"""
    #include <math.h>
    #include <stdint.h>
    #include <stdio.h>
    #include <stdlib.h>
    double fitrig_oracle_global_max(const float* const*, int, int64_t, int64_t, double);
    int fitrig_oracle_tlisi(const float* const*, int, int, int, int, double, int, double, double*, double*, double*, int64_t*, double*, double*);
    int fitrig_oracle_tlisi_windows(const float* const*, int, int, int, int, int, double, int, double, double*, double*, double*, int64_t*, double*, double*);
    void fitrig_oracle_zscore(const double*, int, int64_t, double*, double*, double*);
    int64_t fitrig_oracle_select(const double*, const int64_t*, int, int64_t, int, double, int32_t*, int32_t*, int32_t*, int64_t*, double*, int64_t);
    void fitrig_oracle_spectrum_hsum(const double*, int, int64_t, int, double*, int32_t*, double*);
    int fitrig_oracle_interp_eval(const double*, int, int, int, const double*, const double*, int64_t, double*);
    int fitrig_oracle_localise(const double*, int, int, int, int, int, const int64_t*, int64_t, double*, double*, double*);
    #define CHECK(c) do { if (!(c)) { printf("FAILED %s line %d\n", #c, __LINE__); return 1; } } while (0)
    int main(void) {
      /* P2 (tests/golden/p2_handworked_2x2.json): q = 45/1024 */
      float x0[4] = {1, 2, 3, 4}, x1[4] = {2, 2, 1, 8}, x2[4] = {2, 5, 1, 4};
      const float* s[3] = {x0, x1, x2};
      double M = fitrig_oracle_global_max(s, 3, 2, 2, 1e-6), sd, md, sr, q, tl;
      int64_t arg;
      CHECK(M == 8.0);
      CHECK(fitrig_oracle_tlisi(s, 3, 2, 2, 2, 1e-6, 0, M, &sd, &md, &sr, &arg, &q, &tl) == 0);
      CHECK(sd == 6.0 && md == 3.0 && sr == 2.5 && arg == 1 && q == 45.0 / 1024.0 && tl == 1.0 - 45.0 / 1024.0);
      /* a 5 x 7 image, tiles of 3 (partial edge tiles), windows of 4 every 2, heap buffers sized exactly */
      enum { L = 4, H = 5, W = 7 };
      float* img[L];
      for (int k = 0; k < L; ++k) {
        img[k] = (float*)malloc(sizeof(float) * H * W);
        for (int i = 0; i < H * W; ++i) img[k][i] = (float)(((i * 7 + k * 13) % 11) - 5);
      }
      const float* ip[L] = {img[0], img[1], img[2], img[3]};
      const int Ty = 2, Tx = 3, U = 2, n = U * Ty * Tx;
      double *a = (double*)malloc(sizeof(double) * n), *b = (double*)malloc(sizeof(double) * n), *c = (double*)malloc(sizeof(double) * n);
      double *qq = (double*)malloc(sizeof(double) * n), *tt = (double*)malloc(sizeof(double) * n), *z = (double*)malloc(sizeof(double) * n);
      int64_t* am = (int64_t*)malloc(sizeof(int64_t) * n);
      for (int mode = 0; mode < 3; ++mode)
        CHECK(fitrig_oracle_tlisi(ip, L, H, W, 3, 1e-6, mode, 5.0, a, b, c, am, qq, tt) == 0);
      double mu[2], sg[2];
      fitrig_oracle_zscore(qq, U, Ty * Tx, mu, sg, z);
      int32_t ox[12], oy[12], ou[12];
      int64_t ot[12];
      double oz[12];
      CHECK(fitrig_oracle_select(z, am, U, Ty * Tx, W, -10.0, ox, oy, ou, ot, oz, 12) == 12);
      CHECK(fitrig_oracle_select(z, am, U, Ty * Tx, W, -10.0, ox, oy, ou, ot, oz, 5) == 12);
      {
        const int wy = 2, wx = 3, m = U * wy * wx;  /* n_windows(5,4,2) = 2, n_windows(7,4,2) = 3 */
        double *wa = (double*)malloc(sizeof(double) * m), *wq = (double*)malloc(sizeof(double) * m);
        int64_t* wam = (int64_t*)malloc(sizeof(int64_t) * m);
        CHECK(fitrig_oracle_tlisi_windows(ip, L, H, W, 4, 2, 1e-6, 0, 5.0, wa, NULL, NULL, wam, wq, NULL) == 0);
        free(wa); free(wq); free(wam);
      }
      /* spectrum with harmonic sums on a series of 9 units x 6 tiles */
      {
        enum { UU = 9, NT = 6 };
        double* ser = (double*)malloc(sizeof(double) * UU * NT);
        for (int i = 0; i < UU * NT; ++i) ser[i] = 1e-3 * (1.0 + sin(0.7 * i));
        double eta[NT], mag[(UU / 2) * NT];
        int32_t ks[NT];
        for (int Hh = 1; Hh <= 8; Hh *= 2) fitrig_oracle_spectrum_hsum(ser, UU, NT, Hh, eta, ks, mag);
        for (int t = 0; t < NT; ++t) CHECK(ks[t] >= 1 && ks[t] <= UU / 2 && eta[t] >= 0.0);
        free(ser);
      }
      /* interpolation and localisation on every grid shape class, all four schemes */
      {
        const int shapes[6][2] = {{1, 1}, {1, 4}, {2, 2}, {3, 3}, {4, 5}, {7, 6}};
        for (int sI = 0; sI < 6; ++sI) {
          const int ty = shapes[sI][0], tx = shapes[sI][1];
          double* e = (double*)malloc(sizeof(double) * ty * tx);
          for (int i = 0; i < ty * tx; ++i) e[i] = cos(1.3 * i) + 0.1 * i;
          int64_t* tl2 = (int64_t*)malloc(sizeof(int64_t) * ty * tx);
          for (int i = 0; i < ty * tx; ++i) tl2[i] = i;
          double *px = (double*)malloc(sizeof(double) * ty * tx), *py = (double*)malloc(sizeof(double) * ty * tx), *pv = (double*)malloc(sizeof(double) * ty * tx);
          for (int method = 0; method < 4; ++method) {
            CHECK(fitrig_oracle_localise(e, ty, tx, 4, method, 2, tl2, ty * tx, px, py, pv) == 0);
            double u = 0.5 * (tx - 1), v = 0.5 * (ty - 1), out;
            CHECK(fitrig_oracle_interp_eval(e, ty, tx, method, &u, &v, 1, &out) == 0);
            for (int i = 0; i < ty * tx; ++i) CHECK(pv[i] >= e[i] - 1e-12);  /* the tile centre is on the lattice */
          }
          free(e); free(tl2); free(px); free(py); free(pv);
        }
      }
      for (int k = 0; k < L; ++k) free(img[k]);
      free(a); free(b); free(c); free(qq); free(tt); free(z); free(am);
      printf("SANITIZED OK\n");
      return 0;
    }
""")


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    drv = tmp_path / "driver.c"
    drv.write_text(DRIVER)
    exe = tmp_path / "oracle_san"
    cmd = ["gcc", "-std=c99", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=undefined", "-o", str(exe), str(drv), os.path.join(ROOT, "oracle", "fitrig_oracle.c"), "-lm"]
    built = subprocess.run(cmd, capture_output=True, text=True)
    if built.returncode != 0 and "asan" in (built.stderr or "").lower():
        pytest.skip("this gcc has no libasan")
    assert built.returncode == 0, built.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=120)
    assert run.returncode == 0, run.stdout + run.stderr
    assert "SANITIZED OK" in run.stdout and "runtime error" not in run.stderr and "AddressSanitizer" not in run.stderr
