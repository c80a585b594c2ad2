"""The two C oracles under AddressSanitizer + UndefinedBehaviorSanitizer (gcc), on small inputs that exercise every
entry point: clamped reads at all six faces, windows larger than the volume, rays that miss / graze / cross corners.
A memory error or undefined behaviour aborts the driver with a non-zero status (sanitizers on the
oracle).  The driver is plain C compiled together with the oracle sources; nothing here touches the CUDA path."""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

typedef struct { int32_t n_phase, nz, ny, nx, patch_radius, search_radius; double h, mu; } tnlm_ref_params;
typedef struct { int32_t n_view, nu, nv, nz, ny, nx; double du, dv, sid, sdd, voxel; } tnlmr_ref_geom;
int tnlm_ref_weights(const tnlm_ref_params *, const float *, double *);
int tnlm_ref_jacobi_step(const tnlm_ref_params *, const float *, const float *, const float *, float *);
int tnlm_ref_jacobi_step_at(const tnlm_ref_params *, const float *, const float *, const float *, int64_t, const int64_t *, float *);
int tnlm_ref_enhance(const tnlm_ref_params *, const float *, const float *, float *, int32_t);
int tnlmr_ref_project(const tnlmr_ref_geom *, const double *, const double *, double *);
int tnlmr_ref_backproject(const tnlmr_ref_geom *, const double *, const double *, double *);
int tnlmr_ref_cgls(const tnlmr_ref_geom *, const double *, const double *, double *, int32_t, double *);
int tnlmr_ref_ray(const tnlmr_ref_geom *, const double *, const double *, int64_t *, double *, int32_t);

static float frand(unsigned *s) { *s = *s * 1664525u + 1013904223u; return (float)(*s >> 8) / 16777216.0f; }

int main(void)
{
    unsigned seed = 7;
    int bad = 0;
    const int shapes[4][4] = {{2, 1, 1, 1}, {3, 2, 5, 4}, {2, 4, 3, 7}, {4, 3, 3, 3}};
    for (int c = 0; c < 4; ++c)
        for (int d = 0; d <= 2; ++d)
            for (int M = 0; M <= 3; M += (M == 0 ? 1 : 2)) {
                tnlm_ref_params p = {shapes[c][0], shapes[c][1], shapes[c][2], shapes[c][3], d, M, 0.3, 0.7};
                const size_t n = (size_t)p.n_phase * p.nz * p.ny * p.nx, e = (size_t)(2 * M + 1) * (2 * M + 1) * (2 * M + 1);
                float *f = malloc(n * 4), *g = malloc(n * 4), *r = malloc(n * 4), *o = malloc(n * 4);
                double *w = malloc(n * 2 * e * 8);
                int64_t idx[3] = {0, (int64_t)n / 2, (int64_t)n - 1};
                float o3[3];
                for (size_t i = 0; i < n; ++i) { f[i] = frand(&seed); g[i] = frand(&seed); r[i] = frand(&seed); }
                bad |= tnlm_ref_weights(&p, r, w);
                bad |= tnlm_ref_jacobi_step(&p, f, g, r, o);
                bad |= tnlm_ref_jacobi_step(&p, f, g, NULL, o);
                bad |= tnlm_ref_jacobi_step_at(&p, f, g, r, 3, idx, o3);
                bad |= tnlm_ref_enhance(&p, g, NULL, o, 2);
                bad |= tnlm_ref_enhance(&p, g, f, o, 0);
                for (size_t i = 0; i < n; ++i) bad |= !isfinite(o[i]);
                free(f); free(g); free(r); free(o); free(w);
            }
    const tnlmr_ref_geom geoms[3] = {{3, 7, 5, 4, 5, 6, 1.3, 1.7, 25.0, 41.0, 0.9}, {2, 1, 1, 1, 1, 1, 1.0, 1.0, 5.0, 9.0, 1.0},
                                     {2, 9, 1, 1, 6, 6, 0.7, 1.0, 12.0, 20.0, 1.0}};
    for (int c = 0; c < 3; ++c) {
        const tnlmr_ref_geom *g = &geoms[c];
        const size_t nv = (size_t)g->nz * g->ny * g->nx, nr = (size_t)g->n_view * g->nv * g->nu;
        double ang[3] = {0.0, 1.5707963267948966, 4.0};
        double *f = malloc(nv * 8), *y = malloc(nr * 8), *res = malloc(8 * 8);
        for (size_t i = 0; i < nv; ++i) f[i] = frand(&seed);
        bad |= tnlmr_ref_project(g, ang, f, y);
        bad |= tnlmr_ref_backproject(g, ang, y, f);
        bad |= tnlmr_ref_cgls(g, ang, y, f, 5, res);
        for (size_t i = 0; i < nv; ++i) bad |= !isfinite(f[i]);
        free(f); free(y); free(res);
    }
    {   /* single rays: through a corner, along a face, missing, starting inside */
        const tnlmr_ref_geom g = {1, 1, 1, 2, 3, 4, 1.0, 1.0, 10.0, 20.0, 1.0};
        int64_t vox[32];
        double len[32];
        const double rays[5][6] = {{-5, -5, -5, 5, 5, 5}, {-5, 1.5, 0, 5, 1.5, 0}, {-5, 9, 0, 5, 9, 0}, {0, 0, 0, 7, 0.3, 0.2}, {-5, 0, 1, 5, 0, 1}};
        for (int r = 0; r < 5; ++r) bad |= tnlmr_ref_ray(&g, rays[r], rays[r] + 3, vox, len, 32) < 0;
    }
    printf(bad ? "FAIL\n" : "OK\n");
    return bad;
}
"""


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_oracles_are_clean_under_asan_and_ubsan(tmp_path):
    drv = tmp_path / "driver.c"
    drv.write_text(DRIVER)
    exe = tmp_path / "oracle_san"
    cmd = ["gcc", "-std=c11", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer",
           "-fno-fast-math", "-ffp-contract=off", str(drv), os.path.join(ROOT, "oracle", "tnlm_oracle.c"),
           os.path.join(ROOT, "oracle", "tnlmr_oracle.c"), "-o", str(exe), "-lm"]
    build = subprocess.run(cmd, capture_output=True, text=True)
    if build.returncode != 0 and "sanitize" in build.stderr:
        pytest.skip("this gcc has no sanitizer runtime")
    assert build.returncode == 0, build.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="4")
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=600)
    assert run.returncode == 0 and run.stdout.strip() == "OK", run.stdout + run.stderr
