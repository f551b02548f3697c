"""the oracle built once with -fsanitize=address,undefined and driven through every entry
point on a tiny tilted cone-beam problem (flat and arc detector, all four voxel models, clipped footprints).
A plain C driver includes oracle/sf_oracle.c, so no sanitizer runtime has to be preloaded into Python.  CPU only."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r'''
#include "%(src)s"
#include <stdio.h>
int main(void)
{
    enum { NV = 5, NX = 7, NY = 6, NZ = 5, NU = 9, NVV = 8 };
    double src[NV*3], dc[NV*3], du[NV*3], dv[NV*3];
    for (int i = 0; i < NV; ++i) {
        double th = 6.283185307179586 * i / NV + 0.1, ph = 0.2 * sin(2.0 * th);
        double c = cos(th), s = sin(th), cp = cos(ph), sp = sin(ph);
        /* Rz(th) Rx(ph) applied to (0, 60, 0), (0, -60, 0), ex, ez */
        src[3*i] = -s*cp*60.0; src[3*i+1] = c*cp*60.0; src[3*i+2] = sp*60.0;
        dc[3*i] = s*cp*60.0 + 0.7; dc[3*i+1] = -c*cp*60.0; dc[3*i+2] = -sp*60.0 + 0.3;
        du[3*i] = c; du[3*i+1] = s; du[3*i+2] = 0.0;
        dv[3*i] = s*sp; dv[3*i+1] = -c*sp; dv[3*i+2] = cp;
    }
    double vol[NZ*NY*NX], proj[NV*NVV*NU], out[NZ*NY*NX], q[NV*NVV*NU], F1[NU], F2[NVV], amp, tau[4], st[2];
    int views[NV], rng[4], ijk[6] = {0, 0, 0, NX-1, NY-1, NZ-1};
    float projf[NV*NVV*NU];
    for (int i = 0; i < NV; ++i) views[i] = i;
    for (int i = 0; i < NZ*NY*NX; ++i) vol[i] = 1.0 + 0.01 * i;
    double total = 0.0;
    for (int det = 0; det < 2; ++det)
        for (int model = 0; model < 4; ++model) {
            /* arc detectors need (D - S).u == 0: drop the lateral shift */
            if (det == 1) for (int i = 0; i < NV; ++i) dc[3*i] -= 0.7 * (i == i);
            sfo_geom g = { 3, NX, NY, NZ, 2.0, 2.0, 2.5, 0.5, -0.4, 0.3, NU, NVV, 3.0, 3.5, det, NV, src, dc, du, dv, model };
            if (det == 1) {          /* re-centre exactly: D = S + R n with n = u x v */
                for (int i = 0; i < NV; ++i) {
                    double n[3] = { du[3*i+1]*dv[3*i+2] - du[3*i+2]*dv[3*i+1], du[3*i+2]*dv[3*i] - du[3*i]*dv[3*i+2],
                                    du[3*i]*dv[3*i+1] - du[3*i+1]*dv[3*i] };
                    double sgn = (n[0]*(dc[3*i]-src[3*i]) + n[1]*(dc[3*i+1]-src[3*i+1]) + n[2]*(dc[3*i+2]-src[3*i+2])) < 0 ? -1.0 : 1.0;
                    for (int c = 0; c < 3; ++c) dc[3*i+c] = src[3*i+c] + sgn * 120.0 * n[c];
                }
            }
            sfo_fp(&g, vol, views, NV, proj);
            sfo_bp(&g, proj, views, NV, out);
            sfo_fbp_filter(&g, proj, views, NV, q);
            sfo_bp_recon(&g, q, views, NV, out);
            sfo_bp_voxels(&g, proj, ijk, 2, out);
            for (int i = 0; i < NV*NVV*NU; ++i) projf[i] = (float)proj[i];
            sfo_bp_voxels_f32(&g, projf, ijk, 2, out);
            sfo_footprint(&g, 1, 3, 2, 2, rng, F1, F2, &amp, tau);
            sfo_footprint(&g, 2, 0, 0, 0, rng, F1, F2, &amp, tau);
            double P[3] = {1.0, 2.0, 3.0};
            sfo_det_coords(&g, 0, P, st);
            total += sfo_live_fraction(&g, 2, 1) + proj[7] + out[0];
        }
    /* 2-D */
    {
        sfo_geom g = { 2, NX, NY, 1, 2.0, 2.0, 1.0, 0.0, 0.0, 0.0, NU, 1, 3.0, 1.0, 0, NV, src, dc, du, dv, 0 };
        for (int i = 0; i < NV; ++i) {
            double th = 6.283185307179586 * i / NV;
            src[3*i] = -sin(th)*60.0; src[3*i+1] = cos(th)*60.0; src[3*i+2] = 0.0;
            dc[3*i] = sin(th)*60.0; dc[3*i+1] = -cos(th)*60.0; dc[3*i+2] = 0.0;
            du[3*i] = cos(th); du[3*i+1] = sin(th); du[3*i+2] = 0.0;
        }
        sfo_fp(&g, vol, views, NV, proj);
        sfo_bp(&g, proj, views, NV, out);
        sfo_fbp_filter(&g, proj, views, NV, q);
        sfo_bp_recon(&g, q, views, NV, out);
        total += out[3];
    }
    double tv[4] = {0.0, 0.0, 1.0, 1.0};
    total += sfo_trap_cdf(tv, 0.5) + sfo_num_threads();
    printf("ok %%g\n", total);
    return 0;
}
'''


def test_oracle_is_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    main_c = tmp_path / "drive.c"
    main_c.write_text(DRIVER % {"src": os.path.join(ROOT, "oracle", "sf_oracle.c")})
    exe = tmp_path / "drive"
    cmd = ["gcc", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-o", str(exe), str(main_c), "-lm"]
    build = subprocess.run(cmd, capture_output=True, text=True)
    if build.returncode != 0 and ("asan" in build.stderr.lower() or "sanitize" in build.stderr.lower()):
        pytest.skip("sanitizer runtime not installed: " + build.stderr[-200:])
    assert build.returncode == 0, build.stderr[-2000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", OMP_NUM_THREADS="3")
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=300)
    assert run.returncode == 0 and run.stdout.startswith("ok"), (run.stdout[-500:], run.stderr[-3000:])
    assert "runtime error" not in run.stderr and "AddressSanitizer" not in run.stderr, run.stderr[-3000:]
