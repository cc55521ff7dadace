"""The host oracle under AddressSanitizer and UndefinedBehaviorSanitizer ("sanitizers").

wcsim_oracle.c is compiled with -fsanitize=address,undefined into a scratch directory and a child interpreter (with the
sanitizer runtime preloaded) runs configs[0] and a 2,000-depo fluctuated configs[1] sample through every stage: raster +
scatter with per-depo totals, direct and FFT convolution, noise, drift, digitisation, the impact-position convolution.
Any out-of-bounds access, signed overflow, invalid shift or out-of-range float-to-integer conversion aborts the child.
The CUDA side has no such run: the GPU pool refuses compute-sanitizer.
"""
import os
import shutil
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = textwrap.dedent('''
    import sys
    import numpy as np
    import oracle
    oracle._LIB = sys.argv[1]                      # the instrumented build, not oracle/libwcoracle.so
    oracle.build = lambda force=False: oracle._LIB
    from paper_2203_02479_b200 import synth

    cfg = synth.config(0)
    pl = cfg["planes"][0]
    S, _, st = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], pl["depos"])
    M = oracle.convolve_fft(S, pl["response"], pl["pad_w"], pl["pad_t"])
    Md = oracle.convolve_direct(S, pl["response"])
    assert np.linalg.norm(M - Md) <= 1e-12 * np.linalg.norm(Md)
    oracle.digitize(M, 0.01, 900.0, 12)

    cfg = synth.config(1, n_depos=2000)
    pl = cfg["planes"][0]
    d = {k: v.copy() for k, v in pl["depos"].items()}
    d["q"][::7] *= -1.0
    d["sigma_t"][:3] = 0.0
    d["t0"][3], d["x0"][4] = -1.0, 799.9           # patches that leave the grid
    d["t0"][5] = np.nan                            # skipped
    for fl, norm in ((1, False), (2, False), (1, True)):
        S, tot, st = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=(1 << 63) + 5, fluctuate=fl, normalize=norm,
                                           id_base=(1 << 40) + 17, want_totals=True)
        assert st["skipped"] == 1 and tot.sum() == S.sum()
    Sw, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=3, fluctuate=1, window=(100, 200, 1000, 2000))
    M = oracle.convolve_fft(S, pl["response"], pl["pad_w"], pl["pad_t"])
    px, pt = np.array([0, 5, 799]), np.array([0, 3000, 5999])
    oracle.convolve_points(S, pl["response"], px, pt)
    oracle.noise_add(M, pl["pad_t"], 0xFFFFFFFFFFFFFFFF)
    oracle.noise_points(pl["pad_t"], 7, px, pt)
    K = 2
    Sf = np.zeros((16 * K, 64)); Sf[5, 7] = 1.0; Sf[31, 63] = 2.0
    oracle.convolve_impact(Sf, synth.response_impact(K, 5, 16), K)
    oracle.drift(np.array([10.0, -1.0]), np.zeros(2), np.zeros(2), np.zeros(2), np.array([5e3, 5e3]), v_drift=0.16, D_L=4.0,
                 D_T=8.8, tick=0.5, pitch=0.5)
    oracle.fft(np.arange(16) + 0j)
    print("sanitized oracle ok")
''')


@pytest.mark.skipif(shutil.which("gcc") is None, reason="gcc not on PATH")
def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    ubsan = subprocess.run(["gcc", "-print-file-name=libubsan.so"], capture_output=True, text=True).stdout.strip()
    if not (os.path.isabs(asan) and os.path.exists(asan) and os.path.isabs(ubsan) and os.path.exists(ubsan)):
        pytest.skip("this gcc ships no sanitizer runtimes")
    lib = str(tmp_path / "libwcoracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer",
                           "-o", lib, os.path.join(ROOT, "oracle", "wcsim_oracle.c"), "-lm"])
    env = dict(os.environ, LD_PRELOAD=asan + ":" + ubsan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", PYTHONPATH=ROOT, OMP_NUM_THREADS="4")
    r = subprocess.run([sys.executable, "-c", CHILD, lib], capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, "stdout:\n%s\nstderr:\n%s" % (r.stdout[-2000:], r.stderr[-6000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-6000:]
