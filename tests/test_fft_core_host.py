"""The warp FFT core (csrc/fft_device.cuh) compiled for the CPU with one lane, against a direct DFT.

Covers every radix (2, 3, 4, 5, 8) and every padded size the configs use: P in {16, 32, 40, 64,
128, 160, 192, 256}, P_os in {16, 40, 48, 80, 160, 180, 240, 320}, plus odd mixes.
"""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SIZES = [2, 4, 6, 8, 10, 16, 30, 32, 40, 48, 64, 80, 90, 128, 150, 160, 180, 192, 240, 256, 320, 1000]


@pytest.fixture(scope="module")
def harness(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("fft") / "fft_host_harness")
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-I", os.path.join(ROOT, "paper_1806_07938_b200", "csrc"),
                           os.path.join(ROOT, "tests", "fft_host_harness.cpp"), "-o", exe])
    return exe


def test_fft_core_matches_direct_dft(harness):
    out = subprocess.check_output([harness] + [str(p) for p in SIZES], text=True)
    rows = [line.split() for line in out.strip().splitlines()]
    assert [int(r[0]) for r in rows] == SIZES
    for r in rows:
        f32f, f32i, f64f, f64i = map(float, r[1:])
        assert f32f < 5e-7 and f32i < 5e-7, r
        assert f64f < 5e-15 and f64i < 5e-15, r


def test_static_fft_chain_matches_direct_dft(harness):
    """warp_fft_static (compile-time plan used by the persistent kernel) for every instantiated size."""
    out = subprocess.check_output([harness, "S"], text=True)
    rows = [line.split() for line in out.strip().splitlines()]
    assert [int(r[1]) for r in rows] == [16, 20, 24, 32, 40, 48, 64, 80, 128, 160, 180, 192, 240, 256, 320]
    for r in rows:
        f32f, f32i, f64f, f64i = map(float, r[2:])
        assert f32f < 5e-7 and f32i < 5e-7, r
        assert f64f < 5e-15 and f64i < 5e-15, r


def test_register_two_pass_fft_matches_direct_dft(harness):
    """fft_reg.cuh: the two-pass register split P = A * B (both orders, forward and inverse) the persistent kernel runs."""
    out = subprocess.check_output([harness, "R"], text=True)
    rows = [line.split() for line in out.strip().splitlines()]
    assert [int(r[1]) for r in rows] == [16, 20, 24, 32, 40, 48, 64, 80, 128, 160, 180, 192, 240, 256, 320]
    for r in rows:
        v = list(map(float, r[2:]))
        for f32 in v[0:2] + v[4:6]:
            assert f32 < 5e-7, r
        for f64 in v[2:4] + v[6:8]:
            assert f64 < 5e-15, r
