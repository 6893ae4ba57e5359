"""Pins P1, P2: the oracle's Philox-4x32-10 and uniform conversion against
things other than itself: published known-answer vectors, the C++26 requirement, the CUDA toolkit's
own curand Philox header (a library routine, compiled for the host here), and closed-form moments."""
import ctypes as C
import json
import os
import subprocess

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
GOLDEN = os.path.join(HERE, "golden")


def _kat_rows():
    rows = []
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            lhs, rhs = line.split("->")
            w = [int(x, 16) for x in lhs.split()]
            out = [None if x == "-" else int(x, 16) for x in rhs.split()]
            rows.append((w[:4], w[4:6], out))
    return rows


def test_known_answer_vectors():
    rows = _kat_rows()
    assert len(rows) == 4
    for ctr, key, want in rows:
        got = oracle.philox4x32_10(ctr, key)
        for g, w in zip(got, want):
            if w is not None:
                assert int(g) == w, (ctr, key, [hex(int(x)) for x in got])


def test_cxx26_10000th_value():
    # default seed 20111115; 10000th 32-bit output = word 3 of block 2499
    out = oracle.philox4x32_10([2499, 0, 0, 0], [20111115, 0])
    assert int(out[3]) == 1955073260


CURAND_HDR = "/usr/local/cuda/include/curand_philox4x32_x.h"


@pytest.mark.skipif(not os.path.exists(CURAND_HDR), reason="CUDA toolkit header not present")
def test_against_curand_header(tmp_path):
    """2e5 random (counter, key) pairs against curand_Philox4x32_10 from the toolkit header."""
    src = tmp_path / "ref.cpp"
    src.write_text(
        "#include <cstdint>\n#include <vector_types.h>\n#define QUALIFIERS static inline\n"
        "#include <curand_philox4x32_x.h>\n"
        'extern "C" void ref(const uint32_t* c, const uint32_t* k, uint32_t* o, long n) {\n'
        "  for (long i = 0; i < n; ++i) { uint4 cc = {c[4*i], c[4*i+1], c[4*i+2], c[4*i+3]};\n"
        "    uint2 kk = {k[2*i], k[2*i+1]}; uint4 r = curand_Philox4x32_10(cc, kk);\n"
        "    o[4*i] = r.x; o[4*i+1] = r.y; o[4*i+2] = r.z; o[4*i+3] = r.w; } }\n")
    so = tmp_path / "libref.so"
    subprocess.run(["g++", "-O2", "-shared", "-fPIC", "-I/usr/local/cuda/include", str(src), "-o", str(so)],
                   check=True)
    lib = C.CDLL(str(so))
    n = 200_000
    rng = np.random.default_rng(7)
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    want = np.zeros((n, 4), np.uint32)
    lib.ref(ctr.ctypes.data_as(C.c_void_p), key.ctypes.data_as(C.c_void_p),
            want.ctypes.data_as(C.c_void_p), C.c_long(n))
    step = 97  # every 97th pair through the (slow) per-call ctypes path
    for i in range(0, n, step):
        got = oracle.philox4x32_10(ctr[i], key[i])
        assert np.array_equal(got, want[i]), i


def test_layout_anchors_from_survey():
    """R1-R3: ctr = {lo(i), hi(i), lo(step), hi(step)}, key = {lo(seed), hi(seed)}, key = w0,
    u = ((w3:w2) >> 11) 2^-53 -- against values an independent implementation printed."""
    g = json.load(open(os.path.join(GOLDEN, "survey_p12_vectors.json")))
    seed = g["seed"]
    for a in g["layout_anchors"]:
        i, step = a["i"], a["step"]
        w = oracle.philox4x32_10([i & 0xFFFFFFFF, i >> 32, step & 0xFFFFFFFF, step >> 32],
                                 [seed & 0xFFFFFFFF, seed >> 32])
        assert [f"{int(x):08x}" for x in w] == a["words"]
        key, u = oracle.sd_random(seed, step, i)
        assert key == a["key"]
        assert u == float.fromhex(a["u_hex"])


def test_uniform_conversion_extremes():
    assert oracle.uniform_from_words(0, 0) == 0.0
    assert oracle.uniform_from_words(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    # the low 11 bits of w2 are discarded
    assert oracle.uniform_from_words(0x7FF, 0) == 0.0
    assert oracle.uniform_from_words(0x800, 0) == 2.0 ** -53
    assert oracle.uniform_from_words(0, 0x80000000) == 0.5


def test_uniform_and_key_moments():
    n = 200_000
    us = np.empty(n)
    ks = np.empty(n)
    for i in range(n):
        k, u = oracle.sd_random(42, 3, i)
        us[i] = u
        ks[i] = k
    assert 0.0 <= us.min() and us.max() < 1.0
    # mean 1/2 (sigma 1/sqrt(12 n)), variance 1/12
    assert abs(us.mean() - 0.5) < 5 * (1 / np.sqrt(12 * n))
    assert abs(us.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / n)
    kn = ks / 2.0 ** 32
    assert abs(kn.mean() - 0.5) < 5 * (1 / np.sqrt(12 * n))
    # key and uniform of the same SD come from different words: uncorrelated
    assert abs(np.corrcoef(us, kn)[0, 1]) < 5 / np.sqrt(n)
    # all four byte digits of the key are uniform over 256 bins (chi-square, 255 dof: mean 255, sd 22.6)
    ki = ks.astype(np.uint64)
    for shift in (0, 8, 16, 24):
        h = np.bincount(((ki >> shift) & 0xFF).astype(np.int64), minlength=256)
        chi2 = ((h - n / 256) ** 2 / (n / 256)).sum()
        assert chi2 < 255 + 6 * 22.6
