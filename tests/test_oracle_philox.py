"""Pins for the oracle's Philox4x32-10, keying and word->uniform maps (CPU only)."""
import os
import shutil
import subprocess
import tempfile

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _kat_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            w = [int(t, 16) for t in line.split()]
            rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, expect in rows:
        assert list(oracle.philox4x32_10(ctr, key)) == expect


def test_philox_bijection_and_avalanche():
    # a counter-mode block function must be injective in the counter for a fixed key, and flipping one
    # input bit must flip about half of the 128 output bits (catches a dropped round / wrong lane wiring)
    key = [0xDEADBEEF, 0x12345678]
    outs = set()
    base = np.array(oracle.philox4x32_10([5, 6, 7, 8], key), dtype=np.uint32)
    flips = []
    for word in range(4):
        for bit in range(32):
            ctr = [5, 6, 7, 8]
            ctr[word] ^= (1 << bit)
            o = np.array(oracle.philox4x32_10(ctr, key), dtype=np.uint32)
            outs.add(tuple(int(x) for x in o))
            flips.append(sum(bin(int(a) ^ int(b)).count("1") for a, b in zip(o, base)))
    assert len(outs) == 128
    assert 56 < np.mean(flips) < 72 and min(flips) > 30


def test_keyed_block_packing():
    # reading R7: key=(seed lo, seed hi); c0=lex, c1=sweep, c2=mu|p<<4|sg<<5|hit<<8|domain<<24, c3=draw
    seed = 0x0123456789ABCDEF
    for (lex, sweep, mu, p, sg, hit, dom, draw) in [(0, 0, 0, 0, 0, 0, 0, 0), (123456, 77, 3, 1, 2, 5, 0, 9),
                                                    (1048575, 4000000000, 2, 1, 0, 0, 1, 2)]:
        got = oracle.keyed_block(seed, lex, sweep, mu, p, sg, hit, dom, draw)
        c2 = mu | (p << 4) | (sg << 5) | (hit << 8) | (dom << 24)
        exp = oracle.philox4x32_10([lex, sweep, c2, draw], [seed & 0xFFFFFFFF, seed >> 32])
        assert list(got) == list(exp)
    # every field of the tuple must change the stream
    ref = tuple(oracle.keyed_block(seed, 10, 1, 1, 0, 1, 1, 0, 1))
    variants = [(11, 1, 1, 0, 1, 1, 0, 1), (10, 2, 1, 0, 1, 1, 0, 1), (10, 1, 2, 0, 1, 1, 0, 1), (10, 1, 1, 1, 1, 1, 0, 1),
                (10, 1, 1, 0, 2, 1, 0, 1), (10, 1, 1, 0, 1, 2, 0, 1), (10, 1, 1, 0, 1, 1, 1, 1), (10, 1, 1, 0, 1, 1, 0, 2)]
    for v in variants:
        assert tuple(oracle.keyed_block(seed, *v)) != ref
    assert tuple(oracle.keyed_block(seed + 1, 10, 1, 1, 0, 1, 1, 0, 1)) != ref


def test_word_to_uniform_maps():
    # reading R8: strictly inside (0,1); fp32 mode exactly representable in float
    for w in [0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFE, 0xFFFFFFFF]:
        u64 = oracle.word_to_uniform(w, 0)
        u32 = oracle.word_to_uniform(w, 1)
        assert 0.0 < u64 < 1.0 and 0.0 < u32 < 1.0
        assert u64 == (w + 0.5) / 2.0 ** 32
        assert u32 == ((w >> 9) + 0.5) / 2.0 ** 23
        assert float(np.float32(u32)) == u32
    assert oracle.word_to_uniform(0, 0) == 2.0 ** -33 and oracle.word_to_uniform(0xFFFFFFFF, 1) == 1.0 - 2.0 ** -24


def test_philox_uniformity():
    # words of consecutive counters are uniform: mean 1/2, variance 1/12, no lag-1 correlation (loose 5-sigma bounds)
    n = 20000
    u = np.array([[oracle.word_to_uniform(w, 0) for w in oracle.keyed_block(99, i, 0, 0, 0, 0, 0, 0, 0)] for i in range(n)])
    flat = u.ravel()
    assert abs(flat.mean() - 0.5) < 5 * np.sqrt(1 / 12 / flat.size)
    assert abs(flat.var() - 1 / 12) < 5 * np.sqrt(1 / 180 / flat.size)
    assert abs(np.corrcoef(flat[:-1], flat[1:])[0, 1]) < 5 / np.sqrt(flat.size)


_CURAND_HOST_SRC = r"""
#include <cstdio>
#include <cstdint>
#include <cstdlib>
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
int main(int argc, char** argv) {
  unsigned long long n = strtoull(argv[1], 0, 10);
  uint64_t s = 0x9E3779B97F4A7C15ull;
  for (unsigned long long i = 0; i < n; ++i) {
    uint32_t w[6];
    for (int k = 0; k < 6; ++k) { s ^= s << 13; s ^= s >> 7; s ^= s << 17; w[k] = (uint32_t)(s >> 16); }
    uint4 c; c.x = w[0]; c.y = w[1]; c.z = w[2]; c.w = w[3];
    uint2 k2; k2.x = w[4]; k2.y = w[5];
    uint4 o = curand_Philox4x32_10(c, k2);
    printf("%08x %08x %08x %08x %08x %08x %08x %08x %08x %08x\n", w[0], w[1], w[2], w[3], w[4], w[5], o.x, o.y, o.z, o.w);
  }
  return 0;
}
"""


def test_philox_against_curand_header_on_host():
    """Library cross-check: NVIDIA's own curand_Philox4x32_10 (CUDA toolkit header) compiled for the host."""
    inc = "/usr/local/cuda/include"
    if not os.path.exists(os.path.join(inc, "curand_philox4x32_x.h")) or shutil.which("g++") is None:
        pytest.skip("cuRAND header or g++ not available")
    with tempfile.TemporaryDirectory() as td:
        src = os.path.join(td, "kat.cpp")
        exe = os.path.join(td, "kat")
        with open(src, "w") as f:
            f.write(_CURAND_HOST_SRC)
        r = subprocess.run(["g++", "-O1", "-I", inc, "-D__CUDACC_RTC__=0", "-o", exe, src], capture_output=True, text=True)
        if r.returncode != 0:
            r = subprocess.run(["g++", "-O1", "-I", inc, "-o", exe, src], capture_output=True, text=True)
        if r.returncode != 0:
            pytest.skip("cuRAND header does not compile on the host here: " + r.stderr[-300:])
        out = subprocess.run([exe, "2000"], capture_output=True, text=True, check=True).stdout
    n = 0
    for line in out.splitlines():
        w = [int(t, 16) for t in line.split()]
        assert list(oracle.philox4x32_10(w[0:4], w[4:6])) == w[6:10]
        n += 1
    assert n == 2000
