"""Pins of the oracle's index sampler (Alg. 1 line 1: i.i.d. uniform with replacement), which the
on-device sampler of casgd_outer_steps_sampled must match bit for bit. CPU only.

* Philox4x32-10 against the published known-answer vectors (tests/golden/philox4x32_10_kat.txt);
* against a LIBRARY routine: cuRAND's own curand_Philox4x32_10 (its header is host-callable), compiled into a tiny host
  program with nvcc and run on random counters / keys -- an implementation this repo did not write;
* what the definition fixes: indices in [0, m), a step's indices independent of how many steps are drawn, different
  steps / seeds differ, the multiply-shift map written out with Python integers, uniformity (chi-square) and
  duplicates at the birthday rate (it is WITH replacement).
"""
import os
import subprocess
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _kat():
    rows = []
    for line in open(os.path.join(ROOT, "tests", "golden", "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_philox_matches_the_published_known_answers(oracle_mod):
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert [int(v) for v in oracle_mod.philox4x32_10(ctr, key)] == out


CURAND_HOST = r"""
#include <cstdio>
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>
int main(int argc, char **argv) {
    unsigned c0, c1, c2, c3, k0, k1;
    while (scanf("%x %x %x %x %x %x", &c0, &c1, &c2, &c3, &k0, &k1) == 6) {
        uint4 c = make_uint4(c0, c1, c2, c3);
        uint2 k = make_uint2(k0, k1);
        uint4 r = curand_Philox4x32_10(c, k);
        printf("%08x %08x %08x %08x\n", r.x, r.y, r.z, r.w);
    }
    return 0;
}
"""


def test_philox_matches_curands_own_routine(oracle_mod):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not found")
    rng = np.random.default_rng(7)
    ctr = rng.integers(0, 1 << 32, size=(64, 4), dtype=np.uint64)
    key = rng.integers(0, 1 << 32, size=(64, 2), dtype=np.uint64)
    ctr[0] = 0
    key[0] = 0
    ctr[1] = 0xFFFFFFFF
    with tempfile.TemporaryDirectory() as d:
        src, exe = os.path.join(d, "p.cu"), os.path.join(d, "p")
        open(src, "w").write(CURAND_HOST)
        subprocess.check_call([nvcc, "-O1", "-o", exe, src], stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        text = "\n".join(" ".join(f"{int(v):x}" for v in list(c) + list(k)) for c, k in zip(ctr, key))
        out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout.split()
    lib = np.array([int(t, 16) for t in out], dtype=np.uint32).reshape(64, 4)
    assert np.array_equal(oracle_mod.philox4x32_10(ctr, key), lib)


def test_sampler_definition_written_out(oracle_mod):
    seed, step, sb, m = 0x123456789ABCDEF, (1 << 33) + 5, 37, 5_000_000
    idx = oracle_mod.sample_indices(seed, step, sb, m)
    assert idx.dtype == np.int32 and idx.shape == (sb,)
    for t in (0, 1, 5, 36):
        w = oracle_mod.philox4x32_10([t // 4, step & 0xFFFFFFFF, step >> 32, 0xCA5D], [seed & 0xFFFFFFFF, seed >> 32])[t % 4]
        assert int(idx[t]) == (int(w) * m) >> 32


def test_sampler_is_counter_based_and_uniform_with_replacement(oracle_mod):
    m, sb = 8192, 4096
    a = oracle_mod.sample_indices(42, 7, sb, m)
    assert a.min() >= 0 and a.max() < m
    assert np.array_equal(a[:100], oracle_mod.sample_indices(42, 7, 100, m))       # position t does not depend on sb
    assert not np.array_equal(a, oracle_mod.sample_indices(42, 8, sb, m))          # other step
    assert not np.array_equal(a, oracle_mod.sample_indices(43, 7, sb, m))          # other seed
    # with replacement: sb draws from m values leave about m (1 - exp(-sb/m)) distinct ones
    distinct = len(np.unique(a))
    assert abs(distinct - m * (1 - np.exp(-sb / m))) < 4 * np.sqrt(sb)
    # uniform: chi-square over 64 equal bins of 200 steps' indices
    big = np.concatenate([oracle_mod.sample_indices(42, h, sb, m) for h in range(200)])
    counts = np.bincount(big // (m // 64), minlength=64).astype(np.float64)
    expect = big.size / 64
    chi2 = ((counts - expect) ** 2 / expect).sum()
    assert chi2 < 63 + 6 * np.sqrt(2 * 63)                                          # mean 63, sd sqrt(126)
