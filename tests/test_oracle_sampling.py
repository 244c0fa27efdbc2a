"""Pins for the oracle's sampler O6-O8: Philox4x32-10, the uniform map, greedy, top-k,
and Gumbel-max == softmax sampling (chi-square bound on brute-force enumeration)."""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest
from scipy import stats

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def curand_host(tmp_path_factory):
    """CUDA toolkit's curand_Philox4x32_10 compiled for the HOST (library cross-check)."""
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    out = str(tmp_path_factory.mktemp("curand") / "libcurand_philox_host.so")
    subprocess.run(["nvcc", "-O1", "-shared", "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets",
                    "-o", out, os.path.join(HERE, "helpers", "curand_philox_host.cu")], check=True)
    return C.CDLL(out)


def test_philox_vs_curand_host(curand_host):
    rng = np.random.default_rng(11)
    ctrs = rng.integers(0, 2 ** 32, size=(20000, 4), dtype=np.uint64).astype(np.uint32)
    keys = rng.integers(0, 2 ** 32, size=(20000, 2), dtype=np.uint64).astype(np.uint32)
    # corner counters / keys too
    ctrs[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [1, 0, 0, 0], [0, 0, 0, 1]]
    keys[:4] = [[0, 0], [0xFFFFFFFF] * 2, [0, 1], [1, 0]]
    out = np.empty(4, dtype=np.uint32)
    for c, k in zip(ctrs, keys):
        c = np.ascontiguousarray(c)
        k = np.ascontiguousarray(k)
        curand_host.curand_philox_host(c.ctypes.data_as(C.c_void_p), k.ctypes.data_as(C.c_void_p),
                                       out.ctypes.data_as(C.c_void_p))
        assert np.array_equal(oracle.philox4x32_10(c, k), out)


def test_philox_is_a_bijection_in_one_counter_word():
    # for a fixed key Philox is a permutation of counters: distinct counters -> distinct blocks
    seen = set()
    for c0 in range(4096):
        seen.add(tuple(oracle.philox4x32_10([c0, 5, 2, 9], [123, 456]).tolist()))
    assert len(seen) == 4096


def test_uniform_map_is_exact_and_open():
    # p = ((x >> 9) + 0.5) * 2^-23: smallest, largest, fp32-exact
    assert oracle.uniform(0) == 2.0 ** -24
    assert oracle.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert oracle.uniform(0x1FF) == 2.0 ** -24 and oracle.uniform(0x200) == 1.5 * 2.0 ** -23
    for x in (0, 1 << 9, 0x80000000, 0xFFFFFFFF, 0x12345678):
        p = oracle.uniform(x)
        assert 0.0 < p < 1.0 and float(np.float32(p)) == p


def test_uniform_and_gumbel_statistics():
    # 2^18 draws through the keyed path (seed, req, tau, stream, token): mean/variance of the
    # standard Gumbel are Euler-gamma and pi^2/6; KS test against the Gumbel CDF
    g = np.array([oracle.gumbel(7, q, tau, 1, v) for q in range(64) for tau in range(64) for v in range(64)])
    assert abs(g.mean() - 0.5772156649) < 0.01
    assert abs(g.var() - np.pi ** 2 / 6) < 0.03
    ks = stats.kstest(g, lambda x: np.exp(-np.exp(-x)))
    assert ks.pvalue > 1e-4
    # the four words of one block serve tokens 4b..4b+3 and differ
    blk = [oracle.gumbel(7, 0, 0, 0, v) for v in range(4)]
    assert len(set(blk)) == 4


def test_gumbel_closed_form_values():
    # g(p) = -ln(-ln(1-p)):  p = 1 - 1/e -> 0 ;  p = 1 - exp(-e) -> -1
    assert abs(oracle.lib().oracle_gumbel_from_uniform(1 - np.exp(-1.0))) < 1e-15
    assert abs(oracle.lib().oracle_gumbel_from_uniform(1 - np.exp(-np.e)) + 1.0) < 1e-15
    # small p <-> large g (the winner-relevant tail): g ~ -ln p
    assert abs(oracle.lib().oracle_gumbel_from_uniform(2.0 ** -24) - 24 * np.log(2)) < 1e-6


def test_greedy_equals_numpy_argmax():
    rng = np.random.default_rng(2)
    for trial in range(200):
        M = rng.normal(size=rng.integers(1, 70))
        if trial % 5 == 0 and M.size > 3:           # exact ties: lowest index wins
            M[rng.integers(0, M.size, 3)] = M.max()
        for temp, k in ((0.0, 20), (0.7, 1), (0.0, 1)):
            tok, margin, flags, _ = oracle.sample_cell(M, temp, k, seed=1, req_id=3, tau=4, stream=0)
            assert tok == int(np.argmax(M)) and flags & oracle.FLAG_GREEDY
            srt = np.sort(M)[::-1]
            assert margin == (srt[0] - srt[1] if M.size > 1 else np.inf)


def test_low_temperature_limit_equals_argmax():
    # north_star: greedy sampling (temp -> 0) must equal argmax; through O7-O8 at temp = 1e-4
    rng = np.random.default_rng(3)
    n = 0
    for _ in range(300):
        M = rng.normal(size=64)
        srt = np.sort(M)[::-1]
        if srt[0] - srt[1] <= 4e-3:
            continue
        tok, *_ = oracle.sample_cell(M, 1e-4, 0, seed=9, req_id=1, tau=2, stream=3)
        assert tok == int(np.argmax(M))
        n += 1
    assert n > 200


def _brute_keep(z, k):
    V = z.size
    kk = V if (k <= 0 or k >= V) else k
    thr = np.sort(z)[::-1][kk - 1]
    return z >= thr, thr


def test_topk_brute_force_small_vocab():
    rng = np.random.default_rng(4)
    for trial in range(400):
        V = int(rng.integers(2, 17))
        M = np.round(rng.normal(size=V), 1) if trial % 3 == 0 else rng.normal(size=V)   # with ties
        temp = float(np.float32(rng.uniform(0.5, 1.5)))
        k = int(rng.integers(-1, V + 3))
        if k == 1:
            continue
        seed, q, tau, i = int(rng.integers(1 << 40)), int(rng.integers(1000)), int(rng.integers(100)), int(rng.integers(8))
        tok, margin, flags, thr = oracle.sample_cell(M, temp, k, seed, q, tau, i)
        z = M / np.float64(temp)
        keep, thr_ref = _brute_keep(z, k)
        assert thr == thr_ref and keep[tok]
        kk = V if (k <= 0 or k >= V) else k
        assert keep.sum() >= kk                                     # threshold semantics (C9)
        # independent restatement of O8 on the brute-force keep set
        s = np.array([z[v] + oracle.gumbel(seed, q, tau, i, v) if keep[v] else -np.inf for v in range(V)])
        assert tok == int(np.argmax(s))
        if keep.sum() > 1:
            srt = np.sort(s[keep])[::-1]
            assert abs(margin - (srt[0] - srt[1])) < 1e-12


def test_topk_k_ge_V_is_no_filter_and_k1_is_greedy():
    rng = np.random.default_rng(5)
    M = rng.normal(size=32)
    base = oracle.sample_cell(M, 0.9, 0, 5, 6, 7, 1)[0]
    for k in (-3, 0, 32, 33, 1000):
        assert oracle.sample_cell(M, 0.9, k, 5, 6, 7, 1)[0] == base
    assert oracle.sample_cell(M, 0.9, 1, 5, 6, 7, 1)[0] == int(np.argmax(M))


@pytest.mark.parametrize("V,k,temp", [(4, 0, 1.0), (8, 0, 0.7), (16, 0, 1.3), (16, 5, 0.8), (8, 3, 1.0)])
def test_gumbel_max_matches_softmax_chi_square(V, k, temp):
    """Brute-force enumeration on tiny vocabularies: N = 2^20 draws by sweeping (req_id, tau).
    Stated bound: Pearson chi-square <= chi2.ppf(1 - 1e-6, dof = |keep| - 1); outside keep the
    count must be exactly zero.  Deterministic given the seed."""
    rng = np.random.default_rng(100 + V + k)
    M = rng.normal(size=V) * 1.5
    counts = oracle.sample_sweep(M, temp, k, seed=2024, n_req=1024, n_tau=1024, stream=2)
    N = counts.sum()
    assert N == 1 << 20
    z = M / np.float64(np.float32(temp))
    keep, _ = _brute_keep(z, k)
    assert counts[~keep].sum() == 0
    p = np.exp(z[keep] - z[keep].max())
    p /= p.sum()
    chi2 = float((((counts[keep] - N * p) ** 2) / (N * p)).sum())
    bound = stats.chi2.ppf(1 - 1e-6, df=int(keep.sum()) - 1)
    assert chi2 <= bound, (chi2, bound)


def test_chi_square_detects_a_wrong_sampler():
    # sanity of the pin itself: ignoring the temperature must blow the bound
    rng = np.random.default_rng(104)
    M = rng.normal(size=8) * 1.5
    counts = oracle.sample_sweep(M, 0.7, 0, seed=2024, n_req=512, n_tau=512, stream=2)
    N = counts.sum()
    p = np.exp(M - M.max())
    p /= p.sum()
    chi2 = float((((counts - N * p) ** 2) / (N * p)).sum())
    assert chi2 > 10 * stats.chi2.ppf(1 - 1e-6, df=7)


def test_noise_keys_are_all_used():
    # (seed, request, step, stream, token) each change the draw
    base = oracle.gumbel(1, 2, 3, 4, 5)
    assert base != oracle.gumbel(2, 2, 3, 4, 5)
    assert base != oracle.gumbel(1 + (1 << 32), 2, 3, 4, 5)      # high half of the seed
    assert base != oracle.gumbel(1, 3, 3, 4, 5)
    assert base != oracle.gumbel(1, 2, 4, 4, 5)
    assert base != oracle.gumbel(1, 2, 3, 5, 5)
    assert base != oracle.gumbel(1, 2, 3, 4, 6)
    assert base != oracle.gumbel(1, 2, 3, 4, 9)


def test_close_and_boundary_flags():
    # two survivors with nearly equal perturbed scores -> CLOSE
    M = np.array([0.0, 0.0, -50.0, -50.0])
    g0, g1 = oracle.gumbel(1, 0, 0, 0, 0), oracle.gumbel(1, 0, 0, 0, 1)
    M2 = M.copy()
    M2[1] = g0 - g1 + 1e-3          # s1 = s0 + 1e-3
    tok, margin, flags, _ = oracle.sample_cell(M2, 1.0, 2, 1, 0, 0, 0)
    assert tok == 1 and abs(margin - 1e-3) < 1e-9 and flags & oracle.FLAG_CLOSE
    # an outsider just below the threshold that would win if admitted -> BOUNDARY
    M3 = np.array([5.0, 5.0 - 1e-3, -50.0, -50.0])
    hits = 0
    for tau in range(200):
        tok, margin, flags, _ = oracle.sample_cell(M3, 1.0, 1 + 0, 1, 0, tau, 0)   # greedy: no boundary
        assert not flags & oracle.FLAG_BOUNDARY
        gg0, gg1 = oracle.gumbel(1, 0, tau, 0, 0), oracle.gumbel(1, 0, tau, 0, 1)
        M4 = np.array([5.0, 5.0 - 1e-3, 4.0, -50.0])
        tok, margin, flags, _ = oracle.sample_cell(M4, 1.0, 2, 1, 0, tau, 0)       # keep = {0, 1}
        assert tok in (0, 1)
        M5 = np.array([5.0, 4.0, 4.0 - 1e-3, -50.0])                               # keep = {0, 1}; 2 is near
        tok, margin, flags, _ = oracle.sample_cell(M5, 1.0, 2, 1, 0, tau, 0)
        g2 = oracle.gumbel(1, 0, tau, 0, 2)
        s = [5.0 + gg0, 4.0 + gg1]
        expect = (tok == 1) or (4.0 - 1e-3 + g2 >= max(s) - oracle.TOL)
        assert bool(flags & oracle.FLAG_BOUNDARY) == expect
        hits += int(expect)
    assert 0 < hits < 200


def test_gumbel_key_layout_reading_c12():
    """Reading C12 pins WHICH Philox block and word serve a token: counter = (v >> 2, tau, stream, req_id),
    key = (seed low word, seed high word), output word v & 3.  The keyed entry point must equal the
    composition of the separately pinned pieces (Philox vs the toolkit's generator, the uniform map,
    the Gumbel closed forms) — a swapped counter word or key half would pass every other pin."""
    rng = np.random.default_rng(21)
    gfu = oracle.lib().oracle_gumbel_from_uniform
    for _ in range(400):
        seed = int(rng.integers(0, 2 ** 63)) * 2 + int(rng.integers(0, 2))
        req = int(rng.integers(0, 2 ** 32))
        tau = int(rng.integers(0, 2 ** 20))
        stream = int(rng.integers(0, 64))
        v = int(rng.integers(0, 2 ** 16))
        block = oracle.philox4x32_10([v >> 2, tau, stream, req], [seed & 0xFFFFFFFF, seed >> 32])
        want = gfu(oracle.uniform(int(block[v & 3])))
        assert oracle.gumbel(seed, req, tau, stream, v) == want
    # the five key parts are not interchangeable: swapping any two that differ changes the draw
    base = oracle.gumbel(5, 1, 2, 3, 16)
    assert len({base, oracle.gumbel(5, 2, 1, 3, 16), oracle.gumbel(5, 1, 3, 2, 16), oracle.gumbel(5, 3, 2, 1, 16),
                oracle.gumbel(5, 1, 2, 4, 12), oracle.gumbel(1, 5, 2, 3, 16), oracle.gumbel(5 << 32, 1, 2, 3, 16)}) == 7
