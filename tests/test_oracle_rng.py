"""Pins for the oracle's random source (no GPU).

Philox4x32-10 is pinned against two implementations that are independent of this repo:
torch's at::philox_engine (compiled from the ATen header by this test) and cuRAND's *host*
generator (libcurand, runs on the CPU).  The Random123 known-answer file BASELINE names is
not in the container, so agreement of three implementations stands in.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle as O

TORCH_INC = None
try:
    import torch

    TORCH_INC = os.path.join(os.path.dirname(torch.__file__), "include")
except Exception:  # pragma: no cover
    pass


@pytest.fixture(scope="module")
def aten_philox(tmp_path_factory):
    if TORCH_INC is None or not os.path.exists(os.path.join(TORCH_INC, "ATen/core/PhiloxRNGEngine.h")):
        pytest.skip("ATen Philox header not available")
    exe = str(tmp_path_factory.mktemp("aten") / "aten_philox")
    src = os.path.join(os.path.dirname(__file__), "helpers", "aten_philox_main.cpp")
    subprocess.run(["g++", "-O1", "-std=c++17", f"-I{TORCH_INC}", src, "-o", exe], check=True)

    def run(rows):
        inp = "\n".join(" ".join(str(int(x)) for x in r) for r in rows) + "\n"
        out = subprocess.run([exe], input=inp, capture_output=True, text=True, check=True).stdout
        return [[int(x) for x in line.split()] for line in out.strip().splitlines()]

    return run


def test_philox_matches_aten_on_random_and_layout_counters(aten_philox):
    rng = np.random.default_rng(7)
    rows = [list(rng.integers(0, 2**32, size=6)) for _ in range(200)]
    rows += [[0, 0, 0, 0, 0, 0], [2**32 - 1] * 6]
    # counters of the layout actually used: (k, m, t*J+j, stream<<28|iteration), key = seed halves
    for stream in (0, 1, 2):
        for (k, m, t, J, j, it) in [(0, 0, 0, 1, 0, 0), (255, 15, 19, 1, 0, 0), (8191, 127, 59, 2, 1, 3),
                                    (65535, 255, 49, 1, 0, 499), (3, 2, 1, 3, 2, 2**28 - 1)]:
            rows.append(O.counter(k, m, t, J, j, stream, it) + [4, 0])
    ref = aten_philox(rows)
    for r, o in zip(rows, ref):
        assert O.philox4x32_10(r[:4], r[4:]) == o


def test_counter_layout():
    assert O.counter(5, 6, 7, 2, 1, 1, 9) == [5, 6, 15, (1 << 28) | 9]
    assert O.counter(0, 0, 0, 1, 0, 2, (1 << 28) + 3) == [0, 0, 0, (2 << 28) | 3]  # iteration wraps at 2^28


def test_philox_matches_curand_host_generator():
    try:
        cr = C.CDLL("libcurand.so")
    except OSError:
        try:
            cr = C.CDLL("/usr/local/cuda/lib64/libcurand.so")
        except OSError:
            pytest.skip("libcurand not available")
    for seed in (0, 1, 0x0123456789ABCDEF, 2**64 - 1):
        gen = C.c_void_p()
        assert cr.curandCreateGeneratorHost(C.byref(gen), 161) == 0  # CURAND_RNG_PSEUDO_PHILOX4_32_10
        assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
        n = 4 * 64
        out = (C.c_uint32 * n)()
        assert cr.curandGenerate(gen, out, C.c_size_t(n)) == 0
        cr.curandDestroyGenerator(gen)
        key = (seed & 0xFFFFFFFF, seed >> 32)
        # cuRAND's host ordering: block s of four outputs is subsequence s at offset 0 = counter (0,0,s,0)
        for s in range(64):
            assert O.philox4x32_10((0, 0, s, 0), key) == list(out[4 * s:4 * s + 4])


def test_philox_is_a_bijection_on_counters_sample():
    # distinct counters -> distinct outputs (Philox is a permutation for a fixed key)
    outs = {tuple(O.philox4x32_10((i, j, 0, 0), (1, 2))) for i in range(64) for j in range(64)}
    assert len(outs) == 64 * 64


def test_box_muller_end_points():
    # u1 = 1 (ra all ones) -> rho = 0
    z = O.box_muller(0xFFFFFFFF, 0x12345678)
    assert z[0] == 0.0 and z[1] == 0.0
    # u2 = 0 -> angle 0 -> z = (rho, 0);  u1 = 2^-23 -> rho = sqrt(2*23*ln2)
    z = O.box_muller(0, 0)
    assert z[0] == pytest.approx(np.sqrt(2 * 23 * np.log(2.0)), rel=1e-15) and z[1] == 0.0
    # u2 = 1/4 -> angle pi/2 -> z = (0, rho) ; u1 = 1/2
    z = O.box_muller((2**22 - 1) << 9, 2**21 << 9)
    rho = np.sqrt(2 * np.log(2.0))
    assert abs(z[0]) < 1e-15 and z[1] == pytest.approx(rho, rel=1e-15)
    # low 9 bits are ignored
    assert np.array_equal(O.box_muller(0x000001FF, 0x000001FF), O.box_muller(0, 0))


class _P:  # minimal problem record for state_noise
    K = M = T = 1; dt = 0.1; dyn = 0; dyn_p = [0.33]; u_min = [-1, -1]; u_max = [1, 1]
    sigma_eps = [1, 1]; sigma_w = [1, 1, 1, 1, 1, 1]; alpha = 0.9; lam = 1; gamma = 0
    A = 1; B = 1; C_u = 0; eta = 0; nominal = 0; nom_p = [1, 0, 0, 1]; risk = 2; risk_p = [1, 3]
    noise_kind = 0; noise_p = [0, 0, 0, 0]; seed = 42; circles = None; costmap = None


def _draws(p, n_calls):
    orc = O.Oracle(p)
    return np.array([orc.state_noise(i & 0xFFFF, i >> 16, 0, 1, 0) for i in range(n_calls)])


def test_box_muller16_end_points():
    """State-noise normals: ONE word per pair: radius uniform u1 = (lo16 + 1/2) 2^-16 in (0,1)
    from the low half, angle uniform u2 = (w >> 9) 2^-23 from the top 23 bits."""
    rho_max = np.sqrt(2 * 17 * np.log(2.0))                   # u1 = 2^-17
    z = O.box_muller16(0x00000000)
    assert z[0] == pytest.approx(rho_max, rel=1e-15) and z[1] == 0.0
    z = O.box_muller16(0x40000000)                             # u2 = 1/4 -> angle pi/2
    assert abs(z[0]) < 1e-15 and z[1] == pytest.approx(rho_max, rel=1e-15)
    z = O.box_muller16(0x80000000)                             # u2 = 1/2 -> angle pi
    assert z[0] == pytest.approx(-rho_max, rel=1e-15) and abs(z[1]) < 1e-15
    z = O.box_muller16(0x0000FFFF)                             # u1 = 1 - 2^-17: the smallest radius, never exactly 0
    rho_min = np.sqrt(-2 * np.log1p(-2.0**-17))
    assert np.hypot(*z) == pytest.approx(rho_min, rel=1e-12) and np.hypot(*z) > 0
    assert np.arctan2(z[1], z[0]) == pytest.approx(2 * np.pi * (0xFFFF >> 9) / 2.0**23, rel=1e-9)   # the shared bits turn it
    z = O.box_muller16(0x00007FFF)
    assert np.hypot(*z) == pytest.approx(np.sqrt(-2 * np.log(32767.5 / 65536)), rel=1e-15)
    # roles: the high half only rotates; bits 0..8 only rescale; bits 9..15 do both
    a, b = O.box_muller16(0x00000123), O.box_muller16(0x56780123)
    assert np.hypot(*a) == pytest.approx(np.hypot(*b), rel=1e-15) and a[1] == 0.0 and b[1] != 0.0
    a, b = O.box_muller16(0x12340000), O.box_muller16(0x123401FF)
    assert np.arctan2(a[1], a[0]) == pytest.approx(np.arctan2(b[1], b[0]), rel=1e-14) and np.hypot(*a) > np.hypot(*b)
    a, b = O.box_muller16(0x12340000), O.box_muller16(0x12340200)
    assert np.arctan2(b[1], b[0]) - np.arctan2(a[1], a[0]) == pytest.approx(2 * np.pi * 2.0**-23, rel=1e-6)


def test_box_muller16_exact_lattice_moments():
    """The 2^32 words map to 2^32 points of a polar lattice; its moments are exact finite sums: E z^2 = 1 - 5.3e-6,
    E z^4 = 3 - 2.1e-4, |z| <= 4.855 (the numbers DESIGN.md states).  The radial sum runs over all 65536 radii.  For
    every radius the 65536 free angle bits give equally spaced angles over the full turn (offset by the shared bits), so
    the angular means are exact by symmetry (mean cos = mean cos sin = 0, mean cos^2 = 1/2, mean cos^4 = 3/8)."""
    lo = np.arange(65536, dtype=np.uint64)
    rho = np.array([np.hypot(*O.box_muller16(int(h))) for h in lo[::257]])            # sampled radii via the oracle
    r2_all = -2.0 * np.log((lo.astype(np.float64) + 0.5) / 65536.0)
    assert np.allclose(rho**2, r2_all[::257], rtol=1e-13)
    Ez2, Ez4 = r2_all.mean() / 2.0, (r2_all**2).mean() * 3.0 / 8.0
    assert Ez2 == pytest.approx(1.0 - 5.29e-6, abs=2e-8) and Ez4 == pytest.approx(3.0 - 2.106e-4, abs=1e-6)
    assert np.sqrt(r2_all.max()) == pytest.approx(4.8546, abs=1e-4)
    # angles of one radius (low half fixed, all shared bits included): equally spaced, full turn, exact symmetry
    for low in (0x0000, 0x8001, 0xFE37):
        hi = np.arange(0, 65536, 64)
        pts = np.array([O.box_muller16((int(h) << 16) | low) for h in hi])
        r0 = np.sqrt(-2.0 * np.log((low + 0.5) / 65536.0))
        th = 2 * np.pi * (((hi.astype(np.uint64) << 16) | low) >> 9).astype(np.float64) / 2.0**23
        assert np.allclose(pts[:, 0], r0 * np.cos(th), atol=1e-14) and np.allclose(pts[:, 1], r0 * np.sin(th), atol=1e-14)
        assert abs(pts[:, 0].mean()) < 1e-13 and abs((pts[:, 0] * pts[:, 1]).mean()) < 1e-13
        assert (pts[:, 0] ** 2).mean() == pytest.approx(r0 * r0 / 2, rel=1e-12)
    # distinct words -> distinct points (the shared bits lose nothing)
    ws = np.random.default_rng(3).integers(0, 2**32, 4000)
    assert len({tuple(O.box_muller16(int(w))) for w in ws}) == len(set(int(w) for w in ws))


def test_normal_moments():
    z = _draws(_P, 1 << 17).ravel()  # 2^19 normals
    n = z.size
    assert abs(z.mean()) < 4 / np.sqrt(n)
    assert abs(z.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs((z**4).mean() - 3) < 4 * np.sqrt(96 / n)
    assert abs((z**3).mean()) < 4 * np.sqrt(15 / n)
    assert np.abs(z).max() <= 4.8546
    # the four components of one step are uncorrelated (two pairs from two words)
    zz = z.reshape(-1, 4)
    c = np.corrcoef(zz.T)
    assert np.abs(c - np.eye(4)).max() < 5 / np.sqrt(zz.shape[0])
    # squares too (a pair shares its radius only through independent angles): cov(z0^2, z1^2) = 0 for exact normals
    c2 = np.corrcoef((zz**2).T)
    assert np.abs(c2 - np.eye(4)).max() < 5 / np.sqrt(zz.shape[0])


def test_state_noise_distribution_ks_and_tail_mass():
    """16 bits per uniform must not show in the distribution the CVaR reads: Kolmogorov-Smirnov distance to N(0,1)
    and the tail mass beyond the alpha-quantiles the configs use (0.9, 0.95, 0.99; both tails), on 2^21 draws."""
    from scipy import stats
    z = _draws(_P, 1 << 19).ravel()
    n = z.size
    d = stats.kstest(z, "norm").statistic
    assert d < 1.63 / np.sqrt(n), d                      # 1 % critical value of the KS statistic
    for alpha in (0.9, 0.95, 0.99, 0.999):
        q = stats.norm.ppf(alpha)
        for tail in ((z > q).mean(), (z < -q).mean()):
            assert abs(tail - (1 - alpha)) < 4 * np.sqrt(alpha * (1 - alpha) / n), (alpha, tail)
    # tail mean beyond the quantile = the closed-form Gaussian CVaR (golden file: scipy)
    for alpha, want in ((0.9, 1.7549833), (0.99, 2.6652142)):
        q = stats.norm.ppf(alpha)
        got = z[z > q].mean()
        assert got == pytest.approx(want, abs=4 * 0.6 / np.sqrt((1 - alpha) * n))


def _word(k, m, n, stream, it, seed=_P.seed):
    """Word n of the (k, m, stream, iteration) word stream, from the free functions (pinned above)."""
    key = (seed & 0xFFFFFFFF, seed >> 32)
    return O.philox4x32_10(O.counter(k, m, n // 4, 1, 0, stream, it), key)[n % 4]


def test_state_noise_word_layout_nx4_and_nx6():
    """D:RNG layout: step t of a realisation takes the n_x/2 words (n_x/2) t .. of its word stream, word j -> the
    Box-Muller pair of components (2j, 2j+1): n_x = 4 spends one Philox call on two steps, n_x = 6 three calls on
    four steps."""
    class P6(_P):
        dyn = 1; dyn_p = [4, 0.05, 0.17, 0.17, 30, 30, 0.5]
    orc4, orc6 = O.Oracle(_P), O.Oracle(P6)
    for t in (0, 1, 2, 3, 7, 58):
        w4 = orc4.state_noise(3, 4, t, 1, 6)
        assert w4.shape == (4,)
        assert np.array_equal(w4, np.concatenate([O.box_muller16(_word(3, 4, 2 * t + j, 1, 6)) for j in range(2)]))
        w6 = orc6.state_noise(3, 4, t, 1, 6)
        assert w6.shape == (6,)
        assert np.array_equal(w6, np.concatenate([O.box_muller16(_word(3, 4, 3 * t + j, 1, 6)) for j in range(3)]))
    # steps 2s and 2s+1 of an n_x = 4 realisation share call s and nothing else; no word is used twice
    used = [2 * t + j for t in range(8) for j in range(2)]
    assert used == list(range(16))
    # stream and iteration enter the counter; the PLANT stream is realisation (0, 0), step 0
    assert not np.array_equal(orc4.state_noise(3, 4, 0, 1, 6), orc4.state_noise(3, 4, 0, 2, 6))
    assert np.array_equal(orc4.state_noise(0, 0, 0, 2, 9),
                          np.concatenate([O.box_muller16(_word(0, 0, j, 2, 9)) for j in range(2)]))


def test_jump_noise_word_layout():
    """Jump noise takes n_x/2 + 1 words per step: the pairs, then a word whose HIGH half is the trigger."""
    class PJ(_P):
        noise_kind = 2; noise_p = [1.0, 0, 0, 0]     # always jump: the direction is the normalised Gaussian draw
    class PJh(_P):
        noise_kind = 2; noise_p = [0.5, 0, 0, 0]
    orcj, orch = O.Oracle(PJ), O.Oracle(PJh)
    n_hit = 0
    for t in range(40):
        z = np.concatenate([O.box_muller16(_word(7, 9, 3 * t + j, 1, 2)) for j in range(2)])
        assert np.allclose(orcj.state_noise(7, 9, t, 1, 2), z / np.linalg.norm(z), rtol=1e-13)
        trig = (_word(7, 9, 3 * t + 2, 1, 2) >> 16) / 65536.0
        got = orch.state_noise(7, 9, t, 1, 2)
        assert (np.linalg.norm(got) > 0) == (trig < 0.5)
        n_hit += trig < 0.5
    assert 8 < n_hit < 32


def test_uniform_noise_word_layout():
    class PU(_P):
        noise_kind = 1
    orc = O.Oracle(PU)
    for t in (0, 1, 5):
        u = orc.state_noise(2, 3, t, 1, 4)
        for j in range(2):
            w = _word(2, 3, 2 * t + j, 1, 4)
            assert u[2 * j] == (2 * (w >> 16) + 1) / 65536.0 - 1.0 and u[2 * j + 1] == (2 * (w & 0xFFFF) + 1) / 65536.0 - 1.0


def test_uniform_and_jump_noise_kinds():
    class PU(_P):
        noise_kind = 1; sigma_w = [0.2] * 6
    u = _draws(PU, 1 << 15).ravel()
    assert u.min() > -0.2 and u.max() < 0.2
    assert abs(u.mean()) < 4 * 0.2 / np.sqrt(3 * u.size)
    assert abs(u.var() - 0.2**2 / 3) < 1e-3  # variance of U[-a,a] is a^2/3

    class PJ(_P):
        noise_kind = 2; sigma_w = [0.45] * 6; noise_p = [0.02, 0, 0, 0]
    j = _draws(PJ, 1 << 15)
    nrm = np.linalg.norm(j, axis=1)
    hit = nrm > 0
    assert np.allclose(nrm[hit], 0.45, rtol=1e-12)  # "sudden change of magnitude 0.45" PAPER.md:263
    assert abs(hit.mean() - 0.02) < 4 * np.sqrt(0.02 * 0.98 / hit.size)  # "2% chance"
    # arbitrary direction: mean direction ~ 0
    assert np.abs(j[hit].mean(axis=0)).max() < 5 * 0.45 / np.sqrt(4 * hit.sum())
