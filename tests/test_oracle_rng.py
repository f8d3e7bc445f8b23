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


def test_normal_moments():
    z = _draws(_P, 1 << 17).ravel()  # 2^19 normals
    n = z.size
    assert abs(z.mean()) < 4 / np.sqrt(n)
    assert abs(z.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs((z**4).mean() - 3) < 4 * np.sqrt(96 / n)
    assert abs((z**3).mean()) < 4 * np.sqrt(15 / n)
    assert np.abs(z).max() <= 5.65
    # the four components of one call are uncorrelated
    zz = z.reshape(-1, 4)
    c = np.corrcoef(zz.T)
    assert np.abs(c - np.eye(4)).max() < 5 / np.sqrt(zz.shape[0])


def test_single_track_takes_six_words_per_step_from_the_word_stream():
    """D:RNG layout: step t of an n_x = 6 realisation takes words 6t..6t+5 of its stream, word n = output n%4 of
    call n//4; the n_x = 4 layout at step c IS call c, so it serves as the reference for the call contents."""
    class P6(_P):
        dyn = 1; dyn_p = [4, 0.05, 0.17, 0.17, 30, 30, 0.5]
    orc4, orc6 = O.Oracle(_P), O.Oracle(P6)
    call = lambda c: orc4.state_noise(3, 4, c, 1, 6)          # the four normals of call c
    w_even = orc6.state_noise(3, 4, 4, 1, 6)                   # words 24..29 = call 6 (all), call 7 (outputs 0,1)
    assert w_even.shape == (6,)
    assert np.array_equal(w_even[:4], call(6)) and np.array_equal(w_even[4:], call(7)[:2])
    w_odd = orc6.state_noise(3, 4, 5, 1, 6)                    # words 30..35 = call 7 (outputs 2,3), call 8 (all)
    assert np.array_equal(w_odd[:2], call(7)[2:]) and np.array_equal(w_odd[2:], call(8))
    # consecutive steps never reuse a word: 1.5 calls per step on average, no overlap, no gap
    assert not np.intersect1d(w_even, w_odd).size


def test_jump_noise_word_layout():
    """Jump noise takes n_x + 2 words per step: the components, the trigger, one spare (pairs stay aligned)."""
    class PJ(_P):
        noise_kind = 2; noise_p = [1.0, 0, 0, 0]     # always jump: the direction is the normalised Gaussian draw
    orcj, orc4 = O.Oracle(PJ), O.Oracle(_P)
    call = lambda c: orc4.state_noise(7, 9, c, 1, 2)
    for t in (0, 1, 2, 3):                           # words 6t..6t+3 are the components
        n0 = 6 * t
        z = np.concatenate([call(n0 // 4), call(n0 // 4 + 1)])[n0 % 4: n0 % 4 + 4]
        assert np.allclose(orcj.state_noise(7, 9, t, 1, 2), z / np.linalg.norm(z), rtol=1e-13)


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
