"""Pins for the oracle's E4M3 number line, rounding, dp(S) and scaling exactness.

Each test names the passage of PAPER.md it checks the oracle against; second sources are
torch's CPU float8_e4m3fn cast (a library routine) and exact arithmetic.
"""
import math

import numpy as np
import pytest
import torch

import oracle


def _g(golden, name):
    return {r[0]: r[1] for r in golden(name)}


def test_table_enumeration(golden):
    """126 values, 7 subnormals 2^-9*{1..7}, 8 per binade, max 448."""
    g = _g(golden, "e4m3_thresholds.txt")
    t = oracle.e4m3_table()
    assert len(t) == g["n_positive"]
    assert np.all(np.diff(t) > 0)
    sub = t[t < 2.0 ** g["min_normal_log2"]]
    assert len(sub) == g["n_subnormal"]
    np.testing.assert_array_equal(sub, 2.0 ** g["min_subnormal_log2"] * np.arange(1, 8))
    assert abs(sub[0] - g["subnormal_first"]) < 5e-6 and abs(sub[-1] - g["subnormal_last"]) < 5e-6
    assert len(t) - len(sub) == g["n_normal"]
    assert t[-1] == g["max"] == 1.75 * 2 ** 8
    assert t[7] == 2.0 ** g["min_normal_log2"]
    # every normal binade [2^n, 2^(n+1)) holds 8 equispaced values with LSB 2^(n-3)
    for n in range(-6, 8):
        inb = t[(t >= 2.0 ** n) & (t < 2.0 ** (n + 1))]
        assert len(inb) == g["per_binade"]
        np.testing.assert_array_equal(np.diff(inb), 2.0 ** (n - 3))
    # top binade [256, 512) is cut at 448 (E=15, M=7 is NaN)
    np.testing.assert_array_equal(t[t >= 256], [256, 288, 320, 352, 384, 416, 448])
    # codes are (E<<3)|M and decode back
    for c in range(1, 0x7F):
        assert oracle.e4m3_value(c) == t[c - 1]
        assert oracle.e4m3_value(c | 0x80) == -t[c - 1]
    assert oracle.e4m3_value(0) == 0.0 and math.isnan(oracle.e4m3_value(0x7F))


def test_table_matches_torch_decode():
    """Second source for Eq. 1-2: torch decodes every finite code to the same value."""
    codes = torch.arange(0, 0x7F, dtype=torch.uint8)
    vals = codes.view(torch.float8_e4m3fn).to(torch.float64).numpy()
    np.testing.assert_array_equal(vals[1:], oracle.e4m3_table())
    assert vals[0] == 0.0


def test_round_ties_and_thresholds(golden):
    """PAPER.md:72, 149, 336 + reading R6/R7: RNE, ties to the even code, 2^-10 -> 0."""
    g = _g(golden, "e4m3_thresholds.txt")
    rtz = 2.0 ** g["round_to_zero_log2"]
    assert oracle.round_e4m3(rtz) == 0                       # exact tie 0 | 2^-9 -> even code 0
    assert oracle.round_e4m3(np.nextafter(np.float32(rtz), np.float32(1))) == 1
    assert oracle.round_e4m3(np.nextafter(np.float32(rtz), np.float32(0))) == 0
    assert oracle.round_e4m3(1.5 * 2.0 ** -9) == 2             # tie 1|2 -> 2
    assert oracle.round_e4m3(2.5 * 2.0 ** -9) == 2             # tie 2|3 -> 2
    assert oracle.round_e4m3(7.5 * 2.0 ** -9) == 8             # tie 7|8 -> min normal 2^-6
    assert oracle.round_e4m3(448.0) == 0x7E
    assert oracle.round_e4m3(1e9) == 0x7E                      # satfinite (reading R22)
    assert oracle.round_e4m3(float("inf")) == 0x7E
    assert oracle.round_e4m3(0.0) == 0 and oracle.round_e4m3(-0.0) == 0x80
    assert oracle.round_e4m3(-1.0) == (0x80 | oracle.round_e4m3(1.0))
    assert oracle.round_e4m3(float("nan")) == 0x7F
    assert oracle.round_e4m3(1.0) == 0x38                      # E=7, M=0


def _torch_cast(x32: np.ndarray) -> np.ndarray:
    return torch.from_numpy(x32).to(torch.float8_e4m3fn).view(torch.uint8).numpy()


def test_round_against_torch_cast():
    """Library second source: torch CPU cast agrees on grid points, midpoints, their FP32
    neighbours and a dense log-uniform sample (torch does not saturate: compare x <= 448)."""
    t = np.concatenate([[0.0], oracle.e4m3_table()])
    mids = (t[:-1] + t[1:]) / 2
    pts = np.concatenate([t, mids]).astype(np.float32)
    pts = np.concatenate([pts, np.nextafter(pts, np.float32(np.inf)),
                          np.nextafter(pts, np.float32(-np.inf))])
    rng = np.random.default_rng(1)
    rnd = np.exp2(rng.uniform(-13, np.log2(448.0), size=200_000)).astype(np.float32)
    x = np.concatenate([pts, rnd])
    x = x[(x >= 0) & (x <= 448)]
    mine = np.array([oracle.round_e4m3(v) for v in x], dtype=np.uint8)
    np.testing.assert_array_equal(mine, _torch_cast(x))
    xn = -x[x > 0][:5000]
    np.testing.assert_array_equal(np.array([oracle.round_e4m3(v) for v in xn], dtype=np.uint8),
                                  _torch_cast(xn))


def test_round_is_nearest_bruteforce():
    """Definition: the returned code is a nearest table point (brute force over all 127)."""
    t = np.concatenate([[0.0], oracle.e4m3_table()])
    rng = np.random.default_rng(2)
    x = np.exp2(rng.uniform(-14, 9.5, size=20000)).astype(np.float32)
    for v in x:
        c = oracle.round_e4m3(v)
        err = abs(t[c] - min(float(v), 448.0))
        assert err <= np.min(np.abs(t - min(float(v), 448.0))) + 0.0


def test_dp_values(golden):
    """PAPER.md:287-295 (Thm 6) and 466-472 (App. A)."""
    for S, val, tol in golden("dp_appendix_a.txt"):
        assert abs(oracle.dp(S) - val) <= tol, (S, oracle.dp(S), val)
    assert oracle.dp(448) == 32 / 448
    assert abs(oracle.dp(448) / oracle.dp(256) - 1.142857) < 1e-6
    # Thm 6 (ii), (iii): every non-2^k scale in [2^-6, 448] and every S > 448 is above 2^-4
    pow2 = {2.0 ** k for k in range(-6, 9)}
    for S in np.concatenate([np.exp2(np.linspace(-6, np.log2(448), 4001)), np.arange(1, 449),
                             np.linspace(448.001, 8192, 3000)]):
        if float(S) in pow2:
            continue
        assert oracle.dp(float(S)) > 2.0 ** -4, S
    # footnote 1: dp in (2^-4, 2^-3) for non-2^k S in [2^-6, 448]
    for S in np.exp2(np.linspace(-6, np.log2(448), 997))[1:-1]:
        if float(S) not in pow2:
            assert 2.0 ** -4 < oracle.dp(float(S)) < 2.0 ** -3
    # minimum over [1, 448] is 2^-4, attained exactly at S = 2^k (Thm 6 (i), Thm 7)
    grid = np.arange(1, 449)
    vals = np.array([oracle.dp(float(s)) for s in grid])
    assert vals.min() == 2.0 ** -4
    np.testing.assert_array_equal(grid[vals == vals.min()], [1, 2, 4, 8, 16, 32, 64, 128, 256])


@pytest.mark.parametrize("S", [1.0, 3.0, 16.0, 100.0, 256.0, 448.0])
def test_dp_is_twice_the_max_pointwise_error(S):
    """the maximum pointwise error of P~ = Round(P*S)/S over P in [0,1] is
    dp(S)/2 (attained for these S, whose top gap's midpoint lies inside [0,S])."""
    t = np.concatenate([[0.0], oracle.e4m3_table()])
    mids = (t[:-1] + t[1:]) / 2
    cand = np.concatenate([mids[mids <= S], np.linspace(0, S, 20001)])
    worst = 0.0
    for x in cand:
        c = oracle.round_e4m3(np.float32(x))
        worst = max(worst, abs(t[c] - float(np.float32(x))) / S)
    assert abs(worst - oracle.dp(S) / 2) < 1e-7


@pytest.mark.parametrize("S", [260.0, 300.0, 5.0, 37.0])
def test_dp_bounds_the_pointwise_error(S):
    t = np.concatenate([[0.0], oracle.e4m3_table()])
    for x in np.linspace(0, S, 5001):
        c = oracle.round_e4m3(np.float32(x))
        assert abs(t[c] - float(np.float32(x))) / S <= oracle.dp(S) / 2 + 1e-7


def test_coverage_thresholds(golden):
    """P-domain normal threshold 2^-6/S."""
    min_normal = oracle.e4m3_table()[7]
    for S, printed, rtol in golden("coverage_thresholds.txt"):
        assert abs(min_normal / S - printed) <= rtol * printed
    assert min_normal / 64 == 2.0 ** -12 and min_normal / 256 == 2.0 ** -14


def test_prop5_power_of_two_scaling_is_exact():
    """PAPER.md:259-263 (Prop. 5): x*2^k and x*2^-k are exact in FP32; 1/448 is not."""
    rng = np.random.default_rng(3)
    p = np.exp(-rng.uniform(0, 20, size=100_000)).astype(np.float32)
    for k in range(0, 9):
        S = np.float32(2.0 ** k)
        assert np.array_equal((p * S) * np.float32(1.0 / S), p)
        assert np.array_equal((p * S).astype(np.float64), p.astype(np.float64) * float(S))
    S = np.float32(448.0)
    assert float(np.float32(1.0) / S) != 1.0 / 448.0
    assert not np.array_equal((p * S) * (np.float32(1.0) / S), p)


def test_quantize_roundtrip():
    """Reading R16 (parity unpinned by the paper): per-slab absmax/448; the absmax element
    maps to +-448 and every element is within half an E4M3 step of x/scale."""
    rng = np.random.default_rng(4)
    x = rng.standard_normal((2, 3, 37, 16)).astype(np.float32)
    x[1, 2, 5, 3] = -9.5
    codes, scales = oracle.quantize_e4m3(x)
    assert codes.shape == x.shape and scales.shape == (2, 3)
    t = np.concatenate([[0.0], oracle.e4m3_table()])
    for b in range(2):
        for h in range(3):
            slab = x[b, h]
            amax = np.abs(slab).max()
            assert scales[b, h] == np.float32(amax / np.float32(448.0))
            c = codes[b, h]
            i = np.unravel_index(np.abs(slab).argmax(), slab.shape)
            assert (c[i] & 0x7F) == 0x7E
            y = slab * (np.float32(448.0) / amax)
            np.testing.assert_array_equal(c, _torch_cast(y.astype(np.float32)))
            deq = np.where(c & 0x80, -1.0, 1.0) * t[c & 0x7F]
            gap = np.maximum(2.0 ** -9, 2.0 ** (np.floor(np.log2(np.maximum(np.abs(y), 2.0 ** -6))) - 3))
            assert np.all(np.abs(deq - y) <= gap / 2 + 1e-12)
    z = np.zeros((1, 1, 4, 4), dtype=np.float32)
    cz, sz = oracle.quantize_e4m3(z)
    assert sz[0, 0] == 1.0 and not cz.any()
