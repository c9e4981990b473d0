"""Pins for the oracle's self-supervised decomposition (Eq. 5; Q31): closed forms on
magnitudes 0..N-1, numpy's sort / partition as the library routine, ties, the k = 0 / 100 ends, Eq. 5 as a numpy mean,
central differences of L_s with the classification held fixed, the binary32 magnitude.  CPU only."""
import numpy as np
import pytest

import oracle


def ramp(n, seed=0):
    """dp[i] = mag_i * unit vector, mag a permutation of 0..n-1 (all distinct, exactly representable)."""
    rng = np.random.default_rng(seed)
    mags = rng.permutation(n).astype(np.float32)
    axis = rng.integers(0, 3, n)
    dp = np.zeros((n, 3), np.float32)
    dp[np.arange(n), axis] = mags * rng.choice([-1.0, 1.0], n).astype(np.float32)
    return dp, mags


@pytest.mark.parametrize("n,k", [(1000, 30.0), (1000, 0.1), (777, 12.5), (10, 25.0), (1, 50.0)])
def test_closed_form_on_distinct_integer_magnitudes(n, k):
    dp, mags = ramp(n, n)
    r = oracle.oracle_decompose(dp, k)
    m = int(np.ceil(n * k / 100.0 - 1e-9))
    np.testing.assert_array_equal(r["mag"], mags)
    assert r["tau"] == (float(n - 1 - m) if m < n else -1.0)          # the (m+1)-th largest of 0..n-1
    np.testing.assert_array_equal(r["index"], np.nonzero(mags > n - 1 - m)[0])
    assert len(r["index"]) == m
    static = mags[mags <= n - 1 - m]
    assert r["loss"] == pytest.approx(static.mean() if len(static) else 0.0, rel=1e-15)


def test_numpy_sort_rebuild_random_and_ties_and_ends():
    rng = np.random.default_rng(3)
    dp = rng.standard_normal((5000, 3)).astype(np.float32) * rng.choice([0.0, 1e-3, 1.0], (5000, 1)).astype(np.float32)
    for k in (0.0, 1.0, 30.0, 99.99, 100.0):
        r = oracle.oracle_decompose(dp, k)
        mag = r["mag"]
        m = int(min(5000, max(0, np.ceil(5000 * k / 100.0 - 1e-9))))
        tau = np.inf if m == 0 else (-1.0 if m >= 5000 else np.sort(mag)[::-1][m])
        assert r["tau"] == tau
        np.testing.assert_array_equal(r["index"], np.nonzero(mag > tau)[0].astype(np.int32))
        st = mag[~(mag > tau)]
        assert r["loss"] == pytest.approx(st.astype(np.float64).mean() if len(st) else 0.0, rel=1e-13)
    # one third of the rows are exactly zero: with k = 80 % the threshold falls INTO the tie at 0 -> strictly greater only
    r = oracle.oracle_decompose(dp, 80.0)
    assert r["tau"] == 0.0 and len(r["index"]) == int((r["mag"] > 0).sum()) < 4000
    # all equal: nobody is strictly above the threshold
    same = np.tile(np.array([[3, 4, 0]], np.float32), (100, 1))
    r = oracle.oracle_decompose(same, 30.0)
    assert r["tau"] == 5.0 and len(r["index"]) == 0 and r["loss"] == 5.0


def test_magnitude_is_binary32_without_contraction_and_nan_counts_as_zero():
    rng = np.random.default_rng(5)
    dp = rng.standard_normal((4000, 3)).astype(np.float32) * np.float32(1e-3)
    want = np.sqrt(((dp[:, 0] * dp[:, 0]) + (dp[:, 1] * dp[:, 1])) + (dp[:, 2] * dp[:, 2]))    # numpy: fp32 ops, in order
    assert want.dtype == np.float32
    np.testing.assert_array_equal(oracle.oracle_decompose(dp, 10.0)["mag"], want)
    bad = np.array([[np.nan, 0, 0], [1, 2, 2], [np.inf, 0, 0]], np.float32)
    r = oracle.oracle_decompose(bad, 34.0)                              # m = 2: inf and 3 are the top two
    np.testing.assert_array_equal(r["mag"], [0.0, 3.0, np.inf])
    np.testing.assert_array_equal(r["index"], [1, 2])
    assert r["tau"] == 0.0 and r["loss"] == 0.0 and (r["ddp"] == 0).all()   # the NaN row is static with magnitude 0


def test_gradient_is_the_derivative_of_eq5_with_the_classification_fixed():
    rng = np.random.default_rng(7)
    n = 60
    dp = rng.standard_normal((n, 3)).astype(np.float32)
    r = oracle.oracle_decompose(dp, 25.0, grad_scale=0.5)
    dyn = np.zeros(n, bool); dyn[r["index"]] = True
    ns = n - dyn.sum()
    want = 0.5 * dp.astype(np.float64) / (r["mag"].astype(np.float64)[:, None] * ns)
    want[dyn] = 0
    np.testing.assert_allclose(r["ddp"], want, rtol=2e-7, atol=0)
    # central differences of  0.5 * mean_{static} ||dp||  (static set fixed), in double
    loss = lambda x: 0.5 * np.linalg.norm(x[~dyn], axis=1).sum() / ns
    x0 = dp.astype(np.float64)
    for i in (0, 7, 31):
        for d in range(3):
            xp, xm = x0.copy(), x0.copy()
            xp[i, d] += 1e-6; xm[i, d] -= 1e-6
            assert (loss(xp) - loss(xm)) / 2e-6 == pytest.approx(want[i, d], abs=1e-8)
    assert (r["ddp"][dyn] == 0).all() and np.abs(r["ddp"][~dyn]).sum() > 0
    # a static Gaussian that does not move has no direction to be pulled in
    dp[3] = 0
    assert (oracle.oracle_decompose(dp, 25.0)["ddp"][3] == 0).all()
