"""Pins of the ReSET sampler oracle (oracle/reset_oracle.py) against things other than itself: closed forms, the
hand-worked trace under tests/golden/, published known-answer vectors of the random generator, brute force."""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import reset_oracle as R


def test_entropy_closed_forms():
    for n in (1, 2, 7, 151936):
        assert abs(R.token_entropy(np.full(n, 3.25)) - math.log(n)) <= 1e-12 * max(1.0, math.log(n))   # uniform: log n
    # two-point distribution with odds e^a : 1  ->  H = log(1 + e^a) - a e^a / (1 + e^a)
    for a in (0.0, 1.0, -2.5, 10.0):
        want = math.log1p(math.exp(a)) - a * math.exp(a) / (1 + math.exp(a))
        assert abs(R.token_entropy([a, 0.0]) - want) <= 1e-13
    z = np.array([-1e9, 5.0, -1e9])
    assert R.token_entropy(z) == 0.0                                                # one-hot
    rng = np.random.default_rng(0)
    z = rng.standard_normal(1000) * 3
    assert abs(R.token_entropy(z) - R.token_entropy(z + 123.0)) <= 1e-12            # shift invariance
    p = np.exp(z) / np.exp(z).sum()
    assert abs(R.token_entropy(z) + sum(float(q) * math.log(float(q)) for q in p)) <= 1e-12    # the definition, in a loop


def test_philox_known_answers():
    """Random123 known-answer vectors for philox4x32-10 (Salmon et al., SC'11 reference implementation, kat_vectors)."""
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff, 0xffffffff), (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
            (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]
    for ctr, key, want in kat:
        got = R.philox4x32_10(*ctr, *key)
        assert tuple(int(g[0]) for g in got) == want
    # vectorised call == scalar calls
    v = R.philox4x32_10(np.arange(5), 7, 0, 0, 11, 13)
    for i in range(5):
        s = R.philox4x32_10(i, 7, 0, 0, 11, 13)
        assert all(int(a[i]) == int(b[0]) for a, b in zip(v, s))
    u = R.uniforms(100000, 3, 12345)
    assert u.min() > 0 and u.max() < 1 and abs(u.mean() - 0.5) < 0.005 and abs(u.var() - 1 / 12) < 0.002
    assert np.all((u * 2 ** 24) % 2 == 1)                                            # mid-points of 2^-23 cells: exact in binary32
    assert np.array_equal(u.astype(np.float32).astype(np.float64), u)


def _golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "reset_trace.txt")
    rows = [line.split() for line in open(path) if line.strip() and not line.startswith("#")]
    return {int(r[0]): tuple(float(x) for x in r[1:]) for r in rows}


def test_hand_worked_trace_every_branch():
    """tests/golden/reset_trace.txt: both regimes of Eq. 3 (window spanning the boundary, within-step mean), both
    branches of Eq. 2 (incl. the tie), both branches of Eq. 1 under each of them."""
    H = [0.5] * 16 + [1.5] * 16 + [2.0, 0.0] + [0.25] * 16 + [1.0] * 30 + [3.0] * 20 + [0.1]
    assert len(H) == 101
    st = R.ResetState()
    want = _golden()
    seen = set()
    for t, h in enumerate(H):
        st.H.append(h)
        h_step, h_bar = R.hse(st, t, 32), R.global_mean(st, t)
        tau = R.sat_threshold(h_step, h_bar, 0.6)
        T = R.temperature(h, tau, 0.3, 1.0)
        if t in want:
            g = want[t]
            assert abs(h_step - g[0]) <= 1e-15 and abs(h_bar - g[1]) <= 1e-15 and abs(tau - g[2]) <= 1e-15 and T == g[3], t
            seen.add((t - st.t0 < 32, h_step <= h_bar, h < tau))
        if t == 33:
            st.t0 = 34                    # the token sampled at t = 33 is the delimiter (R16)
    assert len(seen) == 8                 # every (Eq. 3 regime, Eq. 2 branch, Eq. 1 branch) combination is pinned


def test_hse_matches_brute_force_definitions():
    """Eq. 3 against the two estimators of Eq. 4 written as explicit loops."""
    rng = np.random.default_rng(1)
    H = rng.random(300).tolist()
    bounds = {40, 41, 120, 200}
    st = R.ResetState()
    for t, h in enumerate(H):
        st.H.append(h)
        if t - st.t0 < 32:
            lo = max(0, t - 31)
            want = sum(H[lo:t + 1]) / (t + 1 - lo)
        else:
            want = sum(H[st.t0:t + 1]) / (t - st.t0 + 1)
        assert abs(R.hse(st, t, 32) - want) <= 1e-14
        assert abs(R.global_mean(st, t) - sum(H[:t + 1]) / (t + 1)) <= 1e-14
        if t in bounds:
            st.t0 = t + 1


def test_top_p_by_hand_and_brute_force():
    keep = R.top_p_mask(np.array([0.5, 0.3, 0.15, 0.05]), 0.9)
    assert keep.tolist() == [True, True, True, False]           # mass above the 3rd = 0.8 < 0.9; above the 4th = 0.95
    keep = R.top_p_mask(np.array([0.05, 0.5, 0.15, 0.3]), 0.8)
    assert keep.tolist() == [False, True, False, True]          # mass above 0.15 is exactly 0.8: not < 0.8 -> dropped
    keep = R.top_p_mask(np.array([0.25, 0.25, 0.25, 0.25]), 0.1)
    assert keep.tolist() == [True] * 4                          # ties are kept together (R18)
    keep = R.top_p_mask(np.array([0.4, 0.2, 0.2, 0.2]), 0.5)
    assert keep.tolist() == [True, True, True, True]            # above each 0.2: 0.4 < 0.5
    rng = np.random.default_rng(2)
    for _ in range(50):
        p = rng.random(12); p /= p.sum()
        tp = float(rng.random())
        want = [sum(q for q in p if q > pv) < tp for pv in p]   # the definition, O(V^2)
        assert R.top_p_mask(p, tp).tolist() == want


def test_race_samples_the_renormalised_nucleus():
    """exponential race == multinomial over the kept tokens (R19): frequencies over 20000 positions, and the T -> 0 limit."""
    z = np.array([2.0, 1.0, 0.5, 0.0, -1.0, -3.0])
    T, tp = 0.7, 0.9
    p = np.exp(z / T); p /= p.sum()
    keep = R.top_p_mask(p, tp)
    q = np.where(keep, p, 0); q /= q.sum()
    n = 20000
    counts = np.bincount([R.sample_top_p(z, T, tp, t, seed=99) for t in range(n)], minlength=z.size)
    assert counts[~keep].sum() == 0
    chi2 = float((((counts - n * q) ** 2)[keep] / (n * q[keep])).sum())
    assert chi2 < 20.0                                          # 99.9th percentile of chi^2 with <= 4 d.o.f. is 18.5
    assert all(R.sample_top_p(z, 1e-3, 1.0, t, seed=5) == 0 for t in range(200))    # T -> 0: argmax


def test_reset_step_wires_the_equations_together():
    """a full step on logits: the diag values equal the separately computed equations, the delimiter moves t0."""
    rng = np.random.default_rng(3)
    st = R.ResetState()
    V = 500
    for t in range(80):
        z = rng.standard_normal(V) * (4.0 if t % 3 else 0.5)
        tok, d = R.reset_step(st, z, t, tau0=0.6, t_low=0.3, t_high=1.0, w=32, delimiter=7, seed=1,
                              forced_token=7 if t in (20, 55) else None)
        assert d["H"] == R.token_entropy(z) and d["tau"] in (0.6, d["H_step"]) and d["T"] in (0.3, 1.0)
        assert (d["T"] == 0.3) == (d["H"] < d["tau"])
        assert 0 <= tok < V
        assert st.t0 == (0 if t < 20 else 21 if t < 55 else 56)
