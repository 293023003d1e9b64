"""Block evictor: pins of the O(n) oracle statement, then the C++ O(log n) evictor against it."""
import math

import numpy as np
import pytest

from oracle.evictor_oracle import LinearEvictor, branches, delta_t, frequency
from paper_2606_02964_b200 import MsaError, MsaEvictor, MSA_ERR_INVALID_ARG, MSA_ERR_OUT_OF_RANGE, MSA_ERR_OVERLAP

P = dict(alpha=600.0, beta=15.0, tau0=540.0, k5=2.5e-9, c0=3.0e-5)      # seconds; turning point at tau* = 553.8 s


# ------------------------------------------------------------------ oracle pins (nothing here calls the C++ side)
def test_constant_recompute_cost_degenerates_to_lru():
    """with a uniform recovery cost the policy is plain LRU."""
    ev = LinearEvictor(P["alpha"], P["beta"], P["tau0"], k5=0.0, c0=1.0)
    rng = np.random.default_rng(0)
    last = rng.permutation(200).astype(float)
    for b in range(200):
        ev.add(b, int(rng.integers(0, 10_000)), float(last[b]))
    order = [ev.evict(1000.0) for _ in range(200)]
    assert order == list(np.argsort(last))


def test_equal_recency_evicts_the_cheapest_block_first():
    """identical frequency values -> lower recomputation cost goes first, i.e. earlier positions."""
    ev = LinearEvictor(**P)
    pos = np.random.default_rng(1).permutation(300) * 16
    for b in range(300):
        ev.add(b, int(pos[b]), 50.0)
    order = [ev.evict(80.0) for _ in range(300)]
    assert order == list(np.argsort(pos))


def test_eq9_branches_cross_at_the_turning_point_and_eq7_is_linear():
    a, b, t0 = P["alpha"], P["beta"], P["tau0"]
    star = t0 * a / (a - b)
    e1, e2 = branches(star, a, b, t0)
    assert e1 == pytest.approx(e2, rel=1e-12)
    assert frequency(star - 1.0, a, b, t0) == pytest.approx(math.exp(-(star - 1.0) / a))       # first branch inside the lifespan
    assert frequency(star + 1.0, a, b, t0) == pytest.approx(math.exp(-(star + 1.0 - t0) / b))  # steep branch after it
    assert frequency(0.0, a, b, t0) == 1.0
    assert delta_t(4096, 2.0, 3.0) == 2 * 2.0 * 4096 + 3.0
    assert delta_t(100, P["k5"], P["c0"]) - delta_t(99, P["k5"], P["c0"]) == pytest.approx(2 * P["k5"])


def test_each_branch_obeys_the_order_preserving_rule():
    """Eq. (8): for a single exponential the sign of w(B1) - w(B2) never changes with t."""
    rng = np.random.default_rng(2)
    ev = LinearEvictor(**P)
    for b in range(40):
        ev.add(b, int(rng.integers(0, 100_000)), float(rng.uniform(0, 500)))
    for branch in (0, 1):
        s0 = None
        for t in (500.0, 700.0, 2000.0, 9000.0):
            w = np.array([ev.weights(b, t)[branch] for b in range(40)])
            ok = w > 0                                    # deep underflow carries no order
            if ok.sum() < 2:
                continue
            idx = np.flatnonzero(ok)
            s = np.sign(np.log(w[idx])[:, None] - np.log(w[idx])[None, :])
            if s0 is None:
                s0, i0 = s, idx
            else:
                common = np.intersect1d(i0, idx)
                a = np.searchsorted(i0, common)
                b = np.searchsorted(idx, common)
                assert np.array_equal(s0[np.ix_(a, a)], s[np.ix_(b, b)])


def _eq10_lambda(tau, alpha, beta, tau0):
    """Eq. (10), retyped from the paper (not taken from the oracle)."""
    return math.exp((tau - tau0) / beta - tau / alpha)


@pytest.mark.parametrize("tau", [30.0, 200.0, 553.8461538461538, 900.0])
def test_eq10_lambda_moves_the_turning_point_to_the_given_lifespan(tau):
    """Eq. (10): with lambda = exp((tau - tau0)/beta - tau/alpha) the two branch weights of a block of age tau are
    equal (w1 == lambda * w2); a younger block is still weighed by the slow branch w1 (lambda does NOT touch it), an
    older one by lambda * w2 (Algorithm 1 line 8: lambda multiplies the SECOND tree's minimum)."""
    a, b, t0 = P["alpha"], P["beta"], P["tau0"]
    lam = _eq10_lambda(tau, a, b, t0)
    if tau == pytest.approx(t0 * a / (a - b)):
        assert lam == pytest.approx(1.0, rel=1e-9)          # the original turning point needs no correction
    ev = LinearEvictor(lambda_=lam, **P)
    t = 5000.0
    ev.add(0, 4096, t - tau)                 # exactly at the (new) turning point
    ev.add(1, 4096, t - 0.5 * tau)           # younger: inside the lifespan
    ev.add(2, 4096, t - (tau + 60.0))        # older: past it
    d = 2.0 * P["k5"] * 4096 + P["c0"]       # Eq. (7)
    w1, w2 = ev.weights(0, t)
    assert w1 == pytest.approx(lam * w2, rel=1e-12)
    assert ev.weight(0, t) == pytest.approx(w1, rel=1e-12)
    assert ev.weight(1, t) == pytest.approx(math.exp(-0.5 * tau / a) * d, rel=1e-12)
    assert ev.weight(2, t) == pytest.approx(lam * math.exp(-(tau + 60.0 - t0) / b) * d, rel=1e-12)
    assert ev.weight(2, t) < ev.weight(0, t) < ev.weight(1, t)
    assert [ev.evict(t) for _ in range(3)] == [2, 0, 1]


def test_victim_flips_from_the_w1_minimum_to_the_w2_minimum_as_lambda_crosses_w1_over_w2():
    """Algorithm 1 line 8: i = argmin{B1.w1, lambda * B2.w2}.  A = the w1-minimum (young, cheap), B = the w2-minimum
    (old, expensive).  The victim is A for lambda > w1(A)/w2(B) and B below it; the crossing is far from 1, so an
    implementation that put lambda on the other branch (crossing at w2(B)/w1(A)) fails."""
    t = 5000.0
    blocks = {7: (0, t - 100.0), 8: (32768 * 16, t - 700.0)}        # id: (pos, last access)

    def victim(lam):
        ev = LinearEvictor(lambda_=lam, **P)
        for bid, (pos, last) in blocks.items():
            ev.add(bid, pos, last)
        return ev.evict(t)

    dA, dB = 2.0 * P["k5"] * 0 + P["c0"], 2.0 * P["k5"] * 32768 * 16 + P["c0"]
    w1A, w1B = math.exp(-100.0 / P["alpha"]) * dA, math.exp(-700.0 / P["alpha"]) * dB
    w2A, w2B = math.exp(-(100.0 - P["tau0"]) / P["beta"]) * dA, math.exp(-(700.0 - P["tau0"]) / P["beta"]) * dB
    assert w1A < w1B and w2B < w2A                                   # A heads tree 1, B heads tree 2
    cross = w1A / w2B
    assert cross > 50.0                                              # nowhere near its own reciprocal
    assert victim(cross * 1.001) == 7 and victim(cross * 0.999) == 8
    assert victim(1.0) == 8 and victim(1.0 / cross) == 8             # lambda on the wrong branch would return 7 here
    assert victim(cross * cross) == 7


# ------------------------------------------------------------------ C++ evictor against the oracle
@pytest.mark.parametrize("seed,lam", [(10, 1.0), (11, 1.0), (12, 0.05), (13, 40.0)])
def test_cpp_evictor_makes_the_oracles_decisions_on_random_traces(seed, lam):
    rng = np.random.default_rng(seed)
    cpp = MsaEvictor(lambda_=lam, **P)
    ref = LinearEvictor(lambda_=lam, **P)
    t, next_id, live = 0.0, 0, []
    for step in range(4000):
        t += float(rng.exponential(1.5))
        op = rng.random()
        if op < 0.55 or not live:
            pos, last = int(rng.integers(0, 32768)) * 16, t - float(rng.exponential(300.0))
            cpp.add(next_id, pos, last)
            ref.add(next_id, pos, last)
            live.append(next_id)
            next_id += 1
        elif op < 0.75:
            b = live.pop(int(rng.integers(0, len(live))))
            cpp.remove(b)
            ref.remove(b)
        else:
            linear = bool(step & 1)
            b1, b2 = cpp.evict(t, linear=linear), ref.evict(t)
            assert b1 == b2, (step, linear)
            live.remove(b1)
        assert len(cpp) == len(ref) == len(live)
        if live and step % 97 == 0:
            b = live[int(rng.integers(0, len(live)))]
            assert cpp.weight(b, t) == pytest.approx(ref.weight(b, t), rel=1e-9, abs=1e-300)
    cpp.close()


def test_cpp_evictor_error_codes():
    ev = MsaEvictor(**P)
    with pytest.raises(MsaError) as e:
        ev.evict(0.0)
    assert e.value.status == MSA_ERR_OUT_OF_RANGE
    ev.add(7, 0, 0.0)
    with pytest.raises(MsaError) as e:
        ev.add(7, 16, 1.0)
    assert e.value.status == MSA_ERR_OVERLAP
    with pytest.raises(MsaError) as e:
        ev.add(8, -1, 1.0)
    assert e.value.status == MSA_ERR_INVALID_ARG
    with pytest.raises(MsaError) as e:
        ev.remove(9)
    assert e.value.status == MSA_ERR_OUT_OF_RANGE
    with pytest.raises(MsaError) as e:
        MsaEvictor(alpha=-1.0, beta=1.0, tau0=0.0, k5=1.0, c0=1.0)
    assert e.value.status == MSA_ERR_INVALID_ARG
    assert math.isnan(ev.weight(12345, 0.0))
    assert ev.evict(5.0) == 7 and len(ev) == 0


def test_policy_trace_shows_the_two_ended_residency_of_observation_2():
    """under pressure the shared prefix and the suffixes survive, the middle of a sequence goes."""
    from workloads.policy_trace import f3_policy_trace, policy_residency
    sessions, summary = policy_residency()
    assert summary["kept_fraction"] == pytest.approx(0.6, abs=1e-3)
    three = 0
    for x in sessions:
        r = x["resident"]
        assert r[: 512 // 16].all()                                   # the shared prefix is never the victim
        flips = int(np.count_nonzero(r[1:] != r[:-1]))
        assert flips <= 2                                              # at most prefix | evicted middle | suffix
        if flips == 2:
            three += 1
            first_gone = int(np.argmin(r))
            assert r[np.argmax(~r[first_gone:] == False) + first_gone:].all()
    assert three >= 8
    p = f3_policy_trace(layout_only=True)
    assert p.n_req == 48 and p.policy_summary["segments_per_request_max"] == 3
