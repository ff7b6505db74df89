"""CPU oracle of the ReSET sampler step (Sec. 4, :107-139): TEST INFRASTRUCTURE, never on the product path.

Plain NumPy float64, written equation by equation in the paper's order and notation; it shares no code with the CUDA
path (paper_2606_13233_b200/csrc/sampler.cu).  Only tests/, __graft_entry__.smoke() and bench.py's cpu legs import it.

What one step computes for decoding position t (0-based) from the logits z_t over the vocabulary:
  H_t      token entropy of softmax(z_t), natural log                       (Sec. 2.2)
  H_bar    running global mean (1/(t+1)) sum_{i<=t} H_i                      (Sec. 4)
  H_step   hybrid step-entropy estimate HSE, Eq. 3
  tau_t    step-aware threshold SAT, Eq. 2
  T_t      T_low if H_t < tau_t else T_high, Eq. 1 with tau_t
  token    top-p (0.95, App. B.5) sample from softmax(z_t / T_t)
  t0       the next step starts after a sampled step delimiter ("\\n\\n" token, App. B.1)

Readings where the paper is silent (R14-R19):
  R14 H_t is the entropy of the model distribution at temperature 1 (softmax(z_t)), in nats.
  R15 the window W_t of Eq. 3 is the min(w, t+1) most recent positions ending at t (it spans the step boundary,
      PAPER.md:128; before w tokens exist it is shorter, hence the paper's 1/|W_t|).
  R16 the delimiter token belongs to the step it ends: t0 <- t + 1 after it is sampled.
  R17 ties go to the paper's first branch as written: H_step <= H_bar is "confident"; H_t < tau_t sharpens.
  R18 top-p keeps token v iff the probability mass of the STRICTLY more probable tokens is < p (the smallest
      highest-probability prefix whose mass reaches p; all tokens tied with the last one are kept).
  R19 the draw itself is the exponential race used by the paper's serving stack (vLLM):
      argmax_v p_v / e_v with e_v ~ Exp(1), i.e. argmax of z_v/T_t - log(-log u_v) over the kept tokens, ties to
      the lowest index; u_v comes from the counter-based generator Philox4x32-10 (counter = (v, t, 0, 0),
      key = the 64-bit seed), u = ((x0 >> 9) + 0.5) * 2^-23 -- the same generator the CUDA path implements.
"""
from __future__ import annotations

import numpy as np

# ---- Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11) ----------------------------
_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """vectorised over the counter words (uint32 arrays or scalars); returns four uint32 arrays."""
    c0, c1, c2, c3 = [np.atleast_1d(np.asarray(c, dtype=np.uint64)) & _MASK for c in (c0, c1, c2, c3)]
    c0, c1, c2, c3 = np.broadcast_arrays(c0, c1, c2, c3)
    k0, k1 = int(k0) & 0xFFFFFFFF, int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0                                   # 32 x 32 -> 64 bit products
        p1 = _M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & _MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ np.uint64(k0)) & _MASK, lo1, (hi0 ^ c3 ^ np.uint64(k1)) & _MASK, lo0
        k0, k1 = (k0 + _W0) & 0xFFFFFFFF, (k1 + _W1) & 0xFFFFFFFF
    return tuple(c.astype(np.uint32) for c in (c0, c1, c2, c3))


def uniforms(V: int, t: int, seed: int) -> np.ndarray:
    """u_v in (0,1) for v = 0..V-1 at decoding position t (R19): 23 random bits, mid-point of the cell."""
    x0 = philox4x32_10(np.arange(V, dtype=np.uint64), t & 0xFFFFFFFF, 0, 0, seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)[0]
    return ((x0 >> np.uint32(9)).astype(np.float64) + 0.5) * 2.0 ** -23


# ---- the equations -----------------------------------------------------------------------------------------------
def token_entropy(z) -> float:
    """H_t = -sum_v p_t(v) log p_t(v), p_t = softmax(z_t)   (R14)."""
    z = np.asarray(z, dtype=np.float64)
    zs = z - z.max()
    p = np.exp(zs)
    Z = p.sum()
    p = p / Z
    nz = p > 0
    return float(-(p[nz] * np.log(p[nz])).sum())


class ResetState:
    """per-sequence state of Eqs. 2-3: every H_i seen so far and the start t0 of the current step (plain, not
    incremental: the estimator below re-reads the list, so it is the definition itself)."""

    def __init__(self):
        self.H = []          # H_0 .. H_{t-1}
        self.t0 = 0


def hse(state: ResetState, t: int, w: int) -> float:
    """Eq. 3, state.H holds H_0..H_t."""
    H = state.H
    if t - state.t0 < w:                                 # initialization: window of the w most recent tokens (R15)
        win = H[max(0, t - w + 1): t + 1]
        return float(np.sum(win, dtype=np.float64) / len(win))
    seg = H[state.t0: t + 1]                             # within-step running average
    return float(np.sum(seg, dtype=np.float64) / (t - state.t0 + 1))


def global_mean(state: ResetState, t: int) -> float:
    """H_bar = (1/(t+1)) sum_{i=0}^{t} H_i."""
    return float(np.sum(state.H[: t + 1], dtype=np.float64) / (t + 1))


def sat_threshold(h_step: float, h_bar: float, tau0: float) -> float:
    """Eq. 2."""
    return tau0 if h_step <= h_bar else h_step


def temperature(h_t: float, tau_t: float, t_low: float, t_high: float) -> float:
    """Eq. 1 with tau_t substituted."""
    return t_low if h_t < tau_t else t_high


def top_p_mask(p: np.ndarray, top_p: float) -> np.ndarray:
    """R18: keep v iff the mass of strictly more probable tokens is < top_p.  O(V log V), by definition."""
    p = np.asarray(p, dtype=np.float64)
    order = np.argsort(-p, kind="stable")
    ps = p[order]
    csum = np.cumsum(ps)
    # mass strictly above each sorted position: cumulative sum up to the first element of its tie group
    first_of_group = np.concatenate([[True], ps[1:] != ps[:-1]])
    grp_start = np.maximum.accumulate(np.where(first_of_group, np.arange(p.size), 0))
    above = np.where(grp_start > 0, csum[np.maximum(grp_start - 1, 0)], 0.0)
    keep_sorted = above < top_p
    keep = np.zeros(p.size, dtype=bool)
    keep[order] = keep_sorted
    return keep


def sample_top_p(z, T: float, top_p: float, t: int, seed: int) -> int:
    """top-p sample from softmax(z / T) by the exponential race (R18, R19)."""
    z = np.asarray(z, dtype=np.float64)
    zs = (z - z.max()) / T
    p = np.exp(zs)
    p = p / p.sum()
    keep = top_p_mask(p, top_p)
    u = uniforms(z.size, t, seed)
    score = np.where(keep, zs - np.log(-np.log(u)), -np.inf)
    return int(np.argmax(score))                         # first maximum = lowest index


def reset_step(state: ResetState, z, t: int, *, tau0: float, t_low: float, t_high: float, top_p: float = 0.95,
               w: int = 32, delimiter: int = -1, seed: int = 0, forced_token=None):
    """one ReSET decoding step at position t.  Returns (token, diag) with diag = dict(H, H_step, H_bar, tau, T).
    `forced_token` replaces the draw (teacher forcing, for traces with prescribed boundaries)."""
    assert t == len(state.H)
    h_t = token_entropy(z)
    state.H.append(h_t)
    h_step = hse(state, t, w)
    h_bar = global_mean(state, t)
    tau_t = sat_threshold(h_step, h_bar, tau0)
    T_t = temperature(h_t, tau_t, t_low, t_high)
    token = sample_top_p(z, T_t, top_p, t, seed) if forced_token is None else int(forced_token)
    if token == delimiter:
        state.t0 = t + 1                                 # R16
    return token, dict(H=h_t, H_step=h_step, H_bar=h_bar, tau=tau_t, T=T_t)
