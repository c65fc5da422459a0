"""Parity metric of the GPU tests: the relative Frobenius error north_star states PLUS an element-wise bound.

A Frobenius norm alone cannot see a localised fault at full size: one mis-addressed 32 x 32 TMA-store box in a
2048 x 12288 output moves the relative Frobenius error by ~9e-3, under the 1e-2 bf16 tolerance.  So every tensor is
also held, element by element, to

    |got - ref|  <=  C_ELEM * tol * max(rms(ref), rms(ref row))  +  eps_store * |ref|

(DESIGN.md §7): eps_store |ref| is the one rounding of the element's own stored value (bf16: 2^-8, fp32: 2^-23);
the first term bounds the error inherited from upstream roundings, whose standard deviation is <= tol * rms(ref) (that
is what the Frobenius tolerance says).  Were it Gaussian its maximum over n <= 2e9 elements would stay below 6.4
standard deviations; it is heavier-tailed than that (an element that is a short, cancelling sum of large rounded terms
-- e.g. a tokeniser weight gradient summed over 4 patches -- inherits the error of its terms, not of its value:
11.6 standard deviations observed), so C_ELEM = 16.  A wrongly placed tile differs from the reference by ~sqrt(2) rms(ref),
i.e. ~9x this bound at tol = 1e-2 over a whole 32 x 32 box, so a single misplaced box fails.
"""
import numpy as np
import torch

C_ELEM = 16.0
EPS_STORE = {"bf16": 2.0 ** -8, "f32": 2.0 ** -23}


def to_np(got):
    if isinstance(got, torch.Tensor):
        return got.detach().to(torch.float32).cpu().numpy()
    return np.asarray(got)


CHUNK = 1 << 24          # elements per pass: keeps the float64 temporaries of the 6e8-element C5 gradients at ~0.5 GB


def check(name, got, ref, tol, store=None, c_elem=C_ELEM):
    """Assert finite values, rel. Frobenius error <= tol and the element-wise bound; returns the Frobenius error.
    `store`: storage dtype of `got` ("bf16" / "f32"); default: bf16 when tol >= 1e-3 else f32.
    The scale of the element-wise bound is max(rms of the whole tensor, rms of the element's row along the last axis):
    inherited error is proportional to the magnitude of the row it travels with (a token whose softmax weight is
    large has a proportionally large gradient row AND error), never smaller than the tensor-wide floor."""
    ref = np.asarray(ref)
    D = ref.shape[-1] if ref.ndim else 1
    r = ref.reshape(-1, D)
    g = to_np(got).reshape(-1)
    assert g.size == r.size, f"{name}: size {g.size} != reference {r.size}"
    g = g.reshape(-1, D)
    if store is None:
        store = "bf16" if tol >= 1e-3 else "f32"
    rows = r.shape[0]
    step = max(1, CHUNK // D)
    den2 = 0.0
    for a in range(0, rows, step):
        rc = r[a:a + step].astype(np.float64)
        den2 += float((rc * rc).sum())
    rms = (den2 / max(r.size, 1)) ** 0.5
    num2, nbad, worst, worst_at = 0.0, 0, -1.0, (0, 0)
    for a in range(0, rows, step):
        gc = g[a:a + step].astype(np.float64)
        assert np.isfinite(gc).all(), f"{name}: non-finite values"
        rc = r[a:a + step].astype(np.float64)
        diff = np.abs(gc - rc)
        num2 += float((diff * diff).sum())
        scale = np.maximum(np.sqrt((rc * rc).mean(axis=1, keepdims=True)), rms)
        excess = diff - (c_elem * tol * scale + EPS_STORE[store] * np.abs(rc))
        k = np.unravel_index(int(np.argmax(excess)), excess.shape)
        if excess[k] > 0:
            nbad += int((excess > 0).sum())
            if excess[k] > worst:
                worst, worst_at = float(excess[k]), (a + k[0], k[1])
    fro = num2 ** 0.5 / den2 ** 0.5 if den2 > 0 else num2 ** 0.5
    assert fro <= tol, f"{name}: rel Frobenius error {fro:.3e} > {tol:.1e}"
    if nbad:
        idx = np.unravel_index(worst_at[0] * D + worst_at[1], ref.shape)
        raise AssertionError(
            f"{name}: {nbad} element(s) outside the element-wise bound; worst at {tuple(int(i) for i in idx)}: got "
            f"{float(g[worst_at]):.6e} ref {float(r[worst_at]):.6e} (bound exceeded by {worst:.3e}; rms(ref) = {rms:.3e}, "
            f"rel Frobenius {fro:.3e})")
    return fro


def front_oracle_chunked(orc, x, emb, agg_p, dagg, p, heads, chunk, pos=None, round_tok=None):
    """The oracle's front end (tokenize -> var_aggregate -> var_aggregate_bwd -> tokenize_bwd) evaluated over a
    partition of the patches into chunks of `chunk`, calling only oracle/ functions: patches are independent in the
    forward and every parameter gradient is a sum over (b, l), so the chunk results add up to the whole-tensor
    functions exactly (pinned in tests/test_oracle_pins.py) while the fp64 [B, L, V, D] tensors (12 GB each at C3)
    never exist.  `round_tok`: optional storage rounding of the tokens between the two calls (the two-call GPU path
    stores tok in bf16; the fused path never forms it).  Returns agg [B, L, D], dWp, dbp, the aggregation gradients
    and dpos (None without pos)."""
    B, V, Hg, Wg = x.shape
    L = (Hg // p) * (Wg // p)
    out_agg, dWp, dbp, G, dpos = None, None, None, None, None
    for a in range(0, L, chunk):
        ls = np.arange(a, min(a + chunk, L))
        tok_s = orc.tokenize_patches(x, emb["Wp"], emb["bp"], p, ls)
        if round_tok is not None:
            tok_s = round_tok(tok_s)
        agg_s, cache = orc.var_aggregate(tok_s, agg_p, heads, None if pos is None else np.asarray(pos)[ls])
        dtok_s, G_s, dpos_s = orc.var_aggregate_bwd(np.asarray(dagg)[:, ls], agg_p, cache, want_dpos=pos is not None)
        dWp_s, dbp_s = orc.tokenize_bwd_patches(x, dtok_s, p, ls)
        if out_agg is None:
            out_agg = np.empty((B, L, agg_s.shape[-1]), dtype=np.float64)
            dWp, dbp, G = dWp_s, dbp_s, G_s
            if pos is not None:
                dpos = np.empty((L, agg_s.shape[-1]), dtype=np.float64)
        else:
            dWp += dWp_s
            dbp += dbp_s
            for k in G:
                G[k] = G[k] + G_s[k]
        out_agg[:, ls] = agg_s
        if pos is not None:
            dpos[ls] = dpos_s
    return out_agg, dWp, dbp, G, dpos
