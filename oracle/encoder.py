"""TEST INFRASTRUCTURE -- fp64 oracle of the transformer-encoder NER forward.

What it follows.  PAPER.md L43 (§II stage 2) only names the operation ("a configurable
transformer model ... Inference runs on GPU"); BASELINE.json north_star ¶1 lists the steps
("embedding plus L encoder layers (QKV/out/FFN GEMMs, padding-masked variable-length
self-attention, LayerNorm, GELU), then the token-classification head. Per-token argmax")
and SURVEY.md §8(c) O1/O2 fixes the formulas (readings S1-S10: post-LN BERT-style block,
learned absolute positions 0..n-1 per sequence, one token-type vector, biased variance
with eps inside the sqrt, erf GELU, scale 1/sqrt(d_head), bidirectional, ties -> lowest).

Written in the order and notation of O1, one sequence at a time, one head at a time, in
float64 throughout (tier rule: fp64 unless the paper fixes a precision; it fixes none).
``@`` (numpy matmul) and ``scipy.special.erf`` are the only library steps.  No blocking,
no fusion, no batching across sequences: sequences are independent by definition.

Pins: tests/test_oracle_encoder.py (triple-loop brute-force attention, closed forms for
LN/GELU/softmax, padding/packing/permutation invariances, L=0 special case, and a torch
float64 composition of library primitives).
"""
import numpy as np
from scipy.special import erf


def layer_norm(z, g, b, eps):
    """LN(z; g, b)_i = (z_i - mean) / sqrt(var + eps) * g_i + b_i, var biased (O1 last line)."""
    mean = z.mean(axis=-1, keepdims=True)
    var = ((z - mean) ** 2).mean(axis=-1, keepdims=True)
    return (z - mean) / np.sqrt(var + eps) * g + b


def gelu(z):
    """gelu(z) = 0.5 z (1 + erf(z / sqrt 2))  (reading S5)."""
    return 0.5 * z * (1.0 + erf(z / np.sqrt(2.0)))


def softmax_rows(s):
    """p_jm = exp(s_jm - max_m s_jm) / sum_m exp(s_jm - max_m s_jm)."""
    e = np.exp(s - s.max(axis=-1, keepdims=True))
    return e / e.sum(axis=-1, keepdims=True)


def attention_head(q, k, v, n_valid=None):
    """One head of one sequence: softmax_rows(q k^T / sqrt(d)) v over that sequence's keys only.

    n_valid (padded layout only): keys m >= n_valid are padding and get score -inf
    ("padding-masked", north_star ¶1), i.e. probability exactly 0.
    """
    d = q.shape[-1]
    s = (q @ k.T) / np.sqrt(float(d))
    if n_valid is not None:
        s[:, n_valid:] = -np.inf
    return softmax_rows(s) @ v


def forward_sequence(w, desc, ids, n_valid=None):
    """Logits [n, NL] (float64) of ONE sequence of token ids (O1).

    n_valid: see attention_head; rows >= n_valid are then padding rows (values meaningless).
    """
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    H, A, eps = desc["hidden"], desc["heads"], desc["ln_eps"]
    dh = H // A
    n = len(ids)
    pos = np.arange(n)
    x = layer_norm(f8(np.asarray(w["E_w"])[ids]) + f8(np.asarray(w["E_p"])[pos]) + f8(w["E_t"]),
                   f8(w["g_e"]), f8(w["b_e"]), eps)
    for lw in w["layers"]:
        qkv = x @ f8(lw["W_qkv"]).T + f8(lw["b_qkv"])
        q, k, v = qkv[:, :H], qkv[:, H:2 * H], qkv[:, 2 * H:]
        c = np.zeros((n, H))
        for a in range(A):
            sl = slice(a * dh, (a + 1) * dh)
            c[:, sl] = attention_head(q[:, sl], k[:, sl], v[:, sl], n_valid)
        x = layer_norm(x + c @ f8(lw["W_o"]).T + f8(lw["b_o"]), f8(lw["g_1"]), f8(lw["b_1"]), eps)
        f = gelu(x @ f8(lw["W_1"]).T + f8(lw["b_1f"]))
        x = layer_norm(x + f @ f8(lw["W_2"]).T + f8(lw["b_2f"]), f8(lw["g_2"]), f8(lw["b_2"]), eps)
    return x @ f8(w["W_c"]).T + f8(w["b_c"])


def weights_f64(w):
    """Same parameter values as float64 arrays (embedding tables stay as given: they are
    only gathered).  Saves re-converting the matrices for every sequence; no arithmetic."""
    out = {k: (v if k in ("E_w", "E_p", "layers") else np.asarray(v, np.float64)) for k, v in w.items()}
    out["layers"] = [{k: np.asarray(v, np.float64) for k, v in lw.items()} for lw in w["layers"]]
    return out


def forward_packed(w, desc, token_ids, cu_seqlens, seq_subset=None):
    """Logits [T, NL] float64 for a packed batch; rows of sequences not in seq_subset are NaN."""
    w = weights_f64(w)
    token_ids = np.asarray(token_ids)
    cu = np.asarray(cu_seqlens)
    out = np.full((token_ids.shape[0], desc["num_labels"]), np.nan)
    seqs = range(len(cu) - 1) if seq_subset is None else seq_subset
    for i in seqs:
        a, b = int(cu[i]), int(cu[i + 1])
        if b > a:
            out[a:b] = forward_sequence(w, desc, token_ids[a:b])
    return out


def forward_padded(w, desc, ids_padded, lengths):
    """Padded [B, Lmax] layout: every row is run at full width Lmax with the padding keys
    masked by length; logits of padding rows are returned as NaN."""
    w = weights_f64(w)
    B, Lmax = ids_padded.shape
    out = np.full((B, Lmax, desc["num_labels"]), np.nan)
    for i in range(B):
        n = int(lengths[i])
        if n:
            out[i, :n] = forward_sequence(w, desc, ids_padded[i], n_valid=n)[:n]
    return out


def argmax_labels(logits):
    """O2: label_j = min{c : logits_j[c] = max_c' logits_j[c']} (ties -> lowest index)."""
    logits = np.asarray(logits)
    labels = np.zeros(logits.shape[0], np.int32)
    for j in range(logits.shape[0]):
        best = 0
        for c in range(1, logits.shape[1]):
            if logits[j, c] > logits[j, best]:
                best = c
        labels[j] = best
    return labels


def top2_margin(logits):
    """Oracle top-1 minus top-2 logit per token (for the label-agreement rule of north_star)."""
    s = np.sort(np.asarray(logits), axis=1)
    return s[:, -1] - s[:, -2]
