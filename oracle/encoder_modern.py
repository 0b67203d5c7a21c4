"""TEST INFRASTRUCTURE -- fp64 oracle of the ModernBERT-shaped encoder variant.

What it follows.  PAPER.md L43 names the second NER model only by name ("SecureModernBERT-NER"; L95 reports its
accuracy); SURVEY.md §8(f) NEXT-3 lists what distinguishes the shape: "pre-LN, RoPE, GeGLU, alternating local/global
attention, no biases".  The paper prints no formulas, so the forward below is this build's reading D20,
written step by step:

    x      = LN(E_w[ids]; g_e)                                   embedding norm, no position table (RoPE instead)
    layer l = 0 .. L-1:
      h    = LN(x; g_a)                                          pre-norm (every layer, also l = 0)
      qkv  = h W_qkv^T                                           no bias
      q, k = RoPE(q, pos; theta_l), RoPE(k, pos; theta_l)        per head, rotate-half pairing (i, i + d/2)
      s    = q k^T / sqrt(d);  s[i, j] = -inf where layer l is local and |i - j| > window / 2
      x    = x + (softmax_rows(s) v) W_o^T
      h    = LN(x; g_m)
      u    = h W_i^T;  a, g = u[:, :F], u[:, F:]                 GeGLU: act = gelu(a) * g, erf GELU
      x    = x + (gelu(a) * g) W_2^T
    logits = LN(x; g_f) W_c^T + b_c
    layer l is global iff l % global_every == 0 (theta_l = rope_theta_global), else local (rope_theta_local)
    LN(z; g) = (z - mean) / sqrt(var + eps) * g, biased variance, no bias term

float64 throughout; ``@``, ``np.cos`` / ``np.sin`` and ``scipy.special.erf`` are the only library steps; one sequence
and one head at a time.  Pins: tests/test_oracle_encoder_modern.py (RoPE against complex multiplication, hand value,
norm and relative-position properties; band mask against a triple loop; window >= 2n == global, window 0 => c = v;
GeGLU special cases; position-offset invariance of the whole forward; L = 0 closed form; torch float64 library
composition).
"""
import numpy as np
from scipy.special import erf


def layer_norm_nb(z, g, eps):
    """LN without bias: (z - mean) / sqrt(var + eps) * g, var biased."""
    mean = z.mean(axis=-1, keepdims=True)
    var = ((z - mean) ** 2).mean(axis=-1, keepdims=True)
    return (z - mean) / np.sqrt(var + eps) * g


def gelu(z):
    return 0.5 * z * (1.0 + erf(z / np.sqrt(2.0)))


def rope(x, pos, theta):
    """x [n, d] (one head), pos [n]: out[:, i] = x_i cos(a_i) - x_{i+d/2} sin(a_i), out[:, i+d/2] = x_{i+d/2} cos(a_i)
    + x_i sin(a_i), a_i = pos * theta^(-2i/d), i = 0 .. d/2 - 1."""
    n, d = x.shape
    half = d // 2
    inv_freq = theta ** (-2.0 * np.arange(half) / d)
    ang = np.asarray(pos, np.float64)[:, None] * inv_freq[None, :]
    c, s = np.cos(ang), np.sin(ang)
    x1, x2 = x[:, :half], x[:, half:]
    return np.concatenate([x1 * c - x2 * s, x2 * c + x1 * s], axis=1)


def attention_head(q, k, v, window=None):
    """softmax_rows(q k^T / sqrt(d)) v; window (local layers): key j is visible from query i iff |i - j| <= window / 2."""
    n, d = q.shape
    s = (q @ k.T) / np.sqrt(float(d))
    if window is not None:
        i = np.arange(n)
        s = np.where(np.abs(i[:, None] - i[None, :]) <= window // 2, s, -np.inf)
    e = np.exp(s - s.max(axis=-1, keepdims=True))
    return (e / e.sum(axis=-1, keepdims=True)) @ v


def layer_is_global(desc, l):
    return l % desc["global_every"] == 0


def forward_sequence(w, desc, ids, pos0=0):
    """Logits [n, NL] (float64) of ONE sequence.  pos0 shifts every position id (RoPE is relative: the result must not
    depend on it -- used by a pin)."""
    f8 = lambda a: np.asarray(a, dtype=np.float64)
    H, A, F, eps = desc["hidden"], desc["heads"], desc["ffn"], desc["ln_eps"]
    dh = H // A
    n = len(ids)
    pos = np.arange(n) + pos0
    x = layer_norm_nb(f8(np.asarray(w["E_w"])[ids]), f8(w["g_e"]), eps)
    for l, lw in enumerate(w["layers"]):
        glob = layer_is_global(desc, l)
        theta = desc["rope_theta_global"] if glob else desc["rope_theta_local"]
        h = layer_norm_nb(x, f8(lw["g_a"]), eps)
        qkv = h @ f8(lw["W_qkv"]).T
        q, k, v = qkv[:, :H], qkv[:, H:2 * H], qkv[:, 2 * H:]
        c = np.zeros((n, H))
        for a in range(A):
            sl = slice(a * dh, (a + 1) * dh)
            c[:, sl] = attention_head(rope(q[:, sl], pos, theta), rope(k[:, sl], pos, theta), v[:, sl],
                                      None if glob else desc["local_window"])
        x = x + c @ f8(lw["W_o"]).T
        h = layer_norm_nb(x, f8(lw["g_m"]), eps)
        u = h @ f8(lw["W_i"]).T
        x = x + (gelu(u[:, :F]) * u[:, F:]) @ f8(lw["W_2"]).T
    return layer_norm_nb(x, f8(w["g_f"]), eps) @ f8(w["W_c"]).T + f8(w["b_c"])


def forward_packed(w, desc, token_ids, cu_seqlens, seq_subset=None):
    """Logits [T, NL] float64 for a packed batch; rows of sequences not in seq_subset are NaN."""
    token_ids = np.asarray(token_ids)
    cu = np.asarray(cu_seqlens)
    out = np.full((token_ids.shape[0], desc["num_labels"]), np.nan)
    seqs = range(len(cu) - 1) if seq_subset is None else seq_subset
    for i in seqs:
        a, b = int(cu[i]), int(cu[i + 1])
        if b > a:
            out[a:b] = forward_sequence(w, desc, token_ids[a:b])
    return out
