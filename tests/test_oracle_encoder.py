"""Pins for oracle/encoder.py -- CPU only.  Each test is chosen so a plausible slip
(dropped term, wrong sign/index, transposed operand) fails at least one of them."""
import math

import numpy as np
import torch
import torch.nn.functional as F

from harness import gen
from oracle import encoder

DESC = dict(layers=2, hidden=16, heads=2, ffn=24, vocab=50, num_labels=5, max_pos=32, ln_eps=1e-5, dtype=0)


def _w(desc=DESC, seed=1, scale=6.0):
    w = gen.make_weights(desc, seed)
    # scale the matrices up so attention is far from uniform and every term matters
    for lw in w["layers"]:
        for k in ("W_qkv", "W_o", "W_1", "W_2"):
            lw[k] = lw[k] * scale * 5
    w["E_w"] *= scale * 8
    w["E_p"] *= scale * 8
    return w


def test_attention_bruteforce_triple_loop():
    g = np.random.default_rng(0)
    n, d = 7, 4
    q, k, v = g.standard_normal((3, n, d))
    got = encoder.attention_head(q, k, v)
    for j in range(n):
        s = [sum(q[j][t] * k[m][t] for t in range(d)) / 2.0 for m in range(n)]   # sqrt(4) = 2
        mx = max(s)
        e = [math.exp(x - mx) for x in s]
        z = sum(e)
        for t in range(d):
            want = sum(e[m] / z * v[m][t] for m in range(n))
            assert abs(got[j][t] - want) < 1e-12


def test_attention_closed_forms():
    g = np.random.default_rng(1)
    q, k, v = g.standard_normal((3, 6, 8))
    p = encoder.softmax_rows(q @ k.T / math.sqrt(8))
    assert np.allclose(p.sum(1), 1.0, atol=1e-12) and (p > 0).all()
    # zero queries -> uniform mean of V;  n = 1 -> c = v
    assert np.allclose(encoder.attention_head(np.zeros_like(q), k, v), np.tile(v.mean(0), (6, 1)))
    assert np.allclose(encoder.attention_head(q[:1], k[:1], v[:1]), v[:1])
    # masked keys get probability exactly zero
    a = encoder.attention_head(q, k, v, n_valid=4)
    assert np.allclose(a, encoder.attention_head(q, k[:4], v[:4]))


def test_layernorm_and_gelu_closed_forms():
    g = np.random.default_rng(2)
    z = g.standard_normal((5, 64)) * 3 + 1
    one, zero = np.ones(64), np.zeros(64)
    y = encoder.layer_norm(z, one, zero, 1e-5)
    assert np.allclose(y.mean(1), 0, atol=1e-12)
    var = z.var(1)
    assert np.allclose(y.var(1), var / (var + 1e-5), atol=1e-12)
    assert np.allclose(encoder.layer_norm(z + 7.5, one, zero, 1e-5), y, atol=1e-10)      # shift invariance
    gam, bet = g.standard_normal(64), g.standard_normal(64)
    assert np.allclose(encoder.layer_norm(z, gam, bet, 1e-5), y * gam + bet)
    x = np.linspace(-6, 6, 101)
    assert encoder.gelu(np.array([0.0]))[0] == 0.0
    assert np.allclose(encoder.gelu(x) - encoder.gelu(-x), x, atol=1e-12)                # Phi(z)+Phi(-z)=1
    assert abs(encoder.gelu(np.array([1.0]))[0] - 0.5 * (1 + math.erf(1 / math.sqrt(2)))) < 1e-15
    # the tanh approximation is NOT what we compute (reading S5)
    tanh_form = 0.5 * x * (1 + np.tanh(math.sqrt(2 / math.pi) * (x + 0.044715 * x ** 3)))
    assert np.abs(encoder.gelu(x) - tanh_form).max() > 1e-4


def test_padded_equals_packed_and_permutation_invariance():
    w = _w()
    ids, cu, padded, lengths = gen.tokens_uniform(6, 3, 12, DESC["vocab"], 5)
    packed = encoder.forward_packed(w, DESC, ids, cu)
    pad = encoder.forward_padded(w, DESC, padded, lengths)
    for i in range(6):
        a, b = cu[i], cu[i + 1]
        assert np.allclose(pad[i, :lengths[i]], packed[a:b], atol=1e-12, rtol=0)
    # any permutation of the sequences in the pack gives the same per-sequence logits (bit for bit)
    perm = [3, 0, 5, 1, 4, 2]
    ids2 = np.concatenate([ids[cu[i]:cu[i + 1]] for i in perm])
    cu2 = np.concatenate([[0], np.cumsum([lengths[i] for i in perm])])
    packed2 = encoder.forward_packed(w, DESC, ids2, cu2)
    for j, i in enumerate(perm):
        assert np.array_equal(packed2[cu2[j]:cu2[j + 1]], packed[cu[i]:cu[i + 1]])
    # sequences are independent: a sequence alone gives the same rows
    alone = encoder.forward_packed(w, DESC, ids[cu[2]:cu[3]], np.array([0, lengths[2]]))
    assert np.array_equal(alone, packed[cu[2]:cu[3]])


def test_token_permutation_with_zero_positions_and_L0():
    w = _w()
    w["E_p"] = np.zeros_like(w["E_p"])
    ids = np.array([7, 9, 11, 30, 22, 41, 8])
    base = encoder.forward_sequence(w, DESC, ids)
    perm = np.array([4, 2, 6, 0, 1, 5, 3])
    assert np.allclose(encoder.forward_sequence(w, DESC, ids[perm]), base[perm], atol=1e-11)
    # with positions back on, the permutation changes the logits (positions are really added)
    w2 = _w()
    assert np.abs(encoder.forward_sequence(w2, DESC, ids[perm]) - encoder.forward_sequence(w2, DESC, ids)[perm]).max() > 1e-3
    # L = 0 reduces to W_c LN(emb) + b_c
    w0 = dict(w2, layers=[])
    emb = w2["E_w"][ids].astype(np.float64) + w2["E_p"][np.arange(7)] + w2["E_t"]
    mu = emb.mean(1, keepdims=True)
    ln = (emb - mu) / np.sqrt(((emb - mu) ** 2).mean(1, keepdims=True) + 1e-5) * w2["g_e"] + w2["b_e"]
    assert np.allclose(encoder.forward_sequence(w0, dict(DESC, layers=0), ids), ln @ w2["W_c"].T.astype(np.float64) + w2["b_c"], atol=1e-12)


def _torch_forward(w, desc, ids):
    """float64 composition of torch library primitives (test-only cross-check)."""
    t = lambda a: torch.tensor(np.asarray(a), dtype=torch.float64)
    H, A = desc["hidden"], desc["heads"]
    n = len(ids)
    x = t(w["E_w"])[torch.tensor(ids)] + t(w["E_p"])[:n] + t(w["E_t"])
    x = F.layer_norm(x, (H,), t(w["g_e"]), t(w["b_e"]), desc["ln_eps"])
    for lw in w["layers"]:
        qkv = F.linear(x, t(lw["W_qkv"]), t(lw["b_qkv"]))
        q, k, v = [z.reshape(n, A, H // A).transpose(0, 1) for z in qkv.split(H, dim=1)]
        c = F.scaled_dot_product_attention(q, k, v).transpose(0, 1).reshape(n, H)
        x = F.layer_norm(x + F.linear(c, t(lw["W_o"]), t(lw["b_o"])), (H,), t(lw["g_1"]), t(lw["b_1"]), desc["ln_eps"])
        f = F.gelu(F.linear(x, t(lw["W_1"]), t(lw["b_1f"])))
        x = F.layer_norm(x + F.linear(f, t(lw["W_2"]), t(lw["b_2f"])), (H,), t(lw["g_2"]), t(lw["b_2"]), desc["ln_eps"])
    return F.linear(x, t(w["W_c"]), t(w["b_c"])).numpy()


def test_against_torch_float64_library_composition():
    for desc, seed in [(DESC, 3), (dict(gen.DESCS["tiny"]), 4)]:
        w = _w(desc, seed, scale=3.0)
        ids = np.random.default_rng(seed).integers(5, desc["vocab"], 19)
        got = encoder.forward_sequence(w, desc, ids)
        want = _torch_forward(w, desc, ids)
        assert np.abs(got - want).max() < 1e-9 * max(1.0, np.abs(want).max())
        assert np.abs(want).max() > 1e-2           # the comparison is not vacuous


def test_argmax_ties_lowest_index():
    lg = np.array([[0.0, 1.0, 1.0, 0.5], [2.0, 2.0, 2.0, 2.0], [-1.0, -3.0, -0.5, -0.5]])
    assert encoder.argmax_labels(lg).tolist() == [1, 0, 2]
    assert np.allclose(encoder.top2_margin(lg), [0.0, 0.0, 0.0])
    assert np.allclose(encoder.top2_margin(np.array([[0.1, 0.9, 0.3]])), [0.6])
