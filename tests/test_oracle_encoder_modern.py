"""Pins of oracle/encoder_modern.py (NEXT-3, reading D20): each checks the oracle against something other than itself."""
import numpy as np

from harness import gen
from oracle import encoder_modern as em


def test_rope_against_complex_rotation_and_hand_value():
    rng = np.random.default_rng(1)
    n, d, theta = 9, 8, 10000.0
    x = rng.standard_normal((n, d))
    pos = np.arange(n) + 3
    got = em.rope(x, pos, theta)
    # independent formulation: the pair (x_i, x_{i+d/2}) is the complex number x_i + j x_{i+d/2}, rotated by e^{j pos theta^(-2i/d)}
    z = x[:, :d // 2] + 1j * x[:, d // 2:]
    rot = np.exp(1j * pos[:, None] * theta ** (-2.0 * np.arange(d // 2) / d)[None, :])
    want = z * rot
    assert np.allclose(got[:, :d // 2], want.real, atol=1e-13) and np.allclose(got[:, d // 2:], want.imag, atol=1e-13)
    # hand value: d = 2 has one pair with frequency 1; position 1 rotates (1, 0) by one radian
    assert np.allclose(em.rope(np.array([[1.0, 0.0]]), [1], 12345.0), [[np.cos(1.0), np.sin(1.0)]], atol=1e-15)
    # second pair of d = 4 turns at theta^(-1/2): position 4, theta 16 -> one radian as well
    assert np.allclose(em.rope(np.array([[0.0, 1.0, 0.0, 0.0]]), [4], 16.0), [[0.0, np.cos(1.0), 0.0, np.sin(1.0)]], atol=1e-15)
    # position 0 is the identity; rotations keep the norm of every pair; dot products depend on the position difference only
    assert np.array_equal(em.rope(x, np.zeros(n), theta), x)
    assert np.allclose((got ** 2).sum(1), (x ** 2).sum(1))
    q, k = rng.standard_normal((1, d)), rng.standard_normal((1, d))
    a = em.rope(q, [5], theta) @ em.rope(k, [2], theta).T
    b = em.rope(q, [105], theta) @ em.rope(k, [102], theta).T
    assert np.allclose(a, b, atol=1e-12)


def test_local_attention_against_triple_loop():
    rng = np.random.default_rng(2)
    n, d, window = 11, 4, 6
    q, k, v = (rng.standard_normal((n, d)) for _ in range(3))
    got = em.attention_head(q, k, v, window)
    want = np.zeros((n, d))
    for i in range(n):
        num, den = np.zeros(d), 0.0
        for j in range(n):
            if abs(i - j) <= window // 2:
                e = np.exp(sum(q[i, t] * k[j, t] for t in range(d)) / 2.0)
                num += e * v[j]
                den += e
        want[i] = num / den
    assert np.allclose(got, want, atol=1e-12)
    # a window that covers the sequence is global attention; window 0 leaves only the token itself: c = v
    assert np.allclose(em.attention_head(q, k, v, 2 * n), em.attention_head(q, k, v, None), atol=1e-15)
    assert np.allclose(em.attention_head(q, k, v, 0), v, atol=1e-15)


def test_forward_special_cases_and_position_offset():
    d = dict(gen.DESCS["tiny_modern"], layers=4, vocab=600)
    w = gen.make_weights_modern(d, 5)
    ids = gen.rng(7).integers(5, 600, 150)                      # longer than the window: local layers really mask
    base = em.forward_sequence(w, d, ids)
    # RoPE is the only position information: shifting every position changes nothing
    assert np.allclose(em.forward_sequence(w, d, ids, pos0=37), base, atol=1e-9)
    # ... but the order of the tokens matters (a reversed sequence is not the reversed output)
    assert not np.allclose(em.forward_sequence(w, d, ids[::-1])[::-1], base, atol=1e-6)
    # the local window matters: with a window wider than the sequence the logits differ
    assert not np.allclose(em.forward_sequence(w, dict(d, local_window=1000), ids), base, atol=1e-6)
    # ... and with global_every = 1 (all layers global) the window is never used
    dg = dict(d, global_every=1, rope_theta_local=d["rope_theta_global"])
    assert np.allclose(em.forward_sequence(w, dg, ids), em.forward_sequence(w, dict(dg, local_window=2), ids), atol=1e-12)
    # L = 0: logits = LN(LN(E_w[ids]; g_e); g_f) W_c^T + b_c, written out with numpy primitives
    w0 = dict(w, layers=[])
    e = np.asarray(w["E_w"], np.float64)[ids]
    z = (e - e.mean(1, keepdims=True)) / np.sqrt(e.var(1, keepdims=True) + d["ln_eps"]) * w["g_e"]
    z = (z - z.mean(1, keepdims=True)) / np.sqrt(z.var(1, keepdims=True) + d["ln_eps"]) * w["g_f"]
    assert np.allclose(em.forward_sequence(w0, d, ids), z @ np.asarray(w["W_c"], np.float64).T + w["b_c"], atol=1e-10)
    # packed == one sequence at a time
    cu = np.array([0, 40, 40, 150])
    got = em.forward_packed(w, d, ids, cu)
    assert np.allclose(got[:40], em.forward_sequence(w, d, ids[:40]), atol=1e-12)
    assert np.allclose(got[40:], em.forward_sequence(w, d, ids[40:]), atol=1e-12)


def test_geglu_special_cases():
    # gate = 1 gives gelu(a); gelu(a) -> a for large a; gelu(a) - gelu(-a) = a
    a = np.linspace(-6, 6, 25)
    assert np.allclose(em.gelu(a) - em.gelu(-a), a, atol=1e-14)
    assert abs(em.gelu(np.array([12.0]))[0] - 12.0) < 1e-12 and em.gelu(np.array([0.0]))[0] == 0.0


def test_forward_against_torch_library_composition():
    """The same network assembled from torch float64 library primitives (layer_norm, scaled_dot_product_attention with a
    boolean band mask, gelu, complex polar rotation)."""
    import torch
    import torch.nn.functional as Fn
    d = dict(gen.DESCS["tiny_modern"], layers=3, vocab=400, local_window=16)
    w = gen.make_weights_modern(d, 9)
    ids = gen.rng(3).integers(5, 400, 45)
    H, A, F = d["hidden"], d["heads"], d["ffn"]
    dh, n = H // A, len(ids)
    t = lambda a: torch.tensor(np.asarray(a, np.float64))
    ln = lambda z, g: Fn.layer_norm(z, (H,), t(g), None, d["ln_eps"])
    x = ln(t(w["E_w"])[torch.tensor(ids)], w["g_e"])
    pos = torch.arange(n, dtype=torch.float64)
    idx = torch.arange(n)
    band = (idx[:, None] - idx[None, :]).abs() <= d["local_window"] // 2
    for l, lw in enumerate(w["layers"]):
        glob = l % d["global_every"] == 0
        theta = d["rope_theta_global"] if glob else d["rope_theta_local"]
        qkv = ln(x, lw["g_a"]) @ t(lw["W_qkv"]).T
        q, k, v = (qkv[:, i * H:(i + 1) * H].reshape(n, A, dh).transpose(0, 1) for i in range(3))     # [A, n, dh]
        ang = pos[:, None] * theta ** (-2.0 * torch.arange(dh // 2, dtype=torch.float64) / dh)[None, :]
        rot = torch.polar(torch.ones_like(ang), ang)                                                   # e^{j ang}

        def rope(z):
            zc = torch.complex(z[..., :dh // 2], z[..., dh // 2:]) * rot
            return torch.cat([zc.real, zc.imag], dim=-1)
        c = Fn.scaled_dot_product_attention(rope(q), rope(k), v, attn_mask=None if glob else band)
        x = x + c.transpose(0, 1).reshape(n, H) @ t(lw["W_o"]).T
        u = ln(x, lw["g_m"]) @ t(lw["W_i"]).T
        x = x + (Fn.gelu(u[:, :F]) * u[:, F:]) @ t(lw["W_2"]).T
    want = (ln(x, w["g_f"]) @ t(w["W_c"]).T + t(w["b_c"])).numpy()
    assert np.allclose(em.forward_sequence(w, d, ids), want, atol=1e-9)
