"""NEXT-2: the schema-aware direct-field path.  PAPER.md L57 (`anonymization_config`: fields named by the
schema are pseudonymized with a fixed type, NER is skipped) and L111 (that path is 46.9x faster: no encoder).  Here the
caller supplies the field spans (record, char_start, char_end) with a fixed type; the path is
anon_gather_spans -> anon_pseudonymize -> anon_splice_records, no encoder kernel anywhere; the oracle is
decode.gather_spans + crypto.Cache.pseudonymize + decode.splice_records.  Bit-exact."""
import numpy as np
import pytest

from harness import gen

pytestmark = pytest.mark.gpu
KEY = bytes((11 * i + 5) & 255 for i in range(32))


@pytest.mark.parametrize("fixed_type", [2, None])
def test_field_spans_gather_pseudonymize_splice(fixed_type):
    import torch
    import paper_2606_15650_b200 as P
    from oracle import crypto, decode
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    rec = gen.workload_stream(n_records=300, seed=gen.SEED_BASE + 3, n_pool=20000)        # configs[2]-shaped records
    spans = gen.field_spans(rec, 0 if fixed_type is None else fixed_type)
    S, R = len(spans), rec["rec_off"].size - 1
    assert S > 5000 and S == rec["n_entities"]
    text, ro = rec["text"], rec["rec_off"]
    ctx = P.Context(0, workspace_bytes=(64 << 20) + 64 * S + 2 * text.size)
    cache = P.Cache(ctx, 1 << 16, 4 << 20)
    d_text, d_ro = torch.from_numpy(text).to(dev), torch.from_numpy(ro).to(dev)
    d_spans = torch.from_numpy(spans).to(dev)
    span_bytes = torch.zeros(text.size + 16, dtype=torch.uint8, device=dev)
    span_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    span_type = torch.zeros(S, dtype=torch.uint8, device=dev)
    out = torch.zeros(S * 32, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(S, dtype=torch.uint8, device=dev)
    new_text = torch.zeros(text.size + S * 32, dtype=torch.uint8, device=dev)
    new_ro = torch.zeros(R + 1, dtype=torch.int64, device=dev)
    launches0 = None
    ctx.profile(True)
    P.anon_gather_spans(ctx, d_text, d_ro, d_spans, S, span_bytes, span_off, span_type)
    P.anon_pseudonymize(ctx, cache, span_bytes, span_off, None if fixed_type is None else span_type, KEY, 10, gen.TYPE_NAMES_6,
                        out, out_off, hit)
    P.anon_splice_records(ctx, d_text, d_ro, d_spans, S, out, out_off, new_text, new_ro)
    assert ctx.sync() == 0
    prof, launches = ctx.profile_read()
    ctx.profile(False)
    assert launches > 0 and all(prof[k][2] == 0 for k in ("gemm_qkv", "attention", "row", "gemm_out", "gemm_ffn1", "gemm_ffn2"))
    got_ro = new_ro.cpu().numpy()
    got_text = new_text.cpu().numpy()[:got_ro[R]]
    oo = out_off.cpu().numpy()
    got_tok, got_hit = out.cpu().numpy()[:oo[S]], hit.cpu().numpy()
    st = cache.stats()
    cache.close(); ctx.close()
    sp_list = [tuple(int(v) for v in s) for s in spans]
    sb, so = decode.gather_spans(text, ro, sp_list)
    assert np.array_equal(span_off.cpu().numpy(), so) and np.array_equal(span_bytes.cpu().numpy()[:so[-1]], sb)
    oc = crypto.Cache(1 << 16)
    types = None if fixed_type is None else spans[:, 3].astype(np.uint8)
    want = oc.pseudonymize(sb, so, types, KEY, 10, gen.TYPE_NAMES_6)
    oc.close()
    assert np.array_equal(oo, want["out_offsets"]) and np.array_equal(got_tok, want["out_tokens"])
    assert np.array_equal(got_hit, want["hit"]) and st["n_hits"] == int(want["hit"].sum()) > 0
    want_text, want_ro = decode.splice_records(text, ro, sp_list, want["out_tokens"], want["out_offsets"])
    assert np.array_equal(got_ro, want_ro) and np.array_equal(got_text, want_text)
    name = gen.TYPE_NAMES_6[0 if fixed_type is None else fixed_type]
    assert got_text.tobytes().count(("[" + name + "_").encode()) == S
